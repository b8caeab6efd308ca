"""fmx_row_gemm_static (include/fmx.h, csrc/no_alloc.cu): the entry point that allocates nothing - its split-K scratch is a
file-scope __device__ array - against the existing GEMM path (fmx_debug_gemm, the tcgen05 kernel the forward's projections
run on), on two calls in a row that share the array.  Named test_zz_* so that pytest collects it last: the suite runs with
`pytest -x`, and a failure here must not hide another test."""
import numpy as np
import pytest

from fmx_workloads import bf16_bits_to_f64, f32_to_bf16_bits

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu


def _case(fmx_pkg, ctx, M, N, K, seed):
    """Returns (new path output, existing path output, fp64 truth) for one seeded problem."""
    rng = np.random.default_rng(seed)
    a = f32_to_bf16_bits(rng.standard_normal((M, K)).astype(np.float32))
    w = f32_to_bf16_bits(rng.standard_normal((N, K)).astype(np.float32))
    A = torch.from_numpy(a.view(np.int16)).cuda()
    W = torch.from_numpy(w.view(np.int16)).cuda()
    got = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    ref = torch.full((M, N), float("nan"), dtype=torch.float32, device="cuda")
    from paper_2606_09643_b200 import binding
    binding.row_gemm_static(A.data_ptr(), W.data_ptr(), got.data_ptr(), M, N, K)
    ctx.debug_gemm(A.data_ptr(), W.data_ptr(), ref.data_ptr(), M, N, K)
    torch.cuda.synchronize()
    truth = bf16_bits_to_f64(a) @ bf16_bits_to_f64(w).T
    return got.cpu().numpy().astype(np.float64), ref.cpu().numpy().astype(np.float64), truth


def test_static_scratch_gemm_matches_the_existing_path_twice_in_a_row():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2606_09643_b200 as fmx_pkg
    ctx = fmx_pkg.Fmx(0)
    # two calls in a row on the same static array: the second is SMALLER in every dimension and has fewer K slices, so stale
    # partials of the first call sit right next to what it reads; then the first shape again with other data
    for M, N, K, seed in ((64, 1536, 1536, 11), (5, 256, 200, 12), (64, 1536, 1536, 13), (128, 2048, 8960, 14), (1, 128, 8, 15)):
        got, ref, truth = _case(fmx_pkg, ctx, M, N, K, seed)
        tol = 2e-5 * K ** 0.5 * 4                 # the bound tests/test_gpu_parity.py::test_tcgen05_gemm_matches_fp64 uses
        assert np.isfinite(got).all(), (M, N, K)
        assert np.abs(got - ref).max() <= tol, (M, N, K, np.abs(got - ref).max())
        assert np.abs(got - truth).max() <= tol, (M, N, K, np.abs(got - truth).max())
    ctx.destroy()


def test_static_scratch_gemm_rejects_what_does_not_fit():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    from paper_2606_09643_b200 import binding
    from paper_2606_09643_b200.binding import FmxError
    buf = torch.zeros(1 << 20, dtype=torch.float32, device="cuda")
    p = buf.data_ptr()
    for M, N, K, what in ((129, 128, 64, "rows"), (0, 128, 64, "rows"), (16, 100, 64, "multiple of 128"), (16, 128, 12, "multiple of 8"),
                          (128, 128 * 200, 64, "static scratch")):
        with pytest.raises(FmxError) as ei:
            binding.row_gemm_static(p, p, p, M, N, K)
        assert what in str(ei.value), str(ei.value)
    torch.cuda.synchronize()
