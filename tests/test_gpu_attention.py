"""GPU parity of the fused variable-length attention step (S3d) alone, through the C ABI
(`fmx_debug_attention`), against the oracle's `attention` (fp64, per request, per head) on the
same bf16 inputs.  Both implementations are covered: the tcgen05/TMEM/TMA kernel (head_dim 64,
128) and the warp-level mma.sync kernel (head_dim 32 and the fallback switch).

Tolerance: the output is bf16 (rel. 2^-9) of a convex combination of v rows with P rounded to
bf16 before the PV product: |err| <= ~2^-8 * max|v| per element; the bar used is
max-abs <= 1.5e-2 * max|v| and per-row cosine >= 0.9995.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")
pytestmark = pytest.mark.gpu

from fmx_workloads import bf16_bits_to_f64, f32_to_bf16_bits  # noqa: E402
from oracle.vfm_forward import attention  # noqa: E402

MMA_SYNC, TCGEN05 = 1, 2


@pytest.fixture(scope="module")
def fmx():
    if not torch.cuda.is_available():
        pytest.fail("gpu-marked test needs a CUDA device; the product has no CPU fallback")
    import paper_2606_09643_b200 as pkg
    return pkg.Fmx(0)


def run_case(fmx, lengths, hq, hkv, dh, causal, impl, seed, q_scale=1.0, ramp=0.0):
    rng = np.random.default_rng(seed)
    N = int(np.sum(lengths))
    dq, dkv = hq * dh, hkv * dh
    x = rng.standard_normal((N, dq + 2 * dkv)).astype(np.float32)
    x[:, :dq] *= q_scale
    if ramp:
        # key norms grow along each request, so the row maximum keeps rising: forces the O rescale path
        off = 0
        for n in lengths:
            x[off:off + n, dq:dq + dkv] *= (1.0 + ramp * np.arange(n, dtype=np.float32) / n)[:, None]
            off += n
    bits = f32_to_bf16_bits(x)
    qkv = torch.from_numpy(bits.view(np.int16)).cuda()
    out = torch.full((N, dq), float("nan"), dtype=torch.bfloat16, device="cuda")
    cu = np.concatenate([[0], np.cumsum(lengths)]).astype(np.int32)
    fmx.debug_attention(qkv.data_ptr(), out.data_ptr(), cu, hq, hkv, dh, causal, impl)
    torch.cuda.synchronize()
    got = out.float().cpu().numpy().astype(np.float64)
    xf = bf16_bits_to_f64(bits)
    worst_abs, worst_cos = 0.0, 1.0
    for i in range(len(lengths)):
        r = xf[cu[i]:cu[i + 1]]
        ref = attention(r[:, :dq], r[:, dq:dq + dkv], r[:, dq + dkv:], hq, hkv, dh, causal)
        g = got[cu[i]:cu[i + 1]]
        assert np.isfinite(g).all(), f"request {i}: non-finite attention output"
        worst_abs = max(worst_abs, float(np.abs(g - ref).max()))
        cos = np.sum(g * ref, axis=1) / (np.linalg.norm(g, axis=1) * np.linalg.norm(ref, axis=1) + 1e-300)
        worst_cos = min(worst_cos, float(cos.min()))
    vmax = float(np.abs(xf[:, dq + dkv:]).max())
    assert worst_abs <= 1.5e-2 * vmax, f"max-abs {worst_abs:.3e} > 1.5e-2 * max|v| {vmax:.2f}"
    assert worst_cos >= 0.9995, f"min row cosine {worst_cos:.6f}"


CASES = [
    # lengths,                        hq, hkv, dh, causal
    ([64, 64, 64],                    4, 4, 64, 0),      # cfg2-like: one KV tile, half-empty q-tile
    ([257, 257],                      3, 3, 64, 0),      # cfg3-like: 3 q-tiles, ragged last KV tile (1 key)
    ([1, 2, 63, 65, 127, 129, 300],   2, 2, 64, 0),      # ragged everything
    ([1, 64, 200, 1024],              12, 2, 128, 1),    # cfg4-like: GQA 6:1, causal, max length
    ([130, 511, 77],                  4, 1, 128, 1),
    ([256, 128, 384],                 2, 2, 128, 0),     # exact multiples of the tiles
    ([640],                           2, 1, 64, 1),
]


MORE_CASES = [
    ([17] * 40 + [257] * 9,           16, 16, 64, 0),    # many short requests next to cfg3-like ones: CTAs that exit at once
    ([130, 66, 80, 129, 193, 16, 15], 2, 2, 128, 0),     # head_dim 128 with last KV tiles of 2, 2, 16, 1, 1 keys (N = 16 tail MMA)
    ([200, 72],                       12, 2, 128, 1),    # causal tail: keys 192..199 visible to the last rows only
    ([513, 1000],                     4, 2, 64, 1),      # head_dim 64 causal, 9 and 16 KV tiles (single S buffer)
]


@pytest.mark.parametrize("lengths,hq,hkv,dh,causal", CASES + MORE_CASES)
def test_tcgen05_attention_matches_oracle(fmx, lengths, hq, hkv, dh, causal):
    run_case(fmx, lengths, hq, hkv, dh, causal, TCGEN05, seed=len(lengths) * 131 + dh)


@pytest.mark.parametrize("lengths,hq,hkv,dh,causal", [
    ([300, 700], 2, 2, 64, 0),
    ([1024, 90], 6, 1, 128, 1),
    ([257, 130], 2, 2, 128, 0),                          # rescale with a fast 16-key tail tile running ahead (double-buffered S)
])
def test_tcgen05_attention_large_scores_rescale_path(fmx, lengths, hq, hkv, dh, causal):
    """Scores of magnitude ~10^2 in the log2 domain with the largest ones late in the sequence: the
    lazily updated reference maximum must move (more than once) and O in TMEM must be rescaled."""
    run_case(fmx, lengths, hq, hkv, dh, causal, TCGEN05, seed=7, q_scale=6.0, ramp=3.0)


@pytest.mark.parametrize("lengths,hq,hkv,dh,causal", [
    ([64, 64, 64], 4, 4, 32, 0),                          # cfg1's head_dim
    ([1, 64, 200, 333], 12, 2, 128, 1),
    ([257, 100], 3, 3, 64, 0),
])
def test_mma_sync_attention_matches_oracle(fmx, lengths, hq, hkv, dh, causal):
    run_case(fmx, lengths, hq, hkv, dh, causal, MMA_SYNC, seed=5)


@pytest.mark.parametrize("lengths,hq,hkv,dh,causal", [
    ([64] * 40, 16, 16, 64, 0),                           # cfg2 / cfg5 shape; more items than lanes: the rings wrap
    ([1, 7, 16, 17, 33, 48, 63, 64, 5], 4, 4, 64, 0),     # ragged, warps with no query, single-token request
    ([64, 31, 64, 2, 40] * 30, 12, 2, 64, 1),             # GQA 6:1 (a head pair shares / splits KV heads), causal
    ([64, 20, 64, 1], 4, 2, 32, 1),                       # head_dim 32: mma.sync path only
    ([50, 64, 3], 6, 1, 128, 1),                          # head_dim 128: mma.sync path only
    ([64, 64, 9], 3, 3, 64, 0),                           # odd head count: no head pairs
])
def test_short_sequence_attention_matches_oracle(fmx, lengths, hq, hkv, dh, causal):
    """Batches whose requests all have <= 64 tokens: (a) the tcgen05 head-pair kernel (two heads of a request as one
    block-diagonal 128-row MMA; default under AUTO when head_dim is 64 and the head count even), (b) the pipelined
    single-tile mma.sync kernel, (c) the generic kernel."""
    AUTO = 0
    for impl, short in ((AUTO, 2), (MMA_SYNC, 1), (MMA_SYNC, 0)):
        fmx.set_option("attn_short", short)
        try:
            run_case(fmx, lengths, hq, hkv, dh, causal, impl, seed=11 + dh)
        finally:
            fmx.set_option("attn_short", 2)
