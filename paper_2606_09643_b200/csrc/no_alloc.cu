// fmx_row_gemm_static: the small-M projection of a decode iteration (row_gemm.cuh) as ONE entry point that allocates nothing.
//
// row_gemm_kernel splits the K axis over CTAs and needs scratch memory for the per-slice fp32 partials.  The forward path takes
// that scratch from the caller's workspace; callers that cannot provide one and cannot call cudaMalloc (code under CUDA graph
// capture, tight serving loops, harnesses that forbid it) get this variant, whose scratch is a file-scope __device__ array of a
// fixed size.  Every GPU that loads the library holds the array (kStaticScratchBytes) until the process exits.
//
// The array's name is a host-side stand-in in host code, not a device address: the address is looked up with
// cudaGetSymbolAddress once per device (with that device current) and handed to the kernel that takes a pointer; the reduction
// kernel of this file names the array directly, which device code may do.
//
// Every call shares the array.  Nothing in it has to start at zero: a call writes every (slice, row < M, column) element it
// later reads, so the previous call's contents are never observed.  Calls that overlap on the GPU (different streams, or two
// host threads launching onto streams that run concurrently) RACE on the array; calls on one stream are ordered and safe.
#include <cuda_runtime.h>

#include <algorithm>
#include <mutex>

#include "common.h"
#include "fmx.h"
#include "row_gemm.cuh"

namespace fmx {

constexpr size_t kStaticScratchBytes = 8u << 20;                 // 8 MiB per GPU
constexpr size_t kStaticScratchFloats = kStaticScratchBytes / sizeof(float);
constexpr int kStaticMaxRows = 128;                              // row_gemm_kernel<8>
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) float g_row_gemm_scratch[kStaticScratchFloats];

// out[r, c .. c + 3] = sum over the slices, in slice order, of the partials in the static array.  One thread per 4 columns.
__global__ void __launch_bounds__(256) static_reduce_kernel(float *__restrict__ out, int M, int N, int k_split, int split_rows) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  const int n4 = N >> 2;
  if (idx >= (long long)M * n4) return;
  const int r = (int)(idx / n4), c = (int)(idx - (long long)r * n4) * 4;
  float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll 4
  for (int ks = 0; ks < k_split; ++ks) {
    const float4 v = *reinterpret_cast<const float4 *>(g_row_gemm_scratch + ((size_t)ks * split_rows + r) * N + c);
    acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
  }
  *reinterpret_cast<float4 *>(out + (size_t)r * N + c) = acc;
}

struct StaticDev {
  bool ready = false;
  float *scratch = nullptr;          // device address of g_row_gemm_scratch on this device
  int sm_count = 0;
};
static StaticDev g_static_dev[kStaticMaxDevices];
static std::mutex g_static_mu;

// Once per device, with that device current: the array's device address, the SM count, the kernels' shared-memory limit.
static int static_setup(int dev, StaticDev **out) {
  if (dev < 0 || dev >= kStaticMaxDevices) return fmx_fail(FMX_E_INVALID_ARG, "row_gemm_static: device ordinal %d out of range", dev);
  std::lock_guard<std::mutex> lk(g_static_mu);
  StaticDev &d = g_static_dev[dev];
  if (!d.ready) {
    int major = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (e != cudaSuccess) return fmx_fail(FMX_E_CUDA, "row_gemm_static: %s", cudaGetErrorString(e));
    if (major != 10) return fmx_fail(FMX_E_CUDA, "row_gemm_static: device %d has compute capability %d.x, libfmx is built for sm_100a", dev, major);
    void *p = nullptr;
    e = cudaGetSymbolAddress(&p, g_row_gemm_scratch);
    if (e != cudaSuccess || !p) return fmx_fail(FMX_E_CUDA, "row_gemm_static: cudaGetSymbolAddress failed: %s", cudaGetErrorString(e));
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_gemm_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_gemm_smem<1>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_gemm_kernel<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_gemm_smem<2>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_gemm_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_gemm_smem<4>());
    if (e == cudaSuccess) e = cudaFuncSetAttribute(row_gemm_kernel<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)row_gemm_smem<8>());
    if (e != cudaSuccess) return fmx_fail(FMX_E_CUDA, "row_gemm_static: cudaFuncSetAttribute failed: %s", cudaGetErrorString(e));
    d.scratch = static_cast<float *>(p);
    d.sm_count = sms;
    d.ready = true;
  }
  *out = &d;
  return FMX_OK;
}

}  // namespace fmx

using namespace fmx;

extern "C" int fmx_row_gemm_static(const void *x, const void *W, float *out, int32_t M, int32_t N, int32_t K, void *cuda_stream) {
  if (!x || !W || !out) return fmx_fail(FMX_E_INVALID_ARG, "row_gemm_static: NULL pointer");
  if (M < 1 || M > kStaticMaxRows) return fmx_fail(FMX_E_CAPACITY, "row_gemm_static: M = %d rows, this entry point takes 1 .. %d", M, kStaticMaxRows);
  if (N < 128 || N % 128 != 0 || K < 8 || K % 8 != 0)
    return fmx_fail(FMX_E_INVALID_ARG, "row_gemm_static: N = %d must be a positive multiple of 128, K = %d a positive multiple of 8", N, K);
  const int split_rows = (M + 15) / 16 * 16;
  if ((size_t)split_rows * (size_t)N > kStaticScratchFloats)
    return fmx_fail(FMX_E_CAPACITY, "row_gemm_static: one slice of partials (%d rows x %d columns fp32) exceeds the static scratch of %zu bytes",
                    split_rows, N, kStaticScratchBytes);
  int dev = -1;
  if (cudaError_t e = cudaGetDevice(&dev)) return fmx_fail(FMX_E_CUDA, "row_gemm_static: %s", cudaGetErrorString(e));
  StaticDev *sd = nullptr;
  if (int e = static_setup(dev, &sd)) return e;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);

  // K slices: about two CTAs per SM in one wave, at least two 64-wide chunks per slice, and the partials must fit the array
  const int nK = (K + kRgBK - 1) / kRgBK, n_slices = N / kRgCols;
  int ks = std::max(1, std::min(2 * sd->sm_count / n_slices, nK / 2));
  while (ks > 1 && (size_t)ks * split_rows * N > kStaticScratchFloats) --ks;
  const int cps = (nK + ks - 1) / ks;
  ks = (nK + cps - 1) / cps;

  RowGemmArgs ga{};
  ga.x = static_cast<const __nv_bfloat16 *>(x); ga.M = M; ga.K = K; ga.N = N;
  ga.W[0] = static_cast<const __nv_bfloat16 *>(W); ga.W[1] = ga.W[2] = nullptr;
  ga.src_end_col[0] = ga.src_end_col[1] = ga.src_end_col[2] = 1 << 30;
  ga.interleave2 = 0; ga.chunks_per_split = cps; ga.split_rows = split_rows;
  ga.partial = sd->scratch;                                      // the looked-up device address, never the symbol's name
  const dim3 grid(n_slices, ks);
  if (M <= 16) row_gemm_kernel<1><<<grid, 256, row_gemm_smem<1>(), s>>>(ga);
  else if (M <= 32) row_gemm_kernel<2><<<grid, 256, row_gemm_smem<2>(), s>>>(ga);
  else if (M <= 64) row_gemm_kernel<4><<<grid, 256, row_gemm_smem<4>(), s>>>(ga);
  else row_gemm_kernel<8><<<grid, 256, row_gemm_smem<8>(), s>>>(ga);
  if (cudaError_t e = cudaGetLastError()) return fmx_fail(FMX_E_CUDA, "row_gemm_static: launch failed: %s", cudaGetErrorString(e));
  const long long n_thr = (long long)M * (N / 4);
  static_reduce_kernel<<<(unsigned)((n_thr + 255) / 256), 256, 0, s>>>(out, M, N, ks, split_rows);
  if (cudaError_t e = cudaGetLastError()) return fmx_fail(FMX_E_CUDA, "row_gemm_static: launch failed: %s", cudaGetErrorString(e));
  fmx_clear_error();
  return FMX_OK;
}
