// hepf_philox.cu — hepf_philox_normal: the standalone standard-normal stream (BASELINE.json configs[4];
// the paper's PRNG offload, §5.3, replaced by an in-register counter-based generator).
//
// One thread produces one Philox4x32-10 block = two normals = one 16-byte store.  Work is laid out so that a
// warp writes 512 contiguous bytes; the grid is sized in waves of 148 SMs and strides over the pair range.
// Bound: max(HBM write, FP64 pipe) — see DESIGN.md "Kernels".
#include "hepf_common.cuh"

namespace hepf {

constexpr int PN_THREADS = 256;

// Interior of a range: pairs [pair0, pair0 + n_pairs), every one of them fully inside the caller's range, out = the
// 16-byte aligned address of Z[2 * pair0].  One pair = one Philox block = one 128-bit streaming store; a warp writes 512
// contiguous bytes; grid-stride.
__global__ void __launch_bounds__(PN_THREADS)
philox_normal_pairs_kernel(uint32_t k0, uint32_t k1, uint64_t pair0, uint64_t n_pairs, double2* __restrict__ out) {
  const uint64_t stride = (uint64_t)gridDim.x * PN_THREADS;
  for (uint64_t p = (uint64_t)blockIdx.x * PN_THREADS + threadIdx.x; p < n_pairs; p += stride) {
    const uint64_t b = pair0 + p;
    uint32_t x[4];
    philox4x32_10((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1, x);
    double ze, zo; block_normals_ip(x, ze, zo);
    __stcs(out + p, make_double2(ze, zo));
  }
}

// Anything else (a range that starts odd, an 8-byte aligned destination, the odd last element): element-wise stores of
// the members of each pair that fall inside [g_first, g_last).  out[i] = Z[g_first + i].
__global__ void __launch_bounds__(PN_THREADS)
philox_normal_edge_kernel(uint32_t k0, uint32_t k1, uint64_t pair0, uint64_t n_pairs, uint64_t g_first, uint64_t g_last,
                          double* __restrict__ out) {
  const uint64_t stride = (uint64_t)gridDim.x * PN_THREADS;
  for (uint64_t p = (uint64_t)blockIdx.x * PN_THREADS + threadIdx.x; p < n_pairs; p += stride) {
    const uint64_t b = pair0 + p;
    uint32_t x[4];
    philox4x32_10((uint32_t)b, (uint32_t)(b >> 32), 0u, 0u, k0, k1, x);
    double ze, zo; block_normals_ip(x, ze, zo);
    const uint64_t g = 2 * b;
    if (g >= g_first && g < g_last) __stcs(out + (g - g_first), ze);
    if (g + 1 >= g_first && g + 1 < g_last) __stcs(out + (g + 1 - g_first), zo);
  }
}

}  // namespace hepf

using namespace hepf;

extern "C" int hepf_philox_normal(uint64_t seed, uint64_t counter, uint64_t n, double* out, void* stream) {
  if (n == 0) return HEPF_OK;
  if (!out || !aligned(out, 8)) { set_error("hepf_philox_normal: out NULL or misaligned"); return HEPF_ERR_ARG; }
  if (counter + n < counter) { set_error("hepf_philox_normal: counter + n overflows 2^64"); return HEPF_ERR_ARG; }
  const uint64_t g_first = counter, g_last = counter + n;
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const uint64_t cap = (uint64_t)sms * 8 * 4;   // 8 resident blocks of 256 threads per SM, 4 waves
  const uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
  auto grid_for = [cap](uint64_t n_pairs) { const uint64_t want = (n_pairs + PN_THREADS - 1) / PN_THREADS; return (unsigned)(want < cap ? want : cap); };
  cudaStream_t st = (cudaStream_t)stream;
  if (((g_first & 1) == 0) && aligned(out, 16)) {
    const uint64_t n_full = n >> 1;             // whole pairs, then possibly one last even-indexed element
    if (n_full) {
      philox_normal_pairs_kernel<<<grid_for(n_full), PN_THREADS, 0, st>>>(k0, k1, g_first >> 1, n_full, reinterpret_cast<double2*>(out));
      count_launch();
    }
    if (n & 1) {
      philox_normal_edge_kernel<<<1, PN_THREADS, 0, st>>>(k0, k1, (g_last - 1) >> 1, 1, g_last - 1, g_last, out + (n - 1));
      count_launch();
    }
  } else {
    const uint64_t pair0 = g_first >> 1, n_pairs = ((g_last + 1) >> 1) - pair0;
    philox_normal_edge_kernel<<<grid_for(n_pairs), PN_THREADS, 0, st>>>(k0, k1, pair0, n_pairs, g_first, g_last, out);
    count_launch();
  }
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
