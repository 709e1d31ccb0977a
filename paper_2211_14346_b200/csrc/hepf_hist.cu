// hepf_hist.cu — hepf_histogram: device-side histogram of a reconstructed quantity.
//
// Paper: the user's finalize() fills histograms of reconstructed quantities (App. 8.2) and HEP-Frame
// records variables per cut.  Here the winners never leave the GPU for that: one pass over the 128-byte
// records, a shared-memory histogram per block (atomics on shared memory), one global atomic per non-empty bin and block.
// HBM-bound and tiny next to the reconstruction; the bin decision follows the operation sequence of include/hepf.h so
// that the counts are bit-exact against the oracle.
#include "hepf_common.cuh"

namespace hepf {

constexpr int H_THREADS = 256;
constexpr int H_MAX_BINS = 4096;

__device__ __forceinline__ double hist_value(const hepf_best_t& b, int field) {
  switch (field) {
    case HEPF_H_M_TOP: return b.m_top;
    case HEPF_H_M_ANTITOP: return b.m_antitop;
    case HEPF_H_M_WPLUS: return b.m_wplus;
    case HEPF_H_M_WMINUS: return b.m_wminus;
    case HEPF_H_M_HIGGS: return b.m_higgs;
    case HEPF_H_LOGLIK: return b.loglik;
    case HEPF_H_NU_PT: return __dsqrt_rn(__dadd_rn(__dmul_rn(b.nu[0], b.nu[0]), __dmul_rn(b.nu[1], b.nu[1])));
    case HEPF_H_NUBAR_PT: return __dsqrt_rn(__dadd_rn(__dmul_rn(b.nubar[0], b.nubar[0]), __dmul_rn(b.nubar[1], b.nubar[1])));
    default: return (double)b.variation;
  }
}

__global__ void __launch_bounds__(H_THREADS)
histogram_kernel(const hepf_best_t* __restrict__ best, int64_t n, int field, double lo, double inv_w, int nbins,
                 unsigned long long* __restrict__ out) {
  extern __shared__ unsigned int s_h[];          // nbins + 2 counters
  for (int i = threadIdx.x; i < nbins + 2; i += H_THREADS) s_h[i] = 0u;
  __syncthreads();
  const int64_t stride = (int64_t)gridDim.x * H_THREADS;
  for (int64_t k = (int64_t)blockIdx.x * H_THREADS + threadIdx.x; k < n; k += stride) {
    if (!(best[k].status & 1u)) continue;
    const double t = __dmul_rn(__dadd_rn(hist_value(best[k], field), -lo), inv_w);
    if (t != t) continue;                        // NaN: not counted
    const int bin = t < 0.0 ? 0 : (t >= (double)nbins ? nbins + 1 : 1 + (int)t);
    atomicAdd(&s_h[bin], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nbins + 2; i += H_THREADS)
    if (s_h[i]) atomicAdd(&out[i], (unsigned long long)s_h[i]);
}

// the same binning for a plain column of doubles (element k at values[k * stride]); every non-NaN value is filled
__global__ void __launch_bounds__(H_THREADS)
histogram_values_kernel(const double* __restrict__ values, int64_t stride_, int64_t n, double lo, double inv_w, int nbins,
                        unsigned long long* __restrict__ out) {
  extern __shared__ unsigned int s_h[];
  for (int i = threadIdx.x; i < nbins + 2; i += H_THREADS) s_h[i] = 0u;
  __syncthreads();
  const int64_t stride = (int64_t)gridDim.x * H_THREADS;
  for (int64_t k = (int64_t)blockIdx.x * H_THREADS + threadIdx.x; k < n; k += stride) {
    const double t = __dmul_rn(__dadd_rn(__ldcs(values + k * stride_), -lo), inv_w);
    if (t != t) continue;
    const int bin = t < 0.0 ? 0 : (t >= (double)nbins ? nbins + 1 : 1 + (int)t);
    atomicAdd(&s_h[bin], 1u);
  }
  __syncthreads();
  for (int i = threadIdx.x; i < nbins + 2; i += H_THREADS)
    if (s_h[i]) atomicAdd(&out[i], (unsigned long long)s_h[i]);
}

}  // namespace hepf

using namespace hepf;

extern "C" int hepf_histogram_values(const double* values, int64_t stride, int64_t n, double lo, double hi, int32_t nbins,
                                     uint64_t* out, void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (n < 0 || stride < 1 || nbins < 1 || nbins > H_MAX_BINS || !(hi > lo)) {
    set_error("hepf_histogram_values: need n >= 0, stride >= 1, 1 <= nbins <= %d and hi > lo", H_MAX_BINS); return HEPF_ERR_ARG;
  }
  if (!out || !aligned(out, 8) || (n > 0 && (!values || !aligned(values, 8)))) {
    set_error("hepf_histogram_values: values/out NULL or misaligned"); return HEPF_ERR_ARG;
  }
  HEPF_CUDA_TRY(cudaMemsetAsync(out, 0, sizeof(uint64_t) * (size_t)(nbins + 2), stream));
  if (n == 0) return HEPF_OK;
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int64_t want = (n + H_THREADS - 1) / H_THREADS, cap = (int64_t)sms * 8;
  histogram_values_kernel<<<(unsigned)(want < cap ? want : cap), H_THREADS, sizeof(unsigned int) * (size_t)(nbins + 2), stream>>>(
      values, stride, n, lo, (double)nbins / (hi - lo), nbins, reinterpret_cast<unsigned long long*>(out));
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}


extern "C" int hepf_histogram(const hepf_best_t* best, int64_t n, int field, double lo, double hi, int32_t nbins,
                              uint64_t* out, void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  if (n < 0 || nbins < 1 || nbins > H_MAX_BINS || !(hi > lo) || field < HEPF_H_M_TOP || field > HEPF_H_VARIATION) {
    set_error("hepf_histogram: need n >= 0, 1 <= nbins <= %d, hi > lo and a known field", H_MAX_BINS); return HEPF_ERR_ARG;
  }
  if (!out || !aligned(out, 8) || (n > 0 && (!best || !aligned(best, 16)))) {
    set_error("hepf_histogram: best/out NULL or misaligned"); return HEPF_ERR_ARG;
  }
  HEPF_CUDA_TRY(cudaMemsetAsync(out, 0, sizeof(uint64_t) * (size_t)(nbins + 2), stream));
  if (n == 0) return HEPF_OK;
  int dev = 0, sms = 148;
  HEPF_CUDA_TRY(cudaGetDevice(&dev));
  HEPF_CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int64_t want = (n + H_THREADS - 1) / H_THREADS, cap = (int64_t)sms * 8;
  const unsigned grid = (unsigned)(want < cap ? want : cap);
  const double inv_w = (double)nbins / (hi - lo);
  histogram_kernel<<<grid, H_THREADS, sizeof(unsigned int) * (size_t)(nbins + 2), stream>>>(
      best, n, field, lo, inv_w, nbins, reinterpret_cast<unsigned long long*>(out));
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
