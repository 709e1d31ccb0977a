// hepf_api.cu — error plumbing, argument checks, defaults, launch counter, FP64 roof probe.
#include <cstdarg>
#include <cstdio>

#include "hepf_common.cuh"

namespace hepf {

static thread_local char g_err[512] = "";
static thread_local int64_t g_launches = 0;

void set_error(const char* fmt, ...) {
  va_list ap; va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
int cuda_fail(cudaError_t e, const char* what) {
  set_error("CUDA error %d (%s) at %s", (int)e, cudaGetErrorString(e), what);
  return HEPF_ERR_CUDA;
}
void count_launch(int n) { g_launches += n; }

static thread_local bool g_timing = false;
static thread_local cudaEvent_t g_ev[T_SLOTS] = {};
void timing_mark(int slot, cudaStream_t stream) {
  if (!g_timing || slot < 0 || slot >= T_SLOTS) return;
  if (!g_ev[slot] && cudaEventCreate(&g_ev[slot]) != cudaSuccess) return;
  cudaEventRecord(g_ev[slot], stream);
}

int check_events(const hepf_events_t* ev) {
  if (!ev) { set_error("events view is NULL"); return HEPF_ERR_ARG; }
  if (ev->n_events < 0 || ev->stride < ev->n_events || (ev->stride & 1)) {
    set_error("bad n_events/stride (%lld/%lld): need 0 <= n_events <= stride, stride even",
              (long long)ev->n_events, (long long)ev->stride);
    return HEPF_ERR_ARG;
  }
  if (ev->n_events > 0xffffffffll) { set_error("n_events exceeds 2^32-1"); return HEPF_ERR_ARG; }
  const void* ptrs[] = {ev->lep_px, ev->lep_py, ev->lep_pz, ev->lep_e, ev->lep_pt, ev->lep_eta,
                        ev->jet_px, ev->jet_py, ev->jet_pz, ev->jet_e, ev->jet_pt, ev->jet_eta,
                        ev->met_x, ev->met_y, ev->met, ev->mll, ev->flags};
  if (ev->n_events == 0) return HEPF_OK;
  for (const void* p : ptrs)
    if (!p || !aligned(p, 16)) { set_error("event column pointer NULL or not 16-byte aligned"); return HEPF_ERR_ARG; }
  return HEPF_OK;
}

// 8 independent FMA chains per thread: enough ILP to cover the DFMA latency at any occupancy
__global__ void fp64_peak_kernel(int64_t iters, double* sink) {
  double a0 = threadIdx.x * 1e-9, a1 = a0 + 1, a2 = a0 + 2, a3 = a0 + 3, a4 = a0 + 4, a5 = a0 + 5, a6 = a0 + 6, a7 = a0 + 7;
  const double m = 0.999999 + 1e-12 * blockIdx.x, c = 1e-7;
  for (int64_t i = 0; i < iters; i++) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  const double s = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  if (s == 123.456) sink[0] = s;  // never true: keeps the chain alive without a store per thread
}

}  // namespace hepf

using namespace hepf;

extern "C" int hepf_timing_enable(int on) { g_timing = on != 0; return HEPF_OK; }
extern "C" double hepf_timing_ms(int from_slot, int to_slot) {
  if (from_slot < 0 || to_slot < 0 || from_slot >= T_SLOTS || to_slot >= T_SLOTS || !g_ev[from_slot] || !g_ev[to_slot]) return -1.0;
  if (cudaEventSynchronize(g_ev[to_slot]) != cudaSuccess) return -1.0;
  float ms = -1.0f;
  if (cudaEventElapsedTime(&ms, g_ev[from_slot], g_ev[to_slot]) != cudaSuccess) return -1.0;
  return (double)ms;
}
extern "C" const char* hepf_last_error(void) { return g_err; }
extern "C" const char* hepf_version(void) { return "hepf 0.3 (sm_100a)"; }
extern "C" int64_t hepf_launch_count(int reset) {
  int64_t v = g_launches;
  if (reset) g_launches = 0;
  return v;
}

extern "C" void hepf_default_params(hepf_tth_params_t* p) {
  if (!p) return;
  p->m_top = 172.5; p->m_w = 80.4; p->m_higgs = 125.0;
  p->sigma_higgs = 15.0; p->lambda_nu = 40.0;
  p->lep_sigma = 0.01; p->jet_stoch = 0.5; p->jet_const = 0.03;
  p->sigma_scale = 1.0; p->s_min = 0.1;
}

extern "C" int hepf_fp64_peak_probe(int blocks, int threads, int64_t fma_per_thread, double* sink, void* stream) {
  if (blocks <= 0 || threads <= 0 || threads > 1024 || fma_per_thread < 8 || !sink) {
    set_error("hepf_fp64_peak_probe: bad arguments"); return HEPF_ERR_ARG;
  }
  fp64_peak_kernel<<<blocks, threads, 0, (cudaStream_t)stream>>>(fma_per_thread / 8, sink);
  count_launch();
  HEPF_CUDA_TRY(cudaGetLastError());
  return HEPF_OK;
}
