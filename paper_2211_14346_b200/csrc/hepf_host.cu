// hepf_host.cu — hepf_tth_host: the whole path from HOST buffers (the end-to-end entry point bench.py's `e2e` number
// goes through).  Device memory comes from the caller's arena; nothing is allocated here except, once per host thread,
// two copy streams and a few events.
//
// The sample is cut into up to 10 chunks of consecutive events (the first and last ones smaller) and pipelined: every chunk's columns go host -> device on a
// copy-in stream (all enqueued up front), the compute stream waits for chunk c's columns, runs hepf_select and the
// reconstruction on the chunk VIEW (same pointers + offset, event_base + offset: the smearing stream is keyed by the
// global event index, so the records are bit-identical to a single-view run), and the chunk's survivors and records go
// device -> host on a copy-out stream while the next chunk computes.  The reconstruction reads the length of its list
// from device memory (hepf_reconstruct_tth_n's kernels), so the host never waits between a chunk's select and its
// reconstruction: all chunks are enqueued first; only then does the host wait, chunk by chunk, for the survivor count it
// needs to size that chunk's device -> host copies.  With 516 B/event in and a reconstruction of about
// the same duration as the copy, the copies hide behind the kernels.
#include "hepf_common.cuh"

using namespace hepf;

namespace {
constexpr int MAX_CHUNKS = 10;
constexpr int64_t MIN_CHUNK = 32768;      // events; smaller samples are not worth splitting

size_t up256(size_t x) { return (x + 255) / 256 * 256; }

// Chunks of consecutive events; boundaries are multiples of 4 so that every chunk view keeps the 16-byte alignment.  Chunk
// c covers events [start[c], start[c + 1]).  The first and the last chunks are smaller (weights 1 2 4 5 ... 5 4 2 1): the
// kernels cannot start before the first chunk has arrived, and what remains to be done after the last byte has arrived —
// the last chunk's kernels and its copy back — is what the pipeline cannot hide.  Returns the number of chunks.
int chunk_plan(int64_t n, int64_t* start) {
  int nc = (int)(n / MIN_CHUNK); if (nc < 1) nc = 1; if (nc > MAX_CHUNKS) nc = MAX_CHUNKS;
  int wsum = 0, w[MAX_CHUNKS];
  for (int c = 0; c < nc; c++) {
    const int edge = c < nc - 1 - c ? c : nc - 1 - c;
    w[c] = (nc >= 6 && edge < 3) ? (1 << edge) : 5;
    wsum += w[c];
  }
  int64_t acc = 0; start[0] = 0;
  for (int c = 0; c < nc; c++) {
    acc += w[c];
    int64_t e = (n * acc / wsum + 3) / 4 * 4;
    start[c + 1] = (c + 1 == nc || e > n) ? n : e;
  }
  return nc;
}
int64_t longest_chunk(int64_t n) {
  int64_t start[MAX_CHUNKS + 1];
  const int nc = chunk_plan(n, start);
  int64_t m = 1;
  for (int c = 0; c < nc; c++) if (start[c + 1] - start[c] > m) m = start[c + 1] - start[c];
  return m;
}

struct ArenaLayout { size_t cols, flags, idx, count, cutflow, sel_ws[2], reco_ws[2], best, total; };

ArenaLayout layout(int64_t n, int64_t stride) {
  ArenaLayout L{};
  size_t off = 0;
  L.cols = off; off += up256((size_t)64 * stride * sizeof(double));
  L.flags = off; off += up256((size_t)stride * sizeof(uint32_t));
  L.idx = off; off += up256((size_t)(n > 0 ? n : 1) * sizeof(uint32_t));
  L.count = off; off += 256;                                             // one int64 per chunk
  L.cutflow = off; off += up256((size_t)MAX_CHUNKS * HEPF_MAX_CUTS * sizeof(int64_t));
  for (int k = 0; k < 2; k++) {      // one set per compute stream (chunks alternate between two streams)
    L.sel_ws[k] = off; off += up256(hepf_select_workspace_bytes(n));
    L.reco_ws[k] = off; off += up256(hepf_reconstruct_workspace_bytes(longest_chunk(n), 1));   // per chunk: winner keys + nominal objects
  }
  L.best = off; off += up256((size_t)(n > 0 ? n : 1) * sizeof(hepf_best_t));
  L.total = off;
  return L;
}

struct Pipe {                    // per host thread, created on first use
  cudaStream_t in = nullptr, out = nullptr, alt = nullptr;   // alt: second compute stream (odd chunks)
  cudaEvent_t arrived[MAX_CHUNKS] = {}, counted[MAX_CHUNKS] = {}, done[MAX_CHUNKS] = {}, start = nullptr, alt_done = nullptr;
  int64_t* counts = nullptr;     // pinned host memory: one survivor count per chunk
  bool ok = false;
};
thread_local Pipe g_pipe;

int pipe_init() {
  if (g_pipe.ok) return HEPF_OK;
  HEPF_CUDA_TRY(cudaStreamCreateWithFlags(&g_pipe.in, cudaStreamNonBlocking));
  HEPF_CUDA_TRY(cudaStreamCreateWithFlags(&g_pipe.out, cudaStreamNonBlocking));
  HEPF_CUDA_TRY(cudaStreamCreateWithFlags(&g_pipe.alt, cudaStreamNonBlocking));
  HEPF_CUDA_TRY(cudaEventCreateWithFlags(&g_pipe.alt_done, cudaEventDisableTiming));
  HEPF_CUDA_TRY(cudaEventCreateWithFlags(&g_pipe.start, cudaEventDisableTiming));
  for (int c = 0; c < MAX_CHUNKS; c++) {
    HEPF_CUDA_TRY(cudaEventCreateWithFlags(&g_pipe.arrived[c], cudaEventDisableTiming));
    HEPF_CUDA_TRY(cudaEventCreateWithFlags(&g_pipe.done[c], cudaEventDisableTiming));
    HEPF_CUDA_TRY(cudaEventCreateWithFlags(&g_pipe.counted[c], cudaEventDisableTiming));
  }
  HEPF_CUDA_TRY(cudaHostAlloc(reinterpret_cast<void**>(&g_pipe.counts), MAX_CHUNKS * sizeof(int64_t), cudaHostAllocDefault));
  g_pipe.ok = true;
  return HEPF_OK;
}

__global__ void add_offset_kernel(uint32_t* idx, const int64_t* n_dev, uint32_t off) {
  const int64_t n = *n_dev;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) idx[i] += off;
}

// on any failure after work was enqueued: do not return while copies into the caller's buffers are still in flight
int drain(int rc, cudaStream_t stream) {
  cudaStreamSynchronize(g_pipe.in); cudaStreamSynchronize(g_pipe.alt); cudaStreamSynchronize(stream); cudaStreamSynchronize(g_pipe.out);
  return rc;
}
#define HEPF_PIPE_TRY(expr)                                                            \
  do {                                                                                 \
    cudaError_t _e = (expr);                                                           \
    if (_e != cudaSuccess) return drain(::hepf::cuda_fail(_e, #expr), stream);         \
  } while (0)
}  // namespace

extern "C" size_t hepf_tth_host_arena_bytes(int64_t n_events, int32_t n_variations) {
  (void)n_variations;
  if (n_events < 0) return 0;
  int64_t stride = (n_events + 3) / 4 * 4; if (stride < 4) stride = 4;
  return layout(n_events, stride).total + 256;
}

extern "C" int hepf_tth_host(const hepf_events_t* hev, const hepf_cut_t* host_cuts, int n_cuts, int32_t n_variations,
                             uint64_t seed, const hepf_tth_params_t* host_params, uint32_t* host_out_idx,
                             hepf_best_t* host_out_best, int64_t* host_out_count, int64_t* host_out_cutflow, void* arena,
                             size_t arena_bytes, void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  int rc = check_events(hev);
  if (rc != HEPF_OK) return rc;
  if (!host_out_count || (hev->n_events > 0 && !host_out_best)) { set_error("hepf_tth_host: NULL output"); return HEPF_ERR_ARG; }
  if (n_cuts < 0 || n_cuts > HEPF_MAX_CUTS) { set_error("hepf_tth_host: n_cuts must be 0..%d", HEPF_MAX_CUTS); return HEPF_ERR_ARG; }
  const int64_t n = hev->n_events;
  int64_t dstride = (n + 3) / 4 * 4; if (dstride < 4) dstride = 4;
  const ArenaLayout L = layout(n, dstride);
  if (!arena || !aligned(arena, 256) || arena_bytes < L.total) {
    set_error("hepf_tth_host: arena too small or misaligned (%zu < %zu)", arena_bytes, L.total); return HEPF_ERR_CAPACITY;
  }
  rc = pipe_init();
  if (rc != HEPF_OK) return rc;
  char* base = reinterpret_cast<char*>(arena);
  double* dcols = reinterpret_cast<double*>(base + L.cols);
  uint32_t* dflags = reinterpret_cast<uint32_t*>(base + L.flags);
  uint32_t* didx = reinterpret_cast<uint32_t*>(base + L.idx);
  int64_t* dcount = reinterpret_cast<int64_t*>(base + L.count);
  int64_t* dcutflow = reinterpret_cast<int64_t*>(base + L.cutflow);
  hepf_best_t* dbest = reinterpret_cast<hepf_best_t*>(base + L.best);
  // the 16 column groups of the view, in the row order of the device block
  const double* const src[16] = {hev->lep_px, hev->lep_py, hev->lep_pz, hev->lep_e, hev->lep_pt, hev->lep_eta,
                                 hev->jet_px, hev->jet_py, hev->jet_pz, hev->jet_e, hev->jet_pt, hev->jet_eta,
                                 hev->met_x, hev->met_y, hev->met, hev->mll};
  const int rows[16] = {2, 2, 2, 2, 2, 2, 8, 8, 8, 8, 8, 8, 1, 1, 1, 1};
  const double* dptr[16];
  { int64_t row = 0; for (int b = 0; b < 16; b++) { dptr[b] = dcols + row * dstride; row += rows[b]; } }
  int64_t start[MAX_CHUNKS + 1];
  const int nc = chunk_plan(n, start);
  // one 64-row copy per chunk when the host columns are the rows of one [64][stride] block in the device block's row order
  // (the layout hepf_synth and DeviceEvents use); otherwise one copy per column group
  bool one_block = true;
  { int64_t row = 0; for (int b = 0; b < 16; b++) { one_block = one_block && (src[b] == src[0] + row * hev->stride); row += rows[b]; } }
  // ---- host -> device, all chunks, on the copy-in stream (ordered after whatever the caller's stream holds) ----------
  HEPF_PIPE_TRY(cudaEventRecord(g_pipe.start, stream));
  HEPF_PIPE_TRY(cudaStreamWaitEvent(g_pipe.in, g_pipe.start, 0));
  HEPF_PIPE_TRY(cudaStreamWaitEvent(g_pipe.out, g_pipe.start, 0));
  HEPF_PIPE_TRY(cudaStreamWaitEvent(g_pipe.alt, g_pipe.start, 0));
  for (int c = 0; c < nc; c++) {
    const int64_t lo = start[c], len = start[c + 1] - lo;
    if (len <= 0) continue;
    for (int b = 0; b < (one_block ? 1 : 16); b++)
      HEPF_PIPE_TRY(cudaMemcpy2DAsync(const_cast<double*>(dptr[b]) + lo, dstride * sizeof(double), src[b] + lo,
                                      hev->stride * sizeof(double), (size_t)len * sizeof(double), one_block ? 64 : rows[b],
                                      cudaMemcpyHostToDevice, g_pipe.in));
    HEPF_PIPE_TRY(cudaMemcpyAsync(dflags + lo, hev->flags + lo, (size_t)len * sizeof(uint32_t), cudaMemcpyHostToDevice, g_pipe.in));
    HEPF_PIPE_TRY(cudaEventRecord(g_pipe.arrived[c], g_pipe.in));
  }
  // ---- per chunk: select + reconstruct on the chunk view; the survivors and records of chunk c are written at the chunk's
  //      own offset lo (the list length is only known on the device at this point) ----------------------------------------
  for (int c = 0; c < nc; c++) {
    const int64_t lo = start[c], len = start[c + 1] - lo;
    if (len <= 0) { g_pipe.counts[c] = 0; continue; }
    hepf_events_t view = *hev;
    view.n_events = len; view.stride = dstride; view.event_base = hev->event_base + lo;
    const double** vp[16] = {&view.lep_px, &view.lep_py, &view.lep_pz, &view.lep_e, &view.lep_pt, &view.lep_eta,
                             &view.jet_px, &view.jet_py, &view.jet_pz, &view.jet_e, &view.jet_pt, &view.jet_eta,
                             &view.met_x, &view.met_y, &view.met, &view.mll};
    for (int b = 0; b < 16; b++) *vp[b] = dptr[b] + lo;
    view.flags = dflags + lo;
    // chunks alternate between the caller's stream and a second compute stream, so that the persistent search kernel of
    // chunk c + 1 fills the SMs that the tail of chunk c's leaves idle
    const int w = c & 1;
    cudaStream_t cs_ = w ? g_pipe.alt : stream;
    HEPF_PIPE_TRY(cudaStreamWaitEvent(cs_, g_pipe.arrived[c], 0));
    rc = hepf_select(&view, host_cuts, n_cuts, didx + lo, dcount + c, host_out_cutflow ? dcutflow + c * HEPF_MAX_CUTS : nullptr,
                     base + L.sel_ws[w], up256(hepf_select_workspace_bytes(n)), cs_);
    if (rc != HEPF_OK) return drain(rc, stream);
    HEPF_PIPE_TRY(cudaMemcpyAsync(g_pipe.counts + c, dcount + c, sizeof(int64_t), cudaMemcpyDeviceToHost, cs_));
    HEPF_PIPE_TRY(cudaEventRecord(g_pipe.counted[c], cs_));
    rc = reconstruct_impl(&view, didx + lo, dcount + c, len, n_variations, seed, host_params, dbest + lo, base + L.reco_ws[w],
                          up256(hepf_reconstruct_workspace_bytes(longest_chunk(n), 1)), cs_, lo);
    if (rc != HEPF_OK) return drain(rc, stream);
    if (lo > 0) {
      add_offset_kernel<<<256, 256, 0, cs_>>>(didx + lo, dcount + c, (uint32_t)lo);
      count_launch();
    }
    HEPF_PIPE_TRY(cudaEventRecord(g_pipe.done[c], cs_));
  }
  // ---- results device -> host on the copy-out stream: the host learns each chunk's count here, with everything enqueued ----
  int64_t total = 0;
  for (int c = 0; c < nc; c++) {
    const int64_t lo = start[c];
    if (start[c + 1] - lo <= 0) continue;
    HEPF_PIPE_TRY(cudaEventSynchronize(g_pipe.counted[c]));
    const int64_t n_sel = g_pipe.counts[c];
    if (n_sel > 0) {
      HEPF_PIPE_TRY(cudaStreamWaitEvent(g_pipe.out, g_pipe.done[c], 0));
      HEPF_PIPE_TRY(cudaMemcpyAsync(host_out_best + total, dbest + lo, (size_t)n_sel * sizeof(hepf_best_t),
                                    cudaMemcpyDeviceToHost, g_pipe.out));
      if (host_out_idx)
        HEPF_PIPE_TRY(cudaMemcpyAsync(host_out_idx + total, didx + lo, (size_t)n_sel * sizeof(uint32_t),
                                      cudaMemcpyDeviceToHost, g_pipe.out));
    }
    total += n_sel;
  }
  *host_out_count = total;
  HEPF_PIPE_TRY(cudaEventRecord(g_pipe.alt_done, g_pipe.alt));        // the caller's stream ends after both compute streams
  HEPF_PIPE_TRY(cudaStreamWaitEvent(stream, g_pipe.alt_done, 0));
  if (host_out_cutflow && n_cuts > 0) {
    int64_t cf[MAX_CHUNKS * HEPF_MAX_CUTS];
    HEPF_PIPE_TRY(cudaMemcpyAsync(cf, dcutflow, (size_t)nc * HEPF_MAX_CUTS * sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
    HEPF_PIPE_TRY(cudaStreamSynchronize(stream));
    for (int k = 0; k < n_cuts; k++) {
      host_out_cutflow[k] = 0;
      for (int c = 0; c < nc; c++) if (start[c + 1] > start[c]) host_out_cutflow[k] += cf[c * HEPF_MAX_CUTS + k];
    }
  }
  HEPF_PIPE_TRY(cudaStreamSynchronize(g_pipe.out));
  HEPF_PIPE_TRY(cudaStreamSynchronize(stream));
  return HEPF_OK;
}
