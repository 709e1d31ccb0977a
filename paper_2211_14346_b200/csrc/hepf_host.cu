// hepf_host.cu — hepf_tth_host: the whole path from HOST buffers (the end-to-end entry point bench.py's `e2e`
// number goes through): H2D of the event columns -> hepf_select -> hepf_reconstruct_tth -> D2H of the results.
// Device memory comes from the caller's arena; nothing is allocated here.
#include "hepf_common.cuh"

using namespace hepf;

namespace {
size_t up256(size_t x) { return (x + 255) / 256 * 256; }

struct ArenaLayout {
  size_t cols, flags, idx, count, cutflow, sel_ws, reco_ws, best, total;
};

ArenaLayout layout(int64_t n, int64_t stride) {
  ArenaLayout L{};
  size_t off = 0;
  L.cols = off; off += up256((size_t)64 * stride * sizeof(double));
  L.flags = off; off += up256((size_t)stride * sizeof(uint32_t));
  L.idx = off; off += up256((size_t)(n > 0 ? n : 1) * sizeof(uint32_t));
  L.count = off; off += 256;
  L.cutflow = off; off += up256(HEPF_MAX_CUTS * sizeof(int64_t));
  L.sel_ws = off; off += up256(hepf_select_workspace_bytes(n));
  L.reco_ws = off; off += up256(hepf_reconstruct_workspace_bytes(n, 1));
  L.best = off; off += up256((size_t)(n > 0 ? n : 1) * sizeof(hepf_best_t));
  L.total = off;
  return L;
}
}  // namespace

extern "C" size_t hepf_tth_host_arena_bytes(int64_t n_events, int32_t n_variations) {
  (void)n_variations;
  if (n_events < 0) return 0;
  const int64_t stride = n_events + (n_events & 1);
  return layout(n_events, stride < 2 ? 2 : stride).total + 256;
}

extern "C" int hepf_tth_host(const hepf_events_t* hev, const hepf_cut_t* host_cuts, int n_cuts, int32_t n_variations,
                             uint64_t seed, const hepf_tth_params_t* host_params, uint32_t* host_out_idx,
                             hepf_best_t* host_out_best, int64_t* host_out_count, int64_t* host_out_cutflow, void* arena,
                             size_t arena_bytes, void* stream_) {
  cudaStream_t stream = (cudaStream_t)stream_;
  int rc = check_events(hev);
  if (rc != HEPF_OK) return rc;
  if (!host_out_count || (hev->n_events > 0 && !host_out_best)) { set_error("hepf_tth_host: NULL output"); return HEPF_ERR_ARG; }
  const int64_t n = hev->n_events;
  int64_t dstride = n + (n & 1); if (dstride < 2) dstride = 2;
  const ArenaLayout L = layout(n, dstride);
  if (!arena || !aligned(arena, 256) || arena_bytes < L.total) {
    set_error("hepf_tth_host: arena too small or misaligned (%zu < %zu)", arena_bytes, L.total); return HEPF_ERR_CAPACITY;
  }
  char* base = reinterpret_cast<char*>(arena);
  double* dcols = reinterpret_cast<double*>(base + L.cols);
  uint32_t* dflags = reinterpret_cast<uint32_t*>(base + L.flags);
  // device view with a dense stride; copy each column block row by row (host stride may differ)
  hepf_events_t dev = *hev;
  dev.stride = dstride;
  struct Blk { const double* src; const double** dst; int rows; };
  const Blk blks[] = {{hev->lep_px, &dev.lep_px, 2}, {hev->lep_py, &dev.lep_py, 2}, {hev->lep_pz, &dev.lep_pz, 2},
                      {hev->lep_e, &dev.lep_e, 2}, {hev->lep_pt, &dev.lep_pt, 2}, {hev->lep_eta, &dev.lep_eta, 2},
                      {hev->jet_px, &dev.jet_px, 8}, {hev->jet_py, &dev.jet_py, 8}, {hev->jet_pz, &dev.jet_pz, 8},
                      {hev->jet_e, &dev.jet_e, 8}, {hev->jet_pt, &dev.jet_pt, 8}, {hev->jet_eta, &dev.jet_eta, 8},
                      {hev->met_x, &dev.met_x, 1}, {hev->met_y, &dev.met_y, 1}, {hev->met, &dev.met, 1},
                      {hev->mll, &dev.mll, 1}};
  int64_t row = 0;
  for (const Blk& b : blks) {
    double* d = dcols + row * dstride;
    *b.dst = d;
    if (n > 0) {
      if (hev->stride == dstride) {
        HEPF_CUDA_TRY(cudaMemcpyAsync(d, b.src, (size_t)b.rows * dstride * sizeof(double), cudaMemcpyHostToDevice, stream));
      } else {
        HEPF_CUDA_TRY(cudaMemcpy2DAsync(d, dstride * sizeof(double), b.src, hev->stride * sizeof(double),
                                        (size_t)n * sizeof(double), b.rows, cudaMemcpyHostToDevice, stream));
      }
    }
    row += b.rows;
  }
  dev.flags = dflags;
  if (n > 0) HEPF_CUDA_TRY(cudaMemcpyAsync(dflags, hev->flags, (size_t)n * sizeof(uint32_t), cudaMemcpyHostToDevice, stream));
  uint32_t* didx = reinterpret_cast<uint32_t*>(base + L.idx);
  int64_t* dcount = reinterpret_cast<int64_t*>(base + L.count);
  int64_t* dcutflow = reinterpret_cast<int64_t*>(base + L.cutflow);
  hepf_best_t* dbest = reinterpret_cast<hepf_best_t*>(base + L.best);
  rc = hepf_select(&dev, host_cuts, n_cuts, didx, dcount, host_out_cutflow ? dcutflow : nullptr, base + L.sel_ws,
                   up256(hepf_select_workspace_bytes(n)), stream);
  if (rc != HEPF_OK) return rc;
  HEPF_CUDA_TRY(cudaMemcpyAsync(host_out_count, dcount, sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
  HEPF_CUDA_TRY(cudaStreamSynchronize(stream));
  const int64_t n_sel = *host_out_count;
  rc = hepf_reconstruct_tth(&dev, didx, n_sel, n_variations, seed, host_params, dbest, base + L.reco_ws,
                            up256(hepf_reconstruct_workspace_bytes(n, 1)), stream);
  if (rc != HEPF_OK) return rc;
  if (n_sel > 0) {
    HEPF_CUDA_TRY(cudaMemcpyAsync(host_out_best, dbest, (size_t)n_sel * sizeof(hepf_best_t), cudaMemcpyDeviceToHost, stream));
    if (host_out_idx)
      HEPF_CUDA_TRY(cudaMemcpyAsync(host_out_idx, didx, (size_t)n_sel * sizeof(uint32_t), cudaMemcpyDeviceToHost, stream));
  }
  if (host_out_cutflow && n_cuts > 0)
    HEPF_CUDA_TRY(cudaMemcpyAsync(host_out_cutflow, dcutflow, (size_t)n_cuts * sizeof(int64_t), cudaMemcpyDeviceToHost, stream));
  HEPF_CUDA_TRY(cudaStreamSynchronize(stream));
  return HEPF_OK;
}
