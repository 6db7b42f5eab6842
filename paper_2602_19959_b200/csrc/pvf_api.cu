// C-ABI glue: configuration checks, the single workspace pool, weight packing, stage sequencing.
// Declarations and the passages they follow: include/pvf.h.
#include <cstdio>
#include <cstring>
#include <new>
#include <string>
#include <vector>

#include "pvf_internal.cuh"

using namespace pvf;

#define PVF_STR2(x) #x
#define PVF_STR(x) PVF_STR2(x)

struct pvf_ctx {
  pvf_config cfg;
  bool owns_pool = false;
  unsigned char* pool = nullptr;
  size_t pool_bytes = 0;
  int device = 0;
  int sm_count = 148;
  // sub-allocations of the pool
  float* fc_params = nullptr;
  float* conv_f32 = nullptr;      // PyTorch-layout conv params (FP32 path + head of every path)
  UnetParamsF32 conv_ptrs{};
  void* tc_packed = nullptr;
  void* fc_w5img = nullptr;
  int32_t* el_list = nullptr;     // empty-interval elision: work list, its length, UNet(0)
  int32_t* el_count = nullptr;
  float* el_p0 = nullptr;       // tcgen05 image of the 25 -> 800 layer (TF32 / BF16 modes)
  int32_t* perm = nullptr;
  int32_t* seg_off = nullptr;
  int32_t* seg_cnt = nullptr;
  uint32_t* flags = nullptr;
  float* hist = nullptr;
  int32_t hist_events = 0;        // events the histogram buffer holds: max_events, or l2_chunk_events if that is smaller
  // host-io staging (enable_host_io)
  float* st_feat = nullptr;
  int32_t* st_off = nullptr;
  float* st_probs = nullptr;
  float* st_z = nullptr;
  float* st_prob = nullptr;
  int32_t* st_bin = nullptr;
  int32_t* st_count = nullptr;
  uint32_t* st_flags = nullptr;
  // pvf_run_host only: copy streams and events of the chunk pipeline (H2D of chunk k+1 | compute k | D2H k-1)
  static constexpr int kHostChunks = 8;
  cudaStream_t s_in = nullptr, s_out = nullptr;
  cudaEvent_t ev_in[kHostChunks] = {}, ev_comp[kHostChunks] = {}, ev_fork = nullptr, ev_join = nullptr;
  bool suppress_timing = false;
  static constexpr int kTimedRuns = 64;   // ring of per-run event sets (stage timing)
  cudaEvent_t ev[kTimedRuns][5] = {};
  int64_t timed_runs = 0;                 // runs recorded since the last pvf_stage_times_ms
  int32_t last_n_events = 0;      // events whose histograms the buffer holds after the last run ...
  int32_t last_e0 = 0;            // ... and the first of them (non-zero with l2_chunk_events: the last chunk)
  std::string cuda_err;
};

namespace {

size_t align_up(size_t v, size_t a = 256) { return (v + a - 1) / a * a; }

struct Layout {
  size_t fc_params, conv_f32, tc_packed, fc_w5img, el_list, el_count, el_p0, perm, seg_off, seg_cnt, flags, hist;
  size_t st_feat, st_off, st_probs, st_z, st_prob, st_bin, st_count, st_flags, total;
  size_t conv_w_off[6], conv_b_off[6];  // float offsets inside conv_f32
};

void conv_shapes(int C, int shp[6][3]) {
  const int s[6][3] = {{C, kHistCh, 25}, {C, C, 15}, {C, C, 5}, {C, 2 * C, 15}, {C, 2 * C, 25}, {1, C, 1}};
  memcpy(shp, s, sizeof(s));
}

// Which kernels serve the configuration: the tcgen05 kernels (FC with the 25 -> 800 layer on tensor cores + k_unet_tc) for
// every precision, except PVF_PREC_FP32 without CTA pairs = the CUDA-core kernels (k_fc_hist + k_unet_simt), kept as the
// bisecting reference of the GPU side.
bool uses_tc(const pvf_config* c) { return c->precision != PVF_PREC_FP32 || c->unet_cta_pair != 0; }

bool config_ok(const pvf_config* c) {
  if (!c) return false;
  if (c->n_intervals != kIntervals || c->n_bins != kBins) return false;
  if (c->z_min_mm != -200.0f || c->bin_width_mm != 0.1f) return false;
  if (c->fc_in != kFcIn || c->fc_hidden != kFcHidden || c->hist_channels != kHistCh) return false;
  if (c->unet_channels != 64 && c->unet_channels != 32 && c->unet_channels != 16) return false;
  if (c->k_e1 != 25 || c->k_e2 != 15 || c->k_b != 5 || c->k_d2 != 15 || c->k_d1 != 25) return false;
  if (c->leaky_slope != kLeaky) return false;
  if (!(c->peak_threshold == c->peak_threshold)) return false;
  if (c->peak_halfwidth != kPeakHalf || c->max_peaks != kMaxPeaks) return false;
  if (c->precision < PVF_PREC_FP32 || c->precision > PVF_PREC_FP16) return false;
  // split_mask: only bit 0 (e1) is built, for the two formats with a 10-bit mantissa (unet_tc_setup would refuse anything else later)
  if (c->split_mask != 0 && !((c->precision == PVF_PREC_TF32 || c->precision == PVF_PREC_FP16) && c->split_mask == 1)) return false;
  // a perm entry keeps the track index in 29 bits (pvf_internal.cuh kEntryMask): 536 870 911 tracks per call at most
  if (c->max_events < 1 || c->max_tracks < 1 || c->max_tracks > (int64_t)kEntryMask) return false;
  if (c->unet_cta_pair != 0 && c->unet_cta_pair != 1) return false;
  if (c->elide_empty_intervals && !uses_tc(c)) return false;                     // tensor-core kernels only
  if (!(c->boundary_margin_mm >= 0.0f && c->boundary_margin_mm < 4.9f)) return false;
  if (c->l2_chunk_events < 0) return false;
  return true;
}

Layout make_layout(const pvf_config* c) {
  Layout L{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t r = o; o = align_up(o + bytes); return r; };
  L.fc_params = take(sizeof(float) * kFcTotal);
  int shp[6][3];
  conv_shapes(c->unet_channels, shp);
  size_t f = 0;
  for (int k = 0; k < 6; ++k) {
    L.conv_w_off[k] = f; f += (size_t)shp[k][0] * shp[k][1] * shp[k][2]; f = (f + 63) / 64 * 64;
    L.conv_b_off[k] = f; f += shp[k][0]; f = (f + 63) / 64 * 64;
  }
  L.conv_f32 = take(sizeof(float) * f);
  L.tc_packed = take(!uses_tc(c) ? 0 : unet_tc_packed_bytes(c->unet_channels, c->precision, c->split_mask, c->unet_cta_pair));
  const size_t E = (size_t)c->max_events, T = (size_t)c->max_tracks;
  L.fc_w5img = take(!uses_tc(c) ? 0 : fc_tc_packed_bytes());
  L.el_list = take(c->elide_empty_intervals ? sizeof(int32_t) * E * kIntervals : 0);
  L.el_count = take(c->elide_empty_intervals ? 256 : 0);
  L.el_p0 = take(c->elide_empty_intervals ? sizeof(float) * kGlobalBins : 0);
  L.perm = take(sizeof(int32_t) * T * (c->boundary_margin_mm > 0.0f ? 2 : 1));   // NEXT-1: two entries per track
  L.seg_off = take(sizeof(int32_t) * E * kIntervals);
  L.seg_cnt = take(sizeof(int32_t) * E * kIntervals);
  L.flags = take(sizeof(uint32_t) * E);
  const size_t EH = (c->l2_chunk_events > 0 && (size_t)c->l2_chunk_events < E) ? (size_t)c->l2_chunk_events : E;
  L.hist = take(sizeof(float) * (EH * kIntervals * kFcOut + (!uses_tc(c) ? 0 : kFcDumpFloats)));
  if (c->enable_host_io) {
    L.st_feat = take(sizeof(float) * 9 * T);
    L.st_off = take(sizeof(int32_t) * (E + 1));
    L.st_probs = take(sizeof(float) * E * kGlobalBins);
    L.st_z = take(sizeof(float) * E * kMaxPeaks);
    L.st_prob = take(sizeof(float) * E * kMaxPeaks);
    L.st_bin = take(sizeof(int32_t) * E * kMaxPeaks);
    L.st_count = take(sizeof(int32_t) * E);
    L.st_flags = take(sizeof(uint32_t) * E);
  }
  L.total = o;
  return L;
}

pvf_status fail_cuda(pvf_ctx* h, cudaError_t e, const char* where) {
  if (h) h->cuda_err = std::string(where) + ": " + cudaGetErrorString(e);
  return PVF_ERR_CUDA;
}

#define PVF_CUDA(h, call)                                             \
  do {                                                                \
    cudaError_t e__ = (call);                                         \
    if (e__ != cudaSuccess) return fail_cuda((h), e__, #call);        \
  } while (0)

// seg_cnt != nullptr: hist is the pool's histogram as the tensor-core FC kernel leaves it (empty intervals unwritten)
void enqueue_unet(pvf_ctx* h, const float* hist, int n_events, float* out_probs, cudaStream_t s,
                  const int* list = nullptr, const int* n_list = nullptr, const int* seg_cnt = nullptr, bool pdl = false);

bool peaks_ok(const pvf_peaks* p) { return p && p->z_mm && p->prob && p->bin && p->count; }

pvf_status create_impl(const pvf_weights* w, const pvf_config* cfg, void* dev_pool, size_t pool_bytes,
                       pvf_handle* out) {
  if (!out) return PVF_ERR_ARG;
  *out = nullptr;
  if (!w || !cfg) return PVF_ERR_ARG;
  if (!config_ok(cfg)) return PVF_ERR_CONFIG;
  for (int k = 0; k < 6; ++k)
    if (!w->fc_w[k] || !w->fc_b[k] || !w->conv_w[k] || !w->conv_b[k]) return PVF_ERR_ARG;
  const Layout L = make_layout(cfg);
  pvf_ctx* h = new (std::nothrow) pvf_ctx();
  if (!h) return PVF_ERR_ARG;
  h->cfg = *cfg;
  cudaError_t e = cudaGetDevice(&h->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->sm_count, cudaDevAttrMultiProcessorCount, h->device);
  if (e != cudaSuccess) { delete h; return PVF_ERR_CUDA; }
  if (dev_pool) {
    if (pool_bytes < L.total || (reinterpret_cast<uintptr_t>(dev_pool) & 255u)) { delete h; return PVF_ERR_CAPACITY; }
    h->pool = static_cast<unsigned char*>(dev_pool);
  } else {
    void* p = nullptr;
    e = cudaMalloc(&p, L.total);
    if (e != cudaSuccess) { delete h; return PVF_ERR_CUDA; }
    h->pool = static_cast<unsigned char*>(p);
    h->owns_pool = true;
  }
  h->pool_bytes = L.total;
  unsigned char* B = h->pool;
  h->fc_params = reinterpret_cast<float*>(B + L.fc_params);
  h->conv_f32 = reinterpret_cast<float*>(B + L.conv_f32);
  h->tc_packed = B + L.tc_packed;
  h->fc_w5img = B + L.fc_w5img;
  h->el_list = reinterpret_cast<int32_t*>(B + L.el_list);
  h->el_count = reinterpret_cast<int32_t*>(B + L.el_count);
  h->el_p0 = reinterpret_cast<float*>(B + L.el_p0);
  h->perm = reinterpret_cast<int32_t*>(B + L.perm);
  h->seg_off = reinterpret_cast<int32_t*>(B + L.seg_off);
  h->seg_cnt = reinterpret_cast<int32_t*>(B + L.seg_cnt);
  h->flags = reinterpret_cast<uint32_t*>(B + L.flags);
  h->hist = reinterpret_cast<float*>(B + L.hist);
  h->hist_events = (cfg->l2_chunk_events > 0 && cfg->l2_chunk_events < cfg->max_events) ? cfg->l2_chunk_events : cfg->max_events;
  if (cfg->enable_host_io) {
    h->st_feat = reinterpret_cast<float*>(B + L.st_feat);
    h->st_off = reinterpret_cast<int32_t*>(B + L.st_off);
    h->st_probs = reinterpret_cast<float*>(B + L.st_probs);
    h->st_z = reinterpret_cast<float*>(B + L.st_z);
    h->st_prob = reinterpret_cast<float*>(B + L.st_prob);
    h->st_bin = reinterpret_cast<int32_t*>(B + L.st_bin);
    h->st_count = reinterpret_cast<int32_t*>(B + L.st_count);
    h->st_flags = reinterpret_cast<uint32_t*>(B + L.st_flags);
  }
  // ---- pack + upload weights (synchronous copies: create is not on the hot path)
  {
    std::vector<float> fc(kFcTotal);
    memcpy(&fc[kFcW0], w->fc_w[0], sizeof(float) * 225);
    memcpy(&fc[kFcB0], w->fc_b[0], sizeof(float) * 25);
    for (int k = 0; k < 4; ++k) {
      memcpy(&fc[kFcHid + kFcHidStride * k], w->fc_w[k + 1], sizeof(float) * 625);
      memcpy(&fc[kFcHid + kFcHidStride * k + 625], w->fc_b[k + 1], sizeof(float) * 25);
    }
    memcpy(&fc[kFcW5], w->fc_w[5], sizeof(float) * 20000);
    memcpy(&fc[kFcB5], w->fc_b[5], sizeof(float) * 800);
    e = cudaMemcpy(h->fc_params, fc.data(), sizeof(float) * kFcTotal, cudaMemcpyHostToDevice);
  }
  int shp[6][3];
  conv_shapes(cfg->unet_channels, shp);
  for (int k = 0; k < 6 && e == cudaSuccess; ++k) {
    e = cudaMemcpy(h->conv_f32 + L.conv_w_off[k], w->conv_w[k],
                   sizeof(float) * shp[k][0] * shp[k][1] * shp[k][2], cudaMemcpyHostToDevice);
    if (e == cudaSuccess)
      e = cudaMemcpy(h->conv_f32 + L.conv_b_off[k], w->conv_b[k], sizeof(float) * shp[k][0], cudaMemcpyHostToDevice);
    h->conv_ptrs.w[k] = h->conv_f32 + L.conv_w_off[k];
    h->conv_ptrs.b[k] = h->conv_f32 + L.conv_b_off[k];
  }
  if (e == cudaSuccess) {
    if (!uses_tc(cfg)) {
      e = unet_simt_setup(cfg->unet_channels);
      if (e == cudaSuccess) e = fc_hist_setup();
    } else {
      const size_t nb = unet_tc_packed_bytes(cfg->unet_channels, cfg->precision, cfg->split_mask, cfg->unet_cta_pair);
      std::vector<unsigned char> img(nb);
      unet_tc_pack(w, cfg->unet_channels, cfg->precision, cfg->split_mask, cfg->unet_cta_pair, img.data());
      e = cudaMemcpy(h->tc_packed, img.data(), nb, cudaMemcpyHostToDevice);
      if (e == cudaSuccess) e = unet_tc_setup(cfg->unet_channels, cfg->precision, cfg->split_mask, cfg->unet_cta_pair);
      if (e == cudaSuccess) {
        std::vector<unsigned char> fimg(fc_tc_packed_bytes());
        fc_tc_pack(w->fc_w[5], w->fc_b[5], fimg.data());
        e = cudaMemcpy(h->fc_w5img, fimg.data(), fimg.size(), cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = fc_tc_setup();
      }
    }
  }
  // cudaMemcpy from pageable memory returns once the data is staged, not once the DMA has finished, and the caller's
  // (non-blocking) streams are not ordered against the legacy stream: make every upload visible before anything
  // reads it (create is not on the hot path)
  if (e == cudaSuccess) e = cudaDeviceSynchronize();
  if (e == cudaSuccess && cfg->elide_empty_intervals) {
    // UNet(0): one event's worth of zero histograms through the very kernel pvf_run uses, on a private
    // stream (create is not on the hot path); every interval of it is the constant vector
    cudaStream_t cs = nullptr;
    e = cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaMemsetAsync(h->hist, 0, sizeof(float) * kIntervals * kFcOut, cs);
    if (e == cudaSuccess) {
      enqueue_unet(h, h->hist, 1, h->el_p0, cs);
      e = cudaStreamSynchronize(cs);
    }
    if (cs) cudaStreamDestroy(cs);
  }
  if (e == cudaSuccess && cfg->enable_host_io) {
    e = cudaStreamCreateWithFlags(&h->s_in, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->s_out, cudaStreamNonBlocking);
    for (int k = 0; k < pvf_ctx::kHostChunks && e == cudaSuccess; ++k) {
      e = cudaEventCreateWithFlags(&h->ev_in[k], cudaEventDisableTiming);
      if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_comp[k], cudaEventDisableTiming);
    }
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_join, cudaEventDisableTiming);
  }
  if (e == cudaSuccess && cfg->enable_stage_timing)
    for (int r = 0; r < pvf_ctx::kTimedRuns; ++r)
      for (int k = 0; k < 5 && e == cudaSuccess; ++k) e = cudaEventCreate(&h->ev[r][k]);
  if (e != cudaSuccess) {
    fprintf(stderr, "pvf_create: %s\n", cudaGetErrorString(e));
    pvf_destroy(h);
    return PVF_ERR_CUDA;         // unsupported configurations were rejected by config_ok: this is a runtime failure
  }
  *out = h;
  return PVF_OK;
}

void enqueue_unet(pvf_ctx* h, const float* hist, int n_events, float* out_probs, cudaStream_t s, const int* list,
                  const int* n_list, const int* seg_cnt, bool pdl) {
  const int n_int = n_events * kIntervals;
  if (!uses_tc(&h->cfg))
    launch_unet_simt(hist, n_int, h->conv_ptrs, h->cfg.unet_channels, out_probs, pdl, s);
  else
    launch_unet_tc(hist, n_int, h->tc_packed, h->cfg.unet_channels, h->cfg.precision, h->cfg.split_mask,
                   h->cfg.unet_cta_pair, out_probs, h->sm_count, list, n_list, seg_cnt, pdl, s);
}

}  // namespace

// read-only view of a handle for pvf_noalloc.cu (new code only; nothing above uses these)
namespace pvf {
bool handle_view(pvf_handle h, HandleView* v) {
  if (!h || !v) return false;
  v->fc_params = h->fc_params;
  v->device = h->device;
  v->sm_count = h->sm_count;
  v->mfrac = h->cfg.boundary_margin_mm * 0.1f;
  return true;
}
void handle_set_error(pvf_handle h, const char* text) {
  if (h) h->cuda_err = text ? text : "";
}
}  // namespace pvf

extern "C" {

void pvf_default_config(pvf_config* c, int32_t max_events, int64_t max_tracks) {
  if (!c) return;
  memset(c, 0, sizeof(*c));
  c->n_intervals = kIntervals; c->n_bins = kBins; c->z_min_mm = -200.0f; c->bin_width_mm = 0.1f;
  c->fc_in = kFcIn; c->fc_hidden = kFcHidden; c->hist_channels = kHistCh; c->unet_channels = 64;
  c->k_e1 = 25; c->k_e2 = 15; c->k_b = 5; c->k_d2 = 15; c->k_d1 = 25;
  c->leaky_slope = kLeaky; c->peak_threshold = 0.01f; c->peak_halfwidth = kPeakHalf; c->max_peaks = kMaxPeaks;
  c->precision = PVF_PREC_FP32; c->split_mask = 0;
  c->max_events = max_events; c->max_tracks = max_tracks;
  c->enable_stage_timing = 0; c->enable_host_io = 0; c->elide_empty_intervals = 0; c->boundary_margin_mm = 0.0f;
  c->unet_cta_pair = 0;
  c->l2_chunk_events = 0;
}

size_t pvf_workspace_bytes(const pvf_config* cfg) {
  if (!config_ok(cfg)) return 0;
  return make_layout(cfg).total;
}

pvf_status pvf_create(const pvf_weights* w, const pvf_config* cfg, pvf_handle* out) {
  return create_impl(w, cfg, nullptr, 0, out);
}

pvf_status pvf_create_in_pool(const pvf_weights* w, const pvf_config* cfg, void* dev_pool, size_t pool_bytes,
                              pvf_handle* out) {
  if (!dev_pool) return PVF_ERR_ARG;
  return create_impl(w, cfg, dev_pool, pool_bytes, out);
}

pvf_status pvf_run(pvf_handle h, const pvf_tracks* t, int32_t n_events, float* out_probs,
                   const pvf_peaks* pk, void* cuda_stream) {
  if (!h || !t || !cuda_stream || n_events < 0) return PVF_ERR_ARG;
  if (n_events == 0) return PVF_OK;
  if (!out_probs || !peaks_ok(pk) || !t->event_offsets || t->n_tracks < 0) return PVF_ERR_ARG;
  for (int k = 0; k < 9; ++k)
    if (!t->feat[k] && t->n_tracks > 0) return PVF_ERR_ARG;
  if (n_events > h->cfg.max_events || t->n_tracks > h->cfg.max_tracks) return PVF_ERR_CAPACITY;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const bool timing = h->cfg.enable_stage_timing != 0 && !h->suppress_timing;
  cudaEvent_t* ev = h->ev[h->timed_runs % pvf_ctx::kTimedRuns];
  // Programmatic dependent launch (pdl.cuh) chains the kernels of the run: each may start while its predecessor still
  // runs and does its weight-only prologue before it waits for it.  Not with stage timing (an event record between two
  // kernels orders them completely anyway) and not in the elision mode (a memset sits in the chain).
  const bool pdl = !timing && !h->cfg.elide_empty_intervals;
  const bool tc = uses_tc(&h->cfg);
  if (timing) cudaEventRecord(ev[0], s);
  launch_sort(t->feat[0], t->event_offsets, n_events, (int)t->n_tracks, h->perm, h->seg_off, h->seg_cnt, h->flags,
              h->cfg.boundary_margin_mm * 0.1f, s);
  if (timing) cudaEventRecord(ev[1], s);
  // FC + segmented sum, then the UNet -- over the whole batch, or (l2_chunk_events > 0) chunk by chunk through ONE
  // chunk-sized histogram buffer, so that the histograms are written and read back while they are still in the L2
  // cache and never travel to HBM ("memory layout fusion ... explicit workspace reuse"; NEXT-2).
  const int chunk = h->hist_events < n_events ? h->hist_events : n_events;
  float* dump = h->hist + (size_t)h->hist_events * kIntervals * kFcOut;
  if (timing && chunk < n_events) cudaEventRecord(ev[2], s);   // chunked: FC and UNet interleave, their sum is reported as "UNet"
  for (int e0 = 0; e0 < n_events; e0 += chunk) {
    const int ne = n_events - e0 < chunk ? n_events - e0 : chunk;
    const int32_t* so = h->seg_off + (size_t)e0 * kIntervals;
    const int32_t* sc = h->seg_cnt + (size_t)e0 * kIntervals;
    if (!tc)
      launch_fc_hist(t->feat, t->event_offsets, h->perm, so, sc, h->fc_params, ne, h->hist, h->sm_count, pdl, s);
    else
      launch_fc_hist_tc(t->feat, t->event_offsets, h->perm, so, sc, h->fc_params, h->fc_w5img, ne, h->hist, dump,
                        h->sm_count, pdl, s);
    if (timing && chunk >= n_events) cudaEventRecord(ev[2], s);
    float* po = out_probs + (size_t)e0 * kGlobalBins;
    if (h->cfg.elide_empty_intervals) {
      launch_compact_fill(sc, ne * kIntervals, h->el_list, h->el_count, h->el_p0, po, s);
      enqueue_unet(h, h->hist, ne, po, s, h->el_list, h->el_count);   // the list holds non-empty intervals only
    } else {
      // tensor-core modes: k_fc_hist_tc leaves the histograms of empty intervals unwritten, the UNet takes them as zeros
      enqueue_unet(h, h->hist, ne, po, s, nullptr, nullptr, tc ? sc : nullptr, pdl);
    }
  }
  if (timing) cudaEventRecord(ev[3], s);
  launch_peaks(out_probs, n_events, h->cfg.peak_threshold, h->flags, pk->z_mm, pk->prob, pk->bin, pk->count,
               pk->event_flags, pdl, s);
  if (timing) { cudaEventRecord(ev[4], s); ++h->timed_runs; }
  h->last_n_events = chunk < n_events ? (n_events - 1) % chunk + 1 : n_events;   // what the histogram buffer holds now
  h->last_e0 = n_events - h->last_n_events;
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) return fail_cuda(h, e, "pvf_run launch");
  return PVF_OK;
}

pvf_status pvf_run_host(pvf_handle h, const pvf_tracks* t, int32_t n_events, float* host_probs,
                        const pvf_peaks* pk, void* cuda_stream) {
  if (!h || !t || !cuda_stream || n_events < 0) return PVF_ERR_ARG;
  if (!h->cfg.enable_host_io) return PVF_ERR_UNSUPPORTED;
  if (n_events == 0) return PVF_OK;
  if (!peaks_ok(pk) || !t->event_offsets || t->n_tracks < 0) return PVF_ERR_ARG;
  if (n_events > h->cfg.max_events || t->n_tracks > h->cfg.max_tracks) return PVF_ERR_CAPACITY;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  const size_t T = (size_t)t->n_tracks, cap = (size_t)h->cfg.max_tracks, E = (size_t)n_events;
  for (int k = 0; k < 9; ++k)
    if (!t->feat[k] && T > 0) return PVF_ERR_ARG;
  // Large batches run as a pipeline of chunks: the H2D copy of chunk k+1 (stream s_in) and the D2H copy of chunk k-1
  // (stream s_out) overlap the kernels of chunk k on the caller's stream.  Track indices stay absolute (the kernels
  // index everything through event_offsets), so a chunk is just a window [e0, e1) of the same arrays.
  const int n_chunks = n_events >= 4096 ? pvf_ctx::kHostChunks : 1;
  const int32_t* off = t->event_offsets;                     // host pointer here
  // the offsets steer the copies below: ascending, starting at 0, ending at n_tracks -- checked before anything is enqueued
  if (off[0] != 0 || (size_t)off[E] != T) return PVF_ERR_ARG;
  for (size_t e = 0; e < E; ++e)
    if (off[e + 1] < off[e]) return PVF_ERR_ARG;
  pvf_tracks d{};
  for (int k = 0; k < 9; ++k) d.feat[k] = h->st_feat + cap * k;
  d.n_tracks = t->n_tracks;
  // A failing CUDA call inside the pipeline must not leave copies into the caller's host buffers in flight or the
  // handle in "chunked" state: every error path goes through the clean-up at the end.
  cudaError_t ce = cudaSuccess;
  const char* where = "";
#define PVF_TRY(call)                                              \
  do {                                                             \
    if (ce == cudaSuccess) { ce = (call); if (ce != cudaSuccess) where = #call; } \
  } while (0)
  if (n_chunks > 1) {
    PVF_TRY(cudaEventRecord(h->ev_fork, s));                 // the copy streams start after what is already queued on s
    PVF_TRY(cudaStreamWaitEvent(h->s_in, h->ev_fork, 0));
    PVF_TRY(cudaStreamWaitEvent(h->s_out, h->ev_fork, 0));
  }
  h->suppress_timing = n_chunks > 1;                         // stage timing describes whole-batch pvf_run calls only
  pvf_status st = PVF_OK;
  for (int c = 0; c < n_chunks && st == PVF_OK && ce == cudaSuccess; ++c) {
    const size_t e0 = E * c / n_chunks, e1 = E * (c + 1) / n_chunks, ne = e1 - e0;
    const size_t t0 = n_chunks > 1 ? (size_t)off[e0] : 0, t1 = n_chunks > 1 ? (size_t)off[e1] : T;
    cudaStream_t si = n_chunks > 1 ? h->s_in : s, so = n_chunks > 1 ? h->s_out : s;
    for (int k = 0; k < 9; ++k)
      if (t1 > t0)
        PVF_TRY(cudaMemcpyAsync(h->st_feat + cap * k + t0, t->feat[k] + t0, sizeof(float) * (t1 - t0), cudaMemcpyHostToDevice, si));
    {   // offsets (e0, e1] -- plus offsets[e0] for the first chunk -- so that no element is copied twice
      const size_t lo = c == 0 ? e0 : e0 + 1;
      PVF_TRY(cudaMemcpyAsync(h->st_off + lo, off + lo, sizeof(int32_t) * (e1 + 1 - lo), cudaMemcpyHostToDevice, si));
    }
    if (n_chunks > 1) {
      PVF_TRY(cudaEventRecord(h->ev_in[c], si));
      PVF_TRY(cudaStreamWaitEvent(s, h->ev_in[c], 0));
    }
    d.event_offsets = h->st_off + e0;
    pvf_peaks dp{h->st_z + e0 * kMaxPeaks, h->st_prob + e0 * kMaxPeaks, h->st_bin + e0 * kMaxPeaks, h->st_count + e0,
                 h->st_flags + e0};
    if (ce != cudaSuccess) break;
    st = pvf_run(h, &d, (int32_t)ne, h->st_probs + e0 * kGlobalBins, &dp, cuda_stream);
    if (st != PVF_OK) break;
    if (n_chunks > 1) {
      PVF_TRY(cudaEventRecord(h->ev_comp[c], s));
      PVF_TRY(cudaStreamWaitEvent(so, h->ev_comp[c], 0));
    }
    if (host_probs)
      PVF_TRY(cudaMemcpyAsync(host_probs + e0 * kGlobalBins, h->st_probs + e0 * kGlobalBins, sizeof(float) * ne * kGlobalBins,
                                  cudaMemcpyDeviceToHost, so));
    PVF_TRY(cudaMemcpyAsync(pk->z_mm + e0 * kMaxPeaks, dp.z_mm, sizeof(float) * ne * kMaxPeaks, cudaMemcpyDeviceToHost, so));
    PVF_TRY(cudaMemcpyAsync(pk->prob + e0 * kMaxPeaks, dp.prob, sizeof(float) * ne * kMaxPeaks, cudaMemcpyDeviceToHost, so));
    PVF_TRY(cudaMemcpyAsync(pk->bin + e0 * kMaxPeaks, dp.bin, sizeof(int32_t) * ne * kMaxPeaks, cudaMemcpyDeviceToHost, so));
    PVF_TRY(cudaMemcpyAsync(pk->count + e0, dp.count, sizeof(int32_t) * ne, cudaMemcpyDeviceToHost, so));
    if (pk->event_flags)
      PVF_TRY(cudaMemcpyAsync(pk->event_flags + e0, dp.event_flags, sizeof(uint32_t) * ne, cudaMemcpyDeviceToHost, so));
  }
  h->suppress_timing = false;
  if (n_chunks > 1) {                                        // join: the caller's stream is ordered after both copy streams
    PVF_TRY(cudaEventRecord(h->ev_join, h->s_out));
    PVF_TRY(cudaStreamWaitEvent(s, h->ev_join, 0));
    PVF_TRY(cudaEventRecord(h->ev_join, h->s_in));
    PVF_TRY(cudaStreamWaitEvent(s, h->ev_join, 0));
  }
  PVF_TRY(cudaStreamSynchronize(s));
#undef PVF_TRY
  if (ce != cudaSuccess || st != PVF_OK) {                   // nothing may still be writing the caller's buffers
    cudaStreamSynchronize(s);
    if (h->s_in) cudaStreamSynchronize(h->s_in);
    if (h->s_out) cudaStreamSynchronize(h->s_out);
    if (ce != cudaSuccess) return fail_cuda(h, ce, where);
    return st;
  }
  if (st == PVF_OK) h->last_n_events = n_chunks > 1 ? (int32_t)(E - E * (n_chunks - 1) / n_chunks) : n_events;
  return st;
}

pvf_status pvf_find_peaks(pvf_handle h, const float* probs, int32_t n_events, const pvf_peaks* pk, void* cuda_stream) {
  if (!h || !cuda_stream || n_events < 0) return PVF_ERR_ARG;
  if (n_events == 0) return PVF_OK;
  if (!probs || !peaks_ok(pk)) return PVF_ERR_ARG;
  launch_peaks(probs, n_events, h->cfg.peak_threshold, nullptr, pk->z_mm, pk->prob, pk->bin, pk->count,
               pk->event_flags, false, static_cast<cudaStream_t>(cuda_stream));
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) return fail_cuda(h, e, "pvf_find_peaks launch");
  return PVF_OK;
}

pvf_status pvf_run_unet(pvf_handle h, const float* hist, int32_t n_events, float* out_probs, void* cuda_stream) {
  if (!h || !cuda_stream || n_events < 0) return PVF_ERR_ARG;
  if (n_events == 0) return PVF_OK;
  if (!hist || !out_probs) return PVF_ERR_ARG;
  if (n_events > h->cfg.max_events) return PVF_ERR_CAPACITY;
  enqueue_unet(h, hist, n_events, out_probs, static_cast<cudaStream_t>(cuda_stream));
  cudaError_t e = cudaPeekAtLastError();
  if (e != cudaSuccess) return fail_cuda(h, e, "pvf_run_unet launch");
  return PVF_OK;
}

pvf_status pvf_debug_copy_histogram(pvf_handle h, float* dev_out, int32_t n_events, void* cuda_stream) {
  if (!h || !dev_out || !cuda_stream || n_events < 0) return PVF_ERR_ARG;
  if (n_events > h->last_n_events) return PVF_ERR_ARG;
  if (n_events == 0) return PVF_OK;
  if (!uses_tc(&h->cfg)) {
    PVF_CUDA(h, cudaMemcpyAsync(dev_out, h->hist, sizeof(float) * (size_t)n_events * kIntervals * kFcOut,
                                cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(cuda_stream)));
  } else {   // the tensor-core FC kernel writes non-empty intervals only: empty ones are zeros by definition
    launch_copy_hist_masked(h->hist, h->seg_cnt + (size_t)h->last_e0 * kIntervals, n_events * kIntervals, dev_out,
                            static_cast<cudaStream_t>(cuda_stream));
    PVF_CUDA(h, cudaPeekAtLastError());
  }
  return PVF_OK;
}

pvf_status pvf_stage_times_ms(pvf_handle h, float out_ms[4]) {
  if (!h || !out_ms) return PVF_ERR_ARG;
  if (!h->cfg.enable_stage_timing || h->timed_runs == 0) return PVF_ERR_UNSUPPORTED;
  const int64_t n = h->timed_runs < pvf_ctx::kTimedRuns ? h->timed_runs : pvf_ctx::kTimedRuns;
  double acc[4] = {0, 0, 0, 0};
  for (int64_t r = h->timed_runs - n; r < h->timed_runs; ++r) {
    cudaEvent_t* ev = h->ev[r % pvf_ctx::kTimedRuns];
    for (int k = 0; k < 4; ++k) {
      float ms = 0.f;
      PVF_CUDA(h, cudaEventElapsedTime(&ms, ev[k], ev[k + 1]));
      acc[k] += ms;
    }
  }
  for (int k = 0; k < 4; ++k) out_ms[k] = (float)(acc[k] / (double)n);
  h->timed_runs = 0;
  return PVF_OK;
}

int32_t pvf_launches_per_run(pvf_handle h, int32_t n_events) {
  if (!h || n_events <= 0) return 0;
  const int chunks = (n_events + h->hist_events - 1) / h->hist_events;   // 1 unless l2_chunk_events splits the batch
  return 1 /*sort*/ + chunks * (fc_hist_launches(n_events) + 1 /*unet*/ +
                                (h->cfg.elide_empty_intervals ? 2 /*work list, constant fill*/ : 0)) + 1 /*peaks*/;
}

pvf_status pvf_destroy(pvf_handle h) {
  if (!h) return PVF_ERR_ARG;
  for (int r = 0; r < pvf_ctx::kTimedRuns; ++r)
    for (int k = 0; k < 5; ++k)
      if (h->ev[r][k]) cudaEventDestroy(h->ev[r][k]);
  for (int k = 0; k < pvf_ctx::kHostChunks; ++k) {
    if (h->ev_in[k]) cudaEventDestroy(h->ev_in[k]);
    if (h->ev_comp[k]) cudaEventDestroy(h->ev_comp[k]);
  }
  if (h->ev_fork) cudaEventDestroy(h->ev_fork);
  if (h->ev_join) cudaEventDestroy(h->ev_join);
  if (h->s_in) cudaStreamDestroy(h->s_in);
  if (h->s_out) cudaStreamDestroy(h->s_out);
  if (h->owns_pool && h->pool) cudaFree(h->pool);
  delete h;
  return PVF_OK;
}

const char* pvf_status_string(pvf_status s) {
  switch (s) {
    case PVF_OK: return "PVF_OK";
    case PVF_ERR_ARG: return "PVF_ERR_ARG";
    case PVF_ERR_CONFIG: return "PVF_ERR_CONFIG";
    case PVF_ERR_CAPACITY: return "PVF_ERR_CAPACITY";
    case PVF_ERR_CUDA: return "PVF_ERR_CUDA";
    case PVF_ERR_UNSUPPORTED: return "PVF_ERR_UNSUPPORTED";
  }
  return "PVF_ERR_?";
}

const char* pvf_last_cuda_error(pvf_handle h) { return h ? h->cuda_err.c_str() : ""; }

const char* pvf_build_info(void) {
  return "pvfinder-b200 sm_100a nvcc " __VERSION__ " cuda " PVF_STR(CUDART_VERSION);
}

}  // extern "C"
