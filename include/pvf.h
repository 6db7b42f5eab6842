/* pvf.h -- C ABI of the B200-native PVFinder inference hot path.
 *
 * What it computes (section 2, lines 27-31; sizes from BASELINE.json config 0):
 *   tracks (9 features, SoA) -> per-track 6-layer FC 9->25x5->800 -> deterministic sum into one
 *   [8,100] histogram for each of the 40 z-intervals of every event -> 1D UNet (64 channels) per
 *   interval -> sigmoid -> 4000 probabilities per event -> local-maximum peak finding.
 *
 * Shape of the boundary: a spec frozen at init (the paper's TensorSpec), one
 * workspace pool allocated once (the paper's fixed 16 MB arena), per-call non-owning
 * views of caller-owned SoA buffers (TensorView), a single caller-supplied stream with no
 * allocation, no host synchronisation and no default-stream work inside the call,
 * and a status enum for graceful degradation.
 *
 * All entry points are thread-compatible (one handle = one user at a time).  Unless noted,
 * "device" pointers are CUDA device memory owned by the caller, "host" pointers are ordinary
 * host memory.  No PyTorch types appear here.
 */
#ifndef PVF_H
#define PVF_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define PVF_API __attribute__((visibility("default")))
#else
#define PVF_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pvf_ctx* pvf_handle;

typedef enum {
  PVF_OK = 0,
  PVF_ERR_ARG = 1,         /* NULL / negative / inconsistent argument; nothing enqueued */
  PVF_ERR_CONFIG = 2,      /* configuration not supported by this build */
  PVF_ERR_CAPACITY = 3,    /* n_events > max_events or n_tracks > max_tracks; nothing enqueued */
  PVF_ERR_CUDA = 4,        /* a CUDA runtime call failed (see pvf_last_cuda_error) */
  PVF_ERR_UNSUPPORTED = 5  /* valid request this build cannot serve (e.g. stage timing disabled) */
} pvf_status;

/* Arithmetic of the UNet convolutions.  The peak finder is always FP32; the FC stage is always FP32-accurate:
 * FP32 FMAs in PVF_PREC_FP32, and in the tensor-core modes FP32 FMAs for the 25-wide layers plus a 3-pass
 * TF32 hi/lo split with FP32 accumulation for the 25 -> 800 layer. */
typedef enum {
  PVF_PREC_FP32 = 0, /* FP32-accurate.  With unet_cta_pair = 1: tcgen05 -- every product as a kind::tf32 MMA plus one kind::f16
                        correction MMA on BF16 pieces (~2^-20 relative per product).  With
                        unet_cta_pair = 0: FP32 FMA direct convolution on the CUDA cores, the bisecting reference */
  PVF_PREC_TF32 = 1, /* tcgen05 kind::tf32, operands RN-rounded to TF32, FP32 accumulate in TMEM */
  PVF_PREC_BF16 = 2, /* tcgen05 kind::f16 with BF16 operands, FP32 accumulate in TMEM */
  PVF_PREC_FP16 = 3  /* tcgen05 kind::f16 with FP16 operands (the paper's roadmap precision), FP32 accumulation.
                        Operands are rounded to FP16 with saturation to +-inf beyond 65504: histogram values and activations
                        must stay below that (the synthetic workloads peak at a few hundred); with split_mask = 1 it meets the
                        TF32 tolerance */
} pvf_precision;

/* Bits of pvf_peaks.event_flags (data-dependent anomalies never fail the call: PAPER.md:57). */
#define PVF_FLAG_PEAK_OVERFLOW 1u /* more than max_peaks maxima; the first max_peaks are kept */
#define PVF_FLAG_TRACK_DROPPED 2u /* >=1 track outside [z_min, z_min+400mm) or non-finite */
#define PVF_FLAG_NONFINITE 4u     /* >=1 track with non-finite z_poca */
#define PVF_FLAG_BAD_OFFSETS 8u   /* the event's [event_offsets[e], event_offsets[e+1]) is not an ascending range inside
                                     [0, n_tracks]: it was clamped (no access outside the caller's buffers), the
                                     event's result covers the clamped range only */

/* Frozen at pvf_create (the paper's TensorSpec).  Fields marked (fixed) must hold
 * the stated value in this build, anything else returns PVF_ERR_CONFIG. */
typedef struct {
  int32_t n_intervals;     /* (fixed) 40  -- PAPER.md:27 */
  int32_t n_bins;          /* (fixed) 100 -- PAPER.md:27 */
  float z_min_mm;          /* (fixed) -200 */
  float bin_width_mm;      /* (fixed) 0.1 */
  int32_t fc_in;           /* (fixed) 9   -- PAPER.md:27 */
  int32_t fc_hidden;       /* (fixed) 25 */
  int32_t hist_channels;   /* (fixed) 8   -- PAPER.md:29 */
  int32_t unet_channels;   /* 64 (deployed), 32 or 16 (PAPER.md:84 roadmap) */
  int32_t k_e1, k_e2, k_b, k_d2, k_d1; /* (fixed) 25, 15, 5, 15, 25 */
  float leaky_slope;       /* (fixed) 0.01 */
  float peak_threshold;    /* any finite value; config 0 uses 0.01 */
  int32_t peak_halfwidth;  /* (fixed) 3 */
  int32_t max_peaks;       /* (fixed) 32 */
  int32_t precision;       /* pvf_precision */
  int32_t split_mask;      /* PVF_PREC_TF32 and PVF_PREC_FP16 only (the two formats with a 10-bit mantissa): 0, or 1 = the e1
                              layer (raw histogram input, the dominant error of these formats) runs as two passes on 16-bit
                              pieces (BF16 pieces in the TF32 kernel, FP16 pieces in the FP16 kernel).
                              Anything else is PVF_ERR_CONFIG: FP32 accuracy on every layer is PVF_PREC_FP32, not a mask value */
  int32_t max_events;      /* capacity the pool is sized for (>= 1) */
  int64_t max_tracks;      /* capacity the pool is sized for (>= 1, <= 536 870 911 = 2^29 - 1: the sorted list keeps a track index in 29 bits) */
  int32_t enable_stage_timing; /* pre-creates CUDA events around the four stages; default 0 */
  int32_t enable_host_io;  /* reserve pool space for pvf_run_host's device staging; default 0 */
  int32_t elide_empty_intervals; /* tensor-core kernels only; default 0.  1: the UNet runs only over intervals that
                              hold at least one track, every empty interval gets the precomputed vector
                              UNet(0) -- bit-identical output, fewer executed FLOPs (our optimisation, not the
                              method's: SURVEY.md section 8f NEXT-2; reported separately by bench.py) */
  float boundary_margin_mm; /* default 0 = "each track adds to the interval holding its z_poca" (BASELINE.json
                              config 0).  > 0 (< 4.9): a track within this distance of an interval edge also
                              contributes to the neighbouring interval, PAPER.md:49 (NEXT-1; R12) */
  int32_t unet_cta_pair;   /* default 0 (with PVF_PREC_FP32, 0 also selects the CUDA-core kernels).  1: the UNet kernel runs as clusters of two CTAs that
                              share every tcgen05.mma (cta_group::2, M = 256): each CTA keeps its own intervals'
                              activations and half of the weight rows, so the weight stream and the B-operand
                              reads per SM are halved.  Same arithmetic, bit-identical output */
  int32_t l2_chunk_events; /* default 0 = the histogram buffer holds the whole batch (128 KB per event of pool).  > 0:
                              the pool holds the histograms of this many events only, and pvf_run walks the batch in
                              chunks of that size -- FC + sum of a chunk, then its UNet -- so that the histograms are
                              read back while still in the L2 cache instead of travelling through HBM (PAPER.md:86
                              "memory layout fusion ... explicit workspace reuse").  Identical
                              output.  1024 keeps the non-empty histograms (~52 KB per event) inside the 126 MB L2 */
} pvf_config;

/* Fill *cfg with BASELINE.json config 0 (64 channels, FP32) and the given capacities. */
PVF_API void pvf_default_config(pvf_config* cfg, int32_t max_events, int64_t max_tracks);

/* HOST pointers, PyTorch layouts, float32; copied and re-packed at create, not retained. */
typedef struct {
  const float* fc_w[6];   /* Linear weight [out][in] row-major: 25x9, 4 x 25x25, 800x25 */
  const float* fc_b[6];   /* [out] */
  const float* conv_w[6]; /* Conv1d weight [C_out][C_in][K]; order e1, e2, b, d2, d1, head */
  const float* conv_b[6]; /* [C_out] */
} pvf_weights;

/* DEVICE pointers, caller-owned, read-only: Structure-of-Arrays track buffers. */
typedef struct {
  const float* feat[9];         /* each [n_tracks]: z_poca, x_poca, y_poca, e0..e5 (mm) */
  const int32_t* event_offsets; /* [n_events+1] ascending, offsets[0]=0, offsets[n_events]=n_tracks */
  int64_t n_tracks;             /* host scalar */
} pvf_tracks;

/* DEVICE pointers, caller-owned, written by the call. */
typedef struct {
  float* z_mm;          /* [n_events*max_peaks] centroid z; unused slots 0 */
  float* prob;          /* [n_events*max_peaks] P at the peak bin; unused slots 0 */
  int32_t* bin;         /* [n_events*max_peaks] global bin 0..3999 ascending; unused slots -1 */
  int32_t* count;       /* [n_events] = min(found, max_peaks) */
  uint32_t* event_flags;/* [n_events] PVF_FLAG_* bits; may be NULL */
} pvf_peaks;

/* Bytes of device memory the pool needs for this configuration (0 on invalid config). */
PVF_API size_t pvf_workspace_bytes(const pvf_config* cfg);

/* Create a context: validates cfg, packs the weights, makes ONE cudaMalloc for the pool
 * (weights + sort scratch + histogram + staging).  The current CUDA device is used. */
PVF_API pvf_status pvf_create(const pvf_weights* w, const pvf_config* cfg, pvf_handle* out);

/* Same with a caller-supplied device pool (Allen-style fixed pool): ZERO device
 * allocation.  dev_pool must be 256-byte aligned and hold >= pvf_workspace_bytes(cfg). */
PVF_API pvf_status pvf_create_in_pool(const pvf_weights* w, const pvf_config* cfg, void* dev_pool,
                              size_t pool_bytes, pvf_handle* out);

/* The whole hot path for n_events events, enqueued on cuda_stream (a cudaStream_t; NULL is
 * rejected so that nothing can leak onto the default stream).  No allocation, no
 * host sync.  out_probs: device float [n_events, n_intervals*n_bins]; out_peaks: device views.
 * Errors detectable on the host return non-OK and enqueue nothing; n_events == 0 is a no-op.
 * The call may be captured in a CUDA graph (stream capture on cuda_stream) and replayed on new inputs written into the
 * same buffers: it allocates nothing, never synchronises and touches no other stream; the programmatic dependent launches
 * that chain its kernels become programmatic edges of the graph.  Not with enable_stage_timing (event records). */
PVF_API pvf_status pvf_run(pvf_handle h, const pvf_tracks* tracks, int32_t n_events, float* out_probs,
                   const pvf_peaks* out_peaks, void* cuda_stream);

/* Same computation with HOST buffers: H2D of the nine feature arrays + offsets, pvf_run, D2H of
 * probabilities (skipped if host_probs == NULL) and peaks, then one stream synchronise.  Needs
 * enable_host_io.  feat/event_offsets/peaks fields are host pointers here (pinned memory makes the
 * copies asynchronous but is not required; event_offsets[0] must be 0 and event_offsets[n_events] ==
 * n_tracks).  Batches of >= 4096 events run as a pipeline of 8 chunks: the copies use two streams the
 * library created at pvf_create (ordered after / before cuda_stream by events), so that H2D of chunk
 * k+1 and D2H of chunk k-1 overlap the kernels of chunk k; results are identical to pvf_run.  After such
 * a call pvf_debug_copy_histogram sees the last chunk only; stage timing is not recorded. */
PVF_API pvf_status pvf_run_host(pvf_handle h, const pvf_tracks* host_tracks, int32_t n_events,
                        float* host_probs, const pvf_peaks* host_peaks, void* cuda_stream);

/* Peak finder alone on caller-supplied device probabilities [n_events, 4000] (the bit-exactness
 * test of BASELINE.json north_star runs through this entry point). */
PVF_API pvf_status pvf_find_peaks(pvf_handle h, const float* probs, int32_t n_events,
                          const pvf_peaks* out_peaks, void* cuda_stream);

/* UNet + sigmoid alone on a caller-supplied device histogram [n_events,40,8,100] (canonical
 * [B,C,L] layout of PAPER.md:31) -> out_probs [n_events,4000].  Test/diagnostic entry point. */
PVF_API pvf_status pvf_run_unet(pvf_handle h, const float* hist, int32_t n_events, float* out_probs,
                        void* cuda_stream);

/* Copy the histogram of the last pvf_run ([n_events,40,8,100] float, canonical layout) into
 * dev_out, enqueued on cuda_stream.  In the tensor-core modes the pool holds the histograms of the
 * intervals with at least one track only (the UNet kernel takes the others as zeros without reading
 * them); this accessor fills the empty intervals with zeros, so dev_out is always the canonical H.  With
 * l2_chunk_events the buffer holds the LAST chunk of the run only (n_events must not exceed its size). */
PVF_API pvf_status pvf_debug_copy_histogram(pvf_handle h, float* dev_out, int32_t n_events, void* cuda_stream);

/* a0 + a1 + a2 (interval sort, per-track FC, ordered segmented sum; BASELINE.json config 0) for a
 * SMALL batch with NO allocation anywhere in the call: for callers that cannot call cudaMalloc or supply a pool
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  The scratch the two kernels need
 * (the sorted track list perm, seg_off, seg_cnt, per-event flags) does not come from the handle's pool but from ONE
 * file-scope static __device__ array of PVF_NOALLOC_SCRATCH_BYTES (about 149 KB) that every GPU which loads the
 * library holds until the process exits.  Limits: n_events <= PVF_NOALLOC_MAX_EVENTS and n_tracks <=
 * PVF_NOALLOC_MAX_TRACKS, whatever the handle's max_events / max_tracks; beyond them the call returns
 * PVF_ERR_CAPACITY, enqueues nothing and leaves the reason in pvf_last_cuda_error(h).
 *   h              any handle of the current device; only its FC weights (device, uploaded by pvf_create) and its
 *                  boundary_margin_mm are used.  Always runs the FP32 CUDA-core kernels (k_sort, k_fc_hist), whatever
 *                  the handle's precision: the result equals the histogram of a PVF_PREC_FP32 / unet_cta_pair = 0 handle bit
 *                  for bit and that of every other mode within 2e-5 relative to max(|H|, 1).
 *   tracks         device views, as for pvf_run
 *   dev_hist       device float [n_events, 40, 8, 100], canonical layout, every element written (empty intervals = 0)
 *   dev_event_flags  device uint32 [n_events] or NULL: PVF_FLAG_TRACK_DROPPED / NONFINITE / BAD_OFFSETS per event
 *   cuda_stream    a cudaStream_t, not NULL; two kernels are enqueued on it, no host synchronisation
 * The first call on a device resolves the array's device address (cudaGetSymbolAddress, once per device, with that
 * device current -- it may load the module, so make it outside a capture); later calls only launch.  Nothing in the
 * array has to start at zero (every word a call reads it has written before), so it is never cleared and keeps the last
 * call's contents.  ALL calls share the array: two calls that overlap on the GPU (different streams, or different handles)
 * race on it -- keep them on one stream or order them with events.  PVF_ERR_ARG if the current device is not the handle's. */
#define PVF_NOALLOC_MAX_EVENTS 64
#define PVF_NOALLOC_MAX_TRACKS 16384
#define PVF_NOALLOC_SCRATCH_BYTES (2 * 4 * PVF_NOALLOC_MAX_TRACKS + 2 * 4 * 40 * PVF_NOALLOC_MAX_EVENTS + 4 * PVF_NOALLOC_MAX_EVENTS + 768)
PVF_API pvf_status pvf_histogram_noalloc(pvf_handle h, const pvf_tracks* tracks, int32_t n_events, float* dev_hist,
                                         uint32_t* dev_event_flags, void* cuda_stream);

/* Mean stage times in ms over the pvf_run calls made since the previous call of this function (at
 * most the 64 most recent): [0] interval sort, [1] FC + segmented sum, [2] UNet, [3] peaks; measured
 * with CUDA events recorded on the run's stream.  Caller must have synchronised that stream.
 * Needs enable_stage_timing; PVF_ERR_UNSUPPORTED if no run was recorded. */
PVF_API pvf_status pvf_stage_times_ms(pvf_handle h, float out_ms[4]);

/* Number of KERNELS pvf_run enqueues for n_events (host arithmetic; for launch accounting).  The elision mode also enqueues one
 * 4-byte cudaMemsetAsync per chunk (the work-list counter), which is not a kernel and is not counted. */
PVF_API int32_t pvf_launches_per_run(pvf_handle h, int32_t n_events);

PVF_API pvf_status pvf_destroy(pvf_handle h);

PVF_API const char* pvf_status_string(pvf_status s);
PVF_API const char* pvf_last_cuda_error(pvf_handle h); /* "" if none */
PVF_API const char* pvf_build_info(void);              /* arch + compiler string of this library */

#ifdef __cplusplus
}
#endif
#endif /* PVF_H */
