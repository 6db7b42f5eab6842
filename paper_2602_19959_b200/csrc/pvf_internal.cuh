// Internal declarations shared by the kernels and the C-ABI glue (pvf_api.cu).
// The geometry is frozen (include/pvf.h marks the fields "fixed"), BASELINE.json config 0.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "../../include/pvf.h"

namespace pvf {

constexpr int kIntervals = 40;
constexpr int kBins = 100;
constexpr int kGlobalBins = kIntervals * kBins;  // 4000
constexpr int kFcIn = 9;
constexpr int kFcHidden = 25;
constexpr int kHistCh = 8;
constexpr int kFcOut = kHistCh * kBins;          // 800
constexpr int kMaxPeaks = 32;
constexpr int kPeakHalf = 3;
constexpr float kLeaky = 0.01f;

// Packed FC parameters in device memory (floats), see pack_fc() in pvf_api.cu:
//   [0,225)      W0 [25][9]        [225,250)    b0
//   250 + 650*k  W_{k+1} [25][25], then b_{k+1} [25]      (k = 0..3)
//   2850         W5 [800][25]      22850        b5 [800]
constexpr int kFcW0 = 0, kFcB0 = 225, kFcHid = 250, kFcHidStride = 650;
constexpr int kFcW5 = 2850, kFcB5 = 22850, kFcTotal = 23650;

struct ConvShape { int cin, cout, k, len; };

#ifdef __CUDACC__
// DESIGN.md reading O2 (float32, separately rounded add and multiply, no FMA):
//   u = (z + 200f) * 0.1f;  i = floor(u);  zrel = u - i  (exact);  dropped if non-finite or i outside [0,40).
__device__ __forceinline__ int interval_of(float z, float& zrel, bool& nonfinite) {
  nonfinite = !isfinite(z);
  zrel = 0.0f;
  if (nonfinite) return -1;
  const float u = __fmul_rn(__fadd_rn(z, 200.0f), 0.1f);
  const float fl = floorf(u);
  if (!(fl >= 0.0f && fl < (float)kIntervals)) return -1;
  zrel = __fsub_rn(u, fl);
  return (int)fl;
}
// NEXT-1 ("tracks on boundaries of intervals are part of two intervals"; reading R12):
// with margin fraction mfrac = margin_mm * 0.1f > 0 a kept track with zrel < mfrac also contributes to the
// previous interval (zrel + 1), one with zrel >= 1 - mfrac to the next (zrel - 1).  A perm entry carries the
// track index in bits [0,29) and in bits [29,31) which contribution it is: 0 own interval, 1 previous, 2 next.
constexpr int kEntryShift = 29;
constexpr int kEntryMask = (1 << kEntryShift) - 1;
__device__ __forceinline__ int neighbour_code(int iv, float zrel, float mfrac) {
  if (iv < 0 || !(mfrac > 0.0f)) return 0;
  if (iv > 0 && zrel < mfrac) return 1;
  if (iv < kIntervals - 1 && zrel >= __fsub_rn(1.0f, mfrac)) return 2;
  return 0;
}
// interval and relative z of a perm entry; t = the track it refers to
__device__ __forceinline__ int entry_interval(int ent, const float* __restrict__ z_poca, int& t, float& zrel) {
  t = ent & kEntryMask;
  const int which = ent >> kEntryShift;
  bool nf;
  int iv = interval_of(z_poca[t], zrel, nf);
  if (which == 1) { iv -= 1; zrel = __fadd_rn(zrel, 1.0f); }
  else if (which == 2) { iv += 1; zrel = __fsub_rn(zrel, 1.0f); }
  return iv;
}
#endif

// `pdl` on the launchers below: launch with programmatic stream serialization (pdl.cuh) -- the kernel may start while
// its predecessor on the stream still runs and waits for it (griddepcontrol.wait) before it reads what that one wrote.
// a0: interval assignment + stable per-event counting sort (k_sort.cu).  mfrac > 0: boundary tracks get a
// second entry (perm then holds up to 2 entries per track).
void launch_sort(const float* z_poca, const int32_t* event_offsets, int n_events, int n_tracks, int32_t* perm,
                 int32_t* seg_off, int32_t* seg_cnt, uint32_t* flags, float mfrac, cudaStream_t s);

// a1+a2: per-track FC and fixed-order segmented sum into H [n_events,40,8,100] (k_fc.cu)
void launch_fc_hist(const float* const feat[9], const int32_t* event_offsets, const int32_t* perm,
                    const int32_t* seg_off, const int32_t* seg_cnt, const float* fc_params,
                    int n_events, float* hist, int sm_count, bool pdl, cudaStream_t s);
cudaError_t fc_hist_setup();
int fc_hist_launches(int n_events);

// a1+a2, tensor-core version (k_fc_tc.cu): 25 -> 800 layer as 3-pass TF32 tcgen05 MMAs, sum in the epilogue
size_t fc_tc_packed_bytes();
void fc_tc_pack(const float* w5, const float* b5, void* host_dst);
cudaError_t fc_tc_setup();
void launch_fc_hist_tc(const float* const feat[9], const int32_t* event_offsets, const int32_t* perm,
                       const int32_t* seg_off, const int32_t* seg_cnt, const float* fc_params, const void* w5img,
                       int n_events, float* hist, float* dump, int sm_count, bool pdl, cudaStream_t s);
// dump: kFcDumpFloats floats of scratch that the padding lanes of the accumulator tiles write their sums to
constexpr size_t kFcDumpFloats = (size_t)kIntervals * kFcOut + 1024;

// a3, FP32 CUDA-core path (k_unet_simt.cu).  conv params: PyTorch layout, floats.
struct UnetParamsF32 { const float* w[6]; const float* b[6]; };
cudaError_t unet_simt_setup(int channels);
void launch_unet_simt(const float* hist, int n_intervals_total, const UnetParamsF32& p, int channels,
                      float* probs, bool pdl, cudaStream_t s);

// a3, tcgen05/TMEM path (k_unet_tc.cu)
// cta_pair: 0 = one CTA per MMA (cta_group::1); 1 = clusters of two CTAs sharing every MMA (cta_group::2)
size_t unet_tc_packed_bytes(int channels, int precision, int split_mask, int cta_pair);
// packs PyTorch-layout host weights into the shared-memory image order the kernel streams
void unet_tc_pack(const pvf_weights* w, int channels, int precision, int split_mask, int cta_pair, void* host_dst);
cudaError_t unet_tc_setup(int channels, int precision, int split_mask, int cta_pair);
// list / n_list (device, optional): run only over intervals list[0 .. *n_list) (empty-interval elision)
// seg_cnt (device, optional): tracks per interval; intervals with none are taken as zeros without reading hist
void launch_unet_tc(const float* hist, int n_intervals_total, const void* packed_dev, int channels,
                    int precision, int split_mask, int cta_pair, float* probs, int sm_count, const int* list,
                    const int* n_list, const int* seg_cnt, bool pdl, cudaStream_t s);

// NEXT-2, empty-interval elision (k_compact.cu): work list of non-empty intervals + constant fill of the rest
// canonical histogram out of the pool's: out[n] = seg_cnt[n] > 0 ? hist[n] : 0 (debug accessor, tensor-core modes)
void launch_copy_hist_masked(const float* hist, const int32_t* seg_cnt, int n_total, float* out, cudaStream_t s);
void launch_compact_fill(const int32_t* seg_cnt, int n_total, int32_t* list, int32_t* n_list, const float* p0,
                         float* probs, cudaStream_t s);

// pvf_noalloc.cu (pvf_histogram_noalloc) needs three things of a handle; pvf_ctx itself stays private to pvf_api.cu
struct HandleView { const float* fc_params; int device; int sm_count; float mfrac; };
bool handle_view(pvf_handle h, HandleView* v);
void handle_set_error(pvf_handle h, const char* text);    // what pvf_last_cuda_error returns

// a4: peak finder (k_peaks.cu)
void launch_peaks(const float* probs, int n_events, float threshold, const uint32_t* flags_in,
                  float* z_mm, float* prob, int32_t* bin, int32_t* count, uint32_t* flags_out,
                  bool pdl, cudaStream_t s);

}  // namespace pvf
