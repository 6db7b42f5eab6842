// a4 -- peak finder over the 4000 concatenated bins of each event.
//
// PAPER.md:31 "local maximum detection with learned thresholds", PAPER.md:55 (reads the CNN output
// in place); BASELINE.json config 0: prob > 0.01, z = weighted centroid over +-3 bins, at most 32
// peaks per event; north_star: "The peak finder run on identical input probabilities must be
// bit-exact".  Definition (reading O7), all in float32 with round-to-nearest single
// operations (no FMA contraction):
//   peak at g  iff  P[g] > thr  &&  P[g] > P[g-1]  &&  P[g] >= P[g+1]   (out of range = -inf)
//   first 32 in ascending g are kept, count = min(found, 32), overflow flag if found > 32
//   lo = max(g-3,0), hi = min(g+3,3999); s0 = s1 = 0; for j = lo..hi: s0 += P[j]; s1 += P[j]*(j-g)
//   z = ((g + 0.5) + s1/s0) * 0.1 + (-200)
// One warp per event; 32 consecutive bins per step, five steps' loads in flight; ordered compaction by ballot.
#include "pvf_internal.cuh"

namespace pvf {

constexpr int kPeakWarps = 4;

__global__ void __launch_bounds__(kPeakWarps * 32)
k_peaks(const float* __restrict__ probs, int n_events, float thr, const uint32_t* __restrict__ flags_in,
        float* __restrict__ z_mm, float* __restrict__ prob, int32_t* __restrict__ bin,
        int32_t* __restrict__ count, uint32_t* __restrict__ flags_out) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int e = blockIdx.x * kPeakWarps + warp;
  if (e >= n_events) return;
  const float* P = probs + (size_t)e * kGlobalBins;
  const float ninf = __int_as_float(0xff800000);
  int found = 0;
  constexpr int kBatch = 5;                     // 4000 = 25 * 5 * 32: five independent 128-byte loads in flight
  static_assert(kGlobalBins % (32 * kBatch) == 0, "whole batches");   // (25 in flight: 0.107 -> 0.174 ms at 16 k events)
  for (int gb = 0; gb < kGlobalBins; gb += 32 * kBatch) {
    float cv[kBatch];
#pragma unroll
    for (int b = 0; b < kBatch; ++b) cv[b] = P[gb + 32 * b + lane];
    // neighbours across the 32-bin steps: lane 0 needs the last value of the previous step, lane 31 the
    // first of the next one; inside the batch they come from the registers of other lanes
    const float prev_edge = gb > 0 ? P[gb - 1] : ninf;
    const float next_edge = gb + 32 * kBatch < kGlobalBins ? P[gb + 32 * kBatch] : ninf;
#pragma unroll
    for (int b = 0; b < kBatch; ++b) {
      const int g = gb + 32 * b + lane;
      const float c = cv[b];
      float l = __shfl_up_sync(0xffffffffu, c, 1);
      float r = __shfl_down_sync(0xffffffffu, c, 1);
      const float l_in = b > 0 ? __shfl_sync(0xffffffffu, cv[b > 0 ? b - 1 : 0], 31) : prev_edge;
      const float r_in = b + 1 < kBatch ? __shfl_sync(0xffffffffu, cv[b + 1 < kBatch ? b + 1 : b], 0) : next_edge;
      if (lane == 0) l = l_in;
      if (lane == 31) r = r_in;
      const bool is_peak = (c > thr) && (c > l) && (c >= r);
      const unsigned m = __ballot_sync(0xffffffffu, is_peak);
      const int slot = found + __popc(m & ((1u << lane) - 1u));
      if (is_peak && slot < kMaxPeaks) {
        const int lo = max(g - kPeakHalf, 0), hi = min(g + kPeakHalf, kGlobalBins - 1);
        float s0 = 0.0f, s1 = 0.0f;
        for (int j = lo; j <= hi; ++j) {
          const float pj = P[j];
          s0 = __fadd_rn(s0, pj);
          s1 = __fadd_rn(s1, __fmul_rn(pj, (float)(j - g)));
        }
        const float delta = __fdiv_rn(s1, s0);
        const float t = __fadd_rn(__fadd_rn((float)g, 0.5f), delta);
        const float z = __fadd_rn(__fmul_rn(t, 0.1f), -200.0f);
        const size_t o = (size_t)e * kMaxPeaks + slot;
        z_mm[o] = z;
        prob[o] = c;
        bin[o] = g;
      }
      found += __popc(m);
    }
  }
  const int kept = min(found, kMaxPeaks);
  if (lane >= kept) {   // kMaxPeaks == 32 == warp size: lane s clears slot s
    const size_t o = (size_t)e * kMaxPeaks + lane;
    z_mm[o] = 0.0f;
    prob[o] = 0.0f;
    bin[o] = -1;
  }
  if (lane == 0) {
    count[e] = kept;
    if (flags_out) {
      uint32_t f = flags_in ? flags_in[e] : 0u;
      if (found > kMaxPeaks) f |= PVF_FLAG_PEAK_OVERFLOW;
      flags_out[e] = f;
    }
  }
}

void launch_peaks(const float* probs, int n_events, float threshold, const uint32_t* flags_in,
                  float* z_mm, float* prob, int32_t* bin, int32_t* count, uint32_t* flags_out,
                  cudaStream_t s) {
  if (n_events <= 0) return;
  static_assert(kMaxPeaks == 32, "slot clearing assumes one lane per slot");
  const int grid = (n_events + kPeakWarps - 1) / kPeakWarps;
  k_peaks<<<grid, kPeakWarps * 32, 0, s>>>(probs, n_events, threshold, flags_in, z_mm, prob, bin, count, flags_out);
}

}  // namespace pvf
