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
// One CTA of 128 threads per event (one event per thread block).  The event's 4000 probabilities are
// staged in shared memory with coalesced 16-byte loads; thread t then owns the 32 consecutive bins [32 t, 32 t + 32)
// (a padded layout keeps those reads conflict free), counts its maxima, a block-wide exclusive scan turns the counts
// into output slots -- ascending bin order by construction -- and every thread writes the peaks whose slot is < 32.
// One event takes one pass with two block barriers (the first version, one warp walking the 4000 bins, took 23 us
// for a single event).
#include "pvf_internal.cuh"
#include "pdl.cuh"

namespace pvf {

constexpr int kPeakThreads = 128;
constexpr int kPeakRun = 32;                          // consecutive bins per thread: 125 threads x 32 = 4000
static_assert(kGlobalBins % kPeakRun == 0 && kGlobalBins / kPeakRun <= kPeakThreads, "one run per thread");
static_assert(kGlobalBins % 4 == 0, "16-byte loads");

// bin g lives at word g + g / 32: thread t's bins 32 t + j sit in banks (t + j) % 32 -- conflict free for fixed j
__device__ __forceinline__ int pk_slot(int g) { return g + (g >> 5); }

__global__ void __launch_bounds__(kPeakThreads)
k_peaks(const float* __restrict__ probs, int n_events, float thr, const uint32_t* __restrict__ flags_in,
        float* __restrict__ z_mm, float* __restrict__ prob, int32_t* __restrict__ bin,
        int32_t* __restrict__ count, uint32_t* __restrict__ flags_out) {
  __shared__ float sP[kGlobalBins + kGlobalBins / 32];
  __shared__ int s_warp[kPeakThreads / 32];
  const int e = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  pdl_launch_dependents();
  pdl_wait();                                         // the probabilities come from the kernel before this one
  if (e >= n_events) return;
  const float4* P4 = reinterpret_cast<const float4*>(probs + (size_t)e * kGlobalBins);
  constexpr int kLoads = (kGlobalBins / 4 + kPeakThreads - 1) / kPeakThreads;   // 8: all in flight at once (one event: the
  float4 v[kLoads];                                                              // L2 round trips would otherwise add up)
#pragma unroll
  for (int k = 0; k < kLoads; ++k) {
    const int i = tid + k * kPeakThreads;
    if (i < kGlobalBins / 4) v[k] = P4[i];
  }
#pragma unroll
  for (int k = 0; k < kLoads; ++k) {
    const int i = tid + k * kPeakThreads;
    if (i < kGlobalBins / 4) {
      const int s = pk_slot(4 * i);                   // 4 i .. 4 i + 3 never straddle a multiple of 32
      sP[s] = v[k].x; sP[s + 1] = v[k].y; sP[s + 2] = v[k].z; sP[s + 3] = v[k].w;
    }
  }
  __syncthreads();
  const float ninf = __int_as_float(0xff800000);
  const int g0 = tid * kPeakRun;
  const bool has_run = g0 < kGlobalBins;
  // maxima of this thread's run, as a 32-bit mask (bit j = bin g0 + j)
  unsigned mine = 0u;
  if (has_run) {
    float l = g0 > 0 ? sP[pk_slot(g0 - 1)] : ninf;
    float c = sP[pk_slot(g0)];
#pragma unroll 8
    for (int j = 0; j < kPeakRun; ++j) {
      const int g = g0 + j;
      const float r = g + 1 < kGlobalBins ? sP[pk_slot(g + 1)] : ninf;
      if ((c > thr) && (c > l) && (c >= r)) mine |= 1u << j;
      l = c;
      c = r;
    }
  }
  // block-wide exclusive scan of the per-thread counts (thread order = bin order)
  const int cnt = __popc(mine);
  int incl = cnt;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  int before = incl - cnt, found = 0;
#pragma unroll
  for (int w = 0; w < kPeakThreads / 32; ++w) {
    const int t = s_warp[w];
    if (w < warp) before += t;
    found += t;
  }
  // this thread's peaks take slots before, before + 1, ...
  while (mine != 0u && before < kMaxPeaks) {
    const int j = __ffs(mine) - 1;
    mine &= mine - 1u;
    const int g = g0 + j;
    const int lo = max(g - kPeakHalf, 0), hi = min(g + kPeakHalf, kGlobalBins - 1);
    float s0 = 0.0f, s1 = 0.0f;
    for (int k = lo; k <= hi; ++k) {
      const float pj = sP[pk_slot(k)];
      s0 = __fadd_rn(s0, pj);
      s1 = __fadd_rn(s1, __fmul_rn(pj, (float)(k - g)));
    }
    const float delta = __fdiv_rn(s1, s0);
    const float t = __fadd_rn(__fadd_rn((float)g, 0.5f), delta);
    const float z = __fadd_rn(__fmul_rn(t, 0.1f), -200.0f);
    const size_t o = (size_t)e * kMaxPeaks + before;
    z_mm[o] = z;
    prob[o] = sP[pk_slot(g)];
    bin[o] = g;
    ++before;
  }
  const int kept = min(found, kMaxPeaks);
  if (tid < kMaxPeaks && tid >= kept) {               // unused slots
    const size_t o = (size_t)e * kMaxPeaks + tid;
    z_mm[o] = 0.0f;
    prob[o] = 0.0f;
    bin[o] = -1;
  }
  if (tid == 0) {
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
                  bool pdl, cudaStream_t s) {
  if (n_events <= 0) return;
  static_assert(kMaxPeaks <= kPeakThreads, "slot clearing assumes one thread per slot");
  PdlLaunch L(dim3(n_events), dim3(kPeakThreads), 0, s, pdl);
  cudaLaunchKernelEx(&L.cfg, k_peaks, probs, n_events, threshold, flags_in, z_mm, prob, bin, count, flags_out);
}

}  // namespace pvf
