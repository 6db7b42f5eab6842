// Empty-interval elision (NEXT-2 of SURVEY.md section 8f; the paper's "memory layout fusion / workspace
// reuse" roadmap, taken one step further): about 60 % of the 40 z-intervals of a Run-3-like
// event hold no track, and every empty interval yields the same 100 probabilities UNet(0).  With
// pvf_config.elide_empty_intervals the UNet runs only over the non-empty intervals and the others get
// the precomputed vector.  This is OUR optimisation, not the method's: bench.py reports it as a separate
// mode with executed-FLOP accounting.  Results are bit-identical to the plain path because an interval's
// output does not depend on which other intervals share its CTA group.
#include "pvf_internal.cuh"

namespace pvf {

constexpr int kCompactThreads = 256;

// list[0 .. *n_list) = indices n (event * 40 + interval) with seg_cnt[n] > 0.  Ascending inside a block's
// range of 256 intervals; blocks append in arrival order (integer atomic on a work list: the ORDER of the
// list does not influence any result).
__global__ void __launch_bounds__(kCompactThreads)
k_compact_nonempty(const int32_t* __restrict__ seg_cnt, int n_total, int32_t* __restrict__ list,
                   int32_t* __restrict__ n_list) {
  __shared__ int s_warp[kCompactThreads / 32];
  __shared__ int s_base;
  const int n = blockIdx.x * kCompactThreads + threadIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool keep = n < n_total && seg_cnt[n] > 0;
  const unsigned m = __ballot_sync(0xffffffffu, keep);
  if (lane == 0) s_warp[warp] = __popc(m);
  __syncthreads();
  if (threadIdx.x == 0) {
    int tot = 0;
    for (int w = 0; w < kCompactThreads / 32; ++w) { const int c = s_warp[w]; s_warp[w] = tot; tot += c; }
    s_base = tot ? atomicAdd(n_list, tot) : 0;
  }
  __syncthreads();
  if (keep) list[s_base + s_warp[warp] + __popc(m & ((1u << lane) - 1u))] = n;
}

// probs[n, 0..100) = p0 for every interval n without tracks (one warp per interval, coalesced).
__global__ void __launch_bounds__(kCompactThreads)
k_fill_empty(const int32_t* __restrict__ seg_cnt, int n_total, const float* __restrict__ p0,
             float* __restrict__ probs) {
  const int n = blockIdx.x * (kCompactThreads / 32) + (threadIdx.x >> 5);
  const int lane = threadIdx.x & 31;
  if (n >= n_total || seg_cnt[n] > 0) return;
  float* dst = probs + (size_t)n * kBins;
  for (int l = lane; l < kBins; l += 32) dst[l] = p0[l];
}

// out[n, 0..800) = seg_cnt[n] > 0 ? hist[n, 0..800) : 0 (one block per interval).
__global__ void __launch_bounds__(200)
k_copy_hist_masked(const float* __restrict__ hist, const int32_t* __restrict__ seg_cnt, float* __restrict__ out) {
  const size_t n = blockIdx.x;
  const bool live = seg_cnt[n] > 0;
  const float4* src = reinterpret_cast<const float4*>(hist + n * kFcOut);
  float4* dst = reinterpret_cast<float4*>(out + n * kFcOut);
  dst[threadIdx.x] = live ? src[threadIdx.x] : make_float4(0.f, 0.f, 0.f, 0.f);
}

void launch_copy_hist_masked(const float* hist, const int32_t* seg_cnt, int n_total, float* out, cudaStream_t s) {
  if (n_total <= 0) return;
  k_copy_hist_masked<<<n_total, 200, 0, s>>>(hist, seg_cnt, out);
}

void launch_compact_fill(const int32_t* seg_cnt, int n_total, int32_t* list, int32_t* n_list, const float* p0,
                         float* probs, cudaStream_t s) {
  if (n_total <= 0) return;
  cudaMemsetAsync(n_list, 0, sizeof(int32_t), s);
  k_compact_nonempty<<<(n_total + kCompactThreads - 1) / kCompactThreads, kCompactThreads, 0, s>>>(seg_cnt, n_total,
                                                                                                   list, n_list);
  const int per_block = kCompactThreads / 32;
  k_fill_empty<<<(n_total + per_block - 1) / per_block, kCompactThreads, 0, s>>>(seg_cnt, n_total, p0, probs);
}

}  // namespace pvf
