// a0 -- interval assignment + stable per-event counting sort of tracks by z-interval.
//
// PAPER.md:27 (40 intervals x 100 bins over 400 mm), BASELINE.json config 0 ("Each track adds to the
// interval holding its z_poca"), north_star (b) "tracks are sorted by interval and summed in a fixed
// order".  The float32 recipe (reading O2): u = (z + 200f) * 0.1f with separately rounded
// add and multiply, i = floor(u); a track is dropped when z is non-finite or i is outside [0, 40).
//
// One warp per event.  Output: perm[event_offsets[e] + k] = original track index of the k-th kept
// track of event e in (interval, original index) order; seg_off/seg_cnt[e*40 + i] = start (absolute
// index into perm) and length of interval i's run.  Integer shared-memory atomics only count;
// placement uses match/ballot ranks, so the order is the stable one and is reproducible.
#include "pvf_internal.cuh"
#include "pdl.cuh"

namespace pvf {

constexpr int kSortWarps = 4;

__global__ void __launch_bounds__(kSortWarps * 32)
k_sort(const float* __restrict__ z_poca, const int32_t* __restrict__ event_offsets, int n_events,
       int32_t* __restrict__ perm, int32_t* __restrict__ seg_off, int32_t* __restrict__ seg_cnt,
       uint32_t* __restrict__ flags, float mfrac, int two, int n_tracks) {
  __shared__ int s_cnt[kSortWarps][kIntervals];
  __shared__ int s_base[kSortWarps][kIntervals];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int e = blockIdx.x * kSortWarps + warp;
  pdl_launch_dependents();     // the FC kernel may start its prologue (weights to shared memory) now; it waits for
                               // this grid's completion before it reads perm / seg_off / seg_cnt (pdl.cuh)
  if (e >= n_events) return;   // whole warp exits together; no block-level barrier below
  int* cnt = s_cnt[warp];
  int* base = s_base[warp];
  for (int i = lane; i < kIntervals; i += 32) cnt[i] = 0;
  __syncwarp();
  // The offsets are device data the host never sees (data-dependent anomalies degrade per event, they do
  // not fail the call): a range that is not inside [0, n_tracks] or not ascending is clamped -- nothing is ever read
  // or written outside feat[] / perm[] -- and the event is flagged.
  const int lo_raw = event_offsets[e], hi_raw = event_offsets[e + 1];
  const int lo = min(max(lo_raw, 0), n_tracks), hi = min(max(hi_raw, lo), n_tracks);
  const int plo = two ? 2 * lo : lo;        // start of the event's run in perm (two slots per track with NEXT-1)
  uint32_t fl = (lo != lo_raw || hi != hi_raw) ? PVF_FLAG_BAD_OFFSETS : 0u;
  for (int t = lo + lane; t < hi; t += 32) {
    bool nf;
    float zr;
    int iv = interval_of(z_poca[t], zr, nf);
    if (iv >= 0) {
      atomicAdd(&cnt[iv], 1);
      const int nb = neighbour_code(iv, zr, mfrac);      // NEXT-1: boundary tracks count twice
      if (nb) atomicAdd(&cnt[nb == 1 ? iv - 1 : iv + 1], 1);
    } else fl |= PVF_FLAG_TRACK_DROPPED | (nf ? PVF_FLAG_NONFINITE : 0u);
  }
  fl = __reduce_or_sync(0xffffffffu, fl);
  __syncwarp();
  // exclusive scan of the 40 counts (lane handles i = lane and i = lane + 32)
  int c0 = cnt[lane];
  int c1 = (lane + 32 < kIntervals) ? cnt[lane + 32] : 0;
  int s0 = c0;
  for (int d = 1; d < 32; d <<= 1) {
    int v = __shfl_up_sync(0xffffffffu, s0, d);
    if (lane >= d) s0 += v;
  }
  int tot0 = __shfl_sync(0xffffffffu, s0, 31);
  int s1 = c1;
  for (int d = 1; d < 32; d <<= 1) {
    int v = __shfl_up_sync(0xffffffffu, s1, d);
    if (lane >= d) s1 += v;
  }
  base[lane] = s0 - c0;
  seg_off[(size_t)e * kIntervals + lane] = plo + s0 - c0;
  seg_cnt[(size_t)e * kIntervals + lane] = c0;
  if (lane + 32 < kIntervals) {
    base[lane + 32] = tot0 + s1 - c1;
    seg_off[(size_t)e * kIntervals + lane + 32] = plo + tot0 + s1 - c1;
    seg_cnt[(size_t)e * kIntervals + lane + 32] = c1;
  }
  if (lane == 0) flags[e] = fl;
  __syncwarp();
  // stable placement, 32 tracks at a time in original order
  if (!two) {
    for (int c = lo; c < hi; c += 32) {
      const int t = c + lane;
      int key = -1;
      if (t < hi) { bool nf; float zr; key = interval_of(z_poca[t], zr, nf); }
      const unsigned grp = __match_any_sync(0xffffffffu, key);
      const int rank = __popc(grp & ((1u << lane) - 1u));
      int pos = -1;
      if (key >= 0) pos = lo + base[key] + rank;
      __syncwarp();
      if (key >= 0 && rank == 0) base[key] += __popc(grp);
      __syncwarp();
      if (pos >= 0) perm[pos] = t;
    }
  } else {
    // NEXT-1: a lane holds up to two keys (its interval and a neighbour); per interval the entries of the
    // chunk are placed in lane (= track) order, so the order inside a segment stays "ascending track index"
    for (int c = lo; c < hi; c += 32) {
      const int t = c + lane;
      int key = -1, key2 = -1, code = 0;
      if (t < hi) {
        bool nf;
        float zr;
        key = interval_of(z_poca[t], zr, nf);
        code = neighbour_code(key, zr, mfrac);
        if (code) key2 = code == 1 ? key - 1 : key + 1;
      }
      const unsigned present = __ballot_sync(0xffffffffu, key >= 0);
      if (present == 0u) continue;
      for (int k = 0; k < kIntervals; ++k) {
        const bool mine = key == k, mine2 = key2 == k;
        const unsigned m = __ballot_sync(0xffffffffu, mine || mine2);
        if (m == 0u) continue;
        if (mine || mine2) perm[plo + base[k] + __popc(m & ((1u << lane) - 1u))] = t | ((mine ? 0 : code) << kEntryShift);
        __syncwarp();
        if (lane == 0) base[k] += __popc(m);
        __syncwarp();
      }
    }
  }
}

void launch_sort(const float* z_poca, const int32_t* event_offsets, int n_events, int n_tracks, int32_t* perm,
                 int32_t* seg_off, int32_t* seg_cnt, uint32_t* flags, float mfrac, cudaStream_t s) {
  if (n_events <= 0) return;
  const int grid = (n_events + kSortWarps - 1) / kSortWarps;
  k_sort<<<grid, kSortWarps * 32, 0, s>>>(z_poca, event_offsets, n_events, perm, seg_off, seg_cnt, flags, mfrac,
                                          mfrac > 0.0f ? 1 : 0, n_tracks);
}

}  // namespace pvf
