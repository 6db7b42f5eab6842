// a1 + a2 -- per-track fully connected network and deterministic segmented sum into the
// interval histograms H[n_events, 40, 8, 100] (canonical [B, C, L]).
//
// PAPER.md:29 "six FC layers ... combining each track's contribution into a 800-bin histogram
// (8 channels each with 100-bin)"; BASELINE.json config 0: 9->25->25->25->25->25->800,
// LeakyReLU(0.01) hidden, softplus output; north_star (b): sorted by interval, summed in a fixed
// order, no float atomics (PAPER.md:11, 47 determinism).
//
// Mapping: persistent CTAs stride over events.  Per event, tracks are visited in the sorted order
// of a0 in tiles of kThreads: phase A -- thread i runs the five 25-wide layers of sorted track i
// (weights broadcast from shared memory) and parks h[25] in shared memory; phase B -- thread q owns
// outputs o = q + 200*m (m = 0..3) with its four rows of W5 in registers, walks the tile's tracks
// in order, adds softplus(W5 h + b5) into four FP32 accumulators and flushes them to H whenever the
// interval changes.  The 800 contributions per track never touch memory; every H element is written
// exactly once (zeros for empty intervals); the summation order is the sorted order, independent of
// scheduling.
#include "pvf_internal.cuh"
#include "pdl.cuh"

namespace pvf {

constexpr int kFcThreads = 224;     // 7 warps: 200 output owners + 24 spare lanes for phase A
constexpr int kOwners = 200;
constexpr int kHStride = 28;        // h row padded to 7 float4
constexpr int kWRow = 28;           // hidden weight row padded to 7 float4

struct FcSmem {
  float w0[kFcHidden][12];              // W0 [25][9] padded to 12
  float b0[28];
  float wh[4][kFcHidden][kWRow];        // W1..W4 [25][25] padded to 28
  float bh[4][28];
  float h[kFcThreads][kHStride];
  int iv[kFcThreads];
};

__device__ __forceinline__ float leaky(float v) { return v >= 0.0f ? v : kLeaky * v; }

// softplus(v) = max(v,0) + log1p(exp(-|v|))   (reading O3; beta = 1, no threshold)
// Evaluated with the two SFU ops ex2 / lg2: e = exp(-|v|) in (0, 1], log(1 + e) with 1 + e in (1, 2] where
// __logf's absolute error is <= 2^-21.4 (CUDA math API) -- the same order as the FP32 rounding of a
// contribution of size ~0.7, and far below the histogram tolerance.
__device__ __forceinline__ float softplus_f(float v) {
  const float e = __expf(-fabsf(v));
  return fmaxf(v, 0.0f) + __logf(1.0f + e);
}

__global__ void __launch_bounds__(kFcThreads)
k_fc_hist(const float* __restrict__ f0, const float* __restrict__ f1, const float* __restrict__ f2,
          const float* __restrict__ f3, const float* __restrict__ f4, const float* __restrict__ f5,
          const float* __restrict__ f6, const float* __restrict__ f7, const float* __restrict__ f8,
          const int32_t* __restrict__ event_offsets, const int32_t* __restrict__ perm,
          const int32_t* __restrict__ seg_off, const int32_t* __restrict__ seg_cnt,
          const float* __restrict__ par, int n_events, float* __restrict__ hist) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  FcSmem& S = *reinterpret_cast<FcSmem*>(smem_raw);
  const int tid = threadIdx.x;

  pdl_launch_dependents();      // pdl.cuh: the weight staging below may overlap the sort kernel's tail
  // stage the small layers in shared memory (zero padded)
  for (int i = tid; i < kFcHidden * 12; i += kFcThreads) {
    int r = i / 12, c = i % 12;
    S.w0[r][c] = c < kFcIn ? par[kFcW0 + r * kFcIn + c] : 0.0f;
  }
  for (int i = tid; i < 28; i += kFcThreads) S.b0[i] = i < kFcHidden ? par[kFcB0 + i] : 0.0f;
  for (int i = tid; i < 4 * kFcHidden * kWRow; i += kFcThreads) {
    int l = i / (kFcHidden * kWRow), r = (i / kWRow) % kFcHidden, c = i % kWRow;
    S.wh[l][r][c] = c < kFcHidden ? par[kFcHid + l * kFcHidStride + r * kFcHidden + c] : 0.0f;
  }
  for (int i = tid; i < 4 * 28; i += kFcThreads) {
    int l = i / 28, c = i % 28;
    S.bh[l][c] = c < kFcHidden ? par[kFcHid + l * kFcHidStride + kFcHidden * kFcHidden + c] : 0.0f;
  }
  // last layer: four rows of W5 per owner thread, in registers
  float w5[4][kFcHidden];
  float b5[4];
  const bool owner = tid < kOwners;
#pragma unroll
  for (int m = 0; m < 4; ++m) {
    const int o = tid + kOwners * m;
#pragma unroll
    for (int k = 0; k < kFcHidden; ++k) w5[m][k] = owner ? par[kFcW5 + o * kFcHidden + k] : 0.0f;
    b5[m] = owner ? par[kFcB5 + o] : 0.0f;
  }
  __syncthreads();
  pdl_wait();                   // perm / seg_off / seg_cnt come from the sort kernel

  for (int e = blockIdx.x; e < n_events; e += gridDim.x) {
    const size_t seg0 = (size_t)e * kIntervals;
    const int ev_lo = seg_off[seg0];          // start of the event's run of entries in perm
    const int n_kept = seg_off[seg0 + kIntervals - 1] + seg_cnt[seg0 + kIntervals - 1] - ev_lo;
    float* He = hist + (size_t)e * kIntervals * kFcOut;
    float acc[4] = {0.f, 0.f, 0.f, 0.f};
    int cur = 0;   // interval the accumulators belong to
    for (int base = 0; base < n_kept; base += kFcThreads) {
      const int ntile = min(kFcThreads, n_kept - base);
      // ---- phase A: hidden layers, one sorted track per thread
      if (tid < ntile) {
        int t;
        float zrel;
        const int iv = entry_interval(perm[ev_lo + base + tid], f0, t, zrel);   // own or neighbouring interval (NEXT-1)
        S.iv[tid] = iv;
        float x[kFcIn] = {zrel, f1[t], f2[t], f3[t], f4[t], f5[t], f6[t], f7[t], f8[t]};
        float h[28], g[28];
#pragma unroll
        for (int o = 0; o < kFcHidden; ++o) {
          float a = S.b0[o];
#pragma unroll
          for (int i = 0; i < kFcIn; ++i) a = fmaf(S.w0[o][i], x[i], a);
          h[o] = leaky(a);
        }
#pragma unroll
        for (int l = 0; l < 4; ++l) {
#pragma unroll
          for (int o = 0; o < kFcHidden; ++o) {
            float a = S.bh[l][o];
            const float4* wr = reinterpret_cast<const float4*>(S.wh[l][o]);
#pragma unroll
            for (int q = 0; q < 7; ++q) {
              const float4 w = wr[q];
              a = fmaf(w.x, h[4 * q], a);
              if (4 * q + 1 < kFcHidden) a = fmaf(w.y, h[4 * q + 1], a);
              if (4 * q + 2 < kFcHidden) a = fmaf(w.z, h[4 * q + 2], a);
              if (4 * q + 3 < kFcHidden) a = fmaf(w.w, h[4 * q + 3], a);
            }
            g[o] = leaky(a);
          }
#pragma unroll
          for (int o = 0; o < kFcHidden; ++o) h[o] = g[o];
        }
        h[25] = h[26] = h[27] = 0.0f;
        float4* hs = reinterpret_cast<float4*>(S.h[tid]);
#pragma unroll
        for (int q = 0; q < 7; ++q) hs[q] = make_float4(h[4 * q], h[4 * q + 1], h[4 * q + 2], h[4 * q + 3]);
      }
      __syncthreads();
      // ---- phase B: 25 -> 800, softplus, ordered accumulation per interval
      if (owner) {
        for (int k = 0; k < ntile; ++k) {
          const int iv = S.iv[k];
          while (cur < iv) {   // interval finished: flush (zeros for skipped empty intervals)
#pragma unroll
            for (int m = 0; m < 4; ++m) { He[cur * kFcOut + tid + kOwners * m] = acc[m]; acc[m] = 0.f; }
            ++cur;
          }
          const float4* hk = reinterpret_cast<const float4*>(S.h[k]);
          float v[4] = {b5[0], b5[1], b5[2], b5[3]};
#pragma unroll
          for (int q = 0; q < 7; ++q) {
            const float4 hh = hk[q];
#pragma unroll
            for (int m = 0; m < 4; ++m) {
              v[m] = fmaf(w5[m][4 * q], hh.x, v[m]);
              if (4 * q + 1 < kFcHidden) v[m] = fmaf(w5[m][4 * q + 1], hh.y, v[m]);
              if (4 * q + 2 < kFcHidden) v[m] = fmaf(w5[m][4 * q + 2], hh.z, v[m]);
              if (4 * q + 3 < kFcHidden) v[m] = fmaf(w5[m][4 * q + 3], hh.w, v[m]);
            }
          }
#pragma unroll
          for (int m = 0; m < 4; ++m) acc[m] += softplus_f(v[m]);
        }
      }
      __syncthreads();
    }
    if (owner) {
      while (cur < kIntervals) {
#pragma unroll
        for (int m = 0; m < 4; ++m) { He[cur * kFcOut + tid + kOwners * m] = acc[m]; acc[m] = 0.f; }
        ++cur;
      }
    }
  }
}

int fc_hist_launches(int n_events) { return n_events > 0 ? 1 : 0; }

void launch_fc_hist(const float* const feat[9], const int32_t* event_offsets, const int32_t* perm,
                    const int32_t* seg_off, const int32_t* seg_cnt, const float* fc_params,
                    int n_events, float* hist, int sm_count, bool pdl, cudaStream_t s) {
  if (n_events <= 0) return;
  const int grid = min(n_events, sm_count * 2);
  PdlLaunch L(dim3(grid), dim3(kFcThreads), sizeof(FcSmem), s, pdl);
  cudaLaunchKernelEx(&L.cfg, k_fc_hist, feat[0], feat[1], feat[2], feat[3], feat[4], feat[5], feat[6], feat[7], feat[8],
                     event_offsets, perm, seg_off, seg_cnt, fc_params, n_events, hist);
}

cudaError_t fc_hist_setup() {
  return cudaFuncSetAttribute(k_fc_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(FcSmem));
}

}  // namespace pvf
