// a1 + a2, tensor-core version -- per-track fully connected network with the 25 -> 800 output layer on
// tcgen05 (FP32-accurate: 3-pass TF32 hi/lo split) and the deterministic segmented sum into the
// interval histograms H[n_events, 40, 8, 100] done by the epilogue straight out of TMEM.
//
// PAPER.md:29 "six FC layers ... combining each track's contribution into a 800-bin histogram (8
// channels each with 100-bin)"; BASELINE.json config 0 (9->25->25->25->25->25->800, LeakyReLU(0.01),
// softplus) and north_star (a)/(b): MMA for the FC, tracks sorted by interval and summed in a fixed
// order, no float atomics.  DESIGN.md section 4.2.
//
// Mapping.  The last layer is 88 % of the FC FLOPs.  Per tile of up to 128 sorted tracks of one event
//     D[o, t] = sum_k W5x[o, k] * hx[t, k],   k < 25: weights x activations, k = 25: bias x 1, K = 32
// with M = output rows and N = 128 tracks.  So an accumulator lane is one output and an accumulator column
// is one track: the epilogue thread that owns a lane walks the columns in sorted-track order, adds
// softplus(D) into one FP32 register and stores it to H whenever the interval changes -- a sum whose order is fixed
// by the sorted positions, with no cross-lane reduction; only intervals that hold a track are written (k_unet_tc
// takes seg_cnt == 0 as zeros).  Tracks of the same interval share one logarithm per group (16-track chunk or group
// of four; see softplus_front2): sum softplus(v) = sum max(v, 0) + ln 2 lg2(prod (1 + e^-|v|)).
// The packed W5x is pre-scaled by log2(e): D holds t = v log2(e), the sums run in units of log2 and ln 2 is applied per stored sum.
// FP32 accuracy: W5x = W_hi + W_lo and hx = h_hi + h_lo (each part RN-rounded to TF32), three MMAs
// W_hi h_hi + W_hi h_lo + W_lo h_hi accumulate in FP32 in TMEM (the dropped term is ~2^-22 relative).
// CTA pairs: the two CTAs of a cluster serve the two halves of the 800 outputs (400 each, packed densely into
// 3 full accumulator tiles + 16 rows; 128 KB of W5x hi + lo resident in shared memory) for the same strided
// subset of events and share every MMA (cta_group::2, M = 256): each supplies the hidden activations of half of
// the tile's tracks (even / odd sorted positions), so the hidden layers run once per pair.
// Roles: warps 0-11 and 13 epilogue (one accumulator tile quadrant each), warp 12 MMA issuer (leader CTA), warps
// 14-21 = four groups of 64 threads that run the five 25-wide hidden layers (FP32 FMA, thread = track) for
// tiles it, it + 1, it + 2, it + 3 and stage h_hi / h_lo as the B operand (one buffer per group).
#include <cstring>
#include <type_traits>

#include "pvf_internal.cuh"
#include "pdl.cuh"
#include "umma.cuh"

namespace pvf {
using namespace umma;

namespace {

constexpr int kEpiWarps = 13;                // one per (accumulator tile, 32-lane quadrant) that holds outputs
// Warp w runs on scheduler w % 4 and reaches TMEM lanes 32 (w % 4) .. only.  The 13th unit (the 16 rows of tile 3) sits in
// QUADRANT 1 and is served by warp 13, the MMA issuer is warp 12: every scheduler then carries three full epilogue warps
// (the SFU-heavy role) instead of four on scheduler 0.
constexpr int kMmaWarp = 12;
constexpr int kSmallEpiWarp = 13;
constexpr int kSmallRow0 = 3 * 128 + 32;     // accumulator row of the first of the last 16 outputs of a half (384 ..)
constexpr int kHidWarp0 = 14;
#ifndef PVF_FC_HID_GROUPS
#define PVF_FC_HID_GROUPS 4      // measured at 16 k events: 2 groups 2.40 ms, 3: 2.31 ms, 4: 2.16 ms
#endif
constexpr int kHidGroups = PVF_FC_HID_GROUPS;   // groups of two warps, each on its own tile: a CTA runs the hidden layers of HALF of a tile
constexpr int kHidWarps = 2 * kHidGroups;
constexpr int kFtThreads = (kEpiWarps + 1 + kHidWarps) * 32;   // 13 epilogue + 1 MMA + the hidden-layer warps
constexpr int kHalfOut = kFcOut / 2;         // outputs per CTA half, packed densely: row 128 t + r = output 400 half + 128 t + r
constexpr int kTile = 128;                   // tracks per tile (MMA N)
constexpr int kRowsW = 512;                  // 4 channel tiles x 128 rows per CTA half
constexpr int kLboW = kRowsW * 16;           // 8192: next 16-byte K chunk of the A operand
constexpr int kHalfTile = kTile / 2;         // B-operand rows (tracks) this CTA of the pair supplies
constexpr int kLboH = kHalfTile * 16;        // 1024: next 16-byte K chunk of the B operand
constexpr int kWPart = 8 * kLboW;            // 65536 bytes: one part (hi or lo) of W5x for one half
constexpr int kHPart = 8 * kLboH;            // 8192 bytes: one part of hx for this CTA's half of a tile
constexpr int kWRow = 28;

struct FtSmall {                             // the five hidden layers, zero padded
  float w0[kFcHidden][12];
  float b0[28];
  float wh[4][kFcHidden][kWRow];           // TRANSPOSED: wh[l][k][o] = W_{l+1}[o][k] (one row = the weights of input k)
  float bh[4][28];
};

constexpr int OFF_W = 0;                               // [hi | lo][8 chunks][512 rows][16 B]
constexpr int OFF_H = OFF_W + 2 * kWPart;              // [one buffer per hidden-layer group][hi | lo][8 chunks][64 tracks][16 B]
constexpr int OFF_SMALL = OFF_H + 2 * kHidGroups * kHPart;
constexpr int OFF_IV = OFF_SMALL + ((int)sizeof(FtSmall) + 127) / 128 * 128;   // int [4][128]
constexpr int kIvBufs = 8;                   // interval lists of four tiles in flight: the hidden-layer warps of tile
                                             // i + 2 must not wait for the epilogue of tile i (measured: they did)
constexpr int OFF_BARS = OFF_IV + kIvBufs * kTile * 4;
constexpr int FT_SMEM = OFF_BARS + 512;
static_assert(FT_SMEM <= 227 * 1024, "shared memory budget");
// barriers (8 bytes each): h_full[2], peer_h_full[2] (leader: the peer's half is staged), h_empty[2], meta[4],
// acc_full[4], acc_empty[4], peer_acc_empty[4] (leader: the peer's epilogue has drained the tile), iv_full[4], then the
// TMEM slot.
// iv_full[it & 3] ("the interval list of tile it is staged", hidden-layer threads -> epilogue) is indexed like meta[]:
// the hidden-layer threads of tile it + 4 write that list only after meta[it & 3] completed its phase `it`, i.e. after
// EVERY epilogue warp has finished tile it and therefore observed phase `it` of iv_full -- no phase can be skipped.  (The
// 2-deep h_full gave no such guarantee to a slow epilogue warp: hidden(it + 2) is only gated by the MMAs of tile it.)
enum { bHFull = 0, bPHFull = bHFull + kHidGroups, bHEmpty = bPHFull + kHidGroups, bMeta = bHEmpty + kHidGroups,
       bAccFull = bMeta + kIvBufs, bAccEmpty = bAccFull + 4, bPAccEmpty = bAccEmpty + 4, bIvFull = bPAccEmpty + 4,
       bW5 = bIvFull + kIvBufs, bSlot = bW5 + 1 };
static_assert(8 * bSlot + 4 <= 512, "barrier block");
constexpr int kIvLog = 3;
static_assert((1 << kIvLog) == kIvBufs && kIvBufs >= 2 * kHidGroups, "interval lists: a power of two, two per hidden-layer group");
static_assert(FT_SMEM <= 227 * 1024, "shared memory budget");

__device__ __forceinline__ float leaky_ft(float v) { return v >= 0.0f ? v : kLeaky * v; }
__device__ __forceinline__ uint32_t tf32_of(float v) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ void st16(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}
// Packed FP32 pairs (add / fma .f32x2 of sm_100: one issue slot for two values).
__device__ __forceinline__ void add2(float a0, float a1, float b0, float b1, float& o0, float& o1) {
  asm("{\n\t.reg .b64 p, q, r;\n\tmov.b64 p, {%2, %3};\n\tmov.b64 q, {%4, %5};\n\t"
      "add.rn.f32x2 r, p, q;\n\tmov.b64 {%0, %1}, r;\n\t}"
      : "=f"(o0), "=f"(o1) : "f"(a0), "f"(a1), "f"(b0), "f"(b1));
}
__device__ __forceinline__ float lg2_ft(float u) {
  float w;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(w) : "f"(u));
  return w;
}
// softplus(v) = max(v, 0) + ln2 * lg2(1 + 2^(-|v| log2 e)).  The front half for two values: u = 1 + e in (1, 2] and
// m = max(v, 0).  Tracks that are summed into the same interval share ONE logarithm:
//     sum_i softplus(v_i) = sum_i m_i + ln2 * lg2(prod_i u_i)        (16 factors in (1, 2]: prod <= 65536, no overflow)
// which halves the SFU operations of the stage (one ex2 per value, one lg2 per group instead of per value).
// The packed W5x image is scaled by log2(e) (fc_tc_pack), so the accumulators hold t = v log2(e) and the whole sum runs in
// units of log2: softplus(v) / ln 2 = max(t, 0) + lg2(1 + 2^-|t|); the factor ln 2 is applied once per stored sum
// (kLn2 below) instead of one multiply per value in front of the ex2.
// Front half for two values: e = 2^-|t| in (0, 1] and m = max(t, 0); the factor 1 + e is formed where it is used (prod2).
__device__ __forceinline__ void softplus_front2(float t0, float t1, float& e0, float& e1, float& m0, float& m1) {
  const float n0 = -fabsf(t0), n1 = -fabsf(t1);          // operand modifiers of the MUFU, no instructions of their own
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e0) : "f"(n0));
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(e1) : "f"(n1));
  m0 = fmaxf(t0, 0.0f);
  m1 = fmaxf(t1, 0.0f);
}
// Running product of factors (1 + e) as one packed pair: start = (1 + e0, 1 + e1), then P <- P + e P = P (1 + e) per further
// pair of factors -- one fma.rn.f32x2 for two factors (forming 1 + e and multiplying separately took two).
__device__ __forceinline__ unsigned long long prod2_start(float e0, float e1) {
  unsigned long long r;
  asm("{\n\t.reg .b64 p, k;\n\tmov.b64 p, {%1, %2};\n\tmov.b64 k, {%3, %3};\n\tadd.rn.f32x2 %0, p, k;\n\t}"
      : "=l"(r) : "f"(e0), "f"(e1), "f"(1.0f));
  return r;
}
__device__ __forceinline__ void prod2_step(unsigned long long& P, float e0, float e1) {
  asm("{\n\t.reg .b64 q;\n\tmov.b64 q, {%1, %2};\n\tfma.rn.f32x2 %0, q, %0, %0;\n\t}" : "+l"(P) : "f"(e0), "f"(e1));
}
__device__ __forceinline__ float prod2_finish(unsigned long long P) {
  float a, b;
  asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(P));
  return a * b;
}
constexpr float kLn2 = 0.6931471805599453f;

struct Feat9 { const float* f[9]; };

#ifdef PVF_FC_PROF
// Diagnostic build only (-DPVF_FC_PROF): cycles per role and CTA (lane 0 of one warp per role):
// [0] epilogue wait h_full, [1] epilogue wait acc_full, [2] epilogue total; [3] MMA wait h_full, [4] MMA wait acc_empty,
// [5] MMA total; [6] hidden wait h_empty, [7] hidden wait meta, [8] hidden total (group 0), [9] tiles
__device__ unsigned long long g_fc_prof[160][16];
#define FC_PROF_T0() const long long prof_t0 = clock64()
#define FC_PROF_ADD(slot, cond) do { if (cond) g_fc_prof[blockIdx.x][slot] += (unsigned long long)(clock64() - prof_t0); } while (0)
#define FC_PROF_CNT(slot, cond) do { if (cond) g_fc_prof[blockIdx.x][slot] += 1ull; } while (0)
#else
#define FC_PROF_T0() do {} while (0)
#define FC_PROF_ADD(slot, cond) do {} while (0)
#define FC_PROF_CNT(slot, cond) do {} while (0)
#endif

__global__ void __launch_bounds__(kFtThreads, 1)
k_fc_hist_tc(Feat9 F, const int32_t* __restrict__ event_offsets, const int32_t* __restrict__ perm,
             const int32_t* __restrict__ seg_off, const int32_t* __restrict__ seg_cnt,
             const float* __restrict__ par, const unsigned char* __restrict__ w5img, int n_events,
             float* __restrict__ hist, float* __restrict__ dump) {
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t sb = smem_u32(smem);
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  // The two CTAs of a cluster (blockIdx.x = 2 j, 2 j + 1) serve the two halves of the outputs for the SAME events and share
  // every MMA (cta_group::2, M = 256): each supplies its 128 output rows of W5x and the hidden activations of HALF of
  // the tile's tracks (even sorted positions: rank 0, odd: rank 1), so the hidden layers are computed once per pair.
  const int rank = (int)cluster_ctarank();
  const int half = rank;
  FtSmall& S = *reinterpret_cast<FtSmall*>(smem + OFF_SMALL);
  int* s_iv = reinterpret_cast<int*>(smem + OFF_IV);
  auto bar = [&](int k) { return sb + OFF_BARS + 8u * k; };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + OFF_BARS + 8 * bSlot);

  // ---- one-time setup: this half's W5x image, zeroed B buffers, the small layers, barriers, TMEM (weights only:
  // all of it may overlap the tail of the sort kernel, see pdl.cuh)
  pdl_launch_dependents();
  // The 128 KB of W5x go by bulk copies (TMA engine) issued first thing by one thread; they land while the other threads
  // stage the small layers and zero the operand buffers (a load / store loop of all threads took ~4 us, most of what a
  // one-event call spends in this kernel before its first track).
  if (tid == 0) {
    mbar_init(bar(bW5), 1);
    fence_mbar_init();
    mbar_arrive_expect_tx(bar(bW5), (uint32_t)(2 * kWPart));
    for (int k = 0; k < 2 * kWPart / 16384; ++k)
      bulk_g2s(sb + OFF_W + k * 16384, w5img + (size_t)half * 2 * kWPart + (size_t)k * 16384, 16384u, bar(bW5));
  }
  {
    uint4* hz = reinterpret_cast<uint4*>(smem + OFF_H);
    for (int i = tid; i < 2 * kHidGroups * kHPart / 16; i += kFtThreads) hz[i] = make_uint4(0, 0, 0, 0);
  }
  for (int i = tid; i < kFcHidden * 12; i += kFtThreads) {
    const int r = i / 12, c = i % 12;
    S.w0[r][c] = c < kFcIn ? par[kFcW0 + r * kFcIn + c] : 0.0f;
  }
  for (int i = tid; i < 28; i += kFtThreads) S.b0[i] = i < kFcHidden ? par[kFcB0 + i] : 0.0f;
  for (int i = tid; i < 4 * kFcHidden * kWRow; i += kFtThreads) {
    const int l = i / (kFcHidden * kWRow), k = (i / kWRow) % kFcHidden, o = i % kWRow;
    S.wh[l][k][o] = o < kFcHidden ? par[kFcHid + l * kFcHidStride + o * kFcHidden + k] : 0.0f;
  }
  for (int i = tid; i < 4 * 28; i += kFtThreads) {
    const int l = i / 28, c = i % 28;
    S.bh[l][c] = c < kFcHidden ? par[kFcHid + l * kFcHidStride + kFcHidden * kFcHidden + c] : 0.0f;
  }
  if (tid == 0) {
    for (int k = 0; k < kHidGroups; ++k) {
      mbar_init(bar(bHFull + k), kHalfTile); mbar_init(bar(bPHFull + k), kHalfTile); mbar_init(bar(bHEmpty + k), 1);
    }
    for (int k = 0; k < kIvBufs; ++k) { mbar_init(bar(bMeta + k), 32 * kEpiWarps); mbar_init(bar(bIvFull + k), kHalfTile); }
    for (int k = 0; k < 4; ++k) {
      mbar_init(bar(bAccFull + k), 1);
      mbar_init(bar(bAccEmpty + k), k < 3 ? 128 : 32);
      mbar_init(bar(bPAccEmpty + k), k < 3 ? 128 : 32);
    }
    fence_mbar_init();
    mbar_wait(bar(bW5), 0u);                     // this CTA's W5x image has landed (the peer's: before the cluster barrier below)
  }
  if (warp == kMmaWarp) tmem_alloc2(smem_u32(const_cast<uint32_t*>(tmem_slot)), 512);
  fence_proxy_async_smem();
  tc_fence_before_sync();
  cluster_sync_all();
  tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();                                 // perm / seg_off / seg_cnt come from the sort kernel

  // kept (in-range) tracks of event e and the start of its run in perm
  auto kept_of = [&](int e, int& ev_lo) {
    ev_lo = seg_off[(size_t)e * kIntervals];            // start of the event's run of entries in perm
    const size_t s = (size_t)e * kIntervals + kIntervals - 1;
    return seg_off[s] + seg_cnt[s] - ev_lo;
  };

  if (warp < kMmaWarp || warp == kSmallEpiWarp) {
    // ===================== epilogue: lane = output, column = track (sorted order).  The 400 outputs of this half
    // fill accumulator tiles 0-2 and 16 rows of tile 3 (quadrant 1); warp w < 12 owns the 32 rows of quadrant w & 3 of
    // tile w >> 2, warp 13 the 16 rows of tile 3, so every warp has one tile per 128 tracks.
    const int q = warp & 3, mt = warp == kSmallEpiWarp ? 3 : warp >> 2;
    const int r = 32 * q + lane;
    const int ol = warp == kSmallEpiWarp ? 384 + lane : 128 * mt + r;      // output inside this half
    const bool valid = warp == kSmallEpiWarp ? lane < 16 : true;
    const uint32_t lead_pacc = mapa_rank(bar(bPAccEmpty), 0);
    int it = 0;
    [[maybe_unused]] const bool pw = tid == 0;
    FC_PROF_T0();
    for (int e = (int)blockIdx.x >> 1; e < n_events; e += (int)gridDim.x >> 1) {
      int ev_lo;
      const int nk = kept_of(e, ev_lo);
      // output o = c * 100 + l lives at H[e][interval][o]: the dense row index is the offset itself.  Rows that
      // hold no output send their (meaningless) sums to the dump slot, so the boundary stores' predicate stays
      // warp-uniform.
      float* Hc = valid ? hist + (size_t)e * kIntervals * kFcOut + kHalfOut * half + ol : dump + r;   // + iv * 800 (= s_iv)
      float a = 0.f;                             // running sum of the current interval
      int c = 0;                                 // the interval it belongs to, as the offset interval * 800
      for (int base = 0; base < nk; base += kTile, ++it) {
        const int ntile = min(kTile, nk - base);
        const bool last = base + kTile >= nk;
        const int ib = it & (kIvBufs - 1);
        { FC_PROF_T0(); mbar_wait(bar(bIvFull + ib), (uint32_t)((it >> kIvLog) & 1)); FC_PROF_ADD(0, pw); }   // s_iv is staged
        FC_PROF_CNT(9, pw);
        const int* ivs = s_iv + ib * kTile;
        if (base == 0) c = ivs[0];               // the event's first (lowest) non-empty interval
        { FC_PROF_T0(); mbar_wait(bar(bAccFull + mt), (uint32_t)(it & 1)); FC_PROF_ADD(1, pw); }
        tc_fence_after_sync();
        const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) + (uint32_t)(mt * kTile);
        // One chunk of 16 sorted positions.  TAIL (compile time) = the tile's last, partly filled chunk: only that copy of the
        // code masks the columns past the last track (as one body the masking cost every chunk 16 compares + 32 selects).
        auto chunk = [&](const int c0, auto tail_tag) {
          constexpr bool TAIL = decltype(tail_tag)::value;
          // sorted positions c0 .. c0+15: the even ones are columns c0/2 .. of the leader's half of N, the odd ones
          // columns 64 + c0/2 .. of the peer's half
          uint32_t ve[8], vo[8];
          tmem_ld_x8(taddr + (uint32_t)(c0 >> 1), ve);
          tmem_ld_x8(taddr + (uint32_t)(kHalfTile + (c0 >> 1)), vo);
          // Where do intervals change inside these 16 tracks?  The interval list is the same for every lane, so the
          // answer is one warp-uniform 16-bit mask: lane i < 16 compares track c0 + i with its predecessor (the running
          // interval c for the tile's first track), one ballot.  Tracks past the tile's end never start an interval.
          const int nv = TAIL ? ntile - c0 : 16;
          const int pos = c0 + (lane & 15);
          const int iv_prev = pos == 0 ? c : ivs[pos - 1];
          const unsigned mask = __ballot_sync(0xffffffffu, lane < 16 && lane < nv && ivs[pos] != iv_prev);
          tmem_ld_wait();
          // front half of all 16 softplus first: independent, so the SFU pipeline stays full; columns past the
          // tile's last track are computed on stale accumulators and then neutralised (u = 1, m = 0)
          float ev[16], m[16];
#pragma unroll
          for (int k = 0; k < 8; ++k)
            softplus_front2(__uint_as_float(ve[k]), __uint_as_float(vo[k]), ev[2 * k], ev[2 * k + 1], m[2 * k], m[2 * k + 1]);
          if (TAIL) {
#pragma unroll
            for (int i = 0; i < 16; ++i)
              if (i >= nv) { ev[i] = 0.0f; m[i] = 0.0f; }     // factor 1, term 0
          }
#ifdef PVF_FC_NOREDUCE
          // diagnostic build: the FC arithmetic alone (all 16 logarithms, no ordered segmented sum, no histogram stores
          // but the event's last one) -- gives the "FC" share of the fused stage (BASELINE.json config 2)
#pragma unroll
          for (int i = 0; i < 16; ++i) a += lg2_ft(1.0f + ev[i]) + m[i];
#else
          // Ordered accumulation (fixed by the sorted positions, hence reproducible).  Only intervals that hold a track
          // are written -- the UNet kernel never reads the histogram of an empty interval (seg_cnt == 0 means zeros).
          if (mask == 0u) {                      // the whole chunk continues the running interval: one logarithm
            unsigned long long P = prod2_start(ev[0], ev[1]);
#pragma unroll
            for (int k = 1; k < 8; ++k) prod2_step(P, ev[2 * k], ev[2 * k + 1]);
            float t[8];
#pragma unroll
            for (int k = 0; k < 4; ++k) add2(m[4 * k], m[4 * k + 1], m[4 * k + 2], m[4 * k + 3], t[2 * k], t[2 * k + 1]);
            add2(t[0], t[1], t[2], t[3], t[0], t[1]);
            add2(t[4], t[5], t[6], t[7], t[4], t[5]);
            add2(t[0], t[1], t[4], t[5], t[0], t[1]);
            a += lg2_ft(prod2_finish(P)) + (t[0] + t[1]);
          } else {
#pragma unroll
            for (int g = 0; g < 4; ++g) {        // groups of four tracks; the tests are warp-uniform
              const unsigned gb = (mask >> (4 * g)) & 15u;
              if (gb == 0u) {
                unsigned long long P = prod2_start(ev[4 * g], ev[4 * g + 1]);
                prod2_step(P, ev[4 * g + 2], ev[4 * g + 3]);
                float t0, t1;
                add2(m[4 * g], m[4 * g + 1], m[4 * g + 2], m[4 * g + 3], t0, t1);
                a += lg2_ft(prod2_finish(P)) + (t0 + t1);
              } else {                           // an interval starts here: track by track
                const int4 q4 = *reinterpret_cast<const int4*>(ivs + c0 + 4 * g);
                const int iq[4] = {q4.x, q4.y, q4.z, q4.w};
                float u0, u1, u2, u3;
                add2(ev[4 * g], ev[4 * g + 1], 1.0f, 1.0f, u0, u1);
                add2(ev[4 * g + 2], ev[4 * g + 3], 1.0f, 1.0f, u2, u3);
                const float uu[4] = {u0, u1, u2, u3};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                  const float x = lg2_ft(uu[k]) + m[4 * g + k];
                  // Bit k of gb: an interval starts at this track (never set past the tile's last track): the finished sum
                  // goes to H and the sum restarts (0 + x == x exactly).  The compiler predicates the store sequence on the
                  // mask bits (one R2P for the group) -- cheaper than comparing interval ids per track, and cheaper than real
                  // branches (measured: four straight-line cases behind warp-uniform branches, each segment sharing one
                  // logarithm, were 5 % slower: the epilogue is bound by latency, not by issue slots).
                  if (gb & (1u << k)) {
                    Hc[c] = a * kLn2;              // sums run in units of log2 (softplus_front2)
                    a = 0.0f;
                    c = iq[k];
                  }
                  a += x;
                }
              }
            }
          }
#endif
        };
        int c0 = 0;
        for (; c0 + 16 <= ntile; c0 += 16) chunk(c0, std::false_type{});
        if (c0 < ntile) chunk(c0, std::true_type{});
        if (last) Hc[c] = a * kLn2;               // the event's last non-empty interval
        tc_fence_before_sync();
        if (rank == 0) mbar_arrive(bar(bAccEmpty + mt));
        else mbar_arrive_cluster(lead_pacc + 8u * mt);
        mbar_arrive(bar(bMeta + ib));
      }
    }
    FC_PROF_ADD(2, pw);
  } else if (warp == kMmaWarp) {
    // ===================== MMA issuer (leader CTA only; the peer's warp just keeps the TMEM allocation)
    if (rank == 0) {
    constexpr uint32_t idesc = instr_desc(kFmtTF32, 256, kTile);
    constexpr uint32_t hi = (128u >> 4) | (1u << 14);
    constexpr uint32_t a_lbo = (uint32_t)(kLboW >> 4) << 16, b_lbo = (uint32_t)(kLboH >> 4) << 16;
    int it = 0;
    [[maybe_unused]] const bool pw = lane == 0;
    FC_PROF_T0();
    for (int e = (int)blockIdx.x >> 1; e < n_events; e += (int)gridDim.x >> 1) {
      int ev_lo;
      const int nk = kept_of(e, ev_lo);
      for (int base = 0; base < nk; base += kTile, ++it) {
        const int buf = it % kHidGroups;
        {
          FC_PROF_T0();
          mbar_wait(bar(bHFull + buf), (uint32_t)((it / kHidGroups) & 1));       // both halves of the B operand are staged
          mbar_wait(bar(bPHFull + buf), (uint32_t)((it / kHidGroups) & 1));
          FC_PROF_ADD(3, pw);
        }
        tc_fence_after_sync();
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
          {
            FC_PROF_T0();
            mbar_wait(bar(bAccEmpty + mt), (uint32_t)((it & 1) ^ 1));     // both epilogues have drained tile mt
            mbar_wait(bar(bPAccEmpty + mt), (uint32_t)((it & 1) ^ 1));
            FC_PROF_ADD(4, pw);
          }
          tc_fence_after_sync();
          if (elect_one()) {
#pragma unroll
            for (int pass = 0; pass < 3; ++pass) {       // W_hi h_hi, W_hi h_lo, W_lo h_hi
#pragma unroll
              for (int s = 0; s < 4; ++s) {
                const uint32_t a = a_lbo + ((sb + OFF_W + (pass == 2 ? kWPart : 0) + mt * 2048 + s * 2 * kLboW) >> 4);
                const uint32_t b = b_lbo + ((sb + OFF_H + buf * 2 * kHPart + (pass == 1 ? kHPart : 0) + s * 2 * kLboH) >> 4);
                mma2_tf32_lh(tmem_base + (uint32_t)(mt * kTile), a, hi, b, hi, idesc, (pass | s) ? 1u : 0u);
              }
            }
            mma_commit2(bar(bAccFull + mt), 3);            // to both CTAs' barriers
            if (mt == 3) mma_commit2(bar(bHEmpty + buf), 3);
          }
          __syncwarp();
        }
      }
    }
    FC_PROF_ADD(5, pw);
    }
  } else {
    // ===================== hidden layers: two groups of 64 threads for alternating tiles; thread i takes the track
    // at sorted position 2 i + rank of the tile (B-operand row i of this CTA) and also looks up the interval of its
    // neighbour 2 i + 1 - rank, so that both CTAs hold the interval list of the whole tile without exchanging data
    const int g = (warp - kHidWarp0) >> 1, i = tid - 32 * kHidWarp0 - kHalfTile * g;
    const uint32_t hbase = sb + OFF_H + (uint32_t)g * 2 * kHPart + (uint32_t)i * 16u;
    const uint32_t lead_phfull = mapa_rank(bar(bPHFull + g), 0);
    const int p_own = 2 * i + rank, p_other = 2 * i + 1 - rank;
    int it = 0;
    [[maybe_unused]] const bool pw = g == 0 && i == 0;
    FC_PROF_T0();
    for (int e = (int)blockIdx.x >> 1; e < n_events; e += (int)gridDim.x >> 1) {
      int ev_lo;
      const int nk = kept_of(e, ev_lo);
      for (int base = 0; base < nk; base += kTile, ++it) {
        if (it % kHidGroups != g) continue;
        // the track's inputs first (three dependent global loads: perm -> z_poca -> features), THEN the waits for the
        // buffers they go to: the load latency overlaps whatever time the group has to wait anyway
        const bool has_own = base + p_own < nk, has_other = base + p_other < nk;
        int iv_other = 0, iv_own = 0;
        float x[kFcIn] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        if (has_other) {
          int t;
          float zrel;
          iv_other = entry_interval(perm[ev_lo + base + p_other], F.f[0], t, zrel);
        }
        if (has_own) {
          int t;
          iv_own = entry_interval(perm[ev_lo + base + p_own], F.f[0], t, x[0]);   // own or neighbouring interval
#pragma unroll
          for (int k = 1; k < kFcIn; ++k) x[k] = F.f[k][t];
        }
        const uint32_t prev = (uint32_t)(((it / kHidGroups) & 1) ^ 1);
        { FC_PROF_T0(); mbar_wait(bar(bHEmpty + g), prev); FC_PROF_ADD(6, pw); }   // the MMAs that read this buffer have retired
        const int ib = it & (kIvBufs - 1);
        { FC_PROF_T0(); mbar_wait(bar(bMeta + ib), (uint32_t)(((it >> kIvLog) & 1) ^ 1)); FC_PROF_ADD(7, pw); }   // the epilogue is done with s_iv[ib]
        if (has_other) s_iv[ib * kTile + p_other] = iv_other * kFcOut;
        if (has_own) {
          s_iv[ib * kTile + p_own] = iv_own * kFcOut;   // the epilogue wants the interval as its offset in H
          float h[32];
#pragma unroll
          for (int o = 0; o < kFcHidden; ++o) {
            float a = S.b0[o];
#pragma unroll
            for (int k = 0; k < kFcIn; ++k) a = fmaf(S.w0[o][k], x[k], a);
            h[o] = leaky_ft(a);
          }
#pragma unroll 1                  // four identical layers share one copy of the code (I-cache footprint)
          for (int l = 0; l < 4; ++l) {
            // input-major: for every input k the 25 accumulators take one independent FMA each (the weights of input k
            // are one row of the transposed matrix: 7 broadcast 16-byte loads), so no FMA waits for the one before it.
            // (Output-major -- one 25-long dependent chain per output, three chains interleaved by the compiler -- ran
            // the hidden-layer warps at 0.3 instructions per clock and made them the critical path of the kernel.)
            // The 25 accumulators live as 13 packed pairs (fma.rn.f32x2: one issue slot for two outputs); the weight row
            // and the bias arrive as 64-bit pairs straight from the 16-byte loads, so nothing is repacked but the input.
            unsigned long long acc2[14];
            const ulonglong2* br = reinterpret_cast<const ulonglong2*>(S.bh[l]);
#pragma unroll
            for (int q = 0; q < 7; ++q) {
              const ulonglong2 b = br[q];
              acc2[2 * q] = b.x; acc2[2 * q + 1] = b.y;
            }
#pragma unroll
            for (int k = 0; k < kFcHidden; ++k) {
              const ulonglong2* wr = reinterpret_cast<const ulonglong2*>(S.wh[l][k]);
              unsigned long long hh;
              asm("mov.b64 %0, {%1, %1};" : "=l"(hh) : "f"(h[k]));
#pragma unroll
              for (int q = 0; q < 7; ++q) {
                const ulonglong2 w = wr[q];
                asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc2[2 * q]) : "l"(w.x), "l"(hh));
                if (4 * q + 2 < kFcHidden) asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(acc2[2 * q + 1]) : "l"(w.y), "l"(hh));
              }
            }
#pragma unroll
            for (int o = 0; o < kFcHidden; o += 2) {
              float lo, hi2;
              asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi2) : "l"(acc2[o / 2]));
              h[o] = leaky_ft(lo);
              if (o + 1 < kFcHidden) h[o + 1] = leaky_ft(hi2);
            }
          }
          h[25] = 1.0f;                              // multiplies the bias column of W5x
#pragma unroll
          for (int k = 26; k < 32; ++k) h[k] = 0.0f;
#pragma unroll
          for (int c = 0; c < 8; ++c) {
            uint4 vh, vl;
            vh.x = tf32_of(h[4 * c + 0]); vh.y = tf32_of(h[4 * c + 1]);
            vh.z = tf32_of(h[4 * c + 2]); vh.w = tf32_of(h[4 * c + 3]);
            vl.x = tf32_of(h[4 * c + 0] - __uint_as_float(vh.x)); vl.y = tf32_of(h[4 * c + 1] - __uint_as_float(vh.y));
            vl.z = tf32_of(h[4 * c + 2] - __uint_as_float(vh.z)); vl.w = tf32_of(h[4 * c + 3] - __uint_as_float(vh.w));
            st16(hbase + (uint32_t)c * kLboH, vh);
            st16(hbase + kHPart + (uint32_t)c * kLboH, vl);
          }
        }
        fence_proxy_async_smem();
        mbar_arrive(bar(bIvFull + ib));                     // this CTA's epilogue: the interval list is staged
        mbar_arrive(bar(bHFull + g));                       // the leader's MMA issuer: this half of the B operand is staged
        if (rank == 1) mbar_arrive_cluster(lead_phfull);    // the peer's half of the B operand is staged
      }
    }
    FC_PROF_ADD(8, pw);
  }
  __syncwarp();
  tc_fence_before_sync();
  cluster_sync_all();                                       // the pair's shared memory and barriers stay alive until both are done
  if (warp == kMmaWarp) {
    __syncwarp();
    tmem_dealloc2(tmem_base, 512);
  }
}

float tf32_rna_h(float v) {
  uint32_t u;
  memcpy(&u, &v, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return v;
  u = (u + 0x1000u) & 0xffffe000u;
  float r;
  memcpy(&r, &u, 4);
  return r;
}

}  // namespace

size_t fc_tc_packed_bytes() { return (size_t)2 * 2 * kWPart; }      // 2 halves x (hi | lo)

// W5 [800][25] and b5 [800] (PyTorch layouts) -> per half [hi | lo][8 K chunks][512 rows][4 floats];
// row 128*mt + r holds output 400*half + 128*mt + r for the first 384 outputs of a half, rows 416 .. 431 (tile 3, quadrant 1)
// the last 16; all other rows are zero; K index 25 = bias.
void fc_tc_pack(const float* w5, const float* b5, void* host_dst) {
  float* dst = static_cast<float*>(host_dst);
  memset(dst, 0, fc_tc_packed_bytes());
  for (int half = 0; half < 2; ++half)
    for (int row = 0; row < kHalfOut; ++row) {
      const int o = kHalfOut * half + row;
      for (int k = 0; k <= kFcHidden; ++k) {
        // scaled by log2(e) in double, rounded once: the kernel's sums run in units of log2 (softplus_front2)
        const float v = (float)((double)(k < kFcHidden ? w5[o * kFcHidden + k] : b5[o]) * 1.4426950408889634);
        const float hi = tf32_rna_h(v), lo = tf32_rna_h(v - hi);
        const size_t idx = ((size_t)(k / 4) * kRowsW + (row < 384 ? row : kSmallRow0 + row - 384)) * 4 + (k % 4);
        dst[(size_t)half * 2 * (kWPart / 4) + idx] = hi;
        dst[(size_t)half * 2 * (kWPart / 4) + kWPart / 4 + idx] = lo;
      }
    }
}

cudaError_t fc_tc_setup() {
  return cudaFuncSetAttribute(k_fc_hist_tc, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM);
}

void launch_fc_hist_tc(const float* const feat[9], const int32_t* event_offsets, const int32_t* perm,
                       const int32_t* seg_off, const int32_t* seg_cnt, const float* fc_params, const void* w5img,
                       int n_events, float* hist, float* dump, int sm_count, bool pdl, cudaStream_t s) {
  if (n_events <= 0) return;
  Feat9 F;
  for (int k = 0; k < 9; ++k) F.f[k] = feat[k];
  const int gx = n_events < sm_count / 2 ? n_events : sm_count / 2;
  PdlLaunch L(dim3(2 * gx), dim3(kFtThreads), FT_SMEM, s, pdl, 2);   // the two output halves of the same events form a CTA pair
  cudaLaunchKernelEx(&L.cfg, k_fc_hist_tc, F, event_offsets, perm, seg_off, seg_cnt, fc_params,
                     static_cast<const unsigned char*>(w5img), n_events, hist, dump);
}

// include/pvf_debug.h: per-role cycle counters; only a -DPVF_FC_PROF build records them
extern "C" __attribute__((visibility("default"))) int pvf_debug_fc_prof(unsigned long long* host_out, int reset) {
#ifdef PVF_FC_PROF
  cudaDeviceSynchronize();
  if (host_out) cudaMemcpyFromSymbol(host_out, g_fc_prof, sizeof(g_fc_prof));
  if (reset) { static unsigned long long z[160][16]; cudaMemcpyToSymbol(g_fc_prof, z, sizeof(z)); }
  return 0;
#else
  (void)host_out; (void)reset;
  return -1;
#endif
}

}  // namespace pvf
