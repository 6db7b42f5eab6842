// a3, tensor-core path -- the 1D UNet per z-interval as implicit-GEMM convolutions on tcgen05 / TMEM.
//
// PAPER.md:29 "5-layer UNet architecture (64 channels deployed)", PAPER.md:63-76 (the CNN is the
// bottleneck); topology from BASELINE.json config 0 (see k_unet_simt.cu); north_star (c): implicit
// GEMM on tcgen05/TMEM, pool / upsample / concat / activations fused into the epilogues, the
// intermediates stay in shared memory / TMEM.  DESIGN.md "K2" has the derivation of everything here.
//
// Mapping.  A conv layer is  D[m, n] = sum_j sum_ci  A[m + j - p, ci] * W_j[ci, n]  with m = position
// (M), n = output channel (N = C), and one (tap j, 32-byte channel block) per tcgen05.mma of shape
// 128 x C x (8 TF32 | 16 BF16).  Activations live in shared memory in the K-major no-swizzle UMMA
// layout  [channel chunk of 16 B][row][16 B]  (core matrix = 8 rows x 16 B contiguous), so a tap
// shift is a pure bump of the descriptor start address by 16 B per row, the skip concat is a second
// base address, and an epilogue thread (= one row) writes whole 16-byte chunks, conflict free.
// Intervals sit at row stride 128 / 64 / 32 (L = 100 / 50 / 25); the rows between them are zero and
// double as the "same" padding.  One CTA (persistent) takes a group of T intervals through all five
// layers; accumulators of the group's tiles sit side by side in TMEM and each weight slice is
// streamed from L2 exactly once per group (1D bulk copies into a ring of 8 KB stages) and used by
// every tile.  Roles: warp 0 = weight producer, warp 1 = MMA issuer (one thread), warps 2-5 =
// epilogue (TMEM -> registers -> bias, LeakyReLU, TF32/BF16 rounding, pool / upsample -> shared
// memory; the last layer fuses the 1x1 head and the sigmoid and writes the probabilities).
#include <cuda_bf16.h>
#include <cstring>
#include <vector>

#include "pvf_internal.cuh"
#include "umma.cuh"

namespace pvf {
using namespace umma;

namespace {

constexpr int kTcThreads = 192;
constexpr int kStages = 6;
constexpr int kStageBytes = 8192;
constexpr int kHeaderBytes = 2048;          // biases [5][C], head weight [C], head bias
__host__ __device__ constexpr int taps_of(int l) { return (l == 0 || l == 4) ? 25 : (l == 2 ? 5 : 15); }

template <int C, bool BF16>
struct Geo {
  static constexpr int ES = BF16 ? 2 : 4;            // operand element size
  static constexpr int PER = 16 / ES;                // channels per 16-byte chunk
  static constexpr int KPM = 2 * PER;                // channels per MMA (32 bytes of K)
  static constexpr int NCH = C / PER;                // chunks of a C-channel activation
  static constexpr int XCH = BF16 ? 2 : 4;           // chunks of the input buffer X0 (TF32: hi0 hi1 lo0 lo1)
  static constexpr int T = (C == 64) ? (BF16 ? 4 : 2) : (BF16 ? 8 : 4);   // intervals per group
  static constexpr int LEAD1 = 16, LEAD2 = 8, LEAD3 = 8;
  static constexpr int ROWS1 = 128 * T + 32, ROWS2 = 64 * T + 16, ROWS3 = 32 * T + 16;
  static constexpr int LBO1 = ROWS1 * 16, LBO2 = ROWS2 * 16, LBO3 = ROWS3 * 16;
  static constexpr int STEP_BYTES = 2 * C * 16;      // one MMA's B operand: [2 chunks][C][16 B]
  static constexpr int SPS = kStageBytes / STEP_BYTES;   // MMA steps per ring stage
  // shared-memory map (bytes)
  static constexpr int OFF_E1 = 0;
  static constexpr int SZ_L1 = NCH * LBO1;           // a C-channel buffer at L = 100
  static constexpr int SZ_L2 = NCH * LBO2;
  static constexpr int OFF_R = OFF_E1 + SZ_L1;       // overlay region: U1 | (E2, U2) | (P1, P2)
  static constexpr int OFF_X0 = OFF_R + SZ_L1;
  static constexpr int OFF_RING = OFF_X0 + XCH * LBO1;
  static constexpr int OFF_PAR = OFF_RING + kStages * kStageBytes;   // biases + head (floats)
  static constexpr int OFF_BAR = OFF_PAR + kHeaderBytes;
  static constexpr int SMEM = OFF_BAR + 256;
  static constexpr int TMEM_COLS = (T * C <= 32) ? 32 : (T * C <= 64) ? 64 : (T * C <= 128) ? 128 : (T * C <= 256) ? 256 : 512;
  static_assert(2 * SZ_L2 == SZ_L1, "E2 + U2 must tile the overlay region exactly");
  static_assert(SMEM <= 227 * 1024, "shared memory budget");
  static_assert(T * C <= 512, "TMEM budget");
  static_assert(NCH % 2 == 0 && T % 2 == 0, "concat halves must hold whole MMA K blocks; level-2 tiles whole");
};

struct LayerPlan {
  int nkb[5];        // MMA K blocks per tap
  int steps[5];      // taps * nkb
  int w_off[5];      // byte offset of the layer's first step in the packed image
  int total;
};

template <int C, bool BF16>
__host__ __device__ inline LayerPlan make_plan(int split_e1) {
  using G = Geo<C, BF16>;
  LayerPlan P{};
  P.nkb[0] = (!BF16 && split_e1) ? 3 : 1;
  P.nkb[1] = C / G::KPM;
  P.nkb[2] = C / G::KPM;
  P.nkb[3] = 2 * C / G::KPM;
  P.nkb[4] = 2 * C / G::KPM;
  int off = kHeaderBytes;
  for (int l = 0; l < 5; ++l) {
    P.steps[l] = taps_of(l) * P.nkb[l];
    P.w_off[l] = off;
    off += P.steps[l] * G::STEP_BYTES;
  }
  P.total = off;
  return P;
}

__device__ __forceinline__ float lrelu(float v) { return v >= 0.0f ? v : kLeaky * v; }

__device__ __forceinline__ uint32_t to_tf32(float v) {
  uint32_t r;
  asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(v));
  return r;
}
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
  const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
  uint32_t r;
  memcpy(&r, &h, 4);
  return r;
}
__device__ __forceinline__ void st_smem16(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// 16 consecutive channels of one row -> 16-byte chunks (4 for TF32, 2 for BF16) at
// dst + chunk * lbo, chunk counted from c0 / PER.
template <bool BF16>
__device__ __forceinline__ void store_row16(uint32_t dst_row, uint32_t lbo, int c0, const float (&v)[16]) {
  if (BF16) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      uint4 q;
      q.x = pack_bf16(v[8 * k + 0], v[8 * k + 1]);
      q.y = pack_bf16(v[8 * k + 2], v[8 * k + 3]);
      q.z = pack_bf16(v[8 * k + 4], v[8 * k + 5]);
      q.w = pack_bf16(v[8 * k + 6], v[8 * k + 7]);
      st_smem16(dst_row + (uint32_t)(c0 / 8 + k) * lbo, q);
    }
  } else {
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      uint4 q;
      q.x = to_tf32(v[4 * k + 0]);
      q.y = to_tf32(v[4 * k + 1]);
      q.z = to_tf32(v[4 * k + 2]);
      q.w = to_tf32(v[4 * k + 3]);
      st_smem16(dst_row + (uint32_t)(c0 / 4 + k) * lbo, q);
    }
  }
}

__device__ __forceinline__ void zero_rows(uint32_t buf, uint32_t lbo, int nch, int row) {
  for (int c = 0; c < nch; ++c) st_smem16(buf + (uint32_t)c * lbo + (uint32_t)row * 16u, make_uint4(0, 0, 0, 0));
}

enum { kE1 = 0, kE2 = 1, kB = 2, kD2 = 3, kD1 = 4 };

// Epilogue of one 128-row accumulator tile, executed by the four epilogue warps (thread = row m).
template <int C, bool BF16, int MODE>
__device__ __forceinline__ void epilogue_tile(uint32_t smem_base, uint32_t tmem_acc, int tile, int q, int lane,
                                              const float* __restrict__ par, int n_valid_int,
                                              float* __restrict__ probs_group) {
  using G = Geo<C, BF16>;
  const int m = 32 * q + lane;
  const float* bias = par + MODE * C;
  const uint32_t taddr = tmem_acc + ((uint32_t)(32 * q) << 16) + (uint32_t)(tile * C);
  // which interval of the group this row belongs to, its position, and whether it is a real output
  int interval, l;
  bool valid;
  if (MODE == kE1 || MODE == kD1) { interval = tile; l = m; valid = l < 100; }
  else if (MODE == kE2 || MODE == kD2) { interval = 2 * tile + (m >> 6); l = m & 63; valid = l < 50; }
  else { interval = 4 * tile + (m >> 5); l = m & 31; valid = l < 25; }
  const bool exists = interval < G::T;          // level-3 tiles may be wider than the group
  uint32_t dst_full = 0, dst_aux = 0, lbo_full = 0, lbo_aux = 0;
  if (MODE == kE1) {
    dst_full = smem_base + G::OFF_E1 + (uint32_t)(G::LEAD1 + 128 * tile + m) * 16u; lbo_full = G::LBO1;
    dst_aux = smem_base + G::OFF_R + (uint32_t)(G::LEAD2 + 64 * tile + (m >> 1)) * 16u; lbo_aux = G::LBO2;      // P1
    if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_R, G::LBO2, G::NCH, m);
  } else if (MODE == kE2) {
    dst_full = smem_base + G::OFF_R + (uint32_t)(G::LEAD2 + 128 * tile + m) * 16u; lbo_full = G::LBO2;          // E2
    dst_aux = smem_base + G::OFF_R + G::SZ_L2 + (uint32_t)(G::LEAD3 + 64 * tile + (m >> 1)) * 16u; lbo_aux = G::LBO3;  // P2
    if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_R, G::LBO2, G::NCH, m);
    if (tile == 0 && m >= 32 && m < 32 + G::LEAD3) zero_rows(smem_base + G::OFF_R + G::SZ_L2, G::LBO3, G::NCH, m - 32);
  } else if (MODE == kB) {
    dst_full = smem_base + G::OFF_R + G::SZ_L2 + (uint32_t)(G::LEAD2 + 256 * tile + 2 * m) * 16u; lbo_full = G::LBO2;  // U2
    if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_R + G::SZ_L2, G::LBO2, G::NCH, m);
  } else if (MODE == kD2) {
    dst_full = smem_base + G::OFF_R + (uint32_t)(G::LEAD1 + 256 * tile + 2 * m) * 16u; lbo_full = G::LBO1;      // U1
    if (tile == 0 && m < G::LEAD1) zero_rows(smem_base + G::OFF_R, G::LBO1, G::NCH, m);
  }
  float logit = 0.0f;
#pragma unroll 1
  for (int c0 = 0; c0 < C; c0 += 16) {
    uint32_t r[16];
    tmem_ld_x16(taddr + (uint32_t)c0, r);
    tmem_ld_wait();
    float v[16];
#pragma unroll
    for (int i = 0; i < 16; ++i) v[i] = lrelu(__uint_as_float(r[i]) + bias[c0 + i]);
    if (MODE == kD1) {
      const float* hw = par + 5 * C;
#pragma unroll
      for (int i = 0; i < 16; ++i) logit = fmaf(hw[c0 + i], v[i], logit);
      continue;
    }
    if (!valid) {
#pragma unroll
      for (int i = 0; i < 16; ++i) v[i] = 0.0f;
    }
    if (MODE == kE1 || MODE == kE2) {
      store_row16<BF16>(dst_full, lbo_full, c0, v);
      float pv[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) pv[i] = fmaxf(v[i], __shfl_xor_sync(0xffffffffu, v[i], 1));
      if ((lane & 1) == 0) store_row16<BF16>(dst_aux, lbo_aux, c0, pv);
    } else if (exists) {          // kB, kD2: nearest upsample = the same chunk into rows 2m and 2m + 1
      store_row16<BF16>(dst_full, lbo_full, c0, v);
      store_row16<BF16>(dst_full + 16u, lbo_full, c0, v);
    }
  }
  if (MODE == kD1) {
    if (valid && interval < n_valid_int) {
      const float a = logit + par[6 * C];
      probs_group[interval * kBins + l] = 1.0f / (1.0f + expf(-a));
    }
  }
}

// Interval histograms of one group -> X0 (operand-rounded, chunked layout).  128 threads.
template <int C, bool BF16>
__device__ __forceinline__ void load_x0(uint32_t smem_base, const float* __restrict__ hist, long long g0,
                                        int n_valid_int, int split, int tid) {
  using G = Geo<C, BF16>;
  const uint32_t x0 = smem_base + G::OFF_X0;
  if (BF16) {
    for (int it = tid; it < G::T * 100; it += 128) {
      const int t = it / 100, l = it % 100;
      float x[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) x[c] = t < n_valid_int ? __ldg(hist + (g0 + t) * kFcOut + c * kBins + l) : 0.0f;
      uint4 qv;
      qv.x = pack_bf16(x[0], x[1]); qv.y = pack_bf16(x[2], x[3]);
      qv.z = pack_bf16(x[4], x[5]); qv.w = pack_bf16(x[6], x[7]);
      st_smem16(x0 + (uint32_t)(G::LEAD1 + 128 * t + l) * 16u, qv);
    }
  } else {
    for (int it = tid; it < G::T * 200; it += 128) {
      const int t = it / 200, rem = it % 200, qc = rem / 100, l = rem % 100;
      float x[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) x[c] = t < n_valid_int ? __ldg(hist + (g0 + t) * kFcOut + (4 * qc + c) * kBins + l) : 0.0f;
      uint4 hi;
      hi.x = to_tf32(x[0]); hi.y = to_tf32(x[1]); hi.z = to_tf32(x[2]); hi.w = to_tf32(x[3]);
      const uint32_t row = (uint32_t)(G::LEAD1 + 128 * t + l) * 16u;
      st_smem16(x0 + (uint32_t)qc * G::LBO1 + row, hi);
      if (split) {
        uint4 lo;
        lo.x = to_tf32(x[0] - __uint_as_float(hi.x)); lo.y = to_tf32(x[1] - __uint_as_float(hi.y));
        lo.z = to_tf32(x[2] - __uint_as_float(hi.z)); lo.w = to_tf32(x[3] - __uint_as_float(hi.w));
        st_smem16(x0 + (uint32_t)(2 + qc) * G::LBO1 + row, lo);
      }
    }
  }
}

// Compile-time description of conv layer L (0 = e1 ... 4 = d1) as the MMA issuer sees it.
template <int C, bool BF16, int L>
struct Lay {
  using G = Geo<C, BF16>;
  static constexpr int TAPS = taps_of(L);
  static constexpr int PAD = (TAPS - 1) / 2;
  static constexpr int NKB = (L == 0) ? 1 : (L <= 2 ? C / G::KPM : 2 * C / G::KPM);   // K blocks per tap
  static constexpr int STEPS = TAPS * NKB;                                            // (e1 split: x3, runtime)
  static constexpr int LEAD = (L == 0 || L == 4) ? G::LEAD1 : ((L == 1 || L == 3) ? G::LEAD2 : G::LEAD3);
  static constexpr int LBO = (L == 0 || L == 4) ? G::LBO1 : ((L == 1 || L == 3) ? G::LBO2 : G::LBO3);
  static constexpr int NT = (L == 0 || L == 4) ? G::T : ((L == 1 || L == 3) ? G::T / 2 : (G::T + 3) / 4);
  static constexpr int HALF = (L >= 3) ? NKB / 2 : NKB;        // K blocks served by the first source buffer
  static constexpr int SRC0 = (L == 0) ? G::OFF_X0 : (L == 1) ? G::OFF_R : (L == 2) ? G::OFF_R + G::SZ_L2
                              : (L == 3) ? G::OFF_R + G::SZ_L2 /* U2 */ : G::OFF_R /* U1 */;
  static constexpr int SRC1 = (L == 3) ? G::OFF_R /* E2 */ : (L == 4) ? G::OFF_E1 : SRC0;
  // byte offset (from the CTA's shared-memory base) of the first chunk of K block kk
  __host__ __device__ static constexpr int a_off(int kk) {
    return kk < HALF ? SRC0 + 2 * kk * LBO : SRC1 + 2 * (kk - HALF) * LBO;
  }
};

template <bool BF16>
__device__ __forceinline__ void mma_lh(uint32_t d, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi,
                                       uint32_t idesc, uint32_t acc) {
  if (BF16) mma_f16_lh(d, a_lo, a_hi, b_lo, b_hi, idesc, acc);
  else mma_tf32_lh(d, a_lo, a_hi, b_lo, b_hi, idesc, acc);
}

struct RingState { int ring; uint32_t phase; };

// All MMAs of layer L for the group: tap-major over ring stages, every stage used by all NT tiles.
// The warp walks the (uniform) schedule; one elected lane issues a whole stage worth of MMAs whose
// descriptors differ from the stage origin by compile-time constants.
template <int C, bool BF16, int L>
__device__ __forceinline__ void mma_layer(uint32_t sb, uint32_t tmem_acc, uint32_t bar0, RingState& rs,
                                          int steps_rt) {
  using G = Geo<C, BF16>;
  using Y = Lay<C, BF16, L>;
  constexpr int SPS = G::SPS;
  static_assert(Y::HALF % SPS == 0 || SPS % Y::NKB == 0, "a ring stage is either part of one source's K blocks or whole taps");
  constexpr uint32_t idesc = instr_desc(BF16 ? kFmtBF16 : kFmtTF32, 128, C);
  constexpr uint32_t hi = (128u >> 4) | (1u << 14);                    // SBO = 128 B, descriptor version 1
  constexpr uint32_t a_lbo = (uint32_t)(Y::LBO >> 4) << 16;
  constexpr uint32_t b_lbo = (uint32_t)((C * 16) >> 4) << 16;
  const int steps = (L == 0) ? steps_rt : Y::STEPS;
  for (int f = 0; f < steps; f += SPS) {
    const int n = min(SPS, steps - f);
    mbar_wait(bar0 + 8u * rs.ring, rs.phase);
    tc_fence_after_sync();
    const uint32_t b0 = b_lbo + ((sb + G::OFF_RING + rs.ring * kStageBytes) >> 4);
    uint32_t a0 = a_lbo + (sb >> 4);          // stage origin: descriptor low word of tile 0, step f
    if (L == 0) {
      // e1: one K block per step; steps run [pass][tap], pass 1 reads the low-part chunks (split)
    } else if (Y::HALF >= SPS) {
      const int j0 = f / Y::NKB, kk0 = f % Y::NKB;
      const int off = kk0 < Y::HALF ? Y::SRC0 + 2 * kk0 * Y::LBO : Y::SRC1 + 2 * (kk0 - Y::HALF) * Y::LBO;
      a0 += (uint32_t)(off >> 4) + (uint32_t)(Y::LEAD + j0 - Y::PAD);
    } else {
      a0 += (uint32_t)(Y::SRC0 >> 4) + (uint32_t)(Y::LEAD + f / Y::NKB - Y::PAD);
    }
    if (elect_one()) {
#pragma unroll
      for (int i = 0; i < SPS; ++i) {
        if (i < n) {
          uint32_t a;
          if (L == 0) {
            const int step = f + i, pass = step / 25, j = step - 25 * pass;
            a = a0 + (uint32_t)((G::OFF_X0 + (pass == 1 ? 2 * G::LBO1 : 0)) >> 4) + (uint32_t)(Y::LEAD + j - Y::PAD);
          } else if (Y::HALF >= SPS) {
            a = a0 + (uint32_t)(i * ((2 * Y::LBO) >> 4));
          } else {
            a = a0 + (uint32_t)((Y::a_off(i % Y::NKB) - Y::SRC0) >> 4) + (uint32_t)(i / Y::NKB);
          }
          const uint32_t b = b0 + (uint32_t)(i * (G::STEP_BYTES >> 4));
          const uint32_t acc = (i > 0) ? 1u : (f > 0 ? 1u : 0u);
#pragma unroll
          for (int t = 0; t < Y::NT; ++t)
            mma_lh<BF16>(tmem_acc + (uint32_t)(t * C), a + 128u * t, hi, b, hi, idesc, acc);
        }
      }
      mma_commit(bar0 + 8u * (kStages + rs.ring));      // frees the ring slot when these MMAs retire
    }
    __syncwarp();
    if (++rs.ring == kStages) { rs.ring = 0; rs.phase ^= 1u; }
  }
}

template <int C, bool BF16>
__global__ void __launch_bounds__(kTcThreads, 1)
k_unet_tc(const float* __restrict__ hist, int n_int, const unsigned char* __restrict__ wpack, int split_e1,
          float* __restrict__ probs) {
  using G = Geo<C, BF16>;
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t sb = smem_u32(smem);
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // provably warp-uniform role index
  float* par = reinterpret_cast<float*>(smem + G::OFF_PAR);
  const uint32_t bar0 = sb + G::OFF_BAR;
  auto full_bar = [&](int s) { return bar0 + 8u * s; };
  auto empty_bar = [&](int s) { return bar0 + 8u * (kStages + s); };
  const uint32_t accum_bar = bar0 + 8u * (2 * kStages);
  const uint32_t epi_bar = bar0 + 8u * (2 * kStages + 1);
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + G::OFF_BAR + 8 * (2 * kStages + 2));
  const LayerPlan P = make_plan<C, BF16>(split_e1);

  // ---- one-time setup: zero the activation buffers (gap / halo rows must be zero), parameters, barriers
  for (int i = tid; i < G::OFF_RING / 16; i += kTcThreads) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  for (int i = tid; i < 6 * C + 1; i += kTcThreads) par[i] = reinterpret_cast<const float*>(wpack)[i];
  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
    mbar_init(accum_bar, 1);
    mbar_init(epi_bar, 128);
    fence_mbar_init();
  }
  if (warp == 1) tmem_alloc(smem_u32(const_cast<uint32_t*>(tmem_slot)), G::TMEM_COLS);
  fence_proxy_async_smem();
  tc_fence_before_sync();
  __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_acc = *tmem_slot;

  const int n_groups = (n_int + G::T - 1) / G::T;

  if (warp == 0) {
    // ===================== weight producer: streams every layer's MMA steps through the ring
    if (lane == 0) {
      int ring = 0;
      uint32_t phase = 0;
      for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
        for (int l = 0; l < 5; ++l) {
          const unsigned char* src = wpack + P.w_off[l];
          for (int s0 = 0; s0 < P.steps[l]; s0 += G::SPS) {
            const int n = min(G::SPS, P.steps[l] - s0);
            mbar_wait(empty_bar(ring), phase ^ 1u);
            mbar_arrive_expect_tx(full_bar(ring), (uint32_t)(n * G::STEP_BYTES));
            bulk_g2s(sb + G::OFF_RING + ring * kStageBytes, src + (size_t)s0 * G::STEP_BYTES,
                     (uint32_t)(n * G::STEP_BYTES), full_bar(ring));
            if (++ring == kStages) { ring = 0; phase ^= 1u; }
          }
        }
      }
    }
  } else if (warp == 1) {
    // ===================== MMA issuer (whole warp walks the schedule, one elected lane issues)
    RingState rs{0, 0u};
    uint32_t epi_phase = 0;
    for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
#pragma unroll
      for (int l = 0; l < 5; ++l) {
        mbar_wait(epi_bar, epi_phase);
        epi_phase ^= 1u;
        tc_fence_after_sync();
        if (l == 0) mma_layer<C, BF16, 0>(sb, tmem_acc, bar0, rs, P.steps[0]);
        else if (l == 1) mma_layer<C, BF16, 1>(sb, tmem_acc, bar0, rs, 0);
        else if (l == 2) mma_layer<C, BF16, 2>(sb, tmem_acc, bar0, rs, 0);
        else if (l == 3) mma_layer<C, BF16, 3>(sb, tmem_acc, bar0, rs, 0);
        else mma_layer<C, BF16, 4>(sb, tmem_acc, bar0, rs, 0);
        if (elect_one()) mma_commit(accum_bar);
        __syncwarp();
      }
    }
  } else {
    // ===================== epilogue warps (128 threads): thread = accumulator row
    const int q = warp & 3, et = tid - 64;
    uint32_t acc_phase = 0;
    bool first = true;
    for (int g = blockIdx.x; g < n_groups; g += gridDim.x) {
      const long long g0 = (long long)g * G::T;
      const int n_valid = (int)min((long long)G::T, (long long)n_int - g0);
      if (first) {
        load_x0<C, BF16>(sb, hist, g0, n_valid, split_e1, et);
        fence_proxy_async_smem();
        mbar_arrive(epi_bar);
        first = false;
      }
      float* pg = probs + g0 * kBins;
#pragma unroll 1
      for (int l = 0; l < 5; ++l) {
        if (l == 4) {
          // the next group's input is staged while this group's d1 MMAs run (X0 is dead after e1)
          const int gn = g + gridDim.x;
          if (gn < n_groups) {
            const long long gn0 = (long long)gn * G::T;
            load_x0<C, BF16>(sb, hist, gn0, (int)min((long long)G::T, (long long)n_int - gn0), split_e1, et);
          }
        }
        mbar_wait(accum_bar, acc_phase);
        acc_phase ^= 1u;
        tc_fence_after_sync();
        if (l == 0) { for (int t = 0; t < G::T; ++t) epilogue_tile<C, BF16, kE1>(sb, tmem_acc, t, q, lane, par, n_valid, pg); }
        else if (l == 1) { for (int t = 0; t < G::T / 2; ++t) epilogue_tile<C, BF16, kE2>(sb, tmem_acc, t, q, lane, par, n_valid, pg); }
        else if (l == 2) { for (int t = 0; t < (G::T + 3) / 4; ++t) epilogue_tile<C, BF16, kB>(sb, tmem_acc, t, q, lane, par, n_valid, pg); }
        else if (l == 3) { for (int t = 0; t < G::T / 2; ++t) epilogue_tile<C, BF16, kD2>(sb, tmem_acc, t, q, lane, par, n_valid, pg); }
        else { for (int t = 0; t < G::T; ++t) epilogue_tile<C, BF16, kD1>(sb, tmem_acc, t, q, lane, par, n_valid, pg); }
        fence_proxy_async_smem();
        tc_fence_before_sync();
        mbar_arrive(epi_bar);
      }
    }
  }
  tc_fence_before_sync();
  __syncthreads();
  if (warp == 1) {
    __syncwarp();
    tmem_dealloc(tmem_acc, G::TMEM_COLS);
  }
}

// ------------------------------------------------------------------ host side
float tf32_rna(float v) {
  uint32_t u;
  memcpy(&u, &v, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return v;
  u = (u + 0x1000u) & 0xffffe000u;
  float r;
  memcpy(&r, &u, 4);
  return r;
}
uint16_t bf16_rne(float v) {
  uint32_t u;
  memcpy(&u, &v, 4);
  if ((u & 0x7f800000u) == 0x7f800000u) return (uint16_t)(u >> 16);
  u += 0x7fffu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

template <int C, bool BF16>
void pack_impl(const pvf_weights* w, int split_e1, unsigned char* dst) {
  using G = Geo<C, BF16>;
  const LayerPlan P = make_plan<C, BF16>(split_e1);
  memset(dst, 0, P.total);
  float* hdr = reinterpret_cast<float*>(dst);
  for (int l = 0; l < 5; ++l) memcpy(hdr + l * C, w->conv_b[l], sizeof(float) * C);
  memcpy(hdr + 5 * C, w->conv_w[5], sizeof(float) * C);
  hdr[6 * C] = w->conv_b[5][0];
  const int cin[5] = {kHistCh, C, C, 2 * C, 2 * C};
  for (int l = 0; l < 5; ++l) {
    const int K = taps_of(l);
    const float* W = w->conv_w[l];          // [C][cin][K]
    for (int j = 0; j < K; ++j)
      for (int kk = 0; kk < P.nkb[l]; ++kk) {
        // step order inside a layer: [tap][K block]; the e1 split runs [pass][tap] (pass = K block)
        const size_t step_idx = (l == 0) ? (size_t)kk * K + j : (size_t)j * P.nkb[l] + kk;
        unsigned char* step = dst + P.w_off[l] + step_idx * G::STEP_BYTES;
        for (int h = 0; h < 2; ++h)
          for (int n = 0; n < C; ++n)
            for (int e = 0; e < G::PER; ++e) {
              int ci = (2 * kk + h) * G::PER + e;
              int pass = 0;                  // e1 split: k block 0 and 1 carry W_hi, k block 2 carries W_lo
              if (l == 0 && P.nkb[0] == 3) { ci = h * G::PER + e; pass = kk; }
              float v = ci < cin[l] ? W[((size_t)n * cin[l] + ci) * K + j] : 0.0f;
              unsigned char* p = step + ((size_t)h * C + n) * 16 + e * G::ES;
              if (BF16) {
                const uint16_t b = bf16_rne(v);
                memcpy(p, &b, 2);
              } else {
                const float hi = tf32_rna(v);
                const float out = (pass == 2) ? tf32_rna(v - hi) : hi;
                memcpy(p, &out, 4);
              }
            }
      }
  }
}

template <int C, bool BF16>
void launch_impl(const float* hist, int n_int, const void* packed, int split_e1, float* probs, int sm_count,
                 cudaStream_t s) {
  using G = Geo<C, BF16>;
  const int n_groups = (n_int + G::T - 1) / G::T;
  const int grid = n_groups < sm_count ? n_groups : sm_count;
  k_unet_tc<C, BF16><<<grid, kTcThreads, G::SMEM, s>>>(hist, n_int, static_cast<const unsigned char*>(packed),
                                                      split_e1, probs);
}

template <int C, bool BF16>
cudaError_t setup_impl() {
  return cudaFuncSetAttribute(k_unet_tc<C, BF16>, cudaFuncAttributeMaxDynamicSharedMemorySize, Geo<C, BF16>::SMEM);
}

#define PVF_TC_DISPATCH(CALL)                                     \
  do {                                                            \
    const bool bf = precision == PVF_PREC_BF16;                   \
    if (channels == 64) { if (bf) CALL(64, true); else CALL(64, false); }      \
    else if (channels == 32) { if (bf) CALL(32, true); else CALL(32, false); } \
    else { if (bf) CALL(16, true); else CALL(16, false); }        \
  } while (0)

}  // namespace

size_t unet_tc_packed_bytes(int channels, int precision, int split_mask) {
  size_t r = 0;
#define PVF_CALL(C_, B_) r = (size_t)make_plan<C_, B_>(split_mask & 1).total
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
  return r;
}

void unet_tc_pack(const pvf_weights* w, int channels, int precision, int split_mask, void* host_dst) {
#define PVF_CALL(C_, B_) pack_impl<C_, B_>(w, split_mask & 1, static_cast<unsigned char*>(host_dst))
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
}

cudaError_t unet_tc_setup(int channels, int precision, int split_mask) {
  if (channels != 64 && channels != 32 && channels != 16) return cudaErrorInvalidValue;
  if (split_mask & ~1) return cudaErrorInvalidValue;          // only the e1 split is built
  if (precision == PVF_PREC_BF16 && split_mask) return cudaErrorInvalidValue;
  cudaError_t e = cudaSuccess;
#define PVF_CALL(C_, B_) e = setup_impl<C_, B_>()
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
  return e;
}

void launch_unet_tc(const float* hist, int n_intervals_total, const void* packed_dev, int channels, int precision,
                    int split_mask, float* probs, int sm_count, cudaStream_t s) {
  if (n_intervals_total <= 0) return;
#define PVF_CALL(C_, B_) launch_impl<C_, B_>(hist, n_intervals_total, packed_dev, split_mask & 1, probs, sm_count, s)
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
}

}  // namespace pvf
