// a3, tensor-core path -- the 1D UNet per z-interval as implicit-GEMM convolutions on tcgen05 / TMEM.
//
// PAPER.md:29 "5-layer UNet architecture (64 channels deployed)", PAPER.md:63-76 (the CNN is the
// bottleneck); topology from BASELINE.json config 0 (see k_unet_simt.cu); north_star (c): implicit
// GEMM on tcgen05/TMEM, pool / upsample / concat / activations fused into the epilogues, the
// intermediates stay in shared memory / TMEM.  DESIGN.md section 4.3 has the derivation.
//
// Mapping.  A conv layer is  D[m, n] = sum_j sum_ci  A[m + j - p, ci] * W_j[ci, n]  with m = position
// (M), n = output channel.  Taps are taken in (even, odd) pairs that share one read of A:
//     D[m] = E0[m] + E1[m + 1],   E0[m] = sum_u A[m + 2u - p] W_2u,   E1[m'] = sum_u A[m' + 2u - p] W_2u+1
// so one (tap pair u, 32-byte channel block) is one tcgen05.mma of shape 128 x 2C x (8 TF32 | 16 BF16)
// with B = [W_2u | W_2u+1]; the epilogue adds the E1 half of the next row.  Activations live in shared memory in the K-major no-swizzle UMMA
// layout  [channel chunk of 16 B][row][16 B]  (core matrix = 8 rows x 16 B contiguous), so a tap
// shift is a pure bump of the descriptor start address by 16 B per row, the skip concat is a second
// base address, and an epilogue thread (= one row) writes whole 16-byte chunks, conflict free.
// Intervals sit at row stride 128 / 64 / 32 (L = 100 / 50 / 25); the rows between them are zero and
// double as the "same" padding.  One persistent CTA takes a group of T intervals through all five
// layers; each weight slice is streamed from L2 once per group (1D bulk copies into a ring of 16 KB
// stages -- also per CTA of a pair, see Geo::STAGE_BYTES) and used by every tile of the group.
//
// CTA pairs (template parameter CG = 2, the default of the binding): a cluster of two CTAs runs every MMA as
// one tcgen05.mma.cta_group::2 of M = 256 issued by the leader; each CTA keeps its own group's activations
// and accumulators and supplies half of the weight rows (rank 0 the even tap of a pair, rank 1 the odd one).
//
// Schedule.  The MMA issuer never waits for an epilogue in steady state: d1 is split into the half
// that reads the e1 skip (d1E, needs only e1's epilogue) and the half that reads up(d2) (d1U); d1E
// is cut in three parts that run while the epilogues of e2, b and d2 drain, and the NEXT group's e1
// runs before d1U so that its epilogue overlaps d1U:
//     e2 | d1E.1 | b | d1E.2 | d2 | d1E.3 | e1(next) | d1U        (weight image is packed in this order)
// TMEM holds two accumulator regions: A (d1: T/2 low-resolution tiles, polyphase; direct d1: T tiles) and B (e1: T tiles; e2, b,
// d2: its first tiles); FX adds A2 (the upsampled half of d1 accumulates on its own).
// Roles: warp 0 = weight producer, warp 1 = MMA issuer (warp-uniform schedule, one elected lane
// issues; in the peer CTA of a pair it relays "my half of the stage has landed"), warps 2.. = epilogue in
// sets of four (TMEM -> registers -> bias, LeakyReLU, TF32/BF16 rounding, pool / upsample -> shared
// memory; d1's epilogue fuses the 1x1 head + sigmoid and writes out_probs).
// TF32 mode: the e1 layer (raw histogram input) can run as two passes on BF16 pieces (split_mask bit 0).
//
// Polyphase d1 (groups of an even number of intervals, i.e. every format but FX): d1 = conv25(cat[up2(d2), e1]) is computed on
// the LOW-resolution rows i (outputs 2i and 2i + 1 = the two "phases" side by side in N):
//   * the nearest-upsampled half needs no upsampling: out[2i + p] = sum_d d2[i + d] * Wp[d], d = -6 .. 6, with
//     W0[d] = W[2d + 12] + W[2d + 13], W1[d] = W[2d + 11] + W[2d + 12] (taps that read the same low-resolution sample are
//     added on the host) -- 13 MMA steps per K block on HALF as many rows instead of 13 tap pairs on all rows;
//   * the skip half reads e1 de-interleaved (row i holds positions 2i and 2i + 1 as 2C channels): same MMA time as before,
//     no row shift in the epilogue.
// The accumulator tile is [low-resolution row][phase 0: C | phase 1: C]; the epilogue thread of row i computes both
// logits and stores two probabilities.  ~17 % fewer MMA cycles per interval (SURVEY.md H1 "polyphase weights").
//
// FP32-accurate mode (format 3, "FX"; PVF_PREC_FP32 on the tensor cores, BASELINE.json config 0 "FP32"): every product a w is
// taken as  tf32(a) tf32(w)  +  [a - tf32(a)] w  +  a [w - tf32(w)]  -- the first term one kind::tf32 MMA, the two small
// terms ONE kind::f16 MMA over BF16 pieces stacked along K: A' = [a_lo (8 channels) | bf16(a) (the same 8 channels)],
// B' = [bf16(w) | w_lo].  The small terms are 2^-11 of the product, so 8-bit pieces leave ~2^-20 relative error per
// product at 2 MMA time units per (tap pair, 8 channels) -- a three-pass TF32 split needs 3.  Activations live in shared
// memory as three arrays per buffer (HI: TF32 chunks, LO and HB: BF16 chunks; 8 bytes per value), which fits for groups
// of ONE interval; the weight image interleaves a main and a correction step per (tap pair, K block).
#pragma nv_diag_suppress 128   // "loop is not reachable": template branches that return early for some instantiations
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <cstring>
#include <type_traits>
#include <vector>

#include "pvf_internal.cuh"
#include "pdl.cuh"
#include "umma.cuh"

namespace pvf {
using namespace umma;

namespace {

// Epilogue warps come in sets of four (a warp reaches TMEM lanes 32 * (warp % 4) ..): two sets at 64 channels
// (MMA-bound), four at 32 / 16 channels (epilogue work ~ C, MMA work ~ C^2: those widths are epilogue-bound).
constexpr int epi_sets(int C) { return C == 64 ? 2 : 4; }
constexpr int kMaxStages = 8;
constexpr int kStageBytes = 16384;
constexpr int kHeaderBytes = 2048;          // biases [5][C], head weight [C], head bias
constexpr int kBarBytes = 768;

// sub-layers as the MMA issuer sees them
enum { sE1 = 0, sE2 = 1, sB = 2, sD2 = 3, sD1U = 4, sD1E = 5 };
// weight-image segments in streaming order
enum { gE2 = 0, gD1Ea = 1, gB = 2, gD1Eb = 3, gD2 = 4, gD1Ec = 5, gE1 = 6, gD1U = 7, kSegs = 8 };

// BF16: operand format -- 0 = TF32 (4-byte), 1 = BF16, 2 = FP16 (2-byte; everything that only depends on
// the operand size treats 1 and 2 alike)
// CG: CTAs per MMA -- 1, or 2 = a cluster of two CTAs (cta_group::2) that run one M = 256 MMA per step: each CTA
// supplies its own 128 activation rows (its own group of intervals) and HALF of the weight rows (rank 0 the even
// tap of a pair, rank 1 the odd tap), so per CTA the weight stream and the B-operand reads are halved.
// TT: intervals per group, 0 = the default below (an explicit value is for experiments: groups of one interval were
// measured as a small-batch schedule -- 41 -> 35 us for one event -- and dropped again when the polyphase d1, which needs
// an even group, gave the same gain for every batch size with one code path and bit-identical results).
constexpr bool is16(int fmt) { return fmt == 1 || fmt == 2; }

template <int C, int BF16, int CG = 1, int TT = 0>
struct Geo {
  static constexpr bool B16 = is16(BF16);            // 2-byte operands
  static constexpr bool FX = BF16 == 3;              // FP32-accurate: TF32 main array + BF16 correction arrays
  static constexpr int ES = B16 ? 2 : 4;             // operand element size (main array)
  static constexpr int PER = 16 / ES;                // channels per 16-byte chunk (main array)
  static constexpr int KPM = 2 * PER;                // channels per MMA (32 bytes of K)
  static constexpr int NCH = C / PER;                // chunks of a C-channel activation (main array)
  static constexpr int NCHB = FX ? 2 * NCH : NCH;    // chunks per buffer: FX adds LO (NCH/2 chunks of 8 BF16) and HB (same)
  static constexpr int XCH = B16 ? 2 : 4;            // chunks of the input buffer X0 (FX: hi0 hi1 lo hb)
  static constexpr int NKB1 = C / KPM;               // MMA K blocks per tap over C channels
  static constexpr int PH = FX ? 2 : 1;              // MMA steps per (tap pair, K block): FX = main + correction
  static constexpr int NOUT = 2 * C;                 // MMA N: the outputs of an (even, odd) tap pair side by side
  static constexpr int T = TT ? TT : (FX ? 1 : ((C == 64) ? 2 : (C == 32 ? 4 : (B16 ? 8 : 4))));   // intervals per group (TMEM: 4*T*C <= 512)
  // Lead (halo) rows of a chunk.  (12 lead rows at levels 2 / 3 -- chunk pitch 64 mod 128 bytes, so that the chunk pairs an
  // (even, odd) lane pair writes fall into different bank halves -- were measured: C = 32 BF16 5.57 -> 5.98 ms per 8000 events,
  // the tensor core's own operand reads prefer the 128-byte-aligned pitch.)
  static constexpr int LEAD1 = 16, LEAD2 = 8, LEAD3 = 8;
  // rows per chunk = lead halo + T interval slots; reads past the last slot (garbage output rows only)
  // land in the following chunk / buffer, which is always inside the CTA's allocation
  static constexpr int ROWS1 = LEAD1 + 128 * T, ROWS2 = LEAD2 + 64 * T, ROWS3 = LEAD3 + 32 * T;
  static constexpr int LBO1 = ROWS1 * 16, LBO2 = ROWS2 * 16, LBO3 = ROWS3 * 16;
  static constexpr bool PP = (T % 2 == 0);           // polyphase d1 (see the header); FX (groups of one interval) runs d1 directly
  static constexpr int NB = NOUT / CG;               // B-operand rows this CTA holds
  static constexpr int STEP_BYTES = 2 * NB * 16;     // one MMA's B operand in this CTA: [2 chunks][NB rows][16 B]
  // Ring stage.  One stage costs the producer, the relay and the MMA issuer a fixed ~400 cycles of mbarrier round trips
  // each (measured: a single thread issues one bulk copy per ~380 cycles whatever its size), so a stage must hold at least
  // that much tensor work: with the polyphase d1 most steps feed ONE tile (68 cycles), 4-step stages left the tensor pipe
  // idle 30 % of the time.  A CTA of a pair therefore takes 16 KB stages like a single CTA (8 steps at C = 64) whenever
  // three of them fit; the FX format (8-byte activations) keeps 8 KB.
  static constexpr int STAGE_HALF = kStageBytes / CG;
  // shared-memory map (bytes)
  static constexpr int SZ_L1 = NCHB * LBO1;          // a C-channel buffer at L = 100
  static constexpr int SZ_L2 = NCHB * LBO2;          //                     at L = 50
  static constexpr int SZ_E1 = PP ? 2 * SZ_L2 : SZ_L1;   // e1 skip: de-interleaved on level-2 rows (polyphase d1) | level-1 rows
  static constexpr int SZ_R = PP ? 2 * SZ_L2 : SZ_L1;    // (E2 | U2), then d2 in E2's place (polyphase) | U1 over both
  static constexpr int OFF_E1 = 0;                   // e1 skip (dedicated)
  static constexpr int OFF_R = OFF_E1 + SZ_E1;       // overlay: (E2 | U2) then U1 / d2; P2 sits in U2's place
  static constexpr int OFF_XP = OFF_R + SZ_R;        // X0 (input); direct d1: overlaid by P1 = pool(e1)
  // Polyphase: P1 lives in U2's place (second half of R) -- free from d2's MMAs (the last readers of U2) until e2's epilogue
  // writes P2 there, and the NEXT group's e1 epilogue (the writer of P1) only runs after this group's d2 MMAs have retired.
  // XP then holds X0 alone, which is what buys TF32 a fourth 16 KB ring stage.  Direct d1 (FX): U1 covers all of R while the
  // next e1 epilogue runs, so P1 stays in XP.
  static constexpr int OFF_P1 = PP ? OFF_R + SZ_L2 : OFF_XP;
  static constexpr int SZ_XP = PP ? XCH * LBO1 : ((XCH * LBO1 > SZ_L2) ? XCH * LBO1 : SZ_L2);
  static constexpr int OFF_RING = OFF_XP + SZ_XP;
  static constexpr int SETS = epi_sets(C);
  static constexpr int EPI_THREADS = 128 * SETS, THREADS = 64 + EPI_THREADS;
  static constexpr int SCR_BYTES = SETS * 2 * 4 * C * 4;   // epilogue row-exchange scratch: [set][2 buffers][4 warps][C floats]
  static constexpr int RING_FREE = 227 * 1024 - kHeaderBytes - kBarBytes - SCR_BYTES - OFF_RING;
  static constexpr int STAGE_BIG = (kStageBytes / STEP_BYTES > 16) ? 16 * STEP_BYTES : kStageBytes;
  static constexpr int STAGE_HUGE = 16 * STEP_BYTES;       // 16 steps (the most the d1E split points allow), if four fit
  static constexpr int STAGE_BYTES = (RING_FREE / STAGE_HUGE >= 4) ? STAGE_HUGE : (RING_FREE / STAGE_BIG >= 3) ? STAGE_BIG : STAGE_HALF;
  static constexpr int SPS = STAGE_BYTES / STEP_BYTES;   // MMA steps per ring stage
  static constexpr int STAGES_FIT = RING_FREE / STAGE_BYTES;
#ifndef PVF_UNET_MAX_STAGES
#define PVF_UNET_MAX_STAGES 12
#endif
  static constexpr int MAX_STAGES = CG == 2 ? PVF_UNET_MAX_STAGES : kMaxStages;   // measured: depth >= 6 changes nothing (bf16 and tf32)
  static constexpr int STAGES = STAGES_FIT < MAX_STAGES ? STAGES_FIT : MAX_STAGES;   // weight ring depth
  static constexpr int OFF_PAR = OFF_RING + STAGES * STAGE_BYTES;   // biases + head (floats)
  static constexpr int OFF_SCR = OFF_PAR + kHeaderBytes;
  static constexpr int OFF_BAR = OFF_SCR + SCR_BYTES;
  static constexpr int SMEM = OFF_BAR + kBarBytes;
  // mbarriers (8 bytes each): full[S] empty[S] peer_full[S] accum[5] epi[6] peer_epi[6], then the TMEM slot
  static constexpr int BAR_ACCUM = 3 * STAGES, BAR_EPI = BAR_ACCUM + 5, BAR_PEPI = BAR_EPI + 6, BAR_SLOT = BAR_PEPI + 6;
  static_assert(8 * BAR_SLOT + 4 <= kBarBytes, "barrier block");
  // TMEM columns: region A = [0, T*2C) (d1), region B = [T*2C, 2*T*2C) (e1; e2, b, d2 use its head);
  // an accumulator tile is 2C columns: E0 (even taps) | E1 (odd taps)
  static constexpr int COL_A = 0, COL_B = T * NOUT;
  // FX: the two halves of d1 accumulate in SEPARATE tiles (region A for the skip half, A2 for the upsampled half) and
  // the epilogue adds them in FP32: a tensor-core accumulator is not rounded to nearest, and with 400+ accumulating MMAs
  // per tile that rounding is what is left of the error once the products are FP32-accurate (measured on config 1: one
  // tile max |dP| 1.9e-5, two tiles 1.2e-5; a third tile for the last part of the skip half changed nothing)
  static constexpr int COL_A2 = 2 * T * NOUT;
  static constexpr int TMEM_USED = (FX ? 3 : 2) * T * NOUT;
  static constexpr int TMEM_COLS = (TMEM_USED <= 32) ? 32 : (TMEM_USED <= 64) ? 64 : (TMEM_USED <= 128) ? 128
                                   : (TMEM_USED <= 256) ? 256 : 512;
  // d1E parts (steps): run while the epilogues of e2 / b / d2 drain; multiples of every SPS
  static constexpr int D1E_STEPS = 13 * NKB1 * PH * (PP ? 2 : 1);   // 13 tap pairs; polyphase: 13 offsets x 2C channels
  // polyphase: a step feeds T/2 tiles instead of T, so the parts that cover the e2 / b epilogues are twice as many steps
  // (with 16 the issuer waited 3 % of its time for each of the two epilogues)
  static constexpr int D1E_PART = ((PP && C == 64) ? 32 : 16) * PH;   // (narrower widths: measured slower with 32)
  static constexpr int D1E_A = D1E_STEPS < D1E_PART ? D1E_STEPS : D1E_PART;
  static constexpr int D1E_B = (D1E_STEPS - D1E_A) < D1E_PART ? (D1E_STEPS - D1E_A) : D1E_PART;
  static constexpr int D1E_C = D1E_STEPS - D1E_A - D1E_B;
  static_assert(PP || 2 * SZ_L2 == SZ_L1, "E2 + U2 must tile the overlay region exactly (direct d1: U1 overlays both)");
  static constexpr bool kFits = SMEM <= 227 * 1024 && STAGES >= 3;   // checked where a kernel is instantiated (the helper
                                                                     // templates read layout constants from Geo<.., CG = 1>)
  static_assert(TMEM_USED <= 512, "TMEM budget");
  static_assert(NCH % 2 == 0 && (T % 2 == 0 || T == 1), "whole MMA K blocks per source; level-2 tiles whole (or one interval)");
  static_assert(16 % SPS == 0 && SPS % PH == 0, "d1E parts must start on ring-stage boundaries; whole (main, correction) pairs per stage");
  static_assert(!FX || T == 1, "the FP32-accurate format runs on groups of one interval");
};

// Steps and byte offsets of the weight-image segments (host packer, producer and issuer agree on it).
struct Plan {
  int e1_steps;            // 13 tap pairs, x2 with the e1 hi/lo split (TF32 mode)
  int seg_steps[kSegs];
  int seg_off[kSegs];      // bytes from the start of the image
  int total;
};

// With CG = 2 the image is two such images back to back (rank 0 | rank 1), each `total` bytes with its own header.
template <int C, int BF16, int CG>
__host__ __device__ inline Plan make_plan(int split_e1) {
  using G = Geo<C, BF16, CG>;          // (nothing here depends on the group size)
  Plan P{};
  // 16-bit modes: the 8 input channels fill half of an MMA's K = 16, so one e1 step takes TWO tap pairs (7 steps)
  // TF32 with the e1 split: 13 steps [a1 | a2] x [w1 | w1] + 7 steps [a1(pair 2w) | a1(pair 2w+1)] x [w2 | w2]
  // FX: 13 tap pairs x (main, correction)
  // FP16 with the e1 split: the same 13 + 7 steps on FP16 pieces (the BF16 kernel has no split: its tolerance is set by the
  // 8-bit mantissa of every other layer)
  P.e1_steps = G::FX ? 26 : ((split_e1 && BF16 != 1) ? 20 : (G::B16 ? 7 : 13));
  P.seg_steps[gE2] = 8 * G::NKB1 * G::PH;
  P.seg_steps[gD1Ea] = G::D1E_A;
  P.seg_steps[gB] = 3 * G::NKB1 * G::PH;
  P.seg_steps[gD1Eb] = G::D1E_B;
  P.seg_steps[gD2] = 8 * 2 * G::NKB1 * G::PH;
  P.seg_steps[gD1Ec] = G::D1E_C;
  P.seg_steps[gE1] = P.e1_steps;
  P.seg_steps[gD1U] = 13 * G::NKB1 * G::PH;
  int off = kHeaderBytes;
  for (int s = 0; s < kSegs; ++s) {
    P.seg_off[s] = off;
    off += P.seg_steps[s] * G::STEP_BYTES;
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
// two floats -> one 32-bit word of 16-bit operands (FMT 1 = BF16, 2 = FP16), round to nearest even
template <int FMT>
__device__ __forceinline__ uint32_t pack16(float lo, float hi) {
  uint32_t r;
  if (FMT == 2) {
    const __half2 h = __floats2half2_rn(lo, hi);
    memcpy(&r, &h, 4);
  } else {
    const __nv_bfloat162 h = __floats2bfloat162_rn(lo, hi);
    memcpy(&r, &h, 4);
  }
  return r;
}
__device__ __forceinline__ void st_smem16(uint32_t addr, uint4 v) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
}

// 16 consecutive channels of one row -> 16-byte chunks (4 for TF32, 2 for BF16) at
// dst + chunk * lbo, chunk counted from c0 / PER.  FX (NCHM = chunks of the main array): the TF32 chunks, then
// lo = bf16(v - tf32(v)) into the LO array (chunks NCHM ..) and bf16(v) into the HB array (chunks 3 NCHM / 2 ..).
template <int BF16, int NCHM>
__device__ __forceinline__ void store_row16(uint32_t dst_row, uint32_t lbo, int c0, const float (&v)[16]) {
  if (is16(BF16)) {
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      uint4 q;
      q.x = pack16<BF16>(v[8 * k + 0], v[8 * k + 1]);
      q.y = pack16<BF16>(v[8 * k + 2], v[8 * k + 3]);
      q.z = pack16<BF16>(v[8 * k + 4], v[8 * k + 5]);
      q.w = pack16<BF16>(v[8 * k + 6], v[8 * k + 7]);
      st_smem16(dst_row + (uint32_t)(c0 / 8 + k) * lbo, q);
    }
  } else {
    float lo[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      uint4 q;
      q.x = to_tf32(v[4 * k + 0]);
      q.y = to_tf32(v[4 * k + 1]);
      q.z = to_tf32(v[4 * k + 2]);
      q.w = to_tf32(v[4 * k + 3]);
      st_smem16(dst_row + (uint32_t)(c0 / 4 + k) * lbo, q);
      if (BF16 == 3) {
        lo[4 * k + 0] = v[4 * k + 0] - __uint_as_float(q.x); lo[4 * k + 1] = v[4 * k + 1] - __uint_as_float(q.y);
        lo[4 * k + 2] = v[4 * k + 2] - __uint_as_float(q.z); lo[4 * k + 3] = v[4 * k + 3] - __uint_as_float(q.w);
      }
    }
    if (BF16 == 3) {
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        uint4 ql, qh;
        ql.x = pack16<1>(lo[8 * k + 0], lo[8 * k + 1]); ql.y = pack16<1>(lo[8 * k + 2], lo[8 * k + 3]);
        ql.z = pack16<1>(lo[8 * k + 4], lo[8 * k + 5]); ql.w = pack16<1>(lo[8 * k + 6], lo[8 * k + 7]);
        qh.x = pack16<1>(v[8 * k + 0], v[8 * k + 1]); qh.y = pack16<1>(v[8 * k + 2], v[8 * k + 3]);
        qh.z = pack16<1>(v[8 * k + 4], v[8 * k + 5]); qh.w = pack16<1>(v[8 * k + 6], v[8 * k + 7]);
        st_smem16(dst_row + (uint32_t)(NCHM + c0 / 8 + k) * lbo, ql);
        st_smem16(dst_row + (uint32_t)(NCHM + NCHM / 2 + c0 / 8 + k) * lbo, qh);
      }
    }
  }
}

// Pooled row (identical in both lanes of a pair): the even lane stores the first half of the 16 channels,
// the odd lane the second half, so every lane of the store instruction is active.
template <int BF16, int NCHM>
__device__ __forceinline__ void store_pooled16(uint32_t dst_row, uint32_t lbo, int c0, const float (&v)[16], int odd) {
  float h[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) h[i] = odd ? v[8 + i] : v[i];
  if (is16(BF16)) {
    uint4 q;
    q.x = pack16<BF16>(h[0], h[1]); q.y = pack16<BF16>(h[2], h[3]);
    q.z = pack16<BF16>(h[4], h[5]); q.w = pack16<BF16>(h[6], h[7]);
    st_smem16(dst_row + (uint32_t)(c0 / 8 + odd) * lbo, q);
  } else {
    float lo[8];
#pragma unroll
    for (int k = 0; k < 2; ++k) {
      uint4 q;
      q.x = to_tf32(h[4 * k + 0]); q.y = to_tf32(h[4 * k + 1]);
      q.z = to_tf32(h[4 * k + 2]); q.w = to_tf32(h[4 * k + 3]);
      st_smem16(dst_row + (uint32_t)(c0 / 4 + 2 * odd + k) * lbo, q);
      if (BF16 == 3) {
        lo[4 * k + 0] = h[4 * k + 0] - __uint_as_float(q.x); lo[4 * k + 1] = h[4 * k + 1] - __uint_as_float(q.y);
        lo[4 * k + 2] = h[4 * k + 2] - __uint_as_float(q.z); lo[4 * k + 3] = h[4 * k + 3] - __uint_as_float(q.w);
      }
    }
    if (BF16 == 3) {
      uint4 ql, qh;
      ql.x = pack16<1>(lo[0], lo[1]); ql.y = pack16<1>(lo[2], lo[3]); ql.z = pack16<1>(lo[4], lo[5]); ql.w = pack16<1>(lo[6], lo[7]);
      qh.x = pack16<1>(h[0], h[1]); qh.y = pack16<1>(h[2], h[3]); qh.z = pack16<1>(h[4], h[5]); qh.w = pack16<1>(h[6], h[7]);
      st_smem16(dst_row + (uint32_t)(NCHM + c0 / 8 + odd) * lbo, ql);
      st_smem16(dst_row + (uint32_t)(NCHM + NCHM / 2 + c0 / 8 + odd) * lbo, qh);
    }
  }
}

__device__ __forceinline__ void zero_rows(uint32_t buf, uint32_t lbo, int nch, int row) {
  for (int c = 0; c < nch; ++c) st_smem16(buf + (uint32_t)c * lbo + (uint32_t)row * 16u, make_uint4(0, 0, 0, 0));
}

enum { kE1 = 0, kE2 = 1, kB = 2, kD2 = 3, kD1 = 4 };

// Epilogue of channels [cb, ce) of one 128-row accumulator tile, executed by the four warps of one epilogue set
// (thread = row m; named barrier 1 + set among them).  The (tile, channel half) units of a layer go round-robin to
// the sets (whole tiles for d1, whose head sums over all channels).
template <int C, int BF16, int MODE, int TT>
__device__ __forceinline__ void epilogue_tile(uint32_t smem_base, uint32_t tmem_base, int tile, int q, int lane,
                                              const float* __restrict__ par, int n_valid_int,
                                              float* __restrict__ probs_group, float* __restrict__ scr,
                                              const int* __restrict__ list_g, int cb, int ce, int set) {
  using G = Geo<C, BF16, 1, TT>;
  const int m = 32 * q + lane;
  const float* bias = par + MODE * C;
  // accumulator tile: columns [0, C) = E0 (even taps), [C, 2C) = E1 (odd taps); output row m = E0[m] + E1[m+1]
  const uint32_t taddr = tmem_base + ((uint32_t)(32 * q) << 16) +
                         (uint32_t)((MODE == kD1 ? G::COL_A : G::COL_B) + tile * G::NOUT);
  if (MODE == kD1 && G::PP) {
    // polyphase d1: row m = low-resolution position l of interval 2 tile + (m >> 6); columns [0, C) = output 2l,
    // [C, 2C) = output 2l + 1.  No row shift: bias, LeakyReLU, the 1x1 head and the sigmoid per phase.
    const int interval = 2 * tile + (m >> 6), l = m & 63;
    const float* hw = par + 5 * C;
    float logit0 = 0.0f, logit1 = 0.0f;
#pragma unroll 1
    for (int c0 = cb; c0 < ce; c0 += 16) {
      uint32_t r[16], r1[16];
      tmem_ld_x16(taddr + (uint32_t)c0, r);
      tmem_ld_x16(taddr + (uint32_t)(C + c0), r1);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        logit0 = fmaf(hw[c0 + i], lrelu(__uint_as_float(r[i]) + bias[c0 + i]), logit0);
        logit1 = fmaf(hw[c0 + i], lrelu(__uint_as_float(r1[i]) + bias[c0 + i]), logit1);
      }
    }
    if (l < 50 && interval < n_valid_int) {
      const float a0 = logit0 + par[6 * C], a1 = logit1 + par[6 * C];
      // list_g != nullptr: the group's intervals are rows list_g[0..T) of the full output (empty-interval elision)
      const size_t row = list_g ? (size_t)list_g[interval] : (size_t)interval;
      *reinterpret_cast<float2*>(probs_group + row * kBins + 2 * l) =
          make_float2(1.0f / (1.0f + expf(-a0)), 1.0f / (1.0f + expf(-a1)));
    }
    return;
  }
  // Row m + 1 of lane 31 lives in the next warp's TMEM quadrant: lane 0 of every warp publishes its E1 row
  // in shared memory (scr: [4 warps][C], double buffered by the caller), one named barrier per tile.
#pragma unroll 1
  for (int c0 = cb; c0 < ce; c0 += 16) {
    uint32_t r[16];
    tmem_ld_x16(taddr + (uint32_t)(C + c0), r);
    tmem_ld_wait();
    if (MODE == kD1 && G::FX) {
      uint32_t s1[16];
      tmem_ld_x16(taddr + (uint32_t)(G::COL_A2 - G::COL_A + C + c0), s1);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) r[i] = __float_as_uint(__uint_as_float(r[i]) + __uint_as_float(s1[i]));
    }
    if (lane == 0) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        *reinterpret_cast<uint4*>(scr + q * C + c0 + 4 * k) = make_uint4(r[4 * k], r[4 * k + 1], r[4 * k + 2], r[4 * k + 3]);
    }
  }
  asm volatile("bar.sync %0, 128;" ::"r"(1 + set) : "memory");
  const float* nxt = scr + (q < 3 ? q + 1 : 3) * C;   // E1 row of the next quadrant's first lane (q = 3: unused)
  // which interval of the group this row belongs to, its position, and whether it is a real output
  int interval, l;
  bool valid;
  if (MODE == kE1 || MODE == kD1) { interval = tile; l = m; valid = l < 100; }
  else if (MODE == kE2 || MODE == kD2) { interval = 2 * tile + (m >> 6); l = m & 63; valid = l < 50; }
  else { interval = 4 * tile + (m >> 5); l = m & 31; valid = l < 25; }
  const bool exists = interval < G::T;          // level-3 tiles may be wider than the group
  uint32_t dst_full = 0, dst_aux = 0, lbo_full = 0, lbo_aux = 0;
  if (MODE == kE1) {
    if (G::PP) {   // de-interleaved skip: row = low-resolution position, positions 2i / 2i + 1 as channels [0, C) / [C, 2C)
      dst_full = smem_base + G::OFF_E1 + (uint32_t)(G::LEAD2 + 64 * tile + (m >> 1)) * 16u; lbo_full = G::LBO2;
    } else {
      dst_full = smem_base + G::OFF_E1 + (uint32_t)(G::LEAD1 + 128 * tile + m) * 16u; lbo_full = G::LBO1;
    }
    dst_aux = smem_base + G::OFF_P1 + (uint32_t)(G::LEAD2 + 64 * tile + (m >> 1)) * 16u; lbo_aux = G::LBO2;     // P1
    if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_P1, G::LBO2, G::NCHB, m);
  } else if (MODE == kE2) {
    dst_full = smem_base + G::OFF_R + (uint32_t)(G::LEAD2 + 128 * tile + m) * 16u; lbo_full = G::LBO2;          // E2
    dst_aux = smem_base + G::OFF_R + G::SZ_L2 + (uint32_t)(G::LEAD3 + 64 * tile + (m >> 1)) * 16u; lbo_aux = G::LBO3;  // P2
    if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_R, G::LBO2, G::NCHB, m);
    if (tile == 0 && m >= 32 && m < 32 + G::LEAD3) zero_rows(smem_base + G::OFF_R + G::SZ_L2, G::LBO3, G::NCHB, m - 32);
  } else if (MODE == kB) {
    dst_full = smem_base + G::OFF_R + G::SZ_L2 + (uint32_t)(G::LEAD2 + 256 * tile + 2 * m) * 16u; lbo_full = G::LBO2;  // U2
    if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_R + G::SZ_L2, G::LBO2, G::NCHB, m);
  } else if (MODE == kD2) {
    if (G::PP) {   // polyphase d1 reads d2 itself (no upsampled copy): rows as E2's, in E2's place
      dst_full = smem_base + G::OFF_R + (uint32_t)(G::LEAD2 + 128 * tile + m) * 16u; lbo_full = G::LBO2;
      if (tile == 0 && m < G::LEAD2) zero_rows(smem_base + G::OFF_R, G::LBO2, G::NCHB, m);
    } else {
      dst_full = smem_base + G::OFF_R + (uint32_t)(G::LEAD1 + 256 * tile + 2 * m) * 16u; lbo_full = G::LBO1;      // U1
      if (tile == 0 && m < G::LEAD1) zero_rows(smem_base + G::OFF_R, G::LBO1, G::NCHB, m);
    }
  }
  float logit = 0.0f;
#pragma unroll 1
  for (int c0 = cb; c0 < ce; c0 += 16) {
    uint32_t r[16], r1[16];
    tmem_ld_x16(taddr + (uint32_t)c0, r);
    tmem_ld_x16(taddr + (uint32_t)(C + c0), r1);
    tmem_ld_wait();
    if (MODE == kD1 && G::FX) {               // the upsampled half of d1 sits in its own accumulator tile (region A2)
      uint32_t s0[16], s1[16];
      tmem_ld_x16(taddr + (uint32_t)(G::COL_A2 - G::COL_A + c0), s0);
      tmem_ld_x16(taddr + (uint32_t)(G::COL_A2 - G::COL_A + C + c0), s1);
      tmem_ld_wait();
#pragma unroll
      for (int i = 0; i < 16; ++i) {
        r[i] = __float_as_uint(__uint_as_float(r[i]) + __uint_as_float(s0[i]));
        r1[i] = __float_as_uint(__uint_as_float(r1[i]) + __uint_as_float(s1[i]));
      }
    }
    float v[16], nx[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {             // whole-warp broadcast loads (cheaper than 16 predicated scalar loads)
      const float4 n4 = *reinterpret_cast<const float4*>(nxt + c0 + 4 * k);
      nx[4 * k] = n4.x; nx[4 * k + 1] = n4.y; nx[4 * k + 2] = n4.z; nx[4 * k + 3] = n4.w;
    }
#pragma unroll
    for (int i = 0; i < 16; ++i) {
      float up = __shfl_down_sync(0xffffffffu, __uint_as_float(r1[i]), 1);
      if (lane == 31) up = (q < 3) ? nx[i] : 0.0f;
      v[i] = lrelu(__uint_as_float(r[i]) + up + bias[c0 + i]);
    }
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
      float pv[16];
#pragma unroll
      for (int i = 0; i < 16; ++i) pv[i] = fmaxf(v[i], __shfl_xor_sync(0xffffffffu, v[i], 1));
      if (exists) {               // (a level-2 tile is wider than a one-interval group: its upper half has no buffer rows)
        if (MODE == kE1 && G::PP) store_row16<BF16, 2 * G::NCH>(dst_full, lbo_full, c0 + (m & 1) * C, v);
        else store_row16<BF16, G::NCH>(dst_full, lbo_full, c0, v);
        store_pooled16<BF16, G::NCH>(dst_aux, lbo_aux, c0, pv, lane & 1);   // both lanes of a pair hold the same maxima
      }
    } else if (MODE == kD2 && G::PP) {
      if (exists) store_row16<BF16, G::NCH>(dst_full, lbo_full, c0, v);
    } else if (exists) {          // kB, kD2: nearest upsample = the same chunk into rows 2m and 2m + 1;
      // groups of four lanes alternate which of the two rows goes first, so that one store instruction
      // covers all eight 16-byte slots of every 128-byte line evenly (no bank conflicts)
      const uint32_t swz = (uint32_t)((m >> 2) & 1) * 16u;
      store_row16<BF16, G::NCH>(dst_full + swz, lbo_full, c0, v);
      store_row16<BF16, G::NCH>(dst_full + (16u - swz), lbo_full, c0, v);
    }
  }
  if (MODE == kD1) {
    if (valid && interval < n_valid_int) {
      const float a = logit + par[6 * C];
      // list_g != nullptr: the group's intervals are rows list_g[0..T) of the full output (empty-interval elision)
      const size_t row = list_g ? (size_t)list_g[interval] : (size_t)interval;
      probs_group[row * kBins + l] = 1.0f / (1.0f + expf(-a));
    }
  }
}

// Interval histograms of one group -> X0 (operand-rounded, chunked layout).  All epilogue threads.  X0 shares
// its memory with P1, so every row the e1 MMAs can read for a valid output is (re)written: the lead
// rows and the gap rows l >= 100 of every interval as zeros.
// seg_cnt (optional): tracks per interval; an interval without tracks is taken as zeros WITHOUT reading hist
// (the tensor-core FC kernel does not write the histograms of empty intervals).
template <int C, int BF16, int TT>
__device__ __forceinline__ void load_x0(uint32_t smem_base, const float* __restrict__ hist, long long g0,
                                        int n_valid_int, int split, int tid, const int* __restrict__ list,
                                        const int* __restrict__ seg_cnt) {
  using G = Geo<C, BF16, 1, TT>;
  const uint32_t x0 = smem_base + G::OFF_XP;
  const uint4 zero4 = make_uint4(0, 0, 0, 0);
  if (tid < G::LEAD1)
    for (int c = 0; c < G::XCH; ++c) st_smem16(x0 + (uint32_t)c * G::LBO1 + (uint32_t)tid * 16u, zero4);
  if (G::FX) {
    // FP32-accurate format: chunks 0, 1 = TF32 of channels 0-3 / 4-7 (HI), chunk 2 = bf16(x - tf32(x)) (LO), chunk 3 = bf16(x) (HB)
    for (int it = tid; it < G::T * 128; it += G::EPI_THREADS) {
      const int t = it >> 7, l = it & 127;
      bool live = l < 100 && t < n_valid_int;
      const long long src = !live ? 0 : (list ? (long long)list[g0 + t] : g0 + t);
      if (live && seg_cnt != nullptr) live = __ldg(seg_cnt + src) > 0;
      float x[8], r[8];
      uint32_t hi[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        x[c] = live ? __ldg(hist + src * kFcOut + c * kBins + l) : 0.0f;
        hi[c] = to_tf32(x[c]);
        r[c] = x[c] - __uint_as_float(hi[c]);
      }
      uint4 ql, qh;
      ql.x = pack16<1>(r[0], r[1]); ql.y = pack16<1>(r[2], r[3]); ql.z = pack16<1>(r[4], r[5]); ql.w = pack16<1>(r[6], r[7]);
      qh.x = pack16<1>(x[0], x[1]); qh.y = pack16<1>(x[2], x[3]); qh.z = pack16<1>(x[4], x[5]); qh.w = pack16<1>(x[6], x[7]);
      const uint32_t row = (uint32_t)(G::LEAD1 + it) * 16u;
      st_smem16(x0 + row, make_uint4(hi[0], hi[1], hi[2], hi[3]));
      st_smem16(x0 + G::LBO1 + row, make_uint4(hi[4], hi[5], hi[6], hi[7]));
      st_smem16(x0 + 2 * G::LBO1 + row, ql);
      st_smem16(x0 + 3 * G::LBO1 + row, qh);
    }
  } else if (G::B16 && !(split && BF16 == 2)) {
    for (int it = tid; it < G::T * 128; it += G::EPI_THREADS) {
      const int t = it >> 7, l = it & 127;
      bool live = l < 100 && t < n_valid_int;
      const long long src = !live ? 0 : (list ? (long long)list[g0 + t] : g0 + t);
      if (live && seg_cnt != nullptr) live = __ldg(seg_cnt + src) > 0;
      float x[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) x[c] = live ? __ldg(hist + src * kFcOut + c * kBins + l) : 0.0f;
      uint4 qv;
      qv.x = pack16<BF16>(x[0], x[1]); qv.y = pack16<BF16>(x[2], x[3]);
      qv.z = pack16<BF16>(x[4], x[5]); qv.w = pack16<BF16>(x[6], x[7]);
      const uint32_t row = (uint32_t)(G::LEAD1 + it) * 16u;
      st_smem16(x0 + row, qv);
      st_smem16(x0 + G::LBO1 + row, zero4);       // channels 8..15 of the K = 16 MMA: zero
    }
  } else if (split) {
    // TF32 (and FP16) mode with the e1 split: the histogram enters as TWO 16-bit pieces per value, x = a1 + a2 (+ 2^-17 |x|; FP16 pieces: 2^-22),
    // side by side in the K = 16 of one kind::f16 MMA: chunk 0 = a1 of the 8 channels, chunk 1 = a2.  With the
    // weights as [w1 | w1] (pass 0) and [w2 | 0] (pass 1) two MMAs per tap pair give a1 w1 + a2 w1 + a1 w2, i.e.
    // ~2^-16 relative per product (plain TF32: 2^-12) for 2/3 of the MMAs a three-pass TF32 split needs.
    for (int it = tid; it < G::T * 128; it += G::EPI_THREADS) {
      const int t = it >> 7, l = it & 127;
      bool live = l < 100 && t < n_valid_int;
      const long long src = !live ? 0 : (list ? (long long)list[g0 + t] : g0 + t);
      if (live && seg_cnt != nullptr) live = __ldg(seg_cnt + src) > 0;
      // pieces in the format of the MMA that reads them: BF16 in the TF32 kernel, FP16 in the FP16 kernel
      constexpr int PF = BF16 == 2 ? 2 : 1;
      float x[8], r[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        x[c] = live ? __ldg(hist + src * kFcOut + c * kBins + l) : 0.0f;
        r[c] = x[c] - (PF == 2 ? __half2float(__float2half_rn(x[c])) : __bfloat162float(__float2bfloat16_rn(x[c])));
      }
      uint4 q1, q2;
      q1.x = pack16<PF>(x[0], x[1]); q1.y = pack16<PF>(x[2], x[3]); q1.z = pack16<PF>(x[4], x[5]); q1.w = pack16<PF>(x[6], x[7]);
      q2.x = pack16<PF>(r[0], r[1]); q2.y = pack16<PF>(r[2], r[3]); q2.z = pack16<PF>(r[4], r[5]); q2.w = pack16<PF>(r[6], r[7]);
      const uint32_t row = (uint32_t)(G::LEAD1 + it) * 16u;
      st_smem16(x0 + row, q1);
      st_smem16(x0 + G::LBO1 + row, q2);
    }
  } else {
    for (int it = tid; it < G::T * 256; it += G::EPI_THREADS) {
      const int t = it >> 8, qc = (it >> 7) & 1, l = it & 127;
      bool live = l < 100 && t < n_valid_int;
      const long long src = !live ? 0 : (list ? (long long)list[g0 + t] : g0 + t);
      if (live && seg_cnt != nullptr) live = __ldg(seg_cnt + src) > 0;
      float x[4];
#pragma unroll
      for (int c = 0; c < 4; ++c) x[c] = live ? __ldg(hist + src * kFcOut + (4 * qc + c) * kBins + l) : 0.0f;
      uint4 hi;
      hi.x = to_tf32(x[0]); hi.y = to_tf32(x[1]); hi.z = to_tf32(x[2]); hi.w = to_tf32(x[3]);
      const uint32_t row = (uint32_t)(G::LEAD1 + 128 * t + l) * 16u;
      st_smem16(x0 + (uint32_t)qc * G::LBO1 + row, hi);
    }
  }
}

// Compile-time description of sub-layer S as the MMA issuer sees it.
template <int C, int BF16, int S, int TT>
struct Lay {
  using G = Geo<C, BF16, 1, TT>;
  static constexpr bool D1 = (S == sD1U || S == sD1E);
  static constexpr bool POLY = D1 && G::PP;                    // polyphase d1: low-resolution rows, 13 offsets, row step 1
  static constexpr int TAPS = (S == sE1 || D1) ? 25 : (S == sB ? 5 : 15);
  static constexpr int PAD = POLY ? 6 : (TAPS - 1) / 2;        // rows before the output row that the first step reads
  static constexpr int RS = POLY ? 1 : 2;                      // rows per step: a tap pair moves two rows, an offset one
  static constexpr int PAIRS = (TAPS + 1) / 2;                 // (even, odd) tap pairs (the last odd tap is zero) | offsets -6 .. 6
  static constexpr bool HALF_LAST = !POLY;                     // the last tap pair holds one tap only: an N = C step
  static constexpr int NKB = (S == sE1) ? 1 : ((S == sD2 || (S == sD1E && POLY)) ? 2 * G::NKB1 : G::NKB1);     // K blocks per step group
  static constexpr int LEVEL = POLY ? 2 : ((S == sE1 || D1) ? 1 : (S == sB ? 3 : 2));
  static constexpr int LEAD = LEVEL == 1 ? G::LEAD1 : (LEVEL == 2 ? G::LEAD2 : G::LEAD3);
  static constexpr int LBO = LEVEL == 1 ? G::LBO1 : (LEVEL == 2 ? G::LBO2 : G::LBO3);
  static constexpr int NT = LEVEL == 1 ? G::T : (LEVEL == 2 ? (G::T + 1) / 2 : (G::T + 3) / 4);
  static constexpr int HALF = (S == sD2) ? NKB / 2 : NKB;      // K blocks served by the first source buffer
  static constexpr int SRC0 = (S == sE1) ? G::OFF_XP /* X0 */ : (S == sE2) ? G::OFF_P1 /* P1 */
                              : (S == sB) ? G::OFF_R + G::SZ_L2 /* P2 */ : (S == sD2) ? G::OFF_R + G::SZ_L2 /* U2 */
                              : (S == sD1U) ? G::OFF_R /* U1 | polyphase: d2 itself */ : G::OFF_E1 /* E1 */;
  static constexpr int SRC1 = (S == sD2) ? G::OFF_R /* E2 */ : SRC0;
  static constexpr int DCOL = (S == sD1U && G::FX) ? G::COL_A2 : (D1 ? G::COL_A : G::COL_B);
  // byte offset (from the CTA's shared-memory base) of the first chunk of K block kk
  __host__ __device__ static constexpr int a_off(int kk) {
    return kk < HALF ? SRC0 + 2 * kk * LBO : SRC1 + 2 * (kk - HALF) * LBO;
  }
  // FX: the source buffers hold SRC_NCH main chunks, then SRC_NCH / 2 LO chunks, then SRC_NCH / 2 HB chunks; the
  // correction MMA of K block kk reads LO chunk kk and HB chunk kk as the two 16-byte K chunks of its A operand
  static constexpr int SRC_NCH = (S == sE1) ? 2 : G::NCH;
  static constexpr int C_LBO = SRC_NCH / 2 * LBO;              // descriptor LBO of the correction operand (LO -> HB)
  __host__ __device__ static constexpr int c_off(int kk) {
    return (kk < HALF ? SRC0 + kk * LBO : SRC1 + (kk - HALF) * LBO) + SRC_NCH * LBO;
  }
};

template <int BF16, int CG>
__device__ __forceinline__ void mma_lh(uint32_t d, uint32_t a_lo, uint32_t a_hi, uint32_t b_lo, uint32_t b_hi,
                                       uint32_t idesc, uint32_t acc) {
  if (CG == 2) {
    if (is16(BF16)) mma2_f16_lh(d, a_lo, a_hi, b_lo, b_hi, idesc, acc);
    else mma2_tf32_lh(d, a_lo, a_hi, b_lo, b_hi, idesc, acc);
  } else {
    if (is16(BF16)) mma_f16_lh(d, a_lo, a_hi, b_lo, b_hi, idesc, acc);
    else mma_tf32_lh(d, a_lo, a_hi, b_lo, b_hi, idesc, acc);
  }
}

struct RingState { int ring; uint32_t phase; };

#ifdef PVF_UNET_PROF
// Diagnostic build only (-DPVF_UNET_PROF): cycles the MMA issuer spent waiting, per CTA:
// [0..5] wait_epi(k), [6] ring stage full (own half), [7] ring stage full (peer's half), [8] whole role loop
__device__ unsigned long long g_unet_prof[160][16];
#define PVF_PROF_T0() const long long prof_t0 = clock64()
#define PVF_PROF_ADD(slot) do { if ((threadIdx.x & 31) == 0) g_unet_prof[blockIdx.x][slot] += (unsigned long long)(clock64() - prof_t0); } while (0)
#else
#define PVF_PROF_T0() do {} while (0)
#define PVF_PROF_ADD(slot) do {} while (0)
#endif

// MMA steps [f_begin, f_end) of sub-layer S for the group: tap-major over ring stages, every stage
// used by all NT tiles.  The warp walks the (uniform) schedule; one elected lane issues a whole
// stage worth of MMAs whose descriptors differ from the stage origin by compile-time constants.
// f_begin must be a multiple of SPS.  acc0 = 0 starts fresh accumulators at step f_begin.
template <int C, int BF16, int CG, int TT, int S>
__device__ __forceinline__ void mma_seg(uint32_t sb, uint32_t tmem_base, uint32_t bar0, RingState& rs,
                                        int f_begin, int f_end, uint32_t acc0, bool e1x = false) {
  // e1x (sub-layer e1 of the TF32 kernel only): the split e1 runs as kind::f16 MMAs on BF16 pieces (see load_x0)
  // Steps are MMA steps as they sit in the weight image ("physical"); FX has PH = 2 of them -- main (kind::tf32 on the HI
  // array) and correction (kind::f16 on [LO | HB]) -- per (tap pair, K block) ("logical" step).
  using G = Geo<C, BF16, CG, TT>;
  using Y = Lay<C, BF16, S, TT>;
  constexpr int SPS = G::SPS, PH = G::PH, SPL = SPS / PH;
  constexpr bool B16 = G::B16, FX = G::FX;
  static_assert(Y::HALF % SPL == 0 || SPL % Y::NKB == 0,
                "a ring stage is either part of one source's K blocks or whole taps");
  constexpr uint32_t fmt_main = BF16 == 2 ? kFmtF16 : (BF16 == 1 ? kFmtBF16 : kFmtTF32);
  constexpr uint32_t idesc = instr_desc(fmt_main, 128 * CG, G::NOUT);
  constexpr uint32_t idesc_x = instr_desc(kFmtBF16, 128 * CG, G::NOUT);
  // The kernels have an odd number of taps: the last "pair" holds an even tap only, so its steps are MMAs of
  // N = C (half the tensor time, half the B rows; the E1 columns of the accumulator are left alone).
  constexpr uint32_t idesc_h = instr_desc(fmt_main, 128 * CG, G::NOUT / 2);
  constexpr uint32_t idesc_xh = instr_desc(kFmtBF16, 128 * CG, G::NOUT / 2);
  constexpr uint32_t b_lbo_h = (uint32_t)((G::NB / 2 * 16) >> 4) << 16;
  constexpr int LAST0 = Y::HALF_LAST ? (Y::PAIRS - 1) * Y::NKB : (1 << 30);   // first logical step of the last tap pair (not e1)
  constexpr uint32_t hi = (128u >> 4) | (1u << 14);                    // SBO = 128 B, descriptor version 1
  // e1 in the 16-bit modes: the second 16-byte K chunk of A is the SAME 8-channel buffer two rows further down
  // (LBO = 32 bytes), i.e. the input of the next tap pair -- one MMA does tap pairs 2w and 2w + 1
  constexpr uint32_t a_lbo = (S == sE1 && B16) ? (2u << 16) : ((uint32_t)(Y::LBO >> 4) << 16);
  constexpr uint32_t a_lbo_x2 = (2u << 16) - a_lbo;     // added for the second pass of the split e1 (TF32 kernel)
  constexpr uint32_t a_lbo_x2_16 = (2u << 16) - ((uint32_t)(Y::LBO >> 4) << 16);   // subtracted for the FIRST pass in a 16-bit kernel
  constexpr uint32_t c_lbo = (uint32_t)(Y::C_LBO >> 4) << 16;          // FX correction operand: LO chunk -> HB chunk
  constexpr uint32_t b_lbo = (uint32_t)((G::NB * 16) >> 4) << 16;
  const uint32_t dcol = tmem_base + (uint32_t)Y::DCOL;
  for (int f = f_begin; f < f_end; f += SPS) {
    const int n = min(SPS, f_end - f);
    const int lf = f / PH;                      // logical step of the stage's first MMA
    {
      PVF_PROF_T0();
      mbar_wait(bar0 + 8u * rs.ring, rs.phase);
      PVF_PROF_ADD(6);
    }
    if (CG == 2) {
      PVF_PROF_T0();
      mbar_wait_cluster(bar0 + 8u * (2 * G::STAGES + rs.ring), rs.phase);   // the peer's half has landed
      PVF_PROF_ADD(7);
    }
    tc_fence_after_sync();
    const uint32_t b0 = (sb + G::OFF_RING + rs.ring * G::STAGE_BYTES) >> 4;
    uint32_t a0 = a_lbo + (sb >> 4);          // stage origin: descriptor low word of tile 0, logical step lf
    uint32_t c0 = c_lbo + (sb >> 4);          // same for the FX correction operand
    if (S == sE1) {
      // e1: one K block per step; steps run [pass][tap pair]; both passes of the split read the same operand
    } else if (Y::HALF >= SPL) {
      const int j0 = lf / Y::NKB, kk0 = lf % Y::NKB;
      const int off = kk0 < Y::HALF ? Y::SRC0 + 2 * kk0 * Y::LBO : Y::SRC1 + 2 * (kk0 - Y::HALF) * Y::LBO;
      a0 += (uint32_t)(off >> 4) + (uint32_t)(Y::LEAD + Y::RS * j0 - Y::PAD);
      if (FX) {
        const int offc = (kk0 < Y::HALF ? Y::SRC0 + kk0 * Y::LBO : Y::SRC1 + (kk0 - Y::HALF) * Y::LBO) + Y::SRC_NCH * Y::LBO;
        c0 += (uint32_t)(offc >> 4) + (uint32_t)(Y::LEAD + Y::RS * j0 - Y::PAD);
      }
    } else {
      a0 += (uint32_t)(Y::SRC0 >> 4) + (uint32_t)(Y::LEAD + Y::RS * (lf / Y::NKB) - Y::PAD);
      c0 += (uint32_t)(Y::SRC0 >> 4) + (uint32_t)(Y::LEAD + Y::RS * (lf / Y::NKB) - Y::PAD);
    }
    if (elect_one()) {
#pragma unroll
      for (int i = 0; i < SPS; ++i) {
        if (i < n) {
          constexpr int dummy = 0; (void)dummy;
          const int li = i / PH;                 // logical step inside the stage (compile time)
          const bool corr = FX && (i % PH) == 1; // FX: the correction MMA of the logical step
          uint32_t a;
          bool half_n;
          if (S == sE1) {
            // three shapes of e1: 16-bit unsplit (7 steps, K chunks = tap pairs 2 step, 2 step + 1 of the same array: LBO = 2
            // rows), TF32 / FX (13 steps per pass), split (TF32 or FP16 kernel: 13 steps [a1 | a2] with the level-1 LBO, then
            // 7 steps [a1 of pair u | a1 of pair u + 1] with LBO = 2 rows)
            const bool split16 = B16 && e1x;
            const int step = lf + li, pass = step / 13, u = (B16 && !e1x) ? 2 * step : (pass ? 2 * (step - 13) : step);
            a = a0 + (uint32_t)(Y::SRC0 >> 4) + (uint32_t)(Y::LEAD + 2 * u - Y::PAD);
            if (BF16 == 0 && pass) a += a_lbo_x2;              // [a1 of pair u | a1 of pair u + 1]
            if (split16 && !pass) a -= a_lbo_x2_16;            // 16-bit kernel: a_lbo is the 2-row one; pass 0 wants [a1 | a2]
            if (corr) a = c0 + (uint32_t)((Y::SRC0 + Y::SRC_NCH * Y::LBO) >> 4) + (uint32_t)(Y::LEAD + 2 * u - Y::PAD);
            half_n = (B16 && !e1x) ? step == 6 : (step == 12 || step == 19);
          } else if (Y::HALF >= SPL) {
            a = corr ? c0 + (uint32_t)(li * (Y::LBO >> 4)) : a0 + (uint32_t)(li * ((2 * Y::LBO) >> 4));
            half_n = lf + li >= LAST0;
          } else {
            a = corr ? c0 + (uint32_t)((Y::c_off(li % Y::NKB) - Y::SRC0) >> 4) + (uint32_t)(Y::RS * (li / Y::NKB))
                     : a0 + (uint32_t)((Y::a_off(li % Y::NKB) - Y::SRC0) >> 4) + (uint32_t)(Y::RS * (li / Y::NKB));
            half_n = lf + li >= LAST0;
          }
          const uint32_t b = (half_n ? b_lbo_h : b_lbo) + b0 + (uint32_t)(i * (G::STEP_BYTES >> 4));
          const uint32_t acc = (i > 0) ? 1u : (f > f_begin ? 1u : acc0);
#pragma unroll
          for (int t = 0; t < Y::NT; ++t) {
            if ((S == sE1 && BF16 == 0 && e1x) || corr)
              mma_lh<1, CG>(dcol + (uint32_t)(t * G::NOUT), a + 128u * t, hi, b, hi, half_n ? idesc_xh : idesc_x, acc);
            else
              mma_lh<BF16, CG>(dcol + (uint32_t)(t * G::NOUT), a + 128u * t, hi, b, hi, half_n ? idesc_h : idesc, acc);
          }
        }
      }
      // frees the ring slot (in both CTAs of a pair) when these MMAs retire
      if (CG == 2) mma_commit2(bar0 + 8u * (G::STAGES + rs.ring), 3);
      else mma_commit(bar0 + 8u * (G::STAGES + rs.ring));
    }
    __syncwarp();
    if (++rs.ring == G::STAGES) { rs.ring = 0; rs.phase ^= 1u; }
  }
}

template <int C, int BF16, int CG, int TT>
__global__ void __launch_bounds__((Geo<C, BF16, CG, TT>::THREADS), 1)
k_unet_tc(const float* __restrict__ hist, int n_int, const unsigned char* __restrict__ wpack, int split_e1,
          float* __restrict__ probs, const int* __restrict__ list, const int* __restrict__ n_list,
          const int* __restrict__ seg_cnt) {
  // list / n_list (device, optional): process only intervals list[0 .. *n_list) of hist / probs (elision of
  // empty intervals); n_int is then only the capacity the grid was sized for
  pdl_launch_dependents();
  if (n_list != nullptr) { pdl_wait(); n_int = *n_list; }
  using G = Geo<C, BF16, CG, TT>;
  static_assert(G::kFits, "shared memory budget");
  static_assert(!G::FX || CG == 2, "the FP32-accurate format runs as CTA pairs");
  extern __shared__ __align__(1024) unsigned char smem[];
  const uint32_t sb = smem_u32(smem);
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // provably warp-uniform role index
  // CG = 2: the two CTAs of a cluster walk the same schedule in lockstep, each on its own group of intervals;
  // rank 0 (the leader) issues every MMA for both
  const int rank = CG == 2 ? (int)cluster_ctarank() : 0;
  float* par = reinterpret_cast<float*>(smem + G::OFF_PAR);
  // mbarriers: full[s], empty[s] per ring stage (this CTA's half of the weights); peer_full[s] (leader only: the
  // peer's half has landed); accum[k] = "MMAs of layer k retired" (k: e1 e2 b d2 d1; multicast to both CTAs);
  // epi[k] = "this CTA's epilogue k done" (k: x0-staged e1 e2 b d2 d1); peer_epi[k] (leader only: the peer's)
  const uint32_t bar0 = sb + G::OFF_BAR;
  auto accum_bar = [&](int k) { return bar0 + 8u * (G::BAR_ACCUM + k); };
  auto epi_bar = [&](int k) { return bar0 + 8u * (G::BAR_EPI + k); };
  auto pepi_bar = [&](int k) { return bar0 + 8u * (G::BAR_PEPI + k); };
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + G::OFF_BAR + 8 * G::BAR_SLOT);
  const Plan P = make_plan<C, BF16, CG>(split_e1);
  const unsigned char* wimg = wpack + (size_t)rank * P.total;       // this CTA's weight image

  // ---- one-time setup: zero the activation buffers (gap / halo rows must be zero), parameters, barriers
  for (int i = tid; i < G::OFF_RING / 16; i += G::THREADS) reinterpret_cast<uint4*>(smem)[i] = make_uint4(0, 0, 0, 0);
  for (int i = tid; i < 6 * C + 1; i += G::THREADS) par[i] = reinterpret_cast<const float*>(wimg)[i];
  if (tid == 0) {
    for (int s = 0; s < G::STAGES; ++s) {
      mbar_init(bar0 + 8u * s, 1);
      mbar_init(bar0 + 8u * (G::STAGES + s), 1);
      mbar_init(bar0 + 8u * (2 * G::STAGES + s), 1);
    }
    for (int k = 0; k < 5; ++k) mbar_init(accum_bar(k), 1);
    for (int k = 0; k < 6; ++k) { mbar_init(epi_bar(k), G::EPI_THREADS); mbar_init(pepi_bar(k), G::EPI_THREADS); }
    fence_mbar_init();
  }
  if (warp == 1) {
    if (CG == 2) tmem_alloc2(smem_u32(const_cast<uint32_t*>(tmem_slot)), G::TMEM_COLS);
    else tmem_alloc(smem_u32(const_cast<uint32_t*>(tmem_slot)), G::TMEM_COLS);
  }
  fence_proxy_async_smem();
  tc_fence_before_sync();
  if (CG == 2) cluster_sync_all(); else __syncthreads();
  tc_fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  pdl_wait();      // everything above touched weights only; the histograms / seg_cnt come from the kernel before (pdl.cuh)

  // pair-groups: pair p of the grid takes groups CG*pg + rank for pg = p, p + pairs, ...; a CTA whose group lies
  // past the end (odd group count) runs the schedule on zeros and stores nothing
  const int n_groups = (n_int + G::T - 1) / G::T;
  const int n_pg = (n_groups + CG - 1) / CG;
  const int pg0 = (int)blockIdx.x / CG, stride = (int)gridDim.x / CG;

  if (warp == 0) {
    // ===================== weight producer: streams this CTA's image through the ring
    if (lane == 0) {
      RingState rs{0, 0u};
      auto stream = [&](int seg) {
        const unsigned char* src = wimg + P.seg_off[seg];
        const int steps = P.seg_steps[seg];
        for (int f = 0; f < steps; f += G::SPS) {
          const int n = min(G::SPS, steps - f);
          mbar_wait(bar0 + 8u * (G::STAGES + rs.ring), rs.phase ^ 1u);
          mbar_arrive_expect_tx(bar0 + 8u * rs.ring, (uint32_t)(n * G::STEP_BYTES));
          bulk_g2s(sb + G::OFF_RING + rs.ring * G::STAGE_BYTES, src + (size_t)f * G::STEP_BYTES,
                   (uint32_t)(n * G::STEP_BYTES), bar0 + 8u * rs.ring);
          if (++rs.ring == G::STAGES) { rs.ring = 0; rs.phase ^= 1u; }
        }
      };
      bool first = true;
      for (int pg = pg0; pg < n_pg; pg += stride) {
        if (first) { stream(gE1); first = false; }
        const bool has_next = pg + stride < n_pg;
        for (int s = 0; s < kSegs; ++s) {
          if (s == gE1 && !has_next) continue;
          stream(s);
        }
      }
    }
  } else if (warp == 1 && rank == 0) {
    // ===================== MMA issuer (whole warp walks the schedule, one elected lane issues)
    RingState rs{0, 0u};
    uint32_t ph[6] = {0, 0, 0, 0, 0, 0};
    auto wait_epi = [&](int k) {
      PVF_PROF_T0();
      mbar_wait(epi_bar(k), ph[k]);
      if (CG == 2) mbar_wait_cluster(pepi_bar(k), ph[k]);
      PVF_PROF_ADD(k);
      ph[k] ^= 1u;
      tc_fence_after_sync();
    };
    auto commit = [&](int k) {
      if (elect_one()) {
        if (CG == 2) mma_commit2(accum_bar(k), 3); else mma_commit(accum_bar(k));
      }
      __syncwarp();
    };
    bool first = true;
    PVF_PROF_T0();
    for (int pg = pg0; pg < n_pg; pg += stride) {
      const bool has_next = pg + stride < n_pg;
      if (first) {
        wait_epi(0);
        mma_seg<C, BF16, CG, TT, sE1>(sb, tmem_base, bar0, rs, 0, P.e1_steps, 0u, split_e1 != 0);
        commit(0);
      }
      wait_epi(1);                                   // P1 staged, region B drained
      mma_seg<C, BF16, CG, TT, sE2>(sb, tmem_base, bar0, rs, 0, 8 * G::NKB1 * G::PH, 0u);
      commit(1);
      if (!first) wait_epi(5);                       // region A drained by the previous group's d1 epilogue
      mma_seg<C, BF16, CG, TT, sD1E>(sb, tmem_base, bar0, rs, 0, G::D1E_A, 0u);
      wait_epi(2);                                   // E2, P2 staged
      mma_seg<C, BF16, CG, TT, sB>(sb, tmem_base, bar0, rs, 0, 3 * G::NKB1 * G::PH, 0u);
      commit(2);
      mma_seg<C, BF16, CG, TT, sD1E>(sb, tmem_base, bar0, rs, G::D1E_A, G::D1E_A + G::D1E_B, 1u);
      wait_epi(3);                                   // U2 staged
      mma_seg<C, BF16, CG, TT, sD2>(sb, tmem_base, bar0, rs, 0, 8 * 2 * G::NKB1 * G::PH, 0u);
      commit(3);
      mma_seg<C, BF16, CG, TT, sD1E>(sb, tmem_base, bar0, rs, G::D1E_A + G::D1E_B, G::D1E_STEPS, 1u);
      wait_epi(4);                                   // U1 staged, region B drained
      if (has_next) {
        wait_epi(0);                                 // next group's X0 staged
        mma_seg<C, BF16, CG, TT, sE1>(sb, tmem_base, bar0, rs, 0, P.e1_steps, 0u, split_e1 != 0);
        commit(0);
      }
      mma_seg<C, BF16, CG, TT, sD1U>(sb, tmem_base, bar0, rs, 0, 13 * G::NKB1 * G::PH, G::FX ? 0u : 1u);   // FX: its own tile
      commit(4);
      first = false;
    }
    PVF_PROF_ADD(8);
  } else if (warp == 1) {
    // ===================== peer CTA of a pair: relay "my half of ring stage s has landed" to the leader
    if (lane == 0) {
      RingState rs{0, 0u};
      const uint32_t lead_bar0 = mapa_rank(bar0, 0);
      auto relay = [&](int steps) {
        for (int f = 0; f < steps; f += G::SPS) {
          mbar_wait(bar0 + 8u * rs.ring, rs.phase);
          mbar_arrive_cluster(lead_bar0 + 8u * (2 * G::STAGES + rs.ring));
          if (++rs.ring == G::STAGES) { rs.ring = 0; rs.phase ^= 1u; }
        }
      };
      bool first = true;
      for (int pg = pg0; pg < n_pg; pg += stride) {
        if (first) { relay(P.seg_steps[gE1]); first = false; }
        const bool has_next = pg + stride < n_pg;
        for (int s = 0; s < kSegs; ++s) {
          if (s == gE1 && !has_next) continue;
          relay(P.seg_steps[s]);
        }
      }
    }
  } else {
    // ===================== epilogue warps: two sets of 128 threads, thread = accumulator row
    const int q = warp & 3, et = tid - 64, set = (warp - 2) >> 2;
    float* scr0 = reinterpret_cast<float*>(smem + G::OFF_SCR) + set * 2 * 4 * C;
    int ecount = 0;                          // accumulator tiles drained so far (selects the scratch buffer)
    auto scr = [&]() { return scr0 + (ecount++ & 1) * 4 * C; };
    uint32_t pa[5] = {0, 0, 0, 0, 0};
    auto wait_acc = [&](int k) { mbar_wait(accum_bar(k), pa[k]); pa[k] ^= 1u; tc_fence_after_sync(); };
    const uint32_t lead_pepi = CG == 2 ? mapa_rank(pepi_bar(0), 0) : 0u;
    auto done = [&](int k) {
      fence_proxy_async_smem();
      tc_fence_before_sync();
      if (CG == 2 && rank == 1) mbar_arrive_cluster(lead_pepi + 8u * k);
      else mbar_arrive(epi_bar(k));
    };
    bool first = true;
    for (int pg = pg0; pg < n_pg; pg += stride) {
      const long long g0 = ((long long)pg * CG + rank) * G::T;
      const int n_valid = (int)max(0LL, min((long long)G::T, (long long)n_int - g0));
      const bool has_next = pg + stride < n_pg;
      const long long gn0 = ((long long)(pg + stride) * CG + rank) * G::T;
      const int n_valid_next = has_next ? (int)max(0LL, min((long long)G::T, (long long)n_int - gn0)) : 0;
      float* pg_out = list ? probs : probs + g0 * kBins;
      const int* lg = list ? list + g0 : nullptr;
      const int* lgn = list ? list + gn0 : nullptr;
      // The work units of a layer -- (tile, channel half) pairs; whole tiles for d1, whose head sums over all
      // channels, and for C = 16, where a half is less than one 16-channel chunk -- go round-robin to the sets.
      auto layer = [&](auto mode, int nt, int nv, const int* lgx) {
        constexpr int MODE = decltype(mode)::value;
        constexpr int HALVES = (C >= 32 && MODE != kD1) ? 2 : 1;
        for (int u = set; u < nt * HALVES; u += G::SETS) {
          const int t = u / HALVES, cb = (u % HALVES) * (C / HALVES);
          epilogue_tile<C, BF16, MODE, TT>(sb, tmem_base, t, q, lane, par, nv, pg_out, scr(), lgx, cb, cb + C / HALVES, set);
        }
      };
      using std::integral_constant;
      if (first) {
        load_x0<C, BF16, TT>(sb, hist, g0, n_valid, split_e1, et, list, seg_cnt);
        done(0);
        wait_acc(0);
        layer(integral_constant<int, kE1>{}, G::T, n_valid, lg);
        done(1);
        first = false;
      }
      wait_acc(1);
      layer(integral_constant<int, kE2>{}, (G::T + 1) / 2, n_valid, lg);
      done(2);
      if (has_next) {                                // P1 is dead (e2's MMAs retired): stage the next input
        load_x0<C, BF16, TT>(sb, hist, gn0, n_valid_next, split_e1, et, list, seg_cnt);
        done(0);
      }
      wait_acc(2);
      layer(integral_constant<int, kB>{}, (G::T + 3) / 4, n_valid, lg);
      done(3);
      wait_acc(3);
      layer(integral_constant<int, kD2>{}, (G::T + 1) / 2, n_valid, lg);
      done(4);
      if (has_next) {
        wait_acc(0);
        layer(integral_constant<int, kE1>{}, G::T, n_valid_next, lgn);
        done(1);
      }
      wait_acc(4);
      layer(integral_constant<int, kD1>{}, G::PP ? G::T / 2 : G::T, n_valid, lg);
      done(5);
    }
  }
  __syncwarp();
  tc_fence_before_sync();
  if (CG == 2) cluster_sync_all(); else __syncthreads();   // pair: the peer's shared memory and barriers stay alive until both are done
  if (warp == 1) {
    __syncwarp();
    if (CG == 2) tmem_dealloc2(tmem_base, G::TMEM_COLS); else tmem_dealloc(tmem_base, G::TMEM_COLS);
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

uint16_t fp16_rne(float v) {                 // float -> IEEE binary16, round to nearest even, overflow -> inf
  uint32_t u;
  memcpy(&u, &v, 4);
  const uint32_t sign = (u >> 16) & 0x8000u;
  u &= 0x7fffffffu;
  if (u >= 0x7f800000u) return (uint16_t)(sign | (u > 0x7f800000u ? 0x7e00u : 0x7c00u));
  if (u >= 0x477ff000u) return (uint16_t)(sign | 0x7c00u);                 // >= 65520 rounds to inf
  if (u < 0x38800000u) {                                                   // subnormal half (or zero)
    if (u < 0x33000000u) return (uint16_t)sign;
    const int shift = 126 - (int)(u >> 23);                                // 14 .. 24
    const uint32_t mant = (u & 0x7fffffu) | 0x800000u;
    const uint32_t q = mant >> shift, rem = mant & ((1u << shift) - 1u), halfway = 1u << (shift - 1);
    return (uint16_t)(sign | (q + ((rem > halfway || (rem == halfway && (q & 1u))) ? 1u : 0u)));
  }
  const uint32_t r = u + 0xfffu + ((u >> 13) & 1u);                        // round the 13 dropped bits
  return (uint16_t)(sign | ((r - 0x38000000u) >> 13));
}

float fp16_to_float(uint16_t h) {            // IEEE binary16 -> float (exact)
  const uint32_t sign = (uint32_t)(h & 0x8000u) << 16, ex = (h >> 10) & 0x1fu, man = h & 0x3ffu;
  uint32_t u;
  if (ex == 0) {
    if (man == 0) u = sign;
    else {                                   // subnormal: value = man * 2^-24
      float f = (float)man * 5.9604644775390625e-8f;
      memcpy(&u, &f, 4);
      u |= sign;
    }
  } else if (ex == 31) u = sign | 0x7f800000u | (man << 13);
  else u = sign | ((ex + 112u) << 23) | (man << 13);
  float r;
  memcpy(&r, &u, 4);
  return r;
}

// Packs PyTorch-layout conv weights [C_out][C_in][K] into the image the kernel streams: a 2 KB header
// (biases [5][C], head weight [C], head bias) and, per segment in streaming order, per MMA step, the
// B operand [2 chunks][2C rows: C outputs of tap 2u, then of tap 2u+1][16 B of input channels],
// operand-rounded (TF32: RN ties away; BF16: RNE).
// CG = 2: two images back to back; rank r's steps hold B rows [r*C, (r+1)*C) only (rank 0 = the even tap of
// every pair, rank 1 = the odd tap).
template <int C, int BF16, int CG>
void pack_impl(const pvf_weights* w, int split_e1, unsigned char* dst_all) {
  using G = Geo<C, BF16, CG>;
  const Plan P = make_plan<C, BF16, CG>(split_e1);
  memset(dst_all, 0, (size_t)CG * P.total);
  for (int rank = 0; rank < CG; ++rank) {
  unsigned char* dst = dst_all + (size_t)rank * P.total;
  float* hdr = reinterpret_cast<float*>(dst);
  for (int l = 0; l < 5; ++l) memcpy(hdr + l * C, w->conv_b[l], sizeof(float) * C);
  memcpy(hdr + 5 * C, w->conv_w[5], sizeof(float) * C);
  hdr[6 * C] = w->conv_b[5][0];
  struct SegDef { int seg, layer, cin, taps, nkb, ch_base, f0; };
  const int A = G::D1E_A, B = G::D1E_B, N1 = G::NKB1;
  const SegDef defs[kSegs] = {
      {gE2, 1, C, 15, N1, 0, 0},        {gD1Ea, 4, 2 * C, 25, N1, C, 0},     {gB, 2, C, 5, N1, 0, 0},
      {gD1Eb, 4, 2 * C, 25, N1, C, A},  {gD2, 3, 2 * C, 15, 2 * N1, 0, 0},   {gD1Ec, 4, 2 * C, 25, N1, C, A + B},
      {gE1, 0, kHistCh, 25, 1, 0, 0},   {gD1U, 4, 2 * C, 25, N1, 0, 0}};
  constexpr bool B16 = G::B16, FX = G::FX;
  for (const SegDef& d : defs) {
    const float* W = w->conv_w[d.layer];          // [C][cin][taps]
    for (int s = 0; s < P.seg_steps[d.seg]; ++s) {
      const int fp = d.f0 + s;                    // physical step index inside the sub-layer
      const int f = fp / G::PH, part = fp % G::PH;   // logical step; FX: part 0 = main (TF32), part 1 = correction (BF16)
      int u, kk, pass = 0;                        // tap pair, K block
      if (d.seg == gE1 && B16 && !(split_e1 && BF16 == 2)) { u = 2 * f; kk = 0; }   // 16-bit e1: K chunk h of step f holds tap pair 2f + h
      else if (d.seg == gE1) { pass = f / 13; u = f % 13; kk = 0; }   // e1 split runs [pass][tap pair]
      else { u = f / d.nkb; kk = f % d.nkb; }
      unsigned char* step = dst + P.seg_off[d.seg] + (size_t)s * G::STEP_BYTES;
      if (G::PP && d.layer == 4) {
        // polyphase d1 (see the header): step = (offset u - 6, K block); B rows [0, C) = phase 0, [C, 2C) = phase 1.
        //   upsampled half (gD1U):  Wp[u][ci][co] = W[co][ci][2u - p] + W[co][ci][2u - p + 1]     (taps outside 0 .. 24 are absent)
        //   skip half (gD1E*):      K channel q * C + ci = skip channel ci at position 2i + q:  W[co][C + ci][2u + q - p]
        const bool up_half = d.seg == gD1U;
        const int nkb = up_half ? N1 : 2 * N1;
        const int uo = f / nkb, kb = f % nkb;
        for (int h = 0; h < 2; ++h)
          for (int nl = 0; nl < G::NB; ++nl)
            for (int e = 0; e < G::PER; ++e) {
              const int n = rank * G::NB + nl, ph = n / C, co = n % C;
              const int cl = (2 * kb + h) * G::PER + e;
              float v = 0.0f;
              if (up_half) {
                for (int j = 2 * uo - ph; j <= 2 * uo - ph + 1; ++j)
                  if (j >= 0 && j < d.taps) v += W[((size_t)co * d.cin + cl) * d.taps + j];
              } else {
                const int q = cl / C, ci = cl % C, j = 2 * uo + q - ph;
                if (j >= 0 && j < d.taps) v = W[((size_t)co * d.cin + C + ci) * d.taps + j];
              }
              unsigned char* pdst = step + ((size_t)h * G::NB + nl) * 16 + e * G::ES;
              if (B16) {
                const uint16_t b = (BF16 == 2) ? fp16_rne(v) : bf16_rne(v);
                memcpy(pdst, &b, 2);
              } else {
                const float out = tf32_rna(v);
                memcpy(pdst, &out, 4);
              }
            }
        continue;
      }
      if (d.seg == gE1 && (BF16 == 0 || BF16 == 2) && split_e1) {
        // split e1 of the TF32 kernel: BF16 pieces w = w1 + w2; pass 0 (13 steps) holds [w1 | w1] (meets [a1 | a2]),
        // pass 1 (7 steps) [w2 of pair 2w | w2 of pair 2w + 1] (meets [a1 two rows apart])
        if (pass) u = 2 * (f - 13);
        const bool half_x = 2 * u + 1 >= d.taps;
        const int nbx = half_x ? G::NB / 2 : G::NB;
        for (int h = 0; h < 2; ++h)
          for (int nl = 0; nl < nbx; ++nl)
            for (int e = 0; e < 8; ++e) {
              const int n = rank * nbx + nl;
              const int co = n % C, j = 2 * (u + (pass ? h : 0)) + n / C;
              const float v = j < d.taps ? W[((size_t)co * d.cin + e) * d.taps + j] : 0.0f;
              uint16_t w1, w2;                  // pieces in the format of the MMA: BF16 (TF32 kernel) or FP16 (FP16 kernel)
              if (BF16 == 2) {
                w1 = fp16_rne(v);
                w2 = fp16_rne(v - fp16_to_float(w1));
              } else {
                w1 = bf16_rne(v);
                uint32_t w1bits = (uint32_t)w1 << 16;
                float w1f;
                memcpy(&w1f, &w1bits, 4);
                w2 = bf16_rne(v - w1f);
              }
              const uint16_t out = pass == 0 ? w1 : w2;
              memcpy(step + ((size_t)h * nbx + nl) * 16 + e * 2, &out, 2);
            }
        continue;
      }
      // last tap pair (odd tap missing): an N = C step -- half as many B rows, all of the even tap, split over the pair
      const bool half_n = 2 * u + 1 >= d.taps;
      const int nb = half_n ? G::NB / 2 : G::NB;
      if (FX && part == 1) {
        // correction step: K chunk 0 = bf16(w) of the 8 input channels of K block kk (meets a_lo), K chunk 1 =
        // bf16(w - tf32(w)) of the same channels (meets bf16(a))
        for (int h = 0; h < 2; ++h)
          for (int nl = 0; nl < nb; ++nl)
            for (int e = 0; e < 8; ++e) {
              const int n = rank * nb + nl;
              const int co = n % C, j = 2 * u + n / C;
              const int cl = 8 * kk + e;
              const bool real = j < d.taps && ((d.seg == gE1) ? cl < kHistCh : true);
              const float v = real ? W[((size_t)co * d.cin + d.ch_base + cl) * d.taps + j] : 0.0f;
              const uint16_t out = h == 0 ? bf16_rne(v) : bf16_rne(v - tf32_rna(v));
              memcpy(step + ((size_t)h * nb + nl) * 16 + e * 2, &out, 2);
            }
        continue;
      }
      for (int h = 0; h < 2; ++h)
        for (int nl = 0; nl < nb; ++nl)           // rows [0, C): even tap 2u, rows [C, 2C): odd tap 2u + 1
          for (int e = 0; e < G::PER; ++e) {
            const int n = rank * nb + nl;
            const bool e1x2 = d.seg == gE1 && B16;
            const int co = n % C, j = 2 * (u + (e1x2 ? h : 0)) + n / C;
            const int cl = e1x2 ? e : (2 * kk + h) * G::PER + e;   // channel inside the sub-layer's range
            const bool real = j < d.taps && ((d.seg == gE1) ? cl < kHistCh : true);
            const float v = real ? W[((size_t)co * d.cin + d.ch_base + cl) * d.taps + j] : 0.0f;
            unsigned char* p = step + ((size_t)h * nb + nl) * 16 + e * G::ES;
            if (B16) {
              const uint16_t b = (BF16 == 2) ? fp16_rne(v) : bf16_rne(v);
              memcpy(p, &b, 2);
            } else {
              const float hi = tf32_rna(v);
              const float out = hi;
              memcpy(p, &out, 4);
            }
          }
    }
  }
  }
}

template <int C, int BF16, int CG, int TT = 0>
void launch_impl(const float* hist, int n_int, const void* packed, int split_e1, float* probs, int sm_count,
                 const int* list, const int* n_list, const int* seg_cnt, bool pdl, cudaStream_t s) {
  using G = Geo<C, BF16, CG, TT>;
  const int n_groups = (n_int + G::T - 1) / G::T;
#ifndef PVF_UNET_GRID_DIV
#define PVF_UNET_GRID_DIV 1      // experiments only: run on 1/N of the SMs (is a chip-wide resource the limit?)
#endif
  const int n_pg = (n_groups + CG - 1) / CG, max_pairs = sm_count / CG / PVF_UNET_GRID_DIV;
  const int grid = CG * (n_pg < max_pairs ? n_pg : max_pairs);
  PdlLaunch L(dim3(grid), dim3(G::THREADS), G::SMEM, s, pdl, CG);
  cudaLaunchKernelEx(&L.cfg, k_unet_tc<C, BF16, CG, TT>, hist, n_int, static_cast<const unsigned char*>(packed), split_e1,
                     probs, list, n_list, seg_cnt);
}

template <int C, int BF16, int CG>
cudaError_t setup_impl() {
  cudaError_t e = cudaFuncSetAttribute(k_unet_tc<C, BF16, CG, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       Geo<C, BF16, CG, 0>::SMEM);
  return e;
}

#define PVF_TC_DISPATCH_CG(CALL, CG_)                             \
  do {                                                            \
    const int fm = precision == PVF_PREC_BF16 ? 1 : (precision == PVF_PREC_FP16 ? 2 : 0);   \
    if (channels == 64) { if (fm == 1) CALL(64, 1, CG_); else if (fm == 2) CALL(64, 2, CG_); else CALL(64, 0, CG_); }      \
    else if (channels == 32) { if (fm == 1) CALL(32, 1, CG_); else if (fm == 2) CALL(32, 2, CG_); else CALL(32, 0, CG_); } \
    else { if (fm == 1) CALL(16, 1, CG_); else if (fm == 2) CALL(16, 2, CG_); else CALL(16, 0, CG_); }        \
  } while (0)
// PVF_PREC_FP32 on the tensor cores = the FP32-accurate format 3, CTA pairs only
#define PVF_TC_DISPATCH(CALL)                                     \
  do {                                                            \
    if (precision == PVF_PREC_FP32) {                             \
      if (channels == 64) CALL(64, 3, 2); else if (channels == 32) CALL(32, 3, 2); else CALL(16, 3, 2);   \
    } else if (cta_pair) PVF_TC_DISPATCH_CG(CALL, 2); else PVF_TC_DISPATCH_CG(CALL, 1);   \
  } while (0)

}  // namespace

size_t unet_tc_packed_bytes(int channels, int precision, int split_mask, int cta_pair) {
  size_t r = 0;
#define PVF_CALL(C_, B_, G_) r = (size_t)G_ * make_plan<C_, B_, G_>(split_mask & 1).total
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
  return r;
}

void unet_tc_pack(const pvf_weights* w, int channels, int precision, int split_mask, int cta_pair, void* host_dst) {
#define PVF_CALL(C_, B_, G_) pack_impl<C_, B_, G_>(w, split_mask & 1, static_cast<unsigned char*>(host_dst))
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
}

cudaError_t unet_tc_setup(int channels, int precision, int split_mask, int cta_pair) {
  if (channels != 64 && channels != 32 && channels != 16) return cudaErrorInvalidValue;
  if (split_mask & ~1) return cudaErrorInvalidValue;          // only the e1 split is built
  if (precision != PVF_PREC_TF32 && precision != PVF_PREC_FP16 && split_mask) return cudaErrorInvalidValue;   // the split serves the 10-bit formats
  if (precision == PVF_PREC_FP32 && !cta_pair) return cudaErrorInvalidValue;    // FP32 on the tensor cores runs as CTA pairs
  cudaError_t e = cudaSuccess;
#define PVF_CALL(C_, B_, G_) e = setup_impl<C_, B_, G_>()
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
  return e;
}

void launch_unet_tc(const float* hist, int n_intervals_total, const void* packed_dev, int channels, int precision,
                    int split_mask, int cta_pair, float* probs, int sm_count, const int* list, const int* n_list,
                    const int* seg_cnt, bool pdl, cudaStream_t s) {
  if (n_intervals_total <= 0) return;
#define PVF_CALL(C_, B_, G_) \
  launch_impl<C_, B_, G_>(hist, n_intervals_total, packed_dev, split_mask & 1, probs, sm_count, list, n_list, seg_cnt, pdl, s)
  PVF_TC_DISPATCH(PVF_CALL);
#undef PVF_CALL
}

// include/pvf_debug.h: per-CTA wait counters of the MMA issuer; only a -DPVF_UNET_PROF build records them
extern "C" __attribute__((visibility("default"))) int pvf_debug_unet_prof(unsigned long long* host_out, int reset) {
#ifdef PVF_UNET_PROF
  cudaDeviceSynchronize();
  if (host_out) cudaMemcpyFromSymbol(host_out, g_unet_prof, sizeof(g_unet_prof));
  if (reset) { static unsigned long long z[160][16]; cudaMemcpyToSymbol(g_unet_prof, z, sizeof(z)); }
  return 0;
#else
  (void)host_out; (void)reset;
  return -1;
#endif
}

}  // namespace pvf
