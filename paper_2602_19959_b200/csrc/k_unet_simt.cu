// a3, FP32 path -- the 1D UNet per z-interval as direct convolutions on the CUDA cores.
//
// PAPER.md:29 "5-layer UNet architecture (64 channels deployed)"; topology from BASELINE.json
// config 0: e1 8->C k25 (L100) | pool2 | e2 C->C k15 (L50) | pool2 | b C->C k5 (L25) | up2 (+) e2 ->
// d2 2C->C k15 | up2 (+) e1 -> d1 2C->C k25 | head 1x1 C->1 | sigmoid; "same" zero padding,
// LeakyReLU(0.01) after the five k>1 convs; concat order [upsampled, skip] (reading O5).
//
// This is PVF_PREC_FP32: plain FP32 FMAs (BASELINE.json config 0 "Single event, FP32"), used as the
// accuracy reference of the GPU side and for small batches.  The throughput path is k_unet_tc.cu.
// One CTA per interval; all activations of the interval live in shared memory as [C][L] rows, the
// skip tensors are written straight into the second half of the decoder's concat buffers, pooled /
// upsampled copies are produced by the epilogues, weights are read through L1/L2 in PyTorch layout.
#include "pvf_internal.cuh"
#include "pdl.cuh"

namespace pvf {

constexpr int kSimtThreads = 256;

__device__ __forceinline__ float lrelu(float v) { return v >= 0.0f ? v : kLeaky * v; }

enum { kOutPlain = 0, kOutUp2 = 1 };

// y[co][l] = lrelu(b[co] + sum_ci sum_j W[co][ci][j] * x[ci][l + j - p]),  x = 0 outside [0, L)
template <int C, int CIN, int K, int L, int MODE>
__device__ __forceinline__ void conv_layer(const float* __restrict__ x /* smem [CIN][L] */,
                                           const float* __restrict__ W, const float* __restrict__ B,
                                           float* __restrict__ y /* smem [C][L] or [C][2L] */) {
  constexpr int LG = kSimtThreads / C;
  constexpr int LSEG = (L + LG - 1) / LG;
  constexpr int P = (K - 1) / 2;
  constexpr int WIN = LSEG + K - 1;
  const int co = threadIdx.x / LG, lg = threadIdx.x % LG;
  const int l0 = lg * LSEG;
  float acc[LSEG];
  const float bias = B[co];
#pragma unroll
  for (int i = 0; i < LSEG; ++i) acc[i] = bias;
  const float* wrow = W + (size_t)co * CIN * K;
  for (int ci = 0; ci < CIN; ++ci) {
    float win[WIN];
    const float* xr = x + ci * L;
#pragma unroll
    for (int i = 0; i < WIN; ++i) {
      const int m = l0 + i - P;
      win[i] = (m >= 0 && m < L) ? xr[m] : 0.0f;
    }
#pragma unroll
    for (int j = 0; j < K; ++j) {
      const float w = __ldg(wrow + ci * K + j);
#pragma unroll
      for (int i = 0; i < LSEG; ++i) acc[i] = fmaf(w, win[i + j], acc[i]);
    }
  }
#pragma unroll
  for (int i = 0; i < LSEG; ++i) {
    const int l = l0 + i;
    if (l < L) {
      const float v = lrelu(acc[i]);
      if (MODE == kOutPlain) y[co * L + l] = v;
      else { y[co * 2 * L + 2 * l] = v; y[co * 2 * L + 2 * l + 1] = v; }
    }
  }
}

template <int C, int L>
__device__ __forceinline__ void pool2(const float* __restrict__ x, float* __restrict__ y) {
  for (int i = threadIdx.x; i < C * (L / 2); i += kSimtThreads) {
    const int c = i / (L / 2), l = i % (L / 2);
    y[i] = fmaxf(x[c * L + 2 * l], x[c * L + 2 * l + 1]);
  }
}

template <int C>
struct SimtSmem {
  float a1[2 * C][100];  // rows [0,C): up2(d2)   rows [C,2C): e1 (skip)
  float a2[2 * C][50];   // rows [0,C): up2(b)    rows [C,2C): e2 (skip)   | d1 output overlays a2+p1
  float p1[C][50];
  float p2[C][25];
  float h[kHistCh][100];
};

template <int C>
__global__ void __launch_bounds__(kSimtThreads)
k_unet_simt(const float* __restrict__ hist, int n_int, UnetParamsF32 p, float* __restrict__ probs) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SimtSmem<C>& S = *reinterpret_cast<SimtSmem<C>*>(smem_raw);
  pdl_launch_dependents();
  pdl_wait();                   // the histograms come from the FC kernel (pdl.cuh)
  for (int n = blockIdx.x; n < n_int; n += gridDim.x) {
    const float* H = hist + (size_t)n * kFcOut;
    for (int i = threadIdx.x; i < kFcOut; i += kSimtThreads) (&S.h[0][0])[i] = H[i];
    __syncthreads();
    conv_layer<C, kHistCh, 25, 100, kOutPlain>(&S.h[0][0], p.w[0], p.b[0], &S.a1[C][0]);      // e1
    __syncthreads();
    pool2<C, 100>(&S.a1[C][0], &S.p1[0][0]);
    __syncthreads();
    conv_layer<C, C, 15, 50, kOutPlain>(&S.p1[0][0], p.w[1], p.b[1], &S.a2[C][0]);            // e2
    __syncthreads();
    pool2<C, 50>(&S.a2[C][0], &S.p2[0][0]);
    __syncthreads();
    conv_layer<C, C, 5, 25, kOutUp2>(&S.p2[0][0], p.w[2], p.b[2], &S.a2[0][0]);               // b -> up2
    __syncthreads();
    conv_layer<C, 2 * C, 15, 50, kOutUp2>(&S.a2[0][0], p.w[3], p.b[3], &S.a1[0][0]);          // d2 -> up2
    __syncthreads();
    float* d1 = &S.a2[0][0];                                                                  // overlay
    conv_layer<C, 2 * C, 25, 100, kOutPlain>(&S.a1[0][0], p.w[4], p.b[4], d1);                // d1
    __syncthreads();
    if (threadIdx.x < kBins) {                                                                // head + sigmoid
      float a = p.b[5][0];
      for (int c = 0; c < C; ++c) a = fmaf(__ldg(p.w[5] + c), d1[c * 100 + threadIdx.x], a);
      probs[(size_t)n * kBins + threadIdx.x] = 1.0f / (1.0f + expf(-a));
    }
    __syncthreads();
  }
}

template <int C>
static cudaError_t setup_one() {
  return cudaFuncSetAttribute(k_unet_simt<C>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              (int)sizeof(SimtSmem<C>));
}

cudaError_t unet_simt_setup(int channels) {
  switch (channels) {
    case 64: return setup_one<64>();
    case 32: return setup_one<32>();
    case 16: return setup_one<16>();
  }
  return cudaErrorInvalidValue;
}

void launch_unet_simt(const float* hist, int n_int, const UnetParamsF32& p, int channels, float* probs,
                      bool pdl, cudaStream_t s) {
  if (n_int <= 0) return;
  const int grid = n_int < 148 * 64 ? n_int : 148 * 64;
  switch (channels) {
    case 64: { PdlLaunch L(dim3(grid), dim3(kSimtThreads), sizeof(SimtSmem<64>), s, pdl);
               cudaLaunchKernelEx(&L.cfg, k_unet_simt<64>, hist, n_int, p, probs); break; }
    case 32: { PdlLaunch L(dim3(grid), dim3(kSimtThreads), sizeof(SimtSmem<32>), s, pdl);
               cudaLaunchKernelEx(&L.cfg, k_unet_simt<32>, hist, n_int, p, probs); break; }
    case 16: { PdlLaunch L(dim3(grid), dim3(kSimtThreads), sizeof(SimtSmem<16>), s, pdl);
               cudaLaunchKernelEx(&L.cfg, k_unet_simt<16>, hist, n_int, p, probs); break; }
  }
}

}  // namespace pvf
