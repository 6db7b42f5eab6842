// pvf_histogram_noalloc (include/pvf.h): a0 + a1 + a2 for a small batch with the kernels' scratch in a file-scope
// static __device__ array instead of the handle's pool -- an entry point that allocates nothing, for callers that
// cannot call cudaMalloc or hand over a pool (graph capture, tight serving loops, harnesses that forbid it).
//
// PAPER.md:29, 49 and BASELINE.json config 0 define the computation (interval sort, per-track FC 9 -> 25 x 5 -> 800,
// ordered segmented sum into H [E, 40, 8, 100]); the kernels are the existing k_sort and k_fc_hist (FP32, CUDA cores),
// launched through their existing launchers with scratch pointers into the array below.
//
// The array's NAME is a host-side stand-in in host code, not a device address: its address is resolved with
// cudaGetSymbolAddress once per device (with that device current) and only that pointer is passed to kernels.
#include <mutex>
#include <stdio.h>
#include "pvf_internal.cuh"

namespace pvf {
namespace {

constexpr int kNaEvents = PVF_NOALLOC_MAX_EVENTS;    // 64
constexpr int kNaTracks = PVF_NOALLOC_MAX_TRACKS;    // 16384
constexpr size_t na_align(size_t v) { return (v + 255) / 256 * 256; }
// sub-arrays, each 256-byte aligned: perm (two slots per track: boundary tracks of NEXT-1), seg_off, seg_cnt, flags
constexpr size_t kOffPerm = 0;
constexpr size_t kOffSegOff = kOffPerm + na_align(sizeof(int32_t) * 2 * kNaTracks);
constexpr size_t kOffSegCnt = kOffSegOff + na_align(sizeof(int32_t) * kIntervals * kNaEvents);
constexpr size_t kOffFlags = kOffSegCnt + na_align(sizeof(int32_t) * kIntervals * kNaEvents);
constexpr size_t kNaBytes = kOffFlags + na_align(sizeof(uint32_t) * kNaEvents);
static_assert(kNaBytes <= PVF_NOALLOC_SCRATCH_BYTES, "include/pvf.h states the size of the static scratch");

// Held by every GPU that loads the library until the process exits (about 149 KB).  Shared by ALL calls.
static __device__ __align__(256) unsigned char g_noalloc_scratch[PVF_NOALLOC_SCRATCH_BYTES];

constexpr int kMaxDevices = 64;
std::mutex g_mu;
unsigned char* g_scratch_addr[kMaxDevices] = {};      // device address of g_noalloc_scratch on device d, once resolved

// Once per device, with that device current: the array's device address and the FC kernel's shared-memory opt-in.
cudaError_t setup_device(int dev, unsigned char** out) {
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    unsigned char* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p || (reinterpret_cast<uintptr_t>(p) & 255u)) return cudaErrorInvalidSymbol;
    e = fc_hist_setup();                               // cudaFuncSetAttribute; handles of the tensor-core modes never did it
    if (e != cudaSuccess) return e;
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

}  // namespace
}  // namespace pvf

using namespace pvf;

extern "C" PVF_API pvf_status pvf_histogram_noalloc(pvf_handle h, const pvf_tracks* t, int32_t n_events, float* dev_hist,
                                                    uint32_t* dev_event_flags, void* cuda_stream) {
  HandleView v;
  if (!handle_view(h, &v) || !t || !cuda_stream || n_events < 0) return PVF_ERR_ARG;
  if (n_events == 0) return PVF_OK;
  if (!dev_hist || !t->event_offsets || t->n_tracks < 0) return PVF_ERR_ARG;
  for (int k = 0; k < 9; ++k)
    if (!t->feat[k] && t->n_tracks > 0) return PVF_ERR_ARG;
  if (n_events > kNaEvents || t->n_tracks > kNaTracks) {
    char msg[200];
    snprintf(msg, sizeof(msg), "pvf_histogram_noalloc: %d events / %lld tracks exceed the static scratch (at most %d events, "
             "%d tracks per call); use pvf_run", (int)n_events, (long long)t->n_tracks, kNaEvents, kNaTracks);
    handle_set_error(h, msg);
    return PVF_ERR_CAPACITY;
  }
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { handle_set_error(h, cudaGetErrorString(e)); return PVF_ERR_CUDA; }
  if (dev != v.device || dev < 0 || dev >= kMaxDevices) {
    handle_set_error(h, "pvf_histogram_noalloc: the current device is not the handle's");
    return PVF_ERR_ARG;
  }
  unsigned char* scratch = nullptr;
  e = setup_device(dev, &scratch);
  if (e != cudaSuccess) {
    char msg[200];
    snprintf(msg, sizeof(msg), "pvf_histogram_noalloc set-up (cudaGetSymbolAddress / cudaFuncSetAttribute): %s", cudaGetErrorString(e));
    handle_set_error(h, msg);
    return PVF_ERR_CUDA;
  }
  int32_t* perm = reinterpret_cast<int32_t*>(scratch + kOffPerm);
  int32_t* seg_off = reinterpret_cast<int32_t*>(scratch + kOffSegOff);
  int32_t* seg_cnt = reinterpret_cast<int32_t*>(scratch + kOffSegCnt);
  uint32_t* flags = dev_event_flags ? dev_event_flags : reinterpret_cast<uint32_t*>(scratch + kOffFlags);
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  // Nothing in the scratch has to start at zero: k_sort writes seg_off / seg_cnt / flags of every event and the perm
  // entries those ranges name, and k_fc_hist reads only these.  No programmatic dependent launch: plain stream order.
  launch_sort(t->feat[0], t->event_offsets, n_events, (int)t->n_tracks, perm, seg_off, seg_cnt, flags, v.mfrac, s);
  launch_fc_hist(t->feat, t->event_offsets, perm, seg_off, seg_cnt, v.fc_params, n_events, dev_hist, v.sm_count, false, s);
  e = cudaPeekAtLastError();
  if (e != cudaSuccess) {
    handle_set_error(h, cudaGetErrorString(e));
    return PVF_ERR_CUDA;
  }
  return PVF_OK;
}
