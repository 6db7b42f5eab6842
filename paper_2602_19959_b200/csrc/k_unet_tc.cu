// placeholder until the tcgen05 kernel lands
#include "pvf_internal.cuh"
namespace pvf {
size_t unet_tc_packed_bytes(int, int, int) { return 256; }
void unet_tc_pack(const pvf_weights*, int, int, int, void*) {}
cudaError_t unet_tc_setup(int, int, int) { return cudaErrorInvalidValue; }
void launch_unet_tc(const float*, int, const void*, int, int, int, float*, int, cudaStream_t) {}
}
