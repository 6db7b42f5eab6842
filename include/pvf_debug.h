/* pvf_debug.h -- diagnostic entry points of libpvf.so that are NOT part of the product boundary (include/pvf.h).
 *
 * The two tensor-core kernels can be built with per-role cycle counters (PVF_NVCC_EXTRA="-DPVF_FC_PROF -DPVF_UNET_PROF"
 * python -m paper_2602_19959_b200.build --force): clock64() deltas around every mbarrier wait of one lane per role,
 * accumulated per CTA in a device array.  They answer "which role waits for which" (DESIGN.md sections 4.2 / 4.3;
 * the measured tables are under profiles/).  A normal build exports the same two symbols; they then return -1 and
 * touch nothing, so the symbol table does not depend on the build flavour.
 */
#ifndef PVF_DEBUG_H
#define PVF_DEBUG_H

#include "pvf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* host_out: HOST buffer of 160 x 16 unsigned 64-bit counters ([CTA][slot], cycles; NULL = do not read).
 * reset != 0 zeroes the device counters afterwards.  Synchronises the device.  Returns 0, or -1 if the library
 * was built without the counters.
 * k_fc_hist_tc slots: [0] epilogue waits for the interval list, [1] epilogue waits for
 * the accumulator, [2] epilogue total; [3] MMA issuer waits for the B operand, [4] MMA issuer waits for a drained
 * accumulator, [5] MMA issuer total; [6] hidden-layer group 0 waits for its operand buffer, [7] ... for its interval
 * list, [8] hidden-layer group 0 total; [9] tiles processed. */
PVF_API int pvf_debug_fc_prof(unsigned long long* host_out, int reset);

/* k_unet_tc slots: [0..5] MMA issuer waits for epilogue k (x0 staged, e1, e2, b,
 * d2, d1), [6] ... for a ring stage (own half), [7] ... for the peer's half of the stage, [8] issuer total. */
PVF_API int pvf_debug_unet_prof(unsigned long long* host_out, int reset);

#ifdef __cplusplus
}
#endif
#endif /* PVF_DEBUG_H */
