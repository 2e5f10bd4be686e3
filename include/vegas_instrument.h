/* vegas_instrument.h -- measurement hooks of libvegas_b200.so.  NOT part of the boundary of include/vegas.h (the calls
 * SURVEY.md 8(b) lists): bench.py uses them to time the fused kernel alone on the caller's stream and to count the
 * library's own launches (the contract's `roofline.achieved` and `gpu_launches`).  Same C ABI, same error codes. */
#ifndef VEGAS_B200_INSTRUMENT_H
#define VEGAS_B200_INSTRUMENT_H
#include "vegas.h"
#ifdef __cplusplus
extern "C" {
#endif

/* With profiling on, every fused-kernel launch is bracketed by CUDA events on its stream (and the programmatic
 * dependent launch between the chunk launches of the generic kernel is switched off); vegas_kernel_time_ms()
 * synchronises those events and returns their summed duration and the number of launches since the last
 * vegas_reset_counters().  vegas_launch_count() counts ALL kernels of this library launched for the grid (no
 * synchronisation). */
int vegas_set_profiling(vegas_grid* g, int on);
int vegas_kernel_time_ms(vegas_grid* g, double* iterate_kernel_ms, uint64_t* iterate_launches);
uint64_t vegas_launch_count(const vegas_grid* g);
int vegas_reset_counters(vegas_grid* g);

#ifdef __cplusplus
}
#endif
#endif /* VEGAS_B200_INSTRUMENT_H */
