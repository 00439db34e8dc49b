/*
 * lisatdi_bench.h -- measurement instruments of liblisatdi.so: NOT part of the product interface (lisatdi.h).
 * bench.py uses them for the roofline denominator (an FP64 issue-rate probe), for per-kernel device times (CUDA events
 * recorded around every launch of the library) and for the launch count of the timed region.
 */
#ifndef LISATDI_BENCH_H
#define LISATDI_BENCH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* FP64 pipe probe for the roofline denominator: launches a register-resident chain of
 * fused multiply-adds (blocks x 256 threads, 8 independent chains per thread, iters x 64 DFMA per
 * chain step) and writes one value per thread to d_out (blocks * 256 doubles).  *dfma_per_launch
 * receives the number of DFMA the launch executes. */
int ltdi_fp64_probe(double *d_out, int blocks, int iters, void *stream, double *dfma_per_launch);

/* Per-kernel device timing for bench.py's roofline.  While enabled, every kernel launch of the library is
 * bracketed by two CUDA events recorded on the stream it is launched on.  ltdi_profile_read() waits for the
 * recorded events and returns, for kernel id `kernel` (LTDI_KERNEL_*) launched by response `which`
 * (LTDI_RESPONSE_*; the orbit kernel counts under 0), the accumulated device time [ms] and the number of
 * launches since the last ltdi_profile_reset().  Process-global; off by default. */
enum { LTDI_KERNEL_ORBIT = 0,     /* orbit_delay_kernel: S0 */
       LTDI_KERNEL_PREP = 1,      /* per-source parameters and source frames: S1 (batch > 32 or generic orders only) */
       LTDI_KERNEL_ANCHOR = 2,    /* Lagrange weight anchors of the TDI delays (orders 9, 31) */
       LTDI_KERNEL_LINK_FULL = 3, /* link_kernel<.,false>: S2 + S3, Eq. (2.5); hybrid: link_hybrid_kernel, both kinds of link tiles in one launch */
       LTDI_KERNEL_LINK_LFA = 4,  /* link_kernel<.,true>: S6, Eq. (B10) */
       LTDI_KERNEL_TDI = 5,       /* tdi_kernel: S4 + S5 (hybrid: the tiles after the window and, blended, the tiles it touches: S8) */
       LTDI_KERNEL_GENERIC = 6,   /* response_kernel: fused tile kernel of the other Lagrange orders */
       LTDI_KERNEL_TDI_LFA = 7,   /* tdi_kernel, LFA instance: S7 (hybrid: the blocks before the window) */
       LTDI_KERNEL_PLAN = 8,      /* hybrid_plan_kernel: compact tile lists of the hybrid, S8 */
       LTDI_KERNEL_COUNT = 9 };
int ltdi_profile_enable(int on);
int ltdi_profile_read(int kernel, int which, double *total_ms, int64_t *launches);
int ltdi_profile_reset(void);

/* (TDI tile, channel) pairs of the current device that could not use the tile's weight anchors (light times drifting
 * by more than the Taylor bound over a tile, or an integer shift stepping inside it) and took exact per-sample weights
 * instead, since the last reset: a performance diagnostic -- the results are the same to rounding.  Synchronises. */
int ltdi_profile_slow_tiles(int64_t *count, int reset);

/* Number of kernel launches the library has issued in this process (for bench.py's gpu_launches). */
int64_t ltdi_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* LISATDI_BENCH_H */
