/*
 * ah_b200_test.h — test and measurement hooks of libah_b200.so.  NOT part of the product interface
 * (that is ah_b200.h); used by tests/, bench.py and the profiling commands only.
 * Same conventions as ah_b200.h: C ABI, dev_* = device pointers, 0 / negative AH_E* return codes.
 */
#ifndef AH_B200_TEST_H
#define AH_B200_TEST_H

#include "ah_b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/* kernel selection for ah_set_kernel */
#define AH_KERNEL_AUTO 0  /* fused tiled kernel when the lattice allows it, else the site kernel */
#define AH_KERNEL_SITE 1  /* one thread per site, neighbours through L1/L2 (any nx,ny,nz >= 1) */
#define AH_KERNEL_TILED 2 /* z-marching register/shared-memory tiled kernel (needs nx % 64 == 0) */

/* Choose the step kernel (AH_KERNEL_*).  AH_EINVAL if the lattice does not allow it. */
int ah_set_kernel(ah_ctx *ctx, int kernel);

/* The step kernel the context currently launches: AH_KERNEL_SITE or AH_KERNEL_TILED (never AUTO);
 * AH_EINVAL for a null context. */
int ah_get_kernel(const ah_ctx *ctx);

/* Launch geometry the tiled kernel would use for a lattice (host logic only, no device needed; for tests and
 * reports): planes per CTA and number of CTAs.  Returns AH_EINVAL when the lattice does not allow the tiled kernel. */
int ah_tiled_launch_info(int nx, int ny, int nz, int *planes_per_cta, int *n_ctas);

/* Number of kernel launches this context has enqueued since creation (bench.py's gpu_launches). */
int64_t ah_launch_count(const ah_ctx *ctx);

/* Device-side evaluation of the library's fp32 sin/cos kernels' math (tests only): for each of the
 * n device floats in dev_x writes sin and cos as used for link variables, and the plaquette sine. */
int ah_test_trig(const float *dev_x, float *dev_sin, float *dev_cos, float *dev_plaq_sin, size_t n,
                 void *cuda_stream);

/* Same for the tiled step kernel's own trigonometry (tests only): sin/cos of the pi-reduced polynomial pair it
 * uses for link variables (valid for |x| < 2^18; the kernel's domain is |th| < 2^16) and the un-reduced Taylor
 * sine it uses for plaquette angles when a whole warp has |Phi| < 0.5 (dev_small_sin; meaningful for |x| < 0.5). */
int ah_test_trig_fast(const float *dev_x, float *dev_sin, float *dev_cos, float *dev_small_sin, size_t n,
                      void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* AH_B200_TEST_H */
