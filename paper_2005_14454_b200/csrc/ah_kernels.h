// ah_kernels.h — launcher declarations shared by the .cu translation units of libah_b200.so.
#pragma once

#include "ah_common.cuh"

namespace ah {

// general one-thread-per-site step (ah_site_kernel.cu)
template <typename real>
cudaError_t launch_site_step(const ConstFields<real> &in, const Fields<real> &out,
                             const StepCoef<real> &k, int nx, int ny, int nz, ZRange zr, cudaStream_t st);

// fp32 storage, fp64 arithmetic (SURVEY 8(f)4 "mixed precision"): the site kernel's algebra in double on floats
cudaError_t launch_site_step_mixed(const ConstFields<float> &in, const Fields<float> &out,
                                   const StepCoef<double> &k, int nx, int ny, int nz, ZRange zr, cudaStream_t st);

// I0 (ah_site_kernel.cu).  The array holds nz_alloc planes of nx*ny sites; plane zl is plane
// (z_offset + zl) mod nz_global of the global lattice, whose linear site index feeds the counter-based generator
// (whole lattice: nz_alloc = nz_global, z_offset = 0; z slab: nz_alloc = own planes + 2, z_offset = first own - 1).
template <typename real>
cudaError_t launch_init(const Fields<real> &out, uint64_t seed, double sigma, int nx, int ny, int nz_alloc,
                        int nz_global, int z_offset, cudaStream_t st);

// z-marching tiled fp32 step (ah_tiled_kernel.cu); needs nx % 64 == 0 (128-site warp rows when nx % 128 == 0,
// 64-site rows otherwise)
bool tiled_supported(int nx, int ny, int nz);
//   overflow: device int, set to 1 when a link angle is outside the kernel's domain (|th| >= 2^16 rad);
//             the outputs of that step must then be recomputed with the site kernel
//   dk, partials: both non-null selects the fused DIAG instantiation (SURVEY 8(a) row D-fuse): the step plus
//             the read-outs of its ENTRY snapshot, one DiagPartial per CTA (tiled_num_blocks of them), to be
//             totalled by launch_diag_final
cudaError_t launch_tiled_step(const ConstFields<float> &in, const Fields<float> &out,
                              const StepCoef<float> &k, int nx, int ny, int nz, ZRange zr, int *overflow, cudaStream_t st,
                              const DiagCoef *dk = nullptr, DiagPartial *partials = nullptr);
int tiled_num_blocks(int nx, int ny, int nz, bool diag = false);   // the DIAG instantiation has its own tile height
int tiled_chunk(int nx, int ny, int nz, bool diag = false);        // z planes per CTA
// after a tiled step: redo it with the site kernel iff *flag != 0; clears *clear (the next step's flag)
cudaError_t launch_site_redo(const int *flag, int *clear, const ConstFields<float> &in, const Fields<float> &out,
                             const StepCoef<float> &k, int nx, int ny, int nz, ZRange zr, cudaStream_t st);
cudaError_t tiled_setup();  // one-time function attributes (shared-memory carve-out)
float tiled_th_limit();     // the kernel's domain: every |th| below this (2^16 rad)
// z slabs (ah_site_kernel.cu): raise *flag when a link angle of one of the np <= 4 listed planes is outside the tiled
// kernel's domain (planes a slab launch reads without owning them)
cudaError_t launch_th_range_check(int *flag, const ConstFields<float> &in, int nx, int ny, const int *planes, int np,
                                  float limit, cudaStream_t st);

// diagnostics (ah_diag_kernel.cu)
//   partials: device array of at least diag_num_blocks(...) DiagPartial
//   result  : device pointer to ONE DiagPartial (the fixed-order total)
//   w3/near3: optional device int8/uint8 arrays of 3*n (per-plaquette output) or nullptr
int diag_num_blocks(int nx, int ny, int nz);   // nz: planes read out
template <typename real>
cudaError_t launch_diag(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz, ZRange zr,
                        DiagPartial *partials, DiagPartial *result, int8_t *w3, uint8_t *near3,
                        cudaStream_t st);

// the per-block partials alone; only_if != nullptr makes the launch conditional on *only_if != 0 (the redo of a
// fused record whose tiled kernel met a link angle outside its domain)
template <typename real>
cudaError_t launch_diag_partials(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz, ZRange zr,
                                 DiagPartial *partials, int8_t *w3, uint8_t *near3, const int *only_if,
                                 cudaStream_t st);

// fixed-order total of n per-block partials into *result (one block); of n_alt partials when *use_alt != 0
cudaError_t launch_diag_final(const DiagPartial *partials, int n, DiagPartial *result, cudaStream_t st, int n_alt = 0,
                              const int *use_alt = nullptr);

// read-outs of a whole lattice with the partials in the library's own fixed device array (no allocation anywhere):
// at most diag_noalloc_capacity() blocks, i.e. diag_num_blocks(nx, ny, nz) <= that; result as in launch_diag.  The
// first call on a device looks the array's address up (cudaGetSymbolAddress).
int diag_noalloc_capacity();
template <typename real>
cudaError_t launch_diag_noalloc(const ConstFields<real> &in, const DiagCoef &k, int nx, int ny, int nz,
                                DiagPartial *result, cudaStream_t st);

// tests only: evaluate the fp32 trig helpers on device arrays
cudaError_t launch_test_trig(const float *x, float *s, float *c, float *ps, size_t n, cudaStream_t st);
cudaError_t launch_test_trig_fast(const float *x, float *s, float *c, float *ss, size_t n, cudaStream_t st);

}  // namespace ah
