// Launch plumbing of the FFT pass kernels.  The kernel templates of fft_kernels.cuh are instantiated in several
// translation units (fft_unit.cu compiled once per FFT_UNIT value, in parallel: build.py); each unit exports one
// lookup function, and fstat_capi.cu asks them in turn.
#pragma once
#include "fstat_common.cuh"

// Arguments of one FFT pass launch (both passes).
struct FftArgs {
    const float4 *S;          // [n_sky_slots][n_fft] resampled series, tile-blocked: [k2/W1][k1][k2%W1]
    float4 *T;                // [templates of this launch][n_fft] intermediate, tile-blocked: [m1/W2][k2][m1%W2]
    const TmplDesc *tmpl;     // descriptors of the templates of this launch
    const SkyABCD *abcd;      // [n_sky_slots]
    float *twoF;              // output rows of this launch
    uint32_t *gmax;           // top-k mode: [tile][warp] maximum (as topk_key) of the 512 bins each warp of pass 2 writes; else null
    int64_t twoF_stride;      // floats between rows
    const float2 *tw;         // twiddle table of this sub-FFT length
    int64_t n_fft, n_src, n_bins, k_margin;
    double dt;
    int log_other;            // log2 of the other factor (N2 for pass 1, N1 for pass 2)
    int log_w_other;          // log2 W of the other pass (layout of T)
    int log_tiles;            // log2(tiles per template) = log_other - LOGW
    int n_tiles;              // tiles per template * templates in this launch
    int accumulate;           // pass 2: add 2F to what the output row holds (semi-coherent sum over segments)
    int n_tmpl;               // templates of this launch
    int t_fast;               // pass 1: tile order with the template varying fastest (S read from HBM once per launch)
};

// Arguments of the fused sky + FFT pass-1 kernel (sky-varying search): the FFT arguments plus what the sky-dependent
// half needs.  Tiles are (sky group of the launch, column block); f.tmpl / f.T are indexed by template within the launch.
struct FusedArgs {
    FftArgs f;
    PlanGeom g;
    const SkyConst *skies;    // [groups of this launch]
    const double4 *nodes;     // [groups of this launch][n_det][n_nodes] timing nodes
    const float2 *rot;        // [n_src] sidereal-angle table
    const float2 *Y;          // Farrow-filtered series
    const float *wslot;       // [n_det][n_slots]
    const int2 *groups;       // [groups of this launch] (first template within the launch, count)
    uint32_t det_mask;
};

// Arguments of the single-kernel form (both passes, small transforms): the two passes' arguments, the group size G
// (templates whose intermediates share one half of the 2 G-template buffer p1.T = p2.T) and the grid barrier counter
// (zeroed by the host before the launch).
struct SingleArgs {
    FftArgs p1, p2;
    int n_tmpl, group;
    unsigned *counter;
};

struct LaunchCtx {
    cudaStream_t stream;
    int device;
    int n_sm;
};

// Persistent launch of one FFT pass over n_t templates of tiles_per_tmpl tiles each: grid = min(n_tiles, resident CTAs).
typedef cudaError_t (*fft_launch_fn)(const LaunchCtx &ctx, FftArgs &a, int tiles_per_tmpl, int n_t);

// pass: 1 or 2; logn: log2 of the sub-FFT length; logt: log2 of the tile size; elems: register elements per thread (16
// or 32); var: FFT_VAR_* bits of the pass-1 variant (pass 2: 0 or FFT_VAR_FAFB).  Null when the unit has no such kernel.
#define FFT_VAR_SKIPZ 1      // neither stage nor touch the zero padding
#define FFT_VAR_CUBIC 2      // templates with fddot != 0 in the launch
#define FFT_VAR_GENERIC 4    // general (non-affine) address of the transposed store
#define FFT_VAR_FAFB 8       // pass 2 only: store (Fa, Fb) per bin instead of 2F (fstat_debug_compute_fafb; default shapes up to n_fft 2^22)
typedef cudaError_t (*fused_launch_fn)(const LaunchCtx &ctx, FusedArgs &a, int tiles_per_tmpl, int n_groups);
fused_launch_fn fft_find_fused_kernel(int logn, int logt, int var);      // unit 6

// single cooperative kernel (unit 7): *resident = CTAs the launch runs with (all co-resident)
typedef cudaError_t (*single_launch_fn)(const LaunchCtx &ctx, SingleArgs &a, int *resident);
single_launch_fn fft_find_single_kernel(int logn1, int logn2, int var);

#define FFT_N_UNITS 6
fft_launch_fn fft_find_kernel_unit0(int pass, int logn, int logt, int elems, int var);
fft_launch_fn fft_find_kernel_unit1(int pass, int logn, int logt, int elems, int var);
fft_launch_fn fft_find_kernel_unit2(int pass, int logn, int logt, int elems, int var);
fft_launch_fn fft_find_kernel_unit3(int pass, int logn, int logt, int elems, int var);
fft_launch_fn fft_find_kernel_unit4(int pass, int logn, int logt, int elems, int var);
fft_launch_fn fft_find_kernel_unit5(int pass, int logn, int logt, int elems, int var);

inline fft_launch_fn fft_find_kernel(int pass, int logn, int logt, int elems, int var) {
    fft_launch_fn (*const units[FFT_N_UNITS])(int, int, int, int, int) = {
        fft_find_kernel_unit0, fft_find_kernel_unit1, fft_find_kernel_unit2,
        fft_find_kernel_unit3, fft_find_kernel_unit4, fft_find_kernel_unit5};
    for (int u = 0; u < FFT_N_UNITS; ++u)
        if (fft_launch_fn f = units[u](pass, logn, logt, elems, var)) return f;
    return nullptr;
}
