// One translation unit of FFT pass kernel instantiations (compiled once per -DFFT_UNIT=0..5; see fft_launch.cuh).
#include "fft_kernels.cuh"
#include "fft_launch.cuh"

#ifndef FFT_UNIT
#error "compile with -DFFT_UNIT=<0..7>"
#endif

namespace {

template <int LOGN, int LOGT, bool P2, int E, int VAR>
cudaError_t launch_pass(const LaunchCtx &ctx, FftArgs &a, int tiles_per_tmpl, int n_t) {
    using C = FftCfg<LOGN, LOGT, E>;
    constexpr int SMEM = P2 ? C::SMEM_BYTES : C::SMEM_BYTES_P1;
    static thread_local int configured_dev = -1;
    static thread_local int resident = 0;
    auto kern = fft_kernel_ptr<LOGN, LOGT, P2, E, VAR>();
    if (configured_dev != ctx.device) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) return e;
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, C::NT, SMEM);
        if (e != cudaSuccess) return e;
        resident = (per_sm > 0 ? per_sm : 1) * ctx.n_sm;
        configured_dev = ctx.device;
    }
    int lt = 0;
    while ((1 << lt) < tiles_per_tmpl) ++lt;
    a.log_tiles = lt;
    a.n_tiles = tiles_per_tmpl * n_t;
    a.n_tmpl = n_t;
    const int grid = a.n_tiles < resident ? a.n_tiles : resident;
    kern<<<grid, C::NT, SMEM, ctx.stream>>>(a);
    return cudaGetLastError();
}

}  // namespace

#define FFT_CAT2(a, b) a##b
#define FFT_CAT(a, b) FFT_CAT2(a, b)
#define K(P, LN, LT, E, V) if (pass == P && logn == LN && logt == LT && elems == E && var == V) return launch_pass<LN, LT, (P == 2), E, V>;
#define K1(LN, LT) K(1, LN, LT, 16, 0) K(1, LN, LT, 16, FFT_VAR_CUBIC)                                             // pass 1, plain + cubic
#define K1Z(LN, LT) K(1, LN, LT, 16, FFT_VAR_SKIPZ) K(1, LN, LT, 16, FFT_VAR_SKIPZ | FFT_VAR_CUBIC)                 // + padding-skipping variants
#define K1G(LN, LT) K(1, LN, LT, 16, FFT_VAR_GENERIC) K(1, LN, LT, 16, FFT_VAR_GENERIC | FFT_VAR_CUBIC)             // + general store address

#if FFT_UNIT == 6      // fused sky + pass 1 (sky-varying search)
namespace {
template <int LOGN, int LOGT, int VAR>
cudaError_t launch_fused(const LaunchCtx &ctx, FusedArgs &a, int tiles_per_tmpl, int n_groups) {
    using C = FftCfg<LOGN, LOGT, 16>;
    constexpr int SMEM = FusedCfg<LOGN, LOGT>::SMEM_BYTES;
    static thread_local int configured_dev = -1;
    static thread_local int resident = 0;
    auto kern = fft_sky_pass1_kernel<LOGN, LOGT, VAR>;
    if (configured_dev != ctx.device) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) return e;
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, C::NT, SMEM);
        if (e != cudaSuccess) return e;
        resident = (per_sm > 0 ? per_sm : 1) * ctx.n_sm;
        configured_dev = ctx.device;
    }
    int lt = 0;
    while ((1 << lt) < tiles_per_tmpl) ++lt;
    a.f.log_tiles = lt;
    a.f.n_tiles = tiles_per_tmpl * n_groups;
    const int grid = a.f.n_tiles < resident ? a.f.n_tiles : resident;
    kern<<<grid, C::NT, SMEM, ctx.stream>>>(a);
    return cudaGetLastError();
}
}  // namespace
#define KF(LN, LT) if (logn == LN && logt == LT && var == 0) return launch_fused<LN, LT, 0>; \
                   if (logn == LN && logt == LT && var == FFT_VAR_CUBIC) return launch_fused<LN, LT, FFT_VAR_CUBIC>;
#define KFG(LN, LT) if (logn == LN && logt == LT && var == FFT_VAR_GENERIC) return launch_fused<LN, LT, FFT_VAR_GENERIC>; \
                    if (logn == LN && logt == LT && var == (FFT_VAR_GENERIC | FFT_VAR_CUBIC)) return launch_fused<LN, LT, FFT_VAR_GENERIC | FFT_VAR_CUBIC>;
fused_launch_fn fft_find_fused_kernel(int logn, int logt, int var) {
    KF(6, 11) KF(7, 11) KF(8, 11) KF(9, 11) KF(10, 11) KF(11, 11) KF(12, 12)
    KFG(6, 11) KFG(7, 11) KFG(8, 11)
    return nullptr;
}
#elif FFT_UNIT == 7    // both passes in one cooperative kernel (small transforms)
namespace {
template <int LOGN1, int LOGN2, int VAR>
cudaError_t launch_single(const LaunchCtx &ctx, SingleArgs &a, int *resident_out) {
    using SC = SingleCfg<LOGN1, LOGN2, 11, VAR>;
    constexpr int SMEM = SC::SMEM_BYTES, NT = SC::C1::NT;
    static_assert(SC::C1::NT == SC::C2::NT, "both passes run with the same block size");
    static thread_local int configured_dev = -1;
    static thread_local int resident = 0;
    auto kern = fft_single_kernel<LOGN1, LOGN2, 11, VAR>;
    if (configured_dev != ctx.device) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, 100);
        if (e != cudaSuccess) return e;
        int per_sm = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, SMEM);
        if (e != cudaSuccess) return e;
        resident = (per_sm > 0 ? per_sm : 1) * ctx.n_sm;
        configured_dev = ctx.device;
    }
    if (resident_out) *resident_out = resident;
    if (!a.counter) return cudaSuccess;                 // query only
    void *args[] = {&a};
    return cudaLaunchCooperativeKernel((const void *)kern, dim3(resident), dim3(NT), args, SMEM, ctx.stream);
}
}  // namespace
#define KS(L1, L2, V) if (logn1 == L1 && logn2 == L2 && var == (V)) return launch_single<L1, L2, (V)>; \
                      if (logn1 == L1 && logn2 == L2 && var == ((V) | FFT_VAR_CUBIC)) return launch_single<L1, L2, (V) | FFT_VAR_CUBIC>;
single_launch_fn fft_find_single_kernel(int logn1, int logn2, int var) {
    KS(6, 6, FFT_VAR_GENERIC) KS(7, 6, FFT_VAR_GENERIC) KS(7, 7, 0) KS(9, 6, 0) KS(10, 6, 0) KS(10, 7, 0) KS(10, 8, 0)
    return nullptr;
}
#else
fft_launch_fn FFT_CAT(fft_find_kernel_unit, FFT_UNIT)(int pass, int logn, int logt, int elems, int var) {
#if FFT_UNIT == 0      // pass 1, sub-FFT 2^6 .. 2^9
    K1(6, 11) K1(7, 11) K1(8, 11) K1(9, 11) K1(6, 12) K1(7, 12) K1(8, 12) K1(9, 12)
    K(1, 9, 10, 32, 0) K(1, 9, 10, 32, FFT_VAR_CUBIC)                      // one warp per two 2^9-point columns
    K(1, 9, 10, 32, FFT_VAR_GENERIC) K(1, 9, 10, 32, FFT_VAR_GENERIC | FFT_VAR_CUBIC)
    K1G(6, 11) K1G(7, 11) K1G(8, 11) K1G(6, 12) K1G(7, 12) K1G(8, 12)
#elif FFT_UNIT == 1    // pass 1, sub-FFT 2^10, 2^11
    K1(10, 11) K1(10, 12) K1(10, 13) K1Z(10, 11)
    K(1, 10, 10, 32, 0) K(1, 10, 10, 32, FFT_VAR_CUBIC)                    // one warp per 2^10-point column, two radix-32 passes
    K(1, 10, 10, 32, FFT_VAR_GENERIC) K(1, 10, 10, 32, FFT_VAR_GENERIC | FFT_VAR_CUBIC)
    K1(11, 11) K1(11, 12) K1(11, 13) K1Z(11, 11) K1Z(11, 12)
#elif FFT_UNIT == 2    // pass 1, sub-FFT 2^12
    K1(12, 12) K1(12, 13) K1Z(12, 12) K1Z(12, 13)
#elif FFT_UNIT == 3    // pass 2, sub-FFT 2^6 .. 2^9
    K(2, 6, 11, 16, 0) K(2, 7, 11, 16, 0) K(2, 8, 11, 16, 0) K(2, 9, 11, 16, 0)
    K(2, 6, 12, 16, 0) K(2, 7, 12, 16, 0) K(2, 8, 12, 16, 0) K(2, 9, 12, 16, 0) K(2, 9, 12, 32, 0)
    K(2, 6, 12, 16, FFT_VAR_FAFB) K(2, 7, 12, 16, FFT_VAR_FAFB) K(2, 8, 12, 16, FFT_VAR_FAFB) K(2, 9, 12, 32, FFT_VAR_FAFB)   // debug: Fa, Fb out
#elif FFT_UNIT == 4    // pass 2, sub-FFT 2^10, 2^11
    K(2, 10, 11, 16, 0) K(2, 10, 12, 16, 0) K(2, 10, 13, 16, 0) K(2, 10, 12, 32, 0) K(2, 10, 13, 32, 0)
    K(2, 11, 11, 16, 0) K(2, 11, 12, 16, 0) K(2, 11, 13, 16, 0)
    K(2, 10, 12, 32, FFT_VAR_FAFB) K(2, 10, 13, 32, FFT_VAR_FAFB)                                                             // debug: Fa, Fb out
#elif FFT_UNIT == 5    // pass 2, sub-FFT 2^12
    K(2, 12, 12, 16, 0) K(2, 12, 13, 16, 0)
#endif
    return nullptr;
}
#endif
