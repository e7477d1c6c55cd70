// Kernels of the sky-dependent half of the path (H1-H5 of DESIGN.md) in its hoisted form, and the once-per-plan
// tables they use.  PAPER.md:81-84 (steps iii-vi), eq. 3.  Device functions: sky_math.cuh.
#pragma once
#include "sky_math.cuh"

// H3 in Farrow form.  The interpolation weight of tap m, c_m(d) = sinc(d-m) W(d-m) for d in [-1/2, 1/2)
// (S6), is an entire function of d; fstat_setup expands it as c_m(d) = sum_p a[m][p] d^p
// (Chebyshev interpolation of degree FARROW_NC - 1 = 7, converted to powers of d, fp64 -> fp32).  Then
//     z(j0 + d) = sum_m x[j0+m] c_m(d) = sum_p d^p Y_p[j0],   Y_p[j] = sum_m a[m][p] x[j+m]:
// the 2D+1 taps are folded, once per plan and independent of the sky position, into FARROW_NC filtered
// copies of the series (this kernel); per SSB grid point the resampler then reads FARROW_NC complex
// numbers (FARROW_NC / 2 = 4 coalesced float4 loads) and runs one Horner recurrence instead of evaluating 2D+1 weights.
//   series : [n_det][series_stride] float2 (data at +SERIES_PAD, zeros around it)
//   coef   : [2D+1][FARROW_NC] float, row m+D
//   Y      : [n_det][ceil((N+1)/32)][FARROW_NC/2][32] float4 = (Re Y_2c, Im Y_2c, Re Y_2c+1, Im Y_2c+1) (farrow_index, sky_math.cuh)
__global__ void __launch_bounds__(SKY_THREADS)
farrow_filter_kernel(PlanGeom g, const float2 *__restrict__ series, const float *__restrict__ coef, float2 *__restrict__ Y) {
    __shared__ float s_coef[(2 * FSTAT_MAX_DTERMS + 1) * FARROW_NC];
    const int D = g.dterms, X = blockIdx.y;
    for (int e = threadIdx.x; e < (2 * D + 1) * FARROW_NC; e += SKY_THREADS) s_coef[e] = coef[e];
    __syncthreads();
    const int64_t j = (int64_t)blockIdx.x * SKY_THREADS + threadIdx.x;
    if (j > g.n_samples) return;
    const float2 *x = series + (int64_t)X * g.series_stride + SERIES_PAD + j;
    float2 acc[FARROW_NC];
#pragma unroll
    for (int p = 0; p < FARROW_NC; ++p) acc[p] = make_float2(0.f, 0.f);
    for (int m = -D; m <= D; ++m) {
        const float2 xv = __ldg(x + m);
        const float *c = s_coef + (m + D) * FARROW_NC;
#pragma unroll
        for (int p = 0; p < FARROW_NC; ++p) acc[p] = __ffma2_rn(xv, make_float2(c[p], c[p]), acc[p]);
    }
    float4 *out = reinterpret_cast<float4 *>(Y) + (int64_t)X * g.y_det_stride + farrow_index((int)j);
#pragma unroll
    for (int p = 0; p < FARROW_NC / 2; ++p)
        out[FARROW_BLOCK * p] = make_float4(acc[2 * p].x, acc[2 * p].y, acc[2 * p + 1].x, acc[2 * p + 1].y);
}

__global__ void __launch_bounds__(NODE_THREADS)
timing_nodes_kernel(const __grid_constant__ PlanGeom g, const SkyConst *__restrict__ skies, double4 *__restrict__ nodes) {
    const int n = blockIdx.x * NODE_THREADS + threadIdx.x, X = blockIdx.y;
    if (n >= g.n_nodes) return;
    const SkyConst &sc = skies[blockIdx.z];
    const double hstep = (double)(1 << g.log_node) * g.dt;
    const double tau0 = (double)(((int64_t)n << g.log_node) - g.k_margin) * g.dt;
    double d0, s0, d1, s1;
    timing_node(g, sc, X, tau0, d0, s0);
    timing_node(g, sc, X, tau0 + hstep, d1, s1);
    const double m0 = s0 * hstep, m1 = s1 * hstep;
    nodes[((int64_t)blockIdx.z * g.n_det + X) * g.n_nodes + n] =
        make_double4(d0, m0, 3.0 * (d1 - d0) - 2.0 * m0 - m1, 2.0 * (d0 - d1) + m0 + m1);
}

// cos, sin of the Greenwich sidereal angle at every SSB grid point (sky-independent, once per plan; fp64 -> fp32):
// the antenna patterns need it at the detector epoch T = tau - Delta, a rotation by the small angle omega_rot Delta.
__global__ void __launch_bounds__(SKY_THREADS)
sidereal_table_kernel(PlanGeom g, float2 *__restrict__ rot) {
    const int64_t k = (int64_t)blockIdx.x * SKY_THREADS + threadIdx.x;
    if (k >= g.n_src) return;
    double s, c;
    sincos(g.gmst0 + g.omega_rot * ((double)(k - g.k_margin) * g.dt), &s, &c);
    rot[k] = make_float2((float)c, (float)s);
}

// The hoisted form of the sky-dependent half: S written once per sky position and re-read by every spin-down template
// (long fdot banks).  With k = N2 k1 + k2 (the four-step index split of the FFT), a block works on a patch of 32
// adjacent k2 x 32 adjacent k1 of one sky position: warp w takes the rows k1 = k1_0 + w + 8 i (i < 4), lane l the
// grid point k2 = k2_0 + l of each, so that every read of the Farrow-filtered series is 32 consecutive samples
// (512 B per coefficient pair); the 1024 results are transposed through shared memory and written in the tile-blocked
// order FFT pass 1 bulk-loads, as runs of 512 B and more (written point by point that order scatters: one 16-byte piece
// per line, 32 lines per warp store).  What depends on (sky position, detector) only -- antenna coefficients, table
// bases -- is loaded once per thread for the first detector pair instead of once per grid point.
// Block order: sky_major != 0 lets the sky position vary fastest, so that the blocks running at the same time cover
// the same patch for all sky positions of the batch and read the same stretches (+- the spread of the delays) of the
// Farrow-filtered series, which then comes from HBM once per batch instead of once per sky position (used when that
// table exceeds what the L2 holds: 221 MB at config-2 size); otherwise the patch index varies fastest.
//   S      : [n_sky][n_fft] float4 = (Re Ya0, Im Ya0, Re Yb0, Im Yb0); natural order S[k], or
//            (blocked != 0) the tile-blocked order FFT pass 1 bulk-loads: S[k2 / W1][k1][k2 % W1]
#define SKY_PTS 4
#define SKY_PATCH 32
#ifndef SKY_PIN_BASES
#define SKY_PIN_BASES 1
#endif
#ifndef SKY_MIN_BLOCKS
#define SKY_MIN_BLOCKS 5          // 48 registers; measured: 4 blocks +3 %, 6 blocks (40 registers, spills) +4 %
#endif
__global__ void __launch_bounds__(SKY_THREADS, SKY_MIN_BLOCKS)
sky_resample_kernel(const __grid_constant__ PlanGeom g, const SkyConst *__restrict__ skies, const double4 *__restrict__ nodes,
                    const float2 *__restrict__ rot, const float2 *__restrict__ Y, const float *__restrict__ wslot,
                    float4 *__restrict__ S, int blocked, uint32_t det_mask, int n_sky, int n_patches, int sky_major) {
    static_assert(SKY_THREADS == 8 * SKY_PATCH && SKY_PTS * 8 == SKY_PATCH, "8 warps x 4 rows = 32 rows of 32 points");
    __shared__ float4 tile[SKY_PATCH * (SKY_PATCH + 16)];                 // row pitch 32 + W1 elements (W1 <= 16): conflict-free both ways
    const int sky = sky_major ? (int)(blockIdx.x % (unsigned)n_sky) : (int)(blockIdx.x / (unsigned)n_patches);
    const int pb = sky_major ? (int)(blockIdx.x / (unsigned)n_sky) : (int)(blockIdx.x % (unsigned)n_patches);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int k2_0 = (pb & ((1 << (g.log_n2 - 5)) - 1)) << 5, k1_0 = (pb >> (g.log_n2 - 5)) << 5;
    const SkyConst &sc = skies[sky];
    const double4 *nd = nodes + (int64_t)sky * g.n_det * g.n_nodes;
    float4 *Ss = S + (int64_t)sky * g.n_fft;
    // through shared memory when the blocked order breaks a row of 32 adjacent k2 into pieces (W1 < 32 columns per pass-1 tile)
    const bool transpose = blocked && g.log_w1 < 5;
    const int pitch = SKY_PATCH + (1 << min(g.log_w1, 4));
    // the first detector pair (all there is in the two-detector configurations) hoisted out of the loop over grid points
    SkyDetConst d0 = sky_det_const(g, sc, nd, Y, wslot, 0, det_mask);
    SkyDetConst d1 = sky_det_const(g, sc, nd, Y, wslot, 1, det_mask);
#if SKY_PIN_BASES
    // the table bases are uniform values that ptxas would otherwise recompute in every iteration of the loop below
    // (~40 uniform-datapath instructions per grid point): an opaque move pins them in registers
    asm volatile("" : "+l"(d0.nodes), "+l"(d0.y), "+l"(d0.w), "+l"(d1.nodes), "+l"(d1.y), "+l"(d1.w));
#endif
#pragma unroll 1
    for (int i = 0; i < SKY_PTS; ++i) {
        const int k1 = k1_0 + warp + 8 * i, k2 = k2_0 + lane;
        const int k = (k1 << g.log_n2) + k2;                              // n_src <= n_fft <= 2^24
        float2 ya = make_float2(0.f, 0.f), yb = make_float2(0.f, 0.f);
        if (k < g.n_src) {
            const SkyPointCommon c = sky_point_common(g, rot, k);
            {
                const SkyDetPoint o0 = sky_det_point(g, d0, c), o1 = sky_det_point(g, d1, c);
                float4 c0[FARROW_NC / 2], c1[FARROW_NC / 2];
                sky_det_load(o0, c0);
                sky_det_load(o1, c1);
                sky_det_finish(o0, c0, ya, yb);
                sky_det_finish(o1, c1, ya, yb);
            }
            for (int X0 = 2; X0 < g.n_det; X0 += 2) {
                const SkyDetPoint o0 = sky_det_point(g, sky_det_const(g, sc, nd, Y, wslot, X0, det_mask), c);
                const SkyDetPoint o1 = sky_det_point(g, sky_det_const(g, sc, nd, Y, wslot, X0 + 1, det_mask), c);
                float4 c0[FARROW_NC / 2], c1[FARROW_NC / 2];
                sky_det_load(o0, c0);
                sky_det_load(o1, c1);
                sky_det_finish(o0, c0, ya, yb);
                sky_det_finish(o1, c1, ya, yb);
            }
        }
        // blocked mode feeds the FFT kernels, whose element format is (Re Ya, Re Yb, Im Ya, Im Yb)
        const float4 v = blocked ? make_float4(ya.x, yb.x, ya.y, yb.y) : make_float4(ya.x, ya.y, yb.x, yb.y);
        if (transpose) tile[(warp + 8 * i) * pitch + lane] = v;
        else if (k < g.n_src) {                                           // rows of 32 adjacent k2 are contiguous in S
            const int off = blocked ? ((k2 >> g.log_w1) << (g.log_n1 + g.log_w1)) + (k1 << g.log_w1) + (k2 & ((1 << g.log_w1) - 1)) : k;
            Ss[off] = v;
        }
    }
    if (!transpose) return;
    __syncthreads();
    // element e of the patch in output order: run e / (32 W1) = block of W1 columns, then k1, then the column within the block
    const int lw = g.log_w1;
#pragma unroll 1
    for (int i = 0; i < SKY_PTS; ++i) {
        const int e = ((warp + 8 * i) << 5) + lane;
        const int run = e >> (5 + lw), within = e & ((32 << lw) - 1);
        const int k1l = within >> lw, k2l = (run << lw) + (within & ((1 << lw) - 1));
        const int k1 = k1_0 + k1l, k2 = k2_0 + k2l;
        // rows beyond n_src are zero padding: written as zeros (the patch covers whole rows k1 < N1 only)
        if (k1 < (1 << g.log_n1))
            Ss[((k2 >> lw) << (g.log_n1 + lw)) + (k1 << lw) + (k2 & ((1 << lw) - 1))] = tile[k1l * pitch + k2l];
    }
}

// A, B, C (eq. 8, S11): sums of w a^2, w b^2, w a b over the valid detector-frame
// samples.  a(t) and b(t) are linear in the basis u(t) = (1, cos 2th, sin 2th, cos th, sin th) of the
// site's sidereal angle th(t) = gmst0 + omega_rot t' + lon_X, with coefficients that depend on the sky
// position only, so  sum_j w_j a_j^2 = alpha^T M_X alpha  with the sky-independent moment matrix
// M_X = sum_j w_j u_j u_j^T.  This kernel accumulates the 15 distinct entries of M_X once per plan (fp64);
// per sky position A, B, C, D then cost O(25 n_det) flops on the host (fstat_capi.cu).
// grid = (nblk, n_det); each block writes its 15 partial sums; the host adds them in a fixed order.
#define MOM_THREADS 256
#define MOM_PER_THREAD 8
#define MOM_TERMS 15
__global__ void __launch_bounds__(MOM_THREADS)
antenna_moments_kernel(PlanGeom g, const float *__restrict__ wslot, const double *__restrict__ lon,
                       double *__restrict__ partial /* [n_det][gridDim.x][15] */) {
    const int X = blockIdx.y;
    double acc[MOM_TERMS];
#pragma unroll
    for (int q = 0; q < MOM_TERMS; ++q) acc[q] = 0.0;
    const int64_t base = (int64_t)blockIdx.x * (MOM_THREADS * MOM_PER_THREAD);
#pragma unroll 1
    for (int i = 0; i < MOM_PER_THREAD; ++i) {
        const int64_t j = base + i * MOM_THREADS + threadIdx.x;
        if (j >= g.n_samples) break;
        const double tp = (double)j * g.dt;
        const int slot = min((int)floor(tp * g.inv_t_sft), g.n_slots - 1);
        const double w = (double)wslot[X * g.n_slots + slot];
        if (w == 0.0) continue;
        double s1, c1;
        sincos(g.gmst0 + g.omega_rot * tp + lon[X], &s1, &c1);
        const double u[5] = {1.0, c1 * c1 - s1 * s1, 2.0 * s1 * c1, c1, s1};
        int q = 0;
#pragma unroll
        for (int r = 0; r < 5; ++r)
#pragma unroll
            for (int c = r; c < 5; ++c) acc[q++] += w * u[r] * u[c];
    }
    __shared__ double red[MOM_TERMS][MOM_THREADS / 32];
#pragma unroll
    for (int q = 0; q < MOM_TERMS; ++q) {
        double v = acc[q];
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
        if ((threadIdx.x & 31) == 0) red[q][threadIdx.x >> 5] = v;
    }
    __syncthreads();
    if (threadIdx.x < MOM_TERMS) {
        double t = 0.0;
        for (int wv = 0; wv < MOM_THREADS / 32; ++wv) t += red[threadIdx.x][wv];
        partial[((int64_t)X * gridDim.x + blockIdx.x) * MOM_TERMS + threadIdx.x] = t;
    }
}
