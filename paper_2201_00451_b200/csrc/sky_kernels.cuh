// Sky-dependent half of the path (H1-H5 of DESIGN.md): SSB timing, antenna patterns,
// windowed-sinc resampling, SSB heterodyne correction, detector sum.
// PAPER.md:81-84 (steps iii-vi), eq. 3.
#pragma once
#include "fstat_common.cuh"

// sin, cos of a small angle |e| <~ 0.1 rad in double by Taylor series (error < 1e-18 for
// |e| < 0.05: omega_rot * Delta_max = 0.036, omega_orb * Delta_max = 1e-4).
__device__ __forceinline__ void small_sincos(double e, double &s, double &c) {
    const double e2 = e * e;
    s = e * (1.0 + e2 * (-1.0 / 6 + e2 * (1.0 / 120 + e2 * (-1.0 / 5040 + e2 * (1.0 / 362880)))));
    c = 1.0 + e2 * (-0.5 + e2 * (1.0 / 24 + e2 * (-1.0 / 720 + e2 * (1.0 / 40320 + e2 * (-1.0 / 3628800)))));
}

// H1: invert tau = T + Delta_X(T) for the detector epoch T of SSB grid time tau (step iv).
// The trigonometric base values at tau are shared by all detectors and all iterations;
// the epoch shift T - tau = -Delta only rotates them by the small angles omega*Delta.
struct SsbBase {
    double co, so;   // cos, sin of orbital phase at tau
    double cr, sr;   // cos, sin of Greenwich sidereal angle at tau
};

__device__ __forceinline__ SsbBase ssb_base(const PlanGeom &g, double tau) {
    SsbBase b;
    sincos(g.phi_orb0 + g.omega_orb * tau, &b.so, &b.co);
    sincos(g.gmst0 + g.omega_rot * tau, &b.sr, &b.cr);
    return b;
}

// H2: a(t), b(t) from cos/sin of the sidereal angle (fp32).
__device__ __forceinline__ void antenna_ab(const SkyConst &sc, int X, float cth, float sth, float &a, float &b) {
    const float ch = sc.cal[X] * cth + sc.sal[X] * sth;
    const float sh = sc.sal[X] * cth - sc.cal[X] * sth;
    const float c2 = 2.f * ch * ch - 1.f, s2 = 2.f * sh * ch;
    a = sc.ac[X][0] + sc.ac[X][1] * c2 + sc.ac[X][2] * s2 + sc.ac[X][3] * ch + sc.ac[X][4] * sh;
    b = sc.bc[X][0] * c2 + sc.bc[X][1] * s2 + sc.bc[X][2] * ch + sc.bc[X][3] * sh;
}

// Orbital-angle version of small_sincos: |e| = omega_orb * 500 s ~ 1e-4 rad for the Earth (error
// < 1e-30); at the 0.05 rad fstat_setup admits the error is 1.5e-13 (7e-11 s of delay).
__device__ __forceinline__ void tiny_sincos(double e, double &s, double &c) {
    const double e2 = e * e;
    s = e * (1.0 + e2 * (-1.0 / 6 + e2 * (1.0 / 120)));
    c = 1.0 + e2 * (-0.5 + e2 * (1.0 / 24 + e2 * (-1.0 / 720)));
}

// H1 by Newton steps on F(T) = T + Delta_X(T) - tau, from T0 = tau - Delta_X(tau), where
// |T0 - T*| <= |Delta'| |Delta| ~ 1e-4 * 500 s = 0.05 s.  One update leaves
// |F''| (T0 - T*)^2 / 2 ~ 1.3e-10 s^-1 * 2.5e-3 s^2 / 2 = 2e-13 s for the Earth (needed: <~ 3e-8 s,
// SURVEY 7); fstat_setup derives the step count g.n_newton from the ephemeris the same way.
// Returns Delta = tau - T and cos/sin of the sidereal angle at the last evaluation point
// (within 1e-5 s of T: the antenna patterns do not see the difference).
__device__ __forceinline__ double ssb_invert_newton(const PlanGeom &g, const SkyConst &sc, int X, const SsbBase &b,
                                                    double &cth, double &sth) {
    double delta = sc.Pc * b.co + sc.Ps * b.so + sc.Qc[X] * b.cr + sc.Qs[X] * b.sr + sc.Q0[X];
    cth = b.cr; sth = b.sr;
    for (int it = 0; it < g.n_newton; ++it) {
        double se, ce, sr, cr;
        tiny_sincos(g.omega_orb * delta, se, ce);
        small_sincos(g.omega_rot * delta, sr, cr);
        const double co = b.co * ce + b.so * se, so = b.so * ce - b.co * se;      // angles at T_n = tau - delta
        cth = b.cr * cr + b.sr * sr; sth = b.sr * cr - b.cr * sr;
        const double f = (sc.Pc * co + sc.Ps * so + sc.Qc[X] * cth + sc.Qs[X] * sth + sc.Q0[X]) - delta;   // F(T_n)
        const double dp = g.omega_orb * (sc.Ps * co - sc.Pc * so) + g.omega_rot * (sc.Qs[X] * cth - sc.Qc[X] * sth);   // Delta'(T_n)
        delta += f * (1.0 - dp * (1.0 - dp));                                     // 1/(1+dp) to O(dp^3)
    }
    return delta;
}

#define SKY_THREADS 256
#define FARROW_NC 10          // polynomial coefficients per tap (degree 9: 8e-8 max error for Dterms >= 8, 3e-7 for Dterms 1)

// H3 in Farrow form.  The interpolation weight of tap m, c_m(d) = sinc(d-m) W(d-m) for d in [-1/2, 1/2)
// (S6), is an entire function of d; fstat_setup expands it as c_m(d) = sum_p a[m][p] d^p
// (Chebyshev interpolation of degree 9, converted to powers of d, fp64 -> fp32).  Then
//     z(j0 + d) = sum_m x[j0+m] c_m(d) = sum_p d^p Y_p[j0],   Y_p[j] = sum_m a[m][p] x[j+m]:
// the 2D+1 taps are folded, once per plan and independent of the sky position, into FARROW_NC filtered
// copies of the series (this kernel); per SSB grid point the resampler then reads FARROW_NC complex
// numbers (five coalesced float4 loads) and runs one Horner recurrence instead of evaluating 2D+1 weights.
//   series : [n_det][series_stride] float2 (data at +SERIES_PAD, zeros around it)
//   coef   : [2D+1][FARROW_NC] float, row m+D
//   Y      : [n_det][FARROW_NC/2][N+1] float4 = (Re Y_2c, Im Y_2c, Re Y_2c+1, Im Y_2c+1)
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
    // chunk-major: chunk c = (Y_2c, Y_2c+1) of all j contiguous, so that consecutive grid points read consecutive float4
    float4 *out = reinterpret_cast<float4 *>(Y) + (int64_t)X * (FARROW_NC / 2) * (g.n_samples + 1) + j;
#pragma unroll
    for (int p = 0; p < FARROW_NC / 2; ++p)
        out[(int64_t)p * (g.n_samples + 1)] = make_float4(acc[2 * p].x, acc[2 * p].y, acc[2 * p + 1].x, acc[2 * p + 1].y);
}

// ---- H1 on a coarse node grid --------------------------------------------------------------------------------
// The delay Delta(tau) = tau - T(tau) is smooth (sidereal rotation: 21 ms amplitude, one-day period; orbit: 499 s, one
// year), so the exact Newton inversion runs only at nodes M = 2^log_node grid points apart (M dt <= 256 s) and every
// grid point evaluates the cubic Hermite interpolant through the node values and slopes
//     Delta(tau_n + theta M dt) = d0 + theta (m + theta (c2 + theta c3)),   theta in [0, 1),
// in fp64.  Interpolation error (4th derivative) h^4 / 384 < 1e-10 s (measured 6e-11 s at h = 256 s; needed: <~ 3e-8 s,
// SURVEY 7).
//   nodes : [n_sky][n_det][n_nodes] double4 = (d0, m, c2, c3) in seconds
// grid = (ceil(n_nodes / 128), n_det, n_sky), 128 threads.
#define NODE_THREADS 128
__device__ __forceinline__ void timing_node(const PlanGeom &g, const SkyConst &sc, int X, double tau, double &delta, double &slope) {
    const SsbBase b = ssb_base(g, tau);
    double cth, sth;
    delta = ssb_invert_newton(g, sc, X, b, cth, sth);
    // d Delta / d tau = Delta_X'(T) / (1 + Delta_X'(T)) at the converged epoch T = tau - delta
    double se, ce, sr, cr;
    tiny_sincos(g.omega_orb * delta, se, ce);
    small_sincos(g.omega_rot * delta, sr, cr);
    const double co = b.co * ce + b.so * se, so = b.so * ce - b.co * se;
    cth = b.cr * cr + b.sr * sr; sth = b.sr * cr - b.cr * sr;
    const double dp = g.omega_orb * (sc.Ps * co - sc.Pc * so) + g.omega_rot * (sc.Qs[X] * cth - sc.Qc[X] * sth);
    slope = dp / (1.0 + dp);
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

// H1-H5 for SSB grid point k: adds the detectors' contributions to (ya, yb) = (Fa(t), Fb(t)) before the spin-down factor.
//   nodes  : [n_det][n_nodes] double4 of this sky position (timing_nodes_kernel)
//   rot    : [n_src] float2 from sidereal_table_kernel
//   Y      : [n_det][FARROW_NC/2][N+1] float4, the Farrow-filtered series
//   wslot  : [n_det][n_slots] float, 0 in gaps
//   det_mask : bit X set = detector X contributes
// Detectors are taken two at a time: the timing of both first, then the 2 x 80 bytes of Farrow coefficients are requested
// together (these L2 reads are what the thread waits for), then the two Horner recurrences, phase factors and
// antenna weights.  fp64 only for Delta, the fractional sample index and the heterodyne phase.
__device__ __forceinline__ void sky_point(const PlanGeom &g, const SkyConst &sc, const double4 *__restrict__ nodes,
                                          const float2 *__restrict__ rot, const float2 *__restrict__ Y, const float *__restrict__ wslot,
                                          int k, uint32_t det_mask, float2 &ya, float2 &yb) {
    const int krel = k - (int)g.k_margin;
    const double tau = (double)krel * g.dt;
    const int nn = k >> g.log_node;
    const double theta = (double)(k & ((1 << g.log_node) - 1)) * g.inv_node;
    const float2 cs = __ldg(rot + k);
    // band placement: output bin q must land on FFT index q -> multiply by exp(-2 pi i s k / n_fft);
    // (shift * k mod n_fft) / n_fft is exact in fp32 (n_fft <= 2^24 is a power of two, uint32 wrap-around is mod 2^32);
    // + the residual fraction of a bin when f_het is off the bin grid: |value| <= 1/2, k < 2^24 exact in fp32 (error 6e-8 cycles)
    const uint32_t tshift = (g.shift_mod * (uint32_t)k) & (uint32_t)(g.n_fft - 1);
    const float shift_cyc = fmaf((float)k, g.shift_frac_per_k, (float)tshift * (1.0f / (float)g.n_fft));
    const int n_rows = (int)g.n_samples + 1;

    for (int X0 = 0; X0 < g.n_det; X0 += 2) {
        float w[2], d[2], fc[2], ca[2], cb[2];
        const float4 *y[2];
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            const int X = min(X0 + u, g.n_det - 1);
            const double2 *np = reinterpret_cast<const double2 *>(nodes + (int64_t)X * g.n_nodes + nn);
            const double2 n0 = __ldg(np), n1 = __ldg(np + 1);
            const double delta = fma(theta, fma(theta, fma(theta, n1.y, n1.x), n0.y), n0.x);
            const double T = tau - delta;                       // detector epoch - t_start
            w[u] = 0.f;
            // step 3: inside the data and not in a gap (det_mask: the detectors that take part -- all of them, or one
            // for the single-detector statistic)
            if (X0 + u < g.n_det && ((det_mask >> X) & 1u) && T >= 0.0 && T < g.span) {
                const int slot = min((int)(T * g.inv_t_sft), g.n_slots - 1);
                w[u] = wslot[X * g.n_slots + slot];
            }
            // fractional sample index u = krel - Delta/dt = j0 + d,  d in [-1/2, 1/2)
            const double v = -delta * g.inv_dt;
            const double vr = floor(v + 0.5);
            d[u] = (float)(v - vr);
            const int j0 = min(max(krel + (int)vr, 0), n_rows - 1);   // in [0, N] whenever w != 0
            y[u] = reinterpret_cast<const float4 *>(Y) + (int64_t)X * (FARROW_NC / 2) * n_rows + j0;
            // step (iii): SSB heterodyne correction exp(-2 pi i f_het Delta), plus the band shift
            // (phase reduced mod 1 in fp64, then fp32)
            const double cyc = g.f_het * delta;
            fc[u] = (float)(cyc - floor(cyc)) + shift_cyc;
            // sidereal angle at T: rotate the table value by e = omega_rot Delta (|e| < 0.05: Taylor to 1e-9)
            const float e = (float)(g.omega_rot * delta), e2 = e * e;
            const float se = e * fmaf(e2, fmaf(e2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
            const float ce = fmaf(e2, fmaf(e2, 1.0f / 24.0f, -0.5f), 1.0f);
            antenna_ab(sc, X, cs.x * ce + cs.y * se, cs.y * ce - cs.x * se, ca[u], cb[u]);
        }
        float4 c[2][FARROW_NC / 2];
#pragma unroll
        for (int u = 0; u < 2; ++u)
#pragma unroll
            for (int p = 0; p < FARROW_NC / 2; ++p) c[u][p] = __ldg(y[u] + (int64_t)p * n_rows);
#pragma unroll
        for (int u = 0; u < 2; ++u) {
            // z = sum_p d^p Y_p[j0] (Horner, packed re/im)
            const float2 dd = make_float2(d[u], d[u]);
            float2 z = make_float2(c[u][FARROW_NC / 2 - 1].z, c[u][FARROW_NC / 2 - 1].w);
#pragma unroll
            for (int p = FARROW_NC / 2 - 1; p >= 0; --p) {
                if (p < FARROW_NC / 2 - 1) z = __ffma2_rn(z, dd, make_float2(c[u][p].z, c[u][p].w));
                z = __ffma2_rn(z, dd, make_float2(c[u][p].x, c[u][p].y));
            }
            float f = fc[u] - rintf(fc[u]), sp, cp;             // |arg| <= pi, where sin/cos.approx are good to 5e-7 abs
            __sincosf(-6.283185307179586f * f, &sp, &cp);
            const float er = z.x * cp - z.y * sp, ei = z.x * sp + z.y * cp;
            const float wa = w[u] * ca[u], wb = w[u] * cb[u];
            ya.x = fmaf(wa, er, ya.x); ya.y = fmaf(wa, ei, ya.y);
            yb.x = fmaf(wb, er, yb.x); yb.y = fmaf(wb, ei, yb.y);
        }
    }
}

// The hoisted form of the sky-dependent half: one SSB grid point per thread, S written once per sky position and
// re-read by every spin-down template (long fdot banks).  grid = (ceil(n_src/256), n_sky).
//   S      : [n_sky][n_fft] float4 = (Re Ya0, Im Ya0, Re Yb0, Im Yb0); natural order S[k], or
//            (blocked != 0) the tile-blocked order FFT pass 1 bulk-loads: with k = N2*k1 + k2,
//            S[k2 / W1][k1][k2 % W1]
__global__ void __launch_bounds__(SKY_THREADS)
sky_resample_kernel(const __grid_constant__ PlanGeom g, const SkyConst *__restrict__ skies, const double4 *__restrict__ nodes,
                    const float2 *__restrict__ rot, const float2 *__restrict__ Y, const float *__restrict__ wslot,
                    float4 *__restrict__ S, int blocked, uint32_t det_mask) {
    const int k = blockIdx.x * SKY_THREADS + threadIdx.x;          // n_src <= n_fft <= 2^24
    if (k >= g.n_src) return;
    float2 ya = make_float2(0.f, 0.f), yb = make_float2(0.f, 0.f);
    sky_point(g, skies[blockIdx.y], nodes + (int64_t)blockIdx.y * g.n_det * g.n_nodes, rot, Y, wslot, k, det_mask, ya, yb);
    int off = k;
    if (blocked) {
        const int k1 = k >> g.log_n2, k2 = k & ((1 << g.log_n2) - 1);
        off = ((k2 >> g.log_w1) << (g.log_n1 + g.log_w1)) + (k1 << g.log_w1) + (k2 & ((1 << g.log_w1) - 1));
    }
    // blocked mode feeds the FFT kernels, whose element format is (Re Ya, Re Yb, Im Ya, Im Yb)
    S[(int64_t)blockIdx.y * g.n_fft + off] = blocked ? make_float4(ya.x, yb.x, ya.y, yb.y) : make_float4(ya.x, ya.y, yb.x, yb.y);
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
