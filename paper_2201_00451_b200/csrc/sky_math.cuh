// Device functions of the sky-dependent half of the path (H1-H5 of DESIGN.md): SSB timing, antenna patterns,
// windowed-sinc resampling (Farrow form), SSB heterodyne correction, detector sum.  Used by the kernels of
// sky_kernels.cuh (hoisted form) and by the fused sky + FFT pass-1 kernel of fft_kernels.cuh.
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

