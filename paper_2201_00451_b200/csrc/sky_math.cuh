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
// polynomial coefficients per tap weight.  Degree 7: the folded taps differ from the exact windowed-sinc weights by 2e-6
// (root sum of squares over the taps; 7e-6 if all errors add up) for Dterms >= 8 and 2e-5 for Dterms 1, against a
// tolerance of 1e-3 on 2F; degree 9 (10 coefficients, 80 B per sample and detector) gives 1e-8 and costs 25 % more table
// traffic in the kernel that bounds sky-varying searches.
#ifndef FARROW_NC
#define FARROW_NC 8
#endif

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
// ---- H1-H5 per SSB grid point, in pieces that the two forms of the sky-dependent half arrange differently ----------
// (hoisted kernel: detector pairs outside, grid points inside, so that everything that depends on the sky position and
// the detector only is loaded once per thread; fused kernel: one grid point at a time).
//   nodes  : [n_det][n_nodes] double4 of this sky position (timing_nodes_kernel)
//   rot    : [n_src] float2 from sidereal_table_kernel
//   Y      : [n_det][FARROW_NC/2][N+1] float4, the Farrow-filtered series
//   wslot  : [n_det][n_slots] float, 0 in gaps
// fp64 only for Delta, the fractional sample index and the heterodyne phase.  Roundings to integers are done by
// adding 1.5 * 2^52 (fp64 pipe) or 1.5 * 2^23 (fp32) instead of the conversion instructions of the XU pipe.
#define SKY_MAGIC64 6755399441055744.0
#define SKY_MAGIC32 12582912.0f

// Layout of the Farrow-filtered series of one detector: blocks of FARROW_BLOCK = 32 consecutive samples, within a block
// the FARROW_NC / 2 coefficient pairs one after the other, each as 32 float4 = (Re Y_2c, Im Y_2c, Re Y_2c+1, Im Y_2c+1):
// 32 consecutive samples of one pair are 512 contiguous bytes (coalesced for consecutive grid points), and the pairs of
// one sample sit at compile-time offsets from each other (one address computation per sample instead of one per pair).
#define FARROW_BLOCK 32
__host__ __device__ __forceinline__ int farrow_index(int j) { return ((j >> 5) * (FARROW_BLOCK * (FARROW_NC / 2))) + (j & 31); }

// what a grid point contributes to every detector
struct SkyPointCommon {
    int krel;           // k - K_m
    int nn;             // timing node
    double tau;         // SSB time - t_start
    double theta;       // position between the nodes, [0, 1)
    float2 cs;          // cos, sin of the Greenwich sidereal angle at tau
    float shift_cyc;    // band placement ramp (cycles)
};

__device__ __forceinline__ SkyPointCommon sky_point_common(const PlanGeom &g, const float2 *__restrict__ rot, int k) {
    SkyPointCommon c;
    c.krel = k - (int)g.k_margin;
    c.tau = (double)c.krel * g.dt;
    c.nn = k >> g.log_node;
    c.theta = (double)(k & ((1 << g.log_node) - 1)) * g.inv_node;
    c.cs = __ldg(rot + k);
    // band placement: output bin q must land on FFT index q -> multiply by exp(-2 pi i s k / n_fft);
    // (shift * k mod n_fft) / n_fft is exact in fp32 (n_fft <= 2^24 is a power of two, uint32 wrap-around is mod 2^32);
    // + the residual fraction of a bin when f_het is off the bin grid: |value| <= 1/2, k < 2^24 exact in fp32 (error 6e-8 cycles)
    const uint32_t tshift = (g.shift_mod * (uint32_t)k) & (uint32_t)(g.n_fft - 1);
    c.shift_cyc = (float)tshift * g.inv_n_fft;
    if (g.shift_frac_per_k != 0.f) c.shift_cyc = fmaf((float)k, g.shift_frac_per_k, c.shift_cyc);
    return c;
}

// what depends on (sky position, detector) only
struct SkyDetConst {
    float cal, sal, ac[5], bc[4];
    const double4 *nodes;   // this detector's timing nodes
    const float4 *y;        // this detector's Farrow-filtered series
    const float *w;         // this detector's slot weights
    bool on;                // takes part (exists and selected by det_mask)
};

__device__ __forceinline__ SkyDetConst sky_det_const(const PlanGeom &g, const SkyConst &sc, const double4 *__restrict__ nodes,
                                                     const float2 *__restrict__ Y, const float *__restrict__ wslot, int Xu, uint32_t det_mask) {
    const int X = min(Xu, g.n_det - 1);
    SkyDetConst d;
    d.cal = sc.cal[X]; d.sal = sc.sal[X];
#pragma unroll
    for (int q = 0; q < 5; ++q) d.ac[q] = sc.ac[X][q];
#pragma unroll
    for (int q = 0; q < 4; ++q) d.bc[q] = sc.bc[X][q];
    d.nodes = nodes + (int64_t)X * g.n_nodes;
    d.y = reinterpret_cast<const float4 *>(Y) + (int64_t)X * g.y_det_stride;
    d.w = wslot + (int64_t)X * g.n_slots;
    d.on = Xu < g.n_det && ((det_mask >> X) & 1u);
    return d;
}

// per (grid point, detector), before the Farrow coefficients are needed
struct SkyDetPoint {
    float w, d, fc, ca, cb;
    const float4 *y;        // (Y_0, Y_1) of sample j0; the other coefficient pairs follow 32 float4 apart (farrow_index)
};

__device__ __forceinline__ SkyDetPoint sky_det_point(const PlanGeom &g, const SkyDetConst &dc, const SkyPointCommon &c) {
    SkyDetPoint o;
    const double2 *np = reinterpret_cast<const double2 *>(dc.nodes + c.nn);
    const double2 n0 = __ldg(np), n1 = __ldg(np + 1);
    const double delta = fma(c.theta, fma(c.theta, fma(c.theta, n1.y, n1.x), n0.y), n0.x);
    const double T = c.tau - delta;                       // detector epoch - t_start
    o.w = 0.f;
    // step 3: inside the data and not in a gap (dc.on: the detectors that take part -- all of them, or one for the
    // single-detector statistic)
    if (dc.on && T >= 0.0 && T < g.span) {
        const int slot = min(__double2loint(__dadd_rd(T * g.inv_t_sft, SKY_MAGIC64)), g.n_slots - 1);    // floor
        o.w = dc.w[slot];
    }
    // fractional sample index u = krel - Delta/dt = j0 + d,  j0 = floor(u + 1/2), d in [-1/2, 1/2)
    const double v = -delta * g.inv_dt;
    const double vm = __dadd_rd(v + 0.5, SKY_MAGIC64);
    o.d = (float)(v - (vm - SKY_MAGIC64));
    const int n_rows = (int)g.n_samples + 1;
    const int j0 = min(max(c.krel + __double2loint(vm), 0), n_rows - 1);   // in [0, N] whenever w != 0
    o.y = dc.y + farrow_index(j0);
    // step (iii): SSB heterodyne correction exp(-2 pi i f_het Delta), plus the band shift
    // (phase reduced mod 1 in fp64, then fp32)
    const double cyc = g.f_het * delta;
    o.fc = (float)(cyc - ((cyc + SKY_MAGIC64) - SKY_MAGIC64)) + c.shift_cyc;
    // sidereal angle at T: rotate the table value by e = omega_rot Delta (|e| < 0.05: Taylor to 1e-9)
    const float e = (float)(g.omega_rot * delta), e2 = e * e;
    const float se = e * fmaf(e2, fmaf(e2, 1.0f / 120.0f, -1.0f / 6.0f), 1.0f);
    const float ce = fmaf(e2, fmaf(e2, 1.0f / 24.0f, -0.5f), 1.0f);
    // H2: a(t), b(t) from cos/sin of the sidereal angle (fp32), as antenna_ab
    const float cth = c.cs.x * ce + c.cs.y * se, sth = c.cs.y * ce - c.cs.x * se;
    const float ch = dc.cal * cth + dc.sal * sth;
    const float sh = dc.sal * cth - dc.cal * sth;
    const float c2 = 2.f * ch * ch - 1.f, s2 = 2.f * sh * ch;
    o.ca = dc.ac[0] + dc.ac[1] * c2 + dc.ac[2] * s2 + dc.ac[3] * ch + dc.ac[4] * sh;
    o.cb = dc.bc[0] * c2 + dc.bc[1] * s2 + dc.bc[2] * ch + dc.bc[3] * sh;
    return o;
}

__device__ __forceinline__ void sky_det_load(const SkyDetPoint &o, float4 (&c)[FARROW_NC / 2]) {
#pragma unroll
    for (int p = 0; p < FARROW_NC / 2; ++p) c[p] = __ldg(o.y + FARROW_BLOCK * p);
}

__device__ __forceinline__ void sky_det_finish(const SkyDetPoint &o, const float4 (&c)[FARROW_NC / 2], float2 &ya, float2 &yb) {
    // z = sum_p d^p Y_p[j0] (Horner, packed re/im)
    const float2 dd = make_float2(o.d, o.d);
    float2 z = make_float2(c[FARROW_NC / 2 - 1].z, c[FARROW_NC / 2 - 1].w);
#pragma unroll
    for (int p = FARROW_NC / 2 - 1; p >= 0; --p) {
        if (p < FARROW_NC / 2 - 1) z = __ffma2_rn(z, dd, make_float2(c[p].z, c[p].w));
        z = __ffma2_rn(z, dd, make_float2(c[p].x, c[p].y));
    }
    float f = o.fc - ((o.fc + SKY_MAGIC32) - SKY_MAGIC32), sp, cp;      // |arg| <= pi, where sin/cos.approx are good to 5e-7 abs
    __sincosf(-6.283185307179586f * f, &sp, &cp);
    const float er = z.x * cp - z.y * sp, ei = z.x * sp + z.y * cp;
    const float wa = o.w * o.ca, wb = o.w * o.cb;
    ya.x = fmaf(wa, er, ya.x); ya.y = fmaf(wa, ei, ya.y);
    yb.x = fmaf(wb, er, yb.x); yb.y = fmaf(wb, ei, yb.y);
}

// H1-H5 for SSB grid point k: adds the detectors' contributions to (ya, yb) = (Fa(t), Fb(t)) before the spin-down factor.
// Detectors are taken two at a time: the timing of both first, then the 2 x 80 bytes of Farrow coefficients are requested
// together (these L2 reads are what the thread waits for), then the two Horner recurrences, phase factors and
// antenna weights.
__device__ __forceinline__ void sky_point(const PlanGeom &g, const SkyConst &sc, const double4 *__restrict__ nodes,
                                          const float2 *__restrict__ rot, const float2 *__restrict__ Y, const float *__restrict__ wslot,
                                          int k, uint32_t det_mask, float2 &ya, float2 &yb) {
    const SkyPointCommon c = sky_point_common(g, rot, k);
    for (int X0 = 0; X0 < g.n_det; X0 += 2) {
        SkyDetPoint o[2];
        float4 cf[2][FARROW_NC / 2];
#pragma unroll
        for (int u = 0; u < 2; ++u) o[u] = sky_det_point(g, sky_det_const(g, sc, nodes, Y, wslot, X0 + u, det_mask), c);
#pragma unroll
        for (int u = 0; u < 2; ++u) sky_det_load(o[u], cf[u]);
#pragma unroll
        for (int u = 0; u < 2; ++u) sky_det_finish(o[u], cf[u], ya, yb);
    }
}
