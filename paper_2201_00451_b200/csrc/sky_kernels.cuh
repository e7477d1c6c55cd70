// Sky-dependent half of the path (H1-H5 of DESIGN.md): SSB timing, antenna patterns,
// windowed-sinc resampling, SSB heterodyne correction, detector sum.
// PAPER.md:81-84 (steps iii-vi), eq. 3.
#pragma once
#include "fstat_common.cuh"

// Window table, passed by value as a kernel parameter (lands in the constant bank; no
// module-level state shared between plans).
struct WinTable {
    float c[2 * FSTAT_MAX_DTERMS + 1];   // cos(pi m /(D+1/2)), m = -D..D
    float s[2 * FSTAT_MAX_DTERMS + 1];   // sin(pi m /(D+1/2))
};

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

// Returns Delta = tau - T and cos/sin of the sidereal angle at T.
__device__ __forceinline__ double ssb_invert(const PlanGeom &g, const SkyConst &sc, int X, const SsbBase &b,
                                             double &cth, double &sth) {
    double delta = sc.Pc * b.co + sc.Ps * b.so + sc.Qc[X] * b.cr + sc.Qs[X] * b.sr + sc.Q0[X];
    cth = b.cr; sth = b.sr;
#pragma unroll
    for (int it = 0; it < 3; ++it) {      // contraction 1e-4 per step: 5e-2 s -> 5e-6 -> 5e-10 -> 5e-14
        double se, ce, sr, cr;
        small_sincos(g.omega_orb * delta, se, ce);
        small_sincos(g.omega_rot * delta, sr, cr);
        const double co = b.co * ce + b.so * se, so = b.so * ce - b.co * se;     // angle - eps
        cth = b.cr * cr + b.sr * sr; sth = b.sr * cr - b.cr * sr;
        delta = sc.Pc * co + sc.Ps * so + sc.Qc[X] * cth + sc.Qs[X] * sth + sc.Q0[X];
    }
    return delta;
}

// H2: a(t), b(t) from cos/sin of the sidereal angle (fp32).
__device__ __forceinline__ void antenna_ab(const SkyConst &sc, int X, float cth, float sth, float &a, float &b) {
    const float ch = sc.cal[X] * cth + sc.sal[X] * sth;
    const float sh = sc.sal[X] * cth - sc.cal[X] * sth;
    const float c2 = 2.f * ch * ch - 1.f, s2 = 2.f * sh * ch;
    a = sc.ac[X][0] + sc.ac[X][1] * c2 + sc.ac[X][2] * s2 + sc.ac[X][3] * ch + sc.ac[X][4] * sh;
    b = sc.bc[X][0] * c2 + sc.bc[X][1] * s2 + sc.bc[X][2] * ch + sc.bc[X][3] * sh;
}

// H1-H5 for one SSB grid point per thread.  grid = (ceil(n_src/256), n_sky).
//   series : [n_det][series_stride] float2, data starts at +SERIES_PAD (zeros around it)
//   wslot  : [n_det][n_slots] float, 0 in gaps
//   S      : [n_sky][n_fft] float4 = (Re Ya0, Im Ya0, Re Yb0, Im Yb0); natural order S[k], or
//            (blocked != 0) the tile-blocked order FFT pass 1 bulk-loads: with k = N2*k1 + k2,
//            S[k2 / W1][k1][k2 % W1]
__global__ void __launch_bounds__(256)
sky_resample_kernel(const __grid_constant__ PlanGeom g, const __grid_constant__ WinTable win,
                    const SkyConst *__restrict__ skies, const float2 *__restrict__ series,
                    const float *__restrict__ wslot, float4 *__restrict__ S, int blocked) {
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.n_src) return;
    const SkyConst &sc = skies[blockIdx.y];
    const int64_t krel = k - g.k_margin;
    const double tau = (double)krel * g.dt;
    const SsbBase base = ssb_base(g, tau);

    float yar = 0.f, yai = 0.f, ybr = 0.f, ybi = 0.f;
    const int D = g.dterms;
    const float inv_dh = 1.0f / ((float)D + 0.5f);
    // band placement: output bin q must land on FFT index q -> multiply by exp(-2 pi i s k / n_fft)
    const uint64_t tshift = ((uint64_t)g.shift_mod * (uint64_t)k) & (uint64_t)(g.n_fft - 1);
    const double shift_cyc = (double)tshift / (double)g.n_fft;

    for (int X = 0; X < g.n_det; ++X) {
        double cth, sth;
        const double delta = ssb_invert(g, sc, X, base, cth, sth);
        const double T = tau - delta;                       // detector epoch - t_start
        if (!(T >= 0.0 && T < g.span)) continue;            // step 3: outside the data
        const int slot = min((int)floor(T * g.inv_t_sft), g.n_slots - 1);
        const float w = wslot[X * g.n_slots + slot];
        if (w == 0.f) continue;                             // gap
        // fractional sample index u = krel - Delta/dt = j0 + d,  d in [-1/2, 1/2)
        const double v = -delta * g.inv_dt;
        const double vr = floor(v + 0.5);
        const float d = (float)(v - vr);
        const int64_t j0 = krel + (int64_t)vr;
        // kernel coefficients: sinc(d-m) W(d-m) = (-1)^m sin(pi d)/(pi (d-m)) * [0.54 + 0.46 cos(pi (d-m)/(D+1/2))]
        const float spd = sinpif(d) * 0.318309886183790672f;
        float sw, cw;
        sincospif(d * inv_dh, &sw, &cw);
        const float2 *x = series + (int64_t)X * g.series_stride + SERIES_PAD + j0;
        float zr = 0.f, zi = 0.f;
        for (int m = -D; m <= D; ++m) {
            const float2 xv = __ldg(x + m);
            const float wnd = 0.54f + 0.46f * (cw * win.c[m + D] + sw * win.s[m + D]);
            float sinc;
            if (m == 0) sinc = (fabsf(d) < 1e-4f) ? 1.0f - 1.6449340668f * d * d : spd / d;
            else sinc = ((m & 1) ? -spd : spd) / (d - (float)m);
            const float c = sinc * wnd;
            zr = fmaf(xv.x, c, zr); zi = fmaf(xv.y, c, zi);
        }
        // step (iii): SSB heterodyne correction exp(-2 pi i f_het Delta), plus the band shift
        double cyc = g.f_het * delta;
        cyc = (cyc - floor(cyc)) + shift_cyc;
        float sp, cp;
        sincospif(-2.0f * (float)(cyc - floor(cyc)), &sp, &cp);
        const float er = zr * cp - zi * sp, ei = zr * sp + zi * cp;
        float a, b;
        antenna_ab(sc, X, (float)cth, (float)sth, a, b);
        yar = fmaf(w * a, er, yar); yai = fmaf(w * a, ei, yai);
        ybr = fmaf(w * b, er, ybr); ybi = fmaf(w * b, ei, ybi);
    }
    int64_t off = k;
    if (blocked) {
        const int64_t k1 = k >> g.log_n2, k2 = k & (((int64_t)1 << g.log_n2) - 1);
        off = ((k2 >> g.log_w1) << (g.log_n1 + g.log_w1)) + (k1 << g.log_w1) + (k2 & ((1 << g.log_w1) - 1));
    }
    // blocked mode feeds the FFT kernels, whose element format is (Re Ya, Re Yb, Im Ya, Im Yb)
    S[(int64_t)blockIdx.y * g.n_fft + off] = blocked ? make_float4(yar, ybr, yai, ybi) : make_float4(yar, yai, ybr, ybi);
}

// A, B, C (eq. 8): sums of w a^2, w b^2, w a b over the valid detector-frame samples.
// grid = (nblk, n_sky); each block writes one double3 partial; finalize reduces them in
// a fixed order (deterministic).
#define ABC_THREADS 256
#define ABC_PER_THREAD 8
__global__ void __launch_bounds__(ABC_THREADS)
sky_abc_partial_kernel(PlanGeom g, const SkyConst *__restrict__ skies, const float *__restrict__ wslot,
                       double *__restrict__ partial /* [n_sky][gridDim.x][3] */) {
    const SkyConst &sc = skies[blockIdx.y];
    const int64_t total = g.n_samples * g.n_det;
    const double inv2pi = 0.15915494309189533577;
    float sA = 0.f, sB = 0.f, sC = 0.f;
    const int64_t base = (int64_t)blockIdx.x * (ABC_THREADS * ABC_PER_THREAD);
#pragma unroll 1
    for (int i = 0; i < ABC_PER_THREAD; ++i) {
        const int64_t idx = base + i * ABC_THREADS + threadIdx.x;
        if (idx >= total) break;
        const int X = (int)(idx / g.n_samples);
        const int64_t j = idx - (int64_t)X * g.n_samples;
        const double tp = (double)j * g.dt;
        const int slot = min((int)floor(tp * g.inv_t_sft), g.n_slots - 1);
        const float w = wslot[X * g.n_slots + slot];
        if (w == 0.f) continue;
        double rev = (g.gmst0 + g.omega_rot * tp) * inv2pi;
        rev -= floor(rev);
        float sth, cth;
        sincospif(2.0f * (float)rev, &sth, &cth);
        float a, b;
        antenna_ab(sc, X, cth, sth, a, b);
        sA = fmaf(w * a, a, sA); sB = fmaf(w * b, b, sB); sC = fmaf(w * a, b, sC);
    }
    __shared__ double red[3][ABC_THREADS / 32];
    double dA = sA, dB = sB, dC = sC;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        dA += __shfl_down_sync(0xffffffffu, dA, o);
        dB += __shfl_down_sync(0xffffffffu, dB, o);
        dC += __shfl_down_sync(0xffffffffu, dC, o);
    }
    if ((threadIdx.x & 31) == 0) { red[0][threadIdx.x >> 5] = dA; red[1][threadIdx.x >> 5] = dB; red[2][threadIdx.x >> 5] = dC; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double tA = 0, tB = 0, tC = 0;
        for (int wv = 0; wv < ABC_THREADS / 32; ++wv) { tA += red[0][wv]; tB += red[1][wv]; tC += red[2][wv]; }
        double *p = partial + ((int64_t)blockIdx.y * gridDim.x + blockIdx.x) * 3;
        p[0] = tA; p[1] = tB; p[2] = tC;
    }
}

// One block per sky: fixed-order tree reduction of the partials, then the eq. 8 coefficients.
__global__ void __launch_bounds__(256)
sky_abc_finalize_kernel(const double *__restrict__ partial, int nblk, SkyABCD *__restrict__ out, int *__restrict__ err_flag) {
    __shared__ double red[3][256];
    const double *p = partial + (int64_t)blockIdx.x * nblk * 3;
    double tA = 0, tB = 0, tC = 0;
    for (int i = threadIdx.x; i < nblk; i += 256) { tA += p[i * 3]; tB += p[i * 3 + 1]; tC += p[i * 3 + 2]; }
    red[0][threadIdx.x] = tA; red[1][threadIdx.x] = tB; red[2][threadIdx.x] = tC;
    __syncthreads();
    for (int s = 128; s > 0; s >>= 1) {
        if (threadIdx.x < s) {
            red[0][threadIdx.x] += red[0][threadIdx.x + s];
            red[1][threadIdx.x] += red[1][threadIdx.x + s];
            red[2][threadIdx.x] += red[2][threadIdx.x + s];
        }
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        SkyABCD r;
        r.A = red[0][0]; r.B = red[1][0]; r.C = red[2][0];
        r.D = r.A * r.B - r.C * r.C;
        r.bad = !(r.D > 0.0);
        if (r.bad) {
            r.b_over_d = r.a_over_d = r.two_c_over_d = __int_as_float(0x7fc00000);
            atomicExch(err_flag, 1);
        } else {
            r.b_over_d = (float)(r.B / r.D); r.a_over_d = (float)(r.A / r.D); r.two_c_over_d = (float)(2.0 * r.C / r.D);
        }
        out[blockIdx.x] = r;
    }
}
