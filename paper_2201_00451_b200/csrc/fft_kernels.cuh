// Batched four-step Stockham FFT of the pair (Fa(t), Fb(t)) with the spin-down prologue
// and the 2F epilogue fused in (H4b, H6, H7 of DESIGN.md; PAPER.md:84-85 steps vi-vii, eq. 8).
//
//   n_fft = N1 * N2,  k = N2*k1 + k2,  m = m1 + N1*m2
//   pass 1 (one CTA = W adjacent columns k2):   T[k2][m1] = W_N^{k2 m1} sum_k1 y[N2 k1 + k2] W_N1^{k1 m1}
//   pass 2 (one CTA = W adjacent rows   m1):    X[m1 + N1 m2] = sum_k2 T[k2][m1] W_N2^{k2 m2}
//
// An element is a float4 = (Re Fa, Im Fa, Re Fb, Im Fb): both transforms run in lock step and
// share every twiddle.  Each thread keeps 16 elements in registers; shared memory is only the
// exchange buffer between radix passes (one buffer, two barriers per exchange).  The first pass
// reads global memory straight into registers and the last pass writes global memory straight
// from registers, so a sub-FFT of length 2^10 costs two shared-memory round trips.
#pragma once
#include "fstat_common.cuh"

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

// o * exp(-2 pi i j/16), j = 0..7, with the trivial cases spelled out (j is a compile-time
// constant after unrolling).
__device__ __forceinline__ float2 mul_w16(float2 o, int j) {
    const float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    switch (j) {
        case 0: return o;
        case 1: return make_float2(fmaf(o.x, c1, o.y * s1), fmaf(o.y, c1, -o.x * s1));
        case 2: return make_float2((o.x + o.y) * h, (o.y - o.x) * h);
        case 3: return make_float2(fmaf(o.x, s1, o.y * c1), fmaf(o.y, s1, -o.x * c1));
        case 4: return make_float2(o.y, -o.x);
        case 5: return make_float2(fmaf(-o.x, s1, o.y * c1), fmaf(-o.y, s1, -o.x * c1));
        case 6: return make_float2((o.y - o.x) * h, -(o.x + o.y) * h);
        default: return make_float2(fmaf(-o.x, c1, o.y * s1), fmaf(-o.y, c1, -o.x * s1));
    }
}

// In-place forward DFT of length R (kernel exp(-2 pi i rq/R)), natural order in and out.
template <int R> __device__ __forceinline__ void dft(float2 *v) {
    float2 e[R / 2], o[R / 2];
#pragma unroll
    for (int q = 0; q < R / 2; ++q) { e[q] = v[2 * q]; o[q] = v[2 * q + 1]; }
    dft<R / 2>(e);
    dft<R / 2>(o);
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
        const float2 t = mul_w16(o[k], k * (16 / R));
        v[k] = cadd(e[k], t);
        v[k + R / 2] = csub(e[k], t);
    }
}
template <> __device__ __forceinline__ void dft<1>(float2 *) {}

// Radix plan per sub-FFT length 2^LOGN (16 register elements per thread).
template <int LOGN> struct RadixPlan;
template <> struct RadixPlan<6>  { static constexpr int np = 2, r0 = 8,  r1 = 8,  r2 = 1; };
template <> struct RadixPlan<7>  { static constexpr int np = 2, r0 = 16, r1 = 8,  r2 = 1; };
template <> struct RadixPlan<8>  { static constexpr int np = 2, r0 = 16, r1 = 16, r2 = 1; };
template <> struct RadixPlan<9>  { static constexpr int np = 3, r0 = 8,  r1 = 8,  r2 = 8; };
template <> struct RadixPlan<10> { static constexpr int np = 3, r0 = 16, r1 = 16, r2 = 4; };
template <> struct RadixPlan<11> { static constexpr int np = 3, r0 = 16, r1 = 16, r2 = 8; };
template <> struct RadixPlan<12> { static constexpr int np = 3, r0 = 16, r1 = 16, r2 = 16; };

constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }

template <int LOGN> struct FftCfg {
    static constexpr int LOGW = (LOGN == 12) ? 1 : 12 - LOGN;     // tile = 4096 elements (8192 for 2^12)
    static constexpr int W = 1 << LOGW;
    static constexpr int N = 1 << LOGN;
    static constexpr int NT = (N * W) / 16;
    static constexpr int SMEM_BYTES = N * W * 16;
    // twiddle table offsets (float2 entries): pass s >= 1 holds (R_s - 1) * P_s entries, [r-1][k]
    static constexpr int P1 = RadixPlan<LOGN>::r0;
    static constexpr int P2 = P1 * RadixPlan<LOGN>::r1;
    static constexpr int OFF1 = 0;
    static constexpr int OFF2 = (RadixPlan<LOGN>::r1 - 1) * P1;
    static constexpr int TW_ENTRIES = OFF2 + (RadixPlan<LOGN>::np > 2 ? (RadixPlan<LOGN>::r2 - 1) * P2 : 0);
};

// Shared-memory exchange layout: element idx of lane w lives at idx*W + (w ^ swz(idx)) so that
// both "consecutive lanes -> consecutive w" and "consecutive lanes -> consecutive idx" accesses
// of 16-byte elements spread over all banks.
template <int LOGW> __device__ __forceinline__ int sm_phys(int idx, int w) {
    constexpr int W = 1 << LOGW;
    if (LOGW == 0) return idx;
    const int s = (LOGW >= 3) ? (idx & 7) : ((idx >> (3 - LOGW)) & (W - 1));
    return (idx << LOGW) + (w ^ s);
}

// One radix-R Stockham pass on the 16 register elements: twiddle (if P > 1) and DFT.
// Work item bb of this thread is butterfly i = item_i(bb); inputs sit in slots bb*R + r.
template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST>
struct PassIdx {
    static constexpr int LOGR = ilog2c(R);
    static constexpr int NB = 16 / R;                 // butterflies per thread
    static constexpr int NI = (1 << LOGN) / R;        // butterflies per FFT
    __device__ __forceinline__ static void item(int bb, int &i, int &w) {
        const int g = threadIdx.x + bb * NT;
        if (IFAST) { i = g & (NI - 1); w = g >> (LOGN - LOGR); }
        else { w = g & ((1 << LOGW) - 1); i = g >> LOGW; }
    }
    __device__ __forceinline__ static int in_idx(int i, int r) { return i + r * NI; }
    __device__ __forceinline__ static int out_idx(int i, int r) {
        const int k = i & (P - 1);
        return ((i - k) << LOGR) + k + r * P;
    }
};

template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST>
__device__ __forceinline__ void pass_compute(float2 (&a)[16], float2 (&b)[16], const float2 *__restrict__ tw) {
    using PI = PassIdx<R, P, LOGN, LOGW, NT, IFAST>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        if (P > 1) {
            int i, w;
            PI::item(bb, i, w);
            const int k = i & (P - 1);
#pragma unroll
            for (int r = 1; r < R; ++r) {
                const float2 t = __ldg(tw + (r - 1) * P + k);
                a[bb * R + r] = cmul(a[bb * R + r], t);
                b[bb * R + r] = cmul(b[bb * R + r], t);
            }
        }
        dft<R>(&a[bb * R]);
        dft<R>(&b[bb * R]);
    }
}

template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST>
__device__ __forceinline__ void pass_store_smem(const float2 (&a)[16], const float2 (&b)[16], float4 *sm) {
    using PI = PassIdx<R, P, LOGN, LOGW, NT, IFAST>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        int i, w;
        PI::item(bb, i, w);
#pragma unroll
        for (int r = 0; r < R; ++r)
            sm[sm_phys<LOGW>(PI::out_idx(i, r), w)] = make_float4(a[bb * R + r].x, a[bb * R + r].y, b[bb * R + r].x, b[bb * R + r].y);
    }
}

template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST>
__device__ __forceinline__ void pass_load_smem(float2 (&a)[16], float2 (&b)[16], const float4 *sm) {
    using PI = PassIdx<R, P, LOGN, LOGW, NT, IFAST>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        int i, w;
        PI::item(bb, i, w);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 v = sm[sm_phys<LOGW>(PI::in_idx(i, r), w)];
            a[bb * R + r] = make_float2(v.x, v.y);
            b[bb * R + r] = make_float2(v.z, v.w);
        }
    }
}

struct FftArgs {
    const float4 *S;          // [n_sky_slots][n_fft] per-sky resampled series
    float4 *T;                // [n_inflight][n_fft] four-step intermediate
    const TmplDesc *tmpl;     // descriptors of the templates of this launch (blockIdx.y indexes it)
    const SkyABCD *abcd;      // [n_sky_slots]
    float *twoF;              // output rows of this launch: row blockIdx.y
    int64_t twoF_stride;      // floats between rows
    const float2 *tw;         // twiddle table of this sub-FFT length
    int64_t n_fft, n_src, n_bins, k_margin;
    double dt;
    int log_other;            // log2 of the other factor (N2 for pass 1, N1 for pass 2)
};

// ---------------------------------------------------------------------------------------
// Pass 1: spin-down prologue + column FFTs of length N1 = 2^LOGN + four-step twiddle.
// grid = (N2 / W, templates in this launch)
// ---------------------------------------------------------------------------------------
template <int LOGN>
__global__ void __launch_bounds__(FftCfg<LOGN>::NT, (LOGN == 12) ? 1 : 2)
fft_pass1_kernel(FftArgs p) {
    using C = FftCfg<LOGN>;
    using RP = RadixPlan<LOGN>;
    constexpr int LOGW = C::LOGW, NT = C::NT;
    extern __shared__ float4 sm[];
    const TmplDesc td = p.tmpl[blockIdx.y];
    const float4 *__restrict__ S = p.S + (int64_t)td.sky_slot * p.n_fft;
    float4 *__restrict__ T = p.T + (int64_t)blockIdx.y * p.n_fft;
    const int k2_0 = blockIdx.x << LOGW;
    float2 a[16], b[16];

    {   // pass 0 inputs from global memory, times exp(-i Phi_s) (S9)
        using PI = PassIdx<RP::r0, 1, LOGN, LOGW, NT, false>;
#pragma unroll
        for (int bb = 0; bb < PI::NB; ++bb) {
            int i, w;
            PI::item(bb, i, w);
#pragma unroll
            for (int r = 0; r < RP::r0; ++r) {
                const int64_t k = ((int64_t)PI::in_idx(i, r) << p.log_other) + k2_0 + w;
                float4 v = make_float4(0.f, 0.f, 0.f, 0.f);
                if (k < p.n_src) {
                    v = __ldcg(S + k);
                    const double tau = (double)(k - p.k_margin) * p.dt;
                    const double cyc = tau * tau * fma(td.sixth_fddot, tau, td.half_fdot);
                    float sp, cp;
                    sincospif(-2.0f * (float)(cyc - rint(cyc)), &sp, &cp);
                    v = make_float4(v.x * cp - v.y * sp, v.x * sp + v.y * cp, v.z * cp - v.w * sp, v.z * sp + v.w * cp);
                }
                a[bb * RP::r0 + r] = make_float2(v.x, v.y);
                b[bb * RP::r0 + r] = make_float2(v.z, v.w);
            }
        }
    }
    pass_compute<RP::r0, 1, LOGN, LOGW, NT, false>(a, b, nullptr);
    pass_store_smem<RP::r0, 1, LOGN, LOGW, NT, false>(a, b, sm);
    __syncthreads();
    constexpr bool LAST1 = (RP::np == 2);
    pass_load_smem<RP::r1, C::P1, LOGN, LOGW, NT, LAST1>(a, b, sm);
    pass_compute<RP::r1, C::P1, LOGN, LOGW, NT, LAST1>(a, b, p.tw + C::OFF1);
    if (!LAST1) {
        __syncthreads();
        pass_store_smem<RP::r1, C::P1, LOGN, LOGW, NT, false>(a, b, sm);
        __syncthreads();
        pass_load_smem<RP::r2, C::P2, LOGN, LOGW, NT, true>(a, b, sm);
        pass_compute<RP::r2, C::P2, LOGN, LOGW, NT, true>(a, b, p.tw + C::OFF2);
    }
    {   // last pass outputs: m1 = i + r*N1/R (consecutive lanes -> consecutive m1), times W_N^{k2 m1}
        constexpr int RL = LAST1 ? RP::r1 : RP::r2;
        constexpr int PL = LAST1 ? C::P1 : C::P2;
        using PI = PassIdx<RL, PL, LOGN, LOGW, NT, true>;
        const float inv_n = 1.0f / (float)p.n_fft;
#pragma unroll
        for (int bb = 0; bb < PI::NB; ++bb) {
            int i, w;
            PI::item(bb, i, w);
            const int k2 = k2_0 + w;
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                const int m1 = PI::out_idx(i, r);
                const uint32_t t = ((uint32_t)k2 * (uint32_t)m1) & (uint32_t)(p.n_fft - 1);
                float sp, cp;
                sincospif(-2.0f * ((float)t * inv_n), &sp, &cp);
                const float2 tw = make_float2(cp, sp);
                const float2 x = cmul(a[bb * RL + r], tw), y = cmul(b[bb * RL + r], tw);
                __stcg(T + ((int64_t)k2 << LOGN) + m1, make_float4(x.x, x.y, y.x, y.y));
            }
        }
    }
}

// ---------------------------------------------------------------------------------------
// Pass 2: row FFTs of length N2 = 2^LOGN + the 2F combination of eq. 8 (Fig. 1).
// grid = (N1 / W, templates in this launch)
// ---------------------------------------------------------------------------------------
template <int LOGN>
__global__ void __launch_bounds__(FftCfg<LOGN>::NT, (LOGN == 12) ? 1 : 2)
fft_pass2_kernel(FftArgs p) {
    using C = FftCfg<LOGN>;
    using RP = RadixPlan<LOGN>;
    constexpr int LOGW = C::LOGW, NT = C::NT;
    extern __shared__ float4 sm[];
    const TmplDesc td = p.tmpl[blockIdx.y];
    const float4 *__restrict__ T = p.T + (int64_t)blockIdx.y * p.n_fft;
    const int m1_0 = blockIdx.x << LOGW;
    float2 a[16], b[16];
    {
        using PI = PassIdx<RP::r0, 1, LOGN, LOGW, NT, false>;
#pragma unroll
        for (int bb = 0; bb < PI::NB; ++bb) {
            int i, w;
            PI::item(bb, i, w);
#pragma unroll
            for (int r = 0; r < RP::r0; ++r) {
                const float4 v = __ldcg(T + ((int64_t)PI::in_idx(i, r) << p.log_other) + m1_0 + w);
                a[bb * RP::r0 + r] = make_float2(v.x, v.y);
                b[bb * RP::r0 + r] = make_float2(v.z, v.w);
            }
        }
    }
    pass_compute<RP::r0, 1, LOGN, LOGW, NT, false>(a, b, nullptr);
    pass_store_smem<RP::r0, 1, LOGN, LOGW, NT, false>(a, b, sm);
    __syncthreads();
    pass_load_smem<RP::r1, C::P1, LOGN, LOGW, NT, false>(a, b, sm);
    pass_compute<RP::r1, C::P1, LOGN, LOGW, NT, false>(a, b, p.tw + C::OFF1);
    constexpr bool LAST1 = (RP::np == 2);
    if (!LAST1) {
        __syncthreads();
        pass_store_smem<RP::r1, C::P1, LOGN, LOGW, NT, false>(a, b, sm);
        __syncthreads();
        pass_load_smem<RP::r2, C::P2, LOGN, LOGW, NT, false>(a, b, sm);
        pass_compute<RP::r2, C::P2, LOGN, LOGW, NT, false>(a, b, p.tw + C::OFF2);
    }
    {   // epilogue: 2F[q], q = m1 + N1*m2 (consecutive lanes -> consecutive m1)
        constexpr int RL = LAST1 ? RP::r1 : RP::r2;
        constexpr int PL = LAST1 ? C::P1 : C::P2;
        using PI = PassIdx<RL, PL, LOGN, LOGW, NT, false>;
        const SkyABCD ab = p.abcd[td.sky_slot];
        float *__restrict__ out = p.twoF + (int64_t)blockIdx.y * p.twoF_stride;
#pragma unroll
        for (int bb = 0; bb < PI::NB; ++bb) {
            int i, w;
            PI::item(bb, i, w);
#pragma unroll
            for (int r = 0; r < RL; ++r) {
                const int64_t q = ((int64_t)PI::out_idx(i, r) << p.log_other) + m1_0 + w;
                if (q < p.n_bins) {
                    const float2 fa = a[bb * RL + r], fb = b[bb * RL + r];
                    const float twoF = ab.b_over_d * (fa.x * fa.x + fa.y * fa.y) + ab.a_over_d * (fb.x * fb.x + fb.y * fb.y)
                                     - ab.two_c_over_d * (fa.x * fb.x + fa.y * fb.y);
                    __stcs(out + q, twoF);
                }
            }
        }
    }
}
