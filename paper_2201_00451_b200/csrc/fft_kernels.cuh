// Batched four-step Stockham FFT of the pair (Fa(t), Fb(t)) with the spin-down prologue
// and the 2F epilogue fused in (H4b, H6, H7 of DESIGN.md; PAPER.md:84-85 steps vi-vii, eq. 8).
//
//   n_fft = N1 * N2,  k = N2*k1 + k2,  m = m1 + N1*m2
//   pass 1 (one CTA = W adjacent columns k2):   T[k2][m1] = W_N^{k2 m1} sum_k1 y[N2 k1 + k2] W_N1^{k1 m1}
//   pass 2 (one CTA = W adjacent rows   m1):    X[m1 + N1 m2] = sum_k2 T[k2][m1] W_N2^{k2 m2}
//
// An element is a float4 = (Re Fa, Re Fb, Im Fa, Im Fb): both transforms run in lock step and
// share every twiddle.  Each thread keeps E = 16 elements in registers (32 in the two-pass radix-32
// plans of pass 2); shared memory is the exchange buffer between radix passes (one buffer, two
// barriers per exchange).  CTAs are persistent: each loops over tiles, and as soon as the last radix
// pass of a tile has pulled its inputs out of the buffer, the NEXT tile -- one contiguous block of
// global memory thanks to the tile-blocked layouts of S and T -- is copied into it by one thread with
// 1-D bulk TMA (cp.async.bulk + mbarrier; no registers), so the copy flies while the last pass, the
// twiddle / 2F epilogue and the global stores of the current tile execute.
#pragma once
#include "fstat_common.cuh"
#include "fft_launch.cuh"
// Experiment switch ('Tried, not kept'): FFT pass 1 with a staging buffer of its own, so that the next tile's
// bulk copy starts as soon as the current tile's inputs are in registers.  Measured slower (3 instead of 5 CTAs per SM).
#ifndef FFT_P1_DB
#define FFT_P1_DB 0
#endif
#include "sky_math.cuh"
#ifndef FFT_CTAS11
#define FFT_CTAS11 5
#endif
#ifndef FFT_CTAS_WARP
#define FFT_CTAS_WARP 11
#endif

// Packed arithmetic.  Fa and Fb go through identical butterflies with identical twiddles, so
// a register pair holds (Re Fa, Re Fb) or (Im Fa, Im Fb) and every add / multiply / FMA is one
// Blackwell f32x2 instruction (SASS FADD2 / FMUL2 / FFMA2) with the twiddle as a broadcast scalar.
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ float2 mul2s(float2 a, float s) { return __fmul2_rn(a, make_float2(s, s)); }
__device__ __forceinline__ float2 fma2s(float2 a, float s, float2 c) { return __ffma2_rn(a, make_float2(s, s), c); }
// scalar complex product (twiddle recurrences)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}
// (x + i y) * (t.x + i t.y) on a packed pair
__device__ __forceinline__ void pcmul(float2 &x, float2 &y, float2 t) {
    const float2 nx = fma2s(x, t.x, mul2s(y, -t.y));
    const float2 ny = fma2s(x, t.y, mul2s(y, t.x));
    x = nx; y = ny;
}

// (ox + i oy) * exp(-2 pi i j/16), j = 0..7 (j is a compile-time constant after unrolling).
__device__ __forceinline__ void mul_w16(float2 &ox, float2 &oy, int j) {
    const float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    float2 tx, ty;
    switch (j) {
        case 0: return;
        case 1: tx = fma2s(ox, c1, mul2s(oy, s1)); ty = fma2s(oy, c1, mul2s(ox, -s1)); break;
        case 2: tx = mul2s(add2(ox, oy), h); ty = mul2s(sub2(oy, ox), h); break;
        case 3: tx = fma2s(ox, s1, mul2s(oy, c1)); ty = fma2s(oy, s1, mul2s(ox, -c1)); break;
        case 4: tx = oy; ty = make_float2(-ox.x, -ox.y); break;
        case 5: tx = fma2s(ox, -s1, mul2s(oy, c1)); ty = fma2s(oy, -s1, mul2s(ox, -c1)); break;
        case 6: tx = mul2s(sub2(oy, ox), h); ty = mul2s(add2(ox, oy), -h); break;
        default: tx = fma2s(ox, -c1, mul2s(oy, s1)); ty = fma2s(oy, -c1, mul2s(ox, -s1)); break;
    }
    ox = tx; oy = ty;
}

// (ox + i oy) * exp(-2 pi i j/32), j = 0..15 (compile-time constant after unrolling).
__device__ __forceinline__ void mul_w32(float2 &ox, float2 &oy, int j) {
    if ((j & 1) == 0) { mul_w16(ox, oy, j >> 1); return; }
    // cos, sin of 2 pi j / 32 for odd j
    const float c = (j == 1 || j == 15) ? 0.98078528040323043f : (j == 3 || j == 13) ? 0.83146961230254524f
                  : (j == 5 || j == 11) ? 0.55557023301960218f : 0.19509032201612825f;
    const float sn = (j == 1 || j == 15) ? 0.19509032201612825f : (j == 3 || j == 13) ? 0.55557023301960218f
                   : (j == 5 || j == 11) ? 0.83146961230254524f : 0.98078528040323043f;
    const float cc = (j > 8) ? -c : c;                      // cos(2 pi j/32) is negative for j in (8, 16)
    // (x + i y)(cc - i sn) = (x cc + y sn) + i (y cc - x sn)
    const float2 tx = fma2s(ox, cc, mul2s(oy, sn)), ty = fma2s(oy, cc, mul2s(ox, -sn));
    ox = tx; oy = ty;
}

// In-place forward DFT of length R (kernel exp(-2 pi i rq/R)) on packed pairs, natural order.
template <int R> __device__ __forceinline__ void dft(float2 *x, float2 *y) {
    float2 ex[R / 2], ey[R / 2], ox[R / 2], oy[R / 2];
#pragma unroll
    for (int q = 0; q < R / 2; ++q) { ex[q] = x[2 * q]; ey[q] = y[2 * q]; ox[q] = x[2 * q + 1]; oy[q] = y[2 * q + 1]; }
    dft<R / 2>(ex, ey);
    dft<R / 2>(ox, oy);
#pragma unroll
    for (int k = 0; k < R / 2; ++k) {
        mul_w32(ox[k], oy[k], k * (32 / R));
        x[k] = add2(ex[k], ox[k]); y[k] = add2(ey[k], oy[k]);
        x[k + R / 2] = sub2(ex[k], ox[k]); y[k + R / 2] = sub2(ey[k], oy[k]);
    }
}
template <> __device__ __forceinline__ void dft<1>(float2 *, float2 *) {}

// Radix plan per sub-FFT length 2^LOGN and register elements per thread E (16, or 32 for the two-pass plans of pass 2).
template <int LOGN, int E = 16> struct RadixPlan;
template <> struct RadixPlan<6>  { static constexpr int np = 2, r0 = 8,  r1 = 8,  r2 = 1; };
template <> struct RadixPlan<7>  { static constexpr int np = 2, r0 = 16, r1 = 8,  r2 = 1; };
template <> struct RadixPlan<8>  { static constexpr int np = 2, r0 = 16, r1 = 16, r2 = 1; };
template <> struct RadixPlan<9>  { static constexpr int np = 3, r0 = 8,  r1 = 8,  r2 = 8; };
template <> struct RadixPlan<10> { static constexpr int np = 3, r0 = 16, r1 = 16, r2 = 4; };
template <> struct RadixPlan<11> { static constexpr int np = 3, r0 = 16, r1 = 16, r2 = 8; };
template <> struct RadixPlan<12> { static constexpr int np = 3, r0 = 16, r1 = 16, r2 = 16; };
template <> struct RadixPlan<9, 32>  { static constexpr int np = 2, r0 = 32, r1 = 16, r2 = 1; };
template <> struct RadixPlan<10, 32> { static constexpr int np = 2, r0 = 32, r1 = 32, r2 = 1; };

__host__ __device__ constexpr int ilog2c(int v) { return v <= 1 ? 0 : 1 + ilog2c(v >> 1); }

// A tile is 2^LOGT elements = W = 2^(LOGT - LOGN) adjacent sub-FFTs, worked on by 2^LOGT / 16 threads:
// LOGT = 11 (128 threads, 32 KB, 4 CTAs per SM) or 12 (256 threads, 64 KB, 2 CTAs per SM); sub-FFTs of
// length 2^12 use LOGT = 13 (two per tile, so that the other pass still gets 32-byte store runs).
template <int LOGN, int LOGT, int E = 16> struct FftCfg {
    static_assert(LOGT >= LOGN && LOGT >= 10 && LOGT <= 13, "tile must hold at least one sub-FFT");
    static constexpr int LOGW = LOGT - LOGN;
    static constexpr int W = 1 << LOGW;
    // LOGT = 10 with 32 elements per thread: one warp per CTA works on one 2^10-point column (no cross-warp barrier at all)
    static constexpr int MIN_CTAS = (E == 32) ? (LOGT == 13 ? 1 : LOGT == 10 ? FFT_CTAS_WARP : 3) : (LOGT == 11) ? FFT_CTAS11 : (LOGT == 12) ? 2 : 1;
    static constexpr int N = 1 << LOGN;
    static constexpr int NT = (N * W) / E;
    // twiddle table offsets (float2 entries): pass s >= 1 holds (R_s - 1) * P_s entries, [r-1][k]
    static constexpr int P1 = RadixPlan<LOGN, E>::r0;
    static constexpr int P2 = P1 * RadixPlan<LOGN, E>::r1;
    static constexpr int OFF1 = 0;
    static constexpr int OFF2 = (RadixPlan<LOGN, E>::r1 - 1) * P1;
    static constexpr int TW_ENTRIES = OFF2 + (RadixPlan<LOGN, E>::np > 2 ? (RadixPlan<LOGN, E>::r2 - 1) * P2 : 0);
    static constexpr int BUF_ELEMS = (N + N / RadixPlan<LOGN, E>::r0) * W;  // exchange buffer: one pad column of W elements per r0 indices
    // twiddles of the last radix pass of the 2^11-point plan (14 KB) are read from global memory through L1 instead of
    // shared memory: one more CTA per SM with 2^11-element tiles (measured +1 %; at 2^12 points a third CTA per SM costs
    // more in registers than it gains)
    static constexpr bool TW_LAST_GLOBAL = (RadixPlan<LOGN, E>::np > 2) && (LOGN == 11);
    // one-warp CTAs read every twiddle from global memory through L1 (the 8 KB table per warp would halve the warps per SM)
    static constexpr bool TW_ALL_GLOBAL = (NT == 32);
    static constexpr int TW_SMEM_ENTRIES = TW_ALL_GLOBAL ? 0 : TW_LAST_GLOBAL ? OFF2 : TW_ENTRIES;
    static constexpr int SMEM_BYTES = BUF_ELEMS * 16 + TW_SMEM_ENTRIES * 8 + 16;   // exchange buffer + twiddle table + mbarrier
    // pass 1 with a staging buffer of its own (FFT_P1_DB): the next tile's bulk copy starts as soon as the current tile's
    // inputs are in registers instead of after its last exchange
    static constexpr int P1_STAGE_ELEMS = FFT_P1_DB ? N * W : 0;
    static constexpr int SMEM_BYTES_P1 = SMEM_BYTES + P1_STAGE_ELEMS * 16;
    static constexpr int MIN_CTAS_P1 = FFT_P1_DB ? ((228 * 1024 / (SMEM_BYTES_P1 + 1024)) > 5 ? 5 : (228 * 1024 / (SMEM_BYTES_P1 + 1024))) : MIN_CTAS;
};

// Shared-memory exchange layout: element idx of lane w lives at 16-byte chunk
//   ((idx + (idx >> LOGR0)) << LOGW) + w
// i.e. after every r0 = 2^LOGR0 indices one column of W elements is left empty.  The stride-r0 stores of the first
// pass then advance by (r0 + 1) W chunks from lane to lane (conflict-free: 8 distinct chunks per quarter warp for
// every r0 in {8, 16, 32} and W in {1, 2, 4, >= 8}), the index-consecutive loads and stores of the later passes stay
// consecutive within an aligned group of 8 lanes, and -- unlike an XOR swizzle -- every address a thread touches in one
// pass is its base plus a compile-time offset (immediate operands instead of three integer instructions per element).
template <int LOGW, int LOGR0> __device__ __forceinline__ int sm_phys(int idx, int w) {
    return ((idx + (idx >> LOGR0)) << LOGW) + w;
}
// chunk offset of index distance d from a base index: valid when d is a multiple of r0, or d < r0 on an r0-aligned base
template <int LOGW, int LOGR0> __host__ __device__ constexpr int sm_off(int d) { return (d + (d >> LOGR0)) << LOGW; }

// One radix-R Stockham pass on the E register elements: twiddle (if P > 1) and DFT.
// Work item bb of this thread is butterfly i = item_i(bb); inputs sit in slots bb*R + r.
template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST>
struct PassIdx {
    static constexpr int LOGR = ilog2c(R);
    static constexpr int NB = ((1 << (LOGN + LOGW)) / NT) / R;   // butterflies per thread = register elements / R
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

template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST, int E, bool TW_LDG = false>
__device__ __forceinline__ void pass_compute(float2 (&a)[E], float2 (&b)[E], const float2 *__restrict__ tw) {
    using PI = PassIdx<R, P, LOGN, LOGW, NT, IFAST>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        if (P > 1) {
            int i, w;
            PI::item(bb, i, w);
            const int k = i & (P - 1);
#pragma unroll
            for (int r = 1; r < R; ++r) {
                pcmul(a[bb * R + r], b[bb * R + r], TW_LDG ? __ldg(tw + (r - 1) * P + k) : tw[(r - 1) * P + k]);
            }
        }
        dft<R>(&a[bb * R], &b[bb * R]);
    }
}

template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST, int LOGR0, int E>
__device__ __forceinline__ void pass_store_smem(const float2 (&a)[E], const float2 (&b)[E], float4 *sm) {
    using PI = PassIdx<R, P, LOGN, LOGW, NT, IFAST>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        int i, w;
        PI::item(bb, i, w);
        // out_idx(i, r) = out_idx(i, 0) + r P with P = 1 (first pass: base index r0-aligned) or a multiple of r0
        static_assert(P == 1 || (P >> LOGR0) >= 1, "pass stride must be 1 or a multiple of r0");
        float4 *base = sm + sm_phys<LOGW, LOGR0>(PI::out_idx(i, 0), w);
#pragma unroll
        for (int r = 0; r < R; ++r)
            base[sm_off<LOGW, LOGR0>(r * P)] = make_float4(a[bb * R + r].x, a[bb * R + r].y, b[bb * R + r].x, b[bb * R + r].y);
    }
}

template <int R, int P, int LOGN, int LOGW, int NT, bool IFAST, int LOGR0, int E>
__device__ __forceinline__ void pass_load_smem(float2 (&a)[E], float2 (&b)[E], const float4 *sm) {
    using PI = PassIdx<R, P, LOGN, LOGW, NT, IFAST>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        int i, w;
        PI::item(bb, i, w);
        // in_idx = i + r*NI with NI a multiple of r0: base + compile-time offsets
        static_assert((PI::NI >> LOGR0) >= 1, "NI must be a multiple of r0");
        const float4 *base = sm + sm_phys<LOGW, LOGR0>(i, w);
#pragma unroll
        for (int r = 0; r < R; ++r) {
            const float4 v = base[sm_off<LOGW, LOGR0>(r * PI::NI)];
            a[bb * R + r] = make_float2(v.x, v.y);
            b[bb * R + r] = make_float2(v.z, v.w);
        }
    }
}


// exp(-2 pi i x) for a phase x in cycles held in fp64: reduce mod 1 in fp64, sincospif in fp32.
__device__ __forceinline__ float2 expm2pi(double cyc) {
    float sp, cp;
    sincospif(-2.0f * (float)(cyc - rint(cyc)), &sp, &cp);
    return make_float2(cp, sp);
}

// ---- mbarrier + 1-D bulk copy (TMA, cp.async.bulk -> SASS UBLKCP) ------------------------
__device__ __forceinline__ void mbar_init(uint64_t *bar, int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, unsigned parity) {
    const unsigned a = (unsigned)__cvta_generic_to_shared(bar);
    unsigned done = 0;
    while (!done) {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(done) : "r"(a), "r"(parity) : "memory");
    }
}
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gmem_src, unsigned bytes, uint64_t *bar, uint64_t policy) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;\n" ::
                 "r"((unsigned)__cvta_generic_to_shared(smem_dst)), "l"(gmem_src), "r"(bytes),
                 "r"((unsigned)__cvta_generic_to_shared(bar)), "l"(policy) : "memory");
}
// L2 eviction policies: the resampled series S is re-read by every template of the launch
// (evict_last), the four-step intermediate T is written once and read once (evict_first).
__device__ __forceinline__ uint64_t l2_policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t l2_policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(p));
    return p;
}
__device__ __forceinline__ void st_global_hint(float4 *ptr, float4 v, uint64_t policy) {
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;\n" ::
                 "l"(ptr), "f"(v.x), "f"(v.y), "f"(v.z), "f"(v.w), "l"(policy) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory"); }

// One thread starts the copy of a whole tile (contiguous in global memory thanks to the
// tile-blocked layouts) into the exchange buffer; completion is signalled on the mbarrier.
template <int LOGN, int LOGT>
__device__ __forceinline__ void tile_prefetch(float4 *sm, const float4 *__restrict__ src, uint64_t *bar, uint64_t policy,
                                              unsigned n_bytes = FftCfg<LOGN, LOGT>::N * FftCfg<LOGN, LOGT>::W * 16) {
    // n_bytes: the leading part of the tile that is copied (pass 1 skips the rows that are zero padding)
    constexpr unsigned CHUNK = 16384;
    if (threadIdx.x == 0) {
        fence_proxy_async();                      // earlier generic-proxy reads of the buffer are ordered before the async writes
        mbar_expect_tx(bar, n_bytes);
        for (unsigned o = 0; o < n_bytes; o += CHUNK)
            bulk_g2s(reinterpret_cast<char *>(sm) + o, reinterpret_cast<const char *>(src) + o, min(CHUNK, n_bytes - o), bar, policy);
    }
}

// Pass-0 inputs out of the staging layout (linear: element idx of lane w at idx*W + w).
template <int LOGN, int LOGT, int E>
__device__ __forceinline__ void tile_take_inputs(float2 (&a)[E], float2 (&b)[E], const float4 *sm, int r_nz = 32) {
    // r_nz: inputs r >= r_nz of every butterfly are zero padding (not staged, not read)
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    using PI = PassIdx<RP::r0, 1, LOGN, C::LOGW, C::NT, false>;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        const int g = threadIdx.x + bb * C::NT;   // = i*W + w
#pragma unroll
        for (int r = 0; r < RP::r0; ++r) {
            const float4 v = (r < r_nz) ? sm[g + ((r * PI::NI) << C::LOGW)] : make_float4(0.f, 0.f, 0.f, 0.f);
            a[bb * RP::r0 + r] = make_float2(v.x, v.y);
            b[bb * RP::r0 + r] = make_float2(v.z, v.w);
        }
    }
}

// Radix passes of one tile between "inputs of pass 0 are in registers" and "inputs of the last
// pass are in registers and the exchange buffer is free again" (barrier included).
template <int LOGN, int LOGT, int E>
__device__ __forceinline__ void tile_passes(float2 (&a)[E], float2 (&b)[E], float4 *sm, const float2 *__restrict__ tw) {
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    constexpr int LOGW = C::LOGW, NT = C::NT, LOGR0 = ilog2c(RP::r0);
    constexpr bool LAST1 = (RP::np == 2);
    __syncthreads();                                   // every thread has taken its pass-0 inputs
    pass_compute<RP::r0, 1, LOGN, LOGW, NT, false>(a, b, nullptr);
    pass_store_smem<RP::r0, 1, LOGN, LOGW, NT, false, LOGR0>(a, b, sm);
    __syncthreads();
    pass_load_smem<RP::r1, C::P1, LOGN, LOGW, NT, false, LOGR0>(a, b, sm);
    if (!LAST1) {
        pass_compute<RP::r1, C::P1, LOGN, LOGW, NT, false>(a, b, tw + C::OFF1);
        __syncthreads();
        pass_store_smem<RP::r1, C::P1, LOGN, LOGW, NT, false, LOGR0>(a, b, sm);
        __syncthreads();
        pass_load_smem<RP::r2, C::P2, LOGN, LOGW, NT, false, LOGR0>(a, b, sm);
    }
    __syncthreads();                                   // buffer free: the next tile may be prefetched
}

// tw: the shared-memory table; tw_g: the same table in global memory (used for the last pass when it is not in shared memory)
template <int LOGN, int LOGT, int E>
__device__ __forceinline__ void tile_last_pass(float2 (&a)[E], float2 (&b)[E], const float2 *__restrict__ tw, const float2 *__restrict__ tw_g) {
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    if (RP::np == 2 && C::TW_ALL_GLOBAL) pass_compute<RP::r1, C::P1, LOGN, C::LOGW, C::NT, false, E, true>(a, b, tw_g + C::OFF1);
    else if (RP::np == 2) pass_compute<RP::r1, C::P1, LOGN, C::LOGW, C::NT, false>(a, b, tw + C::OFF1);
    else if (C::TW_LAST_GLOBAL) pass_compute<RP::r2, C::P2, LOGN, C::LOGW, C::NT, false, E, true>(a, b, tw_g + C::OFF2);
    else pass_compute<RP::r2, C::P2, LOGN, C::LOGW, C::NT, false>(a, b, tw + C::OFF2);
}

// Spin-down factor exp(-i Phi_s) on the pass-0 inputs of FFT pass 1.  The r0 inputs of one butterfly sit on an
// arithmetic progression tau_r = tau_0 + r*h, and the phase (cycles) is the cubic phi(tau) = tau^2 (c1 + c2 tau):
// its forward differences D1, D2 and the constant D3 are evaluated once per butterfly in fp64 (mod 1), and
// exp(-2 pi i phi(tau_r)) follows by the recurrence e_{r+1} = e_r d_r, d_{r+1} = d_r q_r, q_{r+1} = q_r c (fp32
// complex products).  Without a second spin-down (CUBIC = false) D2 is the same for every butterfly of the
// template: q comes with the template descriptor (computed on the host in fp64) and the q recurrence disappears.
template <int LOGN, int LOGT, int E, bool SKIPZ, bool CUBIC>
__device__ __forceinline__ void spin_down(float2 (&a)[E], float2 (&b)[E], const FftArgs &p, const TmplDesc &td, int k2_0, int r_nz) {
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    using PI = PassIdx<RP::r0, 1, LOGN, C::LOGW, C::NT, false>;
    const double h = (double)((int64_t)PI::NI << p.log_other) * p.dt;
    // one set of formulas for both variants (c2 = 0 folds the cubic terms away at compile time), and a template
    // without second spin-down takes q from its descriptor in both: its 2F bits do not depend on what else is in the launch
    const double c1 = td.half_fdot, c2 = CUBIC ? td.sixth_fddot : 0.0;
    float2 cc = make_float2(1.f, 0.f);
    if (CUBIC) cc = expm2pi(6.0 * c2 * h * h * h);
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        int i, w;
        PI::item(bb, i, w);
        const int64_t k = ((int64_t)i << p.log_other) + k2_0 + w;
        const double tau = (double)(k - p.k_margin) * p.dt;
        const double t3 = 3.0 * c2 * tau;
        float2 e = expm2pi(tau * tau * fma(c2, tau, c1));
        float2 d = expm2pi(h * (fma(2.0 * tau, c1, tau * t3) + h * (c1 + t3 + c2 * h)));
        float2 q = make_float2(td.q_re, td.q_im);             // exp(-2 pi i 2 c1 h^2)
        if (CUBIC && c2 != 0.0) q = expm2pi(h * h * (2.0 * c1 + 2.0 * t3 + 6.0 * c2 * h));
#pragma unroll
        for (int r = 0; r < RP::r0; ++r) {
            if (SKIPZ && r >= r_nz) break;
            pcmul(a[bb * RP::r0 + r], b[bb * RP::r0 + r], e);
            if (r + 1 < RP::r0) {
                e = cmul(e, d);
                d = cmul(d, q);
                if (CUBIC) q = cmul(q, cc);
            }
        }
    }
}

// Epilogue of FFT pass 1: outputs m1 = i + r*NI of column k2 = k2_0 + w, times the four-step twiddle
// W_N^{k2 m1} = W_N^{k2 i} (W_N^{k2 NI})^r (two exact sincospif per butterfly, powers by products), stored
// tile-blocked for pass 2: T[m1 / W2][k2][m1 % W2] -- consecutive lanes (w, then i) fill whole 128-byte lines.
// m1 = i + r NI: when NI is a multiple of W2 the output address is affine in r (one 64-bit multiply-add per element);
// tiny transforms (NI < W2) take the general form (kernel variant GENERIC, AFFINE = false).
template <int LOGN, int LOGT, int E, bool AFFINE>
__device__ __forceinline__ void store_columns(const float2 (&a)[E], const float2 (&b)[E], const FftArgs &p, float4 *__restrict__ T,
                                              int k2_0, uint64_t pol_T) {
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    constexpr int RL = (RP::np == 2) ? RP::r1 : RP::r2;
    constexpr int PL = (RP::np == 2) ? C::P1 : C::P2;
    using PI = PassIdx<RL, PL, LOGN, C::LOGW, C::NT, false>;
    const float inv_n = 1.0f / (float)p.n_fft;
    const uint32_t nmask = (uint32_t)(p.n_fft - 1);
    const int lw2 = p.log_w_other, ln2 = p.log_other;
    const uint32_t rstride_b = ((uint32_t)PI::NI << ln2) * 16u;
#pragma unroll
    for (int bb = 0; bb < PI::NB; ++bb) {
        int i, w;
        PI::item(bb, i, w);
        const uint32_t k2 = (uint32_t)(k2_0 + w);
        float sp, cp;
        sincospif(-2.0f * ((float)((k2 * (uint32_t)i) & nmask) * inv_n), &sp, &cp);
        float2 tw = make_float2(cp, sp);
        sincospif(-2.0f * ((float)((k2 * (uint32_t)PI::NI) & nmask) * inv_n), &sp, &cp);
        const float2 step = make_float2(cp, sp);
        float4 *colbase = T + ((uint32_t)k2 << lw2);
        const char *dst = reinterpret_cast<const char *>(colbase + (((uint32_t)(i >> lw2) << (ln2 + lw2)) + (uint32_t)(i & ((1 << lw2) - 1))));
#pragma unroll
        for (int r = 0; r < RL; ++r) {
            float2 xx = a[bb * RL + r], yy = b[bb * RL + r];
            pcmul(xx, yy, tw);
            const int m1 = i + r * PI::NI;
            float4 *o = AFFINE ? reinterpret_cast<float4 *>(const_cast<char *>(dst) + (uint64_t)rstride_b * (uint32_t)r)
                               : colbase + (((uint32_t)(m1 >> lw2) << (ln2 + lw2)) + (uint32_t)(m1 & ((1 << lw2) - 1)));
            st_global_hint(o, make_float4(xx.x, xx.y, yy.x, yy.y), pol_T);
            if (r + 1 < RL) tw = cmul(tw, step);
        }
    }
}

// ---------------------------------------------------------------------------------------
// Pass 1: spin-down prologue + column FFTs of length N1 = 2^LOGN + four-step twiddle.
// Persistent: grid = min(n_tiles, CTAs that fit the GPU); tile = (template, W adjacent columns).
// ---------------------------------------------------------------------------------------
// VAR (FFT_VAR_* bits, fft_launch.cuh) selects straight-line variants of the tile loop:
//   SKIPZ   do not stage or touch the zero padding (pays when at least half of every column is padding, as in config 4)
//   CUBIC   the launch holds templates with a second spin-down (fddot != 0): third forward difference in the prologue
//   GENERIC the pass-2 tile has more rows than the last radix pass has butterflies (tiny transforms): general store address
// Tile loop over tiles tile0, tile0 + stride, ... < tile_end (tile = template * tiles_per_template + column block); the
// intermediate of template t goes to p.T[t - t_off] (t_off != 0 only in the single-kernel form, which cycles two
// groups of templates through an L2-resident buffer).
template <int LOGN, int LOGT, int E, int VAR>
__device__ __forceinline__ void pass1_tile_loop(const FftArgs &p, float4 *sm, float4 *stage, const float2 *sm_tw, uint64_t *bar, unsigned &parity,
                                                int tile, int tile_end, int stride, int t_off, uint64_t pol_S, uint64_t pol_T) {
    constexpr bool SKIPZ = (VAR & FFT_VAR_SKIPZ) != 0, CUBIC = (VAR & FFT_VAR_CUBIC) != 0, AFFINE = (VAR & FFT_VAR_GENERIC) == 0;
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    constexpr int LOGW = C::LOGW, TILE_ELEMS = C::N * C::W;
    if (tile >= tile_end) return;
    float2 a[E], b[E];
    const int tile_mask = (1 << p.log_tiles) - 1;
    // tile -> (template t, column block x).  Template-major (t = tile / tiles per template) by default; with p.t_fast the
    // template varies fastest, so that the CTAs running at the same time work on the same column blocks of all templates
    // of the launch and the series S, too large to stay in L2 for the length of a template (n_fft >= 2^22), is read from
    // HBM once per launch instead of once per template.
    const bool t_fast = p.t_fast != 0;
    auto tile_t = [&](int tl) { return t_fast ? tl % p.n_tmpl : tl >> p.log_tiles; };
    auto tile_x = [&](int tl) { return t_fast ? tl / p.n_tmpl : tl & tile_mask; };
    TmplDesc td_next = p.tmpl[tile_t(tile)];
    // zero padding: rows k1 >= ceil(n_src / N2) of every column are zero, i.e. the inputs r >= r_nz of every first-pass
    // butterfly (k1 = i + r*NI): they are neither staged nor multiplied by the spin-down factor
    const int r_nz = !SKIPZ ? (int)RP::r0
        : min((int)RP::r0, (int)((((p.n_src + ((int64_t)1 << p.log_other) - 1) >> p.log_other) + (C::N / RP::r0) - 1) / (C::N / RP::r0)));
    const unsigned stage_bytes = (unsigned)min(r_nz * (C::N / RP::r0), (int)C::N) * C::W * 16u;
    tile_prefetch<LOGN, LOGT>(stage, p.S + (int64_t)td_next.sky_slot * p.n_fft + (int64_t)tile_x(tile) * TILE_ELEMS, bar, pol_S, stage_bytes);
    for (; tile < tile_end; tile += stride) {
        const int t = tile_t(tile), x = tile_x(tile);
        const TmplDesc td = td_next;
        const int k2_0 = x << LOGW;
        const int nxt = tile + stride;                  // fetch the next tile's descriptor early
        if (nxt < tile_end) td_next = p.tmpl[tile_t(nxt)];
        mbar_wait(bar, parity);
        parity ^= 1;
        tile_take_inputs<LOGN, LOGT>(a, b, stage, SKIPZ ? r_nz : 32);
        if (FFT_P1_DB) {
            __syncthreads();                            // every thread has taken its inputs: the staging buffer is free
            if (nxt < tile_end)
                tile_prefetch<LOGN, LOGT>(stage, p.S + (int64_t)td_next.sky_slot * p.n_fft + (int64_t)tile_x(nxt) * TILE_ELEMS, bar, pol_S, stage_bytes);
        }
        // times exp(-i Phi_s) (S9)
        spin_down<LOGN, LOGT, E, SKIPZ, CUBIC>(a, b, p, td, k2_0, r_nz);
        tile_passes<LOGN, LOGT>(a, b, sm, sm_tw);
        if (!FFT_P1_DB && nxt < tile_end)
            tile_prefetch<LOGN, LOGT>(sm, p.S + (int64_t)td_next.sky_slot * p.n_fft + (int64_t)tile_x(nxt) * TILE_ELEMS, bar, pol_S, stage_bytes);
        tile_last_pass<LOGN, LOGT>(a, b, sm_tw, p.tw);
        store_columns<LOGN, LOGT, E, AFFINE>(a, b, p, p.T + (int64_t)(t - t_off) * p.n_fft, k2_0, pol_T);
    }
}

// shared-memory carve-up of a pass kernel: exchange buffer | twiddle table | mbarrier
template <int LOGN, int LOGT, int E>
__device__ __forceinline__ void pass_smem_setup(const FftArgs &p, float4 *sm, float2 *&sm_tw, uint64_t *&bar) {
    using C = FftCfg<LOGN, LOGT, E>;
    sm_tw = reinterpret_cast<float2 *>(sm + C::BUF_ELEMS);
    bar = reinterpret_cast<uint64_t *>(sm_tw + C::TW_SMEM_ENTRIES);
    for (int e = threadIdx.x; e < C::TW_SMEM_ENTRIES; e += C::NT) sm_tw[e] = p.tw[e];
    if (threadIdx.x == 0) { mbar_init(bar, 1); fence_proxy_async(); }
    __syncthreads();
}

template <int LOGN, int LOGT, int E, int VAR>
__global__ void __launch_bounds__(FftCfg<LOGN, LOGT, E>::NT, FftCfg<LOGN, LOGT, E>::MIN_CTAS_P1)
fft_pass1_kernel(const __grid_constant__ FftArgs p) {
    extern __shared__ float4 sm[];
    float2 *sm_tw; uint64_t *bar;
    pass_smem_setup<LOGN, LOGT, E>(p, sm, sm_tw, bar);
    unsigned parity = 0;
    float4 *stage = FFT_P1_DB ? reinterpret_cast<float4 *>(reinterpret_cast<char *>(sm) + FftCfg<LOGN, LOGT, E>::SMEM_BYTES) : sm;
    pass1_tile_loop<LOGN, LOGT, E, VAR>(p, sm, stage, sm_tw, bar, parity, blockIdx.x, p.n_tiles, gridDim.x, 0, l2_policy_evict_last(), l2_policy_evict_first());
}

// ---------------------------------------------------------------------------------------
// Sky-varying search (PAPER.md:188 "100 sky locations", :293 2.7e5 sky pointings x 11 spin-downs): FFT pass 1 with
// the sky-dependent half of the path (H1-H5: timing, resampling, heterodyne correction, antenna weights, detector
// sum) in its tile prologue.  Tile = (sky position, W adjacent columns): phase A computes the tile's N1 x W values of
// (Fa(t), Fb(t)) before the spin-down factor from the timing nodes and the Farrow-filtered series (sky_point) into
// shared memory; phase B runs, for every spin-down template of that sky position, spin-down factor -> column FFTs ->
// four-step twiddle -> T.  The resampled series never exists in global memory.  Phase A of one CTA (L2-latency
// bound) overlaps with the FFT phases of the other CTAs on the SM.
// ---------------------------------------------------------------------------------------
template <int LOGN, int LOGT> struct FusedCfg {
    using C = FftCfg<LOGN, LOGT, 16>;
    static constexpr int S_ELEMS = C::N * C::W;                                   // phase-A output, linear layout
    static constexpr int SMEM_BYTES = (S_ELEMS + C::BUF_ELEMS) * 16 + C::TW_SMEM_ENTRIES * 8;
    static constexpr int MIN_CTAS = (228 * 1024 / (SMEM_BYTES + 1024)) < 1 ? 1 : ((228 * 1024 / (SMEM_BYTES + 1024)) > 5 ? 5 : (228 * 1024 / (SMEM_BYTES + 1024)));
};

template <int LOGN, int LOGT, int VAR>
__global__ void __launch_bounds__(FftCfg<LOGN, LOGT, 16>::NT, FusedCfg<LOGN, LOGT>::MIN_CTAS)
fft_sky_pass1_kernel(const __grid_constant__ FusedArgs q) {
    constexpr int E = 16;
    constexpr bool CUBIC = (VAR & FFT_VAR_CUBIC) != 0, AFFINE = (VAR & FFT_VAR_GENERIC) == 0;
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    constexpr int LOGW = C::LOGW, NT = C::NT;
    const FftArgs &p = q.f;
    extern __shared__ float4 sm[];
    float4 *sS = sm, *sX = sm + FusedCfg<LOGN, LOGT>::S_ELEMS;
    float2 *sm_tw = reinterpret_cast<float2 *>(sX + C::BUF_ELEMS);
    for (int e = threadIdx.x; e < C::TW_SMEM_ENTRIES; e += NT) sm_tw[e] = p.tw[e];
    const uint64_t pol_T = l2_policy_evict_first();
    const int tile_mask = (1 << p.log_tiles) - 1;
    float2 a[E], b[E];
    for (int tile = blockIdx.x; tile < p.n_tiles; tile += gridDim.x) {
        const int sg = tile >> p.log_tiles, x = tile & tile_mask;
        const int k2_0 = x << LOGW;
        const int2 grp = q.groups[sg];                  // (first template of this sky position within the launch, count)
        __syncthreads();                                // the previous tile's last template has taken its inputs (and the twiddles are in place)
        {   // phase A
            const SkyConst &sc = q.skies[sg];
            const double4 *nodes = q.nodes + (int64_t)sg * q.g.n_det * q.g.n_nodes;
#pragma unroll 2
            for (int bb = 0; bb < E; ++bb) {
                const int gi = threadIdx.x + bb * NT;                       // = k1 * W + w
                const int k = ((gi >> LOGW) << p.log_other) + k2_0 + (gi & (C::W - 1));
                float2 ya = make_float2(0.f, 0.f), yb = make_float2(0.f, 0.f);
                if (k < (int)p.n_src) sky_point(q.g, sc, nodes, q.rot, q.Y, q.wslot, k, q.det_mask, ya, yb);
                sS[gi] = make_float4(ya.x, yb.x, ya.y, yb.y);
            }
        }
        __syncthreads();
        for (int tt = 0; tt < grp.y; ++tt) {            // phase B
            const int t = grp.x + tt;
            const TmplDesc td = p.tmpl[t];
            tile_take_inputs<LOGN, LOGT>(a, b, sS);
            spin_down<LOGN, LOGT, E, false, CUBIC>(a, b, p, td, k2_0, RP::r0);
            tile_passes<LOGN, LOGT>(a, b, sX, sm_tw);
            tile_last_pass<LOGN, LOGT>(a, b, sm_tw, p.tw);
            store_columns<LOGN, LOGT, E, AFFINE>(a, b, p, p.T + (int64_t)t * p.n_fft, k2_0, pol_T);
        }
    }
}

// ---------------------------------------------------------------------------------------
// Pass 2: row FFTs of length N2 = 2^LOGN + the 2F combination of eq. 8 (Fig. 1).
// Persistent; tile = (template, W adjacent rows m1) = one contiguous block of T.
// ---------------------------------------------------------------------------------------
// E = register elements per thread: 16, or 32 for the two-pass radix-32 plans (sub-FFT 2^9, 2^10: one trip through
// shared memory instead of two).
// FAFB (debug entry point fstat_debug_compute_fafb only): instead of eq. 8 the epilogue stores the spectra themselves,
// (Re Fa, Im Fa, Re Fb, Im Fb) per bin as one float4 -- the vectors the paper's accuracy tooling compares next to 2F
// (PAPER.md:236); p.twoF then points to float4[n_tmpl][n_bins].  A compile-time variant: the product kernels are unchanged.
template <int LOGN, int LOGT, int E, bool FAFB = false>
__device__ __forceinline__ void pass2_tile_loop(const FftArgs &p, float4 *sm, const float2 *sm_tw, uint64_t *bar, unsigned &parity,
                                                int tile, int tile_end, int stride, int t_off, uint64_t pol_T) {
    using C = FftCfg<LOGN, LOGT, E>;
    using RP = RadixPlan<LOGN, E>;
    constexpr int LOGW = C::LOGW, NT = C::NT, TILE_ELEMS = C::N * C::W;
    if (tile >= tile_end) return;
    float2 a[E], b[E];
    const int tile_mask = (1 << p.log_tiles) - 1;
    int2 tm_next = *reinterpret_cast<const int2 *>(&p.tmpl[tile >> p.log_tiles].sky_slot);      // (sky_slot, bin_off)
    tile_prefetch<LOGN, LOGT>(sm, p.T + (int64_t)((tile >> p.log_tiles) - t_off) * p.n_fft + (int64_t)(tile & tile_mask) * TILE_ELEMS, bar, pol_T);
    for (; tile < tile_end; tile += stride) {
        const int t = tile >> p.log_tiles, x = tile & tile_mask;
        const int m1_0 = x << LOGW;
        const int nxt = tile + stride;
        const SkyABCD *abp = p.abcd + tm_next.x;
        const int boff = tm_next.y;
        const float b_over_d = abp->b_over_d, a_over_d = abp->a_over_d, two_c_over_d = abp->two_c_over_d;
        if (nxt < tile_end) tm_next = *reinterpret_cast<const int2 *>(&p.tmpl[nxt >> p.log_tiles].sky_slot);
        mbar_wait(bar, parity);
        parity ^= 1;
        tile_take_inputs<LOGN, LOGT>(a, b, sm);
        tile_passes<LOGN, LOGT>(a, b, sm, sm_tw);
        if (nxt < tile_end)
            tile_prefetch<LOGN, LOGT>(sm, p.T + (int64_t)((nxt >> p.log_tiles) - t_off) * p.n_fft + (int64_t)(nxt & tile_mask) * TILE_ELEMS, bar, pol_T);
        tile_last_pass<LOGN, LOGT>(a, b, sm_tw, p.tw);
        {   // epilogue: 2F[q], q = m1 + N1*m2 (consecutive lanes -> consecutive m1)
            constexpr int RL = (RP::np == 2) ? RP::r1 : RP::r2;
            constexpr int PL = (RP::np == 2) ? C::P1 : C::P2;
            using PI = PassIdx<RL, PL, LOGN, LOGW, NT, false>;
            // bin q of this template goes to output bin q - boff (boff != 0 only in accumulate mode: the track of one
            // signal through segments with different reference times); q in [lo, lo + span) lands inside the row
            float *__restrict__ out = p.twoF + (int64_t)t * p.twoF_stride - boff;
            float tmax = __int_as_float(0xff800000);
            const int nb = (int)p.n_bins;                       // bins fit 32 bits (n_fft <= 2^24)
            const int lo = max(0, boff);
            const unsigned span = (unsigned)max(0, min(nb, nb + boff) - lo);
            const bool acc = p.accumulate != 0;
            const int q_step = PL << p.log_other;               // out_idx(i, r) is linear in r with slope P
#pragma unroll
            for (int bb = 0; bb < PI::NB; ++bb) {
                int i, w;
                PI::item(bb, i, w);
                int q = (PI::out_idx(i, 0) << p.log_other) + m1_0 + w;
#pragma unroll
                for (int r = 0; r < RL; ++r, q += q_step) {
                    if constexpr (FAFB) {
                        if (q < nb)
                            __stcs(reinterpret_cast<float4 *>(p.twoF) + (int64_t)t * nb + q,
                                   make_float4(a[bb * RL + r].x, b[bb * RL + r].x, a[bb * RL + r].y, b[bb * RL + r].y));
                    } else if ((unsigned)(q - lo) < span) {
                        const float2 fa = make_float2(a[bb * RL + r].x, b[bb * RL + r].x);    // unpack (re, im) of Fa, Fb
                        const float2 fb = make_float2(a[bb * RL + r].y, b[bb * RL + r].y);
                        float twoF = b_over_d * (fa.x * fa.x + fa.y * fa.y) + a_over_d * (fb.x * fb.x + fb.y * fb.y)
                                   - two_c_over_d * (fa.x * fb.x + fa.y * fb.y);
                        if (acc) twoF += __ldcs(out + q);
                        __stcs(out + q, twoF);
                        tmax = fmaxf(tmax, twoF);
                    }
                }
            }
            if (p.gmax) {   // H8: per-warp maximum for the top-k selection (topk_kernels.cuh)
                const uint32_t key = __reduce_max_sync(0xffffffffu, topk_key(tmax));
                if ((threadIdx.x & 31) == 0) p.gmax[(int64_t)tile * (NT / 32) + (threadIdx.x >> 5)] = key;
            }
        }
    }
}

template <int LOGN, int LOGT, int E>
__global__ void __launch_bounds__(FftCfg<LOGN, LOGT, E>::NT, FftCfg<LOGN, LOGT, E>::MIN_CTAS)
fft_pass2_kernel(const __grid_constant__ FftArgs p) {
    extern __shared__ float4 sm[];
    float2 *sm_tw; uint64_t *bar;
    pass_smem_setup<LOGN, LOGT, E>(p, sm, sm_tw, bar);
    unsigned parity = 0;
    pass2_tile_loop<LOGN, LOGT, E>(p, sm, sm_tw, bar, parity, blockIdx.x, p.n_tiles, gridDim.x, 0, l2_policy_evict_first());
}

template <int LOGN, int LOGT, int E>
__global__ void __launch_bounds__(FftCfg<LOGN, LOGT, E>::NT, FftCfg<LOGN, LOGT, E>::MIN_CTAS)
fft_pass2_fafb_kernel(const __grid_constant__ FftArgs p) {
    extern __shared__ float4 sm[];
    float2 *sm_tw; uint64_t *bar;
    pass_smem_setup<LOGN, LOGT, E>(p, sm, sm_tw, bar);
    unsigned parity = 0;
    pass2_tile_loop<LOGN, LOGT, E, true>(p, sm, sm_tw, bar, parity, blockIdx.x, p.n_tiles, gridDim.x, 0, l2_policy_evict_first());
}

// ---------------------------------------------------------------------------------------
// Both passes in ONE cooperative kernel for small transforms (n_fft <= 2^18 and a bank whose intermediates fit L2):
// with two launches per batch the path is launch-bound there (~35 us of ramp-up, tail and launch gap per pair against
// 50-100 us of work).  The CTAs (all resident: cooperative launch) run pass 1 over a group of G templates, meet at a
// grid-wide barrier, run pass 2 over the group, and go on to the next group; the intermediates of two consecutive
// groups alternate between the two halves of a 2 G-template buffer that stays L2-resident (L2 evict_last stores,
// never re-fetched from HBM), so one barrier per group is enough: when a CTA writes half (g+1) % 2 in pass 1 of group
// g+1, every CTA has passed barrier g, i.e. finished pass 2 of group g-1, the last reader of that half.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_barrier(unsigned *counter, unsigned &target) {
    __syncthreads();
    if (threadIdx.x == 0) {
        target += gridDim.x;
        __threadfence();                                  // this CTA's stores of T are visible device-wide before it arrives
        atomicAdd(counter, 1u);
        unsigned seen;
        do { asm volatile("ld.acquire.gpu.global.u32 %0, [%1];\n" : "=r"(seen) : "l"(counter) : "memory"); } while ((int)(seen - target) < 0);
        asm volatile("fence.proxy.async.global;\n" ::: "memory");   // the bulk-copy (async proxy) reads that follow see those stores
    }
    __syncthreads();
}

template <int LOGN1, int LOGN2, int LOGT, int VAR>
struct SingleCfg {
    using C1 = FftCfg<LOGN1, LOGT, 16>;
    using C2 = FftCfg<LOGN2, LOGT, 16>;
    static constexpr int BUF = C1::BUF_ELEMS > C2::BUF_ELEMS ? C1::BUF_ELEMS : C2::BUF_ELEMS;
    static constexpr int SMEM_CORE = BUF * 16 + (C1::TW_SMEM_ENTRIES + C2::TW_SMEM_ENTRIES) * 8 + 16;
    static constexpr int SMEM_BYTES = SMEM_CORE + C1::P1_STAGE_ELEMS * 16;
    static constexpr int MIN_CTAS = (228 * 1024 / (SMEM_BYTES + 1024)) > 5 ? 5 : (228 * 1024 / (SMEM_BYTES + 1024));
};

template <int LOGN1, int LOGN2, int LOGT, int VAR>
__global__ void __launch_bounds__(FftCfg<LOGN1, LOGT, 16>::NT, SingleCfg<LOGN1, LOGN2, LOGT, VAR>::MIN_CTAS)
fft_single_kernel(const __grid_constant__ SingleArgs q) {
    using SC = SingleCfg<LOGN1, LOGN2, LOGT, VAR>;
    extern __shared__ float4 sm[];
    float2 *tw1 = reinterpret_cast<float2 *>(sm + SC::BUF), *tw2 = tw1 + SC::C1::TW_SMEM_ENTRIES;
    uint64_t *bar = reinterpret_cast<uint64_t *>(tw2 + SC::C2::TW_SMEM_ENTRIES);
    for (int e = threadIdx.x; e < SC::C1::TW_SMEM_ENTRIES; e += SC::C1::NT) tw1[e] = q.p1.tw[e];
    for (int e = threadIdx.x; e < SC::C2::TW_SMEM_ENTRIES; e += SC::C1::NT) tw2[e] = q.p2.tw[e];
    if (threadIdx.x == 0) { mbar_init(bar, 1); fence_proxy_async(); }
    __syncthreads();
    unsigned parity = 0, target = 0;
    const uint64_t pol_keep = l2_policy_evict_last();
    const int tiles1 = 1 << q.p1.log_tiles, tiles2 = 1 << q.p2.log_tiles;
    for (int g = 0, t0 = 0; t0 < q.n_tmpl; ++g, t0 += q.group) {
        const int t1 = min(t0 + q.group, q.n_tmpl);
        const int t_off = t0 - (g & 1) * q.group;            // template t of this group lives at T[t - t_off]
        pass1_tile_loop<LOGN1, LOGT, 16, VAR>(q.p1, sm, FFT_P1_DB ? reinterpret_cast<float4 *>(reinterpret_cast<char *>(sm) + SC::SMEM_CORE) : sm, tw1, bar, parity, t0 * tiles1 + (int)blockIdx.x, t1 * tiles1, (int)gridDim.x, t_off, pol_keep, pol_keep);
        grid_barrier(q.counter, target);
        pass2_tile_loop<LOGN2, LOGT, 16>(q.p2, sm, tw2, bar, parity, t0 * tiles2 + (int)blockIdx.x, t1 * tiles2, (int)gridDim.x, t_off, pol_keep);
    }
}

// kernel pointer by (sub-FFT, tile, pass, elements, padding variant)
template <int LOGN, int LOGT, bool P2, int E, int VAR>
inline void (*fft_kernel_ptr())(const FftArgs) {
    if constexpr (P2 && (VAR & FFT_VAR_FAFB) != 0) return fft_pass2_fafb_kernel<LOGN, LOGT, E>;
    else if constexpr (P2) return fft_pass2_kernel<LOGN, LOGT, E>;
    else return fft_pass1_kernel<LOGN, LOGT, E, VAR>;
}
