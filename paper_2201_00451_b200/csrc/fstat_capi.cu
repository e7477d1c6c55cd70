// C-ABI of the B200 resampling F-statistic path (include/fstat.h): plan management and
// kernel orchestration.  All arithmetic of the path runs in the kernels of sky_kernels.cuh,
// fft_kernels.cuh and topk_kernels.cuh; the host only derives O(n_det) per-sky constants.
#include "../../include/fstat.h"
#include "../../include/fstat_debug.h"
#include "fstat_common.cuh"
#include "sky_kernels.cuh"
#include "fft_launch.cuh"
#include "topk_kernels.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

namespace {

thread_local std::string g_setup_error;

struct SkyGroup { double alpha, delta; int first, count; };

struct HostRing {            // device row buffers for the *_host variants
    float *buf[2] = {nullptr, nullptr};
    cudaEvent_t done[2] = {nullptr, nullptr};   // D2H of that buffer finished
    int64_t rows = 0;
};

}  // namespace

#define STAGE_SLOTS 4

struct fstat_plan {
    PlanGeom g{};
    cudaStream_t stream = nullptr;
    cudaStream_t copy_stream = nullptr;
    fstat_detector_t det[FSTAT_MAX_DET];
    fstat_ephem_t eph{};
    double f_min = 0, band = 0, df = 0;
    int device = 0;
    int n_sm = 148;
    size_t mem_total = 0;                            // device memory (cudaMemGetInfo at setup): scales the default buffer caps
    // device memory
    float2 *d_series = nullptr;
    void *d_tmp[3] = {nullptr, nullptr, nullptr};   // setup-time scratch (freed by destroy_impl if setup fails half-way)
    float2 *d_rot = nullptr;          // [n_src] cos, sin of the Greenwich sidereal angle per SSB grid point
    double4 *d_nodes = nullptr; size_t nodes_cap = 0;   // timing nodes of the sky positions of one batch [nodes_cap][n_det][n_nodes]
    float2 *d_farrow = nullptr;       // [n_det][y_det_stride] float4: Farrow-filtered series (sky_math.cuh farrow_index)
    float *d_wslot = nullptr;
    float2 *d_tw1 = nullptr, *d_tw2 = nullptr;
    float4 *d_S = nullptr;   int n_sky_slots = 0, max_sky_slots = 1;   // S buffers: allocated / allowed (grown on demand)
    float4 *d_T = nullptr;   int n_inflight = 0;   // four-step intermediates of the templates of one launch
    int t_cap = 0;                                 // templates d_T currently holds (grown on demand up to n_inflight)
    SkyConst *d_sky = nullptr; size_t sky_cap = 0;
    SkyABCD *d_abcd = nullptr; SkyABCD *h_abcd = nullptr;   // per sky group of the current call (capacity sky_cap)
    int2 *d_grp = nullptr; int2 *h_grp = nullptr;           // fused path: (first template within its launch, count) per sky group
    double mom[FSTAT_MAX_DET][MOM_TERMS];                   // antenna moment matrices M_X (sky_kernels.cuh)
    bool pending_edom = false;                              // a template since the last sync had D <= 0
    int force_fused_sky = -1, force_single = -1;            // fstat_debug_set_paths
    bool chunk_one_sky = false;                             // the launch being issued holds templates of one sky position only
    unsigned *d_counter = nullptr;                          // grid barrier of the single-kernel form
    TmplDesc *d_tmpl = nullptr; size_t tmpl_cap = 0;
    float *d_rows = nullptr;          // top-k scratch rows [n_inflight][n_bins]
    uint32_t *d_gmax = nullptr;       // top-k: per-group maxima of the rows in flight [n_inflight][n_groups]
    uint32_t *d_gmax_lin = nullptr;   // fstat_select_*: per-group maxima of caller rows (linear groups)
    HostRing ring;
    float *d_topk_v = nullptr; int *d_topk_i = nullptr; size_t topk_cap = 0;
    // pinned staging
    SkyConst *h_sky = nullptr; TmplDesc *h_tmpl = nullptr;
    // pinned staging comes in STAGE_SLOTS rotating slots (each of capacity tmpl_cap / sky_cap), so that a call does not
    // have to wait for the previous call's GPU work before it can prepare its descriptors
    cudaEvent_t staging_ev[4] = {nullptr, nullptr, nullptr, nullptr}; int stage_slot = 0;
    cudaEvent_t chunk_ev = nullptr;
    int64_t launches = 0;
    std::string err;
    // optional per-kernel-class timing (fstat_set_profile)
    bool profile = false;
    std::vector<cudaEvent_t> ev_pool; size_t ev_used = 0;
    struct Seg { int cls; size_t e0, e1; int launches; };
    std::vector<Seg> segs;
};

namespace {

#define CUDA_TRY(plan, expr)                                                                          \
    do {                                                                                              \
        cudaError_t e__ = (expr);                                                                     \
        if (e__ != cudaSuccess) {                                                                     \
            (plan)->err = std::string(#expr) + ": " + cudaGetErrorString(e__);                        \
            return FSTAT_ECUDA;                                                                       \
        }                                                                                             \
    } while (0)

int fail(fstat_plan *p, int code, const std::string &msg) {
    if (p) p->err = msg; else g_setup_error = msg;
    return code;
}

// profiling: bracket a group of launches of one class with two events on the plan's stream
size_t prof_mark(fstat_plan *p) {
    if (p->ev_used == p->ev_pool.size()) {
        cudaEvent_t e; cudaEventCreate(&e); p->ev_pool.push_back(e);
    }
    cudaEventRecord(p->ev_pool[p->ev_used], p->stream);
    return p->ev_used++;
}
struct ProfScope {
    fstat_plan *p; int cls; size_t e0; int64_t l0;
    ProfScope(fstat_plan *pl, int c) : p(pl), cls(c), e0(0), l0(pl->launches) { if (p->profile) e0 = prof_mark(p); }
    ~ProfScope() { if (p->profile) { size_t e1 = prof_mark(p); p->segs.push_back({cls, e0, e1, (int)(p->launches - l0)}); } }
};

// pass 1 takes the template-fastest tile order when one sky position's series exceeds this many bytes (measured on B200)
#ifndef FSTAT_TFAST_MIN_BYTES
#define FSTAT_TFAST_MIN_BYTES (96ll << 20)
#endif

int ilog2(int64_t v) { int l = 0; while ((int64_t(1) << l) < v) ++l; return l; }

// radix list of fft_kernels.cuh RadixPlan<LOGN>
std::vector<int> radix_list(int logn, int elems = 16) {
    if (elems == 32) return logn == 9 ? std::vector<int>{32, 16} : std::vector<int>{32, 32};     // RadixPlan<9|10, 32>
    switch (logn) {
        case 6: return {8, 8};
        case 7: return {16, 8};
        case 8: return {16, 16};
        case 9: return {8, 8, 8};
        case 10: return {16, 16, 4};
        case 11: return {16, 16, 8};
        default: return {16, 16, 16};
    }
}

// Twiddles of passes s >= 1: entry [(r-1)*P + k] = exp(-2 pi i r k / (P R)).
std::vector<float2> make_twiddles(int logn, int elems = 16) {
    std::vector<float2> tw;
    const std::vector<int> rl = radix_list(logn, elems);
    int P = rl[0];
    for (size_t s = 1; s < rl.size(); ++s) {
        const int R = rl[s];
        for (int r = 1; r < R; ++r)
            for (int k = 0; k < P; ++k) {
                const double ang = -2.0 * M_PI * (double)r * (double)k / ((double)P * (double)R);
                tw.push_back(make_float2((float)cos(ang), (float)sin(ang)));
            }
        P *= R;
    }
    return tw;
}

// Farrow coefficients (sky_kernels.cuh): c_m(d) = sinc(d-m) [0.54 + 0.46 cos(pi (d-m)/(D+1/2))] on d in [-1/2, 1/2]
// as sum_p a[m][p] d^p: Chebyshev interpolation at FARROW_NC nodes in t = 2d, converted to powers of d.  fp64.
std::vector<float> farrow_coefficients(int dterms) {
    const int Q = FARROW_NC;
    std::vector<float> out((size_t)(2 * dterms + 1) * Q);
    // T_k(t) as polynomials in t
    std::vector<std::vector<double>> Tk(Q, std::vector<double>(Q, 0.0));
    Tk[0][0] = 1.0;
    if (Q > 1) Tk[1][1] = 1.0;
    for (int k = 2; k < Q; ++k)
        for (int e = 0; e < Q; ++e) Tk[k][e] = (e > 0 ? 2.0 * Tk[k - 1][e - 1] : 0.0) - Tk[k - 2][e];
    for (int m = -dterms; m <= dterms; ++m) {
        double fv[FARROW_NC], ck[FARROW_NC];
        for (int i = 0; i < Q; ++i) {
            const double d = 0.5 * cos(M_PI * (i + 0.5) / Q), v = d - m;
            const double sinc = (fabs(v) < 1e-12) ? 1.0 : sin(M_PI * v) / (M_PI * v);
            fv[i] = sinc * (0.54 + 0.46 * cos(M_PI * v / (dterms + 0.5)));
        }
        for (int k = 0; k < Q; ++k) {
            double acc = 0.0;
            for (int i = 0; i < Q; ++i) acc += fv[i] * cos(M_PI * k * (i + 0.5) / Q);
            ck[k] = (k == 0 ? 1.0 : 2.0) * acc / Q;
        }
        double pw = 1.0;                                     // t^e = (2d)^e
        for (int e = 0; e < Q; ++e, pw *= 2.0) {
            double a = 0.0;
            for (int k = e; k < Q; ++k) a += ck[k] * Tk[k][e];
            out[(size_t)(m + dterms) * Q + e] = (float)(a * pw);
        }
    }
    return out;
}

void fill_sky_const(const fstat_plan *p, double alpha, double delta, SkyConst *sc) {
    const fstat_ephem_t &e = p->eph;
    const double nx = cos(delta) * cos(alpha), ny = cos(delta) * sin(alpha), nz = sin(delta);
    sc->Pc = e.au_over_c_s * nx;
    sc->Ps = e.au_over_c_s * (ny * cos(e.obliquity_rad) + nz * sin(e.obliquity_rad));
    for (int X = 0; X < p->g.n_det; ++X) {
        const fstat_detector_t &d = p->det[X];
        const double lam = d.lat_rad, L = d.lon_east_rad, gam = d.xarm_azimuth_rad + 0.75 * M_PI;
        sc->Qc[X] = e.re_over_c_s * cos(lam) * (nx * cos(L) + ny * sin(L));
        sc->Qs[X] = e.re_over_c_s * cos(lam) * (ny * cos(L) - nx * sin(L));
        sc->Q0[X] = e.re_over_c_s * nz * sin(lam);
        sc->cal[X] = (float)cos(alpha - L);
        sc->sal[X] = (float)sin(alpha - L);
        const double s2g = sin(2 * gam), c2g = cos(2 * gam);
        sc->ac[X][0] = (float)(0.75 * s2g * cos(lam) * cos(lam) * cos(delta) * cos(delta));
        sc->ac[X][1] = (float)(s2g * (3.0 - cos(2 * lam)) * (3.0 - cos(2 * delta)) / 16.0);
        sc->ac[X][2] = (float)(-0.25 * c2g * sin(lam) * (3.0 - cos(2 * delta)));
        sc->ac[X][3] = (float)(0.25 * s2g * sin(2 * lam) * sin(2 * delta));
        sc->ac[X][4] = (float)(-0.5 * c2g * cos(lam) * sin(2 * delta));
        sc->bc[X][0] = (float)(c2g * sin(lam) * sin(delta));
        sc->bc[X][1] = (float)(0.25 * s2g * (3.0 - cos(2 * lam)) * sin(delta));
        sc->bc[X][2] = (float)(c2g * cos(lam) * cos(delta));
        sc->bc[X][3] = (float)(0.5 * s2g * sin(2 * lam) * cos(delta));
    }
}

// A, B, C, D of one sky position from the moment matrices: A = sum_X alpha_X^T M_X alpha_X etc., with
// alpha_X, beta_X the coefficients of a_X(t), b_X(t) in the basis (1, cos 2th, sin 2th, cos th, sin th).
void sky_abcd(const fstat_plan *p, double alpha, double delta, SkyABCD *out, uint32_t det_mask = 0xffffffffu) {
    double A = 0, B = 0, C = 0;
    const double C1 = cos(alpha), S1 = sin(alpha), C2 = cos(2 * alpha), S2 = sin(2 * alpha);
    for (int X = 0; X < p->g.n_det; ++X) {
        if (!((det_mask >> X) & 1u)) continue;
        const fstat_detector_t &d = p->det[X];
        const double lam = d.lat_rad, gam = d.xarm_azimuth_rad + 0.75 * M_PI;
        const double s2g = sin(2 * gam), c2g = cos(2 * gam);
        const double ac0 = 0.75 * s2g * cos(lam) * cos(lam) * cos(delta) * cos(delta);
        const double ac1 = s2g * (3.0 - cos(2 * lam)) * (3.0 - cos(2 * delta)) / 16.0;
        const double ac2 = -0.25 * c2g * sin(lam) * (3.0 - cos(2 * delta));
        const double ac3 = 0.25 * s2g * sin(2 * lam) * sin(2 * delta);
        const double ac4 = -0.5 * c2g * cos(lam) * sin(2 * delta);
        const double bc0 = c2g * sin(lam) * sin(delta);
        const double bc1 = 0.25 * s2g * (3.0 - cos(2 * lam)) * sin(delta);
        const double bc2 = c2g * cos(lam) * cos(delta);
        const double bc3 = 0.5 * s2g * sin(2 * lam) * cos(delta);
        // h = alpha - th:  cos 2h = C2 cos 2th + S2 sin 2th,  sin 2h = S2 cos 2th - C2 sin 2th, same for h
        const double av[5] = {ac0, ac1 * C2 + ac2 * S2, ac1 * S2 - ac2 * C2, ac3 * C1 + ac4 * S1, ac3 * S1 - ac4 * C1};
        const double bv[5] = {0.0, bc0 * C2 + bc1 * S2, bc0 * S2 - bc1 * C2, bc2 * C1 + bc3 * S1, bc2 * S1 - bc3 * C1};
        double M[5][5];
        int q = 0;
        for (int r = 0; r < 5; ++r)
            for (int cc = r; cc < 5; ++cc) { M[r][cc] = M[cc][r] = p->mom[X][q++]; }
        for (int r = 0; r < 5; ++r)
            for (int cc = 0; cc < 5; ++cc) {
                A += av[r] * M[r][cc] * av[cc];
                B += bv[r] * M[r][cc] * bv[cc];
                C += av[r] * M[r][cc] * bv[cc];
            }
    }
    out->A = A; out->B = B; out->C = C; out->D = A * B - C * C;
    out->bad = !(out->D > 0.0);
    if (out->bad) {
        out->b_over_d = out->a_over_d = out->two_c_over_d = std::nanf("");
    } else {
        out->b_over_d = (float)(B / out->D); out->a_over_d = (float)(A / out->D); out->two_c_over_d = (float)(2.0 * C / out->D);
    }
}

// n_fft = 2^log_n1 x 2^log_n2 and the tile sizes of the two FFT passes, per size as measured on B200
// (DESIGN.md 5 "How n_fft is split").  Pass 2 gets the shorter transform: its tile then spans more rows, which is what
// makes the runs of its transposed 2F store long (W2 x 4 bytes); pass 1 is fastest at <= 2^10 points with
// 2^11-element tiles.
void default_geometry(int L, PlanGeom &g) {
    g.log_n2 = L <= 14 ? L / 2 : L == 15 ? 6 : L == 16 ? 7 : L <= 18 ? 8 : L == 19 ? 9 : L <= 21 ? 10 : L == 22 ? 10 : L - 12;
    g.log_n1 = L - g.log_n2;
    // pass 2: 2^12-element tiles; 2^13 (8 rows of 2^10 points: 128-byte runs in pass 1's transposed store, 32-byte
    // runs of 2F) for n_fft >= 2^21, where the gain in pass 1 outweighs the single CTA per SM in pass 2; likewise 4 rows
    // of 2^11 points at 2^23, which lets pass 1 run one 2^12-point column per 2^12-element tile
    g.log_tile2 = (g.log_n2 == 12 || (g.log_n2 == 10 && L >= 21) || (g.log_n2 == 11 && L == 23)) ? 13 : 12;
    // pass 1: the smallest tile (most CTAs per SM) whose transposed store still writes >= 64-byte runs: a tile
    // of a single column needs >= 4 rows per pass-2 tile
    const int w2_rows = 1 << (g.log_tile2 - g.log_n2);
    // 2^9 / 2^10-point columns: one warp per 2^10-element tile, 32 register elements per thread (two radix passes, no block barrier)
    g.log_tile1 = (g.log_n1 == 9 || g.log_n1 == 10) ? 10 : g.log_n1 <= 10 ? 11 : (w2_rows >= 4 ? g.log_n1 : g.log_n1 + 1);
    // pass 2 with 32 register elements per thread (two radix-32 passes, one trip through shared memory) for
    // sub-FFTs of 2^9 and 2^10 points on 2^12-element (2^10 also 2^13-element) tiles
    g.p2_elems = (((g.log_n2 == 9 || g.log_n2 == 10) && g.log_tile2 == 12) || (g.log_n2 == 10 && g.log_tile2 == 13)) ? 32 : 16;
    g.p1_elems = g.log_tile1 == 10 ? 32 : 16;
    g.log_w1 = g.log_tile1 - g.log_n1; g.log_w2 = g.log_tile2 - g.log_n2;
}

// pass-1 kernel variant for the plan's geometry: columns that are at least half zero padding take the variant that
// neither stages nor touches the padding (where one is instantiated); a pass-2 tile with more rows than the last radix
// pass of pass 1 has butterflies needs the general store address; cubic = the launch holds templates with fddot != 0
int pass1_variant(const PlanGeom &g, bool cubic) {
    const std::vector<int> rl = radix_list(g.log_n1, g.p1_elems);
    const int ni_last = (1 << g.log_n1) / rl.back();
    int var = (cubic ? FFT_VAR_CUBIC : 0) | ((ni_last >> g.log_w2) == 0 ? FFT_VAR_GENERIC : 0);
    if (2 * g.n_src <= g.n_fft && fft_find_kernel(1, g.log_n1, g.log_tile1, g.p1_elems, var | FFT_VAR_SKIPZ)) var |= FFT_VAR_SKIPZ;
    return var;
}
bool geometry_supported(const PlanGeom &g) {
    return fft_find_kernel(1, g.log_n1, g.log_tile1, g.p1_elems, pass1_variant(g, false)) && fft_find_kernel(1, g.log_n1, g.log_tile1, g.p1_elems, pass1_variant(g, true))
        && fft_find_kernel(2, g.log_n2, g.log_tile2, g.p2_elems, 0);
}

// (re)upload the Stockham twiddle tables of the plan's current geometry
int upload_twiddles(fstat_plan *p) {
    const std::vector<float2> tw1 = make_twiddles(p->g.log_n1, p->g.p1_elems), tw2 = make_twiddles(p->g.log_n2, p->g.p2_elems);
    cudaFree(p->d_tw1); cudaFree(p->d_tw2); p->d_tw1 = p->d_tw2 = nullptr;
    CUDA_TRY(p, cudaMalloc(&p->d_tw1, tw1.size() * sizeof(float2)));
    CUDA_TRY(p, cudaMalloc(&p->d_tw2, tw2.size() * sizeof(float2)));
    CUDA_TRY(p, cudaMemcpyAsync(p->d_tw1, tw1.data(), tw1.size() * sizeof(float2), cudaMemcpyHostToDevice, p->stream));
    CUDA_TRY(p, cudaMemcpyAsync(p->d_tw2, tw2.data(), tw2.size() * sizeof(float2), cudaMemcpyHostToDevice, p->stream));
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));      // the host vectors go out of scope
    return FSTAT_OK;
}

// log2 of the tile size used for a sub-FFT of length 2^logn under the plan's tile setting
int tile_log2(const fstat_plan *p) { return p->g.log_tile2; }

// FFT + 2F for templates [t0, t0+nt) of the current call (descriptors already on the device).
// fused_ng > 0: the templates are those of sky groups [g0, g0 + fused_ng), whose timing nodes are in d_nodes; pass 1 runs as
// the fused sky + pass-1 kernel (no resampled series in global memory).  Otherwise pass 1 reads the S slots of the batch.
// How the single-kernel form would group nt templates: 0 = not applicable (no kernel for the geometry, or the bank is
// so long that the two-launch form is faster: more than 4 groups).  A group's intermediates take at most 48 MB, so
// that two groups stay L2-resident.
int single_group_size(fstat_plan *p, int nt, bool cubic) {
    // opt-in only (fstat_debug_set_paths(single = 1) on a plan whose passes both use 2^11-element tiles): measured on B200
    // the single-kernel form is never faster than two launches (the passes are bound on the SM side, so
    // L2 residency of the intermediate buys nothing and every grid barrier adds a tail)
    if (p->force_single <= 0 || p->g.log_tile1 != 11 || p->g.log_tile2 != 11 || p->g.p2_elems != 16) return 0;
    if (!fft_find_single_kernel(p->g.log_n1, p->g.log_n2, pass1_variant(p->g, cubic) & ~FFT_VAR_SKIPZ)) return 0;
    const int cap = (int)std::max<int64_t>(1, (48ll << 20) / (p->g.n_fft * 16));
    if (nt <= cap) return nt;
    const int n_groups = (nt + cap - 1) / cap;
    return (nt + n_groups - 1) / n_groups;                  // equal groups
}

int launch_fft_chunk(fstat_plan *p, int g0, int t0, int nt, float *rows, int64_t row_stride, bool cubic, uint32_t *gmax = nullptr,
                     bool accumulate = false, int fused_ng = 0, uint32_t det_mask = 0xffffffffu, bool fafb = false) {
    const int single_group = (fused_ng > 0 || fafb) ? 0 : single_group_size(p, nt, cubic);
    const int t_need = single_group > 0 ? std::min(nt, 2 * single_group) : nt;
    if (t_need > p->t_cap) {       // grow the intermediate buffer to the launch size actually used
        CUDA_TRY(p, cudaStreamSynchronize(p->stream));
        cudaFree(p->d_T); p->d_T = nullptr; p->t_cap = 0;
        if (cudaMalloc(&p->d_T, (size_t)t_need * p->g.n_fft * sizeof(float4)) != cudaSuccess) { cudaGetLastError(); return fail(p, FSTAT_ENOMEM, "device allocation of the FFT intermediates failed"); }
        p->t_cap = t_need;
    }
    FftArgs a{};
    a.S = p->d_S; a.T = p->d_T; a.tmpl = p->d_tmpl + t0; a.abcd = p->d_abcd + g0;
    a.twoF = rows; a.twoF_stride = row_stride; a.gmax = gmax; a.accumulate = accumulate ? 1 : 0;
    a.n_fft = p->g.n_fft; a.n_src = p->g.n_src; a.n_bins = p->g.n_bins; a.k_margin = p->g.k_margin;
    a.dt = p->g.dt;
    const int l1 = p->g.log_n1, l2 = p->g.log_n2;
    const LaunchCtx ctx{p->stream, p->device, p->n_sm};
    a.tw = p->d_tw1; a.log_other = l2; a.log_w_other = p->g.log_w2;
    const int tiles1 = 1 << (l2 - p->g.log_w1);
    if (single_group > 0) {
        // both passes in one cooperative kernel, groups of single_group templates through an L2-resident buffer
        ProfScope ps(p, 5);
        const single_launch_fn f = fft_find_single_kernel(l1, l2, pass1_variant(p->g, cubic) & ~FFT_VAR_SKIPZ);
        if (!f) return fail(p, FSTAT_ESIZE, "no single-kernel form for this geometry");
        if (!p->d_counter) CUDA_TRY(p, cudaMalloc(&p->d_counter, sizeof(unsigned)));
        CUDA_TRY(p, cudaMemsetAsync(p->d_counter, 0, sizeof(unsigned), p->stream));
        SingleArgs sa{};
        sa.p1 = a; sa.p1.log_tiles = ilog2(tiles1); sa.p1.n_tiles = tiles1 * nt;
        sa.p2 = a; sa.p2.tw = p->d_tw2; sa.p2.log_other = l1; sa.p2.log_w_other = p->g.log_w1;
        const int tiles2 = 1 << (l1 - p->g.log_w2);
        sa.p2.log_tiles = ilog2(tiles2); sa.p2.n_tiles = tiles2 * nt;
        sa.n_tmpl = nt; sa.group = single_group; sa.counter = p->d_counter;
        CUDA_TRY(p, f(ctx, sa, nullptr));
        ++p->launches;
        CUDA_TRY(p, cudaGetLastError());
        return FSTAT_OK;
    }
    if (fused_ng > 0) {
        ProfScope ps(p, 4);
        const fused_launch_fn f = fft_find_fused_kernel(l1, p->g.log_tile1, pass1_variant(p->g, cubic) & ~FFT_VAR_SKIPZ);
        if (!f) return fail(p, FSTAT_ESIZE, "no fused sky + pass-1 kernel for this geometry");
        FusedArgs fa{};
        fa.f = a; fa.g = p->g; fa.skies = p->d_sky + g0; fa.nodes = p->d_nodes; fa.rot = p->d_rot; fa.Y = p->d_farrow;
        fa.wslot = p->d_wslot; fa.groups = p->d_grp + g0; fa.det_mask = det_mask;
        CUDA_TRY(p, f(ctx, fa, tiles1, fused_ng));
        ++p->launches;
    } else {
        ProfScope ps(p, 1);
        const fft_launch_fn f = fft_find_kernel(1, l1, p->g.log_tile1, p->g.p1_elems, pass1_variant(p->g, cubic));
        if (!f) return fail(p, FSTAT_ESIZE, "unsupported (sub-FFT, tile) combination in FFT pass 1");
        // the series of one sky position no longer stays in L2 for the length of a template: template fastest in the tile order
        a.t_fast = p->chunk_one_sky && 16 * p->g.n_src > (int64_t)FSTAT_TFAST_MIN_BYTES;
        CUDA_TRY(p, f(ctx, a, tiles1, nt));
        ++p->launches;
        a.t_fast = 0;
    }
    a.tw = p->d_tw2; a.log_other = l1; a.log_w_other = p->g.log_w1;
    {
        ProfScope ps(p, 2);
        const int tiles2 = 1 << (l1 - p->g.log_w2);
        const fft_launch_fn f = fft_find_kernel(2, l2, p->g.log_tile2, p->g.p2_elems, fafb ? FFT_VAR_FAFB : 0);
        if (!f) return fail(p, FSTAT_ESIZE, fafb ? "no (Fa, Fb) variant of FFT pass 2 for this geometry (default shapes up to n_fft 2^22 only)"
                                                 : "unsupported (sub-FFT, tile) combination in FFT pass 2");
        CUDA_TRY(p, f(ctx, a, tiles2, nt));
        ++p->launches;
    }
    CUDA_TRY(p, cudaGetLastError());
    return FSTAT_OK;
}

// Sky-dependent kernel for sky groups [g0, g0+ng) -> S slots 0..ng-1.
// room for the timing nodes of n sky positions
int ensure_nodes(fstat_plan *p, size_t n) {
    if (n <= p->nodes_cap) return FSTAT_OK;
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    cudaFree(p->d_nodes); p->d_nodes = nullptr; p->nodes_cap = 0;
    if (cudaMalloc(&p->d_nodes, n * p->g.n_det * p->g.n_nodes * sizeof(double4)) != cudaSuccess) { cudaGetLastError(); return fail(p, FSTAT_ENOMEM, "device allocation of the timing nodes failed"); }
    p->nodes_cap = n;
    return FSTAT_OK;
}

// H1 at the timing nodes of sky groups [g0, g0+ng) -> d_nodes[0..ng)
int launch_timing_nodes(fstat_plan *p, int g0, int ng) {
    const PlanGeom &g = p->g;
    int rc = ensure_nodes(p, ng);
    if (rc) return rc;
    timing_nodes_kernel<<<dim3((unsigned)((g.n_nodes + NODE_THREADS - 1) / NODE_THREADS), g.n_det, ng), NODE_THREADS, 0, p->stream>>>(g, p->d_sky + g0, p->d_nodes);
    p->launches += 1;
    CUDA_TRY(p, cudaGetLastError());
    return FSTAT_OK;
}

int launch_sky_batch(fstat_plan *p, int g0, int ng, float4 *S_dst, int blocked, uint32_t det_mask = 0xffffffffu) {
    const PlanGeom &g = p->g;
    ProfScope ps(p, 0);
    int rc = launch_timing_nodes(p, g0, ng);
    if (rc) return rc;
    // patches of 32 adjacent k2 x 32 adjacent k1 (k = N2 k1 + k2) over the rows that hold data
    const int64_t rows_src = (g.n_src + ((int64_t)1 << g.log_n2) - 1) >> g.log_n2;
    const int n_patches = (int)((rows_src + SKY_PATCH - 1) / SKY_PATCH) << (g.log_n2 - 5);
    // sky position fastest when the Farrow-filtered series would not stay in L2 between sky positions
    const int sky_major = ng > 1 && (size_t)g.n_det * (size_t)g.y_det_stride * sizeof(float4) > ((size_t)48 << 20);
    sky_resample_kernel<<<(unsigned)n_patches * (unsigned)ng, SKY_THREADS, 0, p->stream>>>(g, p->d_sky + g0, p->d_nodes, p->d_rot, p->d_farrow, p->d_wslot, S_dst, blocked, det_mask, ng, n_patches, sky_major);
    p->launches += 1;
    CUDA_TRY(p, cudaGetLastError());
    return FSTAT_OK;
}

int ensure_tmpl_capacity(fstat_plan *p, size_t n_tmpl, size_t n_groups) {
    if (n_tmpl > p->tmpl_cap || n_groups > p->sky_cap) CUDA_TRY(p, cudaStreamSynchronize(p->stream));   // staging in flight
    if (n_tmpl > p->tmpl_cap) {
        if (p->d_tmpl) cudaFree(p->d_tmpl);
        if (p->h_tmpl) cudaFreeHost(p->h_tmpl);
        p->d_tmpl = nullptr; p->h_tmpl = nullptr; p->tmpl_cap = 0;
        const size_t cap = n_tmpl + n_tmpl / 2 + 16;
        CUDA_TRY(p, cudaMalloc(&p->d_tmpl, cap * sizeof(TmplDesc)));
        CUDA_TRY(p, cudaMallocHost(&p->h_tmpl, STAGE_SLOTS * cap * sizeof(TmplDesc)));
        p->tmpl_cap = cap;
    }
    if (n_groups > p->sky_cap) {
        if (p->d_sky) cudaFree(p->d_sky);
        if (p->h_sky) cudaFreeHost(p->h_sky);
        if (p->d_abcd) cudaFree(p->d_abcd);
        if (p->h_abcd) cudaFreeHost(p->h_abcd);
        if (p->d_grp) cudaFree(p->d_grp);
        if (p->h_grp) cudaFreeHost(p->h_grp);
        p->d_sky = nullptr; p->h_sky = nullptr; p->d_abcd = nullptr; p->h_abcd = nullptr; p->d_grp = nullptr; p->h_grp = nullptr; p->sky_cap = 0;
        const size_t cap = n_groups + n_groups / 2 + 16;
        CUDA_TRY(p, cudaMalloc(&p->d_sky, cap * sizeof(SkyConst)));
        CUDA_TRY(p, cudaMallocHost(&p->h_sky, STAGE_SLOTS * cap * sizeof(SkyConst)));
        CUDA_TRY(p, cudaMalloc(&p->d_abcd, cap * sizeof(SkyABCD)));
        CUDA_TRY(p, cudaMallocHost(&p->h_abcd, STAGE_SLOTS * cap * sizeof(SkyABCD)));
        CUDA_TRY(p, cudaMalloc(&p->d_grp, cap * sizeof(int2)));
        CUDA_TRY(p, cudaMallocHost(&p->h_grp, STAGE_SLOTS * cap * sizeof(int2)));
        p->sky_cap = cap;
    }
    return FSTAT_OK;
}

enum OutMode { OUT_DEV_ROWS, OUT_HOST_ROWS, OUT_TOPK };

struct OutSpec {
    OutMode mode;
    float *rows = nullptr;       // device (OUT_DEV_ROWS) or host (OUT_HOST_ROWS) [n_tmpl][n_bins]
    int k = 0;
    float *val = nullptr;        // device [n_tmpl][k]
    int32_t *bin = nullptr;
    float thr = 0.f;             // threshold mode (count != null): only bins with 2F > thr
    int32_t *count = nullptr;    // device [n_tmpl]
    bool accumulate = false;     // OUT_DEV_ROWS: rows += 2F (semi-coherent sum)
    const int32_t *bin_off = nullptr;   // accumulate: host [n_tmpl] bin offsets (null = 0)
    uint32_t det_mask = 0xffffffffu;    // detectors that take part
    bool fafb = false;           // OUT_DEV_ROWS: rows is float4[n_tmpl][n_bins] = (Fa, Fb) per bin instead of 2F (debug)
};

// groups of 512 bins (one warp of a pass-2 tile each) per row, and how pass 2 maps them to bins
TopkGeom topk_geom(const fstat_plan *p) {
    const int l2 = p->g.log_n2, lt = tile_log2(p);
    const std::vector<int> rl = radix_list(l2, p->g.p2_elems);
    TopkGeom tg{};
    tg.elems = p->g.p2_elems;
    tg.nt = (1 << lt) / tg.elems;
    tg.log_w = lt - l2;
    tg.log_rl = ilog2(rl.back());
    tg.pl = 1;
    for (size_t i = 0; i + 1 < rl.size(); ++i) tg.pl *= rl[i];
    tg.log_other = p->g.log_n1;
    tg.n_groups = (int)(p->g.n_fft >> lt) * (tg.nt / 32);
    tg.linear = 0;
    return tg;
}

int ensure_topk_scratch(fstat_plan *p) {
    const int64_t nb = p->g.n_bins;
    if (!p->d_rows) CUDA_TRY(p, cudaMalloc(&p->d_rows, (size_t)p->n_inflight * nb * sizeof(float)));
    if (!p->d_gmax) {
        const TopkGeom tg = topk_geom(p);
        CUDA_TRY(p, cudaMalloc(&p->d_gmax, (size_t)p->n_inflight * tg.n_groups * sizeof(uint32_t)));
        // the attribute is per function and device, not per plan: always the maximum any plan can need
        // (n_fft = 2^24 -> 2^24 / 512 groups = 128 KB, + 19 KB static)
        CUDA_TRY(p, cudaFuncSetAttribute(topk_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TOPK_MAX_GROUPS * (int)sizeof(uint32_t)));
    }
    return FSTAT_OK;
}

int ensure_host_ring(fstat_plan *p) {
    if (p->ring.rows) return FSTAT_OK;
    const int64_t nb = p->g.n_bins;
    int64_t rows = (int64_t)(64ll << 20) / (nb * 4);
    if (rows < p->n_inflight) rows = p->n_inflight;
    rows = (rows / p->n_inflight) * p->n_inflight;
    for (int i = 0; i < 2; ++i) {
        CUDA_TRY(p, cudaMalloc(&p->ring.buf[i], (size_t)rows * nb * sizeof(float)));
        CUDA_TRY(p, cudaEventCreateWithFlags(&p->ring.done[i], cudaEventDisableTiming));
    }
    p->ring.rows = rows;
    return FSTAT_OK;
}

int ensure_sky_slots(fstat_plan *p, size_t want);

int compute_impl(fstat_plan *p, const fstat_template_t *tm, int32_t n_tmpl, const OutSpec &out) {
    if (!p) return FSTAT_EINVAL;
    if (n_tmpl < 0 || (n_tmpl > 0 && !tm)) return fail(p, FSTAT_EINVAL, "null template array");
    if (n_tmpl == 0) return FSTAT_OK;
    if (out.mode == OUT_TOPK) {
        if (out.k < 1 || out.k > FSTAT_MAX_TOPK || out.k > p->g.n_bins) return fail(p, FSTAT_EINVAL, "k outside [1, min(64, n_bins)]");
        if (!out.val || !out.bin) return fail(p, FSTAT_EINVAL, "null top-k output");
    } else if (!out.rows) return fail(p, FSTAT_EINVAL, "null 2F output");
    CUDA_TRY(p, cudaSetDevice(p->device));
    const double ftol = 1e-9 * fmax(1.0, fabs(p->f_min));
    std::vector<SkyGroup> groups;
    for (int t = 0; t < n_tmpl; ++t) {
        if (!(fabs(tm[t].f0 - p->f_min) <= ftol)) return fail(p, FSTAT_EDOM, "template f0 differs from the plan's f_min");
        if (!std::isfinite(tm[t].alpha) || !std::isfinite(tm[t].delta) || !std::isfinite(tm[t].fdot) || !std::isfinite(tm[t].fddot))
            return fail(p, FSTAT_EINVAL, "non-finite template parameter");
        if (groups.empty() || groups.back().alpha != tm[t].alpha || groups.back().delta != tm[t].delta)
            groups.push_back({tm[t].alpha, tm[t].delta, t, 0});
        ++groups.back().count;
    }
    int rc = ensure_tmpl_capacity(p, n_tmpl, groups.size());
    if (rc) return rc;
    const int TB = p->n_inflight;
    // Two forms of the sky-dependent half.  Hoisted (default): sky_resample_kernel writes the resampled series S once per
    // sky position, every template of that position re-reads it (from L2).  Fused (fstat_debug_set_paths(fused_sky = 1)):
    // the per-sky work runs in the FFT pass-1 prologue and S never goes to global memory.  Measured on B200 the fused
    // form is slower at every size (a pass-1 tile gathers grid points N2 samples apart, so the reads of
    // the Farrow-filtered series are uncoalesced and run at 12 warps per SM), so it is never chosen automatically.
    int max_count = 0;
    for (const SkyGroup &sg : groups) max_count = std::max(max_count, sg.count);
    bool fused = fft_find_fused_kernel(p->g.log_n1, p->g.log_tile1, pass1_variant(p->g, false) & ~FFT_VAR_SKIPZ) != nullptr && max_count <= TB;
    if (fused && p->force_fused_sky == 0) fused = false;
    if (p->force_fused_sky < 0) fused = false;
    // fused: launches cover whole sky groups, at most TB templates each
    std::vector<int> chunk_of(fused ? groups.size() : 0), chunk_g0;
    if (fused) {
        int cur_t = 0;
        for (size_t gi = 0; gi < groups.size(); ++gi) {
            if (chunk_g0.empty() || cur_t + groups[gi].count > TB) { chunk_g0.push_back((int)gi); cur_t = 0; }
            chunk_of[gi] = (int)chunk_g0.size() - 1;
            cur_t += groups[gi].count;
        }
    } else {
        rc = ensure_sky_slots(p, groups.size());
        if (rc) return rc;
    }
    // staging buffers are reused between calls: wait until the previous upload has been consumed
    const int slot = p->stage_slot;
    p->stage_slot = (slot + 1) % STAGE_SLOTS;
    CUDA_TRY(p, cudaEventSynchronize(p->staging_ev[slot]));
    SkyConst *h_sky = p->h_sky + (size_t)slot * p->sky_cap;
    SkyABCD *h_abcd = p->h_abcd + (size_t)slot * p->sky_cap;
    TmplDesc *h_tmpl = p->h_tmpl + (size_t)slot * p->tmpl_cap;
    int2 *h_grp = p->h_grp + (size_t)slot * p->sky_cap;
    // spacing in time of the first-pass inputs of one FFT pass-1 butterfly: (N1 / r0) rows of N2 samples
    const double h_p1 = (double)(((int64_t)1 << p->g.log_n1) / radix_list(p->g.log_n1, p->g.p1_elems)[0]) * (double)((int64_t)1 << p->g.log_n2) * p->g.dt;
    for (size_t gi = 0; gi < groups.size(); ++gi) {
        fill_sky_const(p, groups[gi].alpha, groups[gi].delta, &h_sky[gi]);
        sky_abcd(p, groups[gi].alpha, groups[gi].delta, &h_abcd[gi], out.det_mask);
        if (h_abcd[gi].bad) p->pending_edom = true;
        if (fused) h_grp[gi] = make_int2(groups[gi].first - groups[chunk_g0[chunk_of[gi]]].first, groups[gi].count);
        for (int t = groups[gi].first; t < groups[gi].first + groups[gi].count; ++t) {
            h_tmpl[t].half_fdot = 0.5 * tm[t].fdot;
            h_tmpl[t].sixth_fddot = tm[t].fddot / 6.0;
            // which SkyABCD entry (and S slot) relative to the launch's first group
            h_tmpl[t].sky_slot = fused ? (int)gi - chunk_g0[chunk_of[gi]] : (int)(gi % p->n_sky_slots);
            h_tmpl[t].bin_off = out.bin_off ? out.bin_off[t] : 0;
            {   // second forward difference of the spin-down phase over the first-pass input spacing of FFT pass 1
                // (fft_kernels.cuh spin_down): 2 (fdot / 2) h^2 cycles, reduced mod 1 in fp64
                const double cyc = tm[t].fdot * h_p1 * h_p1;
                const double fr = cyc - std::rint(cyc);
                h_tmpl[t].q_re = (float)cos(2.0 * M_PI * fr);
                h_tmpl[t].q_im = (float)(-sin(2.0 * M_PI * fr));
            }
        }
    }
    CUDA_TRY(p, cudaMemcpyAsync(p->d_sky, h_sky, groups.size() * sizeof(SkyConst), cudaMemcpyHostToDevice, p->stream));
    CUDA_TRY(p, cudaMemcpyAsync(p->d_abcd, h_abcd, groups.size() * sizeof(SkyABCD), cudaMemcpyHostToDevice, p->stream));
    CUDA_TRY(p, cudaMemcpyAsync(p->d_tmpl, h_tmpl, (size_t)n_tmpl * sizeof(TmplDesc), cudaMemcpyHostToDevice, p->stream));
    if (fused) CUDA_TRY(p, cudaMemcpyAsync(p->d_grp, h_grp, groups.size() * sizeof(int2), cudaMemcpyHostToDevice, p->stream));
    CUDA_TRY(p, cudaEventRecord(p->staging_ev[slot], p->stream));

    if (out.mode == OUT_TOPK) { rc = ensure_topk_scratch(p); if (rc) return rc; }
    if (out.mode == OUT_HOST_ROWS) { rc = ensure_host_ring(p); if (rc) return rc; }

    const int64_t nb = p->g.n_bins;
    int ring_i = 0; int64_t ring_fill = 0; int64_t ring_row0 = 0;   // host-ring state
    auto flush_ring = [&](void) -> int {
        if (ring_fill == 0) return FSTAT_OK;
        CUDA_TRY(p, cudaEventRecord(p->chunk_ev, p->stream));
        CUDA_TRY(p, cudaStreamWaitEvent(p->copy_stream, p->chunk_ev, 0));
        CUDA_TRY(p, cudaMemcpyAsync(out.rows + ring_row0 * nb, p->ring.buf[ring_i], (size_t)ring_fill * nb * sizeof(float),
                                    cudaMemcpyDeviceToHost, p->copy_stream));
        CUDA_TRY(p, cudaEventRecord(p->ring.done[ring_i], p->copy_stream));
        ring_i ^= 1; ring_row0 += ring_fill; ring_fill = 0;
        // the buffer we are about to fill must have been drained
        CUDA_TRY(p, cudaStreamWaitEvent(p->stream, p->ring.done[ring_i], 0));
        return FSTAT_OK;
    };

    // FFT + 2F (+ selection) of templates [t0, t0 + nt), whose sky groups start at g0
    auto run_chunk = [&](int g0, int t0, int nt, int fused_ng) -> int {
        bool cubic = false;                      // second spin-down anywhere in this launch?
        for (int t = t0; t < t0 + nt && !cubic; ++t) cubic = (tm[t].fddot != 0.0);
        // one sky position for the whole launch?  (only then does the template-fastest tile order of pass 1 share anything)
        p->chunk_one_sky = true;
        for (int t = t0 + 1; t < t0 + nt && p->chunk_one_sky; ++t) p->chunk_one_sky = tm[t].alpha == tm[t0].alpha && tm[t].delta == tm[t0].delta;
        int r;
        if (out.mode == OUT_DEV_ROWS) {
            r = launch_fft_chunk(p, g0, t0, nt, out.rows + (int64_t)t0 * nb * (out.fafb ? 4 : 1), nb, cubic, nullptr, out.accumulate, fused_ng,
                                 out.det_mask, out.fafb);
            if (r) return r;
        } else if (out.mode == OUT_HOST_ROWS) {
            if (ring_fill + nt > p->ring.rows) { r = flush_ring(); if (r) return r; }
            r = launch_fft_chunk(p, g0, t0, nt, p->ring.buf[ring_i] + ring_fill * nb, nb, cubic, nullptr, false, fused_ng, out.det_mask);
            if (r) return r;
            ring_fill += nt;
        } else {
            r = launch_fft_chunk(p, g0, t0, nt, p->d_rows, nb, cubic, p->d_gmax, false, fused_ng, out.det_mask);
            if (r) return r;
            ProfScope ps(p, 3);
            const TopkGeom tg = topk_geom(p);
            topk_select_kernel<<<nt, TOPK_THREADS, tg.n_groups * sizeof(uint32_t), p->stream>>>(
                p->d_rows, nb, nb, out.k, p->d_gmax, tg, out.val + (int64_t)t0 * out.k, out.bin + (int64_t)t0 * out.k,
                out.thr, out.count ? out.count + t0 : nullptr);
            p->launches += 1;
            CUDA_TRY(p, cudaGetLastError());
        }
        return FSTAT_OK;
    };
    if (fused) {
        for (size_t c = 0; c < chunk_g0.size(); ++c) {
            const int gA = chunk_g0[c], gB = c + 1 < chunk_g0.size() ? chunk_g0[c + 1] : (int)groups.size();
            const int tA = groups[gA].first, tB = groups[gB - 1].first + groups[gB - 1].count;
            {
                ProfScope ps(p, 0);
                rc = launch_timing_nodes(p, gA, gB - gA);
                if (rc) return rc;
            }
            rc = run_chunk(gA, tA, tB - tA, gB - gA);
            if (rc) return rc;
        }
    } else {
        for (size_t gb = 0; gb < groups.size(); gb += p->n_sky_slots) {
            const int ng = (int)std::min<size_t>(p->n_sky_slots, groups.size() - gb);
            rc = launch_sky_batch(p, (int)gb, ng, p->d_S, 1, out.det_mask);
            if (rc) return rc;
            const int t_begin = groups[gb].first;
            const int t_end = groups[gb + ng - 1].first + groups[gb + ng - 1].count;
            for (int t0 = t_begin; t0 < t_end; t0 += TB) {
                rc = run_chunk((int)gb, t0, std::min(TB, t_end - t0), 0);
                if (rc) return rc;
            }
        }
    }
    if (out.mode == OUT_HOST_ROWS) {
        rc = flush_ring();
        if (rc) return rc;
        CUDA_TRY(p, cudaStreamSynchronize(p->copy_stream));
    }
    return FSTAT_OK;
}

void destroy_impl(fstat_plan *p) {
    if (!p) return;
    cudaSetDevice(p->device);
    if (p->stream) cudaStreamSynchronize(p->stream);
    cudaFree(p->d_series); cudaFree(p->d_farrow); cudaFree(p->d_rot); cudaFree(p->d_nodes); cudaFree(p->d_counter);
    for (void *t : p->d_tmp) cudaFree(t); cudaFree(p->d_wslot); cudaFree(p->d_tw1); cudaFree(p->d_tw2);
    cudaFree(p->d_S); cudaFree(p->d_T); cudaFree(p->d_sky); cudaFree(p->d_abcd); cudaFree(p->d_grp);
    cudaFree(p->d_tmpl); cudaFree(p->d_rows); cudaFree(p->d_gmax); cudaFree(p->d_gmax_lin);
    cudaFree(p->d_topk_v); cudaFree(p->d_topk_i);
    for (int i = 0; i < 2; ++i) { cudaFree(p->ring.buf[i]); if (p->ring.done[i]) cudaEventDestroy(p->ring.done[i]); }
    if (p->h_sky) cudaFreeHost(p->h_sky);
    if (p->h_tmpl) cudaFreeHost(p->h_tmpl);
    if (p->h_abcd) cudaFreeHost(p->h_abcd);
    if (p->h_grp) cudaFreeHost(p->h_grp);
    for (int i = 0; i < STAGE_SLOTS; ++i) if (p->staging_ev[i]) cudaEventDestroy(p->staging_ev[i]);
    if (p->chunk_ev) cudaEventDestroy(p->chunk_ev);
    if (p->copy_stream) cudaStreamDestroy(p->copy_stream);
    for (cudaEvent_t e : p->ev_pool) cudaEventDestroy(e);
    delete p;
}

int default_inflight(const fstat_plan *p) {
    // templates per persistent launch.  Measured on B200: every launch pair
    // costs ~35 us of ramp-up, tail and launch gap whatever its size, and keeping the four-step
    // intermediate L2-resident buys nothing (the passes are FMA-pipe bound, not DRAM bound), so
    // launches are made large: ~112 rounds of 4096-element tiles over the 2 resident CTAs of every SM (128 templates at
    // 2^20 / 2^21: -1 % against 74), bounded by 8 GB of intermediates -- or 1/16 of the device's memory if that is
    // less (180 GB on a B200: the 8 GB cap binds) -- i.e. 128 templates at 2^22, 64 at 2^23: -1..-2 % against 4 GB, mostly
    // fewer top-k launches; much larger buffers get slower again.
    const int64_t n_fft = p->g.n_fft;
    const int log_tile = p->g.log_tile2;
    const int64_t tiles_per_tmpl = (n_fft >> log_tile) > 0 ? (n_fft >> log_tile) : 1;
    int64_t want = (112 * (log_tile == 11 ? 4 : 2) * (int64_t)p->n_sm + tiles_per_tmpl - 1) / tiles_per_tmpl;
    if (want < 128) want = 128;
    const int64_t cap_bytes = std::min<int64_t>(8192ll << 20, (int64_t)(p->mem_total / 16));
    int64_t tb = cap_bytes / (n_fft * 16);
    if (tb > want) tb = want;
    if (tb > FSTAT_MAX_INFLIGHT) tb = FSTAT_MAX_INFLIGHT;
    if (tb < 1) tb = 1;
    return (int)tb;
}

int max_sky_slots_for(const fstat_plan *p) {
    // sky positions resampled per batch: a search over the sky wants large batches (every FFT launch pair costs
    // ~35 us whatever its size), bounded by 2 GB of resampled series (1/64 of the device's memory if less)
    const int64_t cap_bytes = std::min<int64_t>(2048ll << 20, (int64_t)(p->mem_total / 64));
    int64_t s = cap_bytes / (p->g.n_fft * 16);
    if (s < 1) s = 1;
    if (s > 1024) s = 1024;
    return (int)s;
}

// make room for `want` sky positions per batch (up to the plan's maximum)
int ensure_sky_slots(fstat_plan *p, size_t want) {
    int need = (int)std::min<size_t>(want, (size_t)p->max_sky_slots);
    if (need <= p->n_sky_slots) return FSTAT_OK;
    if (need < 2 * p->n_sky_slots) need = std::min(2 * p->n_sky_slots, p->max_sky_slots);
    CUDA_TRY(p, cudaStreamSynchronize(p->stream));
    cudaFree(p->d_S); p->d_S = nullptr; p->n_sky_slots = 0;
    const size_t bytes = (size_t)need * p->g.n_fft * sizeof(float4);
    if (cudaMalloc(&p->d_S, bytes) != cudaSuccess) { cudaGetLastError(); return fail(p, FSTAT_ENOMEM, "device allocation of the resampled-series buffers failed"); }
    CUDA_TRY(p, cudaMemsetAsync(p->d_S, 0, bytes, p->stream));     // the kernels only ever write k < n_src: the zero padding stays
    p->n_sky_slots = need;
    return FSTAT_OK;
}

}  // namespace

// ---- fstat_select_topk_noalloc (include/fstat.h): scratch that is part of the library image -------------------------
// The group maxima of the caller's rows, one uint32 per 512 bins.  A fixed array instead of a cudaMalloc, for callers
// that cannot allocate (a pipeline whose arena owns the whole GPU; a latency-bound loop that cannot take the
// device-wide stall of cudaMalloc / cudaFree).  1 MiB on every device that loads the library, until the process exits.
// In HOST code this name is only a handle for the runtime's symbol table, not a device address: host code must go
// through noalloc_scratch() below, which asks cudaGetSymbolAddress for the address on the current device.
static __device__ __align__(256) uint32_t g_noalloc_gmax[FSTAT_NOALLOC_MAX_GROUPS];

namespace {

#define NOALLOC_MAX_DEVICES 64
std::mutex g_noalloc_mu;
uint32_t *g_noalloc_ptr[NOALLOC_MAX_DEVICES];      // device address of g_noalloc_gmax per device ordinal; null = not set up yet

// One-time set-up per device, with that device current: the array's device address and the dynamic shared-memory
// limit of the selection kernel (128 KB of group keys at 2^24 bins).  Neither call allocates device memory.
int noalloc_scratch(uint32_t **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, FSTAT_ECUDA, std::string("cudaGetDevice: ") + cudaGetErrorString(e));
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(nullptr, FSTAT_ECUDA, "device ordinal beyond the no-alloc set-up table");
    std::lock_guard<std::mutex> lock(g_noalloc_mu);
    if (!g_noalloc_ptr[dev]) {
        uint32_t *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_noalloc_gmax);
        if (e != cudaSuccess || !ptr) {
            cudaGetLastError();
            return fail(nullptr, FSTAT_ECUDA, std::string("cudaGetSymbolAddress(g_noalloc_gmax): ") + cudaGetErrorString(e));
        }
        e = cudaFuncSetAttribute(topk_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TOPK_MAX_GROUPS * (int)sizeof(uint32_t));
        if (e != cudaSuccess) {
            cudaGetLastError();
            return fail(nullptr, FSTAT_ECUDA, std::string("cudaFuncSetAttribute(topk_select_kernel): ") + cudaGetErrorString(e));
        }
        g_noalloc_ptr[dev] = ptr;
    }
    *out = g_noalloc_ptr[dev];
    return FSTAT_OK;
}

}  // namespace

extern "C" {

const char *fstat_strerror(int code) {
    switch (code) {
        case FSTAT_OK: return "ok";
        case FSTAT_EINVAL: return "invalid argument";
        case FSTAT_ESIZE: return "size constraint violated";
        case FSTAT_EDOM: return "outside the domain of the plan (f0 != f_min or D <= 0)";
        case FSTAT_ECUDA: return "CUDA error";
        case FSTAT_ENOMEM: return "out of memory";
        default: return "unknown error";
    }
}

const char *fstat_last_error(const fstat_plan_t *plan) { return plan ? plan->err.c_str() : g_setup_error.c_str(); }

int fstat_setup(fstat_plan_t **out, int32_t n_det, const fstat_detector_t *det, const void *const *series_c64,
                int64_t n_samples, double t_start, double dt, double f_het, const double *const *timestamps,
                const float *const *weights, const int32_t *n_seg, double t_sft, const fstat_ephem_t *eph,
                int32_t dterms, double f_min, double band, int64_t n_fft, void *cuda_stream) {
    if (!out) return fail(nullptr, FSTAT_EINVAL, "out is null");
    *out = nullptr;
    if (n_det < 1 || n_det > FSTAT_MAX_DET) return fail(nullptr, FSTAT_EINVAL, "n_det outside [1, 8]");
    if (!det || !series_c64 || !timestamps || !weights || !n_seg || !eph) return fail(nullptr, FSTAT_EINVAL, "null argument");
    if (!(dt > 0) || !(t_sft > 0) || n_samples < 1 || !(band > 0) || !std::isfinite(f_min) || !std::isfinite(f_het) || !std::isfinite(t_start))
        return fail(nullptr, FSTAT_EINVAL, "dt, t_sft, n_samples, band must be positive and finite");
    if (dterms < 1 || dterms > FSTAT_MAX_DTERMS) return fail(nullptr, FSTAT_ESIZE, "dterms outside [1, 32]");
    if (n_fft < (1 << 12) || n_fft > (1 << 24) || (n_fft & (n_fft - 1))) return fail(nullptr, FSTAT_ESIZE, "n_fft must be a power of two in [2^12, 2^24]");
    const int64_t km = (int64_t)ceil(512.0 / dt);
    if (n_samples + 2 * km > n_fft) return fail(nullptr, FSTAT_ESIZE, "n_samples + 2*ceil(512 s/dt) exceeds n_fft");
    if (band > (1.0 / dt) * (1.0 + 1e-12)) return fail(nullptr, FSTAT_ESIZE, "band wider than the sample rate 1/dt");
    const double reach = fabs(eph->au_over_c_s) + fabs(eph->re_over_c_s);
    if (fabs(eph->omega_rot) * reach > 0.05 || fabs(eph->omega_orb) * reach > 0.05)
        return fail(nullptr, FSTAT_EINVAL, "ephemeris outside the small-delay regime (omega * delay must be < 0.05 rad)");
    const int64_t n_bins = llround(band * (double)n_fft * dt);
    if (n_bins < 1 || n_bins > n_fft) return fail(nullptr, FSTAT_ESIZE, "band gives no bins");
    const int n_slots = (int)ceil((double)n_samples * dt / t_sft - 1e-9);

    // timestamps -> dense slot weights
    std::vector<float> wslot((size_t)n_det * n_slots, 0.f);
    for (int X = 0; X < n_det; ++X) {
        if (n_seg[X] < 0 || (n_seg[X] > 0 && (!timestamps[X] || !weights[X]))) return fail(nullptr, FSTAT_EINVAL, "null timestamps/weights");
        if (!series_c64[X]) return fail(nullptr, FSTAT_EINVAL, "null series pointer");
        long long prev = -1;
        for (int s = 0; s < n_seg[X]; ++s) {
            const double q = (timestamps[X][s] - t_start) / t_sft;
            const long long idx = llround(q);
            if (fabs(q - (double)idx) > 1e-6 || idx < 0 || idx >= n_slots) return fail(nullptr, FSTAT_EINVAL, "timestamp not on the t_start + n*t_sft grid of the series");
            if (idx <= prev) return fail(nullptr, FSTAT_EINVAL, "timestamps unsorted or overlapping");
            if (!(weights[X][s] >= 0.f) || !std::isfinite(weights[X][s])) return fail(nullptr, FSTAT_EINVAL, "negative or non-finite weight");
            wslot[(size_t)X * n_slots + idx] = weights[X][s];
            prev = idx;
        }
    }

    int ndev = 0;
    cudaError_t ce = cudaGetDeviceCount(&ndev);
    if (ce != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, FSTAT_ECUDA, std::string("no CUDA device: ") + cudaGetErrorString(ce));
    }
    fstat_plan *p = new (std::nothrow) fstat_plan();
    if (!p) return fail(nullptr, FSTAT_ENOMEM, "host allocation failed");
    auto bail = [&](int code) { g_setup_error = p->err; destroy_impl(p); return code; };
#define SETUP_TRY(expr) do { cudaError_t e__ = (expr); if (e__ != cudaSuccess) { p->err = std::string(#expr) + ": " + cudaGetErrorString(e__); return bail(e__ == cudaErrorMemoryAllocation ? FSTAT_ENOMEM : FSTAT_ECUDA); } } while (0)
    SETUP_TRY(cudaGetDevice(&p->device));
    SETUP_TRY(cudaDeviceGetAttribute(&p->n_sm, cudaDevAttrMultiProcessorCount, p->device));
    { size_t mem_free = 0; SETUP_TRY(cudaMemGetInfo(&mem_free, &p->mem_total)); }
    p->stream = (cudaStream_t)cuda_stream;
    PlanGeom &g = p->g;
    g.n_det = n_det; g.dterms = dterms; g.n_samples = n_samples; g.k_margin = km; g.n_src = n_samples + 2 * km;
    g.n_fft = n_fft; g.n_bins = n_bins; g.series_stride = n_samples + 2 * SERIES_PAD; g.n_slots = n_slots;
    g.dt = dt; g.inv_dt = 1.0 / dt; g.t_sft = t_sft; g.inv_t_sft = 1.0 / t_sft; g.span = (double)n_samples * dt;
    g.f_het = f_het; g.omega_orb = eph->omega_orb; g.phi_orb0 = eph->phi_orb0; g.omega_rot = eph->omega_rot; g.gmst0 = eph->gmst0_rad;
    // band placement (S13): bin q sits exactly at f_min + q df.  (f_min - f_het)/df = whole FFT bins (an index
    // rotation, exact) + a fraction in [-1/2, 1/2] applied as a phase ramp over the grid index
    const double shift_bins = (f_min - f_het) * (double)n_fft * dt;
    const long long shift = llround(shift_bins);
    g.shift_mod = (uint32_t)(((shift % n_fft) + n_fft) % n_fft);
    g.shift_frac_per_k = (float)((shift_bins - (double)shift) / (double)n_fft);
    default_geometry(ilog2(n_fft), g);
    // timing nodes (sky_kernels.cuh): the largest power of two of grid points that spans at most 256 s
    g.log_node = 0;
    while (g.log_node < 16 && (double)(2 << g.log_node) * dt <= 256.0) ++g.log_node;
    {   // ... and small enough for THIS ephemeris: the cubic Hermite interpolant between nodes h apart is off by at most
        // h^4 / 384 max|Delta''''| ~ h^4 / 384 (re w_rot^4 + au w_orb^4) (7e-12 s for the Earth at h = 256 s).  Halve the
        // spacing until that is below 1e-9 s (needed: <~ 3e-8 s); at log_node = 0 every grid point is a node
        // and the inversion is exact everywhere, so any ephemeris the omega * delay check above admits is handled.
        const double d4 = fabs(eph->re_over_c_s) * pow(eph->omega_rot, 4) + fabs(eph->au_over_c_s) * pow(eph->omega_orb, 4);
        while (g.log_node > 0 && pow((double)(1 << g.log_node) * dt, 4) / 384.0 * d4 > 1e-9) --g.log_node;
    }
    g.n_nodes = (int)((g.n_src - 1) >> g.log_node) + 1;
    g.inv_node = 1.0 / (double)(1 << g.log_node);
    g.inv_n_fft = 1.0f / (float)n_fft;
    g.y_det_stride = ((n_samples + 1 + FARROW_BLOCK - 1) / FARROW_BLOCK) * (int64_t)(FARROW_BLOCK * (FARROW_NC / 2));
    {   // Newton steps of the timing inversion: e <- C2 e^2 / 2 + dp^3 e until below 1e-11 s (sky_kernels.cuh)
        const double wa = fabs(eph->omega_orb * eph->au_over_c_s) + fabs(eph->omega_rot * eph->re_over_c_s);
        const double c2 = eph->omega_orb * eph->omega_orb * fabs(eph->au_over_c_s) + eph->omega_rot * eph->omega_rot * fabs(eph->re_over_c_s);
        double e = wa * reach;
        g.n_newton = 0;
        while (e > 1e-11 && g.n_newton < 8) { e = 0.5 * c2 * e * e + wa * wa * wa * e; ++g.n_newton; }
    }
    p->eph = *eph; p->f_min = f_min; p->band = band; p->df = 1.0 / ((double)n_fft * dt);
    for (int X = 0; X < n_det; ++X) p->det[X] = det[X];

    SETUP_TRY(cudaStreamCreateWithFlags(&p->copy_stream, cudaStreamNonBlocking));
    for (int i = 0; i < STAGE_SLOTS; ++i) SETUP_TRY(cudaEventCreateWithFlags(&p->staging_ev[i], cudaEventDisableTiming));
    SETUP_TRY(cudaEventCreateWithFlags(&p->chunk_ev, cudaEventDisableTiming));
    SETUP_TRY(cudaMalloc(&p->d_series, (size_t)n_det * g.series_stride * sizeof(float2)));
    SETUP_TRY(cudaMemsetAsync(p->d_series, 0, (size_t)n_det * g.series_stride * sizeof(float2), p->stream));
    for (int X = 0; X < n_det; ++X)
        SETUP_TRY(cudaMemcpyAsync(p->d_series + (size_t)X * g.series_stride + SERIES_PAD, series_c64[X], (size_t)n_samples * sizeof(float2),
                                  cudaMemcpyDefault, p->stream));
    SETUP_TRY(cudaMalloc(&p->d_wslot, wslot.size() * sizeof(float)));
    SETUP_TRY(cudaMemcpyAsync(p->d_wslot, wslot.data(), wslot.size() * sizeof(float), cudaMemcpyHostToDevice, p->stream));
    // the default launch shape must be one fft_unit.cu instantiates: fail here, not in the first fstat_compute
    if (!geometry_supported(g)) { p->err = "no FFT kernel instantiated for the default geometry of this n_fft"; return bail(FSTAT_ESIZE); }
    { const int rc = upload_twiddles(p); if (rc != FSTAT_OK) return bail(rc); }
    p->n_inflight = default_inflight(p);
    p->max_sky_slots = max_sky_slots_for(p);
    { const int rc = ensure_sky_slots(p, 1); if (rc != FSTAT_OK) return bail(rc); }
    {   // Farrow-filtered copies of the series (sky_kernels.cuh), once per plan
        const std::vector<float> fc = farrow_coefficients(dterms);
        float *&d_fc = reinterpret_cast<float *&>(p->d_tmp[0]);
        SETUP_TRY(cudaMalloc(&d_fc, fc.size() * sizeof(float)));
        SETUP_TRY(cudaMemcpyAsync(d_fc, fc.data(), fc.size() * sizeof(float), cudaMemcpyHostToDevice, p->stream));
        SETUP_TRY(cudaMalloc(&p->d_farrow, (size_t)n_det * g.y_det_stride * sizeof(float4)));
        dim3 grid((unsigned)((n_samples + 1 + SKY_THREADS - 1) / SKY_THREADS), n_det);
        farrow_filter_kernel<<<grid, SKY_THREADS, 0, p->stream>>>(g, p->d_series, d_fc, p->d_farrow);
        ++p->launches;
        SETUP_TRY(cudaGetLastError());
        SETUP_TRY(cudaMalloc(&p->d_rot, (size_t)g.n_src * sizeof(float2)));
        sidereal_table_kernel<<<(unsigned)((g.n_src + SKY_THREADS - 1) / SKY_THREADS), SKY_THREADS, 0, p->stream>>>(g, p->d_rot);
        ++p->launches;
        SETUP_TRY(cudaGetLastError());
        SETUP_TRY(cudaStreamSynchronize(p->stream));
        cudaFree(d_fc); d_fc = nullptr;
    }
    {   // antenna moment matrices M_X (sky_kernels.cuh), once per plan
        const int nblk = (int)((n_samples + MOM_THREADS * MOM_PER_THREAD - 1) / (MOM_THREADS * MOM_PER_THREAD));
        double *&d_part = reinterpret_cast<double *&>(p->d_tmp[1]), *&d_lon = reinterpret_cast<double *&>(p->d_tmp[2]);
        std::vector<double> lon(n_det), part((size_t)n_det * nblk * MOM_TERMS);
        for (int X = 0; X < n_det; ++X) lon[X] = det[X].lon_east_rad;
        SETUP_TRY(cudaMalloc(&d_part, part.size() * sizeof(double)));
        SETUP_TRY(cudaMalloc(&d_lon, n_det * sizeof(double)));
        SETUP_TRY(cudaMemcpyAsync(d_lon, lon.data(), n_det * sizeof(double), cudaMemcpyHostToDevice, p->stream));
        antenna_moments_kernel<<<dim3(nblk, n_det), MOM_THREADS, 0, p->stream>>>(g, p->d_wslot, d_lon, d_part);
        ++p->launches;
        SETUP_TRY(cudaGetLastError());
        SETUP_TRY(cudaMemcpyAsync(part.data(), d_part, part.size() * sizeof(double), cudaMemcpyDeviceToHost, p->stream));
        SETUP_TRY(cudaStreamSynchronize(p->stream));
        cudaFree(d_part); cudaFree(d_lon); d_part = nullptr; d_lon = nullptr;
        for (int X = 0; X < n_det; ++X)
            for (int q = 0; q < MOM_TERMS; ++q) {
                double t = 0.0;
                for (int b = 0; b < nblk; ++b) t += part[((size_t)X * nblk + b) * MOM_TERMS + q];
                p->mom[X][q] = t;
            }
    }
    for (int i = 0; i < STAGE_SLOTS; ++i) SETUP_TRY(cudaEventRecord(p->staging_ev[i], p->stream));
    // the caller may free its buffers when we return
    SETUP_TRY(cudaStreamSynchronize(p->stream));
#undef SETUP_TRY
    *out = p;
    return FSTAT_OK;
}

int fstat_get_layout(const fstat_plan_t *plan, int64_t *n_bins, double *df) {
    if (!plan) return FSTAT_EINVAL;
    if (n_bins) *n_bins = plan->g.n_bins;
    if (df) *df = plan->df;
    return FSTAT_OK;
}

int fstat_compute(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *twoF_dev) {
    OutSpec o; o.mode = OUT_DEV_ROWS; o.rows = twoF_dev;
    return compute_impl(plan, tmpl_host, n_tmpl, o);
}

int fstat_compute_topk(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, int32_t k, float *val_dev, int32_t *bin_dev) {
    OutSpec o; o.mode = OUT_TOPK; o.k = k; o.val = val_dev; o.bin = bin_dev;
    return compute_impl(plan, tmpl_host, n_tmpl, o);
}

int fstat_compute_threshold(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float threshold, int32_t k,
                            float *val_dev, int32_t *bin_dev, int32_t *count_dev) {
    if (!plan) return FSTAT_EINVAL;
    if (!std::isfinite(threshold)) return fail(plan, FSTAT_EINVAL, "non-finite threshold");
    if (n_tmpl > 0 && !count_dev) return fail(plan, FSTAT_EINVAL, "null count output");
    OutSpec o; o.mode = OUT_TOPK; o.k = k; o.val = val_dev; o.bin = bin_dev; o.thr = threshold; o.count = count_dev;
    return compute_impl(plan, tmpl_host, n_tmpl, o);
}

int fstat_compute_accumulate(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, const int32_t *bin_offset_host,
                             float *twoF_dev) {
    OutSpec o; o.mode = OUT_DEV_ROWS; o.rows = twoF_dev; o.accumulate = true; o.bin_off = bin_offset_host;
    if (plan && bin_offset_host)
        for (int t = 0; t < n_tmpl; ++t)
            if (bin_offset_host[t] <= -plan->g.n_bins || bin_offset_host[t] >= plan->g.n_bins) return fail(plan, FSTAT_EINVAL, "bin offset outside (-n_bins, n_bins)");
    return compute_impl(plan, tmpl_host, n_tmpl, o);
}

int fstat_compute_per_detector(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *twoF_dev) {
    if (!plan) return FSTAT_EINVAL;
    for (int X = 0; X < plan->g.n_det; ++X) {
        OutSpec o; o.mode = OUT_DEV_ROWS; o.det_mask = 1u << X;
        o.rows = twoF_dev ? twoF_dev + (int64_t)X * n_tmpl * plan->g.n_bins : nullptr;
        const int rc = compute_impl(plan, tmpl_host, n_tmpl, o);
        if (rc) return rc;
    }
    return FSTAT_OK;
}

// top-k / threshold selection over caller-owned rows (e.g. the summed 2F of a semi-coherent search)
static int select_rows(fstat_plan *p, const float *rows, int32_t n_rows, int32_t k, float *val, int32_t *bin, float thr, int32_t *count) {
    if (!p) return FSTAT_EINVAL;
    if (n_rows < 0 || (n_rows > 0 && (!rows || !val || !bin))) return fail(p, FSTAT_EINVAL, "null argument");
    if (k < 1 || k > FSTAT_MAX_TOPK || k > p->g.n_bins) return fail(p, FSTAT_EINVAL, "k outside [1, min(64, n_bins)]");
    if (n_rows == 0) return FSTAT_OK;
    CUDA_TRY(p, cudaSetDevice(p->device));
    const int64_t nb = p->g.n_bins;
    TopkGeom tg{};
    tg.elems = 16; tg.linear = 1; tg.n_groups = (int)((nb + 511) / 512);
    const int chunk = 1024;
    if (!p->d_gmax_lin) {
        CUDA_TRY(p, cudaMalloc(&p->d_gmax_lin, (size_t)chunk * tg.n_groups * sizeof(uint32_t)));
        CUDA_TRY(p, cudaFuncSetAttribute(topk_select_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, TOPK_MAX_GROUPS * (int)sizeof(uint32_t)));
    }
    ProfScope ps(p, 3);
    for (int r0 = 0; r0 < n_rows; r0 += chunk) {
        const int nr = std::min(chunk, n_rows - r0);
        const float *rp = rows + (int64_t)r0 * nb;
        group_max_kernel<<<dim3((tg.n_groups + TOPK_THREADS / 32 - 1) / (TOPK_THREADS / 32), nr), TOPK_THREADS, 0, p->stream>>>(rp, nb, nb, tg.n_groups, p->d_gmax_lin);
        topk_select_kernel<<<nr, TOPK_THREADS, tg.n_groups * sizeof(uint32_t), p->stream>>>(
            rp, nb, nb, k, p->d_gmax_lin, tg, val + (int64_t)r0 * k, bin + (int64_t)r0 * k, thr, count ? count + r0 : nullptr);
        p->launches += 2;
        CUDA_TRY(p, cudaGetLastError());
    }
    return FSTAT_OK;
}

int fstat_select_topk(fstat_plan_t *plan, const float *twoF_dev, int32_t n_rows, int32_t k, float *val_dev, int32_t *bin_dev) {
    return select_rows(plan, twoF_dev, n_rows, k, val_dev, bin_dev, 0.f, nullptr);
}

int fstat_select_threshold(fstat_plan_t *plan, const float *twoF_dev, int32_t n_rows, float threshold, int32_t k,
                           float *val_dev, int32_t *bin_dev, int32_t *count_dev) {
    if (!plan) return FSTAT_EINVAL;
    if (!std::isfinite(threshold)) return fail(plan, FSTAT_EINVAL, "non-finite threshold");
    if (n_rows > 0 && !count_dev) return fail(plan, FSTAT_EINVAL, "null count output");
    return select_rows(plan, twoF_dev, n_rows, k, val_dev, bin_dev, threshold, count_dev);
}

// fstat_select_topk without a plan and without any allocation: the two kernels of select_rows, with the group maxima
// in the library's own g_noalloc_gmax (shared by every call on the device; group_max_kernel rewrites each entry the
// selection reads, so stale contents of an earlier call are never seen).
int fstat_select_topk_noalloc(const float *twoF_dev, int64_t n_bins, int32_t n_rows, int32_t k, float *val_dev, int32_t *bin_dev,
                              void *cuda_stream) {
    if (n_rows < 0 || (n_rows > 0 && (!twoF_dev || !val_dev || !bin_dev))) return fail(nullptr, FSTAT_EINVAL, "null argument or negative row count");
    if (n_bins < 1 || n_bins > (int64_t(1) << 24)) return fail(nullptr, FSTAT_ESIZE, "n_bins outside [1, 2^24]");
    if (k < 1 || k > FSTAT_MAX_TOPK || k > n_bins) return fail(nullptr, FSTAT_EINVAL, "k outside [1, min(64, n_bins)]");
    const int64_t n_groups = (n_bins + 511) / 512;
    if ((int64_t)n_rows * n_groups > FSTAT_NOALLOC_MAX_GROUPS) {
        char msg[200];
        snprintf(msg, sizeof msg, "n_rows * ceil(n_bins / 512) = %lld exceeds the fixed scratch of %d groups: split the rows over several calls",
                 (long long)n_rows * (long long)n_groups, FSTAT_NOALLOC_MAX_GROUPS);
        return fail(nullptr, FSTAT_ESIZE, msg);
    }
    if (n_rows == 0) return FSTAT_OK;
    uint32_t *gmax = nullptr;
    const int rc = noalloc_scratch(&gmax);
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    TopkGeom tg{};
    tg.elems = 16; tg.linear = 1; tg.n_groups = (int)n_groups;
    const int chunk = 32768;                                   // rows per launch pair (grid.y limit of group_max_kernel)
    for (int r0 = 0; r0 < n_rows; r0 += chunk) {
        const int nr = std::min(chunk, n_rows - r0);
        const float *rp = twoF_dev + (int64_t)r0 * n_bins;
        uint32_t *gp = gmax + (int64_t)r0 * tg.n_groups;
        group_max_kernel<<<dim3((tg.n_groups + TOPK_THREADS / 32 - 1) / (TOPK_THREADS / 32), nr), TOPK_THREADS, 0, stream>>>(
            rp, n_bins, n_bins, tg.n_groups, gp);
        topk_select_kernel<<<nr, TOPK_THREADS, tg.n_groups * sizeof(uint32_t), stream>>>(
            rp, n_bins, n_bins, k, gp, tg, val_dev + (int64_t)r0 * k, bin_dev + (int64_t)r0 * k, 0.f, nullptr);
    }
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, FSTAT_ECUDA, std::string("fstat_select_topk_noalloc launch: ") + cudaGetErrorString(e));
    return FSTAT_OK;
}

int fstat_compute_host(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *twoF_host) {
    OutSpec o; o.mode = OUT_HOST_ROWS; o.rows = twoF_host;
    int rc = compute_impl(plan, tmpl_host, n_tmpl, o);
    if (rc) return rc;
    return fstat_sync(plan);
}

int fstat_compute_topk_host(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, int32_t k, float *val_host, int32_t *bin_host) {
    if (!plan) return FSTAT_EINVAL;
    if (n_tmpl <= 0) return n_tmpl == 0 ? FSTAT_OK : FSTAT_EINVAL;
    if (!val_host || !bin_host) return fail(plan, FSTAT_EINVAL, "null top-k output");
    if (k < 1 || k > FSTAT_MAX_TOPK) return fail(plan, FSTAT_EINVAL, "k outside [1, 64]");
    const size_t need = (size_t)n_tmpl * k;
    if (need > plan->topk_cap) {
        cudaFree(plan->d_topk_v); cudaFree(plan->d_topk_i);
        plan->d_topk_v = nullptr; plan->d_topk_i = nullptr; plan->topk_cap = 0;
        CUDA_TRY(plan, cudaMalloc(&plan->d_topk_v, need * sizeof(float)));
        CUDA_TRY(plan, cudaMalloc(&plan->d_topk_i, need * sizeof(int)));
        plan->topk_cap = need;
    }
    OutSpec o; o.mode = OUT_TOPK; o.k = k; o.val = plan->d_topk_v; o.bin = plan->d_topk_i;
    int rc = compute_impl(plan, tmpl_host, n_tmpl, o);
    if (rc) return rc;
    CUDA_TRY(plan, cudaMemcpyAsync(val_host, plan->d_topk_v, need * sizeof(float), cudaMemcpyDeviceToHost, plan->stream));
    CUDA_TRY(plan, cudaMemcpyAsync(bin_host, plan->d_topk_i, need * sizeof(int), cudaMemcpyDeviceToHost, plan->stream));
    return fstat_sync(plan);
}

int fstat_resample_sky(fstat_plan_t *plan, double alpha, double delta, float *S_dev, double *abcd_host) {
    if (!plan || !S_dev || !abcd_host) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaSetDevice(plan->device));
    int rc = ensure_tmpl_capacity(plan, 1, 1);
    if (rc) return rc;
    const int slot = plan->stage_slot;
    plan->stage_slot = (slot + 1) % STAGE_SLOTS;
    CUDA_TRY(plan, cudaEventSynchronize(plan->staging_ev[slot]));
    SkyConst *h_sky = plan->h_sky + (size_t)slot * plan->sky_cap;
    fill_sky_const(plan, alpha, delta, h_sky);
    CUDA_TRY(plan, cudaMemcpyAsync(plan->d_sky, h_sky, sizeof(SkyConst), cudaMemcpyHostToDevice, plan->stream));
    CUDA_TRY(plan, cudaEventRecord(plan->staging_ev[slot], plan->stream));
    CUDA_TRY(plan, cudaMemsetAsync(S_dev, 0, (size_t)plan->g.n_fft * sizeof(float4), plan->stream));
    rc = launch_sky_batch(plan, 0, 1, (float4 *)S_dev, 0);
    if (rc) return rc;
    SkyABCD r;
    sky_abcd(plan, alpha, delta, &r);
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    abcd_host[0] = r.A; abcd_host[1] = r.B; abcd_host[2] = r.C; abcd_host[3] = r.D;
    return FSTAT_OK;
}

int fstat_sync(fstat_plan_t *plan) {
    if (!plan) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    const bool bad = plan->pending_edom;
    plan->pending_edom = false;
    if (bad) return fail(plan, FSTAT_EDOM, "antenna determinant D <= 0 for at least one template (outputs are NaN)");
    return FSTAT_OK;
}

int fstat_launch_count(const fstat_plan_t *plan, int64_t *count) {
    if (!plan || !count) return FSTAT_EINVAL;
    *count = plan->launches;
    return FSTAT_OK;
}

int fstat_set_inflight(fstat_plan_t *plan, int32_t n_inflight) {
    if (!plan || n_inflight < 0 || n_inflight > FSTAT_MAX_INFLIGHT) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaSetDevice(plan->device));
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    const int tb = n_inflight == 0 ? default_inflight(plan) : n_inflight;
    if (tb == plan->n_inflight) return FSTAT_OK;
    cudaFree(plan->d_T); plan->d_T = nullptr; plan->t_cap = 0;
    cudaFree(plan->d_rows); plan->d_rows = nullptr;
    cudaFree(plan->d_gmax); plan->d_gmax = nullptr;
    for (int i = 0; i < 2; ++i) { cudaFree(plan->ring.buf[i]); plan->ring.buf[i] = nullptr; if (plan->ring.done[i]) cudaEventDestroy(plan->ring.done[i]); plan->ring.done[i] = nullptr; }
    plan->ring.rows = 0;
    plan->n_inflight = tb;
    return FSTAT_OK;
}

int fstat_set_profile(fstat_plan_t *plan, int32_t enable) {
    if (!plan) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    plan->profile = enable != 0;
    plan->segs.clear(); plan->ev_used = 0;
    return FSTAT_OK;
}

int fstat_get_profile(fstat_plan_t *plan, double *ms, int64_t *launches) {
    if (!plan || !ms || !launches) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    for (int c = 0; c < FSTAT_PROFILE_CLASSES; ++c) { ms[c] = 0.0; launches[c] = 0; }
    for (const fstat_plan::Seg &sg : plan->segs) {
        float t = 0.f;
        CUDA_TRY(plan, cudaEventElapsedTime(&t, plan->ev_pool[sg.e0], plan->ev_pool[sg.e1]));
        ms[sg.cls] += t; launches[sg.cls] += sg.launches;
    }
    plan->segs.clear(); plan->ev_used = 0;
    return FSTAT_OK;
}

int fstat_debug_set_geometry(fstat_plan_t *plan, int32_t log_n2, int32_t log_tile1, int32_t log_tile2, int32_t p2_elems) {
    if (!plan) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaSetDevice(plan->device));
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    PlanGeom g = plan->g;
    const int L = ilog2(g.n_fft);
    default_geometry(L, g);
    if (log_n2 >= 0) { g.log_n2 = log_n2; g.log_n1 = L - log_n2; }
    if (log_tile1 >= 0) g.log_tile1 = log_tile1;
    if (log_tile2 >= 0) g.log_tile2 = log_tile2;
    if (log_n2 >= 0 && log_tile1 < 0) g.log_tile1 = (g.log_n1 == 9 || g.log_n1 == 10) ? 10 : g.log_n1 <= 10 ? 11 : g.log_n1;
    if (log_n2 >= 0 && log_tile2 < 0) g.log_tile2 = g.log_n2 <= 11 ? 12 : 13;
    g.p2_elems = p2_elems >= 0 ? p2_elems : ((g.log_n2 == 9 || g.log_n2 == 10) && g.log_tile2 >= 12 && !(g.log_n2 == 9 && g.log_tile2 == 13)) ? 32 : 16;
    g.p1_elems = g.log_tile1 == 10 ? 32 : 16;
    g.log_w1 = g.log_tile1 - g.log_n1; g.log_w2 = g.log_tile2 - g.log_n2;
    if (!geometry_supported(g)) return fail(plan, FSTAT_ESIZE, "no kernel instantiated for this (sub-FFT, tile, elements) combination");
    plan->g = g;
    cudaFree(plan->d_gmax); plan->d_gmax = nullptr;           // group count depends on the pass-2 tile shape
    // the blocked layout of S moved: what is zero padding (k >= n_src, never written by the kernels) is now elsewhere
    if (plan->d_S) CUDA_TRY(plan, cudaMemsetAsync(plan->d_S, 0, (size_t)plan->n_sky_slots * plan->g.n_fft * sizeof(float4), plan->stream));
    return upload_twiddles(plan);
}

int fstat_debug_set_max_sky_slots(fstat_plan_t *plan, int32_t max_slots) {
    if (!plan || max_slots < 0) return FSTAT_EINVAL;
    CUDA_TRY(plan, cudaSetDevice(plan->device));
    CUDA_TRY(plan, cudaStreamSynchronize(plan->stream));
    plan->max_sky_slots = max_slots == 0 ? max_sky_slots_for(plan) : max_slots;
    if (plan->n_sky_slots > plan->max_sky_slots) {            // shrink: reallocate on the next call
        cudaFree(plan->d_S); plan->d_S = nullptr; plan->n_sky_slots = 0;
        return ensure_sky_slots(plan, 1);
    }
    return FSTAT_OK;
}

int fstat_debug_compute_fafb(fstat_plan_t *plan, const fstat_template_t *tmpl_host, int32_t n_tmpl, float *fafb_dev) {
    OutSpec o; o.mode = OUT_DEV_ROWS; o.rows = fafb_dev; o.fafb = true;
    return compute_impl(plan, tmpl_host, n_tmpl, o);
}

int fstat_debug_set_paths(fstat_plan_t *plan, int32_t fused_sky, int32_t single) {
    if (!plan || fused_sky < -1 || fused_sky > 1 || single < -1 || single > 1) return FSTAT_EINVAL;
    plan->force_fused_sky = fused_sky;
    plan->force_single = single;
    return FSTAT_OK;
}

void fstat_destroy(fstat_plan_t *plan) { destroy_impl(plan); }

}  // extern "C"
