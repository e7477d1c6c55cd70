// Shared definitions of the CUDA path (host + device).  Not used by the oracle.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define FSTAT_MAX_DET 8
#define FSTAT_MAX_DTERMS 32
#define FSTAT_MAX_TOPK 64
#define SERIES_PAD 64            // zero samples kept on both sides of every series

#ifdef __CUDACC__
// Order-preserving map float -> uint32 (NaN lowest, then -inf ... +inf).
__device__ __forceinline__ uint32_t topk_key(float v) {
    const uint32_t b = __float_as_uint(v);
    if (v != v) return 0u;
    return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

#endif

// Per-sky constants, computed on the host in double (cheap, O(n_det)) -- DESIGN.md "H1/H2".
struct SkyConst {
    // Roemer delay: Delta = Pc cos(phi_o) + Ps sin(phi_o) + Qc[X] cos(theta) + Qs[X] sin(theta) + Q0[X]
    // with phi_o = phi_orb0 + omega_orb T', theta = gmst0 + omega_rot T' (longitude folded into Qc, Qs).
    double Pc, Ps;
    double Qc[FSTAT_MAX_DET], Qs[FSTAT_MAX_DET], Q0[FSTAT_MAX_DET];
    // hour angle h = (alpha - lon_X) - theta:  cos h = cal cos(theta) + sal sin(theta), sin h = sal cos(theta) - cal sin(theta)
    float cal[FSTAT_MAX_DET], sal[FSTAT_MAX_DET];
    // a = ac[0] + ac[1] cos2h + ac[2] sin2h + ac[3] cosh + ac[4] sinh ; b = bc[0] cos2h + bc[1] sin2h + bc[2] cosh + bc[3] sinh
    float ac[FSTAT_MAX_DET][5], bc[FSTAT_MAX_DET][4];
};

// Antenna sums of one sky position, written by the device (double) and read by the 2F epilogue.
struct SkyABCD {
    double A, B, C, D;
    float b_over_d, a_over_d, two_c_over_d;   // eq. 8 coefficients
    int bad;                                   // D <= 0
};

// One template as the FFT kernels see it.
struct TmplDesc {
    double half_fdot;     // fdot / 2
    double sixth_fddot;   // fddot / 6
    int32_t sky_slot;     // which S buffer / SkyABCD entry
    int32_t bin_off;      // accumulate mode: 2F of this template's bin q is added to output bin q - bin_off (else 0)
    float q_re, q_im;     // exp(-2 pi i fdot h^2), h = time step between the first-pass inputs of FFT pass 1 (fddot = 0 path)
};

// Geometry of the plan, passed by value to kernels.
struct PlanGeom {
    int n_det;
    int dterms;
    int64_t n_samples;      // N
    int64_t n_src;          // N + 2 K_m
    int64_t n_fft;
    int64_t n_bins;
    int64_t k_margin;       // K_m
    int64_t series_stride;  // N + 2*SERIES_PAD (float2 elements per detector)
    int n_slots;            // slots per detector
    double dt, inv_dt, t_sft, inv_t_sft, span;   // span = N*dt
    double f_het;
    double omega_orb, phi_orb0, omega_rot, gmst0;
    uint32_t shift_mod;     // (round((f_min - f_het)/df)) mod n_fft
    float shift_frac_per_k; // ((f_min - f_het)/df - round(..)) / n_fft: residual band shift in cycles per grid index
    int log_n1, log_n2;     // n_fft = 2^log_n1 * 2^log_n2 (log_n1 >= log_n2)
    int log_w1, log_w2;     // columns / rows per tile of FFT pass 1 / pass 2
    int log_tile1, log_tile2;   // log2 of the tile size of FFT pass 1 / 2 (11 or 12; sub-FFTs of length 2^12 use 13)
    int p1_elems, p2_elems; // register elements per thread of FFT pass 1 / 2 (16 or 32)
    int n_newton;           // Newton steps of the SSB timing inversion (1 for the Earth)
    int log_node, n_nodes;  // timing nodes: every 2^log_node grid points (<= 256 s apart), n_nodes = ((n_src - 1) >> log_node) + 1
    double inv_node;        // 2^-log_node
    float inv_n_fft;        // 1 / n_fft
    int64_t y_det_stride;   // float4 elements of the Farrow-filtered series per detector: 128 * ceil((N + 1) / 32)
};
