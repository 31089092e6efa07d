// rt_direct.cuh -- fused steps 1-4, small-batch variant:
// one thread per (model, wavenumber); the 4-tap bilinear interpolation reads the
// opacity table straight from global memory (coalesced along nu), kappa is never
// materialised, RT state lives in registers.  This is the HBM/L2-bound path for
// B of a few models (the paper's own usage is B = 1 per likelihood call).
// PAPER.md:241 (interpolation), 239 (optical depth), Eq. 2, 4-9 (RT).
#pragma once
#include "common.cuh"

namespace helios {

struct DirectArgs {
    const float* sigma;      // DEVICE [S][nT][nP][stride]
    const float* cia;        // DEVICE [C][nT][stride]
    int S, C, nT, nP, nNu, L;
    long long stride;        // padded row length (floats)
    const int* nu_index;     // DEVICE [stride]  wavenumber grid index of every table column (helios_load_opacity)
    const float* rec;        // DEVICE [B][L][rec_floats]
    int rec_floats;
    const float* model_scale;
    const int* model_flag;
    double nu0, dnu;
    float* flux;             // DEVICE [B][flux_stride]
    long long flux_stride;
    AngleSet ang;
};

constexpr int kDirectThreads = 128;

template <int A>
__global__ void __launch_bounds__(kDirectThreads) k_rt_direct(DirectArgs a) {
    extern __shared__ float srec[];          // [L][rec_floats]
    const int b = blockIdx.y;
    pdl_wait();
    const float* grec = a.rec + (size_t)b * a.L * a.rec_floats;
    for (int i = threadIdx.x; i < a.L * a.rec_floats; i += kDirectThreads) srec[i] = grec[i];
    __syncthreads();

    const int inu = blockIdx.x * kDirectThreads + threadIdx.x;     // column of the (re-ordered) table
    if (inu >= a.nNu) return;
    const int gnu = a.nu_index[inu];                                // its wavenumber grid point
    float* out = a.flux + (size_t)b * a.flux_stride + gnu;
    if (a.model_flag[b]) { *out = __int_as_float(0x7fc00000); return; }

    const double nu_d = a.nu0 + a.dnu * (double)gnu;
    const float nu = (float)nu_d;
    const float nu_lo = (float)(nu_d - (double)nu);
    const float c1nu3 = (float)(kC1 * nu_d * nu_d * nu_d);
    const int PA = 4 * a.S + 2 * a.C;
    const long long plane = (long long)a.nT * a.nP * a.stride;
    const long long s_ip = a.stride, s_iT = (long long)a.nP * a.stride;

    float J[A];
#pragma unroll
    for (int k = 0; k < A; ++k) J[k] = 0.0f;
    float chi_prev = 0.0f, S_prev = 0.0f, hdz_prev = 0.0f, dtc_prev = 0.0f;

    for (int l = 0; l < a.L; ++l) {
        const float* r = srec + l * a.rec_floats;
        const int cell = __float_as_int(r[PA + 3]);
        const int iT = __float_as_int(r[PA + 4]);
        float chi = 0.0f;
        const float* tab = a.sigma + (long long)cell * a.stride + inu;
        for (int s = 0; s < a.S; ++s) {
            const float* t00 = tab + s * plane;
            float v00 = __ldg(t00), v01 = __ldg(t00 + s_ip), v10 = __ldg(t00 + s_iT), v11 = __ldg(t00 + s_iT + s_ip);
            chi = fmaf(r[4 * s + 0], v00, chi);
            chi = fmaf(r[4 * s + 1], v01, chi);
            chi = fmaf(r[4 * s + 2], v10, chi);
            chi = fmaf(r[4 * s + 3], v11, chi);
        }
        for (int c = 0; c < a.C; ++c) {
            const float* a0 = a.cia + ((long long)c * a.nT + iT) * a.stride + inu;
            chi = fmaf(r[4 * a.S + 2 * c + 0], __ldg(a0), chi);
            chi = fmaf(r[4 * a.S + 2 * c + 1], __ldg(a0 + a.stride), chi);
        }
        // S_l = B_nu(T_l) = c1 nu^3 E / (1 - E), E = exp(-c2 nu / T_l)
        const float E = planck_E(r[PA], r[PA + 1], nu, nu_lo);
        const float Sl = planck_from_E(c1nu3, E);
        if (l > 0) {
            const float dtau = fmaf(chi + chi_prev, hdz_prev, dtc_prev);
            const float dS = S_prev - Sl;
            const float q = dS * rcp_approx(dtau);
#pragma unroll
            for (int k = 0; k < A; ++k)
                sc_update(J[k], dtau, q, dS, a.ang.c_exp[k], a.ang.inv_mu[k], a.ang.mu[k]);
        }
        chi_prev = chi; S_prev = Sl; hdz_prev = r[PA + 2]; dtc_prev = r[PA + 5];
    }
    // F+ = 2 pi sum_k w_k mu_k I_k (Eq. 8), I_k = J_k + S_top;  F = f (R/d)^2 F+ (Eq. 9)
    float acc = S_prev * a.ang.wmu_sum;
#pragma unroll
    for (int k = 0; k < A; ++k) acc = fmaf(a.ang.wmu[k], J[k], acc);
    pdl_launch_dependents();
    *out = a.model_scale[b] * acc;
}

}  // namespace helios
