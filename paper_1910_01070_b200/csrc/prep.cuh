// prep.cuh -- step 0 of the hot path: per (model, level) profile
// quantities, interpolation cells/weights and number-density-weighted tap weights.
// fp64 arithmetic, fp32 results.  PAPER.md:55 (levels), 174-221 (first-order
// elements), 484 (isoprofiles, H2/He fill), 241 (interpolation).
#pragma once
#include "common.cuh"

namespace helios {

struct PrepArgs {
    const double* params;     // DEVICE [B][P]
    int B, P, K, S, C, L, nT, nP;
    const double* T_grid;     // DEVICE [nT]
    const double* lvl_p_bar;  // DEVICE [L]
    const int*    lvl_elem;   // DEVICE [L]  finite element the level lies in
    const double* lvl_lw;     // DEVICE [L][kMaxTpNodes]  Lagrange weights of the element's nodes at the level (Eq. 13)
    int tp_order;             // q: element k owns the temperature parameters k q .. k q + q (0: one isothermal value)
    int tp_ratio;             // 1: parameters are (T_1, b_2 .. b_N), T_i = b_i T_{i-1}
    int NT;                   // number of temperature parameters (replaces K in the parameter vector)
    unsigned extras;          // HELIOS_EXTRA_* flags: extra parameters after the VMRs
    int unit_scale;           // 1: model_scale = 2 pi (F+ of Eq. 8, for T_eff); 0: 2 pi f flux_const [/ d^2] (Eq. 9)
    double* model_addvar;     // DEVICE [B]  10^epsilon of Eq. 22 (0 without error inflation)
    const int*    lvl_ip;     // DEVICE [L]  pressure cell
    const double* lvl_u;      // DEVICE [L]  pressure weight in [0,1]
    const int*    lvl_pclamp; // DEVICE [L]  1 if the level pressure is outside the table
    const double* lvl_lnratio;// DEVICE [L]  ln(p_l / p_{l+1}) (0 for the top level)
    double mmw, he_to_h2, flux_const;
    float* rec;               // DEVICE [B][L][rec_floats]
    int rec_floats;
    int slab_layout;          // 0: direct record (4 taps / species), 1: staged-kernel record (common.cuh)
    float* model_x;           // DEVICE [B][x_floats]  staged kernel: x_s 2^32, x_H2 x_c
    int x_floats;
    float* model_scale;       // DEVICE [B]  f * flux_const * 2 pi
    int*   model_flag;        // DEVICE [B]  1 = rejected model (zeroed before the launch, raised by any thread of the model)
    unsigned long long* counters;  // [0] clamped pairs, [1] rejected models
};

constexpr int kMaxTpNodes = 5;    // order <= 4

// Eq. 12: T(level) = sum_i T_dof[k q + i] l_i(xi).  In the ratio form the nodal temperatures are the
// running products T_1 b_2 ... b_j (R28), rebuilt here for the element's q + 1 nodes.
__device__ __forceinline__ double level_temperature(const double* tpar, int q, int ratio, int k, const double* lw) {
    if (q == 0) return tpar[0];
    double T_node = tpar[0];
    if (ratio) { for (int j = 1; j <= k * q; ++j) T_node *= tpar[j]; }
    else T_node = tpar[k * q];
    double T = T_node * lw[0];
    for (int i = 1; i <= q; ++i) {
        T_node = ratio ? T_node * tpar[k * q + i] : tpar[k * q + i];
        T += T_node * lw[i];
    }
    return T;
}

__global__ void __launch_bounds__(128) k_prep(PrepArgs a) {
    int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= a.B * a.L) return;
    int b = idx / a.L, l = idx - b * a.L;
    const double* th = a.params + (size_t)b * a.P;

    bool finite = true;
    for (int i = 0; i < a.P; ++i) finite = finite && isfinite(th[i]);
    float* rec = a.rec + ((size_t)b * a.L + l) * a.rec_floats;
    const int i_extra = 2 + a.NT + a.S;
    const double* tpar = th + 2;
    const double* lvmr = th + 2 + a.NT;
    // Rejected models (helios.h, R31): a non-finite parameter, or an unphysical model -- a level
    // temperature <= 0, VMRs summing to more than 1, f < 0, d <= 0, or a derived quantity that overflows.
    // model_flag is zeroed before the launch; any thread of the model may raise it.
    double T = 0.0, T_up = 0.0, xsum = 0.0;
    bool ok = finite;
    if (finite) {
        T = level_temperature(tpar, a.tp_order, a.tp_ratio, a.lvl_elem[l], a.lvl_lw + (size_t)l * kMaxTpNodes);
        if (l + 1 < a.L)
            T_up = level_temperature(tpar, a.tp_order, a.tp_ratio, a.lvl_elem[l + 1], a.lvl_lw + (size_t)(l + 1) * kMaxTpNodes);
        for (int s = 0; s < a.S; ++s) xsum += pow(10.0, lvmr[s]);
        ok = T > 0.0 && isfinite(T) && (l + 1 >= a.L || (T_up > 0.0 && isfinite(T_up))) && xsum <= 1.0 &&
             isfinite(pow(10.0, th[0])) && th[1] >= 0.0;
        int ie = i_extra;
        if (a.extras & 1u) { ok = ok && th[ie] > 0.0; ++ie; }
        if (a.extras & 2u) { ok = ok && isfinite(pow(10.0, th[ie])); ++ie; }
        if (a.extras & 4u) ok = ok && isfinite(pow(10.0, th[ie])) && isfinite(pow(10.0, th[ie + 1]) * (1.0 + pow(10.0, th[ie + 2])));
    }
    if (!ok && atomicOr(&a.model_flag[b], 1) == 0) atomicAdd(&a.counters[1], 1ULL);
    if (l == 0) {
        double scale = a.unit_scale ? 1.0 : th[1] * a.flux_const;
        int ie = i_extra;
        if (a.extras & 1u) { if (!a.unit_scale) scale /= th[ie] * th[ie]; ++ie; }     // distance, Eq. 9
        a.model_addvar[b] = (ok && (a.extras & 2u)) ? pow(10.0, th[ie]) : 0.0;         // error inflation, Eq. 22
        a.model_scale[b] = ok ? (float)(scale * 2.0 * kPi) : 0.0f;
    }
    if (!ok) {
        for (int i = 0; i < a.rec_floats; ++i) rec[i] = 0.0f;
        if (l == 0 && a.slab_layout) for (int i = 0; i < a.x_floats; ++i) a.model_x[(size_t)b * a.x_floats + i] = 0.0f;
        return;
    }

    const double g = pow(10.0, th[0]);
    const double p = a.lvl_p_bar[l];

    // temperature cell: largest iT with T_grid[iT] <= T, clamped to [0, nT-2]
    int iT = 0;
    for (int k = 0; k < a.nT; ++k) if (a.T_grid[k] <= T) iT = k;
    if (iT > a.nT - 2) iT = a.nT - 2;
    double t = (T - a.T_grid[iT]) / (a.T_grid[iT + 1] - a.T_grid[iT]);
    int clamped = a.lvl_pclamp[l];
    if (t < 0.0) { t = 0.0; clamped = 1; }
    if (t > 1.0) { t = 1.0; clamped = 1; }
    if (clamped) atomicAdd(&a.counters[0], 1ULL);
    const double u = a.lvl_u[l];

    const double n = p * kBarCgs / (kBoltzmann * T);     // cm^-3
    const double x_bg = 1.0 - xsum;
    const double x_h2 = x_bg / (1.0 + a.he_to_h2);
    const double x_he = x_bg * a.he_to_h2 / (1.0 + a.he_to_h2);
    const double am = n / kAmagat;

    int o = 0;
    if (!a.slab_layout) {
        for (int s = 0; s < a.S; ++s) {
            double w = n * pow(10.0, lvmr[s]);
            rec[o++] = (float)(w * (1.0 - t) * (1.0 - u));
            rec[o++] = (float)(w * (1.0 - t) * u);
            rec[o++] = (float)(w * t * (1.0 - u));
            rec[o++] = (float)(w * t * u);
        }
        for (int c = 0; c < a.C; ++c) {
            double w = am * am * x_h2 * (c == 0 ? x_h2 : x_he);
            rec[o++] = (float)(w * (1.0 - t));
            rec[o++] = (float)(w * t);
        }
    } else {
        const double w = n / (double)kSlabXScale;
        rec[o++] = (float)(w * (1.0 - t) * (1.0 - u));
        rec[o++] = (float)(w * (1.0 - t) * u);
        rec[o++] = (float)(w * t * (1.0 - u));
        rec[o++] = (float)(w * t * u);
        rec[o++] = (float)(am * am * (1.0 - t));
        rec[o++] = (float)(am * am * t);
        if (l == 0) {
            float* mx = a.model_x + (size_t)b * a.x_floats;
            int k = 0;
            for (int s = 0; s < a.S; ++s) mx[k++] = (float)(pow(10.0, lvmr[s]) * (double)kSlabXScale);
            for (int c = 0; c < a.C; ++c) mx[k++] = (float)(x_h2 * (c == 0 ? x_h2 : x_he));
            while (k < a.x_floats) mx[k++] = 0.0f;
        }
    }
    // Planck exponent scale and half layer thickness (hydrostatic, ideal gas; R5)
    {
        const double a = kC2 * kLog2e / T;
        const float a_hi = (float)a;
        rec[o++] = a_hi;
        rec[o++] = (float)(a - (double)a_hi);
    }
    double hdz = 0.0, dtc = 0.0;
    if (l + 1 < a.L) {
        double dz = kBoltzmann * 0.5 * (T + T_up) / (a.mmw * kAtomicMass * g) * a.lvl_lnratio[l];
        hdz = 0.5 * dz;
        if (a.extras & 4u) {
            // grey cloud (App. B, R29): tau_c spread uniformly in pressure over [p_top, p_top (1 + phi)];
            // the layer between levels l and l+1 gets the share of its pressure overlap
            const double* cp = th + 2 + a.NT + a.S + ((a.extras & 1u) ? 1 : 0) + ((a.extras & 2u) ? 1 : 0);
            const double tau_c = pow(10.0, cp[0]), p_top_c = pow(10.0, cp[1]), p_bot_c = p_top_c * (1.0 + pow(10.0, cp[2]));
            const double hi = fmin(p, p_bot_c), lo = fmax(a.lvl_p_bar[l + 1], p_top_c);
            if (hi > lo) dtc = tau_c * (hi - lo) / (p_bot_c - p_top_c);
        }
    }
    rec[o++] = (float)hdz;
    if (!a.slab_layout) rec[o++] = __int_as_float(iT * a.nP + a.lvl_ip[l]);
    rec[o++] = __int_as_float(iT);
    rec[o++] = (float)dtc;
    while (o < a.rec_floats) rec[o++] = 0.0f;
}

}  // namespace helios
