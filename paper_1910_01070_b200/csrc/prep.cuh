// prep.cuh -- step 0 of the hot path: per (model, level) profile
// quantities, interpolation cells/weights and number-density-weighted tap weights.
// fp64 arithmetic, fp32 results.  PAPER.md:55 (levels), 174-221 (finite-element
// temperature profile), 484 (isoprofiles, H2/He fill), 241 (interpolation).
//
// One CTA per model: the model-wide quantities (10^VMR, g, flux scale, validity) are computed
// once, in parallel, and shared; the threads then stride over the levels.  (One thread per
// (model, level) repeated ~S+3 double-precision pow() calls in every thread: 20 us for one model.)
#pragma once
#include "common.cuh"
#include "obs.cuh"

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
    float* model_x;           // DEVICE [B][x_floats]  staged kernels: x_s 2^32, x_H2 x_c
    int x_floats;
    float* model_scale;       // DEVICE [B]  f * flux_const * 2 pi
    int*   model_flag;        // DEVICE [B]  1 = rejected model
    unsigned long long* counters;  // [0] clamped pairs, [1] rejected models
    // fused observation (obs.cuh): per (model, bin) the integer accumulator is zeroed and its power-of-two scale set
    unsigned long long* fused_acc; // DEVICE [B][J] or nullptr
    float* fused_q;                // DEVICE [B][J]
    int J;
    const int* row_ptr;            // DEVICE [J + 1]  band of every bin: grid points row_lo[j] .. row_lo[j] + len_j - 1
    const int* row_lo;             // DEVICE [J]
    double nu0, dnu;
};

constexpr int kMaxTpNodes = 5;    // order <= 4
constexpr int kPrepThreads = 128;
constexpr int kPrepMaxSpecies = 64;
constexpr int kPrepMaxLevels = 4096;
constexpr int kPrepMaxTgrid = 256;
constexpr int kPrepIpLevels = 1024;

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

__global__ void __launch_bounds__(kPrepThreads) k_prep(PrepArgs a) {
    __shared__ double sx[kPrepMaxSpecies];     // 10^(log10 VMR)
    __shared__ double sm[8];                   // g, x_h2, x_he, cloud tau, cloud p_top, cloud p_bot
    __shared__ int s_ok;
    __shared__ short s_cell[kPrepMaxLevels];   // temperature cell of every level (cell-walk schedule below)
    __shared__ double s_T[kPrepMaxLevels];     // temperature of every level (each one is needed by three levels)
    __shared__ short s_ip[kPrepIpLevels];      // pressure cell of every level (global memory for longer atmospheres)
    __shared__ double s_Tg[kPrepMaxTgrid];     // the table's temperature grid (global memory when it is longer)
    const int b = blockIdx.x, tid = threadIdx.x;
    pdl_launch_dependents();       // the RT kernel may be scheduled now; it waits for this grid before reading the records
    // static per-level data first, all loads in flight at once: with one model the kernel is a chain of dependent
    // load latencies (the bisection on the temperature grid alone was five round trips to L2)
    const double* Tg = a.nT <= kPrepMaxTgrid ? s_Tg : a.T_grid;
    if (a.nT <= kPrepMaxTgrid) for (int k = tid; k < a.nT; k += kPrepThreads) s_Tg[k] = a.T_grid[k];
    const bool ip_s = a.L <= kPrepIpLevels;
    if (ip_s) for (int l = tid; l < a.L; l += kPrepThreads) s_ip[l] = (short)a.lvl_ip[l];
    auto ip_of = [&](int l) { return ip_s ? (int)s_ip[l] : a.lvl_ip[l]; };
    const double* th = a.params + (size_t)b * a.P;
    const double* tpar = th + 2;
    const double* lvmr = th + 2 + a.NT;
    const int i_extra = 2 + a.NT + a.S;

    bool fin = true;
    for (int i = tid; i < a.P; i += kPrepThreads) fin = fin && isfinite(th[i]);
    const int finite = __syncthreads_and(fin);
    if (tid < a.S) sx[tid] = finite ? exp10(lvmr[tid]) : 0.0;
    __syncthreads();
    // Rejected models (helios.h, R31): a non-finite parameter, or an unphysical model -- VMRs summing
    // to more than 1, f < 0, d <= 0, an overflowing derived quantity, or (below) a level temperature <= 0.
    if (tid == 0) {
        bool ok = finite != 0;
        double xsum = 0.0;
        for (int s = 0; s < a.S; ++s) xsum += sx[s];
        double g = 1.0, scale = 0.0, addvar = 0.0;
        if (ok) {
            g = exp10(th[0]);
            ok = isfinite(g) && xsum <= 1.0 && th[1] >= 0.0;
            scale = a.unit_scale ? 1.0 : th[1] * a.flux_const;
            int ie = i_extra;
            if (a.extras & 1u) { ok = ok && th[ie] > 0.0; if (!a.unit_scale) scale /= th[ie] * th[ie]; ++ie; }   // distance, Eq. 9
            if (a.extras & 2u) { addvar = exp10(th[ie]); ok = ok && isfinite(addvar); ++ie; }                    // Eq. 22
            if (a.extras & 4u) {      // grey cloud (App. B, R29): tau_c uniform in pressure over [p_top, p_top (1 + phi)]
                sm[3] = exp10(th[ie]); sm[4] = exp10(th[ie + 1]); sm[5] = sm[4] * (1.0 + exp10(th[ie + 2]));
                ok = ok && isfinite(sm[3]) && isfinite(sm[5]);
            }
        }
        const double x_bg = 1.0 - xsum;
        sm[0] = g; sm[1] = x_bg / (1.0 + a.he_to_h2); sm[2] = x_bg * a.he_to_h2 / (1.0 + a.he_to_h2);
        sm[6] = scale; sm[7] = addvar;
        s_ok = ok ? 1 : 0;
    }
    __syncthreads();
    const bool model_ok = s_ok != 0;
    const double g = sm[0], x_h2 = sm[1], x_he = sm[2];

    if (a.slab_layout) {
        float* mx = a.model_x + (size_t)b * a.x_floats;
        for (int k = tid; k < a.x_floats; k += kPrepThreads) {
            float v = 0.0f;
            if (model_ok && k < a.S) v = (float)(sx[k] * (double)kSlabXScale);
            else if (model_ok && k < a.S + a.C) v = (float)(x_h2 * (k - a.S == 0 ? x_h2 : x_he));
            mx[k] = v;
        }
    }

    if (model_ok)
        for (int l = tid; l < a.L; l += kPrepThreads)
            s_T[l] = level_temperature(tpar, a.tp_order, a.tp_ratio, a.lvl_elem[l], a.lvl_lw + (size_t)l * kMaxTpNodes);
    __syncthreads();

    bool bad_level = false;
    for (int l = tid; l < a.L; l += kPrepThreads) {
        float* rec = a.rec + ((size_t)b * a.L + l) * a.rec_floats;
        double T = 0.0, T_up = 0.0, T_dn = 0.0;
        bool ok = model_ok;
        if (ok) {
            T = s_T[l];
            if (l + 1 < a.L) T_up = s_T[l + 1];
            if (l > 0) T_dn = s_T[l - 1];
            ok = T > 0.0 && isfinite(T) && (l + 1 >= a.L || (T_up > 0.0 && isfinite(T_up))) && (l == 0 || (T_dn > 0.0 && isfinite(T_dn)));
        }
        if (!ok) {
            bad_level = true;
            for (int i = 0; i < a.rec_floats; ++i) rec[i] = 0.0f;
            s_cell[l] = 0;
            continue;
        }
        const double p = a.lvl_p_bar[l];
        // temperature cell: largest iT with T_grid[iT] <= T, clamped to [0, nT-2]
        int iT = 0;
        for (int hi = a.nT - 1; hi - iT > 1;) {       // bisection: T_grid[iT] <= T < T_grid[hi] (or T outside the grid)
            const int mid = (iT + hi) >> 1;
            if (Tg[mid] <= T) iT = mid; else hi = mid;
        }
        double t = (T - Tg[iT]) / (Tg[iT + 1] - Tg[iT]);
        int clamped = a.lvl_pclamp[l];
        if (t < 0.0) { t = 0.0; clamped = 1; }
        if (t > 1.0) { t = 1.0; clamped = 1; }
        if (clamped) atomicAdd(&a.counters[0], 1ULL);
        s_cell[l] = (short)iT;
        const double u = a.lvl_u[l];
        const double n = p * kBarCgs / (kBoltzmann * T);     // cm^-3
        const double am = n / kAmagat;
        // half layer thickness (hydrostatic, ideal gas; R5) and grey-cloud optical depth of the layer
        // above (levels l, l+1) and of the layer below (levels l-1, l)
        const double hscale = kBoltzmann * 0.25 / (a.mmw * kAtomicMass * g);
        double hdz_up = 0.0, hdz_dn = 0.0, dtc_up = 0.0, dtc_dn = 0.0;
        if (l + 1 < a.L) hdz_up = hscale * (T + T_up) * a.lvl_lnratio[l];
        if (l > 0) hdz_dn = hscale * (T_dn + T) * a.lvl_lnratio[l - 1];
        if (a.extras & 4u) {
            const double tau_c = sm[3], p_top_c = sm[4], p_bot_c = sm[5];
            if (l + 1 < a.L) {
                const double hi = fmin(p, p_bot_c), lo = fmax(a.lvl_p_bar[l + 1], p_top_c);
                if (hi > lo) dtc_up = tau_c * (hi - lo) / (p_bot_c - p_top_c);
            }
            if (l > 0) {
                const double hi = fmin(a.lvl_p_bar[l - 1], p_bot_c), lo = fmax(p, p_top_c);
                if (hi > lo) dtc_dn = tau_c * (hi - lo) / (p_bot_c - p_top_c);
            }
        }
        const double pa = kC2 * kLog2e / T;                  // Planck exponent scale: E = 2^(-pa nu)
        const float pa_hi = (float)pa, pa_lo = (float)(pa - (double)pa_hi);
        int o = 0;
        if (!a.slab_layout) {
            for (int s = 0; s < a.S; ++s) {
                const double w = n * sx[s];
                rec[o++] = (float)(w * (1.0 - t) * (1.0 - u));
                rec[o++] = (float)(w * (1.0 - t) * u);
                rec[o++] = (float)(w * t * (1.0 - u));
                rec[o++] = (float)(w * t * u);
            }
            for (int c = 0; c < a.C; ++c) {
                const double w = am * am * x_h2 * (c == 0 ? x_h2 : x_he);
                rec[o++] = (float)(w * (1.0 - t));
                rec[o++] = (float)(w * t);
            }
            rec[o++] = pa_hi; rec[o++] = pa_lo;
            rec[o++] = (float)hdz_up;
            rec[o++] = __int_as_float(iT * a.nP + ip_of(l));
            rec[o++] = __int_as_float(iT);
            rec[o++] = (float)dtc_up;
        } else {                 // kSlabRecFloats floats, layout in common.cuh
            const double w = n / (double)kSlabXScale;
            rec[o++] = (float)(w * (1.0 - t) * (1.0 - u));
            rec[o++] = (float)(w * (1.0 - t) * u);
            rec[o++] = (float)(w * t * (1.0 - u));
            rec[o++] = (float)(w * t * u);
            rec[o++] = (float)(am * am * (1.0 - t));
            rec[o++] = (float)(am * am * t);
            rec[o++] = pa_hi; rec[o++] = pa_lo;
            rec[o++] = (float)hdz_dn;
            rec[o++] = __int_as_float(iT);
            rec[o++] = (float)dtc_dn;
        }
        while (o < a.rec_floats) rec[o++] = 0.0f;
    }
    const int any_bad = __syncthreads_or(bad_level);
    if (a.slab_layout) {
        // Cell-walk schedule (slot 11 of the staged record, read by the level-parallel kernel): how the table cell of
        // level l relates to the cell of level l - 1 -- 4 same cell, 1 one cell colder, 2 one cell hotter, 3 next
        // pressure cell upwards at the same temperature cell, 0 anything else -- and the distance to the next level
        // that lies in another cell (0: none), so that the kernel can prefetch a cell's corners without scanning.
        for (int l = tid; l < a.L; l += kPrepThreads) {
            int kind = 0;
            if (l > 0) {
                const int iT0 = s_cell[l - 1], ip0 = ip_of(l - 1), iT1 = s_cell[l], ip1 = ip_of(l);
                kind = ip1 == ip0 ? (iT1 == iT0 ? 4 : (iT1 == iT0 - 1 ? 1 : (iT1 == iT0 + 1 ? 2 : 0)))
                                  : ((iT1 == iT0 && ip1 == ip0 - 1) ? 3 : 0);
            }
            int j = l + 1;
            while (j < a.L && s_cell[j] == s_cell[l] && ip_of(j) == ip_of(l)) ++j;
            const int dist = j < a.L ? j - l : 0;
            a.rec[((size_t)b * a.L + l) * a.rec_floats + 11] = __int_as_float(kind | (dist << 8));
        }
    }
    if (a.fused_acc) {
        // the largest value a bin can take for this model: pi f (R/d)^2 max_band B_nu(T_max) (see obs.cuh)
        __shared__ double s_red[kPrepThreads];
        double tmax = 0.0;
        for (int l = tid; l < a.L; l += kPrepThreads) tmax = fmax(tmax, s_T[l]);
        s_red[tid] = tmax;
        __syncthreads();
        for (int o = kPrepThreads / 2; o > 0; o >>= 1) {
            if (tid < o) s_red[tid] = fmax(s_red[tid], s_red[tid + o]);
            __syncthreads();
        }
        tmax = s_red[0];
        const bool ok = model_ok && !any_bad;
        const double amp = 0.5 * sm[6] * 2.0 * kPi;             // model_scale (below) x sum_k w_k mu_k
        for (int j = tid; j < a.J; j += kPrepThreads) {
            const int lo = a.row_lo[j], len = a.row_ptr[j + 1] - a.row_ptr[j];
            float q = 0.0f;
            if (ok && len > 0) q = fused_scale(amp * planck_band_max(a.nu0 + a.dnu * lo, a.nu0 + a.dnu * (lo + len - 1), tmax));
            a.fused_q[(size_t)b * a.J + j] = q;
            a.fused_acc[(size_t)b * a.J + j] = 0ull;
        }
    }
    if (tid == 0) {
        const bool ok = model_ok && !any_bad;
        a.model_flag[b] = ok ? 0 : 1;
        a.model_scale[b] = ok ? (float)(sm[6] * 2.0 * kPi) : 0.0f;
        a.model_addvar[b] = ok ? sm[7] : 0.0;
        if (!ok) atomicAdd(&a.counters[1], 1ULL);
    }
}

}  // namespace helios
