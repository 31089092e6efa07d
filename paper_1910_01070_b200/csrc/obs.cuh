// obs.cuh -- step 5 of the hot path: instrument profile (Eq. 17,
// PAPER.md:229-235), binning and likelihood (Eq. 19,
// PAPER.md:267-270), fused.
//
// "Convolve on the native grid, then bin-average" is linear and model-independent,
// so helios_set_observation() builds ONE banded operator W[J][band] on the device
// (fp64 arithmetic, fp32 storage) and the per-batch kernel applies it:
//     M_j = sum_i W_ji F_i,   W_ji = sum_k b_jk c_ki
//   c_ki = g(nu_i - nu_k; sigma_k) / sum_i' g(nu_i' - nu_k; sigma_k), |nu_i - nu_k| <= 5 sigma_k
//   b_jk = (1/(e_{j+1} - e_j)) * integral over the bin of the hat function of grid point k
//          (= the weight of F_d[k] in the bin mean of the piecewise-linear interpolant).
// DESIGN.md R15, R17, R18.
#pragma once
#include <math_constants.h>

#include "common.cuh"

namespace helios {

struct ObsBuildArgs {
    int nNu, J;
    double nu0, dnu;
    const double* edges;       // DEVICE [J+1]
    const double* inst_sigma;  // DEVICE [nNu] or nullptr
    double* conv_norm;         // DEVICE [nNu]  sum of Gaussian weights actually used
    const int* row_ptr;        // DEVICE [J+1]
    const int* row_lo;         // DEVICE [J]    first grid index of the row's band
    const int* row_klo;        // DEVICE [J]    first / last grid point with non-zero bin weight
    const int* row_khi;
    float* W;                  // DEVICE [row_ptr[J]]
};

__global__ void k_conv_norm(ObsBuildArgs a) {
    int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= a.nNu) return;
    double sg = a.inst_sigma ? a.inst_sigma[k] : 0.0;
    if (!(sg > 0.0)) { a.conv_norm[k] = 1.0; return; }
    int reach = (int)ceil(5.0 * sg / a.dnu) + 1;
    int lo = max(0, k - reach), hi = min(a.nNu - 1, k + reach);
    double nu_k = a.nu0 + a.dnu * k;
    double sum = 0.0;
    for (int i = lo; i <= hi; ++i) {
        double d = (a.nu0 + a.dnu * i) - nu_k;
        if (fabs(d) <= 5.0 * sg) sum += exp(-d * d / (2.0 * sg * sg));
    }
    a.conv_norm[k] = sum;
}

// integral of the unit hat function centred at 0 with half-width 1, from -inf to s
__device__ __forceinline__ double hat_cdf(double s) {
    if (s <= -1.0) return 0.0;
    if (s >= 1.0) return 1.0;
    return s < 0.0 ? 0.5 * (1.0 + s) * (1.0 + s) : 1.0 - 0.5 * (1.0 - s) * (1.0 - s);
}

__global__ void k_build_W(ObsBuildArgs a) {
    const int j = blockIdx.y;
    const int len = a.row_ptr[j + 1] - a.row_ptr[j];
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= len) return;
    const int i = a.row_lo[j] + e;
    const double ea = a.edges[j], eb = a.edges[j + 1];
    const double nu_i = a.nu0 + a.dnu * i;
    double w = 0.0;
    for (int k = a.row_klo[j]; k <= a.row_khi[j]; ++k) {
        const double nu_k = a.nu0 + a.dnu * k;
        const double bjk = (hat_cdf((eb - nu_k) / a.dnu) - hat_cdf((ea - nu_k) / a.dnu)) * a.dnu / (eb - ea);
        if (bjk == 0.0) continue;
        const double sg = a.inst_sigma ? a.inst_sigma[k] : 0.0;
        if (!(sg > 0.0)) { if (i == k) w += bjk; continue; }
        const double d = nu_i - nu_k;
        if (fabs(d) <= 5.0 * sg) w += bjk * exp(-d * d / (2.0 * sg * sg)) / a.conv_norm[k];
    }
    a.W[a.row_ptr[j] + e] = (float)w;
}

struct ObsApplyArgs {
    int J;
    const int* row_ptr;
    const int* row_lo;
    const float* W;
    const float* flux;        // DEVICE [B][flux_stride]
    long long flux_stride;
    const int* model_flag;
    const double* obs;        // DEVICE [J] or nullptr
    const double* inv2var;    // DEVICE [J]  1 / (2 sigma_j^2)
    double logl_const;        // -1/2 sum_j ln(2 pi sigma_j^2)
    float* spectra;           // DEVICE [B][J] or nullptr
    double* logl;             // DEVICE [B] or nullptr
    const double* var;        // DEVICE [J]  sigma_j^2          } error inflation (Eq. 22-23): both non-null,
    const double* addvar;     // DEVICE [B]  10^epsilon of each model } s_j^2 = var_j + addvar_b
    double* partial;          // DEVICE [B][n_chunks] chi-square of each bin chunk (workspace)
    unsigned* arrived;        // DEVICE [B] chunks finished per model; zero between launches (workspace)
};

constexpr int kObsThreads = 256;
constexpr int kObsBinsPerCta = 64;   // 8 warps x 8 bins (large batches); 8 warps x 1 bin for a handful of models

// One CTA per (model, chunk of 64 bins): B * J / 64 CTAs keep every SM busy (one CTA per model
// left 14 warps per SM waiting on dependent L2 loads).  Each warp owns 8 bins: lanes stride the
// band of W, a shuffle tree finishes M_j, lane 0 adds the chi-square term in fp64.  The chunk
// sums go to `partial`; the CTA that finishes a model last (atomic ticket) adds them in chunk
// order, so logL is bitwise reproducible, and only logL is written when spectra == nullptr.
// With a handful of models B * J / 64 CTAs do not fill the GPU and the 8 bins of a warp are 8 chains of dependent
// loads one after the other: kPerWarp = 1 gives every bin its own warp (8 bins per CTA).
template <int kPerWarp>
__global__ void __launch_bounds__(kObsThreads) k_obs_apply(ObsApplyArgs a) {
    __shared__ double warp_sum[kObsThreads / 32];
    __shared__ double tree[kObsThreads];
    __shared__ unsigned ticket;
    const int b = blockIdx.y, chunk = blockIdx.x, n_chunks = gridDim.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    constexpr int kBinsPerCta = kPerWarp * (kObsThreads / 32);
    pdl_wait();                    // the flux (RT kernel) and the model flags (prep kernel) are complete
    const bool bad = a.model_flag[b] != 0;
    const float* F = a.flux + (size_t)b * a.flux_stride;
    const double add = a.addvar ? a.addvar[b] : 0.0;
    double chi2 = 0.0;
    const int j0 = chunk * kBinsPerCta + warp * kPerWarp;
#pragma unroll 2
    for (int j = j0; j < min(j0 + kPerWarp, a.J); ++j) {
        const int p0 = a.row_ptr[j], len = a.row_ptr[j + 1] - p0;
        const float* w = a.W + p0;
        const float* f = F + a.row_lo[j];
        float acc0 = 0.0f, acc1 = 0.0f;
        int i = lane;
        for (; i + 32 < len; i += 64) {
            acc0 = fmaf(w[i], f[i], acc0);
            acc1 = fmaf(w[i + 32], f[i + 32], acc1);
        }
        if (i < len) acc0 = fmaf(w[i], f[i], acc0);
        float acc = acc0 + acc1;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) {
            if (bad) acc = __int_as_float(0x7fc00000);
            if (a.spectra) a.spectra[(size_t)b * a.J + j] = acc;
            if (a.logl) {
                // every bin's term is rounded on its own and then added (explicit _rn intrinsics: no contraction into an
                // FMA with the running sum), so the two variants of this kernel give bitwise the same logL
                const double r = a.obs[j] - (double)acc;
                double term;
                if (a.addvar) {                       // Eq. 23: the normalisation depends on the model too
                    const double s2 = a.var[j] + add;
                    term = __dadd_rn(__ddiv_rn(__dmul_rn(r, r), __dmul_rn(2.0, s2)), __dmul_rn(0.5, log(__dmul_rn(2.0 * kPi, s2))));
                } else {
                    term = __dmul_rn(__dmul_rn(r, r), a.inv2var[j]);
                }
                chi2 = __dadd_rn(chi2, term);
            }
        }
    }
    if (!a.logl) return;
    // chi-square is summed in GROUPS of 8 consecutive bins, in bin order, and the groups in group order: a warp's own
    // sum is a group when it owns 8 bins; with one bin per warp the CTA's 8 bins are a group.  Same grouping in both
    // variants, so logL does not depend on which one ran.
    const int n_groups = (a.J + 7) / 8;
    if (kPerWarp == 8) {
        const int g = chunk * (kObsThreads / 32) + warp;
        if (lane == 0 && g < n_groups) a.partial[(size_t)b * n_groups + g] = chi2;
    } else if (lane == 0) {
        warp_sum[warp] = chi2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        if (kPerWarp != 8) {
            double s = 0.0;
            for (int w = 0; w < kObsThreads / 32; ++w) s += warp_sum[w];
            a.partial[(size_t)b * n_groups + chunk] = s;
        }
        __threadfence();
        ticket = atomicAdd(&a.arrived[b], 1u);
    }
    __syncthreads();
    if (ticket != (unsigned)n_chunks - 1) return;
    // Every chunk of this model is in `partial`: the CTA that arrived last adds the group sums in a FIXED order
    // (thread t takes groups t, t + 256, ...; then a binary tree over the threads), so logL is bitwise reproducible
    // and the same in both variants.  (One thread adding 125 partials one after the other took 4 us of a 12 us kernel.)
    __threadfence();
    double t = 0.0;
    for (int c = threadIdx.x; c < n_groups; c += kObsThreads) t += __ldcg(&a.partial[(size_t)b * n_groups + c]);
    tree[threadIdx.x] = t;
    __syncthreads();
#pragma unroll
    for (int o = kObsThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) tree[threadIdx.x] += tree[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        a.logl[b] = bad ? -CUDART_INF : (a.addvar ? -tree[0] : a.logl_const - tree[0]);
        a.arrived[b] = 0;
    }
}

// ---------------------------------------------------------------------------------------
// Fused variant: the RT kernels apply the operator themselves, in their epilogue, and no high-resolution flux
// is written at all (north_star: "writes only logL when spectra are not requested").  A lane that has just
// finished the flux F of grid point i adds W_ji F to M_j for the handful of bins j whose band holds i
// (the transposed operator, CSR by grid point: wt_ptr / wt_j / wt_w).  The wavenumbers of a warp are
// scattered over the grid (opacity order) and a bin is fed by ~1500 CTAs, so the sums are ATOMIC -- and to keep
// them bitwise reproducible they are INTEGER: every term is scaled by a per-(model, bin) power of two q_bj,
// rounded to a 64-bit integer and added with a 64-bit atomic; integer addition is associative, so the result does
// not depend on the order in which the CTAs arrive.  q_bj = 2^(60 - e) with 2^e > the largest value M_j can take
// for that model, pi f (R/d)^2 max over the band of B_nu(T_max) (every intensity is a convex combination of level
// sources, W rows are non-negative and sum to 1), worked out by k_prep: the sum cannot overflow, and one unit is
// 2^-60 of that bound.  k_obs_final turns the integers back into M_j (exactly, in fp64) and forms chi-square with
// the same grouping and tree as k_obs_apply.
// ---------------------------------------------------------------------------------------
struct FusedObs {
    unsigned long long* acc;   // DEVICE [B][J]  integer sums, zeroed by k_prep; nullptr = not fused (write the flux)
    const float* q;            // DEVICE [B][J]  power-of-two scales (0: model rejected or flux identically 0)
    const int* wt_ptr;         // DEVICE [nNu + 1]
    const int* wt_j;           // DEVICE [nnz]  bin
    const float* wt_w;         // DEVICE [nnz]  W_ji (zeros dropped)
    int J;
};

__device__ __forceinline__ void fused_accumulate(const FusedObs& f, int b, int i, float F) {
    const int t0 = __ldg(f.wt_ptr + i), t1 = __ldg(f.wt_ptr + i + 1);
    unsigned long long* acc = f.acc + (size_t)b * f.J;
    const float* q = f.q + (size_t)b * f.J;
    for (int t = t0; t < t1; ++t) {
        const int j = __ldg(f.wt_j + t);
        const float v = __fmul_rn(__fmul_rn(__ldg(f.wt_w + t), F), __ldg(q + j));       // the scale is a power of two: exact
        atomicAdd(acc + j, (unsigned long long)__float2ll_rn(v));
    }
}

// B_nu(T) at its maximum over [nu_a, nu_b] (the Planck function is unimodal; peak at c2 nu / T = 2.821439...), fp64
__device__ __forceinline__ double planck_band_max(double nu_a, double nu_b, double T) {
    double nu = 2.8214393721220787 * T / kC2;
    nu = fmin(fmax(nu, nu_a), nu_b);
    return kC1 * nu * nu * nu / expm1(kC2 * nu / T);
}
// q_bj for one (model, bin): bound = largest possible M_j; returns 2^(60 - e), bound < 2^e, clamped to the fp32 range
__device__ __forceinline__ float fused_scale(double bound) {
    if (!(bound > 0.0) || !isfinite(bound)) return 0.0f;
    int e;
    frexp(bound, &e);                     // bound = m 2^e, 0.5 <= m < 1
    int qe = 60 - e;
    qe = qe > 127 ? 127 : (qe < -126 ? -126 : qe);
    return __int_as_float((qe + 127) << 23);
}

__global__ void __launch_bounds__(kObsThreads) k_obs_final(ObsApplyArgs a, FusedObs f) {
    __shared__ double tree[kObsThreads];
    const int b = blockIdx.x;
    pdl_wait();                    // the integer sums (RT kernel), scales and flags (prep kernel) are complete
    const bool bad = a.model_flag[b] != 0;
    const unsigned long long* acc = f.acc + (size_t)b * a.J;
    const float* q = f.q + (size_t)b * a.J;
    const double add = a.addvar ? a.addvar[b] : 0.0;
    const int n_groups = (a.J + 7) / 8;
    double t = 0.0;
    for (int g = threadIdx.x; g < n_groups; g += kObsThreads) {       // thread t: groups t, t + 256, ... (k_obs_apply's order)
        double chi2 = 0.0;
        for (int j = 8 * g; j < min(8 * g + 8, a.J); ++j) {
            const float qj = q[j];
            float M = qj > 0.0f ? (float)((double)(long long)acc[j] * (1.0 / (double)qj)) : 0.0f;
            if (bad) M = __int_as_float(0x7fc00000);
            if (a.spectra) a.spectra[(size_t)b * a.J + j] = M;
            if (a.logl) {
                const double r = a.obs[j] - (double)M;
                double term;
                if (a.addvar) {                       // Eq. 23
                    const double s2 = a.var[j] + add;
                    term = __dadd_rn(__ddiv_rn(__dmul_rn(r, r), __dmul_rn(2.0, s2)), __dmul_rn(0.5, log(__dmul_rn(2.0 * kPi, s2))));
                } else {
                    term = __dmul_rn(__dmul_rn(r, r), a.inv2var[j]);
                }
                chi2 = __dadd_rn(chi2, term);
            }
        }
        t += chi2;
    }
    if (!a.logl) return;
    tree[threadIdx.x] = t;
    __syncthreads();
#pragma unroll
    for (int o = kObsThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) tree[threadIdx.x] += tree[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) a.logl[b] = bad ? -CUDART_INF : (a.addvar ? -tree[0] : a.logl_const - tree[0]);
}

// ---------------------------------------------------------------------------------------
// Effective temperature (Sect. 2.6): F_tot = integral of F+ over [nu_a, nu_b]
// (trapezoid on the grid with interpolated end points = sum_i F_i * integral of the hat function of
// grid point i over the window), T_eff = (F_tot / sigma_SB)^(1/4).  One CTA per model, fp64 sums
// combined in a fixed order.
// ---------------------------------------------------------------------------------------
struct TeffArgs {
    int nNu;
    double nu0, dnu, nu_a, nu_b;
    const float* flux;        // DEVICE [B][flux_stride]  F+ (prep ran with unit_scale)
    long long flux_stride;
    const int* model_flag;
    double* teff;             // DEVICE [B]
};

__global__ void __launch_bounds__(256) k_teff(TeffArgs a) {
    __shared__ double part[256];
    const int b = blockIdx.x;
    const float* F = a.flux + (size_t)b * a.flux_stride;
    int ia = (int)floor((a.nu_a - a.nu0) / a.dnu), ib = (int)ceil((a.nu_b - a.nu0) / a.dnu);
    ia = max(ia, 0); ib = min(ib, a.nNu - 1);
    double s = 0.0;
    for (int i = ia + threadIdx.x; i <= ib; i += 256) {
        const double nu_i = a.nu0 + a.dnu * i;
        const double h = (hat_cdf((a.nu_b - nu_i) / a.dnu) - hat_cdf((a.nu_a - nu_i) / a.dnu)) * a.dnu;
        s += h * (double)F[i];
    }
    part[threadIdx.x] = s;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if (threadIdx.x < o) part[threadIdx.x] += part[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const double sigma_sb = 2.0 * kPi * kPi * kPi * kPi * kPi * kBoltzmann * kBoltzmann * kBoltzmann * kBoltzmann /
                                (15.0 * kPlanckH * kPlanckH * kPlanckH * kLightC * kLightC);
        a.teff[b] = a.model_flag[b] ? CUDART_NAN : pow(part[0] / sigma_sb, 0.25);
    }
}

}  // namespace helios
