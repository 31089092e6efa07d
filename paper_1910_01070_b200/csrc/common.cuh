// common.cuh -- constants, record layouts and small device helpers shared by the
// kernels of libhelios_b200 (sm_100a only).  Nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace helios {

// CODATA 2018 (exact SI), cgs
constexpr double kPlanckH   = 6.62607015e-27;     // erg s
constexpr double kLightC    = 2.99792458e10;      // cm / s
constexpr double kBoltzmann = 1.380649e-16;       // erg / K
constexpr double kAtomicMass = 1.66053906660e-24; // g
constexpr double kBarCgs    = 1.0e6;              // dyn / cm^2
// 1 amagat: ideal-gas number density at 273.15 K, 101325 Pa
constexpr double kAmagat    = 1.01325e6 / (kBoltzmann * 273.15);
constexpr double kPi        = 3.14159265358979323846264338327950288;
constexpr double kLog2e     = 1.44269504088896340735992468100189214;
constexpr double kC1        = 2.0 * kPlanckH * kLightC * kLightC;   // 2 h c^2
constexpr double kC2        = kPlanckH * kLightC / kBoltzmann;      // h c / k_B

constexpr int kMaxAngles = 8;
constexpr int kMaxCia = 2;

// Per-(model, level) record written by the prep kernel for the DIRECT kernel, fp32:
//   [0, 4S)        species tap weights  n x_s {(1-t)(1-u), (1-t)u, t(1-u), t u}
//                  for table rows (iT,ip), (iT,ip+1), (iT+1,ip), (iT+1,ip+1)
//   [4S, 4S+2C)    CIA tap weights      am^2 x_H2 x_c {(1-t), t}   rows iT, iT+1
//   +0  planck_a   c2 log2(e) / T_l, high part (B_nu = c1 nu^3 E/(1-E), E = 2^(-planck_a nu))
//   +1  planck_a   low part (fp64 value minus the fp32 high part)
//   +2  hdz        dz_l / 2 of the layer between level l and l+1 (0 at the top level)
//   +3  cell       iT*nP + ip           (int bits)
//   +4  iT                               (int bits)
//   +5  dtau_cloud of the layer above the level (grey cloud, App. B; 0 without)
__host__ __device__ inline int direct_rec_floats(int S, int C) { return (4 * S + 2 * C + 6 + 3) & ~3; }

// Staged ("slab") kernel, fp32.  VMRs are constant with height, so the species
// sum commutes with the bilinear blend: chi_l = sum_corners w_corner G_corner with
// G_corner(nu) = sum_s x_s sigma_s[corner](nu), recomputed only when the model leaves a table cell.
// Per-(model, level) record, kSlabRecFloats floats:
//   0..3  n 2^-32 {(1-t)(1-u), (1-t)u, t(1-u), t u}   weights of G at (iT,ip), (iT,ip+1), (iT+1,ip), (iT+1,ip+1)
//   4..5  am^2 {(1-t), t}                               weights of the CIA mix at iT, iT+1
//   6..7  planck_a high / low      8  hdz of the layer BELOW the level (levels l-1, l; 0 at level 0)      9  iT (int bits)
//   10  dtau_cloud of the layer below      11  cell-walk schedule (int bits): kind | distance to the next cell change << 8 (prep.cuh)
// Per-model vector, slab_x_floats(S, C) floats: x_s 2^32 (S values), then x_H2 x_c (C values).
constexpr int kSlabRecFloats = 12;
constexpr float kSlabXScale = 4294967296.0f;   // 2^32: keeps x_s sigma_s far above the fp32 denormal range
__host__ __device__ inline int slab_x_floats(int S, int C) { return (S + C + 3) & ~3; }

struct AngleSet {
    int   n;
    float c_exp[kMaxAngles];   // log2(e) / mu_k      : e^{-dtau/mu} = 2^(-dtau * c_exp)
    float inv_mu[kMaxAngles];  // 1 / mu_k
    float mu[kMaxAngles];
    float wmu[kMaxAngles];     // w_k mu_k
    float wmu_sum;             // sum_k w_k mu_k ( = 1/2 up to rounding)
    // staged kernel, state H_k = J_k / mu_k (rt_slab.cuh)
    float thr[kMaxAngles];     // kPhiSwitch * mu_k   : small-D branch iff dtau < thr
    float pc[5][kMaxAngles];   // phi(dtau / mu_k) / mu_k = sum_j pc[j][k] dtau^j on the small-D branch
    float wH[kMaxAngles];      // w_k mu_k^2
};

// Chebyshev-node interpolant of phi(D) = (1 - e^{-D})/D on [0, 1/4], degree 4 (|error| < 5e-9);
// Taylor would need degree 6 for the same bound.  Constant term forced to 1.
constexpr double kPhiC1 = -0.49999951482099264, kPhiC2 = 0.16665108206599635, kPhiC3 = -0.041490654102785796,
                 kPhiC4 = 0.00751360621792363;

// Gauss-Legendre rule of order n = 1..8 on [-1,1] mapped to mu in (0,1): mu = (x+1)/2, w = W/2
// (R12).  Compile-time copy for the staged kernel, whose per-angle
// constants are instruction immediates; helios_set_atmosphere() checks it against the Newton
// solution it computes at run time.
constexpr double kGLmu[8][8] = {
    {0.5, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0},
    {0.21132486540518713, 0.7886751345948129, 1.0, 1.0, 1.0, 1.0, 1.0, 1.0},
    {0.1127016653792583, 0.5, 0.8872983346207417, 1.0, 1.0, 1.0, 1.0, 1.0},
    {0.06943184420297371, 0.33000947820757187, 0.6699905217924281, 0.9305681557970262, 1.0, 1.0, 1.0, 1.0},
    {0.04691007703066802, 0.23076534494715845, 0.5, 0.7692346550528415, 0.9530899229693319, 1.0, 1.0, 1.0},
    {0.03376524289842403, 0.16939530676686776, 0.38069040695840156, 0.6193095930415985, 0.8306046932331322, 0.9662347571015759, 1.0, 1.0},
    {0.0254460438286207, 0.12923440720030277, 0.2970774243113014, 0.5, 0.7029225756886985, 0.8707655927996972, 0.9745539561713793, 1.0},
    {0.019855071751231912, 0.10166676129318664, 0.2372337950418355, 0.4082826787521751, 0.5917173212478248, 0.7627662049581645, 0.8983332387068134, 0.9801449282487681},
};
constexpr double kGLw[8][8] = {
    {1.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {0.5, 0.5, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {0.27777777777777785, 0.4444444444444444, 0.27777777777777785, 0.0, 0.0, 0.0, 0.0, 0.0},
    {0.17392742256872679, 0.3260725774312732, 0.3260725774312732, 0.17392742256872679, 0.0, 0.0, 0.0, 0.0},
    {0.11846344252809464, 0.23931433524968315, 0.28444444444444433, 0.23931433524968315, 0.11846344252809464, 0.0, 0.0, 0.0},
    {0.08566224618958514, 0.18038078652406936, 0.23395696728634552, 0.23395696728634552, 0.18038078652406936, 0.08566224618958514, 0.0, 0.0},
    {0.06474248308443487, 0.13985269574463843, 0.19091502525255935, 0.20897959183673465, 0.19091502525255935, 0.13985269574463843, 0.06474248308443487, 0.0},
    {0.05061426814518853, 0.11119051722668721, 0.15685332293894344, 0.18134189168918083, 0.18134189168918083, 0.15685332293894344, 0.11119051722668721, 0.05061426814518853},
};
__host__ __device__ constexpr double cpow(double b, int e) { double r = 1.0; for (int i = 0; i < e; ++i) r *= b; return r; }

// Programmatic dependent launch (sm_90+): the three kernels of a call are launched back to back with the
// programmatic-stream-serialization attribute, so the next kernel's CTAs are scheduled and run their prologue while
// the previous kernel drains; pdl_wait() blocks until the previous kernel has completed and its writes are visible
// (a no-op when the kernel was launched without the attribute).
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

template <class... KArgs, class... Args>
inline cudaError_t launch_kernel(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, bool pdl,
                                 Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

__device__ __forceinline__ float ex2_approx(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ float rcp_approx(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// E = exp(-c2 nu / T) = 2^(-a nu) with a = a_hi + a_lo and nu = nu_hi + nu_lo carried as
// two-float numbers: the exponent reaches ~50 in the Wien tail, where one fp32 rounding of
// a*nu alone costs 3e-6 relative in E -- enough to move logL by more than 1e-3.  The product
// is formed exactly (FMA residual) and the sub-ulp part applied as a first-order factor.
__device__ __forceinline__ float planck_E(float a_hi, float a_lo, float nu_hi, float nu_lo) {
    const float p = a_hi * nu_hi;
    float r = fmaf(a_hi, nu_hi, -p);        // exact low part of the product
    r = fmaf(a_lo, nu_hi, r);
    r = fmaf(a_hi, nu_lo, r);
    const float E0 = ex2_approx(-p);
    return fmaf(E0 * -0.69314718056f, r, E0);
}

// B_nu(T) = c1 nu^3 E / (1 - E)  (Eq. 2, per-wavenumber form; never exp(+x)).
__device__ __forceinline__ float planck_from_E(float c1nu3, float E) {
    return c1nu3 * (E * rcp_approx(1.0f - E));
}

// Short-characteristics update for one angle in deviation form.
// With J = I - S(level) and dS = S_{l-1} - S_l, Eq. 4-6 read
//   J_l = e^{-D} J_{l-1} + phi(D) dS,   phi(D) = (1 - e^{-D})/D,   D = dtau / mu  (Eq. 7)
// (beta = 1 - phi, gamma = phi - e^{-D}).  For D < kPhiSwitch, where (1 - e^{-D})/D cancels
// in fp32, phi comes from a degree-4 near-minimax polynomial (R10).
constexpr float kPhiSwitch = 0.25f;
__device__ __forceinline__ float phi_small(float D) {
    float p = fmaf(D, (float)kPhiC4, (float)kPhiC3);
    p = fmaf(D, p, (float)kPhiC2);
    p = fmaf(D, p, (float)kPhiC1);
    return fmaf(D, p, 1.0f);
}
// Small D: e^{-D} = 1 - D phi(D) exactly, so J_l = J + phi (dS - D J): correctly rounded
// FMAs and no exponential.  (MUFU.EX2 results just below 1 carry a one-sided error of a
// fraction of an ulp; through ~50 transparent layers that biased the flux by -4e-7, which
// the absolute logL tolerance does not allow.)  Large D: hardware 2^x, J_l = e J + (1 - e) t
// with t = mu dS / dtau.  q = dS / dtau is shared by all angles of the layer.
__device__ __forceinline__ void sc_update(float& J, float dtau, float q, float dS,
                                          float c_exp, float inv_mu, float mu) {
    const float D = dtau * inv_mu;
    const float e = ex2_approx(-dtau * c_exp);
    const float t = mu * q;
    const float J_big = fmaf(e, J, fmaf(-e, t, t));
    const float J_small = fmaf(phi_small(D), fmaf(-D, J, dS), J);
    J = (D < kPhiSwitch) ? J_small : J_big;
}

}  // namespace helios
