// rt_slab.cuh -- fused steps 1-4, large-batch variant.
//
// One CTA = NW compute warps + 1 producer warp, working on ONE 64-point wavenumber tile
// for NW models: compute warp w = model w of the group, each lane owns TWO adjacent
// wavenumbers and does all of its fp32 arithmetic as packed pairs (FFMA2/FMUL2/FADD2,
// sm_100 fma.rn.f32x2), which halves the issue slots of an issue-bound kernel.
//
// Table staging.  The levels are a fixed log-p grid, so the pressure cell of
// level l is the same for every model.  Levels are grouped into SEGMENTS of constant pressure
// cell; a segment needs two PLANES of the table, plane(ip) = sigma[all s][all iT][ip][tile]
// (S*nT rows of 256 B).  The producer thread streams the planes through a ring of NB shared
// memory slots with TMA (cp.async.bulk.tensor.4d, one box per species, mbarrier completion);
// consumers release a slot through an "empty" mbarrier when they leave the last segment that
// needs it.  Every table row is therefore read from L2 once per CTA and reused by all NW
// models and all levels of the segment; rows of the CIA tables are staged once.
//
// Cell walk.  VMRs are constant with height, so with G_c = sum_s x_s sigma_s at
// the four corners c of the model's current (T, p) cell, chi_l = n_l sum_c b_c G_c (b = bilinear
// weights): the species sum is redone only for the corners that change when the model enters
// another cell (every ~5 levels), not at every level.  Algebraically identical to interpolating
// each species and then summing; only the fp32 summation order differs.
//
// RT (Eq. 4-9) in the scaled deviation form H_k = (I_k - S_l) / mu_k:
//   large dtau/mu_k:  H <- e H + (1 - e) q,            e = 2^(-dtau log2e / mu_k), q = dS / dtau
//   small dtau/mu_k:  H <- H + P_k(dtau) (dS - dtau H), P_k(dtau) = phi(dtau/mu_k) / mu_k
// (common.cuh, R10); Planck and optical depth as in rt_direct.cuh.
// The thin/thick branch is taken per wavenumber, but a warp whose lanes all agree (for all angles, or for the
// small-mu / large-mu half of them) evaluates only that branch (LayerLimits).
#pragma once
#include <cuda.h>

#include <utility>

#include "common.cuh"
#include "obs.cuh"

namespace helios {

constexpr int kSlabTile = 64;       // wavenumbers per CTA (one 256 B row segment per table row)
constexpr int kSlabMaxRing = 8;
constexpr uint32_t kMbarSuspendNs = 20000;   // try_wait suspend-time hint: sleep in hardware instead of polling

// One segment of the plane schedule with everything that depends on the ring depth NB worked out on the host
// (slot = load index mod NB, parity = (load index / NB) & 1): the kernel does no integer division.
struct __align__(16) SlabSeg {
    int l_begin, l_end;             // levels [l_begin, l_end)
    int hi, lo;                     // slot | parity << 8 of the loads holding plane ip+1 / plane ip
    int shifted;                    // 1: this segment's upper plane is the previous segment's lower plane
    int rel_slot, rel_count;        // slots to release when the segment is done: rel_slot, rel_slot + 1, ... (mod NB)
    int pad;
};

struct SlabArgs {
    int S, C, nT, nNu, L, B;
    const float* rec;               // DEVICE [B][L][kSlabRecFloats]
    const float* model_x;           // DEVICE [B][x_floats]
    int x_floats;
    const float* model_scale;
    const int* model_flag;
    double nu0, dnu;
    const int* nu_index;            // DEVICE [stride]  wavenumber grid index of every table column (helios_load_opacity)
    float* flux;                    // DEVICE [B][flux_stride]  (not written when fused.acc != nullptr)
    long long flux_stride;
    FusedObs fused;                 // observation operator applied in the epilogue (obs.cuh)
    // plane schedule (helios_set_atmosphere), resolved for this launch's ring depth
    const SlabSeg* seg;             // DEVICE [n_seg]
    const int* load_ip;             // DEVICE [n_loads] pressure node of each load, in issue order
    int n_seg, n_loads;
    int ring;                       // NB, number of plane slots
    AngleSet ang;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1, %2;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t"
        "}" ::"r"(smem_u32(bar)), "r"(parity), "r"(kMbarSuspendNs) : "memory");
}
// The producer's wait for a free slot: it has a whole segment of compute (microseconds) to refill it, so it sleeps
// between polls instead of competing with the compute warps of its scheduler for issue slots.
__device__ __forceinline__ void mbar_wait_backoff(uint64_t* bar, uint32_t parity) {
    for (;;) {
        uint32_t done;
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}" : "=r"(done) : "r"(smem_u32(bar)), "r"(parity), "r"(kMbarSuspendNs) : "memory");
        if (done) return;
        __nanosleep(400);
    }
}
// TMA: one box of the 4-D table view {nu, ip, iT, s} / the 3-D CIA view {nu, iT, c} -> shared memory
// (dst: generic pointer to shared memory, or nullptr with the shared-memory byte address in dst_addr)
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2, int c3,
                                            uint32_t dst_addr = 0) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
        ::"r"(dst ? smem_u32(dst) : dst_addr), "l"((uint64_t)tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* tm, uint64_t* bar, int c0, int c1, int c2,
                                            uint32_t dst_addr = 0) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst ? smem_u32(dst) : dst_addr), "l"((uint64_t)tm), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2) : "memory");
}

__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ float4 lds_f4(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}

__device__ __forceinline__ float2 bc2(float v) { return make_float2(v, v); }
__device__ __forceinline__ float2 neg2(float2 v) { return make_float2(-v.x, -v.y); }
// A register copy the compiler may not rename away: keeps the corner values in FIXED registers
// across the level loop, so the (rare) cell changes pay for the moves and the steady state has none.
__device__ __forceinline__ void hard_copy(float2& dst, const float2& src) {
    asm volatile("mov.b32 %0, %2;\n\tmov.b32 %1, %3;" : "=f"(dst.x), "=f"(dst.y) : "f"(src.x), "f"(src.y));
}

__device__ __forceinline__ float2 lds_f2(uint32_t addr) {
    float2 v;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds_f1(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
// ga = sum_s x_s row_a[s], gb = sum_s x_s row_b[s].  qa, qb, x: shared-memory byte addresses;
// rows of consecutive species are `stride` bytes apart.
__device__ __forceinline__ void mix_pair(uint32_t qa, uint32_t qb, uint32_t x, int n, uint32_t stride,
                                         float2& ga, float2& gb) {
    ga = make_float2(0.0f, 0.0f); gb = ga;
#pragma unroll 4
    for (int s = 0; s < n; ++s) {
        const float2 xs = bc2(lds_f1(x));
        ga = __ffma2_rn(xs, lds_f2(qa), ga);
        gb = __ffma2_rn(xs, lds_f2(qb), gb);
        qa += stride; qb += stride; x += 4;
    }
}
__device__ __forceinline__ void mix_one(uint32_t qa, uint32_t x, int n, uint32_t stride, float2& ga) {
    ga = make_float2(0.0f, 0.0f);
#pragma unroll 2
    for (int s = 0; s < n; ++s) {
        ga = __ffma2_rn(bc2(lds_f1(x)), lds_f2(qa), ga);
        qa += stride; x += 4;
    }
}

// One angle of one layer for a pair of wavenumbers (state H = (I - S_l)/mu_k).  All per-angle
// constants are compile-time (Gauss-Legendre order A, node K) and become instruction immediates.
template <int A, int K>
__device__ __forceinline__ void angle_step(float2& H, float2 dtau, float2 ndtau, float2 q, float2 dS) {
    constexpr double mu = kGLmu[A - 1][K];
    constexpr float c_exp = (float)(kLog2e / mu), thr = (float)(0.25 * mu);
    constexpr float p0 = (float)(1.0 / mu), p1 = (float)(kPhiC1 / cpow(mu, 2)), p2 = (float)(kPhiC2 / cpow(mu, 3)),
                    p3 = (float)(kPhiC3 / cpow(mu, 4)), p4 = (float)(kPhiC4 / cpow(mu, 5));
    const float2 arg = __fmul2_rn(ndtau, bc2(c_exp));
    const float2 e = make_float2(ex2_approx(arg.x), ex2_approx(arg.y));
    const float2 big = __ffma2_rn(e, H, __ffma2_rn(neg2(e), q, q));
    float2 P = __ffma2_rn(dtau, bc2(p4), bc2(p3));
    P = __ffma2_rn(dtau, P, bc2(p2));
    P = __ffma2_rn(dtau, P, bc2(p1));
    P = __ffma2_rn(dtau, P, bc2(p0));
    const float2 small = __ffma2_rn(P, __ffma2_rn(ndtau, H, dS), H);
    H.x = dtau.x < thr ? small.x : big.x;
    H.y = dtau.y < thr ? small.y : big.y;
}
template <int A, int... K>
__device__ __forceinline__ void all_angles(float2 (&H)[A], float2 dtau, float2 ndtau, float2 q, float2 dS,
                                           std::integer_sequence<int, K...>) {
    (angle_step<A, K>(H[K], dtau, ndtau, q, dS), ...);
}
// The same update when the branch is known for the whole warp (bitwise the value angle_step selects).
template <int A, int K>
__device__ __forceinline__ void angle_step_thick(float2& H, float2 ndtau, float2 q) {
    constexpr float c_exp = (float)(kLog2e / kGLmu[A - 1][K]);
    const float2 arg = __fmul2_rn(ndtau, bc2(c_exp));
    const float2 e = make_float2(ex2_approx(arg.x), ex2_approx(arg.y));
    H = __ffma2_rn(e, H, __ffma2_rn(neg2(e), q, q));
}
template <int A, int K>
__device__ __forceinline__ void angle_step_thin(float2& H, float2 dtau, float2 ndtau, float2 dS) {
    constexpr double mu = kGLmu[A - 1][K];
    constexpr float p0 = (float)(1.0 / mu), p1 = (float)(kPhiC1 / cpow(mu, 2)), p2 = (float)(kPhiC2 / cpow(mu, 3)),
                    p3 = (float)(kPhiC3 / cpow(mu, 4)), p4 = (float)(kPhiC4 / cpow(mu, 5));
    float2 P = __ffma2_rn(dtau, bc2(p4), bc2(p3));
    P = __ffma2_rn(dtau, P, bc2(p2));
    P = __ffma2_rn(dtau, P, bc2(p1));
    P = __ffma2_rn(dtau, P, bc2(p0));
    H = __ffma2_rn(P, __ffma2_rn(ndtau, H, dS), H);
}
template <int A, int... K>
__device__ __forceinline__ void all_angles_thick(float2 (&H)[A], float2 ndtau, float2 q, std::integer_sequence<int, K...>) {
    (angle_step_thick<A, K>(H[K], ndtau, q), ...);
}
template <int A, int... K>
__device__ __forceinline__ void all_angles_thin(float2 (&H)[A], float2 dtau, float2 ndtau, float2 dS,
                                                std::integer_sequence<int, K...>) {
    (angle_step_thin<A, K>(H[K], dtau, ndtau, dS), ...);
}
// General (per-lane) step in the "w form": H <- H + w (q - H), w = 1 - e^{-D} from ex2 (thick lanes) or from the
// polynomial, w = dtau P_k(dtau) (thin lanes); dtau is clamped to >= 1e-20 by the caller so that q = dS / dtau is finite
// (below that the layer is transparent to every digit either way).
template <int A, int K>
__device__ __forceinline__ void angle_step_w(float2& H, float2 dtau, float2 ndtau, float2 q) {
    constexpr double mu = kGLmu[A - 1][K];
    constexpr float c_exp = (float)(kLog2e / mu), thr = (float)(0.25 * mu);
    constexpr float p0 = (float)(1.0 / mu), p1 = (float)(kPhiC1 / cpow(mu, 2)), p2 = (float)(kPhiC2 / cpow(mu, 3)),
                    p3 = (float)(kPhiC3 / cpow(mu, 4)), p4 = (float)(kPhiC4 / cpow(mu, 5));
    const float2 arg = __fmul2_rn(ndtau, bc2(c_exp));
    const float2 wk = __fadd2_rn(bc2(1.0f), neg2(make_float2(ex2_approx(arg.x), ex2_approx(arg.y))));
    float2 P = __ffma2_rn(dtau, bc2(p4), bc2(p3));
    P = __ffma2_rn(dtau, P, bc2(p2));
    P = __ffma2_rn(dtau, P, bc2(p1));
    P = __ffma2_rn(dtau, P, bc2(p0));
    const float2 wn = __fmul2_rn(dtau, P);
    const float2 w = make_float2(dtau.x < thr ? wn.x : wk.x, dtau.y < thr ? wn.y : wk.y);
    H = __ffma2_rn(w, __fadd2_rn(q, neg2(H)), H);
}
// angles K0 .. K1-1 with one kind of step: 0 general, 1 thick only, 2 thin only, 3 general in the w form, 4 saturated
template <int A, int K0, int K1, int MODE>
__device__ __forceinline__ void angle_range(float2 (&H)[A], float2 dtau, float2 ndtau, float2 q, float2 dS) {
    if constexpr (K0 < K1) {
        if constexpr (MODE == 0) angle_step<A, K0>(H[K0], dtau, ndtau, q, dS);
        if constexpr (MODE == 1) angle_step_thick<A, K0>(H[K0], ndtau, q);
        if constexpr (MODE == 2) angle_step_thin<A, K0>(H[K0], dtau, ndtau, dS);
        if constexpr (MODE == 3) angle_step_w<A, K0>(H[K0], dtau, ndtau, q);
        if constexpr (MODE == 4) H[K0] = __ffma2_rn(make_float2(0.0f, 0.0f), H[K0], q);    // = q, updated in place like the other forms
        angle_range<A, K0 + 1, K1, MODE>(H, dtau, ndtau, q, dS);
    }
}
template <int A, int K>
__device__ __forceinline__ void flux_term(float2& acc, float2 H) {
    constexpr float wH = (float)(kGLw[A - 1][K] * kGLmu[A - 1][K] * kGLmu[A - 1][K]);
    acc = __ffma2_rn(bc2(wH), H, acc);
}
template <int A, int... K>
__device__ __forceinline__ float2 flux_sum(const float2 (&H)[A], float2 S_top, std::integer_sequence<int, K...>) {
    float2 acc = __fmul2_rn(S_top, bc2(0.5f));    // sum_k w_k mu_k = 1/2: the rule integrates mu exactly
    (flux_term<A, K>(acc, H[K]), ...);
    return acc;
}

// Warp-uniform shortcuts of a layer:
//   all-thin   every lane has dtau < 0.25 mu_0        -> only the polynomial branch, for every angle
//   all-thick  every lane has dtau >= 0.25 mu_{A-1}   -> only the ex2 branch, for every angle
// dtau >= 0, so the order of the floats is the order of their bit patterns (REDUX works on integers).
//   saturated  every lane has e^{-dtau/mu_k} < 2^-30 for the n smallest mu_k  -> H_k = e H_k + (1 - e) q = q for those
//              (deep layers: 44 % of the all-thick (warp, layer) pairs at configs[3] are saturated in all 8 angles)
template <int A>
struct LayerLimits {
    static constexpr unsigned all_thick = __builtin_bit_cast(unsigned, (float)(0.25 * kGLmu[A - 1][A - 1]));
    static constexpr unsigned all_thin = __builtin_bit_cast(unsigned, (float)(0.25 * kGLmu[A - 1][0]));
    // dtau above which the n smallest-mu angles are saturated (30 ln 2 = 20.794); n = A, 4, 2, 1
    static constexpr unsigned sat_all = __builtin_bit_cast(unsigned, (float)(20.7944154168 * kGLmu[A - 1][A - 1]));
    static constexpr unsigned sat4 = __builtin_bit_cast(unsigned, (float)(20.7944154168 * kGLmu[A - 1][A >= 4 ? 3 : 0]));
    static constexpr unsigned sat2 = __builtin_bit_cast(unsigned, (float)(20.7944154168 * kGLmu[A - 1][A >= 2 ? 1 : 0]));
    static constexpr unsigned sat1 = __builtin_bit_cast(unsigned, (float)(20.7944154168 * kGLmu[A - 1][0]));
};

// Level records are staged per warp: blocks of kRecBlk levels, double-buffered, copied with cp.async one block ahead
// (a record is read once per wavenumber tile, and every new 32-byte sector of it was an L2 round trip at the top of
// the level iteration: 16 % of all warp stall samples at configs[3]).
#ifndef HELIOS_SLAB_RECBLK
#define HELIOS_SLAB_RECBLK 8
#endif
constexpr int kRecBlk = HELIOS_SLAB_RECBLK;          // power of two; 0 = records straight from global memory
constexpr int kRecRingFloats = 2 * kRecBlk * kSlabRecFloats;
constexpr int kRecBlkDiv = kRecBlk > 0 ? kRecBlk : 1;

// shared memory: [ring][S*nT*64] planes | [C*nT*64] CIA | [NW][x_floats] | [NW][2][kRecBlk] records | mbarriers
__host__ __device__ inline size_t slab_plane_floats(int S, int nT) { return (size_t)S * nT * kSlabTile; }
__host__ __device__ inline size_t slab_fixed_bytes(int C, int nT, int NW, int x_floats) {
    return sizeof(float) * ((size_t)C * nT * kSlabTile + (size_t)NW * x_floats + (size_t)NW * kRecRingFloats) +
           8 * (2 * kSlabMaxRing + 1) + 128;
}

template <int A, int NW, int MINB>
__global__ void __launch_bounds__((NW + 1) * 32, MINB)
k_rt_slab(const __grid_constant__ CUtensorMap tm_sigma, const __grid_constant__ CUtensorMap tm_cia, SlabArgs a) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const size_t plane_floats = slab_plane_floats(a.S, a.nT);
    float* planes = reinterpret_cast<float*>(smem_raw);
    float* cia_s = planes + (size_t)a.ring * plane_floats;
    float* xs_s = cia_s + (size_t)a.C * a.nT * kSlabTile;
    float* rec_s = xs_s + NW * a.x_floats;
    uint64_t* full = reinterpret_cast<uint64_t*>(rec_s + NW * kRecRingFloats);
    uint64_t* empty = full + kSlabMaxRing;
    uint64_t* cia_bar = empty + kSlabMaxRing;

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.y, group = blockIdx.x;
    const int NB = a.ring;

    if (threadIdx.x == 0) {
        for (int i = 0; i < NB; ++i) { mbar_init(&full[i], 1); mbar_init(&empty[i], NW); }
        mbar_init(cia_bar, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        // ===== producer: stream the planes this tile needs, in schedule order =====
        if (lane == 0) {
            const int nu_first = tile * kSlabTile;
            if (a.C > 0) {
                mbar_expect_tx(cia_bar, (uint32_t)(sizeof(float) * a.C * a.nT * kSlabTile));
                for (int c = 0; c < a.C; ++c)
                    tma_load_3d(cia_s + (size_t)c * a.nT * kSlabTile, &tm_cia, cia_bar, nu_first, 0, c);
            }
            if (a.S > 0) {
                int slot = 0, use = 0;
                for (int e = 0; e < a.n_loads; ++e, ++slot) {
                    if (slot == NB) { slot = 0; ++use; }
                    if (use > 0) mbar_wait_backoff(&empty[slot], (uint32_t)((use - 1) & 1));
                    const int ip = a.load_ip[e];
                    float* dst = planes + (size_t)slot * plane_floats;
                    mbar_expect_tx(&full[slot], (uint32_t)(sizeof(float) * plane_floats));
                    for (int s = 0; s < a.S; ++s)
                        tma_load_4d(dst + (size_t)s * a.nT * kSlabTile, &tm_sigma, &full[slot], nu_first, ip, 0, s);
                }
            }
        }
        return;
    }

    // ===== consumers: warp = model, lane = two adjacent wavenumbers =====
    int b = group * NW + warp;
    const bool model_valid = b < a.B;
    if (!model_valid) b = a.B - 1;           // still takes part in the slot hand-shake
    float* xw = xs_s + warp * a.x_floats;
    pdl_wait();                    // records, x and flags come from the prep kernel (the producer streams static tables: no wait)
    for (int i = lane; i < a.x_floats; i += 32) xw[i] = a.model_x[(size_t)b * a.x_floats + i];
    __syncwarp();

    // the lane's two table columns and the wavenumber grid points they hold (the table's nu axis is re-ordered)
    const int inu = tile * kSlabTile + 2 * lane;
    const int2 gnu = __ldg(reinterpret_cast<const int2*>(a.nu_index + inu));
    const double nu_d0 = a.nu0 + a.dnu * (double)gnu.x, nu_d1 = a.nu0 + a.dnu * (double)gnu.y;
    const float2 nu = make_float2((float)nu_d0, (float)nu_d1);
    const float2 nu_lo = make_float2((float)(nu_d0 - (double)nu.x), (float)(nu_d1 - (double)nu.y));
    const float2 c1nu3 = make_float2((float)(kC1 * nu_d0 * nu_d0 * nu_d0), (float)(kC1 * nu_d1 * nu_d1 * nu_d1));
    constexpr uint32_t kRowB = kSlabTile * sizeof(float);   // bytes per table row in a plane
    const uint32_t spB = a.nT * kRowB;        // bytes between species in a plane
    const float* rec_b = a.rec + (size_t)b * a.L * kSlabRecFloats;
    const float4* rp = reinterpret_cast<const float4*>(rec_b);
    const uint32_t rb_a = smem_u32(rec_s + warp * kRecRingFloats);
    const int n_rec16 = a.L * (kSlabRecFloats / 4);                    // 16-byte pieces of this model's records
    auto stage_block = [&](int blk) {                                 // levels blk kRecBlk .. + kRecBlk - 1 -> half blk & 1
        const int piece = blk * kRecBlk * (kSlabRecFloats / 4) + lane;
        if (lane < kRecBlk * (kSlabRecFloats / 4) && piece < n_rec16)
            cp_async_16(rb_a + (uint32_t)(((blk & 1) * kRecBlk * (kSlabRecFloats / 4) + lane) * 16), rp + piece);
        cp_async_commit();
    };
    if (kRecBlk > 0) stage_block(0);
    const uint32_t planes_a = smem_u32(planes) + lane * 8;   // shared-memory byte addresses of this lane's pair
    const uint32_t cia_a = smem_u32(cia_s) + lane * 8;
    const uint32_t xw_a = smem_u32(xw), xc_a = xw_a + a.S * 4;
    const uint32_t plane_bytes = (uint32_t)(plane_floats * sizeof(float));

    float2 H[A];
#pragma unroll
    for (int k = 0; k < A; ++k) H[k] = make_float2(0.0f, 0.0f);
    float2 chi_prev = make_float2(0.0f, 0.0f), S_prev = chi_prev;
    float2 G00 = chi_prev, G01 = chi_prev, G10 = chi_prev, G11 = chi_prev, Gc0 = chi_prev, Gc1 = chi_prev;
    int cur_iT = -2;

    if (a.C > 0) mbar_wait(cia_bar, 0);

    for (int seg = 0; seg < a.n_seg; ++seg) {
        const int4 sg0 = __ldg(reinterpret_cast<const int4*>(a.seg + seg)), sg1 = __ldg(reinterpret_cast<const int4*>(a.seg + seg) + 1);
        const int l_begin = sg0.x, l_end = sg0.y;
        uint32_t pLo = planes_a, pHi = planes_a;
        const bool shifted = sg1.x != 0;      // the previous segment's lower plane is this one's upper plane
        if (a.S > 0) {
            mbar_wait(&full[sg0.z & 0xff], (uint32_t)(sg0.z >> 8));
            mbar_wait(&full[sg0.w & 0xff], (uint32_t)(sg0.w >> 8));
            pHi += (uint32_t)(sg0.z & 0xff) * plane_bytes;
            pLo += (uint32_t)(sg0.w & 0xff) * plane_bytes;
        }
        bool fresh = true;
        for (int l = l_begin; l < l_end; ++l) {
            float4 r0, r1, r2;
            if (kRecBlk > 0) {
                if ((l & (kRecBlkDiv - 1)) == 0) {          // this block has landed (issued a block ago); fetch the next one
                    cp_async_wait_all();
                    __syncwarp();
                    stage_block(l / kRecBlkDiv + 1);
                }
                const uint32_t ra = rb_a + (uint32_t)(l & (2 * kRecBlkDiv - 1)) * (kSlabRecFloats * 4);
                r0 = lds_f4(ra); r1 = lds_f4(ra + 16); r2 = lds_f4(ra + 32);
            } else {
                r0 = __ldcg(rp + 3 * l); r1 = __ldcg(rp + 3 * l + 1); r2 = __ldcg(rp + 3 * l + 2);     // k_prep's output: not .nc under PDL
            }
            const int iT = __float_as_int(r2.y);
            if (fresh || iT != cur_iT) {      // warp-uniform: the model is in another table cell
                const uint32_t lo = pLo + iT * kRowB, hi = pHi + iT * kRowB, qc = cia_a + iT * kRowB;
                if (!fresh && iT == cur_iT - 1) {            // one cell colder: (iT+1) corners are the old iT corners
                    hard_copy(G10, G00); hard_copy(G11, G01); hard_copy(Gc1, Gc0);
                    mix_pair(lo, hi, xw_a, a.S, spB, G00, G01);
                    mix_one(qc, xc_a, a.C, spB, Gc0);
                } else if (!fresh && iT == cur_iT + 1) {     // one cell hotter
                    hard_copy(G00, G10); hard_copy(G01, G11); hard_copy(Gc0, Gc1);
                    mix_pair(lo + kRowB, hi + kRowB, xw_a, a.S, spB, G10, G11);
                    mix_one(qc + kRowB, xc_a, a.C, spB, Gc1);
                } else if (fresh && shifted && iT == cur_iT) {   // next pressure cell, same temperature cell
                    hard_copy(G01, G00); hard_copy(G11, G10);
                    mix_pair(lo, lo + kRowB, xw_a, a.S, spB, G00, G10);
                } else {
                    mix_pair(lo, lo + kRowB, xw_a, a.S, spB, G00, G10);
                    mix_pair(hi, hi + kRowB, xw_a, a.S, spB, G01, G11);
                    mix_pair(qc, qc + kRowB, xc_a, a.C, spB, Gc0, Gc1);
                }
                cur_iT = iT;
                fresh = false;
            }
            float2 chi = __fmul2_rn(bc2(r0.x), G00);
            chi = __ffma2_rn(bc2(r0.y), G01, chi);
            chi = __ffma2_rn(bc2(r0.z), G10, chi);
            chi = __ffma2_rn(bc2(r0.w), G11, chi);
            chi = __ffma2_rn(bc2(r1.x), Gc0, chi);
            chi = __ffma2_rn(bc2(r1.y), Gc1, chi);
            const float2 ah = bc2(r1.z);
            const float2 pr = __fmul2_rn(ah, nu);
            float2 rr = __ffma2_rn(ah, nu, neg2(pr));
            rr = __ffma2_rn(bc2(r1.w), nu, rr);
            rr = __ffma2_rn(ah, nu_lo, rr);
            const float2 E0 = make_float2(ex2_approx(-pr.x), ex2_approx(-pr.y));
            const float2 E = __ffma2_rn(__fmul2_rn(E0, bc2(-0.69314718056f)), rr, E0);
            const float2 om = __fadd2_rn(bc2(1.0f), neg2(E));
            const float2 Sl = __fmul2_rn(c1nu3, __fmul2_rn(E, make_float2(rcp_approx(om.x), rcp_approx(om.y))));
            if (l > 0) {
                // dtau of the layer below this level: trapezoid of chi times the hydrostatic thickness, plus the grey cloud
                const float2 dtau = __ffma2_rn(__fadd2_rn(chi, chi_prev), bc2(r2.x), bc2(r2.z));
                const float2 dS = __fadd2_rn(S_prev, neg2(Sl));
                const float2 ndtau = neg2(dtau);
                const unsigned d_lo = __reduce_min_sync(0xffffffffu, __float_as_uint(fminf(dtau.x, dtau.y)));
                const unsigned d_hi = __reduce_max_sync(0xffffffffu, __float_as_uint(fmaxf(dtau.x, dtau.y)));
                if (d_hi < LayerLimits<A>::all_thin) {
                    all_angles_thin<A>(H, dtau, ndtau, dS, std::make_integer_sequence<int, A>{});
                } else {
                    const float2 q = __fmul2_rn(dS, make_float2(rcp_approx(dtau.x), rcp_approx(dtau.y)));
                    if (d_lo >= LayerLimits<A>::all_thick) {
                        constexpr int N4 = A >= 8 ? 4 : 0, N1 = A >= 4 ? 1 : 0;
                        if (d_lo >= LayerLimits<A>::sat_all) {
                            angle_range<A, 0, A, 4>(H, dtau, ndtau, q, dS);
                        } else if (N4 > 0 && d_lo >= LayerLimits<A>::sat4) {
                            angle_range<A, 0, N4, 4>(H, dtau, ndtau, q, dS);
                            angle_range<A, N4, A, 1>(H, dtau, ndtau, q, dS);
                        } else if (N1 > 0 && d_lo >= LayerLimits<A>::sat1) {
                            angle_range<A, 0, N1, 4>(H, dtau, ndtau, q, dS);
                            angle_range<A, N1, A, 1>(H, dtau, ndtau, q, dS);
                        } else {
                            all_angles_thick<A>(H, ndtau, q, std::make_integer_sequence<int, A>{});
                        }
                    } else {
                        constexpr int GM = 3;
                        const float2 dtc = make_float2(fmaxf(dtau.x, 1e-20f), fmaxf(dtau.y, 1e-20f));
                        const float2 ndtc = neg2(dtc);
                        const float2 qc = __fmul2_rn(dS, make_float2(rcp_approx(dtc.x), rcp_approx(dtc.y)));
                        // many angles: the small-mu half is often thick for every lane while the large-mu half is
                        // still mixed, or the large-mu half thin while the small-mu half is mixed (measured: pays for A >= 6)
                        constexpr int AH = A >= 6 ? A / 2 : 0;
                        constexpr unsigned kLowThick = __builtin_bit_cast(unsigned, (float)(0.25 * kGLmu[A - 1][AH > 0 ? AH - 1 : 0]));
                        constexpr unsigned kHighThin = __builtin_bit_cast(unsigned, (float)(0.25 * kGLmu[A - 1][AH]));
                        if (AH > 0 && d_lo >= kLowThick) {
                            angle_range<A, 0, AH, 1>(H, dtau, ndtau, q, dS);
                            angle_range<A, AH, A, GM>(H, dtc, ndtc, qc, dS);
                        } else if (AH > 0 && d_hi < kHighThin) {
                            angle_range<A, 0, AH, GM>(H, dtc, ndtc, qc, dS);
                            angle_range<A, AH, A, 2>(H, dtau, ndtau, q, dS);
                        } else {
                            angle_range<A, 0, A, GM>(H, dtc, ndtc, qc, dS);
                        }
                    }
                }
            }
            chi_prev = chi; S_prev = Sl;
        }
        if (a.S > 0 && sg1.z > 0) {
            // slots holding loads older than the next segment's are free for the producer
            __syncwarp();
            if (lane == 0) {
                int slot = sg1.y;
                for (int i = 0; i < sg1.z; ++i) { mbar_arrive(&empty[slot]); slot = slot + 1 == NB ? 0 : slot + 1; }
            }
        }
    }

    pdl_launch_dependents();
    if (!model_valid) return;
    const bool one = gnu.x < a.nNu, two = gnu.y < a.nNu;
    const bool rejected = a.model_flag[b] != 0;
    // F+ = 2 pi sum_k w_k mu_k I_k (Eq. 8), I_k = mu_k H_k + S_top;  F = f (R/d)^2 F+ (Eq. 9)
    const float2 acc = flux_sum<A>(H, S_prev, std::make_integer_sequence<int, A>{});
    const float scale = a.model_scale[b];
    if (a.fused.acc) {               // convolve + bin here: integer atomics into M[b][j] (obs.cuh); no flux is written
        if (rejected) return;
        if (one) fused_accumulate(a.fused, b, gnu.x, scale * acc.x);
        if (two) fused_accumulate(a.fused, b, gnu.y, scale * acc.y);
        return;
    }
    float* out = a.flux + (size_t)b * a.flux_stride;       // written in grid order: columns of the padding map to >= nNu
    if (one) out[gnu.x] = rejected ? __int_as_float(0x7fc00000) : scale * acc.x;
    if (two) out[gnu.y] = rejected ? __int_as_float(0x7fc00000) : scale * acc.y;
}

// ---------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------
struct SlabPlan {
    bool ok = false;
    int NW = 0, ring = 0;
    size_t smem = 0, smem_optin = 0;
};

// Picks the models-per-CTA variant and the ring depth that fit the shared memory of one SM.
inline SlabPlan slab_plan(int S, int C, int nT, int A, int n_loads, int want_nw, size_t smem_optin, size_t smem_sm) {
    SlabPlan p;
    if (A < 1 || A > kMaxAngles || nT > 256) return p;
    const int nw = want_nw > 0 ? want_nw : 16;
    if (nw != 8 && nw != 16 && nw != 20 && nw != 24 && nw != 27) return p;
    const int target_ctas = nw == 8 ? 3 : 1;
    const size_t plane = sizeof(float) * slab_plane_floats(S, nT);
    const size_t fixed = slab_fixed_bytes(C, nT, nw, slab_x_floats(S, C));
    for (int ctas = target_ctas; ctas >= 1; --ctas) {
        size_t budget = smem_sm / ctas;
        budget = budget > 1024 ? budget - 1024 : 0;     // per-CTA reservation of the runtime
        if (budget > smem_optin) budget = smem_optin;
        if (budget < fixed) continue;
        int ring = plane ? (int)((budget - fixed) / plane) : 1;
        if (ring > kSlabMaxRing) ring = kSlabMaxRing;
        if (n_loads > 0 && ring > n_loads) ring = n_loads;
        const int need = n_loads >= 3 ? 3 : (n_loads > 0 ? n_loads : 1);
        if (plane && ring < need) continue;
        if (ring < 1) ring = 1;
        p.ok = true; p.NW = nw; p.ring = ring; p.smem = fixed + plane * ring; p.smem_optin = smem_optin;
        return p;
    }
    return p;
}

// `configured` = this CONTEXT has raised the kernel instance's dynamic shared-memory limit (a context lives on one
// device and is used by one host thread at a time, so the flag needs no lock).  The limit is a property of the
// function, shared by every context of the process: it is always set to the device's opt-in maximum, never to the
// size one context happens to need, so contexts with different table shapes cannot lower it for each other.
template <int A, int NW, int MINB>
inline cudaError_t launch_rt_slab_t(const CUtensorMap& tms, const CUtensorMap& tmc, const SlabArgs& a, const SlabPlan& p,
                                    bool& configured, cudaStream_t stream, bool pdl) {
    const size_t smem = p.smem;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_rt_slab<A, NW, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_optin);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const dim3 grid((a.B + NW - 1) / NW, (a.nNu + kSlabTile - 1) / kSlabTile);
    return launch_kernel(k_rt_slab<A, NW, MINB>, grid, dim3((NW + 1) * 32), smem, stream, pdl, tms, tmc, a);
}

struct SlabSmemCache { bool configured[kMaxAngles + 1][5] = {}; };     // [A][models-per-CTA variant], one per context

template <int A>
inline cudaError_t launch_rt_slab_a(const CUtensorMap& tms, const CUtensorMap& tmc, const SlabArgs& a, const SlabPlan& p,
                                    SlabSmemCache& cache, cudaStream_t stream, bool pdl) {
    switch (p.NW) {
        case 8:  return launch_rt_slab_t<A, 8, 3>(tms, tmc, a, p, cache.configured[A][0], stream, pdl);
        case 16: return launch_rt_slab_t<A, 16, 1>(tms, tmc, a, p, cache.configured[A][1], stream, pdl);
        case 20: return launch_rt_slab_t<A, 20, 1>(tms, tmc, a, p, cache.configured[A][2], stream, pdl);
        case 24: return launch_rt_slab_t<A, 24, 1>(tms, tmc, a, p, cache.configured[A][3], stream, pdl);
        case 27: return launch_rt_slab_t<A, 27, 1>(tms, tmc, a, p, cache.configured[A][4], stream, pdl);
        default: return cudaErrorInvalidValue;
    }
}

inline cudaError_t launch_rt_slab(const CUtensorMap& tms, const CUtensorMap& tmc, const SlabArgs& a, const SlabPlan& p,
                                  SlabSmemCache& cache, cudaStream_t stream, bool pdl) {
    switch (a.ang.n) {
        case 1: return launch_rt_slab_a<1>(tms, tmc, a, p, cache, stream, pdl);
        case 2: return launch_rt_slab_a<2>(tms, tmc, a, p, cache, stream, pdl);
        case 3: return launch_rt_slab_a<3>(tms, tmc, a, p, cache, stream, pdl);
        case 4: return launch_rt_slab_a<4>(tms, tmc, a, p, cache, stream, pdl);
        case 5: return launch_rt_slab_a<5>(tms, tmc, a, p, cache, stream, pdl);
        case 6: return launch_rt_slab_a<6>(tms, tmc, a, p, cache, stream, pdl);
        case 7: return launch_rt_slab_a<7>(tms, tmc, a, p, cache, stream, pdl);
        case 8: return launch_rt_slab_a<8>(tms, tmc, a, p, cache, stream, pdl);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace helios
