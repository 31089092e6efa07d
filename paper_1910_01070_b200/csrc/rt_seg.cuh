// rt_seg.cuh -- fused steps 1-4, LEVEL-PARALLEL variant for small batches
// (the paper's own usage is one model per likelihood call).
//
// With a handful of models there are only B * N_nu / 64 warps of work if every warp walks all L
// levels (fewer than two per SM for one model), and each level costs a chain of dependent
// latencies: the staged kernel needs 0.11 ms for ONE model.  But the layer update of Eq. 4,
//     I <- e^{-D} I + (beta S_l + gamma S_{l-1}),
// is an affine map of the incoming intensity, and affine maps compose associatively.  So the
// level loop is cut into chunks: one CTA = one model x one 64-wavenumber tile, warp c = chunk c
// of the layers.  Every warp integrates its chunk for an UNKNOWN incoming state, i.e. it carries,
// per angle, the pair (Psi, C) of  H_out = Psi H_in + C  (H = (I - S)/mu as in rt_slab.cuh; Psi is
// the chunk's transmission, C its own emission), and one warp then chains the 8 pairs bottom-up
// and forms the flux of Eq. 8-9.  All terms are the ones of the sequential recursion; only the
// order of the floating-point operations differs.
//
// Table access: with so few models a table row is used by one warp only, so nothing is shared
// between warps.  Every warp walks the table cells of its own levels (the cell walk of rt_slab.cuh)
// and fetches the rows of a cell's NEW corners (2 S + C rows of 256 B) into a private shared-memory
// buffer one cell change AHEAD with one or two TMA boxes (cp.async.bulk.tensor, all species at once) that
// complete on the warp's mbarrier, so a fetch costs a dozen instructions and its HBM latency is hidden behind
// the levels of the current cell.  Which level enters which cell, and how the new cell relates to the old
// one, is worked out once per model by the prep kernel (record slot 11).  Only the rows the models touch
// are read at all.
#pragma once
#include "common.cuh"
#include "rt_slab.cuh"

namespace helios {

#ifndef HELIOS_SEG_CHUNKS
#define HELIOS_SEG_CHUNKS 8
#endif
constexpr int kSegMaxChunks = HELIOS_SEG_CHUNKS;       // warps per CTA
constexpr int kSegMaxLen = 32;          // layers per chunk (L <= 8 * 32 + 1; longer atmospheres use the staged kernel)

struct SegArgs {
    const float* sigma;       // DEVICE [S][nT][nP][stride]
    const float* cia;         // DEVICE [C][nT][stride]
    long long stride;
    int S, C, nT, nP, nNu, L, B;
    const float* rec;         // DEVICE [B][L][kSlabRecFloats]   (staged-kernel records, common.cuh)
    const float* model_x;     // DEVICE [B][x_floats]
    int x_floats;
    const float* model_scale;
    const int* model_flag;
    const int* lvl_ip;        // DEVICE [L] pressure cell of each level
    const int* nu_index;      // DEVICE [stride]  wavenumber grid index of every table column (helios_load_opacity)
    double nu0, dnu;
    float* flux;              // DEVICE [B][flux_stride]  (not written when fused.acc != nullptr)
    long long flux_stride;
    FusedObs fused;           // observation operator applied in the epilogue (obs.cuh)
    int n_chunks, chunk_len;  // chunk c owns the layers 1 + c len .. min(L - 1, (c + 1) len)  (layer j: levels j-1, j)
};


// A warp's row buffer holds the 2 S + C rows one cell change brings in (a "half" of a cell's corners): for species s the two rows
// 2 s and 2 s + 1 (two pressure nodes of one temperature node, or two temperature nodes of one pressure node),
// then one CIA row per pair.  One TMA box brings in all 2 S species rows (tensor maps of helios_api.cu:
// box {64 nu, 2 p nodes, 1 T node, S} or {64, 1, 2, S}), another the C CIA rows; mix_half reduces a half.
__device__ __forceinline__ void mix_half(uint32_t src, const float* x, int S, int C, int lane, float2& ga, float2& gb, float2& gc) {
    ga = make_float2(0.0f, 0.0f); gb = ga; gc = ga;
    const uint32_t q = src + lane * 8;
#pragma unroll 4
    for (int s = 0; s < S; ++s) {
        const float2 xs = bc2(x[s]);
        ga = __ffma2_rn(xs, lds_f2(q + (2 * s) * kSlabTile * 4), ga);
        gb = __ffma2_rn(xs, lds_f2(q + (2 * s + 1) * kSlabTile * 4), gb);
    }
    for (int c = 0; c < C; ++c) gc = __ffma2_rn(bc2(x[S + c]), lds_f2(q + (2 * S + c) * kSlabTile * 4), gc);
}

// One angle of one layer for the pair (Psi, C): C takes the step of the sequential recursion (the thick, thin and
// general forms of rt_slab.cuh), Psi the homogeneous part of the same step.
// General (per-lane) step in the "w form" of rt_slab.cuh: w = 1 - e^{-D} from ex2 (thick lanes) or from the polynomial,
// w = dtau P_k(dtau) (thin lanes);  C <- C + w (q - C),  Psi <- Psi - w Psi.  dtau is clamped to >= 1e-20 by the caller.
template <int A, int K0>
__device__ __forceinline__ void seg_angles_w(float2 (&Cc)[A], float2 (&Psi)[A], float2 dtau, float2 ndtau, float2 q) {
    if constexpr (K0 < A) {
        constexpr double mu = kGLmu[A - 1][K0];
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
        Cc[K0] = __ffma2_rn(w, __fadd2_rn(q, neg2(Cc[K0])), Cc[K0]);
        Psi[K0] = __ffma2_rn(neg2(w), Psi[K0], Psi[K0]);
        seg_angles_w<A, K0 + 1>(Cc, Psi, dtau, ndtau, q);
    }
}

// The same step when every lane of the warp is on one branch for every angle (LayerLimits of rt_slab.cuh).
template <int A, int K0>
__device__ __forceinline__ void seg_angles_thick(float2 (&Cc)[A], float2 (&Psi)[A], float2 ndtau, float2 q) {
    if constexpr (K0 < A) {
        constexpr float c_exp = (float)(kLog2e / kGLmu[A - 1][K0]);
        const float2 arg = __fmul2_rn(ndtau, bc2(c_exp));
        const float2 e = make_float2(ex2_approx(arg.x), ex2_approx(arg.y));
        Cc[K0] = __ffma2_rn(e, Cc[K0], __ffma2_rn(neg2(e), q, q));
        Psi[K0] = __fmul2_rn(e, Psi[K0]);
        seg_angles_thick<A, K0 + 1>(Cc, Psi, ndtau, q);
    }
}
template <int A, int K0>
__device__ __forceinline__ void seg_angles_thin(float2 (&Cc)[A], float2 (&Psi)[A], float2 dtau, float2 ndtau, float2 dS) {
    if constexpr (K0 < A) {
        constexpr double mu = kGLmu[A - 1][K0];
        constexpr float p0 = (float)(1.0 / mu), p1 = (float)(kPhiC1 / cpow(mu, 2)), p2 = (float)(kPhiC2 / cpow(mu, 3)),
                        p3 = (float)(kPhiC3 / cpow(mu, 4)), p4 = (float)(kPhiC4 / cpow(mu, 5));
        float2 P = __ffma2_rn(dtau, bc2(p4), bc2(p3));
        P = __ffma2_rn(dtau, P, bc2(p2));
        P = __ffma2_rn(dtau, P, bc2(p1));
        P = __ffma2_rn(dtau, P, bc2(p0));
        Cc[K0] = __ffma2_rn(P, __ffma2_rn(ndtau, Cc[K0], dS), Cc[K0]);
        Psi[K0] = __ffma2_rn(__fmul2_rn(ndtau, P), Psi[K0], Psi[K0]);
        seg_angles_thin<A, K0 + 1>(Cc, Psi, dtau, ndtau, dS);
    }
}

// shared memory: [n_chunks][A][2][64] (Psi, C) | [64] S_top | [n_chunks][2 S + C][64] row buffers | [x_floats] x |
//                [n_chunks][chunk_len + 1] records + cells | [n_chunks] mbarriers
__host__ __device__ inline size_t seg_smem_bytes(int A, int n_chunks, int chunk_len, int x_floats, int S, int C) {
    return sizeof(float) * ((size_t)n_chunks * A * 2 * kSlabTile + kSlabTile + (size_t)n_chunks * (2 * S + C) * kSlabTile +
                            x_floats + (size_t)n_chunks * (chunk_len + 1) * (kSlabRecFloats + 4)) + 8 * (size_t)n_chunks + 8;
}

template <int A>
__global__ void __launch_bounds__(kSegMaxChunks * 32, kSegMaxChunks <= 8 ? 3 : 1)
k_rt_seg(const __grid_constant__ CUtensorMap tm_p2, const __grid_constant__ CUtensorMap tm_t2,
         const __grid_constant__ CUtensorMap tm_c, SegArgs a) {
    extern __shared__ __align__(128) float seg_smem[];
    float* ex = seg_smem;
    float* stop = ex + (size_t)a.n_chunks * A * 2 * kSlabTile;
    float* rows = stop + kSlabTile;
    const int half_rows = 2 * a.S + a.C;
    float* xs = rows + (size_t)a.n_chunks * half_rows * kSlabTile;
    float* recs = xs + a.x_floats;
    uint64_t* bars = reinterpret_cast<uint64_t*>(
        (reinterpret_cast<uintptr_t>(recs + (size_t)a.n_chunks * (a.chunk_len + 1) * (kSlabRecFloats + 4)) + 7) & ~(uintptr_t)7);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int b = blockIdx.x, tile = blockIdx.y;
    if (lane == 0) mbar_init(&bars[warp], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const int inu = tile * kSlabTile + 2 * lane;
    const int2 gnu = __ldg(reinterpret_cast<const int2*>(a.nu_index + inu));      // static: in flight before the wait
    pdl_wait();                    // records, x and flags come from the prep kernel
    for (int i = threadIdx.x; i < a.x_floats; i += blockDim.x) xs[i] = a.model_x[(size_t)b * a.x_floats + i];

    // layers j0 .. j1-1 of this chunk need the levels j0-1 .. j1-1
    const int j0 = 1 + warp * a.chunk_len, j1 = min(a.L, j0 + a.chunk_len);
    const int n_lev = j1 > j0 ? j1 - j0 + 1 : 0;
    float* rw = recs + (size_t)warp * (a.chunk_len + 1) * (kSlabRecFloats + 4);     // records, then the pressure cells
    int* ipw = reinterpret_cast<int*>(rw + (a.chunk_len + 1) * kSlabRecFloats);
    const uint32_t half0 = smem_u32(rows) + (uint32_t)warp * half_rows * kSlabTile * 4;
    const uint32_t cia_off = (uint32_t)(2 * a.S) * kSlabTile * 4;
    uint64_t* bar = &bars[warp];
    uint32_t phase = 0;
    const int nu_first = tile * kSlabTile;
    // asynchronous fetch of new corners of cell (iT1, ip1) into the warp's buffer:
    //   what = 1: temperature row iT1, pressure nodes ip1 and ip1 + 1, CIA row iT1      (one cell colder; first half of a new cell)
    //   what = 2: temperature row iT1 + 1, the same                                      (one cell hotter; second half of a new cell)
    //   what = 3: pressure node ip1, temperature rows iT1 and iT1 + 1, no CIA            (next pressure cell upwards)
    auto issue = [&](int what, int iT1, int ip1) {
        if (lane != 0) return;
        const uint32_t sig_bytes = (uint32_t)(2 * a.S) * kSlabTile * 4, cia_bytes = (uint32_t)a.C * kSlabTile * 4;
        const bool with_cia = a.C > 0 && what != 3;
        mbar_expect_tx(bar, sig_bytes + (with_cia ? cia_bytes : 0u));
        const int iTa = what == 2 ? iT1 + 1 : iT1;
        if (a.S > 0) tma_load_4d(nullptr, what == 3 ? &tm_t2 : &tm_p2, bar, nu_first, ip1, iTa, 0, half0);
        if (with_cia) tma_load_3d(nullptr, &tm_c, bar, nu_first, iTa, 0, half0 + cia_off);
    };
    // the chunk's first cell, straight from global memory, so that its fetch is in flight while the records are staged
    int first_iT = 0, first_ip = 0;
    if (lane == 0 && n_lev > 0) {
        first_iT = __float_as_int(__ldcg(a.rec + ((size_t)b * a.L + (j0 - 1)) * kSlabRecFloats + 9));   // written by k_prep while
                                               // this grid may already be resident (programmatic launch): not the read-only (.nc) path
        first_ip = __ldg(a.lvl_ip + j0 - 1);
        issue(1, first_iT, first_ip);          // a new cell = two fetches (what 1 here, what 2 in the level loop)
    }
    {
        const float4* src = reinterpret_cast<const float4*>(a.rec + ((size_t)b * a.L + (j0 - 1)) * kSlabRecFloats);
        for (int i = lane; i < n_lev * (kSlabRecFloats / 4); i += 32) reinterpret_cast<float4*>(rw)[i] = __ldcg(src + i);
        for (int i = lane; i < n_lev; i += 32) ipw[i] = __ldg(a.lvl_ip + j0 - 1 + i);
    }
    __syncthreads();

    const double nu_d0 = a.nu0 + a.dnu * (double)gnu.x, nu_d1 = a.nu0 + a.dnu * (double)gnu.y;
    const float2 nu = make_float2((float)nu_d0, (float)nu_d1);
    const float2 nu_lo = make_float2((float)(nu_d0 - (double)nu.x), (float)(nu_d1 - (double)nu.y));
    const float2 c1nu3 = make_float2((float)(kC1 * nu_d0 * nu_d0 * nu_d0), (float)(kC1 * nu_d1 * nu_d1 * nu_d1));

    float2 Cc[A], Psi[A];
#pragma unroll
    for (int k = 0; k < A; ++k) { Cc[k] = make_float2(0.0f, 0.0f); Psi[k] = make_float2(1.0f, 1.0f); }
    float2 chi_prev = make_float2(0.0f, 0.0f), S_prev = chi_prev;
    float2 G00 = chi_prev, G01 = chi_prev, G10 = chi_prev, G11 = chi_prev, Gc0 = chi_prev, Gc1 = chi_prev;
    auto sched = [&](int i) { return __float_as_int(rw[i * kSlabRecFloats + 11]); };
    auto cell_iT = [&](int i) { return __float_as_int(rw[i * kSlabRecFloats + 9]); };
    // the level after which the rows in flight are needed, and how they relate to the current cell
    int nxt = n_lev, nxt_kind = 0;
    if (n_lev > 0) nxt = 0;                   // the first level's cell is in flight already

    for (int i = 0; i < n_lev; ++i) {
        const float4 r0 = reinterpret_cast<const float4*>(rw)[3 * i], r1 = reinterpret_cast<const float4*>(rw)[3 * i + 1],
                     r2 = reinterpret_cast<const float4*>(rw)[3 * i + 2];
        if (i == nxt) {                       // warp-uniform: the level lies in another table cell; its rows have been fetched
            mbar_wait(bar, phase);
            phase ^= 1u;
            float2 unused;
            if (nxt_kind == 1) {              // one cell colder
                G10 = G00; G11 = G01; Gc1 = Gc0;
                mix_half(half0, xs, a.S, a.C, lane, G00, G01, Gc0);
            } else if (nxt_kind == 2) {       // one cell hotter
                G00 = G10; G01 = G11; Gc0 = Gc1;
                mix_half(half0, xs, a.S, a.C, lane, G10, G11, Gc1);
            } else if (nxt_kind == 3) {       // next pressure cell upwards, same temperature cell
                G01 = G00; G11 = G10;
                mix_half(half0, xs, a.S, 0, lane, G00, G10, unused);
            } else {                          // a new cell: all four corners, in two fetches through the one buffer
                mix_half(half0, xs, a.S, a.C, lane, G00, G01, Gc0);
                __syncwarp();
                issue(2, cell_iT(i), ipw[i]);
                mbar_wait(bar, phase);
                phase ^= 1u;
                mix_half(half0, xs, a.S, a.C, lane, G10, G11, Gc1);
            }
            __syncwarp();                     // every lane has read the buffer before the next fetch overwrites it
            const int dist = sched(i) >> 8;   // next level in another cell (prep.cuh), 0: none
            nxt = dist > 0 ? i + dist : n_lev;
            if (nxt < n_lev) { nxt_kind = sched(nxt) & 0xff; issue(nxt_kind == 0 ? 1 : nxt_kind, cell_iT(nxt), ipw[nxt]); }
        }
        float2 chi = __fmul2_rn(bc2(r0.x), G00);
        chi = __ffma2_rn(bc2(r0.y), G01, chi);
        chi = __ffma2_rn(bc2(r0.z), G10, chi);
        chi = __ffma2_rn(bc2(r0.w), G11, chi);
        chi = __ffma2_rn(bc2(r1.x), Gc0, chi);
        chi = __ffma2_rn(bc2(r1.y), Gc1, chi);
        // S_l = B_nu(T_l) = c1 nu^3 E / (1 - E), E = 2^(-a nu), a nu carried as a two-float product (as rt_slab.cuh)
        const float2 ah = bc2(r1.z);
        const float2 pr = __fmul2_rn(ah, nu);
        float2 rr = __ffma2_rn(ah, nu, neg2(pr));
        rr = __ffma2_rn(bc2(r1.w), nu, rr);
        rr = __ffma2_rn(ah, nu_lo, rr);
        const float2 E0 = make_float2(ex2_approx(-pr.x), ex2_approx(-pr.y));
        const float2 E = __ffma2_rn(__fmul2_rn(E0, bc2(-0.69314718056f)), rr, E0);
        const float2 om = __fadd2_rn(bc2(1.0f), neg2(E));
        const float2 Sl = __fmul2_rn(c1nu3, __fmul2_rn(E, make_float2(rcp_approx(om.x), rcp_approx(om.y))));
        if (i > 0) {
            const float2 dtau = __ffma2_rn(__fadd2_rn(chi, chi_prev), bc2(r2.x), bc2(r2.z));
            const float2 dS = __fadd2_rn(S_prev, neg2(Sl));
            const float2 ndtau = neg2(dtau);
            const unsigned d_lo = __reduce_min_sync(0xffffffffu, __float_as_uint(fminf(dtau.x, dtau.y)));
            const unsigned d_hi = __reduce_max_sync(0xffffffffu, __float_as_uint(fmaxf(dtau.x, dtau.y)));
            if (d_hi < LayerLimits<A>::all_thin) {
                seg_angles_thin<A, 0>(Cc, Psi, dtau, ndtau, dS);
            } else {
                const float2 q = __fmul2_rn(dS, make_float2(rcp_approx(dtau.x), rcp_approx(dtau.y)));
                if (d_lo >= LayerLimits<A>::all_thick) seg_angles_thick<A, 0>(Cc, Psi, ndtau, q);
                else {
                    const float2 dtc = make_float2(fmaxf(dtau.x, 1e-20f), fmaxf(dtau.y, 1e-20f));
                    const float2 qc = __fmul2_rn(dS, make_float2(rcp_approx(dtc.x), rcp_approx(dtc.y)));
                    seg_angles_w<A, 0>(Cc, Psi, dtc, neg2(dtc), qc);
                }
            }
        }
        chi_prev = chi; S_prev = Sl;
    }

    // hand the pair of every angle to the combining warp
    if (warp < a.n_chunks) {
#pragma unroll
        for (int k = 0; k < A; ++k) {
            reinterpret_cast<float2*>(ex + ((size_t)(warp * A + k) * 2 + 0) * kSlabTile)[lane] = Psi[k];
            reinterpret_cast<float2*>(ex + ((size_t)(warp * A + k) * 2 + 1) * kSlabTile)[lane] = Cc[k];
        }
        if (j1 == a.L && n_lev > 0) reinterpret_cast<float2*>(stop)[lane] = S_prev;      // the chunk that holds the top level
    }
    __syncthreads();
    pdl_launch_dependents();
    if (warp != 0) return;

    float2 H[A];
#pragma unroll
    for (int k = 0; k < A; ++k) H[k] = make_float2(0.0f, 0.0f);       // bottom boundary: I = S_0 (R11)
    for (int c = 0; c < a.n_chunks; ++c) {
#pragma unroll
        for (int k = 0; k < A; ++k) {
            const float2 psi = reinterpret_cast<const float2*>(ex + ((size_t)(c * A + k) * 2 + 0) * kSlabTile)[lane];
            const float2 cc = reinterpret_cast<const float2*>(ex + ((size_t)(c * A + k) * 2 + 1) * kSlabTile)[lane];
            H[k] = __ffma2_rn(psi, H[k], cc);
        }
    }
    const bool one = gnu.x < a.nNu, two = gnu.y < a.nNu;
    const bool rejected = a.model_flag[b] != 0;
    const float2 acc = flux_sum<A>(H, reinterpret_cast<const float2*>(stop)[lane], std::make_integer_sequence<int, A>{});
    const float scale = a.model_scale[b];
    if (a.fused.acc) {               // convolve + bin here: integer atomics into M[b][j] (obs.cuh); no flux is written
        if (rejected) return;
        if (one) fused_accumulate(a.fused, b, gnu.x, scale * acc.x);
        if (two) fused_accumulate(a.fused, b, gnu.y, scale * acc.y);
        return;
    }
    float* out = a.flux + (size_t)b * a.flux_stride;
    if (one) out[gnu.x] = rejected ? __int_as_float(0x7fc00000) : scale * acc.x;
    if (two) out[gnu.y] = rejected ? __int_as_float(0x7fc00000) : scale * acc.y;
}

struct SegPlan {
    bool ok = false;
    int n_chunks = 0, chunk_len = 0;
    size_t smem = 0;
};

// Chunking depends on the number of levels only, so within THIS kernel a model's result does not depend on the batch it
// is in.  (Across kernels it does, in the last bits: helios.h, HELIOS_OPT_KERNEL.)
inline SegPlan seg_plan(int L, int A, int S, int C, int x_floats, size_t smem_optin) {
    SegPlan p;
    if (L < 2 || A < 1 || A > kMaxAngles) return p;
    const int layers = L - 1;
    int len = (layers + kSegMaxChunks - 1) / kSegMaxChunks;
    if (len < 4) len = layers < 4 ? layers : 4;       // a chunk re-evaluates its lower boundary level: keep that under 25 %
    if (len > kSegMaxLen) return p;
    p.chunk_len = len;
    p.n_chunks = (layers + len - 1) / len;
    p.smem = seg_smem_bytes(A, p.n_chunks, len, x_floats, S, C);
    p.ok = p.smem <= smem_optin;
    return p;
}

// `configured`: this context has raised the instance's dynamic shared-memory limit to the opt-in maximum (see rt_slab.cuh)
struct SegMaps { CUtensorMap p2, t2, c; };

template <int A>
inline cudaError_t launch_rt_seg_a(const SegMaps& m, const SegArgs& a, size_t smem, size_t smem_optin, bool& configured,
                                   cudaStream_t stream, bool pdl) {
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(k_rt_seg<A>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_optin);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const dim3 grid(a.B, (a.nNu + kSlabTile - 1) / kSlabTile);
    return launch_kernel(k_rt_seg<A>, grid, dim3(a.n_chunks * 32), smem, stream, pdl, m.p2, m.t2, m.c, a);
}

struct SegSmemCache { bool configured[kMaxAngles + 1] = {}; };

inline cudaError_t launch_rt_seg(int A, const SegMaps& m, const SegArgs& a, size_t smem, size_t smem_optin, SegSmemCache& cache,
                                 cudaStream_t stream, bool pdl) {
    switch (A) {
        case 1: return launch_rt_seg_a<1>(m, a, smem, smem_optin, cache.configured[1], stream, pdl);
        case 2: return launch_rt_seg_a<2>(m, a, smem, smem_optin, cache.configured[2], stream, pdl);
        case 3: return launch_rt_seg_a<3>(m, a, smem, smem_optin, cache.configured[3], stream, pdl);
        case 4: return launch_rt_seg_a<4>(m, a, smem, smem_optin, cache.configured[4], stream, pdl);
        case 5: return launch_rt_seg_a<5>(m, a, smem, smem_optin, cache.configured[5], stream, pdl);
        case 6: return launch_rt_seg_a<6>(m, a, smem, smem_optin, cache.configured[6], stream, pdl);
        case 7: return launch_rt_seg_a<7>(m, a, smem, smem_optin, cache.configured[7], stream, pdl);
        case 8: return launch_rt_seg_a<8>(m, a, smem, smem_optin, cache.configured[8], stream, pdl);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace helios
