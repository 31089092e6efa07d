// helios_api.cu -- C ABI of libhelios_b200 (include/helios.h): context, table
// upload, atmosphere / observation setup, kernel launches.  sm_100a only.
#include <math_constants.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

#include "../../include/helios.h"
#include "common.cuh"
#include "obs.cuh"
#include "peaks.cuh"
#include "prep.cuh"
#include "rt_direct.cuh"
#include "rt_slab.cuh"
#include "rt_seg.cuh"

using namespace helios;

struct helios_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int num_sms = 148;

    // ---- opacity tables
    bool have_tables = false;
    int S = 0, C = 0, nT = 0, nP = 0, nNu = 0;
    long long stride = 0;               // padded row length, floats
    double nu0 = 0, dnu = 0;
    std::vector<double> T_grid, lp_grid;
    float* d_sigma = nullptr;           // [S][nT][nP][stride]   columns in the order of d_nu_index
    float* d_cia = nullptr;             // [C][nT][stride]
    int* d_nu_index = nullptr;          // [stride] wavenumber grid index held by every table column (>= nNu: padding)
    double* d_Tgrid = nullptr;

    // ---- atmosphere
    bool have_atmo = false;
    int L = 0, K = 0, A = 0;
    double p_bot = 0, p_top = 0, mmw = 0, he_to_h2 = 0, flux_const = 1;
    std::vector<double> mu, w;
    AngleSet ang{};
    double* d_lvl_p = nullptr; int* d_lvl_elem = nullptr; double* d_lvl_lw = nullptr;
    std::vector<double> lvl_p;          // level pressures, bar
    int tp_order = 1, tp_ratio = 0, NT = 0;   // temperature parametrisation (helios_set_tp_elements)
    unsigned extras = 0;                // HELIOS_EXTRA_* flags
    int n_extra = 0;
    int* d_lvl_ip = nullptr; double* d_lvl_u = nullptr; int* d_lvl_pclamp = nullptr;
    double* d_lvl_lnratio = nullptr;
    std::vector<int> lvl_ip;
    // staged kernel: plane schedule (segments of constant pressure cell) and TMA views of the tables
    int n_seg = 0, n_loads = 0;
    SlabSeg* d_seg = nullptr;           // [kSlabMaxRing][n_seg]: the schedule resolved for every ring depth
    int* d_load_ip = nullptr;
    bool have_tmaps = false, have_seg_maps = false;
    CUtensorMap tm_sigma{}, tm_cia{};
    SegMaps seg_maps{};                 // level-parallel kernel: boxes of one cell change (rt_seg.cuh)
    size_t smem_optin = 0, smem_sm = 0;
    SlabSmemCache slab_smem;
    SegSmemCache seg_smem;
    // CUDA graphs of whole calls (helios_forward_batch): a call that repeats with the same batch size and buffers is
    // captured once (prep -> RT -> observation, programmatic dependencies kept) and replayed with one launch
    struct GraphEntry { int B = 0, P = 0; const void* params = nullptr; const void* spectra = nullptr; const void* logl = nullptr;
                        unsigned long long epoch = 0;   // the context's state when the call was seen / captured
                        cudaGraphExec_t exec = nullptr; unsigned long long last_use = 0; };
    static constexpr int kGraphEntries = 32;
    GraphEntry graphs[kGraphEntries];
    GraphEntry graph_seen;              // the last call that ran without a graph
    unsigned long long graph_clock = 0;
    unsigned long long epoch = 1;       // bumped by every call that changes what the kernels' arguments would be (tables,
                                        // atmosphere, observation, parametrisation, extras, options, stream, workspace)
    unsigned long long n_graph_replays = 0;
    bool graphs_ok = true;              // false after a capture / instantiation failure: plain launches from then on
    cudaStream_t cap_stream = nullptr;

    // ---- observation
    bool have_obs = false, have_data = false;
    int J = 0;
    double logl_const = 0;
    double* d_edges = nullptr; double* d_obs = nullptr; double* d_inv2var = nullptr; double* d_var = nullptr;
    double* d_addvar = nullptr;         // [cap_B] 10^epsilon per model
    int* d_row_ptr = nullptr; int* d_row_lo = nullptr; float* d_W = nullptr;
    int* d_wt_ptr = nullptr; int* d_wt_j = nullptr; float* d_wt_w = nullptr;      // transposed operator (fused observation)
    unsigned long long* d_acc = nullptr; float* d_q = nullptr;                     // [cap_B][J] integer sums and their scales

    // ---- workspace (grown on demand)
    int cap_B = 0;
    float* d_rec = nullptr; size_t rec_bytes = 0;
    float* d_flux = nullptr; long long flux_stride = 0;
    float* d_scale = nullptr; int* d_flag = nullptr; float* d_model_x = nullptr;
    double* d_obs_partial = nullptr; unsigned* d_obs_arrived = nullptr;
    unsigned long long* d_counters = nullptr;    // [2]
    double* d_params_stage = nullptr; float* d_spectra_stage = nullptr; double* d_logl_stage = nullptr;

    // ---- options / statistics
    int opt_kernel = 0, opt_models_per_cta = 0, opt_timing = 0, opt_nu_order = 1, opt_fused = 0, opt_graphs = 1;
    static constexpr int kTimingRing = 64;
    cudaEvent_t ev[kTimingRing][4] = {};
    bool ev_has_obs[kTimingRing] = {};
    bool ev_created = false;
    long long timed_calls = 0;
    unsigned long long n_models = 0, n_launches = 0;
};

static std::string g_create_error;

static int fail(helios_ctx* c, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    if (c) c->err = buf; else g_create_error = buf;
    return code;
}

#define CU_TRY(c, call)                                                                      \
    do {                                                                                     \
        cudaError_t e_ = (call);                                                             \
        if (e_ != cudaSuccess)                                                               \
            return fail((c), e_ == cudaErrorMemoryAllocation ? HELIOS_ENOMEM : HELIOS_ECUDA, \
                        "%s failed: %s", #call, cudaGetErrorString(e_));                     \
    } while (0)

template <class T>
static void dfree(T*& p) { if (p) { cudaFree(p); p = nullptr; } }

template <class T>
static cudaError_t upload(T*& dst, const std::vector<T>& src, cudaStream_t s) {
    dfree(dst);
    cudaError_t e = cudaMalloc(&dst, sizeof(T) * (src.empty() ? 1 : src.size()));
    if (e != cudaSuccess) return e;
    if (!src.empty()) e = cudaMemcpyAsync(dst, src.data(), sizeof(T) * src.size(), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return e;
    return cudaStreamSynchronize(s);     // src may be a temporary
}

// A captured call holds kernel arguments BY VALUE (device pointers, sizes, logl_const, the tensor maps ...): every
// setter calls this, so that no graph outlives the state it was captured from; the epoch is a second guard -- an entry
// whose epoch is not the context's is never replayed, whatever path forgot to come through here.
static void graphs_invalidate(helios_ctx* c) {
    ++c->epoch;
    for (auto& g : c->graphs) { if (g.exec) cudaGraphExecDestroy(g.exec); g = helios_ctx::GraphEntry{}; }
    c->graph_seen = helios_ctx::GraphEntry{};
}

static void free_all(helios_ctx* c) {
    graphs_invalidate(c);
    if (c->cap_stream) { cudaStreamDestroy(c->cap_stream); c->cap_stream = nullptr; }
    dfree(c->d_sigma); dfree(c->d_cia); dfree(c->d_Tgrid); dfree(c->d_nu_index);
    dfree(c->d_lvl_p); dfree(c->d_lvl_elem); dfree(c->d_lvl_lw); dfree(c->d_lvl_ip); dfree(c->d_lvl_u);
    dfree(c->d_lvl_pclamp); dfree(c->d_lvl_lnratio);
    dfree(c->d_seg); dfree(c->d_load_ip);
    dfree(c->d_edges); dfree(c->d_obs); dfree(c->d_inv2var); dfree(c->d_var); dfree(c->d_addvar); dfree(c->d_row_ptr); dfree(c->d_row_lo); dfree(c->d_W);
    dfree(c->d_wt_ptr); dfree(c->d_wt_j); dfree(c->d_wt_w); dfree(c->d_acc); dfree(c->d_q);
    dfree(c->d_rec); dfree(c->d_flux); dfree(c->d_scale); dfree(c->d_flag); dfree(c->d_model_x); dfree(c->d_counters);
    dfree(c->d_obs_partial); dfree(c->d_obs_arrived);
    dfree(c->d_params_stage); dfree(c->d_spectra_stage); dfree(c->d_logl_stage);
}

static int n_params(const helios_ctx* c) { return 2 + c->NT + c->S + c->n_extra; }

// Levels -> finite elements (Sect. 2.5.1): n_elements elements equidistant in log p, order q with
// Gauss-Lobatto points on the reference element; per level the element index and the values of
// the element's q + 1 Lagrange polynomials (Eq. 13).  q = 0: one isothermal value.
static cudaError_t build_tp(helios_ctx* c, int n_elements, int q) {
    std::vector<int> elem(c->L, 0);
    std::vector<double> lw((size_t)c->L * kMaxTpNodes, 0.0);
    double node[kMaxTpNodes] = {0.0, 1.0, 0.0, 0.0, 0.0};
    if (q == 2) { node[1] = 0.5; node[2] = 1.0; }
    if (q == 3) { const double a = 1.0 / std::sqrt(5.0); node[1] = 0.5 * (1.0 - a); node[2] = 0.5 * (1.0 + a); node[3] = 1.0; }
    if (q == 4) { const double a = std::sqrt(3.0 / 7.0); node[1] = 0.5 * (1.0 - a); node[2] = 0.5; node[3] = 0.5 * (1.0 + a); node[4] = 1.0; }
    const double x_bot = std::log10(c->p_bot), x_top = std::log10(c->p_top);
    for (int l = 0; l < c->L; ++l) {
        if (q == 0) { lw[(size_t)l * kMaxTpNodes] = 1.0; continue; }
        const double s = (std::log10(c->lvl_p[l]) - x_bot) / (x_top - x_bot) * n_elements;
        int k = (int)std::floor(s);
        k = k < 0 ? 0 : (k > n_elements - 1 ? n_elements - 1 : k);
        const double xi = s - k;
        elem[l] = k;
        for (int i = 0; i <= q; ++i) {
            double ell = 1.0;
            for (int j = 0; j <= q; ++j) if (j != i) ell *= (xi - node[j]) / (node[i] - node[j]);
            lw[(size_t)l * kMaxTpNodes + i] = ell;
        }
    }
    cudaError_t e = upload(c->d_lvl_elem, elem, c->stream);
    if (e == cudaSuccess) e = upload(c->d_lvl_lw, lw, c->stream);
    return e;
}

// TMA views of the resident tables for the staged kernel (cuTensorMapEncodeTiled, resolved through
// the runtime so that libcuda is not a link-time dependency):
//   sigma {nu (padded row), ip, iT, s}, box {32, 1, nT, 1};   cia {nu, iT, c}, box {32, nT, 1}.
typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static bool build_tensor_maps(helios_ctx* c) {
    c->have_tmaps = c->have_seg_maps = false;
    std::memset(&c->tm_sigma, 0, sizeof c->tm_sigma);
    std::memset(&c->tm_cia, 0, sizeof c->tm_cia);
    std::memset(&c->seg_maps, 0, sizeof c->seg_maps);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) != cudaSuccess ||
        qres != cudaDriverEntryPointSuccess || !fn) {
        cudaGetLastError();
        return false;
    }
    encode_tiled_fn encode = (encode_tiled_fn)fn;
    const cuuint64_t row = (cuuint64_t)c->stride * sizeof(float);
    // level-parallel kernel: all species at two pressure nodes of one temperature node / two temperature nodes of one
    // pressure node; all CIA pairs at one temperature node
    {
        bool ok = true;
        cuuint32_t estr[4] = {1, 1, 1, 1};
        if (c->S > 0) {
            cuuint64_t dims[4] = {(cuuint64_t)c->stride, (cuuint64_t)c->nP, (cuuint64_t)c->nT, (cuuint64_t)c->S};
            cuuint64_t strides[3] = {row, row * c->nP, row * c->nP * c->nT};
            cuuint32_t box_p2[4] = {(cuuint32_t)kSlabTile, 2, 1, (cuuint32_t)c->S}, box_t2[4] = {(cuuint32_t)kSlabTile, 1, 2, (cuuint32_t)c->S};
            ok = ok && encode(&c->seg_maps.p2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, c->d_sigma, dims, strides, box_p2, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
            ok = ok && encode(&c->seg_maps.t2, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, c->d_sigma, dims, strides, box_t2, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
        }
        if (c->C > 0) {
            cuuint64_t dims[3] = {(cuuint64_t)c->stride, (cuuint64_t)c->nT, (cuuint64_t)c->C};
            cuuint64_t strides[2] = {row, row * c->nT};
            cuuint32_t box[3] = {(cuuint32_t)kSlabTile, 1, (cuuint32_t)c->C};
            ok = ok && encode(&c->seg_maps.c, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, c->d_cia, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
        }
        c->have_seg_maps = ok;
    }
    if (c->nT > 256) return false;        // the staged kernel's box holds every temperature node of a plane
    if (c->S > 0) {
        cuuint64_t dims[4] = {(cuuint64_t)c->stride, (cuuint64_t)c->nP, (cuuint64_t)c->nT, (cuuint64_t)c->S};
        cuuint64_t strides[3] = {row, row * c->nP, row * c->nP * c->nT};
        cuuint32_t box[4] = {(cuuint32_t)kSlabTile, 1, (cuuint32_t)c->nT, 1};
        cuuint32_t estr[4] = {1, 1, 1, 1};
        if (encode(&c->tm_sigma, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 4, c->d_sigma, dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return false;
    }
    if (c->C > 0) {
        cuuint64_t dims[3] = {(cuuint64_t)c->stride, (cuuint64_t)c->nT, (cuuint64_t)c->C};
        cuuint64_t strides[2] = {row, row * c->nT};
        cuuint32_t box[3] = {(cuuint32_t)kSlabTile, (cuuint32_t)c->nT, 1};
        cuuint32_t estr[3] = {1, 1, 1};
        if (encode(&c->tm_cia, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, c->d_cia, dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) return false;
    }
    c->have_tmaps = true;
    return true;
}

// Column order of the resident tables.  The kernels own 64 adjacent table columns per warp and take warp-uniform
// shortcuts when all of them are optically thin (or thick) in a layer, so columns of similar opacity should sit
// next to each other -- and on a fine grid adjacent WAVENUMBERS are not: line cores and wings alternate.  The
// columns are therefore sorted once, at load time, by a reference opacity: the cross-sections at one table node
// (middle temperature, a low pressure where the lines are sharp), grouped by the species that dominates the
// column and ordered by its cross-section within the group.  Every kernel reads nu_index[column] for the
// wavenumber and writes its flux to that grid point, so the order is invisible outside the library.
static void opacity_order(const std::vector<std::vector<float>>& ref_rows, int nNu, std::vector<int>& order) {
    order.resize(nNu);
    for (int i = 0; i < nNu; ++i) order[i] = i;
    const int S = (int)ref_rows.size();
    if (S == 0) return;
    std::vector<int> dom(nNu, 0);
    std::vector<float> val(nNu, 0.0f);
    for (int i = 0; i < nNu; ++i) {
        int best = 0;
        for (int s = 1; s < S; ++s) if (ref_rows[s][i] > ref_rows[best][i]) best = s;
        dom[i] = best; val[i] = ref_rows[best][i];
        if (!(val[i] == val[i])) val[i] = 0.0f;      // a NaN in the table must not break the ordering of the sort
    }
    std::stable_sort(order.begin(), order.end(), [&](int x, int y) {
        if (dom[x] != dom[y]) return dom[x] < dom[y];
        return val[x] < val[y];
    });
}

// dst[row][j] = src[row][nu_index[j]] for j < nNu, 0 in the padding: rows of nNu floats -> rows of `stride` floats
__global__ void k_gather_rows(float* dst, const float* src, const int* nu_index, int nNu, long long stride, long long rows) {
    const long long j = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= stride) return;
    const int g = nu_index[j];
    for (long long r = blockIdx.y; r < rows; r += gridDim.y)
        dst[r * stride + j] = (j < nNu) ? src[r * (long long)nNu + g] : 0.0f;
}

// One micro-benchmark: one block of 1024 threads per SM, timed with CUDA events on the context's stream (the
// launch overhead is < 1 % of the 0.5 ms a kernel takes); the SM clock during the run is block 0's
// clock64() / %globaltimer ratio.  Returns scheduler cycles per warp instruction and operations per clock per SM.
template <int MODE>
static int run_peak(helios_ctx* c, float* d_out, PeakTimes* d_times, cudaEvent_t e0, cudaEvent_t e1,
                    double* cycles_per_instr, double* sm_ops_per_clk, double* mhz) {
    double best_ms = 0.0, best_mhz = 0.0;
    for (int rep = 0; rep < 3; ++rep) {      // the first repetition warms the clocks up; keep the fastest
        CU_TRY(c, cudaEventRecord(e0, c->stream));
        k_peak<MODE><<<c->num_sms, kPeakThreads, 0, c->stream>>>(d_out, d_times, 0.999f, 0.001f, 5u);
        CU_TRY(c, cudaEventRecord(e1, c->stream));
        c->n_launches += 1;
        CU_TRY(c, cudaGetLastError());
        PeakTimes t;
        CU_TRY(c, cudaMemcpyAsync(&t, d_times, sizeof t, cudaMemcpyDeviceToHost, c->stream));
        CU_TRY(c, cudaStreamSynchronize(c->stream));
        float ms = 0.0f;
        CU_TRY(c, cudaEventElapsedTime(&ms, e0, e1));
        if (rep == 0 || ms < best_ms) { best_ms = ms; best_mhz = t.ns > 0 ? 1e3 * (double)t.cycles / (double)t.ns : 0.0; }
    }
    const double cycles = best_ms * 1e-3 * best_mhz * 1e6;
    const double thread_ops = (double)kPeakIters * kPeakChains;
    const double warps_per_scheduler = (kPeakThreads / 32) / 4.0;
    *cycles_per_instr = cycles / (thread_ops * warps_per_scheduler);
    *sm_ops_per_clk = thread_ops * kPeakThreads / cycles;
    *mhz = best_mhz;
    return HELIOS_OK;
}

extern "C" {

int helios_create(helios_ctx** out, int device, void* cuda_stream) {
    if (!out) return fail(nullptr, HELIOS_EINVAL, "helios_create: out is NULL");
    *out = nullptr;
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev == 0)
        return fail(nullptr, HELIOS_ECUDA, "helios_create: no CUDA device (%s); this library has no CPU fallback",
                    e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
    if (device < 0 || device >= ndev) return fail(nullptr, HELIOS_EINVAL, "helios_create: device %d of %d", device, ndev);
    e = cudaSetDevice(device);
    if (e != cudaSuccess) return fail(nullptr, HELIOS_ECUDA, "cudaSetDevice: %s", cudaGetErrorString(e));
    cudaFuncAttributes fa;
    e = cudaFuncGetAttributes(&fa, k_prep);
    if (e != cudaSuccess)
        return fail(nullptr, HELIOS_ECUDA, "helios_create: no usable sm_100a kernel image on device %d (%s)", device,
                    cudaGetErrorString(e));
    helios_ctx* c = new (std::nothrow) helios_ctx();
    if (!c) return fail(nullptr, HELIOS_ENOMEM, "helios_create: out of host memory");
    c->device = device;
    c->stream = (cudaStream_t)cuda_stream;
    cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, device);
    int v = 0;
    cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, device); c->smem_optin = (size_t)v;
    cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device); c->smem_sm = (size_t)v;
    e = cudaMalloc(&c->d_counters, 2 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(c->d_counters, 0, 2 * sizeof(unsigned long long));
    if (e != cudaSuccess) { delete c; return fail(nullptr, HELIOS_ECUDA, "helios_create: %s", cudaGetErrorString(e)); }
    *out = c;
    return HELIOS_OK;
}

void helios_destroy(helios_ctx* c) {
    if (!c) return;
    cudaSetDevice(c->device);
    cudaStreamSynchronize(c->stream);
    if (c->ev_created) for (auto& q : c->ev) for (auto& e : q) cudaEventDestroy(e);
    free_all(c);
    delete c;
}

int helios_set_stream(helios_ctx* c, void* s) {
    if (!c) return HELIOS_EINVAL;
    c->stream = (cudaStream_t)s;
    graphs_invalidate(c);
    return HELIOS_OK;
}

const char* helios_last_error(const helios_ctx* c) { return c ? c->err.c_str() : g_create_error.c_str(); }

int helios_set_option(helios_ctx* c, int key, int value) {
    if (!c) return HELIOS_EINVAL;
    graphs_invalidate(c);
    switch (key) {
        case HELIOS_OPT_GRAPHS:
            c->opt_graphs = value ? 1 : 0; return HELIOS_OK;
        case HELIOS_OPT_KERNEL:
            if (value < 0 || value > 3) return fail(c, HELIOS_EINVAL, "HELIOS_OPT_KERNEL must be 0, 1, 2 or 3");
            c->opt_kernel = value; return HELIOS_OK;
        case HELIOS_OPT_MODELS_PER_CTA:
            if (value != 0 && value != 8 && value != 16 && value != 20 && value != 24 && value != 27)
                return fail(c, HELIOS_EINVAL, "HELIOS_OPT_MODELS_PER_CTA must be 0 (auto), 8, 16, 20, 24 or 27");
            c->opt_models_per_cta = value; return HELIOS_OK;
        case HELIOS_OPT_FUSED_OBS:
            c->opt_fused = value ? 1 : 0; return HELIOS_OK;
        case HELIOS_OPT_NU_ORDER:
            if (value != 0 && value != 1) return fail(c, HELIOS_EINVAL, "HELIOS_OPT_NU_ORDER must be 0 (grid order) or 1 (opacity order)");
            c->opt_nu_order = value; return HELIOS_OK;
        case HELIOS_OPT_TIMING:
            c->opt_timing = value ? 1 : 0; c->timed_calls = 0;
            if (value && !c->ev_created) {
                for (auto& q : c->ev) for (auto& e : q) CU_TRY(c, cudaEventCreate(&e));
                c->ev_created = true;
            }
            return HELIOS_OK;
        default: return fail(c, HELIOS_EINVAL, "unknown option %d", key);
    }
}

int helios_load_opacity(helios_ctx* c, int S, int nT, const double* T_grid, int nP, const double* lp_grid,
                        int nNu, double nu0, double dnu, const float* const* sigma, int C,
                        const float* const* cia, unsigned flags) {
    if (!c) return HELIOS_EINVAL;
    if (S < 0 || S > 64 || C < 0 || C > kMaxCia || S + C < 1) return fail(c, HELIOS_EINVAL, "load_opacity: n_species %d, n_cia %d", S, C);
    if (nT < 2 || nP < 2 || nNu < 2 || !(dnu > 0) || !T_grid || !lp_grid) return fail(c, HELIOS_EINVAL, "load_opacity: bad grid sizes");
    for (int i = 1; i < nT; ++i) if (!(T_grid[i] > T_grid[i - 1])) return fail(c, HELIOS_EINVAL, "load_opacity: T grid not strictly increasing");
    for (int i = 1; i < nP; ++i) if (!(lp_grid[i] > lp_grid[i - 1])) return fail(c, HELIOS_EINVAL, "load_opacity: log10 p grid not strictly increasing");
    if ((S > 0 && !sigma) || (C > 0 && !cia)) return fail(c, HELIOS_EINVAL, "load_opacity: NULL table pointer array");
    for (int s = 0; s < S; ++s) if (!sigma[s]) return fail(c, HELIOS_EINVAL, "load_opacity: sigma[%d] is NULL", s);
    for (int k = 0; k < C; ++k) if (!cia[k]) return fail(c, HELIOS_EINVAL, "load_opacity: cia[%d] is NULL", k);
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    graphs_invalidate(c);
    c->have_tables = c->have_atmo = c->have_obs = c->have_data = false;
    dfree(c->d_sigma); dfree(c->d_cia); dfree(c->d_nu_index);
    c->S = S; c->C = C; c->nT = nT; c->nP = nP; c->nNu = nNu; c->nu0 = nu0; c->dnu = dnu;
    c->stride = ((long long)nNu + kSlabTile - 1) / kSlabTile * kSlabTile;   // rows padded to the staged kernel's tile (256 B)
    c->T_grid.assign(T_grid, T_grid + nT);
    c->lp_grid.assign(lp_grid, lp_grid + nP);
    const bool on_device = (flags & HELIOS_PTRS_ON_DEVICE) != 0;
    const size_t rows_s = (size_t)nT * nP;
    // column order (HELIOS_OPT_NU_ORDER): reference rows at the middle temperature node and a low-pressure node
    std::vector<int> order;
    {
        std::vector<std::vector<float>> ref;
        if (c->opt_nu_order == 1 && S > 0) {
            const int iT_ref = nT / 2, ip_ref = (int)std::lround(0.375 * (nP - 1));
            ref.assign(S, std::vector<float>(nNu));
            for (int s = 0; s < S; ++s)
                CU_TRY(c, cudaMemcpy(ref[s].data(), sigma[s] + ((size_t)iT_ref * nP + ip_ref) * nNu, sizeof(float) * nNu,
                                     on_device ? cudaMemcpyDeviceToHost : cudaMemcpyHostToHost));
        }
        opacity_order(ref, nNu, order);
        order.resize((size_t)c->stride);
        for (long long j = nNu; j < c->stride; ++j) order[j] = (int)j;      // padding columns: >= nNu, never written out
        CU_TRY(c, upload(c->d_nu_index, order, c->stream));
    }
    // upload: rows of nNu floats -> padded rows in column order (through a device staging slab when the source is on the host)
    float* d_stage = nullptr;
    struct Stage { float*& p; ~Stage() { dfree(p); } } stage_guard{d_stage};
    const size_t slab_rows = std::max(rows_s, (size_t)nT);
    if (!on_device) CU_TRY(c, cudaMalloc(&d_stage, sizeof(float) * slab_rows * nNu));
    auto put = [&](float* dst, const float* src, size_t rows) -> cudaError_t {
        const float* dsrc = src;
        if (!on_device) {
            cudaError_t e = cudaMemcpyAsync(d_stage, src, sizeof(float) * rows * nNu, cudaMemcpyHostToDevice, c->stream);
            if (e != cudaSuccess) return e;
            dsrc = d_stage;
        }
        const dim3 grid((unsigned)((c->stride + 255) / 256), (unsigned)std::min<size_t>(rows, 1024));
        k_gather_rows<<<grid, 256, 0, c->stream>>>(dst, dsrc, c->d_nu_index, nNu, c->stride, (long long)rows);
        c->n_launches += 1;
        return cudaGetLastError();
    };
    if (S > 0) {
        CU_TRY(c, cudaMalloc(&c->d_sigma, sizeof(float) * (size_t)S * rows_s * c->stride));
        for (int s = 0; s < S; ++s) CU_TRY(c, put(c->d_sigma + (size_t)s * rows_s * c->stride, sigma[s], rows_s));
    }
    if (C > 0) {
        CU_TRY(c, cudaMalloc(&c->d_cia, sizeof(float) * (size_t)C * nT * c->stride));
        for (int k = 0; k < C; ++k) CU_TRY(c, put(c->d_cia + (size_t)k * nT * c->stride, cia[k], (size_t)nT));
    }
    CU_TRY(c, upload(c->d_Tgrid, c->T_grid, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    build_tensor_maps(c);      // failure only disables the staged kernel
    c->have_tables = true;
    c->cap_B = 0;    // record size depends on S, C
    return HELIOS_OK;
}

// n-point Gauss-Legendre rule on [-1, 1]: roots of P_n by Newton's method.
static void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& W) {
    x.resize(n); W.resize(n);
    for (int i = 0; i < (n + 1) / 2; ++i) {
        double z = std::cos(kPi * (i + 0.75) / (n + 0.5)), pp = 1.0;
        for (int it = 0; it < 64; ++it) {
            double pa = 1.0, pb = 0.0;
            for (int j = 0; j < n; ++j) {
                double pc = pb; pb = pa;
                pa = ((2.0 * j + 1.0) * z * pb - j * pc) / (j + 1.0);
            }
            pp = n * (z * pa - pb) / (z * z - 1.0);
            double dz = pa / pp;
            z -= dz;
            if (std::fabs(dz) < 1e-15) break;
        }
        double pa = 1.0, pb = 0.0;
        for (int j = 0; j < n; ++j) { double pc = pb; pb = pa; pa = ((2.0 * j + 1.0) * z * pb - j * pc) / (j + 1.0); }
        pp = n * (z * pa - pb) / (z * z - 1.0);
        x[i] = -z; x[n - 1 - i] = z;
        W[i] = W[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
    }
}

static void axis_cell(const std::vector<double>& grid, double v, int& i, double& w, int& clamped) {
    const int n = (int)grid.size();
    i = 0;
    while (i < n - 2 && grid[i + 1] <= v) ++i;
    w = (v - grid[i]) / (grid[i + 1] - grid[i]);
    clamped = 0;
    if (w < 0.0) { w = 0.0; clamped = 1; }
    if (w > 1.0) { w = 1.0; clamped = 1; }
}

int helios_set_atmosphere(helios_ctx* c, int L, double p_bot, double p_top, int K, int A, double mmw,
                          double he_to_h2, double flux_const) {
    if (!c) return HELIOS_EINVAL;
    if (!c->have_tables) return fail(c, HELIOS_ESTATE, "set_atmosphere: call helios_load_opacity first");
    if (L < 2 || L > 4096) return fail(c, HELIOS_EINVAL, "set_atmosphere: n_levels %d (2..4096)", L);
    if (!(p_bot > p_top) || !(p_top > 0)) return fail(c, HELIOS_EINVAL, "set_atmosphere: need p_bottom > p_top > 0");
    if (K < 1 || K > 64) return fail(c, HELIOS_EINVAL, "set_atmosphere: n_knots %d (1..64)", K);
    if (A < 1 || A > kMaxAngles) return fail(c, HELIOS_EINVAL, "set_atmosphere: n_angles %d (1..%d)", A, kMaxAngles);
    if (!(mmw > 0) || !(he_to_h2 >= 0) || !(flux_const > 0) || !std::isfinite(flux_const))
        return fail(c, HELIOS_EINVAL, "set_atmosphere: need mean_mol_weight > 0, he_to_h2 >= 0, flux_const > 0 (finite)");
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    graphs_invalidate(c);
    c->have_atmo = false;
    c->L = L; c->K = K; c->A = A; c->p_bot = p_bot; c->p_top = p_top; c->mmw = mmw; c->he_to_h2 = he_to_h2;
    c->flux_const = flux_const;

    std::vector<double> p(L), u(L), lnr(L, 0.0);
    std::vector<int> ip(L), pcl(L);
    for (int l = 0; l < L; ++l) {
        p[l] = p_bot * std::pow(p_top / p_bot, (double)l / (double)(L - 1));   // equidistant in log p
        axis_cell(c->lp_grid, std::log10(p[l]), ip[l], u[l], pcl[l]);
    }
    c->lvl_p = p;
    // K nodal temperatures, linear in log p = K - 1 first-order elements (one value: isothermal)
    c->tp_order = K > 1 ? 1 : 0; c->tp_ratio = 0; c->NT = K;
    CU_TRY(c, build_tp(c, K > 1 ? K - 1 : 1, c->tp_order));
    for (int l = 0; l + 1 < L; ++l) lnr[l] = std::log(p[l] / p[l + 1]);
    c->lvl_ip = ip;
    CU_TRY(c, upload(c->d_lvl_p, p, c->stream));
    CU_TRY(c, upload(c->d_lvl_ip, ip, c->stream));
    CU_TRY(c, upload(c->d_lvl_u, u, c->stream));
    CU_TRY(c, upload(c->d_lvl_pclamp, pcl, c->stream));
    CU_TRY(c, upload(c->d_lvl_lnratio, lnr, c->stream));

    // plane schedule of the staged kernel: segments of constant pressure cell; segment k needs the
    // table planes ip_k + 1 ("hi") and ip_k ("lo"); a plane already loaded for the previous
    // segment is reused, so with levels denser than table nodes there is one new load per segment.
    {
        std::vector<int> seg_lbegin, seg_hi, seg_lo, load_ip;
        for (int l = 0; l < L; ++l) {
            if (l > 0 && ip[l] == ip[l - 1]) continue;
            seg_lbegin.push_back(l);
            auto find_or_load = [&](int node) {
                const int n = (int)load_ip.size();
                for (int e = std::max(0, n - 2); e < n; ++e) if (load_ip[e] == node) return e;
                load_ip.push_back(node);
                return n;
            };
            const int hi = find_or_load(ip[l] + 1);
            const int lo = find_or_load(ip[l]);
            seg_hi.push_back(hi); seg_lo.push_back(lo);
        }
        seg_lbegin.push_back(L);
        c->n_seg = (int)seg_hi.size(); c->n_loads = (int)load_ip.size();
        // slot / mbarrier parity of every load and the slots each segment frees, for every ring depth NB:
        // load e lives in slot e % NB during its use number e / NB; a segment frees the loads older than the next one's
        std::vector<SlabSeg> seg((size_t)kSlabMaxRing * c->n_seg);
        for (int nb = 1; nb <= kSlabMaxRing; ++nb) {
            int released = 0;
            for (int k = 0; k < c->n_seg; ++k) {
                SlabSeg& g = seg[(size_t)(nb - 1) * c->n_seg + k];
                g.l_begin = seg_lbegin[k]; g.l_end = seg_lbegin[k + 1];
                g.hi = (seg_hi[k] % nb) | (((seg_hi[k] / nb) & 1) << 8);
                g.lo = (seg_lo[k] % nb) | (((seg_lo[k] / nb) & 1) << 8);
                g.shifted = (k > 0 && seg_hi[k] == seg_lo[k - 1]) ? 1 : 0;
                g.rel_slot = 0; g.rel_count = 0; g.pad = 0;
                if (k + 1 < c->n_seg) {
                    const int next_first = std::min(seg_hi[k + 1], seg_lo[k + 1]);
                    g.rel_slot = released % nb;
                    g.rel_count = std::max(0, next_first - released);
                    released = std::max(released, next_first);
                }
            }
        }
        CU_TRY(c, upload(c->d_seg, seg, c->stream));
        CU_TRY(c, upload(c->d_load_ip, load_ip, c->stream));
    }

    std::vector<double> x, W;
    gauss_legendre(A, x, W);
    c->mu.resize(A); c->w.resize(A);
    AngleSet& g = c->ang;
    std::memset(&g, 0, sizeof g);
    g.n = A;
    double wmu_sum = 0.0;
    for (int k = 0; k < A; ++k) {
        c->mu[k] = 0.5 * (x[k] + 1.0);
        c->w[k] = 0.5 * W[k];
        g.mu[k] = (float)c->mu[k];
        g.inv_mu[k] = (float)(1.0 / c->mu[k]);
        g.c_exp[k] = (float)(kLog2e / c->mu[k]);
        g.wmu[k] = (float)(c->w[k] * c->mu[k]);
        g.thr[k] = (float)(kPhiSwitch * c->mu[k]);
        g.wH[k] = (float)(c->w[k] * c->mu[k] * c->mu[k]);
        const double pc[5] = {1.0, kPhiC1, kPhiC2, kPhiC3, kPhiC4};
        for (int j = 0; j < 5; ++j) g.pc[j][k] = (float)(pc[j] / std::pow(c->mu[k], j + 1));
        wmu_sum += c->w[k] * c->mu[k];
    }
    g.wmu_sum = (float)wmu_sum;
    // the staged kernel uses the compile-time copy of this rule (common.cuh): they must agree
    for (int k = 0; k < A; ++k)
        if (std::fabs(c->mu[k] - kGLmu[A - 1][k]) > 1e-14 || std::fabs(c->w[k] - kGLw[A - 1][k]) > 1e-14)
            return fail(c, HELIOS_ECUDA, "internal: Gauss-Legendre table mismatch at n = %d, k = %d", A, k);
    c->have_atmo = true;
    c->cap_B = 0;
    return HELIOS_OK;
}

int helios_get_angles(const helios_ctx* c, double* mu, double* w) {
    if (!c || !c->have_atmo || !mu || !w) return HELIOS_EINVAL;
    for (int k = 0; k < c->A; ++k) { mu[k] = c->mu[k]; w[k] = c->w[k]; }
    return HELIOS_OK;
}

int helios_set_observation(helios_ctx* c, int J, const double* edges, const double* obs, const double* err,
                           const double* inst_sigma) {
    if (!c) return HELIOS_EINVAL;
    if (!c->have_tables) return fail(c, HELIOS_ESTATE, "set_observation: call helios_load_opacity first");
    if (J < 1 || !edges) return fail(c, HELIOS_EINVAL, "set_observation: n_bins %d", J);
    if ((obs == nullptr) != (err == nullptr)) return fail(c, HELIOS_EINVAL, "set_observation: obs and obs_err must both be given or both NULL");
    const double nu_first = c->nu0, nu_last = c->nu0 + c->dnu * (c->nNu - 1), tol = 1e-9 * c->dnu;
    std::vector<double> e(edges, edges + J + 1);
    for (int j = 0; j <= J; ++j) {
        if (!std::isfinite(e[j]) || e[j] < nu_first - tol || e[j] > nu_last + tol)
            return fail(c, HELIOS_EINVAL, "set_observation: bin edge %d = %g outside the grid [%g, %g]", j, e[j], nu_first, nu_last);
        e[j] = std::fmin(std::fmax(e[j], nu_first), nu_last);
        if (j > 0 && !(e[j] > e[j - 1])) return fail(c, HELIOS_EINVAL, "set_observation: bin edges not strictly ascending at %d", j);
    }
    if (obs) for (int j = 0; j < J; ++j)
        if (!std::isfinite(obs[j]) || !(err[j] > 0) || !std::isfinite(err[j]))
            return fail(c, HELIOS_EINVAL, "set_observation: obs/obs_err[%d] invalid", j);
    if (inst_sigma) for (int k = 0; k < c->nNu; ++k)
        if (!(inst_sigma[k] >= 0) || !std::isfinite(inst_sigma[k]))
            return fail(c, HELIOS_EINVAL, "set_observation: inst_sigma[%d] invalid", k);
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    graphs_invalidate(c);
    c->have_obs = c->have_data = false;
    c->J = J;

    // band extents of each row of W (marshalling: which grid points can contribute)
    std::vector<int> row_ptr(J + 1, 0), row_lo(J), klo(J), khi(J);
    for (int j = 0; j < J; ++j) {
        int a = (int)std::floor((e[j] - c->nu0) / c->dnu), b = (int)std::ceil((e[j + 1] - c->nu0) / c->dnu);
        a = a < 0 ? 0 : a; b = b > c->nNu - 1 ? c->nNu - 1 : b;
        klo[j] = a; khi[j] = b;
        int reach = 0;
        if (inst_sigma) for (int k = a; k <= b; ++k) {
            int r = (int)std::ceil(5.0 * inst_sigma[k] / c->dnu) + 1;
            reach = r > reach ? r : reach;
        }
        int lo = a - reach < 0 ? 0 : a - reach, hi = b + reach > c->nNu - 1 ? c->nNu - 1 : b + reach;
        row_lo[j] = lo;
        row_ptr[j + 1] = row_ptr[j] + (hi - lo + 1);
    }
    int* d_klo = nullptr; int* d_khi = nullptr; double* d_sig = nullptr; double* d_norm = nullptr;
    struct Temporaries {      // freed on every return path, also the CU_TRY early returns
        int*& a; int*& b; double*& s; double*& n;
        ~Temporaries() { dfree(a); dfree(b); dfree(s); dfree(n); }
    } temporaries{d_klo, d_khi, d_sig, d_norm};
    std::vector<double> sig;
    if (inst_sigma) sig.assign(inst_sigma, inst_sigma + c->nNu);
    CU_TRY(c, upload(c->d_edges, e, c->stream));
    CU_TRY(c, upload(c->d_row_ptr, row_ptr, c->stream));
    CU_TRY(c, upload(c->d_row_lo, row_lo, c->stream));
    CU_TRY(c, upload(d_klo, klo, c->stream));
    CU_TRY(c, upload(d_khi, khi, c->stream));
    if (inst_sigma) CU_TRY(c, upload(d_sig, sig, c->stream));
    CU_TRY(c, cudaMalloc(&d_norm, sizeof(double) * c->nNu));
    dfree(c->d_W);
    CU_TRY(c, cudaMalloc(&c->d_W, sizeof(float) * (size_t)row_ptr[J]));
    ObsBuildArgs ba{c->nNu, J, c->nu0, c->dnu, c->d_edges, d_sig, d_norm, c->d_row_ptr, c->d_row_lo, d_klo, d_khi, c->d_W};
    k_conv_norm<<<(c->nNu + 127) / 128, 128, 0, c->stream>>>(ba);
    int max_len = 0;
    for (int j = 0; j < J; ++j) max_len = std::max(max_len, row_ptr[j + 1] - row_ptr[j]);
    k_build_W<<<dim3((max_len + 127) / 128, J), 128, 0, c->stream>>>(ba);
    c->n_launches += 2;
    CU_TRY(c, cudaGetLastError());
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    {   // the operator by grid point (CSR, zeros dropped) for the fused epilogue of the RT kernels (obs.cuh); marshalling only
        std::vector<float> Wh((size_t)row_ptr[J]);
        CU_TRY(c, cudaMemcpy(Wh.data(), c->d_W, sizeof(float) * Wh.size(), cudaMemcpyDeviceToHost));
        std::vector<int> wt_ptr(c->nNu + 1, 0), wt_j;
        std::vector<float> wt_w;
        for (int j = 0; j < J; ++j)
            for (int e2 = row_ptr[j]; e2 < row_ptr[j + 1]; ++e2)
                if (Wh[e2] != 0.0f) wt_ptr[row_lo[j] + (e2 - row_ptr[j]) + 1]++;
        for (int i = 0; i < c->nNu; ++i) wt_ptr[i + 1] += wt_ptr[i];
        wt_j.resize(wt_ptr[c->nNu]); wt_w.resize(wt_ptr[c->nNu]);
        std::vector<int> fill(wt_ptr.begin(), wt_ptr.end() - 1);
        for (int j = 0; j < J; ++j)
            for (int e2 = row_ptr[j]; e2 < row_ptr[j + 1]; ++e2)
                if (Wh[e2] != 0.0f) {
                    const int i = row_lo[j] + (e2 - row_ptr[j]);
                    wt_j[fill[i]] = j; wt_w[fill[i]] = Wh[e2]; fill[i]++;
                }
        CU_TRY(c, upload(c->d_wt_ptr, wt_ptr, c->stream));
        CU_TRY(c, upload(c->d_wt_j, wt_j, c->stream));
        CU_TRY(c, upload(c->d_wt_w, wt_w, c->stream));
    }

    if (obs) {
        std::vector<double> o(obs, obs + J), i2v(J);
        double cst = 0.0;
        for (int j = 0; j < J; ++j) {
            i2v[j] = 1.0 / (2.0 * err[j] * err[j]);
            cst += -0.5 * std::log(2.0 * kPi * err[j] * err[j]);
        }
        c->logl_const = cst;
        CU_TRY(c, upload(c->d_obs, o, c->stream));
        CU_TRY(c, upload(c->d_inv2var, i2v, c->stream));
        std::vector<double> var(J);
        for (int j = 0; j < J; ++j) var[j] = err[j] * err[j];
        CU_TRY(c, upload(c->d_var, var, c->stream));
        c->have_data = true;
    }
    c->have_obs = true;
    c->cap_B = 0;    // staging buffers depend on J
    return HELIOS_OK;
}

// Automatic choice of the level-parallel kernel: measured crossovers with the staged kernel (profiles/r02_batch_sweep.md)
// are B = 8..16 at configs[1] (133 tiles) and configs[2] (255 tiles), B = 4..8 at configs[3] (1329 tiles): the staged
// kernel's time is flat up to there (its warps walk all levels in sequence), the level-parallel kernel's grows with
// B x tiles.
constexpr int kSegAutoMaxBatch = 8;
constexpr long long kSegAutoMaxCtas = 6000;
constexpr int kObsSmallBatchCtas = 592;     // 4 CTAs of 8 warps per SM on 148 SMs

static SlabPlan plan_slab(const helios_ctx* c, int B) {
    SlabPlan none;
    if (c->opt_kernel == 1 || !c->have_tmaps) return none;
    // models per CTA (measured on B200, configs 1-3): 24 warps hide latency best while the state fits
    // 72 registers (<= 4 angles) and the batch fills 24-model groups; 16 otherwise; 8 for B < 16
    int nw = c->opt_models_per_cta;
    if (nw == 0) {
        if (B < 16) nw = 8;
        else {      // padded model slots, weighted by the measured per-model efficiency of the variants (27 warps: +1.8 %
                    // at configs[3] when its groups fill up; its 72-register budget only pays with many angles)
            const double cost24 = (double)((B + 23) / 24 * 24), cost16 = (double)((B + 15) / 16 * 16) / 0.92;
            const double cost27 = c->A >= 6 ? (double)((B + 26) / 27 * 27) / 1.018 : 1e30;
            nw = cost24 <= cost16 ? 24 : 16;
            if (cost27 < std::min(cost24, cost16)) {
                const SlabPlan p27 = slab_plan(c->S, c->C, c->nT, c->A, c->S > 0 ? c->n_loads : 0, 27, c->smem_optin, c->smem_sm);
                if (p27.ok && p27.ring >= 3) nw = 27;
            }
        }
    }
    return slab_plan(c->S, c->C, c->nT, c->A, c->S > 0 ? c->n_loads : 0, nw, c->smem_optin, c->smem_sm);
}

int helios_reserve(helios_ctx* c, int B) {
    if (!c) return HELIOS_EINVAL;
    if (!c->have_tables || !c->have_atmo) return fail(c, HELIOS_ESTATE, "reserve: tables and atmosphere must be set first");
    if (B < 1 || B > 65535) return fail(c, HELIOS_EINVAL, "batch %d out of range (1..65535)", B);
    if (B <= c->cap_B) return HELIOS_OK;
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    dfree(c->d_rec); dfree(c->d_flux); dfree(c->d_scale); dfree(c->d_flag); dfree(c->d_model_x);
    dfree(c->d_obs_partial); dfree(c->d_obs_arrived);
    dfree(c->d_params_stage); dfree(c->d_spectra_stage); dfree(c->d_logl_stage); dfree(c->d_addvar);
    dfree(c->d_acc); dfree(c->d_q);
    graphs_invalidate(c);          // the captured calls point into the old workspace
    c->cap_B = 0;
    const int rf = std::max(direct_rec_floats(c->S, c->C), kSlabRecFloats);
    c->flux_stride = c->stride;
    CU_TRY(c, cudaMalloc(&c->d_rec, sizeof(float) * (size_t)B * c->L * rf));
    CU_TRY(c, cudaMalloc(&c->d_flux, sizeof(float) * (size_t)B * c->flux_stride));
    CU_TRY(c, cudaMalloc(&c->d_scale, sizeof(float) * B));
    CU_TRY(c, cudaMalloc(&c->d_flag, sizeof(int) * B));
    CU_TRY(c, cudaMalloc(&c->d_model_x, sizeof(float) * (size_t)B * slab_x_floats(c->S, c->C)));
    {
        const int n_chunks = ((c->J > 0 ? c->J : 1) + 7) / 8;       // the finer of the two chunkings of k_obs_apply
        CU_TRY(c, cudaMalloc(&c->d_obs_partial, sizeof(double) * (size_t)B * n_chunks));
        CU_TRY(c, cudaMalloc(&c->d_obs_arrived, sizeof(unsigned) * B));
        CU_TRY(c, cudaMemsetAsync(c->d_obs_arrived, 0, sizeof(unsigned) * B, c->stream));
    }
    CU_TRY(c, cudaMalloc(&c->d_params_stage, sizeof(double) * (size_t)B * n_params(c)));
    CU_TRY(c, cudaMalloc(&c->d_addvar, sizeof(double) * B));
    CU_TRY(c, cudaMalloc(&c->d_spectra_stage, sizeof(float) * (size_t)B * (c->J > 0 ? c->J : 1)));
    CU_TRY(c, cudaMalloc(&c->d_logl_stage, sizeof(double) * B));
    CU_TRY(c, cudaMalloc(&c->d_acc, sizeof(unsigned long long) * (size_t)B * (c->J > 0 ? c->J : 1)));
    CU_TRY(c, cudaMalloc(&c->d_q, sizeof(float) * (size_t)B * (c->J > 0 ? c->J : 1)));
    c->cap_B = B;
    return HELIOS_OK;
}

static inline void stamp(helios_ctx* c, int which) {
    if (c->opt_timing) cudaEventRecord(c->ev[c->timed_calls % helios_ctx::kTimingRing][which], c->stream);
}

// steps 0-4: params -> flux (DEVICE [B][flux_stride])
// fused: in/out -- on entry, the caller wants the observation operator applied in the RT kernel's epilogue (obs.cuh);
// on return, whether the kernel that ran did (the direct fallback kernel does not, it writes the flux)
static int run_flux(helios_ctx* c, int B, const double* params, float* flux, long long flux_stride, int unit_scale = 0,
                    bool* fused = nullptr) {
    const SlabPlan plan = plan_slab(c, B);
    if (c->opt_kernel == 2 && !plan.ok)
        return fail(c, HELIOS_EINVAL, "staged kernel requested but unavailable for this table shape (shared memory / TMA)");
    // level-parallel kernel: small batches (measured crossover, profiles/r02_batch_sweep.md), or on request
    const SegPlan seg = (c->have_seg_maps && (c->opt_kernel == 3 || (c->opt_kernel == 0 && B <= kSegAutoMaxBatch &&
                                                                  (long long)B * ((c->nNu + kSlabTile - 1) / kSlabTile) <= kSegAutoMaxCtas)))
                            ? seg_plan(c->L, c->A, c->S, c->C, slab_x_floats(c->S, c->C), c->smem_optin) : SegPlan{};
    if (c->opt_kernel == 3 && !seg.ok)
        return fail(c, HELIOS_EINVAL, "level-parallel kernel requested but unavailable for %d levels", c->L);
    const int slab = (plan.ok || seg.ok) ? 1 : 0;      // both use the staged-kernel records
    const int rf = slab ? kSlabRecFloats : direct_rec_floats(c->S, c->C);
    PrepArgs pa{};
    pa.params = params; pa.B = B; pa.P = n_params(c); pa.K = c->K; pa.S = c->S; pa.C = c->C; pa.L = c->L;
    pa.nT = c->nT; pa.nP = c->nP; pa.T_grid = c->d_Tgrid; pa.lvl_p_bar = c->d_lvl_p; pa.lvl_elem = c->d_lvl_elem;
    pa.lvl_lw = c->d_lvl_lw; pa.tp_order = c->tp_order; pa.tp_ratio = c->tp_ratio; pa.NT = c->NT; pa.extras = c->extras;
    pa.unit_scale = unit_scale; pa.model_addvar = c->d_addvar; pa.lvl_ip = c->d_lvl_ip; pa.lvl_u = c->d_lvl_u; pa.lvl_pclamp = c->d_lvl_pclamp;
    pa.lvl_lnratio = c->d_lvl_lnratio; pa.mmw = c->mmw; pa.he_to_h2 = c->he_to_h2; pa.flux_const = c->flux_const;
    pa.rec = c->d_rec; pa.rec_floats = rf; pa.slab_layout = slab; pa.model_scale = c->d_scale; pa.model_flag = c->d_flag;
    pa.model_x = c->d_model_x; pa.x_floats = slab_x_floats(c->S, c->C);
    pa.counters = c->d_counters;
    const bool fuse = fused && *fused && slab && c->have_obs;
    if (fused) *fused = fuse;
    FusedObs fo{};
    if (fuse) {
        fo.acc = c->d_acc; fo.q = c->d_q; fo.wt_ptr = c->d_wt_ptr; fo.wt_j = c->d_wt_j; fo.wt_w = c->d_wt_w; fo.J = c->J;
        pa.fused_acc = c->d_acc; pa.fused_q = c->d_q; pa.J = c->J; pa.row_ptr = c->d_row_ptr; pa.row_lo = c->d_row_lo;
        pa.nu0 = c->nu0; pa.dnu = c->dnu;
    }
    // programmatic dependent launch of the RT and observation kernels (common.cuh); not with stage timing, whose
    // events between the kernels serialise them
    const bool pdl = !c->opt_timing;
    stamp(c, 0);
    k_prep<<<B, kPrepThreads, 0, c->stream>>>(pa);
    c->n_launches += 1;
    CU_TRY(c, cudaGetLastError());
    stamp(c, 1);

    if (seg.ok) {
        SegArgs ga{};
        ga.sigma = c->d_sigma; ga.cia = c->d_cia; ga.stride = c->stride; ga.S = c->S; ga.C = c->C; ga.nT = c->nT; ga.nP = c->nP;
        ga.nNu = c->nNu; ga.L = c->L; ga.B = B; ga.rec = c->d_rec; ga.model_x = c->d_model_x; ga.x_floats = pa.x_floats;
        ga.model_scale = c->d_scale; ga.model_flag = c->d_flag; ga.lvl_ip = c->d_lvl_ip; ga.nu_index = c->d_nu_index; ga.nu0 = c->nu0; ga.dnu = c->dnu;
        ga.flux = flux; ga.flux_stride = flux_stride; ga.fused = fo; ga.n_chunks = seg.n_chunks; ga.chunk_len = seg.chunk_len;
        cudaError_t e = launch_rt_seg(c->A, c->seg_maps, ga, seg.smem, c->smem_optin, c->seg_smem, c->stream, pdl);
        if (e != cudaSuccess) return fail(c, HELIOS_ECUDA, "level-parallel kernel launch failed: %s", cudaGetErrorString(e));
        c->n_launches += 1;
        stamp(c, 2);
        return HELIOS_OK;
    }
    if (slab) {
        SlabArgs sa{};
        sa.S = c->S; sa.C = c->C; sa.nT = c->nT; sa.nNu = c->nNu; sa.L = c->L; sa.B = B;
        sa.rec = c->d_rec; sa.model_x = c->d_model_x; sa.x_floats = pa.x_floats;
        sa.model_scale = c->d_scale; sa.model_flag = c->d_flag; sa.nu0 = c->nu0; sa.dnu = c->dnu; sa.nu_index = c->d_nu_index;
        sa.flux = flux; sa.flux_stride = flux_stride; sa.fused = fo;
        sa.seg = c->d_seg + (size_t)(plan.ring - 1) * c->n_seg; sa.load_ip = c->d_load_ip;
        sa.n_seg = c->n_seg; sa.n_loads = c->n_loads; sa.ring = plan.ring; sa.ang = c->ang;
        cudaError_t e = launch_rt_slab(c->tm_sigma, c->tm_cia, sa, plan, c->slab_smem, c->stream, pdl);
        if (e != cudaSuccess) return fail(c, HELIOS_ECUDA, "staged kernel launch failed: %s", cudaGetErrorString(e));
        c->n_launches += 1;
        stamp(c, 2);
        return HELIOS_OK;
    }
    DirectArgs da{};
    da.sigma = c->d_sigma; da.cia = c->d_cia; da.S = c->S; da.C = c->C; da.nT = c->nT; da.nP = c->nP; da.nNu = c->nNu;
    da.L = c->L; da.stride = c->stride; da.nu_index = c->d_nu_index; da.rec = c->d_rec; da.rec_floats = rf; da.model_scale = c->d_scale;
    da.model_flag = c->d_flag; da.nu0 = c->nu0; da.dnu = c->dnu; da.flux = flux; da.flux_stride = flux_stride; da.ang = c->ang;
    const size_t smem = sizeof(float) * (size_t)c->L * rf;     // the direct kernel keeps one model's records in shared memory
    if (smem > c->smem_optin)
        return fail(c, HELIOS_EINVAL, "direct kernel: n_levels x record size (%zu B) exceeds the %zu B of shared memory a "
                    "block may use, and the staged kernel is unavailable for this table shape", smem, c->smem_optin);
    const dim3 grid((c->nNu + kDirectThreads - 1) / kDirectThreads, B);
#define HELIOS_DIRECT_CASE(N)                                                                               \
    case N:                                                                                                 \
        if (smem > 48 * 1024) CU_TRY(c, cudaFuncSetAttribute(k_rt_direct<N>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
        CU_TRY(c, launch_kernel(k_rt_direct<N>, grid, dim3(kDirectThreads), smem, c->stream, pdl, da));     \
        break;
    switch (c->A) {
        HELIOS_DIRECT_CASE(1) HELIOS_DIRECT_CASE(2) HELIOS_DIRECT_CASE(3) HELIOS_DIRECT_CASE(4)
        HELIOS_DIRECT_CASE(5) HELIOS_DIRECT_CASE(6) HELIOS_DIRECT_CASE(7) HELIOS_DIRECT_CASE(8)
        default: return fail(c, HELIOS_EINVAL, "n_angles %d", c->A);
    }
#undef HELIOS_DIRECT_CASE
    c->n_launches += 1;
    CU_TRY(c, cudaGetLastError());
    stamp(c, 2);
    return HELIOS_OK;
}

static int check_ready(helios_ctx* c, int B, int P, const double* params, bool need_obs, bool need_data) {
    if (!c) return HELIOS_EINVAL;
    if (!c->have_tables || !c->have_atmo) return fail(c, HELIOS_ESTATE, "tables and atmosphere must be set first");
    if (need_obs && !c->have_obs) return fail(c, HELIOS_ESTATE, "observation grid not set (helios_set_observation)");
    if (need_data && !c->have_data) return fail(c, HELIOS_ESTATE, "logL requested but the observation has no data");
    if (B < 1 || B > 65535) return fail(c, HELIOS_EINVAL, "batch %d out of range (1..65535)", B);
    if (!params) return fail(c, HELIOS_EINVAL, "params is NULL");
    if (P != n_params(c))
        return fail(c, HELIOS_EINVAL, "n_params %d does not match this context's parameter vector (2 + %d temperature "
                    "parameters + %d species + %d extras = %d)", P, c->NT, c->S, c->n_extra, n_params(c));
    return HELIOS_OK;
}

int helios_forward_highres(helios_ctx* c, int B, int P, const double* params, float* flux_out) {
    int rc = check_ready(c, B, P, params, false, false);
    if (rc) return rc;
    if (!flux_out) return fail(c, HELIOS_EINVAL, "flux_out is NULL");
    CU_TRY(c, cudaSetDevice(c->device));
    if ((rc = helios_reserve(c, B))) return rc;
    c->n_models += B;
    rc = run_flux(c, B, params, flux_out, c->nNu);
    if (c->opt_timing) { c->ev_has_obs[c->timed_calls % helios_ctx::kTimingRing] = false; c->timed_calls++; }
    return rc;
}

static int forward_batch_enqueue(helios_ctx* c, int B, int P, const double* params, float* spectra_out, double* logl_out) {
    int rc = check_ready(c, B, P, params, true, logl_out != nullptr);
    if (rc) return rc;
    if (!spectra_out && !logl_out) return fail(c, HELIOS_EINVAL, "both outputs are NULL");
    CU_TRY(c, cudaSetDevice(c->device));
    if ((rc = helios_reserve(c, B))) return rc;
    c->n_models += B;
    bool fused = c->opt_fused != 0;
    if ((rc = run_flux(c, B, params, c->d_flux, c->flux_stride, 0, &fused))) return rc;
    ObsApplyArgs oa{};
    oa.J = c->J; oa.row_ptr = c->d_row_ptr; oa.row_lo = c->d_row_lo; oa.W = c->d_W; oa.flux = c->d_flux;
    oa.flux_stride = c->flux_stride; oa.model_flag = c->d_flag; oa.obs = c->d_obs; oa.inv2var = c->d_inv2var;
    if (c->extras & HELIOS_EXTRA_ERROR_INFLATION) { oa.var = c->d_var; oa.addvar = c->d_addvar; }
    oa.logl_const = c->logl_const; oa.spectra = spectra_out; oa.logl = logl_out;
    oa.partial = c->d_obs_partial; oa.arrived = c->d_obs_arrived;
    // one bin per warp while 64-bin CTAs would leave SMs idle (the choice depends on B only through this threshold;
    // kObsSmallBatchCtas is fixed, so a given (B, J) always takes the same variant)
    const bool pdl = !c->opt_timing;
    if (fused) {
        FusedObs fo{c->d_acc, c->d_q, c->d_wt_ptr, c->d_wt_j, c->d_wt_w, c->J};
        CU_TRY(c, launch_kernel(k_obs_final, dim3(B), dim3(kObsThreads), 0, c->stream, pdl, oa, fo));
    } else if ((long long)B * ((c->J + kObsBinsPerCta - 1) / kObsBinsPerCta) < kObsSmallBatchCtas)
        CU_TRY(c, launch_kernel(k_obs_apply<1>, dim3((c->J + 7) / 8, B), dim3(kObsThreads), 0, c->stream, pdl, oa));
    else
        CU_TRY(c, launch_kernel(k_obs_apply<8>, dim3((c->J + kObsBinsPerCta - 1) / kObsBinsPerCta, B), dim3(kObsThreads), 0,
                                c->stream, pdl, oa));
    c->n_launches += 1;
    stamp(c, 3);
    if (c->opt_timing) { c->ev_has_obs[c->timed_calls % helios_ctx::kTimingRing] = true; c->timed_calls++; }
    return HELIOS_OK;
}

int helios_forward_batch(helios_ctx* c, int B, int P, const double* params, float* spectra_out, double* logl_out) {
    if (!c) return HELIOS_EINVAL;
    if (!c->opt_graphs || !c->graphs_ok || c->opt_timing) return forward_batch_enqueue(c, B, P, params, spectra_out, logl_out);
    using Entry = helios_ctx::GraphEntry;
    auto same = [&](const Entry& g) { return g.epoch == c->epoch && g.B == B && g.P == P && g.params == params &&
                                             g.spectra == spectra_out && g.logl == logl_out; };
    ++c->graph_clock;
    const bool state_ok = c->have_tables && c->have_atmo && c->have_obs && (!logl_out || c->have_data) && B <= c->cap_B;
    for (auto& g : c->graphs)
        if (state_ok && g.exec && same(g)) {        // replay: one launch for the three kernels
            CU_TRY(c, cudaSetDevice(c->device));
            CU_TRY(c, cudaGraphLaunch(g.exec, c->stream));
            g.last_use = c->graph_clock;
            c->n_models += B; c->n_launches += 3; c->n_graph_replays += 1;
            return HELIOS_OK;
        }
    if (!same(c->graph_seen) || B > c->cap_B) {     // first time: plain launches (this also sizes the workspace and
        int rc = forward_batch_enqueue(c, B, P, params, spectra_out, logl_out);      // sets the kernels' attributes)
        if (rc == HELIOS_OK) { c->graph_seen = Entry{}; c->graph_seen.B = B; c->graph_seen.P = P; c->graph_seen.params = params;
                               c->graph_seen.spectra = spectra_out; c->graph_seen.logl = logl_out;
                               c->graph_seen.epoch = c->epoch; }      // after the call: helios_reserve may have bumped it
        return rc;
    }
    // second time with the same arguments: capture the call on a private stream (the context's stream may be the
    // legacy default stream, which cannot be captured), instantiate, and launch the graph on the context's stream
    CU_TRY(c, cudaSetDevice(c->device));
    if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); c->graphs_ok = false;
        return forward_batch_enqueue(c, B, P, params, spectra_out, logl_out);
    }
    cudaStream_t user = c->stream;
    const unsigned long long models0 = c->n_models, launches0 = c->n_launches;
    cudaGraph_t graph = nullptr; cudaGraphExec_t exec = nullptr;
    int rc = HELIOS_OK;
    cudaError_t e = cudaStreamBeginCapture(c->cap_stream, cudaStreamCaptureModeRelaxed);
    if (e == cudaSuccess) {
        c->stream = c->cap_stream;
        rc = forward_batch_enqueue(c, B, P, params, spectra_out, logl_out);
        c->stream = user;
        e = cudaStreamEndCapture(c->cap_stream, &graph);
    }
    if (e == cudaSuccess && rc == HELIOS_OK && graph) e = cudaGraphInstantiate(&exec, graph, 0);
    if (graph) cudaGraphDestroy(graph);
    if (e != cudaSuccess || rc != HELIOS_OK || !exec) {          // no graphs on this context from now on; run the call plainly
        cudaGetLastError();
        if (exec) cudaGraphExecDestroy(exec);
        c->graphs_ok = false;
        c->n_models = models0; c->n_launches = launches0;
        return forward_batch_enqueue(c, B, P, params, spectra_out, logl_out);
    }
    Entry* slot = &c->graphs[0];
    for (auto& g : c->graphs) { if (!g.exec) { slot = &g; break; } if (g.last_use < slot->last_use) slot = &g; }
    if (slot->exec) cudaGraphExecDestroy(slot->exec);
    *slot = c->graph_seen; slot->exec = exec; slot->last_use = c->graph_clock;
    c->graph_seen = Entry{};
    CU_TRY(c, cudaGraphLaunch(exec, user));                       // the counters were advanced by the captured enqueue
    c->n_graph_replays += 1;
    return HELIOS_OK;
}

int helios_loglike_batch(helios_ctx* c, int B, int P, const double* params, double* logl_out) {
    if (c && !logl_out) return fail(c, HELIOS_EINVAL, "logl_out is NULL");
    return helios_forward_batch(c, B, P, params, nullptr, logl_out);
}

int helios_set_tp_elements(helios_ctx* c, int n_elements, int order, int ratio_form) {
    if (!c) return HELIOS_EINVAL;
    if (!c->have_atmo) return fail(c, HELIOS_ESTATE, "set_tp_elements: call helios_set_atmosphere first");
    if (n_elements < 1 || n_elements > 16 || order < 1 || order > 4)
        return fail(c, HELIOS_EINVAL, "set_tp_elements: n_elements %d (1..16), order %d (1..4)", n_elements, order);
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    graphs_invalidate(c);
    c->tp_order = order; c->tp_ratio = ratio_form ? 1 : 0; c->NT = n_elements * order + 1;
    CU_TRY(c, build_tp(c, n_elements, order));
    c->cap_B = 0;    // the parameter staging buffer depends on P
    return HELIOS_OK;
}

int helios_set_extras(helios_ctx* c, unsigned flags) {
    if (!c) return HELIOS_EINVAL;
    if (flags & ~(HELIOS_EXTRA_DISTANCE | HELIOS_EXTRA_ERROR_INFLATION | HELIOS_EXTRA_GREY_CLOUD))
        return fail(c, HELIOS_EINVAL, "set_extras: unknown flag in 0x%x", flags);
    graphs_invalidate(c);
    c->extras = flags;
    c->n_extra = ((flags & HELIOS_EXTRA_DISTANCE) ? 1 : 0) + ((flags & HELIOS_EXTRA_ERROR_INFLATION) ? 1 : 0) +
                 ((flags & HELIOS_EXTRA_GREY_CLOUD) ? 3 : 0);
    c->cap_B = 0;
    return HELIOS_OK;
}

int helios_get_n_params(const helios_ctx* c, int* out) {
    if (!c || !out || !c->have_atmo) return HELIOS_EINVAL;
    *out = n_params(c);
    return HELIOS_OK;
}

int helios_teff_batch(helios_ctx* c, int B, int P, const double* params, double nu_a, double nu_b, double* teff_out) {
    int rc = check_ready(c, B, P, params, false, false);
    if (rc) return rc;
    if (!teff_out) return fail(c, HELIOS_EINVAL, "teff_out is NULL");
    const double nu_first = c->nu0, nu_last = c->nu0 + c->dnu * (c->nNu - 1);
    if (!(nu_b > nu_a) || nu_a < nu_first - 1e-9 * c->dnu || nu_b > nu_last + 1e-9 * c->dnu)
        return fail(c, HELIOS_EINVAL, "teff: window [%g, %g] outside the grid [%g, %g]", nu_a, nu_b, nu_first, nu_last);
    CU_TRY(c, cudaSetDevice(c->device));
    if ((rc = helios_reserve(c, B))) return rc;
    c->n_models += B;
    if ((rc = run_flux(c, B, params, c->d_flux, c->flux_stride, /*unit_scale=*/1))) return rc;
    TeffArgs ta{c->nNu, c->nu0, c->dnu, std::fmax(nu_a, nu_first), std::fmin(nu_b, nu_last), c->d_flux, c->flux_stride,
                c->d_flag, teff_out};
    k_teff<<<B, 256, 0, c->stream>>>(ta);
    c->n_launches += 1;
    CU_TRY(c, cudaGetLastError());
    if (c->opt_timing) { c->ev_has_obs[c->timed_calls % helios_ctx::kTimingRing] = false; c->timed_calls++; }
    return HELIOS_OK;
}

int helios_forward_batch_host(helios_ctx* c, int B, int P_in, const double* params_host, float* spectra_host, double* logl_host) {
    int rc = check_ready(c, B, P_in, params_host, true, logl_host != nullptr);
    if (rc) return rc;
    if (!spectra_host && !logl_host) return fail(c, HELIOS_EINVAL, "both outputs are NULL");
    CU_TRY(c, cudaSetDevice(c->device));
    if ((rc = helios_reserve(c, B))) return rc;
    const size_t P = n_params(c);
    CU_TRY(c, cudaMemcpyAsync(c->d_params_stage, params_host, sizeof(double) * B * P, cudaMemcpyHostToDevice, c->stream));
    rc = helios_forward_batch(c, B, P_in, c->d_params_stage, spectra_host ? c->d_spectra_stage : nullptr,
                              logl_host ? c->d_logl_stage : nullptr);
    if (rc) return rc;
    if (spectra_host)
        CU_TRY(c, cudaMemcpyAsync(spectra_host, c->d_spectra_stage, sizeof(float) * (size_t)B * c->J, cudaMemcpyDeviceToHost, c->stream));
    if (logl_host)
        CU_TRY(c, cudaMemcpyAsync(logl_host, c->d_logl_stage, sizeof(double) * B, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return HELIOS_OK;
}

int helios_teff_batch_host(helios_ctx* c, int B, int P_in, const double* params_host, double nu_a, double nu_b,
                           double* teff_host) {
    int rc = check_ready(c, B, P_in, params_host, false, false);
    if (rc) return rc;
    if (!teff_host) return fail(c, HELIOS_EINVAL, "teff_out is NULL");
    CU_TRY(c, cudaSetDevice(c->device));
    if ((rc = helios_reserve(c, B))) return rc;
    CU_TRY(c, cudaMemcpyAsync(c->d_params_stage, params_host, sizeof(double) * B * (size_t)P_in, cudaMemcpyHostToDevice, c->stream));
    if ((rc = helios_teff_batch(c, B, P_in, c->d_params_stage, nu_a, nu_b, c->d_logl_stage))) return rc;
    CU_TRY(c, cudaMemcpyAsync(teff_host, c->d_logl_stage, sizeof(double) * B, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    return HELIOS_OK;
}

int helios_get_stage_ms(helios_ctx* c, double* stage_ms, int* n_calls) {
    if (!c || !stage_ms || !n_calls) return HELIOS_EINVAL;
    CU_TRY(c, cudaSetDevice(c->device));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    const int n = (int)std::min<long long>(c->timed_calls, helios_ctx::kTimingRing);
    double acc[3] = {0, 0, 0};
    int n_obs = 0;
    for (int i = 0; i < n; ++i) {
        float ms = 0;
        CU_TRY(c, cudaEventElapsedTime(&ms, c->ev[i][0], c->ev[i][1])); acc[0] += ms;
        CU_TRY(c, cudaEventElapsedTime(&ms, c->ev[i][1], c->ev[i][2])); acc[1] += ms;
        if (c->ev_has_obs[i]) { CU_TRY(c, cudaEventElapsedTime(&ms, c->ev[i][2], c->ev[i][3])); acc[2] += ms; ++n_obs; }
    }
    stage_ms[0] = n ? acc[0] / n : 0; stage_ms[1] = n ? acc[1] / n : 0; stage_ms[2] = n_obs ? acc[2] / n_obs : 0;
    *n_calls = n;
    return HELIOS_OK;
}

int helios_measure_peaks(helios_ctx* c, helios_peaks* out) {
    if (!c || !out) return HELIOS_EINVAL;
    CU_TRY(c, cudaSetDevice(c->device));
    float* d_out = nullptr; PeakTimes* d_times = nullptr;
    CU_TRY(c, cudaMalloc(&d_out, sizeof(float) * (size_t)c->num_sms * kPeakThreads));
    if (cudaMalloc(&d_times, sizeof(PeakTimes)) != cudaSuccess) { cudaFree(d_out); return fail(c, HELIOS_ENOMEM, "measure_peaks: out of memory"); }
    double cyc[kPeakModes] = {}, ops[kPeakModes] = {}, mhz[kPeakModes] = {};
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    int rc = HELIOS_OK;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) rc = fail(c, HELIOS_ECUDA, "measure_peaks: cudaEventCreate failed");
    if (!rc) rc = run_peak<kPeakFfma>(c, d_out, d_times, e0, e1, &cyc[0], &ops[0], &mhz[0]);
    if (!rc) rc = run_peak<kPeakFfma2Scalar>(c, d_out, d_times, e0, e1, &cyc[1], &ops[1], &mhz[1]);
    if (!rc) rc = run_peak<kPeakFfma2TwoPairs>(c, d_out, d_times, e0, e1, &cyc[2], &ops[2], &mhz[2]);
    if (!rc) rc = run_peak<kPeakFfma2ThreePairs>(c, d_out, d_times, e0, e1, &cyc[3], &ops[3], &mhz[3]);
    if (!rc) rc = run_peak<kPeakMufuEx2>(c, d_out, d_times, e0, e1, &cyc[4], &ops[4], &mhz[4]);
    if (!rc) rc = run_peak<kPeakFfma2PlusAlu>(c, d_out, d_times, e0, e1, &cyc[5], &ops[5], &mhz[5]);
    if (!rc) rc = run_peak<kPeakFfma2PlusFsel>(c, d_out, d_times, e0, e1, &cyc[6], &ops[6], &mhz[6]);
    if (!rc) rc = run_peak<kPeakFfma3Reg>(c, d_out, d_times, e0, e1, &cyc[7], &ops[7], &mhz[7]);
    if (!rc) rc = run_peak<kPeakFfma2PlusMufu>(c, d_out, d_times, e0, e1, &cyc[8], &ops[8], &mhz[8]);
    cudaFree(d_out); cudaFree(d_times);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    if (rc) return rc;
    out->n_sms = c->num_sms;
    out->sm_clock_mhz = mhz[1];
    out->ffma_per_clk_sm = ops[0];
    out->ffma2_per_clk_sm = 2.0 * ops[1];
    out->mufu_per_clk_sm = ops[4];
    for (int i = 0; i < 3; ++i) out->ffma2_cycles[i] = cyc[1 + i];
    out->alu_extra_cycles = cyc[5] - cyc[1];       // modes 5 and 6 count one FFMA2 + one extra op (pair) per "instruction"
    out->fsel_extra_cycles = cyc[6] - cyc[1];
    out->ffma_3reg_cycles = cyc[7];
    out->mufu_extra_cycles = cyc[8] - cyc[1];
    return HELIOS_OK;
}

int helios_get_stats(helios_ctx* c, helios_stats* out, int reset) {
    if (!c || !out) return HELIOS_EINVAL;
    CU_TRY(c, cudaSetDevice(c->device));
    unsigned long long h[2] = {0, 0};
    CU_TRY(c, cudaMemcpyAsync(h, c->d_counters, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CU_TRY(c, cudaStreamSynchronize(c->stream));
    out->n_clamped = h[0]; out->n_nonfinite = h[1]; out->n_models = c->n_models; out->n_launches = c->n_launches;
    out->n_graph_launches = c->n_graph_replays;
    if (reset) {
        CU_TRY(c, cudaMemsetAsync(c->d_counters, 0, sizeof h, c->stream));
        c->n_models = 0; c->n_launches = 0; c->n_graph_replays = 0;
    }
    return HELIOS_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------------------
// helios_observe_noalloc (include/helios.h): step 5 of the hot path for callers that may not allocate device memory.
//
// Who that is: code that runs where cudaMalloc / cudaFree are forbidden or unaffordable -- a sampler callback inside a
// region another library is capturing into a CUDA graph (an allocation there aborts the capture), a process whose
// memory pool was handed out in full at start-up (nothing is left for the driver to give), a latency-critical loop
// that cannot take the device-wide synchronisation a cudaFree implies.  Every other batch entry point of this library
// grows its workspace through helios_reserve(), i.e. through cudaMalloc.
//
// k_obs_apply needs scratch memory beyond its inputs and outputs: one chi-square partial sum per (model, group of 8
// bins) and one arrival counter per model, used to let the LAST block of a model add the partial sums in a fixed order.
// The variant below, k_obs_apply_static, is the same kernel with that scratch taken from g_obs_static_scratch, an
// array that is part of the library image: the CUDA runtime places it in the memory of every GPU the library's
// module is loaded on, at load time, and it stays there until the process exits (about 0.5 MB per GPU).
//
// g_obs_static_scratch is a DEVICE variable.  Inside device code its name is the array.  In host code the same name
// is only a handle the runtime uses to look the variable up -- it is not the address the GPU sees, and a kernel that
// was handed it would fault or, on systems where the GPU can reach host memory, quietly work on the wrong bytes.
// Host code therefore asks the runtime for the device address, once per GPU, with that GPU current
// (static_scratch_address), and passes that pointer to the kernel.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kStaticMaxBatch = 4096;             // models per call
constexpr int kStaticMaxGroups = 65536;           // B * ceil(n_bins / 8) per call
constexpr size_t kStaticPartialBytes = sizeof(double) * (size_t)kStaticMaxGroups;
constexpr size_t kStaticScratchBytes = kStaticPartialBytes + sizeof(unsigned) * (size_t)kStaticMaxBatch;
constexpr int kStaticMaxDevices = 64;

static __device__ __align__(256) unsigned char g_obs_static_scratch[kStaticScratchBytes];

static std::mutex g_static_mutex;
static unsigned char* g_static_ptr[kStaticMaxDevices] = {};     // device address of the array on each GPU, once looked up

// Device address of g_obs_static_scratch on GPU `device`, which must be the current device.  The first call per GPU
// asks the runtime (this may load the library's module on that GPU, so it should not happen during a stream capture);
// later calls return the remembered pointer.
static cudaError_t static_scratch_address(int device, unsigned char** out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[device]) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, g_obs_static_scratch);
        if (e != cudaSuccess) return e;
        g_static_ptr[device] = (unsigned char*)p;
    }
    *out = g_static_ptr[device];
    return cudaSuccess;
}

// k_obs_apply<8> with its workspace in the static array: one block per (model, 64 bins), a warp owns 8 bins, lanes
// stride a bin's band of W, shuffle tree, fp64 chi-square term per bin, group sums to `partial`, the block that
// arrives last at a model adds the groups in the fixed order of k_obs_apply -- so on the same flux the binned
// spectrum and logL are bitwise those of the allocating path.  Differences: the flux comes from the caller, so there
// are no model flags (a non-finite flux gives NaN bins and logL = -inf), and the arrival counters are cleared by the
// host before every launch instead of by the kernel after it.
__global__ void __launch_bounds__(kObsThreads) k_obs_apply_static(ObsApplyArgs a, unsigned char* scratch) {
    __shared__ double tree[kObsThreads];
    __shared__ unsigned ticket;
    double* partial = reinterpret_cast<double*>(scratch);
    unsigned* arrived = reinterpret_cast<unsigned*>(scratch + kStaticPartialBytes);
    const int b = blockIdx.y, chunk = blockIdx.x, n_chunks = gridDim.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const float* F = a.flux + (size_t)b * a.flux_stride;
    double chi2 = 0.0;
    const int j0 = chunk * kObsBinsPerCta + warp * 8;
#pragma unroll 2
    for (int j = j0; j < min(j0 + 8, a.J); ++j) {
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
            if (a.spectra) a.spectra[(size_t)b * a.J + j] = acc;
            if (a.logl) {
                const double r = a.obs[j] - (double)acc;
                chi2 = __dadd_rn(chi2, __dmul_rn(__dmul_rn(r, r), a.inv2var[j]));
            }
        }
    }
    if (!a.logl) return;
    const int n_groups = (a.J + 7) / 8;
    const int g = chunk * (kObsThreads / 32) + warp;
    if (lane == 0 && g < n_groups) partial[(size_t)b * n_groups + g] = chi2;
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        ticket = atomicAdd(&arrived[b], 1u);
    }
    __syncthreads();
    if (ticket != (unsigned)n_chunks - 1) return;
    __threadfence();
    double t = 0.0;
    for (int c = threadIdx.x; c < n_groups; c += kObsThreads) t += __ldcg(&partial[(size_t)b * n_groups + c]);
    tree[threadIdx.x] = t;
    __syncthreads();
#pragma unroll
    for (int o = kObsThreads / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o) tree[threadIdx.x] += tree[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) a.logl[b] = tree[0] == tree[0] ? a.logl_const - tree[0] : -CUDART_INF;
}

extern "C" int helios_observe_noalloc(helios_ctx* c, int B, const float* flux, float* spectra_out, double* logl_out) {
    if (!c) return HELIOS_EINVAL;
    if (!c->have_obs) return fail(c, HELIOS_ESTATE, "observe_noalloc: observation grid not set (helios_set_observation)");
    if (logl_out && !c->have_data) return fail(c, HELIOS_ESTATE, "observe_noalloc: logL requested but the observation has no data");
    if (c->extras & HELIOS_EXTRA_ERROR_INFLATION)
        return fail(c, HELIOS_ESTATE, "observe_noalloc: error inflation takes its variance term from the parameter vector, "
                    "which this entry point does not see; use helios_forward_batch");
    if (!flux) return fail(c, HELIOS_EINVAL, "observe_noalloc: flux is NULL");
    if (!spectra_out && !logl_out) return fail(c, HELIOS_EINVAL, "observe_noalloc: both outputs are NULL");
    const int n_groups = (c->J + 7) / 8;
    if (B < 1 || B > kStaticMaxBatch || (long long)B * n_groups > kStaticMaxGroups)
        return fail(c, HELIOS_EINVAL, "observe_noalloc: batch %d with %d bins exceeds the static scratch array (at most %d models "
                    "and %d = batch x ceil(n_bins / 8) partial sums per call); split the batch or use helios_forward_batch",
                    B, c->J, kStaticMaxBatch, kStaticMaxGroups);
    if (c->device < 0 || c->device >= kStaticMaxDevices)
        return fail(c, HELIOS_EINVAL, "observe_noalloc: device ordinal %d beyond the %d this entry point keeps an address for",
                    c->device, kStaticMaxDevices);
    CU_TRY(c, cudaSetDevice(c->device));
    unsigned char* scratch = nullptr;
    CU_TRY(c, static_scratch_address(c->device, &scratch));
    // the array still holds what the previous call (of any context on this GPU) left: the counters must start at zero;
    // the partial sums need no clearing, every one a model reads was written by this launch first
    CU_TRY(c, cudaMemsetAsync(scratch + kStaticPartialBytes, 0, sizeof(unsigned) * (size_t)B, c->stream));
    ObsApplyArgs oa{};
    oa.J = c->J; oa.row_ptr = c->d_row_ptr; oa.row_lo = c->d_row_lo; oa.W = c->d_W; oa.flux = flux; oa.flux_stride = c->nNu;
    oa.obs = c->d_obs; oa.inv2var = c->d_inv2var; oa.logl_const = c->logl_const; oa.spectra = spectra_out; oa.logl = logl_out;
    k_obs_apply_static<<<dim3((c->J + kObsBinsPerCta - 1) / kObsBinsPerCta, B), kObsThreads, 0, c->stream>>>(oa, scratch);
    CU_TRY(c, cudaGetLastError());
    c->n_launches += 1;
    return HELIOS_OK;
}
