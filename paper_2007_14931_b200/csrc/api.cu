// api.cu — the C ABI of include/amp.h: argument checking, device-state ownership, the lineshape column
// pool (which columns are already held, which must be recomputed), the choice of normalisation path and
// the launch sequence of one NLL evaluation.  All per-event arithmetic is in the kernels.
#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <new>
#include <string>
#include <vector>

#include "amp_internal.cuh"

using namespace amp;

namespace {

// values of amp_model::colidx below zero.  The plan builders of the tensor-core paths use -2 for "lineshape == 1" in THEIR entry
// lists, so the in-register marker must not be -2: a point whose columns are not held has to be refused there, not read as 1.
enum { COL_NONE = -1, COL_INLINE = -3 };

struct PoolEntry {
    int r = -1;
    double mass = 0, width = 0;
    bool valid_data = false, valid_norm = false;
    long long last_used = -1;
};

}  // namespace

struct amp_model {
    int device = 0;                // the device the model was created on and owns its memory on; every call runs there
    DecayConst dk{};
    std::vector<amp_resonance> res;
    int R = 0, K = 0;
    int slot0[AMP_MAX_RESONANCES]{};
    bool has_z = false;

    Dataset data, norm;
    std::vector<PoolEntry> pool;   // same slot numbering in data.cols and norm.cols
    int pool_cap = 0;

    // parameter points of the last amp_set_params
    int P = 0;
    std::vector<double> couplings;   // [P][K][2]
    std::vector<double> mw;          // [P][R][2]
    std::vector<int> colidx;         // [P][R] pool slot >= 0, or COL_NONE (constant term: no lineshape) / COL_INLINE (evaluated in registers, no column held)
    int miss_streak[AMP_MAX_RESONANCES]{};
    bool was_inline[AMP_MAX_RESONANCES]{};   // evaluated in registers by the previous call
    long long call_id = 0;

    int norm_mode = 0, lineshape_mode = 0;

    // scratch
    double* d_partial = nullptr;   // [2 * AMP_MAX_POINTS][PARTIAL_STRIDE]
    double* d_sums = nullptr;      // [2 * AMP_MAX_POINTS]
    double* d_result = nullptr;    // [4 * AMP_MAX_POINTS + 4]: NLL[P], I[P], domain flag, sum log S [P], sum w S [P]
    int* d_flag = nullptr;
    unsigned int* d_ticket = nullptr;   // last-CTA ticket of the fused single-launch step (0 between launches)
    double* h_pinned = nullptr;    // same layout
    double* h_zc = nullptr;        // [8] mapped pinned host memory: the fused step's kernel writes its result block here (zero copy)
    double zc_seq = 0;             // stamp of the last fused launch
    double* d_npartial = nullptr;  // [DELTAN_MAX_ROWS][PARTIAL_STRIDE] per-CTA partials of k_deltan (deltan.cu)
    double* d_ntot = nullptr;      // [1 + NVAL] its totals, read by k_deltaf's finish
    double* h_zcb = nullptr;       // [4 AMP_MAX_POINTS + 2] the same for the gradient-batch kernel's result block (deltaf.cu)
    double zcb_seq = 0;
    bool zero_copy = true;
    std::vector<double> last_slog, last_swS;   // the two sums of the last amp_nll, per point (amp_nll_terms)

    // batched (P > 1) plan buffers: coefficient fragments, basis entries, sparse items
    unsigned char* d_plan = nullptr;
    unsigned char* h_plan = nullptr;   // pinned
    size_t plan_cap = 0;
    int batch_mode = 0;            // 0 auto (DMMA kernel when eligible), 1 never (loop of single-point kernels)

    // normalisation matrix (a4): Gram matrix of the last lineshape state, its signature, and work buffers
    struct GramKey { int r; double mass, width; int code; };
    std::vector<GramKey> gram_sig;
    std::vector<int2> gram_tiles;
    bool gram_valid = false;
    int gram_KP = 0;
    bool gram_p1 = false;          // the held matrix was built for a single-point call whose masses and widths are gram_mw
    int gram_nent = 0;
    std::vector<double> gram_mw;
    double* d_G = nullptr;         // [KP][KP] dense symmetric realified Gram matrix (sum_j w_j b' b'^T)
    double* d_gt = nullptr;        // [ntile][64]
    double* d_gpartial = nullptr;  // [CTAs][ntile][64]
    size_t gram_cap_KP = 0, gram_cap_tiles = 0;
    unsigned char* d_hk = nullptr; // herk plan: entries, tiles, coefficients
    unsigned char* h_hk = nullptr; // pinned
    size_t hk_cap = 0;
    // scratch of amp_generate, kept between calls (cudaMalloc / cudaFree of ~200 MB per call would cost more than the generation)
    double *toy_x = nullptr, *toy_u = nullptr, *toy_S = nullptr, *toy_cache = nullptr;
    int* toy_count = nullptr;
    unsigned long long* toy_fseen = nullptr;
    long long toy_cap = 0;         // candidates the scratch holds
    long long stat_delta_exact = 0;   // gradient-batch calls repeated without the expansion (guard tripped)
    bool stream_inline = true;     // P == 1: streaming launches evaluate lineshapes in registers even if columns exist
    bool want_matrix = false;      // set_params decided that the normalisation should go through the matrix
    std::vector<double> prev_mw;   // masses and widths of the previous single-point call (static-lineshape detection)

    int stat_launches = 0, stat_columns = 0, stat_norm_path = 0, stat_batched = 0, stat_gram_built = 0;
    cudaEvent_t ev[5]{};           // phase boundaries of the last evaluation (amp_last_call_timing)
    bool ev_valid = false;
    bool split_valid = false;      // ... of the gradient batch's three launches: ev[1], ev[2] lie between them
    bool fused_valid = false;      // the last evaluation was one fused launch (or the gradient-batch launches): ring[ring_last] brackets it
    enum { RING = 256 };
    cudaEvent_t ring[2 * RING]{};  // event pairs around the launches of the fused / gradient-batch evaluations, newest at ring_last
    int ring_last = -1;
    long long ring_calls = 0;      // such evaluations since amp_model_create (amp_recent_launch_ms)
    bool use_delta = false;        // P > 1 and the points are sparse changes of point 0: gradient-batch kernel (delta.cu)
    bool delta_plan_built = false; // delta_chunks hold the program of the current points (compiled lazily when k_deltaf takes the batch)
    bool no_deltaf_once = false;   // amp_set_params called again by evaluate(): the specialised kernel is not to be planned
    struct DeltaChunk { int p0, np, nsorted; std::vector<DeltaContrib> contrib; std::vector<double> slots; };
    std::vector<DeltaChunk> delta_chunks;     // compiled program of the last amp_set_params (points p0 .. p0 + np - 1 per launch)
    bool use_deltaf = false;       // ... and every point is ONE coupling or ONE lineshape change of the paper's resonance lists: deltaf.cu
    DeltaFArgs deltaf{};           // its tables (filled by amp_set_params; pointers and point 0 by evaluate())
    long long stat_deltaf_guard = 0;   // deltaf calls repeated through delta.cu's exact form (guard on r tripped)
    double* d_bkg = nullptr;       // [data.npad] background density b_i at the data events (Eq. 14), 1 on padding
    double purity = 1.0;
    bool has_bkg = false;
    int grad_mode = 0;             // 0: amp_nll_grad picks the shape-specialised kernel where the model allows; 1: always the generic one
    int fused_mode = 0;            // 0: P == 1 steps with floating lineshapes run as one fused launch; 1: separate launches
    std::string err;
};

namespace {

enum { PARTIAL_STRIDE = 2048 };
enum { DELTAN_MAX_ROWS = 1 + 2 * DELTAF_MAX_POS + 8 * DELTAF_MAX_ENT };   // k_deltan: sum w S0, the leaves, eight tile values per entry

amp_status fail(amp_model* m, amp_status s, const std::string& msg) {
    if (m) m->err = msg;
    return s;
}
amp_status cuda_fail(amp_model* m, cudaError_t e, const char* where) {
    return fail(m, e == cudaErrorMemoryAllocation ? AMP_ERR_NOMEM : AMP_ERR_CUDA, std::string(where) + ": " + cudaGetErrorString(e));
}
#define CK(call)                                                  \
    do {                                                          \
        cudaError_t e_ = (call);                                  \
        if (e_ != cudaSuccess) return cuda_fail(m, e_, #call);    \
    } while (0)

// Makes the model's device current for the duration of a call (a process may hold one model per device) and restores the
// caller's device afterwards.
struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(const amp_model* m) {
        int cur = 0;
        if (m && cudaGetDevice(&cur) == cudaSuccess && cur != m->device) { prev = cur; cudaSetDevice(m->device); }
    }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

double h_two_body(double M, double a, double b) {
    const double s = a + b, d = a - b;
    const double k = (M - s) * (M + s) * (M - d) * (M + d);
    return (k >= 0 && M > 0) ? std::sqrt(k) / (2 * M) : std::numeric_limits<double>::quiet_NaN();
}
double h_bw_poly(int L, double z) {
    switch (L) {
        case 0: return 1.0;
        case 1: return 1.0 + z;
        case 2: return (z + 3.0) * z + 9.0;
        case 3: return ((z + 6.0) * z + 45.0) * z + 225.0;
        default: return (((z + 10.0) * z + 135.0) * z + 1575.0) * z + 11025.0;
    }
}

// Constants of one lineshape column (see LineConst).  Returns false if the pole momenta do not exist.
bool make_line_const(const amp_model* m, int r, double mass, double width, LineConst* out) {
    const amp_resonance& R = m->res[r];
    LineConst c{};
    c.kind = R.kind;
    if (R.kind == AMP_CONST) { c.chain = 2; *out = c; return true; }
    if (R.kind == AMP_LASS) {   // Eq. 7: kG = M0^2 Gamma0 / q0, q0 the K momentum at the K0*(1430) mass
        const double q0 = h_two_body(mass, m->dk.mK, m->dk.mpi);
        if (!(q0 > 0) || !(mass > 0) || !(width > 0)) return false;
        c.chain = 0;
        c.M2 = mass * mass;
        c.kG = mass * mass * width / q0;
        c.kN = 1.0;
        *out = c;
        return true;
    }
    double pR0, pB0;
    if (R.kind == AMP_KSTAR) {
        c.chain = 0;
        c.LR = R.J;
        c.LB = R.J == 0 ? 1 : R.J - 1;                          // lowest allowed L_B
        pR0 = h_two_body(mass, m->dk.mK, m->dk.mpi);
        pB0 = h_two_body(m->dk.MB, mass, m->dk.mpsi);
    } else {
        c.chain = 1;
        c.LR = z_class_LR(z_class(R.kind, R.J));                 // 1+ Z -> psi pi in S wave; the other spin-parities: amp_internal.cuh
        c.LB = R.J;                                              // B -> Z K: L_B = J (P wave for the 1+)
        pR0 = h_two_body(mass, m->dk.mpsi, m->dk.mpi);
        pB0 = h_two_body(m->dk.MB, mass, m->dk.mK);
    }
    if (!(pR0 > 0) || !(pB0 > 0) || !(mass > 0) || !(width > 0)) return false;
    c.M2 = mass * mass;
    c.r2 = R.radius * R.radius;
    const double BR0 = h_bw_poly(c.LR, c.r2 * pR0 * pR0), BB0 = h_bw_poly(c.LB, c.r2 * pB0 * pB0);
    const double kF = std::sqrt(BR0 * BB0);
    c.kN = kF / std::pow(m->dk.MB, c.LB);
    c.kG = mass * mass * width * BR0 / std::pow(pR0, 2 * c.LR + 1);
    *out = c;
    return true;
}

__global__ void k_fill(double* __restrict__ p, long long n, double v) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) p[i] = v;
}

void free_toy_scratch(amp_model* m) {
    if (m->toy_x) cudaFree(m->toy_x);
    if (m->toy_u) cudaFree(m->toy_u);
    if (m->toy_S) cudaFree(m->toy_S);
    if (m->toy_cache) cudaFree(m->toy_cache);
    if (m->toy_count) cudaFree(m->toy_count);
    if (m->toy_fseen) cudaFree(m->toy_fseen);
    m->toy_x = m->toy_u = m->toy_S = m->toy_cache = nullptr;
    m->toy_count = nullptr;
    m->toy_fseen = nullptr;
    m->toy_cap = 0;
}

void free_dataset(Dataset& d) {
    if (d.cache) cudaFree(d.cache);
    if (d.cols) cudaFree(d.cols);
    d = Dataset{};
}

// `scratch`: d is a private work set of the caller (the toy generator's candidates): the model's own data / normalisation state is
// left alone and an allocation of the right size is reused
amp_status load_dataset(amp_model* m, Dataset& d, bool is_norm, const double* d_x, const double* d_w, long long n, cudaStream_t s, bool scratch = false) {
    if (!m) return AMP_ERR_INVALID;
    if (n < 0 || (n > 0 && !d_x)) return fail(m, AMP_ERR_INVALID, "load: null events or negative count");
    const long long npad = stream_pad(n > 0 ? n : 1);
    // scratch: the caller's buffer holds at least npad events; otherwise a same-sized reload (pseudo-experiment loops) keeps its
    // allocations (cache and lineshape pool, whose columns are marked stale below): cudaFree + cudaMalloc cost milliseconds
    const bool reuse = scratch ? d.cache != nullptr : (d.cache != nullptr && d.npad == npad);
    if (!reuse) free_dataset(d);
    if (!scratch) {
        for (auto& e : m->pool) (is_norm ? e.valid_norm : e.valid_data) = false;
        if (is_norm) m->gram_valid = false;
        if (!is_norm) { if (m->d_bkg) cudaFree(m->d_bkg); m->d_bkg = nullptr; m->has_bkg = false; m->purity = 1.0; }   // belongs to the old data set
    }
    d.n = n;
    d.npad = npad;
    d.ncache = m->has_z ? NCOL_ALL : NCOL_K;
    d.loaded = false;
    if (!reuse) CK(cudaMalloc(&d.cache, sizeof(double) * (d.ncache + 1) * d.npad));   // tiled: [npad / 512][ncache + 1][512], weight last
    CK(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
    const int grid = kinematics_grid(d.npad);
    KinArgs a{};
    a.dk = m->dk;
    a.x = d_x;
    a.w = d_w;
    a.cache = d.cache;
    a.ncolw = d.ncache + 1;
    a.n = n;
    a.npad = d.npad;
    a.with_z = m->has_z ? 1 : 0;
    a.weight_positive = is_norm ? 0 : 1;
    a.flag = m->d_flag;
    a.partial = m->d_partial;
    CK(launch_kinematics(a, grid, s));
    CK(launch_finalize(m->d_partial, grid, PARTIAL_STRIDE, 1, m->d_sums, s));
    CK(cudaMemcpyAsync(m->h_pinned, m->d_sums, sizeof(double), cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(m->h_pinned + 1, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    int flag;
    std::memcpy(&flag, m->h_pinned + 1, sizeof(int));
    if (flag) {
        if (!scratch) free_dataset(d);
        return fail(m, AMP_ERR_DOMAIN, is_norm ? "amp_load_norm: event outside phase space or bad weight"
                                               : "amp_load_events: event outside phase space or non-positive efficiency");
    }
    d.wsum = m->h_pinned[0];
    if (is_norm && n > 0 && !(d.wsum > 0)) {
        if (!scratch) free_dataset(d);
        return fail(m, AMP_ERR_DOMAIN, "amp_load_norm: weights sum to zero");
    }
    d.loaded = true;
    return AMP_OK;
}

}  // namespace

extern "C" {

const char* amp_version(void) { return "amp4d 0.1 (sm_100a)"; }

const char* amp_status_string(amp_status s) {
    switch (s) {
        case AMP_OK: return "AMP_OK";
        case AMP_ERR_INVALID: return "AMP_ERR_INVALID";
        case AMP_ERR_STATE: return "AMP_ERR_STATE";
        case AMP_ERR_DOMAIN: return "AMP_ERR_DOMAIN";
        case AMP_ERR_CUDA: return "AMP_ERR_CUDA";
        case AMP_ERR_NOMEM: return "AMP_ERR_NOMEM";
    }
    return "?";
}

const char* amp_last_error(const amp_model* m) { return m ? m->err.c_str() : "null model"; }

amp_status amp_model_create(const amp_decay* decay, const amp_resonance* res, int n_res, amp_model** out) {
    if (!decay || !res || !out || n_res < 1 || n_res > AMP_MAX_RESONANCES) return AMP_ERR_INVALID;
    *out = nullptr;
    if (!(decay->m_parent > 0 && decay->m_psi > 0 && decay->m_k > 0 && decay->m_pi > 0) ||
        !(decay->m_parent > decay->m_psi + decay->m_k + decay->m_pi))
        return AMP_ERR_INVALID;
    amp_model* m = new (std::nothrow) amp_model();
    if (!m) return AMP_ERR_NOMEM;
    m->dk = DecayConst{decay->m_parent, decay->m_psi, decay->m_k, decay->m_pi};
    m->R = n_res;
    int K = 0;
    for (int r = 0; r < n_res; ++r) {
        const amp_resonance& a = res[r];
        bool ok = true;
        if (a.kind == AMP_KSTAR) ok = a.J >= 0 && a.J <= 4;
        else if (a.kind == AMP_Z) ok = a.J == 1 || a.J == 2;      // 1+, 2+ (0+ cannot decay to psi pi)
        else if (a.kind == AMP_ZM) ok = a.J >= 0 && a.J <= 2;       // 0-, 1-, 2-
        else if (a.kind == AMP_CONST) ok = a.J == 0;
        else if (a.kind == AMP_LASS) ok = a.J == 0;
        else ok = false;
        if (a.kind != AMP_CONST) ok = ok && a.mass > 0 && a.width > 0 && a.radius >= 0 && std::isfinite(a.mass + a.width + a.radius);
        if (!ok) { delete m; return AMP_ERR_INVALID; }
        m->res.push_back(a);
        m->slot0[r] = K;
        K += (kind_is_z(a.kind) || (a.kind == AMP_KSTAR && a.J >= 1)) ? 3 : 1;
        if (kind_is_z(a.kind)) m->has_z = true;
    }
    int nconst = 0;
    for (int r = 0; r < n_res; ++r) nconst += res[r].kind == AMP_CONST;
    if (K > AMP_MAX_COUPLINGS || nconst > 4) { delete m; return AMP_ERR_INVALID; }
    m->K = K;
    for (int r = 0; r < n_res; ++r) {
        LineConst lc;
        if (!make_line_const(m, r, res[r].mass, res[r].width, &lc)) { delete m; return AMP_ERR_DOMAIN; }
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { delete m; return AMP_ERR_CUDA; }
    if (cudaGetDevice(&m->device) != cudaSuccess) { delete m; return AMP_ERR_CUDA; }
    cudaError_t e = cudaMalloc(&m->d_partial, sizeof(double) * 2 * AMP_MAX_POINTS * PARTIAL_STRIDE);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_sums, sizeof(double) * 2 * AMP_MAX_POINTS);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_result, sizeof(double) * (4 * AMP_MAX_POINTS + 4));
    if (e == cudaSuccess) e = cudaMalloc(&m->d_flag, sizeof(int));
    if (e == cudaSuccess) e = cudaMalloc(&m->d_npartial, sizeof(double) * DELTAN_MAX_ROWS * PARTIAL_STRIDE);
    if (e == cudaSuccess) e = cudaMalloc(&m->d_ntot, sizeof(double) * (1 + 4 * (DELTAF_MAX_POS + DELTAF_MAX_ENT)));
    if (e == cudaSuccess) e = cudaMalloc(&m->d_ticket, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(m->d_ticket, 0, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(m->d_flag, 0, sizeof(int));
    if (e == cudaSuccess) e = cudaMallocHost(&m->h_pinned, sizeof(double) * (4 * AMP_MAX_POINTS + 4));
    if (e == cudaSuccess) e = cudaHostAlloc(&m->h_zc, sizeof(double) * 8, cudaHostAllocMapped);
    if (e == cudaSuccess) { std::memset(m->h_zc, 0, sizeof(double) * 8); m->zero_copy = true; }
    if (e == cudaSuccess) e = cudaHostAlloc(&m->h_zcb, sizeof(double) * (4 * AMP_MAX_POINTS + 2), cudaHostAllocMapped);
    if (e == cudaSuccess) std::memset(m->h_zcb, 0, sizeof(double) * (4 * AMP_MAX_POINTS + 2));
    for (int i = 0; i < 5 && e == cudaSuccess; ++i) e = cudaEventCreate(&m->ev[i]);
    for (int i = 0; i < 2 * amp_model::RING && e == cudaSuccess; ++i) e = cudaEventCreate(&m->ring[i]);
    if (e != cudaSuccess) { amp_model_destroy(m); return e == cudaErrorMemoryAllocation ? AMP_ERR_NOMEM : AMP_ERR_CUDA; }
    *out = m;
    return AMP_OK;
}

amp_status amp_model_destroy(amp_model* m) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    free_dataset(m->data);
    free_dataset(m->norm);
    if (m->d_partial) cudaFree(m->d_partial);
    if (m->d_sums) cudaFree(m->d_sums);
    if (m->d_result) cudaFree(m->d_result);
    if (m->d_flag) cudaFree(m->d_flag);
    if (m->d_ticket) cudaFree(m->d_ticket);
    if (m->d_bkg) cudaFree(m->d_bkg);
    free_toy_scratch(m);
    if (m->h_pinned) cudaFreeHost(m->h_pinned);
    if (m->h_zc) cudaFreeHost(m->h_zc);
    if (m->h_zcb) cudaFreeHost(m->h_zcb);
    if (m->d_npartial) cudaFree(m->d_npartial);
    if (m->d_ntot) cudaFree(m->d_ntot);
    if (m->d_plan) cudaFree(m->d_plan);
    if (m->h_plan) cudaFreeHost(m->h_plan);
    if (m->d_G) cudaFree(m->d_G);
    if (m->d_gt) cudaFree(m->d_gt);
    if (m->d_gpartial) cudaFree(m->d_gpartial);
    if (m->d_hk) cudaFree(m->d_hk);
    if (m->h_hk) cudaFreeHost(m->h_hk);
    for (int i = 0; i < 5; ++i) if (m->ev[i]) cudaEventDestroy(m->ev[i]);
    for (int i = 0; i < 2 * amp_model::RING; ++i) if (m->ring[i]) cudaEventDestroy(m->ring[i]);
    delete m;
    return AMP_OK;
}

int amp_num_couplings(const amp_model* m) { return m ? m->K : -1; }
int amp_num_resonances(const amp_model* m) { return m ? m->R : -1; }

amp_status amp_load_events(amp_model* m, const double* d_x, const double* d_eff, long long n, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    return load_dataset(m, m->data, false, d_x, d_eff, n, (cudaStream_t)stream);
}

amp_status amp_load_norm(amp_model* m, const double* d_x, const double* d_w, long long n_norm, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    if (n_norm < 1) return fail(m, AMP_ERR_INVALID, "amp_load_norm: need at least one normalisation event");
    return load_dataset(m, m->norm, true, d_x, d_w, n_norm, (cudaStream_t)stream);
}

amp_status amp_set_background(amp_model* m, const double* d_bkg, double purity, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    cudaStream_t s = (cudaStream_t)stream;
    if (!d_bkg) {   // back to the signal-only likelihood
        if (m->d_bkg) cudaFree(m->d_bkg);
        m->d_bkg = nullptr; m->has_bkg = false; m->purity = 1.0; m->P = 0;
        return AMP_OK;
    }
    if (!m->data.loaded) return fail(m, AMP_ERR_STATE, "amp_set_background: load the data events first");
    if (!(purity >= 0.0 && purity <= 1.0)) return fail(m, AMP_ERR_INVALID, "amp_set_background: purity must be in [0, 1]");
    if (m->d_bkg) cudaFree(m->d_bkg);
    m->d_bkg = nullptr;
    CK(cudaMalloc(&m->d_bkg, sizeof(double) * m->data.npad));
    k_fill<<<sm_count() * 4, 256, 0, s>>>(m->d_bkg, m->data.npad, 1.0);
    CK(cudaGetLastError());
    CK(cudaMemcpyAsync(m->d_bkg, d_bkg, sizeof(double) * m->data.n, cudaMemcpyDeviceToDevice, s));
    CK(cudaStreamSynchronize(s));
    m->purity = purity;
    m->has_bkg = true;
    m->P = 0;   // parameters must be set again: the evaluation plan depends on the background
    return AMP_OK;
}

amp_status amp_set_norm_mode(amp_model* m, int mode) {
    if (!m || mode < 0 || mode > 2) return AMP_ERR_INVALID;
    m->norm_mode = mode;
    return AMP_OK;
}

amp_status amp_set_batch_mode(amp_model* m, int mode) {
    if (!m || mode < 0 || mode > 4) return AMP_ERR_INVALID;
    m->batch_mode = mode;
    return AMP_OK;
}

amp_status amp_set_fused_mode(amp_model* m, int mode) {
    if (!m || mode < 0 || mode > 1) return AMP_ERR_INVALID;
    m->fused_mode = mode;
    return AMP_OK;
}

amp_status amp_set_grad_mode(amp_model* m, int mode) {
    if (!m || mode < 0 || mode > 1) return AMP_ERR_INVALID;
    m->grad_mode = mode;
    return AMP_OK;
}

amp_status amp_set_lineshape_mode(amp_model* m, int mode) {
    if (!m || mode < 0 || mode > 2) return AMP_ERR_INVALID;
    m->lineshape_mode = mode;
    return AMP_OK;
}

amp_status amp_last_call_stats(const amp_model* m, int* launches, int* columns_recomputed, int* norm_path) {
    if (!m) return AMP_ERR_INVALID;
    if (launches) *launches = m->stat_launches;
    if (columns_recomputed) *columns_recomputed = m->stat_columns;
    if (norm_path) *norm_path = m->stat_norm_path;
    return AMP_OK;
}

amp_status amp_last_call_timing(const amp_model* m, double* ms4) {
    if (!m || !ms4) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    if (m->fused_valid) {   // one launch: everything is reported as the combine phase of both samples
        float t = 0;
        cudaEventSynchronize(m->ring[2 * m->ring_last + 1]);   // (a zero-copy call returns before its end event has landed)
        if (cudaEventElapsedTime(&t, m->ring[2 * m->ring_last], m->ring[2 * m->ring_last + 1]) != cudaSuccess) return AMP_ERR_CUDA;
        ms4[0] = 0; ms4[1] = t; ms4[2] = 0; ms4[3] = 0;
        if (m->split_valid && m->stat_norm_path == 9) {   // normalisation pass 0, pass 1, then the data events
            float t0 = 0, t1 = 0, t2 = 0;
            if (cudaEventElapsedTime(&t0, m->ring[2 * m->ring_last], m->ev[1]) != cudaSuccess || cudaEventElapsedTime(&t1, m->ev[1], m->ev[2]) != cudaSuccess ||
                cudaEventElapsedTime(&t2, m->ev[2], m->ring[2 * m->ring_last + 1]) != cudaSuccess)
                return AMP_ERR_CUDA;
            ms4[1] = t2; ms4[2] = t0; ms4[3] = t1;
        }
        return AMP_OK;
    }
    if (!m->ev_valid) return AMP_ERR_STATE;
    for (int i = 0; i < 4; ++i) {
        float t = 0;
        if (cudaEventElapsedTime(&t, m->ev[i], m->ev[i + 1]) != cudaSuccess) return AMP_ERR_CUDA;
        ms4[i] = t;
    }
    return AMP_OK;
}

amp_status amp_recent_launch_ms(const amp_model* m, int max_calls, double* h_ms, int* n_out) {
    if (!m || !h_ms || !n_out || max_calls < 0) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    const long long have = std::min<long long>(m->ring_calls, amp_model::RING);
    const int n = (int)std::min<long long>(have, max_calls);
    for (int i = 0; i < n; ++i) {   // oldest of the n first
        const int slot = ((m->ring_last - (n - 1 - i)) % amp_model::RING + amp_model::RING) % amp_model::RING;
        float t = 0;
        cudaEventSynchronize(m->ring[2 * slot + 1]);
        if (cudaEventElapsedTime(&t, m->ring[2 * slot], m->ring[2 * slot + 1]) != cudaSuccess) return AMP_ERR_CUDA;
        h_ms[i] = t;
    }
    *n_out = n;
    return AMP_OK;
}

amp_status amp_probe_fp64(int kind, int iters, double* flops, void* stream) {
    if (!flops || kind < 0 || kind > 1 || iters < 1) return AMP_ERR_INVALID;
    return probe_fp64(kind, iters, flops, (cudaStream_t)stream) == cudaSuccess ? AMP_OK : AMP_ERR_CUDA;
}

amp_status amp_probe_hbm_read(long long bytes, double* gbs, void* stream) {
    if (!gbs || bytes < (long long)((NCOL_ALL + 1) * CACHE_TILE * sizeof(double))) return AMP_ERR_INVALID;
    const cudaError_t e = probe_hbm_read(bytes, gbs, (cudaStream_t)stream);
    if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return AMP_ERR_NOMEM; }
    return e == cudaSuccess ? AMP_OK : AMP_ERR_CUDA;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------------
// Parameter points and the lineshape column pool
namespace {

// Make sure both datasets have a column pool of at least `need` slots.  Growing drops all columns.
amp_status ensure_pool(amp_model* m, int need) {
    if (need <= m->pool_cap && (!m->data.loaded || m->data.cols) && (!m->norm.loaded || m->norm.cols)) return AMP_OK;
    int cap = std::max(need, m->pool_cap);
    if (need > m->pool_cap) cap = std::max(need + 4, m->R + 4);
    for (Dataset* d : {&m->data, &m->norm}) {
        if (!d->loaded) continue;
        if (d->cols && cap == m->pool_cap) continue;
        if (d->cols) { cudaFree(d->cols); d->cols = nullptr; }
        CK(cudaMalloc(&d->cols, sizeof(double2) * (size_t)cap * d->npad));
        for (auto& e : m->pool) (d == &m->data ? e.valid_data : e.valid_norm) = false;
    }
    m->pool_cap = cap;
    m->pool.resize(cap);
    return AMP_OK;
}

void fill_stream_args(const amp_model* m, const Dataset& d, int p, int mode, StreamArgs* a, int* ent_of_res = nullptr, int* grp_of_res = nullptr);

// Compile a batch whose points 1..P-1 are sparse changes of point 0 into the gradient-batch kernel's program
// (amp_internal.cuh, DeltaContrib): per chunk of <= 128 points a contribution list and the slot records it refers to.
// False if the batch is not sparse (more than ~3 changed resonances per point on average), touches a constant term's
// coupling, or does not fit the kernel's shared memory: the caller then takes the dense path.
bool build_delta_plan(amp_model* m) {
    const int P = m->P, R = m->R, K = m->K;
    m->delta_chunks.clear();
    if (P < 2) return false;
    for (const auto& rs : m->res)
        if (rs.kind == AMP_LASS) return false;   // LASS terms are not carried by the gradient-batch kernel
    int ent_of_res[AMP_MAX_RESONANCES], grp_of_res[AMP_MAX_RESONANCES];
    {
        StreamArgs tmp;
        fill_stream_args(m, m->norm, 0, MODE_FUSED, &tmp, ent_of_res, grp_of_res);
        if (!delta_fits(tmp.gstart[NSPIN])) return false;
        for (int sp = 6; sp < NSPIN; ++sp) if (tmp.shape[sp]) return false;   // Z's other than 1+: dense path
    }
    size_t total = 0;
    const size_t cap = (size_t)3 * (P - 1) + 8;
    for (int p0 = 1; p0 < P; p0 += DELTA_MAX_SORTED) {
        amp_model::DeltaChunk ch;
        ch.p0 = p0;
        ch.np = std::min((int)DELTA_MAX_SORTED, P - p0);
        ch.nsorted = (ch.np + 31) / 32 * 32;
        std::vector<std::pair<std::vector<double>, int>> known;   // slot record -> offset
        auto add_slot = [&](const std::vector<double>& rec) {
            for (auto& kv : known)
                if (kv.first.size() == rec.size() && std::memcmp(kv.first.data(), rec.data(), rec.size() * sizeof(double)) == 0) return kv.second;
            const int off = (int)ch.slots.size();
            ch.slots.insert(ch.slots.end(), rec.begin(), rec.end());
            known.emplace_back(rec, off);
            return off;
        };
        auto word = [](int lo, int hi) { double d; const int v[2] = {lo, hi}; std::memcpy(&d, v, 8); return d; };
        int prev_slot = -1;
        auto push = [&](int kind, int slot, int r, double a, double b, double c) {
            DeltaContrib dc{};
            const bool isz = r >= 0 && kind_is_z(m->res[r].kind);
            dc.hdr = kind | (slot != prev_slot ? 8 : 0) | (isz ? 32 : 0) | ((r >= 0 ? grp_of_res[r] : 0) << 8);
            dc.slot = slot;
            dc.a = a; dc.b = b; dc.c = c;
            prev_slot = slot;
            ch.contrib.push_back(dc);
        };
        std::vector<size_t> first_of(ch.nsorted + 1, 0);
        for (int q = 0; q < ch.nsorted; ++q) {
            const size_t first = ch.contrib.size();
            first_of[q] = first;
            const int p = p0 + q;
            for (int r = 0; q < ch.np && r < R; ++r) {
                const amp_resonance& rs = m->res[r];
                const int ns = (kind_is_z(rs.kind) || (rs.kind == AMP_KSTAR && rs.J >= 1)) ? 3 : 1;
                const double* c0 = &m->couplings[((size_t)0 * K + m->slot0[r]) * 2];
                const double* cp = &m->couplings[((size_t)p * K + m->slot0[r]) * 2];
                bool dcf[3] = {false, false, false}, anyc = false;
                for (int j = 0; j < ns; ++j) { dcf[j] = cp[2 * j] != c0[2 * j] || cp[2 * j + 1] != c0[2 * j + 1]; anyc |= dcf[j]; }
                if (rs.kind == AMP_CONST) { if (anyc) return false; continue; }
                const double* mw0 = &m->mw[((size_t)0 * R + r) * 2];
                const double* mwp = &m->mw[((size_t)p * R + r) * 2];
                const bool ls = mwp[0] != mw0[0] || mwp[1] != mw0[1];
                if (!anyc && !ls) continue;
                const bool isz = kind_is_z(rs.kind);
                const int Jf = isz ? 1 : rs.J;
                auto term_hdr = [&](int j, bool with_bw, bool unit) {
                    const int l = ns == 3 ? j : 1;   // helicity -1, 0, +1 -> 0, 1, 2
                    return (with_bw ? ent_of_res[r] : 255) | (grp_of_res[r] << 8) | (Jf << 12) | (l << 15) | ((isz ? 1 : 0) << 17) | ((unit ? 1 : 0) << 18);
                };
                // slot = sum_j weight_j [BW_R(0)] g_{R,j}; bw0spec: the slot also carries BW_R(0) for kind-1 contributions
                auto weighted_slot = [&](const double* cc, bool with_bw, int bw0spec) {
                    std::vector<double> rec(1, 0.0);
                    int nt = 0;
                    for (int j = 0; j < ns; ++j) {
                        if (cc[2 * j] == 0.0 && cc[2 * j + 1] == 0.0) continue;
                        rec.push_back(word(term_hdr(j, with_bw, false), 0));
                        rec.push_back(cc[2 * j]);
                        rec.push_back(cc[2 * j + 1]);
                        ++nt;
                    }
                    rec[0] = word(nt, bw0spec);
                    return nt ? add_slot(rec) : -1;
                };
                if (!ls) {
                    // coupling changes only: helicities that move by the same amount share one slot (Eq. 11 ties H_+1 = H_-1 of a 1+ Z)
                    bool done[3] = {false, false, false};
                    for (int j = 0; j < ns; ++j) {
                        if (!dcf[j] || done[j]) continue;
                        const double dre = cp[2 * j] - c0[2 * j], dim = cp[2 * j + 1] - c0[2 * j + 1];
                        std::vector<double> rec(1, 0.0);
                        int nt = 0;
                        for (int j2 = j; j2 < ns; ++j2)
                            if (dcf[j2] && !done[j2] && cp[2 * j2] - c0[2 * j2] == dre && cp[2 * j2 + 1] - c0[2 * j2 + 1] == dim) {
                                done[j2] = true;
                                rec.push_back(word(term_hdr(j2, true, true), 0));
                                rec.push_back(1.0);
                                rec.push_back(0.0);
                                ++nt;
                            }
                        rec[0] = word(nt, -1);
                        push(0, add_slot(rec), r, dre, dim, dre * dre + dim * dim);   // third constant of a kind-0 contribution: |coef|^2
                    }
                } else {
                    LineConst lc;
                    make_line_const(m, r, mwp[0], mwp[1], &lc);
                    const int spec = ent_of_res[r] | (grp_of_res[r] << 8) | ((isz ? 1 : 0) << 12);
                    if (!anyc) {
                        const int sl = weighted_slot(c0, false, spec);        // (BW(p) - BW(0)) sum_j c_j(0) g_j
                        if (sl >= 0) push(1, sl, r, lc.kN, lc.kG, lc.M2);
                    } else {
                        const int s1 = weighted_slot(cp, false, -1);          // BW(p) sum_j c_j(p) g_j
                        if (s1 >= 0) push(2, s1, r, lc.kN, lc.kG, lc.M2);
                        const int s0 = weighted_slot(c0, true, -1);           // - sum_j c_j(0) BW(0) g_j
                        if (s0 >= 0) push(0, s0, r, -1.0, 0.0, 1.0);
                    }
                }
            }
            if (ch.contrib.size() == first) { DeltaContrib e{}; e.hdr = 16; e.slot = -1; ch.contrib.push_back(e); }   // equal to point 0, or padding
            ch.contrib.back().hdr |= 4;
            if (q < ch.np) total += ch.contrib.size() - first;
            if (total > cap || ch.contrib.size() > DELTA_MAX_CONTRIB || ch.slots.size() > DELTA_MAX_SLOTWORDS) return false;
        }
        // Four consecutive points (aligned in the block) that are single contributions of one kind (coupling, or mass / width) on
        // one slot — the gradient pattern — are marked once here (bit 64 of the first header) instead of being recognised by every thread
        first_of[ch.nsorted] = ch.contrib.size();
        for (int q = 0; q + 3 < ch.nsorted; q += 4) {
            bool quad = true;
            const int kind = ch.contrib[first_of[q]].hdr & 3;
            for (int j = 0; j < 4 && quad; ++j) {
                const int h = ch.contrib[first_of[q + j]].hdr;
                quad = first_of[q + j + 1] - first_of[q + j] == 1 && (h & (j ? 28 : 20)) == 4 && (h & 3) == kind && kind < 2;
            }
            if (quad) ch.contrib[first_of[q]].hdr |= 64;
        }
        m->delta_chunks.push_back(std::move(ch));
    }
    return true;
}

// The shape-specialised gradient-batch kernel (deltaf.cu): every point 1..P-1 must be ONE coupling change — a single slot, or the
// helicities -1 and +1 of a Z moving by the same amount (Eq. 11) — or ONE mass / width change of one resonance with its couplings
// unchanged, at most four points per position / resonance, on one of the compiled model shapes.  Fills m->deltaf's tables.
bool build_deltaf_plan(amp_model* m) {
    const int P = m->P, R = m->R, K = m->K;
    if (P < 2 || !m->norm.loaded) return false;
    int ent_of_res[AMP_MAX_RESONANCES], grp_of_res[AMP_MAX_RESONANCES];
    DeltaFArgs& d = m->deltaf;
    fill_stream_args(m, m->norm, 0, MODE_FUSED, &d.a, ent_of_res, grp_of_res);
    DeltaFLayout lay;
    if (!deltaf_layout(d.a, &lay)) return false;
    const int nslot = lay.nslot, nent = lay.nent;
    for (int i = 0; i < DELTAF_MAX_POS; ++i) d.quad_of_pos[i] = (short)(i < lay.npos ? lay.quad_of_pos[i] : 0);
    for (int i = 0; i < DELTAF_MAX_ENT; ++i) d.quad_of_ent[i] = (short)(i < lay.nent ? lay.quad_of_ent[i] : 0);
    const int n0 = d.a.shape[0];
    auto base = [&](int t) { return t < n0 ? t : n0 + 3 * (t - n0); };
    std::memset(d.cq, 0, sizeof(d.cq));
    std::memset(d.cmax, 0, sizeof(d.cmax));
    for (auto& e : d.mw) for (auto& q : e) { q[0] = 1.0; q[1] = 1.0; q[2] = 1.0; }
    d.pos_active = d.ent_active = 0u;
    for (int p = 0; p < AMP_MAX_POINTS; ++p) d.val_of_point[p] = d.pos_of_point[p] = -1;
    int used_pos[DELTAF_MAX_POS] = {}, used_ent[DELTAF_MAX_ENT] = {};
    for (int p = 1; p < P; ++p) {
        int changed = -1;   // the one resonance that differs from point 0
        for (int r = 0; r < R; ++r) {
            bool diff = m->mw[((size_t)p * R + r) * 2] != m->mw[(size_t)r * 2] || m->mw[((size_t)p * R + r) * 2 + 1] != m->mw[(size_t)r * 2 + 1];
            const int ns = (kind_is_z(m->res[r].kind) || (m->res[r].kind == AMP_KSTAR && m->res[r].J >= 1)) ? 3 : 1;
            for (int j = 0; j < ns; ++j)
                for (int c = 0; c < 2; ++c) diff |= m->couplings[((size_t)p * K + m->slot0[r] + j) * 2 + c] != m->couplings[((size_t)(m->slot0[r] + j)) * 2 + c];
            if (!diff) continue;
            if (changed >= 0) return false;
            changed = r;
        }
        if (changed < 0) continue;   // equal to point 0
        if (m->res[changed].kind == AMP_CONST || m->res[changed].kind == AMP_LASS) return false;   // no entry of the specialised shapes
        const int r = changed, t = ent_of_res[r];
        const amp_resonance& rs = m->res[r];
        const bool isz = kind_is_z(rs.kind);
        const int ns = (isz || (rs.kind == AMP_KSTAR && rs.J >= 1)) ? 3 : 1;
        const bool ls = m->mw[((size_t)p * R + r) * 2] != m->mw[(size_t)r * 2] || m->mw[((size_t)p * R + r) * 2 + 1] != m->mw[(size_t)r * 2 + 1];
        double dre[3] = {0, 0, 0}, dim[3] = {0, 0, 0};
        int nchg = 0, jlast = -1;
        for (int j = 0; j < ns; ++j) {
            dre[j] = m->couplings[((size_t)p * K + m->slot0[r] + j) * 2] - m->couplings[(size_t)(m->slot0[r] + j) * 2];
            dim[j] = m->couplings[((size_t)p * K + m->slot0[r] + j) * 2 + 1] - m->couplings[(size_t)(m->slot0[r] + j) * 2 + 1];
            if (dre[j] != 0.0 || dim[j] != 0.0) { ++nchg; jlast = j; }
        }
        LineConst lc0;
        make_line_const(m, r, m->mw[(size_t)r * 2], m->mw[(size_t)r * 2 + 1], &lc0);
        if (ls) {
            if (nchg) return false;                         // lineshape and couplings at once: delta.cu
            if (used_ent[t] >= 4) return false;
            LineConst lcp;
            make_line_const(m, r, m->mw[((size_t)p * R + r) * 2], m->mw[((size_t)p * R + r) * 2 + 1], &lcp);
            if (used_ent[t] == 0)   // unused points of an entry in use sit at point 0 (Delta = 0)
                for (auto& q : d.mw[t]) { q[0] = 1.0; q[1] = lc0.kG; q[2] = lc0.M2; }
            const int j = used_ent[t]++;
            d.mw[t][j][0] = lcp.kN / lc0.kN;
            d.mw[t][j][1] = lcp.kG;
            d.mw[t][j][2] = lcp.M2;
            d.ent_active |= 1u << t;
            d.val_of_point[p] = (short)(4 * lay.quad_of_ent[t] + j);
            continue;
        }
        int pos;
        if (nchg == 1) {
            pos = base(t) + (ns == 3 ? jlast : 0);
        } else if (nchg == 2 && isz && dre[0] == dre[2] && dim[0] == dim[2] && dre[1] == 0.0 && dim[1] == 0.0) {
            pos = nslot + (t - (nent - d.a.shape[5]));      // tied pair of Z number t - oz
            jlast = 0;
        } else {
            return false;
        }
        if (used_pos[pos] >= 4) return false;
        const int j = used_pos[pos]++;
        const double are = dre[jlast] * lc0.kN, aim = dim[jlast] * lc0.kN;
        d.cq[pos][j][0] = are;
        d.cq[pos][j][1] = aim;
        d.cq[pos][j][2] = are * are + aim * aim;
        d.cmax[pos][0] = std::max(d.cmax[pos][0], std::max(std::fabs(are), std::fabs(aim)));
        d.cmax[pos][1] = std::max(d.cmax[pos][1], d.cq[pos][j][2]);
        d.pos_active |= 1u << pos;
        d.val_of_point[p] = (short)(4 * lay.quad_of_pos[pos] + j);
        d.pos_of_point[p] = (short)pos;
    }
    d.P = P;
    return true;
}

}  // namespace

extern "C" amp_status amp_set_params(amp_model* m, int P, const double* h_couplings, const double* h_mass_width) {
    if (!m) return AMP_ERR_INVALID;
    if (P < 1 || P > AMP_MAX_POINTS || !h_couplings) return fail(m, AMP_ERR_INVALID, "amp_set_params: bad P or null couplings");
    const int R = m->R, K = m->K;
    std::vector<double> mw((size_t)P * R * 2);
    for (int p = 0; p < P; ++p)
        for (int r = 0; r < R; ++r) {
            double mass = m->res[r].mass, width = m->res[r].width;
            if (h_mass_width && m->res[r].kind != AMP_CONST) { mass = h_mass_width[((size_t)p * R + r) * 2]; width = h_mass_width[((size_t)p * R + r) * 2 + 1]; }
            // (a gradient batch repeats point 0's masses and widths in all but a few points: those are checked once)
            if (p == 0 || mass != mw[(size_t)r * 2] || width != mw[(size_t)r * 2 + 1]) {
                LineConst lc;
                if (!std::isfinite(mass) || !std::isfinite(width)) return fail(m, AMP_ERR_INVALID, "amp_set_params: non-finite mass or width");
                if (!make_line_const(m, r, mass, width, &lc)) return fail(m, AMP_ERR_DOMAIN, "amp_set_params: pole mass outside the kinematic range or width <= 0");
            }
            mw[((size_t)p * R + r) * 2] = mass;
            mw[((size_t)p * R + r) * 2 + 1] = width;
        }
    for (size_t i = 0; i < (size_t)P * K * 2; ++i)
        if (!std::isfinite(h_couplings[i])) return fail(m, AMP_ERR_INVALID, "amp_set_params: non-finite coupling");
    m->P = P;
    m->couplings.assign(h_couplings, h_couplings + (size_t)P * K * 2);
    m->mw.swap(mw);
    m->call_id++;
    // Normalisation path.  The matrix M pays when it can be reused or shared: a single point whose masses and widths
    // equal those of the previous call (lineshapes are not moving: M is built once, every later call is O(K^2)), or a
    // large batch of points (one Gram pass instead of one pass per point).  Otherwise the direct sum is cheaper.
    const bool mw_same = P == 1 && m->prev_mw.size() == m->mw.size() && std::equal(m->mw.begin(), m->mw.end(), m->prev_mw.begin());
    m->want_matrix = m->norm_mode == 2 || (m->norm_mode == 0 && (P == 1 ? mw_same : (P >= 24 && m->batch_mode != 1)));
    if (P == 1) m->prev_mw = m->mw; else m->prev_mw.clear();
    // P > 1: a batch whose points are sparse changes of point 0 (a gradient step) runs the delta kernel: no column, no matrix
    if (m->has_bkg && P > 1) m->want_matrix = false;   // Eq. 14: the background path streams both samples, point by point (a single
                                                          // point at fixed lineshapes may still hold M: amp_nll_grad reads it)
    // ... through the shape-specialised kernel where every point is one coupling or one lineshape change (batch mode 3: never);
    // the general kernel's program is then compiled only if a call needs it (the guard on r tripped)
    const bool sparse_ok = P > 1 && !m->has_bkg && (m->batch_mode == 0 || m->batch_mode == 3 || m->batch_mode == 4) && m->lineshape_mode != 1 && m->norm_mode != 2;
    m->use_deltaf = sparse_ok && m->batch_mode != 3 && !m->no_deltaf_once && build_deltaf_plan(m);
    m->delta_plan_built = false;
    m->use_delta = m->use_deltaf || (sparse_ok && (m->delta_plan_built = build_delta_plan(m)));
    if (m->use_delta) m->want_matrix = false;
    m->stream_inline = (P == 1 || m->use_delta || m->has_bkg) && m->lineshape_mode != 1;

    // distinct (resonance, mass, width) keys of this call
    struct Key { int r; double mass, width; };
    std::vector<Key> keys;
    std::vector<int> keyidx((size_t)P * R, -1);
    for (int p = 0; p < P; ++p)
        for (int r = 0; r < R; ++r) {
            if (m->res[r].kind == AMP_CONST) continue;
            const double mass = m->mw[((size_t)p * R + r) * 2], width = m->mw[((size_t)p * R + r) * 2 + 1];
            int found = -1;
            for (int k = (int)keys.size() - 1; k >= 0; --k)
                if (keys[k].r == r && keys[k].mass == mass && keys[k].width == width) { found = k; break; }
            if (found < 0) { keys.push_back(Key{r, mass, width}); found = (int)keys.size() - 1; }
            keyidx[(size_t)p * R + r] = found;
        }
    // hit / miss against the pool; a resonance that misses call after call floats: with P == 1 its column
    // is transient and is evaluated in registers by the combine kernel instead of making a round trip
    std::vector<int> keyslot(keys.size(), -1);
    bool res_missed[AMP_MAX_RESONANCES] = {};
    for (size_t k = 0; k < keys.size(); ++k)
        for (int sidx = 0; sidx < (int)m->pool.size(); ++sidx) {
            const PoolEntry& e = m->pool[sidx];
            if (e.r == keys[k].r && e.mass == keys[k].mass && e.width == keys[k].width) { keyslot[k] = sidx; break; }
        }
    // a miss counts towards "floating" only if the pool already holds this resonance at other values
    // (the first, cold fill of the pool says nothing about whether the parameter floats)
    for (size_t k = 0; k < keys.size(); ++k) {
        if (keyslot[k] >= 0) continue;
        bool held = m->was_inline[keys[k].r];
        for (const PoolEntry& e : m->pool) held |= (e.r == keys[k].r);
        if (held) res_missed[keys[k].r] = true;
    }
    for (int r = 0; r < R; ++r) m->miss_streak[r] = res_missed[r] ? m->miss_streak[r] + 1 : 0;
    std::vector<char> inline_key(keys.size(), 0);
    int need = 0;
    for (size_t k = 0; k < keys.size(); ++k) {
        // P == 1: evaluating a Breit-Wigner in registers is cheaper than reading its 16 B column on B200, so
        // unless the caller forces the pool (mode 1) no column is stored or read at all
        const bool want_inline = m->stream_inline && !m->want_matrix;
        inline_key[k] = want_inline;
        if (!want_inline) ++need;
    }
    amp_status st = ensure_pool(m, need);
    if (st != AMP_OK) return st;
    if (need > 0) {
        // re-resolve hits (ensure_pool may have resized the table) and give misses the least recently used slots
        for (size_t k = 0; k < keys.size(); ++k) {
            keyslot[k] = -1;
            for (int sidx = 0; sidx < (int)m->pool.size(); ++sidx) {
                const PoolEntry& e = m->pool[sidx];
                if (e.r == keys[k].r && e.mass == keys[k].mass && e.width == keys[k].width) { keyslot[k] = sidx; break; }
            }
            if (keyslot[k] >= 0) m->pool[keyslot[k]].last_used = m->call_id;
        }
        for (size_t k = 0; k < keys.size(); ++k) {
            if (keyslot[k] >= 0 || inline_key[k]) continue;
            int best = -1;
            for (int sidx = 0; sidx < (int)m->pool.size(); ++sidx)
                if (m->pool[sidx].last_used != m->call_id && (best < 0 || m->pool[sidx].last_used < m->pool[best].last_used)) best = sidx;
            if (best < 0) return fail(m, AMP_ERR_NOMEM, "amp_set_params: lineshape column pool exhausted");
            m->pool[best] = PoolEntry{keys[k].r, keys[k].mass, keys[k].width, false, false, m->call_id};
            keyslot[k] = best;
        }
    }
    m->colidx.assign((size_t)P * R, COL_NONE);
    for (int r = 0; r < R; ++r) m->was_inline[r] = false;
    for (int p = 0; p < P; ++p)
        for (int r = 0; r < R; ++r) {
            const int k = keyidx[(size_t)p * R + r];
            if (k >= 0) m->colidx[(size_t)p * R + r] = inline_key[k] ? COL_INLINE : keyslot[k];
            if (k >= 0 && inline_key[k]) m->was_inline[r] = true;
        }
    return AMP_OK;
}

namespace {

// Recompute the columns of `d` that the current points need and that are not valid yet.
amp_status refresh_columns(amp_model* m, Dataset& d, bool is_norm, cudaStream_t s) {
    std::vector<LineshapeJob> jobs;
    std::vector<char> seen(m->pool.size(), 0);
    for (int p = 0; p < m->P; ++p)
        for (int r = 0; r < m->R; ++r) {
            const int sidx = m->colidx[(size_t)p * m->R + r];
            if (sidx < 0 || seen[sidx]) continue;
            seen[sidx] = 1;
            PoolEntry& e = m->pool[sidx];
            if (is_norm ? e.valid_norm : e.valid_data) continue;
            LineshapeJob j;
            make_line_const(m, e.r, e.mass, e.width, &j.lc);
            j.column = sidx;
            jobs.push_back(j);
            (is_norm ? e.valid_norm : e.valid_data) = true;
        }
    if (jobs.empty() || d.n == 0) return AMP_OK;
    CK(launch_lineshape(d, jobs.data(), (int)jobs.size(), s));
    m->stat_launches += ((int)jobs.size() + MAX_LINE_JOBS - 1) / MAX_LINE_JOBS;
    m->stat_columns += (int)jobs.size();
    return AMP_OK;
}

// Arguments of the streaming kernel for point p on dataset d: resonances grouped by spin, then by
// radius (a barrier group shares its Blatt-Weisskopf factors and momentum powers).
void fill_stream_args(const amp_model* m, const Dataset& d, int p, int mode, StreamArgs* a, int* ent_of_res, int* grp_of_res) {
    std::memset(a, 0, sizeof(*a));
    int t = 0, g = 0;
    auto add_groups = [&](int kind, int J) {
        std::vector<char> done(m->R, 0);
        for (int r = 0; r < m->R; ++r) {
            if (done[r] || m->res[r].kind != kind || m->res[r].J != J) continue;
            BarrierGroup& grp = a->grp[g++];
            grp.r2 = m->res[r].radius * m->res[r].radius;
            grp.first = t;
            for (int r2 = r; r2 < m->R; ++r2) {
                if (done[r2] || m->res[r2].kind != kind || m->res[r2].J != J || m->res[r2].radius != m->res[r].radius) continue;
                done[r2] = 1;
                LineConst lc;
                make_line_const(m, r2, m->mw[((size_t)p * m->R + r2) * 2], m->mw[((size_t)p * m->R + r2) * 2 + 1], &lc);
                if (ent_of_res) { ent_of_res[r2] = t; grp_of_res[r2] = g - 1; }
                ResEntry& e = a->ent[t++];
                e.kN = lc.kN; e.kG = lc.kG; e.M2 = lc.M2;
                const double* cp = &m->couplings[((size_t)p * m->K + m->slot0[r2]) * 2];
                if (J == 0 && kind == AMP_KSTAR) {   // one slot (a spin-0 Z keeps three: lambda' = +-1 multiply a zero d function)
                    e.c0 = make_double2(cp[0], cp[1]);
                    e.cm = e.cp = make_double2(0, 0);
                } else {
                    e.cm = make_double2(cp[0], cp[1]); e.c0 = make_double2(cp[2], cp[3]); e.cp = make_double2(cp[4], cp[5]);
                }
                const size_t ci = (size_t)p * m->R + r2;
                const int sidx = ci < m->colidx.size() ? m->colidx[ci] : -1;
                e.column = (sidx >= 0 && !m->stream_inline) ? sidx : -1;
                if (e.column < 0) {   // lineshape in registers: fold its constant kN into the couplings
                    e.cm.x *= lc.kN; e.cm.y *= lc.kN; e.c0.x *= lc.kN; e.c0.y *= lc.kN; e.cp.x *= lc.kN; e.cp.y *= lc.kN;
                }
            }
            grp.count = t - grp.first;
        }
    };
    a->shape_fixed = 1;
    for (int J = 0; J < 5; ++J) { a->gstart[J] = g; add_groups(AMP_KSTAR, J); }
    for (int zc = 0; zc < NZCLASS; ++zc) { a->gstart[5 + zc] = g; add_groups(z_class_kind(zc), z_class_J(zc)); }
    a->gstart[NSPIN] = g;
    a->lass0 = t;
    for (int r = 0; r < m->R; ++r) {
        if (m->res[r].kind != AMP_LASS) continue;
        LineConst lc;
        make_line_const(m, r, m->mw[((size_t)p * m->R + r) * 2], m->mw[((size_t)p * m->R + r) * 2 + 1], &lc);
        if (ent_of_res) { ent_of_res[r] = t; grp_of_res[r] = 0; }
        ResEntry& e = a->ent[t++];
        e.kN = 1.0; e.kG = lc.kG; e.M2 = lc.M2;
        const double* cp = &m->couplings[((size_t)p * m->K + m->slot0[r]) * 2];
        e.c0 = make_double2(cp[0], cp[1]);
        e.cm = e.cp = make_double2(0, 0);
        const size_t ci = (size_t)p * m->R + r;
        const int sidx = ci < m->colidx.size() ? m->colidx[ci] : -1;
        e.column = (sidx >= 0 && !m->stream_inline) ? sidx : -1;
    }
    a->nlass = t - a->lass0;
    for (int sp = 0; sp < NSPIN; ++sp) {
        const int ng = a->gstart[sp + 1] - a->gstart[sp];
        a->shape[sp] = 0;
        for (int gg = a->gstart[sp]; gg < a->gstart[sp + 1]; ++gg) a->shape[sp] += a->grp[gg].count;
        if (ng > 1) a->shape_fixed = 0;
        a->r2_spin[sp] = ng >= 1 ? a->grp[a->gstart[sp]].r2 : 0.0;
    }
    a->cconst = make_double2(0, 0);
    for (int r = 0; r < m->R; ++r)
        if (m->res[r].kind == AMP_CONST) {
            const double* cp = &m->couplings[((size_t)p * m->K + m->slot0[r]) * 2];
            a->cconst.x += cp[0]; a->cconst.y += cp[1];
        }
    a->cache = d.cache;
    a->ncolw = (m->has_z ? NCOL_ALL : NCOL_K) + 1;
    a->cols = d.cols;
    a->n = d.n;
    a->npad = d.npad;
    a->flag = m->d_flag;
    a->mode = mode;
}

// plain [column][n] copy of the tiled cache (amp_dump_cache)
__global__ void k_dump_cache(const double* __restrict__ cache, int ncolw, int ncols, long long n, double* __restrict__ out) {
    for (long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x; idx < n * ncols; idx += (long long)gridDim.x * blockDim.x) {
        const int c = (int)(idx / n);
        const long long i = idx % n;
        out[idx] = cache[cache_idx(ncolw, c, i)];
    }
}

// nll[p] = -(sum_i log S_i + sum_i log eps_i) + N log I(p), I(p) = sum_j w_j S_j / sum_j w_j
__global__ void k_nll_final(const double* __restrict__ sums, int P, double n_data, double sum_log_eff, double wsum, int want_nll,
                            double* __restrict__ result) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= P) return;
    const double I = sums[P + p] / wsum;
    result[P + p] = I;
    if (want_nll == 2) {          // Eq. 14: sums[p] = sum_i log f_i already holds efficiency, integral and background
        double v = -sums[p];
        if (!isfinite(v) || !(I > 0.0)) v = INFINITY;
        result[p] = v;
    } else if (want_nll) {
        double v = -(sums[p] + sum_log_eff) + n_data * log(I);
        if (!isfinite(v) || !(I > 0.0)) v = INFINITY;
        result[p] = v;
    }
}

// ---- batched (P > 1) path: host-side plan of one launch over points [p0, p0 + Pc) --------------------------------
struct BatchPlan {
    std::vector<double> Adense;
    std::vector<int2> entries, items;
    std::vector<double> itemA;
    int item_start[9];
    int nent;
    std::vector<int> colu;   // distinct pool columns; entries[].x indexes this list
    int point_of_row[BATCH_POINTS];
};

int slot_code(const amp_model* m, int r, int lam) { return (m->res[r].kind << 8) | (m->res[r].J << 4) | (lam + 1); }

// false if the model or the points do not fit the DMMA kernel (too many couplings or extended entries)
bool build_batch_plan(const amp_model* m, int p0, int Pc, BatchPlan* bp) {
    const int R = m->R, K = m->K;
    if (2 * K > BATCH_NKT * 4 || Pc > BATCH_POINTS) return false;
    std::vector<int> slot_res(K), slot_lam(K);
    for (int r = 0; r < R; ++r) {
        const int ns = (kind_is_z(m->res[r].kind) || (m->res[r].kind == AMP_KSTAR && m->res[r].J >= 1)) ? 3 : 1;
        for (int j = 0; j < ns; ++j) { slot_res[m->slot0[r] + j] = r; slot_lam[m->slot0[r] + j] = ns == 3 ? j - 1 : 0; }
    }
    const int nbase = BATCH_NKT * 2;   // complex base entries incl. padding
    bp->entries.assign(nbase, make_int2(-1, 0));
    for (int k = 0; k < K; ++k) {
        const int r = slot_res[k];
        const int col = m->res[r].kind == AMP_CONST ? -2 : m->colidx[(size_t)p0 * R + r];
        if (col == COL_NONE || col == COL_INLINE) return false;   // no column held for this lineshape: not this path
        bp->entries[k] = make_int2(col, slot_code(m, r, slot_lam[k]));
    }
    bp->Adense.assign((size_t)16 * 2 * BATCH_NKT * 32, 0.0);
    struct Item { int row0, octet; double a[2][32]; };
    std::vector<Item> items;
    auto put = [](double (*a)[32], int row, int kk, double cre, double cim) {   // realified rows kk (b_re), kk+1 (b_im) of one k-tile
        a[0][row * 4 + (kk & 3)] = cre;  a[0][row * 4 + (kk & 3) + 1] = -cim;   // Re A
        a[1][row * 4 + (kk & 3)] = cim;  a[1][row * 4 + (kk & 3) + 1] = cre;    // Im A
    };
    // Rows of the GEMM: points that use a lineshape column other than the base one own extra (sparse) blocks; deal
    // them round-robin over the eight warps so every warp multiplies about the same number of blocks.
    std::vector<int> row_of(Pc, -1);
    {
        int next_row[8], nvar = 0;
        for (int w = 0; w < 8; ++w) next_row[w] = 16 * w;
        std::vector<char> is_var(Pc, 0);
        for (int q = 0; q < Pc; ++q)
            for (int r = 0; r < R; ++r)
                if (m->res[r].kind != AMP_CONST && m->colidx[(size_t)(p0 + q) * R + r] != m->colidx[(size_t)p0 * R + r]) is_var[q] = 1;
        for (int q = 0; q < Pc; ++q)
            if (is_var[q]) { const int w = nvar++ % 8; row_of[q] = next_row[w]++; }
        int w = 0;
        for (int q = 0; q < Pc; ++q) {
            if (is_var[q]) continue;
            while (next_row[w] >= 16 * (w + 1)) w = (w + 1) % 8;
            row_of[q] = next_row[w]++;
            w = (w + 1) % 8;
        }
        for (int i = 0; i < BATCH_POINTS; ++i) bp->point_of_row[i] = -1;
        for (int q = 0; q < Pc; ++q) bp->point_of_row[row_of[q]] = q;
    }
    for (int q = 0; q < Pc; ++q) {
        const int p = p0 + q, o = row_of[q] / 8, row = row_of[q] % 8;
        for (int k = 0; k < K; ++k) {
            const int r = slot_res[k];
            const double cre = m->couplings[((size_t)p * K + k) * 2], cim = m->couplings[((size_t)p * K + k) * 2 + 1];
            const int col = m->res[r].kind == AMP_CONST ? -2 : m->colidx[(size_t)p * R + r];
            if (col == COL_NONE || col == COL_INLINE) return false;   // no column held for this lineshape: not this path
            int e = k;
            if (col != bp->entries[k].x) {   // this point uses another lineshape column for this slot: extended entry
                e = -1;
                for (int j = nbase; j < (int)bp->entries.size(); ++j)
                    if (bp->entries[j].x == col && bp->entries[j].y == bp->entries[k].y) { e = j; break; }
                if (e < 0) { bp->entries.push_back(make_int2(col, bp->entries[k].y)); e = (int)bp->entries.size() - 1; }
            }
            const int kk = 2 * e;   // realified row of b_re
            if (e < nbase) {
                double (*a)[32] = nullptr;
                double tmp[2][32] = {};
                a = tmp;
                put(a, row, kk, cre, cim);
                const int kt = kk / 4;
                for (int ri = 0; ri < 2; ++ri)
                    for (int c = 0; c < 2; ++c) {
                        const int lane = row * 4 + (kk & 3) + c;
                        bp->Adense[((((size_t)o * 2 + ri) * BATCH_NKT) + kt) * 32 + lane] = tmp[ri][lane];
                    }
            } else {
                const int row0 = kk / 4 * 4;
                Item* itp = nullptr;
                for (auto& it : items)
                    if (it.row0 == row0 && it.octet == o) { itp = &it; break; }
                if (!itp) { items.push_back(Item{row0, o, {}}); itp = &items.back(); }
                put(itp->a, row, kk, cre, cim);
            }
        }
    }
    if (bp->entries.size() & 1) bp->entries.push_back(make_int2(-1, 0));
    bp->nent = (int)bp->entries.size();
    // pool columns -> indices into the list of distinct columns the kernel stages per tile
    bp->colu.clear();
    for (auto& en : bp->entries) {
        if (en.x < 0) continue;
        int j = 0;
        for (; j < (int)bp->colu.size(); ++j)
            if (bp->colu[j] == en.x) break;
        if (j == (int)bp->colu.size()) bp->colu.push_back(en.x);
        en.x = j;
    }
    if (!batch_fits(bp->nent, (int)bp->colu.size())) return false;
    // items grouped by owning warp (octet / 2)
    bp->items.clear();
    bp->itemA.clear();
    for (int w = 0; w < 8; ++w) {
        bp->item_start[w] = (int)bp->items.size();
        for (auto& it : items)
            if (it.octet / 2 == w) {
                bp->items.push_back(make_int2(it.row0, it.octet & 1));
                for (int ri = 0; ri < 2; ++ri) bp->itemA.insert(bp->itemA.end(), it.a[ri], it.a[ri] + 32);
            }
    }
    bp->item_start[8] = (int)bp->items.size();
    return true;
}

// upload a plan and launch the DMMA kernel on dataset d; partial rows [row0, row0 + Pc)
amp_status run_batch(amp_model* m, const Dataset& d, const BatchPlan& bp, int Pc, int mode, size_t plan_off, double* partial, cudaStream_t s,
                     int* grid_out) {
    const size_t bA = bp.Adense.size() * sizeof(double), bE = bp.entries.size() * sizeof(int2), bI = bp.items.size() * sizeof(int2),
                 bIA = bp.itemA.size() * sizeof(double);
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    const size_t oA = plan_off, oE = oA + al(bA), oI = oE + al(bE), oIA = oI + al(bI), end = oIA + al(bIA);
    if (end > m->plan_cap) return fail(m, AMP_ERR_NOMEM, "batch plan buffer too small");
    std::memcpy(m->h_plan + oA, bp.Adense.data(), bA);
    std::memcpy(m->h_plan + oE, bp.entries.data(), bE);
    if (bI) std::memcpy(m->h_plan + oI, bp.items.data(), bI);
    if (bIA) std::memcpy(m->h_plan + oIA, bp.itemA.data(), bIA);
    CK(cudaMemcpyAsync(m->d_plan + plan_off, m->h_plan + plan_off, end - plan_off, cudaMemcpyHostToDevice, s));
    BatchArgs a{};
    a.cache = d.cache; a.ncolw = d.ncache + 1; a.cols = d.cols; a.n = d.n; a.npad = d.npad;
    a.Adense = reinterpret_cast<const double*>(m->d_plan + oA);
    a.entries = reinterpret_cast<const int2*>(m->d_plan + oE);
    a.items = reinterpret_cast<const int2*>(m->d_plan + oI);
    a.itemA = reinterpret_cast<const double*>(m->d_plan + oIA);
    for (int w = 0; w < 9; ++w) a.item_start[w] = bp.item_start[w];
    for (int i = 0; i < BATCH_POINTS; ++i) a.point_of_row[i] = (short)bp.point_of_row[i];
    a.ncolu = (int)bp.colu.size();
    for (int j = 0; j < a.ncolu; ++j) a.colu[j] = bp.colu[j];
    a.nent = bp.nent; a.nkt = BATCH_NKT; a.P = Pc; a.have_z = m->has_z ? 1 : 0; a.mode = mode;
    a.partial = partial; a.partial_stride = PARTIAL_STRIDE; a.flag = m->d_flag;
    const int grid = batch_grid(d.n);
    CK(launch_batch(a, grid, s));
    m->stat_launches++;
    *grid_out = grid;
    return AMP_OK;
}

// ---- normalisation through the matrix M (a4) -------------------------------------------------------------------
struct HerkPlan {
    std::vector<int2> entries;          // (index into colu | -1 | -2, angular code), nent a multiple of 4
    std::vector<int> colu;
    std::vector<double2> C;             // [P][nent] coefficient of every entry at every point
    std::vector<int2> tiles;            // needed (I <= J) tiles, grouped by owning warp
    std::vector<int4> runs;             // [8][nrun] (I, J0, J1, 0)
    std::vector<int2> runs_out;         // [8][nrun] tile indices of the two products, -1: padding
    int nrun;
    std::vector<amp_model::GramKey> sig;
    int nent;
};

// Extended basis over ALL P points (base = the columns of point 0) and the Gram tiles some point needs.
bool build_herk_plan(const amp_model* m, HerkPlan* hp, int pbase = 0, int npts = -1) {
    const int R = m->R, K = m->K, P = npts < 0 ? m->P : npts;
    std::vector<int> slot_res(K), slot_lam(K);
    for (int r = 0; r < R; ++r) {
        const int ns = (kind_is_z(m->res[r].kind) || (m->res[r].kind == AMP_KSTAR && m->res[r].J >= 1)) ? 3 : 1;
        for (int j = 0; j < ns; ++j) { slot_res[m->slot0[r] + j] = r; slot_lam[m->slot0[r] + j] = ns == 3 ? j - 1 : 0; }
    }
    std::vector<int2> ent(K);           // pool column (or -2) and code, base entries
    for (int k = 0; k < K; ++k) {
        const int r = slot_res[k];
        const int col = m->res[r].kind == AMP_CONST ? -2 : m->colidx[(size_t)pbase * R + r];
        if (col == COL_NONE || col == COL_INLINE) return false;   // no column held for this lineshape: not this path
        ent[k] = make_int2(col, slot_code(m, r, slot_lam[k]));
    }
    std::vector<std::vector<std::pair<int, double2>>> coef(P);
    for (int q = 0; q < P; ++q)
        for (int k = 0; k < K; ++k) {
            const int p = pbase + q;
            const int r = slot_res[k];
            const int col = m->res[r].kind == AMP_CONST ? -2 : m->colidx[(size_t)p * R + r];
            if (col == COL_NONE || col == COL_INLINE) return false;   // no column held for this lineshape: not this path
            int e = k;
            if (col != ent[k].x) {
                e = -1;
                for (int j = K; j < (int)ent.size(); ++j)
                    if (ent[j].x == col && ent[j].y == ent[k].y) { e = j; break; }
                if (e < 0) { ent.push_back(make_int2(col, ent[k].y)); e = (int)ent.size() - 1; }
            }
            coef[q].push_back({e, make_double2(m->couplings[((size_t)p * K + k) * 2], m->couplings[((size_t)p * K + k) * 2 + 1])});
        }
    while (ent.size() % 4) ent.push_back(make_int2(-1, 0));
    hp->nent = (int)ent.size();
    // signature: what each entry is, independent of pool slot numbers
    hp->sig.clear();
    for (auto& en : ent) {
        amp_model::GramKey g{-1, 0, 0, en.y};
        if (en.x >= 0) { g.r = m->pool[en.x].r; g.mass = m->pool[en.x].mass; g.width = m->pool[en.x].width; }
        else g.r = en.x;
        hp->sig.push_back(g);
    }
    hp->colu.clear();
    hp->entries = ent;
    for (auto& en : hp->entries) {
        if (en.x < 0) continue;
        int j = 0;
        for (; j < (int)hp->colu.size(); ++j)
            if (hp->colu[j] == en.x) break;
        if (j == (int)hp->colu.size()) hp->colu.push_back(en.x);
        en.x = j;
    }
    if (!batch_fits(hp->nent, (int)hp->colu.size())) return false;
    hp->C.assign((size_t)P * hp->nent, make_double2(0, 0));
    const int NT = hp->nent / 4;        // row tiles (8 realified rows = 4 complex entries)
    std::vector<char> need((size_t)NT * NT, 0);
    for (int p = 0; p < P; ++p) {
        std::vector<char> used(NT, 0);
        for (auto& ce : coef[p]) {
            hp->C[(size_t)p * hp->nent + ce.first] = ce.second;
            used[ce.first / 4] = 1;   // structural: every entry the point references, whatever its coupling's value
        }
        for (int I = 0; I < NT; ++I)
            if (used[I])
                for (int J = I; J < NT; ++J)
                    if (used[J]) need[(size_t)I * NT + J] = 1;
    }
    std::vector<int2> all;
    for (int I = 0; I < NT; ++I)
        for (int J = I; J < NT; ++J)
            if (need[(size_t)I * NT + J]) all.push_back(make_int2(I, J));
    hp->tiles = all;
    // runs: one row tile with two of its column tiles (three fragment loads feed two DMMAs); dealt to the warps in
    // contiguous, equally long chunks, padded with dummy runs whose results are dropped
    std::vector<int4> runs;
    std::vector<int2> outs;
    for (size_t i = 0; i < all.size();) {
        if (i + 1 < all.size() && all[i + 1].x == all[i].x) {
            runs.push_back(make_int4(all[i].x, all[i].y, all[i + 1].y, 0));
            outs.push_back(make_int2((int)i, (int)i + 1));
            i += 2;
        } else {
            runs.push_back(make_int4(all[i].x, all[i].y, all[i].y, 0));
            outs.push_back(make_int2((int)i, -1));
            i += 1;
        }
    }
    int nrun = ((int)runs.size() + 7) / 8;
    nrun = (nrun + 1) / 2 * 2;
    if (nrun < 2) nrun = 2;
    if (nrun > herk_max_runs()) return false;
    hp->nrun = nrun;
    hp->runs.assign((size_t)8 * nrun, make_int4(0, 0, 0, 0));
    hp->runs_out.assign((size_t)8 * nrun, make_int2(-1, -1));
    const int per = ((int)runs.size() + 7) / 8;
    for (size_t i = 0; i < runs.size(); ++i) {
        const int w = (int)i / per, r = (int)i % per;
        hp->runs[(size_t)w * nrun + r] = runs[i];
        hp->runs_out[(size_t)w * nrun + r] = outs[i];
    }
    return true;
}

bool gram_hit(const amp_model* m, const HerkPlan& hp) {
    if (!m->gram_valid || m->gram_KP != hp.nent * 2 || m->gram_sig.size() != hp.sig.size() || m->gram_tiles.size() != hp.tiles.size()) return false;
    for (size_t i = 0; i < hp.sig.size(); ++i) {
        const auto &a = m->gram_sig[i], &b = hp.sig[i];
        if (a.r != b.r || a.mass != b.mass || a.width != b.width || a.code != b.code) return false;
    }
    for (size_t i = 0; i < hp.tiles.size(); ++i)
        if (m->gram_tiles[i].x != hp.tiles[i].x || m->gram_tiles[i].y != hp.tiles[i].y) return false;
    return true;
}

// G' (re)built if the signature changed; then out[p] = c(p)^H M c(p) (unnormalised: sum_j w_j S_j) for all points
amp_status norm_via_matrix(amp_model* m, const HerkPlan& hp, double* d_out, cudaStream_t s) {
    const int KP = hp.nent * 2, ntile = (int)hp.tiles.size(), P = (int)(hp.C.size() / hp.nent);
    bool hit = gram_hit(m, hp);
    auto al = [](size_t x) { return (x + 255) / 256 * 256; };
    const size_t bE = hp.entries.size() * sizeof(int2), bT = hp.tiles.size() * sizeof(int2), bC = hp.C.size() * sizeof(double2);
    const size_t bR = hp.runs.size() * sizeof(int4), bRO = hp.runs_out.size() * sizeof(int2);
    const size_t oE = 0, oT = al(bE), oC = oT + al(bT), oR = oC + al(bC), oRO = oR + al(bR), end = oRO + al(bRO);
    if (end > m->hk_cap) {
        if (m->d_hk) cudaFree(m->d_hk);
        if (m->h_hk) cudaFreeHost(m->h_hk);
        m->d_hk = m->h_hk = nullptr;
        m->hk_cap = 0;
        CK(cudaMalloc(&m->d_hk, end * 2));
        CK(cudaMallocHost(&m->h_hk, end * 2));
        m->hk_cap = end * 2;
    }
    if ((size_t)KP > m->gram_cap_KP || (size_t)ntile > m->gram_cap_tiles) {
        for (double** b : {&m->d_G, &m->d_gt, &m->d_gpartial}) { if (*b) cudaFree(*b); *b = nullptr; }
        m->gram_valid = false;
        hit = false;
        m->gram_cap_KP = KP;
        m->gram_cap_tiles = ntile;
        CK(cudaMalloc(&m->d_G, sizeof(double) * (size_t)KP * KP));
        CK(cudaMalloc(&m->d_gt, sizeof(double) * (size_t)ntile * 64));
        CK(cudaMalloc(&m->d_gpartial, sizeof(double) * (size_t)herk_grid_max() * ntile * 64));
    }
    std::memcpy(m->h_hk + oE, hp.entries.data(), bE);
    std::memcpy(m->h_hk + oT, hp.tiles.data(), bT);
    std::memcpy(m->h_hk + oC, hp.C.data(), bC);
    std::memcpy(m->h_hk + oR, hp.runs.data(), bR);
    std::memcpy(m->h_hk + oRO, hp.runs_out.data(), bRO);
    CK(cudaMemcpyAsync(m->d_hk, m->h_hk, end, cudaMemcpyHostToDevice, s));
    if (!hit) {
        HerkArgs h{};
        const Dataset& d = m->norm;
        h.b.cache = d.cache; h.b.ncolw = d.ncache + 1; h.b.cols = d.cols; h.b.n = d.n; h.b.npad = d.npad;
        h.b.entries = reinterpret_cast<const int2*>(m->d_hk + oE);
        h.b.nent = hp.nent;
        h.b.ncolu = (int)hp.colu.size();
        for (int j = 0; j < h.b.ncolu; ++j) h.b.colu[j] = hp.colu[j];
        h.b.have_z = m->has_z ? 1 : 0;
        h.runs = reinterpret_cast<const int4*>(m->d_hk + oR);
        h.runs_out = reinterpret_cast<const int2*>(m->d_hk + oRO);
        h.nrun = hp.nrun;
        h.ntile = ntile;
        h.partial = m->d_gpartial;
        const int grid = herk_grid(d.n, hp.nent, (int)hp.colu.size());
        CK(launch_herk(h, grid, s));
        CK(launch_herk_finish(m->d_gpartial, grid, ntile, reinterpret_cast<const int2*>(m->d_hk + oT), KP, m->d_gt, m->d_G, s));
        m->stat_launches += 3;
        m->gram_sig = hp.sig;
        m->gram_tiles = hp.tiles;
        m->gram_KP = KP;
        m->gram_valid = true;
        m->gram_p1 = false;   // (evaluate() marks single-point matrices)
        m->stat_gram_built = 1;
    }
    CK(launch_quadform(m->d_G, KP, reinterpret_cast<const double2*>(m->d_hk + oC), hp.nent, P, d_out, s));
    m->stat_launches++;
    return AMP_OK;
}

amp_status evaluate(amp_model* m, bool want_nll, double* h_nll, double* h_I, cudaStream_t s) {
    if (!m->norm.loaded) return fail(m, AMP_ERR_STATE, "no normalisation sample loaded (amp_load_norm)");
    if (want_nll && !m->data.loaded) return fail(m, AMP_ERR_STATE, "no data events loaded (amp_load_events)");
    if (m->P < 1) return fail(m, AMP_ERR_STATE, "no parameters set (amp_set_params)");
    const int P = m->P;
    m->stat_launches = m->stat_columns = 0;
    m->stat_norm_path = 1;
    amp_status st = ensure_pool(m, 0);
    if (st != AMP_OK) return st;
    m->ev_valid = false;
    if (m->has_bkg && want_nll) {
        // Eq. 14: f_i = purity eps_i S_i / I + (1 - purity) b_i needs I before the data pass: per point one
        // normalisation launch, a fixed-order reduction to sum_j w_j S_j on the device, then the data launch that reads it.
        if (!m->stream_inline) {
            st = refresh_columns(m, m->data, false, s); if (st != AMP_OK) return st;
            st = refresh_columns(m, m->norm, true, s); if (st != AMP_OK) return st;
        }
        CK(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
        const int gd = stream_grid(m->data.n, m->has_z, MODE_DATA), gn = stream_grid(m->norm.n, m->has_z, MODE_NORM);
        StreamArgs a;
        for (int p = 0; p < P; ++p) {
            fill_stream_args(m, m->norm, p, MODE_NORM, &a);
            a.partial = m->d_partial + (size_t)(P + p) * PARTIAL_STRIDE;
            CK(launch_stream(a, gn, s));
        }
        CK(launch_finalize(m->d_partial + (size_t)P * PARTIAL_STRIDE, gn, PARTIAL_STRIDE, P, m->d_sums + P, s));
        for (int p = 0; p < P; ++p) {
            if (m->data.n == 0) { CK(cudaMemsetAsync(m->d_partial + (size_t)p * PARTIAL_STRIDE, 0, sizeof(double), s)); continue; }
            fill_stream_args(m, m->data, p, MODE_DATA_BKG, &a);
            a.partial = m->d_partial + (size_t)p * PARTIAL_STRIDE;
            a.bkg = m->d_bkg; a.purity = m->purity; a.sum_wS = m->d_sums + P + p; a.wsum = m->norm.wsum;
            CK(launch_stream(a, gd, s));
        }
        CK(launch_finalize(m->d_partial, m->data.n > 0 ? gd : 1, PARTIAL_STRIDE, P, m->d_sums, s));
        k_nll_final<<<(P + 127) / 128, 128, 0, s>>>(m->d_sums, P, (double)m->data.n, 0.0, m->norm.wsum, 2, m->d_result);
        CK(cudaGetLastError());
        m->stat_launches = 2 * P + 3;
        m->stat_norm_path = 6;
        m->fused_valid = false;
        CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * 2 * P, cudaMemcpyDeviceToHost, s));
        CK(cudaMemcpyAsync(m->h_pinned + 2 * P, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost, s));
        CK(cudaStreamSynchronize(s));
        int flag;
        std::memcpy(&flag, m->h_pinned + 2 * P, sizeof(int));
        bool bad = flag != 0;
        for (int p = 0; p < P; ++p) {
            h_nll[p] = m->h_pinned[p]; bad |= !std::isfinite(h_nll[p]);
            if (h_I) h_I[p] = m->h_pinned[P + p];
        }
        m->last_slog.assign(P, 0.0); m->last_swS.assign(P, 0.0);
        if (bad) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
        return AMP_OK;
    }
    bool deltaf_tripped = false;
    if (m->use_deltaf) {
        // Gradient batch of the paper's resonance lists: ONE launch of the shape-specialised kernel (deltaf.cu) for all points.
        DeltaFArgs& d = m->deltaf;
        fill_stream_args(m, m->data, 0, MODE_FUSED, &d.a);
        d.a.cache2 = m->norm.cache; d.a.n2 = m->norm.n; d.a.npad2 = m->norm.npad;
        d.a.ticket = m->d_ticket;
        d.a.sum_log_eff = m->data.loaded ? m->data.wsum : 0.0;
        d.a.wsum = m->norm.wsum;
        if (!want_nll) d.a.n = 0;
        d.P = P;
        d.partial = m->d_partial;
        d.stride = PARTIAL_STRIDE;
        d.want_nll = want_nll ? 1 : 0;
        // Result block [4 P + 2]: as for the fused step, mapped host memory that the last CTA fills and stamps (the host spins on the
        // stamp: no D2H copy, no stream-synchronise wake-up)
        const double* res = m->h_pinned;
        if (m->zero_copy) { m->zcb_seq += 1.0; d.result = m->h_zcb; d.seq = m->zcb_seq; res = m->h_zcb; }
        else { d.result = m->d_result; d.seq = 0.0; }
        m->ring_last = (m->ring_last + 1) % amp_model::RING;
        m->ring_calls++;
        CK(cudaEventRecord(m->ring[2 * m->ring_last], s));
        // The normalisation events in kernels of their own first (deltan.cu: their sums do not depend on the point and live in
        // registers there, two passes), then the data events; the last launch's last CTA forms NLL(p), I(p) from all.  Batch mode 4: one launch.
        const bool split = m->batch_mode != 4 && m->norm.n > 0;
        d.npartial = m->d_npartial;
        d.norm_tot = split ? m->d_ntot : nullptr;
        if (split) {
            CK(launch_deltan(d, deltan_grid(d.a.n2), 0, s));
            CK(cudaEventRecord(m->ev[1], s));
            CK(launch_deltan(d, deltan_grid(d.a.n2), 1, s));
            CK(cudaEventRecord(m->ev[2], s));
            d.a.n2 = 0;
        }
        CK(launch_deltaf(d, deltaf_grid(d.a.n, d.a.n2), s));
        CK(cudaEventRecord(m->ring[2 * m->ring_last + 1], s));
        m->split_valid = split;
        m->stat_launches = split ? 3 : 1;
        if (m->zero_copy) {
            volatile double* stamp = m->h_zcb + 4 * P + 1;
            for (unsigned spins = 0; *stamp != m->zcb_seq; ++spins) {
                if ((spins & 0x3fff) == 0x3fff) {   // every 16k spins: has the stream failed or finished without the stamp?
                    const cudaError_t q = cudaStreamQuery(s);
                    if (q != cudaErrorNotReady) { if (q != cudaSuccess) return cuda_fail(m, q, "gradient batch"); if (*stamp == m->zcb_seq) break; return fail(m, AMP_ERR_CUDA, "gradient batch finished without a result"); }
                }
            }
            std::atomic_thread_fence(std::memory_order_acquire);
        } else {
            CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * (4 * P + 1), cudaMemcpyDeviceToHost, s));
            CK(cudaStreamSynchronize(s));
        }
        if (res[2 * P] < 1024.0) {
            m->last_slog.assign(res + 2 * P + 1, res + 3 * P + 1);
            m->last_swS.assign(res + 3 * P + 1, res + 4 * P + 1);
            m->stat_norm_path = 9;
            m->fused_valid = true;
            bool bad = res[2 * P] != 0.0;
            for (int p = 0; p < P; ++p) {
                if (h_nll) { h_nll[p] = res[p]; bad |= !std::isfinite(h_nll[p]); }
                if (h_I) { h_I[p] = res[P + p]; bad |= !(h_I[p] > 0) || !std::isfinite(h_I[p]); }
            }
            if (bad) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
            return AMP_OK;
        }
        // a step so large that some S(p) / S(0) left [0.5, 1.5]: the general kernel below, amplitudes summed term by term
        m->stat_deltaf_guard++;
        deltaf_tripped = true;
        m->ring_calls--;
        m->ring_last = (m->ring_last + amp_model::RING - 1) % amp_model::RING;
    }
    if (m->use_delta && !m->delta_plan_built) {
        if (build_delta_plan(m)) {
            m->delta_plan_built = true;
        } else {
            // a batch the specialised kernel accepted but the general one cannot compile: plan the call again without the former
            const std::vector<double> c = m->couplings, w = m->mw;
            m->no_deltaf_once = true;
            const amp_status rs = amp_set_params(m, P, c.data(), w.data());
            m->no_deltaf_once = false;
            if (rs != AMP_OK) return rs;
            return evaluate(m, want_nll, h_nll, h_I, s);
        }
    }
    if (m->use_delta) {
        // Gradient batch: one fused launch per chunk of <= 128 points besides point 0 (delta.cu)
        int ent_of_res[AMP_MAX_RESONANCES], grp_of_res[AMP_MAX_RESONANCES];
        DeltaArgs d{};
        fill_stream_args(m, m->data, 0, MODE_FUSED, &d.a, ent_of_res, grp_of_res);
        d.a.cache2 = m->norm.cache; d.a.n2 = m->norm.n; d.a.npad2 = m->norm.npad;
        d.a.ticket = m->d_ticket;
        d.a.sum_log_eff = m->data.loaded ? m->data.wsum : 0.0;
        d.a.wsum = m->norm.wsum;
        if (!want_nll) { d.a.n = 0; }
        d.P = P;
        d.partial = m->d_partial;
        d.stride = PARTIAL_STRIDE;
        d.result = m->d_result;
        d.want_nll = want_nll ? 1 : 0;
        size_t need = 4096;
        for (auto& ch : m->delta_chunks) need += ch.contrib.size() * sizeof(DeltaContrib) + ch.slots.size() * sizeof(double) + ch.nsorted * sizeof(int) + 1024;
        if (need > m->plan_cap) {
            if (m->d_plan) cudaFree(m->d_plan);
            if (m->h_plan) cudaFreeHost(m->h_plan);
            m->d_plan = m->h_plan = nullptr;
            m->plan_cap = 0;
            CK(cudaMalloc(&m->d_plan, need * 2));
            CK(cudaMallocHost(&m->h_plan, need * 2));
            m->plan_cap = need * 2;
        }
        // one upload for all chunks, then one launch per chunk
        auto al = [](size_t x) { return (x + 255) / 256 * 256; };
        size_t off = 0;
        std::vector<size_t> offs;
        for (auto& ch : m->delta_chunks) {
            offs.push_back(off);
            const size_t bC = al(ch.contrib.size() * sizeof(DeltaContrib)), bS = al(ch.slots.size() * sizeof(double) + 8);
            std::memcpy(m->h_plan + off, ch.contrib.data(), ch.contrib.size() * sizeof(DeltaContrib));
            if (!ch.slots.empty()) std::memcpy(m->h_plan + off + bC, ch.slots.data(), ch.slots.size() * sizeof(double));
            int* hp = reinterpret_cast<int*>(m->h_plan + off + bC + bS);
            for (int q = 0; q < ch.nsorted; ++q) hp[q] = q < ch.np ? ch.p0 + q : -1;
            off += bC + bS + al(ch.nsorted * sizeof(int));
        }
        m->ring_last = (m->ring_last + 1) % amp_model::RING;
        m->ring_calls++;
        CK(cudaEventRecord(m->ring[2 * m->ring_last], s));
        CK(cudaMemcpyAsync(m->d_plan, m->h_plan, off, cudaMemcpyHostToDevice, s));
        // The kernel expands single-contribution points around point 0 (S(0) + Re(coef T2) + |coef|^2 n); if some point's density
        // falls below 1e-3 S(0) at some event the guard trips (1024 in the flag word) and the call is repeated with the amplitudes
        // summed term by term.  Gradient steps never trip it; a batch that switches a dominant amplitude off can.
        for (int exact = deltaf_tripped ? 1 : 0; exact < 2; ++exact) {
            for (size_t c = 0; c < m->delta_chunks.size(); ++c) {
                const auto& ch = m->delta_chunks[c];
                const size_t bC = al(ch.contrib.size() * sizeof(DeltaContrib)), bS = al(ch.slots.size() * sizeof(double) + 8);
                d.contrib = reinterpret_cast<const DeltaContrib*>(m->d_plan + offs[c]);
                d.slots = reinterpret_cast<const double*>(m->d_plan + offs[c] + bC);
                d.point_of_sorted = reinterpret_cast<const int*>(m->d_plan + offs[c] + bC + bS);
                d.ncontrib = (int)ch.contrib.size();
                d.nslotwords = (int)ch.slots.size();
                d.nsorted = ch.nsorted;
                d.first_chunk = c == 0 ? 1 : 0;
                CK(launch_delta(d, delta_grid(d.a.n, d.a.n2), s, exact != 0));
                m->stat_launches++;
            }
            CK(cudaEventRecord(m->ring[2 * m->ring_last + 1], s));
            CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * (4 * P + 1), cudaMemcpyDeviceToHost, s));
            CK(cudaStreamSynchronize(s));
            if (m->h_pinned[2 * P] < 1024.0) break;
            m->h_pinned[2 * P] = std::fmod(m->h_pinned[2 * P], 1024.0);   // (after the repeat: its own flag word)
            m->stat_delta_exact++;
        }
        m->last_slog.assign(m->h_pinned + 2 * P + 1, m->h_pinned + 3 * P + 1);
        m->last_swS.assign(m->h_pinned + 3 * P + 1, m->h_pinned + 4 * P + 1);
        m->stat_norm_path = 5;
        m->fused_valid = true;
        bool bad = m->h_pinned[2 * P] != 0.0;
        for (int p = 0; p < P; ++p) {
            if (h_nll) { h_nll[p] = m->h_pinned[p]; bad |= !std::isfinite(h_nll[p]); }
            if (h_I) { h_I[p] = m->h_pinned[P + p]; bad |= !(h_I[p] > 0) || !std::isfinite(h_I[p]); }
        }
        if (bad) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
        return AMP_OK;
    }
    if (want_nll && P == 1 && m->stream_inline && m->want_matrix && m->fused_mode == 0 && m->gram_valid && m->gram_p1 && m->gram_mw == m->mw &&
        m->K <= AMP_MAX_COUPLINGS) {
        // Static lineshapes (the paper's default: masses and widths fixed) with the matrix M already held: ONE launch
        // over the data tiles; the last CTA evaluates c^H M c from the device-resident matrix and forms the NLL (MODE_DATA_M).
        StreamArgs a;
        fill_stream_args(m, m->data, 0, MODE_DATA_M, &a);
        a.partial = m->d_partial;
        a.ticket = m->d_ticket;
        a.sum_log_eff = m->data.wsum;
        a.wsum = m->norm.wsum;
        a.qf_G = m->d_G;
        a.qf_KP = m->gram_KP;
        a.qf_nent = m->gram_nent;
        for (int k = 0; k < AMP_MAX_COUPLINGS; ++k)
            a.qf_c[k] = k < m->K ? make_double2(m->couplings[2 * k], m->couplings[2 * k + 1]) : make_double2(0, 0);
        double* res = m->h_pinned;
        if (m->zero_copy) { m->zc_seq += 1.0; a.result = m->h_zc; a.seq = m->zc_seq; res = m->h_zc; }
        else { a.result = m->d_result; a.seq = 0.0; }
        m->ring_last = (m->ring_last + 1) % amp_model::RING;
        m->ring_calls++;
        CK(cudaEventRecord(m->ring[2 * m->ring_last], s));
        CK(launch_stream(a, stream_grid(m->data.n, m->has_z, MODE_DATA), s));
        CK(cudaEventRecord(m->ring[2 * m->ring_last + 1], s));
        if (m->zero_copy) {
            volatile double* stamp = m->h_zc + 5;
            for (unsigned spins = 0; *stamp != m->zc_seq; ++spins) {
                if ((spins & 0x3fff) == 0x3fff) {
                    const cudaError_t q = cudaStreamQuery(s);
                    if (q != cudaErrorNotReady) { if (q != cudaSuccess) return cuda_fail(m, q, "matrix step"); if (*stamp == m->zc_seq) break; return fail(m, AMP_ERR_CUDA, "matrix step finished without a result"); }
                }
            }
            std::atomic_thread_fence(std::memory_order_acquire);
        } else {
            CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * 5, cudaMemcpyDeviceToHost, s));
            CK(cudaStreamSynchronize(s));
        }
        m->last_slog.assign(1, res[3]);
        m->last_swS.assign(1, res[4]);
        m->stat_launches = 1;
        m->stat_norm_path = 2;
        m->fused_valid = true;
        h_nll[0] = res[0];
        if (h_I) h_I[0] = res[1];
        if (res[2] != 0.0 || !std::isfinite(h_nll[0])) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
        return AMP_OK;
    }
    if (want_nll && P == 1 && m->stream_inline && !m->want_matrix && m->fused_mode == 0) {
        // The whole step in ONE launch: lineshapes in registers, combine and both reductions over the data tiles and
        // then the normalisation tiles of one persistent grid; the last CTA forms the NLL (stream.cu, MODE_FUSED).
        StreamArgs a;
        fill_stream_args(m, m->data, 0, MODE_FUSED, &a);
        a.partial = m->d_partial;
        a.partial2 = m->d_partial + PARTIAL_STRIDE;
        a.cache2 = m->norm.cache; a.n2 = m->norm.n; a.npad2 = m->norm.npad;
        a.ticket = m->d_ticket;
        a.sum_log_eff = m->data.wsum;
        a.wsum = m->norm.wsum;
        // Result block: by default mapped host memory (UVA: same pointer on the device) that the last CTA fills and stamps;
        // the host spins on the stamp, which saves the D2H copy and the stream-synchronise wake-up of a synchronous call.
        double* res = m->h_pinned;
        if (m->zero_copy) {
            m->zc_seq += 1.0;
            a.result = m->h_zc;
            a.seq = m->zc_seq;
            res = m->h_zc;
        } else {
            a.result = m->d_result;
            a.seq = 0.0;
        }
        m->ring_last = (m->ring_last + 1) % amp_model::RING;
        m->ring_calls++;
        CK(cudaEventRecord(m->ring[2 * m->ring_last], s));
        CK(launch_stream(a, stream_grid_fused(m->data.n, m->norm.n, m->has_z), s));
        CK(cudaEventRecord(m->ring[2 * m->ring_last + 1], s));
        if (m->zero_copy) {
            volatile double* stamp = m->h_zc + 5;
            for (unsigned spins = 0; *stamp != m->zc_seq; ++spins) {
                if ((spins & 0x3fff) == 0x3fff) {   // every 16k spins: has the stream failed or finished without the stamp?
                    const cudaError_t q = cudaStreamQuery(s);
                    if (q != cudaErrorNotReady) { if (q != cudaSuccess) return cuda_fail(m, q, "fused step"); if (*stamp == m->zc_seq) break; return fail(m, AMP_ERR_CUDA, "fused step finished without a result"); }
                }
            }
            std::atomic_thread_fence(std::memory_order_acquire);
        } else {
            CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * 5, cudaMemcpyDeviceToHost, s));
            CK(cudaStreamSynchronize(s));
        }
        m->last_slog.assign(1, res[3]);
        m->last_swS.assign(1, res[4]);
        m->stat_launches = 1;
        m->stat_norm_path = 4;
        m->fused_valid = true;
        h_nll[0] = res[0];
        if (h_I) h_I[0] = res[1];
        if (res[2] != 0.0 || !std::isfinite(h_nll[0])) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
        return AMP_OK;
    }
    m->fused_valid = false;
    CK(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
    CK(cudaEventRecord(m->ev[0], s));
    m->stat_gram_built = 0;
    HerkPlan hp;
    bool use_matrix = m->want_matrix && build_herk_plan(m, &hp);
    if (use_matrix) {   // the cached matrix may already cover this lineshape state: then no norm column is needed at all
        const bool hit = gram_hit(m, hp);
        if (!hit) { st = refresh_columns(m, m->norm, true, s); if (st != AMP_OK) return st; }
    }
    if (want_nll && !m->stream_inline) { st = refresh_columns(m, m->data, false, s); if (st != AMP_OK) return st; }
    if (!use_matrix && !m->stream_inline) { st = refresh_columns(m, m->norm, true, s); if (st != AMP_OK) return st; }
    CK(cudaEventRecord(m->ev[1], s));
    int gd = stream_grid(m->data.n, m->has_z, MODE_DATA), gn = stream_grid(m->norm.n, m->has_z, MODE_NORM);
    // P > 1: one DMMA launch per dataset and chunk of <= 128 points, if the model and the points fit its plan
    std::vector<BatchPlan> plans;
    // (below ~24 points the streaming kernel, which shares the angular structure, is cheaper per point)
    bool batched = P >= 24 && m->batch_mode != 1;
    if (batched) {
        for (int p0 = 0; p0 < P && batched; p0 += BATCH_POINTS) {
            plans.emplace_back();
            batched = build_batch_plan(m, p0, std::min((int)BATCH_POINTS, P - p0), &plans.back());
        }
    }
    m->stat_batched = batched ? 1 : 0;
    if (batched) m->stat_norm_path = 3;
    if (batched) {
        const size_t per_plan = (size_t)1 << 20, need = per_plan * plans.size() * 2;
        if (need > m->plan_cap) {
            if (m->d_plan) cudaFree(m->d_plan);
            if (m->h_plan) cudaFreeHost(m->h_plan);
            m->d_plan = m->h_plan = nullptr;
            m->plan_cap = 0;
            CK(cudaMalloc(&m->d_plan, need));
            CK(cudaMallocHost(&m->h_plan, need));
            m->plan_cap = need;
        }
        size_t slot = 0;
        if (want_nll) {
            for (size_t c = 0; c < plans.size(); ++c) {
                const int p0 = (int)c * BATCH_POINTS, Pc = std::min((int)BATCH_POINTS, P - p0);
                if (m->data.n > 0) {
                    st = run_batch(m, m->data, plans[c], Pc, MODE_DATA, per_plan * slot++, m->d_partial + (size_t)p0 * PARTIAL_STRIDE, s, &gd);
                    if (st != AMP_OK) return st;
                } else {
                    for (int p = p0; p < p0 + Pc; ++p) CK(cudaMemsetAsync(m->d_partial + (size_t)p * PARTIAL_STRIDE, 0, sizeof(double), s));
                }
            }
        }
        CK(cudaEventRecord(m->ev[2], s));
        for (size_t c = 0; c < plans.size() && !use_matrix; ++c) {
            const int p0 = (int)c * BATCH_POINTS, Pc = std::min((int)BATCH_POINTS, P - p0);
            st = run_batch(m, m->norm, plans[c], Pc, MODE_NORM, per_plan * slot++, m->d_partial + (size_t)(P + p0) * PARTIAL_STRIDE, s, &gn);
            if (st != AMP_OK) return st;
        }
    } else {
    StreamArgs a;
    if (want_nll)
        for (int p = 0; p < P; ++p) {
            if (m->data.n > 0) {
                fill_stream_args(m, m->data, p, MODE_DATA, &a);
                a.partial = m->d_partial + (size_t)p * PARTIAL_STRIDE;
                CK(launch_stream(a, gd, s));
                m->stat_launches++;
            } else {
                CK(cudaMemsetAsync(m->d_partial + (size_t)p * PARTIAL_STRIDE, 0, sizeof(double), s));
            }
        }
    CK(cudaEventRecord(m->ev[2], s));
    for (int p = 0; p < P && !use_matrix; ++p) {
        fill_stream_args(m, m->norm, p, MODE_NORM, &a);
        a.partial = m->d_partial + (size_t)(P + p) * PARTIAL_STRIDE;
        CK(launch_stream(a, gn, s));
        m->stat_launches++;
    }
    }
    if (use_matrix) {
        st = norm_via_matrix(m, hp, m->d_sums + P, s);
        if (st != AMP_OK) return st;
        m->stat_norm_path = 2;
        if (P == 1) { m->gram_p1 = true; m->gram_nent = hp.nent; m->gram_mw = m->mw; }   // later calls at these masses: one launch
    }
    CK(cudaEventRecord(m->ev[3], s));
    if (want_nll) {
        CK(launch_finalize(m->d_partial, m->data.n > 0 ? gd : 1, PARTIAL_STRIDE, P, m->d_sums, s));
        m->stat_launches++;
    }
    if (!use_matrix) CK(launch_finalize(m->d_partial + (size_t)P * PARTIAL_STRIDE, gn, PARTIAL_STRIDE, P, m->d_sums + P, s));
    k_nll_final<<<(P + 127) / 128, 128, 0, s>>>(m->d_sums, P, (double)m->data.n, m->data.loaded ? m->data.wsum : 0.0, m->norm.wsum, want_nll ? 1 : 0,
                                                m->d_result);
    CK(cudaGetLastError());
    m->stat_launches += 2;
    CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * 2 * P, cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(m->h_pinned + 2 * P, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost, s));
    CK(cudaMemcpyAsync(m->h_pinned + 2 * P + 1, m->d_sums, sizeof(double) * 2 * P, cudaMemcpyDeviceToHost, s));
    CK(cudaEventRecord(m->ev[4], s));
    CK(cudaStreamSynchronize(s));
    m->ev_valid = true;
    m->last_slog.assign(m->h_pinned + 2 * P + 1, m->h_pinned + 3 * P + 1);
    m->last_swS.assign(m->h_pinned + 3 * P + 1, m->h_pinned + 4 * P + 1);
    int flag;
    std::memcpy(&flag, m->h_pinned + 2 * P, sizeof(int));
    bool bad = flag != 0;
    for (int p = 0; p < P; ++p) {
        if (h_nll) { h_nll[p] = m->h_pinned[p]; bad |= !std::isfinite(h_nll[p]); }
        if (h_I) { h_I[p] = m->h_pinned[P + p]; bad |= !(h_I[p] > 0) || !std::isfinite(h_I[p]); }
    }
    if (bad) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
    return AMP_OK;
}

}  // namespace

// ---- amp_nll_static: the fused launch with its scratch in a static device array (include/amp.h) -----------------------
// Per point a slice of [2][AMP_STATIC_MAX_CTAS] doubles (the CTAs' sum log S and sum w S) and a 256-byte control block
// (ticket, then flag).  In HOST code the array's name is only a handle for cudaGetSymbolAddress, never a device address.
constexpr size_t STATIC_SLICE_BYTES = 2 * (size_t)AMP_STATIC_MAX_CTAS * sizeof(double) + 256;
static_assert(AMP_STATIC_SCRATCH_BYTES == AMP_STATIC_MAX_POINTS * STATIC_SLICE_BYTES, "include/amp.h states the size");
static __device__ __align__(256) unsigned char g_static_scratch[AMP_STATIC_SCRATCH_BYTES];

// device address of g_static_scratch on the CURRENT device, looked up once per device
cudaError_t static_scratch_address(unsigned char** out) {
    static std::atomic<unsigned char*> addr[AMP_MAX_DEVICES];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= AMP_MAX_DEVICES) return cudaErrorInvalidDevice;
    unsigned char* p = addr[dev].load(std::memory_order_acquire);
    if (!p) {
        e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        addr[dev].store(p, std::memory_order_release);   // (two threads racing here store the same address)
    }
    *out = p;
    return cudaSuccess;
}

extern "C" {

amp_status amp_nll(amp_model* m, double* h_nll, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    if (!h_nll) return fail(m, AMP_ERR_INVALID, "amp_nll: null output");
    return evaluate(m, true, h_nll, nullptr, (cudaStream_t)stream);
}

amp_status amp_nll_static(amp_model* m, double* d_out, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    cudaStream_t s = (cudaStream_t)stream;
    if (!d_out) return fail(m, AMP_ERR_INVALID, "amp_nll_static: null output");
    if (!m->norm.loaded) return fail(m, AMP_ERR_STATE, "no normalisation sample loaded (amp_load_norm)");
    if (!m->data.loaded) return fail(m, AMP_ERR_STATE, "no data events loaded (amp_load_events)");
    if (m->P < 1) return fail(m, AMP_ERR_STATE, "no parameters set (amp_set_params)");
    if (m->has_bkg) return fail(m, AMP_ERR_STATE, "amp_nll_static: not available with a background set (Eq. 14 takes two passes over model-owned buffers)");
    if (m->P > AMP_STATIC_MAX_POINTS) {
        char msg[160];
        std::snprintf(msg, sizeof msg, "amp_nll_static: %d points exceed the static scratch (AMP_STATIC_MAX_POINTS = %d)", m->P, (int)AMP_STATIC_MAX_POINTS);
        return fail(m, AMP_ERR_INVALID, msg);
    }
    const int grid = stream_grid_fused(m->data.n, m->norm.n, m->has_z);
    if (grid > AMP_STATIC_MAX_CTAS) {
        char msg[160];
        std::snprintf(msg, sizeof msg, "amp_nll_static: a grid of %d CTAs exceeds the static scratch (AMP_STATIC_MAX_CTAS = %d)", grid, (int)AMP_STATIC_MAX_CTAS);
        return fail(m, AMP_ERR_INVALID, msg);
    }
    unsigned char* base = nullptr;
    CK(static_scratch_address(&base));
    for (int p = 0; p < m->P; ++p) {
        unsigned char* slice = base + (size_t)p * STATIC_SLICE_BYTES;
        unsigned char* ctl = slice + 2 * (size_t)AMP_STATIC_MAX_CTAS * sizeof(double);
        StreamArgs a;
        fill_stream_args(m, m->data, p, MODE_FUSED, &a);
        // lineshapes always in registers here (pool columns are model-owned buffers that may not exist yet): fold kN as fill_stream_args does
        for (int t = 0; t < a.lass0 + a.nlass; ++t) {
            ResEntry& e = a.ent[t];
            if (e.column < 0) continue;
            e.column = -1;
            if (t < a.lass0) { e.cm.x *= e.kN; e.cm.y *= e.kN; e.c0.x *= e.kN; e.c0.y *= e.kN; e.cp.x *= e.kN; e.cp.y *= e.kN; }
        }
        a.cols = nullptr;
        a.partial = reinterpret_cast<double*>(slice);
        a.partial2 = a.partial + AMP_STATIC_MAX_CTAS;
        a.ticket = reinterpret_cast<unsigned int*>(ctl);
        a.flag = reinterpret_cast<int*>(ctl + 128);
        a.cache2 = m->norm.cache; a.n2 = m->norm.n; a.npad2 = m->norm.npad;
        a.sum_log_eff = m->data.wsum;
        a.wsum = m->norm.wsum;
        a.result = d_out + (size_t)6 * p;
        a.seq = 1.0;
        // the array keeps what the last call (of anyone) left: ticket and flag must start at zero; the partials are overwritten
        CK(cudaMemsetAsync(ctl, 0, 256, s));
        CK(launch_stream(a, grid, s));
    }
    return AMP_OK;
}

amp_status amp_nll_terms(amp_model* m, double* h_sum_log, double* h_sum_wS, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    if (!h_sum_log || !h_sum_wS) return fail(m, AMP_ERR_INVALID, "amp_nll_terms: null output");
    if (m->has_bkg) return fail(m, AMP_ERR_STATE, "amp_nll_terms: not defined with a background set (Eq. 14 does not separate into the two sums)");
    std::vector<double> nll((size_t)std::max(m->P, 1));
    const amp_status st = evaluate(m, true, nll.data(), nullptr, (cudaStream_t)stream);
    if (st != AMP_OK && st != AMP_ERR_DOMAIN) return st;
    for (int p = 0; p < m->P; ++p) { h_sum_log[p] = m->last_slog[p]; h_sum_wS[p] = m->last_swS[p]; }
    return st;
}

amp_status amp_dataset_sums(const amp_model* m, long long* n_data, double* sum_log_eff, long long* n_norm, double* sum_w) {
    if (!m) return AMP_ERR_INVALID;
    if (n_data) *n_data = m->data.loaded ? m->data.n : 0;
    if (sum_log_eff) *sum_log_eff = m->data.loaded ? m->data.wsum : 0.0;
    if (n_norm) *n_norm = m->norm.loaded ? m->norm.n : 0;
    if (sum_w) *sum_w = m->norm.loaded ? m->norm.wsum : 0.0;
    return AMP_OK;
}

amp_status amp_nll_grad(amp_model* m, double* h_nll, double* h_grad, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    if (!h_nll || !h_grad) return fail(m, AMP_ERR_INVALID, "amp_nll_grad: null output");
    cudaStream_t s = (cudaStream_t)stream;
    if (!m->norm.loaded) return fail(m, AMP_ERR_STATE, "no normalisation sample loaded (amp_load_norm)");
    if (!m->data.loaded) return fail(m, AMP_ERR_STATE, "no data events loaded (amp_load_events)");
    if (m->P != 1) return fail(m, AMP_ERR_STATE, "amp_nll_grad: set exactly one parameter point (amp_set_params with P = 1)");
    if (!m->stream_inline) return fail(m, AMP_ERR_STATE, "amp_nll_grad: needs lineshapes in registers (amp_set_lineshape_mode 0 or 2)");
    if (m->K > GRAD_MAX_PAIRS) return fail(m, AMP_ERR_INVALID, "amp_nll_grad: too many couplings");
    int ent_of_res[AMP_MAX_RESONANCES], grp_of_res[AMP_MAX_RESONANCES];
    GradArgs g{};
    fill_stream_args(m, m->data, 0, MODE_FUSED, &g.a, ent_of_res, grp_of_res);
    int nent = g.a.nlass;
    for (int sp = 0; sp < NSPIN; ++sp) nent += g.a.shape[sp];
    if (!grad_fits(nent, g.a.gstart[NSPIN])) return fail(m, AMP_ERR_INVALID, "amp_nll_grad: the model does not fit the kernel's shared memory");
    g.a.cache2 = m->norm.cache; g.a.n2 = m->norm.n; g.a.npad2 = m->norm.npad;
    g.a.ticket = m->d_ticket;
    g.a.sum_log_eff = m->data.wsum;
    g.a.wsum = m->norm.wsum;
    // Static lineshapes (masses and widths as in the previous call): the normalisation side comes from the matrix M —
    // N_k = (M c)_k, sum w S = c^H M c — so only the data events are walked; M is built here if it is not held yet.
    if (m->want_matrix && m->K <= AMP_MAX_COUPLINGS) {
        if (!(m->gram_valid && m->gram_p1 && m->gram_mw == m->mw)) {
            HerkPlan hp;
            if (build_herk_plan(m, &hp, 0, 1)) {
                amp_status st = ensure_pool(m, 0);
                if (st == AMP_OK) st = refresh_columns(m, m->norm, true, s);
                if (st == AMP_OK) st = norm_via_matrix(m, hp, m->d_sums, s);
                if (st != AMP_OK) return st;
                m->gram_p1 = true; m->gram_nent = hp.nent; m->gram_mw = m->mw;
            }
        }
        if (m->gram_valid && m->gram_p1 && m->gram_mw == m->mw) {
            g.a.n2 = 0;
            g.a.qf_G = m->d_G;
            g.a.qf_KP = m->gram_KP;
            g.a.qf_nent = m->gram_nent;
            for (int k = 0; k < AMP_MAX_COUPLINGS; ++k)
                g.a.qf_c[k] = k < m->K ? make_double2(m->couplings[2 * k], m->couplings[2 * k + 1]) : make_double2(0, 0);
        }
    }
    int extra_launches = 0;
    if (m->has_bkg) {   // Eq. 14: the data side needs sum_j w_j S_j before its first event
        g.a.bkg = m->d_bkg;
        g.a.purity = m->purity;
        if (!g.a.qf_G) {   // lineshapes moved: a normalisation launch first (the gradient kernel walks that sample again for N_k)
            StreamArgs a;
            fill_stream_args(m, m->norm, 0, MODE_NORM, &a);
            a.partial = m->d_partial + (size_t)400 * PARTIAL_STRIDE;   // rows the gradient kernel does not use
            const int gn = stream_grid(m->norm.n, m->has_z, MODE_NORM);
            CK(launch_stream(a, gn, s));
            CK(launch_finalize(a.partial, gn, PARTIAL_STRIDE, 1, m->d_sums + 1, s));
            g.a.sum_wS = m->d_sums + 1;
            extra_launches = 2;
        }
    }
    const int K = m->K;
    g.K = K;
    g.npairs = (K + 15) / 16 * 16;
    for (int p = 0; p < GRAD_MAX_PAIRS; ++p) { g.pair_ent[p] = -2; g.pair_lam[p] = 0; g.pair_J[p] = 0; g.pair_grp[p] = 0; g.pair_slot[p] = -1; }
    for (int r = 0; r < m->R; ++r) {
        const amp_resonance& rs = m->res[r];
        const int ns = (kind_is_z(rs.kind) || (rs.kind == AMP_KSTAR && rs.J >= 1)) ? 3 : 1;
        for (int j = 0; j < ns; ++j) {
            const int k = m->slot0[r] + j;
            g.pair_ent[k] = rs.kind == AMP_CONST ? -1 : (signed char)ent_of_res[r];
            g.pair_lam[k] = (signed char)(ns == 3 ? j - 1 : 0);
            g.pair_J[k] = kind_is_z(rs.kind) ? (signed char)(8 + rs.J) : (signed char)rs.J;   // 8 + J: a Z slot of spin J
            g.pair_grp[k] = rs.kind == AMP_CONST ? 0 : (signed char)grp_of_res[r];
            g.pair_slot[k] = (short)k;
        }
    }
    g.partial = m->d_partial;
    g.stride = PARTIAL_STRIDE;
    g.result = m->d_result;
    m->ring_last = (m->ring_last + 1) % amp_model::RING;
    m->ring_calls++;
    CK(cudaEventRecord(m->ring[2 * m->ring_last], s));
    // the paper's resonance lists: every gradient component in a register of the thread that owns the event (gradf.cu)
    const bool fast = m->grad_mode == 0 && gradf_supports(g);
    if (fast) {
        const int n0 = g.a.shape[0];   // accumulators in entry order: one per J = 0 entry, then three (lambda = -1, 0, +1) per entry
        for (int k = 0; k < K; ++k) {
            const int t = g.pair_ent[k];
            g.acc_pair[(t < n0 ? t : n0 + 3 * (t - n0)) + (g.pair_J[k] == 0 ? 0 : g.pair_lam[k] + 1)] = (signed char)k;
        }
        CK(launch_gradf(g, gradf_grid(m->data.n, g.a.n2), s));
    } else {
        CK(launch_grad(g, grad_grid(m->data.n, g.a.n2), s));
    }
    CK(cudaEventRecord(m->ring[2 * m->ring_last + 1], s));
    CK(cudaMemcpyAsync(m->h_pinned, m->d_result, sizeof(double) * (3 + 2 * K), cudaMemcpyDeviceToHost, s));
    CK(cudaStreamSynchronize(s));
    m->stat_launches = 1 + extra_launches;
    m->stat_columns = 0;
    m->stat_norm_path = fast ? 8 : 7;
    m->fused_valid = true;
    h_nll[0] = m->h_pinned[0];
    bool bad = m->h_pinned[2] != 0.0 || !std::isfinite(h_nll[0]);
    for (int i = 0; i < 2 * K; ++i) { h_grad[i] = m->h_pinned[3 + i]; bad |= !std::isfinite(h_grad[i]); }
    if (bad) return fail(m, AMP_ERR_DOMAIN, "non-finite or non-positive PDF value");
    return AMP_OK;
}

amp_status amp_norm_integral(amp_model* m, double* h_I, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    if (!h_I) return fail(m, AMP_ERR_INVALID, "amp_norm_integral: null output");
    return evaluate(m, false, nullptr, h_I, (cudaStream_t)stream);
}

amp_status amp_eval_events(amp_model* m, int p, double* d_out, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    cudaStream_t s = (cudaStream_t)stream;
    if (!m->data.loaded) return fail(m, AMP_ERR_STATE, "no data events loaded (amp_load_events)");
    if (m->P < 1) return fail(m, AMP_ERR_STATE, "no parameters set (amp_set_params)");
    if (p < 0 || p >= m->P || (!d_out && m->data.n > 0)) return fail(m, AMP_ERR_INVALID, "amp_eval_events: bad point index or null output");
    if (m->data.n == 0) return AMP_OK;
    m->stat_launches = m->stat_columns = 0;
    amp_status st = ensure_pool(m, 0);
    if (st != AMP_OK) return st;
    if (!m->stream_inline) {
        st = refresh_columns(m, m->data, false, s);
        if (st != AMP_OK) return st;
    }
    StreamArgs a;
    fill_stream_args(m, m->data, p, MODE_EVAL, &a);
    a.out = d_out;
    CK(launch_stream(a, stream_grid(m->data.n, m->has_z, MODE_EVAL), s));
    m->stat_launches++;
    CK(cudaStreamSynchronize(s));
    return AMP_OK;
}

amp_status amp_generate(amp_model* m, unsigned long long seed, unsigned long long first, long long n_candidates,
                        double f_max, double m_lo, double m_hi, double cos_max,
                        double* d_x_out, long long* d_index_out, long long capacity,
                        long long* h_n_accepted, double* h_f_seen_max, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    cudaStream_t s = (cudaStream_t)stream;
    if (n_candidates < 0 || capacity < 0 || (capacity > 0 && !d_x_out) || !h_n_accepted || !h_f_seen_max)
        return fail(m, AMP_ERR_INVALID, "amp_generate: negative count or null output");
    if (!(m_lo > m->dk.mK + m->dk.mpi) || !(m_hi < m->dk.MB - m->dk.mpsi) || !(m_lo < m_hi) || !(cos_max > 0.0 && cos_max <= 1.0) ||
        !(f_max >= 0.0) || !std::isfinite(f_max))
        return fail(m, AMP_ERR_INVALID, "amp_generate: mass range outside phase space, cos_max outside (0, 1] or bad f_max");
    if (m->P != 1) return fail(m, AMP_ERR_STATE, "amp_generate: needs one parameter point (amp_set_params with P = 1)");
    if (!m->stream_inline) return fail(m, AMP_ERR_STATE, "amp_generate: needs lineshapes in registers (amp_set_lineshape_mode 0 or 2)");
    *h_n_accepted = 0;
    *h_f_seen_max = 0.0;
    if (n_candidates == 0) return AMP_OK;
    m->stat_launches = m->stat_columns = 0;
    const long long CH = 1LL << 21;                       // candidates per block of work (a multiple of the selection block)
    const long long ch = n_candidates < CH ? n_candidates : CH;
    if (m->toy_cap < ch) {
        free_toy_scratch(m);
        const int ncolw = (m->has_z ? NCOL_ALL : NCOL_K) + 1;
        cudaError_t e = cudaMalloc(&m->toy_x, sizeof(double) * 4 * ch);
        if (e == cudaSuccess) e = cudaMalloc(&m->toy_u, sizeof(double) * ch);
        if (e == cudaSuccess) e = cudaMalloc(&m->toy_S, sizeof(double) * stream_pad(ch));
        if (e == cudaSuccess) e = cudaMalloc(&m->toy_cache, sizeof(double) * ncolw * stream_pad(ch));
        if (e == cudaSuccess) e = cudaMalloc(&m->toy_count, sizeof(int) * (toy_blocks(ch) + 1));
        if (e == cudaSuccess) e = cudaMalloc(&m->toy_fseen, sizeof(unsigned long long));
        if (e != cudaSuccess) { free_toy_scratch(m); return cuda_fail(m, e, "amp_generate"); }
        m->toy_cap = ch;
    }
    double *d_x = m->toy_x, *d_u = m->toy_u, *d_S = m->toy_S;
    int* d_count = m->toy_count;
    unsigned long long* d_fseen = m->toy_fseen;
    Dataset tmp{};
    tmp.cache = m->toy_cache;
    auto cleanup = [&]() {};
    cudaError_t e = cudaMemsetAsync(d_fseen, 0, sizeof(unsigned long long), s);
    if (e != cudaSuccess) return cuda_fail(m, e, "amp_generate");
    long long accepted = 0;
    amp_status st = AMP_OK;
    for (long long off = 0; off < n_candidates && st == AMP_OK; off += ch) {
        const long long nc = n_candidates - off < ch ? n_candidates - off : ch;
        ToyArgs t{};
        t.seed = seed;
        t.first = first + (unsigned long long)off;
        t.n = nc;
        t.m_lo = m_lo;
        t.m_span = m_hi - m_lo;
        t.cos_max = cos_max;
        t.f_max = f_max;
        t.x = d_x;
        t.u = d_u;
        t.S = d_S;
        t.count = d_count;
        t.f_seen = d_fseen;
        t.flag = m->d_flag;
        t.x_out = d_x_out;
        t.index_out = d_index_out;
        t.capacity = capacity;
        t.out_base = accepted;
        e = launch_toy_candidates(t, s);
        if (e != cudaSuccess) { st = cuda_fail(m, e, "amp_generate"); break; }
        st = load_dataset(m, tmp, true, d_x, nullptr, nc, s, true);      // kinematics cache of the candidates, weight 1
        if (st != AMP_OK) break;
        StreamArgs a;
        fill_stream_args(m, tmp, 0, MODE_EVAL, &a);
        a.out = d_S;
        e = launch_stream(a, stream_grid(nc, m->has_z, MODE_EVAL), s);
        t.cache = tmp.cache;
        t.ncolw = tmp.ncache + 1;
        if (e == cudaSuccess) e = cudaMemsetAsync(m->d_flag, 0, sizeof(int), s);
        if (e == cudaSuccess) e = launch_toy_select(t, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(m->h_pinned, d_count + toy_blocks(nc), sizeof(int), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(m->h_pinned + 1, m->d_flag, sizeof(int), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaMemcpyAsync(m->h_pinned + 2, d_fseen, sizeof(unsigned long long), cudaMemcpyDeviceToHost, s);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s);
        if (e != cudaSuccess) { st = cuda_fail(m, e, "amp_generate"); break; }
        m->stat_launches += 6;
        int cnt, flag;
        std::memcpy(&cnt, m->h_pinned, sizeof(int));
        std::memcpy(&flag, m->h_pinned + 1, sizeof(int));
        std::memcpy(h_f_seen_max, m->h_pinned + 2, sizeof(double));
        if (flag) { st = fail(m, AMP_ERR_DOMAIN, "amp_generate: a candidate weight p_B q S is not finite"); break; }
        accepted += cnt;
    }
    cleanup();
    CK(cudaMemsetAsync(m->d_flag, 0, sizeof(int), s));
    *h_n_accepted = accepted;
    return st;
}

static const char* const kColNames[NCOL_ALL] = {"m2", "inv_m", "q", "pB", "cosK", "sinK", "cosPsi", "sinPsi", "cosPhi", "sinPhi",
                                                "mZ2", "inv_mZ", "qZ", "pBZ", "cosZ", "sinZ", "cosT", "sinT", "cosPhiT", "sinPhiT", "cosAlpha", "sinAlpha"};
const char* amp_cache_column_name(int i) { return (i >= 0 && i < NCOL_ALL) ? kColNames[i] : nullptr; }

amp_status amp_dump_cache(amp_model* m, int which, double* d_out, int* ncols, void* stream) {
    if (!m || which < 0 || which > 1) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    Dataset& d = which ? m->norm : m->data;
    if (!d.loaded) return fail(m, AMP_ERR_STATE, "amp_dump_cache: dataset not loaded");
    if (ncols) *ncols = d.ncache;
    if (!d_out || d.n == 0) return AMP_OK;
    cudaStream_t s = (cudaStream_t)stream;
    k_dump_cache<<<sm_count() * 4, 256, 0, s>>>(d.cache, d.ncache + 1, d.ncache, d.n, d_out);
    CK(cudaGetLastError());
    CK(cudaStreamSynchronize(s));
    return AMP_OK;
}

amp_status amp_eval_lineshape(amp_model* m, int which, int r, double mass, double width, double* d_out, void* stream) {
    if (!m || which < 0 || which > 1 || r < 0 || r >= m->R || !d_out) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    Dataset& d = which ? m->norm : m->data;
    if (!d.loaded) return fail(m, AMP_ERR_STATE, "amp_eval_lineshape: dataset not loaded");
    cudaStream_t s = (cudaStream_t)stream;
    LineshapeJob j;
    if (!make_line_const(m, r, mass, width, &j.lc)) return fail(m, AMP_ERR_DOMAIN, "amp_eval_lineshape: pole mass outside the kinematic range");
    j.column = 0;
    Dataset tmp = d;   // same cache, private one-column pool
    tmp.cols = nullptr;
    CK(cudaMalloc(&tmp.cols, sizeof(double2) * d.npad));
    cudaError_t e = launch_lineshape(tmp, &j, 1, s);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_out, tmp.cols, sizeof(double2) * d.n, cudaMemcpyDeviceToDevice, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(tmp.cols);
    if (e != cudaSuccess) return cuda_fail(m, e, "amp_eval_lineshape");
    return AMP_OK;
}

amp_status amp_fit_fractions(amp_model* m, int p, double* h_ff, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    cudaStream_t s = (cudaStream_t)stream;
    if (!m->norm.loaded) return fail(m, AMP_ERR_STATE, "no normalisation sample loaded (amp_load_norm)");
    if (m->P < 1) return fail(m, AMP_ERR_STATE, "no parameters set (amp_set_params)");
    if (p < 0 || p >= m->P || !h_ff) return fail(m, AMP_ERR_INVALID, "amp_fit_fractions: bad point index or null output");
    HerkPlan hp;
    if (!build_herk_plan(m, &hp, p, 1))
        return fail(m, AMP_ERR_STATE, "amp_fit_fractions: the lineshape columns of this point are not held; call amp_set_norm_mode(m, 2) before amp_set_params");
    m->stat_launches = m->stat_columns = 0;
    amp_status st = ensure_pool(m, 0);
    if (st != AMP_OK) return st;
    st = refresh_columns(m, m->norm, true, s);
    if (st != AMP_OK) return st;
    // rows of coefficient vectors for the quadratic-form kernel: row 0 = all couplings, row 1 + r = those of resonance r only
    const int R = m->R, nent = hp.nent;
    std::vector<double2> C((size_t)(R + 1) * nent, make_double2(0, 0));
    for (int e = 0; e < nent; ++e) C[e] = hp.C[e];
    for (int r = 0; r < R; ++r) {
        const int ns = (kind_is_z(m->res[r].kind) || (m->res[r].kind == AMP_KSTAR && m->res[r].J >= 1)) ? 3 : 1;
        for (int j = 0; j < ns; ++j) C[(size_t)(1 + r) * nent + m->slot0[r] + j] = hp.C[m->slot0[r] + j];   // single point: entry k = slot k
    }
    hp.C.swap(C);
    double* d_tmp = nullptr;
    CK(cudaMalloc(&d_tmp, sizeof(double) * (R + 1)));
    st = norm_via_matrix(m, hp, d_tmp, s);
    std::vector<double> q((size_t)R + 1);
    cudaError_t e = st == AMP_OK ? cudaMemcpyAsync(q.data(), d_tmp, sizeof(double) * (R + 1), cudaMemcpyDeviceToHost, s) : cudaSuccess;
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(d_tmp);
    if (st != AMP_OK) return st;
    if (e != cudaSuccess) return cuda_fail(m, e, "amp_fit_fractions");
    if (!(q[0] > 0) || !std::isfinite(q[0])) return fail(m, AMP_ERR_DOMAIN, "amp_fit_fractions: the total integral is not positive");
    for (int r = 0; r < R; ++r) h_ff[r] = q[1 + r] / q[0];
    return AMP_OK;
}

amp_status amp_norm_matrix(amp_model* m, int p, double* h_M, void* stream) {
    if (!m) return AMP_ERR_INVALID;
    DeviceGuard on_device(m);
    cudaStream_t s = (cudaStream_t)stream;
    if (!m->norm.loaded) return fail(m, AMP_ERR_STATE, "no normalisation sample loaded (amp_load_norm)");
    if (m->P < 1) return fail(m, AMP_ERR_STATE, "no parameters set (amp_set_params)");
    if (p < 0 || p >= m->P || !h_M) return fail(m, AMP_ERR_INVALID, "amp_norm_matrix: bad point index or null output");
    HerkPlan hp;
    if (!build_herk_plan(m, &hp, p, 1))
        return fail(m, AMP_ERR_STATE, "amp_norm_matrix: the lineshape columns of this point are not held; call amp_set_norm_mode(m, 2) before amp_set_params");
    m->stat_launches = m->stat_columns = 0;
    amp_status st = ensure_pool(m, 0);
    if (st != AMP_OK) return st;
    st = refresh_columns(m, m->norm, true, s);
    if (st != AMP_OK) return st;
    const int KP = hp.nent * 2, K = m->K;
    double* d_tmp = nullptr;
    CK(cudaMalloc(&d_tmp, sizeof(double)));
    st = norm_via_matrix(m, hp, d_tmp, s);
    std::vector<double> G((size_t)KP * KP);
    cudaError_t e = st == AMP_OK ? cudaMemcpyAsync(G.data(), m->d_G, sizeof(double) * G.size(), cudaMemcpyDeviceToHost, s) : cudaSuccess;
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    cudaFree(d_tmp);
    if (st != AMP_OK) return st;
    if (e != cudaSuccess) return cuda_fail(m, e, "amp_norm_matrix");
    for (int k = 0; k < K; ++k)
        for (int l = 0; l < K; ++l) {
            const double* g = &G[(size_t)(2 * k) * KP + 2 * l];
            h_M[((size_t)k * K + l) * 2] = (g[0] + g[KP + 1]) / m->norm.wsum;
            h_M[((size_t)k * K + l) * 2 + 1] = (g[1] - g[KP]) / m->norm.wsum;
        }
    return AMP_OK;
}

}  // extern "C"
