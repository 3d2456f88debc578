// wri_api.cu — C ABI of libwri (include/wri.h): context, validation, launch sequencing.
// All arithmetic of the path runs in the kernels of wri_kernels.cuh / wri_pass.cuh; there is no
// CPU fallback.
#include "../../include/wri.h"
#include "wri_kernels.cuh"
#include "wri_pass.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <thread>
#include <chrono>
#include <type_traits>
#include <utility>
#include <vector>

using namespace wri;

namespace {

thread_local char g_cuda_msg[256] = "no CUDA error recorded";

int cuda_fail(cudaError_t e, const char* what) {
    snprintf(g_cuda_msg, sizeof g_cuda_msg, "CUDA error in %s: %s", what, cudaGetErrorString(e));
    return WRI_ERR_CUDA;
}
#define CK(call)                                                   \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call);      \
    } while (0)

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }
inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
inline int even_up(int n) { return (n + 1) & ~1; }

inline unsigned blocks_for(long long n) { return (unsigned)std::min<long long>((n + 255) / 256, 148 * 16); }
constexpr int kMaxCtas = 512;          // upper bound on the persistent grid (>= SM count)
constexpr int kInitRowBlocks = 64;     // blocks of k_init_rows (extra rows of the generic partials)

struct Tiling {
    int vec;            // complex numbers per thread (2 = 128-bit accesses)
    dim3 block, grid;
    int zc;
    size_t n_tiles;
};

}  // namespace

struct wri_ctx {
    wri_grid g{};
    double h = 0;
    size_t ng = 0;
    std::vector<double> omega;
    wri_sponge sponge{};
    int n_rec = 0, nb_max = 0;
    cudaStream_t stream = nullptr;
    const float* m = nullptr;
    int stencil = WRI_STENCIL_7;
    wri_debug_opts dbg{};
    // library-owned device memory
    float* gtab = nullptr;       // gx | gy | gz
    int* rec = nullptr;          // [n_rec] cell indices
    std::vector<int> rec_ijk;    // host copy [n_rec][3]
    float* coef[2] = {nullptr, nullptr};     // [N_COEF][nb_max] per-column scalars, one bank per parity
    // what the operator / objective entries last put into the constant rows of coef[0] and into src: a
    // call with the same columns skips the five small host-to-device copies (each is a gap on the stream).
    // A solve rewrites those rows on the device (re-packing moves whole banks), so its start clears this.
    std::vector<int> up_idx, up_src;
    float up_lambda = 0.f;
    bool up_cols_valid = false, up_src_valid = false;
    double* stat[2] = {nullptr, nullptr};    // [N_STAT][nb_max]
    int* active[2] = {nullptr, nullptr};     // [nb_max]
    int* iters[2] = {nullptr, nullptr};      // [nb_max]
    int* src = nullptr;          // [nb_max] source cell per caller's column (source-free system)
    bool sf = false;             // the solve in flight has the extra source-weight unknown
    float2* alpha_out = nullptr; // caller's [nb] source-weight estimates (source-free system)
    wri_lsqr_opts opts{};        // warm start / stop-rule reference for the next solves (wri_lsqr_set_opts)
    const unsigned char* rmask = nullptr;   // per-source receiver sets [n_rec][rmask_nb] (wri_set_receiver_mask)
    int rmask_nb = 0;
    int* colmap = nullptr;       // [nb_max] gather map of a grouped solve's start (caller's column per working column)
    // misfit evaluation / Algorithm 2 step (wri_misfit_sf, wri_awri_step)
    float* aw_tol = nullptr;     // [nb_max] the uniform tolerance eps of a misfit evaluation
    double* aw_f = nullptr;      // [2][nb_max] f_pde | f_data of the trial evaluation
    double* aw_ar0 = nullptr;    // [nb_max] alpha1*beta1 of the cold solve at the current model
    int* aw_iters = nullptr;     // [nb_max]
    double* h_aw = nullptr;      // pinned: [2][nb_max] doubles followed by [nb_max] ints
    // paced enqueue: an entry that ends with a stream synchronisation anyway (misfit evaluation, Algorithm 2
    // step, host-buffer solve) enqueues a solve with tolerances a few iterations ahead of the device and
    // stops once the device reports that every column has stopped — instead of enqueuing all maxit
    // iterations, whose launches would each return at once but cost about 2 us apiece (1-3 ms per solve).
    unsigned long long* h_prog = nullptr;   // mapped pinned word written by the finaliser of pass A
    unsigned long long* d_prog = nullptr;   // its device address
    unsigned int solve_id = 0;              // tags the word: a late write of an earlier solve is ignored
    bool pace = false;                      // set by the entries that synchronise at their end
    bool pacing = false;                    // the solve in flight reports its progress
    // caller's workspace
    char* ws = nullptr;
    size_t ws_bytes = 0;
    // solve in flight
    bool solving = false;
    int nb = 0, k = 0, maxit = 0;   // nb = working width at the START of the solve (the device state holds the
                                    // current one); k = iterations ENQUEUED
    int nb0 = 0;                    // caller's batch width
    bool packed = false;            // the working set has a column map; X lives in the workspace
    bool adaptive = false;          // converged columns are compacted away on the device
    float2* u_out = nullptr;
    float2* retire_buf = nullptr;   // adaptive: workspace region [caller's column][cell] for the x of retired columns
    int* retired = nullptr;         // [nb_max] device flags by the caller's column
    int col0 = 0, ncols = 0;        // this group's columns of the caller's batch
    float lambda = 0;
    float2* vec[2][4] = {};         // per parity: U, V, W, X
    float2* U_bot[2] = {nullptr, nullptr};
    float2 *U = nullptr, *V = nullptr, *W = nullptr, *X = nullptr;   // parity 0 (the start works on these)
    double* partials = nullptr;     // generic kernels: [n_tiles + kInitRowBlocks][nb]
    const float* tol = nullptr;
    float* resnorms = nullptr;
    int* iters_out = nullptr;
    Tiling tl{};
    int64_t launches = 0;
    // persistent pass kernel: per-width plans, tensor maps and receiver lists (device tables)
    int num_sms = 0;
    unsigned int* counter = nullptr;      // last-CTA ticket of the pass kernels (device)
    bool rt = false;                      // this solve runs on the persistent pass kernel
    int n_widths = 0;                     // plans of the solve: widths nb, nb-2, ..., (adaptive) or just nb
    int cap_widths = 0, cap_own = 0;
    std::vector<DevPlan> h_plans;
    DevPlan* d_plans = nullptr;
    CUtensorMap* d_maps = nullptr;        // [cap_widths][2][N_MAPS]
    CUtensorMap* d_mmaps = nullptr;       // [cap_widths]
    int* d_own_ptr = nullptr;             // [cap_widths][kMaxCtas + 1]
    int4* d_own = nullptr;                // [cap_widths][cap_own]
    SolveState* d_state = nullptr;
    long long* d_prof = nullptr;          // device counters: widths / launches of the passes that did work (F | A)
    long long prof_host[4] = {0, 0, 0, 0};   // same for the host-sequenced generic path
    size_t smem_f = 0, smem_a = 0;        // dynamic shared memory of the solve's launches (max over its plans)
    double* partials_rt = nullptr;        // [grid][nb]
    bool lazy = false;                    // W, X not cleared: the first pass F must not read them
    // plan cache: the tables above are rebuilt only when one of these changes
    struct PlanKey {
        int nb = 0, adaptive = 0, stencil = 0;
        const void* v[2][4] = {};
        const float* m = nullptr;
        wri_debug_opts dbg{};
    } plan_key;
    bool plan_valid = false;
    // optional per-kernel timing (wri_profile_*)
    bool profiling = false;
    std::vector<cudaEvent_t> ev_pool;     // pairs: start, stop
    std::vector<int> ev_kind;             // per pair: 0 = pass F, 1 = pass A
    size_t ev_used = 0;                   // pairs in use
    std::vector<std::pair<const void*, size_t>> smem_ok;   // kernels already granted their dynamic smem size
    // pipelined host-buffer solves (wri_set_host_pipeline): two staging slots, copy streams, events
    struct PipeSlot {
        float2 *Q = nullptr, *D = nullptr, *X = nullptr, *alpha = nullptr;
        float *tol = nullptr, *res = nullptr;
        int* its = nullptr;
        cudaEvent_t ev_in = nullptr, ev_solve = nullptr, ev_out = nullptr;
    } pipe[2];
    cudaStream_t s_in = nullptr, s_out = nullptr;
    int pipe_nb = 0, pipe_next = 0;       // width the staging was sized for (0 = no pipeline), next slot
};

namespace {

// Tile shape of the generic kernels for batch width nb: threads span the (ix, s) row first, then y;
// blocks march zc planes.
Tiling make_tiling(const wri_ctx* c, int nb) {
    Tiling t;
    t.vec = (nb % 2 == 0) ? 2 : 1;
    const long long items = (long long)c->g.nx * nb / t.vec;       // per x-row
    int tx = 128;
    while (tx > 32 && tx / 2 >= items) tx /= 2;
    int ty = 256 / tx;
    while (ty > 1 && ty / 2 >= c->g.ny) ty /= 2;
    t.block = dim3(tx, ty, 1);
    const unsigned gx = (unsigned)((items + tx - 1) / tx);
    const unsigned gy = (unsigned)((c->g.ny + ty - 1) / ty);
    // planes per tile: enough tiles for >= ~16 waves of 148 SMs x 4 blocks, but at least 8 planes
    int zc = c->g.nz;
    const long long want = 148LL * 4 * 16;
    while (zc > 8 && (long long)gx * gy * ((c->g.nz + zc - 1) / zc) < want) zc = (zc + 1) / 2;
    t.zc = zc;
    const unsigned gz = (unsigned)((c->g.nz + zc - 1) / zc);
    t.grid = dim3(gx, gy, gz);
    t.n_tiles = (size_t)gx * gy * gz;
    return t;
}

// Thread mapping of k_grad: the TPC = nb / vec threads of one cell sit side by side in a block row.
struct GradTiling { Tiling t; int tpc; int shuffle; bool ok; };
GradTiling make_grad_tiling(const wri_ctx* c, int nb) {
    GradTiling G{};
    G.t.vec = (nb % 2 == 0) ? 2 : 1;
    G.tpc = nb / G.t.vec;
    G.ok = G.tpc <= 512;
    if (!G.ok) return G;
    G.shuffle = G.tpc <= 32 && (G.tpc & (G.tpc - 1)) == 0;
    const int tx = G.shuffle ? 128 : G.tpc * std::max(1, 128 / G.tpc);
    int ty = std::max(1, 256 / tx);
    while (ty > 1 && ty / 2 >= c->g.ny) ty /= 2;
    if (G.shuffle && (tx * ty) % 32) ty = 1;
    G.t.block = dim3(tx, ty, 1);
    const long long row_threads = (long long)c->g.nx * G.tpc;
    const unsigned gx = (unsigned)((row_threads + tx - 1) / tx);
    const unsigned gy = (unsigned)((c->g.ny + ty - 1) / ty);
    int zc = c->g.nz;
    const long long want = 148LL * 4 * 4;
    while (zc > 8 && (long long)gx * gy * ((c->g.nz + zc - 1) / zc) < want) zc = (zc + 1) / 2;
    G.t.zc = zc;
    const unsigned gz = (unsigned)((c->g.nz + zc - 1) / zc);
    G.t.grid = dim3(gx, gy, gz);
    G.t.n_tiles = (size_t)gx * gy * gz;
    return G;
}

// Caller's workspace.  Vector regions hold n_g x even(nb) complex64 each: U, V, W always (an odd nb: one
// or two more); with WS_COMPACTION up to nine (the working set of an adaptive solve keeps X in the workspace and has a
// second vector set to re-pack into), with WS_HOST_STAGING the device copy of x for the host entry.
int grad_chunk_for(const wri_ctx* c, int nb);   // column chunk of the gradient pass (below)

struct WsLayout {
    size_t vecs[9], U_bot, partials, partials_rt, gscratch, Xs, Ds, tols, res, its, alphas, U_bot2, total;
    int n_vecs;
};
enum { WS_HOST_STAGING = 1, WS_COMPACTION = 2 };
WsLayout ws_layout(const wri_ctx* c, int nb, int flags, int maxit_cap) {
    WsLayout L{};
    const int nbe = even_up(nb);
    const size_t vec = align_up(c->ng * (size_t)nbe * sizeof(float2), 256);
    const size_t bot = align_up((size_t)std::max(c->n_rec, 1) * nbe * sizeof(float2), 256);
    const Tiling t = make_tiling(c, nb);
    size_t o = 0;
    L.n_vecs = 3;
    for (int i = 0; i < 3; ++i) { L.vecs[i] = o; o += vec; }
    L.U_bot = o; o += bot;
    const GradTiling gt = make_grad_tiling(c, nb);
    L.partials = o;
    o += align_up((std::max(t.n_tiles, gt.ok ? gt.t.n_tiles : 0) + kInitRowBlocks) * nbe * sizeof(double), 256);
    L.partials_rt = o; o += align_up((size_t)kMaxCtas * nbe * sizeof(double), 256);
    // one batch's gradient from the pass kernel, one array per column chunk
    const int gcb = grad_chunk_for(c, nb);
    L.gscratch = o; o += align_up(c->ng * sizeof(float), 256) * (size_t)(gcb ? nb / gcb : 1);
    if (flags & WS_HOST_STAGING) {
        L.Xs = o; o += vec;
        L.Ds = o; o += bot;
        L.tols = o; o += align_up((size_t)nbe * sizeof(float), 256);
        L.res = o; o += align_up((size_t)(maxit_cap + 1) * nbe * sizeof(float), 256);
        L.its = o; o += align_up((size_t)nbe * sizeof(int), 256);
        L.alphas = o; o += align_up((size_t)nbe * sizeof(float2), 256);
    }
    // an odd batch runs on the pass kernel in an even-width working set of its own (X too lives in the
    // workspace then; the host entry keeps its staged q in the V region meanwhile): one or two more regions
    if (nb & 1)
        for (int i = 0; i < ((flags & WS_HOST_STAGING) ? 2 : 1); ++i) { L.vecs[L.n_vecs++] = o; o += vec; }
    if (flags & WS_COMPACTION) {
        while (L.n_vecs < 9) { L.vecs[L.n_vecs++] = o; o += vec; }   // [8]: final x of retired columns
        L.U_bot2 = o; o += bot;
    }
    L.total = o;
    return L;
}
constexpr int kHostMaxitCap = 4096;   // resnorm staging rows reserved for wri_lsqr_batch_host

int upload_columns(wri_ctx* c, int nb, const int32_t* omega_idx, float lambda, int n_real = -1,
                   bool reuse = false) {
    // columns >= n_real are padding of an even-width working set (frequency 0, never active)
    if (n_real < 0) n_real = nb;
    std::vector<float> w2(nb), one(nb, 1.f), lam(nb, lambda), nlam(nb, -lambda), mone(nb, -1.f);
    std::vector<int> idx(nb);
    for (int s = 0; s < nb; ++s) {
        const int j = (omega_idx && s < n_real) ? omega_idx[s] : 0;
        if (j < 0 || j >= (int)c->omega.size()) return WRI_ERR_ARG;
        w2[s] = (float)(c->omega[j] * c->omega[j]);
        idx[s] = j;
    }
    // reuse: an operator / objective entry called again with the same columns and lambda
    if (reuse && c->up_cols_valid && c->up_lambda == lambda && c->up_idx == idx) return WRI_OK;
    c->up_cols_valid = false;
    const size_t NM = c->nb_max;
    float* cf = c->coef[0];
    CK(cudaMemcpyAsync(cf + C_W2 * NM, w2.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(cf + C_ONE * NM, one.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(cf + C_LAM * NM, lam.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(cf + C_NLAM * NM, nlam.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(cf + C_MONE * NM, mone.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    if (reuse) { c->up_idx.swap(idx); c->up_lambda = lambda; c->up_cols_valid = true; }
    return WRI_OK;
}

// source nodes of the source-free system, one per batch column -> c->src (cell indices)
int upload_sources(wri_ctx* c, int nb, const int32_t* src_ijk, bool reuse = false) {
    std::vector<int> cells(nb);
    for (int s = 0; s < nb; ++s) {
        const int ix = src_ijk[3 * s], iy = src_ijk[3 * s + 1], iz = src_ijk[3 * s + 2];
        if (ix < 0 || ix >= c->g.nx || iy < 0 || iy >= c->g.ny || iz < 0 || iz >= c->g.nz) return WRI_ERR_ARG;
        cells[s] = (iz * c->g.ny + iy) * c->g.nx + ix;
    }
    if (reuse && c->up_src_valid && c->up_src == cells) return WRI_OK;
    c->up_src_valid = false;
    // pageable source: the call returns once the data sits in the driver's staging buffer
    CK(cudaMemcpyAsync(c->src, cells.data(), nb * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    if (reuse) { c->up_src.swap(cells); c->up_src_valid = true; }
    return WRI_OK;
}

// Stencil of the discretised Laplacian (reading C-3 / C-23): weights of the centre, the 6 face, the 12
// edge and the 8 corner neighbours, in units of 1/h^2.
struct StencilW { double a0, a1, a2, a3; };
StencilW stencil_weights(int kind) {
    if (kind == WRI_STENCIL_27) return {-128.0 / 30.0, 14.0 / 30.0, 3.0 / 30.0, 1.0 / 30.0};
    return {-6.0, 1.0, 0.0, 0.0};
}

PassParams base_params(const wri_ctx* c, int nb, const Tiling& t) {
    PassParams p{};
    p.m = c->m;
    p.gx = c->gtab;
    p.gy = c->gtab + c->g.nx;
    p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef[0] + C_W2 * (size_t)c->nb_max;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = nb;
    p.zc = t.zc;
    const StencilW w = stencil_weights(c->stencil);
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(w.a0 / (c->h * c->h));
    p.a1 = (float)w.a1; p.a2 = (float)w.a2; p.a3 = (float)w.a3;
    p.sgn = 1.f;
    return p;
}

int profile_event_begin(wri_ctx* c, int kind, cudaEvent_t* e1) {
    *e1 = nullptr;
    if (!c->profiling) return WRI_OK;
    if (c->ev_used * 2 == c->ev_pool.size()) {
        cudaEvent_t a, b;
        CK(cudaEventCreate(&a));
        CK(cudaEventCreate(&b));
        c->ev_pool.push_back(a); c->ev_pool.push_back(b); c->ev_kind.push_back(0);
    }
    cudaEvent_t e0 = c->ev_pool[2 * c->ev_used];
    *e1 = c->ev_pool[2 * c->ev_used + 1];
    c->ev_kind[c->ev_used] = kind;
    c->ev_used++;
    CK(cudaEventRecord(e0, c->stream));
    return WRI_OK;
}

template <int MODE>
int launch_pass(wri_ctx* c, const PassParams& p, const Tiling& t, bool timed = false) {
    const size_t smem = (MODE == MODE_APPLY) ? 0 : (size_t)t.block.x * t.block.y * t.vec * sizeof(double);
    cudaEvent_t e1 = nullptr;
    if (timed) { int rc = profile_event_begin(c, MODE == MODE_F ? 0 : 1, &e1); if (rc) return rc; }
    const bool s27 = c->stencil == WRI_STENCIL_27;
    if (t.vec == 2) {
        if (s27) k_pass<2, MODE, ST_27><<<t.grid, t.block, smem, c->stream>>>(p);
        else     k_pass<2, MODE, ST_7><<<t.grid, t.block, smem, c->stream>>>(p);
    } else {
        if (s27) k_pass<1, MODE, ST_27><<<t.grid, t.block, smem, c->stream>>>(p);
        else     k_pass<1, MODE, ST_7><<<t.grid, t.block, smem, c->stream>>>(p);
    }
    c->launches++;
    CK(cudaGetLastError());
    if (e1) CK(cudaEventRecord(e1, c->stream));
    return WRI_OK;
}

ScalParams scal_params(const wri_ctx* c, const double* partials, int n_rows, const float2* d);

template <int PHASE>
int launch_scalars(wri_ctx* c, const float2* d, int extra_rows = 0) {
    ScalParams s = scal_params(c, c->partials, (int)c->tl.n_tiles + extra_rows, d);
    s.rows_in_pass = c->rt ? 1 : 0;
    s.init_rows = extra_rows > 0;
    const int T = 1024;
    const size_t smem = (size_t)(T + c->nb) * sizeof(double);
    k_scalars<PHASE><<<1, T, smem, c->stream>>>(s);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

// ---- persistent pass kernel: plans, tensor maps, launches ------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)ptr;
    }
    return fn;
}

// 4-D view (column, x, y, z) of a source-interleaved complex64 vector; one element = 8 bytes.
// Out-of-range box elements are zero-filled (the Dirichlet closure of the stencil).
// merged (nb == cb only): (column, x) folded into one dimension of nb*nx contiguous elements, so a box
// row is cb*bx elements (<= 256) — narrow chunks would otherwise move 16-128 byte rows.
// 128-byte L2 promotion: measured 0.7 % faster than 256 B at 128^3 x 64.
int make_tmap(CUtensorMap* tm, const void* base, const wri_ctx* c, int nb, int cb, int bx, int by, bool merged) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return cuda_fail(cudaErrorNotSupported, "cuTensorMapEncodeTiled lookup");
    cuuint64_t gdim[4] = {(cuuint64_t)nb, (cuuint64_t)c->g.nx, (cuuint64_t)c->g.ny, (cuuint64_t)c->g.nz};
    cuuint64_t gstr[3] = {(cuuint64_t)nb * 8, (cuuint64_t)nb * 8 * c->g.nx,
                          (cuuint64_t)nb * 8 * c->g.nx * c->g.ny};
    cuuint32_t box[4] = {(cuuint32_t)cb, (cuuint32_t)bx, (cuuint32_t)by, 1};
    if (merged) {
        gdim[0] = (cuuint64_t)nb * c->g.nx; gdim[1] = (cuuint64_t)c->g.ny; gdim[2] = (cuuint64_t)c->g.nz; gdim[3] = 1;
        gstr[0] = (cuuint64_t)nb * 8 * c->g.nx; gstr[1] = gstr[0] * c->g.ny; gstr[2] = gstr[1] * c->g.nz;
        box[0] = (cuuint32_t)(cb * bx); box[1] = (cuuint32_t)by; box[2] = 1; box[3] = 1;
    }
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, const_cast<void*>(base), gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_msg, sizeof g_cuda_msg, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return WRI_ERR_CUDA;
    }
    return WRI_OK;
}

// 3-D view (x, y, z) of the float32 model; needs a 16-byte row pitch
int make_tmap_model(CUtensorMap* tm, const wri_ctx* c, int bx, int by) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return cuda_fail(cudaErrorNotSupported, "cuTensorMapEncodeTiled lookup");
    cuuint64_t gdim[3] = {(cuuint64_t)c->g.nx, (cuuint64_t)c->g.ny, (cuuint64_t)c->g.nz};
    cuuint64_t gstr[2] = {(cuuint64_t)c->g.nx * 4, (cuuint64_t)c->g.nx * 4 * c->g.ny};
    cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1};
    cuuint32_t estr[3] = {1, 1, 1};
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(c->m), gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_msg, sizeof g_cuda_msg, "cuTensorMapEncodeTiled(model) failed with CUresult %d", (int)r);
        return WRI_ERR_CUDA;
    }
    return WRI_OK;
}

// Column chunk of the pass kernel for batch width nb: the whole width up to 64 columns (one chunk per
// cell), else the largest even divisor <= 64.  0 = the width is served by the generic kernels.
int rt_chunk_for(const wri_ctx* c, int nb) {
    if (c->dbg.generic || nb % 2 || !get_encode_fn()) return 0;
    if (nb <= RT_MAXW) return nb;
    for (int cb = RT_MAXW; cb >= 8; cb -= 2)
        if (nb % cb == 0) return cb;
    return 0;
}

// Column chunk of the gradient pass (MODE_G): its per-cell sum over the columns runs on warp shuffles and
// wants a power-of-two chunk.  The width itself when it is one (4 ... 64 columns), else the largest power of
// two that divides it (48 -> 3 x 16, 192 -> 3 x 64, 24 -> 3 x 8), each chunk with a gradient scratch of its
// own; 0 = generic kernel (odd widths, chunks below 8 columns: the scratch would pass 1/16 of a vector).
int grad_chunk_for(const wri_ctx* c, int nb) {
    if (!rt_chunk_for(c, nb)) return 0;
    int cb = 1;
    while (cb < RT_MAXW && nb % (2 * cb) == 0) cb *= 2;
    if (cb == nb) return nb >= 4 ? cb : 0;
    return cb >= 8 ? cb : 0;
}

// planes per tile and tile count of one pass.  With plenty of tiles the measured preferences hold
// (profiles/r02_width_sweeps.md; an L2 effect: short tiles keep the halo that neighbouring tiles share
// resident across a wave of tiles): pass F 16 planes; pass A 16 planes up to 24 columns and on grids of
// 256 planes and more (256^3 x 32: 0.93 -> 1.00 of the copy bandwidth), 32 otherwise.  With
// few tiles (narrow widths, small grids) the chunk count that minimises rounds x (planes + priming)
// over the persistent grid is taken instead.
PassGeo plan_pass(const wri_ctx* c, const DevPlan& P, bool is_f, int zc_forced) {
    PassGeo G{};
    const int nz = c->g.nz, sms = std::max(1, c->num_sms);
    const long long cols = (long long)P.nchunk * P.ntx * P.nty;
    int zc = is_f ? 16 : ((P.cb <= 24 || nz >= 256) ? 16 : 32);
    if (zc_forced > 0) zc = (zc_forced + 7) / 8 * 8;          // multiples of 8 planes (see the |.|^2 sums of the kernel)
    else if (cols * ((nz + zc - 1) / zc) < 6LL * sms) {
        const double prime = is_f ? 0.6 : 1.2;               // two priming planes in units of a full step
        double best = 1e300;
        for (int z = 8; z < nz + 8; z += 8) {
            const long long tiles = cols * ((nz + z - 1) / z);
            const double cost = (double)((tiles + sms - 1) / sms) * (std::min(z, nz) + prime);
            if (cost < best * 0.999) { best = cost; zc = z; }
        }
    }
    G.zc = zc;
    G.ntz = (nz + zc - 1) / zc;
    G.n_tiles = (int)std::min<long long>(cols * G.ntz, 0x7fffffffLL);
    return G;
}

// Tile geometry for batch width nb (see DevPlan).  The x/y shape minimises, per z-plane of the grid,
// the stencil input the tiles pull through L2 (halo included) plus the issue slots of the 512
// consumer threads (idle ones included), with a penalty for tile rows below 512 contiguous bytes
// and a small one for shapes whose model tile cannot ride in the TMA stage.
int make_plan(const wri_ctx* c, int nb, DevPlan& P, int cb_forced = 0) {
    std::memset(&P, 0, sizeof P);
    const int cb = cb_forced > 0 ? cb_forced : rt_chunk_for(c, nb);
    if (!cb || nb % cb) return WRI_ERR_ARG;
    P.nb = nb; P.cb = cb; P.hp = cb / 2; P.nchunk = nb / cb;
    const int maxcells = RT_NT / P.hp;
    const int nx = c->g.nx, ny = c->g.ny;
    const bool m_al = (nx % 4 == 0) && aligned16(c->m);
    double best = 1e300;
    int btx = 1, bty = 1;
    if (c->dbg.txc > 0 && c->dbg.tyc > 0 && c->dbg.txc * c->dbg.tyc <= maxcells) { btx = c->dbg.txc; bty = c->dbg.tyc; }
    else
        for (int tyc = 1; tyc <= std::min(maxcells, 64); ++tyc)
            for (int txc = 1; txc * tyc <= maxcells && txc <= 254; ++txc) {
                // three F stages (halo box + three centre boxes) must fit
                const size_t stage = align_up((size_t)(txc + 2) * (tyc + 2) * cb * 8, 128) +
                                     3 * align_up((size_t)txc * tyc * cb * 8, 128) + 128;
                if (2 * stage + 24576 > (size_t)RT_SMEM_MAX) continue;
                const double ntx = (nx + txc - 1) / txc, nty = (ny + tyc - 1) / tyc;
                // (from 16 columns on idle consumer threads cost little — 384 busy ones keep pass A at its
                // rate — and contiguous tile rows below 2 KB cost a lot: 48 columns as 8 x 2 cells run 4 %
                // faster than as 4 x 5, profiles/r02_width_sweeps.md)
                const bool long_rows = cb >= 10 || cb == 6;      // (2, 4 and 8 columns: measured no gain)
                double cost = ntx * nty * ((txc + 2.0) * (tyc + 2.0) + (long_rows ? 0.25 : 0.75) * maxcells);
                const int row_bytes = txc * cb * 8;
                if (row_bytes < 512 && txc < nx) cost *= 1.0 + 0.25 * (512 - row_bytes) / 512.0;
                if (long_rows && row_bytes < 2048 && txc < nx) cost *= 1.0 + (2048 - row_bytes) / 2048.0;
                // below 32 columns a box row should carry (column, x) folded into one dimension
                if (cb < 32 && !(P.nchunk == 1 && cb * (txc + 2) <= 256)) cost *= 1.2;
                // tile rows that do not start on 128-byte lines: measured 6-10 % slower in both passes
                // (widths 6, 10: profiles/r02_width_sweeps.md)
                if (row_bytes % 128 != 0 && txc < nx) cost *= 1.2;
                if (!(m_al && txc % 4 == 0)) cost *= 1.3;    // model tile by plain loads: pass A 0.98 -> 0.80 at 48 columns
                if (cost < best) { best = cost; btx = txc; bty = tyc; }
            }
    P.txc = btx; P.tyc = bty;
    P.items = btx * bty * P.hp;
    P.ntx = (nx + btx - 1) / btx;
    P.nty = (ny + bty - 1) / bty;
    P.merged = (P.nchunk == 1 && cb * (btx + 2) <= 256) ? 1 : 0;
    P.m_tma = (m_al && btx % 4 == 0) ? 1 : 0;
    // pass F reads the model by plain loads: +1 to +4 % at every width (profiles/r02_width_sweeps.md)
    P.f_m_ldg = c->dbg.m_ldg_f == 2 ? 0 : 1;
    P.row_b = (btx + 2) * cb * 8;
    P.cell_b = cb * 8;
    P.in_bytes = (btx + 2) * (bty + 2) * cb * 8;
    P.in_span = (int)align_up(P.in_bytes, 128);
    P.ctr_bytes = btx * bty * cb * 8;
    P.ctr_span = (int)align_up(P.ctr_bytes, 128);
    P.m_bytes = P.m_tma ? btx * bty * 4 : 0;
    P.m_span = (int)align_up(P.m_bytes, 128);
    P.f = plan_pass(c, P, true, c->dbg.zc_f);
    P.a = plan_pass(c, P, false, c->dbg.zc_a);
    // ring depth of pass A: near 150 KB of stages in flight per SM (measured optimum,
    // profiles/r01_v6_stages.md: a deeper ring costs L2 hits on the stencil halo, a shallower one
    // leaves the copy engine idle), within the shared memory that is left
    const int nxyz = c->g.nx + c->g.ny + c->g.nz;
    auto depth = [&](int nstream, double target, int lo, int hi, int forced) {
        const int stage = rt_stage_bytes(P, nstream);
        int n = forced > 0 ? std::min(forced, RT_MAX_STAGES)
                           : std::max(lo, std::min((int)std::floor(target / stage + 0.5), hi));
        while (n > 2 && rt_smem_bytes(P, nstream, n, nxyz) > (size_t)RT_SMEM_MAX) --n;
        return n;
    };
    // pass F: three stages.  A fourth costs 4-8 % wherever the stage is small enough to afford it (widths
    // 18, 22, 26, 34, 44, 46: profiles/r02_width_sweeps.md) — more loads in flight than the L2 keeps halos for
    P.f.nstage = depth(3, 120e3, 2, cb < 8 ? 4 : 3, c->dbg.nstage_f);
    P.a.nstage = depth(1, 150e3, 3, 10, c->dbg.nstage_a);
    if (rt_smem_bytes(P, 3, P.f.nstage, nxyz) > (size_t)RT_SMEM_MAX) return WRI_ERR_ARG;
    return WRI_OK;
}

// opt-in to > 48 KB of dynamic shared memory, once per (context, kernel).  The attribute belongs to the
// function on the device, not to the context: it is always raised to the same ceiling, so that two
// contexts with different needs cannot lower it under one another.
int allow_smem(wri_ctx* c, const void* fn, size_t bytes) {
    if (bytes > (size_t)RT_SMEM_MAX) return WRI_ERR_ARG;
    for (auto& e : c->smem_ok)
        if (e.first == fn) return WRI_OK;
    CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, RT_SMEM_MAX));
    c->smem_ok.emplace_back(fn, (size_t)RT_SMEM_MAX);
    return WRI_OK;
}

// receivers (x column chunks) inside each CTA's tiles of pass A, in the order the CTA walks its tiles
// (same tile numbering as the kernel): CSR over CTAs + {receiver, cell, tile, entries of this tile}
void build_own(const wri_ctx* c, const DevPlan& P, int grid, std::vector<int>& ptr, std::vector<int4>& own) {
    const int nent = c->n_rec * P.nchunk;
    struct Ent { int cta, tile, r; };
    std::vector<Ent> ents(nent);
    for (int e = 0; e < nent; ++e) {
        const int r = e / P.nchunk, chunk = e % P.nchunk;
        const int tx = c->rec_ijk[3 * r] / P.txc, ty = c->rec_ijk[3 * r + 1] / P.tyc;
        const int tz = c->rec_ijk[3 * r + 2] / P.a.zc;
        const int t = (int)((((long long)tz * P.nty + ty) * P.ntx + tx) * P.nchunk + chunk);
        ents[e] = {t % grid, t, r};
    }
    std::sort(ents.begin(), ents.end(), [](const Ent& a, const Ent& b) {
        return a.cta != b.cta ? a.cta < b.cta : a.tile != b.tile ? a.tile < b.tile : a.r < b.r;
    });
    ptr.assign(kMaxCtas + 1, 0);
    own.assign(std::max(nent, 1), make_int4(-1, -1, -1, 0));
    for (int e = 0; e < nent; ++e) ptr[ents[e].cta + 1]++;
    for (int b = 0; b < kMaxCtas; ++b) ptr[b + 1] += ptr[b];
    for (int e = 0; e < nent;) {
        int f = e;
        while (f < nent && ents[f].cta == ents[e].cta && ents[f].tile == ents[e].tile) ++f;
        for (int j = e; j < f; ++j) {
            const int r = ents[j].r;
            const int cell = (c->rec_ijk[3 * r + 2] * c->g.ny + c->rec_ijk[3 * r + 1]) * c->g.nx + c->rec_ijk[3 * r];
            own[j] = make_int4(r, cell, ents[j].tile, j == e ? f - e : 0);
        }
        e = f;
    }
}

int rt_grid(const wri_ctx* c) { return std::max(1, std::min(c->num_sms, kMaxCtas)); }

// Plans, tensor maps and receiver lists of the solve that is starting: one entry per width the working
// set can have (nb, nb-2, ..., 2 for an adaptive solve, else nb alone), for both vector sets.  Cached:
// rebuilt only when the widths, the vector slots, the model pointer or the options change.
int rt_setup(wri_ctx* c) {
    wri_ctx::PlanKey key;
    key.nb = c->nb; key.adaptive = c->adaptive; key.stencil = c->stencil; key.m = c->m; key.dbg = c->dbg;
    for (int p = 0; p < 2; ++p)
        for (int q = 0; q < 4; ++q) key.v[p][q] = c->vec[p][q];
    auto same = [](const wri_ctx::PlanKey& a, const wri_ctx::PlanKey& b) {
        if (a.nb != b.nb || a.adaptive != b.adaptive || a.stencil != b.stencil || a.m != b.m) return false;
        for (int p = 0; p < 2; ++p)
            for (int q = 0; q < 4; ++q)
                if (a.v[p][q] != b.v[p][q]) return false;
        const wri_debug_opts &x = a.dbg, &y = b.dbg;
        return x.nstage_f == y.nstage_f && x.nstage_a == y.nstage_a && x.zc_f == y.zc_f && x.zc_a == y.zc_a &&
               x.txc == y.txc && x.tyc == y.tyc && x.generic == y.generic && x.m_ldg_f == y.m_ldg_f;
    };
    if (c->plan_valid && same(key, c->plan_key)) return WRI_OK;
    c->plan_valid = false;
    const int nw = c->adaptive ? c->nb / 2 : 1;
    const int own_cap = std::max(1, c->n_rec * std::max(1, c->nb / std::max(2, rt_chunk_for(c, c->nb))));
    if (nw > c->cap_widths || own_cap > c->cap_own) {
        // the tables are in use by nothing: every earlier solve of this context was enqueued on the same
        // stream, and cudaFree waits for the device
        cudaFree(c->d_plans); cudaFree(c->d_maps); cudaFree(c->d_mmaps); cudaFree(c->d_own_ptr); cudaFree(c->d_own);
        c->d_plans = nullptr; c->d_maps = nullptr; c->d_mmaps = nullptr; c->d_own_ptr = nullptr; c->d_own = nullptr;
        c->cap_widths = std::max(nw, c->cap_widths);
        c->cap_own = std::max(own_cap, c->cap_own);
        CK(cudaMalloc(&c->d_plans, (size_t)c->cap_widths * sizeof(DevPlan)));
        CK(cudaMalloc(&c->d_maps, (size_t)c->cap_widths * 2 * N_MAPS * sizeof(CUtensorMap)));
        CK(cudaMalloc(&c->d_mmaps, (size_t)c->cap_widths * sizeof(CUtensorMap)));
        CK(cudaMalloc(&c->d_own_ptr, (size_t)c->cap_widths * (kMaxCtas + 1) * sizeof(int)));
        CK(cudaMalloc(&c->d_own, (size_t)c->cap_widths * c->cap_own * sizeof(int4)));
    }
    c->h_plans.assign(nw, DevPlan{});
    std::vector<CUtensorMap> maps((size_t)nw * 2 * N_MAPS), mmaps(nw);
    std::vector<int> own_ptr((size_t)nw * (kMaxCtas + 1), 0);
    std::vector<int4> own((size_t)nw * c->cap_own, make_int4(-1, -1, -1, 0));
    const int nxyz = c->g.nx + c->g.ny + c->g.nz;
    c->smem_f = c->smem_a = 0;
    int rc;
    for (int wi = 0; wi < nw; ++wi) {
        const int w = c->nb - 2 * wi;
        DevPlan& P = c->h_plans[wi];
        if ((rc = make_plan(c, w, P))) return rc;
        c->smem_f = std::max(c->smem_f, rt_smem_bytes(P, 3, P.f.nstage, nxyz));
        c->smem_a = std::max(c->smem_a, rt_smem_bytes(P, 1, P.a.nstage, nxyz));
        for (int par = 0; par < (c->adaptive ? 2 : 1); ++par) {
            CUtensorMap* M = &maps[((size_t)wi * 2 + par) * N_MAPS];
            const bool mg = P.merged != 0;
            float2* const* v = c->vec[par];
            if ((rc = make_tmap(&M[MP_V_HALO], v[1], c, w, P.cb, P.txc + 2, P.tyc + 2, mg))) return rc;
            if ((rc = make_tmap(&M[MP_U_HALO], v[0], c, w, P.cb, P.txc + 2, P.tyc + 2, mg))) return rc;
            if ((rc = make_tmap(&M[MP_U_CTR], v[0], c, w, P.cb, P.txc, P.tyc, mg))) return rc;
            if ((rc = make_tmap(&M[MP_V_CTR], v[1], c, w, P.cb, P.txc, P.tyc, mg))) return rc;
            if ((rc = make_tmap(&M[MP_W_CTR], v[2], c, w, P.cb, P.txc, P.tyc, mg))) return rc;
            if ((rc = make_tmap(&M[MP_X_CTR], v[3], c, w, P.cb, P.txc, P.tyc, mg))) return rc;
        }
        if (P.m_tma && (rc = make_tmap_model(&mmaps[wi], c, P.txc, P.tyc))) return rc;
        if (c->n_rec) {
            std::vector<int> ptr;
            std::vector<int4> ow;
            build_own(c, P, rt_grid(c), ptr, ow);
            std::copy(ptr.begin(), ptr.end(), own_ptr.begin() + (size_t)wi * (kMaxCtas + 1));
            std::copy(ow.begin(), ow.begin() + std::min<size_t>(ow.size(), c->cap_own), own.begin() + (size_t)wi * c->cap_own);
        }
    }
    // pageable sources: each call returns once the data sits in the driver's staging buffer
    CK(cudaMemcpyAsync(c->d_plans, c->h_plans.data(), nw * sizeof(DevPlan), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_maps, maps.data(), maps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_mmaps, mmaps.data(), mmaps.size() * sizeof(CUtensorMap), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_own_ptr, own_ptr.data(), own_ptr.size() * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->d_own, own.data(), own.size() * sizeof(int4), cudaMemcpyHostToDevice, c->stream));
    c->n_widths = nw;
    c->plan_key = key;
    c->plan_valid = true;
    return WRI_OK;
}

ScalParams scal_params(const wri_ctx* c, const double* partials, int n_rows, const float2* d) {
    ScalParams s{};
    s.partials = partials;
    s.n_tiles = n_rows;
    s.nb = c->nb; s.nb_max = c->nb_max;
    s.n_rec = c->n_rec; s.rec = c->rec;
    s.V = c->V; s.U_bot = c->U_bot[0]; s.d = d;
    s.coef = c->coef[0]; s.stat = c->stat[0]; s.active = c->active[0]; s.iters = c->iters[0];
    s.tol = c->tol; s.resnorms = c->resnorms; s.iters_out = c->iters_out;
    s.progress = c->pacing ? c->d_prog : nullptr;
    s.solve_id = c->solve_id;
    s.k = c->k; s.maxit = c->maxit; s.lambda = c->lambda;
    s.rows_in_pass = 1;
    s.colmap = c->packed ? c->colmap : nullptr;
    s.nb_out = c->nb0;
    s.src = c->sf ? c->src : nullptr;
    s.U = c->U;
    s.alpha_out = c->sf ? c->alpha_out : nullptr;
    s.warm = c->opts.warm_start;
    s.X = c->X;
    s.ar_ref = c->opts.ar_ref_dev;
    s.ar0_out = c->opts.ar0_out_dev;
    s.rmask = c->rmask;
    return s;
}

void rt_common(const wri_ctx* c, RtParams& p) {
    const StencilW w = stencil_weights(c->stencil);
    p.m = c->m;
    p.gtab = c->gtab;
    p.counter = c->counter;
    p.prof = c->d_prof;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb_max = c->nb_max;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.a0h = (float)(w.a0 / (c->h * c->h));
    p.a1 = (float)w.a1; p.a2 = (float)w.a2; p.a3 = (float)w.a3;
    for (int par = 0; par < 2; ++par) {
        p.coef[par] = c->coef[par]; p.stat[par] = c->stat[par];
        p.active[par] = c->active[par]; p.iters[par] = c->iters[par];
    }
}

template <int MODE, bool TRK = false>
const void* rt_kernel(const wri_ctx* c) {
    return c->stencil == WRI_STENCIL_27 ? (const void*)k_pass_rt<MODE, ST_27, TRK>
                                        : (const void*)k_pass_rt<MODE, ST_7, TRK>;
}

// parameters of one pass of the solve in flight (the same for every iteration: what changes lives
// in the device-resident state)
template <int MODE>
RtParams rt_solve_params(const wri_ctx* c, int phase) {
    RtParams p{};
    rt_common(c, p);
    p.st = c->d_state;
    p.plans = c->d_plans; p.maps = c->d_maps; p.mmaps = c->d_mmaps;
    p.own_ptr_tab = c->d_own_ptr; p.own_tab = c->d_own;
    p.own_ptr_stride = kMaxCtas + 1; p.own_stride = c->cap_own;
    for (int par = 0; par < 2; ++par) {
        for (int q = 0; q < 4; ++q) p.vec[par][q] = c->vec[par][q];
        p.U_bot[par] = c->U_bot[par];
    }
    p.partials = c->partials_rt;
    p.sgn = (MODE == MODE_F) ? 1.f : -1.f;
    p.phase = phase;
    // streams known to be zero are neither cleared nor read: V in the start's adjoint pass, W and X in
    // the first forward pass of a cold batch solve (c->lazy)
    p.has_old = (MODE == MODE_A) ? (phase != PH_INIT_A) : 1;
    p.lazy = c->lazy;
    p.packed = c->packed; p.adaptive = c->adaptive;
    p.retire_buf = c->retire_buf; p.retired = c->retired;
    p.maxit = c->maxit;
    p.n_rec = c->n_rec; p.rec = c->rec;
    p.fin = scal_params(c, c->partials_rt, rt_grid(c), nullptr);
    return p;
}

template <int MODE>
int launch_rt(wri_ctx* c, int phase) {
    // every launch of a solve asks for the same (maximal) amount of dynamic shared memory: kernels that
    // alternate between different sizes make the SMs re-partition their L1 / shared memory in between
    if (std::max(c->smem_f, c->smem_a) > (size_t)RT_SMEM_MAX) return WRI_ERR_ARG;
    const size_t smem = RT_SMEM_MAX;
    const void* fn = rt_kernel<MODE>(c);
    int rc = allow_smem(c, fn, smem);
    if (rc) return rc;
    RtParams p = rt_solve_params<MODE>(c, phase);
    p.it = c->k;
    CUtensorMap dummy{};
    cudaEvent_t e1 = nullptr;
    if (phase != PH_INIT_A && (rc = profile_event_begin(c, MODE == MODE_F ? 0 : 1, &e1))) return rc;
    void* args[] = {&dummy, &dummy, &dummy, &p};
    // programmatic dependent launch: the next pass's CTAs move in while this one's last CTA still runs
    // its finaliser, and wait (griddepcontrol.wait at the top of the kernel) for the launch to complete
    cudaLaunchAttribute attr{};
    attr.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr.val.programmaticStreamSerializationAllowed = 1;
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(rt_grid(c)); cfg.blockDim = dim3(RT_NT + 32);
    cfg.dynamicSmemBytes = smem; cfg.stream = c->stream;
    cfg.attrs = &attr; cfg.numAttrs = 1;
    CK(cudaLaunchKernelExC(&cfg, fn, args));
    c->launches++;
    if (c->adaptive && phase != PH_INIT_A) {
        // the re-packing variant of the same pass: exactly one of the two does the work (decided on the
        // device from the solve state), the other returns at once
        const void* fn_t = rt_kernel<MODE, true>(c);
        if ((rc = allow_smem(c, fn_t, smem))) return rc;
        CK(cudaLaunchKernelExC(&cfg, fn_t, args));
        c->launches++;
    }
    if (e1) CK(cudaEventRecord(e1, c->stream));
    return WRI_OK;
}

MoveParams move_params(const wri_ctx* c) {
    MoveParams p{};
    p.st = c->d_state; p.plans = c->d_plans;
    for (int par = 0; par < 2; ++par) {
        for (int q = 0; q < 4; ++q) p.vec[par][q] = c->vec[par][q];
        p.U_bot[par] = c->U_bot[par];
        p.coef[par] = c->coef[par]; p.stat[par] = c->stat[par];
        p.active[par] = c->active[par]; p.iters[par] = c->iters[par];
    }
    p.u_out = c->u_out; p.resnorms = c->resnorms;
    p.n_g = (long long)c->ng; p.nb_out = c->nb0; p.nb_max = c->nb_max; p.maxit = c->maxit; p.n_rec = c->n_rec;
    p.packed = c->packed;
    p.R = c->adaptive ? c->retire_buf : nullptr;
    p.retired = c->retired;
    p.col0 = c->col0; p.ncols = c->ncols;
    return p;
}

// A static launch of the pass kernel (operator entries, gradient pass, warm start): plan and tensor
// maps travel as kernel parameters, nothing is read from the solve state.
struct StaticLaunch {
    DevPlan P;
    CUtensorMap in, old, m;
    size_t smem;
    int grid;
};
int static_plan(wri_ctx* c, int nb, const void* in, const void* old, StaticLaunch& S, size_t reserve = 0,
                int cb_forced = 0) {
    int rc = make_plan(c, nb, S.P, cb_forced);
    if (rc) return rc;
    DevPlan& P = S.P;
    // one light stream: long tiles (128 planes: 0.88 -> 0.90 of the copy bandwidth at 128^3 x 64) and the
    // deepest ring that fits (measured for the operator entries: deeper is better)
    // (one chunk per cell, grids below 256 planes: at 256^3 x 32 and at 128^3 x 192 it costs 10 %)
    if (!c->dbg.zc_a && P.a.zc < 128 && P.nchunk == 1 && c->g.nz < 256 &&
        (long long)P.ntx * P.nty >= 6LL * rt_grid(c)) {
        P.a.zc = 128;
        P.a.ntz = (c->g.nz + 127) / 128;
        P.a.n_tiles = P.nchunk * P.ntx * P.nty * P.a.ntz;
    }
    const int nxyz = c->g.nx + c->g.ny + c->g.nz;
    int n = c->dbg.nstage_a > 0 ? c->dbg.nstage_a : RT_MAX_STAGES;
    n = std::min(n, RT_MAX_STAGES);
    while (n > 2 && rt_smem_bytes(P, 1, n, nxyz) + reserve > (size_t)RT_SMEM_MAX) --n;
    P.a.nstage = n;
    S.smem = rt_smem_bytes(P, 1, n, nxyz) + reserve;
    S.grid = std::min(P.a.n_tiles, rt_grid(c));
    const bool mg = P.merged != 0;
    if ((rc = make_tmap(&S.in, in, c, nb, P.cb, P.txc + 2, P.tyc + 2, mg))) return rc;
    if ((rc = make_tmap(&S.old, old ? old : in, c, nb, P.cb, P.txc, P.tyc, mg))) return rc;
    if (P.m_tma) { if ((rc = make_tmap_model(&S.m, c, P.txc, P.tyc))) return rc; }
    else S.m = S.old;
    return WRI_OK;
}

template <int MODE>
int launch_static(wri_ctx* c, StaticLaunch& S, RtParams& p) {
    const void* fn = rt_kernel<MODE>(c);
    int rc = allow_smem(c, fn, S.smem);
    if (rc) return rc;
    rt_common(c, p);
    p.st = nullptr;
    p.plan0 = S.P;
    void* args[] = {&S.in, &S.old, &S.m, &p};
    CK(cudaLaunchKernel(fn, dim3(S.grid), dim3(RT_NT + 32), args, S.smem, c->stream));
    c->launches++;
    return WRI_OK;
}

// out = lambda * A in (sgn = +1) or lambda * A^H in (sgn = -1): the pass kernel without its in-place
// stream, scalar phase and receiver rows; the generic kernel for odd widths.  No workspace is touched.
int apply_operator(wri_ctx* c, int nb, const float2* in, float2* out, float sgn) {
    if (!c->solving && rt_chunk_for(c, nb)) {
        StaticLaunch S;
        int rc = static_plan(c, nb, in, nullptr, S);
        if (rc) return rc;
        RtParams p{};
        p.sgn = sgn; p.phase = -1; p.has_old = 0;
        p.ca_static = c->coef[0] + C_LAM * (size_t)c->nb_max;
        p.out = out;
        return launch_static<MODE_A>(c, S, p);
    }
    const Tiling t = make_tiling(c, nb);
    PassParams p = base_params(c, nb, t);
    p.in = in; p.out = out;
    p.ca = c->coef[0] + C_LAM * (size_t)c->nb_max;
    p.sgn = sgn;
    return launch_pass<MODE_APPLY>(c, p, t);
}

int check_batch_args(const wri_ctx* c, int nb) {
    if (!c) return WRI_ERR_ARG;
    if (nb <= 0 || nb > c->nb_max) return WRI_ERR_ARG;
    if (c->rmask && c->rmask_nb != nb) return WRI_ERR_ARG;       // the receiver mask was given for another width
    if ((long long)c->ng * even_up(nb) > 0x7fffffffLL * 1LL) return WRI_ERR_ARG;   // element indices stay below 2^31
    return WRI_OK;
}

}  // namespace

extern "C" {

const char* wri_strerror(int code) {
    switch (code) {
        case WRI_OK: return "ok";
        case WRI_ERR_ARG: return "invalid argument (null pointer, bad size, nb > nb_max, or misaligned buffer)";
        case WRI_ERR_RECEIVER_RANGE: return "receiver node outside the grid";
        case WRI_ERR_RECEIVER_DUP: return "duplicate receiver node";
        case WRI_ERR_WORKSPACE: return "workspace missing or too small";
        case WRI_ERR_CUDA: return g_cuda_msg;
        case WRI_ERR_STATE: return "call out of order";
        case WRI_ERR_NUMERIC: return "objective is not finite";
        case WRI_ERR_SCRATCH_LIMIT:
            return "wri_objective_gradient_static: grid x batch width needs more than the "
                   "WRI_STATIC_SCRATCH_BYTES (4 MiB) of built-in scratch; use wri_objective_gradient with a workspace";
        default: return "unknown error code";
    }
}

int wri_create(wri_ctx** out, wri_grid grid, double h, int32_t n_omega, const double* omega_host,
               const float* m_dev, wri_sponge sponge, int32_t n_rec, const int32_t* rec_ijk_host,
               int32_t nb_max, void* cuda_stream) {
    if (!out) return WRI_ERR_ARG;
    *out = nullptr;
    if (grid.nx <= 0 || grid.ny <= 0 || grid.nz <= 0 || !(h > 0.0) || n_omega <= 0 || !omega_host ||
        !m_dev || n_rec < 0 || (n_rec > 0 && !rec_ijk_host) || nb_max <= 0 || sponge.width < 0 ||
        sponge.power < 0)
        return WRI_ERR_ARG;
    const size_t ng = (size_t)grid.nx * grid.ny * grid.nz;
    if (ng > 0x7fffffffULL) return WRI_ERR_ARG;
    // receivers: validated on the host before any CUDA call (reading C-8)
    std::vector<int> cells(n_rec);
    for (int r = 0; r < n_rec; ++r) {
        const int ix = rec_ijk_host[3 * r], iy = rec_ijk_host[3 * r + 1], iz = rec_ijk_host[3 * r + 2];
        if (ix < 0 || ix >= grid.nx || iy < 0 || iy >= grid.ny || iz < 0 || iz >= grid.nz)
            return WRI_ERR_RECEIVER_RANGE;
        cells[r] = (iz * grid.ny + iy) * grid.nx + ix;
    }
    {
        std::vector<int> sorted(cells);
        std::sort(sorted.begin(), sorted.end());
        if (std::adjacent_find(sorted.begin(), sorted.end()) != sorted.end()) return WRI_ERR_RECEIVER_DUP;
    }
    int ndev = 0;
    CK(cudaGetDeviceCount(&ndev));
    if (ndev <= 0) return cuda_fail(cudaErrorNoDevice, "wri_create");

    wri_ctx* c = new wri_ctx();
    c->g = grid; c->h = h; c->ng = ng;
    c->omega.assign(omega_host, omega_host + n_omega);
    c->sponge = sponge; c->n_rec = n_rec;
    c->nb_max = even_up(nb_max);                     // an odd batch runs in an even-width working set
    c->stream = (cudaStream_t)cuda_stream;
    c->m = m_dev;
    const int NM = c->nb_max;

    // sponge profile per axis, computed in double and rounded once; gamma = max over axes
    const int L = sponge.width;
    std::vector<float> gt((size_t)grid.nx + grid.ny + grid.nz, 0.f);
    auto fill = [&](float* dst, int n, bool lo, bool hi) {
        for (int i = 0; i < n; ++i) {
            double d = 0.0;
            if (L > 0) {
                if (lo) d = std::max(d, (double)(L - i));
                if (hi) d = std::max(d, (double)(i - (n - 1 - L)));
                dst[i] = (float)((double)sponge.gamma_max * std::pow(d / (double)L, (double)sponge.power));
                if (d == 0.0) dst[i] = 0.f;
            }
        }
    };
    fill(gt.data(), grid.nx, sponge.faces & 1u, sponge.faces & 2u);
    fill(gt.data() + grid.nx, grid.ny, sponge.faces & 4u, sponge.faces & 8u);
    fill(gt.data() + grid.nx + grid.ny, grid.nz, sponge.faces & 16u, sponge.faces & 32u);

    auto fail = [&](int code) { wri_destroy(c); return code; };
#define CKC(call)                                                          \
    do {                                                                   \
        cudaError_t e__ = (call);                                          \
        if (e__ != cudaSuccess) return fail(cuda_fail(e__, #call));        \
    } while (0)
    CKC(cudaMalloc(&c->gtab, gt.size() * sizeof(float)));
    CKC(cudaMemcpy(c->gtab, gt.data(), gt.size() * sizeof(float), cudaMemcpyHostToDevice));
    CKC(cudaMalloc(&c->rec, std::max(n_rec, 1) * sizeof(int)));
    if (n_rec) CKC(cudaMemcpy(c->rec, cells.data(), n_rec * sizeof(int), cudaMemcpyHostToDevice));
    c->rec_ijk.assign(rec_ijk_host, rec_ijk_host + 3 * (size_t)n_rec);
    for (int b = 0; b < 2; ++b) {
        CKC(cudaMalloc(&c->coef[b], (size_t)N_COEF * NM * sizeof(float)));
        CKC(cudaMemset(c->coef[b], 0, (size_t)N_COEF * NM * sizeof(float)));
        CKC(cudaMalloc(&c->stat[b], (size_t)N_STAT * NM * sizeof(double)));
        CKC(cudaMemset(c->stat[b], 0, (size_t)N_STAT * NM * sizeof(double)));
        CKC(cudaMalloc(&c->active[b], NM * sizeof(int)));
        CKC(cudaMalloc(&c->iters[b], NM * sizeof(int)));
        CKC(cudaMemset(c->active[b], 0, NM * sizeof(int)));
        CKC(cudaMemset(c->iters[b], 0, NM * sizeof(int)));
    }
    CKC(cudaMalloc(&c->colmap, NM * sizeof(int)));
    CKC(cudaMalloc(&c->retired, NM * sizeof(int)));
    CKC(cudaMalloc(&c->src, NM * sizeof(int)));
    CKC(cudaMalloc(&c->aw_tol, NM * sizeof(float)));
    CKC(cudaMalloc(&c->aw_f, (size_t)2 * NM * sizeof(double)));
    CKC(cudaMalloc(&c->aw_ar0, NM * sizeof(double)));
    CKC(cudaMalloc(&c->aw_iters, NM * sizeof(int)));
    CKC(cudaMallocHost(&c->h_aw, (size_t)NM * (2 * sizeof(double) + sizeof(int))));
    CKC(cudaHostAlloc((void**)&c->h_prog, 64, cudaHostAllocMapped));
    *c->h_prog = 0;
    CKC(cudaHostGetDevicePointer((void**)&c->d_prog, c->h_prog, 0));
    CKC(cudaMalloc(&c->counter, sizeof(unsigned int)));
    CKC(cudaMemset(c->counter, 0, sizeof(unsigned int)));
    CKC(cudaMalloc(&c->d_state, sizeof(SolveState)));
    CKC(cudaMemset(c->d_state, 0, sizeof(SolveState)));
    CKC(cudaMalloc(&c->d_prof, 4 * sizeof(long long)));
    CKC(cudaMemset(c->d_prof, 0, 4 * sizeof(long long)));
    {
        int dev = 0;
        CKC(cudaGetDevice(&dev));
        CKC(cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, dev));
    }
#undef CKC
    *out = c;
    return WRI_OK;
}

int wri_destroy(wri_ctx* c) {
    if (!c) return WRI_OK;
    cudaFree(c->gtab); cudaFree(c->rec); cudaFree(c->counter);
    for (int b = 0; b < 2; ++b) { cudaFree(c->coef[b]); cudaFree(c->stat[b]); cudaFree(c->active[b]); cudaFree(c->iters[b]); }
    cudaFree(c->colmap); cudaFree(c->src); cudaFree(c->retired);
    cudaFree(c->aw_tol); cudaFree(c->aw_f); cudaFree(c->aw_ar0); cudaFree(c->aw_iters);
    if (c->h_aw) cudaFreeHost(c->h_aw);
    if (c->h_prog) cudaFreeHost(c->h_prog);
    cudaFree(c->d_plans); cudaFree(c->d_maps); cudaFree(c->d_mmaps); cudaFree(c->d_own_ptr); cudaFree(c->d_own);
    cudaFree(c->d_state); cudaFree(c->d_prof);
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    for (auto& sl : c->pipe) {
        if (sl.ev_in) cudaEventDestroy(sl.ev_in);
        if (sl.ev_solve) cudaEventDestroy(sl.ev_solve);
        if (sl.ev_out) cudaEventDestroy(sl.ev_out);
    }
    if (c->s_in) cudaStreamDestroy(c->s_in);
    if (c->s_out) cudaStreamDestroy(c->s_out);
    delete c;
    return WRI_OK;
}

int wri_set_model(wri_ctx* c, const float* m_dev) {
    if (!c || !m_dev) return WRI_ERR_ARG;
    c->m = m_dev;
    return WRI_OK;
}

int wri_set_stencil(wri_ctx* c, int32_t stencil) {
    if (!c || (stencil != WRI_STENCIL_7 && stencil != WRI_STENCIL_27)) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    c->stencil = stencil;
    return WRI_OK;
}

int wri_plan_info(wri_ctx* c, int32_t nb, int32_t* out16) {
    if (!c || !out16 || nb <= 0 || nb > c->nb_max) return WRI_ERR_ARG;
    DevPlan P;
    int rc = make_plan(c, nb, P);
    if (rc) return rc;
    const int v[16] = {P.cb, P.nchunk, P.txc, P.tyc, P.items, P.merged, P.m_tma, P.f.zc, P.f.nstage, P.f.n_tiles,
                       P.a.zc, P.a.nstage, P.a.n_tiles, rt_stage_bytes(P, 3), rt_stage_bytes(P, 1), rt_grid(c)};
    for (int i = 0; i < 16; ++i) out16[i] = v[i];
    return WRI_OK;
}

int wri_set_debug_opts(wri_ctx* c, const wri_debug_opts* o) {
    if (!c) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    c->dbg = o ? *o : wri_debug_opts{};
    return WRI_OK;
}

size_t wri_workspace_bytes(const wri_ctx* c, int32_t nb, int32_t flags) {
    if (!c || nb <= 0 || nb > c->nb_max) return 0;
    return ws_layout(c, nb, flags & (WS_HOST_STAGING | WS_COMPACTION), kHostMaxitCap).total;
}

int wri_set_workspace(wri_ctx* c, void* ws_dev, size_t bytes) {
    if (!c || !ws_dev || !aligned16(ws_dev)) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    c->ws = (char*)ws_dev;
    c->ws_bytes = bytes;
    return WRI_OK;
}

int wri_set_receiver_mask(wri_ctx* c, int32_t nb, const uint8_t* mask_dev) {
    if (!c || (mask_dev && (nb <= 0 || nb > c->nb_max))) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    c->rmask = mask_dev;
    c->rmask_nb = mask_dev ? nb : 0;
    return WRI_OK;
}

int wri_lsqr_set_opts(wri_ctx* c, const wri_lsqr_opts* opts) {
    if (!c) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    c->opts = opts ? *opts : wri_lsqr_opts{};
    return WRI_OK;
}

int64_t wri_launch_count(const wri_ctx* c) { return c ? c->launches : 0; }

int wri_profile_enable(wri_ctx* c, int32_t on) {
    if (!c) return WRI_ERR_ARG;
    c->profiling = on != 0;
    return WRI_OK;
}

int wri_profile_read(wri_ctx* c, double* ms_f, int64_t* n_f, int64_t* cols_f, double* ms_a, int64_t* n_a,
                     int64_t* cols_a) {
    if (!c || !ms_f || !n_f || !cols_f || !ms_a || !n_a || !cols_a) return WRI_ERR_ARG;
    // launches that did work and their widths are counted on the device (the width of an adaptive
    // solve is not known to the host); the events bracket every launch, no-ops included
    long long h[4] = {0, 0, 0, 0};
    CK(cudaMemcpyAsync(h, c->d_prof, sizeof h, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemsetAsync(c->d_prof, 0, sizeof h, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    *ms_f = *ms_a = 0.0;
    for (size_t i = 0; i < c->ev_used; ++i) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]));
        if (c->ev_kind[i] == 0) *ms_f += ms;
        else *ms_a += ms;
    }
    *cols_f = h[0] + c->prof_host[0]; *n_f = h[1] + c->prof_host[1];
    *cols_a = h[2] + c->prof_host[2]; *n_a = h[3] + c->prof_host[3];
    c->prof_host[0] = c->prof_host[1] = c->prof_host[2] = c->prof_host[3] = 0;
    c->ev_used = 0;
    return WRI_OK;
}

int wri_apply_M(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, float lambda,
                const void* x_dev, void* ytop_dev, void* ybot_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!x_dev || !ytop_dev || (c->n_rec && !ybot_dev) || !aligned16(x_dev) || !aligned16(ytop_dev))
        return WRI_ERR_ARG;
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda, -1, true))) return rc;
    if ((rc = apply_operator(c, nb, (const float2*)x_dev, (float2*)ytop_dev, 1.f))) return rc;
    if (c->n_rec) {
        const long long n = (long long)c->n_rec * nb;
        k_gather<<<(unsigned)std::min<long long>((n + 255) / 256, 1184), 256, 0, c->stream>>>(
            (const float2*)x_dev, c->rec, c->n_rec, nb, (float2*)ybot_dev, c->rmask);
        c->launches++;
        CK(cudaGetLastError());
    }
    return WRI_OK;
}

int wri_apply_MH(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, float lambda,
                 const void* ytop_dev, const void* ybot_dev, void* x_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!x_dev || !ytop_dev || (c->n_rec && !ybot_dev) || !aligned16(x_dev) || !aligned16(ytop_dev))
        return WRI_ERR_ARG;
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda, -1, true))) return rc;
    if ((rc = apply_operator(c, nb, (const float2*)ytop_dev, (float2*)x_dev, -1.f))) return rc;
    if (c->n_rec) {
        const long long n = (long long)c->n_rec * nb;
        k_scatter_add<<<(unsigned)std::min<long long>((n + 255) / 256, 1184), 256, 0, c->stream>>>(
            (float2*)x_dev, c->rec, c->n_rec, nb, (const float2*)ybot_dev, c->rmask);
        c->launches++;
        CK(cudaGetLastError());
    }
    return WRI_OK;
}

int wri_apply_S(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                float lambda, const void* x_dev, const void* xalpha_dev, void* ytop_dev, void* ybot_dev) {
    if (!src_ijk_host || !xalpha_dev) return WRI_ERR_ARG;
    int rc = wri_apply_M(c, nb, omega_idx_host, lambda, x_dev, ytop_dev, ybot_dev);
    if (rc) return rc;
    if ((rc = upload_sources(c, nb, src_ijk_host, true))) return rc;
    k_src_forward<<<(nb + 127) / 128, 128, 0, c->stream>>>((float2*)ytop_dev, c->src, nb, lambda,
                                                          (const float2*)xalpha_dev);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

int wri_apply_SH(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                 float lambda, const void* ytop_dev, const void* ybot_dev, void* x_dev, void* xalpha_dev) {
    if (!src_ijk_host || !xalpha_dev) return WRI_ERR_ARG;
    int rc = wri_apply_MH(c, nb, omega_idx_host, lambda, ytop_dev, ybot_dev, x_dev);
    if (rc) return rc;
    if ((rc = upload_sources(c, nb, src_ijk_host, true))) return rc;
    k_src_adjoint<<<(nb + 127) / 128, 128, 0, c->stream>>>((const float2*)ytop_dev, c->src, nb, lambda,
                                                          (float2*)xalpha_dev);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

int wri_objective_gradient(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host,
                           const int32_t* src_ijk_host, const void* alpha_dev, const void* q_dev,
                           const void* u_dev, const void* d_dev, float lambda, double* f_pde_dev,
                           double* f_data_dev, float* g_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!u_dev || !aligned16(u_dev) || (q_dev && !aligned16(q_dev)) || (c->n_rec && !d_dev) || !f_pde_dev ||
        !f_data_dev || (src_ijk_host && !alpha_dev))
        return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    const GradTiling G = make_grad_tiling(c, nb);
    if (!G.ok) return WRI_ERR_ARG;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    const WsLayout L = ws_layout(c, nb, 0, kHostMaxitCap);
    if (c->ws_bytes < L.total) return WRI_ERR_WORKSPACE;
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda, -1, true))) return rc;
    if (src_ijk_host && (rc = upload_sources(c, nb, src_ijk_host, true))) return rc;
    const StencilW sw = stencil_weights(c->stencil);
    double* partials = (double*)(c->ws + L.partials);
    int n_rows = (int)G.t.n_tiles;
    // pass kernel when the batch is one power-of-two chunk per cell (64 / 32 / 16 / 8 / 4 columns): the
    // per-cell sum over the columns runs on warp shuffles; the generic kernel otherwise
    const int cb = grad_chunk_for(c, nb);
    if (cb) {
        StaticLaunch S;
        if ((rc = static_plan(c, nb, u_dev, q_dev, S, RT_G_SCRATCH, cb))) return rc;
        float* g_scr = g_dev ? (float*)(c->ws + L.gscratch) : nullptr;
        RtParams p{};
        p.sgn = 1.f; p.phase = -1;
        p.has_old = q_dev != nullptr;
        p.partials = (double*)(c->ws + L.partials_rt);
        p.gsrc = src_ijk_host ? c->src : nullptr;
        p.galpha = (const float2*)alpha_dev;
        p.g = g_scr;
        p.lam2 = lambda * lambda;
        if ((rc = launch_static<MODE_G>(c, S, p))) return rc;
        if (g_dev) {
            k_add_f32<<<blocks_for((long long)c->ng), 256, 0, c->stream>>>(g_dev, g_scr, (long long)c->ng, nb / cb);
            c->launches++;
            CK(cudaGetLastError());
        }
        partials = p.partials;
        n_rows = S.grid;
    } else {
        GradParams p{};
        p.u = (const float2*)u_dev; p.q = (const float2*)q_dev;
        p.src = src_ijk_host ? c->src : nullptr; p.alpha = (const float2*)alpha_dev;
        p.m = c->m;
        p.gx = c->gtab; p.gy = c->gtab + c->g.nx; p.gz = c->gtab + c->g.nx + c->g.ny;
        p.w2 = c->coef[0] + C_W2 * (size_t)c->nb_max;
        p.g = g_dev;
        p.partials = partials;
        p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = nb; p.zc = G.t.zc;
        p.tpc = G.tpc; p.shuffle = G.shuffle;
        p.ih2 = (float)(1.0 / (c->h * c->h));
        p.m6ih2 = (float)(sw.a0 / (c->h * c->h));
        p.a1 = (float)sw.a1; p.a2 = (float)sw.a2; p.a3 = (float)sw.a3;
        p.lam2 = lambda * lambda;
        const size_t smem = (size_t)G.t.block.x * G.t.block.y * G.t.vec * sizeof(double);
        const bool s27 = c->stencil == WRI_STENCIL_27;
        if (G.t.vec == 2) {
            if (s27) k_grad<2, ST_27><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
            else     k_grad<2, ST_7><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
        } else {
            if (s27) k_grad<1, ST_27><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
            else     k_grad<1, ST_7><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
        }
        c->launches++;
        CK(cudaGetLastError());
    }
    k_objective<<<(nb + OBJ_CPB - 1) / OBJ_CPB, 1024, 1024 * sizeof(double), c->stream>>>(
        partials, n_rows, nb, (const float2*)u_dev, (const float2*)d_dev, c->rec, c->n_rec,
        (double)lambda * (double)lambda, f_pde_dev, f_data_dev, c->rmask);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

}  // extern "C"

// ---- objective / gradient without device allocation ----------------------------------------------
// Scratch of wri_objective_gradient_static (include/wri.h): the [n_tiles][nb] column sums of |r|^2 that
// k_grad writes and k_objective folds.  Part of the library image: every GPU that loads libwri holds
// these WRI_STATIC_SCRATCH_BYTES until the process exits.  In host code the name below is only a
// stand-in for the symbol — the kernels get the address cudaGetSymbolAddress returns for the current
// device, looked up once per device.
constexpr size_t kStaticScratchDoubles = WRI_STATIC_SCRATCH_BYTES / sizeof(double);
static __device__ __align__(256) double g_static_partials[kStaticScratchDoubles];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
double* g_static_ptr[kStaticMaxDevices] = {};

// device address of g_static_partials on the current device (the one the context's buffers live on)
int static_scratch_ptr(double** out) {
    int dev = -1;
    CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kStaticMaxDevices) return WRI_ERR_ARG;
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[dev]) {
        void* ptr = nullptr;
        CK(cudaGetSymbolAddress(&ptr, g_static_partials));
        if (!ptr) return WRI_ERR_CUDA;
        g_static_ptr[dev] = static_cast<double*>(ptr);
    }
    *out = g_static_ptr[dev];
    return WRI_OK;
}

}  // namespace

extern "C" int wri_objective_gradient_static(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host,
                                             const int32_t* src_ijk_host, const void* alpha_dev,
                                             const void* q_dev, const void* u_dev, const void* d_dev,
                                             float lambda, double* f_pde_dev, double* f_data_dev,
                                             float* g_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!u_dev || !aligned16(u_dev) || (q_dev && !aligned16(q_dev)) || (c->n_rec && !d_dev) || !f_pde_dev ||
        !f_data_dev || (src_ijk_host && !alpha_dev))
        return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    GradTiling G = make_grad_tiling(c, nb);
    if (!G.ok) return WRI_ERR_ARG;
    // taller tiles until the per-tile sums fit the static array; refused when even whole columns do not
    while (G.t.n_tiles * (size_t)nb > kStaticScratchDoubles && G.t.zc < c->g.nz) {
        G.t.zc = std::min(c->g.nz, G.t.zc * 2);
        G.t.grid.z = (unsigned)((c->g.nz + G.t.zc - 1) / G.t.zc);
        G.t.n_tiles = (size_t)G.t.grid.x * G.t.grid.y * G.t.grid.z;
    }
    if (G.t.n_tiles * (size_t)nb > kStaticScratchDoubles) return WRI_ERR_SCRATCH_LIMIT;
    double* partials = nullptr;
    if ((rc = static_scratch_ptr(&partials))) return rc;
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda, -1, true))) return rc;
    if (src_ijk_host && (rc = upload_sources(c, nb, src_ijk_host, true))) return rc;
    const StencilW sw = stencil_weights(c->stencil);
    GradParams p{};
    p.u = (const float2*)u_dev; p.q = (const float2*)q_dev;
    p.src = src_ijk_host ? c->src : nullptr; p.alpha = (const float2*)alpha_dev;
    p.m = c->m;
    p.gx = c->gtab; p.gy = c->gtab + c->g.nx; p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef[0] + C_W2 * (size_t)c->nb_max;
    p.g = g_dev;
    p.partials = partials;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = nb; p.zc = G.t.zc;
    p.tpc = G.tpc; p.shuffle = G.shuffle;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(sw.a0 / (c->h * c->h));
    p.a1 = (float)sw.a1; p.a2 = (float)sw.a2; p.a3 = (float)sw.a3;
    p.lam2 = lambda * lambda;
    const size_t smem = (size_t)G.t.block.x * G.t.block.y * G.t.vec * sizeof(double);
    const bool s27 = c->stencil == WRI_STENCIL_27;
    if (G.t.vec == 2) {
        if (s27) k_grad<2, ST_27><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
        else     k_grad<2, ST_7><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
    } else {
        if (s27) k_grad<1, ST_27><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
        else     k_grad<1, ST_7><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
    }
    c->launches++;
    CK(cudaGetLastError());
    k_objective<<<(nb + OBJ_CPB - 1) / OBJ_CPB, 1024, 1024 * sizeof(double), c->stream>>>(
        partials, (int)G.t.n_tiles, nb, (const float2*)u_dev, (const float2*)d_dev, c->rec, c->n_rec,
        (double)lambda * (double)lambda, f_pde_dev, f_data_dev, c->rmask);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

// ---- solver entries ----------------------------------------------------------------------------

namespace {

// One group of a solve.  col0, ncols: the caller's columns [col0, col0 + ncols) are solved in a
// compact working set of even width nbw >= ncols carved out of the workspace (nbw = 0: all nb columns
// in the caller's own layout).  Columns are independent systems (reading C-9).
int lsqr_begin_impl(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev,
                    const void* d_dev, float lambda, const float* tol_dev, int32_t maxit,
                    void* u_out_dev, float* resnorms_dev, int32_t* iters_dev, bool host_staged,
                    const int32_t* src_ijk_host = nullptr, void* alpha_out_dev = nullptr,
                    int col0 = 0, int ncols = 0, bool batch = false) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    const bool sf = src_ijk_host != nullptr;          // source-free system: q may be absent (b_top = 0)
    if ((!q_dev && !sf) || (c->n_rec && !d_dev) || !u_out_dev || maxit < 0 ||
        (q_dev && !aligned16(q_dev)) || !aligned16(u_out_dev) || q_dev == u_out_dev || (sf && !alpha_out_dev))
        return WRI_ERR_ARG;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    const int base_flags = host_staged ? WS_HOST_STAGING : 0;
    if (c->ws_bytes < ws_layout(c, nb, base_flags, kHostMaxitCap).total) return WRI_ERR_WORKSPACE;
    const WsLayout L = ws_layout(c, nb, base_flags | WS_COMPACTION, kHostMaxitCap);
    const bool ws_big = c->ws_bytes >= L.total;               // the spare vector regions of WS_COMPACTION are there
    const int n_rgn = ws_big ? 8 : ws_layout(c, nb, base_flags, kHostMaxitCap).n_vecs;
    bool grouped = ncols > 0;
    if (!grouped) { col0 = 0; ncols = nb; }
    int nbw = grouped ? even_up(ncols) : nb;
    // the pass kernel serves even widths; an odd batch runs padded when the workspace has a spare region
    bool rt = rt_chunk_for(c, nbw) != 0;
    if (!grouped && (nb % 2) && batch && n_rgn >= 4 && rt_chunk_for(c, nb + 1)) { grouped = true; nbw = nb + 1; rt = true; }
    // adaptive accuracy: with tolerances, converged columns are compacted out of the working set on the device
    const bool adaptive = rt && batch && tol_dev && ws_big && nbw <= RT_MAXW && nbw >= 4 && !c->dbg.no_compact;
    const bool packed = grouped || adaptive;

    // vector slots: nbw-wide pieces of the nb-wide regions (the V region is skipped while the host
    // entry's staged q sits there: it must survive until the last group has started)
    std::vector<float2*> slots;
    {
        const size_t slot = align_up(c->ng * (size_t)nbw * sizeof(float2), 256);
        const size_t region = align_up(c->ng * (size_t)even_up(nb) * sizeof(float2), 256);
        for (int rgn = 0; rgn < n_rgn; ++rgn) {
            if (rgn == 1 && host_staged && q_dev && grouped) continue;
            for (size_t o = 0; o + slot <= region; o += slot) slots.push_back((float2*)(c->ws + L.vecs[rgn] + o));
        }
    }
    const size_t need = adaptive ? 8 : packed ? 4 : 3;
    if (slots.size() < need) return WRI_ERR_WORKSPACE;
    if ((rc = upload_columns(c, nbw, omega_idx_host ? omega_idx_host + col0 : nullptr, lambda, ncols))) return rc;
    if (sf && (rc = upload_sources(c, nb, src_ijk_host))) return rc;
    c->sf = sf;
    c->alpha_out = (float2*)alpha_out_dev;
    c->nb = nbw; c->nb0 = nb; c->k = 0; c->maxit = maxit; c->lambda = lambda;
    c->packed = packed; c->adaptive = adaptive; c->rt = rt;
    c->partials = (double*)(c->ws + L.partials);
    c->partials_rt = (double*)(c->ws + L.partials_rt);
    c->u_out = (float2*)u_out_dev;
    c->col0 = col0; c->ncols = ncols;
    c->retire_buf = ws_big ? (float2*)(c->ws + L.vecs[8]) : nullptr;
    if (adaptive) CK(cudaMemsetAsync(c->retired, 0, c->nb_max * sizeof(int), c->stream));
    std::memset(c->vec, 0, sizeof c->vec);
    for (int q = 0; q < 3; ++q) c->vec[0][q] = slots[q];
    c->vec[0][3] = packed ? slots[3] : (float2*)u_out_dev;
    if (adaptive) for (int q = 0; q < 4; ++q) c->vec[1][q] = slots[4 + q];
    c->U = c->vec[0][0]; c->V = c->vec[0][1]; c->W = c->vec[0][2]; c->X = c->vec[0][3];
    // receiver rows: nbw-wide pieces of the nb-wide region(s)
    c->U_bot[0] = (float2*)(c->ws + L.U_bot);
    c->U_bot[1] = ws_big ? (float2*)(c->ws + L.U_bot2) : c->U_bot[0] + (size_t)std::max(c->n_rec, 1) * nbw;
    if (adaptive && !ws_big) return WRI_ERR_WORKSPACE;
    c->tol = tol_dev; c->resnorms = resnorms_dev; c->iters_out = iters_dev;
    c->tl = make_tiling(c, nbw);

    // initial device state (pageable source: staged by the driver before the call returns)
    SolveState st;
    std::memset(&st, 0, sizeof st);
    st.nb = nbw; st.n_active = nbw;
    for (int j = 0; j < RT_MAXW; ++j) st.colmap[0][j] = st.colmap[1][j] = (j < ncols) ? col0 + j : -1;
    CK(cudaMemcpyAsync(c->d_state, &st, sizeof st, cudaMemcpyHostToDevice, c->stream));
    if (packed) {
        std::vector<int> cm(nbw);
        for (int j = 0; j < nbw; ++j) cm[j] = (j < ncols) ? col0 + j : -1;
        CK(cudaMemcpyAsync(c->colmap, cm.data(), nbw * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    }
    if (rt && (rc = rt_setup(c))) return rc;
    const size_t vbytes = c->ng * (size_t)nbw * sizeof(float2);
    const size_t NM = c->nb_max;

    // beta1 u1 = b = [lambda q ; d]   (q is consumed before V is written: the host entry stages q in
    // the V region)
    PassParams p = base_params(c, nbw, c->tl);
    p.partials = c->partials;
    p.in = (const float2*)q_dev; p.out = c->U; p.ca = c->coef[0] + C_LAM * NM;
    auto gather_in = [&](float2* dst, const void* src) -> int {      // dst[:, j] = src[:, col0 + j]
        k_gather_cols<<<blocks_for((long long)c->ng * nbw), 256, 0, c->stream>>>(
            dst, (const float2*)src, c->colmap, (long long)c->ng, nbw, nb);
        c->launches++;
        CK(cudaGetLastError());
        return WRI_OK;
    };
    if (packed && c->opts.warm_start && (rc = gather_in(c->X, u_out_dev))) return rc;
    if (q_dev) {
        if (grouped) {                    // the group's columns of q, compact, in the (still unused) W slot
            if ((rc = gather_in(c->W, q_dev))) return rc;
            p.in = c->W;
        }
        if ((rc = launch_pass<MODE_INIT>(c, p, c->tl))) return rc;
    } else {
        CK(cudaMemsetAsync(c->U, 0, vbytes, c->stream));
        CK(cudaMemsetAsync(c->partials, 0, c->tl.n_tiles * nbw * sizeof(double), c->stream));
    }
    if (c->opts.warm_start) {
        // warm start: u_out holds x0; top rows of r0 = b - S x0:  U <- U - lambda A x0  (and its ||.||^2)
        PassParams r = p;
        r.in = c->X; r.out = c->U; r.sgn = 1.f;
        r.ca = c->coef[0] + C_NLAM * NM; r.cb = c->coef[0] + C_MONE * NM;
        if ((rc = launch_pass<MODE_A>(c, r, c->tl))) return rc;
    }
    // x0 = 0, w = 0, v = 0.  On the pass kernel V is not read by the start's adjoint pass, and in a cold
    // batch solve of at least one iteration (lazy) W and X are not read by the first forward pass,
    // which writes them: no clearing needed.  (The stepping entries clear everything: their state can
    // be looked at before the first iteration.)
    c->lazy = batch && rt && !c->opts.warm_start && maxit >= 1;
    if (!c->opts.warm_start && !c->lazy) CK(cudaMemsetAsync(c->X, 0, vbytes, c->stream));
    if (!c->lazy) CK(cudaMemsetAsync(c->W, 0, vbytes, c->stream));
    if (!rt) CK(cudaMemsetAsync(c->V, 0, vbytes, c->stream));
    {
        // receiver rows of b spread over blocks, then beta1 and the first coefficients in one block
        ScalParams s = scal_params(c, c->partials, (int)c->tl.n_tiles, (const float2*)d_dev);
        k_init_rows<<<kInitRowBlocks, 256, 256 * sizeof(double), c->stream>>>(s, c->partials, (int)c->tl.n_tiles);
        c->launches++;
        CK(cudaGetLastError());
    }
    if ((rc = launch_scalars<PH_INIT_B>(c, (const float2*)d_dev, kInitRowBlocks))) return rc;
    // alpha1 v1 = M^H u1
    if (rt) {
        if ((rc = launch_rt<MODE_A>(c, PH_INIT_A))) return rc;
    } else {
        p.in = c->U; p.out = c->V; p.sgn = -1.f;
        p.ca = c->coef[0] + C_CA_A * NM; p.cb = c->coef[0] + C_CB_A * NM;
        if ((rc = launch_pass<MODE_A>(c, p, c->tl))) return rc;
        if ((rc = launch_scalars<PH_INIT_A>(c, nullptr))) return rc;
    }
    c->solving = true;
    return WRI_OK;
}

// Enqueue of a solve with tolerances from an entry that synchronises at its end: at most kAhead
// iterations ahead of the device, and no further once every column has stopped.
int iterate_paced(wri_ctx* c, int n_steps) {
    constexpr int kAhead = 16;
    volatile unsigned long long* prog = c->h_prog;
    using clock = std::chrono::steady_clock;
    unsigned long long seen = ~0ull;
    clock::time_point since = clock::now();
    for (int i = 0; i < n_steps; ++i) {
        for (;;) {
            const unsigned long long w = *prog;
            const bool mine = (unsigned int)(w >> 32) == c->solve_id;
            if (mine && (w & 1ull)) return WRI_OK;                    // every column has stopped
            const int k_dev = mine ? (int)((w & 0xffffffffull) >> 1) : 0;
            if (c->k - k_dev < kAhead) break;
            // the word has not moved for a long time: ask the stream whether anything is still in flight
            // (an error, or a device that cannot reach the word) rather than wait for ever.  Rare on
            // purpose: a stream query in a tight loop slows the kernels in flight.
            const clock::time_point now = clock::now();
            if (w != seen) { seen = w; since = now; }
            else if (now - since > std::chrono::milliseconds(200)) {
                const cudaError_t e = cudaStreamQuery(c->stream);
                if (e == cudaSuccess) break;
                if (e != cudaErrorNotReady) return cuda_fail(e, "paced enqueue");
                since = now;
            }
            std::this_thread::sleep_for(std::chrono::microseconds(20));
        }
        const int rc = wri_lsqr_iterate(c, 1);
        if (rc) return rc;
    }
    return WRI_OK;
}

// A batch is worked through in groups of at most 64 columns, each in a compact even-width working set
// of its own inside the workspace; a group that is the whole (even, <= 64 wide) batch works in the
// caller's own layout.  With several chunks per cell a tile row is a 512-byte piece of a wider cell
// record and the passes reach 0.84-0.88 of the copy bandwidth; compact groups run at the single-chunk
// rate.  The stepping entries keep all columns in lock-step.
int solve_groups(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev, const void* d_dev,
                 float lambda, const float* tol_dev, int32_t maxit, void* u_out_dev, float* resnorms_dev,
                 int32_t* iters_dev, bool host_staged, const int32_t* src_ijk_host, void* alpha_out_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    // groups need four 64-wide vector slots inside the nb-wide regions of the workspace; a batch that has
    // no room for them (e.g. 80 or 96 columns without the compaction regions) runs in lock-step
    bool split = nb > RT_MAXW && !c->dbg.no_groups && rt_chunk_for(c, RT_MAXW) != 0 && c->ws;
    if (split) {
        const int flags = host_staged ? WS_HOST_STAGING : 0;
        const bool ws_big = c->ws_bytes >= ws_layout(c, nb, flags | WS_COMPACTION, kHostMaxitCap).total;
        const size_t slot = align_up(c->ng * (size_t)RT_MAXW * sizeof(float2), 256);
        const size_t region = align_up(c->ng * (size_t)even_up(nb) * sizeof(float2), 256);
        const size_t regions = (ws_big ? 8 : 3) - ((host_staged && q_dev) ? 1 : 0);
        split = regions * (region / slot) >= 4;
    }
    const int gw = split ? RT_MAXW : nb;
    for (int col0 = 0; col0 < nb; col0 += gw) {
        const int ncols = std::min(gw, nb - col0);
        // (the generic kernels' host-sequenced solve has no device-side stop to report)
        c->pacing = c->pace && tol_dev && maxit > 0 && rt_chunk_for(c, even_up(split ? ncols : nb)) != 0;
        if (c->pacing) ++c->solve_id;
        if ((rc = lsqr_begin_impl(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev,
                                  resnorms_dev, iters_dev, host_staged, src_ijk_host, alpha_out_dev, col0,
                                  split ? ncols : 0, true))) {
            c->pacing = false;
            return rc;
        }
        if (!c->rt) c->pacing = false;
        rc = c->pacing ? iterate_paced(c, maxit) : wri_lsqr_iterate(c, maxit);
        c->pacing = false;
        if (rc) { c->solving = false; return rc; }
        if ((rc = wri_lsqr_end(c))) return rc;
    }
    return WRI_OK;
}

}  // namespace

extern "C" {

int wri_lsqr_begin(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev,
                   const void* d_dev, float lambda, const float* tol_dev, int32_t maxit,
                   void* u_out_dev, float* resnorms_dev, int32_t* iters_dev) {
    return lsqr_begin_impl(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev,
                           resnorms_dev, iters_dev, false);
}

int wri_lsqr_sf_begin(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                      const void* q_dev, const void* d_dev, float lambda, const float* tol_dev,
                      int32_t maxit, void* u_out_dev, void* alpha_out_dev, float* resnorms_dev,
                      int32_t* iters_dev) {
    if (!src_ijk_host) return WRI_ERR_ARG;
    return lsqr_begin_impl(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev,
                           resnorms_dev, iters_dev, false, src_ijk_host, alpha_out_dev);
}

int wri_lsqr_iterate(wri_ctx* c, int32_t n_steps) {
    if (!c || n_steps < 0) return WRI_ERR_ARG;
    if (!c->solving) return WRI_ERR_STATE;
    if (c->k + n_steps > c->maxit) return WRI_ERR_ARG;
    int rc;
    const size_t NM = c->nb_max;
    for (int i = 0; i < n_steps; ++i) {
        c->k++;
        if (c->rt) {
            // two launches per iteration: the last CTA of each pass runs the scalar recurrences.  The
            // launches read the solve state on the device (width, parity, iteration count) and return at
            // once when every column has stopped; nothing comes back to the host.
            if ((rc = launch_rt<MODE_F>(c, PH_F))) return rc;
            if ((rc = launch_rt<MODE_A>(c, PH_A))) return rc;
        } else {
            PassParams p = base_params(c, c->nb, c->tl);
            p.partials = c->partials;
            // pass F: U <- (lambda/alpha) A V - (alpha/beta) U ; deferred x, w updates
            p.in = c->V; p.out = c->U; p.W = c->W; p.X = c->X; p.sgn = 1.f;
            p.ca = c->coef[0] + C_CA_F * NM; p.cb = c->coef[0] + C_CB_F * NM; p.cv = c->coef[0] + C_CV_F * NM;
            p.cx = c->coef[0] + C_CX * NM; p.cw = c->coef[0] + C_CW * NM;
            if ((rc = launch_pass<MODE_F>(c, p, c->tl, true))) return rc;
            if ((rc = launch_scalars<PH_F>(c, nullptr))) return rc;
            // pass A: V <- (lambda/beta) A^H U - (beta/alpha) V
            p.in = c->U; p.out = c->V; p.W = nullptr; p.X = nullptr; p.sgn = -1.f;
            p.ca = c->coef[0] + C_CA_A * NM; p.cb = c->coef[0] + C_CB_A * NM;
            if ((rc = launch_pass<MODE_A>(c, p, c->tl, true))) return rc;
            if ((rc = launch_scalars<PH_A>(c, nullptr))) return rc;
            if (c->profiling) { c->prof_host[0] += c->nb; c->prof_host[1]++; c->prof_host[2] += c->nb; c->prof_host[3]++; }
        }
    }
    return WRI_OK;
}

int wri_lsqr_end(wri_ctx* c) {
    if (!c) return WRI_ERR_ARG;
    if (!c->solving) return WRI_ERR_STATE;
    const size_t NM = c->nb_max;
    if (!c->rt) {
        // host-sequenced solve: the state the closing kernel reads is written now
        SolveState st;
        std::memset(&st, 0, sizeof st);
        st.nb = c->nb; st.k = c->k;
        CK(cudaMemcpyAsync(c->d_state, &st, sizeof st, cudaMemcpyHostToDevice, c->stream));
    }
    // last deferred update x_k = X + cx W (scattered to the caller's columns where the working set has
    // a column map); history rows after the last iteration performed are held
    k_finish<<<c->num_sms * 8, 256, 0, c->stream>>>(move_params(c));
    c->launches++;
    CK(cudaGetLastError());
    k_clear_cx<<<(c->nb_max + 127) / 128, 128, 0, c->stream>>>(c->coef[0] + C_CX * NM, c->coef[1] + C_CX * NM, c->nb_max);
    c->launches++;
    CK(cudaGetLastError());
    c->solving = false;
    return WRI_OK;
}

int wri_lsqr_batch(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev,
                   const void* d_dev, float lambda, const float* tol_dev, int32_t maxit,
                   void* u_out_dev, float* resnorms_dev, int32_t* iters_dev) {
    return solve_groups(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev, resnorms_dev,
                        iters_dev, false, nullptr, nullptr);
}

int wri_lsqr_sf_batch(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                      const void* q_dev, const void* d_dev, float lambda, const float* tol_dev,
                      int32_t maxit, void* u_out_dev, void* alpha_out_dev, float* resnorms_dev,
                      int32_t* iters_dev) {
    if (!src_ijk_host) return WRI_ERR_ARG;
    return solve_groups(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev, resnorms_dev,
                        iters_dev, false, src_ijk_host, alpha_out_dev);
}

}  // extern "C"

namespace {

int lsqr_batch_host_impl(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                         const void* q_host, const void* d_host, float lambda, const float* tol_host,
                         int32_t maxit, void* u_out_host, void* alpha_out_host, float* resnorms_host,
                         int32_t* iters_host) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    const bool sf = src_ijk_host != nullptr;
    if ((!q_host && !sf) || (c->n_rec && !d_host) || !u_out_host || !resnorms_host || maxit < 0 ||
        maxit > kHostMaxitCap || (sf && !alpha_out_host))
        return WRI_ERR_ARG;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    const WsLayout L = ws_layout(c, nb, WS_HOST_STAGING, kHostMaxitCap);
    if (c->ws_bytes < L.total) return WRI_ERR_WORKSPACE;
    const size_t vbytes = c->ng * (size_t)nb * sizeof(float2);
    const size_t dbytes = (size_t)c->n_rec * nb * sizeof(float2);
    float2* Xs = (float2*)(c->ws + L.Xs);
    float2* Ds = (float2*)(c->ws + L.Ds);
    float* tols = (float*)(c->ws + L.tols);
    float* res = (float*)(c->ws + L.res);
    int* its = (int*)(c->ws + L.its);
    // q is staged in the V slot: the start consumes q before it clears V
    float2* Qs = q_host ? (float2*)(c->ws + L.vecs[1]) : nullptr;
    float2* As = (float2*)(c->ws + L.alphas);
    if (c->opts.warm_start) {                 // x0 (alpha0) arrive in the output buffers
        CK(cudaMemcpyAsync(Xs, u_out_host, vbytes, cudaMemcpyHostToDevice, c->stream));
        if (sf) CK(cudaMemcpyAsync(As, alpha_out_host, nb * sizeof(float2), cudaMemcpyHostToDevice, c->stream));
    }
    if (Qs) CK(cudaMemcpyAsync(Qs, q_host, vbytes, cudaMemcpyHostToDevice, c->stream));
    if (dbytes) CK(cudaMemcpyAsync(Ds, d_host, dbytes, cudaMemcpyHostToDevice, c->stream));
    if (tol_host) CK(cudaMemcpyAsync(tols, tol_host, nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    c->pace = true;                          // this entry synchronises at its end
    rc = solve_groups(c, nb, omega_idx_host, Qs, Ds, lambda, tol_host ? tols : nullptr, maxit, Xs, res, its,
                      true, src_ijk_host, sf ? As : nullptr);
    c->pace = false;
    if (rc) return rc;
    CK(cudaMemcpyAsync(u_out_host, Xs, vbytes, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemcpyAsync(resnorms_host, res, (size_t)(maxit + 1) * nb * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    if (iters_host) CK(cudaMemcpyAsync(iters_host, its, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    if (sf) CK(cudaMemcpyAsync(alpha_out_host, As, nb * sizeof(float2), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return WRI_OK;
}

}  // namespace

extern "C" {

int wri_lsqr_batch_host(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_host,
                        const void* d_host, float lambda, const float* tol_host, int32_t maxit,
                        void* u_out_host, float* resnorms_host, int32_t* iters_host) {
    if (!q_host) return WRI_ERR_ARG;
    return lsqr_batch_host_impl(c, nb, omega_idx_host, nullptr, q_host, d_host, lambda, tol_host, maxit,
                                u_out_host, nullptr, resnorms_host, iters_host);
}

int wri_lsqr_sf_batch_host(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                           const void* q_host, const void* d_host, float lambda, const float* tol_host,
                           int32_t maxit, void* u_out_host, void* alpha_out_host, float* resnorms_host,
                           int32_t* iters_host) {
    if (!src_ijk_host) return WRI_ERR_ARG;
    return lsqr_batch_host_impl(c, nb, omega_idx_host, src_ijk_host, q_host, d_host, lambda, tol_host, maxit,
                                u_out_host, alpha_out_host, resnorms_host, iters_host);
}

int wri_lsqr_peek(const wri_ctx* c, wri_lsqr_view* v) {
    if (!c || !v) return WRI_ERR_ARG;
    if (!c->U) return WRI_ERR_STATE;
    const size_t NM = c->nb_max;
    // the working width, the iteration count and the vector set in use live on the device
    SolveState st;
    std::memset(&st, 0, sizeof st);
    st.nb = c->nb; st.k = c->k;
    if (c->rt) {
        CK(cudaStreamSynchronize(c->stream));
        CK(cudaMemcpy(&st, c->d_state, sizeof st, cudaMemcpyDeviceToHost));
    }
    const int par = st.parity & 1;
    v->nb = st.nb; v->k = st.k;
    v->U_top = c->vec[par][0]; v->U_bot = c->U_bot[par]; v->V = c->vec[par][1]; v->W = c->vec[par][2];
    v->X = c->vec[par][3];
    const double* stat = c->stat[par];
    const float* coef = c->coef[par];
    v->alpha = stat + S_ALPHA * NM; v->beta = stat + S_BETA * NM;
    v->rhobar = stat + S_RHOBAR * NM; v->phibar = stat + S_PHIBAR * NM;
    v->ar0 = stat + S_AR0 * NM;
    v->cx = coef + C_CX * NM;
    v->cw = coef + C_CW * NM;
    v->active = c->active[par]; v->iters = c->iters[par];
    v->nb_max = c->nb_max;
    v->sf_state = c->sf ? stat + S_VA_RE * NM : nullptr;
    return WRI_OK;
}

}  // extern "C"

// ---- pipelined host-buffer solves ------------------------------------------------------------------
namespace {

struct PipeLayout { size_t Q, D, X, alpha, tol, res, its, slot; };
PipeLayout pipe_layout(const wri_ctx* c, int nb) {
    PipeLayout L{};
    const size_t vec = align_up(c->ng * (size_t)nb * sizeof(float2), 256);
    const size_t bot = align_up((size_t)std::max(c->n_rec, 1) * nb * sizeof(float2), 256);
    size_t o = 0;
    L.Q = o; o += vec;
    L.X = o; o += vec;
    L.D = o; o += bot;
    L.alpha = o; o += align_up((size_t)nb * sizeof(float2), 256);
    L.tol = o; o += align_up((size_t)nb * sizeof(float), 256);
    L.res = o; o += align_up((size_t)(kHostMaxitCap + 1) * nb * sizeof(float), 256);
    L.its = o; o += align_up((size_t)nb * sizeof(int), 256);
    L.slot = o;
    return L;
}

int host_async_impl(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                    const void* q_host, const void* d_host, float lambda, const float* tol_host, int32_t maxit,
                    void* u_out_host, void* alpha_out_host, float* resnorms_host, int32_t* iters_host) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    const bool sf = src_ijk_host != nullptr;
    if ((!q_host && !sf) || (c->n_rec && !d_host) || !u_out_host || !resnorms_host || maxit < 0 ||
        maxit > kHostMaxitCap || (sf && !alpha_out_host))
        return WRI_ERR_ARG;
    if (!c->pipe_nb || nb > c->pipe_nb) return WRI_ERR_WORKSPACE;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    wri_ctx::PipeSlot& S = c->pipe[c->pipe_next];
    c->pipe_next ^= 1;
    const size_t vbytes = c->ng * (size_t)nb * sizeof(float2);
    const size_t dbytes = (size_t)c->n_rec * nb * sizeof(float2);
    // inputs: the slot's previous solve has consumed them and its results have left
    CK(cudaStreamWaitEvent(c->s_in, S.ev_solve, 0));
    CK(cudaStreamWaitEvent(c->s_in, S.ev_out, 0));
    if (c->opts.warm_start) {
        CK(cudaMemcpyAsync(S.X, u_out_host, vbytes, cudaMemcpyHostToDevice, c->s_in));
        if (sf) CK(cudaMemcpyAsync(S.alpha, alpha_out_host, nb * sizeof(float2), cudaMemcpyHostToDevice, c->s_in));
    }
    if (q_host) CK(cudaMemcpyAsync(S.Q, q_host, vbytes, cudaMemcpyHostToDevice, c->s_in));
    if (dbytes) CK(cudaMemcpyAsync(S.D, d_host, dbytes, cudaMemcpyHostToDevice, c->s_in));
    if (tol_host) CK(cudaMemcpyAsync(S.tol, tol_host, nb * sizeof(float), cudaMemcpyHostToDevice, c->s_in));
    CK(cudaEventRecord(S.ev_in, c->s_in));
    // the solve, on the context's stream
    CK(cudaStreamWaitEvent(c->stream, S.ev_in, 0));
    CK(cudaStreamWaitEvent(c->stream, S.ev_out, 0));
    if ((rc = solve_groups(c, nb, omega_idx_host, q_host ? S.Q : nullptr, S.D, lambda, tol_host ? S.tol : nullptr,
                           maxit, S.X, S.res, S.its, false, src_ijk_host, sf ? S.alpha : nullptr)))
        return rc;
    CK(cudaEventRecord(S.ev_solve, c->stream));
    // results
    CK(cudaStreamWaitEvent(c->s_out, S.ev_solve, 0));
    CK(cudaMemcpyAsync(u_out_host, S.X, vbytes, cudaMemcpyDeviceToHost, c->s_out));
    CK(cudaMemcpyAsync(resnorms_host, S.res, (size_t)(maxit + 1) * nb * sizeof(float), cudaMemcpyDeviceToHost, c->s_out));
    if (iters_host) CK(cudaMemcpyAsync(iters_host, S.its, nb * sizeof(int), cudaMemcpyDeviceToHost, c->s_out));
    if (sf) CK(cudaMemcpyAsync(alpha_out_host, S.alpha, nb * sizeof(float2), cudaMemcpyDeviceToHost, c->s_out));
    CK(cudaEventRecord(S.ev_out, c->s_out));
    return WRI_OK;
}

}  // namespace

extern "C" {

size_t wri_host_pipeline_bytes(const wri_ctx* c, int32_t nb) {
    if (!c || nb <= 0 || nb > c->nb_max) return 0;
    return 2 * pipe_layout(c, nb).slot;
}

int wri_set_host_pipeline(wri_ctx* c, int32_t nb, void* buf_dev, size_t bytes) {
    if (!c) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    if (c->s_out) { CK(cudaStreamSynchronize(c->s_out)); CK(cudaStreamSynchronize(c->s_in)); }
    if (!buf_dev) { c->pipe_nb = 0; return WRI_OK; }
    if (nb <= 0 || nb > c->nb_max || !aligned16(buf_dev)) return WRI_ERR_ARG;
    const PipeLayout L = pipe_layout(c, nb);
    if (bytes < 2 * L.slot) return WRI_ERR_WORKSPACE;
    if (!c->s_in) {
        CK(cudaStreamCreateWithFlags(&c->s_in, cudaStreamNonBlocking));
        CK(cudaStreamCreateWithFlags(&c->s_out, cudaStreamNonBlocking));
        for (auto& sl : c->pipe) {
            CK(cudaEventCreateWithFlags(&sl.ev_in, cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&sl.ev_solve, cudaEventDisableTiming));
            CK(cudaEventCreateWithFlags(&sl.ev_out, cudaEventDisableTiming));
        }
    }
    for (int i = 0; i < 2; ++i) {
        char* b = (char*)buf_dev + (size_t)i * L.slot;
        wri_ctx::PipeSlot& S = c->pipe[i];
        S.Q = (float2*)(b + L.Q); S.X = (float2*)(b + L.X); S.D = (float2*)(b + L.D);
        S.alpha = (float2*)(b + L.alpha); S.tol = (float*)(b + L.tol); S.res = (float*)(b + L.res);
        S.its = (int*)(b + L.its);
    }
    c->pipe_nb = nb;
    c->pipe_next = 0;
    return WRI_OK;
}

int wri_lsqr_batch_host_async(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_host,
                              const void* d_host, float lambda, const float* tol_host, int32_t maxit,
                              void* u_out_host, float* resnorms_host, int32_t* iters_host) {
    if (!q_host) return WRI_ERR_ARG;
    return host_async_impl(c, nb, omega_idx_host, nullptr, q_host, d_host, lambda, tol_host, maxit, u_out_host,
                           nullptr, resnorms_host, iters_host);
}

int wri_lsqr_sf_batch_host_async(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host,
                                 const int32_t* src_ijk_host, const void* q_host, const void* d_host,
                                 float lambda, const float* tol_host, int32_t maxit, void* u_out_host,
                                 void* alpha_out_host, float* resnorms_host, int32_t* iters_host) {
    if (!src_ijk_host) return WRI_ERR_ARG;
    return host_async_impl(c, nb, omega_idx_host, src_ijk_host, q_host, d_host, lambda, tol_host, maxit,
                           u_out_host, alpha_out_host, resnorms_host, iters_host);
}

int wri_host_wait(wri_ctx* c) {
    if (!c) return WRI_ERR_ARG;
    if (c->s_in) CK(cudaStreamSynchronize(c->s_in));
    CK(cudaStreamSynchronize(c->stream));
    if (c->s_out) CK(cudaStreamSynchronize(c->s_out));
    return WRI_OK;
}

}  // extern "C"

// ---- misfit evaluation and one outer iteration of Algorithm 2 -------------------------------------
namespace {

// Lines 4-5 (or 7-8) of Algorithm 2 for one group of columns: source-free solve to tolerance eps,
// then eq. 8-9 at the solution.  f_host (optional) receives sum_s (f_pde + f_data), iters_host the
// column iterations spent; either one makes the call synchronise the stream.
int misfit_impl(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                const void* d_dev, float lambda, float eps, int32_t maxit, int32_t warm, void* u_dev,
                void* alpha_dev, double* ar0_dev, double* f_pde_dev, double* f_data_dev, float* g_dev,
                int32_t* iters_dev, double* f_host, int64_t* iters_host) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!src_ijk_host || !u_dev || !alpha_dev || !f_pde_dev || !f_data_dev || !(eps >= 0.f) || maxit < 0 ||
        (warm && !ar0_dev))
        return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    std::vector<float> tol(nb, eps);
    CK(cudaMemcpyAsync(c->aw_tol, tol.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    int32_t* its = iters_dev ? iters_dev : c->aw_iters;
    const wri_lsqr_opts saved = c->opts;
    c->opts = wri_lsqr_opts{};
    if (warm) { c->opts.warm_start = 1; c->opts.ar_ref_dev = ar0_dev; }
    else c->opts.ar0_out_dev = ar0_dev;
    c->pace = f_host || iters_host;         // the call synchronises at its end: enqueue a little ahead only
    rc = wri_lsqr_sf_batch(c, nb, omega_idx_host, src_ijk_host, nullptr, d_dev, lambda,
                           eps > 0.f ? c->aw_tol : nullptr, maxit, u_dev, alpha_dev, nullptr, its);
    c->pace = false;
    c->opts = saved;
    if (rc) return rc;
    if ((rc = wri_objective_gradient(c, nb, omega_idx_host, src_ijk_host, alpha_dev, nullptr, u_dev, d_dev,
                                     lambda, f_pde_dev, f_data_dev, g_dev)))
        return rc;
    if (f_host || iters_host) {
        double* hf = c->h_aw;
        int* hi = reinterpret_cast<int*>(c->h_aw + 2 * (size_t)c->nb_max);
        CK(cudaMemcpyAsync(hf, f_pde_dev, nb * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaMemcpyAsync(hf + c->nb_max, f_data_dev, nb * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaMemcpyAsync(hi, its, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
        CK(cudaStreamSynchronize(c->stream));
        double f = 0.0;
        int64_t n = 0;
        for (int s = 0; s < nb; ++s) { f += hf[s] + hf[c->nb_max + s]; n += hi[s]; }   // fixed order
        if (f_host) *f_host = f;
        if (iters_host) *iters_host = n;
    }
    return WRI_OK;
}

}  // namespace

extern "C" {

int wri_misfit_sf(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                  const void* d_dev, float lambda, float eps, int32_t maxit, int32_t warm, void* u_dev,
                  void* alpha_dev, double* ar0_dev, double* f_pde_dev, double* f_data_dev, float* g_dev,
                  int32_t* iters_dev, double* f_host) {
    return misfit_impl(c, nb, omega_idx_host, src_ijk_host, d_dev, lambda, eps, maxit, warm, u_dev, alpha_dev,
                       ar0_dev, f_pde_dev, f_data_dev, g_dev, iters_dev, f_host, nullptr);
}

int wri_awri_step(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                  const void* d_dev, float lambda, float eps, int32_t maxit, const wri_awri_opts* o,
                  float* m_dev, float* m_trial_dev, float* g_dev, void* u_dev, void* alpha_dev,
                  void* u_trial_dev, void* alpha_trial_dev, double* f_cols_dev, wri_awri_report* rep) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!o || !m_dev || !m_trial_dev || !g_dev || !u_dev || !alpha_dev || !u_trial_dev || !alpha_trial_dev ||
        !f_cols_dev || !rep || !(eps > 0.f) || o->max_halvings < 0 || o->max_halvings >= WRI_AWRI_MAX_TRACE ||
        m_dev == m_trial_dev || u_dev == u_trial_dev)
        return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    const float* m_saved = c->m;
    auto leave = [&](int code) { c->m = m_saved; return code; };
    memset(rep, 0, sizeof *rep);
    double* f_pde = f_cols_dev;
    double* f_data = f_cols_dev + nb;
    for (int h = 0;; ++h) {
        // line 4-5: x-bar, f, g at the current model (after a "go back": optionally continued from x-bar)
        double f = 0.0, f_trial = 0.0;
        int64_t it0 = 0, it1 = 0;
        c->m = m_dev;
        CK(cudaMemsetAsync(g_dev, 0, c->ng * sizeof(float), c->stream));
        const int warm = (o->warm_restart && h > 0) ? 1 : 0;
        if ((rc = misfit_impl(c, nb, omega_idx_host, src_ijk_host, d_dev, lambda, eps, maxit, warm, u_dev,
                              alpha_dev, c->aw_ar0, f_pde, f_data, g_dev, nullptr, &f, &it0)))
            return leave(rc);
        // eq. 8-9 are sums over every rank's columns: the caller's collective adds the objective and the
        // gradient, so that all ranks hold the same f, g and take the same decision below
        if (o->reduce && o->reduce(o->user, &f, g_dev, (int64_t)c->ng, (void*)c->stream) != 0) return leave(WRI_ERR_ARG);
        // line 6: the trial model
        if (o->update) {
            if (o->update(o->user, m_dev, g_dev, m_trial_dev, (void*)c->stream) != 0) return leave(WRI_ERR_ARG);
        } else {
            k_model_step<<<blocks_for((long long)c->ng), 256, 0, c->stream>>>(
                m_trial_dev, m_dev, g_dev, o->step, o->m_min, o->m_max, (long long)c->ng);
            c->launches++;
            CK(cudaGetLastError());
        }
        // line 7-8: x-tilde and f-tilde at the trial model (cold solve, objective only)
        c->m = m_trial_dev;
        if ((rc = misfit_impl(c, nb, omega_idx_host, src_ijk_host, d_dev, lambda, eps, maxit, 0, u_trial_dev,
                              alpha_trial_dev, nullptr, c->aw_f, c->aw_f + c->nb_max, nullptr, nullptr,
                              &f_trial, &it1)))
            return leave(rc);
        c->m = m_dev;
        if (o->reduce && o->reduce(o->user, &f_trial, nullptr, 0, (void*)c->stream) != 0) return leave(WRI_ERR_ARG);
        rep->trace_eps[h] = eps; rep->trace_f[h] = f; rep->trace_f_trial[h] = f_trial;
        rep->n_trace = h + 1;
        rep->f = f; rep->f_trial = f_trial; rep->eps = eps; rep->n_halvings = h;
        rep->lsqr_iters += it0 + it1;
        // the objective at the current model must be a number; a trial objective that is not
        // (an update that produced a non-physical model) counts as a rejected step
        if (!std::isfinite(f)) return leave(WRI_ERR_NUMERIC);
        if (std::isfinite(f_trial) && f_trial <= f) {       // line 9 / 12-13
            CK(cudaMemcpyAsync(m_dev, m_trial_dev, c->ng * sizeof(float), cudaMemcpyDeviceToDevice, c->stream));
            rep->accepted = 1;
            break;
        }
        if (h == o->max_halvings) break;                    // reading C-20: give up, model unchanged
        eps *= 0.5f;                                        // line 10-11
    }
    return leave(WRI_OK);
}

}  // extern "C"
