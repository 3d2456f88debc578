// wri_api.cu — C ABI of libwri (include/wri.h): context, validation, launch sequencing.
// All arithmetic of the path runs in the kernels of wri_kernels.cuh; there is no CPU fallback.
#include "../../include/wri.h"
#include "wri_kernels.cuh"
#include "wri_tma.cuh"

#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
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

inline unsigned blocks_for(long long n) { return (unsigned)std::min<long long>((n + 255) / 256, 148 * 16); }
constexpr int kMaxCtas = 512;          // upper bound on the persistent grid (>= SM count)
constexpr int kMinChunk = 2;           // narrowest column chunk of the TMA path

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
    // library-owned device memory
    float* gtab = nullptr;       // gx | gy | gz
    int* rec = nullptr;          // [n_rec] cell indices
    std::vector<int> rec_ijk;    // host copy [n_rec][3]
    int* own_ptr = nullptr;      // [kMaxCtas + 1] pass A: CSR of the receivers inside each CTA's tiles
    int4* own = nullptr;         // [n_rec * max chunks] {receiver, cell, tile, group size}
    std::vector<int> h_own_ptr;
    std::vector<int4> h_own;
    float* coef = nullptr;       // [N_COEF][nb_max]   current bank of the per-column scalars
    double* stat = nullptr;      // [N_STAT][nb_max]
    int* active = nullptr;       // [nb_max]
    int* iters = nullptr;        // [nb_max]
    float* coef_alt = nullptr;   // second bank: column compaction gathers into it and swaps
    double* stat_alt = nullptr;
    int* active_alt = nullptr;
    int* iters_alt = nullptr;
    int* src = nullptr;          // [nb_max] source cell per caller's column (source-free system)
    bool sf = false;             // the solve in flight has the extra source-weight unknown
    float2* alpha_out = nullptr; // caller's [nb] source-weight estimates (source-free system)
    wri_lsqr_opts opts{};        // warm start / stop-rule reference for the next solves (wri_lsqr_set_opts)
    const unsigned char* rmask = nullptr;   // per-source receiver sets [n_rec][rmask_nb] (wri_set_receiver_mask)
    int rmask_nb = 0;
    int* colmap = nullptr;       // [nb_max] working column -> caller's column (-1 = padding)
    int* idx = nullptr;          // [3][nb_max] scratch: gather map | retire source | retire destination
    int* h_active = nullptr;     // pinned host copy of the active flags
    // misfit evaluation / Algorithm 2 step (wri_misfit_sf, wri_awri_step)
    float* aw_tol = nullptr;     // [nb_max] the uniform tolerance eps of a misfit evaluation
    double* aw_f = nullptr;      // [2][nb_max] f_pde | f_data of the trial evaluation
    double* aw_ar0 = nullptr;    // [nb_max] alpha1*beta1 of the cold solve at the current model
    int* aw_iters = nullptr;     // [nb_max]
    double* h_aw = nullptr;      // pinned: [2][nb_max] doubles followed by [nb_max] ints
    // caller's workspace
    char* ws = nullptr;
    size_t ws_bytes = 0;
    // solve in flight
    bool solving = false;
    int nb = 0, k = 0, maxit = 0;   // nb = WORKING width (shrinks when converged columns are compacted away)
    int nb0 = 0;                    // caller's batch width
    bool packed = false;            // X lives in the workspace (after the first compaction); else X = u_out
    bool can_compact = false, all_done = false;
    int check_every = 0;            // iterations between host looks at the active flags (0 = never)
    std::vector<int> h_colmap;      // host copy of colmap
    std::vector<char> retired;      // per caller's column: x and history are final in the caller's buffers
    std::vector<float2*> free_slots;   // workspace vector slots not holding a live vector
    float2 *U_bot_alt = nullptr, *u_out = nullptr;
    float lambda = 0;
    float2 *U = nullptr, *V = nullptr, *W = nullptr, *X = nullptr, *U_bot = nullptr;
    double* partials = nullptr;
    const float* tol = nullptr;
    float* resnorms = nullptr;
    int* iters_out = nullptr;
    Tiling tl{};
    int64_t launches = 0;
    // persistent TMA pass kernel (nb % 16 == 0): column chunk width, tiling, tensor maps
    int num_sms = 0;
    unsigned int* counter = nullptr;      // last-CTA ticket (device)
    int tma_cb = 0;                       // 0 = not used for this solve
    struct TmaPlan {                      // one per pass (tile shapes may differ between F and A)
        int txc = 0, tyc = 0, ntx = 0, nty = 0, ntz = 0, zc = 0, nchunk = 0, tiles = 0, grid = 0;
        CUtensorMap in{}, old{}, w{}, x{}, m{};
        int m_tma = 0;                    // model tile rides in the TMA stage
        int merged = 0;                   // tensor maps fold (column, x)
    } planF, planA, planG;
    double* partials_tma = nullptr;       // [grid][nb]
    bool wx_zero = false;                 // W, X not cleared: the first pass F must not read them
    // optional per-kernel timing (wri_profile_*)
    bool profiling = false;
    std::vector<cudaEvent_t> ev_pool;     // pairs: start, stop
    std::vector<int> ev_kind;             // per pair: 0 = pass F, 1 = pass A
    std::vector<int> ev_cols;             // per pair: working batch width of that launch
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

// Tile shape for batch width nb: threads span the (ix, s) row first, then y; blocks march zc planes.
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

struct WsLayout {
    size_t U, V, W, U_bot, partials, partials_tma, gscratch, Xs, Ds, tols, res, its, alphas, B3, B4, U_bot2, total;
};
enum { WS_HOST_STAGING = 1, WS_COMPACTION = 2 };
WsLayout ws_layout(const wri_ctx* c, int nb, int flags, int maxit_cap) {
    WsLayout L{};
    const size_t vec = align_up(c->ng * (size_t)nb * sizeof(float2), 256);
    const size_t bot = align_up((size_t)std::max(c->n_rec, 1) * nb * sizeof(float2), 256);
    const Tiling t = make_tiling(c, nb);
    size_t o = 0;
    L.U = o; o += vec;
    L.V = o; o += vec;
    L.W = o; o += vec;
    L.U_bot = o; o += bot;
    const GradTiling gt = make_grad_tiling(c, nb);
    L.partials = o; o += align_up(std::max(t.n_tiles, gt.ok ? gt.t.n_tiles : 0) * nb * sizeof(double), 256);
    L.partials_tma = o; o += align_up((size_t)kMaxCtas * nb * sizeof(double), 256);
    L.gscratch = o; o += align_up(c->ng * sizeof(float), 256);       // one batch's gradient (TMA path)
    if (flags & WS_HOST_STAGING) {
        L.Xs = o; o += vec;
        L.Ds = o; o += bot;
        L.tols = o; o += align_up((size_t)nb * sizeof(float), 256);
        L.res = o; o += align_up((size_t)(maxit_cap + 1) * nb * sizeof(float), 256);
        L.its = o; o += align_up((size_t)nb * sizeof(int), 256);
        L.alphas = o; o += align_up((size_t)nb * sizeof(float2), 256);
    }
    if (flags & WS_COMPACTION) {
        L.B3 = o; o += vec;
        L.B4 = o; o += vec;
        L.U_bot2 = o; o += bot;
    }
    L.total = o;
    return L;
}
constexpr int kHostMaxitCap = 4096;   // resnorm staging rows reserved for wri_lsqr_batch_host

int upload_columns(wri_ctx* c, int nb, const int32_t* omega_idx, float lambda) {
    std::vector<float> w2(nb), one(nb, 1.f), lam(nb, lambda), nlam(nb, -lambda), mone(nb, -1.f);
    for (int s = 0; s < nb; ++s) {
        const int j = omega_idx ? omega_idx[s] : 0;
        if (j < 0 || j >= (int)c->omega.size()) return WRI_ERR_ARG;
        w2[s] = (float)(c->omega[j] * c->omega[j]);
    }
    const size_t NM = c->nb_max;
    CK(cudaMemcpyAsync(c->coef + C_W2 * NM, w2.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->coef + C_ONE * NM, one.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->coef + C_LAM * NM, lam.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->coef + C_NLAM * NM, nlam.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->coef + C_MONE * NM, mone.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    return WRI_OK;
}

// source nodes of the source-free system, one per batch column -> c->src (cell indices)
int upload_sources(wri_ctx* c, int nb, const int32_t* src_ijk) {
    std::vector<int> cells(nb);
    for (int s = 0; s < nb; ++s) {
        const int ix = src_ijk[3 * s], iy = src_ijk[3 * s + 1], iz = src_ijk[3 * s + 2];
        if (ix < 0 || ix >= c->g.nx || iy < 0 || iy >= c->g.ny || iz < 0 || iz >= c->g.nz) return WRI_ERR_ARG;
        cells[s] = (iz * c->g.ny + iy) * c->g.nx + ix;
    }
    // pageable source: the call returns once the data sits in the driver's staging buffer
    CK(cudaMemcpyAsync(c->src, cells.data(), nb * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    return WRI_OK;
}

PassParams base_params(const wri_ctx* c, int nb, const Tiling& t) {
    PassParams p{};
    p.m = c->m;
    p.gx = c->gtab;
    p.gy = c->gtab + c->g.nx;
    p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef + C_W2 * (size_t)c->nb_max;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = nb;
    p.zc = t.zc;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(-6.0 / (c->h * c->h));
    p.sgn = 1.f;
    return p;
}

template <int MODE>
int launch_pass(wri_ctx* c, const PassParams& p, const Tiling& t, bool timed = false) {
    const size_t smem = (MODE == MODE_APPLY) ? 0 : (size_t)t.block.x * t.block.y * t.vec * sizeof(double);
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    if (timed && c->profiling) {
        if (c->ev_used * 2 == c->ev_pool.size()) {
            cudaEvent_t a, b;
            CK(cudaEventCreate(&a));
            CK(cudaEventCreate(&b));
            c->ev_pool.push_back(a); c->ev_pool.push_back(b); c->ev_kind.push_back(0); c->ev_cols.push_back(0);
        }
        e0 = c->ev_pool[2 * c->ev_used]; e1 = c->ev_pool[2 * c->ev_used + 1];
        c->ev_kind[c->ev_used] = (MODE == MODE_F) ? 0 : 1;
        c->ev_cols[c->ev_used] = c->nb;
        c->ev_used++;
        CK(cudaEventRecord(e0, c->stream));
    }
    if (t.vec == 2) k_pass<2, MODE><<<t.grid, t.block, smem, c->stream>>>(p);
    else            k_pass<1, MODE><<<t.grid, t.block, smem, c->stream>>>(p);
    c->launches++;
    CK(cudaGetLastError());
    if (e1) CK(cudaEventRecord(e1, c->stream));
    return WRI_OK;
}

ScalParams scal_params(const wri_ctx* c, const double* partials, int n_rows, const float2* d);

template <int PHASE>
int launch_scalars(wri_ctx* c, const float2* d) {
    ScalParams s = scal_params(c, c->partials, (int)c->tl.n_tiles, d);
    s.rows_in_pass = c->tma_cb ? 1 : 0;
    const int T = 1024;
    const size_t smem = (size_t)(T + c->nb) * sizeof(double);
    k_scalars<PHASE><<<1, T, smem, c->stream>>>(s);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}


// ---- TMA path -------------------------------------------------------------------------------
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
// row is cb*bx elements (<= 256) — narrow chunks would otherwise move 32-128 byte rows
int make_tmap(CUtensorMap* tm, const void* base, const wri_ctx* c, int nb, int cb, int bx, int by,
              bool merged = false) {
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
    // 128-byte L2 promotion: measured 0.7 % faster than 256 B at 128^3 x 64 (whole step 0.924 against 0.918)
    CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_128B;
    if (const char* e = getenv("WRI_L2PROMO")) promo = (CUtensorMapL2promotion)atoi(e);
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_UINT64, 4, const_cast<void*>(base), gdim, gstr, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                    promo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_msg, sizeof g_cuda_msg, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
        return WRI_ERR_CUDA;
    }
    return WRI_OK;
}

// Tile shapes per column-chunk width and pass.  A tile row is TXC cells = TXC*CB*8 contiguous
// bytes; TXC*TYC*CB = 1024 complex (F: 512 consumer threads, 1 item each; A: 256 x 2 items).
#ifndef WRI_F_TX
#define WRI_F_TX 4
#endif
#ifndef WRI_F_TY
#define WRI_F_TY 4
#endif
#ifndef WRI_A_TX
#define WRI_A_TX 4
#endif
#ifndef WRI_A_TY
#define WRI_A_TY 4
#endif
#ifndef WRI_F_NT
#define WRI_F_NT 512
#endif
#ifndef WRI_A_NT
#define WRI_A_NT 512
#endif
template <int CB, int MODE> struct CfgFor {
    static constexpr int S = 64 / CB;   // narrower chunks -> proportionally more cells per tile row
    typedef TileCfg<CB, (MODE == MODE_F ? WRI_F_TX : WRI_A_TX) * (S >= 2 ? 2 : 1),
                    (MODE == MODE_F ? WRI_F_TY : WRI_A_TY) * (S >= 4 ? 2 : 1),
                    (MODE == MODE_F ? WRI_F_NT : WRI_A_NT), PassTraits<MODE>::NSTAGE> type;
};

// 48 columns: 4 x 4 cells x 48 columns = 768 complex per plane, 384 consumer threads (one item each)
#ifndef WRI_F48_NT
#define WRI_F48_NT 384
#endif
#ifndef WRI_A48_NT
#define WRI_A48_NT 384
#endif
#ifndef WRI_A48_STAGES
#define WRI_A48_STAGES 8
#endif
template <int MODE> struct CfgFor<48, MODE> {
    typedef TileCfg<48, 4, 4, (MODE == MODE_F ? WRI_F48_NT : WRI_A48_NT),
                    (MODE == MODE_F ? PassTraits<MODE_F>::NSTAGE : WRI_A48_STAGES)> type;
};

// 8 / 4 columns (the tail of a shrinking batch): 16 x 8 / 16 x 16 cells, always one chunk per cell
template <int MODE> struct CfgFor<8, MODE> {
    typedef TileCfg<8, 16, 8, (MODE == MODE_F ? WRI_F_NT : WRI_A_NT), PassTraits<MODE>::NSTAGE> type;
};
template <int MODE> struct CfgFor<4, MODE> {
    typedef TileCfg<4, 16, 16, (MODE == MODE_F ? WRI_F_NT : WRI_A_NT), PassTraits<MODE>::NSTAGE> type;
};
// 56 / 40 / 24 columns (widths a shrinking batch passes through): one item per consumer thread
template <int MODE> struct CfgFor<56, MODE> {
    typedef TileCfg<56, 4, 4, 448, (MODE == MODE_F ? PassTraits<MODE_F>::NSTAGE : WRI_A48_STAGES)> type;
};
template <int MODE> struct CfgFor<40, MODE> {
    typedef TileCfg<40, 4, 4, 320, (MODE == MODE_F ? PassTraits<MODE_F>::NSTAGE : WRI_A48_STAGES)> type;
};
template <int MODE> struct CfgFor<24, MODE> {
    typedef TileCfg<24, 8, 4, 384, (MODE == MODE_F ? PassTraits<MODE_F>::NSTAGE : WRI_A48_STAGES)> type;
};
// 2 columns (one 16-byte item per cell): 32 x 16 cells
template <int MODE> struct CfgFor<2, MODE> {
    typedef TileCfg<2, 32, 16, (MODE == MODE_F ? WRI_F_NT : WRI_A_NT), PassTraits<MODE>::NSTAGE> type;
};

int tma_chunk_for(int nb) {
    const char* off = getenv("WRI_NO_TMA");
    if (off && off[0] == '1') return 0;
    if (nb % 64 == 0) return 64;
    if (nb == 56 || nb == 40 || nb == 24) return nb;
    if (nb % 48 == 0) return 48;
    if (nb % 32 == 0) return 32;
    if (nb % 16 == 0) return 16;
    if (nb == 8 || nb == 4 || nb == 2) return nb;
    return 0;
}

// opt-in to > 48 KB of dynamic shared memory, once per (context, kernel, size): the attribute is per
// device, so it is not cached in a process-wide static
int allow_smem(wri_ctx* c, const void* fn, size_t bytes) {
    for (auto& e : c->smem_ok)
        if (e.first == fn) {
            if (e.second >= bytes) return WRI_OK;
            CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
            e.second = bytes;
            return WRI_OK;
        }
    CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes));
    c->smem_ok.emplace_back(fn, bytes);
    return WRI_OK;
}

template <class Cfg, int MODE>
size_t tma_smem_bytes(const wri_ctx* c) {
    return (size_t)Cfg::NSTAGE *
               (Cfg::IN_SPAN + PassTraits<MODE>::NSTREAM * Cfg::CTR_BYTES + Cfg::M_BYTES) +
           2 * Cfg::NSTAGE * 8 + (size_t)c->nb * 8 + (size_t)Cfg::NT * 2 * 8 +
           (size_t)(c->g.nx + c->g.ny + c->g.nz) * 4 + (size_t)6 * c->nb * 4;
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

// tiling + tensor maps of one pass for the solve that is starting
template <class Cfg>
int tma_plan(wri_ctx* c, wri_ctx::TmaPlan& P, const void* in, const void* old, bool is_f,
             bool rec_lists = true) {
    P.txc = Cfg::TXC; P.tyc = Cfg::TYC;
    P.nchunk = c->nb / Cfg::CB;
    P.ntx = (c->g.nx + P.txc - 1) / P.txc;
    P.nty = (c->g.ny + P.tyc - 1) / P.tyc;
    const long long per_plane = (long long)P.nchunk * P.ntx * P.nty;
    // planes per tile: 32, except pass F with one 64-column chunk per cell: 16 — measured
    // (profiles/r01_v6_stages.md): shorter tiles shorten the time between the waves of tiles, so more of
    // the halo shared across a wave boundary is still in L2, at the price of two more halo planes per
    // tile; at 128^3 x 64 pass F gains (0.929 -> 0.947), pass A loses (0.938 -> 0.907), and at 32 or 48
    // columns (256^3, 200x200x160) F does not gain either.  WRI_ZC / WRI_ZC_F / WRI_ZC_A override.
    // (pass F at 32 columns: 128 planes, 0.945 -> 0.957 at 256^3 x 32)
    int zc = std::min(c->g.nz, (is_f && Cfg::CB == 64 && P.nchunk == 1) ? 16 : (is_f && Cfg::CB == 32) ? 128 : 32);
    const char* zenv = getenv(is_f ? "WRI_ZC_F" : "WRI_ZC_A");
    if (!zenv) zenv = getenv("WRI_ZC");
    if (zenv && atoi(zenv) > 0) zc = std::min(c->g.nz, atoi(zenv));
    else
        while (zc > 8 && per_plane * ((c->g.nz + zc - 1) / zc) < 16LL * c->num_sms) zc = (zc + 1) / 2;
    P.zc = zc;
    P.ntz = (c->g.nz + zc - 1) / zc;
    const long long tiles = per_plane * P.ntz;
    if (tiles > 0x7fffffffLL) return WRI_ERR_ARG;
    P.tiles = (int)tiles;
    P.grid = (int)std::min<long long>(tiles, std::min(c->num_sms, kMaxCtas));
    int rc;
    const bool mg = P.nchunk == 1 && Cfg::CB * (P.txc + 2) <= 256 && !getenv("WRI_NO_MERGE");
    P.merged = mg;
    if ((rc = make_tmap(&P.in, in, c, c->nb, Cfg::CB, P.txc + 2, P.tyc + 2, mg))) return rc;
    if ((rc = make_tmap(&P.old, old, c, c->nb, Cfg::CB, P.txc, P.tyc, mg))) return rc;
    if (is_f) {
        if ((rc = make_tmap(&P.w, c->W, c, c->nb, Cfg::CB, P.txc, P.tyc, mg))) return rc;
        if ((rc = make_tmap(&P.x, c->X, c, c->nb, Cfg::CB, P.txc, P.tyc, mg))) return rc;
    } else {
        P.w = P.old; P.x = P.old;          // unused by pass A
    }
    if (!is_f && c->n_rec && rec_lists) {
        // receivers (x column chunks) inside each CTA's tiles, in the order the CTA walks its
        // tiles (same tile numbering as the kernel)
        const int G = P.grid, nent = c->n_rec * P.nchunk;
        struct Ent { int cta, tile, r; };
        std::vector<Ent> ents(nent);
        for (int e = 0; e < nent; ++e) {
            const int r = e / P.nchunk, chunk = e % P.nchunk;
            const int tx = c->rec_ijk[3 * r] / P.txc, ty = c->rec_ijk[3 * r + 1] / P.tyc;
            const int tz = c->rec_ijk[3 * r + 2] / P.zc;
            const int t = (int)((((long long)tz * P.nty + ty) * P.ntx + tx) * P.nchunk + chunk);
            ents[e] = {t % G, t, r};
        }
        std::sort(ents.begin(), ents.end(), [](const Ent& a, const Ent& b) {
            return a.cta != b.cta ? a.cta < b.cta : a.tile != b.tile ? a.tile < b.tile : a.r < b.r;
        });
        c->h_own_ptr.assign(G + 1, 0);
        c->h_own.resize(nent);
        for (int e = 0; e < nent; ++e) c->h_own_ptr[ents[e].cta + 1]++;
        for (int b = 0; b < G; ++b) c->h_own_ptr[b + 1] += c->h_own_ptr[b];
        for (int e = 0; e < nent;) {
            int f = e;
            while (f < nent && ents[f].cta == ents[e].cta && ents[f].tile == ents[e].tile) ++f;
            for (int j = e; j < f; ++j) {
                const int r = ents[j].r;
                const int cell = (c->rec_ijk[3 * r + 2] * c->g.ny + c->rec_ijk[3 * r + 1]) * c->g.nx + c->rec_ijk[3 * r];
                c->h_own[j] = make_int4(r, cell, ents[j].tile, j == e ? f - e : 0);
            }
            e = f;
        }
        CK(cudaMemcpyAsync(c->own_ptr, c->h_own_ptr.data(), (G + 1) * sizeof(int), cudaMemcpyHostToDevice, c->stream));
        CK(cudaMemcpyAsync(c->own, c->h_own.data(), nent * sizeof(int4), cudaMemcpyHostToDevice, c->stream));
    }
    P.m_tma = (c->g.nx % 4 == 0) && (P.txc % 4 == 0) && aligned16(c->m);
    if (P.m_tma) { if ((rc = make_tmap_model(&P.m, c, P.txc, P.tyc))) return rc; }
    else P.m = P.old;                       // unused placeholder
    return WRI_OK;
}

// One place that turns the run-time column-chunk width into its tile configuration: f is called with
// std::integral_constant<int, CB> for the CB that tma_chunk_for() returned.
template <class F>
int dispatch_cb(int cb, F&& f) {
    switch (cb) {
        case 64: return f(std::integral_constant<int, 64>{});
        case 56: return f(std::integral_constant<int, 56>{});
        case 48: return f(std::integral_constant<int, 48>{});
        case 40: return f(std::integral_constant<int, 40>{});
        case 32: return f(std::integral_constant<int, 32>{});
        case 24: return f(std::integral_constant<int, 24>{});
        case 8:  return f(std::integral_constant<int, 8>{});
        case 4:  return f(std::integral_constant<int, 4>{});
        case 2:  return f(std::integral_constant<int, 2>{});
        default: return f(std::integral_constant<int, 16>{});
    }
}

int tma_setup(wri_ctx* c) {
    c->tma_cb = tma_chunk_for(c->nb);
    if (!c->tma_cb) return WRI_OK;
    if (!get_encode_fn()) { c->tma_cb = 0; return WRI_OK; }
    return dispatch_cb(c->tma_cb, [&](auto cb) -> int {
        constexpr int CB = decltype(cb)::value;
        int rc = tma_plan<typename CfgFor<CB, MODE_F>::type>(c, c->planF, c->V, c->U, true);
        if (rc) return rc;
        return tma_plan<typename CfgFor<CB, MODE_A>::type>(c, c->planA, c->U, c->V, false);
    });
}

ScalParams scal_params(const wri_ctx* c, const double* partials, int n_rows, const float2* d) {
    ScalParams s{};
    s.partials = partials;
    s.n_tiles = n_rows;
    s.nb = c->nb; s.nb_max = c->nb_max;
    s.n_rec = c->n_rec; s.rec = c->rec;
    s.V = c->V; s.U_bot = c->U_bot; s.d = d;
    s.coef = c->coef; s.stat = c->stat; s.active = c->active; s.iters = c->iters;
    s.tol = c->tol; s.resnorms = c->resnorms; s.iters_out = c->iters_out;
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

// Ring depth per pass and plan.  Measured on B200 (profiles/r01_v6_stages.md): the adjoint pass is
// sensitive to the prefetch distance (more stages in flight cost L2 hits on the stencil halo), with
// the optimum near 130-160 KB of stages in flight: 6 stages for one 64-column chunk per cell, 5 for 32
// columns or several chunks, 7-8 for the narrower widths with their smaller stages; pass F at 3 (2 for
// 32-column chunks, 4 for 40).
template <class Cfg, int MODE>
int ring_depth(int nchunk) {
    int n;
    if (MODE == MODE_F) n = Cfg::CB == 32 ? 2 : Cfg::CB == 40 ? 4 : 3;
    else if (MODE == MODE_G) n = Cfg::NSTAGE;     // one light stream: the deepest ring the stage layout allows
    else if (Cfg::CB == 64) n = nchunk == 1 ? 6 : 5;
    else if (Cfg::CB == 32) n = 5;
    else if (Cfg::CB == 56) n = 6;
    else if (Cfg::CB == 48) n = 7;
    else if (Cfg::CB == 40 || Cfg::CB == 24) n = 8;
    else n = 7;                                   // 16, 8, 4, 2 columns: small stages, deeper ring
    if (const char* e = getenv(MODE == MODE_F ? "WRI_F_NSTAGE" : "WRI_A_NSTAGE"))
        if (atoi(e) > 0) n = atoi(e);
    return std::max(2, std::min(n, (int)Cfg::NSTAGE));
}

template <class Cfg, int MODE>
int launch_tma_cfg(wri_ctx* c, int phase) {
    const wri_ctx::TmaPlan& P = (MODE == MODE_F) ? c->planF : c->planA;
    const size_t smem = tma_smem_bytes<Cfg, MODE>(c);
    int rc_attr = allow_smem(c, (const void*)k_pass_tma<Cfg, MODE>, smem);
    if (rc_attr) return rc_attr;
    const size_t NM = c->nb_max;
    TmaPassParams p{};
    p.m = c->m;
    p.gx = c->gtab; p.gy = c->gtab + c->g.nx; p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef + C_W2 * NM;
    p.partials = c->partials_tma; p.counter = c->counter;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = c->nb;
    p.zc = P.zc; p.ntx = P.ntx; p.nty = P.nty; p.ntz = P.ntz;
    p.nchunk = P.nchunk; p.n_tiles = P.tiles;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(-6.0 / (c->h * c->h));
    p.phase = phase;
    // streams known to be zero are neither cleared nor read: V in the start's adjoint pass, W and X in the
    // first forward pass of a cold batch solve (c->wx_zero)
    p.has_q = (MODE == MODE_A) ? (phase != PH_INIT_A) : (MODE == MODE_F ? !c->wx_zero : 1);
    p.nstage = ring_depth<Cfg, MODE>(P.nchunk);
    p.m_tma = P.m_tma;
    p.merged = P.merged;
    p.fin = scal_params(c, c->partials_tma, P.grid, nullptr);
    p.n_rec = c->n_rec; p.rec = c->rec; p.U_bot = c->U_bot; p.V = c->V;
    p.ct = c->coef + C_CT_A * NM; p.own_ptr = c->own_ptr; p.own = c->own;
    if (MODE == MODE_F) {
        p.out = c->U; p.W = c->W; p.X = c->X; p.sgn = 1.f;
        p.ca = c->coef + C_CA_F * NM; p.cb = c->coef + C_CB_F * NM; p.cv = c->coef + C_CV_F * NM;
        p.cx = c->coef + C_CX * NM; p.cw = c->coef + C_CW * NM;
    } else {
        p.out = c->V; p.sgn = -1.f;
        p.ca = c->coef + C_CA_A * NM; p.cb = c->coef + C_CB_A * NM;
        p.cv = p.cx = p.cw = p.ca;
    }
    cudaEvent_t e1 = nullptr;
    if (c->profiling && phase != PH_INIT_A) {
        if (c->ev_used * 2 == c->ev_pool.size()) {
            cudaEvent_t a, b;
            CK(cudaEventCreate(&a));
            CK(cudaEventCreate(&b));
            c->ev_pool.push_back(a); c->ev_pool.push_back(b); c->ev_kind.push_back(0); c->ev_cols.push_back(0);
        }
        cudaEvent_t e0 = c->ev_pool[2 * c->ev_used];
        e1 = c->ev_pool[2 * c->ev_used + 1];
        c->ev_kind[c->ev_used] = (MODE == MODE_F) ? 0 : 1;
        c->ev_cols[c->ev_used] = c->nb;
        c->ev_used++;
        CK(cudaEventRecord(e0, c->stream));
    }
    k_pass_tma<Cfg, MODE><<<P.grid, Cfg::NT + 32, smem, c->stream>>>(P.in, P.old, P.w, P.x, P.m, p);
    c->launches++;
    CK(cudaGetLastError());
    if (e1) CK(cudaEventRecord(e1, c->stream));
    return WRI_OK;
}

template <int MODE>
int launch_tma(wri_ctx* c, int phase) {
    return dispatch_cb(c->tma_cb, [&](auto cb) -> int {
        return launch_tma_cfg<typename CfgFor<decltype(cb)::value, MODE>::type, MODE>(c, phase);
    });
}

// objective + gradient through the TMA pipeline (one chunk per cell, power-of-two column pairs)
template <int CB>
int launch_tma_grad(wri_ctx* c, const float2* u, const float2* q, const int* src, const float2* alpha,
                    float* g, float lambda) {
    // pass A's tile shape, 512 consumer threads (one item each): this pass is bound by
    // instruction issue, not by DRAM, and 4 warps per scheduler hide the shared-memory latency
    typedef typename CfgFor<CB, MODE_A>::type CfgA;
    typedef TileCfg<CB, CfgA::TXC, CfgA::TYC, WRI_F_NT, WRI_A_STAGES> Cfg;
    int rc = tma_plan<Cfg>(c, c->planG, u, q ? q : u, false, false);
    if (rc) return rc;
    const wri_ctx::TmaPlan& P = c->planG;
    const size_t smem = tma_smem_bytes<Cfg, MODE_G>(c);
    if ((rc = allow_smem(c, (const void*)k_pass_tma<Cfg, MODE_G>, smem))) return rc;
    const size_t NM = c->nb_max;
    TmaPassParams p{};
    p.m = c->m;
    p.gx = c->gtab; p.gy = c->gtab + c->g.nx; p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef + C_W2 * NM;
    p.ca = p.cb = p.cv = p.cx = p.cw = p.w2;      // unused by MODE_G
    p.partials = c->partials_tma; p.counter = c->counter;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = c->nb;
    p.zc = P.zc; p.ntx = P.ntx; p.nty = P.nty; p.ntz = P.ntz;
    p.nchunk = P.nchunk; p.n_tiles = P.tiles;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(-6.0 / (c->h * c->h));
    p.sgn = 1.f;
    p.m_tma = P.m_tma; p.merged = P.merged;
    p.nstage = ring_depth<Cfg, MODE_G>(P.nchunk);
    p.has_q = q != nullptr; p.gsrc = src; p.galpha = alpha; p.g = g; p.lam2 = lambda * lambda;
    k_pass_tma<Cfg, MODE_G><<<P.grid, Cfg::NT + 32, smem, c->stream>>>(P.in, P.old, P.old, P.old, P.m, p);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

// out = lambda * A in (sgn = +1) or lambda * A^H in (sgn = -1) through the TMA pipeline: pass A's kernel
// without its in-place stream, scalar phase and receiver rows.  No workspace is touched.
template <int CB>
int launch_tma_apply(wri_ctx* c, const float2* in, float2* out, float sgn) {
    typedef typename CfgFor<CB, MODE_A>::type Cfg;
    int rc = tma_plan<Cfg>(c, c->planG, in, in, false, false);
    if (rc) return rc;
    const wri_ctx::TmaPlan& P = c->planG;
    const size_t smem = tma_smem_bytes<Cfg, MODE_A>(c);
    if ((rc = allow_smem(c, (const void*)k_pass_tma<Cfg, MODE_A>, smem))) return rc;
    const size_t NM = c->nb_max;
    TmaPassParams p{};
    p.m = c->m;
    p.gx = c->gtab; p.gy = c->gtab + c->g.nx; p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef + C_W2 * NM;
    p.ca = c->coef + C_LAM * NM;
    p.cb = p.cv = p.cx = p.cw = p.ca;                 // unused without the in-place stream
    p.partials = nullptr; p.counter = c->counter;
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = c->nb;
    p.zc = P.zc; p.ntx = P.ntx; p.nty = P.nty; p.ntz = P.ntz;
    p.nchunk = P.nchunk; p.n_tiles = P.tiles;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(-6.0 / (c->h * c->h));
    p.sgn = sgn;
    p.phase = -1; p.has_q = 0; p.n_rec = 0;
    p.m_tma = P.m_tma; p.merged = P.merged;
    p.nstage = Cfg::NSTAGE;                           // no in-place stream: the deepest ring (measured 7 > 6 > 5)
    p.out = out;
    k_pass_tma<Cfg, MODE_A><<<P.grid, Cfg::NT + 32, smem, c->stream>>>(P.in, P.old, P.old, P.old, P.m, p);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

// operator part of wri_apply_M / _MH: TMA pipeline when the width has a tile configuration, else k_pass
int apply_operator(wri_ctx* c, int nb, const float2* in, float2* out, float sgn) {
    const int cb = (c->solving || getenv("WRI_APPLY_GENERIC") || !get_encode_fn()) ? 0 : tma_chunk_for(nb);
    if (cb) {
        const int nb_saved = c->nb;
        c->nb = nb;
        const int rc = dispatch_cb(cb, [&](auto t) -> int {
            return launch_tma_apply<decltype(t)::value>(c, in, out, sgn);
        });
        c->nb = nb_saved;
        return rc;
    }
    const Tiling t = make_tiling(c, nb);
    PassParams p = base_params(c, nb, t);
    p.in = in; p.out = out;
    p.ca = c->coef + C_LAM * (size_t)c->nb_max;
    p.sgn = sgn;
    return launch_pass<MODE_APPLY>(c, p, t);
}

int check_batch_args(const wri_ctx* c, int nb) {
    if (!c) return WRI_ERR_ARG;
    if (nb <= 0 || nb > c->nb_max) return WRI_ERR_ARG;
    if (c->rmask && c->rmask_nb != nb) return WRI_ERR_ARG;       // the receiver mask was given for another width
    if ((long long)c->ng * nb > 0x7fffffffLL * 1LL) return WRI_ERR_ARG;   // element indices stay below 2^31
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
    c->sponge = sponge; c->n_rec = n_rec; c->nb_max = nb_max;
    c->stream = (cudaStream_t)cuda_stream;
    c->m = m_dev;

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
    CKC(cudaMalloc(&c->own_ptr, (kMaxCtas + 1) * sizeof(int)));
    CKC(cudaMalloc(&c->own, (size_t)std::max(n_rec, 1) * (nb_max / kMinChunk + 1) * sizeof(int4)));
    CKC(cudaMalloc(&c->coef, (size_t)N_COEF * nb_max * sizeof(float)));
    CKC(cudaMemset(c->coef, 0, (size_t)N_COEF * nb_max * sizeof(float)));
    CKC(cudaMalloc(&c->stat, (size_t)N_STAT * nb_max * sizeof(double)));
    CKC(cudaMemset(c->stat, 0, (size_t)N_STAT * nb_max * sizeof(double)));
    CKC(cudaMalloc(&c->active, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->iters, nb_max * sizeof(int)));
    CKC(cudaMemset(c->active, 0, nb_max * sizeof(int)));
    CKC(cudaMemset(c->iters, 0, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->coef_alt, (size_t)N_COEF * nb_max * sizeof(float)));
    CKC(cudaMalloc(&c->stat_alt, (size_t)N_STAT * nb_max * sizeof(double)));
    CKC(cudaMalloc(&c->active_alt, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->iters_alt, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->colmap, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->src, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->idx, (size_t)3 * nb_max * sizeof(int)));
    CKC(cudaMallocHost(&c->h_active, nb_max * sizeof(int)));
    CKC(cudaMalloc(&c->aw_tol, nb_max * sizeof(float)));
    CKC(cudaMalloc(&c->aw_f, (size_t)2 * nb_max * sizeof(double)));
    CKC(cudaMalloc(&c->aw_ar0, nb_max * sizeof(double)));
    CKC(cudaMalloc(&c->aw_iters, nb_max * sizeof(int)));
    CKC(cudaMallocHost(&c->h_aw, (size_t)nb_max * (2 * sizeof(double) + sizeof(int))));
    CKC(cudaMalloc(&c->counter, sizeof(unsigned int)));
    CKC(cudaMemset(c->counter, 0, sizeof(unsigned int)));
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
    cudaFree(c->gtab); cudaFree(c->rec); cudaFree(c->coef); cudaFree(c->stat);
    cudaFree(c->active); cudaFree(c->iters); cudaFree(c->counter);
    cudaFree(c->own_ptr); cudaFree(c->own);
    cudaFree(c->coef_alt); cudaFree(c->stat_alt); cudaFree(c->active_alt); cudaFree(c->iters_alt);
    cudaFree(c->colmap); cudaFree(c->idx); cudaFree(c->src);
    if (c->h_active) cudaFreeHost(c->h_active);
    cudaFree(c->aw_tol); cudaFree(c->aw_f); cudaFree(c->aw_ar0); cudaFree(c->aw_iters);
    if (c->h_aw) cudaFreeHost(c->h_aw);
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
    CK(cudaStreamSynchronize(c->stream));
    *ms_f = *ms_a = 0.0; *n_f = *n_a = 0; *cols_f = *cols_a = 0;
    for (size_t i = 0; i < c->ev_used; ++i) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]));
        if (c->ev_kind[i] == 0) { *ms_f += ms; ++*n_f; *cols_f += c->ev_cols[i]; }
        else { *ms_a += ms; ++*n_a; *cols_a += c->ev_cols[i]; }
    }
    c->ev_used = 0;
    return WRI_OK;
}

int wri_apply_M(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, float lambda,
                const void* x_dev, void* ytop_dev, void* ybot_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!x_dev || !ytop_dev || (c->n_rec && !ybot_dev) || !aligned16(x_dev) || !aligned16(ytop_dev))
        return WRI_ERR_ARG;
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda))) return rc;
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
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda))) return rc;
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
    if ((rc = upload_sources(c, nb, src_ijk_host))) return rc;
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
    if ((rc = upload_sources(c, nb, src_ijk_host))) return rc;
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
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda))) return rc;
    if (src_ijk_host && (rc = upload_sources(c, nb, src_ijk_host))) return rc;
    GradParams p{};
    p.u = (const float2*)u_dev; p.q = (const float2*)q_dev;
    p.src = src_ijk_host ? c->src : nullptr; p.alpha = (const float2*)alpha_dev;
    p.m = c->m;
    p.gx = c->gtab; p.gy = c->gtab + c->g.nx; p.gz = c->gtab + c->g.nx + c->g.ny;
    p.w2 = c->coef + C_W2 * (size_t)c->nb_max;
    p.g = g_dev;
    p.partials = (double*)(c->ws + L.partials);
    p.nx = c->g.nx; p.ny = c->g.ny; p.nz = c->g.nz; p.nb = nb; p.zc = G.t.zc;
    p.tpc = G.tpc; p.shuffle = G.shuffle;
    p.ih2 = (float)(1.0 / (c->h * c->h));
    p.m6ih2 = (float)(-6.0 / (c->h * c->h));
    p.lam2 = lambda * lambda;
    // TMA pipeline when the batch is one power-of-two chunk per cell (64 / 32 / 16 / 8 / 4 columns);
    // the generic kernel otherwise (odd widths, 48, several chunks)
    int cb = tma_chunk_for(nb);
    if ((cb & (cb - 1)) || cb == 2 || cb != nb || !get_encode_fn() || getenv("WRI_GRAD_GENERIC")) cb = 0;
    int n_rows = (int)G.t.n_tiles;
    if (cb) {
        c->nb = nb;
        c->partials_tma = (double*)(c->ws + L.partials_tma);
        float* g_user = g_dev;
        if (g_dev) g_dev = (float*)(c->ws + L.gscratch);
        switch (cb) {
            case 64: rc = launch_tma_grad<64>(c, p.u, p.q, p.src, p.alpha, g_dev, lambda); break;
            case 32: rc = launch_tma_grad<32>(c, p.u, p.q, p.src, p.alpha, g_dev, lambda); break;
            case 16: rc = launch_tma_grad<16>(c, p.u, p.q, p.src, p.alpha, g_dev, lambda); break;
            case 8:  rc = launch_tma_grad<8>(c, p.u, p.q, p.src, p.alpha, g_dev, lambda); break;
            default: rc = launch_tma_grad<4>(c, p.u, p.q, p.src, p.alpha, g_dev, lambda); break;
        }
        if (rc) return rc;
        if (g_user) {
            k_add_f32<<<blocks_for((long long)c->ng), 256, 0, c->stream>>>(g_user, g_dev, (long long)c->ng);
            c->launches++;
            CK(cudaGetLastError());
        }
        p.partials = c->partials_tma;
        n_rows = c->planG.grid;
    } else {
        const size_t smem = (size_t)G.t.block.x * G.t.block.y * G.t.vec * sizeof(double);
        if (G.t.vec == 2) k_grad<2><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
        else              k_grad<1><<<G.t.grid, G.t.block, smem, c->stream>>>(p);
        c->launches++;
        CK(cudaGetLastError());
    }
    k_objective<<<(nb + OBJ_CPB - 1) / OBJ_CPB, 1024, 1024 * sizeof(double), c->stream>>>(p.partials, n_rows, nb, p.u,
                                                             (const float2*)d_dev, c->rec, c->n_rec,
                                                             (double)lambda * (double)lambda, f_pde_dev,
                                                             f_data_dev, c->rmask);
    c->launches++;
    CK(cudaGetLastError());
    return WRI_OK;
}

// ---- solver entries ----------------------------------------------------------------------------
}  // extern "C"

namespace {

int lsqr_begin_impl(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev,
                    const void* d_dev, float lambda, const float* tol_dev, int32_t maxit,
                    void* u_out_dev, float* resnorms_dev, int32_t* iters_dev, bool host_staged,
                    const int32_t* src_ijk_host = nullptr, void* alpha_out_dev = nullptr,
                    int col0 = 0, int nbw = 0, bool lazy_start = false) {
    // col0, nbw: a GROUPED solve works on the caller's columns [col0, col0 + nbw) only, in a compact
    // nbw-wide working set of its own (nbw = 0: all nb columns, working set = the caller's layout)
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    const bool grouped = nbw > 0 && nbw < nb;
    if (!grouped) { col0 = 0; nbw = nb; }
    const bool sf = src_ijk_host != nullptr;          // source-free system: q may be absent (b_top = 0)
    if ((!q_dev && !sf) || (c->n_rec && !d_dev) || !u_out_dev || maxit < 0 ||
        (q_dev && !aligned16(q_dev)) || !aligned16(u_out_dev) || q_dev == u_out_dev || (sf && !alpha_out_dev))
        return WRI_ERR_ARG;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    const int base_flags = host_staged ? WS_HOST_STAGING : 0;
    if (c->ws_bytes < ws_layout(c, nb, base_flags, kHostMaxitCap).total) return WRI_ERR_WORKSPACE;
    const WsLayout L = ws_layout(c, nb, base_flags | WS_COMPACTION, kHostMaxitCap);
    if ((rc = upload_columns(c, nbw, omega_idx_host ? omega_idx_host + col0 : nullptr, lambda))) return rc;
    if (sf && (rc = upload_sources(c, nb, src_ijk_host))) return rc;
    c->sf = sf;
    c->alpha_out = (float2*)alpha_out_dev;

    c->nb = nbw; c->nb0 = nb; c->k = 0; c->maxit = maxit; c->lambda = lambda;
    c->packed = grouped; c->all_done = false;
    c->U_bot = (float2*)(c->ws + L.U_bot);
    c->partials = (double*)(c->ws + L.partials);
    c->partials_tma = (double*)(c->ws + L.partials_tma);
    c->u_out = (float2*)u_out_dev;
    c->free_slots.clear();
    const bool ws_compact = c->ws_bytes >= L.total;           // the two spare vectors are there
    if (!grouped) {
        c->U = (float2*)(c->ws + L.U); c->V = (float2*)(c->ws + L.V); c->W = (float2*)(c->ws + L.W);
        c->X = (float2*)u_out_dev;
        if (ws_compact) {
            c->free_slots.push_back((float2*)(c->ws + L.B3));
            c->free_slots.push_back((float2*)(c->ws + L.B4));
            c->U_bot_alt = (float2*)(c->ws + L.U_bot2);
        }
    } else {
        // nbw-wide slots carved out of the nb-wide vector regions; the V region is skipped when the
        // host entry has staged q there (it must survive until the last group has started)
        const size_t slot = align_up(c->ng * (size_t)nbw * sizeof(float2), 256);
        const size_t region = align_up(c->ng * (size_t)nb * sizeof(float2), 256);
        std::vector<float2*> slots;
        size_t bases[5] = {L.U, L.V, L.W, L.B3, L.B4};
        for (int rgn = 0; rgn < (ws_compact ? 5 : 3); ++rgn) {
            if (rgn == 1 && host_staged && q_dev) continue;
            for (size_t o = 0; o + slot <= region; o += slot) slots.push_back((float2*)(c->ws + bases[rgn] + o));
        }
        if (slots.size() < 4) return WRI_ERR_WORKSPACE;
        c->U = slots[0]; c->V = slots[1]; c->W = slots[2]; c->X = slots[3];
        for (size_t i = 4; i < slots.size(); ++i) c->free_slots.push_back(slots[i]);
        // the receiver-row region holds nb columns: first half the rows, second half the spare
        c->U_bot_alt = c->U_bot + (size_t)std::max(c->n_rec, 1) * nbw;
        std::vector<int> cm(nbw);
        for (int j = 0; j < nbw; ++j) cm[j] = col0 + j;
        CK(cudaMemcpyAsync(c->colmap, cm.data(), nbw * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    }
    c->tol = tol_dev; c->resnorms = resnorms_dev; c->iters_out = iters_dev;
    c->tl = make_tiling(c, nbw);
    if ((rc = tma_setup(c))) return rc;
    // Convergence is watched from the host only when tolerances are given: every check_every
    // iterations (~2 ms of device work) the active flags are read back; converged columns are
    // compacted away when the workspace has room for it and the batch is on the TMA path.
    c->can_compact = tol_dev && c->tma_cb && c->free_slots.size() >= 2 && !getenv("WRI_NO_COMPACT");
    c->check_every = 0;
    if (tol_dev) {
        const double t_iter = 80.0 * (double)c->ng * nbw / 6.0e12;
        c->check_every = (int)std::min(32.0, std::max(1.0, std::ceil(2.0e-3 / t_iter)));
    }
    c->h_colmap.resize(nbw);
    for (int s = 0; s < nbw; ++s) c->h_colmap[s] = col0 + s;
    c->retired.assign(nb, 0);
    const size_t vbytes = c->ng * (size_t)nbw * sizeof(float2);
    const size_t NM = c->nb_max;

    // beta1 u1 = b = [lambda q ; d]   (q is consumed before V is cleared: the host entry
    // stages q in the V slot)
    PassParams p = base_params(c, nbw, c->tl);
    p.partials = c->partials;
    p.in = (const float2*)q_dev; p.out = c->U; p.ca = c->coef + C_LAM * NM;
    auto gather_in = [&](float2* dst, const void* src) -> int {      // dst[:, j] = src[:, col0 + j]
        k_gather_cols<<<blocks_for((long long)c->ng * nbw), 256, 0, c->stream>>>(
            dst, (const float2*)src, c->colmap, (long long)c->ng, nbw, nb);
        c->launches++;
        CK(cudaGetLastError());
        return WRI_OK;
    };
    if (grouped && c->opts.warm_start && (rc = gather_in(c->X, u_out_dev))) return rc;
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
        r.ca = c->coef + C_NLAM * NM; r.cb = c->coef + C_MONE * NM;
        if ((rc = launch_pass<MODE_A>(c, r, c->tl))) return rc;
    }
    // x0 = 0, w = 0, v = 0.  On the TMA path V is not read by the start's adjoint pass, and in a cold
    // batch solve of at least one iteration (lazy_start) W and X are not read by the first forward pass,
    // which writes them: no clearing needed.  (The stepping entries clear everything: their state can
    // be looked at before the first iteration.)
    c->wx_zero = lazy_start && c->tma_cb && !c->opts.warm_start && maxit >= 1;
    if (!c->opts.warm_start && !c->wx_zero) CK(cudaMemsetAsync(c->X, 0, vbytes, c->stream));
    if (!c->wx_zero) CK(cudaMemsetAsync(c->W, 0, vbytes, c->stream));
    if (!c->tma_cb) CK(cudaMemsetAsync(c->V, 0, vbytes, c->stream));
    if ((rc = launch_scalars<PH_INIT_B>(c, (const float2*)d_dev))) return rc;
    // alpha1 v1 = M^H u1
    if (c->tma_cb) {
        if ((rc = launch_tma<MODE_A>(c, PH_INIT_A))) return rc;
    } else {
        p.in = c->U; p.out = c->V; p.sgn = -1.f;
        p.ca = c->coef + C_CA_A * NM; p.cb = c->coef + C_CB_A * NM;
        if ((rc = launch_pass<MODE_A>(c, p, c->tl))) return rc;
        if ((rc = launch_scalars<PH_INIT_A>(c, nullptr))) return rc;
    }
    c->solving = true;
    return WRI_OK;
}


// x and history of the listed working columns become final in the caller's buffers:
// u_out[:, dst] = X[:, src] + cx[src] W[:, src]; resnorms rows k+1..maxit held at phibar.
int retire_columns(wri_ctx* c, const std::vector<int>& src, const std::vector<int>& dst) {
    const int n = (int)src.size();
    if (!n) return WRI_OK;
    const size_t NM = c->nb_max;
    int* d_src = c->idx + NM;
    int* d_dst = c->idx + 2 * NM;
    CK(cudaMemcpyAsync(d_src, src.data(), n * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(d_dst, dst.data(), n * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    k_retire_cols<<<blocks_for((long long)c->ng * n), 256, 0, c->stream>>>(
        c->u_out, c->X, c->W, c->coef + C_CX * NM, d_src, d_dst, n, (long long)c->ng, c->nb, c->nb0);
    c->launches++;
    CK(cudaGetLastError());
    if (c->k < c->maxit && c->resnorms) {
        k_hold_history<<<blocks_for((long long)(c->maxit - c->k) * n), 256, 0, c->stream>>>(
            c->resnorms, c->stat + S_PHIBAR * NM, d_src, d_dst, n, c->k + 1, c->maxit, c->nb0);
        c->launches++;
        CK(cudaGetLastError());
    }
    for (int t = 0; t < n; ++t) c->retired[dst[t]] = 1;
    return WRI_OK;
}

// working widths the TMA path serves: 2, 4, multiples of 8 up to 64, then multiples of 16
int round_up16(int n) { return n <= 2 ? 2 : n <= 4 ? 4 : n <= 64 ? (n + 7) / 8 * 8 : (n + 15) / 16 * 16; }

// Re-pack the working set to the columns still active (plus zero padding up to the next supported width).
int compact_columns(wri_ctx* c, const int* act) {
    std::vector<int> keep, rs, rd;
    for (int j = 0; j < c->nb; ++j) {
        const int so = c->h_colmap[j];
        if (act[j]) keep.push_back(j);
        else if (so >= 0 && !c->retired[so]) { rs.push_back(j); rd.push_back(so); }
    }
    const int new_nb = round_up16((int)keep.size());
    if (new_nb >= c->nb) return WRI_OK;
    int rc = retire_columns(c, rs, rd);
    if (rc) return rc;
    std::vector<int> map(new_nb, -1), cm(new_nb, -1);
    for (size_t i = 0; i < keep.size(); ++i) { map[i] = keep[i]; cm[i] = c->h_colmap[keep[i]]; }
    const size_t NM = c->nb_max;
    CK(cudaMemcpyAsync(c->idx, map.data(), new_nb * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->colmap, cm.data(), new_nb * sizeof(int), cudaMemcpyHostToDevice, c->stream));
    // vectors: gather each into a free slot, then its old slot becomes free (X = u_out is the caller's)
    float2** vecs[4] = {&c->U, &c->V, &c->W, &c->X};
    for (int i = 0; i < 4; ++i) {
        if (c->free_slots.empty()) return WRI_ERR_STATE;
        float2* dst = c->free_slots.front();
        c->free_slots.erase(c->free_slots.begin());
        float2* src = *vecs[i];
        k_gather_cols<<<blocks_for((long long)c->ng * new_nb), 256, 0, c->stream>>>(
            dst, src, c->idx, (long long)c->ng, new_nb, c->nb);
        c->launches++;
        CK(cudaGetLastError());
        if (!(i == 3 && !c->packed)) c->free_slots.push_back(src);
        *vecs[i] = dst;
    }
    if (c->n_rec) {
        k_gather_cols<<<blocks_for((long long)c->n_rec * new_nb), 256, 0, c->stream>>>(
            c->U_bot_alt, c->U_bot, c->idx, (long long)c->n_rec, new_nb, c->nb);
        c->launches++;
        CK(cudaGetLastError());
        std::swap(c->U_bot, c->U_bot_alt);
    }
    k_gather_scalars<<<(new_nb + 127) / 128, 128, 0, c->stream>>>(
        c->coef_alt, c->coef, c->stat_alt, c->stat, c->active_alt, c->active, c->iters_alt, c->iters,
        c->idx, new_nb, (int)NM);
    c->launches++;
    CK(cudaGetLastError());
    std::swap(c->coef, c->coef_alt); std::swap(c->stat, c->stat_alt);
    std::swap(c->active, c->active_alt); std::swap(c->iters, c->iters_alt);
    c->h_colmap = cm;
    c->nb = new_nb;
    c->packed = true;
    c->tl = make_tiling(c, new_nb);
    return tma_setup(c);
}

// host look at the active flags: early exit when every column has stopped, compaction when the
// active count has dropped below the next supported width
int check_active(wri_ctx* c) {
    CK(cudaMemcpyAsync(c->h_active, c->active, c->nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    int n_act = 0;
    for (int j = 0; j < c->nb; ++j) n_act += c->h_active[j] != 0;
    if (n_act == 0) { c->all_done = true; return WRI_OK; }
    if (c->can_compact && round_up16(n_act) < c->nb) return compact_columns(c, c->h_active);
    return WRI_OK;
}

// A batch wider than one 64-column chunk per cell is solved as successive 64-column GROUPS, each in a
// compact working set of its own (columns are independent systems; reading C-9: a
// column's result does not depend on its batch).  With several chunks per cell a tile row is a 512-byte
// piece of a wider cell record and the passes reach 0.84-0.88 of the copy bandwidth; compact groups
// run at the single-chunk rate (0.92).  The stepping entries keep all columns in lock-step.
int group_width(const wri_ctx* c, int nb) {
    if (getenv("WRI_NO_GROUPS")) return 0;
    return (nb > 64 && nb % 64 == 0 && tma_chunk_for(64) == 64 && get_encode_fn()) ? 64 : 0;
}

int solve_groups(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev, const void* d_dev,
                 float lambda, const float* tol_dev, int32_t maxit, void* u_out_dev, float* resnorms_dev,
                 int32_t* iters_dev, bool host_staged, const int32_t* src_ijk_host, void* alpha_out_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    const int gw = group_width(c, nb);
    for (int col0 = 0; col0 < nb; col0 += (gw ? gw : nb)) {
        if ((rc = lsqr_begin_impl(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev,
                                  resnorms_dev, iters_dev, host_staged, src_ijk_host, alpha_out_dev, col0, gw, true)))
            return rc;
        if ((rc = wri_lsqr_iterate(c, maxit))) { c->solving = false; return rc; }
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
    for (int i = 0; i < n_steps && !c->all_done; ++i) {
        c->k++;
        const size_t NM = c->nb_max;
        if (c->tma_cb) {
            // two launches per iteration: the last CTA of each pass runs the scalar recurrences
            if ((rc = launch_tma<MODE_F>(c, PH_F))) return rc;
            c->wx_zero = false;
            if ((rc = launch_tma<MODE_A>(c, PH_A))) return rc;
        } else {
            PassParams p = base_params(c, c->nb, c->tl);
            p.partials = c->partials;
            // pass F: U <- (lambda/alpha) A V - (alpha/beta) U ; deferred x, w updates
            p.in = c->V; p.out = c->U; p.W = c->W; p.X = c->X; p.sgn = 1.f;
            p.ca = c->coef + C_CA_F * NM; p.cb = c->coef + C_CB_F * NM; p.cv = c->coef + C_CV_F * NM;
            p.cx = c->coef + C_CX * NM; p.cw = c->coef + C_CW * NM;
            if ((rc = launch_pass<MODE_F>(c, p, c->tl, true))) return rc;
            if ((rc = launch_scalars<PH_F>(c, nullptr))) return rc;
            // pass A: V <- (lambda/beta) A^H U - (beta/alpha) V
            p.in = c->U; p.out = c->V; p.W = nullptr; p.X = nullptr; p.sgn = -1.f;
            p.ca = c->coef + C_CA_A * NM; p.cb = c->coef + C_CB_A * NM;
            if ((rc = launch_pass<MODE_A>(c, p, c->tl, true))) return rc;
            if ((rc = launch_scalars<PH_A>(c, nullptr))) return rc;
        }
        if (c->check_every && c->k % c->check_every == 0 && c->k < c->maxit)
            if ((rc = check_active(c))) return rc;
    }
    return WRI_OK;
}

int wri_lsqr_end(wri_ctx* c) {
    if (!c) return WRI_ERR_ARG;
    if (!c->solving) return WRI_ERR_STATE;
    const size_t NM = c->nb_max;
    int rc;
    if (!c->packed && c->k == c->maxit) {
        // X is the caller's buffer: apply the last deferred update in place
        const long long n = (long long)c->ng * c->nb;
        k_flush_x<<<148 * 8, 256, 0, c->stream>>>(c->X, c->W, c->coef + C_CX * NM, n, c->nb);
        c->launches++;
        CK(cudaGetLastError());
    } else {
        // stopped early and / or compacted: every column not yet final is retired now
        std::vector<int> rs, rd;
        for (int j = 0; j < c->nb; ++j) {
            const int so = c->h_colmap[j];
            if (so >= 0 && !c->retired[so]) { rs.push_back(j); rd.push_back(so); }
        }
        if ((rc = retire_columns(c, rs, rd))) return rc;
    }
    CK(cudaMemsetAsync(c->coef + C_CX * NM, 0, c->nb * sizeof(float), c->stream));
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
    float2* Qs = q_host ? (float2*)(c->ws + L.V) : nullptr;
    float2* As = (float2*)(c->ws + L.alphas);
    if (c->opts.warm_start) {                 // x0 (alpha0) arrive in the output buffers
        CK(cudaMemcpyAsync(Xs, u_out_host, vbytes, cudaMemcpyHostToDevice, c->stream));
        if (sf) CK(cudaMemcpyAsync(As, alpha_out_host, nb * sizeof(float2), cudaMemcpyHostToDevice, c->stream));
    }
    if (Qs) CK(cudaMemcpyAsync(Qs, q_host, vbytes, cudaMemcpyHostToDevice, c->stream));
    if (dbytes) CK(cudaMemcpyAsync(Ds, d_host, dbytes, cudaMemcpyHostToDevice, c->stream));
    if (tol_host) CK(cudaMemcpyAsync(tols, tol_host, nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    if ((rc = solve_groups(c, nb, omega_idx_host, Qs, Ds, lambda, tol_host ? tols : nullptr, maxit, Xs, res, its,
                           true, src_ijk_host, sf ? As : nullptr)))
        return rc;
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
    v->nb = c->nb; v->k = c->k;
    v->U_top = c->U; v->U_bot = c->U_bot; v->V = c->V; v->W = c->W; v->X = c->X;
    v->alpha = c->stat + S_ALPHA * NM; v->beta = c->stat + S_BETA * NM;
    v->rhobar = c->stat + S_RHOBAR * NM; v->phibar = c->stat + S_PHIBAR * NM;
    v->ar0 = c->stat + S_AR0 * NM;
    v->cx = c->coef + C_CX * NM;
    v->cw = c->coef + C_CW * NM;
    v->active = c->active; v->iters = c->iters;
    v->nb_max = c->nb_max;
    v->sf_state = c->sf ? c->stat + S_VA_RE * NM : nullptr;
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
    rc = wri_lsqr_sf_batch(c, nb, omega_idx_host, src_ijk_host, nullptr, d_dev, lambda,
                           eps > 0.f ? c->aw_tol : nullptr, maxit, u_dev, alpha_dev, nullptr, its);
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
        rep->trace_eps[h] = eps; rep->trace_f[h] = f; rep->trace_f_trial[h] = f_trial;
        rep->n_trace = h + 1;
        rep->f = f; rep->f_trial = f_trial; rep->eps = eps; rep->n_halvings = h;
        rep->lsqr_iters += it0 + it1;
        if (!(f_trial > f)) {                               // line 9 / 12-13
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
