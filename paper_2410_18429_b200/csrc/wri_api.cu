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

constexpr int kMaxCtas = 512;          // upper bound on the persistent grid (>= SM count)
constexpr int kMinChunk = 16;          // narrowest column chunk of the TMA path

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
    float* coef = nullptr;       // [N_COEF][nb_max]
    double* stat = nullptr;      // [N_STAT][nb_max]
    int* active = nullptr;       // [nb_max]
    int* iters = nullptr;        // [nb_max]
    // caller's workspace
    char* ws = nullptr;
    size_t ws_bytes = 0;
    // solve in flight
    bool solving = false;
    int nb = 0, k = 0, maxit = 0;
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
    } planF, planA;
    double* partials_tma = nullptr;       // [grid][nb]
    // optional per-kernel timing (wri_profile_*)
    bool profiling = false;
    std::vector<cudaEvent_t> ev_pool;     // pairs: start, stop
    std::vector<int> ev_kind;             // per pair: 0 = pass F, 1 = pass A
    size_t ev_used = 0;                   // pairs in use
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

struct WsLayout {
    size_t U, V, W, U_bot, partials, partials_tma, Xs, Ds, tols, res, its, total;
};
WsLayout ws_layout(const wri_ctx* c, int nb, int host_staging, int maxit_cap) {
    WsLayout L{};
    size_t vec = align_up(c->ng * (size_t)nb * sizeof(float2), 256);
    if (const char* e = getenv("WRI_PAD")) vec += (size_t)atoll(e);
    const size_t bot = align_up((size_t)std::max(c->n_rec, 1) * nb * sizeof(float2), 256);
    const Tiling t = make_tiling(c, nb);
    size_t o = 0;
    L.U = o; o += vec;
    L.V = o; o += vec;
    L.W = o; o += vec;
    L.U_bot = o; o += bot;
    L.partials = o; o += align_up(t.n_tiles * nb * sizeof(double), 256);
    L.partials_tma = o; o += align_up((size_t)kMaxCtas * nb * sizeof(double), 256);
    if (host_staging) {
        L.Xs = o; o += vec;
        L.Ds = o; o += bot;
        L.tols = o; o += align_up((size_t)nb * sizeof(float), 256);
        L.res = o; o += align_up((size_t)(maxit_cap + 1) * nb * sizeof(float), 256);
        L.its = o; o += align_up((size_t)nb * sizeof(int), 256);
    }
    L.total = o;
    return L;
}
constexpr int kHostMaxitCap = 4096;   // resnorm staging rows reserved for wri_lsqr_batch_host

int upload_columns(wri_ctx* c, int nb, const int32_t* omega_idx, float lambda) {
    std::vector<float> w2(nb), one(nb, 1.f), lam(nb, lambda);
    for (int s = 0; s < nb; ++s) {
        const int j = omega_idx ? omega_idx[s] : 0;
        if (j < 0 || j >= (int)c->omega.size()) return WRI_ERR_ARG;
        w2[s] = (float)(c->omega[j] * c->omega[j]);
    }
    const size_t NM = c->nb_max;
    CK(cudaMemcpyAsync(c->coef + C_W2 * NM, w2.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->coef + C_ONE * NM, one.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(c->coef + C_LAM * NM, lam.data(), nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
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
            c->ev_pool.push_back(a); c->ev_pool.push_back(b); c->ev_kind.push_back(0);
        }
        e0 = c->ev_pool[2 * c->ev_used]; e1 = c->ev_pool[2 * c->ev_used + 1];
        c->ev_kind[c->ev_used] = (MODE == MODE_F) ? 0 : 1;
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

template <int PHASE>
int launch_scalars(wri_ctx* c, const float2* d) {
    ScalParams s{};
    s.partials = c->partials;
    s.n_tiles = (int)c->tl.n_tiles;
    s.nb = c->nb; s.nb_max = c->nb_max;
    s.n_rec = c->n_rec; s.rec = c->rec;
    s.V = c->V; s.U_bot = c->U_bot; s.d = d;
    s.coef = c->coef; s.stat = c->stat; s.active = c->active; s.iters = c->iters;
    s.tol = c->tol; s.resnorms = c->resnorms; s.iters_out = c->iters_out;
    s.k = c->k; s.maxit = c->maxit; s.lambda = c->lambda;
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
int make_tmap(CUtensorMap* tm, const void* base, const wri_ctx* c, int nb, int cb, int bx, int by) {
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return cuda_fail(cudaErrorNotSupported, "cuTensorMapEncodeTiled lookup");
    cuuint64_t gdim[4] = {(cuuint64_t)nb, (cuuint64_t)c->g.nx, (cuuint64_t)c->g.ny, (cuuint64_t)c->g.nz};
    cuuint64_t gstr[3] = {(cuuint64_t)nb * 8, (cuuint64_t)nb * 8 * c->g.nx,
                          (cuuint64_t)nb * 8 * c->g.nx * c->g.ny};
    cuuint32_t box[4] = {(cuuint32_t)cb, (cuuint32_t)bx, (cuuint32_t)by, 1};
    cuuint32_t estr[4] = {1, 1, 1, 1};
    CUtensorMapL2promotion promo = CU_TENSOR_MAP_L2_PROMOTION_L2_256B;
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
#define WRI_A_NT 256
#endif
template <int CB, int MODE> struct CfgFor {
    static constexpr int S = 64 / CB;   // narrower chunks -> proportionally more cells per tile row
    typedef TileCfg<CB, (MODE == MODE_F ? WRI_F_TX : WRI_A_TX) * (S >= 2 ? 2 : 1),
                    (MODE == MODE_F ? WRI_F_TY : WRI_A_TY) * (S >= 4 ? 2 : 1),
                    (MODE == MODE_F ? WRI_F_NT : WRI_A_NT)> type;
};

int tma_chunk_for(int nb) {
    const char* off = getenv("WRI_NO_TMA");
    if (off && off[0] == '1') return 0;
    if (nb % 64 == 0) return 64;
    if (nb % 32 == 0) return 32;
    if (nb % 16 == 0) return 16;
    return 0;
}

template <class Cfg, int MODE>
size_t tma_smem_bytes(const wri_ctx* c) {
    return (size_t)PassTraits<MODE>::NSTAGE *
               (Cfg::IN_BYTES + PassTraits<MODE>::NSTREAM * Cfg::CTR_BYTES + Cfg::M_BYTES) +
           2 * PassTraits<MODE>::NSTAGE * 8 + (size_t)c->nb * 8 + (size_t)Cfg::NT * 2 * 8 +
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
int tma_plan(wri_ctx* c, wri_ctx::TmaPlan& P, const void* in, const void* old, bool is_f) {
    P.txc = Cfg::TXC; P.tyc = Cfg::TYC;
    P.nchunk = c->nb / Cfg::CB;
    P.ntx = (c->g.nx + P.txc - 1) / P.txc;
    P.nty = (c->g.ny + P.tyc - 1) / P.tyc;
    const long long per_plane = (long long)P.nchunk * P.ntx * P.nty;
    int zc = std::min(c->g.nz, 32);
    const char* zenv = getenv("WRI_ZC");
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
    if ((rc = make_tmap(&P.in, in, c, c->nb, Cfg::CB, P.txc + 2, P.tyc + 2))) return rc;
    if ((rc = make_tmap(&P.old, old, c, c->nb, Cfg::CB, P.txc, P.tyc))) return rc;
    if (is_f) {
        if ((rc = make_tmap(&P.w, c->W, c, c->nb, Cfg::CB, P.txc, P.tyc))) return rc;
        if ((rc = make_tmap(&P.x, c->X, c, c->nb, Cfg::CB, P.txc, P.tyc))) return rc;
    } else {
        P.w = P.old; P.x = P.old;          // unused by pass A
    }
    if (!is_f && c->n_rec) {
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

int tma_setup(wri_ctx* c) {
    c->tma_cb = tma_chunk_for(c->nb);
    if (!c->tma_cb) return WRI_OK;
    if (!get_encode_fn()) { c->tma_cb = 0; return WRI_OK; }
    int rc;
    switch (c->tma_cb) {
        case 64:
            if ((rc = tma_plan<CfgFor<64, MODE_F>::type>(c, c->planF, c->V, c->U, true))) return rc;
            return tma_plan<CfgFor<64, MODE_A>::type>(c, c->planA, c->U, c->V, false);
        case 32:
            if ((rc = tma_plan<CfgFor<32, MODE_F>::type>(c, c->planF, c->V, c->U, true))) return rc;
            return tma_plan<CfgFor<32, MODE_A>::type>(c, c->planA, c->U, c->V, false);
        default:
            if ((rc = tma_plan<CfgFor<16, MODE_F>::type>(c, c->planF, c->V, c->U, true))) return rc;
            return tma_plan<CfgFor<16, MODE_A>::type>(c, c->planA, c->U, c->V, false);
    }
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
    return s;
}

template <class Cfg, int MODE>
int launch_tma_cfg(wri_ctx* c, int phase) {
    static size_t attr_bytes = 0;
    const wri_ctx::TmaPlan& P = (MODE == MODE_F) ? c->planF : c->planA;
    const size_t smem = tma_smem_bytes<Cfg, MODE>(c);
    if (smem > attr_bytes) {
        CK(cudaFuncSetAttribute(k_pass_tma<Cfg, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        attr_bytes = smem;
    }
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
    p.m_tma = P.m_tma;
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
            c->ev_pool.push_back(a); c->ev_pool.push_back(b); c->ev_kind.push_back(0);
        }
        cudaEvent_t e0 = c->ev_pool[2 * c->ev_used];
        e1 = c->ev_pool[2 * c->ev_used + 1];
        c->ev_kind[c->ev_used] = (MODE == MODE_F) ? 0 : 1;
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
    switch (c->tma_cb) {
        case 64: return launch_tma_cfg<typename CfgFor<64, MODE>::type, MODE>(c, phase);
        case 32: return launch_tma_cfg<typename CfgFor<32, MODE>::type, MODE>(c, phase);
        default: return launch_tma_cfg<typename CfgFor<16, MODE>::type, MODE>(c, phase);
    }
}

int check_batch_args(const wri_ctx* c, int nb) {
    if (!c) return WRI_ERR_ARG;
    if (nb <= 0 || nb > c->nb_max) return WRI_ERR_ARG;
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
    for (cudaEvent_t e : c->ev_pool) cudaEventDestroy(e);
    delete c;
    return WRI_OK;
}

int wri_set_model(wri_ctx* c, const float* m_dev) {
    if (!c || !m_dev) return WRI_ERR_ARG;
    c->m = m_dev;
    return WRI_OK;
}

size_t wri_workspace_bytes(const wri_ctx* c, int32_t nb, int32_t host_staging) {
    if (!c || nb <= 0 || nb > c->nb_max) return 0;
    return ws_layout(c, nb, host_staging, kHostMaxitCap).total;
}

int wri_set_workspace(wri_ctx* c, void* ws_dev, size_t bytes) {
    if (!c || !ws_dev || !aligned16(ws_dev)) return WRI_ERR_ARG;
    if (c->solving) return WRI_ERR_STATE;
    c->ws = (char*)ws_dev;
    c->ws_bytes = bytes;
    return WRI_OK;
}

int64_t wri_launch_count(const wri_ctx* c) { return c ? c->launches : 0; }

int wri_profile_enable(wri_ctx* c, int32_t on) {
    if (!c) return WRI_ERR_ARG;
    c->profiling = on != 0;
    return WRI_OK;
}

int wri_profile_read(wri_ctx* c, double* ms_f, int64_t* n_f, double* ms_a, int64_t* n_a) {
    if (!c || !ms_f || !n_f || !ms_a || !n_a) return WRI_ERR_ARG;
    CK(cudaStreamSynchronize(c->stream));
    *ms_f = *ms_a = 0.0; *n_f = *n_a = 0;
    for (size_t i = 0; i < c->ev_used; ++i) {
        float ms = 0.f;
        CK(cudaEventElapsedTime(&ms, c->ev_pool[2 * i], c->ev_pool[2 * i + 1]));
        if (c->ev_kind[i] == 0) { *ms_f += ms; ++*n_f; } else { *ms_a += ms; ++*n_a; }
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
    const Tiling t = make_tiling(c, nb);
    PassParams p = base_params(c, nb, t);
    p.in = (const float2*)x_dev; p.out = (float2*)ytop_dev;
    p.ca = c->coef + C_LAM * (size_t)c->nb_max;
    p.sgn = 1.f;
    if ((rc = launch_pass<MODE_APPLY>(c, p, t))) return rc;
    if (c->n_rec) {
        const long long n = (long long)c->n_rec * nb;
        k_gather<<<(unsigned)std::min<long long>((n + 255) / 256, 1184), 256, 0, c->stream>>>(
            (const float2*)x_dev, c->rec, c->n_rec, nb, (float2*)ybot_dev);
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
    const Tiling t = make_tiling(c, nb);
    PassParams p = base_params(c, nb, t);
    p.in = (const float2*)ytop_dev; p.out = (float2*)x_dev;
    p.ca = c->coef + C_LAM * (size_t)c->nb_max;
    p.sgn = -1.f;
    if ((rc = launch_pass<MODE_APPLY>(c, p, t))) return rc;
    if (c->n_rec) {
        const long long n = (long long)c->n_rec * nb;
        k_scatter_add<<<(unsigned)std::min<long long>((n + 255) / 256, 1184), 256, 0, c->stream>>>(
            (float2*)x_dev, c->rec, c->n_rec, nb, (const float2*)ybot_dev);
        c->launches++;
        CK(cudaGetLastError());
    }
    return WRI_OK;
}

int wri_lsqr_begin(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev,
                   const void* d_dev, float lambda, const float* tol_dev, int32_t maxit,
                   void* u_out_dev, float* resnorms_dev, int32_t* iters_dev) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!q_dev || (c->n_rec && !d_dev) || !u_out_dev || !resnorms_dev || maxit < 0 ||
        !aligned16(q_dev) || !aligned16(u_out_dev) || q_dev == u_out_dev)
        return WRI_ERR_ARG;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    const WsLayout L = ws_layout(c, nb, 0, 0);
    if (c->ws_bytes < L.total) return WRI_ERR_WORKSPACE;
    if ((rc = upload_columns(c, nb, omega_idx_host, lambda))) return rc;

    c->nb = nb; c->k = 0; c->maxit = maxit; c->lambda = lambda;
    c->U = (float2*)(c->ws + L.U); c->V = (float2*)(c->ws + L.V); c->W = (float2*)(c->ws + L.W);
    c->U_bot = (float2*)(c->ws + L.U_bot);
    c->partials = (double*)(c->ws + L.partials);
    c->partials_tma = (double*)(c->ws + L.partials_tma);
    c->X = (float2*)u_out_dev;
    c->tol = tol_dev; c->resnorms = resnorms_dev; c->iters_out = iters_dev;
    c->tl = make_tiling(c, nb);
    if ((rc = tma_setup(c))) return rc;
    const size_t vbytes = c->ng * (size_t)nb * sizeof(float2);
    const size_t NM = c->nb_max;

    // beta1 u1 = b = [lambda q ; d]   (q is consumed before V is cleared: the host entry
    // stages q in the V slot)
    PassParams p = base_params(c, nb, c->tl);
    p.partials = c->partials;
    p.in = (const float2*)q_dev; p.out = c->U; p.ca = c->coef + C_LAM * NM;
    if ((rc = launch_pass<MODE_INIT>(c, p, c->tl))) return rc;
    CK(cudaMemsetAsync(c->X, 0, vbytes, c->stream));
    CK(cudaMemsetAsync(c->W, 0, vbytes, c->stream));
    CK(cudaMemsetAsync(c->V, 0, vbytes, c->stream));
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

int wri_lsqr_iterate(wri_ctx* c, int32_t n_steps) {
    if (!c || n_steps < 0) return WRI_ERR_ARG;
    if (!c->solving) return WRI_ERR_STATE;
    if (c->k + n_steps > c->maxit) return WRI_ERR_ARG;
    const size_t NM = c->nb_max;
    int rc;
    for (int i = 0; i < n_steps; ++i) {
        c->k++;
        if (c->tma_cb) {
            // two launches per iteration: the last CTA of each pass runs the scalar recurrences
            if ((rc = launch_tma<MODE_F>(c, PH_F))) return rc;
            if ((rc = launch_tma<MODE_A>(c, PH_A))) return rc;
            continue;
        }
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
    return WRI_OK;
}

int wri_lsqr_end(wri_ctx* c) {
    if (!c) return WRI_ERR_ARG;
    if (!c->solving) return WRI_ERR_STATE;
    const long long n = (long long)c->ng * c->nb;
    const size_t NM = c->nb_max;
    k_flush_x<<<148 * 8, 256, 0, c->stream>>>(c->X, c->W, c->coef + C_CX * NM, n, c->nb);
    c->launches++;
    CK(cudaGetLastError());
    CK(cudaMemsetAsync(c->coef + C_CX * NM, 0, c->nb * sizeof(float), c->stream));
    c->solving = false;
    return WRI_OK;
}

int wri_lsqr_batch(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_dev,
                   const void* d_dev, float lambda, const float* tol_dev, int32_t maxit,
                   void* u_out_dev, float* resnorms_dev, int32_t* iters_dev) {
    int rc = wri_lsqr_begin(c, nb, omega_idx_host, q_dev, d_dev, lambda, tol_dev, maxit, u_out_dev,
                            resnorms_dev, iters_dev);
    if (rc) return rc;
    if ((rc = wri_lsqr_iterate(c, maxit))) { c->solving = false; return rc; }
    return wri_lsqr_end(c);
}

int wri_lsqr_batch_host(wri_ctx* c, int32_t nb, const int32_t* omega_idx_host, const void* q_host,
                        const void* d_host, float lambda, const float* tol_host, int32_t maxit,
                        void* u_out_host, float* resnorms_host, int32_t* iters_host) {
    int rc = check_batch_args(c, nb);
    if (rc) return rc;
    if (!q_host || (c->n_rec && !d_host) || !u_out_host || !resnorms_host || maxit < 0 ||
        maxit > kHostMaxitCap)
        return WRI_ERR_ARG;
    if (!c->ws) return WRI_ERR_WORKSPACE;
    const WsLayout L = ws_layout(c, nb, 1, kHostMaxitCap);
    if (c->ws_bytes < L.total) return WRI_ERR_WORKSPACE;
    const size_t vbytes = c->ng * (size_t)nb * sizeof(float2);
    const size_t dbytes = (size_t)c->n_rec * nb * sizeof(float2);
    float2* Xs = (float2*)(c->ws + L.Xs);
    float2* Ds = (float2*)(c->ws + L.Ds);
    float* tols = (float*)(c->ws + L.tols);
    float* res = (float*)(c->ws + L.res);
    int* its = (int*)(c->ws + L.its);
    // q is staged in the V slot: wri_lsqr_begin consumes q before it clears V
    float2* Qs = (float2*)(c->ws + L.V);
    CK(cudaMemcpyAsync(Qs, q_host, vbytes, cudaMemcpyHostToDevice, c->stream));
    if (dbytes) CK(cudaMemcpyAsync(Ds, d_host, dbytes, cudaMemcpyHostToDevice, c->stream));
    if (tol_host) CK(cudaMemcpyAsync(tols, tol_host, nb * sizeof(float), cudaMemcpyHostToDevice, c->stream));
    rc = wri_lsqr_batch(c, nb, omega_idx_host, Qs, Ds, lambda, tol_host ? tols : nullptr, maxit, Xs, res, its);
    if (rc) return rc;
    CK(cudaMemcpyAsync(u_out_host, Xs, vbytes, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaMemcpyAsync(resnorms_host, res, (size_t)(maxit + 1) * nb * sizeof(float), cudaMemcpyDeviceToHost, c->stream));
    if (iters_host) CK(cudaMemcpyAsync(iters_host, its, nb * sizeof(int), cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return WRI_OK;
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
    return WRI_OK;
}

}  // extern "C"
