// wri_kernels.cuh — sm_100a device code of libwri (see include/wri.h for the operations).
//
// Layout: complex64 vectors are source-interleaved, element (c, s) at c*nb + s with
// c = (iz*ny + iy)*nx + ix.  One x-row of the grid is therefore a contiguous run of
// RL = nx*nb complex numbers; x-neighbours are +-nb elements away, y-neighbours +-RL,
// z-neighbours +-RL*ny.  A thread owns VEC consecutive columns of one cell (16 B when
// VEC = 2) and marches along z with a three-plane register pipeline, so each element of
// the stencil input is fetched from HBM once per pass; x/y neighbours are re-read through
// L1/L2 (they are the centre loads of neighbouring threads of the same tile).
//
// Every LSQR vector operation is fused into the two stencil passes:
//   pass F : U <- ca * A V  - cb * U,  ||U||^2 partials,  X += cx W,  W <- cv V - cw W
//   pass A : V <- ca * A^H U - cb * V, ||V||^2 partials
// with per-column coefficients (lazy normalisation: U, V stay un-normalised).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace wri {

enum PassMode { MODE_APPLY = 0, MODE_A = 1, MODE_F = 2, MODE_INIT = 3, MODE_G = 4 };

// per-column float coefficients, one row of nb_max each
enum Coef { C_CA_F = 0, C_CB_F, C_CV_F, C_CX, C_CW, C_CA_A, C_CB_A, C_CT_A, C_W2, C_ONE, C_LAM, C_NLAM, C_MONE, N_COEF };
// per-column double state, one row of nb_max each
// (S_VA.. S_XA: the source-weight entries of V, W, X in the source-free system, re/im pairs;
//  V's entry is stored un-normalised like V itself)
enum Stat { S_ALPHA = 0, S_BETA, S_RHOBAR, S_PHIBAR, S_AR0,
            S_VA_RE, S_VA_IM, S_WA_RE, S_WA_IM, S_XA_RE, S_XA_IM, N_STAT };

// ---------------------------------------------------------------------------------------------
// Persistent pass kernel (wri_pass.cuh): tile plan per working width and the device-resident state
// of the solve in flight.
constexpr int RT_NT = 512;            // consumer threads (one 16-byte item each)
constexpr int RT_MAXW = 64;           // widest column chunk (and widest working set that can be compacted)
constexpr int RT_MAX_STAGES = 12;
constexpr int RT_SMEM_MAX = 232448 - 1024;  // 227 KB of shared memory per CTA, less the static part
constexpr int RT_MIN_STAGE_AREA = 20480;   // the CTA epilogue re-uses the (idle) stages as scratch
constexpr int RT_G_SCRATCH = (RT_NT / 32) * 4 * 32 * 4 + 16;   // gradient pass: four planes of terms per consumer warp

enum StencilKind { ST_7 = 0, ST_27 = 1 };
enum MapSlot { MP_V_HALO = 0, MP_U_CTR, MP_W_CTR, MP_X_CTR, MP_U_HALO, MP_V_CTR, N_MAPS };

struct PassGeo {          // per pass: planes per tile, tile count, ring depth
    int zc, ntz, n_tiles, nstage;
};

struct DevPlan {          // tile geometry of one working width
    int nb, cb, hp, nchunk;           // batch width, column chunk, column pairs per chunk, chunks per cell
    int txc, tyc, items;              // cells per tile (x, y); consumer threads with work = txc*tyc*hp
    int ntx, nty;
    int merged, m_tma;                // tensor maps fold (column, x); the model tile rides in the stage
    int f_m_ldg, pad0;                // ... except in pass F (plain loads there)
    int row_b, cell_b;                // bytes per row / per cell of the halo box in shared memory
    int in_bytes, in_span;            // halo box: bytes delivered, room taken (128 B granules)
    int ctr_bytes, ctr_span;          // centre box
    int m_bytes, m_span;              // model tile (float per cell)
    PassGeo f, a;
};

struct SolveState {       // device-resident state of the solve in flight
    int widx, nb, k, n_active;
    int all_done, parity, pending, pending_widx;   // pending: iteration whose passes re-pack the set (0: none)
    // pending re-packing of the working set (decided by the finaliser of pass A, carried out by the
    // two passes of the next iteration, see k_pass_rt):
    int map[RT_MAXW];                 // new column j <- old column map[j] (-1 = padding)
    int dest[RT_MAXW];                // old column c -> new column (>= 0); -1: c leaves; <= -2: c leaves and its
                                      // threads zero-fill the padding column -2 - dest[c] of the new set
    int ret_dst[RT_MAXW];             // old column c -> caller's column that receives its final x (-1: none)
    int colmap[2][RT_MAXW];           // per parity: working column -> caller's column (-1 = padding)
};

struct PassParams {
    const float2* in;      // stencil input [n_g][nb]
    float2* out;           // result; also the "old" vector of the axpy (in place)
    float2* W;             // MODE_F only
    float2* X;             // MODE_F only
    const float* m;        // [n_g] squared slowness
    const float* gx;       // [nx] sponge profile per axis, gamma = max(gx,gy,gz)
    const float* gy;
    const float* gz;
    const float* w2;       // [nb] omega^2 per column
    const float* ca;       // [nb] scale of the operator term (includes lambda)
    const float* cb;       // [nb] scale of the old vector
    const float* cv;       // [nb] MODE_F: scale of V in the w update
    const float* cx;       // [nb] MODE_F
    const float* cw;       // [nb] MODE_F
    double* partials;      // [n_tiles][nb] squared-norm partial sums
    int nx, ny, nz, nb;
    int zc;                // planes per tile
    float ih2;             // 1/h^2
    float m6ih2;           // centre weight a0/h^2 (-6/h^2 for the 7-point stencil)
    float a1, a2, a3;      // 27-point stencil: weights of the face / edge / corner neighbours (units of 1/h^2)
    float sgn;             // +1: A, -1: A^H (conjugated diagonal)
};

template <int VEC> struct CV { float2 a[VEC]; };

template <int VEC> __device__ __forceinline__ CV<VEC> ldg_ro(const float2* p);
template <> __device__ __forceinline__ CV<1> ldg_ro<1>(const float2* p) {
    CV<1> r; r.a[0] = __ldg(p); return r;
}
template <> __device__ __forceinline__ CV<2> ldg_ro<2>(const float2* p) {
    float4 t = __ldg(reinterpret_cast<const float4*>(p));
    CV<2> r; r.a[0] = make_float2(t.x, t.y); r.a[1] = make_float2(t.z, t.w); return r;
}
// streaming load of data that is read once and rewritten in place
template <int VEC> __device__ __forceinline__ CV<VEC> ld_rw(const float2* p);
template <> __device__ __forceinline__ CV<1> ld_rw<1>(const float2* p) {
    CV<1> r; r.a[0] = __ldcs(p); return r;
}
template <> __device__ __forceinline__ CV<2> ld_rw<2>(const float2* p) {
    float4 t = __ldcs(reinterpret_cast<const float4*>(p));
    CV<2> r; r.a[0] = make_float2(t.x, t.y); r.a[1] = make_float2(t.z, t.w); return r;
}
template <int VEC> __device__ __forceinline__ void st_v(float2* p, const CV<VEC>& v);
template <> __device__ __forceinline__ void st_v<1>(float2* p, const CV<1>& v) { *p = v.a[0]; }
template <> __device__ __forceinline__ void st_v<2>(float2* p, const CV<2>& v) {
    *reinterpret_cast<float4*>(p) = make_float4(v.a[0].x, v.a[0].y, v.a[1].x, v.a[1].y);
}
template <int VEC> __device__ __forceinline__ CV<VEC> zero_v() {
    CV<VEC> r;
#pragma unroll
    for (int k = 0; k < VEC; ++k) r.a[k] = make_float2(0.f, 0.f);
    return r;
}

// Block-level, fixed-order reduction of per-thread column sums into partials[tile][0..nb).
// Slot (ty, tx, k) holds column (col0 + tx*VEC + k) % nb; thread j sums the slots of column j
// in increasing (ty, position) order, so the result does not depend on scheduling.
template <int VEC>
__device__ __forceinline__ void block_column_sums(const double (&acc)[VEC], int col0, int nb,
                                                  double* __restrict__ dst) {
    extern __shared__ double red[];
    const int TX = blockDim.x, TY = blockDim.y;
    const int slot = (threadIdx.y * TX + threadIdx.x) * VEC;
#pragma unroll
    for (int k = 0; k < VEC; ++k) red[slot + k] = acc[k];
    __syncthreads();
    const int width = TX * VEC;
    const int tid = threadIdx.y * TX + threadIdx.x;
    for (int j = tid; j < nb; j += TX * TY) {
        int t0 = j - col0;
        if (t0 < 0) t0 += nb;
        double s = 0.0;
        for (int ty = 0; ty < TY; ++ty)
            for (int t = t0; t < width; t += nb) s += red[ty * width + t];
        dst[j] = s;
    }
}


// 27-point stencil (generic kernels): weighted sum of the 26 neighbours of one cell for VEC columns,
// a1 * faces + a2 * edges + a3 * corners, zero outside the grid.  Plain loads through L1/L2 — the
// generic kernels are the fallback path; the persistent pass kernel keeps the planes in registers.
template <int VEC>
__device__ __forceinline__ void nbr27(const float2* __restrict__ in, size_t off, int nb, int RL, size_t plane,
                                      int ix, int iy, int iz, int nx, int ny, int nz, float a1, float a2, float a3,
                                      float (&sr)[VEC], float (&si)[VEC]) {
    float cr[3][VEC], ci[3][VEC];
#pragma unroll
    for (int q = 0; q < 3; ++q)
#pragma unroll
        for (int k = 0; k < VEC; ++k) cr[q][k] = ci[q][k] = 0.f;
    for (int dz = -1; dz <= 1; ++dz) {
        if (iz + dz < 0 || iz + dz >= nz) continue;
        for (int dy = -1; dy <= 1; ++dy) {
            if (iy + dy < 0 || iy + dy >= ny) continue;
            for (int dx = -1; dx <= 1; ++dx) {
                if (ix + dx < 0 || ix + dx >= nx) continue;
                const int cls = (dx != 0) + (dy != 0) + (dz != 0);
                if (cls == 0) continue;
                const long long o = (long long)off + dz * (long long)plane + dy * (long long)RL + dx * (long long)nb;
                const CV<VEC> v = ldg_ro<VEC>(in + o);
#pragma unroll
                for (int k = 0; k < VEC; ++k) { cr[cls - 1][k] += v.a[k].x; ci[cls - 1][k] += v.a[k].y; }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < VEC; ++k) {
        sr[k] = fmaf(a1, cr[0][k], fmaf(a2, cr[1][k], a3 * cr[2][k]));
        si[k] = fmaf(a1, ci[0][k], fmaf(a2, ci[1][k], a3 * ci[2][k]));
    }
}

template <int VEC, int MODE, int STENCIL>
__global__ void __launch_bounds__(256)
k_pass(const PassParams p) {
    const int nb = p.nb;
    const int RL = p.nx * nb;                               // complex elements per x-row
    const int e0 = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    const int iy = blockIdx.y * blockDim.y + threadIdx.y;
    const int z0 = blockIdx.z * p.zc;
    const int z1 = min(z0 + p.zc, p.nz);
    const bool live = (e0 < RL) && (iy < p.ny);
    const int col0 = (int)(((long long)blockIdx.x * blockDim.x * VEC) % nb);

    double acc[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) acc[k] = 0.0;

    if (live) {
        const int ix = e0 / nb;
        const int s0 = e0 - ix * nb;
        float w2[VEC], ca[VEC], cb[VEC], cv[VEC], cx[VEC], cw[VEC];
#pragma unroll
        for (int k = 0; k < VEC; ++k) {
            w2[k] = p.w2[s0 + k];
            ca[k] = p.ca[s0 + k];
            cb[k] = (MODE == MODE_A || MODE == MODE_F) ? p.cb[s0 + k] : 0.f;
            cv[k] = (MODE == MODE_F) ? p.cv[s0 + k] : 0.f;
            cx[k] = (MODE == MODE_F) ? p.cx[s0 + k] : 0.f;
            cw[k] = (MODE == MODE_F) ? p.cw[s0 + k] : 0.f;
        }
        const bool has_xm = ix > 0, has_xp = ix < p.nx - 1;
        const bool has_ym = iy > 0, has_yp = iy < p.ny - 1;
        const size_t plane = (size_t)RL * p.ny;
        const float gxy = fmaxf(p.gx[ix], p.gy[iy]);

        size_t off = ((size_t)z0 * p.ny + iy) * RL + e0;
        size_t moff = ((size_t)z0 * p.ny + iy) * p.nx + ix;
        CV<VEC> prev = zero_v<VEC>(), cur, nxt;
        cur = ldg_ro<VEC>(p.in + off);
        if (MODE != MODE_INIT && z0 > 0) prev = ldg_ro<VEC>(p.in + off - plane);

#pragma unroll 1
        for (int z = z0; z < z1; ++z) {
            nxt = zero_v<VEC>();
            if (z + 1 < p.nz && (MODE != MODE_INIT || z + 1 < z1)) nxt = ldg_ro<VEC>(p.in + off + plane);
            CV<VEC> r;
            if (MODE != MODE_INIT) {
                CV<VEC> xm = zero_v<VEC>(), xp = zero_v<VEC>(), ym = zero_v<VEC>(), yp = zero_v<VEC>();
                float s27r[VEC], s27i[VEC];
                if (STENCIL == ST_27) {
                    nbr27<VEC>(p.in, off, nb, RL, plane, ix, iy, z, p.nx, p.ny, p.nz, p.a1, p.a2, p.a3, s27r, s27i);
                } else {
                    if (has_xm) xm = ldg_ro<VEC>(p.in + off - nb);
                    if (has_xp) xp = ldg_ro<VEC>(p.in + off + nb);
                    if (has_ym) ym = ldg_ro<VEC>(p.in + off - RL);
                    if (has_yp) yp = ldg_ro<VEC>(p.in + off + RL);
                }
                CV<VEC> old, wv, xv;
                if (MODE == MODE_A || MODE == MODE_F) old = ld_rw<VEC>(p.out + off);
                if (MODE == MODE_F) { wv = ld_rw<VEC>(p.W + off); xv = ld_rw<VEC>(p.X + off); }
                const float mc = __ldg(p.m + moff);
                const float g = fmaxf(gxy, p.gz[z]);
#pragma unroll
                for (int k = 0; k < VEC; ++k) {
                    const float wm = w2[k] * mc;
                    const float dr = wm + p.m6ih2;          // Re diag = -6/h^2 + w^2 m
                    const float di = p.sgn * wm * g;        // Im diag = +-w^2 m gamma
                    const float sr = (STENCIL == ST_27) ? s27r[k]
                        : ((xm.a[k].x + xp.a[k].x) + (ym.a[k].x + yp.a[k].x)) + (prev.a[k].x + nxt.a[k].x);
                    const float si = (STENCIL == ST_27) ? s27i[k]
                        : ((xm.a[k].y + xp.a[k].y) + (ym.a[k].y + yp.a[k].y)) + (prev.a[k].y + nxt.a[k].y);
                    float ar = fmaf(p.ih2, sr, fmaf(dr, cur.a[k].x, -di * cur.a[k].y));
                    float ai = fmaf(p.ih2, si, fmaf(dr, cur.a[k].y, di * cur.a[k].x));
                    if (MODE == MODE_A || MODE == MODE_F) {
                        ar = fmaf(ca[k], ar, -cb[k] * old.a[k].x);
                        ai = fmaf(ca[k], ai, -cb[k] * old.a[k].y);
                    } else {
                        ar *= ca[k]; ai *= ca[k];
                    }
                    r.a[k] = make_float2(ar, ai);
                    if (MODE == MODE_F) {
                        xv.a[k].x = fmaf(cx[k], wv.a[k].x, xv.a[k].x);
                        xv.a[k].y = fmaf(cx[k], wv.a[k].y, xv.a[k].y);
                        wv.a[k].x = fmaf(cv[k], cur.a[k].x, -cw[k] * wv.a[k].x);
                        wv.a[k].y = fmaf(cv[k], cur.a[k].y, -cw[k] * wv.a[k].y);
                    }
                }
                if (MODE == MODE_F) { st_v<VEC>(p.X + off, xv); st_v<VEC>(p.W + off, wv); }
            } else {
#pragma unroll
                for (int k = 0; k < VEC; ++k)
                    r.a[k] = make_float2(ca[k] * cur.a[k].x, ca[k] * cur.a[k].y);
            }
            st_v<VEC>(p.out + off, r);
            if (MODE != MODE_APPLY) {
#pragma unroll
                for (int k = 0; k < VEC; ++k)
                    acc[k] += (double)fmaf(r.a[k].x, r.a[k].x, r.a[k].y * r.a[k].y);
            }
            prev = cur; cur = nxt;
            off += plane;
            moff += (size_t)p.nx * p.ny;
        }
    }
    if (MODE != MODE_APPLY) {
        const size_t tile = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
        block_column_sums<VEC>(acc, col0, nb, p.partials + tile * nb);
    }
}

// ---------------------------------------------------------------------------------------------
// Receiver rows (P and P^T are exact indexing).

// Per-source receiver sets P_s ("P_i"): rmask[r][s] = 1 when receiver r records column s,
// 0 when that row is absent from P_s (its entry of P_s v is 0 and its datum is ignored); null = all.
// ybot[r][s] = x[rec[r]][s]            (bit-exact copy)
__global__ void k_gather(const float2* __restrict__ x, const int* __restrict__ rec, int n_rec, int nb,
                         float2* __restrict__ ybot, const unsigned char* __restrict__ rmask) {
    const long long n = (long long)n_rec * nb;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(i / nb), s = (int)(i - (long long)r * nb);
        ybot[i] = (!rmask || rmask[i]) ? x[(size_t)rec[r] * nb + s] : make_float2(0.f, 0.f);
    }
}

// x[rec[r]][s] += ybot[r][s]           (receivers are unique, so this is race-free)
__global__ void k_scatter_add(float2* __restrict__ x, const int* __restrict__ rec, int n_rec, int nb,
                              const float2* __restrict__ ybot, const unsigned char* __restrict__ rmask) {
    const long long n = (long long)n_rec * nb;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const int r = (int)(i / nb), s = (int)(i - (long long)r * nb);
        if (rmask && !rmask[i]) continue;
        float2* d = x + (size_t)rec[r] * nb + s;
        const float2 a = *d, b = ybot[i];
        *d = make_float2(a.x + b.x, a.y + b.y);
    }
}

// Source column of S = [lambda A, -lambda e; P, 0] (eq. 6), one entry per batch column:
//   forward : ytop[src[s]][s] -= lambda * a[s]            (after ytop = lambda A x)
//   adjoint : xa[s] = -lambda * ytop[src[s]][s]           (e is a real unit vector)
__global__ void k_src_forward(float2* __restrict__ ytop, const int* __restrict__ src, int nb, float lambda,
                              const float2* __restrict__ a) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < nb) {
        float2* y = ytop + (size_t)src[s] * nb + s;
        const float2 t = *y, as = a[s];
        *y = make_float2(fmaf(-lambda, as.x, t.x), fmaf(-lambda, as.y, t.y));
    }
}
__global__ void k_src_adjoint(const float2* __restrict__ ytop, const int* __restrict__ src, int nb, float lambda,
                              float2* __restrict__ xa) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s < nb) {
        const float2 t = ytop[(size_t)src[s] * nb + s];
        xa[s] = make_float2(-lambda * t.x, -lambda * t.y);
    }
}

// ---------------------------------------------------------------------------------------------
// Per-column scalar recurrences + receiver rows, one block.  Phases:
enum ScalPhase { PH_INIT_B = 0, PH_INIT_A = 1, PH_F = 2, PH_A = 3 };

struct ScalParams {
    const double* partials;   // [n_tiles][nb]
    int n_tiles;
    int nb, nb_max;
    int n_rec;
    const int* rec;           // [n_rec] cell indices
    float2* V;                // [n_g][nb]
    float2* U_bot;            // [n_rec][nb]
    const float2* d;          // PH_INIT_B: data rows [n_rec][nb]
    float* coef;              // [N_COEF][nb_max]
    double* stat;             // [N_STAT][nb_max]
    int* active;              // [nb]
    int* iters;               // [nb]
    const float* tol;         // [nb] or null
    float* resnorms;          // [maxit+1][nb]
    int* iters_out;           // [nb] or null
    // paced enqueue (entries that end with a stream synchronisation): the finaliser of pass A reports
    // (solve id, iteration, every column stopped) in one 8-byte word of mapped host memory; null otherwise
    unsigned long long* progress;
    unsigned int solve_id;
    int k;                    // iteration number (PH_A), for resnorms / iters
    int maxit;
    float lambda;
    int rows_in_pass;         // 1: the pass kernels own the receiver rows (wri_pass.cuh); the
                              //    finaliser only reduces partials and runs the recurrences
    const int* colmap;        // [nb] working column -> caller's column (-1 = padding); null = identity
    int nb_out;               // caller's batch width: row stride of resnorms
    // source-free system S = [lambda A, -lambda e; P, 0]: one more unknown per column
    const int* src;           // [nb_out] source cell of the CALLER's column, or null (known-source system)
    float2* U;                // [n_g][nb] top rows of u (its source-node entry takes the -lambda e column)
    float2* alpha_out;        // [nb_out] source-weight estimate of x_k, c64
    // warm start (x0 in X / alpha_out on entry) and the reference of the stop rule
    int warm;
    const float2* X;          // [n_g][nb] x0 (PH_INIT_B: receiver rows of the residual)
    const double* ar_ref;     // [nb] or null: arnorm_k <= tol * ar_ref instead of tol * alpha1 beta1
    double* ar0_out;          // [nb] or null: alpha1 beta1 of this solve
    const unsigned char* rmask;   // [n_rec][nb_out] per-source receiver sets by the CALLER's column, or null
    // device-resident solve state (persistent pass kernel): iteration counter, active count, the
    // decision to re-pack the working set (PH_A)
    SolveState* st;           // null: host-sequenced solve (generic kernels)
    int adaptive;             // PH_A may ask for a re-packing of the working set
    int widx;                 // index of the current width's plan
    // PH_A of an iteration whose passes re-packed the vectors (trans): the finaliser moves the
    // per-column state to the other bank and switches the solve state over
    int trans;
    int nb_new;               // width of the new working set
    float* coef2; double* stat2; int* active2; int* iters2;   // the other bank
    float2* U_bot2;
    int* retired;             // [nb_out] by the CALLER's column: its final x sits in the side buffer (adaptive solves)
    int init_rows;            // PH_INIT_B: k_init_rows has formed U_bot; its |.|^2 sums are extra rows of partials
};

// sum over tiles of partials[.][s] in fixed order; result for column s in colsum[s] (shared).
// Runs while every other SM waits (last CTA of a pass), so the loads are issued four at a time and the
// groups are folded in two levels (groups of 8, then those): the longest dependent chain is
// n_tiles / Gc / 4 load rounds + Gc / 8 + 8 additions instead of n_tiles / Gc + Gc.
__device__ __forceinline__ void reduce_partials(const ScalParams& p, double* scratch, double* colsum) {
    const int nb = p.nb, T = blockDim.x;
    for (int base = 0; base < nb; base += T) {           // nb > T handled in column chunks
        const int ncol = min(nb - base, T);
        const int g = threadIdx.x / ncol, cl = threadIdx.x % ncol, s = base + cl;
        const int Gc = max(1, T / ncol);
        double a = 0.0;
        if (g < Gc) {
            int b = g;
            for (; b + 7 * Gc < p.n_tiles; b += 8 * Gc) {           // 8 loads in flight, added in order
                double t[8];
#pragma unroll
                for (int j = 0; j < 8; ++j) t[j] = __ldcg(p.partials + (size_t)(b + j * Gc) * nb + s);
#pragma unroll
                for (int j = 0; j < 8; ++j) a += t[j];
            }
            for (; b < p.n_tiles; b += 4 * Gc) {                     // the rest, still four at a time
                double t[4];
#pragma unroll
                for (int j = 0; j < 4; ++j)
                    t[j] = (b + j * Gc < p.n_tiles) ? __ldcg(p.partials + (size_t)(b + j * Gc) * nb + s) : 0.0;
#pragma unroll
                for (int j = 0; j < 4; ++j) a += t[j];
            }
        }
        scratch[threadIdx.x] = a;
        __syncthreads();
        int ng = Gc;                                                 // groups left to fold
        if (Gc > 8) {
            const int h = threadIdx.x / ncol;                        // thread (h, cl), h < 8: groups h, h + 8, ...
            double t = 0.0;
            if (h < 8)
                for (int gg = h; gg < Gc; gg += 8) t += scratch[gg * ncol + cl];
            __syncthreads();
            if (h < 8) scratch[h * ncol + cl] = t;
            __syncthreads();
            ng = 8;
        }
        if (threadIdx.x < ncol) {
            double t = 0.0;
            for (int gg = 0; gg < ng; ++gg) t += scratch[gg * ncol + threadIdx.x];
            colsum[base + threadIdx.x] = t;
        }
        __syncthreads();
    }
}

// fixed-order sum over receivers of |U_bot[r][s]|^2, added to colsum[s]
__device__ __forceinline__ void add_receiver_norms(const ScalParams& p, double* scratch, double* colsum) {
    const int nb = p.nb, T = blockDim.x;
    for (int base = 0; base < nb; base += T) {
        const int ncol = min(nb - base, T);
        const int Gc = max(1, T / ncol);
        const int g = threadIdx.x / ncol, s = base + threadIdx.x % ncol;
        double a = 0.0;
        if (g < Gc)
            for (int r = g; r < p.n_rec; r += Gc) {
                const float2 u = p.U_bot[(size_t)r * nb + s];
                a += (double)fmaf(u.x, u.x, u.y * u.y);
            }
        scratch[threadIdx.x] = a;
        __syncthreads();
        if (threadIdx.x < ncol) {
            double t = 0.0;
            for (int gg = 0; gg < Gc; ++gg) t += scratch[gg * ncol + threadIdx.x];
            colsum[base + threadIdx.x] += t;
        }
        __syncthreads();
    }
}

// Runs in ONE block (any size): the standalone k_scalars kernel, or the last CTA of the
// persistent pass kernel.  sh: (blockDim.x + nb) doubles of shared memory.
template <int PHASE>
__device__ __forceinline__ void finalize_phase(const ScalParams& p, double* sh) {
    double* scratch = sh;                   // [blockDim.x]
    double* colsum = sh + blockDim.x;       // [nb]
    const int nb = p.nb, NM = p.nb_max;
    float* cf = p.coef;
    double* st = p.stat;

    // The per-column state is needed after the partial sums have been folded; asking for it now lets
    // those trips to L2 overlap (this code runs in one CTA while the rest of the grid has finished).
    if ((PHASE == PH_F || PHASE == PH_A) && threadIdx.x < nb) {
        const int s = threadIdx.x;
        auto pf = [](const void* a) { asm volatile("prefetch.global.L1 [%0];" ::"l"(a)); };
        pf(p.active + s);
        if (p.colmap) pf(p.colmap + s);
        if (p.tol) pf(p.tol + s);
#pragma unroll
        for (int r = S_ALPHA; r <= S_AR0; ++r) pf(st + r * NM + s);
        if (p.src) pf(st + S_VA_RE * NM + s);
        pf(cf + (PHASE == PH_F ? C_CA_F : C_CA_A) * NM + s);
    }

    const long long nrs = (long long)p.n_rec * nb;
    if (PHASE == PH_INIT_B && !p.init_rows) {
        // U_bot = d (exact copy), then beta1 = ||[lambda q ; d]||
        // (d is the CALLER's [n_rec][nb_out] array: a grouped solve works on a subset of its columns)
        for (long long i = threadIdx.x; i < nrs; i += blockDim.x) {
            const int r = (int)(i / nb), s = (int)(i - (long long)r * nb);
            const int so = p.colmap ? p.colmap[s] : s;
            float2 dv = so >= 0 ? p.d[(size_t)r * p.nb_out + so] : make_float2(0.f, 0.f);
            if (p.warm) {
                // warm start: bottom rows of r0 = b - S x0, i.e. d - x0 at the receiver nodes
                const float2 xv = p.X[(size_t)p.rec[r] * nb + s];
                dv = make_float2(dv.x - xv.x, dv.y - xv.y);
            }
            if (p.rmask && so >= 0 && !p.rmask[(size_t)r * p.nb_out + so]) dv = make_float2(0.f, 0.f);
            p.U_bot[i] = dv;
        }
        __syncthreads();
    }
    if (PHASE == PH_F && !p.rows_in_pass) {
        // bottom rows of the forward pass just done:  U_bot <- cv * V[rec] - cb * U_bot
        for (long long i = threadIdx.x; i < nrs; i += blockDim.x) {
            const int r = (int)(i / nb), s = (int)(i - (long long)r * nb);
            const float cv = cf[C_CV_F * NM + s], cb = cf[C_CB_F * NM + s];
            const float2 v = p.V[(size_t)p.rec[r] * nb + s];
            const float2 u = p.U_bot[i];
            const int so = p.colmap ? p.colmap[s] : s;
            const bool on = !p.rmask || so < 0 || p.rmask[(size_t)r * p.nb_out + so];
            p.U_bot[i] = on ? make_float2(fmaf(cv, v.x, -cb * u.x), fmaf(cv, v.y, -cb * u.y)) : make_float2(0.f, 0.f);
        }
        __syncthreads();
    }
    reduce_partials(p, scratch, colsum);
    if ((PHASE == PH_INIT_B && !p.init_rows) || (PHASE == PH_F && !p.rows_in_pass)) add_receiver_norms(p, scratch, colsum);

    for (int s = threadIdx.x; s < nb; s += blockDim.x) {
        const int so = p.colmap ? p.colmap[s] : s;           // caller's column of working column s
        const int sc = (p.src && so >= 0) ? p.src[so] : -1;  // source cell (source-free system) or -1
        double cs = colsum[s];
        if (sc >= 0 && PHASE != PH_INIT_B && p.active[s]) {
            // the extra column -lambda e of S and its row of S^H (one entry per column):
            double va_re = st[S_VA_RE * NM + s], va_im = st[S_VA_IM * NM + s];
            float2* up = p.U + (size_t)sc * nb + s;
            const float2 o = __ldcg(up);
            if (PHASE == PH_F) {
                // u_top[src] -= (lambda/alpha) v_a ; the squared norm follows by the difference
                const double ca = (double)cf[C_CA_F * NM + s];
                const float2 n = make_float2((float)((double)o.x - ca * va_re), (float)((double)o.y - ca * va_im));
                *up = n;
                cs += ((double)n.x * n.x + (double)n.y * n.y) - ((double)o.x * o.x + (double)o.y * o.y);
            } else {
                // v_a <- -(lambda/beta) u_top[src] - (beta/alpha) v_a  (first pass: old v_a = 0)
                const double ca = (double)cf[C_CA_A * NM + s], cb = (double)cf[C_CB_A * NM + s];
                va_re = -ca * (double)o.x - cb * va_re;
                va_im = -ca * (double)o.y - cb * va_im;
                st[S_VA_RE * NM + s] = va_re; st[S_VA_IM * NM + s] = va_im;
                cs += va_re * va_re + va_im * va_im;
            }
        }
        if (PHASE == PH_INIT_B) {
            for (int r = S_VA_RE; r <= S_XA_IM; ++r) st[r * NM + s] = 0.0;
            if (p.alpha_out && !p.warm && so >= 0) p.alpha_out[so] = make_float2(0.f, 0.f);
            if (p.warm && sc >= 0) {
                // r0_top = lam q - lam (A x0 - a0 e): the pass before left lam q - lam A x0 in U
                const float2 a0 = p.alpha_out[so];
                st[S_XA_RE * NM + s] = (double)a0.x; st[S_XA_IM * NM + s] = (double)a0.y;
                float2* up = p.U + (size_t)sc * nb + s;
                const float2 o = __ldcg(up);
                const float2 n = make_float2((float)((double)o.x + (double)p.lambda * a0.x),
                                             (float)((double)o.y + (double)p.lambda * a0.y));
                *up = n;
                cs += ((double)n.x * n.x + (double)n.y * n.y) - ((double)o.x * o.x + (double)o.y * o.y);
            }
        }
        const double nrm = sqrt(fmax(cs, 0.0));
        if (PHASE == PH_INIT_B) {
            // beta1 u1 = b.  b = 0 => x = 0, nothing to iterate (reading C-7).
            const double beta = nrm;
            st[S_BETA * NM + s] = beta;
            st[S_PHIBAR * NM + s] = beta;
            st[S_ALPHA * NM + s] = 0.0;
            st[S_RHOBAR * NM + s] = 0.0;
            st[S_AR0 * NM + s] = 0.0;
            const int act = beta > 0.0;
            p.active[s] = act;
            p.iters[s] = 0;
            if (p.iters_out && so >= 0) p.iters_out[so] = 0;
            if (p.resnorms && so >= 0) p.resnorms[so] = (float)beta;
            // first adjoint pass: V = (lambda/beta) A^H U + (1/beta) P^T U_bot, old V = 0 with cb = 1
            cf[C_CA_A * NM + s] = act ? (float)((double)p.lambda / beta) : 0.f;
            cf[C_CT_A * NM + s] = act ? (float)(1.0 / beta) : 0.f;
            cf[C_CB_A * NM + s] = 1.f;
            cf[C_CX * NM + s] = 0.f;
            cf[C_CW * NM + s] = 0.f;
        } else if (PHASE == PH_INIT_A) {
            // alpha1 v1 = M^H u1 ; w1 = v1 ; phibar = beta1 ; rhobar = alpha1
            const double alpha = nrm, beta = st[S_BETA * NM + s];
            int act = p.active[s];
            st[S_ALPHA * NM + s] = alpha;
            st[S_RHOBAR * NM + s] = alpha;
            st[S_AR0 * NM + s] = (p.ar_ref && so >= 0 && p.ar_ref[so] > 0.0) ? p.ar_ref[so] : alpha * beta;
            if (p.ar0_out && so >= 0) p.ar0_out[so] = alpha * beta;
            if (act && !(alpha > 0.0)) { act = 0; p.active[s] = 0; }
            cf[C_CA_F * NM + s] = act ? (float)((double)p.lambda / alpha) : 0.f;
            cf[C_CV_F * NM + s] = act ? (float)(1.0 / alpha) : 0.f;
            cf[C_CB_F * NM + s] = act ? (float)(alpha / beta) : 0.f;
            if (sc >= 0) {                                    // w1 = v1, x0 = 0
                st[S_WA_RE * NM + s] = act ? st[S_VA_RE * NM + s] / alpha : 0.0;
                st[S_WA_IM * NM + s] = act ? st[S_VA_IM * NM + s] / alpha : 0.0;
            }
        } else if (PHASE == PH_F) {
            // beta_{k+1} = ||M v_k - alpha_k u_k||
            const int act = p.active[s];
            if (act) {
                const double beta = nrm, alpha = st[S_ALPHA * NM + s];
                st[S_BETA * NM + s] = beta;
                const bool ok = beta > 0.0;
                cf[C_CA_A * NM + s] = ok ? (float)((double)p.lambda / beta) : 0.f;
                cf[C_CT_A * NM + s] = ok ? (float)(1.0 / beta) : 0.f;
                cf[C_CB_A * NM + s] = ok ? (float)(beta / alpha) : 0.f;
            } else {
                cf[C_CA_A * NM + s] = 0.f; cf[C_CT_A * NM + s] = 0.f; cf[C_CB_A * NM + s] = 0.f;
                cf[C_CX * NM + s] = 0.f;          // a stopped column's last x update has been applied
            }
        } else {  // PH_A
            int act = p.active[s];
            if (act) {
                // alpha_{k+1} = ||M^H u_{k+1} - beta_{k+1} v_k||, then the plane rotation
                const double alpha = nrm, beta = st[S_BETA * NM + s];
                const double rhobar = st[S_RHOBAR * NM + s], phibar = st[S_PHIBAR * NM + s];
                const double rho = hypot(rhobar, beta);
                const double c = rhobar / rho, sn = beta / rho;
                const double theta = sn * alpha;
                const double phi = c * phibar;
                const double phibar_n = sn * phibar;
                st[S_ALPHA * NM + s] = alpha;
                st[S_RHOBAR * NM + s] = -c * alpha;
                st[S_PHIBAR * NM + s] = phibar_n;
                p.iters[s] = p.k;
                if (p.iters_out) p.iters_out[so] = p.k;
                const double arnorm = phibar_n * alpha * fabs(c);
                const float tol = p.tol ? p.tol[so] : 0.f;
                bool stop = !(beta > 0.0) || !(alpha > 0.0);
                if (tol > 0.f && arnorm <= (double)tol * st[S_AR0 * NM + s]) stop = true;
                cf[C_CX * NM + s] = (float)(phi / rho);
                if (sc >= 0) {
                    // the alpha entries of x and w are updated at once (the vectors' updates are
                    // deferred to the next pass F):  x_a += (phi/rho) w_a ; w_a = v_a/alpha - (theta/rho) w_a
                    const double t1 = phi / rho, t2 = theta / rho;
                    const double wr = st[S_WA_RE * NM + s], wi = st[S_WA_IM * NM + s];
                    const double xr = st[S_XA_RE * NM + s] + t1 * wr, xi = st[S_XA_IM * NM + s] + t1 * wi;
                    st[S_XA_RE * NM + s] = xr; st[S_XA_IM * NM + s] = xi;
                    if (!stop) {
                        st[S_WA_RE * NM + s] = st[S_VA_RE * NM + s] / alpha - t2 * wr;
                        st[S_WA_IM * NM + s] = st[S_VA_IM * NM + s] / alpha - t2 * wi;
                    }
                    if (p.alpha_out) p.alpha_out[so] = make_float2((float)xr, (float)xi);
                }
                if (stop) {
                    act = 0; p.active[s] = 0;
                    cf[C_CW * NM + s] = 0.f;
                    cf[C_CA_F * NM + s] = 0.f; cf[C_CV_F * NM + s] = 0.f; cf[C_CB_F * NM + s] = 0.f;
                } else {
                    cf[C_CW * NM + s] = (float)(theta / rho);
                    cf[C_CA_F * NM + s] = (float)((double)p.lambda / alpha);
                    cf[C_CV_F * NM + s] = (float)(1.0 / alpha);
                    cf[C_CB_F * NM + s] = (float)(alpha / beta);
                }
            } else {
                cf[C_CW * NM + s] = 0.f;
                cf[C_CA_F * NM + s] = 0.f; cf[C_CV_F * NM + s] = 0.f; cf[C_CB_F * NM + s] = 0.f;
            }
            if (so >= 0 && p.resnorms) p.resnorms[(size_t)p.k * p.nb_out + so] = (float)st[S_PHIBAR * NM + s];
        }
    }
    __syncthreads();

    if (PHASE == PH_A && p.st && threadIdx.x == 0) {
        // device-resident solve state: iteration count, live columns, and — with adaptive accuracy —
        // the decision to re-pack the working set.  Re-packing rides on the two passes of the next
        // iteration (they write their results at the new width, see k_pass_rt), so it costs one extra
        // write of U and nothing else: it is asked for as soon as the even width that holds the live
        // columns is narrower than the working set.
        SolveState* st = p.st;
        int n_act = 0;
        for (int s = 0; s < nb; ++s) n_act += p.active[s] != 0;
        st->k = p.k;
        st->n_active = n_act;
        if (p.progress) {
            *p.progress = ((unsigned long long)p.solve_id << 32) | ((unsigned long long)(unsigned)p.k << 1) |
                          (n_act == 0 ? 1ull : 0ull);
            __threadfence_system();
        }
        if (n_act == 0) st->all_done = 1;
        else if (p.adaptive && !p.trans) {
            const int w_new = max(2, (n_act + 1) & ~1);
            if (w_new < nb && p.k < p.maxit) {
                // order of the new set: first the old pairs (2i, 2i+1) whose columns both go on — they stay
                // aligned pairs, so the passes that re-pack store them with one 16-byte store per thread —,
                // then the columns that lost their partner, then (at most one) padding column, zero-filled
                // by the threads of a column that leaves
                int nk = 0;
                for (int s = 0; s < nb; ++s) {
                    st->dest[s] = -1;
                    st->ret_dst[s] = p.active[s] ? -1 : p.colmap[s];
                }
                for (int s = 0; s + 1 < nb; s += 2)
                    if (p.active[s] && p.active[s + 1]) {
                        st->map[nk] = s; st->dest[s] = nk; ++nk;
                        st->map[nk] = s + 1; st->dest[s + 1] = nk; ++nk;
                    }
                for (int s = 0; s < nb; ++s)
                    if (p.active[s] && st->dest[s] < 0) { st->map[nk] = s; st->dest[s] = nk; ++nk; }
                for (int s = 0, j = nk; s < nb && j < w_new; ++s)
                    if (!p.active[s]) { st->dest[s] = -2 - j; st->map[j] = -1; ++j; }
                st->pending_widx = p.widx + (nb - w_new) / 2;
                st->pending = p.k + 1;          // the passes of the next iteration re-pack
            }
        }
    }

    if (PHASE == PH_A && p.st && p.trans) {
        // This iteration's passes wrote U, V, W, X of the live columns into the other vector set at the
        // new width (and the final x of the leaving columns into the caller's u_out).  The per-column
        // state follows: scalars, receiver rows, column map; the residual history of the columns that
        // left is held at the stop value (reading C-9).  Then the solve state switches over.
        __syncthreads();
        SolveState* st = p.st;
        const int a = st->parity, nbn = p.nb_new;
        for (int j = threadIdx.x; j < nbn; j += blockDim.x) {
            const int m = st->map[j];
            for (int r = 0; r < N_COEF; ++r) p.coef2[r * NM + j] = m >= 0 ? cf[r * NM + m] : 0.f;
            for (int r = 0; r < N_STAT; ++r) p.stat2[r * NM + j] = m >= 0 ? p.stat[r * NM + m] : 0.0;
            p.active2[j] = m >= 0 ? p.active[m] : 0;
            p.iters2[j] = m >= 0 ? p.iters[m] : 0;
            st->colmap[a ^ 1][j] = m >= 0 ? st->colmap[a][m] : -1;
        }
        for (int j = nbn + threadIdx.x; j < RT_MAXW; j += blockDim.x) st->colmap[a ^ 1][j] = -1;
        for (long long i = threadIdx.x; i < (long long)p.n_rec * nbn; i += blockDim.x) {
            const long long r = i / nbn;
            const int m = st->map[(int)(i - r * nbn)];
            p.U_bot2[i] = m >= 0 ? p.U_bot[r * nb + m] : make_float2(0.f, 0.f);
        }
        for (int s = threadIdx.x; s < nb; s += blockDim.x)
            if (st->ret_dst[s] >= 0) p.retired[st->ret_dst[s]] = 1;
        if (p.resnorms)
            for (long long i = threadIdx.x; i < (long long)(p.maxit - p.k) * nb; i += blockDim.x) {
                const int row = (int)(i / nb), s = (int)(i - (long long)row * nb);
                const int so = st->ret_dst[s];
                if (so >= 0) p.resnorms[(size_t)(p.k + 1 + row) * p.nb_out + so] = (float)p.stat[S_PHIBAR * NM + s];
            }
        __syncthreads();
        if (threadIdx.x == 0) {
            st->parity = a ^ 1;
            st->widx = st->pending_widx;
            st->nb = nbn;
            st->pending = 0;
        }
    }

    if ((PHASE == PH_INIT_B || PHASE == PH_F) && !p.rows_in_pass) {
        // fold P^T into the coming adjoint pass:  V <- ca A^H U - cb (V - (ct/cb) P^T U_bot)
        for (long long i = threadIdx.x; i < nrs; i += blockDim.x) {
            const int r = (int)(i / nb), s = (int)(i - (long long)r * nb);
            const float cb = cf[C_CB_A * NM + s];
            if (cb != 0.f) {
                const float f = cf[C_CT_A * NM + s] / cb;
                const float2 u = p.U_bot[i];
                float2* v = p.V + (size_t)p.rec[r] * nb + s;
                float2 t = *v;
                t.x = fmaf(-f, u.x, t.x);
                t.y = fmaf(-f, u.y, t.y);
                *v = t;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Column gather for the start of a grouped solve (the re-packing of a shrinking working set during
// an adaptive solve rides on the pass kernels themselves, wri_pass.cuh).

// dst[c][j] = src[c][map[j]] (map[j] < 0 -> 0), widths nb_dst <= nb_src; dst and src are distinct buffers
__global__ void k_gather_cols(float2* __restrict__ dst, const float2* __restrict__ src,
                              const int* __restrict__ map, long long n_rows, int nb_dst, int nb_src) {
    const long long n = n_rows * nb_dst;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        const long long c = i / nb_dst;
        const int j = (int)(i - c * nb_dst);
        const int m = map[j];
        dst[i] = m >= 0 ? __ldcs(src + c * nb_src + m) : make_float2(0.f, 0.f);
    }
}

// Arguments shared by the kernels that move a solve's state around on the device.
struct MoveParams {
    SolveState* st;
    const DevPlan* plans;
    float2* vec[2][4];        // per parity: U, V, W, X
    float2* U_bot[2];
    float* coef[2];
    double* stat[2];
    int* active[2];
    int* iters[2];
    float2* u_out;            // caller's [n_g][nb_out]
    float* resnorms;          // caller's [maxit+1][nb_out] or null
    long long n_g;
    int nb_out, nb_max, maxit, n_rec;
    int packed;
    // adaptive solves: the final x of the columns that left the working set, column by column
    // ([caller's column][cell]), and which columns those are; this group's columns of the caller's batch
    const float2* R;
    const int* retired;
    int col0, ncols;
};

// End of a solve: the last deferred update x_k = X + cx W is applied and, where the working set has
// a column map (grouped / adaptive solves: X lives in the workspace), scattered to the caller's
// u_out; the residual history of the rows after the last iteration performed is held (reading C-9).
__global__ void __launch_bounds__(256)
k_finish(const MoveParams p) {
    const SolveState* st = p.st;
    __shared__ int s_cm[RT_MAXW];
    __shared__ float s_cx[RT_MAXW];
    const int a = st->parity, nb = st->nb, k = st->k;
    const size_t NM = p.nb_max;
    const float* cxr = p.coef[a] + C_CX * NM;
    const long long gs = (long long)gridDim.x * blockDim.x, g0 = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (p.packed) {
        if (threadIdx.x < RT_MAXW) {
            s_cm[threadIdx.x] = st->colmap[a][threadIdx.x];
            s_cx[threadIdx.x] = threadIdx.x < nb ? cxr[threadIdx.x] : 0.f;
        }
        __syncthreads();
        const float2* X = p.vec[a][3];
        const float2* W = p.vec[a][2];
        if (p.R) {
            // adaptive solve: the caller's rows are put together in shared memory, 32 cells at a time —
            // the columns still in the working set from X (+ cx W), the ones that left from the side
            // buffer (read along the cells) — and written as whole rows: full sectors both ways
            constexpr int CH = 32;
            __shared__ float2 tile[CH][RT_MAXW + 1];
            __shared__ int s_ok[RT_MAXW];
            const int ncols = p.ncols, col0 = p.col0;
            if (threadIdx.x < RT_MAXW) s_ok[threadIdx.x] = threadIdx.x < ncols && p.retired[col0 + threadIdx.x] ? 2 : 0;
            __syncthreads();
            if (threadIdx.x < nb && s_cm[threadIdx.x] >= 0) s_ok[s_cm[threadIdx.x] - col0] = 1;
            __syncthreads();
            for (long long c0 = (long long)blockIdx.x * CH; c0 < p.n_g; c0 += (long long)gridDim.x * CH) {
                const int nc = (int)min((long long)CH, p.n_g - c0);
                for (int idx = threadIdx.x; idx < nc * nb; idx += blockDim.x) {
                    const int c = idx / nb, j = idx - c * nb, so = s_cm[j];
                    if (so < 0) continue;
                    const long long i = (c0 + c) * nb + j;
                    float2 x = __ldcs(X + i);
                    const float cx = s_cx[j];
                    if (cx != 0.f) {
                        const float2 w = __ldcs(W + i);
                        x.x = fmaf(cx, w.x, x.x);
                        x.y = fmaf(cx, w.y, x.y);
                    }
                    tile[c][so - col0] = x;
                }
                for (int idx = threadIdx.x; idx < ncols * CH; idx += blockDim.x) {
                    const int jj = idx / CH, t = idx - jj * CH;
                    if (s_ok[jj] == 2 && t < nc) tile[t][jj] = __ldcs(p.R + (size_t)(col0 + jj) * p.n_g + c0 + t);
                }
                __syncthreads();
                for (int idx = threadIdx.x; idx < nc * ncols; idx += blockDim.x) {
                    const int c = idx / ncols, jj = idx - c * ncols;
                    if (s_ok[jj]) p.u_out[(c0 + c) * p.nb_out + col0 + jj] = tile[c][jj];
                }
                __syncthreads();
            }
        } else
        for (long long i = g0; i < p.n_g * nb; i += gs) {
            const long long c = i / nb;
            const int j = (int)(i - c * nb), so = s_cm[j];
            if (so < 0) continue;
            float2 x = __ldcs(X + i);
            const float cx = s_cx[j];
            if (cx != 0.f) {
                const float2 w = __ldcs(W + i);
                x.x = fmaf(cx, w.x, x.x);
                x.y = fmaf(cx, w.y, x.y);
            }
            p.u_out[c * p.nb_out + so] = x;
        }
    } else {
        float2* X = p.vec[a][3];                                 // = u_out, same layout
        const float2* W = p.vec[a][2];
        for (long long i = g0; i < p.n_g * nb; i += gs) {
            const float cx = cxr[(int)(i % nb)];
            if (cx != 0.f) {
                const float2 w = __ldcs(W + i);
                float2 x = X[i];
                x.x = fmaf(cx, w.x, x.x);
                x.y = fmaf(cx, w.y, x.y);
                X[i] = x;
            }
        }
    }
    if (p.resnorms)
        for (long long i = g0; i < (long long)(p.maxit - k) * nb; i += gs) {
            const int row = (int)(i / nb), j = (int)(i - (long long)row * nb);
            const int so = p.packed ? st->colmap[a][j] : j;
            if (so >= 0) p.resnorms[(size_t)(k + 1 + row) * p.nb_out + so] = (float)p.stat[a][S_PHIBAR * NM + j];
        }
}

// the pending x-update coefficients are spent once k_finish has run
__global__ void k_clear_cx(float* cx0, float* cx1, int n) {
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j < n) { cx0[j] = 0.f; cx1[j] = 0.f; }
}

// Golub-Kahan start, receiver rows of b = [lambda q ; d] spread over the blocks:  U_bot = d (exact
// copy; warm start: d - x0 at the receiver nodes; masked rows of per-source receiver sets = 0) and
// per-block column sums of |U_bot|^2 into rows n_rows0 + blockIdx.x of partials.  blockDim.x is a
// any size; thread (i, s): rows blockIdx.x + (i + j*rpb) * gridDim.x, column s.
__global__ void __launch_bounds__(256)
k_init_rows(const ScalParams p, double* __restrict__ partials, int n_rows0) {
    extern __shared__ double sh_rows[];                      // [blockDim.x]
    const int nb = p.nb, T = blockDim.x;
    for (int base = 0; base < nb; base += T) {
        const int ncol = min(nb - base, T);
        const int rpb = T / ncol;                            // rows in flight per block
        const int i = threadIdx.x / ncol, s = base + threadIdx.x % ncol;
        double a = 0.0;
        if (i < rpb) {
            const int so = p.colmap ? p.colmap[s] : s;
            for (int r = blockIdx.x + i * gridDim.x; r < p.n_rec; r += rpb * gridDim.x) {
                float2 dv = so >= 0 ? p.d[(size_t)r * p.nb_out + so] : make_float2(0.f, 0.f);
                if (p.warm) {
                    const float2 xv = p.X[(size_t)p.rec[r] * nb + s];
                    dv = make_float2(dv.x - xv.x, dv.y - xv.y);
                }
                if (p.rmask && so >= 0 && !p.rmask[(size_t)r * p.nb_out + so]) dv = make_float2(0.f, 0.f);
                p.U_bot[(size_t)r * nb + s] = dv;
                a += (double)fmaf(dv.x, dv.x, dv.y * dv.y);
            }
        }
        sh_rows[threadIdx.x] = a;
        __syncthreads();
        if (threadIdx.x < ncol) {
            double t = 0.0;
            for (int g = 0; g < rpb; ++g) t += sh_rows[g * ncol + threadIdx.x];
            partials[(size_t)(n_rows0 + blockIdx.x) * nb + base + threadIdx.x] = t;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------------------------------------
// Objective and gradient of the reduced problem (eq. 4, 98-110 eq. 8-9), at given
// wavefields u (and source weights):   r = A u - q - alpha e,
//   f_pde[s]  = 1/2 lambda^2 ||r_s||^2,   f_data[s] = 1/2 ||P u_s - d_s||^2,
//   g[c]     += sum_s lambda^2 omega_s^2 Re[ conj((1 + i gamma_c) u_cs) r_cs ]
// (eq. 9 with dA/dm_c = omega^2 (1 + i gamma_c) of this build's sponge; the sum over the batch
// columns is the paper's sum over sources and frequencies).  Same thread mapping and z march as
// k_pass; the threads of one cell are TPC = nb / VEC consecutive threads of a block row (the
// host makes blockDim.x a multiple of TPC), reduced in a fixed order — warp shuffles when TPC is
// a power of two <= 32, shared memory otherwise — so g is bit-reproducible.
struct GradParams {
    const float2* u;       // [n_g][nb]
    const float2* q;       // [n_g][nb] or null
    const int* src;        // [nb] source cells or null
    const float2* alpha;   // [nb] source weights (with src)
    const float* m;
    const float *gx, *gy, *gz;
    const float* w2;       // [nb]
    float* g;              // [n_g], accumulated; may be null
    double* partials;      // [n_tiles][nb] sums of |r|^2
    int nx, ny, nz, nb, zc;
    int tpc;               // threads per cell
    int shuffle;           // 1: tpc is a power of two <= 32
    float ih2, m6ih2, lam2;
    float a1, a2, a3;      // 27-point stencil weights (see PassParams)
};

template <int VEC, int STENCIL>
__global__ void __launch_bounds__(512)
k_grad(const GradParams p) {
    extern __shared__ double red[];                          // block_column_sums scratch; reused per plane
    const int nb = p.nb;
    const int RL = p.nx * nb;
    const int e0 = (blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    const int iy = blockIdx.y * blockDim.y + threadIdx.y;
    const int z0 = blockIdx.z * p.zc;
    const int z1 = min(z0 + p.zc, p.nz);
    const bool live = (e0 < RL) && (iy < p.ny);
    const int tlin = threadIdx.y * blockDim.x + threadIdx.x;
    float* gsm = reinterpret_cast<float*>(red);              // [blockDim.x * blockDim.y] per-thread g terms

    double acc[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) acc[k] = 0.0;

    const int ix = live ? e0 / nb : 0;
    const int s0 = live ? e0 - ix * nb : 0;
    float w2[VEC];
    int srcc[VEC];
    float2 al[VEC];
#pragma unroll
    for (int k = 0; k < VEC; ++k) {
        w2[k] = live ? p.w2[s0 + k] : 0.f;
        srcc[k] = (live && p.src) ? p.src[s0 + k] : -1;
        al[k] = (live && p.src) ? p.alpha[s0 + k] : make_float2(0.f, 0.f);
    }
    const bool has_xm = ix > 0, has_xp = ix < p.nx - 1;
    const bool has_ym = iy > 0, has_yp = iy < p.ny - 1;
    const size_t plane = (size_t)RL * p.ny;
    const float gxy = live ? fmaxf(p.gx[ix], p.gy[iy]) : 0.f;
    size_t off = live ? ((size_t)z0 * p.ny + iy) * RL + e0 : 0;
    size_t cell = live ? ((size_t)z0 * p.ny + iy) * p.nx + ix : 0;
    CV<VEC> prev = zero_v<VEC>(), cur = zero_v<VEC>(), nxt;
    if (live) {
        cur = ldg_ro<VEC>(p.u + off);
        if (z0 > 0) prev = ldg_ro<VEC>(p.u + off - plane);
    }

#pragma unroll 1
    for (int z = z0; z < z1; ++z) {
        float gterm = 0.f;
        if (live) {
            nxt = zero_v<VEC>();
            if (z + 1 < p.nz) nxt = ldg_ro<VEC>(p.u + off + plane);
            CV<VEC> xm = zero_v<VEC>(), xp = zero_v<VEC>(), ym = zero_v<VEC>(), yp = zero_v<VEC>();
            float s27r[VEC], s27i[VEC];
            if (STENCIL == ST_27) {
                nbr27<VEC>(p.u, off, nb, RL, plane, ix, iy, z, p.nx, p.ny, p.nz, p.a1, p.a2, p.a3, s27r, s27i);
            } else {
                if (has_xm) xm = ldg_ro<VEC>(p.u + off - nb);
                if (has_xp) xp = ldg_ro<VEC>(p.u + off + nb);
                if (has_ym) ym = ldg_ro<VEC>(p.u + off - RL);
                if (has_yp) yp = ldg_ro<VEC>(p.u + off + RL);
            }
            CV<VEC> qv = zero_v<VEC>();
            if (p.q) qv = ld_rw<VEC>(p.q + off);
            const float mc = __ldg(p.m + cell);
            const float gam = fmaxf(gxy, p.gz[z]);
#pragma unroll
            for (int k = 0; k < VEC; ++k) {
                const float wm = w2[k] * mc;
                const float dr = wm + p.m6ih2, di = wm * gam;
                const float sr = (STENCIL == ST_27) ? s27r[k]
                    : ((xm.a[k].x + xp.a[k].x) + (ym.a[k].x + yp.a[k].x)) + (prev.a[k].x + nxt.a[k].x);
                const float si = (STENCIL == ST_27) ? s27i[k]
                    : ((xm.a[k].y + xp.a[k].y) + (ym.a[k].y + yp.a[k].y)) + (prev.a[k].y + nxt.a[k].y);
                float rr = fmaf(p.ih2, sr, fmaf(dr, cur.a[k].x, -di * cur.a[k].y)) - qv.a[k].x;
                float ri = fmaf(p.ih2, si, fmaf(dr, cur.a[k].y, di * cur.a[k].x)) - qv.a[k].y;
                if ((int)cell == srcc[k]) { rr -= al[k].x; ri -= al[k].y; }
                acc[k] += (double)fmaf(rr, rr, ri * ri);
                // Re[conj((1 + i gamma) u) r] = Re t + gamma Im t,  t = conj(u) r
                const float tr = fmaf(cur.a[k].x, rr, cur.a[k].y * ri);
                const float ti = fmaf(cur.a[k].x, ri, -cur.a[k].y * rr);
                gterm = fmaf(w2[k], fmaf(gam, ti, tr), gterm);
            }
            prev = cur; cur = nxt;
        }
        if (p.g) {
            if (p.shuffle) {
                for (int d = p.tpc >> 1; d > 0; d >>= 1) gterm += __shfl_down_sync(0xffffffffu, gterm, d, p.tpc);
                if (live && (threadIdx.x % p.tpc) == 0) p.g[cell] += p.lam2 * gterm;
            } else {
                gsm[tlin] = gterm;
                __syncthreads();
                if (live && (threadIdx.x % p.tpc) == 0) {
                    float t = 0.f;
                    for (int j = 0; j < p.tpc; ++j) t += gsm[tlin + j];
                    p.g[cell] += p.lam2 * t;
                }
                __syncthreads();
            }
        }
        off += plane;
        cell += (size_t)p.nx * p.ny;
    }
    const size_t tile = ((size_t)blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x;
    const int col0 = (int)(((long long)blockIdx.x * blockDim.x * VEC) % nb);
    __syncthreads();
    block_column_sums<VEC>(acc, col0, nb, p.partials + tile * nb);
}

// trial model of Algorithm 2 line 6 with the built-in steepest-descent update:
// m_trial = clamp(m - step * g, m_min, m_max)   (the l-BFGS direction is the caller's)
__global__ void k_model_step(float* __restrict__ m_trial, const float* __restrict__ m, const float* __restrict__ g,
                             float step, float m_min, float m_max, long long n) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x)
        m_trial[i] = fminf(fmaxf(fmaf(-step, g[i], m[i]), m_min), m_max);
}

// g += t[0] + t[1] + ...  (the batch's gradient from the pass kernel, one array per column chunk, added
// in chunk order into the caller's accumulated gradient)
__global__ void k_add_f32(float* __restrict__ g, const float* __restrict__ t, long long n, int nchunk) {
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
         i += (long long)gridDim.x * blockDim.x) {
        float a = t[i];
        for (int k = 1; k < nchunk; ++k) a += t[(size_t)k * n + i];
        g[i] += a;
    }
}

// f_pde[s] = 1/2 lambda^2 sum_tiles partials[.][s];  f_data[s] = 1/2 sum_r |u[rec_r][s] - d[r][s]|^2
// Block b owns OBJ_CPB consecutive columns (T / OBJ_CPB row groups each); fixed summation order.
constexpr int OBJ_CPB = 8;
__global__ void __launch_bounds__(1024)
k_objective(const double* __restrict__ partials, int n_tiles, int nb, const float2* __restrict__ u,
            const float2* __restrict__ d, const int* __restrict__ rec, int n_rec, double lam2,
            double* __restrict__ f_pde, double* __restrict__ f_data, const unsigned char* __restrict__ rmask) {
    extern __shared__ double sh_obj[];                       // [blockDim.x]
    const int T = blockDim.x;
    const int base = blockIdx.x * OBJ_CPB;
    const int ncol = min(nb - base, OBJ_CPB);
    const int Gc = T / OBJ_CPB;
    const int g = threadIdx.x / OBJ_CPB, cl = threadIdx.x % OBJ_CPB, s = base + cl;
    for (int pass = 0; pass < 2; ++pass) {
        double a = 0.0;
        if (cl < ncol) {
            if (pass == 0) {
                int b = g;
                for (; b + 7 * Gc < n_tiles; b += 8 * Gc) {          // 8 loads in flight, added in order
                    double t[8];
#pragma unroll
                    for (int j = 0; j < 8; ++j) t[j] = __ldcg(partials + (size_t)(b + j * Gc) * nb + s);
#pragma unroll
                    for (int j = 0; j < 8; ++j) a += t[j];
                }
                for (; b < n_tiles; b += Gc) a += __ldcg(partials + (size_t)b * nb + s);
            } else {
                for (int r = g; r < n_rec; r += Gc) {
                    if (rmask && !rmask[(size_t)r * nb + s]) continue;
                    const float2 uv = u[(size_t)rec[r] * nb + s], dv = d[(size_t)r * nb + s];
                    const double er = (double)uv.x - (double)dv.x, ei = (double)uv.y - (double)dv.y;
                    a += er * er + ei * ei;
                }
            }
        }
        sh_obj[threadIdx.x] = a;
        __syncthreads();
        if (threadIdx.x < ncol) {
            double t = 0.0;
            for (int gg = 0; gg < Gc; ++gg) t += sh_obj[gg * OBJ_CPB + threadIdx.x];
            if (pass == 0) f_pde[base + threadIdx.x] = 0.5 * lam2 * t;
            else f_data[base + threadIdx.x] = 0.5 * t;
        }
        __syncthreads();
    }
}

template <int PHASE>
__global__ void __launch_bounds__(1024)
k_scalars(const ScalParams p) {
    extern __shared__ double sh_scal[];
    finalize_phase<PHASE>(p, sh_scal);
}

}  // namespace wri
