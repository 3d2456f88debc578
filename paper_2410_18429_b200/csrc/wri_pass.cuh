// wri_pass.cuh — persistent, TMA-fed stencil + LSQR pass for sm_100a with the batch width as a
// RUN-TIME parameter (the hot kernel of libwri).
//
// One CTA per SM walks a fixed (static round-robin) list of tiles.  A tile is txc x tyc cells x cb
// batch columns, marched over zc planes; all of it comes from a DevPlan that the kernel reads from
// device memory, so that the same launch (grid, block, shared memory, arguments) serves every
// width a shrinking batch passes through.  A producer warp streams, per plane p,
//     the stencil input tile with a one-cell x/y halo      box (cb, txc+2, tyc+2, 1)
//     the in-place streams of plane p-1 (old | W | X)      box (cb, txc,   tyc,   1)
// into a ring of shared-memory stages with cp.async.bulk.tensor (TMA).  Out-of-grid halo cells and
// planes -1 / nz are zero-filled by the TMA unit, which IS the Dirichlet closure of the stencil —
// no boundary branches in the kernel.  512 consumer threads own one 16-byte item (one cell, two
// columns) each, keep the z pipeline in registers (centre plane, neighbour-plane contribution,
// running in-plane sum) and write results straight to HBM with 128-bit stores.
//
// Solve state on the device (SolveState): working width, iteration count, parity of the vector
// set in use, the re-packing that the last finaliser asked for.  Every launch of a solve reads it
// first; once every column has stopped the launches return at once.  No host round trip anywhere
// in an LSQR solve, with or without tolerances.  Re-packing a shrinking working set is done by
// the passes themselves (TRK instances: results stored into the other vector set at the new
// width); the launches of a solve are chained by programmatic dependent launch.
//
// The squared-norm partials are accumulated per column in a fixed order (thread -> CTA row of
// partials[] -> last CTA); the last CTA to finish reduces the rows and runs the per-column scalar
// recurrences (finalize_phase), so an LSQR iteration is two launches.  Receiver rows: pass F's
// prologue (P v) and a per-tile correction in pass A (P^T).  The same kernel serves the
// objective / gradient pass (MODE_G) and, without its in-place stream, the operator entries.
#pragma once
#include <cuda.h>
#include "wri_kernels.cuh"

namespace wri {

struct RtParams {
    SolveState* st;                   // null: static launch (plan0, maps passed as kernel parameters)
    const DevPlan* plans;             // [n_widths]
    const CUtensorMap* maps;          // [n_widths][2][N_MAPS]
    const CUtensorMap* mmaps;         // [n_widths] model-tile maps
    const int* own_ptr_tab;           // pass A: [n_widths][own_ptr_stride] CSR of the receivers inside each CTA's tiles
    const int4* own_tab;              // [n_widths][own_stride] {receiver, cell, tile, entries of this tile}
    int own_ptr_stride, own_stride;
    DevPlan plan0;
    float2* vec[2][4];                // per parity: U, V, W, X
    float2* U_bot[2];
    float* coef[2];
    double* stat[2];
    int* active[2];
    int* iters[2];
    const float* m;
    const float* gtab;                // gx | gy | gz
    double* partials;                 // [gridDim.x][nb]
    unsigned int* counter;            // last-block ticket
    long long* prof;                  // [4] widths / launches of the passes that did work: F | A
    int nx, ny, nz, nb_max;
    float ih2, a0h, a1, a2, a3, sgn;  // stencil: centre a0/h^2, weights of face / edge / corner neighbours
    int phase;                        // ScalPhase run by the last CTA; < 0: none (operator application)
    int has_old;                      // MODE_A / MODE_G: the second stream (old vector / q) is present
    int lazy;                         // MODE_F: W and X are known to be zero before the first iteration
    int packed;                       // the working set has a column map (grouped / adaptive solves)
    int adaptive;                     // the finaliser may decide to re-pack the working set (both vector sets exist)
    int* retired;                     // adaptive: [nb_out] flags by the caller's column, set when a column leaves
    float2* retire_buf;               // adaptive: [caller's column][cell] final x of the columns that leave (k_finish
                                      // moves them to the caller's u_out as whole rows)
    int maxit;
    int n_rec;
    const int* rec;                   // [n_rec] cell indices
    const float* ca_static;           // static launches: [nb] scale of the operator term
    float2* out;                      // static launches: result vector
    ScalParams fin;                   // template of the finaliser's arguments (banks patched by parity)
    // MODE_G (objective + gradient, eq. 4 / 9): the optional stream is q
    const int* gsrc;                  // [nb] source cells or null
    const float2* galpha;             // [nb] source weights (with gsrc)
    float* g;                         // [n_g] this batch's gradient (overwritten) or null
    float lam2;
    int it;                           // iteration this launch belongs to (host count, 1-based)
};

template <int MODE> struct RtTraits;
template <> struct RtTraits<MODE_F> { static constexpr int NSTREAM = 3; };
template <> struct RtTraits<MODE_A> { static constexpr int NSTREAM = 1; };
template <> struct RtTraits<MODE_G> { static constexpr int NSTREAM = 1; };

__host__ __device__ inline int rt_stage_bytes(const DevPlan& pl, int nstream) {
    return pl.in_span + nstream * pl.ctr_span + pl.m_span;
}
// dynamic shared memory of a launch: ring + barriers + column sums + scratch + tables
__host__ __device__ inline size_t rt_smem_bytes(const DevPlan& pl, int nstream, int nstage, int nxyz) {
    size_t ring = (size_t)nstage * rt_stage_bytes(pl, nstream);
    if (ring < (size_t)RT_MIN_STAGE_AREA) ring = RT_MIN_STAGE_AREA;
    return ring + 2 * RT_MAX_STAGES * 8 + (size_t)pl.nb * 8 + (size_t)RT_NT * 8 + (size_t)nxyz * 4 +
           (size_t)6 * pl.nb * 4 + 64;
}

// rows x columns work with a fixed-order per-column sum: row i of `nrows`, local column s of
// `ncols` -> fn(i, s) returns a double that is added to colacc[coloff(i) + s].  Rows are taken
// NT/ncols at a time; within a round thread s adds the rows in increasing order, so the result
// does not depend on scheduling.  Called by the NT consumer threads only (named barrier 1).
template <int NT, class Fn, class Off>
__device__ __forceinline__ void rows_by_columns(int nrows, int ncols, int tid, double* red, double* colacc,
                                                Fn fn, Off coloff) {
    for (int cbase = 0; cbase < ncols; cbase += NT) {
        const int nc = min(ncols - cbase, NT);
        const int rpr = NT / nc;                                // rows per round
        const int i = tid / nc, s = cbase + tid % nc;
        for (int row0 = 0; row0 < nrows; row0 += rpr) {
            double a = 0.0;
            if (i < rpr && row0 + i < nrows) a = fn(row0 + i, s);
            red[tid] = a;
            asm volatile("bar.sync 1, %0;" ::"r"(NT) : "memory");
            if (tid < nc) {
                const int nr = min(rpr, nrows - row0);
                for (int j = 0; j < nr; ++j) colacc[coloff(row0 + j) + cbase + tid] += red[j * nc + tid];
            }
            asm volatile("bar.sync 1, %0;" ::"r"(NT) : "memory");
        }
    }
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra LAB_DONE;\n"
        "bra LAB_WAIT;\n"
        "LAB_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
// L2 eviction-priority policies: the in-place streams (old | W | X) are touched once per pass,
// the stencil input is re-read by the neighbouring tiles and should outlive them in L2.
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
__device__ __forceinline__ void tma_load_4d_hint(uint32_t dst, const CUtensorMap* tm, uint32_t bar,
                                                 int c0, int c1, int c2, int c3, uint64_t pol) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint"
        " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;" ::"r"(dst), "l"(tm), "r"(bar),
        "r"(c0), "r"(c1), "r"(c2), "r"(c3), "l"(pol) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, uint32_t bar,
                                            int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst), "l"(tm), "r"(bar),
        "r"(c0), "r"(c1), "r"(c2) : "memory");
}
// a tensor map that lives in global memory (the per-width table) is made visible to the TMA unit
__device__ __forceinline__ void tmap_acquire(const CUtensorMap* tm) {
    asm volatile("fence.proxy.tensormap::generic.acquire.gpu [%0], 128;" ::"l"(tm) : "memory");
}
__device__ __forceinline__ void stg128_hint(float2* ptr, const float4& v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(ptr), "f"(v.x), "f"(v.y),
                 "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void stg64_hint(float2* ptr, float a, float b, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v2.f32 [%0], {%1, %2}, %3;" ::"l"(ptr), "f"(a), "f"(b), "l"(pol) : "memory");
}
// one column of a result that is being re-packed: d >= 0 its column in the new set, d <= -2 this column
// leaves and zero-fills the padding column -2 - d instead, -1 nothing to store
__device__ __forceinline__ void put_col(float2* base, size_t cell_off, int d, float a, float b, uint64_t pol) {
    if (d >= 0) stg64_hint(base + cell_off + d, a, b, pol);
    else if (d <= -2) stg64_hint(base + cell_off + (-2 - d), 0.f, 0.f, pol);
}
// the two columns of a thread: one 16-byte store when they stay an aligned pair in the new set (the
// finaliser orders the new set so that this is the rule), else column by column
__device__ __forceinline__ void put_pair(float2* base, size_t cell_off, int d0, int d1, bool pair16, const float4& v,
                                         uint64_t pol) {
    if (pair16) stg128_hint(base + cell_off + d0, v, pol);
    else {
        put_col(base, cell_off, d0, v.x, v.y, pol);
        put_col(base, cell_off, d1, v.z, v.w, pol);
    }
}
__device__ __forceinline__ void consumer_sync(int nthreads) {
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}
// loads from the ring by 32-bit shared-space address (no generic-to-shared conversion per plane)
__device__ __forceinline__ float4 lds128(uint32_t addr) {
    float4 v;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "r"(addr));
    return v;
}
__device__ __forceinline__ float lds32(uint32_t addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}
__device__ __forceinline__ void sts32(uint32_t addr, float v) {
    asm volatile("st.shared.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
__device__ __forceinline__ float4 f4add(const float4& a, const float4& b) {
    return make_float4(a.x + b.x, a.y + b.y, a.z + b.z, a.w + b.w);
}
__device__ __forceinline__ float4 f4zero() { return make_float4(0.f, 0.f, 0.f, 0.f); }

struct TrueT { static constexpr bool value = true; };
struct FalseT { static constexpr bool value = false; };

// Column sums of an [nrows][ncols] row-major matrix of doubles in shared memory, in a fixed order,
// added to colacc[off + j]: blocks of rows first (about sqrt(nrows) groups), then the groups.
template <int NT>
__device__ __forceinline__ void column_sums(const double* mat, int nrows, int ncols, int tid, double* part,
                                            double* colacc, int off) {
    int G = 1;
    while (G * G < nrows) ++G;                                  // ~sqrt(nrows) groups
    G = max(1, min(G, NT / ncols));
    const int rpg = (nrows + G - 1) / G;
    const int g = tid / ncols, j = tid - g * ncols;
    if (g < G) {
        double a = 0.0;
        const int r1 = min(nrows, (g + 1) * rpg);
        for (int r = g * rpg; r < r1; ++r) a += mat[r * ncols + j];
        part[g * ncols + j] = a;
    }
    consumer_sync(NT);
    if (tid < ncols) {
        double t = 0.0;
        for (int gg = 0; gg < G; ++gg) t += part[gg * ncols + tid];
        colacc[off + tid] += t;
    }
    consumer_sync(NT);
}

template <int MODE, int STENCIL, bool TRK>
__global__ void __launch_bounds__(RT_NT + 32, 1)
k_pass_rt(const __grid_constant__ CUtensorMap pm_in, const __grid_constant__ CUtensorMap pm_old,
          const __grid_constant__ CUtensorMap pm_m, const __grid_constant__ RtParams p) {
    constexpr int NT = RT_NT;
    constexpr int NSTREAM = RtTraits<MODE>::NSTREAM;

    // ---- state of the solve in flight (uniform over the grid; written only by finalisers of
    //      earlier launches)
    // Programmatic dependent launch: the passes of a solve are enqueued with the stream-serialisation
    // attribute, so a CTA of the next launch may take an SM as soon as this launch's CTA there has left;
    // it waits here until the whole launch before it has completed and its writes are visible.  (Without
    // the attribute both instructions do nothing.)
    asm volatile("griddepcontrol.wait;" ::: "memory");
    int par = 0, widx = 0, k_done = 0, nbn = 0;
    bool trans = false;
    if (p.st) {
        if (p.st->all_done) return;
        k_done = p.st->k;
        if (k_done >= p.maxit && p.phase != PH_INIT_A) return;
        par = p.st->parity;
        widx = p.st->widx;
        // Re-packing of a shrinking working set (adaptive accuracy): when the finaliser of the last
        // iteration asked for it, both passes of this iteration run as usual on the old vector set but
        // store their results column by column into the other set at the new width — pass F the
        // updated W and X (and the final x of every column that leaves, into the caller's u_out), pass
        // A the new V and a copy of U.  No separate compaction pass over the vectors.
        // The re-packing variant is a kernel of its own (TRK), so that the code of the plain passes is
        // not touched by it: an adaptive solve enqueues both per pass and the one that does not apply
        // returns at once.
        // (pending holds the number of the iteration that re-packs; p.it is this launch's iteration as the
        // host counts it — the plain pass A that asks for a re-packing is followed, in the same iteration,
        // by a launch of the re-packing variant, which must not take the request for its own)
        trans = p.adaptive && p.st->pending == p.it && p.phase != PH_INIT_A;
        if (trans != TRK) return;
        if (trans) nbn = p.plans[p.st->pending_widx].nb;
    }

    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ DevPlan s_pl;
    __shared__ unsigned int s_ticket;
    __shared__ int s_dest[RT_MAXW], s_ret[RT_MAXW];
    const int tid = threadIdx.x;
    {
        const int* src = reinterpret_cast<const int*>(p.st ? p.plans + widx : &p.plan0);
        if (tid < (int)(sizeof(DevPlan) / 4)) reinterpret_cast<int*>(&s_pl)[tid] = src[tid];
        if (TRK && tid < RT_MAXW) {
            s_dest[tid] = p.st->dest[tid];
            s_ret[tid] = p.st->ret_dst[tid];
        }
    }
    __syncthreads();
    const DevPlan& pl = s_pl;
    const PassGeo geo = (MODE == MODE_F) ? pl.f : pl.a;
    // the model tile rides in the TMA stage, except in pass F where the plan may ask for plain loads (its
    // stage already takes four tensor loads per plane; a fifth, tiny one costs 2-3 % from 24 columns on)
    const bool m_tma = pl.m_tma && !(MODE == MODE_F && pl.f_m_ldg);
    const int nb = pl.nb, cb = pl.cb, hp = pl.hp;
    const int nstage = geo.nstage;
    const int STAGE_BYTES = rt_stage_bytes(pl, NSTREAM);
    const int IN_SPAN = pl.in_span, CTR_SPAN = pl.ctr_span;
    const int M_OFF = IN_SPAN + NSTREAM * CTR_SPAN;

    int ring = nstage * STAGE_BYTES;
    if (ring < RT_MIN_STAGE_AREA) ring = RT_MIN_STAGE_AREA;
    unsigned char* stages = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + ring);                   // full[], empty[]
    double* colacc = reinterpret_cast<double*>(bars + 2 * RT_MAX_STAGES);        // [nb]
    double* red = colacc + nb;                                                    // [NT]
    float* tab_g = reinterpret_cast<float*>(red + NT);                            // gx | gy | gz
    float* tab_c = tab_g + (p.nx + p.ny + p.nz);                                  // w2|ca|cb|cv|cx|cw, [6][nb]
    // MODE_G: per consumer warp, the gradient terms of four planes (RT_G_SCRATCH bytes behind the tables)
    float* gbuf_all = reinterpret_cast<float*>((reinterpret_cast<uintptr_t>(tab_c + 6 * nb) + 15) & ~(uintptr_t)15);
    const uint32_t gbuf_w = smem_u32(gbuf_all) + (uint32_t)(threadIdx.x >> 5) * 512u;   // this warp's 4 x 32 terms
    const int lhp = 31 - __clz(max(hp, 1));                                            // log2(hp) where hp is a power of two

    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + RT_MAX_STAGES);
    const size_t NM = p.nb_max;
    const float* cf = p.coef[par];

    const int live_warps = (pl.items + 31) / 32;               // consumer warps with work
    if (tid == 0) {
        for (int s = 0; s < nstage; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, live_warps);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int j = tid; j < nb; j += blockDim.x) {
        colacc[j] = 0.0;
        tab_c[j] = cf[C_W2 * NM + j];
        float ca, cbv = 0.f, cv = 0.f, cx = 0.f, cw = 0.f;
        if (MODE == MODE_F) {
            ca = cf[C_CA_F * NM + j]; cbv = cf[C_CB_F * NM + j]; cv = cf[C_CV_F * NM + j];
            cx = cf[C_CX * NM + j]; cw = cf[C_CW * NM + j];
        } else if (p.st) {
            ca = cf[C_CA_A * NM + j]; cbv = cf[C_CB_A * NM + j];
        } else {
            ca = p.ca_static ? p.ca_static[j] : 1.f;
        }
        tab_c[nb + j] = ca;
        tab_c[2 * nb + j] = cbv;
        tab_c[3 * nb + j] = cv;
        tab_c[4 * nb + j] = cx;
        tab_c[5 * nb + j] = cw;
    }
    for (int j = tid; j < p.nx + p.ny + p.nz; j += blockDim.x) tab_g[j] = p.gtab[j];
    __syncthreads();

    float2* const vU = p.vec[par][0];
    float2* const vV = p.vec[par][1];
    float2* const vW = p.vec[par][2];
    float2* const vX = p.vec[par][3];
    float2* const out = p.st ? ((MODE == MODE_F) ? vU : vV) : p.out;
    float2* const U_bot = p.U_bot[par];
    // the other vector set, written at width nbn while the working set is being re-packed
    float2* const nU = p.vec[par ^ 1][0];
    float2* const nV = p.vec[par ^ 1][1];
    float2* const nW = p.vec[par ^ 1][2];
    float2* const nX = p.vec[par ^ 1][3];
    // pass F's W / X streams are skipped when both are known to be zero (first pass of a cold solve)
    const bool has_old = (MODE == MODE_F) || p.has_old;
    const bool has_wx = (MODE == MODE_F) && !(p.lazy && k_done == 0);

    if (tid >= NT) {
        // ------------------------------------------------------------------ producer warp
        // (all 32 lanes walk the loops together; lane 0 issues)
        const bool issuer = (tid == NT);
        const bool mg = pl.merged != 0;
        const CUtensorMap *tm_in, *tm_old, *tm_w = nullptr, *tm_x = nullptr, *tm_m;
        if (p.st) {
            const CUtensorMap* base = p.maps + ((size_t)widx * 2 + par) * N_MAPS;
            tm_in = base + (MODE == MODE_F ? MP_V_HALO : MP_U_HALO);
            tm_old = base + (MODE == MODE_F ? MP_U_CTR : MP_V_CTR);
            tm_w = base + MP_W_CTR;
            tm_x = base + MP_X_CTR;
            tm_m = p.mmaps + widx;
            if (issuer) {
                tmap_acquire(tm_in); tmap_acquire(tm_old);
                if (MODE == MODE_F) { tmap_acquire(tm_w); tmap_acquire(tm_x); }
                if (m_tma) tmap_acquire(tm_m);
            }
        } else {
            tm_in = &pm_in; tm_old = &pm_old; tm_m = &pm_m;
        }
        const uint64_t pol_stream = policy_evict_first();
        const uint64_t pol_in = policy_evict_last();
        const uint32_t tx_first = pl.in_bytes;
        const uint32_t tx_full = pl.in_bytes + (has_old ? (has_wx ? 3 : 1) * pl.ctr_bytes : 0) +
                                 (m_tma ? pl.m_bytes : 0);
        int stage = 0;
        uint32_t phase = 0;
        for (int t = blockIdx.x; t < geo.n_tiles; t += gridDim.x) {
            int r = t;
            const int chunk = r % pl.nchunk; r /= pl.nchunk;
            const int tx = r % pl.ntx; r /= pl.ntx;
            const int ty = r % pl.nty;
            const int tz = r / pl.nty;
            const int z0 = tz * geo.zc, z1 = min(z0 + geo.zc, p.nz);
            const int c0 = chunk * cb, x0 = tx * pl.txc, y0 = ty * pl.tyc;
            for (int plz = z0 - 1; plz <= z1; ++plz) {
                if (issuer) {
                    mbar_wait(empty0 + 8 * stage, phase ^ 1);
                    const bool streams = plz >= z0 + 1;
                    const uint32_t fb = full0 + 8 * stage;
                    mbar_expect_tx(fb, streams ? tx_full : tx_first);
                    const uint32_t dst = smem_u32(stages + stage * STAGE_BYTES);
                    tma_load_4d_hint(dst, tm_in, fb, mg ? (x0 - 1) * cb : c0, mg ? y0 - 1 : x0 - 1,
                                     mg ? plz : y0 - 1, mg ? 0 : plz, pol_in);
                    if (streams) {
                        const int a0 = mg ? x0 * cb : c0, a1 = mg ? y0 : x0, a2 = mg ? plz - 1 : y0,
                                  a3 = mg ? 0 : plz - 1;
                        if (has_old) tma_load_4d_hint(dst + IN_SPAN, tm_old, fb, a0, a1, a2, a3, pol_stream);
                        if (has_wx) {
                            tma_load_4d_hint(dst + IN_SPAN + CTR_SPAN, tm_w, fb, a0, a1, a2, a3, pol_stream);
                            tma_load_4d_hint(dst + IN_SPAN + 2 * CTR_SPAN, tm_x, fb, a0, a1, a2, a3, pol_stream);
                        }
                        if (m_tma) tma_load_3d(dst + M_OFF, tm_m, fb, x0, y0, plz - 1);
                    }
                }
                __syncwarp();
                if (++stage == nstage) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ------------------------------------------------------------------ consumers
        const bool live = tid < pl.items;
        const int cellt = live ? tid / hp : 0;                  // cell of the tile this thread owns
        const int cp = live ? tid - cellt * hp : 0;             // column pair within the chunk
        const int cxj = cellt % pl.txc, cyj = cellt / pl.txc;
        const int ROW_B = pl.row_b, CELL_B = pl.cell_b;
        const int sm_ctr = (cyj + 1) * ROW_B + (cxj + 1) * CELL_B + cp * 16;   // centre in the halo tile
        const int io = IN_SPAN + (live ? tid : 0) * 16;         // this item in the centre boxes
        const int mo = M_OFF + (cyj * pl.txc + cxj) * 4;
        const uint64_t pol_st = policy_evict_first();
        int stage = 0;
        uint32_t phase = 0;
        uint32_t sb_cur = smem_u32(stages);                     // shared-space address of the stage in use
        const uint32_t ring_b = (uint32_t)(nstage * STAGE_BYTES);

        // pass A: receivers inside this CTA's tiles (host-built per width, in tile order)
        int own_cur = 0, own_end = 0;
        int4 own_nxt = make_int4(-1, -1, -1, 0);
        const int* own_ptr = p.own_ptr_tab + (size_t)widx * p.own_ptr_stride;
        const int4* own = p.own_tab + (size_t)widx * p.own_stride;
        if (MODE == MODE_A && p.st && p.n_rec > 0) {
            own_cur = own_ptr[blockIdx.x];
            own_end = own_ptr[blockIdx.x + 1];
            if (own_cur < own_end) own_nxt = __ldg(own + own_cur);
        }
        if (MODE == MODE_F && p.n_rec > (int)blockIdx.x) {
            // receiver rows of u = M v - alpha u:  U_bot <- cv V[rec] - cb U_bot  (V is read-only in
            // this pass), rows blockIdx.x, +gridDim.x, ...; their |.|^2 joins this CTA's column sums.
            // Runs while the producer warp fills the pipeline.
            const int nrows = (p.n_rec - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
            const int* colmap = p.packed ? p.st->colmap[par] : nullptr;
            rows_by_columns<NT>(nrows, nb, tid, red, colacc,
                [&](int i, int s) -> double {
                    const int r = blockIdx.x + i * gridDim.x;
                    const size_t e = (size_t)r * nb + s;
                    const float2 v = __ldcg(vV + (size_t)p.rec[r] * nb + s);
                    const float2 u = __ldcg(U_bot + e);
                    const float cvs = tab_c[3 * nb + s], cbs = tab_c[2 * nb + s];
                    float2 n = make_float2(fmaf(cvs, v.x, -cbs * u.x), fmaf(cvs, v.y, -cbs * u.y));
                    if (p.fin.rmask) {                                  // per-source receiver sets
                        const int so = colmap ? colmap[s] : s;
                        if (so >= 0 && !p.fin.rmask[(size_t)r * p.fin.nb_out + so]) n = make_float2(0.f, 0.f);
                    }
                    U_bot[e] = n;
                    return (double)fmaf(n.x, n.x, n.y * n.y);
                },
                [](int) { return 0; });
        }

        double acc[2] = {0.0, 0.0};                             // this thread's two columns, all tiles

        // One tile, marched over its planes.  M_TMA / HAS_OLD are compile-time copies of pl.m_tma and
        // of "the old-vector stream is present".  Register pipeline along z, per item:
        //   c_prev  centre of plane z,  s_prev  what plane z gives to its z-neighbours (7-point: the
        //   centre itself; 27-point: a1 c + a2 e + a3 d),  lap  in-plane sum of plane z plus the
        //   contribution of plane z-1.  When plane z+1 arrives, plane z is emitted.
        auto run_tile = [&](auto m_tma_c, auto has_old_c, auto trans_c, const int t) {
            constexpr bool M_TMA = decltype(m_tma_c)::value, HAS_OLD = decltype(has_old_c)::value;
            constexpr bool TR = decltype(trans_c)::value && MODE != MODE_G;   // this iteration re-packs the working set
            int r = t;
            const int chunk = r % pl.nchunk; r /= pl.nchunk;
            const int tx = r % pl.ntx; r /= pl.ntx;
            const int ty = r % pl.nty;
            const int tz = r / pl.nty;
            const int z0 = tz * geo.zc, z1 = min(z0 + geo.zc, p.nz);
            const int col = chunk * cb + cp * 2;

            float w2[2], ca[2], cbk[2], cv[2], cx[2], cw[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                w2[e] = tab_c[col + e]; ca[e] = tab_c[nb + col + e]; cbk[e] = tab_c[2 * nb + col + e];
                cv[e] = tab_c[3 * nb + col + e];
                cx[e] = tab_c[4 * nb + col + e];
                cw[e] = tab_c[5 * nb + col + e];
            }
            const int d0 = TR ? s_dest[col] : -1, d1 = TR ? s_dest[col + 1] : -1;   // columns in the new set
            const int r0 = TR ? s_ret[col] : -1, r1 = TR ? s_ret[col + 1] : -1;     // caller's columns of leaving ones
            const bool pair16 = TR && d0 >= 0 && !(d0 & 1) && d1 == d0 + 1;
            const size_t n_g = (size_t)p.nx * p.ny * p.nz;
            int gsrc0 = -1, gsrc1 = -1;
            float2 gal0 = make_float2(0.f, 0.f), gal1 = gal0;
            // MODE_G: each column chunk has a gradient scratch of its own (the host adds them in chunk order)
            float* const gq = (MODE == MODE_G && p.g) ? p.g + (size_t)chunk * n_g : nullptr;
            if (MODE == MODE_G && p.gsrc) {
                gsrc0 = p.gsrc[col]; gsrc1 = p.gsrc[col + 1];
                gal0 = p.galpha[col]; gal1 = p.galpha[col + 1];
            }
            const int ix = tx * pl.txc + cxj, iy = ty * pl.tyc + cyj;
            const bool valid = live && ix < p.nx && iy < p.ny;
            const int ixc = min(ix, p.nx - 1), iyc = min(iy, p.ny - 1);
            const float gxy = fmaxf(tab_g[ixc], tab_g[p.nx + iyc]);
            int cell = (z0 * p.ny + iyc) * p.nx + ixc;          // cell of the plane being emitted
            unsigned int off = (unsigned int)cell * nb + col;  // its element offset (< 2^31, checked by the host)
            float m_cur = 0.f, m_nxt = 0.f;
            float4 cA = f4zero(), cB = f4zero(), sA = f4zero(), sB = f4zero(), lap = f4zero();
            float acc32[2] = {0.f, 0.f};
            const unsigned int plane_e = (unsigned int)(p.nx * p.ny) * nb;
            const int plane_m = p.nx * p.ny;
            const float* gz_tab = tab_g + p.nx + p.ny;

            // step plz: c_new <- centre of plane plz; emit plane plz-1; then lap <- in-plane sum of plz
            // plus the contribution of plane plz-1
            auto plane = [&](const int plz, float4& c_prev, float4& c_new, float4& s_prev, float4& s_new) {
                if (!M_TMA && plz >= z0 && plz < z1) m_nxt = __ldg(p.m + cell + (plz > z0 ? plane_m : 0));
                const bool emit = plz >= z0 + 1;
                float gzv = 0.f;                                // sponge profile of the plane being emitted, read
                if (emit) gzv = gz_tab[plz - 1];                // before the wait so that its latency hides behind it
                mbar_wait(full0 + 8 * stage, phase);
                const uint32_t sb = sb_cur;                     // this stage's shared-space address
                c_new = lds128(sb + sm_ctr);
                float4 t_new;                                   // in-plane part of the stencil on plane plz
                {
                    const float4 a = lds128(sb + sm_ctr - CELL_B), b = lds128(sb + sm_ctr + CELL_B);
                    const float4 c = lds128(sb + sm_ctr - ROW_B), d = lds128(sb + sm_ctr + ROW_B);
                    const float4 e4 = f4add(f4add(a, b), f4add(c, d));
                    if (STENCIL == ST_27) {
                        const float4 a2 = lds128(sb + sm_ctr - ROW_B - CELL_B), b2 = lds128(sb + sm_ctr - ROW_B + CELL_B);
                        const float4 c2 = lds128(sb + sm_ctr + ROW_B - CELL_B), d2 = lds128(sb + sm_ctr + ROW_B + CELL_B);
                        const float4 d4 = f4add(f4add(a2, b2), f4add(c2, d2));
                        s_new = make_float4(fmaf(p.a1, c_new.x, fmaf(p.a2, e4.x, p.a3 * d4.x)),
                                            fmaf(p.a1, c_new.y, fmaf(p.a2, e4.y, p.a3 * d4.y)),
                                            fmaf(p.a1, c_new.z, fmaf(p.a2, e4.z, p.a3 * d4.z)),
                                            fmaf(p.a1, c_new.w, fmaf(p.a2, e4.w, p.a3 * d4.w)));
                        t_new = make_float4(fmaf(p.a1, e4.x, p.a2 * d4.x), fmaf(p.a1, e4.y, p.a2 * d4.y),
                                            fmaf(p.a1, e4.z, p.a2 * d4.z), fmaf(p.a1, e4.w, p.a2 * d4.w));
                    } else {
                        t_new = e4;
                    }
                }
                const float4& zn = (STENCIL == ST_27) ? s_new : c_new;   // what plane plz gives plane plz-1
                const float4& zp = (STENCIL == ST_27) ? s_prev : c_prev; // what plane plz-1 gives plane plz
                float4 o_old = f4zero();
                if (emit) {
                    if (HAS_OLD) o_old = lds128(sb + io);
                    if (M_TMA) m_cur = lds32(sb + mo);
                }
                // pass A / G: the stage is free once its loads are done.  Pass F reads W and X from
                // the stage just before it uses them (fewer live registers) and releases it after.
                auto release = [&]() {
                    __syncwarp();
                    if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * stage);
                    sb_cur += STAGE_BYTES;
                    if (++stage == nstage) { stage = 0; phase ^= 1; sb_cur -= ring_b; }
                };
                if (MODE != MODE_F) release();

                if (emit) {
                    const float g = fmaxf(gxy, gzv);
                    const float4 cc = c_prev;
                    const float s0 = lap.x + zn.x, s1 = lap.y + zn.y, s2 = lap.z + zn.z, s3 = lap.w + zn.w;
                    if (MODE == MODE_G) {
                        // r = A u - q - alpha e;  |r|^2 sums;  g[c] += lam^2 sum_s w2_s (Re t + gamma Im t),
                        // t = conj(u) r  (= Re[conj((1 + i gamma) u) r], eq. 9 with this build's sponge)
                        float gterm = 0.f;
                        {
                            const float wm = w2[0] * m_cur;
                            const float dr = wm + p.a0h, di = wm * g;
                            float r_re = fmaf(p.ih2, s0, fmaf(dr, cc.x, -di * cc.y)) - o_old.x;
                            float r_im = fmaf(p.ih2, s1, fmaf(dr, cc.y, di * cc.x)) - o_old.y;
                            if (cell == gsrc0) { r_re -= gal0.x; r_im -= gal0.y; }
                            if (valid) acc32[0] += fmaf(r_re, r_re, r_im * r_im);
                            const float tr = fmaf(cc.x, r_re, cc.y * r_im), ti = fmaf(cc.x, r_im, -cc.y * r_re);
                            gterm = w2[0] * fmaf(g, ti, tr);
                        }
                        {
                            const float wm = w2[1] * m_cur;
                            const float dr = wm + p.a0h, di = wm * g;
                            float r_re = fmaf(p.ih2, s2, fmaf(dr, cc.z, -di * cc.w)) - o_old.z;
                            float r_im = fmaf(p.ih2, s3, fmaf(dr, cc.w, di * cc.z)) - o_old.w;
                            if (cell == gsrc1) { r_re -= gal1.x; r_im -= gal1.y; }
                            if (valid) acc32[1] += fmaf(r_re, r_re, r_im * r_im);
                            const float tr = fmaf(cc.z, r_re, cc.w * r_im), ti = fmaf(cc.z, r_im, -cc.w * r_re);
                            gterm = fmaf(w2[1], fmaf(g, ti, tr), gterm);
                        }
                        if (p.g && hp >= 4) {
                            // Sum over the batch columns of a cell: the hp threads of a cell are consecutive
                            // lanes (the host sends only power-of-two hp <= 32 down this path).  The terms of
                            // FOUR planes are parked in the warp's scratch and folded together — a lane takes
                            // four neighbouring terms (one plane, one cell), then hp/4 lanes are folded by
                            // shuffles: 1 + log2(hp/4) dependent steps per four planes instead of log2(hp)
                            // per plane (the chain of shuffles was the longest stall of this pass).  Fixed
                            // order; planes are emitted in aligned blocks of four (tiles start at multiples
                            // of 8 planes).  Pure stores (no load in the pipeline's critical path): this
                            // batch's gradient goes to a scratch array, k_add_f32 accumulates it afterwards.
                            // (hp is a power of two here: shifts and masks, no division in the loop)
                            const int lane = tid & 31, slot = (plz - 1) & 3;
                            sts32(gbuf_w + 128 * slot + 4 * lane, gterm);
                            if (slot == 3 || plz == z1) {
                                __syncwarp();
                                const float4 v4 = lds128(gbuf_w + 16 * lane);
                                float sum = (v4.x + v4.y) + (v4.z + v4.w);
                                const int qpc = hp >> 2;                       // lanes per (plane, cell) now
                                if (qpc > 4) sum += __shfl_down_sync(0xffffffffu, sum, 4, qpc);
                                if (qpc > 2) sum += __shfl_down_sync(0xffffffffu, sum, 2, qpc);
                                if (qpc > 1) sum += __shfl_down_sync(0xffffffffu, sum, 1, qpc);
                                const int pl = lane >> 3, cw = ((lane & 7) << 2) >> lhp;
                                // cell of (first plane of the block, cell cw of this warp) from a lane that owns it
                                const int c0 = __shfl_sync(0xffffffffu, valid ? cell - slot * plane_m : -1, cw << lhp);
                                if ((lane & (qpc - 1)) == 0 && pl <= slot && c0 >= 0) gq[c0 + pl * plane_m] = p.lam2 * sum;
                                __syncwarp();
                            }
                        } else if (p.g) {
                            for (int dlt = hp >> 1; dlt > 0; dlt >>= 1)
                                gterm += __shfl_down_sync(0xffffffffu, gterm, dlt, hp);
                            if (cp == 0 && valid) gq[cell] = p.lam2 * gterm;
                        }
                    } else {
                        float4 rr;
                        {
                            const float wm = w2[0] * m_cur;
                            const float dr = wm + p.a0h, di = p.sgn * wm * g;
                            const float ar = fmaf(p.ih2, s0, fmaf(dr, cc.x, -di * cc.y));
                            const float ai = fmaf(p.ih2, s1, fmaf(dr, cc.y, di * cc.x));
                            rr.x = fmaf(ca[0], ar, -cbk[0] * o_old.x);
                            rr.y = fmaf(ca[0], ai, -cbk[0] * o_old.y);
                        }
                        {
                            const float wm = w2[1] * m_cur;
                            const float dr = wm + p.a0h, di = p.sgn * wm * g;
                            const float ar = fmaf(p.ih2, s2, fmaf(dr, cc.z, -di * cc.w));
                            const float ai = fmaf(p.ih2, s3, fmaf(dr, cc.w, di * cc.z));
                            rr.z = fmaf(ca[1], ar, -cbk[1] * o_old.z);
                            rr.w = fmaf(ca[1], ai, -cbk[1] * o_old.w);
                        }
                        if (valid) {
                            const size_t offn = (size_t)cell * nbn;
                            if (!TR || MODE == MODE_F) {
                                stg128_hint(out + off, rr, pol_st);
                            } else {
                                // pass A of a re-packing iteration: the new V and a copy of U (its centre
                                // value is in registers) go to the new set
                                put_pair(nV, offn, d0, d1, pair16, rr, pol_st);
                                put_pair(nU, offn, d0, d1, pair16, cc, pol_st);
                            }
                            acc32[0] += fmaf(rr.x, rr.x, rr.y * rr.y);
                            acc32[1] += fmaf(rr.z, rr.z, rr.w * rr.w);
                            if (MODE == MODE_F) {
                                float4 o_w = f4zero(), o_x = f4zero();
                                if (has_wx) {
                                    o_w = lds128(sb + io + CTR_SPAN);
                                    o_x = lds128(sb + io + 2 * CTR_SPAN);
                                }
                                float4 xn, wn;
                                xn.x = fmaf(cx[0], o_w.x, o_x.x);
                                xn.y = fmaf(cx[0], o_w.y, o_x.y);
                                xn.z = fmaf(cx[1], o_w.z, o_x.z);
                                xn.w = fmaf(cx[1], o_w.w, o_x.w);
                                wn.x = fmaf(cv[0], cc.x, -cw[0] * o_w.x);
                                wn.y = fmaf(cv[0], cc.y, -cw[0] * o_w.y);
                                wn.z = fmaf(cv[1], cc.z, -cw[1] * o_w.z);
                                wn.w = fmaf(cv[1], cc.w, -cw[1] * o_w.w);
                                if (!TR) {
                                    stg128_hint(vX + off, xn, pol_st);
                                    stg128_hint(vW + off, wn, pol_st);
                                } else {
                                    // pass F of a re-packing iteration: X and W go to the new set; a column
                                    // that leaves has just received its last update, x_k = X + cx W
                                    put_pair(nX, offn, d0, d1, pair16, xn, pol_st);
                                    put_pair(nW, offn, d0, d1, pair16, wn, pol_st);
                                    // (column by column in a side buffer: the threads of neighbouring cells
                                    // fill its sectors; straight into u_out these would be 8-byte pieces
                                    // of 32-byte sectors, read-modify-write in DRAM)
                                    if (r0 >= 0) stg64_hint(p.retire_buf + (size_t)r0 * n_g + cell, xn.x, xn.y, pol_st);
                                    if (r1 >= 0) stg64_hint(p.retire_buf + (size_t)r1 * n_g + cell, xn.z, xn.w, pol_st);
                                }
                            }
                        }
                    }
                    off += plane_e;
                    cell += plane_m;
                    // |.|^2 in fp32 over one aligned block of 8 planes, then fp64: tiles start at multiples
                    // of 8 planes, so these partial sums — and with them a column's result — do not depend
                    // on the tile geometry of the width the column happens to run at (reading C-9)
                    if (((plz - 1) & 7) == 7) {
                        acc[0] += (double)acc32[0]; acc[1] += (double)acc32[1];
                        acc32[0] = acc32[1] = 0.f;
                    }
                }
                if (MODE == MODE_F) release();
                lap = f4add(t_new, zp);
                if (!M_TMA) m_cur = m_nxt;
            };
            for (int plz = z0 - 1; plz <= z1; plz += 2) {
                plane(plz, cA, cB, sA, sB);
                if (plz + 1 > z1) break;
                plane(plz + 1, cB, cA, sB, sA);
            }
            acc[0] += (double)acc32[0];
            acc[1] += (double)acc32[1];
            return chunk;
        };

        // warps without work (tiles of fewer than 512 items) stay out of the pipeline: the empty
        // barriers count the live warps only; everybody meets again at the named barriers below
        const bool warp_live = (tid >> 5) < live_warps;
        for (int t = blockIdx.x; t < geo.n_tiles; t += gridDim.x) {
            int chunk = t % pl.nchunk;
            if (warp_live) {
                if constexpr (TRK) {                             // (a re-packing iteration always has its old stream)
                    if (m_tma) chunk = run_tile(TrueT{}, TrueT{}, TrueT{}, t);
                    else          chunk = run_tile(FalseT{}, TrueT{}, TrueT{}, t);
                } else if (m_tma) {
                    if (has_old) chunk = run_tile(TrueT{}, TrueT{}, FalseT{}, t);
                    else         chunk = run_tile(TrueT{}, FalseT{}, FalseT{}, t);
                } else {
                    if (has_old) chunk = run_tile(FalseT{}, TrueT{}, FalseT{}, t);
                    else         chunk = run_tile(FalseT{}, FalseT{}, FalseT{}, t);
                }
            }
            if (pl.nchunk > 1) {
                // several chunks per cell: a thread's columns change from tile to tile, so its sums
                // are folded into the CTA's column sums tile by tile
                double* mat = red;                               // [items][2] does not fit red: use two rounds
                for (int e = 0; e < 2; ++e) {
                    consumer_sync(NT);
                    mat[tid] = live ? acc[e] : 0.0;
                    consumer_sync(NT);
                    if (tid < hp) {
                        double s = 0.0;
                        for (int kx = tid; kx < pl.items; kx += hp) s += mat[kx];
                        colacc[chunk * cb + 2 * tid + e] += s;
                    }
                }
                consumer_sync(NT);
                acc[0] = acc[1] = 0.0;
            }
            if (MODE == MODE_A && own_nxt.z == t) {
                // P^T rows: the receivers inside the tile just written get  V += ct U_bot ; the
                // squared-norm sums are corrected by |V + ct U_bot|^2 - |V|^2.
                consumer_sync(NT);                               // the tile's stores are done
                const int cnt = own_nxt.w;
                const float* ct = cf + C_CT_A * NM;
                rows_by_columns<NT>(cnt, cb, tid, red, colacc,
                    [&](int i, int s) -> double {
                        const int4 en = (i == 0) ? own_nxt : __ldg(own + own_cur + i);
                        const int c = chunk * cb + s;
                        float2* vp = out + (size_t)en.y * nb + c;
                        if (TRK) {                               // V of this iteration lives in the new set
                            if (s_dest[c] < 0) return 0.0;       // (a column that leaves is no longer iterated)
                            vp = nV + (size_t)en.y * nbn + s_dest[c];
                        }
                        const float2 v = __ldcg(vp);
                        const float2 u = __ldcg(U_bot + (size_t)en.x * nb + c);
                        const float cts = ct[c];
                        const float2 n = make_float2(fmaf(cts, u.x, v.x), fmaf(cts, u.y, v.y));
                        *vp = n;
                        return ((double)n.x * n.x + (double)n.y * n.y) - (double)fmaf(v.x, v.x, v.y * v.y);
                    },
                    [&](int) { return chunk * cb; });
                own_cur += cnt;
                own_nxt = (own_cur < own_end) ? __ldg(own + own_cur) : make_int4(-1, -1, -1, 0);
            }
        }
        if (pl.nchunk == 1) {
            // one chunk per cell: thread tid owns columns (2 cp, 2 cp + 1) for the whole launch; fold
            // the per-thread sums into the CTA's column sums once, through the (idle) stages
            consumer_sync(NT);                                   // every stage has been consumed
            double* mat = reinterpret_cast<double*>(stages);     // [items][2] = [cells][cb]
            double* part = mat + 2 * NT;
            if (live) { mat[2 * tid] = acc[0]; mat[2 * tid + 1] = acc[1]; }
            consumer_sync(NT);
            column_sums<NT>(mat, pl.items / hp, cb, tid, part, colacc, 0);
        }
    }

    // ---------------------------------------------------------------------- CTA epilogue
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    __syncthreads();
    if (p.partials)
        for (int j = tid; j < nb; j += blockDim.x) p.partials[(size_t)blockIdx.x * nb + j] = colacc[j];
    __threadfence();
    __syncthreads();
    if (tid == 0) s_ticket = atomicAdd(p.counter, 1u);
    __syncthreads();
    if (s_ticket == gridDim.x - 1) {
        __threadfence();
        double* sh = reinterpret_cast<double*>(smem);           // stages are idle now
        if (MODE != MODE_G && p.phase >= 0) {                   // phase < 0: no scalar phase (operator application)
            ScalParams f = p.fin;
            f.nb = nb;
            f.n_tiles = gridDim.x;
            f.V = vV; f.U = vU; f.X = vX; f.U_bot = U_bot;
            f.coef = p.coef[par]; f.stat = p.stat[par]; f.active = p.active[par]; f.iters = p.iters[par];
            f.colmap = p.packed ? p.st->colmap[par] : nullptr;
            f.k = k_done + 1;
            f.st = p.st;
            f.adaptive = p.adaptive;
            f.widx = widx;
            f.trans = trans;
            f.nb_new = nbn;
            f.coef2 = p.coef[par ^ 1]; f.stat2 = p.stat[par ^ 1]; f.active2 = p.active[par ^ 1];
            f.iters2 = p.iters[par ^ 1]; f.U_bot2 = p.U_bot[par ^ 1];
            f.retired = p.retired;
            switch (p.phase) {
                case PH_INIT_A: finalize_phase<PH_INIT_A>(f, sh); break;
                case PH_F:      finalize_phase<PH_F>(f, sh); break;
                default:        finalize_phase<PH_A>(f, sh); break;
            }
        }
        __syncthreads();
        if (tid == 0) {
            *p.counter = 0u;
            if (p.st && p.phase != PH_INIT_A && p.prof) {
                p.prof[MODE == MODE_F ? 0 : 2] += nb;
                p.prof[MODE == MODE_F ? 1 : 3] += 1;
            }
        }
    }
}

}  // namespace wri
