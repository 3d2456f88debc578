// wri_tma.cuh — persistent, TMA-fed stencil + LSQR pass for sm_100a (the hot kernel).
//
// One CTA per SM walks a fixed (static round-robin) list of tiles.  A tile is TXC x TYC cells
// x CB batch columns, marched over zc planes.  A producer warp streams, per plane p,
//     the stencil input tile with a one-cell x/y halo      box (CB, TXC+2, TYC+2, 1)
//     the in-place streams of plane p-1 (old | W | X)      box (CB, TXC,   TYC,   1)
// into a ring of shared-memory stages with cp.async.bulk.tensor (TMA).  Out-of-grid halo cells
// and planes -1 / nz are zero-filled by the TMA unit, which IS the Dirichlet closure of the
// 7-point stencil — no boundary branches in the kernel.  The consumer threads (one 16-byte item
// each, up to 512) keep the z pipeline (c_{z-1}, c_z, in-plane neighbour sum n_z) in registers, so
// every stage is consumed entirely at its own step, and write results straight to HBM with 128-bit
// stores.  The ring depth in use is a run-time parameter (TmaPassParams::nstage <= Cfg::NSTAGE).
//
// The squared-norm partials are accumulated per column in a fixed order (thread -> tile ->
// CTA row of partials[]); the last CTA to finish reduces the rows and runs the per-column scalar
// recurrences (finalize_phase), so an LSQR iteration is two launches.  Receiver rows: pass F's
// prologue (P v) and a per-tile correction in pass A (P^T).  The same kernel serves the
// objective / gradient pass (MODE_G) and, without its in-place stream, the operator entries.
#pragma once
#include <cuda.h>
#include "wri_kernels.cuh"

#ifndef WRI_HINTS
#define WRI_HINTS 2     // 0 none, 1 streams evict_first, 2 + stencil input evict_last, 3 + output evict_last
#endif

namespace wri {

template <int CB_, int TXC_, int TYC_, int NT_, int NSTAGE_>
struct TileCfg {
    static constexpr int CB = CB_, TXC = TXC_, TYC = TYC_;
    static constexpr int NT = NT_;                              // consumer threads
    static constexpr int NSTAGE = NSTAGE_;                      // LARGEST depth of the shared-memory ring (p.nstage <= NSTAGE is used)
    static constexpr int ITEMS = TXC * TYC * CB / 2;            // 16-byte items per plane
    static constexpr int IPT = ITEMS / NT;                      // items per thread
    static constexpr int IN_BYTES = (TXC + 2) * (TYC + 2) * CB * 8;   // bytes the halo box delivers
    static constexpr int IN_SPAN = (IN_BYTES + 127) / 128 * 128;       // room it takes in a stage (TMA destinations: 128 B)
    static constexpr int CTR_BYTES = TXC * TYC * CB * 8;
    static constexpr int M_BYTES = (TXC * TYC * 4 + 127) / 128 * 128;   // model tile (float per cell)
    static_assert(ITEMS % NT == 0, "tile must give every consumer thread the same work");
    static_assert(NT % (CB / 2) == 0, "a thread must keep one column pair");
    static_assert(CTR_BYTES % 128 == 0, "TMA destinations need 128 B alignment");
};

struct TrueT { static constexpr bool value = true; };
struct FalseT { static constexpr bool value = false; };

template <int MODE> struct PassTraits;
#ifndef WRI_F_STAGES
#define WRI_F_STAGES 4
#endif
#ifndef WRI_A_STAGES
#define WRI_A_STAGES 7
#endif
template <> struct PassTraits<MODE_F> { static constexpr int NSTREAM = 3, NSTAGE = WRI_F_STAGES; };   // largest depths
template <> struct PassTraits<MODE_A> { static constexpr int NSTREAM = 1, NSTAGE = WRI_A_STAGES; };
template <> struct PassTraits<MODE_G> { static constexpr int NSTREAM = 1, NSTAGE = WRI_A_STAGES; };   // stream = q (optional)

struct TmaPassParams {
    float2* out;           // result vector (its old values arrive through tm_old)
    float2* W;
    float2* X;
    const float* m;
    const float *gx, *gy, *gz;
    const float *w2, *ca, *cb, *cv, *cx, *cw;
    double* partials;      // [gridDim.x][nb]
    unsigned int* counter; // last-block ticket
    int nx, ny, nz, nb;
    int zc, ntx, nty, ntz, nchunk, n_tiles;
    float ih2, m6ih2, sgn;
    int m_tma;             // 1: the model tile rides in the TMA stage (needs nx % 4 == 0)
    int merged;            // 1: tensor maps fold (column, x) into one dimension (nchunk == 1)
    int phase;             // ScalPhase run by the last CTA
    int nstage;            // ring depth in use (<= Cfg::NSTAGE), chosen per plan by the host
    // receiver rows, spread over the CTAs (keeps them off the last CTA's serial tail)
    int n_rec;
    const int* rec;        // [n_rec] cell indices
    float2* U_bot;         // [n_rec][nb]
    const float2* V;       // pass F: the stencil input as a plain pointer (rows of P v)
    const float* ct;       // pass A: [nb] scale of P^T U_bot
    const int* own_ptr;    // pass A: [gridDim.x + 1] CSR over own
    const int4* own;       // pass A: receivers inside this CTA's tiles, sorted by tile:
                           //         {receiver, cell, tile, entries in this tile (at its first entry)};
                           //         with column chunks, one entry per (receiver, chunk)
    ScalParams fin;
    // MODE_G (objective + gradient, eq. 4 / 9): out is unused; the optional stream is q
    int has_q;             // MODE_A / MODE_G: the second stream (old vector / q) is present; 0 = plain operator
                           // MODE_F: the W and X streams are read; 0 = they are known to be zero (first pass of a
                           // cold solve: they are written, never read, so they need no clearing beforehand)
                           // application out = ca * A in (wri_apply_M / _MH through this pipeline)
    const int* gsrc;       // [nb] source cells or null
    const float2* galpha;  // [nb] source weights (with gsrc)
    float* g;              // [n_g] this batch's gradient (overwritten) or null
    float lam2;
};

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
#ifdef WRI_RELAXED_ARRIVE
    asm volatile("mbarrier.arrive.relaxed.cta.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
#else
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
#endif
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
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* tm, uint32_t bar,
                                            int c0, int c1, int c2, int c3) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5, %6}], [%2];" ::"r"(dst), "l"(tm), "r"(bar),
        "r"(c0), "r"(c1), "r"(c2), "r"(c3) : "memory");
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
__device__ __forceinline__ void stg128_hint(float2* ptr, const float4& v, uint64_t pol) {
    asm volatile("st.global.L2::cache_hint.v4.f32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(ptr), "f"(v.x), "f"(v.y),
                 "f"(v.z), "f"(v.w), "l"(pol) : "memory");
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap* tm, uint32_t bar,
                                            int c0, int c1, int c2) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes"
        " [%0], [%1, {%3, %4, %5}], [%2];" ::"r"(dst), "l"(tm), "r"(bar),
        "r"(c0), "r"(c1), "r"(c2) : "memory");
}
__device__ __forceinline__ void consumer_sync(int nthreads) {
    asm volatile("bar.sync 1, %0;" ::"r"(nthreads) : "memory");
}
__device__ __forceinline__ float4 lds128(const unsigned char* base, int byte_off) {
    return *reinterpret_cast<const float4*>(base + byte_off);
}

template <class Cfg, int MODE>
__global__ void __launch_bounds__(Cfg::NT + 32, 1)
k_pass_tma(const __grid_constant__ CUtensorMap tm_in, const __grid_constant__ CUtensorMap tm_old,
           const __grid_constant__ CUtensorMap tm_w, const __grid_constant__ CUtensorMap tm_x,
           const __grid_constant__ CUtensorMap tm_m, const TmaPassParams p) {
    constexpr int CB = Cfg::CB, TXC = Cfg::TXC, TYC = Cfg::TYC, NT = Cfg::NT, IPT = Cfg::IPT;
    constexpr int NSTREAM = PassTraits<MODE>::NSTREAM, NSTAGE = Cfg::NSTAGE;
    constexpr int M_OFF = Cfg::IN_SPAN + NSTREAM * Cfg::CTR_BYTES;
    constexpr int STAGE_BYTES = M_OFF + Cfg::M_BYTES;
    constexpr int HP = CB / 2;                                  // column pairs per cell
    constexpr int ROW_B = (TXC + 2) * CB * 8;                   // bytes per halo-tile row
    constexpr int CELL_B = CB * 8;

    extern __shared__ __align__(128) unsigned char smem[];
    unsigned char* stages = smem;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + NSTAGE * STAGE_BYTES);   // full[NSTAGE], empty[NSTAGE]
    double* colacc = reinterpret_cast<double*>(bars + 2 * NSTAGE);               // [nb]
    double* red = colacc + p.nb;                                                  // [NT*2]
    float* tab_g = reinterpret_cast<float*>(red + 2 * NT);                        // gx | gy | gz
    float* tab_c = tab_g + (p.nx + p.ny + p.nz);                                  // w2|ca|cb|cv|cx|cw, [6][nb]
    __shared__ unsigned int s_ticket;

    const int tid = threadIdx.x;
    const uint32_t full0 = smem_u32(bars), empty0 = smem_u32(bars + NSTAGE);

    if (tid == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(full0 + 8 * s, 1);
            mbar_init(empty0 + 8 * s, NT / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    for (int j = tid; j < p.nb; j += blockDim.x) {
        colacc[j] = 0.0;
        tab_c[j] = p.w2[j];
        tab_c[p.nb + j] = p.ca[j];
        tab_c[2 * p.nb + j] = p.cb[j];
        tab_c[3 * p.nb + j] = (MODE == MODE_F) ? p.cv[j] : 0.f;
        tab_c[4 * p.nb + j] = (MODE == MODE_F) ? p.cx[j] : 0.f;
        tab_c[5 * p.nb + j] = (MODE == MODE_F) ? p.cw[j] : 0.f;
    }
    for (int j = tid; j < p.nx + p.ny + p.nz; j += blockDim.x) tab_g[j] = p.gx[j];   // gx|gy|gz are contiguous
    __syncthreads();

    if (tid >= NT) {
        // ------------------------------------------------------------------ producer warp
        // (all 32 lanes walk the loops together; lane 0 issues)
        const bool issuer = (tid == NT);
        // merged maps (narrow chunks, one chunk per cell): the column index is folded into x, so a
        // box row is CB*(TXC+2) contiguous elements instead of CB:  (x*CB, y, z, 0)
        const bool mg = p.merged != 0;
#if WRI_HINTS >= 1
        const uint64_t pol_stream = policy_evict_first();
#endif
#if WRI_HINTS >= 2
        const uint64_t pol_in = policy_evict_last();
#endif
        int stage = 0;
        uint32_t phase = 0;
        for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
            int r = t;
            const int chunk = r % p.nchunk; r /= p.nchunk;
            const int tx = r % p.ntx; r /= p.ntx;
            const int ty = r % p.nty;
            const int tz = r / p.nty;
            const int z0 = tz * p.zc, z1 = min(z0 + p.zc, p.nz);
            const int c0 = chunk * CB, x0 = tx * TXC, y0 = ty * TYC;
            for (int pl = z0 - 1; pl <= z1; ++pl) {
                if (issuer) {
                    mbar_wait(empty0 + 8 * stage, phase ^ 1);
                    const bool streams = pl >= z0 + 1;
                    const bool old_stream = (MODE == MODE_F) || p.has_q;
                    const bool wx_streams = (MODE == MODE_F) && p.has_q;     // F's first pass of a cold solve: W = X = 0
                    const uint32_t fb = full0 + 8 * stage;
                    mbar_expect_tx(fb, Cfg::IN_BYTES + (streams ? (old_stream ? (wx_streams || MODE != MODE_F ? NSTREAM : 1) * Cfg::CTR_BYTES : 0) +
                                                            (p.m_tma ? TXC * TYC * 4 : 0) : 0));
                    const uint32_t dst = smem_u32(stages + stage * STAGE_BYTES);
#if WRI_HINTS >= 2
                    tma_load_4d_hint(dst, &tm_in, fb, mg ? (x0 - 1) * CB : c0, mg ? y0 - 1 : x0 - 1, mg ? pl : y0 - 1, mg ? 0 : pl, pol_in);
#else
                    tma_load_4d(dst, &tm_in, fb, mg ? (x0 - 1) * CB : c0, mg ? y0 - 1 : x0 - 1, mg ? pl : y0 - 1, mg ? 0 : pl);
#endif
                    if (streams) {
#if WRI_HINTS >= 1
                        if (old_stream)
                        tma_load_4d_hint(dst + Cfg::IN_SPAN, &tm_old, fb, mg ? x0 * CB : c0, mg ? y0 : x0, mg ? pl - 1 : y0, mg ? 0 : pl - 1, pol_stream);
                        if (wx_streams) {
                            tma_load_4d_hint(dst + Cfg::IN_SPAN + Cfg::CTR_BYTES, &tm_w, fb, mg ? x0 * CB : c0, mg ? y0 : x0, mg ? pl - 1 : y0, mg ? 0 : pl - 1, pol_stream);
                            tma_load_4d_hint(dst + Cfg::IN_SPAN + 2 * Cfg::CTR_BYTES, &tm_x, fb, mg ? x0 * CB : c0, mg ? y0 : x0, mg ? pl - 1 : y0, mg ? 0 : pl - 1, pol_stream);
                        }
#else
                        if (old_stream)
                        tma_load_4d(dst + Cfg::IN_SPAN, &tm_old, fb, mg ? x0 * CB : c0, mg ? y0 : x0, mg ? pl - 1 : y0, mg ? 0 : pl - 1);
                        if (wx_streams) {
                            tma_load_4d(dst + Cfg::IN_SPAN + Cfg::CTR_BYTES, &tm_w, fb, mg ? x0 * CB : c0, mg ? y0 : x0, mg ? pl - 1 : y0, mg ? 0 : pl - 1);
                            tma_load_4d(dst + Cfg::IN_SPAN + 2 * Cfg::CTR_BYTES, &tm_x, fb, mg ? x0 * CB : c0, mg ? y0 : x0, mg ? pl - 1 : y0, mg ? 0 : pl - 1);
                        }
#endif
                        if (p.m_tma) tma_load_3d(dst + M_OFF, &tm_m, fb, x0, y0, pl - 1);
                    }
                }
                __syncwarp();
                if (++stage == p.nstage) { stage = 0; phase ^= 1; }
            }
        }
    } else {
        // ------------------------------------------------------------------ consumers
        const int cp = tid % HP;                                // column pair within the chunk
#if WRI_HINTS >= 1
        const uint64_t pol_st = policy_evict_first();
        const uint64_t pol_out = (WRI_HINTS >= 3) ? policy_evict_last() : pol_st;
#endif
        int stage = 0;
        uint32_t phase = 0;
        // static item geometry: item j of this thread is cell (cxj, cyj) of the tile
        int sm_ctr[IPT];                                        // byte offset of the centre in the halo tile
        int cxj[IPT], cyj[IPT];
#pragma unroll
        for (int j = 0; j < IPT; ++j) {
            const int cell = (tid + j * NT) / HP;
            cxj[j] = cell % TXC;
            cyj[j] = cell / TXC;
            sm_ctr[j] = (cyj[j] + 1) * ROW_B + (cxj[j] + 1) * CELL_B + cp * 16;
        }

        int own_cur = 0, own_end = 0;
        int4 own_nxt = make_int4(-1, -1, -1, 0);
        if (MODE == MODE_A && p.n_rec > 0) {
            own_cur = p.own_ptr[blockIdx.x];
            own_end = p.own_ptr[blockIdx.x + 1];
            if (own_cur < own_end) own_nxt = __ldg(p.own + own_cur);
        }
        if (MODE == MODE_F && p.n_rec > (int)blockIdx.x) {
            // receiver rows of u = M v - alpha u:  U_bot <- cv V[rec] - cb U_bot  (V is read-only in
            // this pass), rows blockIdx.x, +gridDim.x, ...; their |.|^2 joins this CTA's column sums.
            // Runs while the producer warp fills the pipeline.
            const int nrows = (p.n_rec - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;
            const int nb = p.nb;
            rows_by_columns<NT>(nrows, nb, tid, red, colacc,
                [&](int i, int s) -> double {
                    const int r = blockIdx.x + i * gridDim.x;
                    const size_t e = (size_t)r * nb + s;
                    const float2 v = __ldcg(p.V + (size_t)p.rec[r] * nb + s);
                    const float2 u = __ldcg(p.U_bot + e);
                    const float cvs = tab_c[3 * nb + s], cbs = tab_c[2 * nb + s];
                    float2 n = make_float2(fmaf(cvs, v.x, -cbs * u.x), fmaf(cvs, v.y, -cbs * u.y));
                    if (p.fin.rmask) {                                  // per-source receiver sets
                        const int so = p.fin.colmap ? p.fin.colmap[s] : s;
                        if (so >= 0 && !p.fin.rmask[(size_t)r * p.fin.nb_out + so]) n = make_float2(0.f, 0.f);
                    }
                    p.U_bot[e] = n;
                    return (double)fmaf(n.x, n.x, n.y * n.y);
                },
                [](int) { return 0; });
        }

        // One tile, marched over its planes.  M_TMA / HAS_OLD are compile-time copies of p.m_tma and of
        // "the old-vector stream is present" so that the plane loop carries no such branches.  The
        // three centre planes (z-1, z, z+1) rotate through three register sets by NAME (the loop is
        // unrolled by three), the in-plane neighbour sum is overwritten after its use: no register
        // copies per plane.  |.|^2 is summed in fp32 over the <= 32 planes of the tile, then in fp64.
        auto run_tile = [&](auto m_tma_c, auto has_old_c, const int t, double (&acc)[2], int& chunk_out) {
            constexpr bool M_TMA = decltype(m_tma_c)::value, HAS_OLD = decltype(has_old_c)::value;
            int r = t;
            const int chunk = r % p.nchunk; r /= p.nchunk;
            const int tx = r % p.ntx; r /= p.ntx;
            const int ty = r % p.nty;
            const int tz = r / p.nty;
            const int z0 = tz * p.zc, z1 = min(z0 + p.zc, p.nz);
            const int col = chunk * CB + cp * 2;
            chunk_out = chunk;

            float w2[2], ca[2], cb[2], cv[2], cx[2], cw[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                w2[e] = tab_c[col + e]; ca[e] = tab_c[p.nb + col + e]; cb[e] = tab_c[2 * p.nb + col + e];
                cv[e] = tab_c[3 * p.nb + col + e];
                cx[e] = tab_c[4 * p.nb + col + e];
                cw[e] = tab_c[5 * p.nb + col + e];
            }
            int gsrc0 = -1, gsrc1 = -1;
            float2 gal0 = make_float2(0.f, 0.f), gal1 = gal0;
            if (MODE == MODE_G && p.gsrc) {
                gsrc0 = p.gsrc[col]; gsrc1 = p.gsrc[col + 1];
                gal0 = p.galpha[col]; gal1 = p.galpha[col + 1];
            }
            bool valid[IPT];
            float gxy[IPT], m_cur[IPT], m_nxt[IPT];
            size_t off[IPT];                                    // element offset of (cell, plane being emitted)
            int cell[IPT];                                      // its cell index
            float4 cA[IPT], cB[IPT], cC[IPT], n_cur[IPT];
#pragma unroll
            for (int j = 0; j < IPT; ++j) {
                const int ix = tx * TXC + cxj[j], iy = ty * TYC + cyj[j];
                valid[j] = ix < p.nx && iy < p.ny;
                const int ixc = min(ix, p.nx - 1), iyc = min(iy, p.ny - 1);
                gxy[j] = fmaxf(tab_g[ixc], tab_g[p.nx + iyc]);
                cell[j] = (z0 * p.ny + iyc) * p.nx + ixc;
                off[j] = (size_t)cell[j] * p.nb + col;
                m_cur[j] = 0.f;
                m_nxt[j] = 0.f;
                cA[j] = cB[j] = cC[j] = n_cur[j] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            float acc32[2] = {0.f, 0.f};
            const size_t plane_e = (size_t)p.nx * p.ny * p.nb;
            const int plane_m = p.nx * p.ny;
            const float* gz_tab = tab_g + p.nx + p.ny;

            // step pl: c_new <- centre of plane pl; emit plane pl-1 from (c_prev, c_cur, c_new, n_cur);
            // then n_cur <- in-plane neighbour sum of plane pl
            auto plane = [&](const int pl, float4 (&c_prev)[IPT], float4 (&c_cur)[IPT], float4 (&c_new)[IPT]) {
                if (!M_TMA && pl >= z0 && pl < z1) {
#pragma unroll
                    for (int j = 0; j < IPT; ++j) m_nxt[j] = __ldg(p.m + cell[j] + (pl > z0 ? plane_m : 0));
                }
                mbar_wait(full0 + 8 * stage, phase);
                const unsigned char* sb = stages + stage * STAGE_BYTES;
                float4 n_new[IPT], o_old[IPT], o_w[IPT], o_x[IPT];
                const bool emit = pl >= z0 + 1;
#pragma unroll
                for (int j = 0; j < IPT; ++j) {
                    c_new[j] = lds128(sb, sm_ctr[j]);
                    const float4 a = lds128(sb, sm_ctr[j] - CELL_B), b = lds128(sb, sm_ctr[j] + CELL_B);
                    const float4 c = lds128(sb, sm_ctr[j] - ROW_B), d = lds128(sb, sm_ctr[j] + ROW_B);
                    n_new[j] = make_float4((a.x + b.x) + (c.x + d.x), (a.y + b.y) + (c.y + d.y),
                                           (a.z + b.z) + (c.z + d.z), (a.w + b.w) + (c.w + d.w));
                    if (emit) {
                        const int io = Cfg::IN_SPAN + (tid + j * NT) * 16;
                        o_old[j] = HAS_OLD ? lds128(sb, io) : make_float4(0.f, 0.f, 0.f, 0.f);
                        if (M_TMA)
                            m_cur[j] = *reinterpret_cast<const float*>(sb + M_OFF + (cyj[j] * TXC + cxj[j]) * 4);
                    }
                }
                // pass A / G: the stage is free once its loads are done.  Pass F reads W and X from
                // the stage just before it uses them (fewer live registers) and releases it after.
                auto release = [&]() {
                    __syncwarp();
                    if ((tid & 31) == 0) mbar_arrive(empty0 + 8 * stage);
                    if (++stage == p.nstage) { stage = 0; phase ^= 1; }
                };
                if (MODE != MODE_F) release();

                if (emit) {
                    const float gzv = gz_tab[pl - 1];
#pragma unroll
                    for (int j = 0; j < IPT; ++j) {
                        const float g = fmaxf(gxy[j], gzv);
                        const float4 cc = c_cur[j];
                        // neighbour sums (x, y from this plane; z from the planes before / after)
                        const float s0 = n_cur[j].x + (c_prev[j].x + c_new[j].x);
                        const float s1 = n_cur[j].y + (c_prev[j].y + c_new[j].y);
                        const float s2 = n_cur[j].z + (c_prev[j].z + c_new[j].z);
                        const float s3 = n_cur[j].w + (c_prev[j].w + c_new[j].w);
                        if (MODE == MODE_G) {
                            // r = A u - q - alpha e;  |r|^2 sums;  g[c] += lam^2 sum_s w2_s (Re t + gamma Im t),
                            // t = conj(u) r  (= Re[conj((1 + i gamma) u) r], eq. 9 with this build's sponge)
                            float gterm = 0.f;
                            {
                                const float wm = w2[0] * m_cur[j];
                                const float dr = wm + p.m6ih2, di = wm * g;
                                float r_re = fmaf(p.ih2, s0, fmaf(dr, cc.x, -di * cc.y)) - o_old[j].x;
                                float r_im = fmaf(p.ih2, s1, fmaf(dr, cc.y, di * cc.x)) - o_old[j].y;
                                if (cell[j] == gsrc0) { r_re -= gal0.x; r_im -= gal0.y; }
                                if (valid[j]) acc32[0] += fmaf(r_re, r_re, r_im * r_im);
                                const float tr = fmaf(cc.x, r_re, cc.y * r_im), ti = fmaf(cc.x, r_im, -cc.y * r_re);
                                gterm = w2[0] * fmaf(g, ti, tr);
                            }
                            {
                                const float wm = w2[1] * m_cur[j];
                                const float dr = wm + p.m6ih2, di = wm * g;
                                float r_re = fmaf(p.ih2, s2, fmaf(dr, cc.z, -di * cc.w)) - o_old[j].z;
                                float r_im = fmaf(p.ih2, s3, fmaf(dr, cc.w, di * cc.z)) - o_old[j].w;
                                if (cell[j] == gsrc1) { r_re -= gal1.x; r_im -= gal1.y; }
                                if (valid[j]) acc32[1] += fmaf(r_re, r_re, r_im * r_im);
                                const float tr = fmaf(cc.z, r_re, cc.w * r_im), ti = fmaf(cc.z, r_im, -cc.w * r_re);
                                gterm = fmaf(w2[1], fmaf(g, ti, tr), gterm);
                            }
                            if (p.g) {
                                // the HP threads of one cell are consecutive lanes (HP is a power of two <= 32)
#pragma unroll
                                for (int dlt = HP >> 1; dlt > 0; dlt >>= 1)
                                    gterm += __shfl_down_sync(0xffffffffu, gterm, dlt, HP);
                                // pure store (no load in the pipeline's critical path): this batch's
                                // gradient goes to a scratch array, k_add_f32 accumulates it afterwards
                                if (cp == 0 && valid[j]) p.g[cell[j]] = p.lam2 * gterm;
                            }
                        } else {
                            float4 rr;
                            {
                                const float wm = w2[0] * m_cur[j];
                                const float dr = wm + p.m6ih2, di = p.sgn * wm * g;
                                const float ar = fmaf(p.ih2, s0, fmaf(dr, cc.x, -di * cc.y));
                                const float ai = fmaf(p.ih2, s1, fmaf(dr, cc.y, di * cc.x));
                                rr.x = fmaf(ca[0], ar, -cb[0] * o_old[j].x);
                                rr.y = fmaf(ca[0], ai, -cb[0] * o_old[j].y);
                            }
                            {
                                const float wm = w2[1] * m_cur[j];
                                const float dr = wm + p.m6ih2, di = p.sgn * wm * g;
                                const float ar = fmaf(p.ih2, s2, fmaf(dr, cc.z, -di * cc.w));
                                const float ai = fmaf(p.ih2, s3, fmaf(dr, cc.w, di * cc.z));
                                rr.z = fmaf(ca[1], ar, -cb[1] * o_old[j].z);
                                rr.w = fmaf(ca[1], ai, -cb[1] * o_old[j].w);
                            }
                            if (valid[j]) {
#if WRI_HINTS >= 1
                                stg128_hint(p.out + off[j], rr, pol_out);
#else
                                *reinterpret_cast<float4*>(p.out + off[j]) = rr;
#endif
                                acc32[0] += fmaf(rr.x, rr.x, rr.y * rr.y);
                                acc32[1] += fmaf(rr.z, rr.z, rr.w * rr.w);
                                if (MODE == MODE_F) {
                                    const int io = Cfg::IN_SPAN + (tid + j * NT) * 16;
                                    if (p.has_q) {
                                        o_w[j] = lds128(sb, io + Cfg::CTR_BYTES);
                                        o_x[j] = lds128(sb, io + 2 * Cfg::CTR_BYTES);
                                    } else {
                                        o_w[j] = o_x[j] = make_float4(0.f, 0.f, 0.f, 0.f);
                                    }
                                    float4 xn, wn;
                                    xn.x = fmaf(cx[0], o_w[j].x, o_x[j].x);
                                    xn.y = fmaf(cx[0], o_w[j].y, o_x[j].y);
                                    xn.z = fmaf(cx[1], o_w[j].z, o_x[j].z);
                                    xn.w = fmaf(cx[1], o_w[j].w, o_x[j].w);
                                    wn.x = fmaf(cv[0], cc.x, -cw[0] * o_w[j].x);
                                    wn.y = fmaf(cv[0], cc.y, -cw[0] * o_w[j].y);
                                    wn.z = fmaf(cv[1], cc.z, -cw[1] * o_w[j].z);
                                    wn.w = fmaf(cv[1], cc.w, -cw[1] * o_w[j].w);
#if WRI_HINTS >= 1
                                    stg128_hint(p.X + off[j], xn, pol_st);
                                    stg128_hint(p.W + off[j], wn, pol_st);
#else
                                    *reinterpret_cast<float4*>(p.X + off[j]) = xn;
                                    *reinterpret_cast<float4*>(p.W + off[j]) = wn;
#endif
                                }
                            }
                        }
                        off[j] += plane_e;
                        cell[j] += plane_m;
                    }
                }
                if (MODE == MODE_F) release();
#pragma unroll
                for (int j = 0; j < IPT; ++j) {
                    n_cur[j] = n_new[j];
                    if (!M_TMA) m_cur[j] = m_nxt[j];
                }
            };
            for (int pl = z0 - 1; pl <= z1; pl += 3) {
                plane(pl, cA, cB, cC);
                if (pl + 1 > z1) break;
                plane(pl + 1, cB, cC, cA);
                if (pl + 2 > z1) break;
                plane(pl + 2, cC, cA, cB);
            }
            acc[0] = (double)acc32[0];
            acc[1] = (double)acc32[1];
        };

        for (int t = blockIdx.x; t < p.n_tiles; t += gridDim.x) {
            double acc[2];
            int chunk;
            const bool has_old = (MODE == MODE_F) || p.has_q;
            if (p.m_tma) {
                if (has_old) run_tile(TrueT{}, TrueT{}, t, acc, chunk);
                else         run_tile(TrueT{}, FalseT{}, t, acc, chunk);
            } else {
                if (has_old) run_tile(FalseT{}, TrueT{}, t, acc, chunk);
                else         run_tile(FalseT{}, FalseT{}, t, acc, chunk);
            }
            // fold this tile's per-thread sums into the CTA's per-column sums, fixed order
            red[tid * 2] = acc[0];
            red[tid * 2 + 1] = acc[1];
            consumer_sync(NT);
            if (tid < CB) {
                const int e = tid & 1, c2 = tid >> 1;
                double s = 0.0;
#pragma unroll 4
                for (int k = 0; k < NT / HP; ++k) s += red[(c2 + k * HP) * 2 + e];
                colacc[chunk * CB + tid] += s;
            }
            consumer_sync(NT);
            if (MODE == MODE_A && own_nxt.z == t) {
                // P^T rows: the receivers inside the tile just written get  V += ct U_bot ; the
                // squared-norm sums are corrected by |V + ct U_bot|^2 - |V|^2.
                const int cnt = own_nxt.w, nb = p.nb;
                rows_by_columns<NT>(cnt, CB, tid, red, colacc,
                    [&](int i, int s) -> double {
                        const int4 en = (i == 0) ? own_nxt : __ldg(p.own + own_cur + i);
                        const int c = chunk * CB + s;
                        float2* vp = p.out + (size_t)en.y * nb + c;
                        const float2 v = __ldcg(vp);
                        const float2 u = __ldcg(p.U_bot + (size_t)en.x * nb + c);
                        const float cts = p.ct[c];
                        const float2 n = make_float2(fmaf(cts, u.x, v.x), fmaf(cts, u.y, v.y));
                        *vp = n;
                        return ((double)n.x * n.x + (double)n.y * n.y) - (double)fmaf(v.x, v.x, v.y * v.y);
                    },
                    [&](int) { return chunk * CB; });
                own_cur += cnt;
                own_nxt = (own_cur < own_end) ? __ldg(p.own + own_cur) : make_int4(-1, -1, -1, 0);
            }
        }
    }

    // ---------------------------------------------------------------------- CTA epilogue
    __syncthreads();
    if (p.partials)
        for (int j = tid; j < p.nb; j += blockDim.x) p.partials[(size_t)blockIdx.x * p.nb + j] = colacc[j];
    __threadfence();
    __syncthreads();
    if (tid == 0) s_ticket = atomicAdd(p.counter, 1u);
    __syncthreads();
    if (s_ticket == gridDim.x - 1) {
        __threadfence();
        double* sh = reinterpret_cast<double*>(smem);           // stages are idle now
        if (MODE != MODE_G && p.phase >= 0)                     // phase < 0: no scalar phase (operator application)
        switch (p.phase) {
            case PH_INIT_A: finalize_phase<PH_INIT_A>(p.fin, sh); break;
            case PH_F:      finalize_phase<PH_F>(p.fin, sh); break;
            default:        finalize_phase<PH_A>(p.fin, sh); break;
        }
        __syncthreads();
        if (tid == 0) *p.counter = 0u;
    }
}

}  // namespace wri
