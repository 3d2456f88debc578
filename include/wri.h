/*
 * wri.h — C ABI of libwri: batched LSQR on the data-augmented Helmholtz system of
 * 3D wavefield reconstruction inversion, hand-written CUDA for sm_100a (B200).
 *
 *   min_u || lambda (A(m) u - q) ||^2 + || P u - d ||^2          (eq. 4-6,
 *                                                                 source weight fixed: q = alpha e)
 *   A(m) = Laplacian_h + omega^2 diag(m) (1 + i gamma)            (2nd-order 7-point
 *                                                                 stencil + gamma sponge per
 *                                                                 BASELINE.json north_star)
 *   M = [lambda A ; P],  M^H = [lambda A^H , P^T],  P = sampling of receiver nodes
 *   solver: LSQR (Paige & Saunders 1982; "Algorithm 1"), batched over
 *   sources / frequencies ("grouping", eq. 12) with per-column scalars,
 *   tolerance and active mask.
 *
 * Conventions
 *   cell index       c = (iz*ny + iy)*nx + ix          (x fastest, z = depth), n_g = nx*ny*nz
 *   batched vectors  complex64 (float re, float im), source-interleaved: element (c, s) at
 *                    index c*nb + s, s = batch column; "c64 [n_g][nb]" below
 *   pointers         *_dev  = device memory on the context's GPU, 16-byte aligned;
 *                    *_host = host memory.  Nothing is a torch type.
 *   ownership        the caller owns every buffer it passes, including the workspace; the
 *                    library owns only the opaque context and a few KB of device scalars.
 *                    Inputs are never written.  Outputs must not alias inputs.
 *   execution        all work is enqueued on the CUDA stream given at wri_create; calls return
 *                    after enqueue (the *_host entry synchronises the stream before returning).
 *   errors           int return, 0 = WRI_OK, negative = error (table below); no exceptions,
 *                    no exit().  Numerical breakdown (b = 0, beta = 0, alpha = 0) is not an
 *                    error: the column stops (reading C-7).
 *   no CPU fallback  every entry that computes needs a CUDA device and fails with
 *                    WRI_ERR_CUDA without one.
 */
#ifndef WRI_H_
#define WRI_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define WRI_OK                    0
#define WRI_ERR_ARG              -1   /* null pointer, non-positive size, nb > nb_max, misaligned  */
#define WRI_ERR_RECEIVER_RANGE   -2   /* a receiver node lies outside the grid                     */
#define WRI_ERR_RECEIVER_DUP     -3   /* two receivers on one node (P^T must be a pure scatter)    */
#define WRI_ERR_WORKSPACE        -4   /* workspace missing or too small                            */
#define WRI_ERR_CUDA             -5   /* CUDA runtime error; text via wri_strerror                 */
#define WRI_ERR_STATE            -6   /* call out of order (e.g. iterate before begin)             */
#define WRI_ERR_NUMERIC          -7   /* wri_awri_step: the objective at the current model is not finite */
#define WRI_ERR_SCRATCH_LIMIT    -8   /* wri_objective_gradient_static: needs more than WRI_STATIC_SCRATCH_BYTES */

typedef struct wri_ctx wri_ctx;                 /* opaque, library-owned */

typedef struct { int32_t nx, ny, nz; } wri_grid;

/* Sponge: gamma(ix,iy,iz) = gamma_max * ( max(dx,dy,dz) / width )^power,
 * d_axis(i) = max(width - i, i - (n_axis-1-width), 0) on the listed faces (reading C-4).   */
typedef struct {
    int32_t  width;       /* cells; 0 = no sponge                                   */
    float    gamma_max;   /* 1.0 in BASELINE.json configs                            */
    int32_t  power;       /* 2 = quadratic                                           */
    uint32_t faces;       /* bit0..5 = x-,x+,y-,y+,z-,z+ ; 0x3F = all six            */
} wri_sponge;

/* wri_create — build a context for one grid / model / receiver set (north_star:
 * "wri_create(grid,h,omega,m,sponge,receivers)").
 *   omega_host   [n_omega] angular frequencies (rad/s); a batch column picks one by index
 *   m_dev        [n_g] float32 squared slowness (s^2/m^2), BORROWED until wri_set_model/destroy
 *   rec_ijk_host [n_rec][3] = (ix,iy,iz) receiver nodes; validated before any CUDA call:
 *                out of range -> WRI_ERR_RECEIVER_RANGE, duplicates -> WRI_ERR_RECEIVER_DUP
 *   nb_max       largest batch width later calls may use
 *   cuda_stream  cudaStream_t (NULL = default stream)                                        */
int wri_create(wri_ctx** out, wri_grid grid, double h,
               int32_t n_omega, const double* omega_host,
               const float* m_dev, wri_sponge sponge,
               int32_t n_rec, const int32_t* rec_ijk_host,
               int32_t nb_max, void* cuda_stream);

/* m changes every outer iteration of the inversion (Algorithm 2). */
int wri_set_model(wri_ctx* ctx, const float* m_dev);

/* Discretisation of the Laplacian in A(m) (PAPER.md:56 says only "discretized 3D Laplacian"; readings
 * C-3 and C-23 of DESIGN.md), sticky for every later call of the context:
 *   WRI_STENCIL_7   2nd-order 7-point star (north_star; the default)
 *   WRI_STENCIL_27  2nd-order 27-point box with an isotropic leading error term: centre -128/30, the
 *                   6 face neighbours 14/30, the 12 edge neighbours 3/30, the 8 corner neighbours 1/30,
 *                   all over h^2; zero (Dirichlet) outside the grid, so A stays complex-symmetric.
 * The mass term omega^2 m (1 + i gamma) stays on the diagonal.  Same bytes per iteration as the
 * 7-point stencil (the halo is still one cell).                                                  */
#define WRI_STENCIL_7  0
#define WRI_STENCIL_27 1
int wri_set_stencil(wri_ctx* ctx, int32_t stencil);

/* Tuning and test switches of the kernels behind the entries (all zero = the library's own choices;
 * NULL restores that).  Results do not depend on them beyond rounding order, except that no_compact /
 * no_groups / generic select code paths whose results the tests compare with the default ones.
 *   nstage_f / nstage_a   depth of the shared-memory ring of the forward / adjoint pass
 *   zc_f / zc_a           planes per tile
 *   txc / tyc             cells per tile in x / y
 *   no_compact            keep converged columns in the working set (they stay frozen, no re-packing)
 *   no_groups             run a batch wider than 64 columns in lock-step instead of 64-column groups
 *   generic               use the plain (non-TMA) kernels for every width
 *   m_ldg_f               pass F reads the model by plain loads (1) / through its TMA stage (2)     */
typedef struct {
    int32_t nstage_f, nstage_a, zc_f, zc_a, txc, tyc;
    int32_t no_compact, no_groups, generic, m_ldg_f;
} wri_debug_opts;
int wri_set_debug_opts(wri_ctx* ctx, const wri_debug_opts* opts);

/* Tile plan the pass kernel would use for batch width nb (introspection for bench.py and the tuning
 * tables under profiles/): out16 = { column chunk, chunks per cell, cells per tile in x, in y, consumer
 * threads with work, merged tensor maps, model tile by TMA, pass F: planes per tile, ring depth, tiles,
 * pass A: planes per tile, ring depth, tiles, bytes per stage of pass F, of pass A, persistent grid }.
 * WRI_ERR_ARG when the width is served by the generic kernels (odd widths).                        */
int wri_plan_info(wri_ctx* ctx, int32_t nb, int32_t* out16);

/* Workspace for wri_lsqr_* and wri_objective_gradient at batch width nb (u, v, w vectors, receiver
 * rows, reduction partials, one float32 [n_g] gradient scratch per power-of-two column chunk of the
 * gradient pass: 1 for 64 columns, 3 for 48 or 192).  flags: WRI_WS_HOST_STAGING adds room for the device copies wri_lsqr_batch_host
 * needs; WRI_WS_COMPACTION adds six more vectors: with per-column tolerances the working set then
 * lives entirely in the workspace, has a second vector set and a side buffer, so that converged columns can be
 * compacted out of it on the device (without it such a solve still stops early once every column
 * has converged, but converged columns keep costing bandwidth).  An odd batch width is given one
 * spare vector (two with host staging) whatever the flags: wri_lsqr_batch runs it in an even-width
 * working set on the fast kernel.
 * The caller allocates (e.g. a torch uint8 tensor) and hands it over; it must stay alive and
 * untouched while a solve is in flight.                                                      */
#define WRI_WS_HOST_STAGING 1
#define WRI_WS_COMPACTION   2
size_t wri_workspace_bytes(const wri_ctx* ctx, int32_t nb, int32_t flags);
int    wri_set_workspace(wri_ctx* ctx, void* ws_dev, size_t bytes);

/* y = M x: ytop = lambda * A x  (c64 [n_g][nb]),  ybot = x at the receiver
 * nodes (c64 [n_rec][nb], exact copies).  omega_idx_host [nb] (NULL = all 0).  No workspace. */
int wri_apply_M(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, float lambda,
                const void* x_dev, void* ytop_dev, void* ybot_dev);

/* x = M^H y = lambda * A^H ytop + P^T ybot  (conjugate transpose, reading C-2). */
int wri_apply_MH(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, float lambda,
                 const void* ytop_dev, const void* ybot_dev, void* x_dev);

/* wri_lsqr_batch — nb independent LSQR solves, b_s = [lambda q_s ; d_s], x0 = 0.  Up to 64 columns run in
 * lock-step (two kernel launches per iteration for all of them); a wider batch whose width is a multiple
 * of 64 is worked through as successive 64-column groups, each in a compact working set inside the same
 * workspace (columns are independent systems, so a column's result does not depend on the grouping).
 *   q_dev        c64 [n_g][nb]     d_dev  c64 [n_rec][nb]
 *   tol_dev      float [nb] or NULL; column s stops at the first k with
 *                ||M^H r_k|| / ||M^H b|| <= tol_s  (LSQR's running estimate, reading C-6);
 *                tol_s <= 0 (or NULL) runs exactly maxit iterations
 *   u_out_dev    c64 [n_g][nb]     the wavefields x_k at each column's stop iteration
 *   resnorms_dev float [maxit+1][nb]: ||b - M x_k|| for k = 0..maxit, held at the last value
 *                after a column stops (reading C-9); may be NULL (no history wanted)
 *   iters_dev    int32 [nb] iterations performed per column (may be NULL)
 * Equivalent to wri_lsqr_begin + wri_lsqr_iterate(maxit) + wri_lsqr_end.  Needs a workspace.
 * The call only enqueues work, with or without tolerances: the state of the solve (iteration
 * count, active flags, working width) lives on the device.  With tolerances the finaliser of
 * each iteration counts the live columns; as soon as they fit a narrower (even) width, the two
 * passes of the next iteration store their results into a second vector set at that width, so
 * stopped columns leave the working set without a separate pass over the vectors (adaptive
 * accuracy; "the active mask shrinking as sources converge", BASELINE.json
 * configs[3]); once every column has stopped the remaining launches return at once.  A column's
 * result does not depend on the batch it runs in (bit-identical with and without re-packing). */
int wri_lsqr_batch(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                   const void* q_dev, const void* d_dev, float lambda,
                   const float* tol_dev, int32_t maxit,
                   void* u_out_dev, float* resnorms_dev, int32_t* iters_dev);

/* ---- Source-free system (the system the paper states, eq. 4-6) ---------------
 *
 *     S = [ lambda A   -lambda e ]      x = [ u     ]      b = [ lambda q ]   (paper: q = 0)
 *         [ P           0        ]          [ alpha ]          [ d        ]
 *
 * The source weight alpha of every column is one more complex unknown; e is the real unit
 * vector at that column's source node.  S^H y = [lambda A^H y_top + P^T y_bot ;
 * -lambda y_top[src]].  All norms run over the stacked vectors including the alpha entry.
 *   src_ijk_host  [nb][3] = (ix,iy,iz) source node per batch column (columns of one source at
 *                 several frequencies repeat it); outside the grid -> WRI_ERR_ARG
 *   xalpha / alpha_out   c64 [nb], device
 *   q_dev         may be NULL (the paper's b = [0; d]); given, it is a known part of the source
 * wri_apply_S / wri_apply_SH are the operator entries; wri_lsqr_sf_* mirror wri_lsqr_* (same
 * stop rule, histories, compaction, stepping through wri_lsqr_iterate / _end / _peek), and
 * alpha_out_dev receives the source-weight estimate of x_k (the paper's on-the-fly source
 * estimation).                                                                    */
int wri_apply_S (wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                 float lambda, const void* x_dev, const void* xalpha_dev, void* ytop_dev, void* ybot_dev);
int wri_apply_SH(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                 float lambda, const void* ytop_dev, const void* ybot_dev, void* x_dev, void* xalpha_dev);
int wri_lsqr_sf_batch(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                      const void* q_dev, const void* d_dev, float lambda, const float* tol_dev,
                      int32_t maxit, void* u_out_dev, void* alpha_out_dev, float* resnorms_dev,
                      int32_t* iters_dev);
int wri_lsqr_sf_begin(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                      const void* q_dev, const void* d_dev, float lambda, const float* tol_dev,
                      int32_t maxit, void* u_out_dev, void* alpha_out_dev, float* resnorms_dev,
                      int32_t* iters_dev);
int wri_lsqr_sf_batch_host(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                           const int32_t* src_ijk_host, const void* q_host, const void* d_host,
                           float lambda, const float* tol_host, int32_t maxit, void* u_out_host,
                           void* alpha_out_host, float* resnorms_host, int32_t* iters_host);

/* Objective and gradient of the reduced problem at given wavefields (eq. 4,
 * 98-110 eq. 8-9; "does not involve additional PDE solvers"), per batch column s:
 *     r_s       = A u_s - q_s - alpha_s e_s
 *     f_pde[s]  = 1/2 lambda^2 || r_s ||^2          f_data[s] = 1/2 || P u_s - d_s ||^2
 *     g[c]     += sum_s lambda^2 omega_s^2 Re[ conj((1 + i gamma_c) u_cs) r_cs ]
 * f_pde + f_data = f2 of eq. 4 (= 1/2 ||S x - b||^2, eq. 5); g is eq. 9 with dA/dm_c =
 * omega^2 (1 + i gamma_c) of this build's sponge (equal to the printed formula where gamma = 0;
 * the real part is implied, m is real).  The sum over the batch is the paper's sum over sources
 * and frequencies; g_dev (float32 [n_g]) is ACCUMULATED so that several batches add up — clear
 * it first; NULL skips the gradient.  src_ijk_host/alpha_dev (c64 [nb]) and q_dev are each
 * optional: the source-free solve passes the first pair, the known-source solve passes q_dev.
 * f_pde_dev, f_data_dev: double [nb].  Needs a workspace; nb <= 1024.  Bit-reproducible.       */
int wri_objective_gradient(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                           const int32_t* src_ijk_host, const void* alpha_dev, const void* q_dev,
                           const void* u_dev, const void* d_dev, float lambda,
                           double* f_pde_dev, double* f_data_dev, float* g_dev);

/* wri_objective_gradient without a workspace and without any device allocation, for callers that may
 * not call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it).
 * Same operation, arguments, outputs and accumulation rule as wri_objective_gradient (eq. 4, eq. 8-9,
 * PAPER.md:71-76, 98-110); every width runs the generic gradient kernel, whose per-tile column sums of
 * |r|^2 go to a scratch array that is part of the library image: WRI_STATIC_SCRATCH_BYTES of device
 * memory on every GPU that loads the library, held until the process exits.  The scratch need is
 * (number of thread-block tiles) x nb doubles; the tiles are made taller until that fits, and a case
 * that does not fit even with tiles as tall as the grid (128^3 x 64, 256^3 x 64 and 200 x 200 x 160 x 48
 * fit; 128^3 x 192 and wider do not) is refused with WRI_ERR_SCRATCH_LIMIT before anything is
 * launched or written.  The call does no cudaMalloc / cudaFree and calls no
 * allocating library routine; it needs no wri_set_workspace.  Like every entry it must be called with
 * the context's GPU current: the array's device address is looked up for the current device
 * (cudaGetSymbolAddress, once per device).  As in wri_objective_gradient, the per-column tables (omega^2,
 * lambda, source cells; a few KB) go host -> device by cudaMemcpyAsync into buffers the context already
 * owns, so the call itself is not capturable into a CUDA graph as it stands.  Nothing in the scratch has to start at
 * zero (every entry that is read is written first by the same call).  ALL calls on one GPU share the
 * array, whatever their context or stream: calls that can overlap on the GPU (different streams,
 * different contexts, different host threads without ordering) race on it and return garbage sums —
 * order them on one stream or with events.  f_pde / f_data agree with wri_objective_gradient to
 * double rounding of a differently grouped sum, g to float rounding (the power-of-two widths use
 * another kernel there).                                                                          */
#define WRI_STATIC_SCRATCH_BYTES (4u << 20)
int wri_objective_gradient_static(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                                  const int32_t* src_ijk_host, const void* alpha_dev, const void* q_dev,
                                  const void* u_dev, const void* d_dev, float lambda,
                                  double* f_pde_dev, double* f_data_dev, float* g_dev);

/* Per-source receiver sets P_i ("P_i is the restriction operator for source i").
 * mask_dev: uint8 [n_rec][nb], 1 = receiver r records batch column s, 0 = that row is absent from
 * P_s: its entry of P_s v is 0, its datum d[r][s] is ignored, P_s^T adds nothing there.  Sticky for
 * every later call of batch width nb (apply, solve, objective / gradient, misfit); other widths are
 * refused with WRI_ERR_ARG while a mask is set; NULL restores "every receiver records every column"
 * (the default, north_star's shared P).  The array is BORROWED: it must stay valid and unchanged
 * while calls that use it are in flight.                                                        */
int wri_set_receiver_mask(wri_ctx* ctx, int32_t nb, const uint8_t* mask_dev);

/* Options of the solves that follow (all wri_lsqr_* / wri_lsqr_sf_* begin and batch entries);
 * sticky until set again, NULL restores the defaults (all zero).
 *   warm_start   1: u_out_dev (and alpha_out_dev) hold x0 (alpha0) on entry.  Algorithm 1 leaves
 *                x0 free; the solve runs LSQR on the residual system
 *                r0 = b - S x0 and accumulates into x0, so x_k = x0 + dx_k and resnorms[k] =
 *                ||b - S x_k|| of the original system.  Used to re-solve after a model update
 *                or with a tighter tolerance (Algorithm 2).
 *   ar_ref_dev   double [nb] or NULL: reference of the stop rule, ||S^H r_k|| <= tol * ar_ref
 *                (default: this solve's own alpha1*beta1 = ||S^H r0||).  A warm start passes the
 *                cold solve's value so that tol keeps its meaning (reading C-17).
 *   ar0_out_dev  double [nb] or NULL: receives alpha1*beta1 of the solve.
 * The device arrays must stay valid while a solve is in flight.                                  */
typedef struct {
    int32_t       warm_start;
    const double* ar_ref_dev;
    double*       ar0_out_dev;
} wri_lsqr_opts;
int wri_lsqr_set_opts(wri_ctx* ctx, const wri_lsqr_opts* opts);

/* ---- Misfit evaluation and the adaptive outer step (Algorithm 2) -------------
 *
 * wri_misfit_sf — one misfit evaluation of the source-free problem for a group of nb columns
 * ("a single misfit function calculation", the unit of the paper's Table 1):
 *     x_bar_s = argmin || S_s x - [0; d_s] ||   by LSQR, every column to the tolerance eps (eq. 7)
 *     f_pde[s], f_data[s], g += ...             as wri_objective_gradient at (u_bar, alpha_bar) (eq. 8-9)
 *   eps        LSQR tolerance of every column (0: exactly maxit iterations)
 *   warm       1: u_dev / alpha_dev hold a start point and ar0_dev the cold solve's alpha1*beta1
 *              (the stop rule stays relative to it, reading C-17); 0: cold solve, ar0_dev (may be
 *              NULL) receives alpha1*beta1
 *   u_dev      c64 [n_g][nb], alpha_dev c64 [nb]: the minimisers on return
 *   g_dev      float [n_g], ACCUMULATED (clear it first), or NULL for the objective alone
 *   iters_dev  int32 [nb] or NULL
 *   f_host     HOST double or NULL: sum_s (f_pde + f_data), summed in column order; asking for it
 *              synchronises the stream.  The call then blocks until the result is there anyway, so
 *              with eps > 0 it enqueues its solve only 16 iterations ahead of the device (which
 *              reports its progress in a word of mapped host memory) and stops once every column
 *              has stopped, instead of enqueuing all maxit iterations; same results, and the
 *              1-3 ms of launches that would each return at once are not paid.  wri_awri_step and
 *              the host-buffer solves with tolerances (wri_lsqr_batch_host, wri_lsqr_sf_batch_host)
 *              do the same.  The device-buffer solves enqueue everything and return.
 * Needs a workspace (with WRI_WS_COMPACTION room converged columns are compacted away).
 *
 * wri_awri_step — lines 4-14 of Algorithm 2 for one group of columns and the model in m_dev:
 *     4-5  x_bar, f, g at m with tolerance eps            7-8  x_tilde, f_tilde at m_tilde
 *     6    m_tilde = update(m, g)                          9-11 f_tilde > f: eps <- eps/2, back to 4
 *                                                          13   else m <- m_tilde
 * The quasi-Newton direction of line 6 is the caller's (l-BFGS is outside this library):
 * opts->update(user, m_dev, g_dev, m_trial_dev, cuda_stream) must ENQUEUE the computation of
 * m_trial on the given stream and return 0; with update == NULL the built-in steepest-descent
 * update m_tilde = clamp(m - step * g, m_min, m_max) is used.  Algorithm 2 does not bound the
 * "go back" loop: after max_halvings halvings the step is reported as rejected and m_dev is left
 * unchanged (reading C-20).  A trial objective that is not finite counts as a rejected step; a
 * non-finite objective at the current model returns WRI_ERR_NUMERIC with m_dev unchanged.  warm_restart = 1 continues the re-solve of line 4 from x_bar.
 * The comparison of line 9 is made on the host in double (one stream synchronisation per
 * evaluation).  During the call the context's model pointer is switched between m_dev and
 * m_trial_dev and restored on return.
 *   m_dev        float [n_g]: m^(k) on entry, m^(k+1) on return if accepted
 *   m_trial_dev  float [n_g] scratch (the last trial model on return)
 *   g_dev        float [n_g]: gradient at m^(k) with the final eps (overwritten)
 *   u_dev, alpha_dev / u_trial_dev, alpha_trial_dev   wavefields and source weights at m^(k) / m_tilde
 *   f_cols_dev   double [2][nb]: f_pde | f_data per column at m^(k)
 *   report       HOST                                                                          */
#define WRI_AWRI_MAX_TRACE 16
typedef int (*wri_update_fn)(void* user, const float* m_dev, const float* g_dev, float* m_trial_dev,
                             void* cuda_stream);
/* Sum over ranks (column sharding): eq. 8-9 are sums over all sources and frequencies.
 * reduce(user, f_host, g_dev, n_g, cuda_stream) must replace *f_host (HOST double) by its sum over the
 * ranks and, when g_dev is not NULL, ENQUEUE on the given stream the all-reduce of the float32 [n_g]
 * gradient; return 0.  Every rank then holds the same f, f_tilde and g, and takes the same decision. */
typedef int (*wri_reduce_fn)(void* user, double* f_host, float* g_dev, int64_t n_g, void* cuda_stream);
typedef struct {
    int32_t       max_halvings;     /* < WRI_AWRI_MAX_TRACE                                      */
    int32_t       warm_restart;
    wri_update_fn update;           /* NULL: built-in steepest descent with the fields below     */
    void*         user;
    float         step, m_min, m_max;
    wri_reduce_fn reduce;           /* NULL: this process holds every column                     */
} wri_awri_opts;
typedef struct {
    int32_t accepted, n_halvings, n_trace;
    float   eps;                    /* tolerance in force at the end                              */
    double  f, f_trial;             /* of the last round                                          */
    int64_t lsqr_iters;             /* column iterations spent by all solves of the step          */
    float   trace_eps[WRI_AWRI_MAX_TRACE];
    double  trace_f[WRI_AWRI_MAX_TRACE], trace_f_trial[WRI_AWRI_MAX_TRACE];
} wri_awri_report;
int wri_misfit_sf(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                  const void* d_dev, float lambda, float eps, int32_t maxit, int32_t warm,
                  void* u_dev, void* alpha_dev, double* ar0_dev, double* f_pde_dev, double* f_data_dev,
                  float* g_dev, int32_t* iters_dev, double* f_host);
int wri_awri_step(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host, const int32_t* src_ijk_host,
                  const void* d_dev, float lambda, float eps, int32_t maxit, const wri_awri_opts* opts,
                  float* m_dev, float* m_trial_dev, float* g_dev, void* u_dev, void* alpha_dev,
                  void* u_trial_dev, void* alpha_trial_dev, double* f_cols_dev, wri_awri_report* report);

/* Same solve with HOST buffers: copies q, d (and tol) to the device, solves, copies u_out,
 * resnorms and iters back, then synchronises the stream.  Needs a workspace sized with
 * host_staging = 1.  Pinned host memory makes the copies asynchronous but is not required.   */
int wri_lsqr_batch_host(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                        const void* q_host, const void* d_host, float lambda,
                        const float* tol_host, int32_t maxit,
                        void* u_out_host, float* resnorms_host, int32_t* iters_host);

/* Pipelined host-buffer solves.  An inversion walks through many source groups / frequencies
 * (PAPER.md:221); with HOST buffers the copies of one solve (q in, u out: 2 x n_g*nb*8 bytes) can
 * ride under the neighbouring solves: while solve i runs, the inputs of solve i+1 are uploaded and
 * the results of solve i-1 downloaded, on two copy streams of the library's own.
 *   wri_host_pipeline_bytes / wri_set_host_pipeline   two staging slots (q, d, x, tol, history per
 *                slot) in a device buffer the caller allocates for batch widths up to nb; NULL drops it
 *   wri_lsqr_batch_host_async / wri_lsqr_sf_batch_host_async   same arguments and results as the
 *                _host entries, but the call returns once everything is ENQUEUED (with tolerances:
 *                once the solve itself has finished); the host buffers — PINNED memory, or nothing
 *                overlaps — must stay valid, and the outputs must not be read, until wri_host_wait
 *   wri_host_wait   blocks until every enqueued solve has delivered its results
 * Solves still execute one after the other on the context's stream, so results are those of the
 * _host entries bit for bit.  Call wri_host_wait before using any other entry of the context.   */
size_t wri_host_pipeline_bytes(const wri_ctx* ctx, int32_t nb);
int    wri_set_host_pipeline(wri_ctx* ctx, int32_t nb, void* buf_dev, size_t bytes);
int    wri_lsqr_batch_host_async(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                                 const void* q_host, const void* d_host, float lambda,
                                 const float* tol_host, int32_t maxit,
                                 void* u_out_host, float* resnorms_host, int32_t* iters_host);
int    wri_lsqr_sf_batch_host_async(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                                    const int32_t* src_ijk_host, const void* q_host, const void* d_host,
                                    float lambda, const float* tol_host, int32_t maxit, void* u_out_host,
                                    void* alpha_out_host, float* resnorms_host, int32_t* iters_host);
int    wri_host_wait(wri_ctx* ctx);

/* Stepping form of the same solve (outer drivers, teacher-forced parity tests).
 *   begin   : Golub-Kahan start  beta1 u1 = b, alpha1 v1 = M^H u1, w1 = v1, x0 = 0
 *   iterate : n_steps more iterations (total must not exceed maxit)
 *   end     : applies the last deferred x update; u_out/resnorms/iters are final afterwards  */
int wri_lsqr_begin(wri_ctx* ctx, int32_t nb, const int32_t* omega_idx_host,
                   const void* q_dev, const void* d_dev, float lambda,
                   const float* tol_dev, int32_t maxit,
                   void* u_out_dev, float* resnorms_dev, int32_t* iters_dev);
int wri_lsqr_iterate(wri_ctx* ctx, int32_t n_steps);
int wri_lsqr_end(wri_ctx* ctx);

/* Device-side LSQR state between wri_lsqr_iterate calls (valid after the stream is synced).
 * The vectors are stored UN-normalised (lazy normalisation):
 *   after k iterations: u_{k+1} = U / beta, v_{k+1} = V / alpha, W = w_k, X = x_{k-1}; the
 *   updates x_k = X + cx * W and w_{k+1} = V/alpha - cw * W are applied by the next iteration
 *   (x_k also by wri_lsqr_end).
 * Pointers are into the caller's workspace / u_out buffer and the context's scalar block.    */
typedef struct {
    int32_t nb, k;                   /* working batch width (shrinks when converged columns   */
                                     /* are compacted away), iterations enqueued so far       */
    const void*   U_top;             /* c64 [n_g][nb]                                          */
    const void*   U_bot;             /* c64 [n_rec][nb]                                        */
    const void*   V;                 /* c64 [n_g][nb]                                          */
    const void*   W;                 /* c64 [n_g][nb]                                          */
    const void*   X;                 /* c64 [n_g][nb] (= u_out_dev)                            */
    const double* alpha;             /* [nb] each, device                                      */
    const double* beta;
    const double* rhobar;
    const double* phibar;
    const double* ar0;               /* alpha1 * beta1                                         */
    const float*  cx;                /* [nb] pending x-update coefficient phi_k/rho_k          */
    const float*  cw;                /* [nb] pending w-update coefficient theta_{k+1}/rho_k:   */
                                     /*      w_{k+1} = V/alpha - cw * W                        */
    const int32_t* active;           /* [nb] 1 while the column iterates                       */
    const int32_t* iters;            /* [nb]                                                   */
    int32_t nb_max;                  /* row stride of sf_state                                 */
    const double* sf_state;          /* source-free solves (else NULL): [6][nb_max] rows        */
                                     /* Re v_a, Im v_a, Re w_a, Im w_a, Re x_a, Im x_a — the     */
                                     /* alpha entries of V (un-normalised like V), of w_{k+1}   */
                                     /* and of x_k (these two are NOT deferred)                 */
} wri_lsqr_view;
int wri_lsqr_peek(const wri_ctx* ctx, wri_lsqr_view* view);

/* Kernels launched by this context since creation (bench.py's gpu_launches). */
int64_t wri_launch_count(const wri_ctx* ctx);

/* Per-kernel timing for the roofline report: while enabled, the two stencil passes of every
 * LSQR iteration are bracketed by CUDA events on the context's stream.  wri_profile_read
 * synchronises the stream and returns, for pass F (forward operator + x/w update) and pass A
 * (adjoint operator) since the last read: the summed durations (ms), the launch counts and the
 * summed working batch widths of those launches (so that bytes moved = bytes per cell-column
 * x n_g x cols even when compaction narrows the batch); then resets the counters.           */
int wri_profile_enable(wri_ctx* ctx, int32_t on);
int wri_profile_read(wri_ctx* ctx, double* ms_pass_f, int64_t* n_pass_f, int64_t* cols_pass_f,
                     double* ms_pass_a, int64_t* n_pass_a, int64_t* cols_pass_a);

int wri_destroy(wri_ctx* ctx);

/* Static text for an error code; for WRI_ERR_CUDA the last CUDA error string seen. */
const char* wri_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* WRI_H_ */
