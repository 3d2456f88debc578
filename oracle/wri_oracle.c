/*
 * wri_oracle.c — TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, complex128 CPU oracle for the hot path of 3D wavefield
 * reconstruction inversion: the stacked operator M = [lambda*A ; P], its adjoint,
 * and LSQR on  min_u || lambda (A u - q) ||^2 + || P u - d ||^2 .
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may call this.  It shares no code, header, table or helper
 * with the CUDA path under paper_2410_18429_b200/.
 *
 * What each function follows:
 *   ref_gamma      sponge profile: BASELINE.json configs[0] ("gamma rising
 *                  quadratically from 0 to 1"), reading C-4.
 *   ref_apply_A    A = omega^2 diag(m)(1+i gamma) + Laplacian
 *                  ("A_j(m) = omega_j^2 diag(m) + Delta"); 2nd-order 7-point
 *                  stencil and the (1+i gamma) sponge are fixed by
 *                  BASELINE.json north_star; zero (Dirichlet) outside the grid,
 *                  DESIGN.md reading C-3.  op->stencil = 1 selects the 27-point
 *                  box discretisation of the same Laplacian (SURVEY.md §8(f)
 *                  NEXT-4, reading C-23), written out as its definition.
 *   ref_apply_M    M v = [lambda A v ; P v], PAPER.md:78-85 (eq. 5-6) with the
 *                  source weight fixed (reading C-5); P = sampling of receiver
 *                  nodes.
 *   ref_apply_MH   M^H y = lambda A^H y_top + P^T y_bot (PAPER.md:95, 118 write
 *                  "T"; conjugate transpose is meant, reading C-2).  A and A^H
 *                  share one stencil routine (apply_A_impl) with a flag that
 *                  conjugates the diagonal; the adjoint dot test and
 *                  test_adjoint_of_A_alone_and_symmetry pin that flag.
 *   ref_lsqr       Paige & Saunders (1982) LSQR, the algorithm the paper names
 *                  and cites.  Algorithm 1 as
 *                  printed is garbled (reading C-1); the recurrences below are
 *                  the standard ones in the standard order.
 *   ref_lsqr_step  exactly one iteration of the loop body of ref_lsqr on a
 *                  caller-supplied state (for teacher-forced parity).
 *
 * Index conventions: cell c = (iz*ny + iy)*nx + ix  (x fastest, z = depth).
 * One column (one source/frequency) per call; complex numbers are C99
 * double complex (re, im pairs in memory).
 *
 * Pins (tests/test_oracle_*.py; the source-free and gradient functions at the
 * end of this file list theirs in their own headers): adjoint dot test, closed-form eigenpairs
 * (periodic plane wave, Dirichlet sine modes), printed sponge values, dense
 * LAPACK least squares on 8^3, SciPy LSQR, CGLS, estimate-vs-true residuals,
 * monotone ||r||, consistent system, breakdown cases.  27-point stencil
 * (tests/test_oracle_stencil27.py): closed-form symbol on the periodic box and on
 * Dirichlet sine modes, second-order convergence to the continuous Laplacian,
 * dot test, dense least squares.  round_c64 (tests/test_oracle_c64floor.py):
 * flag off is bit-identical to the plain solver; with it the iterates stay
 * within float32 rounding of the plain ones on a well-conditioned problem.
 * Unpinned: nothing in this file.  (Free-running complex64-vs-complex128
 * agreement on configs[0] is a property of the problem, C-12.)
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef double complex zc;

typedef struct {
    int32_t nx, ny, nz;
    double h;            /* grid spacing (m)                                  */
    double omega;        /* angular frequency (rad/s)                         */
    int32_t sponge_width;/* L, cells                                          */
    double gamma_max;
    int32_t power;       /* exponent of the profile                           */
    uint32_t faces;      /* bit0..5 = x-,x+,y-,y+,z-,z+                        */
    int32_t periodic;    /* TEST ONLY: wrap neighbours (closed-form pin P2a)  */
    int32_t stencil;     /* 0: 7-point star (north_star); 1: 27-point box, reading C-23 */
    int32_t round_c64;   /* TEST ONLY: LSQR keeps u, v, w, x in complex64 STORAGE (rounded
                          * after every step; all arithmetic stays complex128) — the
                          * attainable floor of a complex64 solver, SURVEY C-12(iii)       */
} ref_op;

/* depth into the sponge along one axis, in cells: max(L - i, i - (n-1-L), 0)
 * on the listed faces (reading C-4). */
static double sponge_depth(int i, int n, int L, int lo_on, int hi_on) {
    double d = 0.0;
    if (lo_on && (double)(L - i) > d) d = (double)(L - i);
    if (hi_on && (double)(i - (n - 1 - L)) > d) d = (double)(i - (n - 1 - L));
    return d;
}

/* gamma[c] = gamma_max * ( max(dx,dy,dz) / L )^p */
void ref_gamma(const ref_op *op, double *gamma) {
    const int nx = op->nx, ny = op->ny, nz = op->nz, L = op->sponge_width;
    for (int iz = 0; iz < nz; ++iz)
        for (int iy = 0; iy < ny; ++iy)
            for (int ix = 0; ix < nx; ++ix) {
                double g = 0.0;
                if (L > 0) {
                    double dx = sponge_depth(ix, nx, L, op->faces & 1u, op->faces & 2u);
                    double dy = sponge_depth(iy, ny, L, op->faces & 4u, op->faces & 8u);
                    double dz = sponge_depth(iz, nz, L, op->faces & 16u, op->faces & 32u);
                    double d = dx;
                    if (dy > d) d = dy;
                    if (dz > d) d = dz;
                    g = op->gamma_max * pow(d / (double)L, (double)op->power);
                }
                gamma[((size_t)iz * ny + iy) * nx + ix] = g;
            }
}

/* neighbour value with the boundary rule: zero outside, or wrap if periodic */
static zc nb(const ref_op *op, const zc *v, int ix, int iy, int iz) {
    const int nx = op->nx, ny = op->ny, nz = op->nz;
    if (op->periodic) {
        ix = (ix + nx) % nx;
        iy = (iy + ny) % ny;
        iz = (iz + nz) % nz;
    } else if (ix < 0 || ix >= nx || iy < 0 || iy >= ny || iz < 0 || iz >= nz) {
        return 0.0;
    }
    return v[((size_t)iz * ny + iy) * nx + ix];
}

/* y = A v  (conj_diag = 0)   or   y = A^H v  (conj_diag = 1).
 * The Laplacian part is real and symmetric under either boundary rule; the
 * only complex entries of A are on its diagonal, so A^H differs from A by
 * conjugating the diagonal. */
static void apply_A_impl(const ref_op *op, const double *m, const double *gamma,
                         const zc *v, zc *y, int conj_diag) {
    const int nx = op->nx, ny = op->ny, nz = op->nz;
    const double ih2 = 1.0 / (op->h * op->h);
    const double w2 = op->omega * op->omega;
    for (int iz = 0; iz < nz; ++iz)
        for (int iy = 0; iy < ny; ++iy)
            for (int ix = 0; ix < nx; ++ix) {
                size_t c = ((size_t)iz * ny + iy) * nx + ix;
                zc lap;
                if (op->stencil == 1) {
                    /* 27-point box stencil (reading C-23): the member of the family
                     *   h^2 Lap_h = a0 v_c + a1 sum(6 faces) + a2 sum(12 edges) + a3 sum(8 corners)
                     * that is consistent (a0 + 6 a1 + 12 a2 + 8 a3 = 0, a1 + 4 a2 + 4 a3 = 1), has an
                     * isotropic leading error term (a2 + 2 a3 = 1/6) and a3 = 1/30:
                     *   a0 = -128/30, a1 = 14/30, a2 = 3/30, a3 = 1/30. */
                    zc sum[4] = {0.0, 0.0, 0.0, 0.0};
                    for (int dz = -1; dz <= 1; ++dz)
                        for (int dy = -1; dy <= 1; ++dy)
                            for (int dx = -1; dx <= 1; ++dx)
                                sum[(dx != 0) + (dy != 0) + (dz != 0)] += nb(op, v, ix + dx, iy + dy, iz + dz);
                    lap = (-128.0 * sum[0] + 14.0 * sum[1] + 3.0 * sum[2] + 1.0 * sum[3]) / 30.0;
                } else {
                    lap = nb(op, v, ix - 1, iy, iz) + nb(op, v, ix + 1, iy, iz) +
                          nb(op, v, ix, iy - 1, iz) + nb(op, v, ix, iy + 1, iz) +
                          nb(op, v, ix, iy, iz - 1) + nb(op, v, ix, iy, iz + 1) -
                          6.0 * v[c];
                }
                zc mass = w2 * m[c] * (1.0 + I * gamma[c]);
                if (conj_diag) mass = conj(mass);
                y[c] = lap * ih2 + mass * v[c];
            }
}

void ref_apply_A(const ref_op *op, const double *m, const zc *v, zc *y) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    ref_gamma(op, gamma);
    apply_A_impl(op, m, gamma, v, y, 0);
    free(gamma);
}

void ref_apply_AH(const ref_op *op, const double *m, const zc *v, zc *y) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    ref_gamma(op, gamma);
    apply_A_impl(op, m, gamma, v, y, 1);
    free(gamma);
}

/* M v = [ lambda * A v ; v[rec[r]] ] */
static void apply_M_g(const ref_op *op, const double *m, const double *gamma, double lambda,
                      int32_t n_rec, const int64_t *rec, const zc *v, zc *ytop, zc *ybot) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    apply_A_impl(op, m, gamma, v, ytop, 0);
    for (size_t c = 0; c < ng; ++c) ytop[c] *= lambda;
    for (int32_t r = 0; r < n_rec; ++r) ybot[r] = v[rec[r]];
}

/* M^H y = lambda * A^H y_top ; then x[rec[r]] += y_bot[r] */
static void apply_MH_g(const ref_op *op, const double *m, const double *gamma, double lambda,
                       int32_t n_rec, const int64_t *rec, const zc *ytop, const zc *ybot, zc *x) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    apply_A_impl(op, m, gamma, ytop, x, 1);
    for (size_t c = 0; c < ng; ++c) x[c] *= lambda;
    for (int32_t r = 0; r < n_rec; ++r) x[rec[r]] += ybot[r];
}

void ref_apply_M(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                 const int64_t *rec, const zc *v, zc *ytop, zc *ybot) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    ref_gamma(op, gamma);
    apply_M_g(op, m, gamma, lambda, n_rec, rec, v, ytop, ybot);
    free(gamma);
}

void ref_apply_MH(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                  const int64_t *rec, const zc *ytop, const zc *ybot, zc *x) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    ref_gamma(op, gamma);
    apply_MH_g(op, m, gamma, lambda, n_rec, rec, ytop, ybot, x);
    free(gamma);
}

/* Euclidean norm of the stacked vector [a ; b], plain left-to-right sum */
static double norm2(const zc *a, size_t na, const zc *b, size_t nb_) {
    double s = 0.0;
    for (size_t i = 0; i < na; ++i) s += creal(a[i]) * creal(a[i]) + cimag(a[i]) * cimag(a[i]);
    for (size_t i = 0; i < nb_; ++i) s += creal(b[i]) * creal(b[i]) + cimag(b[i]) * cimag(b[i]);
    return sqrt(s);
}

/* TEST ONLY (op->round_c64): complex64 storage of a vector — each component is
 * rounded to float and promoted back. */
static void round_vec(zc *a, size_t n) {
    for (size_t i = 0; i < n; ++i) a[i] = (double)(float)creal(a[i]) + I * (double)(float)cimag(a[i]);
}

/* LSQR state of one column, all vectors NORMALISED as in Paige & Saunders:
 * ||u|| = ||v|| = 1 (unless broken down). */
typedef struct {
    zc *u_top;      /* [n_g]   */
    zc *u_bot;      /* [n_rec] */
    zc *v;          /* [n_g]   */
    zc *w;          /* [n_g]   */
    zc *x;          /* [n_g]   */
    double alpha, beta, rhobar, phibar;
    /* outputs of the last step */
    double rho, c, s, theta, phi, arnorm;
    int32_t stop;   /* 0 running, 1 beta==0, 2 alpha==0 */
} ref_state;

/* One LSQR iteration (loop body of O-2):
 *   u = M v - alpha u ; beta = ||u|| ; u /= beta
 *   v = M^H u - beta v ; alpha = ||v|| ; v /= alpha
 *   rho = hypot(rhobar, beta) ; c = rhobar/rho ; s = beta/rho ; theta = s alpha
 *   rhobar = -c alpha ; phi = c phibar ; phibar = s phibar
 *   x += (phi/rho) w ; w = v - (theta/rho) w
 * Breakdown (reading C-7): beta == 0 or alpha == 0 finishes the valid updates
 * of this step and raises st->stop; nothing divides by zero. */
static void lsqr_step_g(const ref_op *op, const double *m, const double *gamma, double lambda,
                        int32_t n_rec, const int64_t *rec, ref_state *st, zc *tmp_top, zc *tmp_bot) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double alpha = st->alpha, beta;

    apply_M_g(op, m, gamma, lambda, n_rec, rec, st->v, tmp_top, tmp_bot);
    for (size_t i = 0; i < ng; ++i) st->u_top[i] = tmp_top[i] - alpha * st->u_top[i];
    for (int32_t r = 0; r < n_rec; ++r) st->u_bot[r] = tmp_bot[r] - alpha * st->u_bot[r];
    beta = norm2(st->u_top, ng, st->u_bot, (size_t)n_rec);

    if (beta > 0.0) {
        for (size_t i = 0; i < ng; ++i) st->u_top[i] /= beta;
        for (int32_t r = 0; r < n_rec; ++r) st->u_bot[r] /= beta;
        apply_MH_g(op, m, gamma, lambda, n_rec, rec, st->u_top, st->u_bot, tmp_top);
        for (size_t i = 0; i < ng; ++i) st->v[i] = tmp_top[i] - beta * st->v[i];
        alpha = norm2(st->v, ng, NULL, 0);
        if (alpha > 0.0)
            for (size_t i = 0; i < ng; ++i) st->v[i] /= alpha;
    } else {
        alpha = 0.0;
    }

    double rho = hypot(st->rhobar, beta);
    double c = st->rhobar / rho;
    double s = beta / rho;
    double theta = s * alpha;
    double phi = c * st->phibar;
    st->rhobar = -c * alpha;
    st->phibar = s * st->phibar;

    double t1 = phi / rho, t2 = theta / rho;
    for (size_t i = 0; i < ng; ++i) {
        st->x[i] += t1 * st->w[i];
        st->w[i] = st->v[i] - t2 * st->w[i];
    }
    if (op->round_c64) {
        round_vec(st->u_top, ng); round_vec(st->u_bot, (size_t)n_rec);
        round_vec(st->v, ng); round_vec(st->w, ng); round_vec(st->x, ng);
    }
    st->alpha = alpha;
    st->beta = beta;
    st->rho = rho; st->c = c; st->s = s; st->theta = theta; st->phi = phi;
    st->arnorm = st->phibar * alpha * fabs(c);
    st->stop = (beta == 0.0) ? 1 : (alpha == 0.0 ? 2 : 0);
}

void ref_lsqr_step(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                   const int64_t *rec, ref_state *st) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    zc *tmp_top = (zc *)malloc(ng * sizeof(zc));
    zc *tmp_bot = (zc *)malloc(((size_t)n_rec + 1) * sizeof(zc));
    ref_gamma(op, gamma);
    lsqr_step_g(op, m, gamma, lambda, n_rec, rec, st, tmp_top, tmp_bot);
    free(gamma); free(tmp_top); free(tmp_bot);
}

/*
 * LSQR on  min_x || M x - b ||,  b = [lambda q ; d],  x0 = 0  (O-2).
 *
 * tol > 0 : stop at the first k with  phibar*alpha*|c| <= tol * alpha1*beta1
 *           (relative normal-equations residual estimate, reading C-6);
 * tol <= 0: run exactly maxit iterations (unless breakdown).
 * resnorms[k] = phibar after iteration k (= ||b - M x_k||), resnorms[0] = ||b||;
 * arnorms[k]  = phibar*alpha*|c| (= ||M^H (b - M x_k)||), arnorms[0] = alpha1*beta1;
 * both are held at their last value after the column stops (reading C-9).
 * x_snap (may be NULL): x after every snap_stride-th iteration,
 *   x_snap[(k/snap_stride - 1)*n_g + c]  for k = snap_stride, 2*snap_stride, ...
 * Returns the number of iterations performed.
 */
int32_t ref_lsqr(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                 const int64_t *rec, const zc *q, const zc *d, double tol, int32_t maxit,
                 zc *x, double *resnorms, double *arnorms, zc *x_snap, int32_t snap_stride) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    zc *tmp_top = (zc *)malloc(ng * sizeof(zc));
    zc *tmp_bot = (zc *)malloc(((size_t)n_rec + 1) * sizeof(zc));
    ref_state st;
    memset(&st, 0, sizeof st);
    st.u_top = (zc *)malloc(ng * sizeof(zc));
    st.u_bot = (zc *)malloc(((size_t)n_rec + 1) * sizeof(zc));
    st.v = (zc *)malloc(ng * sizeof(zc));
    st.w = (zc *)malloc(ng * sizeof(zc));
    st.x = x;
    ref_gamma(op, gamma);
    int32_t iters = 0;

    for (size_t i = 0; i < ng; ++i) { st.u_top[i] = lambda * q[i]; x[i] = 0.0; }
    for (int32_t r = 0; r < n_rec; ++r) st.u_bot[r] = d[r];
    double beta = norm2(st.u_top, ng, st.u_bot, (size_t)n_rec);
    double ar0 = 0.0, last_r = beta, last_ar = 0.0;
    resnorms[0] = beta;
    if (arnorms) arnorms[0] = 0.0;

    if (beta > 0.0) {
        for (size_t i = 0; i < ng; ++i) st.u_top[i] /= beta;
        for (int32_t r = 0; r < n_rec; ++r) st.u_bot[r] /= beta;
        apply_MH_g(op, m, gamma, lambda, n_rec, rec, st.u_top, st.u_bot, st.v);
        double alpha = norm2(st.v, ng, NULL, 0);
        ar0 = alpha * beta;
        last_ar = ar0;
        if (arnorms) arnorms[0] = ar0;
        if (alpha > 0.0) {
            for (size_t i = 0; i < ng; ++i) { st.v[i] /= alpha; st.w[i] = st.v[i]; }
            if (op->round_c64) {
                round_vec(st.u_top, ng); round_vec(st.u_bot, (size_t)n_rec);
                round_vec(st.v, ng); round_vec(st.w, ng);
            }
            st.alpha = alpha; st.beta = beta; st.phibar = beta; st.rhobar = alpha;
            for (int32_t k = 1; k <= maxit; ++k) {
                lsqr_step_g(op, m, gamma, lambda, n_rec, rec, &st, tmp_top, tmp_bot);
                iters = k;
                last_r = st.phibar; last_ar = st.arnorm;
                resnorms[k] = last_r;
                if (arnorms) arnorms[k] = last_ar;
                if (x_snap && snap_stride > 0 && k % snap_stride == 0)
                    memcpy(x_snap + (size_t)(k / snap_stride - 1) * ng, x, ng * sizeof(zc));
                if (st.stop) break;
                if (tol > 0.0 && st.arnorm <= tol * ar0) break;
            }
        }
    }
    for (int32_t k = iters + 1; k <= maxit; ++k) {
        resnorms[k] = last_r;
        if (arnorms) arnorms[k] = last_ar;
    }
    free(gamma); free(tmp_top); free(tmp_bot);
    free(st.u_top); free(st.u_bot); free(st.v); free(st.w);
    return iters;
}

/* ===========================================================================
 * Source-free system: the system the paper actually
 * states, PAPER.md:76-85 (eq. 4-6), with the source weight alpha UNKNOWN:
 *
 *     S = [ lambda A   -lambda e ]      x = [ u     ]      b = [ 0 ]
 *         [ P           0        ]          [ alpha ]          [ d ]
 *
 * e = real unit vector at the source node `src` ("e_i is a unit
 * vector representing the location of the i-th source").
 *   ref_apply_S    S [u; a]   = [ lambda (A u - a e) ; P u ]
 *   ref_apply_SH   S^H [yt;yb] = [ lambda A^H yt + P^T yb ; -lambda yt[src] ]
 *                  (e is real, so e^H yt = yt[src]; conjugate transpose per
 *                  reading C-2)
 *   ref_lsqr_sf    the same Paige & Saunders recurrences as ref_lsqr on S, b;
 *                  norms run over the stacked vectors including the alpha entry
 *   ref_lsqr_sf_step  one loop body on a caller-supplied state
 * Pins (tests/test_oracle_sf.py): adjoint dot test, dense LAPACK least squares
 * on 8^3 incl. the alpha entry, recovery of alpha_true on consistent data,
 * SciPy LSQR on the assembled sparse S, agreement with ref_lsqr when the alpha
 * column is removed.
 * ======================================================================== */

static void apply_S_g(const ref_op *op, const double *m, const double *gamma, double lambda,
                      int32_t n_rec, const int64_t *rec, int64_t src, const zc *u, zc a,
                      zc *ytop, zc *ybot) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    apply_A_impl(op, m, gamma, u, ytop, 0);
    ytop[src] -= a;                                  /* A u - alpha e            */
    for (size_t c = 0; c < ng; ++c) ytop[c] *= lambda;
    for (int32_t r = 0; r < n_rec; ++r) ybot[r] = u[rec[r]];
}

static void apply_SH_g(const ref_op *op, const double *m, const double *gamma, double lambda,
                       int32_t n_rec, const int64_t *rec, int64_t src, const zc *ytop,
                       const zc *ybot, zc *xu, zc *xa) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    apply_A_impl(op, m, gamma, ytop, xu, 1);
    for (size_t c = 0; c < ng; ++c) xu[c] *= lambda;
    for (int32_t r = 0; r < n_rec; ++r) xu[rec[r]] += ybot[r];
    *xa = -lambda * ytop[src];                       /* (-lambda e)^H y_top      */
}

void ref_apply_S(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                 const int64_t *rec, int64_t src, const zc *u, const zc *a, zc *ytop, zc *ybot) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    ref_gamma(op, gamma);
    apply_S_g(op, m, gamma, lambda, n_rec, rec, src, u, *a, ytop, ybot);
    free(gamma);
}

void ref_apply_SH(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                  const int64_t *rec, int64_t src, const zc *ytop, const zc *ybot, zc *xu, zc *xa) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    ref_gamma(op, gamma);
    apply_SH_g(op, m, gamma, lambda, n_rec, rec, src, ytop, ybot, xu, xa);
    free(gamma);
}

/* LSQR state of one source-free column: the x-space vectors v, w, x carry one
 * more complex entry (the alpha component), all NORMALISED as in ref_state. */
typedef struct {
    zc *u_top;      /* [n_g]   */
    zc *u_bot;      /* [n_rec] */
    zc *v;          /* [n_g]   */
    zc *w;          /* [n_g]   */
    zc *x;          /* [n_g]   */
    zc v_a, w_a, x_a;               /* alpha entries of v, w, x */
    double alpha, beta, rhobar, phibar;     /* LSQR scalars (alpha here is Golub-Kahan's, */
                                            /* not the source weight)                     */
    double rho, c, s, theta, phi, arnorm;
    int32_t stop;
} ref_state_sf;

static double abs2(zc z) { return creal(z) * creal(z) + cimag(z) * cimag(z); }

/* One LSQR iteration on S (same loop body and order as lsqr_step_g). */
static void lsqr_sf_step_g(const ref_op *op, const double *m, const double *gamma, double lambda,
                           int32_t n_rec, const int64_t *rec, int64_t src, ref_state_sf *st,
                           zc *tmp_top, zc *tmp_bot) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double alpha = st->alpha, beta;
    zc tmp_a;

    apply_S_g(op, m, gamma, lambda, n_rec, rec, src, st->v, st->v_a, tmp_top, tmp_bot);
    for (size_t i = 0; i < ng; ++i) st->u_top[i] = tmp_top[i] - alpha * st->u_top[i];
    for (int32_t r = 0; r < n_rec; ++r) st->u_bot[r] = tmp_bot[r] - alpha * st->u_bot[r];
    beta = norm2(st->u_top, ng, st->u_bot, (size_t)n_rec);

    if (beta > 0.0) {
        for (size_t i = 0; i < ng; ++i) st->u_top[i] /= beta;
        for (int32_t r = 0; r < n_rec; ++r) st->u_bot[r] /= beta;
        apply_SH_g(op, m, gamma, lambda, n_rec, rec, src, st->u_top, st->u_bot, tmp_top, &tmp_a);
        for (size_t i = 0; i < ng; ++i) st->v[i] = tmp_top[i] - beta * st->v[i];
        st->v_a = tmp_a - beta * st->v_a;
        double nv = norm2(st->v, ng, NULL, 0);
        alpha = sqrt(nv * nv + abs2(st->v_a));
        if (alpha > 0.0) {
            for (size_t i = 0; i < ng; ++i) st->v[i] /= alpha;
            st->v_a /= alpha;
        }
    } else {
        alpha = 0.0;
    }

    double rho = hypot(st->rhobar, beta);
    double c = st->rhobar / rho;
    double s = beta / rho;
    double theta = s * alpha;
    double phi = c * st->phibar;
    st->rhobar = -c * alpha;
    st->phibar = s * st->phibar;

    double t1 = phi / rho, t2 = theta / rho;
    for (size_t i = 0; i < ng; ++i) {
        st->x[i] += t1 * st->w[i];
        st->w[i] = st->v[i] - t2 * st->w[i];
    }
    st->x_a += t1 * st->w_a;
    st->w_a = st->v_a - t2 * st->w_a;
    if (op->round_c64) {          /* the alpha entries live in double on the GPU too: not rounded */
        round_vec(st->u_top, ng); round_vec(st->u_bot, (size_t)n_rec);
        round_vec(st->v, ng); round_vec(st->w, ng); round_vec(st->x, ng);
    }
    st->alpha = alpha;
    st->beta = beta;
    st->rho = rho; st->c = c; st->s = s; st->theta = theta; st->phi = phi;
    st->arnorm = st->phibar * alpha * fabs(c);
    st->stop = (beta == 0.0) ? 1 : (alpha == 0.0 ? 2 : 0);
}

void ref_lsqr_sf_step(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                      const int64_t *rec, int64_t src, ref_state_sf *st) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    zc *tmp_top = (zc *)malloc(ng * sizeof(zc));
    zc *tmp_bot = (zc *)malloc(((size_t)n_rec + 1) * sizeof(zc));
    ref_gamma(op, gamma);
    lsqr_sf_step_g(op, m, gamma, lambda, n_rec, rec, src, st, tmp_top, tmp_bot);
    free(gamma); free(tmp_top); free(tmp_bot);
}

/* LSQR on  min_x || S x - b ||,  b = [lambda q ; d]  (the paper's b = [0 ; d] is q = NULL),
 * x0 = 0.  Same histories and hold-last convention as ref_lsqr.
 * Stop rule: arnorm_k <= tol * ar_ref, with ar_ref = alpha1*beta1 of THIS system when the
 * argument is <= 0 (reading C-6), else the caller's reference (warm starts, reading C-17:
 * the tolerance stays relative to the cold problem's ||S^H b||).  x_u [n_g] and x_a [1]
 * receive the wavefield and the source-weight estimate.  Returns the iterations performed. */
int32_t ref_lsqr_sf(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                    const int64_t *rec, int64_t src, const zc *q, const zc *d, double tol,
                    double ar_ref, int32_t maxit,
                    zc *x_u, zc *x_a, double *resnorms, double *arnorms) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    zc *tmp_top = (zc *)malloc(ng * sizeof(zc));
    zc *tmp_bot = (zc *)malloc(((size_t)n_rec + 1) * sizeof(zc));
    ref_state_sf st;
    memset(&st, 0, sizeof st);
    st.u_top = (zc *)malloc(ng * sizeof(zc));
    st.u_bot = (zc *)malloc(((size_t)n_rec + 1) * sizeof(zc));
    st.v = (zc *)malloc(ng * sizeof(zc));
    st.w = (zc *)malloc(ng * sizeof(zc));
    st.x = x_u;
    ref_gamma(op, gamma);
    int32_t iters = 0;

    for (size_t i = 0; i < ng; ++i) { st.u_top[i] = q ? lambda * q[i] : 0.0; x_u[i] = 0.0; }
    for (int32_t r = 0; r < n_rec; ++r) st.u_bot[r] = d[r];
    double beta = norm2(st.u_top, ng, st.u_bot, (size_t)n_rec);
    double ar0 = 0.0, last_r = beta, last_ar = 0.0;
    resnorms[0] = beta;
    if (arnorms) arnorms[0] = 0.0;

    if (beta > 0.0) {
        for (size_t i = 0; i < ng; ++i) st.u_top[i] /= beta;
        for (int32_t r = 0; r < n_rec; ++r) st.u_bot[r] /= beta;
        apply_SH_g(op, m, gamma, lambda, n_rec, rec, src, st.u_top, st.u_bot, st.v, &st.v_a);
        double nv = norm2(st.v, ng, NULL, 0);
        double alpha = sqrt(nv * nv + abs2(st.v_a));
        last_ar = alpha * beta;
        if (arnorms) arnorms[0] = last_ar;
        ar0 = ar_ref > 0.0 ? ar_ref : alpha * beta;
        if (alpha > 0.0) {
            for (size_t i = 0; i < ng; ++i) { st.v[i] /= alpha; st.w[i] = st.v[i]; }
            st.v_a /= alpha; st.w_a = st.v_a;
            if (op->round_c64) {
                round_vec(st.u_top, ng); round_vec(st.u_bot, (size_t)n_rec);
                round_vec(st.v, ng); round_vec(st.w, ng);
            }
            st.alpha = alpha; st.beta = beta; st.phibar = beta; st.rhobar = alpha;
            for (int32_t k = 1; k <= maxit; ++k) {
                lsqr_sf_step_g(op, m, gamma, lambda, n_rec, rec, src, &st, tmp_top, tmp_bot);
                iters = k;
                last_r = st.phibar; last_ar = st.arnorm;
                resnorms[k] = last_r;
                if (arnorms) arnorms[k] = last_ar;
                if (st.stop) break;
                if (tol > 0.0 && st.arnorm <= tol * ar0) break;
            }
        }
    }
    *x_a = st.x_a;
    for (int32_t k = iters + 1; k <= maxit; ++k) {
        resnorms[k] = last_r;
        if (arnorms) arnorms[k] = last_ar;
    }
    free(gamma); free(tmp_top); free(tmp_bot);
    free(st.u_top); free(st.u_bot); free(st.v); free(st.w);
    return iters;
}

/* ===========================================================================
 * Objective and gradient of the reduced problem,
 * PAPER.md:71-76 (eq. 4), 98-110 (eq. 8-9), for ONE column at a given (u, alpha):
 *
 *   r      = A(m) u - q - alpha e                    (q dense and/or alpha e; either may be absent)
 *   f_pde  = 1/2 lambda^2 || r ||^2                  (eq. 5: the 1/2 covers both terms of eq. 4)
 *   f_data = 1/2 || P u - d ||^2
 *   g[c]  += lambda^2 omega^2 Re[ conj((1 + i gamma_c) u_c) r_c ]
 *
 * Eq. 9 prints  lambda^2 omega^2 diag(conj(u)) (A u - alpha e)  for the paper's
 * real-coefficient A = omega^2 diag(m) + Laplacian; m is real, so the real part
 * is meant, and with the sponge of this build dA/dm_c = omega^2 (1 + i gamma_c),
 * which gives the factor above (it reduces to eq. 9 where gamma = 0).  By
 * variable projection this partial derivative at the minimiser
 * (u-bar, alpha-bar) IS the gradient of f4(m); "does not involve additional PDE
 * solvers".  g is ACCUMULATED (the paper sums over sources and frequencies).
 * Pins (tests/test_oracle_sf.py): central finite differences of f in m at fixed
 * (u, alpha); finite differences of f4(m) through a converged solve on 6^3.
 * ======================================================================== */
void ref_objective_gradient(const ref_op *op, const double *m, double lambda, int32_t n_rec,
                            const int64_t *rec, int64_t src /* < 0: none */, const zc *alpha_src,
                            const zc *q /* may be NULL */, const zc *u, const zc *d,
                            double *f_pde, double *f_data, double *g /* [n_g], += ; may be NULL */) {
    size_t ng = (size_t)op->nx * op->ny * op->nz;
    double *gamma = (double *)malloc(ng * sizeof(double));
    zc *r = (zc *)malloc(ng * sizeof(zc));
    ref_gamma(op, gamma);
    apply_A_impl(op, m, gamma, u, r, 0);
    if (q) for (size_t c = 0; c < ng; ++c) r[c] -= q[c];
    if (src >= 0) r[src] -= *alpha_src;
    double sp = 0.0, sd = 0.0;
    for (size_t c = 0; c < ng; ++c) sp += abs2(r[c]);
    for (int32_t k = 0; k < n_rec; ++k) sd += abs2(u[rec[k]] - d[k]);
    *f_pde = 0.5 * lambda * lambda * sp;
    *f_data = 0.5 * sd;
    if (g) {
        const double w2 = op->omega * op->omega;
        for (size_t c = 0; c < ng; ++c)
            g[c] += lambda * lambda * w2 * creal(conj((1.0 + I * gamma[c]) * u[c]) * r[c]);
    }
    free(gamma); free(r);
}
