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
 *                  DESIGN.md reading C-3.
 *   ref_apply_M    M v = [lambda A v ; P v], PAPER.md:78-85 (eq. 5-6) with the
 *                  source weight fixed (reading C-5); P = sampling of receiver
 *                  nodes.
 *   ref_apply_MH   M^H y = lambda A^H y_top + P^T y_bot (PAPER.md:95, 118 write
 *                  "T"; conjugate transpose is meant, reading C-2).  A^H is
 *                  written out here as its own stencil (conjugated diagonal),
 *                  not derived from ref_apply_A, so the adjoint dot test pins
 *                  both.
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
 * Pins (tests/test_oracle_*.py): adjoint dot test, closed-form eigenpairs
 * (periodic plane wave, Dirichlet sine modes), printed sponge values, dense
 * LAPACK least squares on 8^3, SciPy LSQR, CGLS, estimate-vs-true residuals,
 * monotone ||r||, consistent system, breakdown cases.
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
                zc lap = nb(op, v, ix - 1, iy, iz) + nb(op, v, ix + 1, iy, iz) +
                         nb(op, v, ix, iy - 1, iz) + nb(op, v, ix, iy + 1, iz) +
                         nb(op, v, ix, iy, iz - 1) + nb(op, v, ix, iy, iz + 1) -
                         6.0 * v[c];
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
