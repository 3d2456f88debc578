"""Pins of the oracle's source-free system S = [lam A, -lam e; P, 0] (eq. 4-6),
its LSQR, and the objective / gradient of eq. 4, 8, 9 (CPU only).

None of these re-types the oracle's formulas: S is checked against the already pinned M plus
the block structure the paper prints, the solver against LAPACK / SciPy / a direct Helmholtz
solve, and the gradient against finite differences of the objective.
"""
import math

import numpy as np
import pytest
import scipy.sparse.linalg as spla

from oracle import oracle as O


def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _cn(rng, n):
    return (rng.standard_normal(n) + 1j * rng.standard_normal(n)) / math.sqrt(2)


def _problem(nx, ny, nz, n_rec, seed, L=2, f=5.0, h=10.0):
    rng = _rng(seed)
    op = O.Operator(nx, ny, nz, h, 2 * math.pi * f, L)
    v = rng.uniform(1500.0, 4500.0, op.ng)
    m = 1.0 / v ** 2
    cells = rng.choice(op.ng, size=n_rec, replace=False).astype(np.int64)
    src = int(rng.integers(op.ng))
    return op, m, cells, src, rng


def _dense_M(op, m, lam, rec):
    n = op.ng
    Mtx = np.zeros((n + rec.size, n), dtype=complex)
    e = np.zeros(n, complex)
    for j in range(n):
        e[j] = 1.0
        t, b = O.apply_M(op, m, lam, rec, e)
        Mtx[:n, j], Mtx[n:, j] = t, b
        e[j] = 0.0
    return Mtx


def _dense_S(op, m, lam, rec, src):
    """eq. 6 assembled from the pinned M: S = [ M | (-lam e ; 0) ]."""
    n = op.ng
    S = np.zeros((n + rec.size, n + 1), dtype=complex)
    S[:, :n] = _dense_M(op, m, lam, rec)
    S[src, n] = -lam
    return S


@pytest.fixture(scope="module")
def tiny():
    op, m, rec, src, rng = _problem(8, 8, 8, 12, seed=31, L=2)
    lam = 20.0
    d = _cn(rng, rec.size)
    return op, m, rec, src, lam, d, _dense_S(op, m, lam, rec, src)


# ---------------------------------------------------------------- operator
@pytest.mark.parametrize("shape", [(7, 5, 9), (8, 8, 8), (1, 6, 5)])
def test_sf_adjoint_dot(shape):
    op, m, rec, src, rng = _problem(*shape, n_rec=7, seed=41)
    lam = 3.7
    u, a = _cn(rng, op.ng), complex(_cn(rng, 1)[0])
    yt, yb = _cn(rng, op.ng), _cn(rng, rec.size)
    St, Sb = O.apply_S(op, m, lam, rec, src, u, a)
    xu, xa = O.apply_SH(op, m, lam, rec, src, yt, yb)
    lhs = np.vdot(yt, St) + np.vdot(yb, Sb)                  # <y, S x>
    rhs = np.vdot(xu, u) + np.conj(xa) * a                   # <S^H y, x>
    assert abs(lhs - rhs) / abs(lhs) < 1e-12


def test_sf_operator_is_M_plus_the_source_column(tiny):
    """S [u; a] = M u + a (-lam e; 0)  and  S^H y = [M^H y; -lam y_top[src]] (eq. 6)."""
    op, m, rec, src, lam, d, S = tiny
    rng = _rng(42)
    u, a = _cn(rng, op.ng), complex(_cn(rng, 1)[0])
    St, Sb = O.apply_S(op, m, lam, rec, src, u, a)
    ref = S @ np.concatenate([u, [a]])
    assert np.linalg.norm(np.concatenate([St, Sb]) - ref) < 1e-13 * np.linalg.norm(ref)
    y = _cn(rng, op.ng + rec.size)
    xu, xa = O.apply_SH(op, m, lam, rec, src, y[:op.ng], y[op.ng:])
    refh = S.conj().T @ y
    assert np.linalg.norm(np.concatenate([xu, [xa]]) - refh) < 1e-13 * np.linalg.norm(refh)
    # the source column only touches the source node, with a minus sign
    St0, _ = O.apply_S(op, m, lam, rec, src, u, 0.0)
    diff = St - St0
    assert diff[src] == pytest.approx(-lam * a, rel=1e-12)
    diff[src] = 0
    assert not diff.any()


# ---------------------------------------------------------------- solver
def test_sf_lsqr_converges_to_dense_least_squares(tiny):
    """eq. 7: the minimiser of || S x - [0; d] || by LAPACK, alpha entry included."""
    op, m, rec, src, lam, d, S = tiny
    b = np.concatenate([np.zeros(op.ng), d])
    x_ls = np.linalg.lstsq(S, b, rcond=None)[0]
    out = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=700)
    x = np.concatenate([out["x"], [out["alpha_src"]]])
    assert np.linalg.norm(x - x_ls) < 1e-9 * np.linalg.norm(x_ls)
    assert abs(out["alpha_src"] - x_ls[-1]) < 1e-8 * abs(x_ls[-1])


def test_sf_lsqr_matches_scipy_lsqr(tiny):
    op, m, rec, src, lam, d, _ = tiny
    n, nr = op.ng, rec.size

    def mv(x):
        t, b = O.apply_S(op, m, lam, rec, src, x[:n], complex(x[n]))
        return np.concatenate([t, b])

    def rmv(y):
        xu, xa = O.apply_SH(op, m, lam, rec, src, y[:n], y[n:])
        return np.concatenate([xu, [xa]])

    A = spla.LinearOperator((n + nr, n + 1), dtype=complex, matvec=mv, rmatvec=rmv)
    b = np.concatenate([np.zeros(n), d])
    for K in (1, 3, 6, 25):
        ref = spla.lsqr(A, b, atol=0, btol=0, conlim=0, iter_lim=K)
        out = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=K)
        x = np.concatenate([out["x"], [out["alpha_src"]]])
        if K <= 6:
            assert np.linalg.norm(x - ref[0]) < 1e-10 * np.linalg.norm(ref[0])   # rounding order only
            assert out["resnorms"][K] == pytest.approx(ref[3], rel=1e-11)
            assert out["arnorms"][K] == pytest.approx(ref[7], rel=1e-9)
        else:
            # the 12 receiver rows are degenerate singular values far above the rest of the
            # spectrum (C-12): Lanczos vectors lose orthogonality within ~7 steps even
            # in fp64, so two correct implementations drift apart in x; the residual is robust
            assert np.linalg.norm(x - ref[0]) < 1e-3 * np.linalg.norm(ref[0])
            assert out["resnorms"][K] == pytest.approx(ref[3], rel=1e-6)


def test_sf_recovers_the_source_weight_on_consistent_data():
    """d = P u_true with A u_true = alpha_true e (direct solve): the data-augmented system is
    consistent, so LSQR must return u_true, alpha_true and a vanishing residual — the paper's
    on-the-fly source estimate (Table 3)."""
    op, m, rec, src, rng = _problem(6, 7, 6, 10, seed=43, L=2)
    n = op.ng
    Amat = np.zeros((n, n), complex)
    e = np.zeros(n, complex)
    for j in range(n):
        e[j] = 1.0
        Amat[:, j] = O.apply_A(op, m, e)
        e[j] = 0.0
    alpha_true = 2.5 - 1.5j
    rhs = np.zeros(n, complex)
    rhs[src] = alpha_true
    u_true = np.linalg.solve(Amat, rhs)
    d = u_true[rec]
    out = O.lsqr_sf(op, m, 1e3, rec, src, d, tol=0.0, maxit=900)
    assert out["resnorms"][-1] < 1e-9 * out["resnorms"][0]
    assert abs(out["alpha_src"] - alpha_true) < 1e-6 * abs(alpha_true)
    assert np.linalg.norm(out["x"] - u_true) < 1e-6 * np.linalg.norm(u_true)


def test_sf_with_alpha_fixed_is_the_known_source_system(tiny):
    """Fixing alpha at the source-free estimate turns eq. 6 into north_star's M u = [lam q; d],
    q = alpha e: the already pinned ref_lsqr must land on the same wavefield."""
    op, m, rec, src, lam, d, _ = tiny
    sf = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=700)
    q = np.zeros(op.ng, complex)
    q[src] = sf["alpha_src"]
    ks = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=700)
    assert np.linalg.norm(ks["x"] - sf["x"]) < 1e-8 * np.linalg.norm(sf["x"])


def test_sf_estimates_stop_rule_and_step_entry(tiny):
    op, m, rec, src, lam, d, S = tiny
    K = 30
    out = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=K)
    b = np.concatenate([np.zeros(op.ng), d])
    assert out["resnorms"][0] == pytest.approx(np.linalg.norm(d), rel=1e-14)
    assert np.all(np.diff(out["resnorms"]) <= 1e-14 * out["resnorms"][0])
    x = np.concatenate([out["x"], [out["alpha_src"]]])
    r = b - S @ x
    assert out["resnorms"][K] == pytest.approx(np.linalg.norm(r), rel=1e-11)
    assert out["arnorms"][K] == pytest.approx(np.linalg.norm(S.conj().T @ r), rel=1e-8)
    # tolerance mode: first crossing, history held
    ar = out["arnorms"]
    tol = 1.0001 * ar[15] / ar[0]                       # crossed at iteration 15 at the latest
    ar = out["arnorms"]
    k_stop = int(np.argmax(ar[1:] <= tol * ar[0])) + 1
    assert ar[k_stop] <= tol * ar[0]
    t = O.lsqr_sf(op, m, lam, rec, src, d, tol=tol, maxit=K)
    assert t["iters"] == k_stop
    assert np.all(t["resnorms"][k_stop:] == t["resnorms"][k_stop])
    short = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=k_stop)
    assert np.array_equal(short["x"], t["x"]) and short["alpha_src"] == t["alpha_src"]
    # zero data: nothing to iterate
    z = O.lsqr_sf(op, m, lam, rec, src, np.zeros(rec.size), tol=0.0, maxit=5)
    assert z["iters"] == 0 and not z["x"].any() and z["alpha_src"] == 0 and not z["resnorms"].any()

    # the step entry replays the loop: start by hand, then K steps
    beta = np.linalg.norm(d)
    u_bot = d / beta
    v, va = O.apply_SH(op, m, lam, rec, src, np.zeros(op.ng), u_bot)
    alpha = math.sqrt(np.linalg.norm(v) ** 2 + abs(va) ** 2)
    st = dict(u_top=np.zeros(op.ng, complex), u_bot=u_bot, v=v / alpha, w=v / alpha,
              x=np.zeros(op.ng, complex), v_a=va / alpha, w_a=va / alpha, x_a=0.0,
              alpha=alpha, beta=beta, rhobar=alpha, phibar=beta)
    for _ in range(7):
        st = O.lsqr_sf_step(op, m, lam, rec, src, st)
    seven = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=7)
    # (the start above is computed by numpy, so equality holds up to summation order)
    assert np.linalg.norm(st["x"] - seven["x"]) < 1e-12 * np.linalg.norm(seven["x"])
    assert abs(st["x_a"] - seven["alpha_src"]) < 1e-12 * np.linalg.norm(seven["x"])   # one entry of [x; x_a]
    assert st["phibar"] == pytest.approx(seven["resnorms"][7], rel=1e-13)


# ---------------------------------------------------------------- objective and gradient
def test_objective_is_half_the_squared_lsqr_residual(tiny):
    """f3 = 1/2 ||S x - b||^2 (eq. 5) = f_pde + f_data of eq. 4 = 1/2 phibar_k^2 at an LSQR iterate."""
    op, m, rec, src, lam, d, S = tiny
    out = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=20)
    fp, fd = O.objective_gradient(op, m, lam, rec, out["x"], d, src=src, alpha_src=out["alpha_src"])
    assert fp + fd == pytest.approx(0.5 * out["resnorms"][20] ** 2, rel=1e-11)
    x = np.concatenate([out["x"], [out["alpha_src"]]])
    r = S @ x - np.concatenate([np.zeros(op.ng), d])
    assert fp == pytest.approx(0.5 * np.linalg.norm(r[:op.ng]) ** 2, rel=1e-12)
    assert fd == pytest.approx(0.5 * np.linalg.norm(r[op.ng:]) ** 2, rel=1e-12)
    # dense q instead of alpha e gives the same number
    q = np.zeros(op.ng, complex)
    q[src] = out["alpha_src"]
    fp2, fd2 = O.objective_gradient(op, m, lam, rec, out["x"], d, q=q)
    assert fp2 == pytest.approx(fp, rel=1e-13) and fd2 == fd


def test_gradient_matches_finite_differences_at_fixed_wavefield():
    """f is quadratic in m at fixed (u, alpha): central differences are exact up to rounding.
    Checked inside the sponge too (the (1 + i gamma) factor of dA/dm)."""
    op, m, rec, src, rng = _problem(9, 8, 10, 9, seed=44, L=2)
    lam = 7.0
    u, a, d = _cn(rng, op.ng), complex(_cn(rng, 1)[0]), _cn(rng, rec.size)
    g = np.zeros(op.ng)
    O.objective_gradient(op, m, lam, rec, u, d, src=src, alpha_src=a, g=g)
    gam = O.gamma(op).reshape(-1)
    assert (gam > 0.5).any() and (gam == 0).any()
    for trial in range(4):
        dm = rng.standard_normal(op.ng) * m.mean()
        if trial == 0:
            dm = np.where(gam > 0.5, dm, 0.0)            # sponge cells only
        eps = 1e-3
        fp1, fd1 = O.objective_gradient(op, m + eps * dm, lam, rec, u, d, src=src, alpha_src=a)
        fp0, fd0 = O.objective_gradient(op, m - eps * dm, lam, rec, u, d, src=src, alpha_src=a)
        fdiff = (fp1 - fp0) / (2 * eps)
        assert fd1 == fd0
        assert fdiff == pytest.approx(float(g @ dm), rel=1e-6)        # cancellation in f1 - f0
    # accumulation over columns: a second call adds
    g2 = g.copy()
    O.objective_gradient(op, m, lam, rec, u, d, src=src, alpha_src=a, g=g2)
    assert np.allclose(g2, 2 * g, rtol=1e-15)


def test_gradient_of_the_reduced_objective_by_variable_projection():
    """eq. 8-9: d f4 / dm = partial derivative at the minimiser (u-bar, alpha-bar), with no
    further solve.  f4(m +- eps dm) is evaluated independently through LAPACK least squares."""
    op, m, rec, src, rng = _problem(6, 6, 6, 8, seed=45, L=2)
    lam = 15.0
    d = _cn(rng, rec.size)
    b = np.concatenate([np.zeros(op.ng), d])

    def f4(mm):
        S = _dense_S(op, mm, lam, rec, src)
        x = np.linalg.lstsq(S, b, rcond=None)[0]
        return 0.5 * np.linalg.norm(S @ x - b) ** 2, x

    _, xbar = f4(m)
    g = np.zeros(op.ng)
    O.objective_gradient(op, m, lam, rec, xbar[:-1], d, src=src, alpha_src=xbar[-1], g=g)
    dm = rng.standard_normal(op.ng) * m.mean()
    eps = 1e-4
    fd = (f4(m + eps * dm)[0] - f4(m - eps * dm)[0]) / (2 * eps)
    assert fd == pytest.approx(float(g @ dm), rel=1e-5)


# ---------------------------------------------------------------- known part of the source, warm start
def test_sf_with_a_known_source_part_and_warm_start(tiny):
    """b = [lam q; d] with the weight still unknown, and x0 != 0 (Algorithm 1 leaves x0 free):
    both must land on LAPACK's minimiser; a warm start from zero is the cold start; a warm start
    at the minimiser has nothing left to do once the stop rule refers to the cold ||S^H b||."""
    op, m, rec, src, lam, d, S = tiny
    rng = _rng(46)
    q = _cn(rng, op.ng) * 1e-3
    b = np.concatenate([lam * q, d])
    x_ls = np.linalg.lstsq(S, b, rcond=None)[0]
    cold = O.lsqr_sf(op, m, lam, rec, src, d, tol=0.0, maxit=700, q=q)
    x = np.concatenate([cold["x"], [cold["alpha_src"]]])
    assert np.linalg.norm(x - x_ls) < 1e-9 * np.linalg.norm(x_ls)
    assert cold["resnorms"][0] == pytest.approx(np.linalg.norm(b), rel=1e-14)
    # warm start from zero = cold start (up to the rounding of (lam q) / lam * lam)
    w0 = O.lsqr_sf_warm(op, m, lam, rec, src, d, np.zeros(op.ng), 0.0, maxit=5, q=q)
    c0 = O.lsqr_sf(op, m, lam, rec, src, d, maxit=5, q=q)
    assert np.linalg.norm(w0["x"] - c0["x"]) < 1e-10 * np.linalg.norm(c0["x"])
    assert np.allclose(w0["resnorms"], c0["resnorms"], rtol=1e-12)
    # warm start from a random point converges to the same minimiser; resnorms[0] = ||b - S x0||
    x0, a0 = _cn(rng, op.ng), complex(_cn(rng, 1)[0])
    warm = O.lsqr_sf_warm(op, m, lam, rec, src, d, x0, a0, maxit=700, q=q)
    xw = np.concatenate([warm["x"], [warm["alpha_src"]]])
    assert np.linalg.norm(xw - x_ls) < 1e-9 * np.linalg.norm(x_ls)
    assert warm["resnorms"][0] == pytest.approx(np.linalg.norm(b - S @ np.concatenate([x0, [a0]])), rel=1e-12)
    # from a partly converged iterate, with the cold reference: fewer iterations than the cold solve
    tol = 1e-6
    full = O.lsqr_sf(op, m, lam, rec, src, d, tol=tol, maxit=700, q=q)
    part = O.lsqr_sf(op, m, lam, rec, src, d, tol=1e-3, maxit=700, q=q)
    ar_cold = full["arnorms"][0]
    cont = O.lsqr_sf_warm(op, m, lam, rec, src, d, part["x"], part["alpha_src"], tol=tol, maxit=700, q=q,
                          ar_ref=ar_cold)
    assert 0 < cont["iters"] < full["iters"]
    r = b - S @ np.concatenate([cont["x"], [cont["alpha_src"]]])
    assert np.linalg.norm(S.conj().T @ r) <= 1.01 * tol * ar_cold
    # at the minimiser nothing is left: the first look at the rule stops it
    done = O.lsqr_sf_warm(op, m, lam, rec, src, d, x_ls[:-1], x_ls[-1], tol=tol, maxit=50, q=q, ar_ref=ar_cold)
    assert done["iters"] <= 1
    assert np.linalg.norm(done["x"] - x_ls[:-1]) < 1e-9 * np.linalg.norm(x_ls)
