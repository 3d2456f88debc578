"""Pins of the CPU oracle against what the paper and the mathematics fix (CPU only).

Each test is chosen so that a plausible mistake in oracle/wri_oracle.c (dropped term,
wrong sign or index, transposed operand, missing conjugate) fails at least one of them.
Pin numbers follow DESIGN.md / SURVEY.md section 8(c).
"""
import math
import os

import numpy as np
import pytest
import scipy.sparse.linalg as spla

from oracle import oracle as O

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


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
    return op, m, cells, rng


# ---------------------------------------------------------------- C-P1 adjoint dot test
@pytest.mark.parametrize("shape", [(7, 5, 9), (13, 11, 6), (8, 8, 8), (1, 6, 5)])
def test_adjoint_dot(shape):
    op, m, rec, rng = _problem(*shape, n_rec=7, seed=11)
    lam = 3.7
    x = _cn(rng, op.ng)
    yt, yb = _cn(rng, op.ng), _cn(rng, rec.size)
    Mt, Mb = O.apply_M(op, m, lam, rec, x)
    MHy = O.apply_MH(op, m, lam, rec, yt, yb)
    lhs = np.vdot(yt, Mt) + np.vdot(yb, Mb)        # <y, M x>
    rhs = np.vdot(MHy, x)                            # <M^H y, x>
    assert abs(lhs - rhs) / abs(lhs) < 1e-12


def test_adjoint_of_A_alone_and_symmetry():
    """A is complex-symmetric (reading C-3): A^H y = conj(A conj y)."""
    op, m, _, rng = _problem(9, 7, 6, 1, seed=12)
    y = _cn(rng, op.ng)
    a = O.apply_A(op, m, y, adjoint=True)
    b = np.conj(O.apply_A(op, m, np.conj(y)))
    assert np.linalg.norm(a - b) <= 1e-15 * np.linalg.norm(a)
    # and A is not Hermitian once the sponge is on (the conjugate matters)
    assert np.linalg.norm(a - O.apply_A(op, m, y)) > 1e-6 * np.linalg.norm(a)


# ---------------------------------------------------------------- C-P2 closed-form eigenpairs
@pytest.mark.parametrize("p", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (2, 3, 1)])
def test_plane_wave_periodic_box(p):
    """north_star (b): plane wave in a periodic undamped homogeneous box is an eigenvector
    with eigenvalue -(4/h^2) sum_a sin^2(k_a h/2) + omega^2 m."""
    nx, ny, nz, h = 8, 10, 12, 12.5
    op = O.Operator(nx, ny, nz, h, 2 * math.pi * 4.0, 0, periodic=True)
    m0 = 1.0 / 2000.0 ** 2
    m = np.full(op.ng, m0)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    kx, ky, kz = 2 * math.pi * p[0] / nx, 2 * math.pi * p[1] / ny, 2 * math.pi * p[2] / nz
    v = np.exp(1j * (kx * x + ky * y + kz * z)).reshape(-1)
    lam = -(4 / h ** 2) * (math.sin(kx / 2) ** 2 + math.sin(ky / 2) ** 2 + math.sin(kz / 2) ** 2) \
        + op.omega ** 2 * m0
    r = O.apply_A(op, m, v) - lam * v
    assert np.linalg.norm(r) < 1e-13 * abs(lam) * np.linalg.norm(v) + 1e-16


@pytest.mark.parametrize("p", [(1, 1, 1), (2, 1, 3), (5, 4, 2)])
def test_sine_modes_dirichlet_box(p):
    """Production boundary (zero outside the grid): prod_a sin(pi p_a (i_a+1)/(N_a+1)) is an
    eigenvector with eigenvalue -(4/h^2) sum_a sin^2(pi p_a / (2 (N_a+1))) + omega^2 m."""
    nx, ny, nz, h = 7, 9, 6, 10.0
    op = O.Operator(nx, ny, nz, h, 2 * math.pi * 6.0, 0)
    m0 = 1.0 / 2500.0 ** 2
    m = np.full(op.ng, m0)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    v = (np.sin(math.pi * p[0] * (x + 1) / (nx + 1)) * np.sin(math.pi * p[1] * (y + 1) / (ny + 1))
         * np.sin(math.pi * p[2] * (z + 1) / (nz + 1))).reshape(-1).astype(complex)
    lam = -(4 / h ** 2) * sum(math.sin(math.pi * pa / (2 * (na + 1))) ** 2
                              for pa, na in zip(p, (nx, ny, nz))) + op.omega ** 2 * m0
    r = O.apply_A(op, m, v) - lam * v
    assert np.linalg.norm(r) < 1e-13 * abs(lam) * np.linalg.norm(v)


def test_axes_are_not_interchanged():
    """x is the fastest axis, z the slowest: a mode that varies along x only must see the
    x-eigenvalue (catches swapped strides on non-cubic grids)."""
    nx, ny, nz, h = 5, 1, 1, 10.0
    op = O.Operator(nx, ny, nz, h, 0.0, 0)
    v = np.sin(math.pi * (np.arange(nx) + 1) / (nx + 1)).astype(complex)
    lam = -(4 / h ** 2) * math.sin(math.pi / (2 * (nx + 1))) ** 2 - 4 / h ** 2  # y,z: single cell, -2/h^2 each
    r = O.apply_A(op, np.zeros(op.ng), v) - lam * v
    assert np.linalg.norm(r) < 1e-15


# ---------------------------------------------------------------- sponge (reading C-4)
def test_sponge_profile_printed_values():
    depth, g_ref = np.loadtxt(os.path.join(GOLDEN, "sponge_profile.txt"), unpack=True)
    n, L = 32, 8
    op = O.Operator(n, n, n, 10.0, 1.0, L)
    g = O.gamma(op)                       # [nz, ny, nx]
    mid = n // 2
    for d, gr in zip(depth.astype(int), g_ref):
        i_lo, i_hi = L - d, n - 1 - L + d
        for line in (g[mid, mid, :], g[mid, :, mid], g[:, mid, mid]):
            assert line[i_lo] == pytest.approx(gr, abs=1e-15)
            assert line[i_hi] == pytest.approx(gr, abs=1e-15)
    assert np.all(g[L:n - L, L:n - L, L:n - L] == 0.0)
    assert g.max() == 1.0 and g[0, 0, 0] == 1.0             # corners: max rule keeps gamma <= 1
    assert g[2, mid, 5] == pytest.approx((6 / 8) ** 2)        # max(dz=6, dx=3)
    # face mask: only the z- face listed
    g2 = O.gamma(O.Operator(n, n, n, 10.0, 1.0, L, faces=0x10))
    assert g2[0, mid, mid] == 1.0 and g2[n - 1, mid, mid] == 0.0 and g2[mid, mid, 0] == 0.0


def test_mass_term_carries_one_plus_i_gamma():
    """(A 1)[c] = omega^2 m (1 + i gamma) at a cell whose six neighbours are inside the grid
    (the Laplacian of a constant vanishes there): pins the sign and placement of i*gamma."""
    n, L = 12, 4
    op = O.Operator(n, n, n, 10.0, 2 * math.pi * 5, L)
    rng = _rng(5)
    m = 1.0 / rng.uniform(1500, 4000, op.ng) ** 2
    y = O.apply_A(op, m, np.ones(op.ng, complex)).reshape(n, n, n)
    g = O.gamma(op)
    mm = m.reshape(n, n, n)
    inner = (slice(1, n - 1),) * 3
    np.testing.assert_allclose(y[inner].real, op.omega ** 2 * mm[inner], rtol=1e-10)
    np.testing.assert_allclose(y[inner].imag, op.omega ** 2 * mm[inner] * g[inner], rtol=1e-10, atol=1e-20)
    assert y[1, 6, 6].imag > 0      # +i gamma, depth 3 of 4 -> gamma = 9/16
    assert y[1, 6, 6].imag / y[1, 6, 6].real == pytest.approx(9 / 16, rel=1e-10)


# ---------------------------------------------------------------- receivers
def test_receiver_sampling_is_exact_indexing():
    op, m, rec, rng = _problem(6, 5, 4, 9, seed=3)
    v = _cn(rng, op.ng)
    _, yb = O.apply_M(op, m, 2.0, rec, v)
    assert np.array_equal(yb, v[rec])
    x = O.apply_MH(op, m, 2.0, rec, np.zeros(op.ng), np.arange(1, 10) * (1 + 2j))
    ref = np.zeros(op.ng, complex)
    ref[rec] = np.arange(1, 10) * (1 + 2j)
    assert np.array_equal(x, ref)
    ijk = np.array([[1, 2, 3], [0, 0, 0], [5, 4, 3]])
    assert list(O.rec_cells(6, 5, 4, ijk)) == [(3 * 5 + 2) * 6 + 1, 0, (3 * 5 + 4) * 6 + 5]


# ---------------------------------------------------------------- LSQR pins
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


@pytest.fixture(scope="module")
def tiny():
    """8^3 grid, sponge 2, 12 receivers, lambda such that cond(M) is moderate."""
    op, m, rec, rng = _problem(8, 8, 8, 12, seed=21, L=2, f=5.0, h=10.0)
    lam = 20.0
    q, d = _cn(rng, op.ng) * 1e-3, _cn(rng, rec.size)
    return op, m, rec, lam, q, d, _dense_M(op, m, lam, rec)


def test_lsqr_converges_to_dense_least_squares(tiny):
    """C-P3: eq. 4/7 minimiser by LAPACK on the dense (n_g+n_r) x n_g matrix."""
    op, m, rec, lam, q, d, Mtx = tiny
    b = np.concatenate([lam * q, d])
    x_ls = np.linalg.lstsq(Mtx, b, rcond=None)[0]
    out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=600)
    assert np.linalg.norm(out["x"] - x_ls) < 1e-10 * np.linalg.norm(x_ls)
    # and it is NOT converged early on: the oracle must be compared iterate by iterate
    early = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=10)
    assert np.linalg.norm(early["x"] - x_ls) > 1e-3 * np.linalg.norm(x_ls)


def test_lsqr_matches_scipy_lsqr(tiny):
    """C-P4: SciPy's Paige-Saunders LSQR on the same operator, fixed K."""
    op, m, rec, lam, q, d, _ = tiny
    n, nr = op.ng, rec.size
    A = spla.LinearOperator(
        (n + nr, n), dtype=complex,
        matvec=lambda x: np.concatenate(O.apply_M(op, m, lam, rec, x)),
        rmatvec=lambda y: O.apply_MH(op, m, lam, rec, y[:n], y[n:]))
    b = np.concatenate([lam * q, d])
    for K in (1, 7, 30):
        ref = spla.lsqr(A, b, atol=0, btol=0, conlim=0, iter_lim=K)
        out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=K)
        assert np.linalg.norm(out["x"] - ref[0]) < 1e-11 * np.linalg.norm(ref[0])
        assert out["resnorms"][K] == pytest.approx(ref[3], rel=1e-11)      # r1norm
        assert out["arnorms"][K] == pytest.approx(ref[7], rel=1e-9)        # arnorm


def test_lsqr_matches_cgls(tiny):
    """C-P5: CGLS iterates equal LSQR iterates in exact arithmetic."""
    op, m, rec, lam, q, d, Mtx = tiny
    b = np.concatenate([lam * q, d])
    K = 25
    x = np.zeros(op.ng, complex)
    r = b.copy()
    s = Mtx.conj().T @ r
    p = s.copy()
    g = np.vdot(s, s).real
    for _ in range(K):
        t = Mtx @ p
        a = g / np.vdot(t, t).real
        x += a * p
        r -= a * t
        s = Mtx.conj().T @ r
        g_new = np.vdot(s, s).real
        p = s + (g_new / g) * p
        g = g_new
    out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=K)
    assert np.linalg.norm(out["x"] - x) < 1e-9 * np.linalg.norm(x)


def test_estimates_equal_true_residuals_and_monotone(tiny):
    """C-P6 / C-P7: phibar_k = ||b - M x_k||, phibar alpha |c| = ||M^H (b - M x_k)||;
    ||r_k|| never increases (LSQR minimises it over the Krylov space, reading C-13)."""
    op, m, rec, lam, q, d, Mtx = tiny
    b = np.concatenate([lam * q, d])
    K = 40
    out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=K, snap_stride=1)
    assert out["resnorms"][0] == pytest.approx(np.linalg.norm(b), rel=1e-14)
    assert out["arnorms"][0] == pytest.approx(np.linalg.norm(Mtx.conj().T @ b), rel=1e-12)
    for k in range(1, K + 1):
        r = b - Mtx @ out["x_snap"][k - 1]
        assert out["resnorms"][k] == pytest.approx(np.linalg.norm(r), rel=1e-11)
        assert out["arnorms"][k] == pytest.approx(np.linalg.norm(Mtx.conj().T @ r), rel=1e-8)
    assert np.all(np.diff(out["resnorms"]) <= 0)
    assert out["arnorms"][K] < 0.2 * out["arnorms"][0]


def test_consistent_system_recovers_wavefield():
    """C-P8: q = A u*, d = P u*  =>  x_k -> u*, ||r_k|| -> 0 (pins the lambda weighting of b)."""
    op, m, rec, rng = _problem(6, 6, 6, 10, seed=8, L=2)
    lam = 50.0
    ustar = _cn(rng, op.ng)
    q = O.apply_A(op, m, ustar)
    d = ustar[rec]
    out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=800)
    assert np.linalg.norm(out["x"] - ustar) < 1e-8 * np.linalg.norm(ustar)
    assert out["resnorms"][-1] < 1e-9 * out["resnorms"][0]


def test_stopping_rule_hold_last_and_breakdown(tiny):
    """C-6 / C-7 / C-9: first crossing of the relative normal-equations residual; history
    held after the stop; b = 0 gives x = 0 in 0 iterations; tol = 0 runs exactly maxit."""
    op, m, rec, lam, q, d, _ = tiny
    full = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=60)
    assert full["iters"] == 60
    tol = 0.05
    rel = full["arnorms"] / full["arnorms"][0]
    k_first = int(np.argmax(rel[1:] <= tol)) + 1
    out = O.lsqr(op, m, lam, rec, q, d, tol=tol, maxit=60)
    assert out["iters"] == k_first
    assert np.array_equal(out["resnorms"][:k_first + 1], full["resnorms"][:k_first + 1])
    assert np.all(out["resnorms"][k_first:] == out["resnorms"][k_first])
    z = O.lsqr(op, m, lam, rec, np.zeros(op.ng), np.zeros(rec.size), tol=0.0, maxit=5)
    assert z["iters"] == 0 and not z["x"].any() and not z["resnorms"].any()


def test_one_unknown_is_solved_in_one_step_and_stays_finite():
    """Degenerate 1-cell grid: M is 2x1, LSQR is exact after one iteration and later
    iterations must not produce NaN/Inf."""
    op = O.Operator(1, 1, 1, 10.0, 2 * math.pi * 5, 0)
    m = np.array([1 / 2000.0 ** 2])
    rec = np.array([0], dtype=np.int64)
    lam, q, d = 30.0, np.array([0.3 - 0.2j]), np.array([1.0 + 2.0j])
    a = lam * (-6 / 100.0 + op.omega ** 2 * m[0])
    x_exact = (np.conj(a) * lam * q[0] + d[0]) / (abs(a) ** 2 + 1)
    out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=1)
    assert out["x"][0] == pytest.approx(x_exact, rel=1e-13)
    out = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=6)
    assert np.all(np.isfinite(out["x"])) and np.all(np.isfinite(out["resnorms"]))
    assert out["x"][0] == pytest.approx(x_exact, rel=1e-10)


def test_step_entry_reproduces_the_loop_and_batch_is_columnwise(tiny):
    """ref_lsqr_step chained from the initial state equals ref_lsqr bit for bit; a batch is
    exactly its columns solved alone, in any order, threaded or not (C-P9)."""
    op, m, rec, lam, q, d, _ = tiny
    b_top, b_bot = lam * q, d.copy()
    beta = math.sqrt((np.abs(b_top) ** 2).sum() + (np.abs(b_bot) ** 2).sum())
    u_top, u_bot = b_top / beta, b_bot / beta
    v = O.apply_MH(op, m, lam, rec, u_top, u_bot)
    alpha = math.sqrt((np.abs(v) ** 2).sum())
    v = v / alpha
    st = dict(u_top=u_top, u_bot=u_bot, v=v, w=v.copy(), x=np.zeros(op.ng, complex),
              alpha=alpha, beta=beta, rhobar=alpha, phibar=beta)
    for _ in range(5):
        st = O.lsqr_step(op, m, lam, rec, st)
    ref = O.lsqr(op, m, lam, rec, q, d, tol=0.0, maxit=5)
    assert np.linalg.norm(st["x"] - ref["x"]) <= 1e-14 * np.linalg.norm(ref["x"])
    assert st["phibar"] == pytest.approx(ref["resnorms"][5], rel=1e-14)

    rng = _rng(99)
    Q = np.stack([q, 2 * q, _cn(rng, op.ng)], axis=1)
    D = np.stack([d, -d, _cn(rng, rec.size)], axis=1)
    op2 = O.Operator(op.nx, op.ny, op.nz, op.h, 2 * math.pi * 7.0, op.sponge_width)
    ops = [op, op, op2]
    tols = [0.0, 0.1, 0.0]
    a = O.lsqr_batch(ops, m, lam, rec, Q, D, tols, maxit=20, threads=1)
    b = O.lsqr_batch(ops, m, lam, rec, Q, D, tols, maxit=20, threads=3)
    c = O.lsqr_batch(ops[::-1], m, lam, rec, Q[:, ::-1], D[:, ::-1], tols[::-1], maxit=20)
    for k in ("x", "resnorms", "iters"):
        assert np.array_equal(a[k], b[k])
        assert np.array_equal(a[k], c[k][..., ::-1])
    assert np.array_equal(a["x"][:, 0], O.lsqr(op, m, lam, rec, q, d, maxit=20)["x"])
    assert a["iters"][1] < 20 and a["iters"][0] == 20
