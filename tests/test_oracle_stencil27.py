"""Pins of the oracle's 27-point discretisation of the Laplacian (
PAPER.md:56 says only "discretized 3D Laplacian"; reading C-23).  CPU only.

h^2 Lap_h = a0 v_c + a1 sum(6 faces) + a2 sum(12 edges) + a3 sum(8 corners) with
(a0, a1, a2, a3) = (-128, 14, 3, 1) / 30.  The box stencil is a polynomial in the one-dimensional
shifts T_a = S_a^+ + S_a^-:  a0 + a1 sum_a T_a + a2 sum_{a<b} T_a T_b + a3 T_x T_y T_z,  so every
eigenvector of the T_a — plane waves on the periodic box, sine modes under the zero (Dirichlet)
closure — is an eigenvector with the closed-form symbol below.  Three independent wave vectors pin
the four weights together with consistency (second-order convergence)."""
import math

import numpy as np
import pytest

from oracle import oracle as O

A0, A1, A2, A3 = -128.0 / 30.0, 14.0 / 30.0, 3.0 / 30.0, 1.0 / 30.0


def _symbol(t):
    """eigenvalue of h^2 Lap_h for eigenvalues t = (tx, ty, tz) of the one-dimensional T_a"""
    tx, ty, tz = t
    return A0 + A1 * (tx + ty + tz) + A2 * (tx * ty + tx * tz + ty * tz) + A3 * tx * ty * tz


def test_weights_are_the_isotropic_consistent_member():
    # consistency: constants are annihilated, second moments give the Laplacian
    assert A0 + 6 * A1 + 12 * A2 + 8 * A3 == pytest.approx(0.0, abs=1e-15)
    assert A1 + 4 * A2 + 4 * A3 == pytest.approx(1.0, abs=1e-15)
    # isotropic leading error term: coefficient of x^2 y^2 is twice that of x^4
    assert A2 + 2 * A3 == pytest.approx(1.0 / 6.0, abs=1e-15)


@pytest.mark.parametrize("p", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (2, 3, 1), (3, 1, 5)])
def test_plane_wave_periodic_box(p):
    nx, ny, nz, h = 8, 10, 12, 12.5
    op = O.Operator(nx, ny, nz, h, 2 * math.pi * 4.0, 0, periodic=True, stencil=1)
    m0 = 1.0 / 2000.0 ** 2
    m = np.full(op.ng, m0)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    th = (2 * math.pi * p[0] / nx, 2 * math.pi * p[1] / ny, 2 * math.pi * p[2] / nz)
    v = np.exp(1j * (th[0] * x + th[1] * y + th[2] * z)).reshape(-1)
    lam = _symbol([2 * math.cos(t) for t in th]) / h ** 2 + op.omega ** 2 * m0
    r = O.apply_A(op, m, v) - lam * v
    assert np.linalg.norm(r) < 1e-13 * max(abs(lam), 1 / h ** 2) * np.linalg.norm(v)


@pytest.mark.parametrize("p", [(1, 1, 1), (2, 1, 3), (5, 4, 2)])
def test_sine_modes_dirichlet_box(p):
    """production boundary: zero outside the grid, corners and edges included"""
    nx, ny, nz, h = 7, 9, 6, 10.0
    op = O.Operator(nx, ny, nz, h, 2 * math.pi * 6.0, 0, stencil=1)
    m0 = 1.0 / 2500.0 ** 2
    m = np.full(op.ng, m0)
    z, y, x = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    v = (np.sin(math.pi * p[0] * (x + 1) / (nx + 1)) * np.sin(math.pi * p[1] * (y + 1) / (ny + 1))
         * np.sin(math.pi * p[2] * (z + 1) / (nz + 1))).reshape(-1).astype(complex)
    t = [2 * math.cos(math.pi * pa / (na + 1)) for pa, na in zip(p, (nx, ny, nz))]
    lam = _symbol(t) / h ** 2 + op.omega ** 2 * m0
    r = O.apply_A(op, m, v) - lam * v
    assert np.linalg.norm(r) < 1e-13 * abs(lam) * np.linalg.norm(v)


def test_second_order_convergence_to_the_continuous_laplacian():
    """u = sin(a x) sin(b y) sin(c z) on the unit cube (zero on the faces): Lap u = -(a^2+b^2+c^2) u;
    the error of Lap_h u falls by 4 when h halves (catches a wrong normalisation of the weights)."""
    errs = []
    for n in (7, 15, 31):                                    # h = 1/8, 1/16, 1/32
        h = 1.0 / (n + 1)
        op = O.Operator(n, n, n, h, 0.0, 0, stencil=1)
        g = (np.arange(n) + 1) * h
        z, y, x = np.meshgrid(g, g, g, indexing="ij")
        a, b, c = math.pi, 2 * math.pi, math.pi
        u = (np.sin(a * x) * np.sin(b * y) * np.sin(c * z)).reshape(-1)
        lap = O.apply_A(op, np.zeros(op.ng), u.astype(complex)).real
        errs.append(np.abs(lap + (a * a + b * b + c * c) * u).max())
    assert 3.5 < errs[0] / errs[1] < 4.5 and 3.8 < errs[1] / errs[2] < 4.2


def test_mass_term_sponge_and_adjoint_are_those_of_the_seven_point_operator():
    """the two discretisations differ by a real symmetric matrix only: the diagonal mass term with
    its (1 + i gamma) factor is shared, A stays complex-symmetric, and the dot test holds"""
    rng = np.random.Generator(np.random.PCG64(3))
    op7 = O.Operator(9, 7, 6, 10.0, 2 * math.pi * 5.0, 2)
    op27 = O.Operator(9, 7, 6, 10.0, 2 * math.pi * 5.0, 2, stencil=1)
    m = 1.0 / rng.uniform(1500.0, 4500.0, op7.ng) ** 2
    v = (rng.standard_normal(op7.ng) + 1j * rng.standard_normal(op7.ng))
    diff = O.apply_A(op27, m, v) - O.apply_A(op7, m, v)       # (Lap27 - Lap7) v: no m, no gamma in it
    diff0 = O.apply_A(op27, np.zeros(op7.ng), v) - O.apply_A(op7, np.zeros(op7.ng), v)
    assert np.linalg.norm(diff - diff0) < 1e-12 * np.linalg.norm(diff0)
    a = O.apply_A(op27, m, v, adjoint=True)
    assert np.linalg.norm(a - np.conj(O.apply_A(op27, m, np.conj(v)))) <= 1e-15 * np.linalg.norm(a)
    rec = rng.choice(op7.ng, size=5, replace=False).astype(np.int64)
    yt = rng.standard_normal(op7.ng) + 1j * rng.standard_normal(op7.ng)
    yb = rng.standard_normal(5) + 1j * rng.standard_normal(5)
    Mt, Mb = O.apply_M(op27, m, 2.5, rec, v)
    lhs = np.vdot(yt, Mt) + np.vdot(yb, Mb)
    rhs = np.vdot(O.apply_MH(op27, m, 2.5, rec, yt, yb), v)
    assert abs(lhs - rhs) / abs(lhs) < 1e-12


def test_lsqr_on_the_27_point_system_reaches_the_dense_least_squares_solution():
    n = 6
    rng = np.random.Generator(np.random.PCG64(8))
    op = O.Operator(n, n, n, 10.0, 2 * math.pi * 5.0, 2, stencil=1)
    m = 1.0 / rng.uniform(1500.0, 4500.0, op.ng) ** 2
    rec = rng.choice(op.ng, size=9, replace=False).astype(np.int64)
    lam = 1.0
    cols = []
    for j in range(op.ng):
        e = np.zeros(op.ng, dtype=complex)
        e[j] = 1.0
        t, b = O.apply_M(op, m, lam, rec, e)
        cols.append(np.concatenate([t, b]))
    M = np.stack(cols, axis=1)
    q = rng.standard_normal(op.ng) + 1j * rng.standard_normal(op.ng)
    d = rng.standard_normal(9) + 1j * rng.standard_normal(9)
    b = np.concatenate([lam * q, d])
    x_ref = np.linalg.lstsq(M, b, rcond=None)[0]
    out = O.lsqr(op, m, lam, rec, q, d, maxit=400)
    assert np.linalg.norm(out["x"] - x_ref) < 1e-9 * np.linalg.norm(x_ref)
