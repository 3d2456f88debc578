"""Parity of the source-free system S = [lam A, -lam e; P, 0], x = [u; alpha] (PAPER.md:76-85,
eq. 4-6) on the GPU against the complex128 oracle: operator
entries <= 1e-5, teacher-forced LSQR steps <= 1e-5, free-running history / wavefield / source
weight after 50 iterations <= 1e-3, adaptive masks with compaction, host entry."""
import math

import numpy as np
import pytest

import workloads
from oracle import oracle as O
from gpu_util import c64_floor, gpu_state_column_sf, ops_for, rel

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _wri(w, nb_max=None):
    from paper_2410_18429_b200 import Wri
    return Wri.from_workload(w, nb_max=nb_max)


def _cn(rng, shape):
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / math.sqrt(2)).astype(np.complex64)


def _src_cells(w):
    return O.rec_cells(w.nx, w.ny, w.nz, w.src_ijk)


SHAPES = [
    ("config1", dict(grid=(37, 41, 29), nb=1)),
    ("config2", dict(grid=(20, 33, 18), nb=3)),
    ("config2", dict(grid=(48, 40, 36), nb=48)),
    ("config3", dict(grid=(50, 50, 40), nb=16)),
    ("config2", dict(grid=(21, 18, 37), nb=64)),
]


@pytest.mark.parametrize("name,kw", SHAPES)
def test_apply_S_and_SH_match_oracle(torch_cuda, name, kw):
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    rng = np.random.Generator(np.random.PCG64(17))
    x, xa = _cn(rng, (w.ng, w.nb)), _cn(rng, (w.nb,))
    yt, yb = _cn(rng, (w.ng, w.nb)), _cn(rng, (w.n_rec, w.nb))
    xd, xad, ytd, ybd = (torch.from_numpy(a).cuda() for a in (x, xa, yt, yb))
    St, Sb = ctx.apply_S(xd, xad, w.lam, w.src_ijk, w.omega_idx)
    SHx, SHa = ctx.apply_SH(ytd, ybd, w.lam, w.src_ijk, w.omega_idx)
    St, Sb, SHx, SHa = (t.cpu().numpy() for t in (St, Sb, SHx, SHa))
    rec, src = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk), _src_cells(w)
    assert np.array_equal(Sb, x[rec, :])
    ops = ops_for(w)
    for s in sorted(set([0, w.nb // 2, w.nb - 1])):
        rt, _ = O.apply_S(ops[s], w.m, w.lam, rec, src[s], x[:, s], xa[s])
        assert rel(St[:, s], rt) < 1e-5
        # the source node itself, where the extra column lands
        assert abs(St[src[s], s] - rt[src[s]]) < 1e-5 * max(abs(rt[src[s]]), np.abs(rt).max())
        rx, ra = O.apply_SH(ops[s], w.m, w.lam, rec, src[s], yt[:, s], yb[:, s])
        assert rel(SHx[:, s], rx) < 1e-5
        assert abs(SHa[s] - ra) < 1e-6 * abs(ra)
    lhs = np.vdot(yt.astype(complex), St.astype(complex)) + np.vdot(yb.astype(complex), Sb.astype(complex))
    rhs = np.vdot(SHx.astype(complex), x.astype(complex)) + np.vdot(SHa.astype(complex), xa.astype(complex))
    assert abs(lhs - rhs) / abs(lhs) < 2e-5


TF_CASES = [
    ("config1", dict(grid=(24, 20, 28), nb=4), 8),      # generic kernel + one-block scalar kernels
    ("config2", dict(grid=(20, 33, 18), nb=3), 8),
    ("config2", dict(grid=(21, 18, 37), nb=64), 5),     # persistent TMA kernel, last-CTA finaliser
    ("config3", dict(grid=(27, 25, 20), nb=48), 5),
    ("config1", dict(grid=(32, 32, 32), nb=16), 6),
]


def _abs_terms_of_u_src(w, op, gam, c, pv):
    """Sum of the magnitudes of the terms that form (beta u)_top[src] = lam (A v)[src] - lam v_a
    - alpha u_top[src]: float32 arithmetic leaves an absolute error of about eps times this in
    that one entry (the stencil terms cancel for a smooth field).  Tolerance helper only."""
    nx, ny = w.nx, w.ny
    ix, iy, iz = c % nx, (c // nx) % ny, c // (nx * ny)
    v = pv["v"]
    nbrs = 0.0
    for dx, dy, dz in ((1, 0, 0), (-1, 0, 0), (0, 1, 0), (0, -1, 0), (0, 0, 1), (0, 0, -1)):
        jx, jy, jz = ix + dx, iy + dy, iz + dz
        if 0 <= jx < nx and 0 <= jy < ny and 0 <= jz < w.nz:
            nbrs += abs(v[(jz * ny + jy) * nx + jx])
    ih2 = 1.0 / w.h ** 2
    diag = abs(-6.0 * ih2 + op.omega ** 2 * float(w.m[c]) * (1 + 1j * gam[c]))
    return w.lam * (ih2 * nbrs + diag * abs(v[c]) + abs(pv["v_a"])) + pv["alpha"] * abs(pv["u_top"][c])


@pytest.mark.parametrize("name,kw,K", TF_CASES)
def test_sf_teacher_forced_steps(torch_cuda, name, kw, K, record_property):
    torch = torch_cuda
    tol = 1e-5
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    rec, src = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk), _src_cells(w)
    ops = ops_for(w)
    gam = O.gamma(ops[0]).reshape(-1)
    d = torch.from_numpy(w.D).cuda()
    ctx.lsqr_sf_begin(d, w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx)
    st = ctx.lsqr_peek()
    for s in range(w.nb):
        b_bot = w.D[:, s].astype(complex)
        beta1 = np.linalg.norm(b_bot)
        assert st["beta"][s] == pytest.approx(beta1, rel=1e-6)
        v1, va1 = O.apply_SH(ops[s], w.m, w.lam, rec, src[s], np.zeros(w.ng), b_bot / beta1)
        a1 = math.sqrt(np.linalg.norm(v1) ** 2 + abs(va1) ** 2)
        g = gpu_state_column_sf(st, s)
        assert rel(g["v"], v1 / a1) < tol
        assert g["alpha"] == pytest.approx(a1, rel=tol)
        assert abs(g["v_a"] - va1 / a1) < tol and abs(g["w_a"] - va1 / a1) < tol and g["x_a"] == 0
    worst_kappa = worst_err_a = 0.0
    for k in range(1, K + 1):
        prev = st
        ctx.lsqr_iterate(1)
        st = ctx.lsqr_peek()
        for s in range(w.nb):
            pv = gpu_state_column_sf(prev, s)
            ref = O.lsqr_sf_step(ops[s], w.m, w.lam, rec, src[s], pv)
            got = gpu_state_column_sf(st, s)
            errs = [rel(got[n], ref[n]) for n in ("u_top", "v", "w", "x")]
            errs.append(float(np.linalg.norm(got["u_bot"] - ref["u_bot"])))
            # alpha entries: error relative to the (unit-norm / x-norm) vector they belong to.
            # v_a = (-lam u_top[src] - beta v_a_old) / alpha is ONE entry formed from the complex64
            # value u_top[src]: its float32 rounding (eps |u|) is amplified by lam/alpha, and the
            # two terms cancel, so the bound is 8 eps_32 kappa with kappa the step's amplification
            # in the oracle's arithmetic (same rule as configs[0], C-12)
            kappa = (w.lam * _abs_terms_of_u_src(w, ops[s], gam, src[s], pv) / ref["beta"]
                     + ref["beta"] * abs(pv["v_a"])) / ref["alpha"]
            tol_a = max(tol, 8 * 6e-8 * kappa)
            worst_kappa = max(worst_kappa, kappa)
            worst_err_a = max(worst_err_a, abs(got["v_a"] - ref["v_a"]))
            assert abs(got["v_a"] - ref["v_a"]) < tol_a, (k, s, kappa)
            assert abs(got["w_a"] - ref["w_a"]) / max(1.0, np.linalg.norm(ref["w"])) < tol_a, (k, s, kappa)
            errs.append(abs(got["x_a"] - ref["x_a"]) / math.sqrt(np.linalg.norm(ref["x"]) ** 2 + abs(ref["x_a"]) ** 2))
            errs += [abs(got[n] - ref[n]) / abs(ref[n]) for n in ("alpha", "beta", "phibar", "rhobar")]
            assert max(errs) < tol, (k, s, errs)
            # the source node of u_top carries the -lam e column: check it on its own
            c = src[s]
            assert abs(got["u_top"][c] - ref["u_top"][c]) < \
                max(1e-7, 8 * 6e-8 * _abs_terms_of_u_src(w, ops[s], gam, c, pv) / ref["beta"])
    ctx.lsqr_end()
    # the data-dependent gate of the alpha entries (8 eps kappa) is logged so that it cannot grow unseen
    print("source-free teacher-forced %s %s: largest kappa %.1f (gate %.2e), largest |v_a error| %.2e"
          % (name, kw, worst_kappa, max(tol, 8 * 6e-8 * worst_kappa), worst_err_a))
    record_property("largest_kappa", "%.3e" % worst_kappa)
    record_property("largest_v_a_error", "%.3e" % worst_err_a)
    assert worst_kappa < 1000 and worst_err_a < 1e-4         # measured: kappa <= 588, error <= 4.2e-5


def _true_residuals(w, op, rec, src_cell, s, x, a):
    """||b - S [x; a]|| and ||S^H (b - S [x; a])|| in the oracle's arithmetic, b = [0; d]."""
    t, b = O.apply_S(op, w.m, w.lam, rec, src_cell, x.astype(complex), complex(a))
    rt, rb = -t, w.D[:, s].astype(complex) - b
    gx, ga = O.apply_SH(op, w.m, w.lam, rec, src_cell, rt, rb)
    return (math.sqrt(np.linalg.norm(rt) ** 2 + np.linalg.norm(rb) ** 2),
            math.sqrt(np.linalg.norm(gx) ** 2 + abs(ga) ** 2))


@pytest.mark.parametrize("name,kw,cols", [
    ("config1", dict(grid=(32, 32, 32), nb=16), [0, 7, 15]),
    ("config2", dict(grid=(32, 28, 24), nb=64), [0, 21, 42, 63]),
    ("config2", dict(grid=(20, 33, 18), nb=3), [0, 1, 2]),
])
def test_sf_free_running_50_iterations(torch_cuda, name, kw, cols):
    """With b = [0; d] the start vector lies in the span of the (degenerate, dominant) receiver
    singular vectors, so the Lanczos process loses orthogonality within a few steps and the
    iterates at a given k are rounding-determined even in complex128 (a 1e-12 perturbation of d
    moves the oracle's own x_10 by 3e-3; C-16, same mechanism as C-12).  What is
    attainable and checked: k <= 3 within 1e-3 of the oracle; at k = 50 the GPU's [u; alpha] is as
    good a solution as the oracle's (true residual, oracle arithmetic), its own residual estimate
    is honest, the history is monotone and stays near the oracle's; results are deterministic."""
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    d = torch.from_numpy(w.D).cuda()
    rec, src = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk), _src_cells(w)
    ops = ops_for(w)

    def run(K):
        out = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx)
        torch.cuda.synchronize()
        return [t.cpu().numpy() for t in out]

    u, a, res, it = run(3)
    ref = O.lsqr_sf_batch(ops, w.m, w.lam, rec, src, w.D, None, maxit=3, threads=4, columns=cols)
    for j, s in enumerate(cols):
        xn = math.sqrt(np.linalg.norm(ref["x"][:, j]) ** 2 + abs(ref["alpha_src"][j]) ** 2)
        assert rel(res[:, s], ref["resnorms"][:, j]) < 1e-3
        assert rel(u[:, s], ref["x"][:, j]) < 1e-3
        assert abs(a[s] - ref["alpha_src"][j]) < 1e-3 * xn

    K = 50
    u, a, res, it = run(K)
    assert (it == K).all()
    ref = O.lsqr_sf_batch(ops, w.m, w.lam, rec, src, w.D, None, maxit=K, threads=4, columns=cols)
    from dataclasses import replace
    for j, s in enumerate(cols):
        r_true, _ = _true_residuals(w, ops[s], rec, src[s], s, u[:, s], a[s])
        assert abs(res[K, s] / r_true - 1.0) < 1e-3                 # the GPU's estimate is honest
        assert np.all(np.diff(res[:, s]) <= 1e-6 * res[0, s])       # monotone ||r_k||
        # against the attainable floor: the oracle's complex64-storage emulation of the same column
        # (reading C-16; measured on CPU in tests/test_oracle_c64floor.py)
        fx, fh, _ = c64_floor(lambda dd, r: O.lsqr_sf(replace(ops[s], round_c64=r), w.m, w.lam, rec, src[s], dd,
                                                      maxit=K), w.D[:, s].astype(complex))
        dev_x, dev_h = rel(u[:, s], ref["x"][:, j]), rel(res[:, s], ref["resnorms"][:, j])
        print("b = [0; d] %s column %d k = %d: GPU deviation x %.3e history %.3e; complex64 floor x %.3e "
              "history %.3e" % (name, s, K, dev_x, dev_h, fx, fh))
        assert dev_x <= 2.0 * fx + 1e-3 and dev_h <= 2.0 * fh + 1e-3
        assert abs(r_true / ref["resnorms"][K, j] - 1.0) <= 2.0 * c64_floor.last_residual + 1e-3, \
            (s, r_true, ref["resnorms"][K, j])
    u2, a2, res2, _ = run(K)
    assert np.array_equal(u2, u) and np.array_equal(a2, a) and np.array_equal(res2, res)


def test_sf_adaptive_masks_compaction_and_host_entry(torch_cuda, monkeypatch):
    """Per-column tolerances: stop iterations follow the oracle's, converged columns are compacted
    away without changing the others' results, and the host-buffer entry returns the same."""
    torch = torch_cuda
    w = workloads.make("config3", grid=(40, 40, 32), nb=32)
    maxit = 60
    rng = np.random.Generator(np.random.PCG64(5))
    tol = (10.0 ** rng.uniform(-2.0, -0.5, w.nb)).astype(np.float32)
    tol[3] = 0.0                                            # one column runs to maxit
    ctx = _wri(w)
    d, told = torch.from_numpy(w.D).cuda(), torch.from_numpy(tol).cuda()
    u, a, res, it = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, told, maxit=maxit, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    u, a, res, it = u.cpu().numpy(), a.cpu().numpy(), res.cpu().numpy(), it.cpu().numpy()
    assert it[3] == maxit and len(set(it.tolist())) > 3
    rec, src = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk), _src_cells(w)
    cols = [0, 3, 11, 20, 31]
    ops = ops_for(w)
    ref = O.lsqr_sf_batch(ops, w.m, w.lam, rec, src, w.D, tol, maxit=maxit, threads=5, columns=cols)
    for j, s in enumerate(cols):
        k = int(it[s])
        # iterates are rounding-determined (see test_sf_free_running_50_iterations), so the stop
        # iteration may shift by a few steps of the convergence staircase; what must hold is the
        # stop RULE on the GPU's own result, evaluated in the oracle's arithmetic:
        r_true, ar_true = _true_residuals(w, ops[s], rec, src[s], s, u[:, s], a[s])
        ar0 = ref["arnorms"][0, j]
        assert abs(res[k, s] / r_true - 1.0) < 1e-3
        if tol[s] > 0:
            assert ar_true <= 1.5 * tol[s] * ar0, (s, k, ar_true / ar0, tol[s])
            assert abs(k - int(ref["iters"][j])) <= max(3, int(0.3 * ref["iters"][j])), (s, k, ref["iters"][j])
        assert np.all(res[k:, s] == res[k, s])
        assert np.all(np.diff(res[:, s]) <= 1e-6 * res[0, s])
    # without compaction: bit-identical per column
    ctx.set_debug_opts(no_compact=1)
    u2, a2, res2, it2 = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, told, maxit=maxit, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    ctx.set_debug_opts()
    assert np.array_equal(it2.cpu().numpy(), it)
    assert np.array_equal(res2.cpu().numpy(), res)
    assert np.array_equal(a2.cpu().numpy(), a)
    assert np.array_equal(u2.cpu().numpy(), u)
    # host-buffer entry
    uh, ah, resh, ith = ctx.lsqr_sf_batch_host(torch.from_numpy(w.D).pin_memory(), w.lam, w.src_ijk,
                                               torch.from_numpy(tol).pin_memory(), maxit=maxit,
                                               omega_idx=w.omega_idx)
    assert np.array_equal(ith.numpy(), it) and np.array_equal(ah.numpy(), a)
    assert np.array_equal(uh.numpy(), u) and np.array_equal(resh.numpy(), res)


def test_sf_known_part_of_the_source_and_bad_source_node(torch_cuda):
    """q given together with the unknown weight (b = [lam q; d]) and argument checking."""
    torch = torch_cuda
    from paper_2410_18429_b200.binding import WriError, WRI_ERR_ARG
    w = workloads.make("config1", grid=(24, 20, 28), nb=16)
    ctx = _wri(w)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    u, a, res, it = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=10, omega_idx=w.omega_idx, q=q)
    torch.cuda.synchronize()
    s = 5
    b0 = math.sqrt(np.linalg.norm(w.lam * w.Q[:, s].astype(complex)) ** 2 + np.linalg.norm(w.D[:, s].astype(complex)) ** 2)
    assert float(res[0, s]) == pytest.approx(b0, rel=1e-6)
    assert np.all(np.diff(res.cpu().numpy()[:, s]) <= 0)
    bad = w.src_ijk.copy()
    bad[2, 0] = w.nx
    with pytest.raises(WriError) as e:
        ctx.lsqr_sf_batch(d, w.lam, bad, None, maxit=2, omega_idx=w.omega_idx)
    assert e.value.code == WRI_ERR_ARG


@pytest.mark.parametrize("name,kw", [
    ("config1", dict(grid=(32, 32, 32), nb=16)),       # TMA path
    ("config2", dict(grid=(20, 33, 18), nb=3)),        # generic path
])
def test_sf_warm_start_and_stop_rule_reference(torch_cuda, name, kw):
    """Warm start (wri_lsqr_set_opts): the start of the residual system (r0 = b - S x0, teacher-forced
    against the oracle's operator), x_k = x0 + dx_k against the oracle's warm start for k <= 3, the
    history is ||b - S x_k|| of the original system, and continuing a loose solve to a tight
    tolerance with the cold reference needs fewer iterations than the cold tight solve."""
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    rec, src = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk), _src_cells(w)
    ops = ops_for(w)
    rng = np.random.Generator(np.random.PCG64(29))
    d, q = torch.from_numpy(w.D).cuda(), torch.from_numpy(w.Q).cuda()
    x0 = (_cn(rng, (w.ng, w.nb)) * np.float32(1e-2)).astype(np.complex64)
    a0 = (_cn(rng, (w.nb,)) * np.float32(1e-2)).astype(np.complex64)
    K = 3
    ctx.set_opts(warm_start=True)
    out = (torch.from_numpy(x0).cuda(), torch.from_numpy(a0).cuda(),
           torch.empty((K + 1, w.nb), dtype=torch.float32, device="cuda"),
           torch.empty(w.nb, dtype=torch.int32, device="cuda"))
    u, a, res, it = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx, q=q, out=out)
    torch.cuda.synchronize()
    u, a, res = u.cpu().numpy(), a.cpu().numpy(), res.cpu().numpy()
    for s in sorted(set([0, w.nb // 2, w.nb - 1])):
        ref = O.lsqr_sf_warm(ops[s], w.m, w.lam, rec, src[s], w.D[:, s], x0[:, s], a0[s], maxit=K, q=w.Q[:, s])
        assert rel(res[:, s], ref["resnorms"]) < 1e-3
        assert rel(u[:, s], ref["x"]) < 1e-3
        assert abs(a[s] - ref["alpha_src"]) < 1e-3 * math.sqrt(np.linalg.norm(ref["x"]) ** 2 + abs(ref["alpha_src"]) ** 2)
        # resnorms[0] is the residual of the ORIGINAL system at x0
        t, b = O.apply_S(ops[s], w.m, w.lam, rec, src[s], x0[:, s], a0[s])
        r0 = math.sqrt(np.linalg.norm(w.lam * w.Q[:, s].astype(complex) - t) ** 2
                       + np.linalg.norm(w.D[:, s].astype(complex) - b) ** 2)
        assert res[0, s] == pytest.approx(r0, rel=1e-5)

    # loose solve, then continue to a tight tolerance with the cold reference
    ctx.set_opts(ar0_out=torch.zeros(w.nb, dtype=torch.float64, device="cuda"))
    ar0 = ctx._opt_keep[1]
    maxit = 150
    loose = torch.full((w.nb,), 3e-2, dtype=torch.float32, device="cuda")
    tight = torch.full((w.nb,), 3e-3, dtype=torch.float32, device="cuda")
    ul, al, resl, itl = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, loose, maxit=maxit, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    ar_cold = ar0.clone()
    assert (ar_cold > 0).all()
    ctx.set_opts()
    ut, at, rest, itt = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, tight, maxit=maxit, omega_idx=w.omega_idx)
    ctx.set_opts(warm_start=True, ar_ref=ar_cold)
    out = (ul.clone(), al.clone(), torch.empty_like(resl), torch.empty_like(itl))
    uc, ac, resc, itc = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, tight, maxit=maxit, omega_idx=w.omega_idx, out=out)
    torch.cuda.synchronize()
    ctx.set_opts()
    itl, itt, itc = itl.cpu().numpy(), itt.cpu().numpy(), itc.cpu().numpy()
    assert (itl < itt).all() and (itt < maxit).all()
    assert (itc < itt).all(), (itl, itt, itc)
    # the continued solution satisfies the tight rule (oracle arithmetic) and starts where the loose one ended
    uc, ac, resc = uc.cpu().numpy(), ac.cpu().numpy(), resc.cpu().numpy()
    for s in (0, w.nb - 1):
        r_true, ar_true = _true_residuals(w, ops[s], rec, src[s], s, uc[:, s], ac[s])
        assert ar_true <= 1.5 * 3e-3 * float(ar_cold[s])
        assert resc[0, s] == pytest.approx(float(resl[itl[s], s]), rel=1e-4)
        assert abs(resc[itc[s], s] / r_true - 1.0) < 1e-3
