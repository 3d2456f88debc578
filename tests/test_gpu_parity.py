"""Parity of the CUDA path (through the C ABI) against the complex128 oracle, element by element,
on the same seeded, once-rounded inputs.  Tolerances are BASELINE.json north_star's:
receiver indexing bit-exact; one complex64 operator application <= 1e-5 relative L2;
residual history and u after 50 iterations <= 1e-3 relative L2 (configs[0] caveat: DESIGN.md C-12).
"""
import math

import numpy as np
import pytest

import workloads
from oracle import oracle as O
from gpu_util import c64_floor, gpu_state_column, ops_for, rel

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


SHAPES = [
    ("config1", dict(grid=(37, 41, 29), nb=1)),
    ("config1", dict(grid=(37, 41, 29), nb=2)),
    ("config2", dict(grid=(20, 33, 18), nb=3)),
    ("config2", dict(grid=(24, 17, 40), nb=5)),
    ("config2", dict(grid=(48, 40, 36), nb=48)),
    ("config3", dict(grid=(50, 50, 40), nb=16)),
    ("config4", dict(grid=(32, 32, 32), nb=32)),
]


@pytest.mark.parametrize("name,kw", SHAPES)
def test_apply_M_and_MH_match_oracle(torch_cuda, name, kw):
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    rng = np.random.Generator(np.random.PCG64(7))
    x = _cn(rng, (w.ng, w.nb))
    yt, yb = _cn(rng, (w.ng, w.nb)), _cn(rng, (w.n_rec, w.nb))
    xd, ytd, ybd = (torch.from_numpy(a).cuda() for a in (x, yt, yb))
    oi = w.omega_idx
    Mt, Mb = ctx.apply_M(xd, w.lam, oi)
    MH = ctx.apply_MH(ytd, ybd, w.lam, oi)
    Mt, Mb, MH = Mt.cpu().numpy(), Mb.cpu().numpy(), MH.cpu().numpy()
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    assert np.array_equal(Mb, x[rec, :])                    # receiver indexing: bit-exact
    ops = ops_for(w)
    cols = sorted(set([0, w.nb // 2, w.nb - 1]))
    for s in cols:
        rt, rb = O.apply_M(ops[s], w.m, w.lam, rec, x[:, s])
        assert rel(Mt[:, s], rt) < 1e-5
        rh = O.apply_MH(ops[s], w.m, w.lam, rec, yt[:, s], yb[:, s])
        assert rel(MH[:, s], rh) < 1e-5
    # adjoint dot test on the GPU results (float32 arithmetic)
    lhs = np.vdot(yt.astype(complex), Mt.astype(complex)) + np.vdot(yb.astype(complex), Mb.astype(complex))
    rhs = np.vdot(MH.astype(complex), x.astype(complex))
    assert abs(lhs - rhs) / abs(lhs) < 2e-5


def test_receivers_on_faces_and_corners_are_exact(torch_cuda):
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri
    nx, ny, nz, nb = 9, 7, 6, 4
    rec = np.array([[0, 0, 0], [8, 6, 5], [8, 0, 0], [0, 6, 5], [4, 3, 0], [4, 3, 5], [0, 3, 2]], dtype=np.int32)
    m = torch.full((nx * ny * nz,), 1 / 2000.0 ** 2, device="cuda")
    ctx = Wri((nx, ny, nz), 10.0, [2 * math.pi * 5], m, 2, rec, nb)
    rng = np.random.Generator(np.random.PCG64(3))
    x = _cn(rng, (nx * ny * nz, nb))
    _, yb = ctx.apply_M(torch.from_numpy(x).cuda(), 1.0)
    cells = O.rec_cells(nx, ny, nz, rec)
    assert np.array_equal(yb.cpu().numpy(), x[cells])
    ybot = _cn(rng, (len(rec), nb))
    out = ctx.apply_MH(torch.zeros((nx * ny * nz, nb), dtype=torch.complex64, device="cuda"),
                       torch.from_numpy(ybot).cuda(), 1.0).cpu().numpy()
    ref = np.zeros_like(x)
    ref[cells] = ybot
    assert np.array_equal(out, ref)                          # P^T is a pure scatter


TF_CASES = [
    ("config0", {}, 14),
    ("config1", dict(grid=(24, 20, 28), nb=4), 10),
    ("config2", dict(grid=(20, 33, 18), nb=3), 10),
    ("config3", dict(grid=(40, 40, 32), nb=6), 10),
    # persistent TMA kernel: column chunks of 64 / 32 / 16, ragged tiles, mixed frequencies
    ("config2", dict(grid=(21, 18, 37), nb=64), 5),
    ("config4", dict(grid=(19, 22, 35), nb=32), 5),
    ("config3", dict(grid=(27, 25, 20), nb=48), 5),
    ("config1", dict(grid=(32, 32, 32), nb=16), 5),
    ("config1", dict(grid=(21, 34, 19), nb=8), 4),
    ("config2", dict(grid=(30, 17, 22), nb=4), 4),
    ("config4", dict(grid=(35, 18, 21), nb=2), 4),                     # 2-column tiles (32 x 16 cells)
    ("config2", dict(grid=(22, 19, 36), nb=56), 4),                    # widths of a shrinking batch
    ("config3", dict(grid=(23, 21, 20), nb=40), 4),
    ("config2", dict(grid=(26, 18, 35), nb=24), 4),
]


def _step_tolerance(name, op, w, rec, prev, ref):
    """1e-5 relative L2 per step.  On configs[0] (lambda = 1) single steps cancel strongly
    (the receiver block of u shrinks by 1-2 orders in one step, C-12), so float32
    operands of size `a` leave an error eps*a in a result of size 1: there the bound is
    8 eps_32 * kappa with kappa the step's cancellation factor in the oracle's arithmetic."""
    if name != "config0":
        return 1e-5
    none = np.zeros(0, dtype=np.int64)
    mt, mb = O.apply_M(op, w.m, w.lam, rec, prev["v"])
    a_bot = (np.linalg.norm(mb) + prev["alpha"] * np.linalg.norm(prev["u_bot"])) / ref["beta"]
    k_u = (math.sqrt(np.linalg.norm(mt) ** 2 + np.linalg.norm(mb) ** 2) + prev["alpha"]) / ref["beta"]
    ah = O.apply_MH(op, w.m, w.lam, none, ref["u_top"], np.zeros(0))
    k_v = (np.linalg.norm(ah) + np.linalg.norm(ref["u_bot"]) + ref["beta"] + a_bot) / ref["alpha"]
    return max(1e-5, 8 * 6e-8 * max(k_u, k_v))


@pytest.mark.parametrize("name,kw,K", TF_CASES)
def test_teacher_forced_steps(torch_cuda, name, kw, K, record_property):
    """Every iteration: load the GPU's state k-1 into the oracle's single step and compare the
    step-k outputs (u, v, w, x, alpha, beta, phibar, rhobar).  This is the correctness gate that
    holds on every config, including configs[0] where free-running complex64 cannot track
    complex128."""
    torch = torch_cuda
    tol = 1e-5
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = ops_for(w)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    ctx.lsqr_begin(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    st = ctx.lsqr_peek()
    # start vectors against the oracle's definition
    for s in range(w.nb):
        b_top = w.lam * w.Q[:, s].astype(complex)
        b_bot = w.D[:, s].astype(complex)
        beta1 = math.sqrt((abs(b_top) ** 2).sum() + (abs(b_bot) ** 2).sum())
        assert st["beta"][s] == pytest.approx(beta1, rel=1e-6)
        v1 = O.apply_MH(ops[s], w.m, w.lam, rec, b_top / beta1, b_bot / beta1)
        g = gpu_state_column(st, s)
        assert rel(g["v"], v1 / np.linalg.norm(v1)) < tol
        assert g["alpha"] == pytest.approx(np.linalg.norm(v1), rel=tol)
    worst_tol = worst_err = 0.0
    for k in range(1, K + 1):
        prev = st
        ctx.lsqr_iterate(1)
        st = ctx.lsqr_peek()
        for s in range(w.nb):
            pv = gpu_state_column(prev, s)
            ref = O.lsqr_step(ops[s], w.m, w.lam, rec, pv)
            got = gpu_state_column(st, s)
            tol_k = _step_tolerance(name, ops[s], w, rec, pv, ref)
            errs = [rel(got[n], ref[n]) for n in ("u_top", "v", "w", "x")]
            if w.n_rec:   # receiver rows: error relative to the whole (unit-norm) vector u
                errs.append(float(np.linalg.norm(got["u_bot"] - ref["u_bot"])))
            errs += [abs(got[n] - ref[n]) / abs(ref[n]) for n in ("alpha", "beta", "phibar", "rhobar")]
            assert max(errs) < tol_k, (k, s, tol_k, errs)
            worst_tol, worst_err = max(worst_tol, tol_k), max(worst_err, max(errs))
    ctx.lsqr_end()
    # the data-dependent gate of configs[0] (8 eps kappa) is logged so that it cannot grow unseen
    print("teacher-forced %s %s: largest step tolerance %.2e (kappa %.0f), largest error %.2e"
          % (name, kw, worst_tol, worst_tol / (8 * 6e-8), worst_err))
    record_property("largest_step_tolerance", "%.3e" % worst_tol)
    record_property("largest_step_error", "%.3e" % worst_err)
    assert worst_tol < 2e-4                                  # kappa stays below ~400 on every case


def _free_run(torch, w, K, cols=None, threads=8):
    ctx = _wri(w)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    cols = list(range(w.nb)) if cols is None else cols
    ref = O.lsqr_batch(ops_for(w), w.m, w.lam, rec, w.Q, w.D, None, maxit=K, threads=threads, columns=cols)
    return u.cpu().numpy()[:, cols], res.cpu().numpy()[:, cols], it.cpu().numpy()[cols], ref


def test_free_running_config1_50_iterations(torch_cuda):
    """configs[1] (64^3 x 16 sources, lambda = 10): residual history and u after 50 iterations
    within 1e-3 relative L2 of the complex128 oracle."""
    w = workloads.make("config1")
    u, res, it, ref = _free_run(torch_cuda, w, 50, cols=[0, 5, 10, 15])
    assert (it == 50).all()
    for j in range(u.shape[1]):
        assert rel(res[:, j], ref["resnorms"][:, j]) < 1e-3
        assert rel(u[:, j], ref["x"][:, j]) < 1e-3


@pytest.mark.parametrize("name,kw,cols", [
    ("config2", dict(grid=(40, 36, 44), nb=6), None),
    ("config4", dict(grid=(48, 48, 48), nb=8), None),
    ("config3", dict(grid=(50, 50, 40), nb=12), None),
    ("config2", dict(grid=(45, 38, 70), nb=64), [0, 21, 42, 63]),      # TMA path, 3 z-chunks
    ("config4", dict(grid=(40, 44, 36), nb=32), [0, 13, 31]),
    ("config3", dict(grid=(50, 50, 40), nb=48), [0, 17, 47]),
    ("config1", dict(grid=(45, 38, 36), nb=16), [0, 9, 15]),           # merged (column, x) tensor maps
    ("config1", dict(grid=(37, 41, 40), nb=8), None),                  # 8- and 4-column tiles
    ("config4", dict(grid=(33, 35, 34), nb=4), None),
    ("config3", dict(grid=(70, 37, 34), nb=2), None),                  # 2-column tiles, ragged in x and y
    ("config2", dict(grid=(30, 27, 34), nb=56), [0, 30, 55]),
    ("config3", dict(grid=(30, 27, 34), nb=40), [0, 21, 39]),
    ("config3", dict(grid=(42, 27, 34), nb=24), [0, 11, 23]),
])
def test_free_running_scaled_configs(torch_cuda, name, kw, cols):
    w = workloads.make(name, **kw)
    u, res, it, ref = _free_run(torch_cuda, w, 50, cols=cols)
    for j in range(u.shape[1]):
        assert rel(res[:, j], ref["resnorms"][:, j]) < 1e-3
        assert rel(u[:, j], ref["x"][:, j]) < 1e-3


def test_config0_free_running_is_bounded_by_the_storage_floor(torch_cuda):
    """configs[0] (lambda = 1): complex64 storage cannot follow the complex128 iterates beyond
    k ~ 3 (C-12, a property of the problem).  Check what is attainable: k <= 3 within
    1e-3, and the TRUE residual of the GPU's x_50 (oracle arithmetic) within 25 % of the
    oracle's own ||r_50||."""
    torch = torch_cuda
    w = workloads.make("config0")
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    op = ops_for(w)[0]
    u3, res3, _, ref3 = _free_run(torch, w, 3)
    assert rel(u3[:, 0], ref3["x"][:, 0]) < 1e-3
    assert rel(res3[:, 0], ref3["resnorms"][:, 0]) < 1e-3
    u, res, it, ref = _free_run(torch, w, 50)
    x = u[:, 0].astype(complex)
    t, b = O.apply_M(op, w.m, w.lam, rec, x)
    r_true = math.sqrt((abs(w.lam * w.Q[:, 0].astype(complex) - t) ** 2).sum()
                       + (abs(w.D[:, 0].astype(complex) - b) ** 2).sum())
    assert abs(res[50, 0] / r_true - 1.0) < 0.05             # the GPU's own estimate is honest
    assert np.all(np.diff(res[:, 0]) <= 1e-6 * res[0, 0])    # monotone ||r_k||
    # against the attainable floor (the oracle's complex64-storage emulation, measured on CPU in
    # tests/test_oracle_c64floor.py): the GPU deviates from complex128 by no more than twice that
    from dataclasses import replace
    q0, d0 = w.Q[:, 0].astype(complex), w.D[:, 0].astype(complex)
    fx, fh, _ = c64_floor(lambda dd, r: O.lsqr(replace(op, round_c64=r), w.m, w.lam, rec, q0, dd, maxit=50), d0)
    dev_x, dev_h = rel(u[:, 0], ref["x"][:, 0]), rel(res[:, 0], ref["resnorms"][:, 0])
    print("configs[0] k = 50: GPU deviation x %.3e history %.3e; complex64 floor x %.3e history %.3e"
          % (dev_x, dev_h, fx, fh))
    assert dev_x <= 2.0 * fx and dev_h <= 2.0 * fh
    # ... and the TRUE residual of its x_50 (oracle arithmetic) is as far from the oracle's as the floor's
    fr = c64_floor.last_residual
    print("configs[0] k = 50: true residual of the GPU's x / oracle's %.4f; floor of that ratio 1 +- %.4f"
          % (r_true / ref["resnorms"][50, 0], fr))
    assert abs(r_true / ref["resnorms"][50, 0] - 1.0) <= 2.0 * fr + 1e-3


def test_adaptive_masks_config3(torch_cuda):
    """configs[3]-shaped: per-source tolerance, shrinking mask.  Stop iteration within +-2
    (or 2 %) of the oracle's; x compared with the oracle run to the GPU's own stop iteration."""
    torch = torch_cuda
    w = workloads.make("config3", grid=(50, 50, 40), nb=12)
    w.tol[:] = np.array([1e-1, 3e-2, 1e-2, 5e-2, 2e-2, 8e-2, 1e-1, 6e-2, 1.5e-2, 4e-2, 2.5e-2, 0.0],
                        dtype=np.float32)
    maxit = 120
    ctx = _wri(w)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    tol = torch.from_numpy(w.tol).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, tol, maxit=maxit, omega_idx=w.omega_idx)
    u, res, it = u.cpu().numpy(), res.cpu().numpy(), it.cpu().numpy()
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = ops_for(w)
    ref = O.lsqr_batch(ops, w.m, w.lam, rec, w.Q, w.D, w.tol, maxit=maxit, threads=8)
    assert it[-1] == maxit                                   # tol = 0 runs to maxit
    assert len(set(it.tolist())) > 4                         # the mask really shrinks
    for s in range(w.nb):
        assert abs(int(it[s]) - int(ref["iters"][s])) <= max(2, 0.02 * ref["iters"][s]), (s, it[s], ref["iters"][s])
        k = int(it[s])
        same = O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=0.0, maxit=k)
        if k <= 60:
            assert rel(u[:, s], same["x"]) < 1e-3
            assert rel(res[:k + 1, s], same["resnorms"]) < 1e-3
        else:
            # beyond ~60 iterations float32 Lanczos vectors lose orthogonality and the iterates
            # drift (C-12); the residual history stays robust
            assert rel(res[:k + 1, s], same["resnorms"]) < 5e-3
            assert rel(u[:, s], same["x"]) < 5e-2
        assert np.all(res[k:, s] == res[k, s])               # history held after the stop


def test_column_compaction_matches_uncompacted_and_oracle(torch_cuda, monkeypatch):
    """48 columns on the TMA path with tolerances spread over two decades: converged columns are
    compacted out of the working set (48 -> 32 -> 16 -> 8 -> 4 columns) and the solve returns once all have
    stopped.  Stop iterations, wavefields and histories must match the same solve without
    compaction and the oracle."""
    torch = torch_cuda
    w = workloads.make("config3", grid=(50, 50, 40), nb=48)
    rng = np.random.Generator(np.random.PCG64(5))
    w.tol[:] = (10.0 ** rng.uniform(-2.0, -0.7, w.nb)).astype(np.float32)
    w.tol[7] = 0.0                                           # one column runs to maxit
    maxit = 90
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    tol = torch.from_numpy(w.tol).cuda()

    def run(no_compact):
        ctx = _wri(w)
        ctx.set_debug_opts(no_compact=int(no_compact))
        out = [t.cpu().numpy() for t in ctx.lsqr_batch(q, d, w.lam, tol, maxit=maxit, omega_idx=w.omega_idx)]
        return out, ctx.lsqr_peek()["nb"], ctx.launch_count()

    (u, res, it), nb_end, n1 = run(False)
    (u0, res0, it0), nb_end0, n0 = run(True)
    assert nb_end0 == 48 and nb_end <= 8                     # the working set really shrank (48 -> ... -> a few)
    assert np.array_equal(it, it0) and it[7] == maxit and len(set(it.tolist())) > 8
    assert np.isfinite(u.view(np.float32)).all()
    for s in range(w.nb):
        assert rel(u[:, s], u0[:, s]) < 2e-5, s
        assert rel(res[:, s], res0[:, s]) < 1e-6, s
        assert np.all(res[it[s]:, s] == res[it[s], s])       # history held after the stop
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = ops_for(w)
    for s in (0, 7, 19, 33, 47):
        ref = O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=float(w.tol[s]), maxit=maxit)
        assert abs(int(it[s]) - int(ref["iters"])) <= 2, (s, it[s], ref["iters"])
        same = O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=0.0, maxit=int(it[s]))
        lim = 1e-3 if it[s] <= 60 else 5e-2
        assert rel(u[:, s], same["x"]) < lim, (s, it[s])
        assert rel(res[:it[s] + 1, s], same["resnorms"]) < 5e-3

    # every column converges early: the solve stops before maxit and still fills the history
    w.tol[:] = 5e-2
    tol2 = torch.from_numpy(w.tol).cuda()
    ctx = _wri(w)
    u2, res2, it2 = [t.cpu().numpy() for t in ctx.lsqr_batch(q, d, w.lam, tol2, maxit=maxit, omega_idx=w.omega_idx)]
    assert it2.max() < maxit and ctx.lsqr_peek()["k"] < maxit
    for s in (0, 21, 47):
        same = O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=0.0, maxit=int(it2[s]))
        assert rel(u2[:, s], same["x"]) < 1e-3
        assert np.all(res2[it2[s]:, s] == res2[it2[s], s]) and res2[maxit, s] > 0


def test_degenerate_columns_and_determinism(torch_cuda):
    """b = 0 column -> x = 0, iters = 0, no NaN anywhere; no receivers; two runs bit-identical."""
    torch = torch_cuda
    w = workloads.make("config1", grid=(20, 18, 16), nb=4)
    w.Q[:, 2] = 0
    w.D[:, 2] = 0
    ctx = _wri(w)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    a = [t.cpu().numpy() for t in ctx.lsqr_batch(q, d, w.lam, None, maxit=20, omega_idx=w.omega_idx)]
    b = [t.cpu().numpy() for t in ctx.lsqr_batch(q, d, w.lam, None, maxit=20, omega_idx=w.omega_idx)]
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    u, res, it = a
    assert np.isfinite(u.view(np.float32)).all() and np.isfinite(res).all()
    assert it[2] == 0 and not u[:, 2].any() and not res[:, 2].any()
    assert (it[[0, 1, 3]] == 20).all()
    # a column's answer does not depend on its neighbours' data
    w2 = workloads.make("config1", grid=(20, 18, 16), nb=4)
    w2.Q[:, 2] = 0
    w2.D[:, 2] = 0
    w2.Q[:, 1] *= 3.0
    q2 = torch.from_numpy(w2.Q).cuda()
    u2 = ctx.lsqr_batch(q2, d, w.lam, None, maxit=20, omega_idx=w.omega_idx)[0].cpu().numpy()
    assert np.array_equal(u2[:, 0], u[:, 0]) and np.array_equal(u2[:, 3], u[:, 3])


def test_no_receivers_and_host_entry(torch_cuda):
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri
    w = workloads.make("config1", grid=(16, 16, 16), nb=2)
    m = torch.from_numpy(w.m).cuda()
    ctx0 = Wri((w.nx, w.ny, w.nz), w.h, w.omegas, m, w.sponge_width, np.zeros((0, 3), np.int32), w.nb)
    q = torch.from_numpy(w.Q).cuda()
    d0 = torch.zeros((0, w.nb), dtype=torch.complex64, device="cuda")
    u, res, it = ctx0.lsqr_batch(q, d0, w.lam, None, maxit=15)
    none = np.zeros(0, dtype=np.int64)
    ref = O.lsqr(ops_for(w)[0], w.m, w.lam, none, w.Q[:, 0], np.zeros(0), maxit=15)
    assert rel(u.cpu().numpy()[:, 0], ref["x"]) < 1e-3
    # host-buffer entry gives the same bits as the device entry
    ctx = _wri(w)
    dd = torch.from_numpy(w.D).cuda()
    a = [t.cpu().numpy() for t in ctx.lsqr_batch(q, dd, w.lam, None, maxit=15, omega_idx=w.omega_idx)]
    qh, dh = torch.from_numpy(w.Q).pin_memory(), torch.from_numpy(w.D).pin_memory()
    b = [t.numpy() for t in ctx.lsqr_batch_host(qh, dh, w.lam, None, maxit=15, omega_idx=w.omega_idx)]
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_wide_batches_are_solved_in_64_column_groups(torch_cuda, monkeypatch):
    """nb = 128: wri_lsqr_batch works through two compact 64-column groups.
    Each group must give exactly what a separate solve of those 64 columns gives (a column's
    result does not depend on its batch, C-9), the lock-step 128-column solve (debug option no_groups) the
    same within rounding, the oracle within 1e-3; with tolerances, the source-free system, a warm
    start and the host entry as well."""
    torch = torch_cuda
    w = workloads.make("config2", grid=(24, 28, 40), nb=128)
    K = 30
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    ctx = _wri(w)
    u, res, it = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    assert (it.cpu().numpy() == K).all()
    for g in range(2):
        sl = slice(64 * g, 64 * g + 64)
        ug, rg, _ = ctx.lsqr_batch(q[:, sl].contiguous(), d[:, sl].contiguous(), w.lam, None, maxit=K,
                                   omega_idx=w.omega_idx[sl])
        assert torch.equal(torch.view_as_real(u[:, sl]), torch.view_as_real(ug))
        assert torch.equal(res[:, sl], rg)
    ctx.set_debug_opts(no_groups=1)
    u1, res1, _ = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    ctx.set_debug_opts()
    assert rel(u.cpu().numpy(), u1.cpu().numpy()) < 1e-5
    assert rel(res.cpu().numpy(), res1.cpu().numpy()) < 1e-6
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    cols = [0, 63, 64, 127]
    ref = O.lsqr_batch(ops_for(w), w.m, w.lam, rec, w.Q, w.D, None, maxit=K, threads=4, columns=cols)
    for j, s in enumerate(cols):
        assert rel(res[:, s].cpu().numpy(), ref["resnorms"][:, j]) < 1e-3
        assert rel(u[:, s].cpu().numpy(), ref["x"][:, j]) < 1e-3

    # per-column tolerances: groups compact on their own; same stop iterations as the lock-step solve
    rng = np.random.Generator(np.random.PCG64(5))
    tolh = (10.0 ** rng.uniform(-2.5, -0.5, w.nb)).astype(np.float32)
    tolh[7] = 0.0
    tol = torch.from_numpy(tolh).cuda()
    ut, rt, itt = ctx.lsqr_batch(q, d, w.lam, tol, maxit=80, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    ctx.set_debug_opts(no_groups=1)
    ut1, rt1, itt1 = ctx.lsqr_batch(q, d, w.lam, tol, maxit=80, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    ctx.set_debug_opts()
    assert torch.equal(itt, itt1) and int(itt[7]) == 80 and len(set(itt.cpu().tolist())) > 8
    assert rel(ut.cpu().numpy(), ut1.cpu().numpy()) < 1e-5
    assert rel(rt.cpu().numpy(), rt1.cpu().numpy()) < 1e-6

    # source-free system, then a warm continuation with the cold reference, grouped vs lock-step
    outs = {}
    for mode in ("groups", "lockstep"):
        if mode == "lockstep":
            ctx.set_debug_opts(no_groups=1)
        ar0 = torch.zeros(w.nb, dtype=torch.float64, device="cuda")
        ctx.set_opts(ar0_out=ar0)
        us, al, rs, its = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=12, omega_idx=w.omega_idx)
        ctx.set_opts(warm_start=True, ar_ref=ar0)
        us2, al2, rs2, its2 = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=8, omega_idx=w.omega_idx,
                                                out=(us.clone(), al.clone(),
                                                     torch.empty((9, w.nb), dtype=torch.float32, device="cuda"),
                                                     torch.empty(w.nb, dtype=torch.int32, device="cuda")))
        ctx.set_opts()
        torch.cuda.synchronize()
        outs[mode] = [t.cpu().numpy() for t in (us, al, rs, us2, al2, rs2, ar0)]
        if mode == "lockstep":
            ctx.set_debug_opts()
    for a, b in zip(outs["groups"], outs["lockstep"]):
        assert rel(a, b) < 2e-5
    assert np.all(outs["groups"][5][-1] < outs["groups"][2][-1])       # the continuation went on converging

    # host entry
    qh, dh = torch.from_numpy(w.Q).pin_memory(), torch.from_numpy(w.D).pin_memory()
    uh, rh, ith = ctx.lsqr_batch_host(qh, dh, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    assert np.array_equal(uh.numpy(), u.cpu().numpy()) and np.array_equal(rh.numpy(), res.cpu().numpy())


def test_pipelined_host_entry_equals_the_serial_one(torch_cuda):
    """wri_lsqr_batch_host_async: four solves with different inputs enqueued back to back (uploads
    and downloads ride under the neighbouring solves on the library's copy streams); after
    wri_host_wait every result equals the serial host entry's bit for bit; with tolerances and a
    128-column (grouped) batch as well."""
    torch = torch_cuda
    w = workloads.make("config2", grid=(24, 28, 40), nb=128)
    ctx = _wri(w)
    rng = np.random.Generator(np.random.PCG64(3))
    K = 12
    ins, outs = [], []
    tolh = (10.0 ** rng.uniform(-2.0, -0.7, w.nb)).astype(np.float32)
    for i in range(4):
        scale = np.float32(1.0 + 0.25 * i)
        q = torch.from_numpy((w.Q * scale).astype(np.complex64)).pin_memory()
        d = torch.from_numpy(np.roll(w.D, i, axis=1).copy()).pin_memory()
        tol = torch.from_numpy(tolh).pin_memory() if i == 2 else None
        ins.append((q, d, tol))
    for q, d, tol in ins:                                        # all enqueued before anything is read
        outs.append(ctx.lsqr_batch_host_async(q, d, w.lam, tol, maxit=K, omega_idx=w.omega_idx))
    ctx.host_wait()
    for (q, d, tol), (u, res, it) in zip(ins, outs):
        us, rs, its = ctx.lsqr_batch_host(q, d, w.lam, tol, maxit=K, omega_idx=w.omega_idx)
        assert np.array_equal(u.numpy(), us.numpy())
        assert np.array_equal(res.numpy(), rs.numpy()) and np.array_equal(it.numpy(), its.numpy())
    assert len(set(outs[2][2].numpy().tolist())) > 3             # the tolerance case really stopped early
    assert not np.array_equal(outs[0][0].numpy(), outs[1][0].numpy())
    # the source-free system through the pipeline, a known-source solve in between
    sf = [ctx.lsqr_sf_batch_host_async(ins[i][1], w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx)
          for i in (0, 1)]
    mid = ctx.lsqr_batch_host_async(ins[3][0], ins[3][1], w.lam, None, maxit=K, omega_idx=w.omega_idx)
    sf.append(ctx.lsqr_sf_batch_host_async(ins[2][1], w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx))
    ctx.host_wait()
    assert np.array_equal(mid[0].numpy(), outs[3][0].numpy())
    for i, (u, a, res, it) in zip((0, 1, 2), sf):
        us, as_, rs, its = ctx.lsqr_sf_batch_host(ins[i][1], w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx)
        assert np.array_equal(u.numpy(), us.numpy()) and np.array_equal(a.numpy(), as_.numpy())
        assert np.array_equal(res.numpy(), rs.numpy()) and np.array_equal(it.numpy(), its.numpy())


def test_two_contexts_and_a_side_stream(torch_cuda):
    """Two contexts (different grids, widths, receiver sets) used alternately, one of them on a
    non-default CUDA stream: each gives what it gives alone (no state shared between contexts; all
    work of a context is enqueued on the stream given at create)."""
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri
    wa = workloads.make("config1", grid=(32, 28, 24), nb=16)
    wb = workloads.make("config3", grid=(26, 30, 22), nb=48)
    side = torch.cuda.Stream()
    ca = _wri(wa)
    with torch.cuda.stream(side):
        mb = torch.from_numpy(wb.m).cuda()
        cb = Wri((wb.nx, wb.ny, wb.nz), wb.h, wb.omegas, mb, wb.sponge_width, wb.rec_ijk, wb.nb,
                 stream=side.cuda_stream)
        qb, db = torch.from_numpy(wb.Q).cuda(), torch.from_numpy(wb.D).cuda()
    qa, da = torch.from_numpy(wa.Q).cuda(), torch.from_numpy(wa.D).cuda()
    side.synchronize()
    K = 10
    ua0, ra0, _ = ca.lsqr_batch(qa, da, wa.lam, None, maxit=K, omega_idx=wa.omega_idx)
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        ub0, rb0, _ = cb.lsqr_batch(qb, db, wb.lam, None, maxit=K, omega_idx=wb.omega_idx)
    side.synchronize()
    ua0, ra0, ub0, rb0 = (t.clone() for t in (ua0, ra0, ub0, rb0))
    # interleaved, stepping entries, both in flight at once
    ua, ra, _ = ca.lsqr_begin(qa, da, wa.lam, None, maxit=K, omega_idx=wa.omega_idx)
    with torch.cuda.stream(side):
        ub, rb, _ = cb.lsqr_begin(qb, db, wb.lam, None, maxit=K, omega_idx=wb.omega_idx)
    for _ in range(K // 2):
        ca.lsqr_iterate(2)
        cb.lsqr_iterate(2)
    ca.lsqr_end()
    cb.lsqr_end()
    torch.cuda.synchronize()
    side.synchronize()
    assert torch.equal(ra, ra0) and torch.equal(torch.view_as_real(ua), torch.view_as_real(ua0))
    assert torch.equal(rb, rb0) and torch.equal(torch.view_as_real(ub), torch.view_as_real(ub0))
    rec = O.rec_cells(wb.nx, wb.ny, wb.nz, wb.rec_ijk)
    ref = O.lsqr(ops_for(wb)[5], wb.m, wb.lam, rec, wb.Q[:, 5], wb.D[:, 5], tol=0.0, maxit=K)
    assert rel(ub[:, 5].cpu().numpy(), ref["x"]) < 1e-3 and rel(rb[:, 5].cpu().numpy(), ref["resnorms"]) < 1e-3


def test_operator_entries_reuse_their_column_tables_only_when_the_columns_are_the_same(torch_cuda):
    """The operator / objective entries keep the per-column tables (omega^2, lambda, source cells) of their
    last call on the device and skip the upload when a call names the same columns.  One context called with
    changing frequencies per column, lambda, source nodes and width, with a re-packing adaptive solve in
    between (it rewrites those tables on the device): every result is bit-identical to the same single call
    on a fresh context."""
    torch = torch_cuda
    w = workloads.make("config2", grid=(24, 20, 28), nb=12)            # three frequencies, 4 columns each
    assert len(set(w.omega_idx.tolist())) == 3
    rng = np.random.Generator(np.random.PCG64(21))
    x = torch.from_numpy(_cn(rng, (w.ng, w.nb))).cuda()
    yb = torch.from_numpy(_cn(rng, (w.n_rec, w.nb))).cuda()
    al = torch.from_numpy(_cn(rng, (w.nb,))).cuda()
    d = torch.from_numpy(w.D).cuda()
    q = torch.from_numpy(w.Q).cuda()
    idx_a = w.omega_idx.copy()
    idx_b = np.ascontiguousarray(w.omega_idx[::-1])                    # other frequency per column
    src_a = w.src_ijk.copy()
    src_b = np.ascontiguousarray(w.src_ijk[::-1])
    assert not np.array_equal(src_a, src_b)

    def call(ctx, kind, idx, lam, src, nb):
        xs, ybs, als, ds = x[:, :nb].contiguous(), yb[:, :nb].contiguous(), al[:nb].contiguous(), d[:, :nb].contiguous()
        if kind == "M":
            t, b = ctx.apply_M(xs, lam, idx[:nb])
            return [t, b]
        if kind == "MH":
            return [ctx.apply_MH(xs, ybs, lam, idx[:nb])]
        if kind == "S":
            return list(ctx.apply_S(xs, als, lam, src[:nb], idx[:nb]))
        if kind == "SH":
            return list(ctx.apply_SH(xs, ybs, lam, src[:nb], idx[:nb]))
        g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
        fp, fd = ctx.objective_gradient(xs, ds, lam, omega_idx=idx[:nb], src_ijk=src[:nb], alpha=als, g=g)
        return [fp, fd, g]

    seq = [("M", idx_a, w.lam, src_a, 12), ("M", idx_a, w.lam, src_a, 12),        # same: tables reused
           ("MH", idx_a, w.lam, src_a, 12), ("M", idx_b, w.lam, src_a, 12),       # other frequencies
           ("MH", idx_b, 0.5 * w.lam, src_a, 12),                                  # other lambda
           ("S", idx_b, 0.5 * w.lam, src_a, 12), ("SH", idx_b, 0.5 * w.lam, src_b, 12),   # other source nodes
           ("G", idx_a, w.lam, src_b, 12), ("G", idx_a, w.lam, src_b, 12), ("G", idx_a, w.lam, src_a, 12),
           ("M", idx_a, w.lam, src_a, 8), ("M", idx_a, w.lam, src_a, 12),         # other width and back
           "solve",
           ("M", idx_a, w.lam, src_a, 12), ("G", idx_a, w.lam, src_a, 12), ("SH", idx_a, w.lam, src_a, 12)]
    ctx = _wri(w)
    ctx.ensure_workspace(w.nb, compaction=True)
    tol = torch.from_numpy(np.geomspace(1e-1, 1e-3, w.nb).astype(np.float32)).cuda()
    for step in seq:
        if step == "solve":
            # a source-free adaptive solve: writes the tables for its own columns and re-packs them on the device
            _, _, _, it = ctx.lsqr_sf_batch(d, w.lam, src_b, tol, maxit=80, omega_idx=idx_b)
            torch.cuda.synchronize()
            assert len(set(it.cpu().numpy().tolist())) > 1
            continue
        got = call(ctx, *step)
        fresh = _wri(w)
        want = call(fresh, *step)
        torch.cuda.synchronize()
        for a, b in zip(got, want):
            va = torch.view_as_real(a) if a.is_complex() else a
            vb = torch.view_as_real(b) if b.is_complex() else b
            assert torch.equal(va, vb), step[0]
        fresh.close()
    ctx.close()
