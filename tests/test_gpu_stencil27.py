"""GPU parity of the 27-point discretisation of the Laplacian (PAPER.md:56
"discretized 3D Laplacian"; reading C-23) against the oracle's definition (oracle stencil = 1,
pinned in tests/test_oracle_stencil27.py).  Same bars as the 7-point stencil (BASELINE.json north_star):
receiver rows bit-exact, one operator application <= 1e-5, teacher-forced LSQR step <= 1e-5, residual
history and u after 50 iterations <= 1e-3; objective and gradient (eq. 8-9) <= 1e-5.  Covers the persistent
pass kernel (even widths, several tile shapes, ragged tiles), the generic kernel (stepping entry at an odd
width) and the padded odd-width batch solve."""
import math
from dataclasses import replace

import numpy as np
import pytest

import workloads
from oracle import oracle as O
from gpu_util import gpu_state_column, rel

pytestmark = pytest.mark.gpu

WRI_STENCIL_27 = 1


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _wri27(w):
    from paper_2410_18429_b200 import Wri
    ctx = Wri.from_workload(w)
    ctx.set_stencil(WRI_STENCIL_27)
    return ctx


def _ops27(w):
    return [O.Operator(w.nx, w.ny, w.nz, w.h, w.omegas[j], w.sponge_width, w.gamma_max, w.power, w.faces,
                       stencil=1) for j in w.omega_idx]


def _cn(rng, shape):
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / math.sqrt(2)).astype(np.complex64)


SHAPES = [
    ("config1", dict(grid=(37, 41, 29), nb=1)),      # generic kernel
    ("config2", dict(grid=(24, 17, 40), nb=5)),
    ("config1", dict(grid=(37, 41, 29), nb=2)),      # pass kernel, every width class
    ("config3", dict(grid=(33, 30, 21), nb=6)),
    ("config3", dict(grid=(50, 50, 40), nb=16)),
    ("config2", dict(grid=(48, 40, 36), nb=48)),
    ("config2", dict(grid=(21, 18, 37), nb=64)),
]


@pytest.mark.parametrize("name,kw", SHAPES)
def test_apply_M_and_MH_27_match_oracle(torch_cuda, name, kw):
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri27(w)
    rng = np.random.Generator(np.random.PCG64(11))
    x = _cn(rng, (w.ng, w.nb))
    yt, yb = _cn(rng, (w.ng, w.nb)), _cn(rng, (w.n_rec, w.nb))
    xd, ytd, ybd = (torch.from_numpy(a).cuda() for a in (x, yt, yb))
    Mt, Mb = ctx.apply_M(xd, w.lam, w.omega_idx)
    MH = ctx.apply_MH(ytd, ybd, w.lam, w.omega_idx)
    Mt, Mb, MH = Mt.cpu().numpy(), Mb.cpu().numpy(), MH.cpu().numpy()
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    assert np.array_equal(Mb, x[rec, :])                                  # P: bit-exact indexing
    ops = _ops27(w)
    ops7 = [replace(op, stencil=0) for op in ops]
    for s in sorted(set([0, w.nb // 2, w.nb - 1])):
        rt, _ = O.apply_M(ops[s], w.m, w.lam, rec, x[:, s])
        assert rel(Mt[:, s], rt) < 1e-5
        rh = O.apply_MH(ops[s], w.m, w.lam, rec, yt[:, s], yb[:, s])
        assert rel(MH[:, s], rh) < 1e-5
        # ... and it is NOT the 7-point operator (the two differ by O(1) on a random field)
        r7, _ = O.apply_M(ops7[s], w.m, w.lam, rec, x[:, s])
        assert rel(Mt[:, s], r7) > 1e-2
    lhs = np.vdot(yt.astype(complex), Mt.astype(complex)) + np.vdot(yb.astype(complex), Mb.astype(complex))
    rhs = np.vdot(MH.astype(complex), x.astype(complex))
    assert abs(lhs - rhs) / abs(lhs) < 2e-5
    ctx.close()


TF_CASES = [
    ("config1", dict(grid=(24, 20, 28), nb=4), 6),
    ("config2", dict(grid=(20, 33, 18), nb=3), 5),       # generic kernel + one-block scalar kernels
    ("config3", dict(grid=(27, 25, 20), nb=48), 4),
    ("config2", dict(grid=(21, 18, 37), nb=64), 4),
    ("config1", dict(grid=(21, 34, 19), nb=8), 4),
]


@pytest.mark.parametrize("name,kw,K", TF_CASES)
def test_teacher_forced_steps_27(torch_cuda, name, kw, K):
    """Every iteration: the GPU's state k-1 goes through the oracle's single step (27-point operator) and
    the step-k outputs are compared, 1e-5."""
    torch = torch_cuda
    tol = 1e-5
    w = workloads.make(name, **kw)
    ctx = _wri27(w)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = _ops27(w)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    ctx.lsqr_begin(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    st = ctx.lsqr_peek()
    for s in range(w.nb):
        b_top, b_bot = w.lam * w.Q[:, s].astype(complex), w.D[:, s].astype(complex)
        beta1 = math.sqrt((abs(b_top) ** 2).sum() + (abs(b_bot) ** 2).sum())
        v1 = O.apply_MH(ops[s], w.m, w.lam, rec, b_top / beta1, b_bot / beta1)
        g = gpu_state_column(st, s)
        assert rel(g["v"], v1 / np.linalg.norm(v1)) < tol
        assert g["alpha"] == pytest.approx(np.linalg.norm(v1), rel=tol)
    for k in range(1, K + 1):
        prev = st
        ctx.lsqr_iterate(1)
        st = ctx.lsqr_peek()
        for s in range(w.nb):
            ref = O.lsqr_step(ops[s], w.m, w.lam, rec, gpu_state_column(prev, s))
            got = gpu_state_column(st, s)
            errs = [rel(got[n], ref[n]) for n in ("u_top", "v", "w", "x")]
            errs.append(float(np.linalg.norm(got["u_bot"] - ref["u_bot"])))
            errs += [abs(got[n] - ref[n]) / abs(ref[n]) for n in ("alpha", "beta", "phibar", "rhobar")]
            assert max(errs) < tol, (k, s, errs)
    ctx.lsqr_end()
    ctx.close()


FREE_CASES = [
    ("config1", dict(grid=(40, 36, 32)), [0, 7, 15]),            # configs[1]: 16 columns, pass kernel
    ("config1", dict(grid=(30, 27, 34), nb=5), [0, 2, 4]),       # odd width: padded working set
    ("config3", dict(grid=(42, 27, 34), nb=24), [0, 11, 23]),
]


@pytest.mark.parametrize("name,kw,cols", FREE_CASES)
def test_free_running_50_iterations_27(torch_cuda, name, kw, cols):
    """Residual history and u after 50 free-running iterations within 1e-3 of the oracle (north_star)."""
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri27(w)
    K = 50
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    assert (it.cpu().numpy() == K).all()
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ref = O.lsqr_batch(_ops27(w), w.m, w.lam, rec, w.Q, w.D, None, maxit=K, threads=3, columns=cols)
    resh, uh = res.cpu().numpy(), u.cpu().numpy()
    for j, s in enumerate(cols):
        assert rel(resh[:, s], ref["resnorms"][:, j]) < 1e-3, s
        assert rel(uh[:, s], ref["x"][:, j]) < 1e-3, s
    assert np.all(np.diff(resh, axis=0) <= 1e-6 * resh[0][None, :])        # ||r_k|| never grows
    ctx.close()


def test_adaptive_solve_27_does_not_depend_on_the_repacking(torch_cuda):
    """Per-column tolerances with the 27-point stencil: the re-packing variants of the passes have their
    own ST_27 instances; results bit-identical to the run that keeps every column in the working set."""
    torch = torch_cuda
    w = workloads.make("config3", grid=(40, 40, 32), nb=16)
    ctx = _wri27(w)
    ctx.ensure_workspace(w.nb, compaction=True)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    tol = torch.from_numpy(w.tol).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, tol, maxit=120, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    ith = it.cpu().numpy()
    assert len(set(ith.tolist())) > 4 and ith.min() < 120
    ctx.set_debug_opts(no_compact=1)
    u2, res2, it2 = ctx.lsqr_batch(q, d, w.lam, tol, maxit=120, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    assert torch.equal(it, it2) and torch.equal(res, res2)
    assert torch.equal(torch.view_as_real(u), torch.view_as_real(u2))
    # one column against the oracle at its own stop iteration
    s = int(np.argmax(ith < 120))
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    r = O.lsqr(_ops27(w)[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=0.0, maxit=int(ith[s]))
    assert rel(u[:, s].cpu().numpy(), r["x"]) < 1e-3
    ctx.close()


@pytest.mark.parametrize("name,kw", [("config1", dict(grid=(24, 20, 28), nb=16)),     # pass kernel (MODE_G)
                                      ("config3", dict(grid=(27, 25, 20), nb=48)),     # pass kernel, 3 chunks of 16
                                      ("config2", dict(grid=(20, 33, 18), nb=5))])     # generic k_grad
def test_objective_and_gradient_27(torch_cuda, name, kw):
    """eq. 4 and eq. 9 with the 27-point A: f_pde, f_data per column and the group gradient, 1e-5."""
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri27(w)
    rng = np.random.Generator(np.random.PCG64(5))
    u = _cn(rng, (w.ng, w.nb))
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    out = ctx.objective_gradient(torch.from_numpy(u).cuda(), torch.from_numpy(w.D).cuda(), w.lam,
                                 omega_idx=w.omega_idx, q=torch.from_numpy(w.Q).cuda(), g=g)
    f_pde, f_data = (t.cpu().numpy() for t in out[:2])
    ops = _ops27(w)
    gsum = np.zeros(w.ng)
    for s in range(w.nb):
        gs = np.zeros(w.ng)
        fp, fd = O.objective_gradient(ops[s], w.m.astype(np.float64), w.lam, rec, u[:, s].astype(complex),
                                      w.D[:, s], q=w.Q[:, s].astype(complex), g=gs)
        assert f_pde[s] == pytest.approx(fp, rel=1e-5) and f_data[s] == pytest.approx(fd, rel=1e-5), s
        gsum += gs
    assert rel(g.cpu().numpy(), gsum) < 1e-5
    ctx.close()
