"""Per-source receiver sets P_i on the GPU: a 0/1 mask [n_rec][nb] selects, per batch
column, the receivers that record it.  The oracle needs nothing new: it takes the receiver list of
a column as an argument, so column s is checked against the oracle run with rec[mask[:, s]] and
d[mask[:, s], s].  Operator entries bit-exact / 1e-5, LSQR 1e-3, objective 1e-5 as elsewhere."""
import math

import numpy as np
import pytest

import workloads
from oracle import oracle as O
from gpu_util import ops_for, rel

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _cn(rng, shape):
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / math.sqrt(2)).astype(np.complex64)


def _mask(rng, n_rec, nb):
    m = (rng.uniform(size=(n_rec, nb)) < 0.6).astype(np.uint8)
    m[:, 0] = 1                     # one column with every receiver
    m[:, 1] = 0                     # one with none: pure PDE rows (b_bot = 0)
    m[0, 2:] = 1
    return m


@pytest.mark.parametrize("name,kw,K", [
    ("config1", dict(grid=(24, 20, 28), nb=16), 30),        # TMA path
    ("config2", dict(grid=(20, 33, 18), nb=5), 30),         # generic path
    ("config2", dict(grid=(24, 28, 26), nb=128), 12),       # two 64-column groups
])
def test_receiver_mask_operator_solve_objective(torch_cuda, name, kw, K):
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri
    from paper_2410_18429_b200.binding import WriError
    w = workloads.make(name, **kw)
    ctx = Wri.from_workload(w)
    rng = np.random.Generator(np.random.PCG64(17))
    mask = _mask(rng, w.n_rec, w.nb)
    md = torch.from_numpy(mask).cuda()
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = ops_for(w)
    ctx.set_receiver_mask(md)

    # operator entries
    x, yt, yb = _cn(rng, (w.ng, w.nb)), _cn(rng, (w.ng, w.nb)), _cn(rng, (w.n_rec, w.nb))
    xd, ytd, ybd = (torch.from_numpy(a).cuda() for a in (x, yt, yb))
    Mt, Mb = ctx.apply_M(xd, w.lam, w.omega_idx)
    MH = ctx.apply_MH(ytd, ybd, w.lam, w.omega_idx).cpu().numpy()
    assert np.array_equal(Mb.cpu().numpy(), np.where(mask[:, :] == 1, x[rec, :], 0))      # bit-exact rows
    cols = [0, 1, 2, w.nb - 1]
    for s in cols:
        sel = mask[:, s] == 1
        ref = O.apply_MH(ops[s], w.m, w.lam, rec[sel], yt[:, s], yb[sel, s])
        assert rel(MH[:, s], ref) < 1e-5, s

    # solve: column s against the oracle on its own receiver subset
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    u, res = u.cpu().numpy(), res.cpu().numpy()
    for s in cols:
        sel = mask[:, s] == 1
        r = O.lsqr(ops[s], w.m, w.lam, rec[sel], w.Q[:, s], w.D[sel, s], tol=0.0, maxit=K)
        assert rel(res[:, s], r["resnorms"]) < 1e-3, s
        assert rel(u[:, s], r["x"]) < 1e-3, s
    # the mask changes the answer where it hides receivers
    ctx.set_receiver_mask(None)
    u_all, _, _ = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    u_all = u_all.cpu().numpy()
    assert rel(u_all[:, 0], u[:, 0]) < 1e-6 and rel(u_all[:, 1], u[:, 1]) > 1e-2

    # objective / gradient at given wavefields
    ctx.set_receiver_mask(md)
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    ud = torch.from_numpy(x).cuda()
    fp, fd = ctx.objective_gradient(ud, d, w.lam, omega_idx=w.omega_idx, q=q, g=g)
    fp, fd = fp.cpu().numpy(), fd.cpu().numpy()
    for s in cols:
        sel = mask[:, s] == 1
        rfp, rfd = O.objective_gradient(ops[s], w.m, w.lam, rec[sel], x[:, s], w.D[sel, s], q=w.Q[:, s])
        assert fp[s] == pytest.approx(rfp, rel=1e-5) and fd[s] == pytest.approx(rfd, rel=1e-5, abs=1e-30)
    assert fd[1] == 0.0

    # a mask given for one width is refused at another
    if w.nb > 2:
        with pytest.raises(WriError):
            ctx.apply_M(xd[:, :2].contiguous(), w.lam, w.omega_idx[:2])
    ctx.set_receiver_mask(None)


def test_receiver_mask_source_free_with_tolerances(torch_cuda):
    """Source-free system, per-column tolerances and compaction with a mask: stop iterations within
    the complex64 band of the oracle's (C-16), true residual of the GPU's [u; alpha] (oracle
    arithmetic, on the column's own receivers) equal to its reported one."""
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri
    w = workloads.make("config3", grid=(40, 40, 32), nb=16)
    ctx = Wri.from_workload(w)
    rng = np.random.Generator(np.random.PCG64(19))
    mask = _mask(rng, w.n_rec, w.nb)
    mask[:, 1] = mask[:, 3]          # (a column without any receiver has b = 0: nothing to solve)
    ctx.set_receiver_mask(torch.from_numpy(mask).cuda())
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    srcc = O.rec_cells(w.nx, w.ny, w.nz, w.src_ijk)
    ops = ops_for(w)
    d = torch.from_numpy(w.D).cuda()
    tolh = (10.0 ** rng.uniform(-2.5, -1.0, w.nb)).astype(np.float32)
    u, al, res, it = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, torch.from_numpy(tolh).cuda(), maxit=200,
                                       omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    u, al, res, it = u.cpu().numpy(), al.cpu().numpy(), res.cpu().numpy(), it.cpu().numpy()
    assert len(set(it.tolist())) > 4
    for s in (0, 1, 5, 15):
        sel = mask[:, s] == 1
        r = O.lsqr_sf(ops[s], w.m, w.lam, rec[sel], int(srcc[s]), w.D[sel, s], tol=float(tolh[s]), maxit=200)
        # (the stop estimate is not monotone, C-13: the first crossing may come a little earlier too)
        assert abs(int(it[s]) - r["iters"]) <= max(2, math.ceil(0.4 * r["iters"])), (s, it[s], r["iters"])
        t, b = O.apply_S(ops[s], w.m, w.lam, rec[sel], int(srcc[s]), u[:, s].astype(complex), complex(al[s]))
        r_true = math.sqrt(float(np.vdot(t, t).real) + float(np.sum(np.abs(w.D[sel, s].astype(complex) - b) ** 2)))
        assert res[it[s], s] == pytest.approx(r_true, rel=2e-3), s
        assert res[it[s], s] == pytest.approx(r["resnorms"][r["iters"]], rel=5e-3), s
