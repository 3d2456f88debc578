"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (same grid,
batch width, tile configuration and entry point; fewer iterations where the oracle needs them).

The complex128 oracle solves sampled columns one by one (columns are independent systems,
PAPER.md:221); every column is additionally checked through properties that hold at any size:
receiver rows bit-exact, ||r_k|| monotone (LSQR minimises it over the Krylov space, DESIGN.md
C-13), the residual history equal to the TRUE residual ||b - M x_k|| of the returned wavefield,
history held after a stop (C-9), and bit-identical results run to run.
Tolerances: BASELINE.json north_star (operator 1e-5, history and u 1e-3 relative L2).
"""
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


def _wri(w):
    from paper_2410_18429_b200 import Wri
    return Wri.from_workload(w)


def _true_residual_norms(torch, ctx, w, q, d, u):
    """||[lam q; d] - M u|| per column: M u from the library's operator entry (checked against
    the oracle on sampled columns in the same test), norms in float64 with torch."""
    top, bot = ctx.apply_M(u, w.lam, w.omega_idx)
    rt = (w.lam * q - top).to(torch.complex128)
    rb = (d - bot).to(torch.complex128)
    n2 = (rt.real ** 2 + rt.imag ** 2).sum(0) + (rb.real ** 2 + rb.imag ** 2).sum(0)
    return n2.sqrt().cpu().numpy()


def _check_operator_columns(torch, ctx, w, x, cols, rec, stencil=0):
    top, bot = ctx.apply_M(x, w.lam, w.omega_idx)
    xh = x.cpu().numpy()
    assert np.array_equal(bot.cpu().numpy(), xh[rec, :])          # P: bit-exact indexing
    ops = ops_for(w, stencil)
    for s in cols:
        rt, _ = O.apply_M(ops[s], w.m, w.lam, rec, xh[:, s])
        assert rel(top[:, s].cpu().numpy(), rt) < 1e-5, s


def _fixed_k_case(torch, w, K, cols, threads, stencil=0):
    ctx = _wri(w)
    ctx.set_stencil(stencil)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    resh, ith = res.cpu().numpy(), it.cpu().numpy()
    # every column: iteration count, monotone history, history = true residual of the result
    assert (ith == K).all()
    assert np.isfinite(resh).all()
    assert np.all(np.diff(resh, axis=0) <= 1e-6 * resh[0][None, :])
    r_true = _true_residual_norms(torch, ctx, w, q, d, u)
    assert np.max(np.abs(resh[K] / r_true - 1.0)) < 1e-3
    # the operator entry used above, and the solve itself, against the oracle on sampled columns
    _check_operator_columns(torch, ctx, w, u, cols[:2], rec, stencil)
    ref = O.lsqr_batch(ops_for(w, stencil), w.m, w.lam, rec, w.Q, w.D, None, maxit=K, threads=threads, columns=cols)
    for j, s in enumerate(cols):
        assert rel(resh[:, s], ref["resnorms"][:, j]) < 1e-3, s
        assert rel(u[:, s].cpu().numpy(), ref["x"][:, j]) < 1e-3, s
    # bit-reproducible run to run
    u2, res2, _ = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    assert torch.equal(res, res2)
    assert torch.equal(torch.view_as_real(u), torch.view_as_real(u2))
    ctx.close()


def test_config2_128cubed_x64src_50_iterations(torch_cuda):
    """The headline workload (BASELINE.json metric: 128^3 x 64 sources, f = 6 Hz, lambda = 10):
    residual history and u after 50 iterations within 1e-3 of the oracle on columns 0, 31, 63."""
    w = workloads.make("config2", freqs=(6.0,))
    assert (w.nx, w.ny, w.nz, w.nb, w.n_rec) == (128, 128, 128, 64, 1024)
    _fixed_k_case(torch_cuda, w, 50, [0, 31, 63], threads=3)


def test_config2_128cubed_x64src_27_point_stencil(torch_cuda):
    """The headline workload with the 27-point discretisation (reading C-23), the configuration
    `bench.py --stencil 27` times: 50 iterations, columns 0 and 63 against the oracle's 27-point operator."""
    w = workloads.make("config2", freqs=(6.0,))
    _fixed_k_case(torch_cuda, w, 50, [0, 63], threads=2, stencil=1)


def test_config2_128cubed_x192col_three_frequencies(torch_cuda):
    """configs[2] in full: 64 sources x {4, 6, 8} Hz in one 192-column batch (solved as three compact
    64-column groups); one column per frequency against the oracle, 50 iterations."""
    w = workloads.make("config2")
    assert w.nb == 192 and len(set(w.omega_idx.tolist())) == 3
    _fixed_k_case(torch_cuda, w, 50, [5, 100, 191], threads=3)


def test_config4_256cubed_x32src(torch_cuda):
    """configs[4] (256^3 x 32 sources, 4096 receivers, sponge 16): 50 iterations, columns 0 and 31."""
    w = workloads.make("config4")
    assert (w.nx, w.ny, w.nz, w.nb, w.n_rec) == (256, 256, 256, 32, 4096)
    _fixed_k_case(torch_cuda, w, 50, [0, 31], threads=2)


def test_config3_vsp_adaptive_full_size(torch_cuda):
    """configs[3] (200 x 200 x 160, 48 sources, borehole receivers, per-source tolerances in
    [1e-3, 1e-1], maxit = 300, compaction of the shrinking batch): the three columns with the
    loosest tolerances are re-solved by the oracle (stop iteration within +-2, x and history at the
    GPU's own stop iteration within 1e-3); all 48 through the size-independent properties."""
    torch = torch_cuda
    w = workloads.make("config3")
    assert (w.nx, w.ny, w.nz, w.nb, w.n_rec) == (200, 200, 160, 48, 120)
    ctx = _wri(w)
    ctx.ensure_workspace(w.nb, compaction=True)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    tol = torch.from_numpy(w.tol).cuda()
    u, res, it = ctx.lsqr_batch(q, d, w.lam, tol, maxit=w.maxit, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    resh, ith = res.cpu().numpy(), it.cpu().numpy()
    assert np.isfinite(resh).all()
    assert ith.min() >= 1 and ith.max() <= w.maxit
    assert len(set(ith.tolist())) > 8                            # the mask really shrinks
    assert np.all(np.diff(resh, axis=0) <= 1e-6 * resh[0][None, :])
    for s in range(w.nb):
        assert np.all(resh[ith[s]:, s] == resh[ith[s], s])        # held after the stop (C-9)
    # looser tolerance never needs more iterations on these statistically alike columns by much:
    # rank correlation between tol and iters is strongly negative
    rk = lambda a: np.argsort(np.argsort(a))
    assert np.corrcoef(rk(w.tol), rk(ith))[0, 1] < -0.8
    r_true = _true_residual_norms(torch, ctx, w, q, d, u)
    final = resh[ith, np.arange(w.nb)]
    # long-running columns drift at float32 (C-12): 1e-3 up to 60 iterations, 5e-3 beyond
    lim = np.where(ith <= 60, 1e-3, 5e-3)
    assert np.all(np.abs(final / r_true - 1.0) < lim)
    loose = [int(s) for s in np.argsort(-w.tol)[:3]]
    _check_operator_columns(torch, ctx, w, u, loose[:1], rec)
    ops = ops_for(w)

    def one(s):
        r = O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=float(w.tol[s]), maxit=w.maxit)
        k = int(ith[s])
        same = r if int(r["iters"]) == k else O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s],
                                                       tol=0.0, maxit=k)
        return s, int(r["iters"]), same

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(3) as ex:
        outs = list(ex.map(one, loose))
    for s, k_ref, same in outs:
        k = int(ith[s])
        assert abs(k - k_ref) <= 2, (s, k, k_ref)
        assert rel(resh[:k + 1, s], same["resnorms"][:k + 1]) < 1e-3, s
        assert rel(u[:, s].cpu().numpy(), same["x"]) < 1e-3, s
    ctx.close()


def test_config3_vsp_tightest_columns_through_the_repacking(torch_cuda):
    """configs[3] at full size, the columns that live longest: the adaptive solve is cut at maxit = 50.
    By then the loose half of the batch has stopped and the working set has been re-packed about ten
    times (48 -> ~22 columns); the three columns with the TIGHTEST tolerances have run all 50
    iterations through every one of those re-packings.  Their wavefield and residual history at
    k = 50 against the oracle's fixed-K solve, 1e-3 relative L2 (north_star)."""
    torch = torch_cuda
    w = workloads.make("config3")
    ctx = _wri(w)
    ctx.ensure_workspace(w.nb, compaction=True)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    tol = torch.from_numpy(w.tol).cuda()
    K = 50
    u, res, it = ctx.lsqr_batch(q, d, w.lam, tol, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    resh, ith = res.cpu().numpy(), it.cpu().numpy()
    assert (ith < K).sum() >= 20 and (ith == K).sum() >= 10       # the batch really shrank on the way
    tight = [int(s) for s in np.argsort(w.tol)[:3]]
    assert all(ith[s] == K for s in tight)
    ref = O.lsqr_batch(ops_for(w), w.m, w.lam, rec, w.Q, w.D, None, maxit=K, threads=3, columns=tight)
    for j, s in enumerate(tight):
        assert rel(resh[:, s], ref["resnorms"][:, j]) < 1e-3, s
        assert rel(u[:, s].cpu().numpy(), ref["x"][:, j]) < 1e-3, s
    # and the same columns do not depend on the re-packing: bit-identical to the plain fixed-K solve
    u2, res2, _ = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    for s in tight:
        assert torch.equal(res[:, s], res2[:, s]), s
        assert torch.equal(torch.view_as_real(u[:, s]), torch.view_as_real(u2[:, s])), s
    ctx.close()


def test_config2_128cubed_x64src_source_free_and_misfit(torch_cuda):
    """The headline grid and batch width through the paper's own system (source weight unknown,
    b = [0; d]) and one misfit evaluation (solve to a tolerance + eq. 8-9), in bench.py's launch
    configuration.  Sampled columns against the oracle where complex64 can follow it (k <= 3, C-16);
    every column through oracle-independent properties; the group gradient against the oracle's
    eq. 9 evaluated on the GPU's own wavefields (all 64 columns)."""
    torch = torch_cuda
    w = workloads.make("config2", freqs=(6.0,))
    ctx = _wri(w)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    srcc = O.rec_cells(w.nx, w.ny, w.nz, w.src_ijk)
    ops = ops_for(w)
    d = torch.from_numpy(w.D).cuda()
    m64 = w.m.astype(np.float64)
    # three free-running iterations: x and the history follow the oracle
    u3, a3, res3, _ = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=3, omega_idx=w.omega_idx)
    torch.cuda.synchronize()
    cols = [0, 31, 63]
    for s in cols:
        r = O.lsqr_sf(ops[s], m64, w.lam, rec, int(srcc[s]), w.D[:, s], tol=0.0, maxit=3)
        assert rel(res3[:, s].cpu().numpy(), r["resnorms"]) < 1e-3, s
        assert rel(u3[:, s].cpu().numpy(), r["x"]) < 1e-3, s
        assert abs(complex(a3[s].item()) - r["alpha_src"]) <= 1e-3 * abs(r["alpha_src"]), s
    # misfit evaluation at eps = 1e-2
    eps, maxit = 1e-2, 200
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    out = ctx.misfit_sf(d, w.lam, w.src_ijk, eps, maxit, omega_idx=w.omega_idx, g=g)
    it = out["iters"].cpu().numpy()
    assert it.min() >= 1 and it.max() < maxit
    f_cols = (out["f_pde"] + out["f_data"]).cpu().numpy()
    assert out["f"] == pytest.approx(float(f_cols.sum()), rel=1e-12)
    u, al = out["u"].cpu().numpy(), out["alpha"].cpu().numpy()
    gsum = np.zeros(w.ng)

    def one(s):
        gs = np.zeros(w.ng)
        fp, fd = O.objective_gradient(ops[s], m64, w.lam, rec, u[:, s].astype(complex), w.D[:, s],
                                      src=int(srcc[s]), alpha_src=complex(al[s]), g=gs)
        return s, fp + fd, gs

    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(8) as ex:
        for s, f_true, gs in ex.map(one, range(w.nb)):
            assert f_cols[s] == pytest.approx(f_true, rel=1e-5), s          # honest objective, every column
            gsum += gs
    assert rel(g.cpu().numpy(), gsum) < 1e-5
    # the stop rule holds in oracle arithmetic (sampled columns), and the oracle stops in the same band
    ar0 = out["ar0"].cpu().numpy()
    for s in cols:
        t, b = O.apply_S(ops[s], m64, w.lam, rec, int(srcc[s]), u[:, s].astype(complex), complex(al[s]))
        xu, xa = O.apply_SH(ops[s], m64, w.lam, rec, int(srcc[s]), -t, w.D[:, s].astype(complex) - b)
        ar_true = float(np.sqrt(np.vdot(xu, xu).real + abs(xa) ** 2))
        assert ar_true <= 1.05 * eps * ar0[s], s
        r = O.lsqr_sf(ops[s], m64, w.lam, rec, int(srcc[s]), w.D[:, s], tol=eps, maxit=maxit)
        assert abs(int(it[s]) - r["iters"]) <= max(2, int(0.4 * r["iters"])), (s, it[s], r["iters"])
        assert f_cols[s] == pytest.approx(0.5 * r["resnorms"][r["iters"]] ** 2, rel=5e-3), s
        assert ar0[s] == pytest.approx(r["arnorms"][0], rel=1e-5), s
    ctx.close()


def test_config3_vsp_objective_and_gradient_full_size(torch_cuda):
    """configs[3]'s grid and width (200 x 200 x 160, 48 columns: the gradient pass runs as three chunks of
    16 columns) through eq. 4 / eq. 9 at a random wavefield with a known source q and a source weight on
    top: f_pde, f_data of every column and the group gradient against the oracle, 1e-5."""
    torch = torch_cuda
    from concurrent.futures import ThreadPoolExecutor
    w = workloads.make("config3")
    assert (w.nx, w.ny, w.nz, w.nb) == (200, 200, 160, 48)
    ctx = _wri(w)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    srcc = O.rec_cells(w.nx, w.ny, w.nz, w.src_ijk)
    ops = ops_for(w)
    gen = torch.Generator(device="cuda").manual_seed(11)
    u = torch.view_as_complex(torch.randn((w.ng, w.nb, 2), dtype=torch.float32, device="cuda", generator=gen))
    al = torch.view_as_complex(torch.randn((w.nb, 2), dtype=torch.float32, device="cuda", generator=gen))
    q, d = torch.from_numpy(w.Q).cuda(), torch.from_numpy(w.D).cuda()
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    fp, fd = ctx.objective_gradient(u, d, w.lam, omega_idx=w.omega_idx, q=q, src_ijk=w.src_ijk, alpha=al, g=g)
    torch.cuda.synchronize()
    fp, fd, uh, alh = fp.cpu().numpy(), fd.cpu().numpy(), u.cpu().numpy(), al.cpu().numpy()
    m64 = w.m.astype(np.float64)

    def one(s):
        gs = np.zeros(w.ng)
        a, b = O.objective_gradient(ops[s], m64, w.lam, rec, uh[:, s].astype(complex), w.D[:, s],
                                    q=w.Q[:, s].astype(complex), src=int(srcc[s]), alpha_src=complex(alh[s]), g=gs)
        return s, a, b, gs

    gsum = np.zeros(w.ng)
    with ThreadPoolExecutor(8) as ex:
        for s, a, b, gs in ex.map(one, range(w.nb)):
            assert fp[s] == pytest.approx(a, rel=1e-5) and fd[s] == pytest.approx(b, rel=1e-5), s
            gsum += gs
    assert rel(g.cpu().numpy(), gsum) < 1e-5
    ctx.close()
