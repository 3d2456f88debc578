"""Parity of wri_objective_gradient (eq. 4, 8, 9) against
the complex128 oracle: objective terms per column and the gradient summed over the batch columns,
<= 1e-5 relative (float32 arithmetic, float64 sums); accumulation and determinism bit-exact."""
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


def _wri(w):
    from paper_2410_18429_b200 import Wri
    return Wri.from_workload(w)


def _cn(rng, shape):
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / math.sqrt(2)).astype(np.complex64)


def _oracle(w, u, d, q=None, alpha=None, cols=None):
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    src = O.rec_cells(w.nx, w.ny, w.nz, w.src_ijk)
    ops = ops_for(w)
    g = np.zeros(w.ng)
    fp, fd = np.zeros(w.nb), np.zeros(w.nb)
    for s in range(w.nb):
        fp[s], fd[s] = O.objective_gradient(
            ops[s], w.m, w.lam, rec, u[:, s], d[:, s], q=None if q is None else q[:, s],
            src=-1 if alpha is None else int(src[s]), alpha_src=0.0 if alpha is None else complex(alpha[s]), g=g)
    return fp, fd, g


CASES = [
    ("config1", dict(grid=(17, 13, 11), nb=1), "sf"),        # one thread per cell
    ("config2", dict(grid=(20, 33, 18), nb=3), "sf"),        # 3 threads per cell: shared-memory reduction
    ("config2", dict(grid=(24, 17, 40), nb=5), "q"),
    ("config1", dict(grid=(32, 32, 32), nb=16), "sf"),       # shuffle reduction, width 8
    ("config3", dict(grid=(27, 25, 20), nb=48), "both"),     # pass kernel, 3 chunks of 16 columns
    ("config2", dict(grid=(21, 18, 37), nb=64), "sf"),       # one warp per cell, three frequencies
    ("config4", dict(grid=(19, 22, 35), nb=32), "q"),
    ("config2", dict(grid=(12, 14, 10), nb=192), "sf"),      # pass kernel, 3 chunks of 64 columns
    ("config3", dict(grid=(30, 26, 22), nb=24), "sf"),       # 3 chunks of 8 (four lanes per cell, no shuffle step)
    ("config3", dict(grid=(22, 19, 24), nb=40), "both"),     # 5 chunks of 8
    ("config2", dict(grid=(16, 12, 18), nb=128), "q"),       # 2 chunks of 64
    ("config3", dict(grid=(20, 23, 17), nb=12), "sf"),       # chunk of 4 would be too narrow: generic, 6 threads per cell
    ("config3", dict(grid=(18, 20, 16), nb=44), "both"),     # likewise (4 x 11): generic, 22 threads per cell
]


@pytest.mark.parametrize("name,kw,mode", CASES)
def test_objective_and_gradient_match_oracle(torch_cuda, name, kw, mode):
    torch = torch_cuda
    w = workloads.make(name, **kw)
    ctx = _wri(w)
    rng = np.random.Generator(np.random.PCG64(23))
    u = _cn(rng, (w.ng, w.nb))
    alpha = _cn(rng, (w.nb,)) if mode in ("sf", "both") else None
    q = (_cn(rng, (w.ng, w.nb)) * np.float32(1e-3)).astype(np.complex64) if mode in ("q", "both") else None
    ud, dd = torch.from_numpy(u).cuda(), torch.from_numpy(w.D).cuda()
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    kwargs = dict(omega_idx=w.omega_idx, g=g)
    if alpha is not None:
        kwargs.update(src_ijk=w.src_ijk, alpha=torch.from_numpy(alpha).cuda())
    if q is not None:
        kwargs.update(q=torch.from_numpy(q).cuda())
    fp, fd = ctx.objective_gradient(ud, dd, w.lam, **kwargs)
    torch.cuda.synchronize()
    rfp, rfd, rg = _oracle(w, u, w.D, q=q, alpha=alpha)
    assert np.allclose(fp.cpu().numpy(), rfp, rtol=1e-5, atol=0)
    assert np.allclose(fd.cpu().numpy(), rfd, rtol=1e-5, atol=0)
    g1 = g.cpu().numpy()
    assert rel(g1, rg) < 1e-5
    # the source cells, where the -alpha e term lands, on their own
    if alpha is not None:
        src = O.rec_cells(w.nx, w.ny, w.nz, w.src_ijk)
        assert np.allclose(g1[src], rg[src], rtol=1e-4, atol=1e-5 * np.abs(rg).max())
    # accumulation: a second call adds the same numbers (x + x is exact in float32)
    fp2, fd2 = ctx.objective_gradient(ud, dd, w.lam, **kwargs)
    torch.cuda.synchronize()
    assert np.array_equal(g.cpu().numpy(), 2 * g1)
    assert np.array_equal(fp2.cpu().numpy(), fp.cpu().numpy()) and np.array_equal(fd2.cpu().numpy(), fd.cpu().numpy())
    # g = NULL computes the objective only
    kwargs["g"] = None
    fp3, _ = ctx.objective_gradient(ud, dd, w.lam, **kwargs)
    assert np.array_equal(fp3.cpu().numpy(), fp.cpu().numpy())


@pytest.mark.parametrize("nb", [16, 48, 192])
def test_pass_kernel_and_generic_kernel_agree(torch_cuda, nb):
    """The same evaluation through the pass kernel (one chunk, 3 x 16, 3 x 64) and through the generic
    kernel (debug option): objective to fp64 rounding of a differently grouped sum, gradient to 1e-5."""
    torch = torch_cuda
    w = workloads.make("config2", grid=(20, 18, 24), nb=nb)
    ctx = _wri(w)
    rng = np.random.Generator(np.random.PCG64(31))
    u = torch.from_numpy(_cn(rng, (w.ng, w.nb))).cuda()
    al = torch.from_numpy(_cn(rng, (w.nb,))).cuda()
    d = torch.from_numpy(w.D).cuda()
    out = []
    for generic in (0, 1):
        ctx.set_debug_opts(generic=generic)
        g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
        n0 = ctx.launch_count()
        fp, fd = ctx.objective_gradient(u, d, w.lam, omega_idx=w.omega_idx, src_ijk=w.src_ijk, alpha=al, g=g)
        torch.cuda.synchronize()
        out.append((fp.cpu().numpy(), fd.cpu().numpy(), g.cpu().numpy(), ctx.launch_count() - n0))
    (fp0, fd0, g0, l0), (fp1, fd1, g1, l1) = out
    assert (l0, l1) == (3, 2)                        # pass kernel + k_add_f32 + k_objective | k_grad + k_objective
    assert np.allclose(fp0, fp1, rtol=1e-6) and np.array_equal(fd0, fd1)
    assert rel(g0, g1) < 1e-5
    ctx.close()


def test_objective_equals_half_squared_residual_of_the_solve(torch_cuda):
    """After a source-free solve f_pde + f_data = 1/2 ||S x - b||^2 = 1/2 phibar_K^2 (eq. 5), and for the
    known-source solve likewise with q; the gradient agrees with the oracle's on the oracle's
    inputs rounded to complex64."""
    torch = torch_cuda
    w = workloads.make("config1", grid=(32, 32, 32), nb=16)
    ctx = _wri(w)
    d, q = torch.from_numpy(w.D).cuda(), torch.from_numpy(w.Q).cuda()
    K = 30
    u, a, res, it = ctx.lsqr_sf_batch(d, w.lam, w.src_ijk, None, maxit=K, omega_idx=w.omega_idx)
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    fp, fd = ctx.objective_gradient(u, d, w.lam, omega_idx=w.omega_idx, src_ijk=w.src_ijk, alpha=a, g=g)
    torch.cuda.synchronize()
    f = (fp + fd).cpu().numpy()
    assert np.allclose(f, 0.5 * res[K].cpu().numpy().astype(np.float64) ** 2, rtol=2e-3)
    rfp, rfd, rg = _oracle(w, u.cpu().numpy(), w.D, alpha=a.cpu().numpy())
    assert np.allclose(fp.cpu().numpy(), rfp, rtol=1e-4) and np.allclose(fd.cpu().numpy(), rfd, rtol=1e-5)
    assert rel(g.cpu().numpy(), rg) < 1e-4          # r = A u - alpha e cancels strongly at a near-solution
    u2, res2, _ = ctx.lsqr_batch(q, d, w.lam, None, maxit=K, omega_idx=w.omega_idx)
    fp, fd = ctx.objective_gradient(u2, d, w.lam, omega_idx=w.omega_idx, q=q)
    torch.cuda.synchronize()
    assert np.allclose((fp + fd).cpu().numpy(), 0.5 * res2[K].cpu().numpy().astype(np.float64) ** 2, rtol=2e-3)
