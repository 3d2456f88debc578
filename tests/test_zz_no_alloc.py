"""wri_objective_gradient_static (include/wri.h): the objective / gradient entry (eq. 4,
98-110 eq. 8-9) for callers that may not allocate device memory.  Its scratch is a 4 MiB array in the
library image; it needs no workspace.  Checked here against the existing wri_objective_gradient at the
tolerance of the gradient tests (1e-5 relative), on two calls in a row that share the array: a wide case
first, then a narrower one whose rows land on the first call's leftovers, then the first case again.
Also: the call works on a context that never had a workspace, does not move torch's allocator
counters, and refuses a case beyond the limit before writing anything.

Collected last on purpose (the suite runs with pytest -x)."""
import math

import numpy as np
import pytest

import workloads
from gpu_util import rel

pytestmark = pytest.mark.gpu

TOL = 1e-5


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available()
    return torch


def _cn(rng, shape):
    return ((rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / math.sqrt(2)).astype(np.complex64)


class _Case:
    """Inputs on the device, outputs of both paths preallocated."""

    def __init__(self, torch, name, kw, seed, source_free):
        from paper_2410_18429_b200 import Wri
        self.w = w = workloads.make(name, **kw)
        rng = np.random.Generator(np.random.PCG64(seed))
        self.u = torch.from_numpy(_cn(rng, (w.ng, w.nb))).cuda()
        self.d = torch.from_numpy(w.D).cuda()
        self.q = None if source_free else torch.from_numpy(w.Q).cuda()
        self.src = w.src_ijk if source_free else None
        self.alpha = torch.from_numpy(_cn(rng, (w.nb,))).cuda() if source_free else None
        # the existing path: its own context with a workspace
        self.ref_ctx = Wri.from_workload(w)
        g_ref = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
        fp, fd = self.ref_ctx.objective_gradient(self.u, self.d, w.lam, omega_idx=w.omega_idx, q=self.q,
                                                 src_ijk=self.src, alpha=self.alpha, g=g_ref)
        torch.cuda.synchronize()
        self.ref = (fp.cpu().numpy(), fd.cpu().numpy(), g_ref.cpu().numpy())
        # the new path: a context that never gets a workspace; outputs allocated before the calls
        self.ctx = Wri.from_workload(w)
        self.f_pde = torch.empty(w.nb, dtype=torch.float64, device="cuda")
        self.f_data = torch.empty(w.nb, dtype=torch.float64, device="cuda")
        self.g = torch.empty(w.ng, dtype=torch.float32, device="cuda")

    def call_static(self):
        w = self.w
        self.f_pde.fill_(float("nan"))
        self.f_data.fill_(float("nan"))
        self.g.zero_()
        self.ctx.objective_gradient_static(self.u, self.d, w.lam, self.f_pde, self.f_data, omega_idx=w.omega_idx,
                                           q=self.q, src_ijk=self.src, alpha=self.alpha, g=self.g)

    def check(self, torch):
        torch.cuda.synchronize()
        fp, fd, g = self.ref
        got_fp, got_fd, got_g = self.f_pde.cpu().numpy(), self.f_data.cpu().numpy(), self.g.cpu().numpy()
        assert np.all(np.isfinite(got_fp)) and np.all(np.isfinite(got_fd))
        assert np.max(np.abs(got_fp - fp) / np.abs(fp)) < TOL
        assert np.max(np.abs(got_fd - fd) / np.abs(fd)) < TOL
        assert rel(got_g, g) < TOL

    def close(self):
        self.ref_ctx.close()
        self.ctx.close()


def test_static_scratch_entry_matches_the_workspace_path_on_calls_in_a_row(torch_cuda):
    torch = torch_cuda
    # A: 16 columns on the persistent pass kernel in the existing path (generic kernel in the new one), known source;
    # B: 5 columns (odd width, generic kernel in both), source-free right-hand side, other grid: fewer and
    #    shorter scratch rows than A, so its sums sit on top of A's
    a = _Case(torch, "config1", dict(grid=(40, 36, 32), nb=16), seed=3, source_free=False)
    b = _Case(torch, "config2", dict(grid=(24, 17, 40), nb=5), seed=4, source_free=True)
    try:
        torch.cuda.synchronize()
        before = torch.cuda.memory_stats()
        n_alloc = (before["allocation.all.allocated"], before["segment.all.allocated"])
        launches = a.ctx.launch_count()
        a.call_static()
        b.call_static()                      # second call straight behind the first, same stream
        assert a.ctx.launch_count() == launches + 2          # gradient kernel + objective fold, nothing else
        a.check(torch)
        b.check(torch)
        a.call_static()                      # and back: the array now holds B's rows
        a.check(torch)
        b.call_static()
        b.call_static()                      # same case twice: g is cleared by the caller in between
        b.check(torch)
        after = torch.cuda.memory_stats()
        assert (after["allocation.all.allocated"], after["segment.all.allocated"]) == n_alloc
        # bit-reproducible, like the existing entry
        g1, fp1 = a.g.clone(), a.f_pde.clone()
        a.call_static()
        torch.cuda.synchronize()
        assert torch.equal(a.g, g1) and torch.equal(a.f_pde, fp1)
    finally:
        a.close()
        b.close()


def test_static_scratch_entry_with_the_27_point_stencil_and_a_receiver_mask(torch_cuda):
    """The other template instances of the kernel and the per-source receiver sets go through the same entry."""
    torch = torch_cuda
    c = _Case(torch, "config3", dict(grid=(33, 30, 21), nb=6), seed=8, source_free=True)
    try:
        rng = np.random.Generator(np.random.PCG64(9))
        mask = torch.from_numpy((rng.random((c.w.n_rec, c.w.nb)) < 0.7).astype(np.uint8)).cuda()
        for ctx in (c.ref_ctx, c.ctx):
            ctx.set_stencil(1)
            ctx.set_receiver_mask(mask)
        g_ref = torch.zeros(c.w.ng, dtype=torch.float32, device="cuda")
        fp, fd = c.ref_ctx.objective_gradient(c.u, c.d, c.w.lam, omega_idx=c.w.omega_idx, src_ijk=c.src,
                                              alpha=c.alpha, g=g_ref)
        torch.cuda.synchronize()
        c.ref = (fp.cpu().numpy(), fd.cpu().numpy(), g_ref.cpu().numpy())
        c.call_static()
        c.check(torch)
        c.call_static()
        c.check(torch)
    finally:
        c.close()


@pytest.mark.parametrize("grid,nb", [((128, 128, 128), 64),      # the headline size: 4096 tiles x 64 columns, half the array
                                     ((24, 24, 256), 512)])      # 4608 tiles x 512 columns at the usual tile height:
def test_static_scratch_entry_at_sizes_near_its_limit(torch_cuda, grid, nb):   # fits only with tiles as tall as the grid
    """Sizes the header names as fitting: the result equals the workspace path's (1e-5) and, for the tall
    grid, the entry gets there by making its tiles taller (the default tiling would need 18.9 MB of sums)."""
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri
    w = workloads.make("config2", grid=grid, nb=4)
    rng = np.random.Generator(np.random.PCG64(17))
    gen = torch.Generator(device="cuda").manual_seed(5)
    u = torch.view_as_complex(torch.randn((w.ng, nb, 2), dtype=torch.float32, device="cuda", generator=gen))
    d = torch.view_as_complex(torch.randn((w.n_rec, nb, 2), dtype=torch.float32, device="cuda", generator=gen))
    al = torch.view_as_complex(torch.randn((nb, 2), dtype=torch.float32, device="cuda", generator=gen))
    idx = rng.integers(0, len(w.omegas), nb).astype(np.int32)
    src = np.stack([rng.integers(2, w.nx - 2, nb), rng.integers(2, w.ny - 2, nb), rng.integers(2, w.nz - 2, nb)],
                   axis=1).astype(np.int32)
    ref_ctx = Wri.from_workload(w, nb_max=nb)
    g_ref = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    fp, fd = ref_ctx.objective_gradient(u, d, w.lam, omega_idx=idx, src_ijk=src, alpha=al, g=g_ref)
    ctx = Wri.from_workload(w, nb_max=nb)
    f_pde = torch.empty(nb, dtype=torch.float64, device="cuda")
    f_data = torch.empty(nb, dtype=torch.float64, device="cuda")
    g = torch.zeros(w.ng, dtype=torch.float32, device="cuda")
    try:
        for _ in range(2):                   # two calls in a row on the shared array
            g.zero_()
            ctx.objective_gradient_static(u, d, w.lam, f_pde, f_data, omega_idx=idx, src_ijk=src, alpha=al, g=g)
            torch.cuda.synchronize()
            assert float(((f_pde - fp).abs() / fp.abs()).max()) < TOL
            assert float(((f_data - fd).abs() / fd.abs()).max()) < TOL
            assert float((g - g_ref).norm() / g_ref.norm()) < TOL
    finally:
        ref_ctx.close()
        ctx.close()


def test_static_scratch_entry_refuses_sizes_beyond_its_array(torch_cuda):
    """48 x 48 x 16 x 300 columns: one cell per thread-block row, so 48 x 48 tiles x 300 doubles = 5.5 MB
    of sums even with tiles as tall as the grid -> WRI_ERR_SCRATCH_LIMIT with a message that names the
    limit, nothing launched and the outputs untouched."""
    torch = torch_cuda
    from paper_2410_18429_b200 import Wri, WriError
    from paper_2410_18429_b200.binding import WRI_ERR_SCRATCH_LIMIT, WRI_STATIC_SCRATCH_BYTES
    assert WRI_STATIC_SCRATCH_BYTES == 4 << 20
    nb = 300
    w = workloads.make("config2", grid=(48, 48, 16), nb=4)
    ctx = Wri.from_workload(w, nb_max=nb)
    try:
        u = torch.zeros((w.ng, nb), dtype=torch.complex64, device="cuda")
        d = torch.zeros((w.n_rec, nb), dtype=torch.complex64, device="cuda")
        f_pde = torch.full((nb,), -7.0, dtype=torch.float64, device="cuda")
        f_data = torch.full((nb,), -7.0, dtype=torch.float64, device="cuda")
        launches = ctx.launch_count()
        with pytest.raises(WriError) as ei:
            ctx.objective_gradient_static(u, d, w.lam, f_pde, f_data)
        assert ei.value.code == WRI_ERR_SCRATCH_LIMIT
        assert "WRI_STATIC_SCRATCH_BYTES" in str(ei.value) and "4 MiB" in str(ei.value)
        torch.cuda.synchronize()
        assert ctx.launch_count() == launches
        assert bool((f_pde == -7.0).all()) and bool((f_data == -7.0).all())
    finally:
        ctx.close()
