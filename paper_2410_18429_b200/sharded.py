"""Column sharding of the misfit evaluation over N ranks (one process per GPU, torch.distributed).

The systems S_ij are independent across sources and frequencies, so every rank
solves its own block of batch columns with no exchange inside LSQR.  The objective and the gradient
are SUMS over sources and frequencies (eq. 8-9): one all-reduce of the float32
[n_g] gradient and of the objective per misfit evaluation is the only collective of the method
(NCCL over NVLink on GPUs; 8 MB at 128^3 against >= 60 ms of solves, so it is not fused into a
kernel).  Every rank ends up with the same f and g, hence takes the same accept / reject decision
in Algorithm 2 without further communication.

Plumbing only: the arithmetic of a rank's block runs in libwri (Wri.misfit_sf); `evaluate` is
injectable so that the reduction logic can be exercised on CPU ranks (gloo) in the tests.
"""
from __future__ import annotations


def column_range(nb: int, rank: int, world: int):
    """Contiguous block [lo, hi) of the nb batch columns owned by `rank`; blocks differ by at most one."""
    base, rem = divmod(int(nb), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


class ShardedMisfit:
    """f4(m) = sum over ALL columns of 1/2 ||S x_bar - b||^2 and its gradient on N ranks.

    evaluate(lo, hi, eps, maxit, g, warm) -> (f_local: float, iters_local: int, state)
        the rank-local misfit of columns [lo, hi): adds the block's gradient into g (a float32
        [n_g] tensor on the rank's device, cleared by this class) and returns the block's objective;
        `warm` is the state a previous call returned (or None), for warm restarts.
    dist: torch.distributed (initialised) or None for a single process.
    """

    def __init__(self, nb_total, evaluate, n_g, device, dist=None):
        import torch
        self._t = torch
        self.dist = dist if (dist is not None and dist.is_initialized()) else None
        self.rank = self.dist.get_rank() if self.dist else 0
        self.world = self.dist.get_world_size() if self.dist else 1
        self.nb_total = int(nb_total)
        self.lo, self.hi = column_range(nb_total, self.rank, self.world)
        self.evaluate = evaluate
        self.g = torch.zeros(int(n_g), dtype=torch.float32, device=device)

    def misfit(self, eps, maxit, want_gradient=True, warm=None):
        """Returns (f, g, iters, state): f and iters summed over all ranks, g all-reduced in place
        (None when want_gradient is False), state = this rank's warm-start state."""
        t = self._t
        g = self.g if want_gradient else None
        if g is not None:
            g.zero_()
        if self.hi > self.lo:
            f_loc, it_loc, state = self.evaluate(self.lo, self.hi, eps, maxit, g, warm)
        else:
            f_loc, it_loc, state = 0.0, 0, None              # more ranks than columns
        if self.dist:
            s = t.tensor([float(f_loc), float(it_loc)], dtype=t.float64, device=self.g.device)
            self.dist.all_reduce(s, op=self.dist.ReduceOp.SUM)
            if g is not None:
                self.dist.all_reduce(g, op=self.dist.ReduceOp.SUM)
            f_loc, it_loc = float(s[0]), int(round(float(s[1])))
        return float(f_loc), g, int(it_loc), state

    def reduce(self, f, g=None):
        """Sum over ranks of an objective value and, in place, of a gradient tensor: the `reduce`
        argument of Wri.awri_step (wri_awri_opts.reduce).  Returns the summed objective."""
        if not self.dist:
            return float(f)
        t = self._t
        s = t.tensor([float(f)], dtype=t.float64, device=self.g.device)
        self.dist.all_reduce(s, op=self.dist.ReduceOp.SUM)
        if g is not None:
            self.dist.all_reduce(g, op=self.dist.ReduceOp.SUM)
        return float(s[0])

    def awri_step(self, awri_step_fn, /, *args, **kw):
        """One outer step of Algorithm 2 over all ranks' columns.  The decision logic (lines 4-14, the
        eps halving, the warm restart) lives in ONE place, the library's wri_awri_step; this is a
        pass-through that hands it the collective: awri_step_fn is Wri.awri_step bound to this rank's
        columns (or, on CPU ranks in the tests, the oracle's step), called as
        awri_step_fn(*args, reduce=self.reduce, **kw) — positional-only here, so that the step's own
        keyword arguments (step=, m_min=, ...) pass through untouched.
        Every rank sees the same f, f_tilde and g, hence takes the same decision."""
        return awri_step_fn(*args, reduce=self.reduce, **kw)


def wri_evaluator(ctx, d, lam, src_ijk, omega_idx, rmask=None):
    """evaluate() for ShardedMisfit on a GPU rank: Wri.misfit_sf on the rank's block of columns.
    d [n_rec, nb_total] (complex64, device), src_ijk [nb_total, 3], omega_idx [nb_total];
    rmask: optional per-source receiver sets, uint8 [n_rec, nb_total] (the rank's columns are cut
    out and handed to wri_set_receiver_mask)."""

    def evaluate(lo, hi, eps, maxit, g, warm):
        if rmask is not None:
            ctx.set_receiver_mask(rmask[:, lo:hi].contiguous())
        out = ctx.misfit_sf(d[:, lo:hi].contiguous(), lam, src_ijk[lo:hi], eps, maxit,
                            omega_idx=None if omega_idx is None else omega_idx[lo:hi], g=g, warm=warm)
        return out["f"], int(out["iters"].sum().item()), (out["u"], out["alpha"], out["ar0"])

    return evaluate
