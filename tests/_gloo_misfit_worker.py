"""Worker of tests/test_sharding.py::test_two_rank_gloo_misfit_and_adaptive_step (2 processes, gloo,
CPU).  Each rank evaluates the misfit of its block of columns with the CPU oracle (the stand-in for
Wri.misfit_sf on a box without GPUs); paper_2410_18429_b200.sharded does the partition, the
all-reduce of objective and gradient, and the Algorithm 2 step; rank 0 writes what it saw."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

from oracle import awri as A  # noqa: E402
from paper_2410_18429_b200.sharded import ShardedMisfit  # noqa: E402
from test_oracle_awri import _problem  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank = dist.get_rank()
    ops, m, rec, src, D, _ = _problem((9, 8, 7), 10, 5, seed=61)
    lam = 20.0
    model = {"m": m.copy()}

    def evaluate(lo, hi, eps, maxit, g, warm):
        r = A.misfit_sf(ops[lo:hi], model["m"], lam, rec, src[lo:hi], D[:, lo:hi], eps, maxit,
                        want_gradient=g is not None)
        if g is not None:
            g += torch.from_numpy(r["g"]).to(torch.float32)
        return r["f"], int(r["iters"].sum()), None

    sm = ShardedMisfit(5, evaluate, ops[0].ng, "cpu", dist)
    f, g, iters, _ = sm.misfit(1e-8, 2000)
    out = {"rank_cols": [sm.lo, sm.hi], "f": f, "g": g.double().numpy().tolist(), "iters": iters}

    # Algorithm 2 step with a rejection forced first (stateful update), then an accepted descent step
    t = 0.5 * float(np.abs(m).mean() / np.abs(g.numpy()).max())
    calls = [0]

    def update(mm, gg):
        sign = +1.0 if calls[0] == 0 else -1.0
        calls[0] += 1
        return mm + sign * t * gg

    # the decision logic is the step's own (the library's wri_awri_step on GPU ranks; here, on CPU
    # ranks, the oracle's); ShardedMisfit.awri_step only hands it the collective
    def oracle_step(*a, reduce, **k):
        return A.awri_step(*a, reduce=lambda f, gg: reduce(f, None if gg is None else torch.from_numpy(gg)), **k)

    lo, hi = sm.lo, sm.hi
    step = sm.awri_step(oracle_step, ops[lo:hi], m.copy(), lam, rec, src[lo:hi], D[:, lo:hi], 2e-3, 2000, update,
                        max_halvings=4)
    out["step"] = {k: step[k] for k in ("accepted", "n_halvings", "eps", "f", "f_trial", "lsqr_iters", "trace")}
    out["m_next"] = np.asarray(step["m"]).tolist()
    out["t"] = t
    gathered = [None] * dist.get_world_size()
    dist.all_gather_object(gathered, out)
    if rank == 0:
        with open(sys.argv[1], "w") as fh:
            json.dump(gathered, fh)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
