"""Worker of tests/test_sharding.py, launched by torch.distributed.run with 2 processes (gloo, CPU).
Each rank takes its block of batch columns (workloads.column_range), solves them with the CPU oracle
(the stand-in for the GPU solve on a box without GPUs) and the ranks combine with bench.py's own
aggregation; rank 0 writes what it saw to the file given as argv[1]."""
import json
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import bench  # noqa: E402
import workloads  # noqa: E402
from oracle import oracle as O  # noqa: E402


def main():
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    w = workloads.make("config3", grid=(14, 12, 10), nb=5)
    w.tol[:] = np.array([1e-1, 0.0, 3e-2, 1e-2, 5e-2], dtype=np.float32)
    lo, hi = workloads.column_range(w.nb, rank, world)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = [O.Operator(w.nx, w.ny, w.nz, w.h, w.omegas[j], w.sponge_width, w.gamma_max, w.power, w.faces)
           for j in w.omega_idx]
    out = O.lsqr_batch(ops, w.m, w.lam, rec, w.Q, w.D, w.tol, maxit=40, threads=1, columns=list(range(lo, hi)))
    my_time = 1.0 + rank                       # synthetic per-rank step time: the job takes the MAX
    (t_max,), (it_sum, ncols) = bench.reduce_over_ranks([my_time], [int(out["iters"].sum()), hi - lo], dist)
    gathered = [None] * world
    dist.all_gather_object(gathered, (lo, hi, out["iters"].tolist(), out["x"][:, 0].real.sum().item()))
    if rank == 0:
        with open(sys.argv[1], "w") as f:
            json.dump({"t_max": t_max, "it_sum": it_sum, "ncols": ncols, "parts": gathered, "world": world}, f)
    dist.destroy_process_group()


if __name__ == "__main__":
    main()
