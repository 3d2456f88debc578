"""N > 1: columns are independent systems, so the path shards by batch columns with
no data-path collective.  World-size-2 gloo run on CPU: the two ranks' column blocks tile the batch,
each rank's results equal the single-process ones bit for bit, and bench.py's aggregation takes the
MAX of the times and the SUM of the iteration counts."""
import json
import os
import socket
import subprocess
import sys

import numpy as np

import workloads
from oracle import oracle as O

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_two_rank_gloo_column_sharding(tmp_path):
    out = tmp_path / "gloo.json"
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "tests", "_gloo_worker.py"), str(out)]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    got = json.loads(out.read_text())
    assert got["world"] == 2 and got["t_max"] == 2.0 and got["ncols"] == 5
    # single-process answer on the same workload
    w = workloads.make("config3", grid=(14, 12, 10), nb=5)
    w.tol[:] = np.array([1e-1, 0.0, 3e-2, 1e-2, 5e-2], dtype=np.float32)
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = [O.Operator(w.nx, w.ny, w.nz, w.h, w.omegas[j], w.sponge_width, w.gamma_max, w.power, w.faces)
           for j in w.omega_idx]
    ref = O.lsqr_batch(ops, w.m, w.lam, rec, w.Q, w.D, w.tol, maxit=40, threads=1)
    covered = []
    for lo, hi, iters, chk in got["parts"]:
        covered += list(range(lo, hi))
        assert iters == ref["iters"][lo:hi].tolist()
        assert chk == ref["x"][:, lo].real.sum().item()        # bit-identical first column of the block
    assert covered == list(range(w.nb))
    assert got["it_sum"] == int(ref["iters"].sum())
    assert len(set(ref["iters"].tolist())) > 2                  # the tolerances really differ


def test_reference_arm_is_rank0_only():
    """bench.py --impl reference under N ranks: ranks other than 0 print nothing and exit 0."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "config1_64cubed_x16src", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == ""
