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
import pytest

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


def test_two_rank_gloo_misfit_and_adaptive_step(tmp_path):
    """paper_2410_18429_b200.sharded on 2 gloo ranks: the blocks tile the columns, the all-reduced
    objective and gradient equal the single-process ones (eq. 8-9 are sums over columns), both ranks
    see identical numbers and take the same Algorithm 2 decisions as the single-process oracle."""
    from oracle import awri as A
    from test_oracle_awri import _problem
    out = tmp_path / "gloo_misfit.json"
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "tests", "_gloo_misfit_worker.py"), str(out)]
    env = dict(os.environ, OMP_NUM_THREADS="1")
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, env=env, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    a, b = json.loads(out.read_text())
    assert a["rank_cols"] == [0, 3] and b["rank_cols"] == [3, 5]
    for k in ("f", "g", "iters", "m_next"):
        assert a[k] == b[k], k                                   # every rank holds the same result
    for k in a["step"]:                                          # ... and took the same decisions
        if k != "lsqr_iters":                                    # (iterations are counted per rank)
            assert a["step"][k] == b["step"][k], k
    ops, m, rec, src, D, _ = _problem((9, 8, 7), 10, 5, seed=61)
    ref = A.misfit_sf(ops, m, 20.0, rec, src, D, 1e-8, 2000)
    assert a["f"] == pytest.approx(ref["f"], rel=1e-13)
    assert a["iters"] == int(ref["iters"].sum())
    assert np.allclose(a["g"], ref["g"], rtol=1e-6, atol=1e-6 * np.abs(ref["g"]).max())    # float32 reduction buffer
    calls = [0]
    t = a["t"]

    def upd(mm, gg):
        sign = +1.0 if calls[0] == 0 else -1.0
        calls[0] += 1
        return mm + sign * t * gg

    rs = A.awri_step(ops, m, 20.0, rec, src, D, 2e-3, 2000, upd, max_halvings=4)
    st = a["step"]
    assert a["step"]["lsqr_iters"] + b["step"]["lsqr_iters"] == rs["lsqr_iters"]
    assert st["accepted"] and rs["accepted"] and st["n_halvings"] == rs["n_halvings"] == 1
    assert st["eps"] == pytest.approx(rs["eps"], rel=1e-15)
    for (e, f, ft), (er, fr, ftr) in zip(st["trace"], rs["trace"]):
        # (the trial model comes from the float32 all-reduce buffer of the gradient)
        assert e == pytest.approx(er) and f == pytest.approx(fr, rel=1e-9) and ft == pytest.approx(ftr, rel=1e-5)
    assert np.allclose(a["m_next"], rs["m"], rtol=1e-6)


def test_column_range_tiles_the_batch():
    from paper_2410_18429_b200.sharded import column_range
    for nb in (1, 5, 48, 64, 192):
        for world in (1, 2, 3, 8):
            parts = [column_range(nb, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == nb
            assert all(parts[i][1] == parts[i + 1][0] for i in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
            assert parts == [workloads.column_range(nb, r, world) for r in range(world)]


def test_reference_arm_is_rank0_only():
    """bench.py --impl reference under N ranks: ranks other than 0 print nothing and exit 0."""
    env = dict(os.environ, RANK="1", WORLD_SIZE="2", LOCAL_RANK="1")
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "config1_64cubed_x16src", "--steps", "1", "--warmup", "0"],
                       capture_output=True, text=True, timeout=300, env=env, cwd=ROOT)
    assert r.returncode == 0 and r.stdout.strip() == ""
