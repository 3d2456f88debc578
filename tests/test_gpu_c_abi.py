"""The C ABI on its own: tests/c_abi/abi_demo.c (plain C99 + the CUDA runtime, no Python, no torch in
the process) is built against include/wri.h and libwri.so, run on a seeded problem, and its results
are compared with the CPU oracle: receiver rows bit-exact, operator 1e-5, LSQR history and x 1e-3."""
import math
import os
import shutil
import subprocess

import numpy as np
import pytest

import workloads
from oracle import oracle as O
from gpu_util import ops_for, rel

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_c_program_through_the_abi(tmp_path):
    from paper_2410_18429_b200 import lib_path
    gcc = shutil.which("gcc")
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    assert gcc and os.path.exists(os.path.join(cuda, "include", "cuda_runtime.h"))
    exe = tmp_path / "abi_demo"
    libdir = os.path.dirname(lib_path())
    subprocess.check_call([gcc, "-std=c99", "-O1", "-o", str(exe), os.path.join(ROOT, "tests", "c_abi", "abi_demo.c"),
                           "-I" + os.path.join(cuda, "include"), "-L" + os.path.join(cuda, "lib64"), "-L" + libdir,
                           "-l:libwri.so", "-lcudart", "-Wl,-rpath," + libdir, "-Wl,-rpath," + os.path.join(cuda, "lib64")])
    w = workloads.make("config2", grid=(24, 20, 36), nb=16)
    K = 8
    fin, fout = tmp_path / "in.bin", tmp_path / "out.bin"
    with open(fin, "wb") as f:
        f.write(np.array([w.nx, w.ny, w.nz, w.nb, w.n_rec, w.sponge_width, K, len(w.omegas)], dtype=np.int32).tobytes())
        f.write(np.array([w.h, w.lam], dtype=np.float64).tobytes())
        f.write(np.array(w.omegas, dtype=np.float64).tobytes())
        f.write(np.ascontiguousarray(w.omega_idx, dtype=np.int32).tobytes())
        f.write(np.ascontiguousarray(w.rec_ijk, dtype=np.int32).tobytes())
        f.write(np.ascontiguousarray(w.m, dtype=np.float32).tobytes())
        f.write(np.ascontiguousarray(w.Q, dtype=np.complex64).tobytes())
        f.write(np.ascontiguousarray(w.D, dtype=np.complex64).tobytes())
    r = subprocess.run([str(exe), str(fin), str(fout)], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stderr
    assert r.stdout.startswith("launches ") and int(r.stdout.split()[1]) > 2 * K
    raw = np.fromfile(fout, dtype=np.uint8)
    nv, nd = w.ng * w.nb, w.n_rec * w.nb
    o = 0
    ytop = raw[o:o + nv * 8].view(np.complex64).reshape(w.ng, w.nb); o += nv * 8
    ybot = raw[o:o + nd * 8].view(np.complex64).reshape(w.n_rec, w.nb); o += nd * 8
    u = raw[o:o + nv * 8].view(np.complex64).reshape(w.ng, w.nb); o += nv * 8
    res = raw[o:o + (K + 1) * w.nb * 4].view(np.float32).reshape(K + 1, w.nb); o += (K + 1) * w.nb * 4
    it = raw[o:o + w.nb * 4].view(np.int32); o += w.nb * 4
    f_pde = raw[o:o + w.nb * 8].view(np.float64); o += w.nb * 8
    f_data = raw[o:o + w.nb * 8].view(np.float64); o += w.nb * 8
    g = raw[o:o + w.ng * 4].view(np.float32); o += w.ng * 4
    assert o == raw.size
    rec = O.rec_cells(w.nx, w.ny, w.nz, w.rec_ijk)
    ops = ops_for(w)
    assert np.array_equal(ybot, w.Q[rec, :])
    assert (it == K).all()
    for s in (0, 7, 15):
        rt, _ = O.apply_M(ops[s], w.m, w.lam, rec, w.Q[:, s])
        assert rel(ytop[:, s], rt) < 1e-5
        ref = O.lsqr(ops[s], w.m, w.lam, rec, w.Q[:, s], w.D[:, s], tol=0.0, maxit=K)
        assert rel(res[:, s], ref["resnorms"]) < 1e-3 and rel(u[:, s], ref["x"]) < 1e-3
    # eq. 4 / eq. 9 at the program's own u, from the entry that allocates nothing (scratch in the library image)
    gsum = np.zeros(w.ng)
    for s in range(w.nb):
        fp, fd = O.objective_gradient(ops[s], w.m.astype(np.float64), w.lam, rec, u[:, s].astype(complex), w.D[:, s],
                                      q=w.Q[:, s].astype(complex), g=gsum)
        assert f_pde[s] == pytest.approx(fp, rel=1e-5) and f_data[s] == pytest.approx(fd, rel=1e-5), s
    assert rel(g, gsum) < 1e-5
