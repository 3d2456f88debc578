"""Seeded input generators: determinism, shapes, value ranges, receiver validity (CPU only)."""
import math

import numpy as np
import pytest

import workloads


@pytest.mark.parametrize("name,kw", [
    ("config0", {}),
    ("config1", dict(grid=(24, 20, 28), nb=5)),
    ("config2", dict(grid=(20, 24, 16), nb=6)),
    ("config3", dict(grid=(40, 40, 32), nb=7)),
    ("config4", dict(grid=(32, 32, 32), nb=4)),
])
def test_generators_are_seeded_and_well_formed(name, kw):
    a, b = workloads.make(name, **kw), workloads.make(name, **kw)
    for f in ("m", "Q", "D", "rec_ijk", "tol", "omega_idx"):
        assert np.array_equal(getattr(a, f), getattr(b, f))
    assert a.m.dtype == np.float32 and a.Q.dtype == np.complex64 and a.D.dtype == np.complex64
    assert a.m.shape == (a.ng,) and a.Q.shape == (a.ng, a.nb) and a.D.shape == (a.n_rec, a.nb)
    v = 1.0 / np.sqrt(a.m.astype(np.float64))
    assert 1200.0 < v.min() and v.max() < 5600.0
    r = a.rec_ijk.astype(np.int64)
    assert (r >= 0).all() and (r[:, 0] < a.nx).all() and (r[:, 1] < a.ny).all() and (r[:, 2] < a.nz).all()
    cells = (r[:, 2] * a.ny + r[:, 1]) * a.nx + r[:, 0]
    assert np.unique(cells).size == cells.size
    assert ((a.Q != 0).sum(axis=0) == 1).all()          # point sources
    assert a.omega_idx.max() < len(a.freqs)


def test_config_sizes_match_baseline_json():
    w = workloads.make("config1")
    assert (w.nx, w.ny, w.nz, w.nb, w.n_rec, w.maxit, w.lam, w.sponge_width) == (64, 64, 64, 16, 256, 100, 10.0, 10)
    assert list(w.rec_ijk[0]) == [2, 2, 2] and list(w.rec_ijk[17]) == [6, 6, 2]
    assert list(w.src_ijk[0]) == [8, 8, 3] and list(w.src_ijk[5]) == [24, 24, 3]
    ric = (2 / math.sqrt(math.pi)) * (36 / 512) * math.exp(-36 / 64)
    assert abs(w.Q[(3 * 64 + 8) * 64 + 8, 0]) == pytest.approx(ric, rel=1e-6)
    qn = np.linalg.norm(w.Q.astype(complex), axis=0)
    dn = np.linalg.norm(w.D.astype(complex), axis=0)
    np.testing.assert_allclose(dn, qn, rtol=1e-5)
    w0 = workloads.make("config0")
    assert (w0.nb, w0.n_rec, w0.maxit, w0.lam, w0.sponge_width) == (1, 16, 50, 1.0, 8)
    assert w0.Q[(4 * 32 + 16) * 32 + 16, 0] == 1.0
    w3 = workloads.make("config3", grid=(50, 50, 40))
    assert w3.nb == 48 and (w3.tol >= 1e-3).all() and (w3.tol <= 1e-1).all()


def test_column_range_partitions():
    for nb, world in [(64, 2), (48, 5), (3, 4), (192, 8)]:
        got = [workloads.column_range(nb, r, world) for r in range(world)]
        assert got[0][0] == 0 and got[-1][1] == nb
        assert all(got[i][1] == got[i + 1][0] for i in range(world - 1))
        sizes = [b - a for a, b in got]
        assert max(sizes) - min(sizes) <= 1
