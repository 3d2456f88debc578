"""Seeded generators for BASELINE.json configs[0..4] (recipes: DESIGN.md "Input recipe").

No method arithmetic here: velocity models, point sources, receiver node lists
and random data only.  Everything is built in float64 and rounded once to
float32 (m) / complex64 (Q, D); the CUDA path and the oracle both read the
rounded arrays.

Structure follows the paper's workloads: point sources near the surface,
receivers on a surface grid or down a borehole, layered models with compact
anomalies, single frequencies of 4-10 Hz.
The paper's own models exist only as figures, so these stand in for them.

Layouts: cell c = (iz*ny + iy)*nx + ix; Q[c, s], D[r, s] are source-interleaved
(column s fastest).
"""
from __future__ import annotations

import math
import os
from dataclasses import dataclass, field

import numpy as np

CONFIG_NAMES = ("config0", "config1", "config2", "config3", "config4")

_GOLDEN = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))),
                       "tests", "golden")


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    h: float
    freqs: tuple            # unique frequencies (Hz); omega = 2*pi*f
    omega_idx: np.ndarray   # int32 [nb], index into freqs per column
    m: np.ndarray           # float32 [n_g], squared slowness s^2/m^2
    sponge_width: int
    rec_ijk: np.ndarray     # int32 [n_r, 3] = (ix, iy, iz)
    Q: np.ndarray           # complex64 [n_g, nb]
    D: np.ndarray           # complex64 [n_r, nb]
    lam: float
    tol: np.ndarray         # float32 [nb]; 0 => run exactly maxit
    maxit: int
    seed: int
    src_ijk: np.ndarray = field(default=None)   # int32 [nb, 3]
    gamma_max: float = 1.0
    power: int = 2
    faces: int = 0x3F

    @property
    def ng(self):
        return self.nx * self.ny * self.nz

    @property
    def nb(self):
        return int(self.Q.shape[1])

    @property
    def n_rec(self):
        return int(self.rec_ijk.shape[0])

    @property
    def omegas(self):
        return tuple(2.0 * math.pi * f for f in self.freqs)


def column_range(nb: int, rank: int, world: int):
    """Contiguous block of batch columns owned by `rank` (columns are independent
    systems, so sharding needs no exchange)."""
    base, rem = divmod(nb, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


# ----------------------------------------------------------------------------- helpers

def _rng(seed):
    return np.random.Generator(np.random.PCG64(seed))


def _cn(rng, shape):
    """Standard complex Gaussian CN(0,1) = (N(0,1) + i N(0,1)) / sqrt(2)."""
    return (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) / math.sqrt(2.0)


def _lattice(n: int, k: int) -> np.ndarray:
    """k nodes evenly spread over n cells: floor((i + 0.5) n / k)."""
    return np.floor((np.arange(k) + 0.5) * n / k).astype(np.int64)


def _ricker(f, f0):
    return (2.0 / math.sqrt(math.pi)) * (f * f / f0 ** 3) * math.exp(-(f * f) / (f0 * f0))


def _coords(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                          np.arange(nx, dtype=np.float64), indexing="ij")
    return x, y, z


def _add_anomalies(v, rng, n, amp, sigma, L, signs="seeded"):
    nz, ny, nx = v.shape
    x, y, z = _coords(nx, ny, nz)
    for _ in range(n):
        cx = rng.uniform(L, nx - 1 - L)
        cy = rng.uniform(L, ny - 1 - L)
        cz = rng.uniform(L, nz - 1 - L)
        sgn = 1.0 if signs == "plus" else (1.0 if rng.uniform() < 0.5 else -1.0)
        r2 = (x - cx) ** 2 + (y - cy) ** 2 + (z - cz) ** 2
        v *= 1.0 + sgn * amp * np.exp(-r2 / (2.0 * sigma * sigma))
    return v


def _unique_nodes(ijk, nx, ny):
    ijk = np.asarray(ijk, dtype=np.int64).reshape(-1, 3)
    cell = (ijk[:, 2] * ny + ijk[:, 1]) * nx + ijk[:, 0]
    _, first = np.unique(cell, return_index=True)
    return ijk[np.sort(first)].astype(np.int32)


def _grid_nodes(xs, ys, iz):
    gx, gy = np.meshgrid(xs, ys, indexing="xy")
    return np.stack([gx.ravel(), gy.ravel(), np.full(gx.size, iz)], axis=1)


def _point_sources(ng, nx, ny, src_ijk, amps):
    nb = len(src_ijk)
    Q = np.zeros((ng, nb), dtype=np.complex64)
    for s, (ix, iy, iz) in enumerate(src_ijk):
        Q[(int(iz) * ny + int(iy)) * nx + int(ix), s] = amps[s]
    return Q


def _gaussian_data(rng, n_rec, Q):
    """CN data scaled column-wise so that ||d_s|| = ||q_s||."""
    nb = Q.shape[1]
    D = _cn(rng, (n_rec, nb))
    qn = np.sqrt((np.abs(Q.astype(np.complex128)) ** 2).sum(axis=0))
    dn = np.sqrt((np.abs(D) ** 2).sum(axis=0))
    return (D * (qn / dn)[None, :]).astype(np.complex64)


def _select(n_full, nb):
    if nb is None or nb >= n_full:
        return np.arange(n_full)
    return np.unique(np.round(np.linspace(0, n_full - 1, nb)).astype(np.int64))


def _scale_L(L_full, n, n_full):
    return int(max(2, min(round(L_full * n / n_full), (n - 2) // 2)))


def _finish(name, grid, h, freqs, col_f, v, L, rec, src, amps, lam, tol, maxit, seed, rng, D=None):
    nx, ny, nz = grid
    ng = nx * ny * nz
    m = (1.0 / (v * v)).reshape(-1).astype(np.float32)
    rec = _unique_nodes(rec, nx, ny)
    src = np.asarray(src, dtype=np.int32).reshape(-1, 3)
    Q = _point_sources(ng, nx, ny, src, amps)
    if D is None:
        D = _gaussian_data(rng, rec.shape[0], Q)
    nb = Q.shape[1]
    tol = np.zeros(nb, dtype=np.float32) if tol is None else np.asarray(tol, dtype=np.float32)
    return Workload(name=name, nx=nx, ny=ny, nz=nz, h=float(h), freqs=tuple(freqs),
                    omega_idx=np.asarray(col_f, dtype=np.int32), m=m, sponge_width=int(L),
                    rec_ijk=rec, Q=Q, D=D, lam=float(lam), tol=tol, maxit=int(maxit),
                    seed=seed, src_ijk=src)


# ----------------------------------------------------------------------------- configs

def _config0(grid, nb, freqs, seed):
    """32^3, h=10, v=2000, 1 source at (16,16,4), f=5 Hz, sponge 8, 16 receivers at z=2,
    lambda=1, 50 iterations.  d = P u_true + 1% noise; P u_true comes from the stored
    fixture tests/golden/config0_Pu_true.txt (written by tests/golden/make_config0.py,
    which calls only oracle/)."""
    if grid is not None or nb is not None or freqs is not None:
        raise ValueError("config0 has a stored data fixture and cannot be resized")
    seed = 1001 if seed is None else seed
    rng = _rng(seed)
    nx = ny = nz = 32
    v = np.full((nz, ny, nx), 2000.0)
    xs = _lattice(nx, 4)
    rec = _grid_nodes(xs, xs, 2)
    pu = np.loadtxt(os.path.join(_GOLDEN, "config0_Pu_true.txt")).view(np.complex128).reshape(-1)
    assert pu.size == 16
    rms = math.sqrt(float((np.abs(pu) ** 2).mean()))
    D = (pu + 0.01 * rms * _cn(rng, 16)).reshape(16, 1).astype(np.complex64)
    return _finish("config0", (nx, ny, nz), 10.0, (5.0,), [0], v, 8, rec, [(16, 16, 4)], [1.0],
                   1.0, None, 50, seed, rng, D=D)


def config0_true_model():
    """v_true of configs[0]: v * (1 + 0.10 exp(-r^2 / 2 sigma^2)), sigma = 3 cells, centred."""
    x, y, z = _coords(32, 32, 32)
    r2 = (x - 15.5) ** 2 + (y - 15.5) ** 2 + (z - 15.5) ** 2
    v = 2000.0 * (1.0 + 0.10 * np.exp(-r2 / (2.0 * 9.0)))
    return (1.0 / (v * v)).reshape(-1)


def _config1(grid, nb, freqs, seed):
    """64^3, h=10, three flat layers 1500/2500/3500 + one +-15% anomaly (sigma 5), f=6 Hz,
    sponge 10, 16 sources at z=3 (4x4), 256 receivers at z=2 (16x16), lambda=10, K=100."""
    seed = 1002 if seed is None else seed
    rng = _rng(seed)
    nx, ny, nz = grid or (64, 64, 64)
    L = _scale_L(10, nx, 64)
    iz = np.arange(nz)
    vz = np.where(iz < round(nz * 21 / 64), 1500.0, np.where(iz < round(nz * 43 / 64), 2500.0, 3500.0))
    v = np.broadcast_to(vz[:, None, None], (nz, ny, nx)).copy()
    v = _add_anomalies(v, rng, 1, 0.15, 5.0 * nx / 64, L)
    f = (freqs or (6.0,))[0]
    sx, sy = _lattice(nx, 4), _lattice(ny, 4)
    src = _grid_nodes(sx, sy, 3)
    sel = _select(len(src), nb)
    src = src[sel]
    kx, ky = min(16, nx // 2), min(16, ny // 2)
    rec = _grid_nodes(_lattice(nx, kx), _lattice(ny, ky), 2)
    amps = [_ricker(f, 8.0)] * len(src)
    return _finish("config1", (nx, ny, nz), 10.0, (f,), [0] * len(src), v, L, rec, src, amps,
                   10.0, None, 100, seed, rng)


def _config2(grid, nb, freqs, seed):
    """128^3, h=12.5, v = 1500 + 3000 iz/(nz-1) + 5 anomalies +-20% (sigma 6), f in {4,6,8},
    64 sources (8x8, z=3), 1024 receivers (32x32, z=2), sponge 12, lambda=10, K=200.
    Column b = jf*64 + is."""
    seed = 1003 if seed is None else seed
    rng = _rng(seed)
    nx, ny, nz = grid or (128, 128, 128)
    L = _scale_L(12, nx, 128)
    vz = 1500.0 + 3000.0 * np.arange(nz) / (nz - 1)
    v = np.broadcast_to(vz[:, None, None], (nz, ny, nx)).copy()
    v = _add_anomalies(v, rng, 5, 0.20, 6.0 * nx / 128, L)
    freqs = tuple(freqs or (4.0, 6.0, 8.0))
    src1 = _grid_nodes(_lattice(nx, 8), _lattice(ny, 8), 3)
    src_all = np.concatenate([src1] * len(freqs))
    colf_all = np.repeat(np.arange(len(freqs)), len(src1))
    sel = _select(len(src_all), nb)
    src, col_f = src_all[sel], colf_all[sel]
    kx, ky = min(32, nx // 2), min(32, ny // 2)
    rec = _grid_nodes(_lattice(nx, kx), _lattice(ny, ky), 2)
    amps = [_ricker(freqs[j], 8.0) for j in col_f]
    return _finish("config2", (nx, ny, nz), 12.5, freqs, col_f, v, L, rec, src, amps,
                   10.0, None, 200, seed, rng)


def _config3(grid, nb, freqs, seed):
    """VSP: 200x200x160, h=10, six dipping layers 1800..4000 (dips 0-15 deg) + high-velocity
    lens, 48 surface sources on 4 rings x 12 azimuths around a vertical borehole at the
    grid centre, 120 borehole receivers iz=20..139, f=10 Hz, lambda=5, per-source
    tol in [1e-3, 1e-1] (log-uniform), maxit=300."""
    seed = 1004 if seed is None else seed
    rng = _rng(seed)
    nx, ny, nz = grid or (200, 200, 160)
    L = _scale_L(12, nx, 200)
    x, y, z = _coords(nx, ny, nz)
    cx, cy = nx // 2, ny // 2
    vl = np.linspace(1800.0, 4000.0, 6)
    layer = np.zeros((nz, ny, nx), dtype=np.int64)
    for k in range(1, 6):
        dip = math.radians(rng.uniform(0.0, 15.0))
        az = rng.uniform(0.0, 2.0 * math.pi)
        zk = nz * k / 6.0 + math.tan(dip) * ((x - cx) * math.cos(az) + (y - cy) * math.sin(az))
        layer += (z >= zk)
    v = vl[layer]
    ax, ay, azl = 30.0 * nx / 200, 30.0 * ny / 200, 8.0 * nz / 160
    lens = ((x - cx) / ax) ** 2 + ((y - cy) / ay) ** 2 + ((z - 0.55 * nz) / azl) ** 2 <= 1.0
    v = np.where(lens, 4500.0, v)
    f = (freqs or (10.0,))[0]
    src = []
    for ir, r in enumerate((20, 40, 60, 80)):
        rr = r * nx / 200.0
        for ia in range(12):
            a = math.radians(30.0 * ia + 15.0 * ir)
            src.append((int(round(cx + rr * math.cos(a))), int(round(cy + rr * math.sin(a))), 3))
    src = np.array(src)
    sel = _select(len(src), nb)
    src = src[sel]
    z0, z1 = int(round(nz * 20 / 160)), int(round(nz * 139 / 160))
    rec = np.stack([np.full(z1 - z0 + 1, cx), np.full(z1 - z0 + 1, cy), np.arange(z0, z1 + 1)], axis=1)
    tol = 10.0 ** (-3.0 + 2.0 * rng.uniform(size=48))
    tol = tol[sel]
    return _finish("config3", (nx, ny, nz), 10.0, (f,), [0] * len(src), v, L, rec, src,
                   [1.0] * len(src), 5.0, tol, 300, seed, rng)


def _config4(grid, nb, freqs, seed):
    """256^3, h=10, ten random layers (>= 8 cells thick, v ~ U[1500,4500]) + 8 anomalies
    +-15% (sigma 8), f=8 Hz, sponge 16, 32 sources (8x4, z=3), 4096 receivers (64x64, z=2),
    lambda=10, K=150."""
    seed = 1005 if seed is None else seed
    rng = _rng(seed)
    nx, ny, nz = grid or (256, 256, 256)
    L = _scale_L(16, nx, 256)
    tmin = max(1, round(8 * nz / 256))
    extra = rng.dirichlet(np.ones(10)) * (nz - 10 * tmin)
    edges = np.concatenate([[0.0], np.cumsum(tmin + extra)])
    vl = rng.uniform(1500.0, 4500.0, size=10)
    li = np.clip(np.searchsorted(edges, np.arange(nz) + 0.5) - 1, 0, 9)
    v = np.broadcast_to(vl[li][:, None, None], (nz, ny, nx)).copy()
    v = _add_anomalies(v, rng, 8, 0.15, 8.0 * nx / 256, L)
    f = (freqs or (8.0,))[0]
    src = _grid_nodes(_lattice(nx, 8), _lattice(ny, 4), 3)
    sel = _select(len(src), nb)
    src = src[sel]
    kx, ky = min(64, nx // 2), min(64, ny // 2)
    rec = _grid_nodes(_lattice(nx, kx), _lattice(ny, ky), 2)
    return _finish("config4", (nx, ny, nz), 10.0, (f,), [0] * len(src), v, L, rec, src,
                   [1.0] * len(src), 10.0, None, 150, seed, rng)


_MAKERS = {"config0": _config0, "config1": _config1, "config2": _config2,
           "config3": _config3, "config4": _config4}


def make(name: str, grid=None, nb=None, freqs=None, seed=None) -> Workload:
    """Build a workload.  grid=(nx,ny,nz) / nb / freqs shrink or reshape it for tests
    (geometry scales with the grid; columns are sub-sampled evenly)."""
    return _MAKERS[name](grid, nb, freqs, seed)
