"""ctypes front end of the complex128 CPU oracle (oracle/wri_oracle.c).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
imports nothing from the CUDA package and the CUDA package imports nothing
from here.

All arithmetic lives in wri_oracle.c (see its header for the PAPER.md passages
each function follows); this file only marshals numpy arrays and loops over
batch columns (columns are independent systems).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "wri_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile wri_oracle.c with gcc -O2 (no -ffast-math) into oracle/liboracle.so."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".%d.tmp" % os.getpid()
        subprocess.check_call(
            ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


class _RefOp(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
                ("h", C.c_double), ("omega", C.c_double),
                ("sponge_width", C.c_int32), ("gamma_max", C.c_double),
                ("power", C.c_int32), ("faces", C.c_uint32), ("periodic", C.c_int32),
                ("stencil", C.c_int32), ("round_c64", C.c_int32)]


class _RefState(C.Structure):
    _fields_ = [("u_top", C.c_void_p), ("u_bot", C.c_void_p), ("v", C.c_void_p),
                ("w", C.c_void_p), ("x", C.c_void_p),
                ("alpha", C.c_double), ("beta", C.c_double),
                ("rhobar", C.c_double), ("phibar", C.c_double),
                ("rho", C.c_double), ("c", C.c_double), ("s", C.c_double),
                ("theta", C.c_double), ("phi", C.c_double), ("arnorm", C.c_double),
                ("stop", C.c_int32)]


class _RefStateSF(C.Structure):
    _fields_ = [("u_top", C.c_void_p), ("u_bot", C.c_void_p), ("v", C.c_void_p),
                ("w", C.c_void_p), ("x", C.c_void_p),
                ("v_a", C.c_double * 2), ("w_a", C.c_double * 2), ("x_a", C.c_double * 2),
                ("alpha", C.c_double), ("beta", C.c_double),
                ("rhobar", C.c_double), ("phibar", C.c_double),
                ("rho", C.c_double), ("c", C.c_double), ("s", C.c_double),
                ("theta", C.c_double), ("phi", C.c_double), ("arnorm", C.c_double),
                ("stop", C.c_int32)]


_lib = None


def _L():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        P = C.c_void_p
        lib.ref_gamma.argtypes = [C.POINTER(_RefOp), P]
        lib.ref_apply_A.argtypes = [C.POINTER(_RefOp), P, P, P]
        lib.ref_apply_AH.argtypes = [C.POINTER(_RefOp), P, P, P]
        lib.ref_apply_M.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, P, P, P]
        lib.ref_apply_MH.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, P, P, P]
        lib.ref_lsqr_step.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P,
                                      C.POINTER(_RefState)]
        lib.ref_lsqr.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, P, P,
                                 C.c_double, C.c_int32, P, P, P, P, C.c_int32]
        lib.ref_lsqr.restype = C.c_int32
        I64 = C.c_int64
        lib.ref_apply_S.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, I64, P, P, P, P]
        lib.ref_apply_SH.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, I64, P, P, P, P]
        lib.ref_lsqr_sf_step.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, I64,
                                         C.POINTER(_RefStateSF)]
        lib.ref_lsqr_sf.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, I64, P, P,
                                    C.c_double, C.c_double, C.c_int32, P, P, P, P]
        lib.ref_lsqr_sf.restype = C.c_int32
        lib.ref_objective_gradient.argtypes = [C.POINTER(_RefOp), P, C.c_double, C.c_int32, P, I64,
                                               P, P, P, P, P, P, P]
        for f in (lib.ref_gamma, lib.ref_apply_A, lib.ref_apply_AH, lib.ref_apply_M,
                  lib.ref_apply_MH, lib.ref_lsqr_step, lib.ref_apply_S, lib.ref_apply_SH,
                  lib.ref_lsqr_sf_step, lib.ref_objective_gradient):
            f.restype = None
        _lib = lib
    return _lib


@dataclass
class Operator:
    """Grid, frequency and sponge of one column's Helmholtz operator."""
    nx: int
    ny: int
    nz: int
    h: float
    omega: float
    sponge_width: int = 0
    gamma_max: float = 1.0
    power: int = 2
    faces: int = 0x3F
    periodic: bool = False   # test-only boundary rule for the plane-wave pin
    stencil: int = 0         # 0: 7-point star, 1: 27-point box (reading C-23)
    round_c64: bool = False  # test-only: LSQR vectors stored in complex64 (attainable-floor emulation)

    @property
    def ng(self) -> int:
        return self.nx * self.ny * self.nz

    def _c(self) -> _RefOp:
        return _RefOp(self.nx, self.ny, self.nz, float(self.h), float(self.omega),
                      int(self.sponge_width), float(self.gamma_max), int(self.power),
                      int(self.faces), int(bool(self.periodic)), int(self.stencil),
                      int(bool(self.round_c64)))


def _f64(a, n):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1))
    assert a.size == n, (a.size, n)
    return a


def _c128(a, n):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.complex128).reshape(-1))
    assert a.size == n, (a.size, n)
    return a


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def rec_cells(nx: int, ny: int, nz: int, rec_ijk) -> np.ndarray:
    """(ix,iy,iz) receiver nodes -> cell indices c = (iz*ny+iy)*nx+ix (int64)."""
    r = np.asarray(rec_ijk, dtype=np.int64).reshape(-1, 3)
    return np.ascontiguousarray((r[:, 2] * ny + r[:, 1]) * nx + r[:, 0])


def gamma(op: Operator) -> np.ndarray:
    g = np.empty(op.ng, dtype=np.float64)
    _L().ref_gamma(C.byref(op._c()), _ptr(g))
    return g.reshape(op.nz, op.ny, op.nx)


def apply_A(op: Operator, m, v, adjoint: bool = False) -> np.ndarray:
    m = _f64(m, op.ng)
    v = _c128(v, op.ng)
    y = np.empty(op.ng, dtype=np.complex128)
    (_L().ref_apply_AH if adjoint else _L().ref_apply_A)(C.byref(op._c()), _ptr(m), _ptr(v), _ptr(y))
    return y


def apply_M(op: Operator, m, lam: float, rec: np.ndarray, v):
    m = _f64(m, op.ng)
    v = _c128(v, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    ytop = np.empty(op.ng, dtype=np.complex128)
    ybot = np.empty(max(rec.size, 1), dtype=np.complex128)
    _L().ref_apply_M(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), _ptr(v),
                     _ptr(ytop), _ptr(ybot))
    return ytop, ybot[:rec.size]


def apply_MH(op: Operator, m, lam: float, rec: np.ndarray, ytop, ybot) -> np.ndarray:
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    ytop = _c128(ytop, op.ng)
    ybot = _c128(ybot, rec.size) if rec.size else np.zeros(1, dtype=np.complex128)
    x = np.empty(op.ng, dtype=np.complex128)
    _L().ref_apply_MH(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), _ptr(ytop),
                      _ptr(ybot), _ptr(x))
    return x


def lsqr(op: Operator, m, lam: float, rec: np.ndarray, q, d, tol: float = 0.0,
         maxit: int = 50, snap_stride: int = 0) -> dict:
    """One column of LSQR on min ||M x - [lam q; d]||, x0 = 0."""
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    q = _c128(q, op.ng)
    d = _c128(d, rec.size) if rec.size else np.zeros(1, dtype=np.complex128)
    x = np.empty(op.ng, dtype=np.complex128)
    res = np.empty(maxit + 1, dtype=np.float64)
    ar = np.empty(maxit + 1, dtype=np.float64)
    nsnap = maxit // snap_stride if snap_stride > 0 else 0
    snap = np.zeros((max(nsnap, 1), op.ng), dtype=np.complex128)
    it = _L().ref_lsqr(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), _ptr(q), _ptr(d),
                       float(tol), int(maxit), _ptr(x), _ptr(res), _ptr(ar),
                       _ptr(snap) if nsnap else None, int(snap_stride))
    return {"x": x, "resnorms": res, "arnorms": ar, "iters": int(it),
            "x_snap": snap[:nsnap] if nsnap else None}


def lsqr_step(op: Operator, m, lam: float, rec: np.ndarray, state: dict) -> dict:
    """One LSQR iteration on a normalised state
    {u_top,u_bot,v,w,x (complex128), alpha,beta,rhobar,phibar}; returns the new state
    plus rho,c,s,theta,phi,arnorm,stop."""
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    arrs = {k: _c128(state[k], op.ng).copy() for k in ("u_top", "v", "w", "x")}
    arrs["u_bot"] = (_c128(state["u_bot"], rec.size).copy() if rec.size
                     else np.zeros(1, dtype=np.complex128))
    st = _RefState()
    for k, a in arrs.items():
        setattr(st, k, a.ctypes.data)
    for k in ("alpha", "beta", "rhobar", "phibar"):
        setattr(st, k, float(state[k]))
    _L().ref_lsqr_step(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), C.byref(st))
    out = dict(arrs)
    out["u_bot"] = arrs["u_bot"][:rec.size]
    for k in ("alpha", "beta", "rhobar", "phibar", "rho", "c", "s", "theta", "phi", "arnorm"):
        out[k] = getattr(st, k)
    out["stop"] = int(st.stop)
    return out


def lsqr_batch(ops, m, lam: float, rec: np.ndarray, Q, D, tols=None, maxit: int = 50,
               threads: int = 1, columns=None) -> dict:
    """Column loop over source-interleaved inputs Q[n_g, nb], D[n_r, nb].

    ops: one Operator per column (frequencies may differ, reading C-10).
    Returns X[n_g, ncols], resnorms[maxit+1, ncols], arnorms, iters[ncols] for the
    requested columns (default: all).  threads > 1 runs independent columns on a
    thread pool (ctypes releases the GIL); each column's arithmetic is unchanged.
    """
    Q = np.asarray(Q)
    D = np.asarray(D)
    nb = Q.shape[1]
    cols = list(range(nb)) if columns is None else list(columns)
    tols = np.zeros(nb) if tols is None else np.asarray(tols, dtype=np.float64)

    def one(s):
        return lsqr(ops[s], m, lam, rec, Q[:, s], D[:, s] if D.size else D.reshape(0),
                    tol=float(tols[s]), maxit=maxit)

    if threads > 1 and len(cols) > 1:
        _L()
        with ThreadPoolExecutor(max_workers=threads) as ex:
            outs = list(ex.map(one, cols))
    else:
        outs = [one(s) for s in cols]
    return {"x": np.stack([o["x"] for o in outs], axis=1),
            "resnorms": np.stack([o["resnorms"] for o in outs], axis=1),
            "arnorms": np.stack([o["arnorms"] for o in outs], axis=1),
            "iters": np.array([o["iters"] for o in outs], dtype=np.int32)}


# ---------------------------------------------------------------------------------------------
# Source-free system S = [lam A, -lam e; P, 0], x = [u; alpha], b = [0; d]

def _drec(d, rec):
    return _c128(d, rec.size) if rec.size else np.zeros(1, dtype=np.complex128)


def apply_S(op: Operator, m, lam: float, rec: np.ndarray, src: int, u, a):
    m = _f64(m, op.ng)
    u = _c128(u, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    a = np.array([a], dtype=np.complex128)
    ytop = np.empty(op.ng, dtype=np.complex128)
    ybot = np.empty(max(rec.size, 1), dtype=np.complex128)
    _L().ref_apply_S(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), int(src), _ptr(u),
                     _ptr(a), _ptr(ytop), _ptr(ybot))
    return ytop, ybot[:rec.size]


def apply_SH(op: Operator, m, lam: float, rec: np.ndarray, src: int, ytop, ybot):
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    ytop = _c128(ytop, op.ng)
    ybot = _drec(ybot, rec)
    xu = np.empty(op.ng, dtype=np.complex128)
    xa = np.empty(1, dtype=np.complex128)
    _L().ref_apply_SH(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), int(src),
                      _ptr(ytop), _ptr(ybot), _ptr(xu), _ptr(xa))
    return xu, complex(xa[0])


def lsqr_sf(op: Operator, m, lam: float, rec: np.ndarray, src: int, d, tol: float = 0.0,
            maxit: int = 50, q=None, ar_ref: float = 0.0) -> dict:
    """One column of LSQR on min ||S [u; alpha] - [lam q; d]||, x0 = 0 (q = None: the paper's
    b = [0; d]).  ar_ref > 0 replaces alpha1*beta1 as the reference of the stop rule."""
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    d = _drec(d, rec)
    qq = _c128(q, op.ng) if q is not None else None
    x = np.empty(op.ng, dtype=np.complex128)
    xa = np.zeros(1, dtype=np.complex128)
    res = np.empty(maxit + 1, dtype=np.float64)
    ar = np.empty(maxit + 1, dtype=np.float64)
    it = _L().ref_lsqr_sf(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), int(src),
                          _ptr(qq) if qq is not None else None, _ptr(d), float(tol), float(ar_ref),
                          int(maxit), _ptr(x), _ptr(xa), _ptr(res), _ptr(ar))
    return {"x": x, "alpha_src": complex(xa[0]), "resnorms": res, "arnorms": ar, "iters": int(it)}


def lsqr_sf_warm(op: Operator, m, lam: float, rec: np.ndarray, src: int, d, x0, a0, tol: float = 0.0,
                 maxit: int = 50, q=None, ar_ref: float = 0.0) -> dict:
    """Warm start (Algorithm 1 leaves x0 free), written out as its definition:
    r0 = b - S [x0; a0];  [dx; da] = LSQR on S with right-hand side r0 from zero;  x = x0 + dx.
    resnorms[k] is then ||b - S x_k|| of the ORIGINAL system."""
    x0 = _c128(x0, op.ng)
    t, bb = apply_S(op, m, lam, rec, src, x0, a0)
    b_top = (lam * _c128(q, op.ng) if q is not None else np.zeros(op.ng, dtype=np.complex128))
    r_top = b_top - t
    r_bot = _drec(d, np.ascontiguousarray(rec, dtype=np.int64))[:np.size(rec)] - bb
    out = lsqr_sf(op, m, lam, rec, src, r_bot, tol=tol, maxit=maxit, q=r_top / lam, ar_ref=ar_ref)
    out["x"] = x0 + out["x"]
    out["alpha_src"] = complex(a0) + out["alpha_src"]
    return out


def lsqr_sf_step(op: Operator, m, lam: float, rec: np.ndarray, src: int, state: dict) -> dict:
    """One LSQR iteration on a normalised source-free state: the keys of lsqr_step plus the
    alpha entries v_a, w_a, x_a of v, w, x."""
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    arrs = {k: _c128(state[k], op.ng).copy() for k in ("u_top", "v", "w", "x")}
    arrs["u_bot"] = _drec(state["u_bot"], rec).copy()
    st = _RefStateSF()
    for k, a in arrs.items():
        setattr(st, k, a.ctypes.data)
    for k in ("v_a", "w_a", "x_a"):
        z = complex(state[k])
        getattr(st, k)[0] = z.real
        getattr(st, k)[1] = z.imag
    for k in ("alpha", "beta", "rhobar", "phibar"):
        setattr(st, k, float(state[k]))
    _L().ref_lsqr_sf_step(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), int(src),
                          C.byref(st))
    out = dict(arrs)
    out["u_bot"] = arrs["u_bot"][:rec.size]
    for k in ("v_a", "w_a", "x_a"):
        out[k] = complex(getattr(st, k)[0], getattr(st, k)[1])
    for k in ("alpha", "beta", "rhobar", "phibar", "rho", "c", "s", "theta", "phi", "arnorm"):
        out[k] = getattr(st, k)
    out["stop"] = int(st.stop)
    return out


def lsqr_sf_batch(ops, m, lam: float, rec: np.ndarray, src_cells, D, tols=None, maxit: int = 50,
                  threads: int = 1, columns=None) -> dict:
    """Column loop of lsqr_sf over D[n_r, nb]; src_cells[nb] = source node of each column."""
    D = np.asarray(D)
    nb = len(src_cells)
    cols = list(range(nb)) if columns is None else list(columns)
    tols = np.zeros(nb) if tols is None else np.asarray(tols, dtype=np.float64)

    def one(s):
        return lsqr_sf(ops[s], m, lam, rec, int(src_cells[s]), D[:, s] if D.size else D.reshape(0),
                       tol=float(tols[s]), maxit=maxit)

    if threads > 1 and len(cols) > 1:
        _L()
        with ThreadPoolExecutor(max_workers=threads) as ex:
            outs = list(ex.map(one, cols))
    else:
        outs = [one(s) for s in cols]
    return {"x": np.stack([o["x"] for o in outs], axis=1),
            "alpha_src": np.array([o["alpha_src"] for o in outs], dtype=np.complex128),
            "resnorms": np.stack([o["resnorms"] for o in outs], axis=1),
            "arnorms": np.stack([o["arnorms"] for o in outs], axis=1),
            "iters": np.array([o["iters"] for o in outs], dtype=np.int32)}


def objective_gradient(op: Operator, m, lam: float, rec: np.ndarray, u, d, q=None, src: int = -1,
                       alpha_src: complex = 0.0, g=None):
    """f_pde = lam^2/2 ||A u - q - alpha e||^2, f_data = 1/2 ||P u - d||^2 and, when g (float64
    [n_g]) is given, g += lam^2 omega^2 Re[conj((1+i gamma) u) r]  (eq. 4, 9)."""
    m = _f64(m, op.ng)
    rec = np.ascontiguousarray(rec, dtype=np.int64)
    u = _c128(u, op.ng)
    d = _drec(d, rec)
    qq = _c128(q, op.ng) if q is not None else None
    a = np.array([alpha_src], dtype=np.complex128)
    fp = C.c_double(0.0)
    fd = C.c_double(0.0)
    if g is not None:
        assert g.dtype == np.float64 and g.flags.c_contiguous and g.size == op.ng
    _L().ref_objective_gradient(C.byref(op._c()), _ptr(m), float(lam), rec.size, _ptr(rec), int(src),
                                _ptr(a), _ptr(qq) if qq is not None else None, _ptr(u), _ptr(d),
                                C.byref(fp), C.byref(fd), _ptr(g) if g is not None else None)
    return fp.value, fd.value
