"""ctypes binding of libwri.so — same names as include/wri.h, marshalling only."""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


class WriError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libwri error %d: %s" % (code, msg))
        self.code = code


class wri_grid(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32)]


class wri_sponge(C.Structure):
    _fields_ = [("width", C.c_int32), ("gamma_max", C.c_float), ("power", C.c_int32),
                ("faces", C.c_uint32)]


class wri_lsqr_opts(C.Structure):
    _fields_ = [("warm_start", C.c_int32), ("ar_ref_dev", C.c_void_p), ("ar0_out_dev", C.c_void_p)]


class wri_lsqr_view(C.Structure):
    _fields_ = [("nb", C.c_int32), ("k", C.c_int32),
                ("U_top", C.c_void_p), ("U_bot", C.c_void_p), ("V", C.c_void_p),
                ("W", C.c_void_p), ("X", C.c_void_p),
                ("alpha", C.c_void_p), ("beta", C.c_void_p), ("rhobar", C.c_void_p),
                ("phibar", C.c_void_p), ("ar0", C.c_void_p), ("cx", C.c_void_p), ("cw", C.c_void_p),
                ("active", C.c_void_p), ("iters", C.c_void_p),
                ("nb_max", C.c_int32), ("sf_state", C.c_void_p)]


WRI_AWRI_MAX_TRACE = 16
wri_update_fn = C.CFUNCTYPE(C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p)
wri_reduce_fn = C.CFUNCTYPE(C.c_int, C.c_void_p, C.POINTER(C.c_double), C.c_void_p, C.c_int64, C.c_void_p)


class wri_awri_opts(C.Structure):
    _fields_ = [("max_halvings", C.c_int32), ("warm_restart", C.c_int32), ("update", wri_update_fn),
                ("user", C.c_void_p), ("step", C.c_float), ("m_min", C.c_float), ("m_max", C.c_float),
                ("reduce", wri_reduce_fn)]


class wri_debug_opts(C.Structure):
    _fields_ = [(n, C.c_int32) for n in ("nstage_f", "nstage_a", "zc_f", "zc_a", "txc", "tyc",
                                         "no_compact", "no_groups", "generic", "m_ldg_f")]


class wri_awri_report(C.Structure):
    _fields_ = [("accepted", C.c_int32), ("n_halvings", C.c_int32), ("n_trace", C.c_int32),
                ("eps", C.c_float), ("f", C.c_double), ("f_trial", C.c_double), ("lsqr_iters", C.c_int64),
                ("trace_eps", C.c_float * WRI_AWRI_MAX_TRACE), ("trace_f", C.c_double * WRI_AWRI_MAX_TRACE),
                ("trace_f_trial", C.c_double * WRI_AWRI_MAX_TRACE)]


WRI_OK = 0
WRI_ERR_ARG = -1
WRI_ERR_RECEIVER_RANGE = -2
WRI_ERR_RECEIVER_DUP = -3
WRI_ERR_WORKSPACE = -4
WRI_ERR_CUDA = -5
WRI_ERR_STATE = -6
WRI_ERR_NUMERIC = -7
WRI_ERR_SCRATCH_LIMIT = -8
WRI_STATIC_SCRATCH_BYTES = 4 << 20
WRI_STENCIL_7 = 0
WRI_STENCIL_27 = 1
WRI_WS_HOST_STAGING = 1
WRI_WS_COMPACTION = 2

_lib = None


def lib_path() -> str:
    return os.path.join(_HERE, "libwri.so")


def load_library():
    """Load libwri.so (must have been built: python -m paper_2410_18429_b200.build)."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        # the in-tree library is missing (fresh checkout): build it with nvcc, loudly; never a CPU fallback
        import sys
        sys.stderr.write("paper_2410_18429_b200: libwri.so missing, building it with nvcc for sm_100a ...\n")
        try:
            from . import build as _build
            _build.build()
        except Exception as e:
            raise WriError(WRI_ERR_CUDA, "libwri.so is not built and building it failed (%s); run python -m "
                                         "paper_2410_18429_b200.build; there is no CPU fallback" % (e,))
    if not os.path.exists(path):
        raise WriError(WRI_ERR_CUDA, "libwri.so is not built (run python -m paper_2410_18429_b200.build); "
                                     "there is no CPU fallback")
    lib = C.CDLL(path)
    P, I32, F32, F64 = C.c_void_p, C.c_int32, C.c_float, C.c_double
    lib.wri_create.argtypes = [C.POINTER(P), wri_grid, F64, I32, P, P, wri_sponge, I32, P, I32, P]
    lib.wri_set_model.argtypes = [P, P]
    lib.wri_set_stencil.argtypes = [P, I32]
    lib.wri_set_debug_opts.argtypes = [P, C.POINTER(wri_debug_opts)]
    lib.wri_plan_info.argtypes = [P, I32, P]
    lib.wri_workspace_bytes.argtypes = [P, I32, I32]
    lib.wri_workspace_bytes.restype = C.c_size_t
    lib.wri_set_workspace.argtypes = [P, P, C.c_size_t]
    lib.wri_apply_M.argtypes = [P, I32, P, F32, P, P, P]
    lib.wri_apply_MH.argtypes = [P, I32, P, F32, P, P, P]
    solve = [P, I32, P, P, P, F32, P, I32, P, P, P]
    lib.wri_lsqr_batch.argtypes = solve
    lib.wri_lsqr_batch_host.argtypes = solve
    lib.wri_lsqr_batch_host_async.argtypes = solve
    lib.wri_host_pipeline_bytes.argtypes = [P, I32]
    lib.wri_host_pipeline_bytes.restype = C.c_size_t
    lib.wri_set_host_pipeline.argtypes = [P, I32, P, C.c_size_t]
    lib.wri_host_wait.argtypes = [P]
    lib.wri_lsqr_begin.argtypes = solve
    lib.wri_apply_S.argtypes = [P, I32, P, P, F32, P, P, P, P]
    lib.wri_apply_SH.argtypes = [P, I32, P, P, F32, P, P, P, P]
    solve_sf = [P, I32, P, P, P, P, F32, P, I32, P, P, P, P]
    lib.wri_lsqr_sf_batch.argtypes = solve_sf
    lib.wri_lsqr_sf_begin.argtypes = solve_sf
    lib.wri_lsqr_sf_batch_host.argtypes = solve_sf
    lib.wri_lsqr_sf_batch_host_async.argtypes = solve_sf
    lib.wri_objective_gradient.argtypes = [P, I32, P, P, P, P, P, P, F32, P, P, P]
    lib.wri_objective_gradient_static.argtypes = [P, I32, P, P, P, P, P, P, F32, P, P, P]
    lib.wri_lsqr_set_opts.argtypes = [P, C.POINTER(wri_lsqr_opts)]
    lib.wri_set_receiver_mask.argtypes = [P, I32, P]
    lib.wri_misfit_sf.argtypes = [P, I32, P, P, P, F32, F32, I32, I32, P, P, P, P, P, P, P, P]
    lib.wri_awri_step.argtypes = [P, I32, P, P, P, F32, F32, I32, C.POINTER(wri_awri_opts), P, P, P, P, P, P, P,
                                  P, C.POINTER(wri_awri_report)]
    lib.wri_lsqr_iterate.argtypes = [P, I32]
    lib.wri_lsqr_end.argtypes = [P]
    lib.wri_lsqr_peek.argtypes = [P, C.POINTER(wri_lsqr_view)]
    lib.wri_launch_count.argtypes = [P]
    lib.wri_launch_count.restype = C.c_int64
    lib.wri_profile_enable.argtypes = [P, I32]
    lib.wri_profile_read.argtypes = [P, P, P, P, P, P, P]
    lib.wri_destroy.argtypes = [P]
    lib.wri_strerror.argtypes = [C.c_int]
    lib.wri_strerror.restype = C.c_char_p
    _lib = lib
    return lib


def _ck(code):
    if code != WRI_OK:
        raise WriError(code, load_library().wri_strerror(code).decode())


def _dptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _i32(a):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a, a.ctypes.data_as(C.c_void_p)


class Wri:
    """One wri_ctx: grid + model + receivers on the current CUDA device and stream.

    Tensors are torch CUDA tensors: m float32 [n_g]; batched vectors complex64 [n_g, nb]
    (source-interleaved), receiver rows complex64 [n_rec, nb].
    """

    def __init__(self, grid, h, omegas, m, sponge_width, rec_ijk, nb_max, gamma_max=1.0, power=2,
                 faces=0x3F, stream=None):
        import torch
        lib = load_library()
        self._torch = torch
        self.nx, self.ny, self.nz = (int(g) for g in grid)
        self.ng = self.nx * self.ny * self.nz
        self.nb_max = int(nb_max)
        om = np.ascontiguousarray(omegas, dtype=np.float64)
        rec = np.ascontiguousarray(rec_ijk, dtype=np.int32).reshape(-1, 3)
        self.n_rec = rec.shape[0]
        self.m = m
        self._ws = None
        self._keep = []
        if stream is None and torch.cuda.is_available():
            stream = torch.cuda.current_stream().cuda_stream
        h_ctx = C.c_void_p()
        _ck(lib.wri_create(C.byref(h_ctx), wri_grid(self.nx, self.ny, self.nz), float(h), om.size,
                           om.ctypes.data_as(C.c_void_p), _dptr(m),
                           wri_sponge(int(sponge_width), float(gamma_max), int(power), int(faces)),
                           self.n_rec, rec.ctypes.data_as(C.c_void_p) if self.n_rec else None,
                           self.nb_max, C.c_void_p(stream or 0)))
        self._h = h_ctx
        self._lib = lib

    @classmethod
    def from_workload(cls, w, device="cuda", nb_max=None):
        import torch
        m = torch.from_numpy(w.m).to(device)
        return cls((w.nx, w.ny, w.nz), w.h, w.omegas, m, w.sponge_width, w.rec_ijk,
                   nb_max or w.nb, gamma_max=w.gamma_max, power=w.power, faces=w.faces)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.wri_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- workspace
    def workspace_bytes(self, nb, host_staging=False, compaction=False):
        flags = (WRI_WS_HOST_STAGING if host_staging else 0) | (WRI_WS_COMPACTION if compaction else 0)
        return int(self._lib.wri_workspace_bytes(self._h, int(nb), flags))

    def ensure_workspace(self, nb, host_staging=False, compaction=False):
        # sticky: a workspace once sized for host staging / compaction keeps that room
        self._ws_hs = getattr(self, "_ws_hs", False) or bool(host_staging)
        self._ws_cp = getattr(self, "_ws_cp", False) or bool(compaction)
        need = self.workspace_bytes(nb, self._ws_hs, self._ws_cp)
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = self._torch.empty(need, dtype=self._torch.uint8, device=self.m.device)
            _ck(self._lib.wri_set_workspace(self._h, _dptr(self._ws), self._ws.numel()))
        return self._ws

    def set_model(self, m):
        self.m = m
        _ck(self._lib.wri_set_model(self._h, _dptr(m)))

    def set_stencil(self, stencil):
        """WRI_STENCIL_7 (default) or WRI_STENCIL_27; sticky."""
        _ck(self._lib.wri_set_stencil(self._h, int(stencil)))

    def plan_info(self, nb):
        """Tile plan of the pass kernel for batch width nb (wri_plan_info), or None (generic kernels)."""
        out = (C.c_int32 * 16)()
        if self._lib.wri_plan_info(self._h, int(nb), out) != WRI_OK:
            return None
        keys = ("cb", "nchunk", "txc", "tyc", "items", "merged", "m_tma", "zc_f", "nstage_f", "tiles_f",
                "zc_a", "nstage_a", "tiles_a", "stage_bytes_f", "stage_bytes_a", "grid")
        return dict(zip(keys, (int(v) for v in out)))

    def set_debug_opts(self, **kw):
        """Tuning / test switches (wri_debug_opts); no arguments restores the defaults."""
        o = wri_debug_opts()
        for k, v in kw.items():
            if not hasattr(o, k):
                raise TypeError("unknown debug option %r" % (k,))
            setattr(o, k, int(v))
        _ck(self._lib.wri_set_debug_opts(self._h, C.byref(o)))

    # ---- operator
    def apply_M(self, x, lam, omega_idx=None, out=None):
        """out = (ytop, ybot) to reuse buffers."""
        t = self._torch
        nb = x.shape[1]
        if out is not None:
            ytop, ybot = out
        else:
            ytop = t.empty_like(x)
            ybot = t.empty((self.n_rec, nb), dtype=t.complex64, device=x.device)
        keep, oi = _i32(omega_idx)
        _ck(self._lib.wri_apply_M(self._h, nb, oi, float(lam), _dptr(x), _dptr(ytop), _dptr(ybot)))
        return ytop, ybot

    def apply_MH(self, ytop, ybot, lam, omega_idx=None, out=None):
        t = self._torch
        nb = ytop.shape[1]
        x = out if out is not None else t.empty_like(ytop)
        keep, oi = _i32(omega_idx)
        _ck(self._lib.wri_apply_MH(self._h, nb, oi, float(lam), _dptr(ytop), _dptr(ybot), _dptr(x)))
        return x

    def apply_S(self, x, xalpha, lam, src_ijk, omega_idx=None):
        """S [x; xalpha] of the source-free system: (ytop, ybot)."""
        t = self._torch
        nb = x.shape[1]
        ytop = t.empty_like(x)
        ybot = t.empty((self.n_rec, nb), dtype=t.complex64, device=x.device)
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_apply_S(self._h, nb, oi, si, float(lam), _dptr(x), _dptr(xalpha), _dptr(ytop),
                                  _dptr(ybot)))
        return ytop, ybot

    def apply_SH(self, ytop, ybot, lam, src_ijk, omega_idx=None):
        """S^H [ytop; ybot]: (x, xalpha)."""
        t = self._torch
        nb = ytop.shape[1]
        x = t.empty_like(ytop)
        xa = t.empty(nb, dtype=t.complex64, device=ytop.device)
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_apply_SH(self._h, nb, oi, si, float(lam), _dptr(ytop), _dptr(ybot), _dptr(x),
                                   _dptr(xa)))
        return x, xa

    # ---- solver
    def _outputs(self, nb, maxit, device):
        t = self._torch
        u = t.empty((self.ng, nb), dtype=t.complex64, device=device)
        res = t.empty((maxit + 1, nb), dtype=t.float32, device=device)
        it = t.empty(nb, dtype=t.int32, device=device)
        return u, res, it

    def lsqr_batch(self, q, d, lam, tol=None, maxit=50, omega_idx=None, out=None):
        nb = q.shape[1]
        self.ensure_workspace(nb, compaction=tol is not None)
        u, res, it = out if out is not None else self._outputs(nb, maxit, q.device)
        keep, oi = _i32(omega_idx)
        _ck(self._lib.wri_lsqr_batch(self._h, nb, oi, _dptr(q), _dptr(d), float(lam), _dptr(tol),
                                     int(maxit), _dptr(u), _dptr(res), _dptr(it)))
        return u, res, it

    def lsqr_batch_host(self, q, d, lam, tol=None, maxit=50, omega_idx=None, out=None):
        """Host-buffer entry: q, d, tol and the outputs are CPU tensors (pinned for speed)."""
        t = self._torch
        nb = q.shape[1]
        self.ensure_workspace(nb, host_staging=True, compaction=tol is not None)
        if out is None:
            out = (t.empty((self.ng, nb), dtype=t.complex64).pin_memory(),
                   t.empty((maxit + 1, nb), dtype=t.float32).pin_memory(),
                   t.empty(nb, dtype=t.int32).pin_memory())
        u, res, it = out
        keep, oi = _i32(omega_idx)
        _ck(self._lib.wri_lsqr_batch_host(self._h, nb, oi, _dptr(q), _dptr(d), float(lam), _dptr(tol),
                                          int(maxit), _dptr(u), _dptr(res), _dptr(it)))
        return u, res, it

    def ensure_host_pipeline(self, nb):
        """Device staging for the pipelined host-buffer entries (two slots)."""
        need = int(self._lib.wri_host_pipeline_bytes(self._h, int(nb)))
        buf = getattr(self, "_pipe", None)
        if buf is None or buf.numel() < need or getattr(self, "_pipe_nb", 0) < nb:
            self._pipe = self._torch.empty(need, dtype=self._torch.uint8, device=self.m.device)
            self._pipe_nb = int(nb)
            _ck(self._lib.wri_set_host_pipeline(self._h, int(nb), _dptr(self._pipe), self._pipe.numel()))

    def lsqr_batch_host_async(self, q, d, lam, tol=None, maxit=50, omega_idx=None, out=None):
        """Pipelined host-buffer solve: returns after enqueue; q, d, tol and out = (u, resnorms,
        iters) are PINNED CPU tensors that must stay alive, and out unread, until host_wait()."""
        t = self._torch
        nb = q.shape[1]
        self.ensure_workspace(nb, compaction=tol is not None)
        self.ensure_host_pipeline(nb)
        if out is None:
            out = (t.empty((self.ng, nb), dtype=t.complex64).pin_memory(),
                   t.empty((maxit + 1, nb), dtype=t.float32).pin_memory(),
                   t.empty(nb, dtype=t.int32).pin_memory())
        u, res, it = out
        keep, oi = _i32(omega_idx)
        self._async_keep = getattr(self, "_async_keep", []) + [(q, d, tol, u, res, it)]
        _ck(self._lib.wri_lsqr_batch_host_async(self._h, nb, oi, _dptr(q), _dptr(d), float(lam), _dptr(tol),
                                                int(maxit), _dptr(u), _dptr(res), _dptr(it)))
        return u, res, it

    def lsqr_sf_batch_host_async(self, d, lam, src_ijk, tol=None, maxit=50, omega_idx=None, q=None, out=None):
        """Pipelined host-buffer solve of the source-free system; out = (u, alpha, resnorms, iters),
        pinned CPU tensors; see lsqr_batch_host_async."""
        t = self._torch
        nb = d.shape[1]
        self.ensure_workspace(nb, compaction=tol is not None)
        self.ensure_host_pipeline(nb)
        if out is None:
            out = (t.empty((self.ng, nb), dtype=t.complex64).pin_memory(),
                   t.empty(nb, dtype=t.complex64).pin_memory(),
                   t.empty((maxit + 1, nb), dtype=t.float32).pin_memory(),
                   t.empty(nb, dtype=t.int32).pin_memory())
        u, a, res, it = out
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        self._async_keep = getattr(self, "_async_keep", []) + [(q, d, tol, u, a, res, it)]
        _ck(self._lib.wri_lsqr_sf_batch_host_async(self._h, nb, oi, si, _dptr(q), _dptr(d), float(lam),
                                                   _dptr(tol), int(maxit), _dptr(u), _dptr(a), _dptr(res),
                                                   _dptr(it)))
        return u, a, res, it

    def host_wait(self):
        _ck(self._lib.wri_host_wait(self._h))
        self._async_keep = []

    def lsqr_begin(self, q, d, lam, tol=None, maxit=50, omega_idx=None):
        nb = q.shape[1]
        self.ensure_workspace(nb, compaction=tol is not None)
        u, res, it = self._outputs(nb, maxit, q.device)
        keep, oi = _i32(omega_idx)
        self._keep = [q, d, tol, u, res, it]
        _ck(self._lib.wri_lsqr_begin(self._h, nb, oi, _dptr(q), _dptr(d), float(lam), _dptr(tol),
                                     int(maxit), _dptr(u), _dptr(res), _dptr(it)))
        return u, res, it

    def set_opts(self, warm_start=False, ar_ref=None, ar0_out=None):
        """Options of the solves that follow: warm start from the contents of the output buffers,
        reference of the stop rule (float64 [nb] CUDA tensor), receiver of alpha1*beta1."""
        self._opt_keep = (ar_ref, ar0_out)
        o = wri_lsqr_opts(int(bool(warm_start)), _dptr(ar_ref), _dptr(ar0_out))
        _ck(self._lib.wri_lsqr_set_opts(self._h, C.byref(o)))

    def set_receiver_mask(self, mask):
        """Per-source receiver sets: mask uint8 [n_rec, nb] CUDA tensor (1 = recorded), None = all."""
        self._rmask_keep = mask
        _ck(self._lib.wri_set_receiver_mask(self._h, 0 if mask is None else int(mask.shape[1]), _dptr(mask)))

    # ---- source-free system (unknown source weight per column)
    def lsqr_sf_batch(self, d, lam, src_ijk, tol=None, maxit=50, omega_idx=None, q=None, out=None):
        """out = (u, alpha, resnorms, iters) to reuse buffers; with set_opts(warm_start=True) u and
        alpha hold the start point on entry."""
        t = self._torch
        nb = d.shape[1]
        self.ensure_workspace(nb, compaction=tol is not None)
        if out is not None:
            u, a, res, it = out
        else:
            u, res, it = self._outputs(nb, maxit, d.device)
            a = t.empty(nb, dtype=t.complex64, device=d.device)
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_lsqr_sf_batch(self._h, nb, oi, si, _dptr(q), _dptr(d), float(lam), _dptr(tol),
                                        int(maxit), _dptr(u), _dptr(a), _dptr(res), _dptr(it)))
        return u, a, res, it

    def lsqr_sf_batch_host(self, d, lam, src_ijk, tol=None, maxit=50, omega_idx=None, q=None, out=None):
        t = self._torch
        nb = d.shape[1]
        self.ensure_workspace(nb, host_staging=True, compaction=tol is not None)
        if out is None:
            out = (t.empty((self.ng, nb), dtype=t.complex64).pin_memory(),
                   t.empty(nb, dtype=t.complex64).pin_memory(),
                   t.empty((maxit + 1, nb), dtype=t.float32).pin_memory(),
                   t.empty(nb, dtype=t.int32).pin_memory())
        u, a, res, it = out
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_lsqr_sf_batch_host(self._h, nb, oi, si, _dptr(q), _dptr(d), float(lam),
                                             _dptr(tol), int(maxit), _dptr(u), _dptr(a), _dptr(res),
                                             _dptr(it)))
        return u, a, res, it

    def lsqr_sf_begin(self, d, lam, src_ijk, tol=None, maxit=50, omega_idx=None, q=None):
        t = self._torch
        nb = d.shape[1]
        self.ensure_workspace(nb, compaction=tol is not None)
        u, res, it = self._outputs(nb, maxit, d.device)
        a = t.empty(nb, dtype=t.complex64, device=d.device)
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        self._keep = [q, d, tol, u, a, res, it]
        _ck(self._lib.wri_lsqr_sf_begin(self._h, nb, oi, si, _dptr(q), _dptr(d), float(lam), _dptr(tol),
                                        int(maxit), _dptr(u), _dptr(a), _dptr(res), _dptr(it)))
        return u, a, res, it

    def objective_gradient(self, u, d, lam, omega_idx=None, q=None, src_ijk=None, alpha=None, g=None):
        """(f_pde [nb], f_data [nb]) float64 tensors; g (float32 [n_g]) is accumulated in place."""
        t = self._torch
        nb = u.shape[1]
        self.ensure_workspace(nb)
        fp = t.empty(nb, dtype=t.float64, device=u.device)
        fd = t.empty(nb, dtype=t.float64, device=u.device)
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_objective_gradient(self._h, nb, oi, si, _dptr(alpha), _dptr(q), _dptr(u), _dptr(d),
                                             float(lam), _dptr(fp), _dptr(fd), _dptr(g)))
        return fp, fd

    def objective_gradient_static(self, u, d, lam, f_pde, f_data, omega_idx=None, q=None, src_ijk=None,
                                  alpha=None, g=None):
        """wri_objective_gradient_static: the same operation with the scratch in the library image — no
        workspace, no device allocation here or in the library.  The caller passes the outputs f_pde,
        f_data (float64 [nb], device); g (float32 [n_g]) is accumulated in place.  Raises WriError
        (WRI_ERR_SCRATCH_LIMIT) when grid x width needs more than WRI_STATIC_SCRATCH_BYTES."""
        t = self._torch
        nb = u.shape[1]
        for f in (f_pde, f_data):
            if f.dtype != t.float64 or f.numel() != nb or not f.is_contiguous() or f.device != u.device:
                raise ValueError("f_pde / f_data: contiguous float64 [nb] on the device of u")
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_objective_gradient_static(self._h, nb, oi, si, _dptr(alpha), _dptr(q), _dptr(u),
                                                    _dptr(d), float(lam), _dptr(f_pde), _dptr(f_data),
                                                    _dptr(g)))

    def misfit_sf(self, d, lam, src_ijk, eps, maxit, omega_idx=None, g=None, warm=None, want_f=True):
        """One misfit evaluation (wri_misfit_sf).  warm = (u, alpha, ar0) from an earlier evaluation
        continues from it.  Returns dict(u, alpha, ar0, f_pde, f_data, iters, f); f is a host float
        (None with want_f=False: then nothing synchronises)."""
        t = self._torch
        nb = d.shape[1]
        self.ensure_workspace(nb, compaction=eps > 0)
        if warm is not None:
            u, a, ar0 = warm
        else:
            u = t.empty((self.ng, nb), dtype=t.complex64, device=d.device)
            a = t.empty(nb, dtype=t.complex64, device=d.device)
            ar0 = t.empty(nb, dtype=t.float64, device=d.device)
        fp = t.empty(nb, dtype=t.float64, device=d.device)
        fd = t.empty(nb, dtype=t.float64, device=d.device)
        it = t.empty(nb, dtype=t.int32, device=d.device)
        f = C.c_double(0.0)
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        _ck(self._lib.wri_misfit_sf(self._h, nb, oi, si, _dptr(d), float(lam), float(eps), int(maxit),
                                    int(warm is not None), _dptr(u), _dptr(a), _dptr(ar0), _dptr(fp),
                                    _dptr(fd), _dptr(g), _dptr(it), C.byref(f) if want_f else None))
        return dict(u=u, alpha=a, ar0=ar0, f_pde=fp, f_data=fd, iters=it, f=f.value if want_f else None)

    def awri_step(self, m, d, lam, src_ijk, eps, maxit, omega_idx=None, max_halvings=8, warm_restart=False,
                  update=None, step=0.0, m_min=0.0, m_max=float("inf"), reduce=None):
        """Lines 4-14 of Algorithm 2 (wri_awri_step) on the model tensor m (float32 [n_g], updated in
        place when the step is accepted).  update(m, g, m_trial): enqueue m_trial on the current
        stream (torch ops on the three tensors); None = built-in clamp(m - step g, m_min, m_max).
        reduce(f, g) -> f_sum: sum over ranks of the objective (a float) and, when g is not None,
        in-place all-reduce of the gradient tensor (column sharding); None = single process."""
        t = self._torch
        nb = d.shape[1]
        self.ensure_workspace(nb, compaction=True)
        dev = d.device
        m_trial = t.empty_like(m)
        g = t.empty(self.ng, dtype=t.float32, device=dev)
        u, ut = (t.empty((self.ng, nb), dtype=t.complex64, device=dev) for _ in range(2))
        a, at = (t.empty(nb, dtype=t.complex64, device=dev) for _ in range(2))
        fc = t.empty((2, nb), dtype=t.float64, device=dev)
        err = []

        def _cb(user, m_ptr, g_ptr, mt_ptr, stream):
            try:
                update(m, g, m_trial)
                return 0
            except Exception as e:                      # never raise across the C ABI
                err.append(e)
                return 1

        def _red(user, f_ptr, g_ptr, n_g, stream):
            try:
                f_ptr[0] = float(reduce(float(f_ptr[0]), g if g_ptr else None))
                return 0
            except Exception as e:
                err.append(e)
                return 1

        cb = wri_update_fn(_cb) if update is not None else wri_update_fn()
        rb = wri_reduce_fn(_red) if reduce is not None else wri_reduce_fn()
        o = wri_awri_opts(int(max_halvings), int(bool(warm_restart)), cb, None, float(step), float(m_min),
                          float(m_max), rb)
        rep = wri_awri_report()
        keep, oi = _i32(omega_idx)
        keep2, si = _i32(src_ijk)
        rc = self._lib.wri_awri_step(self._h, nb, oi, si, _dptr(d), float(lam), float(eps), int(maxit),
                                     C.byref(o), _dptr(m), _dptr(m_trial), _dptr(g), _dptr(u), _dptr(a),
                                     _dptr(ut), _dptr(at), _dptr(fc), C.byref(rep))
        if err:
            raise err[0]
        _ck(rc)
        n = rep.n_trace
        return dict(accepted=bool(rep.accepted), n_halvings=rep.n_halvings, eps=rep.eps, f=rep.f,
                    f_trial=rep.f_trial, lsqr_iters=rep.lsqr_iters, g=g, m_trial=m_trial, u=u, alpha=a,
                    u_trial=ut, alpha_trial=at, f_cols=fc,
                    trace=[(rep.trace_eps[i], rep.trace_f[i], rep.trace_f_trial[i]) for i in range(n)])

    def lsqr_iterate(self, n_steps=1):
        _ck(self._lib.wri_lsqr_iterate(self._h, int(n_steps)))

    def lsqr_end(self):
        _ck(self._lib.wri_lsqr_end(self._h))

    def lsqr_peek(self):
        """Copies of the device LSQR state as numpy arrays (synchronises)."""
        t = self._torch
        v = wri_lsqr_view()
        _ck(self._lib.wri_lsqr_peek(self._h, C.byref(v)))
        t.cuda.synchronize()
        nb = v.nb

        def grab(ptr, shape, dtype):
            typestr = {np.complex64: "<c8", np.float64: "<f8", np.float32: "<f4", np.int32: "<i4"}[dtype]
            view = t.as_tensor(_DevArray(ptr, tuple(int(x) for x in shape), typestr), device=self.m.device)
            return view.clone().cpu().numpy()

        out = {"nb": nb, "k": v.k}
        for name in ("U_top", "V", "W", "X"):
            out[name] = grab(getattr(v, name), (self.ng, nb), np.complex64)
        out["U_bot"] = grab(v.U_bot, (self.n_rec, nb), np.complex64) if self.n_rec else \
            np.zeros((0, nb), np.complex64)
        for name in ("alpha", "beta", "rhobar", "phibar", "ar0"):
            out[name] = grab(getattr(v, name), (nb,), np.float64)
        out["cx"] = grab(v.cx, (nb,), np.float32)
        out["cw"] = grab(v.cw, (nb,), np.float32)
        out["active"] = grab(v.active, (nb,), np.int32)
        out["iters"] = grab(v.iters, (nb,), np.int32)
        if v.sf_state:
            sf = grab(v.sf_state, (6, v.nb_max), np.float64)[:, :nb]
            out["v_a"] = sf[0] + 1j * sf[1]
            out["w_a"] = sf[2] + 1j * sf[3]
            out["x_a"] = sf[4] + 1j * sf[5]
        return out

    def profile_enable(self, on=True):
        _ck(self._lib.wri_profile_enable(self._h, int(bool(on))))

    def profile_read(self):
        """(ms_pass_f, n_pass_f, cols_pass_f, ms_pass_a, n_pass_a, cols_pass_a) since the last read;
        synchronises."""
        mf, ma = C.c_double(), C.c_double()
        nf, na, cf, ca = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int64()
        _ck(self._lib.wri_profile_read(self._h, C.byref(mf), C.byref(nf), C.byref(cf), C.byref(ma),
                                       C.byref(na), C.byref(ca)))
        return mf.value, nf.value, cf.value, ma.value, na.value, ca.value

    def launch_count(self):
        return int(self._lib.wri_launch_count(self._h))


class _DevArray:
    """Raw device pointer exposed through __cuda_array_interface__ (read-only view for torch)."""

    def __init__(self, ptr, shape, typestr):
        self.__cuda_array_interface__ = {"data": (int(ptr), False), "shape": shape,
                                         "typestr": typestr, "version": 2}
