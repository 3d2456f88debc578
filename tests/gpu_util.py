"""Helpers shared by the -m gpu parity tests: oracle operators per column, GPU state ->
Paige-Saunders state in float64."""
import numpy as np

from oracle import oracle as O


def ops_for(w):
    """One oracle Operator per batch column of a workload."""
    return [O.Operator(w.nx, w.ny, w.nz, w.h, w.omegas[j], w.sponge_width, w.gamma_max, w.power, w.faces)
            for j in w.omega_idx]


def rel(a, b):
    a = np.asarray(a, dtype=np.complex128).reshape(-1)
    b = np.asarray(b, dtype=np.complex128).reshape(-1)
    nb = np.linalg.norm(b)
    return float(np.linalg.norm(a - b) / nb) if nb > 0 else float(np.linalg.norm(a))


def gpu_state_column(st, s):
    """Normalised LSQR state of column s after st['k'] iterations, from the device state
    (un-normalised U, V; lagging W, X; include/wri.h wri_lsqr_view), in float64."""
    alpha, beta = float(st["alpha"][s]), float(st["beta"][s])
    W = st["W"][:, s].astype(np.complex128)
    V = st["V"][:, s].astype(np.complex128)
    v = V / alpha
    return dict(u_top=st["U_top"][:, s].astype(np.complex128) / beta,
                u_bot=st["U_bot"][:, s].astype(np.complex128) / beta,
                v=v,
                w=v - float(st["cw"][s]) * W,
                x=st["X"][:, s].astype(np.complex128) + float(st["cx"][s]) * W,
                alpha=alpha, beta=beta, rhobar=float(st["rhobar"][s]), phibar=float(st["phibar"][s]))


def gpu_state_column_sf(st, s):
    """Same for a source-free solve: adds the alpha entries of v, w, x (sf_state of
    wri_lsqr_view: v_a un-normalised like V; w_a and x_a are not deferred)."""
    g = gpu_state_column(st, s)
    g["v_a"] = complex(st["v_a"][s]) / g["alpha"]
    g["w_a"] = complex(st["w_a"][s])
    g["x_a"] = complex(st["x_a"][s])
    return g
