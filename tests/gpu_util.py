"""Helpers shared by the -m gpu parity tests: oracle operators per column, GPU state ->
Paige-Saunders state in float64."""
import numpy as np

from oracle import oracle as O


def ops_for(w, stencil=0):
    """One oracle Operator per batch column of a workload (stencil: 0 = 7-point, 1 = 27-point)."""
    return [O.Operator(w.nx, w.ny, w.nz, w.h, w.omegas[j], w.sponge_width, w.gamma_max, w.power, w.faces,
                       stencil=stencil)
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


def c64_floor(solve, d, members=3):
    """Attainable floor of a complex64 solver on one column: the deviation
    from the complex128 iterates of the oracle's own complex64-STORAGE emulation (round_c64), taken as
    the largest over a few members whose data differ by one float32 rounding (6e-8 relative) — the
    onset of the orthogonality loss moves by an iteration or two between such members, so a single one
    can sit on the lucky side at a given k.  solve(d, round_c64) -> dict with "x" and "resnorms".
    Returns (floor_x, floor_history, reference); c64_floor.last_residual holds the floor of the LAST
    residual norm alone, |res_K / ref_K - 1| (the history norm is dominated by its early entries)."""
    ref = solve(d, False)
    fx = fh = 0.0
    c64_floor.last_residual = 0.0
    for i in range(members):
        dd = d
        if i:
            rng = np.random.Generator(np.random.PCG64(100 + i))
            dd = d * (1.0 + 6e-8 * (rng.standard_normal(d.size) + 1j * rng.standard_normal(d.size)))
        e = solve(dd, True)
        fx = max(fx, rel(e["x"], ref["x"]))
        fh = max(fh, rel(e["resnorms"], ref["resnorms"]))
        c64_floor.last_residual = max(c64_floor.last_residual,
                                      abs(float(e["resnorms"][-1]) / float(ref["resnorms"][-1]) - 1.0))
    return fx, fh, ref
