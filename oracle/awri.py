"""Oracle for one outer iteration of the adaptive scheme (Algorithm 2) and for
the misfit evaluation it is made of (eq. 7-9).

TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports only oracle/oracle.py
(the complex128 column solver and the objective/gradient of wri_oracle.c) and numpy.

misfit_sf   lines 4-5 (and 7-8) of Algorithm 2 for one group of columns:
              x_bar_s = argmin || S_s x - b_s ||   by LSQR to tolerance eps (eq. 7; reading C-6)
              f = sum_s 1/2 || S_s x_bar_s - b_s ||^2                       (eq. 8)
              g = sum_s lambda^2 omega_s^2 Re[conj((1+i gamma) u_s) (A u_s - alpha_s e_s)]  (eq. 9, C-18)
            in the paper's order: solve every column, then evaluate f and g at the solutions.
awri_step   lines 4-14 of Algorithm 2, written out in the paper's order:
              4:  x_bar   <- solve at m with tolerance eps
              5:  f, g    <- objective and gradient at (m, x_bar)
              6:  m_tilde <- update(m, g)          (the l-BFGS direction is the CALLER's: out of scope)
              7:  x_tilde <- solve at m_tilde with tolerance eps
              8:  f_tilde <- objective at (m_tilde, x_tilde)
              9-11: f_tilde > f  =>  eps <- 0.5 eps, go back to line 4
              13: else m <- m_tilde
            Readings (C-20): Algorithm 2 has no bound on the "go back" loop; a cap
            max_halvings is added, after which the step is returned as rejected with m unchanged.
            Line 9 compares numbers: a trial objective that is not finite (an update that left
            the physical range) counts as "f_tilde > f" (rejected); a non-finite f at the
            current model is an error.
            When the loop goes back to line 4 the re-solve at the same m may continue from
            x_bar (Algorithm 1 leaves x0 free; warm=True), with the stop rule still relative to
            the cold problem's ||S^H b|| (C-17); warm=False solves from zero as printed.
Pins: tests/test_oracle_awri.py.
"""
from __future__ import annotations

import numpy as np

from . import oracle as O


def misfit_sf(ops, m, lam, rec, src_cells, D, eps, maxit, x0=None, a0=None, ar_ref=None,
              want_gradient=True):
    """One misfit evaluation of the source-free problem for the columns of D[n_r, nb].

    x0 [n_g, nb], a0 [nb], ar_ref [nb]: warm start and the cold solve's alpha1*beta1 (C-17).
    Returns f (float), f_cols [nb], g [n_g] float64 or None, U [n_g, nb], alpha [nb],
    iters [nb], ar0 [nb] (alpha1*beta1 of a cold solve; the given ar_ref on a warm one)."""
    D = np.asarray(D)
    nb = D.shape[1]
    ng = ops[0].ng
    U = np.empty((ng, nb), dtype=np.complex128)
    alpha = np.empty(nb, dtype=np.complex128)
    iters = np.zeros(nb, dtype=np.int32)
    ar0 = np.zeros(nb)
    for s in range(nb):                                       # line 4 / 7: every column's solve
        if x0 is None:
            r = O.lsqr_sf(ops[s], m, lam, rec, int(src_cells[s]), D[:, s], tol=float(eps), maxit=maxit)
            ar0[s] = r["arnorms"][0]
        else:
            ref = float(ar_ref[s]) if ar_ref is not None else 0.0
            r = O.lsqr_sf_warm(ops[s], m, lam, rec, int(src_cells[s]), D[:, s], x0[:, s], a0[s],
                               tol=float(eps), maxit=maxit, ar_ref=ref)
            ar0[s] = ref if ref > 0.0 else r["arnorms"][0]
        U[:, s], alpha[s], iters[s] = r["x"], r["alpha_src"], r["iters"]
    g = np.zeros(ng) if want_gradient else None
    f_cols = np.zeros(nb)
    for s in range(nb):                                       # line 5 / 8: eq. 8 and eq. 9
        fp, fd = O.objective_gradient(ops[s], m, lam, rec, U[:, s], D[:, s], src=int(src_cells[s]),
                                      alpha_src=alpha[s], g=g)
        f_cols[s] = fp + fd
    return dict(f=float(f_cols.sum()), f_cols=f_cols, g=g, U=U, alpha=alpha, iters=iters, ar0=ar0)


def awri_step(ops, m, lam, rec, src_cells, D, eps, maxit, update, max_halvings=8, warm=False, reduce=None):
    """Lines 4-14 of Algorithm 2 for the model m (float array [n_g]).  update(m, g) -> m_tilde.
    reduce(f, g) -> f: the sums of eq. 8-9 taken over column blocks held elsewhere (column sharding,
    PAPER.md:221): returns the summed objective and sums g (a float64 array, or None) in place;
    None = these are all the columns.

    Returns dict(accepted, m (the next model), eps (the tolerance in force at the end),
    n_halvings, f, f_trial, g (gradient at the entry model with the final eps), lsqr_iters
    (all column iterations spent), trace [(eps, f, f_trial), ...])."""
    m = np.asarray(m)
    eps = float(eps)
    trace = []
    total = 0
    prev = None
    for h in range(max_halvings + 1):
        if warm and prev is not None:                         # line 4 after a "go back"
            cur = misfit_sf(ops, m, lam, rec, src_cells, D, eps, maxit, x0=prev["U"], a0=prev["alpha"],
                            ar_ref=prev["ar0"])
        else:
            cur = misfit_sf(ops, m, lam, rec, src_cells, D, eps, maxit)          # lines 4-5
        total += int(cur["iters"].sum())
        if reduce is not None:
            cur["f"] = reduce(cur["f"], cur["g"])
        if not np.isfinite(cur["f"]):
            raise FloatingPointError("objective at the current model is not finite")
        m_t = update(m, cur["g"])                                                  # line 6
        tri = misfit_sf(ops, m_t, lam, rec, src_cells, D, eps, maxit, want_gradient=False)  # lines 7-8
        total += int(tri["iters"].sum())
        if reduce is not None:
            tri["f"] = reduce(tri["f"], None)
        trace.append((eps, cur["f"], tri["f"]))
        if np.isfinite(tri["f"]) and tri["f"] <= cur["f"]:                         # line 9 / 12-13
            return dict(accepted=True, m=m_t, eps=eps, n_halvings=h, f=cur["f"], f_trial=tri["f"],
                        g=cur["g"], lsqr_iters=total, trace=trace)
        if h == max_halvings:
            break
        eps *= 0.5                                                                 # line 10
        prev = cur
    return dict(accepted=False, m=m, eps=eps, n_halvings=max_halvings, f=cur["f"], f_trial=tri["f"],
                g=cur["g"], lsqr_iters=total, trace=trace)
