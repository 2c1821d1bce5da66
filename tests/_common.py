"""Shared helpers for the parity tests (test code only: may import the oracle)."""
import numpy as np

from oracle import tfs_oracle as O

TOL = 1e-4          # BASELINE.json north_star: 1e-4 relative on every Upsilon and per-segment product


def to_complex(coeff):
    c = np.asarray(coeff, dtype=np.float64)
    return c[..., 0] + 1j * c[..., 1]


def oracle_eval(coeff, weight, gap, params, Nt, Nf, dt, N_seg, **opts):
    g = O.Grid(Nt, Nf, dt)
    W = None if weight is None else np.asarray(weight, dtype=np.float64)
    return O.evaluate(params, to_complex(coeff), W, gap, g, N_seg, O.Opts(**opts))


def add_injections(coeff, weight, gap, inj_list, Nt, Nf, dt, **opts):
    """coeff += injected signals (oracle-made, untruncated dense templates); float32 in, float32 out."""
    g = O.Grid(Nt, Nf, dt)
    W = None if weight is None else np.asarray(weight, dtype=np.float64)
    for p, rho in inj_list:
        S = O.injection(p, rho, W, gap, g, O.Opts(**opts))
        coeff[..., 0] += S.real.astype(np.float32)
        coeff[..., 1] += S.imag.astype(np.float32)
    return coeff


def parity_report(gpu, ora, N_seg):
    """Errors under the DESIGN.md C12 criterion.  Returns dict of worst normalised errors (<= 1 passes
    at TOL) and the plain relative error on Upsilon."""
    zg, zo = np.asarray(gpu["seg_dh"]), np.asarray(ora["seg_dh"])
    hg, ho = np.asarray(gpu["seg_hh"], dtype=np.float64), np.asarray(ora["seg_hh"])
    ug, uo = np.asarray(gpu["upsilon"], dtype=np.float64), np.asarray(ora["upsilon"])
    Pg, Po = np.asarray(gpu["seg_power"], dtype=np.float64), np.asarray(ora["seg_power"])
    n_eff = np.maximum((ho > 0).sum(axis=1), 1)
    with np.errstate(divide="ignore", invalid="ignore"):
        e_hh = np.where(ho > 0, np.abs(hg - ho) / np.where(ho > 0, ho, 1.0), np.abs(hg))
        e_z = np.abs(zg - zo) / np.maximum(np.maximum(np.abs(zo), np.sqrt(2.0 * ho)), 1e-300)
        e_z = np.where(ho > 0, e_z, np.abs(zg))
        e_u = np.abs(ug - uo) / np.maximum(uo, 2.0 * n_eff)
        e_P = np.abs(Pg - Po) / np.maximum(Po, 2.0)
        rel_u = np.where(uo > 0, np.abs(ug - uo) / np.where(uo > 0, uo, 1.0), np.abs(ug))
    return dict(hh=float(e_hh.max(initial=0.0)), z=float(e_z.max(initial=0.0)), ups=float(e_u.max(initial=0.0)),
                P=float(e_P.max(initial=0.0)), rel_ups=float(rel_u.max(initial=0.0)),
                n_active=int((uo > 0).sum()))


def assert_parity(gpu, ora, N_seg, tol=TOL, label=""):
    r = parity_report(gpu, ora, N_seg)
    msg = f"{label} parity {r}"
    assert r["hh"] <= tol, msg
    assert r["z"] <= tol, msg
    assert r["ups"] <= tol, msg
    assert r["P"] <= tol, msg
    return r
