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


def oracle_eval_multi(coeff, weight, gap, params, Nt, Nf, dt, N_segs, **opts):
    """Oracle results for several N_seg at once: the dense template of a row is built once
    (O.dense_template) and O.segment_products / O.combine run once per N_seg -- the same calls
    O.evaluate makes, so the values are identical to calling it per N_seg.  Returns {N_seg: dict}."""
    g = O.Grid(Nt, Nf, dt)
    o = O.Opts(**opts)
    D = to_complex(coeff)
    W = None if weight is None else np.asarray(weight, dtype=np.float64)
    params = np.atleast_2d(np.asarray(params, dtype=np.float64))
    n = len(params)
    out = {N: dict(upsilon=np.zeros(n), seg_power=np.zeros((n, N)), seg_dh=np.zeros((n, N), dtype=np.complex128),
                   seg_hh=np.zeros((n, N))) for N in N_segs}
    for i, p in enumerate(params):
        if not np.all(np.isfinite(p)) or p[0] <= 0:
            continue
        Hd = O.dense_template(p[0], p[1], p[2], p[7], g, o, gap, truncate=True)
        T = np.array([p[3] + 1j * p[4], p[5] + 1j * p[6]])
        for N in N_segs:
            z, hh = O.segment_products(Hd, T[: D.shape[0]], D, W, gap, N)
            P, U = O.combine(z, hh)
            r = out[N]
            r["upsilon"][i], r["seg_power"][i], r["seg_dh"][i], r["seg_hh"][i] = U, P, z, hh
    return out


def add_injections(coeff, weight, gap, inj_list, Nt, Nf, dt, truncate=False, **opts):
    """coeff += injected signals (oracle-made dense templates: untruncated by default; truncate=True keeps
    only the window that `opts` defines, e.g. half_width=100 at full size where filling every bin of a
    4096 x 3072 grid takes minutes per signal); float32 in, float32 out."""
    g = O.Grid(Nt, Nf, dt)
    W = None if weight is None else np.asarray(weight, dtype=np.float64)
    for p, rho in inj_list:
        S = O.injection(p, rho, W, gap, g, O.Opts(**opts), truncate=truncate)
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
