"""Helpers of the GPU parity tests: run a workload through the C ABI (libmppi) and through the
float64 oracle on the same seeded inputs and compare element by element.

Tolerances are BASELINE.json:north_star's: per-sample cost |dJ| <= 1e-4 max(|J|, 1) [R-20];
samples whose oracle gate-plane crossing margin is below 1e-5 m are counted separately [R-19];
weights abs 1e-5; u_new abs 1e-4 N.
"""
from __future__ import annotations

import numpy as np

COST_RTOL = 1e-4
W_ATOL = 1e-5
U_ATOL = 1e-4
MARGIN = 1e-5

STATS: list[str] = []           # one line per compared iteration: achieved errors
REPORT: list[str] = []          # "reported separately" lines, printed at the end of the session


def oracle_track(wl):
    from oracle import oracle as O
    return O.Track(gates=wl.gates, ref=wl.ref, path=wl.path, closed=wl.closed,
                   prev_front=getattr(wl, "prev_front", None))


def make_ctx(wl, **opts):
    from paper_2509_14726_b200 import binding as Bd
    m = Bd.Mppi(wl.params, **opts)
    m.set_track(wl)
    return m


def to_dev(wl):
    import torch
    return (torch.from_numpy(wl.x0.copy()).cuda(), torch.from_numpy(wl.start.copy()).cuda(),
            torch.from_numpy(wl.u_nom.copy()).cuda())


def gpu_step(m, x0, start, u_nom, seed, it, **kw):
    import torch
    u_new, cost, w = m.step(x0, start, u_nom, seed, it, **kw)
    torch.cuda.synchronize()
    r = dict(u_new=u_new.cpu().numpy(), cost=cost.cpu().numpy(), weights=w.cpu().numpy())
    if getattr(m, "_v", None) is not None:
        r["v_new"] = m._v[1].cpu().numpy()
    return r


def oracle_step(wl, x0, start, u_nom, seed, it, want_du=False, params=None, v_nom=None):
    from oracle import oracle as O
    return O.step(params or wl.params, oracle_track(wl), np.asarray(x0, np.float64),
                  np.asarray(start, np.int32), np.asarray(u_nom, np.float64), seed, it, want_du=want_du,
                  v_nom=None if v_nom is None else np.asarray(v_nom, np.float64))


def compare(tag, g, o, lam, gate_objective, cost_floor=1.0):
    """Asserts parity of one iteration; returns a small stats dict.  cost_floor: the smallest magnitude
    the cost error is measured against (1 by [R-20]; objective 4 passes the size of the progress reward
    its positive terms cancel against [R-38])."""
    Jg, Jo = g["cost"].astype(np.float64), o["cost"]
    assert np.isfinite(Jg).all(), f"{tag}: non-finite GPU cost"
    flagged = (o["margin"] < MARGIN) if gate_objective else np.zeros_like(Jo, dtype=bool)
    err = np.abs(Jg - Jo) / np.maximum(np.abs(Jo), cost_floor)
    ok = err <= COST_RTOL
    n_flag = int(flagged.sum())
    assert ok[~flagged].all(), (f"{tag}: {int((~ok & ~flagged).sum())} costs out of tolerance, worst rel "
                               f"{err[~flagged].max():.3e} at {np.unravel_index(np.argmax(np.where(flagged, 0, err)), err.shape)}")
    assert n_flag <= max(2, 0.01 * Jo.size), f"{tag}: {n_flag} samples within {MARGIN} m of a crossing decision"
    if n_flag:
        REPORT.append(f"{tag}: {n_flag} samples with crossing margin < {MARGIN} m reported separately "
                      f"({int((~ok & flagged).sum())} of them differ)")

    wg, wo = g["weights"].astype(np.float64), o["weights"]
    assert np.allclose(wg.sum(-1), 1.0, atol=2e-5), f"{tag}: weights do not sum to 1"
    # [R-19] weight rule: first-order sensitivity of the softmax to the observed cost error
    dJ = float(np.abs(Jg - Jo)[~flagged].max()) if (~flagged).any() else 0.0
    sens = float((wo * (1.0 - wo)).max()) * 2.0 * dJ / lam
    decided_by_flagged = bool(((wo > 1e-6) | (wg > 1e-6))[flagged & ~ok].any()) if n_flag else False
    werr = float(np.abs(wg - wo).max())
    uerr = float(np.abs(g["u_new"].astype(np.float64) - o["u_new"]).max())
    strict = werr <= W_ATOL and uerr <= U_ATOL
    if not strict:
        # allowed only when fp32 cannot resolve the decision: then the GPU must still be the exact
        # softmax / update of ITS OWN costs
        assert sens > 0.5 * W_ATOL or decided_by_flagged, (
            f"{tag}: weights err {werr:.3e}, u_new err {uerr:.3e} (sensitivity bound {sens:.2e})")
        z = np.exp(-(Jg - Jg.min(-1, keepdims=True)) / lam)
        w_self = z / z.sum(-1, keepdims=True)
        assert np.abs(wg - w_self).max() <= W_ATOL, f"{tag}: weights are not the softmax of the GPU costs"
        if o.get("du") is not None:
            u_self = o["u_nom"] + np.einsum("bk,bktn->btn", w_self, o["du"])
            assert np.abs(g["u_new"] - u_self).max() <= U_ATOL, f"{tag}: u_new inconsistent with its weights"
        REPORT.append(f"{tag}: near-tied minimum (sensitivity {sens:.2e}, flagged-decided {decided_by_flagged}): "
                      f"weights err {werr:.2e}, u_new err {uerr:.2e} reported separately")
    st = dict(cost_rel=float(err[~flagged].max()) if (~flagged).any() else 0.0, w=werr, u=uerr,
              flagged=n_flag, ess=float(1.0 / (wo ** 2).sum(-1).min()))
    STATS.append(f"{tag}: cost rel {st['cost_rel']:.2e}  weights {werr:.2e}  u_new {uerr:.2e}  ESS {st['ess']:.1f}  flagged {n_flag}")
    return st
