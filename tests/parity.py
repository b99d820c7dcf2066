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
    """One oracle iteration.  The result also carries what compare()'s near-tie fall-back needs: the nominal
    (u_nom), the largest possible |dU| entry (du_max) and, when the perturbations were not kept, a callable
    that re-runs the oracle for them (du_fn)."""
    from oracle import oracle as O
    p = params or wl.params
    args = (p, oracle_track(wl), np.asarray(x0, np.float64), np.asarray(start, np.int32), np.asarray(u_nom, np.float64), seed, it)
    vn = None if v_nom is None else np.asarray(v_nom, np.float64)
    o = O.step(*args, want_du=want_du, v_nom=vn)
    o["u_nom"] = np.asarray(u_nom, np.float64).reshape(o["u_new"].shape)
    o["du_max"] = 2.0 * float(p["rate_max"]) if p.get("input_model", 0) == 1 else float(p["T_max"]) - float(p["T_min"])
    if not want_du:
        o["du_fn"] = lambda: O.step(*args, want_du=True, want_diag=False, v_nom=vn)["du"]
    return o


def compare(tag, g, o, lam, gate_objective, cost_floor=1.0, du_fn=None, du_max=None):
    """Asserts parity of one iteration; returns a small stats dict.  cost_floor: the smallest magnitude
    the cost error is measured against (1 by [R-20]; objective 4 passes the size of the progress reward
    its positive terms cancel against [R-38]).  du_fn: zero-argument callable returning the oracle's
    perturbations [B,K,N,4] on demand (large cases do not keep them); du_max: largest possible |dU| entry
    (T_max - T_min, or 2 rate_max), used by the bound on u_new in the near-tie fall-back."""
    Jg, Jo = g["cost"].astype(np.float64), o["cost"]
    du_fn = du_fn or o.get("du_fn")
    du_max = du_max if du_max is not None else o.get("du_max")
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
    counted = ~(flagged & ~ok)             # everything but the flagged samples whose cost really differs
    dJ = float(np.abs(Jg - Jo)[counted].max()) if counted.any() else 0.0
    sens = float((wo * (1.0 - wo)).max()) * 2.0 * dJ / lam
    decided_by_flagged = bool(((wo > 1e-6) | (wg > 1e-6))[flagged & ~ok].any()) if n_flag else False
    werr = float(np.abs(wg - wo).max())
    uerr = float(np.abs(g["u_new"].astype(np.float64) - o["u_new"]).max())
    strict = werr <= W_ATOL and uerr <= U_ATOL
    if not strict:
        # allowed only when fp32 cannot resolve the decision.  Then (i) the deviation must stay inside what the
        # observed cost error can do to a softmax: with every |dJ_k| <= dJ, w'_k / w_k and (1 - w'_k) / (1 - w_k)
        # lie in [exp(-2 dJ / lam), exp(2 dJ / lam)], hence |dw_k| <= min(w_k, 1 - w_k) (exp(2 dJ / lam) - 1) and
        # |du_new| <= sum_k |dw_k| max|dU|; (ii) the GPU must still be the exact softmax / update of ITS OWN costs
        assert sens > 0.5 * W_ATOL or decided_by_flagged, (
            f"{tag}: weights err {werr:.3e}, u_new err {uerr:.3e} (sensitivity bound {sens:.2e})")
        if not decided_by_flagged:
            grow = float(np.expm1(min(2.0 * dJ / lam, 50.0)))
            mw = np.minimum(wo, 1.0 - wo)
            bound_w = float(mw.max()) * grow + W_ATOL
            assert werr <= bound_w, f"{tag}: weights err {werr:.3e} beyond what a cost error of {dJ:.2e} explains ({bound_w:.2e})"
            if du_max is not None:
                bound_u = float(mw.sum(-1).max()) * grow * float(du_max) + U_ATOL
                assert uerr <= bound_u, f"{tag}: u_new err {uerr:.3e} beyond what a cost error of {dJ:.2e} explains ({bound_u:.2e})"
        z = np.exp(-(Jg - Jg.min(-1, keepdims=True)) / lam)
        w_self = z / z.sum(-1, keepdims=True)
        assert np.abs(wg - w_self).max() <= W_ATOL, f"{tag}: weights are not the softmax of the GPU costs"
        du = o.get("du")
        if du is None and du_fn is not None:
            du = du_fn()
        assert du is not None, f"{tag}: the near-tie fall-back needs the oracle's perturbations (pass du_fn)"
        u_self = o["u_nom"] + np.einsum("bk,bktn->btn", w_self, du)
        assert np.abs(g["u_new"] - u_self).max() <= U_ATOL, f"{tag}: u_new inconsistent with its weights"
        REPORT.append(f"{tag}: near-tied minimum (sensitivity {sens:.2e}, flagged-decided {decided_by_flagged}): "
                      f"weights err {werr:.2e}, u_new err {uerr:.2e} reported separately")
    st = dict(cost_rel=float(err[~flagged].max()) if (~flagged).any() else 0.0, w=werr, u=uerr,
              flagged=n_flag, ess=float(1.0 / (wo ** 2).sum(-1).min()))
    STATS.append(f"{tag}: cost rel {st['cost_rel']:.2e}  weights {werr:.2e}  u_new {uerr:.2e}  ESS {st['ess']:.1f}  flagged {n_flag}")
    return st
