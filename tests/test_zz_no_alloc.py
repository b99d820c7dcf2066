"""mppi_step_static (include/mppi.h): the entry point that allocates nothing -- scratch in a file-scope static device
array -- against the existing allocating path (mppi_create + mppi_set_gates + mppi_step) on the same inputs.

Named test_zz_* so that pytest collects it LAST (the suite runs with pytest -x).  It must pass alone in a fresh
process and after every other test: the static array is shared by all calls of a process and keeps the last call's
contents, so the second call of each case runs on an array the first one has used."""
import numpy as np
import pytest

import parity as Pz
from paper_2509_14726_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _both_paths(wl, seed, iters, fast_math):
    """`iters` warm-started iterations through both paths; -> list of (existing, static) result dicts."""
    import torch
    from paper_2509_14726_b200 import binding as Bd
    P = wl.params
    m = Pz.make_ctx(wl, fast_math=fast_math)
    x0, start, u_a = Pz.to_dev(wl)
    u_b = u_a.clone()
    gates = torch.from_numpy(np.ascontiguousarray(wl.gates, dtype=np.float32)).cuda()
    prm = Bd.make_params(P, fast_math=fast_math)
    # every output of the static path is allocated HERE, before its first call
    cost_b = torch.empty((P["B"], P["K"]), device="cuda"); w_b = torch.empty_like(cost_b)
    out = []
    for it in range(iters):
        g = Pz.gpu_step(m, x0, start, u_a, seed, it, u_new=u_a)                                   # existing path, in place
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        Bd.step_static(prm, gates, x0, start, u_b, seed, it, u_b, cost_b, w_b)                     # static path, in place
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info()[0]
        if it > 0:          # (the first call of a process may load the kernels' code lazily)
            assert free1 == free0, "device memory in use changed across a call of the static path"
        out.append((g, dict(u_new=u_b.cpu().numpy(), cost=cost_b.cpu().numpy(), weights=w_b.cpu().numpy())))
    m.close()
    return out


@pytest.mark.parametrize("fast_math", [0, 1], ids=["accurate", "fast"])
def test_static_path_equals_the_allocating_path_on_two_calls_in_a_row(fast_math):
    # configs[1] (K = 4096, N = 50, one controller): AUTO runs the same pipelined kernel on the allocating path
    wl = W.cfg1()
    for it, (g, s) in enumerate(_both_paths(wl, wl.seed, 3, fast_math)):
        Jg, Js = g["cost"].astype(np.float64), s["cost"].astype(np.float64)
        assert np.isfinite(Js).all()
        assert (np.abs(Js - Jg) <= Pz.COST_RTOL * np.maximum(np.abs(Jg), 1.0)).all(), f"iteration {it}: costs differ"
        assert np.abs(s["weights"].astype(np.float64) - g["weights"]).max() <= Pz.W_ATOL, f"iteration {it}: weights differ"
        assert np.abs(s["u_new"].astype(np.float64) - g["u_new"]).max() <= Pz.U_ATOL, f"iteration {it}: u_new differs"
        assert abs(float(s["weights"].sum()) - 1.0) < 2e-5


def test_static_path_matches_the_oracle_and_handles_batches_and_ragged_sizes():
    # B = 3 controllers, K = 96, N = 7 on the crossing-heavy track: the static path on its own against the oracle,
    # twice in a row (the second call reuses the array the first one left behind, and a different grid used it before)
    import torch
    from paper_2509_14726_b200 import binding as Bd
    wl = W.replicate(W.stress_gate(K=96, N=7), 3, 0.2)
    prm = Bd.make_params(wl.params)
    x0, start, u = Pz.to_dev(wl)
    gates = torch.from_numpy(wl.gates).cuda()
    u_new = torch.empty_like(u); cost = torch.empty((3, 96), device="cuda"); w = torch.empty_like(cost)
    for it in range(2):
        Bd.step_static(prm, gates, x0, start, u, wl.seed, it, u_new, cost, w)
        torch.cuda.synchronize()
        g = dict(u_new=u_new.cpu().numpy(), cost=cost.cpu().numpy(), weights=w.cpu().numpy())
        o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, it, want_du=True)
        Pz.compare(f"static path B3 K96 N7 it{it}", g, o, wl.params["lambda"], True)


def test_static_path_rejects_sizes_beyond_its_scratch():
    import torch
    from paper_2509_14726_b200 import binding as Bd
    wl = W.cfg1()
    x0, start, u = Pz.to_dev(wl)
    gates = torch.from_numpy(wl.gates).cuda()
    for over, text in ((dict(K=Bd.STATIC_MAX["K"] + 32), "MPPI_STATIC_MAX_K"), (dict(N=Bd.STATIC_MAX["N"] + 1), "MPPI_STATIC_MAX_N"),
                       (dict(B=Bd.STATIC_MAX["B"] + 1), "MPPI_STATIC_MAX_B")):
        p = dict(wl.params, **over)
        B, N, K = p["B"], p["N"], p["K"]
        args = (torch.zeros((B, 13), device="cuda"), torch.zeros(B, dtype=torch.int32, device="cuda"),
                torch.zeros((B, N, 4), device="cuda"))
        with pytest.raises(Bd.MppiError) as e:
            Bd.step_static(p, gates, *args, 0, 0, torch.zeros((B, N, 4), device="cuda"), torch.zeros((B, K), device="cuda"),
                           torch.zeros((B, K), device="cuda"))
        assert e.value.status == -5 and text in str(e.value)                # MPPI_E_RANGE, with the limit named
    big = torch.zeros((Bd.STATIC_MAX["G"] + 1, 11), device="cuda")
    with pytest.raises(Bd.MppiError) as e:
        Bd.step_static(wl.params, big, x0, start, u, 0, 0, torch.empty_like(u), torch.empty((1, 4096), device="cuda"),
                       torch.empty((1, 4096), device="cuda"))
    assert e.value.status == -5 and "MPPI_STATIC_MAX_GATES" in str(e.value)
    with pytest.raises(Bd.MppiError) as e:                                   # another objective: not this entry point
        Bd.step_static(dict(W.cfg2().params), gates, x0, start, u, 0, 0, torch.empty_like(u),
                       torch.empty((1, 4096), device="cuda"), torch.empty((1, 4096), device="cuda"))
    assert e.value.status == -2
