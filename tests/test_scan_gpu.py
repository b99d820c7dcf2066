"""GPU parity tests of the time-parallel latency kernel (MPPI_VARIANT_SCAN = 5, csrc/mppi_scan.cuh): every rollout is
split over 16 lanes along the horizon and the chunks are joined by scans.  Its states equal the sequential RK4's to
rounding only, so -- as for every kernel -- the reference is the float64 oracle, element by element through the C ABI,
within north_star's tolerances (tests/parity.py)."""
from __future__ import annotations

import numpy as np
import pytest

import parity as Pz
from paper_2509_14726_b200 import workloads as W

pytestmark = pytest.mark.gpu
SCAN = 5
MATH = [dict(fast_math=0), dict(fast_math=1)]


def run_case(wl, tag, it=0, **opts):
    m = Pz.make_ctx(wl, **opts)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, it)
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, it, want_du=wl.params["K"] * wl.params["N"] * wl.params["B"] <= 1 << 22)
    o["u_nom"] = wl.u_nom.astype(np.float64)
    st = Pz.compare(tag, g, o, wl.params["lambda"], wl.params["objective"] in (0, 3))
    info = m.info()
    m.close()
    return g, o, st, info


@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
@pytest.mark.parametrize("K,N,B", [(32, 1, 1), (64, 16, 1), (96, 17, 2), (256, 20, 1), (480, 33, 3), (1024, 48, 2),
                                   (4096, 50, 1), (4096, 64, 1), (2048, 49, 5), (16384, 20, 1)])
def test_sizes_chunks_and_ragged_blocks(K, N, B, math):
    # chunk lengths 1..4 (N = 1 .. 64), horizons that leave lanes idle or half-filled (17, 33, 49, 50), blocks of 8 .. 32
    # samples incl. a ragged last block (K = 4096 on 148 SMs: 147 blocks of 28), several controllers, more blocks than
    # SMs (K = 16384), crossing-heavy track
    wl = W.cfg4(K=K, N=N, B=B) if B > 1 else W.stress_gate(K=K, N=N)
    g, o, st, info = run_case(wl, f"scan K{K} N{N} B{B} {math}", variant=SCAN, **math)
    assert info["rollout_warps_per_block"] == 16 and info["block_threads"] % 32 == 0 and 128 <= info["block_threads"] <= 512
    spb = info["block_threads"] // 16
    assert info["blocks_per_controller"] == -(-K // spb) and info["local_bytes_per_thread"] == 0
    if B == 1 and N >= 30:
        assert int((o["ncross"] > 0).sum()) > 0


def test_cfg1_ten_warm_started_iterations():
    # configs[1] as stated: 10 warm-started iterations, the oracle teacher-forced with the GPU's nominal [R-14]
    wl = W.cfg1()
    m = Pz.make_ctx(wl, variant=SCAN)
    info = m.info()
    assert info["blocks_per_controller"] > 128 or info["sm_count"] <= 128     # a lone controller spreads over every SM
    x0, start, u = Pz.to_dev(wl)
    crossings = 0
    for it in range(wl.iters):
        u_in = u.cpu().numpy()
        g = Pz.gpu_step(m, x0, start, u, wl.seed, it, u_new=u)          # in place
        o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, it, want_du=True)
        o["u_nom"] = u_in.astype(np.float64)
        Pz.compare(f"scan cfg1 it{it}", g, o, wl.params["lambda"], True)
        crossings += int((o["ncross"] > 0).sum())
        np.testing.assert_array_equal(u.cpu().numpy(), g["u_new"])
    assert crossings > 0
    m.close()


@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_crossings_in_every_chunk(math):
    # the hypothesis rounds of the gate objective: passes and misses, several target switches per horizon, spread over
    # the chunks -- both branches of the crossing test must be well populated
    wl = W.stress_gate(K=4096, N=64)
    g, o, st, _ = run_case(wl, f"scan stress N64 {math}", variant=SCAN, **math)
    assert (o["ncross"][0] >= 1).mean() > 0.1
    wl = W.stress_gate(K=2048, N=30)
    run_case(wl, f"scan stress N30 {math}", variant=SCAN, **math)
    # a slalom of eight gates 1.4 m apart flown at 9 m/s: three to six target switches in one horizon, i.e. as many
    # rounds of re-scoring, in chunks next to each other
    wl = W.stress_gate(K=2048, N=64)
    G = 8
    gates = np.zeros((G, 11), np.float32)
    gates[:, 0] = 1.0 + 1.4 * np.arange(G); gates[:, 2] = 2.0
    gates[:, 3] = 1.0; gates[:, 7] = 1.0; gates[:, 9] = 1.2; gates[:, 10] = 0.9
    wl.gates = gates
    wl.x0[:] = 0.0; wl.x0[:, 2] = 2.0; wl.x0[:, 3] = 1.0; wl.x0[:, 7] = 9.0
    wl.start[:] = 0
    g, o, st, _ = run_case(wl, f"scan slalom {math}", variant=SCAN, **math)
    nc = o["ncross"][0]
    assert (nc >= 3).mean() > 0.5 and nc.max() >= 5, (np.bincount(nc),)


@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
@pytest.mark.parametrize("near_mode", [0, 1])
def test_the_papers_own_gate_objective(near_mode, math):
    # objective 3 (eq.(6),(7) with squared distances, Q_near term, temporal check with previous-iteration flags): on the
    # configs[1] track at full size, and crossing-heavy with RANDOM flags so that registered and unregistered passes of
    # the start gate both occur, in both readings of the near term
    wl = W.gate_paper()
    wl.params["near_mode"] = near_mode
    run_case(wl, f"scan gate_paper near{near_mode} {math}", variant=SCAN, **math)
    for K, N, B in ((2048, 30, 1), (1024, 64, 1), (512, 37, 3)):
        wl = W.stress_gate_paper(K=K, N=N)
        wl.params["near_mode"] = near_mode
        if B > 1:
            wl = W.replicate(wl, B, 0.2)
        g, o, st, _ = run_case(wl, f"scan stress_gate_paper K{K} N{N} B{B} near{near_mode} {math}", variant=SCAN, **math)
        assert int((o["ncross"] > 0).sum()) > 0


def test_mixing_weights_strict():
    # many samples carry weight: every warp of every block takes part in the block partial; strict bounds
    wl = W.cfg1(K=2048, N=50)
    o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    wl.params["lambda"] = float(np.float32(0.25 * o0["cost"].std()))
    g, o, st, _ = run_case(wl, "scan flat-cfg1", variant=SCAN)
    assert st["ess"] > 20
    assert st["w"] <= Pz.W_ATOL and st["u"] <= Pz.U_ATOL


def test_unnormalised_start_quaternion_and_spinning_start():
    # x0 is taken as given (the first step's stage attitudes are not normalised, as in the sequential RK4): lane 0 starts
    # its chunk from q0 itself.  Also a fast-spinning start, where the body-rate scan (the complex affine maps) matters.
    wl = W.stress_gate(K=1024, N=40)
    wl.x0[:, 3:7] *= np.float32(1.07)
    wl.x0[:, 10:13] = np.array([6.0, -4.0, 9.0], np.float32)
    run_case(wl, "scan q0 x 1.07, spinning", variant=SCAN)
    run_case(wl, "scan q0 x 1.07, spinning, fast", variant=SCAN, fast_math=1)


@pytest.mark.parametrize("name,B", [("cfg1", 1), ("stress_gate", 3), ("gate_paper", 2)])
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_optimize_chain_equals_the_steps(name, B, math):
    # mppi_optimize: programmatic dependent launch without a graph, one graph launch with use_graph -- both must equal
    # the chain of single steps bit for bit, repeatedly (a race would show as a run-to-run difference)
    import torch
    wl = W.replicate(W.ALL[name](), B, 0.2) if B > 1 else W.ALL[name]()
    x0, start, u0 = Pz.to_dev(wl)
    m = Pz.make_ctx(wl, variant=SCAN, **math)
    u = u0.clone()
    n = 6
    for it in range(n):
        if it == n - 1:
            u_in = u.cpu().numpy()
        _, c_ref, w_ref = m.step(x0, start, u, wl.seed, it, u_new=u)
    torch.cuda.synchronize()
    for graph in (0, 1):
        m2 = Pz.make_ctx(wl, variant=SCAN, use_graph=graph, **math)
        for rep in range(4):
            u2 = u0.clone()
            _, c2, w2 = m2.optimize(x0, start, u2, wl.seed, 0, n)
            torch.cuda.synchronize()
            assert torch.equal(u2, u) and torch.equal(c2, c_ref) and torch.equal(w2, w_ref), (graph, rep)
        m2.close()
    o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, n - 1, want_du=True)
    g = dict(u_new=u.cpu().numpy(), cost=c_ref.cpu().numpy(), weights=w_ref.cpu().numpy())
    Pz.compare(f"scan optimize chain {name} B{B} {math}", g, o, wl.params["lambda"], wl.params["objective"] in (0, 3))
    m.close()


def test_sigma_zero_saturated_nominal_and_diverged_samples():
    wl = W.cfg0(K=128, N=10)
    wl.params["sigma"] = 0.0
    g, o, _, _ = run_case(wl, "scan sigma0", variant=SCAN)
    np.testing.assert_allclose(g["weights"], 1.0 / 128, rtol=1e-6)
    np.testing.assert_array_equal(g["u_new"], wl.u_nom)
    assert np.ptp(g["cost"]) == 0.0
    wl = W.cfg0(K=256, N=12)
    wl.u_nom[:] = 7.0
    wl.params["lambda"] = float(np.float32(1e-4))
    g, o, _, _ = run_case(wl, "scan saturated", variant=SCAN)
    assert g["weights"][0, int(np.argmin(o["cost"][0]))] > 0.999
    # [R-41]: a third of the samples at the cost cap get weight 0, the update stays finite
    wl = W.stress_gate(K=2048, N=30)
    wl.params["gate_miss_penalty"] = 3.0e38
    m = Pz.make_ctx(wl, variant=SCAN)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    m.close()
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True)
    capped = o["cost"][0] == 3.0e38
    flagged = o["margin"][0] < Pz.MARGIN
    assert capped.mean() > 0.1 and np.isfinite(g["cost"]).all() and np.isfinite(g["u_new"]).all()
    assert (((g["cost"][0] == np.float32(3.0e38)) == capped)[~flagged]).all()
    assert (g["weights"][0][capped & ~flagged] == 0.0).all() and abs(g["weights"].sum() - 1.0) < 2e-5


def test_what_the_variant_rejects_and_what_auto_picks():
    from paper_2509_14726_b200 import binding as Bd
    wl = W.cfg0(K=256, N=20)
    for over in (dict(Jy=np.float32(1.2e-3)), dict(N=65), dict(pipeline=1), dict(block_threads=64)):
        with pytest.raises(Bd.MppiError) as e:
            Bd.Mppi(wl.params, variant=SCAN, **over)
        assert e.value.status == -2, over                                 # MPPI_E_PARAM
    for make in (W.cfg2, W.cfg3, W.rate_gate_paper):
        with pytest.raises(Bd.MppiError) as e:
            Bd.Mppi(make().params, variant=SCAN)
        assert e.value.status == -2
    # AUTO: the lone gate-progress controller goes to this kernel, a batch that needs more than one wave of its
    # blocks does not, nor does an airframe with Jx != Jy (its body-rate equations are not linear in omega_xy)
    m = Pz.make_ctx(W.cfg1()); info = m.info(); m.close()
    assert info["rollout_warps_per_block"] == 16
    m = Pz.make_ctx(W.cfg4(B=2)); info = m.info(); m.close()
    assert info["rollout_warps_per_block"] != 16
    wl = W.cfg1(); wl.params["Jy"] = np.float32(1.3e-3)
    m = Pz.make_ctx(wl); info = m.info(); m.close()
    assert info["rollout_warps_per_block"] != 16


def test_run_to_run_determinism_and_host_entry():
    import torch
    wl = W.cfg1()
    m = Pz.make_ctx(wl, variant=SCAN, fast_math=1)
    x0, start, u = Pz.to_dev(wl)
    a = Pz.gpu_step(m, x0, start, u, 3, 11)
    for _ in range(5):
        b = Pz.gpu_step(m, x0, start, u, 3, 11)
        for key in ("u_new", "cost", "weights"):
            np.testing.assert_array_equal(a[key], b[key])
    h = m.step_host(wl.x0, wl.start, wl.u_nom, 3, 11)
    np.testing.assert_array_equal(h[0], a["u_new"])
    m.close()


@pytest.mark.parametrize("fuzz_seed", [1, 2, 3])
def test_random_tracks_states_and_sizes(fuzz_seed):
    # seeded fuzz over what the kernel's special handling depends on: the number of gates (1: the target index never
    # changes value; 2, 3: it wraps inside a horizon), gates in a row at random spacing so that chunks hold zero to
    # several passes, random start index, speed, spin and attitude, horizons 1 .. 64, block sizes from K and B, both gate
    # objectives with random flags and both readings of the near term, both math modes, sigma from small to large
    rng = np.random.default_rng(1000 + fuzz_seed)
    crossed, multi = 0, 0
    for case in range(14):
        obj = int(rng.choice([0, 3]))
        K = int(rng.choice([32, 64, 160, 256, 512, 1024])); N = int(rng.integers(1, 65)); B = int(rng.integers(1, 4))
        G = int(rng.choice([1, 2, 3, 5, 8]))
        wl = W.stress_gate(K=K, N=N)
        gates = np.zeros((G, 11), np.float32)
        gates[:, 0] = 1.0 + np.cumsum(rng.uniform(0.6, 2.2, G)); gates[:, 1] = rng.uniform(-0.15, 0.15, G); gates[:, 2] = 2.0 + rng.uniform(-0.15, 0.15, G)
        gates[:, 3] = 1.0; gates[:, 7] = 1.0; gates[:, 9] = rng.uniform(0.7, 1.2, G); gates[:, 10] = rng.uniform(0.6, 1.0, G)
        wl.gates = gates
        x0 = np.zeros((1, 13), np.float32)
        x0[0, 0:3] = [0.0, rng.uniform(-0.3, 0.3), 2.0 + rng.uniform(-0.3, 0.3)]
        q = np.array([1.0, 0, 0, 0]) + rng.normal(0, 0.05, 4); x0[0, 3:7] = q / np.linalg.norm(q)
        x0[0, 7:10] = [rng.uniform(2.0, 12.0), rng.normal(0, 0.5), rng.normal(0, 0.5)]
        x0[0, 10:13] = rng.normal(0, 3.0, 3)
        wl.x0 = x0
        wl.start[:] = 0 if rng.uniform() < 0.7 else int(rng.integers(-3, 12))
        wl.params["sigma"] = np.float32(rng.choice([0.3, 1.0, 2.5]))
        wl.params["lambda"] = np.float32(rng.choice([0.05, 0.5, 5.0]))
        if obj == 3:
            wl.params.update(objective=3, q_near=np.float32(2.0), r_near=np.float32(1.5), near_mode=int(rng.integers(0, 2)))
            wl.prev_front = (rng.uniform(size=(1, N + 1)) < 0.6).astype(np.int32)
        if B > 1:
            wl = W.replicate(wl, B, 0.2)
        math = int(rng.integers(0, 2))
        tag = f"scan fuzz {fuzz_seed}/{case}: obj {obj} K {K} N {N} B {B} G {G} math {math}"
        g, o, st, _ = run_case(wl, tag, it=case, variant=SCAN, fast_math=math)
        crossed += int((o["ncross"] >= 1).sum()); multi += int((o["ncross"] >= 2).sum())
    assert crossed > 1000 and multi > 100, (crossed, multi)       # the re-scoring rounds really ran
