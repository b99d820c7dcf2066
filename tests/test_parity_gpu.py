"""GPU parity: the CUDA path behind the C ABI against the float64 oracle, element by element, on
the same seeded inputs -- the five BASELINE.json configs at full size in the launch configuration
bench.py times, plus stress, ragged and degenerate cases.  Tolerances: tests/parity.py."""
import numpy as np
import pytest

import parity as Pz
from paper_2509_14726_b200 import workloads as W

pytestmark = pytest.mark.gpu


def run_case(wl, tag, it=0, **opts):
    m = Pz.make_ctx(wl, **opts)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, it)
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, it, want_du=wl.params["K"] * wl.params["N"] * wl.params["B"] <= 1 << 22)
    o["u_nom"] = wl.u_nom.astype(np.float64)
    st = Pz.compare(tag, g, o, wl.params["lambda"], wl.params["objective"] == 0)
    m.close()
    return g, o, st


# fused pipeline with the latency / scalar throughput / packed fp32x2 throughput kernels; two-pass
# pipeline with the packed (AUTO picks it when K % 64 == 0) and the scalar rollout kernel
PIPES = [dict(pipeline=0, variant=4), dict(pipeline=0, variant=2), dict(pipeline=0, variant=1), dict(pipeline=0, variant=3),
         dict(pipeline=1), dict(pipeline=1, variant=1)]
PIPE_IDS = ["fused_pipe", "fused_lat", "fused_thr", "fused_pk", "two_pass", "two_pass_thr"]
MATH = [dict(fast_math=0), dict(fast_math=1)]


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_cfg0_tiny_gate(pipe, math):
    g, o, st = run_case(W.cfg0(), f"cfg0[{pipe},{math}]", **pipe, **math)
    assert st["ess"] > 1.5            # the config really mixes several samples


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_cfg1_ten_warm_started_iterations(pipe):
    # [R-14] no shift, same x0, u_nom <- u_new, iter = 0..9; the oracle is teacher-forced with the
    # GPU's nominal of each iteration (fp32 -> fp64) so that every iteration is an exact comparison
    import torch
    wl = W.cfg1()
    m = Pz.make_ctx(wl, **pipe)
    x0, start, u = Pz.to_dev(wl)
    crossings = 0
    for it in range(wl.iters):
        u_in = u.cpu().numpy()
        g = Pz.gpu_step(m, x0, start, u, wl.seed, it, u_new=u)          # in place
        o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, it, want_du=True)
        o["u_nom"] = u_in.astype(np.float64)
        Pz.compare(f"cfg1[{pipe}] it{it}", g, o, wl.params["lambda"], True)
        crossings += int((o["ncross"] > 0).sum())
        np.testing.assert_array_equal(u.cpu().numpy(), g["u_new"])
    assert crossings > 0
    m.close()


def test_cfg1_optimize_graph_equals_step_chain():
    import torch
    wl = W.cfg1()
    x0, start, u0 = Pz.to_dev(wl)
    m = Pz.make_ctx(wl)
    u = u0.clone()
    for it in range(wl.iters):
        _, c_ref, w_ref = m.step(x0, start, u, wl.seed, it, u_new=u)
    for graph in (0, 1):
        m2 = Pz.make_ctx(wl, use_graph=graph)
        for rep in range(2):                       # second replay goes through SetParams
            u2 = u0.clone()
            _, c2, w2 = m2.optimize(x0, start, u2, wl.seed, 0, wl.iters)
            torch.cuda.synchronize()
            assert torch.equal(u2, u) and torch.equal(c2, c_ref) and torch.equal(w2, w_ref)
        m2.close()
    m.close()


@pytest.mark.parametrize("name,B", [("cfg1", 1), ("cfg2", 1), ("gate_paper", 2), ("stress_gate", 3)])
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_optimize_chain_by_programmatic_dependent_launch_equals_the_steps(name, B, math):
    # mppi_optimize without a graph chains the pipelined kernel's iterations by programmatic dependent launch: iteration
    # i + 1 starts while iteration i publishes and combines, draws the state-independent half of its noise, then waits
    # before it reads the nominal.  Must equal the chain of single steps bit for bit, repeatedly (a race would show as a
    # run-to-run difference), and the last iteration must match the oracle fed with the chain's own nominal.
    import torch
    wl = W.replicate(W.ALL[name](), B, 0.2) if B > 1 else W.ALL[name]()
    x0, start, u0 = Pz.to_dev(wl)
    m = Pz.make_ctx(wl, variant=4, **math)
    u = u0.clone()
    n = 6
    for it in range(n):
        if it == n - 1:
            u_in = u.cpu().numpy()
        _, c_ref, w_ref = m.step(x0, start, u, wl.seed, it, u_new=u)
    torch.cuda.synchronize()
    for rep in range(5):
        u2 = u0.clone()
        _, c2, w2 = m.optimize(x0, start, u2, wl.seed, 0, n)
        torch.cuda.synchronize()
        assert torch.equal(u2, u) and torch.equal(c2, c_ref) and torch.equal(w2, w_ref), rep
    o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, n - 1, want_du=True)
    g = dict(u_new=u2.cpu().numpy(), cost=c2.cpu().numpy(), weights=w2.cpu().numpy())
    Pz.compare(f"optimize chain (PDL) {name} B{B} {math}", g, o, wl.params["lambda"], wl.params["objective"] in (0, 3))
    m.close()


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_cfg2_tracking(pipe, math):
    run_case(W.cfg2(), f"cfg2[{pipe},{math}]", **pipe, **math)


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_cfg3_contouring(pipe, math):
    run_case(W.cfg3(), f"cfg3[{pipe},{math}]", **pipe, **math)


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_stress_gate_crossings(pipe, math):
    wl = W.stress_gate(K=4096, N=30)
    g, o, st = run_case(wl, f"stress[{pipe},{math}]", **pipe, **math)
    nc = o["ncross"]
    assert (nc > 0).mean() > 0.3 and (nc == 0).mean() > 0.1      # pass and miss branches both taken


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
@pytest.mark.parametrize("name", ["stress_gate", "cfg2"])
def test_asymmetric_inertia(name, pipe):
    # Jx != Jy: the yaw-rate derivative gets its gyroscopic term (the packed kernel then leaves its
    # symmetric-airframe short-cut, rk4_step2<false>); every kernel against the oracle, fast math
    wl = W.stress_gate(K=4096, N=30) if name == "stress_gate" else W.cfg2()
    wl.params.update(Jx=1.0e-3, Jy=1.6e-3, Jz=2.1e-3)
    g, o, st = run_case(wl, f"asym_{name}[{pipe}]", fast_math=1, **pipe)
    wl0 = W.stress_gate(K=4096, N=30) if name == "stress_gate" else W.cfg2()
    wl0.params.update(Jx=1.3e-3, Jy=1.3e-3, Jz=2.1e-3)
    o0 = Pz.oracle_step(wl0, wl0.x0, wl0.start, wl0.u_nom, wl0.seed, 0)
    assert (np.abs(o0["cost"] - o["cost"]) > 1e-3 * np.abs(o["cost"])).mean() > 0.5      # the asymmetry matters


def test_cfg4_closed_loop_teacher_forced():
    # [R-17] configs[4] as stated: 64 drones, 500 control steps, closed loop on the GPU (plant + shift kernel) --
    # the loop bench.py times.  At control step 0, every 50th and the last one the oracle gets the GPU loop's
    # actual (x, start, u_nom, iter) and is compared for that one step (iteration AND plant step).
    # With configs[4]'s sigma = 1.5 N, lambda = 0.5 the drones pass one gate and then lose height (DESIGN.md
    # section 10, "Finding"): the late checks compare rollouts from states far below the track.
    import torch
    from oracle import oracle as O
    wl = W.cfg4()
    assert wl.iters == 500
    m = Pz.make_ctx(wl)
    x, start, u = Pz.to_dev(wl)
    trk = Pz.oracle_track(wl)
    checked, passes = 0, np.zeros(wl.params["B"], np.int64)
    for step in range(wl.iters):
        check = step % 50 == 0 or step == wl.iters - 1
        if check:
            x_in, s_in, u_in = x.cpu().numpy(), start.cpu().numpy(), u.cpu().numpy()
        s_before = start.clone()
        u_new, cost, w = m.step(x, start, u, wl.seed, step)
        if check:
            torch.cuda.synchronize()
            g = dict(u_new=u_new.cpu().numpy(), cost=cost.cpu().numpy(), weights=w.cpu().numpy())
            o = Pz.oracle_step(wl, x_in, s_in, u_in, wl.seed, step)
            Pz.compare(f"cfg4 step{step}", g, o, wl.params["lambda"], True)
            xo, so, uo = O.sim_step(wl.params, trk, x_in, s_in, g["u_new"])
        m.sim_step(x, start, u_new, u_nom_next=u)
        passes += (start != s_before).cpu().numpy()
        if check:
            torch.cuda.synchronize()
            np.testing.assert_allclose(x.cpu().numpy(), xo, rtol=3e-6, atol=2e-5)
            np.testing.assert_array_equal(u.cpu().numpy(), uo.astype(np.float32))
            # the plant's gate decision may differ only if the plant sat within the margin
            assert (start.cpu().numpy() == so).mean() >= 0.98
            checked += 1
    assert checked == 11
    assert passes.max() >= 1            # the loop really flies through gates
    Pz.STATS.append(f"cfg4 closed loop, 500 control steps: gate passes per drone min {passes.min()} / median "
                    f"{int(np.median(passes))} / max {passes.max()}; final height min {float(x[:, 2].min()):.1f} m")
    m.close()


def _sim_step_case(kind, rate):
    """B drones whose start indices / positions exercise every branch of mppi_sim_step under tracking and
    search-contouring (include/mppi.h: mppi_sim_step; Alg. 1 l.2-3 PAPER.md:177-178)."""
    K, N = 256, 20
    if kind == "track":
        base = W.cfg2(K=K, N=N, extra_rows=3)                 # M = N + 1 + 3: the start row clamps at 3
        B = 4
        wl = W.replicate(base, B, 0.2)
        wl.start = np.array([0, 1, 3, 7], np.int32)           # advances, advances, stays clamped, pulled back
    else:
        base = W.cfg3(K=K, N=N)
        pts = base.path.astype(np.float64)
        P = len(pts)
        spec = [(P - 3, P - 3, 8.0), (P - 3, -1, 8.0), (100, 100, 5.0), (100, 80, 5.0), (100, -1, 0.0), (250, 255, 3.0)]
        B = len(spec)
        wl = W.replicate(base, B, 0.0)
        for b, (at, hint, speed) in enumerate(spec):          # next to vertex `at`, flying along the path
            tan = pts[(at + 1) % P] - pts[(at - 1) % P]; tan /= np.linalg.norm(tan)
            wl.x0[b, 0:3] = (pts[at] + np.array([0.05, -0.03, 0.04])).astype(np.float32)
            wl.x0[b, 7:10] = (speed * tan).astype(np.float32)
            wl.start[b] = hint
    if rate:
        wl = W._rate_model(wl, wl.name + "_rate")
    return wl


@pytest.mark.parametrize("rate", [0, 1], ids=["thrusts", "rate_model"])
@pytest.mark.parametrize("kind", ["track", "contour"])
def test_sim_step_tracking_and_contouring_match_the_oracle(kind, rate):
    # the closed-loop glue under objectives 1 and 2, both input models: every control step of a short loop is
    # compared with orc_sim_step from the GPU loop's own inputs [R-17] -- plant state, start index (tracking:
    # +1 clamped at M - 1 - N; contouring: windowed / global nearest vertex incl. the seam), shifted nominal
    import torch
    from oracle import oracle as O
    wl = _sim_step_case(kind, rate)
    p = wl.params
    m = Pz.make_ctx(wl)
    x, start, u = Pz.to_dev(wl)
    trk = Pz.oracle_track(wl)
    pts = None if wl.path is None else wl.path.astype(np.float64)
    seen = []
    for step in range(6):
        x_in, s_in, u_in = x.cpu().numpy(), start.cpu().numpy(), u.cpu().numpy()
        g = Pz.gpu_step(m, x, start, u, wl.seed, step)
        o = Pz.oracle_step(wl, x_in, s_in, u_in, wl.seed, step, want_du=True)
        Pz.compare(f"sim {kind} rate{rate} step{step}", g, o, p["lambda"], False)
        xo, so, uo = O.sim_step(p, trk, x_in, s_in, g["u_new"])
        m.sim_step(x, start, torch.from_numpy(g["u_new"]).cuda(), u_nom_next=u); torch.cuda.synchronize()
        np.testing.assert_allclose(x.cpu().numpy(), xo, rtol=3e-6, atol=2e-5)
        np.testing.assert_array_equal(u.cpu().numpy(), uo.astype(np.float32))
        sg = start.cpu().numpy()
        if kind == "track":
            np.testing.assert_array_equal(sg, so)
        else:
            for b in np.nonzero(sg != so)[0]:             # only an fp32-unresolvable tie may pick the other vertex
                da, db = (np.sum((xo[b, 0:3] - pts[i]) ** 2) for i in (sg[b], so[b]))
                assert abs(da - db) <= 1e-5 * max(da, db), (step, b, sg[b], so[b])
        seen.append(sg.copy())
    seen = np.array(seen)
    if kind == "track":
        np.testing.assert_array_equal(seen[:, 0], [1, 2, 3, 3, 3, 3])
        np.testing.assert_array_equal(seen[-1], [3, 3, 3, 3])
    else:
        P = len(pts)
        assert seen[-1, 0] < 50 and seen[-1, 1] < 50          # crossed the seam (started at P - 3)
        assert seen[0, 3] <= 96                               # hint 80: the window 64..96 does not reach vertex ~100
        assert abs(int(seen[0, 4]) - 100) <= 1                # global search finds it
    m.close()


# ---- the reduction arithmetic with many contributing samples (ESS >> 1) -------------------------

@pytest.mark.parametrize("name", ["cfg1", "cfg2", "cfg3"])
@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_flat_weights_exercise_the_update(name, pipe):
    wl = W.ALL[name](K=2048, N=50)
    o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    wl.params["lambda"] = float(np.float32(0.25 * o0["cost"].std()))
    g, o, st = run_case(wl, f"flat-{name}[{pipe}]", **pipe)
    assert st["ess"] > 20
    assert st["w"] <= Pz.W_ATOL and st["u"] <= Pz.U_ATOL


@pytest.mark.parametrize("name", ["cfg1", "cfg2", "rate_gate_paper", "rate_track"])
@pytest.mark.parametrize("opts", [dict(variant=3), dict(variant=1), dict(variant=3, store_noise=1), dict(variant=1, store_noise=1, block_threads=64)],
                         ids=["packed_adaptive", "scalar_adaptive", "packed_stored", "scalar_stored"])
def test_mixing_weights_dense_update_from_stored_noise(name, opts):
    # eq.(5) PAPER.md:91-95 when MANY samples carry weight: the fused throughput kernels then keep dU and sum it from
    # memory (mppi_rollout.cuh, warp_noise_partial) instead of re-deriving the noise.  store_noise = 1 takes that path
    # from the first iteration on; otherwise the previous iteration's combine switches it on (StepArgs::hint), so
    # iteration 0 re-derives and iterations 1, 2 read back.  All must meet the strict bounds.  N = 37 leaves a ragged
    # last group of the eight-step butterfly, B = 3 checks the per-controller hint.
    wl = W.replicate(W.ALL[name](K=1024, N=37), 3, 0.2)
    o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    wl.params["lambda"] = float(np.float32(0.25 * np.median(o0["cost"].std(-1))))
    m = Pz.make_ctx(wl, **opts)
    x0, start, u = Pz.to_dev(wl)
    for it in range(3):
        u_in = u.cpu().numpy()
        g = Pz.gpu_step(m, x0, start, u, wl.seed, it, u_new=u)        # warm start in place
        o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, it, want_du=True)
        st = Pz.compare(f"mixing-{name}[{opts}] it{it}", g, o, wl.params["lambda"], False)
        assert st["ess"] > 20
        assert st["w"] <= Pz.W_ATOL and st["u"] <= Pz.U_ATOL
    m.close()


def test_noise_matches_oracle_and_pipelines_agree():
    import torch
    wl = W.cfg0(K=512, N=37)
    outs = {}
    # "fused" names the pipelined kernel: under AUTO this shape now goes to the time-parallel kernel (variant 5), whose
    # states equal the others' to rounding only (another association order of the same RK4: mppi_scan.cuh); its noise
    # is the same stream bit for bit, its costs are compared below with a tolerance
    for name, opts in dict(fused=dict(pipeline=0, variant=4, store_noise=1), two=dict(pipeline=1),
                           thr=dict(pipeline=0, variant=1, store_noise=1),
                           pk=dict(pipeline=0, variant=3, store_noise=1),
                           scan=dict(pipeline=0, variant=5, store_noise=1)).items():
        m = Pz.make_ctx(wl, **opts)
        x0, start, u = Pz.to_dev(wl)
        outs[name] = Pz.gpu_step(m, x0, start, u, 5, 7)
        outs[name]["du"] = m.debug_noise().cpu().numpy()      # [B,N,K,4]
        m.close()
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, 5, 7, want_du=True)
    du_o = np.transpose(o["du"], (0, 2, 1, 3))
    np.testing.assert_allclose(outs["fused"]["du"], du_o, rtol=0, atol=3e-6)
    np.testing.assert_array_equal(outs["fused"]["du"], outs["two"]["du"])
    np.testing.assert_array_equal(outs["scan"]["du"], outs["two"]["du"])
    np.testing.assert_allclose(outs["scan"]["cost"], outs["two"]["cost"], rtol=2e-5, atol=2e-5)
    np.testing.assert_allclose(outs["scan"]["weights"], outs["two"]["weights"], rtol=0, atol=1e-5)
    np.testing.assert_allclose(outs["scan"]["u_new"], outs["two"]["u_new"], rtol=0, atol=1e-4)
    # the packed fp32x2 kernel performs, per half, the scalar kernel's operations in the same order
    for key in ("du", "cost"):
        np.testing.assert_array_equal(outs["thr"][key], outs["pk"][key])
    # (the update is summed over differently shaped blocks: equal up to the summation order)
    np.testing.assert_allclose(outs["thr"]["weights"], outs["pk"]["weights"], rtol=0, atol=2e-6)
    np.testing.assert_allclose(outs["thr"]["u_new"], outs["pk"]["u_new"], rtol=0, atol=2e-5)
    np.testing.assert_array_equal(outs["fused"]["cost"], outs["two"]["cost"])
    np.testing.assert_allclose(outs["fused"]["weights"], outs["two"]["weights"], rtol=0, atol=2e-6)
    np.testing.assert_allclose(outs["fused"]["u_new"], outs["two"]["u_new"], rtol=0, atol=2e-5)
    # clamp really acts: some perturbations are cut at the thrust limits
    T = wl.u_nom[:, :, None, :] + outs["fused"]["du"]
    assert T.min() >= 0.0 and T.max() <= 7.0 and (T == 0.0).any()
    m = Pz.make_ctx(wl)
    assert m.debug_noise() is None
    m.close()


@pytest.mark.parametrize("K,N,B,consumers", [(32, 1, 1, 1), (64, 33, 1, 1), (4096, 50, 1, 1), (8192, 50, 1, 2),
                                             (16384, 20, 1, 4), (512, 20, 3, 1), (4096, 256, 1, 1), (96, 7, 1, 1)])
def test_latency_variant_shapes(K, N, B, consumers):
    # the warp-specialised kernel: C rollout warps per 256-thread block, C picked from the grid size
    wl = W.cfg4(K=K, N=N, B=B) if B > 1 else W.stress_gate(K=K, N=N)
    m = Pz.make_ctx(wl, variant=2)
    info = m.info()
    assert info["block_threads"] == 256 and info["blocks_per_controller"] == K // (32 * consumers)
    m.close()
    run_case(wl, f"lat K{K} N{N} B{B}", variant=2)
    # the pipelined kernel (three warps per rollout): always 32 samples per 256-thread block
    m = Pz.make_ctx(wl, variant=4)
    info = m.info()
    assert info["block_threads"] == 256 and info["blocks_per_controller"] == K // 32
    m.close()
    run_case(wl, f"pipe K{K} N{N} B{B}", variant=4)


# ---- ragged / degenerate / maximum sizes ----------------------------------------------------------

@pytest.mark.parametrize("K,N,tpb", [(32, 1, 32), (32, 33, 32), (64, 20, 64), (96, 7, 32), (256, 256, 256),
                                     (1024, 64, 128), (8192, 50, 256)])
@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_sizes_and_block_shapes(K, N, tpb, pipe):
    wl = W.stress_gate(K=K, N=N)
    if pipe.get("variant") == 3 and (K % (2 * tpb) != 0 or tpb > 128):
        from paper_2509_14726_b200 import binding as Bd
        with pytest.raises(Bd.MppiError) as e:                 # two samples per thread: tpb <= 128, 2*tpb divides K
            Pz.make_ctx(wl, block_threads=tpb, **pipe)
        assert e.value.status == -2
        return
    run_case(wl, f"sizes K{K} N{N} tpb{tpb} [{pipe}]", block_threads=tpb, **pipe)


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_sigma_zero_is_uniform(pipe):
    wl = W.cfg0(K=128, N=10)
    wl.params["sigma"] = 0.0
    g, o, _ = run_case(wl, f"sigma0[{pipe}]", **pipe)
    np.testing.assert_allclose(g["weights"], 1.0 / 128, rtol=1e-6)
    np.testing.assert_array_equal(g["u_new"], wl.u_nom)
    assert np.ptp(g["cost"]) == 0.0


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_saturated_nominal_and_tiny_lambda(pipe):
    wl = W.cfg0(K=256, N=12)
    wl.u_nom[:] = 7.0
    wl.params["lambda"] = float(np.float32(1e-4))
    g, o, _ = run_case(wl, f"saturated[{pipe}]", **pipe)
    k = int(np.argmin(o["cost"][0]))
    assert g["weights"][0, k] > 0.999                       # lambda -> 0: the arg-min sample
    assert g["u_new"].max() <= 7.0 and g["u_new"].min() >= 0.0


def test_multi_controller_batches_are_independent():
    # B = 3 controllers with different states, starts and nominals; controller b of the batch
    # equals a B = 1 run given the same counter word b -> checked against the oracle per b
    wl = W.cfg4(K=512, N=20, B=3)
    wl.start[:] = [0, 2, 3]
    wl.u_nom[1] += 0.2
    run_case(wl, "B3 gate", it=4)
    wl2 = W.cfg2(K=256, N=16, extra_rows=8)
    wl2.params["B"] = 2
    wl2.x0 = np.repeat(wl2.x0, 2, 0); wl2.x0[1, 0:3] += 0.1
    wl2.start = np.array([0, 5], np.int32)
    wl2.u_nom = np.repeat(wl2.u_nom, 2, 0)
    run_case(wl2, "B2 track")


def test_contour_hint_and_open_path():
    wl = W.cfg3(K=512, N=30)
    run_case(wl, "contour global")
    wl.start[:] = 470                                      # windowed search around a hint
    run_case(wl, "contour hint")
    wl.closed = False                                      # open path: no wrap, clipped window
    wl.start[:] = -1
    run_case(wl, "contour open")
    wl.x0[0, 0:3] = wl.path[3] + np.float32([0.05, 0.0, 0.02])
    wl.start[:] = 2
    run_case(wl, "contour open near start")


@pytest.mark.parametrize("pipe", [dict(pipeline=0, variant=2), dict(pipeline=0, variant=3), dict(pipeline=0, variant=1),
                                  dict(pipeline=1)], ids=["fused_lat", "fused_pk", "fused_thr", "two_pass"])
@pytest.mark.parametrize("window,closed,near_end", [(5, True, True), (40, True, False), (7, False, True), (16, False, True)])
def test_contour_window_sizes(window, closed, near_end, pipe):
    # the search runs on the padded copy of the points: windows other than the unrolled default (16),
    # wrap-around of a closed path and the clipped window at both ends of an open one
    wl = W.cfg3(K=1024, N=30)
    wl.params["window"] = window
    wl.closed = closed
    if near_end:                      # start next to the seam / the end: the window reaches past index P - 1
        wl.x0[0, 0:3] = wl.path[-2] + np.float32([0.03, -0.02, 0.01])
        wl.start[:] = wl.path.shape[0] - 3
    run_case(wl, f"contour W{window} closed{closed} [{pipe}]", fast_math=1, **pipe)


def test_determinism_and_host_entry_point():
    import torch
    wl = W.stress_gate(K=1024, N=30)
    for opts in PIPES:
        m = Pz.make_ctx(wl, **opts)
        x0, start, u = Pz.to_dev(wl)
        a = Pz.gpu_step(m, x0, start, u, 9, 1)
        b = Pz.gpu_step(m, x0, start, u, 9, 1)
        for k in a:
            np.testing.assert_array_equal(a[k], b[k])
        c = Pz.gpu_step(m, x0, start, u, 9, 2)
        assert not np.array_equal(a["cost"], c["cost"])     # iter feeds the counter
        d = Pz.gpu_step(m, x0, start, u, 10, 1)
        assert not np.array_equal(a["cost"], d["cost"])     # seed feeds the key
        un, co, we = m.step_host(wl.x0, wl.start, wl.u_nom, 9, 1)
        np.testing.assert_array_equal(un, a["u_new"]); np.testing.assert_array_equal(co, a["cost"])
        np.testing.assert_array_equal(we, a["weights"])
        # the pre-marshalled form of the same call, with and without the optional outputs
        un2, co2 = np.empty_like(un), np.empty_like(co)
        m.step_host_fn(wl.x0, wl.start, wl.u_nom, un2, cost=co2)(9, 1)
        np.testing.assert_array_equal(un2, un); np.testing.assert_array_equal(co2, co)
        un3 = np.empty_like(un)
        m.step_host_fn(wl.x0, wl.start, wl.u_nom, un3)(9, 1)
        np.testing.assert_array_equal(un3, un)
        assert m.launch_count() == (7 if opts["pipeline"] == 0 else 14)
        m.close()


@pytest.mark.parametrize("case", ["contour_max_path_max_horizon", "track_max_horizon_many_samples", "gate_max_horizon"])
def test_auto_falls_back_when_the_latency_kernels_do_not_fit(case):
    # AUTO picks the pipelined / latency kernel from the warp count alone, before the track is known; at the limits of
    # include/mppi.h (MPPI_MAX_N = 256, MPPI_MAX_PATH = 2048) their rings / thrust tables do not fit in 227 KB of
    # shared memory beside the track.  The first step must then move to a kernel that fits instead of failing.
    if case == "contour_max_path_max_horizon":
        wl = W.cfg3(K=4096, N=256)
        a = 2 * np.pi * np.arange(2048) / 2048
        wl.path = np.stack([5 * np.cos(a), 5 * np.sin(a), 1.5 + 0.2 * np.sin(3 * a)], 1).astype(np.float32)
    elif case == "track_max_horizon_many_samples":
        wl = W.cfg2(K=16384, N=256)
    else:
        wl = W.cfg1(K=2048, N=256)
    wl.params["sigma"] = float(np.float32(0.3))
    wl.params["dt"] = float(np.float32(0.005))             # 256 steps = 1.28 s of horizon (at 0.02 s the fp32 error of 5 s of free flight is the test)
    m = Pz.make_ctx(wl)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    info = m.info()
    assert info["dynamic_smem_bytes"] <= 227 * 1024
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True)
    Pz.compare(f"auto fallback {case} ({info['block_threads']} thr x {info['grid_blocks']})", g, o, wl.params["lambda"],
               wl.params["objective"] == 0)
    m.close()
    # an explicit request for a kernel that does not fit still fails cleanly
    if case != "gate_max_horizon":
        from paper_2509_14726_b200 import binding as Bd
        m = Pz.make_ctx(wl, variant=2 if case.startswith("contour") else 4)
        with pytest.raises(Bd.MppiError) as e:
            m.step(x0, start, u, wl.seed, 0)
        assert e.value.status == -2
        m.close()


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_diverged_samples_get_no_weight(pipe):
    # [R-41] a sample whose cost is not representable (here: a miss penalty of 3e38 on a third of the samples) is
    # reported as 3.0e38 and gets weight 0; the others are untouched and the update stays finite
    wl = W.stress_gate(K=2048, N=30)
    wl.params["gate_miss_penalty"] = 3.0e38
    m = Pz.make_ctx(wl, **pipe)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    m.close()
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True)
    capped = o["cost"][0] == 3.0e38
    assert capped.mean() > 0.1 and (~capped).mean() > 0.1
    flagged = o["margin"][0] < Pz.MARGIN
    assert np.isfinite(g["cost"]).all() and np.isfinite(g["u_new"]).all() and np.isfinite(g["weights"]).all()
    same = (g["cost"][0] == np.float32(3.0e38)) == capped
    assert same[~flagged].all()
    assert (g["weights"][0][capped & ~flagged] == 0.0).all()
    ok = ~capped & ~flagged
    assert (np.abs(g["cost"][0][ok] - o["cost"][0][ok]) <= 1e-4 * np.maximum(np.abs(o["cost"][0][ok]), 1.0)).all()
    assert abs(g["weights"].sum() - 1.0) < 2e-5
    if not flagged.any():
        assert np.abs(g["u_new"] - o["u_new"]).max() <= Pz.U_ATOL


def test_rate_model_divergent_rollouts_stay_finite():
    # sigma = 60 N/s on the thrust rates: the explicit RK4 itself diverges on the tumbling samples (DESIGN.md section
    # 10): fp32 costs overflow to Inf and Inf - Inf.  Outputs must stay finite, weights normalised, u_new in range
    wl = W.rate_stress(K=2048, N=50)
    wl.params.update(sigma=float(np.float32(60.0)), rate_max=float(np.float32(100.0)))
    for opts in (dict(variant=1), dict(variant=3), dict(variant=4), dict(pipeline=1)):
        m = Pz.make_ctx(wl, **opts)
        x0, start, u = Pz.to_dev(wl)
        g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
        m.close()
        assert np.isfinite(g["cost"]).all() and np.isfinite(g["weights"]).all() and np.isfinite(g["u_new"]).all(), opts
        assert abs(g["weights"].sum() - 1.0) < 2e-5 and np.abs(g["u_new"]).max() <= 100.0
        assert (g["cost"] == np.float32(3.0e38)).any(), "the case is meant to contain diverged samples"


@pytest.mark.parametrize("opts", [dict(variant=4), dict(variant=1, block_threads=32), dict(variant=3, block_threads=32)],
                         ids=["pipelined_512_blocks", "scalar_512_blocks", "packed_256_blocks"])
@pytest.mark.parametrize("mixing", [False, True], ids=["lambda_as_stated", "mixing"])
def test_many_blocks_per_controller(opts, mixing):
    # more than 256 partials per controller take the block-wide form of the last-block combine (the per-warp form
    # keeps at most eight (m, Z) pairs per lane); exactly 256 is its boundary
    wl = W.replicate(W.cfg1(K=16384, N=10), 2, 0.2)
    if mixing:
        o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
        wl.params["lambda"] = float(np.float32(0.25 * np.median(o0["cost"].std(-1))))
    g, o, st = run_case(wl, f"many blocks [{opts}, mixing {mixing}]", **opts)
    if mixing:
        assert st["ess"] > 100 and st["w"] <= Pz.W_ATOL and st["u"] <= Pz.U_ATOL


@pytest.mark.parametrize("sweep_seed", [20251105, 7, 99])
def test_random_small_configurations_against_the_oracle(sweep_seed):
    # seeded sweep over objective x input model x sizes x kernel variant x pipeline x math mode: every combination the
    # library accepts must match the oracle; what it rejects must be rejected with MPPI_E_PARAM, not run wrongly
    from paper_2509_14726_b200 import binding as Bd
    rng = np.random.default_rng(sweep_seed)
    ran, rejected = 0, 0
    for case in range(60):
        obj = int(rng.integers(0, 4))
        rate = int(rng.integers(0, 2))
        K = int(rng.choice([32, 64, 96, 128, 256, 512]))
        N = int(rng.integers(1, 41))
        B = int(rng.integers(1, 4))
        make = (W.stress_gate, W.cfg2, W.cfg3, W.stress_gate_paper)[obj]
        wl = make(K=K, N=N)
        if obj == 3:
            wl.params["near_mode"] = int(rng.integers(0, 2))
        if rate:
            wl = W._rate_model(wl, wl.name + "_rate")
        wl = W.replicate(wl, B, 0.2)
        if obj == 2:
            wl.start[:] = rng.integers(-1, 500, B)               # hint or global search
        opts = dict(variant=int(rng.choice([0, 1, 2, 3, 4, 5])), pipeline=int(rng.integers(0, 2)), fast_math=int(rng.integers(0, 2)))
        if rng.integers(0, 3) == 0:
            opts["block_threads"] = int(rng.choice([32, 64, 128]))
        tag = f"random case {sweep_seed}/{case}: obj {obj} rate {rate} K {K} N {N} B {B} {opts}"
        try:
            m = Pz.make_ctx(wl, **opts)
            x0, start, u = Pz.to_dev(wl)
            g = Pz.gpu_step(m, x0, start, u, wl.seed, case)
        except Bd.MppiError as e:
            assert e.status == -2, tag                           # MPPI_E_PARAM: an unsupported combination
            rejected += 1
            continue
        o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, case, want_du=True)
        Pz.compare(tag, g, o, wl.params["lambda"], obj in (0, 3))
        m.close()
        ran += 1
    assert ran >= 25 and rejected >= 3, (ran, rejected)        # (variant 5 takes the gate objective with thrust inputs only)


def test_seed_high_word_reaches_the_key():
    wl = W.cfg0(K=64, N=5)
    wl.seed = (0xDEADBEEF << 32) | 0x12345678
    run_case(wl, "64-bit seed", it=0xFFFFFFFF)


def test_error_paths_on_device():
    import torch
    from paper_2509_14726_b200 import binding as Bd
    wl = W.cfg0(K=64, N=8)
    m = Bd.Mppi(wl.params)
    x0, start, u = Pz.to_dev(wl)
    with pytest.raises(Bd.MppiError) as e:
        m.step(x0, start, u, 0, 0)
    assert e.value.status == -3                                           # MPPI_E_NO_TRACK
    bad = wl.gates.copy(); bad[0, 3:6] *= 1.01
    with pytest.raises(Bd.MppiError) as e:
        m.set_gates(bad)
    assert e.value.status == -4                                           # MPPI_E_TRACK
    m.set_gates(wl.gates)
    buf = torch.zeros(2 * u.numel(), device="cuda")
    a = buf[: u.numel()].view_as(u); b = buf[4: 4 + u.numel()].view_as(u)
    with pytest.raises(Bd.MppiError) as e:
        m.step(x0, start, a, 0, 0, u_new=b)
    assert e.value.status == -5                                           # MPPI_E_RANGE
    with pytest.raises(ValueError):
        m.step(x0, start, u.double(), 0, 0)
    m.close()
    m = Bd.Mppi(W.cfg2(K=64, N=8).params)
    with pytest.raises(Bd.MppiError) as e:
        m.set_reference(np.zeros((8, 13), np.float32))                    # M < N+1
    assert e.value.status == -4
    m.close()
    m = Bd.Mppi(W.cfg3(K=64, N=8).params)
    with pytest.raises(Bd.MppiError) as e:
        m.set_path(np.zeros((10, 3), np.float32))                         # P < 2 window + 1
    assert e.value.status == -4
    m.close()


# ---- the paper's own J_gate (eq.(6),(7) + temporal check), objective 3 ----------

@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
def test_gate_paper_objective(pipe, math):
    # configs[1] geometry, squared progress + Q_near term, no flags (all in front)
    g, o, st = run_case(W.gate_paper(), f"gate_paper[{pipe},{math}]", **pipe, **math)
    # the near term is active for a good share of the samples: their costs differ from pure progress
    wl = W.gate_paper(); wl.params["q_near"] = 0.0
    o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    assert (np.abs(o0["cost"] - o["cost"]) > 1e-3).mean() > 0.1


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_gate_paper_temporal_check_at_scale(pipe):
    # crossing-heavy case with random previous-iteration flags: registered passes, ignored passes and
    # misses all occur; the GPU must take every one of those decisions like the oracle
    wl = W.stress_gate_paper(K=4096, N=30)
    g, o, st = run_case(wl, f"stress_paper[{pipe}]", **pipe)
    wl_all = W.stress_gate_paper(K=4096, N=30); wl_all.prev_front = None
    o_all = Pz.oracle_step(wl_all, wl.x0, wl.start, wl.u_nom, wl.seed, 0)
    reg, geo = o["ncross"][0] > 0, o_all["ncross"][0] > 0
    assert reg.mean() > 0.1 and (geo & ~reg).mean() > 0.1
    # and the flags really change the GPU result
    m = Pz.make_ctx(wl_all, **pipe)
    x0, start, u = Pz.to_dev(wl_all)
    g_all = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    m.close()
    assert (np.abs(g_all["cost"] - g["cost"]) > 1.0).mean() > 0.1


@pytest.mark.parametrize("pipe", PIPES, ids=PIPE_IDS)
def test_gate_paper_near_mode_1(pipe):
    # eq.(7)'s near term measured against the horizon's START gate, before and after the switch [R-40]: the
    # crossing-heavy case (two thirds of the samples pass gate 0 and then sit within r_near BEHIND it) through
    # every kernel; the two readings must really differ on the samples that pass
    wl = W.stress_gate_paper(K=4096, N=30)
    wl.params["near_mode"] = 1
    g, o, st = run_case(wl, f"stress_paper near_mode 1 [{pipe}]", **pipe)
    o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, params=dict(wl.params, near_mode=0))
    passed = o["ncross"][0] > 0
    assert passed.mean() > 0.1 and (np.abs(o["cost"][0] - o0["cost"][0])[passed] > 1e-3).mean() > 0.5


@pytest.mark.parametrize("pipe", [dict(pipeline=0, variant=4), dict(pipeline=0, variant=1), dict(pipeline=0, variant=3), dict(pipeline=1)],
                         ids=["fused_pipe", "fused", "fused_pk", "two_pass"])
def test_gate_paper_near_mode_1_rate_model(pipe):
    wl = W._rate_model(W.stress_gate_paper(K=2048, N=30), "rate_stress_paper_near1", sigma=np.float32(12.0), rate_max=np.float32(20.0))
    wl.params["near_mode"] = 1
    g, o, st = run_case(wl, f"rate stress_paper near_mode 1 [{pipe}]", **pipe)
    o0 = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, params=dict(wl.params, near_mode=0))
    assert (np.abs(o["cost"][0] - o0["cost"][0]) > 1e-3).mean() > 0.1


@pytest.mark.parametrize("near_mode", [0, 1])
def test_front_flags_and_closed_loop_feed(near_mode):
    # the flags of the new nominal feed the next control iteration (shifted by the one control step
    # that elapsed); every iteration is compared with the oracle, teacher-forced [R-17]
    import torch
    from oracle import oracle as O
    B, K, N = 4, 1024, 30
    wl = W.stress_gate_paper(K=K, N=N)
    p = dict(wl.params, B=B, near_mode=near_mode)
    rng = np.random.default_rng(2)
    x0 = np.repeat(wl.x0, B, 0); x0[:, 0:3] += rng.uniform(-0.2, 0.2, (B, 3)).astype(np.float32)
    from paper_2509_14726_b200 import binding as Bd
    m = Bd.Mppi(p); m.set_gates(wl.gates)
    x = torch.from_numpy(x0).cuda(); start = torch.zeros(B, dtype=torch.int32, device="cuda")
    u = torch.from_numpy(np.repeat(wl.u_nom, B, 0)).cuda()
    front = None
    seen_zero = False
    for step in range(6):
        x_in, s_in, u_in = x.cpu().numpy(), start.cpu().numpy(), u.cpu().numpy()
        m.set_prev_front(front)
        u_new, cost, w = m.step(x, start, u, 7, step)
        torch.cuda.synchronize()
        trk = O.Track(gates=wl.gates, prev_front=None if front is None else front.cpu().numpy())
        o = O.step(p, trk, x_in, s_in, u_in, 7, step, want_du=True)
        o["u_nom"] = u_in.astype(np.float64)
        gdict = dict(u_new=u_new.cpu().numpy(), cost=cost.cpu().numpy(), weights=w.cpu().numpy())
        Pz.compare(f"paper loop near_mode {near_mode} step{step}", gdict, o, p["lambda"], True)
        # flags of the new nominal from the current state, against the oracle's
        f = m.front_flags(x, start, u_new); torch.cuda.synchronize()
        fg = f.cpu().numpy()
        for b in range(B):
            fo, mg = O.front_flags(p, trk, x_in[b], int(s_in[b]), gdict["u_new"][b])
            assert mg < 1e-5 or np.array_equal(fg[b], fo), (step, b)
            assert fg[b, 0] == (1 if fo[0] else 0)
        seen_zero |= bool((fg == 0).any())
        # plant step, shift of the nominal and of the flags by one control step (last repeated)
        m.sim_step(x, start, u_new, u_nom_next=u)
        front = torch.cat([f[:, 1:], f[:, -1:]], dim=1).contiguous()
    assert seen_zero                        # the nominal really crosses the gate plane within the horizon
    m.close()


# ---- the paper's own input model (thrust rates, thrust states, drag, rate limit) ----

RATE_PIPES = [dict(pipeline=0, variant=4), dict(pipeline=0, variant=1), dict(pipeline=0, variant=1, block_threads=64), dict(pipeline=1),
              dict(pipeline=0, variant=3), dict(pipeline=1, variant=3, block_threads=64)]


RATE_IDS = ["fused_pipe", "fused", "fused_tpb64", "two_pass", "fused_pk", "two_pass_pk64"]


@pytest.mark.parametrize("pipe", RATE_PIPES, ids=RATE_IDS)
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
@pytest.mark.parametrize("name", ["rate_gate_paper", "rate_track"])
def test_rate_model_objectives(name, pipe, math):
    wl = W.ALL[name]()
    g, o, st = run_case(wl, f"{name}[{pipe},{math}]", **pipe, **math)
    # drag and the rate limit are really in play: switching them off changes the costs
    wl0 = W.ALL[name](); wl0.params.update(drag_x=0.0, drag_y=0.0, drag_z=0.0, w_limit=0.0)
    o0 = Pz.oracle_step(wl0, wl0.x0, wl0.start, wl0.u_nom, wl0.seed, 0)
    assert (np.abs(o0["cost"] - o["cost"]) > 1e-3 * np.abs(o["cost"])).mean() > 0.5


@pytest.mark.parametrize("pipe", RATE_PIPES, ids=RATE_IDS)
@pytest.mark.parametrize("name", ["rate_gate_paper", "rate_track"])
def test_rate_model_anisotropic_drag(name, pipe):
    # drag_x != drag_y: the scalar and packed kernels leave the axisymmetric short-cut of f_dyn
    # (fdyn_general<false>: all three body axes projected); Jx != Jy on top
    wl = W.ALL[name]()
    wl.params.update(drag_x=np.float32(0.8), drag_y=np.float32(0.05), drag_z=np.float32(0.1), Jx=1.0e-3, Jy=1.5e-3)
    g, o, st = run_case(wl, f"aniso_{name}[{pipe}]", fast_math=1, **pipe)
    wl0 = W.ALL[name]()
    wl0.params.update(drag_x=np.float32(0.425), drag_y=np.float32(0.425), drag_z=np.float32(0.1), Jx=1.0e-3, Jy=1.5e-3)
    o0 = Pz.oracle_step(wl0, wl0.x0, wl0.start, wl0.u_nom, wl0.seed, 0)
    assert (np.abs(o0["cost"] - o["cost"]) > 2e-4 * np.abs(o["cost"])).mean() > 0.2       # the anisotropy matters


@pytest.mark.parametrize("pipe", RATE_PIPES, ids=RATE_IDS)
def test_rate_model_saturation_and_crossings(pipe):
    wl = W.rate_stress(K=4096, N=30)
    g, o, st = run_case(wl, f"rate_stress[{pipe}]", **pipe)
    nc = o["ncross"]
    assert (nc > 0).mean() > 0.1 and (nc == 0).mean() > 0.1
    assert (np.abs(o["du"]) == wl.params["rate_max"]).mean() > 0.05          # rate clamp acts at scale


@pytest.mark.parametrize("K,N,B", [(32, 1, 1), (64, 7, 3), (96, 23, 2), (256, 100, 1), (2048, 50, 2)])
@pytest.mark.parametrize("name", ["rate_gate_paper", "rate_track", "rate_stress"])
def test_rate_model_pipelined_kernel_sizes(name, K, N, B):
    # the pipelined latency kernel of the rate model: ragged last chunk (N % 5 != 0), a single step, the
    # longest horizon its rings take, several controllers; against the oracle and against the scalar kernel
    if name == "rate_stress":
        N = min(N, 30)    # its sigma = 12 N/s is tuned for 30 steps: longer horizons leave the fp32 range
    wl = W.replicate(W.ALL[name](K=K, N=N), B, 0.2)
    if N >= 100:          # two seconds of sigma = 5 N/s rate noise tumble past the stability limit of explicit RK4
        wl.params["sigma"] = np.float32(1.0)
    if wl.prev_front is not None:
        wl.prev_front = np.random.default_rng(2).integers(0, 2, (B, N + 1)).astype(np.int32)
    m = Pz.make_ctx(wl, variant=4)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, 9, 2)
    assert m.info()["block_threads"] == 320 and m.info()["rollout_warps_per_block"] == 5     # chosen at the first step
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, 9, 2, want_du=True)
    o["u_nom"] = wl.u_nom.astype(np.float64)
    Pz.compare(f"{name} pipe K{K} N{N} B{B}", g, o, wl.params["lambda"], wl.params["objective"] == 0)
    m2 = Pz.make_ctx(wl, variant=1)
    g2 = Pz.gpu_step(m2, x0, start, u, 9, 2)
    np.testing.assert_allclose(g["cost"], g2["cost"], rtol=2e-4, atol=2e-4)
    g_again = Pz.gpu_step(m, x0, start, u, 9, 2)                  # run-to-run determinism
    for k in ("cost", "weights", "u_new"):
        np.testing.assert_array_equal(g[k], g_again[k])
    m.close(); m2.close()


def test_rate_model_contouring_batch_and_warm_start():
    # contouring under the rate model, B = 3, three warm-started iterations (teacher-forced)
    import torch
    wl = W._rate_model(W.cfg3(K=512, N=30), "rate_contour")
    B = 3
    wl.params = dict(wl.params, B=B)
    wl.x0 = np.repeat(wl.x0, B, 0); wl.x0[1, 0:3] += np.float32([0.1, -0.1, 0.05]); wl.x0[2, 13:17] += np.float32(0.3)
    wl.start = np.repeat(wl.start, B, 0); wl.u_nom = np.repeat(wl.u_nom, B, 0)
    m = Pz.make_ctx(wl)
    x0, start, u = Pz.to_dev(wl)
    for it in range(3):
        u_in = u.cpu().numpy()
        g = Pz.gpu_step(m, x0, start, u, wl.seed, it, u_new=u)
        o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, it, want_du=True)
        o["u_nom"] = u_in.astype(np.float64)
        Pz.compare(f"rate_contour it{it}", g, o, wl.params["lambda"], False)
    un, co, we = m.step_host(wl.x0, wl.start, u_in, wl.seed, 2)
    np.testing.assert_array_equal(co, g["cost"])
    m.close()


def test_rate_model_rejects_what_it_does_not_support():
    from paper_2509_14726_b200 import binding as Bd
    wl = W.rate_gate_paper(K=64, N=8)
    for bad in (dict(variant=2), dict(variant=3, K=96), dict(variant=3, block_threads=256), dict(variant=4, pipeline=1), dict(variant=4, block_threads=64),
                dict(variant=4, N=101), dict(rate_max=0.0)):
        with pytest.raises(Bd.MppiError) as e:
            Bd.Mppi(wl.params, **bad)
        assert e.value.status == -2
    with pytest.raises(Bd.MppiError) as e:
        Bd.Mppi(W.cfg0().params, drag_x=0.1)                    # drag needs the rate model
    assert e.value.status == -2


def test_rate_model_closed_loop_with_flags():
    # the paper's model + the paper's J_gate in a closed loop: plant step on the 17-entry rows, flags of
    # the new nominal fed to the next control step; every step teacher-forced against the oracle [R-17]
    import torch
    from oracle import oracle as O
    from paper_2509_14726_b200 import binding as Bd
    B, K, N = 4, 1024, 30
    wl = W.rate_gate_paper(K=K, N=N)
    p = dict(wl.params, B=B)
    rng = np.random.default_rng(4)
    x0 = np.repeat(wl.x0, B, 0); x0[:, 0:3] += rng.uniform(-0.2, 0.2, (B, 3)).astype(np.float32)
    m = Bd.Mppi(p); m.set_gates(wl.gates)
    x = torch.from_numpy(x0).cuda(); start = torch.zeros(B, dtype=torch.int32, device="cuda")
    u = torch.from_numpy(np.repeat(wl.u_nom, B, 0)).cuda()
    front = None
    for step in range(5):
        x_in, s_in, u_in = x.cpu().numpy(), start.cpu().numpy(), u.cpu().numpy()
        m.set_prev_front(front)
        u_new, cost, w = m.step(x, start, u, 3, step)
        torch.cuda.synchronize()
        trk = O.Track(gates=wl.gates, prev_front=None if front is None else front.cpu().numpy())
        o = O.step(p, trk, x_in, s_in, u_in, 3, step, want_du=True)
        o["u_nom"] = u_in.astype(np.float64)
        g = dict(u_new=u_new.cpu().numpy(), cost=cost.cpu().numpy(), weights=w.cpu().numpy())
        Pz.compare(f"rate loop step{step}", g, o, p["lambda"], True)
        f = m.front_flags(x, start, u_new); torch.cuda.synchronize()
        for b in range(B):
            fo, mg = O.front_flags(p, trk, x_in[b], int(s_in[b]), g["u_new"][b])
            assert mg < 1e-5 or np.array_equal(f.cpu().numpy()[b], fo), (step, b)
        xo, so, uo = O.sim_step(p, trk, x_in, s_in, g["u_new"])
        m.sim_step(x, start, u_new, u_nom_next=u); torch.cuda.synchronize()
        np.testing.assert_allclose(x.cpu().numpy(), xo, rtol=3e-6, atol=2e-5)
        np.testing.assert_array_equal(u.cpu().numpy(), uo.astype(np.float32))
        np.testing.assert_array_equal(start.cpu().numpy(), so)
        front = torch.cat([f[:, 1:], f[:, -1:]], dim=1).contiguous()
    assert not np.array_equal(x.cpu().numpy()[:, 13:], x0[:, 13:])      # the thrust states moved
    m.close()


# ---- the paper's own contouring formulation (objective 4; readings R-33..R-37) --------

V_ATOL = 1e-4        # m/s^2 on the fifth column of the update: north_star's u_new bound carried over


def _cp_check(tag, wl, g, o):
    # [R-38] eq.(9) sums a reward -mu v_theta against positive error terms: J can cancel to ~0 while both
    # parts are ~ mu v_theta_max N; the fp32 error scales with the parts, so that is the floor of the bound
    # Tried in round 2: with the thrust combinations carried as states (ThrustDiff) the full-size cases meet plain
    # [R-20] (32 of 34 objective-4 cases), but two small-K closed-loop cases keep costs that cancel to |J| < 1 with an
    # error of 7-9e-4 -- a compensated (Kahan) sum of the stage terms changes that from 8.6e-4 to 7.3e-4 only: the
    # error is the fp32 state error times the cost gradient (q_c = 200 on e_c^2), not the summation.  The floor stays.
    floor = max(1.0, float(wl.params["mu_progress"]) * float(wl.params["v_theta_max"]) * wl.params["N"])
    st = Pz.compare(tag, g, o, wl.params["lambda"], False, cost_floor=floor)
    verr = float(np.abs(g["v_new"].astype(np.float64) - o["v_new"]).max())
    Pz.STATS.append(f"{tag}: v_new {verr:.2e}")
    if verr > V_ATOL:
        # as for u_new in parity.compare: allowed only where fp32 cannot resolve the weights (a "reported
        # separately" line exists for this tag); the column must then be the exact update of the GPU's weights
        assert any(r.startswith(tag + ": near-tied") for r in Pz.REPORT), f"{tag}: v_new err {verr:.3e}"
        v_self = o["v_nom"] + np.einsum("bk,bkt->bt", g["weights"].astype(np.float64), o["dv"])
        assert np.abs(g["v_new"] - v_self).max() <= V_ATOL, f"{tag}: v_new inconsistent with its weights"
    return st


@pytest.mark.parametrize("pipe", [dict(variant=1), dict(variant=1, block_threads=64), dict(variant=1, block_threads=256), dict(variant=4), dict(),
                                  dict(variant=3), dict(variant=3, block_threads=32)],
                         ids=["fused", "fused_tpb64", "fused_tpb256", "fused_pipe", "auto", "fused_pk", "fused_pk_tpb32"])
@pytest.mark.parametrize("math", MATH, ids=["accurate", "fast"])
@pytest.mark.parametrize("regime", [dict(), {"sigma": np.float32(2.0), "lambda": np.float32(1000.0)}], ids=["argmin", "mixing"])
def test_contour_paper_full_size(pipe, math, regime):
    # "argmin": the workload as it stands -- like the paper's lambda = 0.01 (Table I) the softmax picks one
    # sample (ESS 1); "mixing": a temperature at the scale of the cost spread, so that the weights and
    # both updates average over tens of samples
    wl = W.contour_paper()
    wl.params.update(regime)
    rng = np.random.default_rng(5)
    wl.v_nom = rng.uniform(-3, 3, wl.v_nom.shape).astype(np.float32)       # a non-trivial nominal fifth column
    m = Pz.make_ctx(wl, **pipe, **math)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True, v_nom=wl.v_nom)
    o["u_nom"] = wl.u_nom.astype(np.float64); o["v_nom"] = wl.v_nom.astype(np.float64)
    st = _cp_check(f"contour_paper[{pipe},{math},{sorted(regime)}]", wl, g, o)
    assert (st["ess"] > 10) == bool(regime)
    assert (np.abs(o["dv"] + wl.v_nom[:, None, :] ) == wl.params["dv_max"]).any()      # the fifth input's clamp acts
    assert np.abs(o["v_new"] - wl.v_nom).max() > 0.05                                  # and the update moves it
    m.close()


def test_contour_paper_batch_warm_start_open_path_and_speed_limits():
    # B = 3 on the OPEN form of the path, theta_0 near both ends and v_theta,0 at both limits, four
    # warm-started iterations in place (u and v); teacher-forced against the oracle [R-17]
    import torch
    wl = W.contour_paper(K=1024, N=40)
    B = 3
    wl.closed = 0
    wl.params = dict(wl.params, B=B, sigma=np.float32(2.0))
    wl.params["lambda"] = np.float32(300.0)                      # mixing regime: ESS 15..70 over the four iterations
    L = float(np.linalg.norm(np.diff(wl.path.astype(np.float64), axis=0), axis=1).sum())
    wl.x0 = np.repeat(wl.x0, B, 0)
    wl.x0[1, 17:19] = np.float32([L - 0.3, 10.0]); wl.x0[1, 0:3] = wl.path[-2]
    wl.x0[2, 17:19] = np.float32([0.05, 0.0]); wl.x0[2, 0:3] = wl.path[0] + np.float32([0.1, 0.0, -0.1])
    wl.start = np.repeat(wl.start, B, 0); wl.u_nom = np.repeat(wl.u_nom, B, 0)
    wl.v_nom = np.repeat(wl.v_nom, B, 0)
    _open_path_iterations(wl, dict(variant=1), 128)              # scalar kernel of the rate model
    _open_path_iterations(wl, dict(), 320)                       # AUTO: 96 warps, the path fits -> the pipelined kernel
    _open_path_iterations(wl, dict(variant=3), 128)              # packed fp32x2 kernel (K = 1024: 4 blocks of 256 samples)


def _open_path_iterations(wl, opts, threads):
    import torch
    m = Pz.make_ctx(wl, **opts)
    x0, start, u = Pz.to_dev(wl)
    v = torch.from_numpy(wl.v_nom.copy()).cuda()
    m.set_progress(v)                                            # in place
    for it in range(4):
        u_in, v_in = u.cpu().numpy(), v.cpu().numpy()
        g = Pz.gpu_step(m, x0, start, u, wl.seed, it, u_new=u)
        o = Pz.oracle_step(wl, wl.x0, wl.start, u_in, wl.seed, it, want_du=True, v_nom=v_in)
        o["u_nom"] = u_in.astype(np.float64); o["v_nom"] = v_in.astype(np.float64)
        assert _cp_check(f"contour_paper open {opts} it{it}", wl, g, o)["ess"] > 10
    assert np.abs(v.cpu().numpy()).max() > 0.1
    # mppi_optimize runs the same four iterations in one call
    u2 = torch.from_numpy(wl.u_nom.copy()).cuda(); v2 = torch.from_numpy(wl.v_nom.copy()).cuda()
    m.set_progress(v2)
    m.optimize(x0, start, u2, wl.seed, 0, 4); torch.cuda.synchronize()
    np.testing.assert_array_equal(u2.cpu().numpy(), u.cpu().numpy())
    np.testing.assert_array_equal(v2.cpu().numpy(), v.cpu().numpy())
    assert m.info()["kernels_per_step"] == 1                     # the fifth column rides in the fused update
    assert m.info()["block_threads"] == threads
    m.close()


def test_rate_model_stored_noise_matches_the_oracle():
    # store_noise = 1: the clamped rate perturbations dU the kernels rolled out, pipelined and scalar kernel
    wl = W.rate_gate_paper(K=256, N=23)
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, 5, 7, want_du=True)
    du_o = np.transpose(o["du"], (0, 2, 1, 3))
    outs = {}
    for name, opts in dict(pipe=dict(variant=4, store_noise=1), thr=dict(variant=1, store_noise=1)).items():
        m = Pz.make_ctx(wl, **opts)
        x0, start, u = Pz.to_dev(wl)
        outs[name] = Pz.gpu_step(m, x0, start, u, 5, 7)
        du = m.debug_noise().cpu().numpy()                      # [B,N,K,4]
        np.testing.assert_allclose(du, du_o, rtol=0, atol=1e-5)
        outs[name]["du"] = du
        m.close()
    np.testing.assert_array_equal(outs["pipe"]["du"], outs["thr"]["du"])
    assert (np.abs(wl.u_nom[:, :, None, :] + outs["pipe"]["du"]) == wl.params["rate_max"]).any()     # the rate clamp acts


def test_rate_model_auto_kernel_choice():
    # input_model = 1 under AUTO: pipelined kernel with deep rings up to one block per SM, with shallow rings (two
    # blocks per SM) up to twice the SM count when they fit, else the scalar kernel -- decided at the first step
    sm = Pz.make_ctx(W.cfg0()).info()["sm_count"]
    for K, N, B, threads in ((4096, 50, 1, 320), (8192, 20, 1, 320), (8192, 50, 1, 128), (4096, 50, 3, 128)):
        wl = W.replicate(W.rate_gate_paper(K=K, N=N), B, 0.2)
        m = Pz.make_ctx(wl)
        x0, start, u = Pz.to_dev(wl)
        g = Pz.gpu_step(m, x0, start, u, 2, 0)
        assert m.info()["block_threads"] == threads, (K, N, B, m.info())
        if threads == 320:
            assert m.info()["grid_blocks"] <= (1 if N == 50 else 2) * sm
        o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, 2, 0, want_du=True)
        o["u_nom"] = wl.u_nom.astype(np.float64)
        Pz.compare(f"rate auto K{K} N{N} B{B}", g, o, wl.params["lambda"], False)
        m.close()


def test_table1_sizes():
    # the sizes of the paper's own Table I (M = 8192, K = 20, dt = 0.03, lambda = 0.01) under the paper's J_gate
    # and the paper's contouring, thrust-rate model
    wl = W.table1("gate")
    m = Pz.make_ctx(wl)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True)
    o["u_nom"] = wl.u_nom.astype(np.float64)
    # [R-20] as it stands.  (Round 1 measured this case against |p_0 - c|^2; the error turned out to sit in the soft
    # body-rate limit next to omega_max, fed by the rounding of the thrust states' differences, and went away with the
    # thrust combinations carried as states: profiles/README_r02a.md, mppi_rate.cuh ThrustDiff.)
    Pz.compare("table1_gate", g, o, wl.params["lambda"], False)
    m.close()
    wl = W.table1("contour")
    m = Pz.make_ctx(wl)
    x0, start, u = Pz.to_dev(wl)
    g = Pz.gpu_step(m, x0, start, u, wl.seed, 0)
    o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, wl.seed, 0, want_du=True, v_nom=wl.v_nom)
    o["u_nom"] = wl.u_nom.astype(np.float64); o["v_nom"] = wl.v_nom.astype(np.float64)
    _cp_check("table1_contour", wl, g, o)
    m.close()


def test_contour_paper_auto_falls_back_when_the_path_does_not_fit():
    # AUTO takes the pipelined kernel for a lone controller only if the path fits in shared memory beside its rings:
    # 500 points do, 1800 do not (-> scalar kernel); an explicit PIPELINED request then fails with MPPI_E_PARAM
    from paper_2509_14726_b200 import binding as Bd
    wl = W.contour_paper(K=256, N=20)
    long_path = W.spline_path(W.circle_gates()[:, 0:3], 1800)
    for path, threads in ((wl.path, 320), (long_path, 128)):
        wl.path = path
        m = Pz.make_ctx(wl)
        x0, start, u = Pz.to_dev(wl)
        g = Pz.gpu_step(m, x0, start, u, 4, 1)
        assert m.info()["block_threads"] == threads
        o = Pz.oracle_step(wl, wl.x0, wl.start, wl.u_nom, 4, 1, want_du=True, v_nom=wl.v_nom)
        o["u_nom"] = wl.u_nom.astype(np.float64); o["v_nom"] = wl.v_nom.astype(np.float64)
        _cp_check(f"contour_paper auto P{len(path)}", wl, g, o)
        m.close()
    m = Pz.make_ctx(wl, variant=4)
    x0, start, u = Pz.to_dev(wl)
    with pytest.raises(Bd.MppiError) as e:
        m.step(x0, start, u, 4, 1)
    assert e.value.status == -2
    m.close()


def test_contour_paper_rejects_what_it_does_not_support():
    import torch
    from paper_2509_14726_b200 import binding as Bd
    wl = W.contour_paper(K=64, N=8)
    for bad in (dict(input_model=0, drag_x=0.0, drag_y=0.0, drag_z=0.0, w_limit=0.0), dict(pipeline=1), dict(use_graph=1),
                dict(dv_max=0.0), dict(v_theta_max=0.0), dict(sigma_v=-1.0), dict(r_dv=-1.0)):
        with pytest.raises(Bd.MppiError) as e:
            Bd.Mppi(wl.params, **bad)
        assert e.value.status == -2, bad
    m = Bd.Mppi(wl.params); m.set_path(wl.path, wl.closed)
    x0, start, u = Pz.to_dev(wl)
    with pytest.raises(Bd.MppiError) as e:
        m.step(x0, start, u, 1, 0)                              # mppi_set_progress not called
    assert e.value.status == -3
    v = torch.zeros((1, 8), device="cuda")
    m.set_progress(v, torch.empty_like(v))
    with pytest.raises(Bd.MppiError) as e:
        m.optimize(x0, start, u, 1, 0, 2)                       # needs the in-place form
    assert e.value.status == -5
    with pytest.raises(Bd.MppiError) as e:
        m.step_host(wl.x0, wl.start, wl.u_nom, 1, 0)
    assert e.value.status == -2
    m.close()
    m = Bd.Mppi(W.cfg3().params)
    with pytest.raises(Bd.MppiError) as e:
        m.set_progress(torch.zeros((1, 50), device="cuda"))    # another objective
    assert e.value.status == -2
    m.close()


# ---- closed-loop lap experiment (paper_2509_14726_b200/closed_loop.py) ---------------

@pytest.mark.parametrize("kind,iters", [("gate", 1), ("gate_paper", 2)])
def test_lap_experiment_gate_objectives(kind, iters):
    from paper_2509_14726_b200 import closed_loop as CL
    # K = 4096 as in DESIGN.md's table: with half as many samples the paper's J_gate does not reliably hold the lap
    # (2 of 4 drones miss a gate and never return), and which drones do depends on the last bits of the update
    wl = W.lap(kind, B=4, K=4096, steps=700)
    m = Pz.make_ctx(wl)
    log = CL.fly(m, wl, 700, iters_per_step=iters, prev_front_feedback=(kind == "gate_paper"))
    m.close()
    assert np.isfinite(log.x).all()
    mt = CL.lap_metrics(log, wl.gates, laps=1)
    G = wl.gates.shape[0]
    for b, q in enumerate(mt):
        assert q["flight_time_s"] is not None and q["flight_time_s"] < 14.0, (b, q)     # a lap of 31 m
        assert q["wp_dist_max"] <= np.hypot(0.75, 0.75) + 1e-6                         # inside the opening
        assert 2.0 < q["speed_mean"] < 15.0
        # the device's own gate counter (float32 plant test) agrees with the float64 host replay
        assert int(log.start[-1, b]) == q["passes"] % G


def test_lap_experiment_tracking_and_contouring():
    from paper_2509_14726_b200 import closed_loop as CL
    wl = W.lap("track", B=4, K=2048, steps=400)
    m = Pz.make_ctx(wl)
    log = CL.fly(m, wl, 400)
    m.close()
    assert (CL.tracking_rmse(log, wl.ref) < 0.6).all()
    np.testing.assert_array_equal(log.start[-1], 400)          # the reference clock advanced one row per step
    wl = W.lap("contour", B=4, K=2048, steps=400)
    m = Pz.make_ctx(wl)
    log = CL.fly(m, wl, 400)
    m.close()
    assert (CL.contour_rms(log, wl.path) < 0.3).all()
    travelled = np.linalg.norm(np.diff(log.x[:, :, 0:3].astype(np.float64), axis=0), axis=-1).sum(0)
    assert (travelled > 15.0).all()                            # it really flies along the path


def test_contour_paper_closed_loop_teacher_forced():
    # the paper's contouring in a closed loop: iteration (u and v updated in place), plant step on rows of 19,
    # shift of both nominals; every step compared with the oracle from the GPU's own inputs [R-17]
    import torch
    from oracle import oracle as O
    B, K, N = 3, 1024, 30
    wl = W.lap("contour_paper", B=B, K=K, N=N)
    p = wl.params
    m = Pz.make_ctx(wl)
    x, start, u = Pz.to_dev(wl)
    v = torch.from_numpy(wl.v_nom.copy()).cuda()
    m.set_progress(v)
    for step in range(5):
        x_in, u_in, v_in = x.cpu().numpy(), u.cpu().numpy(), v.cpu().numpy()
        g = Pz.gpu_step(m, x, start, u, 5, step, u_new=u)
        o = O.step(p, O.Track(path=wl.path, closed=wl.closed), x_in, wl.start, u_in, 5, step, want_du=True, v_nom=v_in)
        o["u_nom"] = u_in.astype(np.float64); o["v_nom"] = v_in.astype(np.float64)
        _cp_check(f"contour_paper loop step{step}", wl, g, o)
        xo, uo, vo = O.sim_step_progress(p, x_in, g["u_new"], g["v_new"])
        m.sim_step_progress(x, u, v); torch.cuda.synchronize()
        np.testing.assert_allclose(x.cpu().numpy(), xo, rtol=3e-6, atol=2e-5)
        np.testing.assert_array_equal(u.cpu().numpy(), uo.astype(np.float32))
        np.testing.assert_array_equal(v.cpu().numpy(), vo.astype(np.float32))
    assert (x.cpu().numpy()[:, 17] > wl.x0[:, 17] + 0.1).all()            # theta moved on
    # out-of-place form gives the same plant step
    x2 = torch.from_numpy(x_in).cuda(); u2 = torch.from_numpy(g["u_new"]).cuda(); v2 = torch.from_numpy(g["v_new"]).cuda()
    un = torch.empty_like(u2); vn = torch.empty_like(v2)
    m.sim_step_progress(x2, u2, v2, u_nom_next=un, v_nom_next=vn); torch.cuda.synchronize()
    np.testing.assert_array_equal(x2.cpu().numpy(), x.cpu().numpy())
    np.testing.assert_array_equal(un.cpu().numpy(), u.cpu().numpy()); np.testing.assert_array_equal(vn.cpu().numpy(), v.cpu().numpy())
    m.close()


def test_lap_experiment_contour_paper():
    from paper_2509_14726_b200 import closed_loop as CL
    wl = W.lap("contour_paper", B=4, K=2048, steps=500)
    m = Pz.make_ctx(wl)
    log = CL.fly(m, wl, 500)
    m.close()
    assert np.isfinite(log.x).all()
    for b, q in enumerate(CL.progress_metrics(log, wl.path)):
        assert q["laps"] > 1.5 and len(q["lap_times_s"]) >= 1 and q["lap_times_s"][0] < 8.0, (b, q)   # 31 m per lap
        assert q["dist_to_progress_point_max"] < 1.5, (b, q)       # the vehicle stays with its progress state
        assert 3.0 < q["speed_mean"] < 12.0
    assert (CL.contour_rms(log, wl.path) < 0.4).all()
    assert log.x[:, :, 2].min() > 0.5                              # and in the air (the path is at z = 1.5 m)


def test_lap_experiment_on_the_figure_eight():
    # the stand-in for the paper's Figure-8 track: the 7-gate lemniscate of configs[1], gate heights
    # 1-3 m.  The gate objective must complete a lap through all seven gates in order; the paper's contouring must
    # carry its progress state once around the spline path through the gate centres, the vehicle staying with it
    from paper_2509_14726_b200 import closed_loop as CL
    wl = W.lap("gate", B=4, K=4096, track="figure8")
    m = Pz.make_ctx(wl)
    log = CL.fly(m, wl, 700)
    m.close()
    assert np.isfinite(log.x).all()
    for b, q in enumerate(CL.lap_metrics(log, wl.gates, laps=1)):
        assert q["flight_time_s"] is not None and q["flight_time_s"] < 13.0, (b, q)     # 60 m per lap
        assert q["wp_dist_max"] <= np.hypot(0.75, 0.75) + 1e-6
        assert int(log.start[-1, b]) == q["passes"] % wl.gates.shape[0]                 # device counter = float64 replay
    wl = W.lap("contour_paper", B=4, K=4096, track="figure8")
    m = Pz.make_ctx(wl)
    log = CL.fly(m, wl, 700)
    m.close()
    for b, q in enumerate(CL.progress_metrics(log, wl.path)):
        assert q["laps"] > 1.2 and q["dist_to_progress_point_max"] < 2.5, (b, q)
    assert (CL.contour_rms(log, wl.path) < 0.5).all()
    assert log.x[:, :, 2].min() > 0.3                                                   # gate heights are 1-3 m
