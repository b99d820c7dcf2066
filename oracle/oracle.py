"""ctypes front end of the float64 CPU oracle (oracle/mppi_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It holds no arithmetic of the
method; every number comes out of the C file, which cites PAPER.md passage by passage.
Nothing here imports, links or reads the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "mppi_oracle.c"
_LIB = _HERE / "libmppi_oracle.so"

OBJ_GATE, OBJ_TRACK, OBJ_CONTOUR, OBJ_GATE_PAPER, OBJ_CONTOUR_PAPER = 0, 1, 2, 3, 4


def build(force: bool = False) -> Path:
    """Compile the oracle with gcc: -O2, OpenMP over samples, no fast-math, no FMA contraction.

    MPPI_ORACLE_SANITIZE=1 in the environment builds (and loads) an AddressSanitizer + UndefinedBehaviorSanitizer
    variant instead (same source, -O1 -g; libmppi_oracle_san.so).  The interpreter must then be started with the
    sanitizer runtimes preloaded:
        MPPI_ORACLE_SANITIZE=1 ASAN_OPTIONS=detect_leaks=0 \
        LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)" \
        python -m pytest tests -q -m "not gpu"
    """
    san = os.environ.get("MPPI_ORACLE_SANITIZE", "") not in ("", "0")
    lib = _HERE / "libmppi_oracle_san.so" if san else _LIB
    if force or not lib.exists() or lib.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = lib.with_suffix(f".{os.getpid()}.tmp")
        opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if san else ["-O2"]
        cmd = ["gcc", "-std=c11", *opt, "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-shared", "-fPIC", "-Wall", "-Wextra", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, lib)
    return lib


class _Params(C.Structure):
    _fields_ = [("K", C.c_int32), ("N", C.c_int32), ("B", C.c_int32), ("objective", C.c_int32),
                ("dt", C.c_double), ("lambda_", C.c_double), ("sigma", C.c_double),
                ("mass", C.c_double), ("Jx", C.c_double), ("Jy", C.c_double), ("Jz", C.c_double),
                ("arm", C.c_double), ("c_tau", C.c_double), ("g", C.c_double),
                ("T_min", C.c_double), ("T_max", C.c_double), ("w_omega", C.c_double),
                ("gate_miss_penalty", C.c_double), ("gate_pass_bonus", C.c_double),
                ("Qp", C.c_double), ("Qv", C.c_double), ("Qq", C.c_double), ("Qw", C.c_double),
                ("R", C.c_double), ("q_contour", C.c_double), ("q_lag", C.c_double),
                ("mu_progress", C.c_double), ("window", C.c_int32), ("near_mode", C.c_int32),
                ("q_near", C.c_double), ("r_near", C.c_double),
                ("input_model", C.c_int32), ("pad2_", C.c_int32), ("rate_max", C.c_double),
                ("drag_x", C.c_double), ("drag_y", C.c_double), ("drag_z", C.c_double),
                ("w_limit", C.c_double), ("omega_max", C.c_double),
                ("sigma_v", C.c_double), ("dv_max", C.c_double), ("v_theta_max", C.c_double), ("r_dv", C.c_double)]


class _Track(C.Structure):
    _fields_ = [("G", C.c_int32), ("M", C.c_int32), ("P", C.c_int32), ("closed", C.c_int32),
                ("gates", C.POINTER(C.c_double)), ("ref", C.POINTER(C.c_double)),
                ("pts", C.POINTER(C.c_double)), ("v_nom", C.POINTER(C.c_double)),
                ("v_new", C.POINTER(C.c_double)), ("dv_out", C.POINTER(C.c_double)),
                ("prev_front", C.POINTER(C.c_int32))]


_PARAM_KEYS = [f for f, _ in _Params._fields_ if f not in ("pad_", "pad2_")]
_OPTIONAL = {"near_mode": 0, "q_near": 0.0, "r_near": 0.0, "input_model": 0, "rate_max": 0.0, "drag_x": 0.0, "drag_y": 0.0,
             "drag_z": 0.0, "w_limit": 0.0, "omega_max": 0.0, "sigma_v": 0.0, "dv_max": 0.0, "v_theta_max": 0.0,
             "r_dv": 0.0}
_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_up = C.POINTER(C.c_uint32)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(str(build()))
        L = _lib
        L.orc_philox4x32_10.argtypes = [_up, _up, _up]
        L.orc_philox4x32_10.restype = None
        L.orc_uniform.argtypes = [C.c_uint32]
        L.orc_uniform.restype = C.c_double
        L.orc_normals.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, _dp]
        L.orc_normals.restype = None
        L.orc_fdyn.argtypes = [C.POINTER(_Params), _dp, _dp, _dp]
        L.orc_fdyn.restype = None
        L.orc_rk4_step.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_double, _dp]
        L.orc_rk4_step.restype = None
        L.orc_path_eval.argtypes = [_dp, _dp, _dp, C.c_int32, C.c_int32, C.c_double, C.c_double, _dp, _dp]
        L.orc_path_eval.restype = None
        L.orc_normal5.argtypes = [C.c_uint64, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32]
        L.orc_normal5.restype = C.c_double
        L.orc_progress_step.argtypes = [C.POINTER(_Params), C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.orc_progress_step.restype = None
        L.orc_rk4_rate_step.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_double, _dp]
        L.orc_rk4_rate_step.restype = None
        L.orc_rate_limit_cost.argtypes = [C.POINTER(_Params), _dp]
        L.orc_rate_limit_cost.restype = C.c_double
        L.orc_gate_step.argtypes = [C.POINTER(_Params), C.POINTER(_Track), _dp, _dp, _dp, _ip, _dp,
                                    _ip]
        L.orc_gate_step.restype = C.c_double
        L.orc_gate_paper_step.argtypes = [C.POINTER(_Params), C.POINTER(_Track), _dp, _dp, _dp, _ip,
                                          C.c_int32, C.c_int32, _dp, _ip]
        L.orc_gate_paper_step.restype = C.c_double
        L.orc_front_flags.argtypes = [C.POINTER(_Params), C.POINTER(_Track), _dp, C.c_int32, _dp, _ip, _dp]
        L.orc_front_flags.restype = None
        L.orc_track_state_term.argtypes = [C.POINTER(_Params), _dp, _dp]
        L.orc_track_state_term.restype = C.c_double
        L.orc_track_stage.argtypes = [C.POINTER(_Params), _dp, _dp, _dp]
        L.orc_track_stage.restype = C.c_double
        L.orc_path_prepare.argtypes = [_dp, C.c_int32, C.c_int32, _dp, _dp]
        L.orc_path_prepare.restype = C.c_double
        L.orc_path_nearest.argtypes = [_dp, C.c_int32, C.c_int32, _dp, C.c_int32, C.c_int32]
        L.orc_path_nearest.restype = C.c_int32
        L.orc_contour_step.argtypes = [C.POINTER(_Params), C.POINTER(_Track), _dp, _dp, C.c_double,
                                       _dp, _dp, _ip, _dp]
        L.orc_contour_step.restype = C.c_double
        L.orc_weights_update.argtypes = [C.c_int32, C.c_int32, C.c_double, _dp, _dp, _dp, _dp, _dp]
        L.orc_weights_update.restype = None
        L.orc_step.argtypes = [C.POINTER(_Params), C.POINTER(_Track), _dp, _ip, _dp, C.c_uint64,
                               C.c_uint32, _dp, _dp, _dp, _dp, _dp, _ip, _ip]
        L.orc_step.restype = C.c_int
        L.orc_sim_step.argtypes = [C.POINTER(_Params), C.POINTER(_Track), _dp, _ip, _dp, _dp]
        L.orc_sim_step.restype = C.c_int
        L.orc_sim_step_progress.argtypes = [C.POINTER(_Params), _dp, _dp, _dp, _dp, _dp]
        L.orc_sim_step_progress.restype = C.c_int
        L.orc_num_threads.argtypes = []
        L.orc_num_threads.restype = C.c_int
    return _lib


def _d(a):
    return a.ctypes.data_as(_dp)


def _i(a):
    return a.ctypes.data_as(_ip)


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None:
        a = a.reshape(shape)
    return a


def make_params(p: dict) -> _Params:
    """dict (keys of include/mppi.h's mppi_params; 'lambda' accepted for lambda_) -> C struct.
    Values are converted exactly (a float32 input becomes the same real number in double)."""
    s = _Params()
    src = dict(p)
    if "lambda" in src:
        src["lambda_"] = src.pop("lambda")
    for k in _PARAM_KEYS:
        if k not in src:
            if k in _OPTIONAL:                      # the paper-variant extensions (objective 3, NEXT-2)
                src[k] = _OPTIONAL[k]
            else:
                raise KeyError(f"oracle params: missing '{k}'")
        v = src[k]
        setattr(s, k, int(v) if k in ("K", "N", "B", "objective", "window", "input_model", "near_mode") else float(v))
    return s


class Track:
    """Holds float64 copies of the track arrays and the C view of them."""

    def __init__(self, gates=None, ref=None, path=None, closed=True, prev_front=None):
        self.gates = _f64(gates, (-1, 11)) if gates is not None else None
        self.ref = _f64(ref, (-1, 13)) if ref is not None else None
        self.path = _f64(path, (-1, 3)) if path is not None else None
        self.c = _Track()
        self.c.G = 0 if self.gates is None else self.gates.shape[0]
        self.c.M = 0 if self.ref is None else self.ref.shape[0]
        self.c.P = 0 if self.path is None else self.path.shape[0]
        self.c.closed = 1 if closed else 0
        null = C.cast(None, _dp)
        self.c.gates = _d(self.gates) if self.gates is not None else null
        self.c.ref = _d(self.ref) if self.ref is not None else null
        self.c.pts = _d(self.path) if self.path is not None else null
        self.prev_front = (np.ascontiguousarray(np.asarray(prev_front, dtype=np.int32))
                           if prev_front is not None else None)
        self.c.prev_front = _i(self.prev_front) if self.prev_front is not None else C.cast(None, _ip)


# ---- thin wrappers -----------------------------------------------------------------------

def philox4x32_10(ctr, key):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return [int(v) for v in o]


def uniform(r: int) -> float:
    return lib().orc_uniform(int(r) & 0xFFFFFFFF)


def normals(seed, k, t, it, b):
    z = np.zeros(4)
    lib().orc_normals(int(seed), int(k), int(t), int(it), int(b), _d(z))
    return z


def fdyn(params, x, T):
    P = make_params(params)
    x = _f64(x, (13,)); T = _f64(T, (4,)); out = np.zeros(13)
    lib().orc_fdyn(C.byref(P), _d(x), _d(T), _d(out))
    return out


def rk4_step(params, x, T, dt=None):
    P = make_params(params)
    x = _f64(x, (13,)); T = _f64(T, (4,)); out = np.zeros(13)
    lib().orc_rk4_step(C.byref(P), _d(x), _d(T), float(P.dt if dt is None else dt), _d(out))
    return out


def path_eval(pts, closed, theta):
    """[R-36] -> (P(theta), unit tangent at theta, path length L) for a caller-supplied path."""
    pts = _f64(pts, (-1, 3)); n = pts.shape[0]
    s = np.zeros(n); tan = np.zeros((n, 3))
    L = lib().orc_path_prepare(_d(pts), n, 1 if closed else 0, _d(s), _d(tan))
    pos = np.zeros(3); tg = np.zeros(3)
    lib().orc_path_eval(_d(pts), _d(s), _d(tan), n, 1 if closed else 0, L, float(theta), _d(pos), _d(tg))
    return pos, tg, L


def normal5(seed, k, t, it, b):
    return lib().orc_normal5(int(seed), int(k), int(t), int(it), int(b))


def progress_step(params, theta, v, dv):
    P = make_params(params)
    a = np.zeros(1); b = np.zeros(1)
    lib().orc_progress_step(C.byref(P), float(theta), float(v), float(dv), _d(a), _d(b))
    return float(a[0]), float(b[0])


def rk4_rate_step(params, x, u, dt=None):
    """One RK4 step of the 17-state thrust-rate model [R-27],[R-29]."""
    P = make_params(params)
    x = _f64(x, (17,)); u = _f64(u, (4,)); out = np.zeros(17)
    lib().orc_rk4_rate_step(C.byref(P), _d(x), _d(u), float(P.dt if dt is None else dt), _d(out))
    return out


def rate_limit_cost(params, omega):
    P = make_params(params)
    return lib().orc_rate_limit_cost(C.byref(P), _d(_f64(omega, (3,))))


def gate_step(params, track: Track, p_prev, p, omega, gate):
    """-> (step cost, new gate index, margin, number of valid passes)."""
    P = make_params(params)
    g = C.c_int32(int(gate)); m = C.c_double(np.inf); n = C.c_int32(0)
    J = lib().orc_gate_step(C.byref(P), C.byref(track.c), _d(_f64(p_prev, (3,))), _d(_f64(p, (3,))),
                            _d(_f64(omega, (3,))), C.byref(g), C.byref(m), C.byref(n))
    return J, g.value, m.value, n.value


def gate_paper_step(params, track: Track, p_prev, p, omega, gate, gate0, front_ok):
    """The paper's J_gate, one step -> (step cost, new gate index, margin, registered passes)."""
    P = make_params(params)
    g = C.c_int32(int(gate)); m = C.c_double(np.inf); n = C.c_int32(0)
    J = lib().orc_gate_paper_step(C.byref(P), C.byref(track.c), _d(_f64(p_prev, (3,))), _d(_f64(p, (3,))),
                                  _d(_f64(omega, (3,))), C.byref(g), int(gate0), int(front_ok),
                                  C.byref(m), C.byref(n))
    return J, g.value, m.value, n.value


def front_flags(params, track: Track, x0, start, u):
    """[R-26] -> (front[N+1] int32, margin) of the noise-free rollout of u from x0."""
    P = make_params(params)
    u = _f64(u, (P.N, 4)); f = np.zeros(P.N + 1, np.int32); m = C.c_double(np.inf)
    lib().orc_front_flags(C.byref(P), C.byref(track.c), _d(_f64(x0, (17 if P.input_model == 1 else 13,))), int(start), _d(u), _i(f), C.byref(m))
    return f, m.value


def track_state_term(params, x, xr):
    P = make_params(params)
    return lib().orc_track_state_term(C.byref(P), _d(_f64(x, (13,))), _d(_f64(xr, (13,))))


def track_stage(params, x, T, xr):
    P = make_params(params)
    return lib().orc_track_stage(C.byref(P), _d(_f64(x, (13,))), _d(_f64(T, (4,))),
                                 _d(_f64(xr, (13,))))


def path_prepare(pts, closed=True):
    """-> (s[P], tangents[P,3], L)."""
    pts = _f64(pts, (-1, 3)); n = pts.shape[0]
    s = np.zeros(n); tan = np.zeros((n, 3))
    L = lib().orc_path_prepare(_d(pts), n, 1 if closed else 0, _d(s), _d(tan))
    return s, tan, L


def path_nearest(pts, closed, p, centre, W):
    pts = _f64(pts, (-1, 3))
    return lib().orc_path_nearest(_d(pts), pts.shape[0], 1 if closed else 0, _d(_f64(p, (3,))),
                                  int(centre), int(W))


def contour_step(params, track: Track, p, omega, idx, theta_prev):
    """-> (step cost, new index, new theta)."""
    P = make_params(params)
    s, tan, L = path_prepare(track.path, bool(track.c.closed))
    i = C.c_int32(int(idx)); th = C.c_double(float(theta_prev))
    J = lib().orc_contour_step(C.byref(P), C.byref(track.c), _d(s), _d(tan), L, _d(_f64(p, (3,))),
                               _d(_f64(omega, (3,))), C.byref(i), C.byref(th))
    return J, i.value, th.value


def weights_update(lam, cost, du, u_nom):
    """cost [K], du [K,N,4], u_nom [N,4] -> (weights [K], u_new [N,4])   eq.(4),(5)."""
    cost = _f64(cost, (-1,)); K = cost.shape[0]
    u_nom = _f64(u_nom, (-1, 4)); N = u_nom.shape[0]
    du = _f64(du, (K, N, 4))
    w = np.zeros(K); un = np.zeros((N, 4))
    lib().orc_weights_update(K, N, float(lam), _d(cost), _d(du), _d(u_nom), _d(w), _d(un))
    return w, un


def step(params, track: Track, x0, start, u_nom, seed, it, want_du=False, want_diag=True, v_nom=None):
    """One MPPI iteration.  Returns dict(u_new [B,N,4], cost [B,K], weights [B,K],
    du [B,K,N,4] | None, margin [B,K], ncross [B,K], aux_end [B,K]); under OBJ_CONTOUR_PAPER (v_nom
    [B,N] required) also v_new [B,N] and dv [B,K,N] | None."""
    P = make_params(params)
    B, K, N = P.B, P.K, P.N
    xdim = 19 if P.objective == OBJ_CONTOUR_PAPER else (17 if P.input_model == 1 else 13)
    x0 = _f64(x0, (B, xdim)); u_nom = _f64(u_nom, (B, N, 4))
    v_new = dv = None
    if P.objective == OBJ_CONTOUR_PAPER:
        v_nom = _f64(v_nom, (B, N)); v_new = np.zeros((B, N)); dv = np.zeros((B, K, N)) if want_du else None
        track.c.v_nom = _d(v_nom); track.c.v_new = _d(v_new)
        track.c.dv_out = _d(dv) if dv is not None else C.cast(None, _dp)
    start = np.ascontiguousarray(np.asarray(start, dtype=np.int32).reshape(B))
    u_new = np.zeros((B, N, 4)); cost = np.zeros((B, K)); w = np.zeros((B, K))
    du = np.zeros((B, K, N, 4)) if want_du else None
    margin = np.zeros((B, K)) if want_diag else None
    ncross = np.zeros((B, K), dtype=np.int32) if want_diag else None
    aux_end = np.zeros((B, K), dtype=np.int32) if want_diag else None
    nd = C.cast(None, _dp); ni = C.cast(None, _ip)
    rc = lib().orc_step(C.byref(P), C.byref(track.c), _d(x0), _i(start), _d(u_nom), int(seed),
                        int(it), _d(u_new), _d(cost), _d(w), _d(du) if want_du else nd,
                        _d(margin) if want_diag else nd, _i(ncross) if want_diag else ni,
                        _i(aux_end) if want_diag else ni)
    if rc != 0:
        raise RuntimeError(f"orc_step failed ({rc})")
    return dict(u_new=u_new, cost=cost, weights=w, du=du, margin=margin, ncross=ncross,
                aux_end=aux_end, v_new=v_new, dv=dv)


def sim_step(params, track: Track, x, start, u_new):
    """Closed-loop glue: -> (x_next [B,13], start_next [B], u_nom_next [B,N,4])."""
    P = make_params(params)
    B, N = P.B, P.N
    x = _f64(x, (B, 17 if P.input_model == 1 else 13)).copy(); u_new = _f64(u_new, (B, N, 4))
    start = np.ascontiguousarray(np.asarray(start, dtype=np.int32).reshape(B)).copy()
    nxt = np.zeros((B, N, 4))
    rc = lib().orc_sim_step(C.byref(P), C.byref(track.c), _d(x), _i(start), _d(u_new), _d(nxt))
    if rc != 0:
        raise RuntimeError(f"orc_sim_step failed ({rc})")
    return x, start, nxt


def sim_step_progress(params, x, u_new, v_new):
    """Closed-loop glue under OBJ_CONTOUR_PAPER [R-39]: -> (x_next [B,19], u_nom_next [B,N,4], v_nom_next [B,N])."""
    P = make_params(params)
    B, N = P.B, P.N
    x = _f64(x, (B, 19)).copy(); u_new = _f64(u_new, (B, N, 4)); v_new = _f64(v_new, (B, N))
    nu = np.zeros((B, N, 4)); nv = np.zeros((B, N))
    rc = lib().orc_sim_step_progress(C.byref(P), _d(x), _d(u_new), _d(nu), _d(v_new), _d(nv))
    if rc != 0:
        raise RuntimeError(f"orc_sim_step_progress failed ({rc})")
    return x, nu, nv


def num_threads() -> int:
    return int(lib().orc_num_threads())
