"""Thin Python binding of libmppi (include/mppi.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for device
buffers and streams, nothing else.  There is no fallback: if libmppi.so is missing or cannot be
loaded, importing this module raises (build it with `python -m paper_2509_14726_b200.build`).
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libmppi.so"

OBJ_GATE, OBJ_TRACK, OBJ_CONTOUR, OBJ_GATE_PAPER, OBJ_CONTOUR_PAPER = 0, 1, 2, 3, 4
PIPE_FUSED, PIPE_TWO_PASS = 0, 1
VARIANT_AUTO, VARIANT_THROUGHPUT, VARIANT_LATENCY, VARIANT_PACKED, VARIANT_PIPELINED, VARIANT_SCAN = 0, 1, 2, 3, 4, 5

EXPORTS = ["mppi_default_params", "mppi_create", "mppi_destroy", "mppi_set_gates",
           "mppi_set_reference", "mppi_set_path", "mppi_step", "mppi_optimize", "mppi_step_host",
           "mppi_sim_step", "mppi_set_prev_front", "mppi_front_flags", "mppi_set_progress", "mppi_sim_step_progress", "mppi_debug_noise", "mppi_get_info", "mppi_launch_count",
           "mppi_error_string", "mppi_last_error", "mppi_measure_fma_peak", "mppi_measure_copy_bw", "mppi_measure_issue_rates", "mppi_measure_launch_floor",
           "mppi_step_static", "mppi_step_static_error"]


class MppiParams(C.Structure):
    """mppi_params of include/mppi.h, field for field."""
    _fields_ = [("struct_size", C.c_uint32), ("K", C.c_int32), ("N", C.c_int32), ("B", C.c_int32),
                ("objective", C.c_int32), ("dt", C.c_float), ("lambda_", C.c_float),
                ("sigma", C.c_float), ("mass", C.c_float), ("Jx", C.c_float), ("Jy", C.c_float),
                ("Jz", C.c_float), ("arm", C.c_float), ("c_tau", C.c_float), ("g", C.c_float),
                ("T_min", C.c_float), ("T_max", C.c_float), ("w_omega", C.c_float),
                ("gate_miss_penalty", C.c_float), ("gate_pass_bonus", C.c_float),
                ("Qp", C.c_float), ("Qv", C.c_float), ("Qq", C.c_float), ("Qw", C.c_float),
                ("R", C.c_float), ("q_contour", C.c_float), ("q_lag", C.c_float),
                ("mu_progress", C.c_float), ("window", C.c_int32), ("pipeline", C.c_int32),
                ("use_graph", C.c_int32), ("block_threads", C.c_int32), ("fast_math", C.c_int32),
                ("store_noise", C.c_int32), ("variant", C.c_int32), ("q_near", C.c_float),
                ("r_near", C.c_float), ("input_model", C.c_int32), ("rate_max", C.c_float),
                ("drag_x", C.c_float), ("drag_y", C.c_float), ("drag_z", C.c_float),
                ("sigma_v", C.c_float), ("dv_max", C.c_float), ("v_theta_max", C.c_float), ("r_dv", C.c_float),
                ("w_limit", C.c_float), ("omega_max", C.c_float), ("near_mode", C.c_int32)]


class MppiInfo(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("block_threads", C.c_int32), ("grid_blocks", C.c_int32),
                ("blocks_per_controller", C.c_int32), ("regs_per_thread", C.c_int32),
                ("static_smem_bytes", C.c_int32), ("dynamic_smem_bytes", C.c_int32),
                ("local_bytes_per_thread", C.c_int32), ("max_blocks_per_sm", C.c_int32),
                ("sm_count", C.c_int32), ("kernels_per_step", C.c_int32), ("samples_per_thread", C.c_int32),
                ("rollout_warps_per_block", C.c_int32), ("l2_bytes", C.c_int32),
                ("scratch_bytes", C.c_int64)]


def _load():
    if not LIB_PATH.exists():
        raise RuntimeError(f"{LIB_PATH} is missing: the CUDA library has not been built "
                           "(python -m paper_2509_14726_b200.build). There is no CPU fallback.")
    L = C.CDLL(str(LIB_PATH))
    vp, fp, ip = C.c_void_p, C.c_void_p, C.c_void_p
    L.mppi_default_params.argtypes = [C.POINTER(MppiParams)]
    L.mppi_create.argtypes = [C.POINTER(MppiParams), C.POINTER(vp)]
    L.mppi_destroy.argtypes = [vp]
    L.mppi_set_gates.argtypes = [vp, fp, C.c_int]
    L.mppi_set_reference.argtypes = [vp, fp, C.c_int]
    L.mppi_set_path.argtypes = [vp, fp, C.c_int, C.c_int]
    L.mppi_step.argtypes = [vp, fp, ip, fp, C.c_uint64, C.c_uint32, fp, fp, fp, vp]
    L.mppi_optimize.argtypes = [vp, fp, ip, fp, C.c_uint64, C.c_uint32, C.c_int, fp, fp, vp]
    L.mppi_step_host.argtypes = [vp, fp, ip, fp, C.c_uint64, C.c_uint32, fp, fp, fp, vp]
    L.mppi_sim_step.argtypes = [vp, fp, ip, fp, fp, vp]
    L.mppi_set_progress.argtypes = [vp, fp, fp]
    L.mppi_sim_step_progress.argtypes = [vp, fp, fp, fp, fp, fp, vp]
    L.mppi_set_prev_front.argtypes = [vp, ip]
    L.mppi_front_flags.argtypes = [vp, fp, ip, fp, ip, vp]
    L.mppi_debug_noise.argtypes = [vp]
    L.mppi_debug_noise.restype = C.c_void_p
    L.mppi_get_info.argtypes = [vp, C.POINTER(MppiInfo)]
    L.mppi_launch_count.argtypes = [vp]
    L.mppi_launch_count.restype = C.c_int64
    L.mppi_error_string.argtypes = [C.c_int]
    L.mppi_error_string.restype = C.c_char_p
    L.mppi_last_error.argtypes = [vp]
    L.mppi_last_error.restype = C.c_char_p
    L.mppi_measure_fma_peak.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.mppi_measure_copy_bw.argtypes = [C.c_int64, C.c_int, C.POINTER(C.c_double)]
    L.mppi_measure_issue_rates.argtypes = [C.POINTER(C.c_double), C.c_int]
    L.mppi_measure_launch_floor.argtypes = [C.c_int, C.POINTER(C.c_double)]
    L.mppi_step_static.argtypes = [C.POINTER(MppiParams), fp, C.c_int, fp, ip, fp, C.c_uint64, C.c_uint32, fp, fp, fp, vp]
    L.mppi_step_static_error.argtypes = []
    L.mppi_step_static_error.restype = C.c_char_p
    for name in EXPORTS:
        getattr(L, name)            # AttributeError here = the library is stale: rebuild it
    return L


lib = _load()


class MppiError(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = int(status)
        text = lib.mppi_error_string(int(status)).decode()
        super().__init__(f"libmppi: {text} ({status})" + (f": {detail}" if detail else ""))


def default_params() -> MppiParams:
    p = MppiParams()
    rc = lib.mppi_default_params(C.byref(p))
    if rc:
        raise MppiError(rc)
    return p


def make_params(d: dict | None = None, **over) -> MppiParams:
    """dict with the keys of mppi_params ('lambda' accepted for lambda_) -> C struct."""
    p = default_params()
    src = dict(d or {})
    src.update(over)
    if "lambda" in src:
        src["lambda_"] = src.pop("lambda")
    names = {f for f, _ in MppiParams._fields_}
    for k, v in src.items():
        if k not in names or k == "struct_size":
            raise KeyError(f"mppi_params has no field '{k}'")
        setattr(p, k, v)
    return p


def _host_f32(a, shape):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float32))
    try:
        return a.reshape(shape)
    except ValueError:
        raise ValueError(f"expected shape {shape}, got {a.shape}") from None


def _stream_ptr(stream):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


class Mppi:
    """One libmppi context.  Device arguments are torch CUDA tensors (float32 / int32,
    contiguous); the methods check shape, dtype and device and pass raw pointers through."""

    def __init__(self, params=None, **over):
        if isinstance(params, MppiParams):
            base = {f: getattr(params, f) for f, _ in MppiParams._fields_ if f != "struct_size"}
        else:
            base = dict(params or {})
        self.params = make_params(base, **over)
        h = C.c_void_p()
        rc = lib.mppi_create(C.byref(self.params), C.byref(h))
        if rc:
            raise MppiError(rc, lib.mppi_last_error(None).decode())
        self._h = h
        self.K, self.N, self.B = self.params.K, self.params.N, self.params.B
        self._v = None
        self.xdim = 19 if self.params.objective == OBJ_CONTOUR_PAPER else 17 if self.params.input_model == 1 else 13

    # -- lifetime
    def close(self):
        if getattr(self, "_h", None):
            lib.mppi_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, rc):
        if rc:
            raise MppiError(rc, lib.mppi_last_error(self._h).decode())

    # -- tracks (host arrays)
    def set_gates(self, gates):
        g = _host_f32(gates, (-1, 11))
        self._ck(lib.mppi_set_gates(self._h, g.ctypes.data, g.shape[0]))

    def set_reference(self, ref):
        r = np.ascontiguousarray(np.asarray(ref, dtype=np.float32)).reshape(-1, 13)
        self._ck(lib.mppi_set_reference(self._h, r.ctypes.data, r.shape[0]))

    def set_path(self, pts, closed=True):
        p = np.ascontiguousarray(np.asarray(pts, dtype=np.float32)).reshape(-1, 3)
        self._ck(lib.mppi_set_path(self._h, p.ctypes.data, p.shape[0], 1 if closed else 0))

    def set_track(self, wl):
        """Convenience: feed whichever of gates / ref / path a workloads.Workload carries."""
        if wl.gates is not None:
            self.set_gates(wl.gates)
        if getattr(wl, "prev_front", None) is not None:
            import torch
            self.set_prev_front(torch.from_numpy(np.ascontiguousarray(wl.prev_front, dtype=np.int32)).cuda())
        if wl.ref is not None:
            self.set_reference(wl.ref)
        if wl.path is not None:
            self.set_path(wl.path, wl.closed)
        if getattr(wl, "v_nom", None) is not None and self.params.objective == OBJ_CONTOUR_PAPER:
            import torch
            v = torch.from_numpy(np.ascontiguousarray(wl.v_nom, dtype=np.float32)).cuda()
            self.set_progress(v, torch.empty_like(v))

    # -- device calls
    @staticmethod
    def _dev(t, shape, dtype):
        import torch
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()
                and tuple(t.shape) == tuple(shape)):
            raise ValueError(f"need a contiguous CUDA {dtype} tensor of shape {tuple(shape)}")
        return C.c_void_p(t.data_ptr())

    def step(self, x0, start, u_nom, seed, it, u_new=None, cost=None, weights=None, stream=None):
        import torch
        B, N, K = self.B, self.N, self.K
        dev = x0.device
        u_new = torch.empty((B, N, 4), dtype=torch.float32, device=dev) if u_new is None else u_new
        cost = torch.empty((B, K), dtype=torch.float32, device=dev) if cost is None else cost
        weights = torch.empty((B, K), dtype=torch.float32, device=dev) if weights is None else weights
        self._ck(lib.mppi_step(self._h, self._dev(x0, (B, self.xdim), torch.float32),
                               self._dev(start, (B,), torch.int32),
                               self._dev(u_nom, (B, N, 4), torch.float32), C.c_uint64(int(seed)),
                               C.c_uint32(int(it)), self._dev(u_new, (B, N, 4), torch.float32),
                               self._dev(cost, (B, K), torch.float32),
                               self._dev(weights, (B, K), torch.float32), _stream_ptr(stream)))
        return u_new, cost, weights

    def optimize(self, x0, start, u, seed, it0, n_iters, cost=None, weights=None, stream=None):
        import torch
        B, N, K = self.B, self.N, self.K
        dev = x0.device
        cost = torch.empty((B, K), dtype=torch.float32, device=dev) if cost is None else cost
        weights = torch.empty((B, K), dtype=torch.float32, device=dev) if weights is None else weights
        self._ck(lib.mppi_optimize(self._h, self._dev(x0, (B, self.xdim), torch.float32),
                                   self._dev(start, (B,), torch.int32),
                                   self._dev(u, (B, N, 4), torch.float32), C.c_uint64(int(seed)),
                                   C.c_uint32(int(it0)), int(n_iters),
                                   self._dev(cost, (B, K), torch.float32),
                                   self._dev(weights, (B, K), torch.float32), _stream_ptr(stream)))
        return u, cost, weights

    def step_host(self, x0, start, u_nom, seed, it, u_new=None, cost=None, weights=None,
                  want_cost=True, stream=None):
        """Host buffers in, host buffers out (numpy, or pinned torch CPU tensors via .numpy())."""
        B, N, K = self.B, self.N, self.K
        x0 = _host_f32(x0, (B, self.xdim)); u_nom = _host_f32(u_nom, (B, N, 4))
        start = np.ascontiguousarray(np.asarray(start, dtype=np.int32)).reshape(B)
        u_new = np.empty((B, N, 4), np.float32) if u_new is None else u_new
        if want_cost:
            cost = np.empty((B, K), np.float32) if cost is None else cost
            weights = np.empty((B, K), np.float32) if weights is None else weights
        self._ck(lib.mppi_step_host(self._h, x0.ctypes.data, start.ctypes.data, u_nom.ctypes.data,
                                    C.c_uint64(int(seed)), C.c_uint32(int(it)), u_new.ctypes.data,
                                    cost.ctypes.data if cost is not None else None,
                                    weights.ctypes.data if weights is not None else None,
                                    _stream_ptr(stream)))
        return u_new, cost, weights

    def step_host_fn(self, x0, start, u_nom, u_new, cost=None, weights=None, stream=None):
        """Pre-marshalled mppi_step_host: checks the (numpy, C-contiguous) host buffers once and
        returns f(seed, it) that only passes the stored pointers through -- for control loops that
        call every cycle with the same buffers.  The arrays must stay alive and in place."""
        B, N, K = self.B, self.N, self.K

        def chk(a, shape, dtype):
            if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"]
                    and a.size == int(np.prod(shape))):
                raise ValueError(f"need a C-contiguous {np.dtype(dtype).name} array with {int(np.prod(shape))} elements")
            return C.c_void_p(a.ctypes.data)
        px0, pst, pu = chk(x0, (B, self.xdim), np.float32), chk(start, (B,), np.int32), chk(u_nom, (B, N, 4), np.float32)
        pun = chk(u_new, (B, N, 4), np.float32)
        pc = chk(cost, (B, K), np.float32) if cost is not None else None
        pw = chk(weights, (B, K), np.float32) if weights is not None else None
        ps = _stream_ptr(stream)
        h, fn, ck, u64, u32 = self._h, lib.mppi_step_host, self._ck, C.c_uint64, C.c_uint32

        def call(seed, it):
            ck(fn(h, px0, pst, pu, u64(seed), u32(it), pun, pc, pw, ps))
        return call

    def sim_step(self, x, start, u_new, u_nom_next=None, stream=None):
        import torch
        B, N = self.B, self.N
        u_nom_next = torch.empty_like(u_new) if u_nom_next is None else u_nom_next
        self._ck(lib.mppi_sim_step(self._h, self._dev(x, (B, self.xdim), torch.float32),
                                   self._dev(start, (B,), torch.int32),
                                   self._dev(u_new, (B, N, 4), torch.float32),
                                   self._dev(u_nom_next, (B, N, 4), torch.float32),
                                   _stream_ptr(stream)))
        return x, start, u_nom_next

    def set_progress(self, v_nom, v_new=None):
        """Objective 4: v_nom / v_new CUDA float32 tensors [B, N] (kept alive here); v_new=None = in place."""
        import torch
        v_new = v_nom if v_new is None else v_new
        self._v = (v_nom, v_new)
        self._ck(lib.mppi_set_progress(self._h, self._dev(v_nom, (self.B, self.N), torch.float32),
                                       self._dev(v_new, (self.B, self.N), torch.float32)))

    def sim_step_progress(self, x, u_new, v_new, u_nom_next=None, v_nom_next=None, stream=None):
        """Objective 4: plant step on rows of 19 + shift of both nominals (in place when the outputs are None)."""
        import torch
        B, N = self.B, self.N
        u_nom_next = u_new if u_nom_next is None else u_nom_next
        v_nom_next = v_new if v_nom_next is None else v_nom_next
        self._ck(lib.mppi_sim_step_progress(self._h, self._dev(x, (B, 19), torch.float32),
                                            self._dev(u_new, (B, N, 4), torch.float32),
                                            self._dev(u_nom_next, (B, N, 4), torch.float32),
                                            self._dev(v_new, (B, N), torch.float32),
                                            self._dev(v_nom_next, (B, N), torch.float32), _stream_ptr(stream)))
        return x, u_nom_next, v_nom_next

    def set_prev_front(self, prev_front):
        """prev_front: CUDA int32 tensor [B, N+1] (kept alive by this object), or None."""
        import torch
        if prev_front is None:
            self._prev_front = None
            self._ck(lib.mppi_set_prev_front(self._h, None))
            return
        self._prev_front = prev_front
        self._ck(lib.mppi_set_prev_front(self._h, self._dev(prev_front, (self.B, self.N + 1), torch.int32)))

    def front_flags(self, x0, start, u, out=None, stream=None):
        import torch
        B, N = self.B, self.N
        out = torch.empty((B, N + 1), dtype=torch.int32, device=x0.device) if out is None else out
        self._ck(lib.mppi_front_flags(self._h, self._dev(x0, (B, self.xdim), torch.float32),
                                      self._dev(start, (B,), torch.int32),
                                      self._dev(u, (B, N, 4), torch.float32),
                                      self._dev(out, (B, N + 1), torch.int32), _stream_ptr(stream)))
        return out

    def debug_noise(self):
        """dU [B,N,K,4] of the last step as a torch tensor copy, or None if the context keeps none."""
        import torch
        ptr = lib.mppi_debug_noise(self._h)
        if not ptr:
            return None
        shape = (self.B, self.N, self.K, 4)

        class _View:
            __cuda_array_interface__ = {"shape": shape, "typestr": "<f4", "data": (int(ptr), False),
                                        "version": 3, "strides": None}
        torch.cuda.synchronize()
        return torch.as_tensor(_View(), device="cuda").clone()

    def info(self) -> dict:
        o = MppiInfo()
        o.struct_size = C.sizeof(MppiInfo)
        self._ck(lib.mppi_get_info(self._h, C.byref(o)))
        return {f: getattr(o, f) for f, _ in MppiInfo._fields_ if f != "struct_size"}

    def launch_count(self) -> int:
        return int(lib.mppi_launch_count(self._h))


def measure_fma_peak(reps=5):
    t, f = C.c_double(), C.c_double()
    rc = lib.mppi_measure_fma_peak(int(reps), C.byref(t), C.byref(f))
    if rc:
        raise MppiError(rc)
    return t.value, f.value


def measure_copy_bw(nbytes=1 << 30, reps=5):
    g = C.c_double()
    rc = lib.mppi_measure_copy_bw(int(nbytes), int(reps), C.byref(g))
    if rc:
        raise MppiError(rc)
    return g.value


ISSUE_RATE_CLASSES = ("ffma_rrr", "ffma_const", "ffma2_rrr", "fmul", "fadd", "philox_half_round", "mufu", "fmnmx")


def measure_issue_rates() -> dict:
    """cycles per warp-instruction per SM sub-partition at saturation, by instruction class (mppi_measure_issue_rates)."""
    a = (C.c_double * len(ISSUE_RATE_CLASSES))()
    rc = lib.mppi_measure_issue_rates(a, len(ISSUE_RATE_CLASSES))
    if rc:
        raise MppiError(rc)
    return dict(zip(ISSUE_RATE_CLASSES, (float(v) for v in a)))


def measure_launch_floor(reps=400) -> float:
    """median event-to-event time of an empty 128 x 256 kernel behind a busy GPU, microseconds."""
    v = C.c_double()
    rc = lib.mppi_measure_launch_floor(int(reps), C.byref(v))
    if rc:
        raise MppiError(rc)
    return v.value


STATIC_MAX = dict(K=8192, N=64, B=4, G=64)      # MPPI_STATIC_MAX_* of include/mppi.h


def step_static(params, gates, x0, start, u_nom, seed, it, u_new, cost, weights, stream=None):
    """mppi_step_static: one gate-progress iteration that allocates nothing (scratch in a static device array; limits
    STATIC_MAX).  params: dict / MppiParams; every other argument a contiguous CUDA tensor the CALLER allocated:
    gates [G,11] f32, x0 [B,13] f32, start [B] i32, u_nom / u_new [B,N,4] f32, cost / weights [B,K] f32.
    Calls on one device must not overlap on the GPU."""
    import torch
    P = params if isinstance(params, MppiParams) else make_params(params)
    B, N, K = P.B, P.N, P.K
    G = int(gates.shape[0])
    dev = Mppi._dev
    rc = lib.mppi_step_static(C.byref(P), dev(gates, (G, 11), torch.float32), G, dev(x0, (B, 13), torch.float32),
                              dev(start, (B,), torch.int32), dev(u_nom, (B, N, 4), torch.float32), C.c_uint64(int(seed)),
                              C.c_uint32(int(it)), dev(u_new, (B, N, 4), torch.float32), dev(cost, (B, K), torch.float32),
                              dev(weights, (B, K), torch.float32), _stream_ptr(stream))
    if rc:
        raise MppiError(rc, lib.mppi_step_static_error().decode())
    return u_new, cost, weights
