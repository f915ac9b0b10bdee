"""ctypes binding of libdg (include/dg.h).  Same names as the C entry points, minus the prefix."""
from __future__ import annotations

import ctypes as C
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libdg.so")

DG_TUNE_ROWS_PER_CTA = 1
DG_TUNE_FUSED_CFL = 2
DG_TUNE_GEN_PREFETCH = 3
DG_TUNE_RK4_FORM = 4
DG_TUNE_STAGE_IMPL = 5

EXPORTS = [
    "dg_workspace_bytes", "dg_init", "dg_set_state", "dg_set_state_host", "dg_get_state",
    "dg_get_state_host", "dg_rhs", "dg_cfl_dt", "dg_step", "dg_step_debug", "dg_run_host",
    "dg_time", "dg_set_time", "dg_launch_count", "dg_set_tuning", "dg_stage_timing",
    "dg_stage_time_ms", "dg_stage_times_ms", "dg_probe_fp64_peak", "dg_last_error", "dg_destroy",
    "dg_rk_stages", "dg_limit", "dg_torque", "dg_torque_normalised",
    "dg_step_begin", "dg_substep", "dg_substep_part", "dg_step_end", "dg_halo_layout",
    "dg_static_setup", "dg_torque_static", "dg_static_last_error",
]


class DGError(RuntimeError):
    pass


class DGParams(C.Structure):
    """Mirror of ``dg_params`` (include/dg.h)."""
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32),
        ("x0", C.c_double), ("x1", C.c_double), ("y0", C.c_double), ("y1", C.c_double),
        ("order", C.c_int32), ("rk", C.c_int32), ("bc", C.c_int32), ("eos", C.c_int32),
        ("gamma", C.c_double), ("h_aspect", C.c_double),
        ("gm_star", C.c_double), ("eps_star", C.c_double),
        ("q_planet", C.c_double), ("r_planet", C.c_double), ("eps_planet", C.c_double),
        ("omega_planet", C.c_double), ("phase0", C.c_double),
        ("damp_r0", C.c_double), ("damp_r1", C.c_double), ("t0", C.c_double),
        ("limiter", C.c_int32), ("lim_eps", C.c_double),
        ("flux", C.c_int32),
        ("damp_in_r0", C.c_double), ("damp_in_r1", C.c_double),
        ("halo_south", C.c_int32), ("halo_north", C.c_int32),
        ("damp_mode", C.c_int32),
    ]


def params_struct(p: dict) -> DGParams:
    s = DGParams()
    for name, _ in DGParams._fields_:
        setattr(s, name, p[name])
    return s


_lib = None


def load_library(path: str | None = None):
    """dlopen libdg.so and declare the signatures.  Fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or _LIB_PATH
    if not os.path.exists(path):
        raise DGError(f"{path} not found: build it with `python -m paper_1805_01443_b200.build` "
                      "(there is no CPU fallback)")
    L = C.CDLL(path)
    vp, d, i, ll = C.c_void_p, C.c_double, C.c_int, C.c_longlong
    PP = C.POINTER(DGParams)
    sig = {
        "dg_workspace_bytes": (C.c_size_t, [PP]),
        "dg_init": (i, [PP, vp, C.c_size_t, vp, C.POINTER(vp)]),
        "dg_set_state": (i, [vp, vp]), "dg_set_state_host": (i, [vp, vp]),
        "dg_get_state": (i, [vp, vp]), "dg_get_state_host": (i, [vp, vp]),
        "dg_rhs": (i, [vp, d, vp]),
        "dg_cfl_dt": (i, [vp, d, C.POINTER(d)]),
        "dg_step": (i, [vp, d]), "dg_step_debug": (i, [vp, d, vp]),
        "dg_run_host": (i, [vp, vp, i, d, vp]),
        "dg_time": (d, [vp]), "dg_set_time": (i, [vp, d]),
        "dg_launch_count": (ll, [vp]),
        "dg_set_tuning": (i, [vp, i, i]),
        "dg_stage_timing": (i, [vp, i]),
        "dg_stage_time_ms": (i, [vp, C.POINTER(d), C.POINTER(ll)]),
        "dg_stage_times_ms": (i, [vp, C.POINTER(d), ll, C.POINTER(ll)]),
        "dg_probe_fp64_peak": (i, [vp, C.POINTER(d)]),
        "dg_last_error": (C.c_char_p, [vp]),
        "dg_destroy": (None, [vp]),
        "dg_step_begin": (i, [vp, d]), "dg_substep": (i, [vp]), "dg_substep_part": (i, [vp, i]), "dg_step_end": (i, [vp]),
        "dg_halo_layout": (i, [vp, C.POINTER(C.c_size_t), C.POINTER(C.c_size_t)]),
        "dg_rk_stages": (i, [i]), "dg_limit": (i, [vp]), "dg_torque": (i, [vp, d, C.POINTER(d)]),
        "dg_torque_normalised": (i, [vp, d, d, C.POINTER(d)]),
        "dg_static_setup": (i, []), "dg_torque_static": (i, [PP, vp, d, vp, vp]),
        "dg_static_last_error": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(L, name)
        fn.restype, fn.argtypes = res, args
    _lib = L
    return L


def static_setup():
    """dg_static_setup: look up the library's static scratch on the current device (once per device)."""
    L = load_library()
    if L.dg_static_setup() != 0:
        raise DGError(L.dg_static_last_error().decode())


def torque_static(params: dict, U, t: float, out, stream=None):
    """dg_torque_static: torque of Eq.(6) from a modal DEVICE state ``U`` into the DEVICE tensor ``out`` (3 doubles),
    on ``stream`` (default: torch's current stream).  No context, no workspace, nothing allocated, nothing synchronised."""
    import torch
    L = load_library()
    for x in (U, out):
        if not (x.is_cuda and x.dtype == torch.float64 and x.is_contiguous()):
            raise DGError("torque_static: U and out must be contiguous fp64 CUDA tensors")
    m = int(params["order"])
    if U.numel() != int(params["ny"]) * int(params["nx"]) * 4 * m * m or out.numel() < 3:
        raise DGError("torque_static: U must hold ny*nx*4*m*m doubles and out at least 3")
    ps = params_struct(params)
    s = stream if stream is not None else torch.cuda.current_stream()
    e = L.dg_torque_static(C.byref(ps), U.data_ptr(), float(t), out.data_ptr(), s.cuda_stream)
    if e != 0:
        raise DGError(f"dg_torque_static: {e}: {L.dg_static_last_error().decode()}")
    return out


class DG:
    """One DG context on the current CUDA device.

    ``params``: dict with the fields of ``dg_params`` (see ``workloads.make_params``).
    Device buffers are torch tensors (fp64, cuda); host buffers are torch CPU tensors or NumPy
    arrays (pinned torch tensors make the copies asynchronous).
    """

    def __init__(self, params: dict, stream=None, extra_workspace_bytes: int = 0):
        import torch
        if not torch.cuda.is_available():
            raise DGError("no CUDA device: libdg has no CPU fallback")
        self._torch = torch
        self.L = load_library()
        self.params = dict(params)
        self.m = int(params["order"])
        self.shape = (int(params["ny"]), int(params["nx"]), 4, self.m, self.m)
        self.ncoef = 1
        for s in self.shape:
            self.ncoef *= s
        ps = params_struct(params)
        nbytes = self.L.dg_workspace_bytes(C.byref(ps))
        if nbytes == 0:
            raise DGError("invalid dg_params")
        nbytes += int(extra_workspace_bytes)             # e.g. two state arrays for DG_TUNE_RK4_FORM = 0 (include/dg.h)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device="cuda")
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self.stream = stream if stream is not None else torch.cuda.current_stream()
        self._h = C.c_void_p()
        e = self.L.dg_init(C.byref(ps), C.c_void_p(self._ws_ptr), nbytes,
                           C.c_void_p(self.stream.cuda_stream), C.byref(self._h))
        if e != 0:
            raise DGError(f"dg_init failed ({e})")

    # -- helpers ------------------------------------------------------------------------------
    def _chk(self, e: int, what: str):
        if e != 0:
            msg = self.L.dg_last_error(self._h)
            raise DGError(f"{what} failed ({e}): {msg.decode() if msg else ''}")

    def _dev(self, t, n=None):
        torch = self._torch
        assert t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
        assert t.numel() == (self.ncoef if n is None else n), (t.shape, self.shape)
        return C.c_void_p(t.data_ptr())

    def _host(self, a):
        torch = self._torch
        if isinstance(a, torch.Tensor):
            assert not a.is_cuda and a.dtype == torch.float64 and a.is_contiguous()
            assert a.numel() == self.ncoef
            return C.c_void_p(a.data_ptr())
        import numpy as np
        assert isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags.c_contiguous
        assert a.size == self.ncoef
        return C.c_void_p(a.ctypes.data)

    def new_device_state(self, extra=()):
        return self._torch.empty(tuple(extra) + self.shape, dtype=self._torch.float64, device="cuda")

    # -- the C entry points -------------------------------------------------------------------
    def set_state(self, U_dev):
        self._chk(self.L.dg_set_state(self._h, self._dev(U_dev)), "dg_set_state")

    def set_state_host(self, U_host):
        self._chk(self.L.dg_set_state_host(self._h, self._host(U_host)), "dg_set_state_host")

    def get_state(self, out=None):
        out = self.new_device_state() if out is None else out
        self._chk(self.L.dg_get_state(self._h, self._dev(out)), "dg_get_state")
        return out

    def get_state_host(self, out):
        self._chk(self.L.dg_get_state_host(self._h, self._host(out)), "dg_get_state_host")
        return out

    def rhs(self, t: float, out=None):
        out = self.new_device_state() if out is None else out
        self._chk(self.L.dg_rhs(self._h, float(t), self._dev(out)), "dg_rhs")
        return out

    def cfl_dt(self, cfl: float) -> float:
        dt = C.c_double()
        self._chk(self.L.dg_cfl_dt(self._h, float(cfl), C.byref(dt)), "dg_cfl_dt")
        return dt.value

    def step(self, dt: float):
        self._chk(self.L.dg_step(self._h, float(dt)), "dg_step")

    def step_debug(self, dt: float, out=None):
        rk = int(self.L.dg_rk_stages(int(self.params["rk"])))
        out = self.new_device_state((rk,)) if out is None else out
        self._chk(self.L.dg_step_debug(self._h, float(dt), self._dev(out, rk * self.ncoef)), "dg_step_debug")
        return out

    def step_begin(self, dt: float):
        self._chk(self.L.dg_step_begin(self._h, float(dt)), "dg_step_begin")

    def substep(self):
        self._chk(self.L.dg_substep(self._h), "dg_substep")

    def substep_part(self, part: int):
        self._chk(self.L.dg_substep_part(self._h, int(part)), "dg_substep_part")

    def step_end(self):
        self._chk(self.L.dg_step_end(self._h), "dg_step_end")

    @property
    def rk_stages(self) -> int:
        return int(self.L.dg_rk_stages(int(self.params["rk"])))

    def halo_rows(self):
        """Views into the workspace (flat fp64 tensors, internal layout): (first row, last row) of the array the
        next stage kernel reads, and (south halo, north halo) (None at a domain boundary)."""
        off = (C.c_size_t * 4)()
        nb = C.c_size_t()
        self._chk(self.L.dg_halo_layout(self._h, off, C.byref(nb)), "dg_halo_layout")
        base = self._ws_ptr - self.workspace.data_ptr()

        def view(o):
            if o == C.c_size_t(-1).value:
                return None
            return self.workspace[base + o: base + o + nb.value].view(self._torch.float64)

        return (view(off[0]), view(off[1])), (view(off[2]), view(off[3]))

    def limit(self):
        self._chk(self.L.dg_limit(self._h), "dg_limit")

    def torque(self, t: float) -> float:
        g = C.c_double()
        self._chk(self.L.dg_torque(self._h, float(t), C.byref(g)), "dg_torque")
        return g.value

    def torque_normalised(self, t: float, sigma_p: float) -> float:
        g = C.c_double()
        self._chk(self.L.dg_torque_normalised(self._h, float(t), float(sigma_p), C.byref(g)), "dg_torque_normalised")
        return g.value

    def run_host(self, U_in, nsteps: int, cfl: float, U_out):
        self._chk(self.L.dg_run_host(self._h, self._host(U_in), int(nsteps), float(cfl),
                                     self._host(U_out)), "dg_run_host")
        return U_out

    @property
    def time(self) -> float:
        return float(self.L.dg_time(self._h))

    @time.setter
    def time(self, t: float):
        self._chk(self.L.dg_set_time(self._h, float(t)), "dg_set_time")

    @property
    def launch_count(self) -> int:
        return int(self.L.dg_launch_count(self._h))

    def set_tuning(self, key: int, value: int):
        self._chk(self.L.dg_set_tuning(self._h, int(key), int(value)), "dg_set_tuning")

    def stage_timing(self, enable: bool):
        self._chk(self.L.dg_stage_timing(self._h, 1 if enable else 0), "dg_stage_timing")

    def stage_time_ms(self):
        ms, n = C.c_double(), C.c_longlong()
        self._chk(self.L.dg_stage_time_ms(self._h, C.byref(ms), C.byref(n)), "dg_stage_time_ms")
        return ms.value, n.value

    def stage_times_ms(self, capacity: int = 4096):
        buf, n = (C.c_double * capacity)(), C.c_longlong()
        self._chk(self.L.dg_stage_times_ms(self._h, buf, capacity, C.byref(n)), "dg_stage_times_ms")
        return list(buf[:n.value])

    def probe_fp64_peak(self) -> float:
        tf = C.c_double()
        self._chk(self.L.dg_probe_fp64_peak(self._h, C.byref(tf)), "dg_probe_fp64_peak")
        return tf.value

    def close(self):
        if getattr(self, "_h", None):
            self.L.dg_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
