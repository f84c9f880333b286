"""Thin Python binding of libphx (include/phx.h): argument marshalling only.

Every step of the method runs in the CUDA kernels of libphx.so.  PyTorch is used for device memory
(the workspace tensor), streams and pinned host buffers.  There is no CPU fallback: if the shared
library is missing, or there is no CUDA device, the calls raise.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libphx.so")

PHX_OK, PHX_ERR_INVALID_ARG, PHX_ERR_BAD_STATE, PHX_ERR_UNSUPPORTED, PHX_ERR_CUDA, PHX_ERR_WORKSPACE = range(6)
PHX_WARN_UNSTABLE = 100
PHX_C32, PHX_C64 = 0, 1
PHX_SCALAR, PHX_RESERVOIR, PHX_SPINOR, PHX_SPINOR_RESERVOIR = range(4)
PHX_HOST, PHX_DEVICE = 0, 1
PHX_PSI, PHX_PSI_MINUS, PHX_N, PHX_N_MINUS = range(4)
PHX_BC_PERIODIC, PHX_BC_ZERO = 0, 1
PHX_VARIANT_AUTO, PHX_VARIANT_STAGE, PHX_VARIANT_STEP, PHX_VARIANT_RESIDENT = 0, 1, 3, 4
PHX_NCOEF = 18

MODELS = {"scalar": PHX_SCALAR, "reservoir": PHX_RESERVOIR, "spinor": PHX_SPINOR, "spinor_reservoir": PHX_SPINOR_RESERVOIR}
PRECS = {"c32": PHX_C32, "c64": PHX_C64}
FIELDS = {"psi_p": PHX_PSI, "psi_m": PHX_PSI_MINUS, "n_p": PHX_N, "n_m": PHX_N_MINUS}
PHX_INT_RK4, PHX_INT_DP54 = 0, 1
INTEGRATORS = {"rk4": PHX_INT_RK4, "dp54": PHX_INT_DP54}
EXPORTS = ("phx_workspace_bytes", "phx_create_grid", "phx_set_params", "phx_set_potential_pump", "phx_set_drive",
           "phx_set_field", "phx_read_field", "phx_step_rk4", "phx_step_adaptive", "phx_get_adaptive_state", "phx_set_time",
           "phx_get_step", "phx_set_step",
           "phx_ensemble_mean_density", "phx_get_coeffs", "phx_debug_noise_u32", "phx_select_variant",
           "phx_get_variant", "phx_get_launch_count", "phx_set_tuning", "phx_sync", "phx_last_error",
           "phx_destroy_grid", "phx_step_rk4_static", "phx_check_finite")
PHX_STATIC_SCRATCH_BYTES = 8 << 20


class phx_grid_desc(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("batch", C.c_int32), ("dx", C.c_double), ("dy", C.c_double),
                ("prec", C.c_int32), ("model", C.c_int32), ("noise", C.c_int32), ("bc_x", C.c_int32),
                ("bc_y", C.c_int32), ("integrator", C.c_int32), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("stream", C.c_void_p)]


class phx_params(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("hbar", "m", "g", "g_x", "g_r", "R", "gamma_c", "gamma_r", "beta", "dt",
                                          "noise_scale", "density_offset", "omega")] + [("seed", C.c_uint32)]


class phx_adaptive(C.Structure):
    _fields_ = [("atol", C.c_double), ("rtol", C.c_double), ("h_init", C.c_double), ("h_min", C.c_double),
                ("h_max", C.c_double), ("max_attempts", C.c_int64)]


class phx_adaptive_state(C.Structure):
    _fields_ = [("t", C.c_double), ("h_next", C.c_double), ("n_accept", C.c_int64), ("n_reject", C.c_int64),
                ("attempts", C.c_int64), ("err_last", C.c_double)]


class PhxError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"libphx status {status}: {msg}")
        self.status = status


_lib = None


def lib():
    """Loads libphx.so (built in-tree by paper_2411_18341_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: run `python -m paper_2411_18341_b200.build` (no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint64
        L.phx_workspace_bytes.restype = C.c_size_t
        L.phx_workspace_bytes.argtypes = [vp]
        sigs = {
            "phx_create_grid": [vp, vp], "phx_set_params": [vp, vp], "phx_set_potential_pump": [vp, vp, vp, i32],
            "phx_set_drive": [vp, vp, i32], "phx_set_field": [vp, i32, vp, i32], "phx_read_field": [vp, i32, vp, i32],
            "phx_step_rk4": [vp, i64], "phx_get_step": [vp, vp], "phx_set_step": [vp, u64],
            "phx_step_adaptive": [vp, C.c_double, vp], "phx_get_adaptive_state": [vp, vp, vp, vp, vp, vp, i64, vp],
            "phx_set_time": [vp, C.c_double, C.c_double],
            "phx_ensemble_mean_density": [vp, i32, vp, i32], "phx_get_coeffs": [vp, vp, i32],
            "phx_debug_noise_u32": [vp, u64, vp, i32], "phx_select_variant": [vp, i32], "phx_get_variant": [vp, vp],
            "phx_get_launch_count": [vp, vp], "phx_set_tuning": [vp, C.c_char_p, i32], "phx_sync": [vp],
            "phx_check_finite": [vp, vp],
            "phx_step_rk4_static": [i32, i32, C.c_double, C.c_double, i32, i32, i32, vp, vp, vp, vp, i64, vp],
        }
        for name, args in sigs.items():
            fn = getattr(L, name)
            fn.restype = i32
            fn.argtypes = args
        L.phx_last_error.restype = C.c_char_p
        L.phx_last_error.argtypes = [vp]
        L.phx_destroy_grid.restype = None
        L.phx_destroy_grid.argtypes = [vp]
        _lib = L
    return _lib


def make_params(**kw) -> phx_params:
    d = dict(hbar=1.0, m=0.5, g=0.0, g_x=0.0, g_r=0.0, R=0.0, gamma_c=0.0, gamma_r=0.0, beta=0.0, dt=0.0,
             noise_scale=1.0, density_offset=0.0, omega=0.0, seed=0)
    for k in kw:
        if k not in d:
            raise KeyError(k)
    d.update(kw)
    return phx_params(**d)


def _addr(buf):
    """(address, phx_mem) of a numpy array (host) or torch tensor (host or device); None -> (None, HOST)."""
    if buf is None:
        return None, PHX_HOST
    if isinstance(buf, np.ndarray):
        if not buf.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be C-contiguous")
        return buf.ctypes.data, PHX_HOST
    import torch
    if isinstance(buf, torch.Tensor):
        if not buf.is_contiguous():
            raise ValueError("tensor must be contiguous")
        return buf.data_ptr(), (PHX_DEVICE if buf.is_cuda else PHX_HOST)
    raise TypeError(type(buf))


class Grid:
    """One phx_grid handle plus the torch tensor that backs its workspace.  Method names mirror the C ABI."""

    def __init__(self, nx, ny, dx, dy, model="scalar", prec="c32", batch=1, noise=False, bc=(0, 0), stream=None,
                 device="cuda:0", integrator="rk4"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("libphx needs a CUDA device (no CPU fallback)")
        self._lib = lib()
        self.nx, self.ny, self.batch, self.model, self.prec = int(nx), int(ny), int(batch), model, prec
        self.cdtype = np.complex64 if prec == "c32" else np.complex128
        self.rdtype = np.float32 if prec == "c32" else np.float64
        self.desc = phx_grid_desc(self.nx, self.ny, self.batch, float(dx), float(dy), PRECS[prec], MODELS[model],
                                  int(bool(noise)), int(bc[0]), int(bc[1]), INTEGRATORS[integrator], None, 0, None)
        nbytes = self._lib.phx_workspace_bytes(C.byref(self.desc))
        if nbytes == 0:
            raise PhxError(PHX_ERR_INVALID_ARG, "invalid grid descriptor")
        self.device = torch.device(device)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        aligned = (base + 255) // 256 * 256
        self.desc.workspace = aligned
        self.desc.workspace_bytes = nbytes
        self.stream = stream
        self.desc.stream = None if stream is None else stream.cuda_stream
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            st = self._lib.phx_create_grid(C.byref(self._h), C.byref(self.desc))
        if st != PHX_OK:
            raise PhxError(st, "phx_create_grid failed")

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, st, allow_warn=True):
        if st == PHX_OK or (allow_warn and st >= 100):
            return st
        raise PhxError(st, self._lib.phx_last_error(self._h).decode())

    def _field_shape_dtype(self, field):
        f = FIELDS[field] if isinstance(field, str) else field
        return f, (self.batch, self.ny, self.nx), (self.cdtype if f in (PHX_PSI, PHX_PSI_MINUS) else self.rdtype)

    # -- C ABI, one to one -------------------------------------------------------------------------
    def set_params(self, params=None, **kw):
        p = params if params is not None else make_params(**kw)
        return self._check(self._lib.phx_set_params(self._h, C.byref(p)))

    def set_potential_pump(self, V=None, P=None):
        pv, wv = _addr(None if V is None else self._as_T(V, self.rdtype))
        pp, wp = _addr(None if P is None else self._as_T(P, self.rdtype))
        where = wv if V is not None else wp
        if V is not None and P is not None and wv != wp:
            raise ValueError("V and P must live in the same memory space")
        self._keep = (V, P)
        return self._check(self._lib.phx_set_potential_pump(self._h, pv, pp, where))

    def set_drive(self, E=None):
        p, w = _addr(None if E is None else self._as_T(E, self.cdtype))
        return self._check(self._lib.phx_set_drive(self._h, p, w))

    def _as_T(self, a, dt):
        if isinstance(a, np.ndarray):
            return np.ascontiguousarray(a, dtype=dt)
        return a

    def set_field(self, field, src):
        f, shape, dt = self._field_shape_dtype(field)
        src = self._as_T(src, dt)
        if int(np.prod(src.shape)) != int(np.prod(shape)):
            raise ValueError(f"field {field}: expected {shape}, got {tuple(src.shape)}")
        p, w = _addr(src)
        return self._check(self._lib.phx_set_field(self._h, f, p, w))

    def read_field(self, field, out=None):
        f, shape, dt = self._field_shape_dtype(field)
        if out is None:
            out = np.empty(shape, dtype=dt)
        p, w = _addr(out)
        self._check(self._lib.phx_read_field(self._h, f, p, w))
        return out

    def step_rk4(self, n_steps=1):
        return self._check(self._lib.phx_step_rk4(self._h, int(n_steps)))

    def step_adaptive(self, t_end, atol, rtol, h_init, h_min=1e-12, h_max=1e30, max_attempts=1 << 40):
        ctl = phx_adaptive(float(atol), float(rtol), float(h_init), float(h_min), float(h_max), int(max_attempts))
        return self._check(self._lib.phx_step_adaptive(self._h, float(t_end), C.byref(ctl)))

    def get_adaptive_state(self, log_cap=1 << 16):
        """Integrator state and the attempt log of the last phx_step_adaptive call (synchronises)."""
        st = phx_adaptive_state()
        acc, q = np.zeros(log_cap, np.int32), np.zeros(log_cap, np.int32)
        h, err = np.zeros(log_cap), np.zeros(log_cap)
        n = C.c_int64(0)
        self._check(self._lib.phx_get_adaptive_state(self._h, C.byref(st), acc.ctypes.data, q.ctypes.data, h.ctypes.data,
                                                     err.ctypes.data, log_cap, C.byref(n)))
        k = n.value
        return {"t": st.t, "h_next": st.h_next, "n_accept": st.n_accept, "n_reject": st.n_reject, "attempts": st.attempts,
                "err_last": st.err_last, "accept": acc[:k], "q": q[:k], "h": h[:k], "err": err[:k]}

    def set_time(self, t, h_next=0.0):
        return self._check(self._lib.phx_set_time(self._h, float(t), float(h_next)))

    def get_step(self):
        v = C.c_uint64()
        self._check(self._lib.phx_get_step(self._h, C.byref(v)))
        return v.value

    def set_step(self, step):
        return self._check(self._lib.phx_set_step(self._h, int(step)))

    def ensemble_mean_density(self, field="psi_p", out=None):
        f = FIELDS[field]
        if out is None:
            out = np.empty((self.ny, self.nx), dtype=self.rdtype)
        p, w = _addr(out)
        self._check(self._lib.phx_ensemble_mean_density(self._h, f, p, w))
        return out

    def check_finite(self):
        flag = C.c_int32(0)
        self._check(self._lib.phx_check_finite(self._h, C.byref(flag)))
        return bool(flag.value)

    def get_coeffs(self):
        out = np.zeros(PHX_NCOEF, dtype=np.float64)
        self._check(self._lib.phx_get_coeffs(self._h, out.ctypes.data, PHX_NCOEF))
        return out

    def debug_noise_u32(self, step, out=None):
        if out is None:
            out = np.empty((self.batch, self.ny, self.nx, 4), dtype=np.uint32)
        p, w = _addr(out)
        self._check(self._lib.phx_debug_noise_u32(self._h, int(step), p, w))
        return out

    def select_variant(self, variant):
        return self._check(self._lib.phx_select_variant(self._h, int(variant)))

    def get_variant(self):
        v = C.c_int32()
        self._check(self._lib.phx_get_variant(self._h, C.byref(v)))
        return v.value

    def get_launch_count(self):
        v = C.c_uint64()
        self._check(self._lib.phx_get_launch_count(self._h, C.byref(v)))
        return v.value

    def set_tuning(self, key, value):
        return self._check(self._lib.phx_set_tuning(self._h, key.encode(), int(value)))

    def sync(self):
        return self._check(self._lib.phx_sync(self._h))

    def last_error(self):
        return self._lib.phx_last_error(self._h).decode()

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.phx_destroy_grid(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def grid_from_workload(w, variant=PHX_VARIANT_AUTO, stream=None, upload=True, **overrides) -> "Grid":
    """Convenience for tests and bench: a Grid configured from a workloads.Workload."""
    g = Grid(w.nx, w.ny, w.dx, w.dy, model=w.model, prec=w.prec, batch=w.batch, noise=w.noise, stream=stream,
             **overrides)
    g.set_params(make_params(seed=w.seed, **w.params))
    if w.V is not None or w.P is not None:
        g.set_potential_pump(w.V, w.P)
    if variant != PHX_VARIANT_AUTO:
        g.select_variant(variant)
    if upload:
        for name, arr in w.fields.items():
            g.set_field(name, arr)
    return g


def step_rk4_static(psi_in, psi_out, dx, dy, params, V=None, n_steps=1, bc=(0, 0), stream=None):
    """phx_step_rk4_static: RK4 steps of the scalar model without a handle, a workspace or any allocation (include/phx.h).
    psi_in / psi_out / V: torch CUDA tensors [ny][nx] (complex64 or complex128; V float32 / float64) on the current device;
    enqueues on `stream` (a torch stream, default: the current one) and does not synchronise."""
    import torch
    ny, nx = psi_in.shape[-2], psi_in.shape[-1]
    prec = PHX_C64 if psi_in.dtype == torch.complex128 else PHX_C32
    if stream is None:
        stream = torch.cuda.current_stream(psi_in.device)
    st = lib().phx_step_rk4_static(nx, ny, float(dx), float(dy), prec, int(bc[0]), int(bc[1]), C.byref(params),
                                   None if V is None else V.data_ptr(), psi_in.data_ptr(), psi_out.data_ptr(), int(n_steps),
                                   stream.cuda_stream)
    if st != PHX_OK:
        need = 3 * ((nx * ny * (16 if prec == PHX_C64 else 8) + 255) // 256 * 256) + 256
        msg = {PHX_ERR_WORKSPACE: f"phx_step_rk4_static: a {nx} x {ny} grid needs {need} bytes of scratch, the static array holds "
                                  f"{PHX_STATIC_SCRATCH_BYTES}",
               PHX_ERR_INVALID_ARG: "phx_step_rk4_static: invalid argument",
               PHX_ERR_CUDA: "phx_step_rk4_static: CUDA runtime failure"}.get(st, "phx_step_rk4_static failed")
        raise PhxError(st, msg)
