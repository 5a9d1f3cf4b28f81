"""ctypes binding of libcavity.so (include/cavity.h).  Argument marshalling only: every step of the path
runs in the CUDA kernels behind the C ABI.  There is no CPU fallback; a missing library or a missing
CUDA device raises.

`import torch` happens before the library is loaded: libcavity.so takes its device memory from PyTorch's
caching allocator and enqueues on PyTorch's current stream.
"""
import ctypes as C
import os

import numpy as np

ENGINE_AUTO, ENGINE_STREAM, ENGINE_RESIDENT = 0, 1, 2
_ENGINES = {"auto": ENGINE_AUTO, "stream": ENGINE_STREAM, "resident": ENGINE_RESIDENT}

# every symbol include/cavity.h and include/cavity_debug.h declare
SYMBOLS = ("cav_create", "cav_destroy", "cav_set_fields", "cav_get_fields", "cav_step", "cav_step_async", "cav_sync",
           "cav_poisson", "cav_get_diag", "cav_set_engine", "cav_set_resident_plan", "cav_trace_sweeps", "cav_describe", "cav_launch_count",
           "cav_last_elapsed_ms", "cav_strerror", "cav_set_sweep", "cav_step_res", "cav_run_to_steady", "cav_debug_set_epoch",
           "cav_measure_fp64_peak", "cav_plan_check", "cav_debug_unit_roundtrip", "cav_diag_noalloc", "cav_noalloc_max_n")

SWEEP_REDBLACK, SWEEP_JACOBI, SWEEP_COMPACT9 = 0, 1, 2
_SWEEPS = {"redblack": SWEEP_REDBLACK, "jacobi": SWEEP_JACOBI, "compact9": SWEEP_COMPACT9}

_lib = None


class CavDiag(C.Structure):
    _fields_ = [("t", C.c_double), ("step", C.c_longlong), ("res_inf", C.c_double), ("res_l2", C.c_double),
                ("kinetic_energy", C.c_double), ("enstrophy", C.c_double)]


class CavMonitor(C.Structure):
    _fields_ = [("steps", C.c_int), ("converged", C.c_int), ("res_psi", C.c_double), ("res_omega", C.c_double)]


class CavityError(RuntimeError):
    def __init__(self, what, code):
        msg = lib().cav_strerror(code).decode() if _lib is not None else "?"
        super().__init__("%s failed: %s (code %d)" % (what, msg, code))
        self.code = code


def lib_path():
    return os.path.join(os.path.dirname(os.path.abspath(__file__)), "libcavity.so")


def lib():
    """Loads libcavity.so (building it first if the sources are newer).  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    import torch  # noqa: F401  (loads libc10 / libc10_cuda, which libcavity.so links against)
    path = lib_path()
    if os.environ.get("CAVITY_NO_BUILD", "0") != "1":
        from .build import build
        path = build()
    if not os.path.exists(path):
        raise RuntimeError("libcavity.so is missing (%s); run python -m paper_0809_3098_b200.build" % path)
    L = C.CDLL(path)
    dp = C.POINTER(C.c_double)
    L.cav_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_double, C.c_double, C.c_double, C.c_int]
    L.cav_destroy.argtypes = [C.c_void_p]
    L.cav_destroy.restype = None
    L.cav_set_fields.argtypes = [C.c_void_p, dp, dp]
    L.cav_get_fields.argtypes = [C.c_void_p, dp, dp]
    L.cav_step.argtypes = [C.c_void_p, C.c_int]
    L.cav_step_async.argtypes = [C.c_void_p, C.c_int]
    L.cav_sync.argtypes = [C.c_void_p]
    L.cav_poisson.argtypes = [C.c_void_p, C.c_int, dp]
    L.cav_get_diag.argtypes = [C.c_void_p, C.POINTER(CavDiag)]
    L.cav_set_engine.argtypes = [C.c_void_p, C.c_int]
    L.cav_set_resident_plan.argtypes = [C.c_void_p, C.c_int, C.c_int]
    L.cav_trace_sweeps.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_longlong), C.c_int, C.POINTER(C.c_int)]
    L.cav_describe.argtypes = [C.c_void_p, C.c_char_p, C.c_int]
    L.cav_launch_count.argtypes = [C.c_void_p]
    L.cav_launch_count.restype = C.c_longlong
    L.cav_last_elapsed_ms.argtypes = [C.c_void_p, C.POINTER(C.c_float)]
    L.cav_set_sweep.argtypes = [C.c_void_p, C.c_int]
    L.cav_step_res.argtypes = [C.c_void_p, dp, dp]
    L.cav_run_to_steady.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.POINTER(CavMonitor)]
    L.cav_debug_set_epoch.argtypes = [C.c_void_p, C.c_uint]
    L.cav_measure_fp64_peak.argtypes = [C.c_void_p, dp, dp]
    L.cav_plan_check.argtypes = [C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_longlong)]
    L.cav_debug_unit_roundtrip.argtypes = [dp, dp, C.c_int, C.c_uint, C.POINTER(C.c_int)]
    L.cav_diag_noalloc.argtypes = [C.c_int, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.cav_noalloc_max_n.argtypes = []
    L.cav_strerror.argtypes = [C.c_int]
    L.cav_strerror.restype = C.c_char_p
    _lib = L
    return L


def _p(a):
    return a.ctypes.data_as(C.POINTER(C.c_double)) if a is not None else None


def _chk(rc, what):
    if rc != 0:
        raise CavityError(what, rc)


def _field(a, N, name):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.shape != (N + 1, N + 1):
        raise ValueError("%s must have shape (N+1, N+1) = (%d, %d), row j = y index" % (name, N + 1, N + 1))
    return a


def unit_roundtrip(values, tag):
    """Testing aid: values (float64, length a multiple of 4, any bit patterns) through the exchange-unit encoding on the device.
    Returns (restored values, number of units whose tags did not validate)."""
    v = np.ascontiguousarray(values, dtype=np.float64)
    assert v.ndim == 1 and v.size % 4 == 0 and v.size > 0
    out = np.empty_like(v)
    bad = C.c_int()
    _chk(lib().cav_debug_unit_roundtrip(_p(v), _p(out), v.size // 4, int(tag), C.byref(bad)), "cav_debug_unit_roundtrip")
    return out, bad.value


def noalloc_max_n():
    """Largest N cav_diag_noalloc accepts (its scratch is a fixed array inside the library)."""
    return int(lib().cav_noalloc_max_n())


def diag_noalloc(N, psi_dev, omega_dev, out4_dev, pitch=None, stream=0):
    """cav_diag_noalloc: the a4 diagnostics of fields the caller holds on the device, for callers that may not allocate device
    memory (no context, no cudaMalloc, no PyTorch allocator; see include/cavity.h for who that is and for the limits).
    psi_dev, omega_dev, out4_dev: device addresses (int) or objects with data_ptr() (torch CUDA tensors of float64); pitch =
    doubles per row (default N + 1: dense); stream = a cudaStream_t as an int (0 = default stream).  Only enqueues: out4_dev
    (res_inf, res_l2, kinetic_energy, enstrophy) is valid once the stream has run that far.  Calls that can overlap on the GPU
    race on the library's one scratch array; the first call on a device should precede any stream capture."""
    def addr(x):
        return C.c_void_p(int(x.data_ptr()) if hasattr(x, "data_ptr") else int(x))
    _chk(lib().cav_diag_noalloc(int(N), int(N + 1 if pitch is None else pitch), addr(psi_dev), addr(omega_dev), addr(out4_dev),
                                C.c_void_p(int(stream))), "cav_diag_noalloc")


def plan_check(N, sweep="redblack", T=0, sms=148, smem_bytes=232448):
    """Host logic only (no device): the resident plan of an (N + 1)^2 grid and the consistency of its halo-exchange pattern.
    Returns (rc, plan dict or None, counts dict)."""
    plan = (C.c_int * 9)()
    counts = (C.c_longlong * 5)()
    rc = lib().cav_plan_check(int(N), _SWEEPS[sweep], int(T), int(sms), int(smem_bytes), plan, counts)
    names = ("ntx", "nty", "CW", "CH", "halo", "T", "warps", "smem_bytes", "EB")
    cn = ("fetched", "stored", "unmatched", "unfetched", "misfit")
    return rc, (dict(zip(names, plan)) if rc != -4 else None), dict(zip(cn, counts))


class Cavity:
    """One cav_ctx.  Fields are numpy (N+1, N+1) float64 arrays indexed [j, i] (row N = lid)."""

    def __init__(self, N, Re, dt, sor_omega, sweeps_per_stage, engine="auto", resident_T=0):
        self.N = int(N)
        self._h = C.c_void_p()
        L = lib()
        import torch
        if torch.cuda.is_available():
            torch.cuda.init()          # libcavity.so allocates through PyTorch's caching allocator
        _chk(lib().cav_create(C.byref(self._h), int(N), float(Re), float(dt), float(sor_omega),
                              int(sweeps_per_stage)), "cav_create")
        if engine != "auto":
            self.set_engine(engine)
        if resident_T:
            self.set_resident_plan(resident_T)

    def close(self):
        if getattr(self, "_h", None):
            lib().cav_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_engine(self, engine):
        _chk(lib().cav_set_engine(self._h, _ENGINES[engine] if isinstance(engine, str) else int(engine)),
             "cav_set_engine")

    def set_sweep(self, kind):
        """'redblack' (default), 'jacobi' or 'compact9' (or the CAV_SWEEP_* integer)."""
        _chk(lib().cav_set_sweep(self._h, _SWEEPS[kind] if isinstance(kind, str) else int(kind)), "cav_set_sweep")

    def step_res(self):
        """One time step; returns (RES_psi, RES_omega) of that step (eq 26-27 of the paper)."""
        rp, rw = C.c_double(), C.c_double()
        _chk(lib().cav_step_res(self._h, C.byref(rp), C.byref(rw)), "cav_step_res")
        return rp.value, rw.value

    def run_to_steady(self, max_steps, check_every, tol_psi, tol_omega):
        m = CavMonitor()
        _chk(lib().cav_run_to_steady(self._h, int(max_steps), int(check_every), float(tol_psi), float(tol_omega),
                                     C.byref(m)), "cav_run_to_steady")
        return {"steps": m.steps, "converged": bool(m.converged), "res_psi": m.res_psi, "res_omega": m.res_omega}

    def debug_set_epoch(self, epoch):
        _chk(lib().cav_debug_set_epoch(self._h, int(epoch) & 0xFFFFFFFF), "cav_debug_set_epoch")

    def set_resident_plan(self, T=0, variant=-1):
        _chk(lib().cav_set_resident_plan(self._h, int(T), int(variant)), "cav_set_resident_plan")

    def trace_sweeps(self, nsweeps, slots_per_tile=64):
        """(ntiles, slots) int64 array of %globaltimer stamps in ns (see include/cavity_debug.h: cav_trace_sweeps)."""
        out = np.zeros((1024, slots_per_tile), dtype=np.int64)
        nt = C.c_int()
        _chk(lib().cav_trace_sweeps(self._h, int(nsweeps), out.ctypes.data_as(C.POINTER(C.c_longlong)),
                                    int(slots_per_tile), C.byref(nt)), "cav_trace_sweeps")
        return out[:nt.value]

    def set_fields(self, psi, omega):
        psi = None if psi is None else _field(psi, self.N, "psi")
        omega = _field(omega, self.N, "omega")
        _chk(lib().cav_set_fields(self._h, _p(psi), _p(omega)), "cav_set_fields")

    def get_fields(self, psi_out=None, omega_out=None):
        psi = np.empty((self.N + 1, self.N + 1)) if psi_out is None else psi_out
        w = np.empty((self.N + 1, self.N + 1)) if omega_out is None else omega_out
        _chk(lib().cav_get_fields(self._h, _p(psi), _p(w)), "cav_get_fields")
        return psi, w

    def step(self, nsteps=1):
        _chk(lib().cav_step(self._h, int(nsteps)), "cav_step")

    def step_async(self, nsteps=1):
        _chk(lib().cav_step_async(self._h, int(nsteps)), "cav_step_async")

    def sync(self):
        _chk(lib().cav_sync(self._h), "cav_sync")

    def poisson(self, nsweeps, want_residual=True):
        r = C.c_double()
        _chk(lib().cav_poisson(self._h, int(nsweeps), C.byref(r) if want_residual else None), "cav_poisson")
        return r.value if want_residual else None

    def diag(self):
        d = CavDiag()
        _chk(lib().cav_get_diag(self._h, C.byref(d)), "cav_get_diag")
        return {"t": d.t, "step": d.step, "res_inf": d.res_inf, "res_l2": d.res_l2,
                "kinetic_energy": d.kinetic_energy, "enstrophy": d.enstrophy}

    def measure_fp64_peak(self):
        """(fp64 FMA instructions per second per lane summed over the GPU, nominal SM clock in MHz) of a DFMA-chain kernel."""
        r, mhz = C.c_double(), C.c_double()
        _chk(lib().cav_measure_fp64_peak(self._h, C.byref(r), C.byref(mhz)), "cav_measure_fp64_peak")
        return r.value, mhz.value

    def describe(self):
        buf = C.create_string_buffer(1024)
        _chk(lib().cav_describe(self._h, buf, 1024), "cav_describe")
        return buf.value.decode()

    def launch_count(self):
        return int(lib().cav_launch_count(self._h))

    def last_elapsed_ms(self):
        ms = C.c_float()
        _chk(lib().cav_last_elapsed_ms(self._h, C.byref(ms)), "cav_last_elapsed_ms")
        return float(ms.value)
