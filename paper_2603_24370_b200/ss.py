"""Thin ctypes binding of libss.so (include/ss.h).  Argument marshalling only: every step of the
path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

There is no CPU fallback: importing this module without the built library raises, and
creating a solver without a CUDA device raises SSError(SS_ERR_CUDA).
"""
from __future__ import annotations

import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libss.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(
        f"{LIB_PATH} is missing: build it with `python -m paper_2603_24370_b200.build` "
        "(nvcc, sm_100a).  There is no CPU fallback.")
_lib = C.CDLL(LIB_PATH)

THEORY_CHIRAL_MAGNET, THEORY_ABELIAN_HIGGS, THEORY_BABY_SKYRME = 0, 1, 2
POT_STANDARD, POT_EASY_PLANE, POT_BROKEN = 0, 1, 2
F64, F32 = 0, 1
OK, ERR_ARG, ERR_UNSUPPORTED, ERR_CUDA, ERR_WORKSPACE, ERR_STATE, ERR_NONFINITE, ERR_TOO_LARGE = \
    0, -1, -2, -3, -4, -5, -6, -7
RK4, VERLET = 0, 1
OBS_ENERGY, OBS_CHARGE, OBS_ORDER = 0, 1, 2
NOALLOC_MAX_SITES = 2048 * 2048   # SS_NOALLOC_MAX_SITES of include/ss.h
FLAG_NO_GRAPH = 1
FLAG_NO_RESIDENT = 2
FLAG_NO_SLABS = 4

EXPORTS = ["ss_workspace_bytes", "ss_create", "ss_destroy", "ss_set_fields", "ss_get_fields",
           "ss_set_fields_host", "ss_get_fields_host", "ss_profile_step", "ss_kernel_name",
           "ss_step", "ss_energy", "ss_charge", "ss_kinetic", "ss_status", "ss_arrests",
           "ss_launch_count", "ss_strerror", "ss_render", "ss_schedule_name",
           "ss_render_noalloc"]


class ss_params(C.Structure):
    _fields_ = [("dtype", C.c_int), ("batch", C.c_int), ("dt", C.c_double),
                ("kappa", C.c_double), ("B", C.c_double), ("K", C.c_double),
                ("B_batch", C.POINTER(C.c_double)), ("lam", C.c_double),
                ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("stream", C.c_void_p), ("arrest_log_capacity", C.c_int64),
                ("integrator", C.c_int), ("flags", C.c_int),
                ("chunks_per_segment", C.c_int), ("dmi_d", C.POINTER(C.c_double)),
                ("mu", C.c_double), ("potential", C.c_int), ("potential_n", C.c_int),
                ("demag", C.c_double), ("demag_cycles", C.c_int)]


_dp = C.POINTER(C.c_double)
_lib.ss_workspace_bytes.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(ss_params)]
_lib.ss_workspace_bytes.restype = C.c_size_t
_lib.ss_create.argtypes = [C.POINTER(C.c_void_p), C.c_int, C.c_int, C.c_int, C.c_double,
                           C.POINTER(ss_params)]
_lib.ss_destroy.argtypes = [C.c_void_p]
_lib.ss_set_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ss_get_fields.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ss_set_fields_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ss_get_fields_host.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ss_profile_step.argtypes = [C.c_void_p, C.c_int, _dp, C.c_int, C.POINTER(C.c_int)]
_lib.ss_kernel_name.argtypes = [C.c_void_p, C.c_int]
_lib.ss_kernel_name.restype = C.c_char_p
_lib.ss_schedule_name.argtypes = [C.c_void_p]
_lib.ss_schedule_name.restype = C.c_char_p
_lib.ss_step.argtypes = [C.c_void_p, C.c_int64]
for _n in ("ss_energy", "ss_charge", "ss_kinetic"):
    getattr(_lib, _n).argtypes = [C.c_void_p, _dp]
_lib.ss_status.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_int64),
                           C.POINTER(C.c_int)]
_lib.ss_arrests.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_int64), C.c_int64,
                            C.POINTER(C.c_int64)]
_lib.ss_launch_count.argtypes = [C.c_void_p]
_lib.ss_render.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, _dp]
_lib.ss_launch_count.restype = C.c_int64
_lib.ss_render_noalloc.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(ss_params),
                                   C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
_lib.ss_strerror.argtypes = [C.c_int]
_lib.ss_strerror.restype = C.c_char_p


class SSError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {_lib.ss_strerror(code).decode()} ({code})")


def strerror(code: int) -> str:
    return _lib.ss_strerror(int(code)).decode()


def _check(rc, where, allow=()):
    if rc != OK and rc not in allow:
        raise SSError(rc, where)
    return rc


def _params(dtype, batch, dt, kappa, B, K, lam, B_batch, log_cap, flags, cps=0, integrator=0,
            dmi=None, mu=0.0, pot=0, potN=3, demag=0.0, demag_cycles=0):
    p = ss_params()
    p.demag, p.demag_cycles = float(demag), int(demag_cycles)
    p.mu, p.potential, p.potential_n = float(mu), int(pot), int(potN)
    p.dtype, p.batch, p.dt = int(dtype), int(batch), float(dt)
    p.kappa, p.B, p.K, p.lam = float(kappa), float(B), float(K), float(lam)
    keep = None
    if B_batch is not None:
        keep = (C.c_double * int(batch))(*[float(x) for x in B_batch])
        p.B_batch = C.cast(keep, _dp)
    p.arrest_log_capacity = int(log_cap)
    p.integrator, p.flags = int(integrator), int(flags)
    p.chunks_per_segment = int(cps)
    if dmi is not None:
        flat = [float(x) for v in dmi for x in (v if hasattr(v, "__len__") else (v,))]
        assert len(flat) == 6
        keep = (keep, (C.c_double * 6)(*flat))
        p.dmi_d = C.cast(keep[1], _dp)
    return p, keep


def workspace_bytes(theory, Nx, Ny, dtype=F64, batch=1, log_cap=0) -> int:
    p, _ = _params(dtype, batch, 0.0, 0, 0, 0, 0, None, log_cap, 0)
    return _lib.ss_workspace_bytes(int(theory), int(Nx), int(Ny), C.byref(p))


class Solver:
    """ss_create ... ss_destroy around torch-owned device memory and the current torch stream."""

    def __init__(self, theory, Nx, Ny, h, *, dtype=F64, batch=1, dt=0.0, kappa=0.0, B=0.0, K=0.0,
                 lam=0.0, B_batch=None, log_cap=0, flags=0, cps=0, integrator=RK4, dmi=None,
                 mu=0.0, pot=POT_STANDARD, potN=3, demag=0.0, demag_cycles=0, device="cuda:0",
                 stream=None):
        self.theory, self.Nx, self.Ny, self.batch = int(theory), int(Nx), int(Ny), int(batch)
        self.C = 4 if theory == THEORY_ABELIAN_HIGGS else 3
        self.dtype = dtype
        self.log_cap = int(log_cap) if log_cap else 4096
        self.torch_dtype = torch.float64 if dtype == F64 else torch.float32
        self.device = torch.device(device)
        self._h = C.c_void_p()
        p, keep = _params(dtype, batch, dt, kappa, B, K, lam, B_batch, log_cap, flags, cps,
                          integrator, dmi, mu, pot, potN, demag, demag_cycles)
        nbytes = _lib.ss_workspace_bytes(self.theory, self.Nx, self.Ny, C.byref(p))
        if nbytes == 0:
            # invalid or over a limit: ss_create tells which (it checks before touching memory)
            _check(_lib.ss_create(C.byref(self._h), self.theory, self.Nx, self.Ny, float(h),
                                  C.byref(p)), "ss_create")
            raise SSError(ERR_ARG, "ss_workspace_bytes")
        if not torch.cuda.is_available():
            raise SSError(ERR_CUDA, "ss_create (no CUDA device; libss has no CPU path)")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
        p.workspace = self.workspace.data_ptr()
        p.workspace_bytes = nbytes
        p.stream = self.stream.cuda_stream
        # the library binds the solver to the workspace's device; no call needs it to be current
        _check(_lib.ss_create(C.byref(self._h), self.theory, self.Nx, self.Ny, float(h),
                              C.byref(p)), "ss_create")

    @property
    def shape(self):
        return (self.batch, self.C, self.Ny, self.Nx)

    def close(self):
        if getattr(self, "_h", None) and self._h.value and _lib is not None:
            _lib.ss_destroy(self._h)
            self._h = C.c_void_p()

    __del__ = close

    def _dev(self, t, name):
        if t is None:
            return None
        if not (t.is_cuda and t.dtype == self.torch_dtype and t.is_contiguous()
                and tuple(t.shape) == self.shape):
            raise ValueError(f"{name}: need a contiguous {self.torch_dtype} CUDA tensor of shape "
                             f"{self.shape}")
        return C.c_void_p(t.data_ptr())

    def _after_current(self):
        """the solver's stream waits for work already queued on torch's current stream"""
        cur = torch.cuda.current_stream(self.device)
        if cur != self.stream:
            self.stream.wait_stream(cur)

    def _before_current(self):
        """torch's current stream waits for what the solver's stream has queued"""
        cur = torch.cuda.current_stream(self.device)
        if cur != self.stream:
            cur.wait_stream(self.stream)

    def set_fields(self, fields, vel=None):
        self._after_current()               # the inputs may still be being produced there
        _check(_lib.ss_set_fields(self._h, self._dev(fields, "fields"), self._dev(vel, "vel")),
               "ss_set_fields")

    def get_fields(self, want_vel=True):
        f = torch.empty(self.shape, dtype=self.torch_dtype, device=self.device)
        v = torch.empty_like(f) if want_vel else None
        self._after_current()               # f, v were allocated on torch's current stream
        with torch.cuda.stream(self.stream):
            _check(_lib.ss_get_fields(self._h, C.c_void_p(f.data_ptr()),
                                      C.c_void_p(v.data_ptr()) if want_vel else None),
                   "ss_get_fields")
        self._before_current()              # the outputs are used on torch's current stream
        return (f, v) if want_vel else f

    def _host(self, t, name):
        if t is None:
            return None
        if not (not t.is_cuda and t.dtype == self.torch_dtype and t.is_contiguous()
                and tuple(t.shape) == self.shape):
            raise ValueError(f"{name}: need a contiguous {self.torch_dtype} CPU tensor of shape "
                             f"{self.shape}")
        return C.c_void_p(t.data_ptr())

    def set_fields_host(self, fields, vel=None):
        """fields / vel: CPU tensors (pinned for asynchronous copies)."""
        _check(_lib.ss_set_fields_host(self._h, self._host(fields, "fields"),
                                       self._host(vel, "vel")), "ss_set_fields_host")

    def get_fields_host(self, fields=None, vel=None):
        """Fill the given CPU tensors (either may be None); synchronises the stream."""
        _check(_lib.ss_get_fields_host(self._h, self._host(fields, "fields"),
                                       self._host(vel, "vel")), "ss_get_fields_host")

    def step(self, k=1):
        _check(_lib.ss_step(self._h, int(k)), "ss_step")

    def profile_step(self, reps=1):
        """[(kernel name, average ms)] of one flow step, kernels launched one by one."""
        cap = 8192                          # a demagnetisation step has a few hundred kernels
        buf = (C.c_double * cap)()
        n = C.c_int()
        _check(_lib.ss_profile_step(self._h, int(reps), buf, cap, C.byref(n)), "ss_profile_step")
        return [(_lib.ss_kernel_name(self._h, i).decode(), buf[i]) for i in range(n.value)]

    def _scalar(self, fn, name, strict):
        out = (C.c_double * self.batch)()
        _check(fn(self._h, out), name, allow=() if strict else (ERR_NONFINITE,))
        return [out[i] for i in range(self.batch)]

    def energy(self, strict=True):
        return self._scalar(_lib.ss_energy, "ss_energy", strict)

    def charge(self, strict=True):
        return self._scalar(_lib.ss_charge, "ss_charge", strict)

    def kinetic(self, strict=True):
        return self._scalar(_lib.ss_kinetic, "ss_kinetic", strict)

    def status(self):
        steps = C.c_int64()
        na = (C.c_int64 * self.batch)()
        nf = (C.c_int * self.batch)()
        rc = _check(_lib.ss_status(self._h, C.byref(steps), na, nf), "ss_status",
                    allow=(ERR_NONFINITE,))
        return dict(steps=steps.value, n_arrests=list(na), nonfinite=list(nf), rc=rc)

    def arrests(self, lattice=0):
        cap = self.log_cap
        buf = (C.c_int64 * cap)()
        cnt = C.c_int64()
        _check(_lib.ss_arrests(self._h, int(lattice), buf, cap, C.byref(cnt)), "ss_arrests")
        return [int(buf[i]) for i in range(min(cnt.value, cap))], cnt.value

    def render(self, observable=OBS_ENERGY, lattice=0, strict=True):
        """(rgba [Ny][Nx] uint8x4 CUDA tensor, (min, max)) of one observable (headless).
        strict=False tolerates non-finite interior values (drawn magenta)."""
        img = torch.empty((self.Ny, self.Nx, 4), dtype=torch.uint8, device=self.device)
        mm = (C.c_double * 2)()
        self._after_current()
        with torch.cuda.stream(self.stream):
            _check(_lib.ss_render(self._h, int(observable), int(lattice),
                                  C.c_void_p(img.data_ptr()), mm), "ss_render",
                   allow=() if strict else (ERR_NONFINITE,))
        self._before_current()
        return img, (mm[0], mm[1])

    def schedule(self) -> str:
        return _lib.ss_schedule_name(self._h).decode()

    def launch_count(self) -> int:
        return _lib.ss_launch_count(self._h)


def render_noalloc(theory, h, fields, minmax, *, rgba=None, nonfinite=None, observable=OBS_ENERGY,
                   dtype=F64, kappa=0.0, B=0.0, K=0.0, lam=0.0, dmi=None, mu=0.0, pot=POT_STANDARD,
                   potN=3, stream=None) -> None:
    """ss_render_noalloc: extrema (and image) of one observable of ONE lattice `fields`
    ([C][Ny][Nx] CUDA tensor) with no handle, no workspace and no device allocation: the caller
    passes every output -- minmax (2 float64), rgba ([Ny][Nx][4] uint8, optional), nonfinite
    (1 int32, optional), all CUDA tensors on the device of `fields`.  Asynchronous on `stream`
    (default: torch's current stream).  Lattices of more than NOALLOC_MAX_SITES sites are
    rejected; calls that overlap on the GPU race on the library's static scratch."""
    C_, Ny, Nx = (int(x) for x in fields.shape)
    want = torch.float64 if dtype == F64 else torch.float32
    if not (fields.is_cuda and fields.is_contiguous() and fields.dtype == want and
            C_ == (4 if theory == THEORY_ABELIAN_HIGGS else 3)):
        raise ValueError("fields: need a contiguous [C][Ny][Nx] CUDA tensor of the solver dtype")
    if not (minmax.is_cuda and minmax.dtype == torch.float64 and minmax.numel() == 2 and
            minmax.is_contiguous() and minmax.device == fields.device):
        raise ValueError("minmax: need 2 contiguous float64 on the device of fields")
    if rgba is not None and not (rgba.is_cuda and rgba.dtype == torch.uint8 and rgba.is_contiguous()
                                 and tuple(rgba.shape) == (Ny, Nx, 4) and rgba.device == fields.device):
        raise ValueError("rgba: need a contiguous [Ny][Nx][4] uint8 CUDA tensor")
    if nonfinite is not None and not (nonfinite.is_cuda and nonfinite.dtype == torch.int32 and
                                      nonfinite.numel() == 1 and nonfinite.device == fields.device):
        raise ValueError("nonfinite: need 1 int32 on the device of fields")
    p, keep = _params(dtype, 1, 0.0, kappa, B, K, lam, None, 0, 0, dmi=dmi, mu=mu, pot=pot, potN=potN)
    st = stream if stream is not None else torch.cuda.current_stream(fields.device)
    p.stream = st.cuda_stream
    _check(_lib.ss_render_noalloc(int(theory), Nx, Ny, float(h), C.byref(p), int(observable),
                                  C.c_void_p(fields.data_ptr()),
                                  C.c_void_p(rgba.data_ptr()) if rgba is not None else None,
                                  C.c_void_p(minmax.data_ptr()),
                                  C.c_void_p(nonfinite.data_ptr()) if nonfinite is not None else None),
           "ss_render_noalloc")
    del keep


def solver_for(w, *, dtype=F64, flags=0, device="cuda:0", log_cap=0, cps=0,
               integrator=RK4, demag_cycles=0) -> Solver:
    """Solver configured from a workloads.Workload (sizes and parameters only)."""
    return Solver(w.theory, w.Nx, w.Ny, w.h, dtype=dtype, batch=w.batch, dt=w.dt, kappa=w.kappa,
                  B=w.B, K=w.K, lam=w.lam, B_batch=w.B_batch, log_cap=log_cap, flags=flags,
                  cps=cps, integrator=integrator, dmi=getattr(w, "dmi", None),
                  mu=getattr(w, "mu", 0.0), pot=getattr(w, "pot", 0), potN=getattr(w, "potN", 3),
                  demag=getattr(w, "demag", 0.0), demag_cycles=demag_cycles,
                  device=device)
