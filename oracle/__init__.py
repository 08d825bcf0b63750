"""ctypes front end of the CPU oracle (oracle/oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It shares nothing with paper_2603_24370_b200 (the CUDA
path): no kernels, headers, constants or helpers.  It compiles oracle.c with gcc on
first use (``build()``); building the checker is not using it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")

CM, AH, BS = 0, 1, 2
POT_STANDARD, POT_EASY_PLANE, POT_BROKEN = 0, 1, 2
_dp = C.POINTER(C.c_double)


def build(force: bool = False) -> str:
    """gcc -O2 -fopenmp -ffp-contract=off: every expression is evaluated as written."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-Wall", "-shared", "-fPIC",
             "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Model(C.Structure):
    _fields_ = [("theory", C.c_int), ("Nx", C.c_int), ("Ny", C.c_int), ("h", C.c_double),
                ("kappa", C.c_double), ("B", C.c_double), ("K", C.c_double),
                ("lam", C.c_double), ("dmi", C.c_int), ("d", C.c_double * 6),
                ("pot", C.c_int), ("potN", C.c_int), ("mu", C.c_double), ("demag", C.c_double)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_stencil.argtypes = [C.c_int, _dp, _dp, C.c_int, C.c_int, C.c_double]
        L.orc_tree_sum.argtypes = [_dp, C.c_size_t]
        L.orc_tree_sum.restype = C.c_double
        L.orc_tree_sum2d.argtypes = [_dp, C.c_int, C.c_int]
        L.orc_tree_sum2d.restype = C.c_double
        L.orc_cm_energy_bond.argtypes = [_dp, C.c_int, C.c_int] + [C.c_double] * 4
        L.orc_cm_energy_bond.restype = C.c_double
        L.orc_cm_energy_bond_d.argtypes = [_dp, C.c_int, C.c_int] + [C.c_double] * 4 + [_dp]
        L.orc_cm_energy_bond_d.restype = C.c_double
        L.orc_ah_energy_bond.argtypes = [_dp, C.c_int, C.c_int, C.c_double, C.c_double]
        L.orc_ah_energy_bond.restype = C.c_double
        L.orc_bs_energy_plain.argtypes = [C.POINTER(_Model), _dp]
        L.orc_bs_energy_plain.restype = C.c_double
        L.orc_poisson_solve.argtypes = [_dp, _dp, C.c_int, C.c_int, C.c_double]
        L.orc_poisson_solve.restype = C.c_int
        L.orc_demag_potential.argtypes = [C.POINTER(_Model), _dp, _dp]
        L.orc_demag_energy_plain.argtypes = [C.POINTER(_Model), _dp]
        L.orc_demag_energy_plain.restype = C.c_double
        L.orc_energy_charge.argtypes = [C.POINTER(_Model), _dp, C.c_int, _dp, _dp, _dp, _dp]
        L.orc_gradient.argtypes = [C.POINTER(_Model), _dp, _dp]
        L.orc_accel.argtypes = [C.POINTER(_Model), _dp, _dp]
        L.orc_flow_create.argtypes = [C.POINTER(_Model), C.c_double]
        L.orc_flow_create.restype = C.c_void_p
        L.orc_flow_destroy.argtypes = [C.c_void_p]
        L.orc_flow_set.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_flow_step.argtypes = [C.c_void_p, C.c_int64]
        L.orc_flow_step_verlet.argtypes = [C.c_void_p, C.c_int64]
        L.orc_flow_get.argtypes = [C.c_void_p, _dp, _dp]
        L.orc_flow_scalars.argtypes = [C.c_void_p, _dp, _dp, _dp, C.POINTER(C.c_int64),
                                       C.POINTER(C.c_int64), C.POINTER(C.c_int),
                                       C.POINTER(C.c_int)]
        L.orc_flow_arrests.argtypes = [C.c_void_p, C.POINTER(C.c_int64), C.c_int64]
        L.orc_flow_arrests.restype = C.c_int64
        L.orc_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a


def threads() -> int:
    """OpenMP threads the oracle's loops run on."""
    return int(lib().orc_threads())


def ncomp(theory: int) -> int:
    return 4 if theory == AH else 3


def model(theory, Nx, Ny, h, kappa=0.0, B=0.0, K=0.0, lam=0.0, dmi=None, mu=0.0,
          pot=POT_STANDARD, potN=3, demag=0.0):
    """dmi: None = kappa n.(curl n) (BASELINE), else the six numbers (d_x, d_y) of
    PAPER.md:196 eq. (5): e_DMI = kappa sum_mu d_mu . (n x d_mu n).
    Baby Skyrme (theory BS): kappa = Skyrme coupling, V proportional to mu^2,
    pot in POT_*, potN = N of the Z_N-symmetric "broken" potential."""
    m = _Model(int(theory), int(Nx), int(Ny), float(h), float(kappa), float(B), float(K),
               float(lam))
    m.pot, m.potN, m.mu = int(pot), int(potN), float(mu)
    m.demag = float(demag)     # chiral magnet: g = mu0 Ms^2 of PAPER.md:196 eq. (5), (6); 0 = off
    if dmi is not None:
        m.dmi = 1
        m.d = (C.c_double * 6)(*[float(x) for x in np.asarray(dmi).reshape(6)])
    return m


def stencil(op: str, f, h):
    """op in Dx, Dy, Lx, Ly, DxDy applied to one [Ny][Nx] plane (interior; halo 0)."""
    f = _f64(f)
    out = np.empty_like(f)
    lib().orc_stencil({"Dx": 0, "Dy": 1, "Lx": 2, "Ly": 3, "DxDy": 4}[op], _p(f), _p(out),
                      f.shape[1], f.shape[0], float(h))
    return out


def tree_sum(v):
    v = _f64(v).ravel()
    return lib().orc_tree_sum(_p(v), v.size)


def tree_sum2d(v):
    v = _f64(v)
    return lib().orc_tree_sum2d(_p(v), v.shape[1], v.shape[0])


def poisson_solve(rho, h, guess=None):
    """(Lx + Ly) psi = rho on the interior, psi = 0 on the halo (eq. 2; conjugate gradients)."""
    rho = _f64(rho)
    psi = np.zeros_like(rho) if guess is None else _f64(guess).copy()
    lib().orc_poisson_solve(_p(rho), _p(psi), rho.shape[1], rho.shape[0], float(h))
    return psi


def demag_potential(m, f):
    """psi with lap psi = D_x n1 + D_y n2 (eq. 6 in units phi = mu0 Ms psi)."""
    f = _f64(f)
    psi = np.empty((m.Ny, m.Nx))
    lib().orc_demag_potential(C.byref(m), _p(f), _p(psi))
    return psi


def energy_bond(m, f):
    """Plain bond-sum definition of E_h (straight summation)."""
    f = _f64(f)
    if m.theory == BS:
        return lib().orc_bs_energy_plain(C.byref(m), _p(f))
    if m.theory == CM:
        Ed = lib().orc_demag_energy_plain(C.byref(m), _p(f)) if m.demag != 0.0 else 0.0
        if m.dmi:
            d = np.array(list(m.d))
            return Ed + lib().orc_cm_energy_bond_d(_p(f), m.Nx, m.Ny, m.h, m.kappa, m.B, m.K, _p(d))
        return Ed + lib().orc_cm_energy_bond(_p(f), m.Nx, m.Ny, m.h, m.kappa, m.B, m.K)
    return lib().orc_ah_energy_bond(_p(f), m.Nx, m.Ny, m.h, m.lam)


def energy_charge(m, f, literal=False, densities=False):
    """(E, Q) with the canonical tree; literal=True: AH eq.(1)-only diagnostic energy."""
    f = _f64(f)
    E, Q = C.c_double(), C.c_double()
    de = np.empty((m.Ny, m.Nx)) if densities else None
    dq = np.empty((m.Ny, m.Nx)) if densities else None
    lib().orc_energy_charge(C.byref(m), _p(f), int(literal), C.byref(E), C.byref(Q), _p(de),
                            _p(dq))
    return (E.value, Q.value, de, dq) if densities else (E.value, Q.value)


def gradient(m, f):
    f = _f64(f)
    G = np.empty_like(f)
    lib().orc_gradient(C.byref(m), _p(f), _p(G))
    return G


def accel(m, f):
    f = _f64(f)
    a = np.empty_like(f)
    lib().orc_accel(C.byref(m), _p(f), _p(a))
    return a


class Flow:
    """Arrested Newton flow on host arrays [C][Ny][Nx]."""

    def __init__(self, m, dt=0.0, integrator="rk4"):
        """integrator: "rk4" or "verlet" (one gradient per step, DESIGN R15)."""
        assert integrator in ("rk4", "verlet")
        self.integrator = integrator
        self.m = m
        self.shape = (ncomp(m.theory), m.Ny, m.Nx)
        self._h = lib().orc_flow_create(C.byref(m), float(dt))

    def __del__(self):
        if getattr(self, "_h", None):
            try:
                lib().orc_flow_destroy(self._h)
            except TypeError:      # interpreter shutdown: the module globals are already gone
                pass
            self._h = None

    def set_fields(self, phi, vel=None):
        phi = _f64(phi)
        assert phi.shape == self.shape
        vel = None if vel is None else _f64(vel)
        lib().orc_flow_set(self._h, _p(phi), _p(vel))

    def step(self, k=1):
        if self.integrator == "rk4":
            lib().orc_flow_step(self._h, int(k))
        else:
            lib().orc_flow_step_verlet(self._h, int(k))

    def get_fields(self):
        phi, vel = np.empty(self.shape), np.empty(self.shape)
        lib().orc_flow_get(self._h, _p(phi), _p(vel))
        return phi, vel

    def scalars(self):
        E, Q, KE = C.c_double(), C.c_double(), C.c_double()
        n, na = C.c_int64(), C.c_int64()
        nf, vz = C.c_int(), C.c_int()
        lib().orc_flow_scalars(self._h, C.byref(E), C.byref(Q), C.byref(KE), C.byref(n),
                               C.byref(na), C.byref(nf), C.byref(vz))
        return dict(E=E.value, Q=Q.value, KE=KE.value, steps=n.value, n_arrests=na.value,
                    nonfinite=nf.value, v_is_zero=vz.value)

    @property
    def energy(self):
        return self.scalars()["E"]

    @property
    def charge(self):
        return self.scalars()["Q"]

    def arrests(self):
        n = self.scalars()["n_arrests"]
        out = (C.c_int64 * max(n, 1))()
        lib().orc_flow_arrests(self._h, out, n)
        return [int(out[i]) for i in range(n)]


# ---------------------------------------------------------------- headless visualisation (R17)
# CPU restatement of the colour map of ss_render (DESIGN R17, own definition: the paper,
# PAPER.md:158-160, gives no formula): observable over the interior, its extrema, then
# t = (v - min) / (max - min) through a 5-stop piecewise-linear map, one IEEE fp64 operation at a
# time in this order, bytes by floor(x + 0.5); halo sites are 0.
_STOPS = np.array([[0, 0, 128], [0, 128, 255], [255, 255, 255], [255, 128, 0], [128, 0, 0]],
                  dtype=np.float64)


def observable(m, f, which):
    """which: 0 energy density e_i, 1 charge / flux density q_i, 2 order parameter (CM n3, AH |phi|);
    [Ny][Nx] with NaN on the halo."""
    f = _f64(f)
    out = np.full((m.Ny, m.Nx), np.nan)
    I = (slice(2, m.Ny - 2), slice(2, m.Nx - 2))
    if which == 2:
        v = np.sqrt(f[0] * f[0] + f[1] * f[1]) if m.theory == AH else f[2]
    else:
        _, _, de, dq = energy_charge(m, f, densities=True)
        v = de if which == 0 else dq
    out[I] = v[I]
    return out


def colormap(values):
    """values [Ny][Nx] (NaN = halo) -> ([Ny][Nx][4] uint8 RGBA, (min, max))."""
    ok = ~np.isnan(values)
    mn, mx = float(values[ok].min()), float(values[ok].max())
    span = mx - mn
    v = np.where(ok, values, mn)
    t = (v - mn) / span if span > 0.0 else np.full_like(v, 0.5)
    t4 = t * 4.0
    seg = np.minimum(t4.astype(np.int64), 3)
    u = t4 - seg
    img = np.zeros(values.shape + (4,), dtype=np.uint8)
    for k in range(3):
        c0, c1 = _STOPS[seg, k], _STOPS[seg + 1, k]
        x = (c0 + (c1 - c0) * u) + 0.5
        img[..., k] = np.floor(x).astype(np.int64).astype(np.uint8)
    img[..., 3] = 255
    img[~ok] = 0
    return img, (mn, mx)
