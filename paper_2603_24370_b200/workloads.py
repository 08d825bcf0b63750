"""Seeded synthetic inputs shaped like the paper's workloads (BASELINE.json configs 1-5).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of
the method's arithmetic: no stencil, energy, gradient, flow or reduction lives here —
only initial fields (ansaetze + noise), parameters and sizes.  numpy only; it imports
neither the CUDA binding nor oracle/.  Arrays are fp64 [C][Ny][Nx] (x fastest), Nx, Ny
INCLUDE the frozen halo of width 2 (DESIGN R4).  Recipe: DESIGN.md "Input recipe".

The paper uses no public dataset; its use cases are skyrmions in chiral magnets
 and vortices in Abelian-Higgs / Ginzburg-Landau models
(PAPER.md:83, :322).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED0 = 260324370
CM, AH, BS = 0, 1, 2
POT_STANDARD, POT_EASY_PLANE, POT_BROKEN = 0, 1, 2   # baby-Skyrme potentials
HALO = 2

# DMI vectors (d_x, d_y) of PAPER.md:196 eq. (5), e_DMI = kappa sum_mu d_mu . (n x d_mu n)
# (DESIGN R16).  BLOCH is BASELINE's kappa n.(curl n); NEEL its rotation by 90 degrees about e3 in
# spin space (interfacial DMI); D2D its spin mirror y -> -y (the paper's dmi_term="Heusler",
# PAPER.md:141, which selects the antiskyrmion sector).
DMI_BLOCH = ((-1.0, 0.0, 0.0), (0.0, -1.0, 0.0))
DMI_NEEL = ((0.0, -1.0, 0.0), (1.0, 0.0, 0.0))
DMI_D2D = ((1.0, 0.0, 0.0), (0.0, -1.0, 0.0))


@dataclass
class Workload:
    name: str
    theory: int
    Nx: int
    Ny: int
    h: float
    dt: float
    kappa: float = 0.0
    B: float = 0.0
    K: float = 0.0
    lam: float = 0.0
    mu: float = 0.0                   # baby Skyrme: V proportional to mu^2
    demag: float = 0.0                # chiral magnet: g = mu0 Ms^2 of the demagnetisation term
    pot: int = 0                      # baby Skyrme: POT_*
    potN: int = 3                     # baby Skyrme: N of the Z_N-symmetric potential
    batch: int = 1
    steps: int = 0
    B_batch: np.ndarray | None = None
    dmi: tuple | None = None          # None = DMI_BLOCH through the library's default path
    fields: np.ndarray | None = field(default=None, repr=False)   # [batch][C][Ny][Nx] fp64

    @property
    def C(self) -> int:
        return 4 if self.theory == AH else 3

    @property
    def interior_sites(self) -> int:
        return self.batch * (self.Nx - 4) * (self.Ny - 4)


def _rng(config: int, seed_offset: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED0 + config + seed_offset))


def coords(Nx: int, Ny: int, h: float):
    """x_i = (i - (Nx-1)/2) h, y_j = (j - (Ny-1)/2) h as [Ny][Nx] meshes."""
    x = (np.arange(Nx) - (Nx - 1) / 2.0) * h
    y = (np.arange(Ny) - (Ny - 1) / 2.0) * h
    return np.meshgrid(x, y)


def interior_mask(Nx: int, Ny: int) -> np.ndarray:
    m = np.zeros((Ny, Nx), dtype=bool)
    m[HALO:Ny - HALO, HALO:Nx - HALO] = True
    return m


def skyrmion_ansatz(Nx, Ny, h, centres=((0.0, 0.0),), mirror=False) -> np.ndarray:
    """Hedgehog profile f = pi exp(-r/2), n = (sin f cos th, sin f sin th, cos f); several
    centres are superposed stereographically: w = sum_k tan(f_k/2) e^{i th_k},
    n = (2 Re w, 2 Im w, 1-|w|^2)/(1+|w|^2).  mirror: th -> -th (opposite degree)."""
    X, Y = coords(Nx, Ny, h)
    w = np.zeros((Ny, Nx), dtype=np.complex128)
    for cx, cy in centres:
        dx, dy = X - cx, Y - cy
        r = np.hypot(dx, dy)
        f = np.pi * np.exp(-r / 2.0)
        th = np.arctan2(dy, dx)
        if mirror:
            th = -th
        t = np.tan(np.minimum(f / 2.0, np.pi / 2.0 - 1e-9))
        w += t * np.exp(1j * th)
    a2 = np.abs(w) ** 2
    n = np.stack([2.0 * w.real, 2.0 * w.imag, 1.0 - a2]) / (1.0 + a2)
    return n


def _normalise(n: np.ndarray) -> np.ndarray:
    return n / np.sqrt((n * n).sum(axis=0, keepdims=True))


def _cm_finish(n, Nx, Ny, rng, noise):
    """Add U(-noise, noise) per component on the interior, renormalise, vacuum halo."""
    eta = rng.uniform(-noise, noise, size=(3, Ny, Nx)) if noise > 0 else 0.0
    n = _normalise(n + eta)
    m = interior_mask(Nx, Ny)
    n[0][~m] = 0.0
    n[1][~m] = 0.0
    n[2][~m] = 1.0
    return n


def _reject_sample(rng, count, lo, hi, min_sep):
    pts = []
    while len(pts) < count:
        p = rng.uniform(lo, hi, size=2)
        if all(np.hypot(*(p - q)) >= min_sep for q in pts):
            pts.append(p)
    return [tuple(map(float, p)) for p in pts]


def cm_single(N=64, h=0.2, B=0.6, K=0.0, noise=0.01, config=1, steps=1000, seed_offset=0,
              mirror=False) -> Workload:
    """Config 1: one centred skyrmion ansatz + noise, vacuum halo."""
    rng = _rng(config, seed_offset)
    n = _cm_finish(skyrmion_ansatz(N, N, h, mirror=mirror), N, N, rng, noise)
    return Workload(f"cm_single_{N}", CM, N, N, h, 0.5 * h, kappa=1.0, B=B, K=K, steps=steps,
                    fields=n[None])


def cm_multi(N=1024, h=0.2, count=16, noise=0.01, config=2, steps=10000, margin=12.0,
             min_sep=16.0) -> Workload:
    """Config 2: `count` skyrmions at rejection-sampled non-overlapping centres."""
    rng = _rng(config)
    L = N * h
    centres = _reject_sample(rng, count, -L / 2 + margin, L / 2 - margin, min_sep)
    n = _cm_finish(skyrmion_ansatz(N, N, h, centres), N, N, rng, noise)
    return Workload(f"cm_multi_{N}", CM, N, N, h, 0.5 * h, kappa=1.0, B=0.6, steps=steps,
                    fields=n[None])


def vortex_ansatz(Nx, Ny, h, centres):
    """phi = prod_k tanh(r_k) e^{i th_k};  A = sum_k tanh^2(r_k) grad th_k,
    grad th_k = (-(y-y_k), (x-x_k))/r_k^2 (regular at each core)."""
    X, Y = coords(Nx, Ny, h)
    phi = np.ones((Ny, Nx), dtype=np.complex128)
    A1 = np.zeros((Ny, Nx))
    A2 = np.zeros((Ny, Nx))
    for cx, cy in centres:
        dx, dy = X - cx, Y - cy
        r = np.hypot(dx, dy)
        rs = np.where(r > 0, r, 1.0)
        t = np.tanh(r)
        phi *= np.where(r > 0, t * (dx + 1j * dy) / rs, 0.0)
        g = np.where(r > 0, (t / rs) ** 2, 1.0)
        A1 += -dy * g
        A2 += dx * g
    return np.stack([phi.real, phi.imag, A1, A2])


def ah_vortices(N=2048, h=0.1, lam=1.0, count=4, noise=1e-3, config=3, steps=20000,
                min_sep=4.0, centres=None) -> Workload:
    """Config 3: N vortices in the central box [-L/8, L/8]^2; noise on the interior only,
    halo = noise-free ansatz (frozen)."""
    rng = _rng(config)
    L = N * h
    if centres is None:
        centres = _reject_sample(rng, count, -L / 8, L / 8, min_sep)
    f = vortex_ansatz(N, N, h, centres)
    if noise > 0:
        eta = rng.uniform(-noise, noise, size=(4, N, N))
        f = f + eta * interior_mask(N, N)[None]
    return Workload(f"ah_vortices_{N}_lam{lam:g}", AH, N, N, h, 0.5 * h, lam=lam, steps=steps,
                    fields=f[None])


def cm_quench(N=4096, h=0.2, K=0.3, config=4, steps=5000) -> Workload:
    """Config 4: i.i.d. N(0,1) per component, normalised (random unit vectors); vacuum halo."""
    rng = _rng(config)
    n = rng.standard_normal(size=(3, N, N))
    n = _cm_finish(n, N, N, rng, 0.0)
    return Workload(f"cm_quench_{N}", CM, N, N, h, 0.5 * h, kappa=1.0, B=0.6, K=K, steps=steps,
                    fields=n[None])


def cm_sweep(batch=256, N=256, h=0.2, noise=0.01, config=5, steps=5000) -> Workload:
    """Config 5: `batch` independent lattices, B_b = 0.2 + 0.8 U[0,1) drawn first."""
    rng = _rng(config)
    Bb = 0.2 + 0.8 * rng.random(batch)
    base = skyrmion_ansatz(N, N, h)
    f = np.empty((batch, 3, N, N))
    for b in range(batch):
        f[b] = _cm_finish(base.copy(), N, N, rng, noise)
    return Workload(f"cm_sweep_{batch}x{N}", CM, N, N, h, 0.5 * h, kappa=1.0, B=0.6, batch=batch,
                    steps=steps, B_batch=Bb, fields=f)


def bs_single(N=128, h=0.2, kappa=1.0, mu=1.0, pot=POT_STANDARD, potN=3, noise=0.01, count=1,
              config=6, steps=2000, batch=1, seed_offset=0) -> Workload:
    """Baby skyrmions (SURVEY 8(f) NEXT-2b; not a BASELINE config): `count`
    hedgehogs (the chiral-magnet ansatz, degree -1 each) at rejection-sampled centres (one:
    centred) plus noise, renormalised; vacuum halo m = e3."""
    rng = _rng(config, seed_offset)
    L = N * h
    f = np.empty((batch, 3, N, N))
    for b in range(batch):
        centres = [(0.0, 0.0)] if count == 1 else _reject_sample(rng, count, -L / 4, L / 4, 5.0)
        f[b] = _cm_finish(skyrmion_ansatz(N, N, h, centres), N, N, rng, noise)
    return Workload(f"bs_{N}_pot{pot}", BS, N, N, h, 0.5 * h, kappa=kappa, mu=mu, pot=pot, potN=potN,
                    batch=batch, steps=steps, fields=f)


def bs_bench() -> Workload:
    """The baby-Skyrme bench workload: 2048^2, 32 hedgehogs, standard potential."""
    return bs_single(N=2048, count=32, steps=2000)


def cm_demag_bench() -> Workload:
    """Demagnetisation bench workload (not a BASELINE config): config 2's
    multi-skyrmion recipe at 2048^2 with Neel DMI and g = mu0 Ms^2 = 1."""
    w = cm_multi(N=2048, count=64, margin=12.0, min_sep=16.0)
    w.name, w.demag, w.dmi, w.K = "cm_demag_2048", 1.0, DMI_NEEL, 0.1
    return w


def baseline_config(c: int, **kw) -> Workload:
    """BASELINE.json configs[c-1] at full size (override sizes with kw for scaled copies)."""
    return {1: cm_single, 2: cm_multi, 3: ah_vortices, 4: cm_quench, 5: cm_sweep}[c](**kw)
