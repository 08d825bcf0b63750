"""Pins for the oracle's discrete energies, gradients and charges (DESIGN R1-R3, R9).

Nothing here re-types the oracle's formulas: the gradient is pinned to brute-force
differences of the plain bond-sum energy, the energies to closed forms / vacuum /
continuum quadrature, the charges to integers.
"""
import math

import numpy as np
import pytest
from scipy import integrate

import oracle
from paper_2603_24370_b200 import workloads as W

INT = (slice(None), slice(2, -2), slice(2, -2))


def _fd_gradient(m, f, eps=1e-6):
    """(1/h^2) dE_bond/df by central differences over every interior degree of freedom."""
    G = np.zeros_like(f)
    C, Ny, Nx = f.shape
    for c in range(C):
        for j in range(2, Ny - 2):
            for i in range(2, Nx - 2):
                fp, fm = f.copy(), f.copy()
                fp[c, j, i] += eps
                fm[c, j, i] -= eps
                G[c, j, i] = (oracle.energy_bond(m, fp) - oracle.energy_bond(m, fm)) / (2 * eps)
    return G / m.h ** 2


@pytest.mark.parametrize("halo", ["vacuum", "random"])
def test_cm_gradient_is_exact_derivative_of_bond_energy(halo):
    rng = np.random.default_rng(11)
    m = oracle.model(oracle.CM, 8, 8, 0.2, kappa=0.9, B=0.6, K=0.3)
    f = rng.standard_normal((3, 8, 8))          # non-unit on purpose: ambient-space gradient
    if halo == "vacuum":
        mask = W.interior_mask(8, 8)
        f[:, ~mask] = np.array([0.0, 0.0, 1.0])[:, None]
    G = oracle.gradient(m, f)
    Gfd = _fd_gradient(m, f)
    assert np.abs(G - Gfd)[INT].max() <= 1e-8 * np.abs(Gfd).max()


def test_ah_gradient_is_exact_derivative_of_bond_energy():
    rng = np.random.default_rng(12)
    m = oracle.model(oracle.AH, 8, 8, 0.1, lam=1.7)
    f = rng.standard_normal((4, 8, 8))
    G = oracle.gradient(m, f)
    Gfd = _fd_gradient(m, f)
    assert np.abs(G - Gfd)[INT].max() <= 1e-8 * np.abs(Gfd).max()
    # rectangular lattice, different seed: catches an Nx/Ny mix-up
    m = oracle.model(oracle.AH, 9, 7, 0.3, lam=0.5)
    f = rng.standard_normal((4, 7, 9))
    Gfd = _fd_gradient(m, f)
    assert np.abs(oracle.gradient(m, f) - Gfd)[INT].max() <= 1e-8 * np.abs(Gfd).max()


@pytest.mark.parametrize("theory,shape", [(oracle.CM, (3, 11, 14)), (oracle.AH, (4, 12, 9))])
def test_site_form_equals_bond_form(theory, shape):
    rng = np.random.default_rng(5)
    f = rng.standard_normal(shape)
    m = oracle.model(theory, shape[2], shape[1], 0.25, kappa=1.3, B=0.4, K=0.2, lam=2.0)
    Eb = oracle.energy_bond(m, f)
    Es, _ = oracle.energy_charge(m, f)
    assert abs(Es - Eb) <= 1e-13 * max(abs(Eb), 1.0) * 10


def test_cm_vacuum():
    m = oracle.model(oracle.CM, 12, 10, 0.2, kappa=1.0, B=0.6, K=0.3)
    f = np.zeros((3, 10, 12))
    f[2] = 1.0
    E, Q = oracle.energy_charge(m, f)
    assert E == 0.0 and Q == 0.0 and oracle.energy_bond(m, f) == 0.0
    G = oracle.gradient(m, f)
    assert np.all(G[0][2:-2, 2:-2] == 0.0) and np.all(G[1][2:-2, 2:-2] == 0.0)
    assert np.allclose(G[2][2:-2, 2:-2], -(0.6 + 2 * 0.3), rtol=0, atol=1e-15)
    assert np.all(oracle.accel(m, f) == 0.0)


def test_ah_vacuum():
    m = oracle.model(oracle.AH, 10, 12, 0.1, lam=1.0)
    f = np.zeros((4, 12, 10))
    f[0] = 1.0
    E, Q = oracle.energy_charge(m, f)
    assert E == 0.0 and Q == 0.0 and oracle.energy_bond(m, f) == 0.0
    assert np.all(oracle.gradient(m, f) == 0.0)
    # a pure gauge transform of the vacuum by a constant phase is also a zero
    f[0], f[1] = math.cos(0.7), math.sin(0.7)
    assert abs(oracle.energy_charge(m, f)[0]) < 1e-13


def test_cm_helix_closed_form():
    # textbook spin spiral n = (0, sin qx, cos qx) on every site incl. halo
    h, q, kappa, B, K = 0.2, 0.83, 1.1, 0.6, 0.3
    Nx, Ny = 24, 16
    X, _ = W.coords(Nx, Ny, h)
    f = np.stack([np.zeros_like(X), np.sin(q * X), np.cos(q * X)])
    m = oracle.model(oracle.CM, Nx, Ny, h, kappa=kappa, B=B, K=K)
    s = (8 * math.sin(q * h) - math.sin(2 * q * h)) / (6 * h)
    t2 = (30 - 32 * math.cos(q * h) + 2 * math.cos(2 * q * h)) / (12 * h * h)
    _, _, de, dq = oracle.energy_charge(m, f, densities=True)
    deep = (slice(4, -4), slice(4, -4))
    e_ref = ((4 / 3) * (1 - math.cos(q * h)) - (1 / 12) * (1 - math.cos(2 * q * h))) / h ** 2 \
        + kappa * s + B * (1 - np.cos(q * X)) + K * np.sin(q * X) ** 2
    assert np.abs(de - e_ref)[deep].max() < 1e-12
    assert np.abs(dq)[deep].max() < 1e-14          # coplanar texture: no charge
    G = oracle.gradient(m, f)
    G_ref = (t2 + 2 * kappa * s) * f
    G_ref[2] -= B + 2 * K * f[2]
    assert np.abs(G - G_ref)[INT].max() < 1e-11
    # kappa -> -kappa flips the DMI sign (a wrong sign would pass a symmetric test only)
    m2 = oracle.model(oracle.CM, Nx, Ny, h, kappa=-kappa, B=B, K=K)
    _, _, de2, _ = oracle.energy_charge(m2, f, densities=True)
    assert np.abs((de - de2) - 2 * kappa * s)[deep].max() < 1e-12


def test_cm_charge_is_integer_degree():
    w = W.cm_single(N=64, noise=0.0)
    m = oracle.model(oracle.CM, 64, 64, w.h, kappa=1.0, B=0.6)
    _, Q = oracle.energy_charge(m, w.fields[0])
    assert abs(Q + 1.0) < 5e-3                      # hedgehog ansatz: degree -1
    w2 = W.cm_single(N=64, noise=0.0, mirror=True)
    assert abs(oracle.energy_charge(m, w2.fields[0])[1] - 1.0) < 5e-3
    w3 = W.cm_multi(N=512, count=5, noise=0.0)
    m3 = oracle.model(oracle.CM, 512, 512, w3.h, kappa=1.0, B=0.6)
    assert abs(oracle.energy_charge(m3, w3.fields[0])[1] + 5.0) < 1e-2
    # unit-sphere area element: n -> -n flips the sign of q
    assert abs(oracle.energy_charge(m, -w.fields[0])[1] - 1.0) < 5e-3


def test_ah_vortex_flux_and_ansatz_energy():
    """Single vortex f = tanh r, a = tanh^2 r: flux = 1 and the literal lattice energy
    converges at 4th order to the 1-D radial quadrature of the continuum functional."""
    lam = 1.0

    def dens(r):
        f, a = math.tanh(r), math.tanh(r) ** 2
        fp = 1 - f * f
        ap = 2 * f * fp
        return r * (fp ** 2 + (1 - a) ** 2 * f ** 2 / r ** 2 + ap ** 2 / r ** 2
                    + (lam / 4) * (1 - f * f) ** 2)
    I, _ = integrate.quad(dens, 1e-12, 40.0, limit=400, epsabs=1e-13, epsrel=1e-13)
    assert abs(I - 1.449699006) < 1e-8               # SURVEY 8(c6) value reproduced
    errs = []
    for N, h in ((200, 0.1), (400, 0.05)):
        w = W.ah_vortices(N=N, h=h, lam=lam, noise=0.0, centres=[(0.0, 0.0)])
        m = oracle.model(oracle.AH, N, N, h, lam=lam)
        EA, Nv = oracle.energy_charge(m, w.fields[0], literal=True)
        assert abs(Nv - 1.0) < 1e-6
        errs.append(abs(EA / math.pi - I))
    assert errs[0] < 1e-4 and 10.0 < errs[0] / errs[1] < 24.0
    # anti-vortex (complex conjugate, A -> -A) has flux -1 and the same energy
    f = w.fields[0].copy()
    f[1:] *= -1.0
    EA2, Nv2 = oracle.energy_charge(m, f, literal=True)
    assert abs(Nv2 + 1.0) < 1e-6 and abs(EA2 - EA) < 1e-9


def test_ah_gauge_covariance_of_energy():
    # E_h is invariant under a CONSTANT phase rotation exactly, and the site form follows
    rng = np.random.default_rng(2)
    f = rng.standard_normal((4, 10, 10))
    m = oracle.model(oracle.AH, 10, 10, 0.2, lam=1.3)
    c, s = math.cos(1.1), math.sin(1.1)
    g = f.copy()
    g[0], g[1] = c * f[0] - s * f[1], s * f[0] + c * f[1]
    assert abs(oracle.energy_bond(m, f) - oracle.energy_bond(m, g)) < 1e-11
    G, Gg = oracle.gradient(m, f), oracle.gradient(m, g)
    assert np.abs(Gg[0] - (c * G[0] - s * G[1])).max() < 1e-10
    assert np.abs(Gg[2:] - G[2:]).max() < 1e-10
