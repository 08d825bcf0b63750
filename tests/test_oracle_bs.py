"""Pins for the oracle's baby-Skyrme theory (PAPER.md:323 Table 2, :90; DESIGN R18;
SURVEY 8(f) NEXT-2b).  None of them re-types the oracle's formulas: brute-force differences of
the plain energy, closed forms by 1-D quadrature, the Belavin-Polyakov lump, Derrick's scaling
argument and its virial identity at a relaxed minimum."""
import math

import numpy as np
import pytest
from scipy.integrate import quad

import oracle
from paper_2603_24370_b200 import workloads as W

POTS = [(oracle.POT_STANDARD, 3), (oracle.POT_EASY_PLANE, 3), (oracle.POT_BROKEN, 3),
        (oracle.POT_BROKEN, 2)]


def _model(N, h=0.2, kappa=1.0, mu=1.0, pot=oracle.POT_STANDARD, potN=3, Ny=None):
    return oracle.model(oracle.BS, N, Ny or N, h, kappa=kappa, mu=mu, pot=pot, potN=potN)


@pytest.mark.parametrize("pot,potN", POTS)
@pytest.mark.parametrize("halo", ["vacuum", "random"])
def test_gradient_is_the_exact_derivative_of_the_plain_energy(pot, potN, halo):
    # 12 x 10 lattice (8 x 6 interior): the exact gradient has radius 4, every interior degree of
    # freedom of a random NON-unit field is differentiated by central differences of the plain sum
    rng = np.random.default_rng(11 + pot + potN)
    Nx, Ny, h = 12, 10, 0.2
    m = _model(Nx, h, kappa=0.7, mu=1.3, pot=pot, potN=potN, Ny=Ny)
    f = 0.5 * rng.standard_normal((3, Ny, Nx)) + np.array([0.0, 0.0, 1.0])[:, None, None]
    if halo == "vacuum":
        f[:, ~W.interior_mask(Nx, Ny)] = np.array([0.0, 0.0, 1.0])[:, None]
    G = oracle.gradient(m, f)
    eps = 1e-4          # E is O(100) with a 1/h^4 term: rounding, not truncation, limits smaller steps
    worst = 0.0
    for c in range(3):
        for j in range(2, Ny - 2):
            for i in range(2, Nx - 2):
                fp, fm = f.copy(), f.copy()
                fp[c, j, i] += eps
                fm[c, j, i] -= eps
                d = (oracle.energy_bond(m, fp) - oracle.energy_bond(m, fm)) / (2 * eps) / (h * h)
                worst = max(worst, abs(d - G[c, j, i]) / max(1.0, abs(d)))
    assert worst < 1e-7, worst
    assert np.all(G[:, ~W.interior_mask(Nx, Ny)] == 0.0)


@pytest.mark.parametrize("pot,potN", POTS)
def test_site_form_equals_plain_sum(pot, potN):
    rng = np.random.default_rng(5)
    for Nx, Ny in ((12, 10), (21, 17)):
        m = _model(Nx, 0.15, kappa=0.9, mu=0.8, pot=pot, potN=potN, Ny=Ny)
        f = rng.standard_normal((3, Ny, Nx))
        E, _ = oracle.energy_charge(m, f)
        Ep = oracle.energy_bond(m, f)
        assert abs(E - Ep) <= 1e-12 * abs(Ep)


@pytest.mark.parametrize("pot,potN", POTS)
def test_vacuum_is_a_zero_energy_fixed_point(pot, potN):
    m = _model(16, pot=pot, potN=potN)
    f = np.zeros((3, 16, 16))
    f[2] = 1.0
    E, Q = oracle.energy_charge(m, f)
    assert E == 0.0 and Q == 0.0 and oracle.energy_bond(m, f) == 0.0
    assert np.all(oracle.accel(m, f) == 0.0)              # G is parallel to m: no tangent force


def _profile(r):
    return math.pi * math.exp(-r / 2.0)


def test_hedgehog_closed_forms_by_quadrature():
    """n = (sin f cos th, sin f sin th, cos f), f = pi exp(-r/2): |d1 n x d2 n| = |f' sin f| / r, so
    E4 = (kappa^2/2) 2 pi int (f' sin f)^2 / r dr, E0 = mu^2 2 pi int (1 - cos f) r dr (standard
    potential), E2 = pi int (f'^2 + sin^2 f / r^2) r dr.  The lattice values converge to them."""
    kappa, mu = 0.8, 0.6
    R = 12.8

    def fp(r):
        return -0.5 * _profile(r)
    # the lattice integrates over the interior square of half-width R - 2.5 h; the integrands
    # decay like exp(-r), so the quadrature runs over the inscribed disc and beyond: tail < 1e-4
    I4 = quad(lambda r: (fp(r) * math.sin(_profile(r))) ** 2 / r if r > 0 else 0.0, 0, 40,
              limit=200)[0]
    I0 = quad(lambda r: (1 - math.cos(_profile(r))) * r, 0, 40, limit=200)[0]
    I2 = quad(lambda r: (fp(r) ** 2 + (math.sin(_profile(r)) / r) ** 2) * r if r > 0 else 0.0,
              0, 40, limit=200)[0]
    E4c, E0c, E2c = 0.5 * kappa ** 2 * 2 * math.pi * I4, mu ** 2 * 2 * math.pi * I0, math.pi * I2
    errs = []
    for N, h in ((128, 0.2), (256, 0.1)):
        w = W.bs_single(N=N, h=h, noise=0.0)
        f = w.fields[0]
        E_full, Q = oracle.energy_charge(_model(N, h, kappa=kappa, mu=mu), f)
        E_nok, _ = oracle.energy_charge(_model(N, h, kappa=0.0, mu=mu), f)
        E_nomu, _ = oracle.energy_charge(_model(N, h, kappa=kappa, mu=0.0), f)
        E4, E0 = E_full - E_nok, E_full - E_nomu
        E2 = E_full - E4 - E0
        errs.append((abs(E4 / E4c - 1), abs(E0 / E0c - 1), abs(E2 / E2c - 1)))
        assert abs(Q + 1.0) < 2e-3
    # every term within a few 1e-3 of its closed form at h = 0.2 and within 1e-3 at h = 0.1 (a
    # wrong coefficient, power of h or derivative count is off by a factor >= 2); the Skyrme term,
    # the new code, converges at 4th order
    assert max(errs[0]) < 3e-3 and max(errs[1]) < 1e-3, errs
    assert errs[1][0] < errs[0][0] / 8.0, errs


def test_belavin_polyakov_lump_saturates_the_sigma_model_bound():
    """kappa = mu = 0: E = E2 >= 4 pi |Q| with equality for the lump u = (x + i y)/lam,
    m = (2 Re u, 2 Im u, |u|^2 - 1)/(1 + |u|^2) (m -> e3 at infinity).  On a box of half-width R
    the missing tail is 4 pi lam^2/(lam^2 + R^2)."""
    N, h, lam = 160, 0.1, 1.0
    X, Y = W.coords(N, N, h)
    u2 = (X * X + Y * Y) / lam ** 2
    f = np.stack([2 * X / lam, 2 * Y / lam, u2 - 1.0]) / (1.0 + u2)
    m = _model(N, h, kappa=0.0, mu=0.0)
    E, Q = oracle.energy_charge(m, f)
    R = (N / 2 - 2) * h
    tail = lam ** 2 / (lam ** 2 + R ** 2)                    # of a disc; the square keeps a bit more
    assert abs(abs(Q) - 1.0) < 1.2 * tail
    assert E >= 4 * math.pi * abs(Q) * (1 - 1e-4)            # the bound, up to O(h^4)
    assert abs(E / (4 * math.pi) - 1.0) < 1.5 * tail


def test_derrick_scaling_of_the_three_terms():
    """Under x -> x/s (a hedgehog s times larger) E2 is invariant, E4 -> E4/s^2, E0 -> s^2 E0:
    fixes the powers of h and the derivative counts of the three terms."""
    def terms(s, N, h):
        X, Y = W.coords(N, N, h)
        r = np.hypot(X, Y) / s
        th = np.arctan2(Y, X)
        fr = np.pi * np.exp(-r / 2.0)
        f = np.stack([np.sin(fr) * np.cos(th), np.sin(fr) * np.sin(th), np.cos(fr)])
        f[:, ~W.interior_mask(N, N)] = np.array([0.0, 0.0, 1.0])[:, None]
        full = oracle.energy_charge(_model(N, h, kappa=1.0, mu=1.0), f)[0]
        nok = oracle.energy_charge(_model(N, h, kappa=0.0, mu=1.0), f)[0]
        nomu = oracle.energy_charge(_model(N, h, kappa=1.0, mu=0.0), f)[0]
        E4, E0 = full - nok, full - nomu
        return full - E4 - E0, E4, E0
    a = terms(1.0, 256, 0.1)
    b = terms(2.0, 256, 0.2)                                 # same lattice in units of the soliton
    assert abs(b[0] / a[0] - 1.0) < 1e-10                    # E2: exactly scale invariant on it
    assert abs(b[1] / a[1] - 0.25) < 1e-10 and abs(b[2] / a[2] - 4.0) < 1e-10
    c = terms(2.0, 512, 0.1)                                 # same soliton, finer lattice
    assert abs(c[1] / a[1] - 0.25) < 5e-3 and abs(c[2] / a[2] - 4.0) < 5e-3
    assert abs(c[0] / a[0] - 1.0) < 5e-3


def test_relaxed_baby_skyrmion_obeys_the_derrick_virial_identity():
    """At a minimum E(s) = E2 + E4/s^2 + E0 s^2 is stationary at s = 1: E4 = E0.  The arrested
    flow (gradient with the radius-4 Skyrme force, projection, arrest) must find that state from
    an ansatz that violates it; energy falls monotonically except at logged arrests; the degree
    stays -1 and |m| = 1."""
    N, h, kappa, mu = 80, 0.2, 1.0, 1.0
    w = W.bs_single(N=N, h=h, kappa=kappa, mu=mu)
    m = _model(N, h, kappa=kappa, mu=mu)

    def split(f):
        full = oracle.energy_charge(m, f)[0]
        E4 = full - oracle.energy_charge(_model(N, h, kappa=0.0, mu=mu), f)[0]
        E0 = full - oracle.energy_charge(_model(N, h, kappa=kappa, mu=0.0), f)[0]
        return full, E4, E0
    _, E4i, E0i = split(w.fields[0])
    assert abs(E4i / E0i - 1.0) > 0.3                        # the ansatz is far from virial
    fl = oracle.Flow(m, w.dt)
    fl.set_fields(w.fields[0])
    E = [fl.energy]
    for _ in range(1500):
        fl.step(1)
        E.append(fl.energy)
    arrests = set(fl.arrests())
    assert len(arrests) >= 1
    for n in range(1, len(E)):
        assert (E[n] > E[n - 1]) == (n in arrests)
    phi, _ = fl.get_fields()
    full, E4, E0 = split(phi)
    assert full < E[0] and abs(E4 / E0 - 1.0) < 2e-2
    assert abs(fl.charge + 1.0) < 2e-3
    assert np.abs((phi * phi).sum(0) - 1.0).max() < 4e-15
    assert full > 4 * math.pi                                # E >= E2 + 2 sqrt(E4 E0) > 4 pi |Q|
