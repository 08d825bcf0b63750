"""Pins for the oracle's demagnetisation term (eq. (5) last term, :199-205 eq. (6);
DESIGN R19): the Poisson solve inverts the separately pinned eq. (2) operator,
converges at 4th order to an analytic potential, vanishes for divergence-free textures, and the
energy / gradient pair is exact."""
import numpy as np
import pytest

import oracle
from paper_2603_24370_b200 import workloads as W


def test_poisson_solve_inverts_the_pinned_stencil_operator():
    # psi* arbitrary on the interior, 0 on the halo; rho = (Lx + Ly) psi* from the stencil routine
    # that tests/test_oracle_stencils.py pins; the solve must give psi* back
    rng = np.random.default_rng(3)
    for Nx, Ny, h in ((20, 14, 0.2), (37, 50, 0.13)):
        ps = rng.standard_normal((Ny, Nx)) * W.interior_mask(Nx, Ny)
        rho = oracle.stencil("Lx", ps, h) + oracle.stencil("Ly", ps, h)
        got = oracle.poisson_solve(rho, h)
        assert np.abs(got - ps).max() <= 1e-12 * np.abs(ps).max()
        assert np.all(got[~W.interior_mask(Nx, Ny)] == 0.0)
        # a starting guess does not change the answer
        got2 = oracle.poisson_solve(rho, h, guess=rng.standard_normal((Ny, Nx)))
        assert np.abs(got2 - ps).max() <= 1e-12 * np.abs(ps).max()


def test_poisson_solve_converges_at_fourth_order_to_an_analytic_potential():
    # psi = exp(-r^2 / 2 s^2) (1e-14 at the wall), lap psi = (r^2/s^4 - 2/s^2) psi
    s, L = 1.0, 17.6
    errs = []
    for N in (44, 88, 176):
        h = L / N
        X, Y = W.coords(N, N, h)
        r2 = X * X + Y * Y
        psi = np.exp(-r2 / (2 * s * s))
        rho = (r2 / s ** 4 - 2 / s ** 2) * psi
        got = oracle.poisson_solve(rho, h)
        errs.append(np.abs(got - psi).max())
    assert 12.0 < errs[0] / errs[1] < 20.0 and 12.0 < errs[1] / errs[2] < 20.0, errs
    assert errs[2] < 1e-5


def _cm(N, g, dmi=None, Ny=None):
    return oracle.model(oracle.CM, N, Ny or N, 0.2, kappa=1.0, B=0.6, K=0.1, dmi=dmi, demag=g)


def test_divergence_free_textures_have_no_demag_field():
    # n1 depends on y only, n2 on x only: D_x n1 + D_y n2 = 0 exactly -> psi = 0, E_d = 0
    N = 24
    X, Y = W.coords(N, N, 0.2)
    f = np.stack([np.sin(Y), np.cos(0.7 * X), 0.3 + 0 * X])
    m0, m1 = _cm(N, 0.0), _cm(N, 2.5)
    # (eq. (1) as printed leaves a rounding residue of a few 1e-16 on a constant row)
    assert np.abs(oracle.demag_potential(m1, f)).max() < 1e-13
    E0, E1 = oracle.energy_charge(m0, f)[0], oracle.energy_charge(m1, f)[0]
    assert abs(E1 - E0) <= 1e-13 * abs(E0)
    assert np.abs(oracle.gradient(m1, f) - oracle.gradient(m0, f)).max() < 1e-11


def test_demag_energy_is_positive_and_equals_minus_half_g_psi_rho():
    # summation by parts with the exact solve: (g/2) sum_bonds J (dpsi)^2 = -(g/2) h^2 sum psi rho
    w = W.cm_single(N=48, noise=0.05)
    f, h, g = w.fields[0], w.h, 1.7
    m0, m1 = _cm(48, 0.0), _cm(48, g)
    Ed = oracle.energy_bond(m1, f) - oracle.energy_bond(m0, f)
    psi = oracle.demag_potential(m1, f)
    rho = oracle.stencil("Dx", f[0], h) + oracle.stencil("Dy", f[1], h)
    assert Ed > 0.0
    assert abs(Ed + 0.5 * g * h * h * float((psi * rho).sum())) <= 1e-10 * Ed
    # site form == plain sum
    E1, _ = oracle.energy_charge(m1, f)
    assert abs(E1 - oracle.energy_bond(m1, f)) <= 1e-12 * abs(E1)


@pytest.mark.parametrize("halo", ["vacuum", "random"])
def test_gradient_with_demag_is_the_exact_derivative(halo):
    # every evaluation of the plain energy solves its own Poisson problem; random non-unit field
    rng = np.random.default_rng(9)
    Nx, Ny, h = 10, 9, 0.2
    m = oracle.model(oracle.CM, Nx, Ny, h, kappa=0.8, B=0.4, K=0.2, demag=1.9)
    f = rng.standard_normal((3, Ny, Nx))
    if halo == "vacuum":
        f[:, ~W.interior_mask(Nx, Ny)] = np.array([0.0, 0.0, 1.0])[:, None]
    G = oracle.gradient(m, f)
    eps, worst = 1e-5, 0.0
    for c in range(3):
        for j in range(2, Ny - 2):
            for i in range(2, Nx - 2):
                fp, fm = f.copy(), f.copy()
                fp[c, j, i] += eps
                fm[c, j, i] -= eps
                d = (oracle.energy_bond(m, fp) - oracle.energy_bond(m, fm)) / (2 * eps) / (h * h)
                worst = max(worst, abs(d - G[c, j, i]) / max(1.0, abs(d)))
    assert worst < 1e-7, worst


def test_demag_separates_bloch_and_neel_skyrmions():
    """"the inclusion of demagnetization breaks the degeneracy between different
    DMI realizations".  A Bloch skyrmion (helicity pi/2) is divergence-free in the continuum, a
    Neel hedgehog is not: E_d(Neel) >> E_d(Bloch) ~ discretisation error."""
    N, h, g = 96, 0.2, 1.0
    X, Y = W.coords(N, N, h)
    r, th = np.hypot(X, Y), np.arctan2(Y, X)
    fr = np.pi * np.exp(-r / 2.0)
    neel = np.stack([np.sin(fr) * np.cos(th), np.sin(fr) * np.sin(th), np.cos(fr)])
    bloch = np.stack([-np.sin(fr) * np.sin(th), np.sin(fr) * np.cos(th), np.cos(fr)])
    m = _cm(N, g)
    Ed = {}
    for name, f in (("neel", neel), ("bloch", bloch)):
        f[:, ~W.interior_mask(N, N)] = np.array([0.0, 0.0, 1.0])[:, None]
        Ed[name] = oracle.energy_bond(m, f) - oracle.energy_bond(_cm(N, 0.0), f)
    assert Ed["neel"] > 1.0 and Ed["bloch"] < 1e-3 * Ed["neel"], Ed


def test_flow_with_demag_keeps_the_arrest_invariants():
    w = W.cm_single(N=40)
    m = oracle.model(oracle.CM, 40, 40, w.h, kappa=1.0, B=0.6, demag=0.8)
    for integ in ("rk4", "verlet"):
        fl = oracle.Flow(m, w.dt, integrator=integ)
        fl.set_fields(w.fields[0])
        E = [fl.energy]
        for _ in range(60):
            fl.step(1)
            E.append(fl.energy)
        arrests = set(fl.arrests())
        assert E[-1] < E[0]
        for n in range(1, len(E)):
            assert (E[n] > E[n - 1]) == (n in arrests)
        phi, vel = fl.get_fields()
        assert np.abs((phi * phi).sum(0) - 1.0).max() < 4e-15
