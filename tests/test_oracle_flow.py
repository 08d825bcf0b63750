"""Pins for the oracle's arrested Newton flow (PAPER.md:117-127, :129+154; DESIGN R5-R8)."""
import math
import os

import numpy as np
import pytest

import oracle
from paper_2603_24370_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "survey_scratch_anchors.txt")


def _gold():
    d = {}
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        k, *v = line.split()
        d[k] = [float(x) for x in v]
    return d


def _cm_flow(w):
    m = oracle.model(oracle.CM, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K)
    fl = oracle.Flow(m, w.dt)
    fl.set_fields(w.fields[0])
    return m, fl


def test_default_time_step_is_half_courant():
    # C = dt/dx = 0.5 by default -> dt<=0 must behave exactly like dt = h/2
    w = W.cm_single(N=24)
    m = oracle.model(oracle.CM, 24, 24, w.h, kappa=1.0, B=0.6)
    a, b = oracle.Flow(m, 0.0), oracle.Flow(m, 0.5 * w.h)
    for fl in (a, b):
        fl.set_fields(w.fields[0])
        fl.step(5)
    assert np.array_equal(a.get_fields()[0], b.get_fields()[0])


def test_rk4_order_unconstrained():
    """AH from rest, no arrest inside the window: field error ratio ~16 on halving dt,
    drift of E_h + KE ratio ~32 (classical RK4)."""
    w = W.ah_vortices(N=28, h=0.2, lam=1.0, noise=0.0, centres=[(0.1, -0.2)])
    m = oracle.model(oracle.AH, 28, 28, 0.2, lam=1.0)
    T = 0.32

    def run(dt):
        fl = oracle.Flow(m, dt)
        fl.set_fields(w.fields[0])
        E0 = fl.energy
        fl.step(round(T / dt))
        s = fl.scalars()
        assert s["n_arrests"] == 0
        return fl.get_fields(), (s["E"] + s["KE"]) - E0
    (ref, vref), _ = run(T / 256)
    errs, drifts = [], []
    for dt in (T / 4, T / 8, T / 16):
        (phi, vel), dr = run(dt)
        errs.append(max(np.abs(phi - ref).max(), np.abs(vel - vref).max()))
        drifts.append(abs(dr))
    assert 12.0 < errs[0] / errs[1] < 20.0 and 12.0 < errs[1] / errs[2] < 20.0
    assert 24.0 < drifts[0] / drifts[1] < 40.0


def test_constrained_scheme_is_first_order_in_dt():
    """SURVEY 8(c6) "Constrained scheme ... error ratio ~2" (survey scratch: 2.02).  Chiral magnet
    from rest, no arrest inside the window, fixed final time: with the projection of
    PAPER.md:129+154 applied to every stage field and stage gradient and NO centripetal term
    (DESIGN R7) the RK4 stages are consistent only to first order on the sphere, so field and
    velocity errors halve with dt -- where the unconstrained theory shows ~16
    (test_rk4_order_unconstrained).  A different placement of the projections (projecting only
    the final field, or adding the -|v|^2 n term) changes this order."""
    w = W.cm_single(N=32, noise=0.0)
    m = oracle.model(oracle.CM, 32, 32, w.h, kappa=1.0, B=0.6)
    T = 0.2

    def run(dt):
        fl = oracle.Flow(m, dt)
        fl.set_fields(w.fields[0])
        fl.step(round(T / dt))
        assert fl.scalars()["n_arrests"] == 0
        return fl.get_fields()
    ref, vref = run(T / 512)
    ef, ev = [], []
    for dt in (T / 4, T / 8, T / 16, T / 32):
        phi, vel = run(dt)
        ef.append(np.abs(phi - ref).max())
        ev.append(np.abs(vel - vref).max())
    for e in (ef, ev):
        for a, b in zip(e, e[1:]):
            assert 1.8 < a / b < 2.4, (ef, ev)


def test_newton_flow_is_second_order_in_time_from_rest():
    # phi(dt) - phi(0) = -dt^2/2 G + O(dt^4) from rest (eq. 3): catches a wrong mass / sign
    w = W.ah_vortices(N=20, h=0.2, lam=1.0, noise=0.05, centres=[(0.0, 0.0)])
    m = oracle.model(oracle.AH, 20, 20, 0.2, lam=1.0)
    G = oracle.gradient(m, w.fields[0])
    dt = 1e-3
    fl = oracle.Flow(m, dt)
    fl.set_fields(w.fields[0])
    fl.step(1)
    phi, vel = fl.get_fields()
    assert np.abs((phi - w.fields[0]) + 0.5 * dt * dt * G).max() < 1e-10
    assert np.abs(vel + dt * G).max() < 1e-3 * dt * np.abs(G).max()


def test_constraint_and_tangency():
    w = W.cm_single(N=32)
    m, fl = _cm_flow(w)
    for _ in range(40):
        fl.step(1)
        n, v = fl.get_fields()
        assert np.abs((n * n).sum(0) - 1.0).max() < 4e-15
        assert np.abs((n * v).sum(0)).max() < 1e-14
    # halo never changes
    mask = W.interior_mask(32, 32)
    assert np.array_equal(n[:, ~mask], w.fields[0][:, ~mask])


def test_arrest_invariants_and_survey_anchors():
    g = _gold()
    w0 = W.cm_single(noise=0.0)
    m, fl = _cm_flow(w0)
    assert abs(fl.energy - g["E0_no_noise"][0]) < 5e-9
    w = W.cm_single()
    m, fl = _cm_flow(w)
    E = [fl.energy]
    logged_v_zero = True
    for n in range(1, 1001):
        fl.step(1)
        s = fl.scalars()
        E.append(s["E"])
        if s["v_is_zero"]:
            logged_v_zero &= bool(np.all(fl.get_fields()[1] == 0.0))
    arrests = fl.arrests()
    assert arrests[:4] == [int(x) for x in g["first_arrests"]]
    assert logged_v_zero
    assert E[1] < E[0]                                   # first step from rest descends
    assert E[-1] < E[0]
    aset = set(arrests)
    for n in range(1, 1001):                              # eq. (4), strict >
        assert (E[n] > E[n - 1]) == (n in aset)
    for a, b in zip(arrests, arrests[1:]):                # a step from rest is a descent step
        if abs(E[a] - E[a - 1]) > 1e-12 * abs(E[a]):
            assert b != a + 1
    assert abs(E[-1] - g["E_converged"][0]) < 1e-9
    assert abs(fl.charge - g["Q_converged"][0]) < 1e-7
    # same minimum for a different noise seed
    m, fl2 = _cm_flow(W.cm_single(seed_offset=17))
    fl2.step(1000)
    assert abs(fl2.energy - g["E_converged"][0]) < 1e-9


def test_initial_velocity_and_restart_roundtrip():
    # get_fields -> set_fields continues the same trajectory if E_prev is re-primed one step
    w = W.cm_single(N=32)
    m, a = _cm_flow(w)
    a.step(7)
    phi, vel = a.get_fields()
    assert a.scalars()["v_is_zero"] == 0
    b = oracle.Flow(m, w.dt)
    b.set_fields(phi, vel)
    a.step(3)
    b.step(3)
    assert np.abs(a.get_fields()[0] - b.get_fields()[0]).max() < 1e-15
    assert b.scalars()["steps"] == 3


@pytest.mark.parametrize("lam", [1.0, 2.0])
def test_bogomolny_bound(lam):
    """lambda = 1: relaxed E -> pi |N| (E_A tight, E_h within the boundary functional);
    lambda = 2 (type II): E > pi |N|."""
    N, h = 100, 0.2
    w = W.ah_vortices(N=N, h=h, lam=lam, noise=1e-3, centres=[(0.0, 0.0)])
    m = oracle.model(oracle.AH, N, N, h, lam=lam)
    fl = oracle.Flow(m, w.dt)
    fl.set_fields(w.fields[0])
    E0 = fl.energy
    fl.step(1500)
    phi, _ = fl.get_fields()
    EA, Nv = oracle.energy_charge(m, phi, literal=True)
    assert abs(Nv - 1.0) < 1e-4 and fl.energy < E0
    if lam == 1.0:
        assert abs(EA / math.pi - 1.0) < 1e-4
        assert abs(fl.energy / math.pi - 1.0) < 2e-2
    else:
        assert EA / math.pi > 1.1 and fl.energy / math.pi > 1.1
