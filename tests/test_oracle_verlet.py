"""Pins for the oracle's one-gradient-per-step integrator (velocity Verlet with the paper's
projection and arrest; "such as", DESIGN R15).  None of them re-types its formula:
they are the textbook properties of velocity Verlet (second order, bounded energy error), agreement with the separately pinned RK4 flow in the limit dt -> 0, the
constraint, the arrest invariants of eq. (4) and the survey's converged energy of config 1."""
import os

import numpy as np

import oracle
from paper_2603_24370_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "survey_scratch_anchors.txt")


def _gold(key):
    for line in open(GOLD):
        if line.startswith(key + " "):
            return [float(x) for x in line.split()[1:]]
    raise KeyError(key)


def _ah():
    w = W.ah_vortices(N=28, h=0.2, lam=1.0, noise=0.0, centres=[(0.1, -0.2)])
    return w, oracle.model(oracle.AH, 28, 28, 0.2, lam=1.0)


def _run(m, f0, dt, steps, integrator, vel=None):
    fl = oracle.Flow(m, dt, integrator=integrator)
    fl.set_fields(f0, vel)
    E0 = fl.energy
    fl.step(steps)
    s = fl.scalars()
    return fl.get_fields(), s, (s["E"] + s["KE"]) - E0


def test_second_order_and_limit_equals_rk4():
    w, m = _ah()
    T = 0.32
    (ref, vref), s, _ = _run(m, w.fields[0], T / 256, 256, "rk4")
    assert s["n_arrests"] == 0
    errs, verrs = [], []
    for n in (8, 16, 32):
        (phi, vel), s, _ = _run(m, w.fields[0], T / n, n, "verlet")
        assert s["n_arrests"] == 0
        errs.append(np.abs(phi - ref).max())
        verrs.append(np.abs(vel - vref).max())
    for e in (errs, verrs):
        assert 3.6 < e[0] / e[1] < 4.4 and 3.6 < e[1] / e[2] < 4.4, e   # O(dt^2)
    assert errs[2] < 1e-4


def test_first_order_variants_are_excluded():
    # a symplectic-Euler-like scheme (one full kick) would converge with ratio 2, and a scheme
    # with a wrong kick coefficient would not converge to the RK4 trajectory at all: the
    # velocity error at fixed time must shrink by 4 per halving down to the 1e-6 level
    w, m = _ah()
    T = 0.16
    (_, vref), _, _ = _run(m, w.fields[0], T / 512, 512, "rk4")
    e = [np.abs(_run(m, w.fields[0], T / n, n, "verlet")[0][1] - vref).max() for n in (16, 32, 64)]
    assert 3.7 < e[0] / e[1] < 4.3 and 3.7 < e[1] / e[2] < 4.3, e
    assert e[2] < 2e-6


def test_energy_error_is_second_order():
    # E_h + KE is conserved by the continuous flow; velocity Verlet's error in it is O(dt^2)
    w, m = _ah()
    T = 0.32
    d = []
    for n in (8, 16, 32):
        _, s, drift = _run(m, w.fields[0], T / n, n, "verlet")
        assert s["n_arrests"] == 0
        d.append(abs(drift))
    assert 3.4 < d[0] / d[1] < 4.6 and 3.4 < d[1] / d[2] < 4.6, d


def test_constraint_tangency_and_arrest_invariants():
    w = W.cm_single(N=32)
    m = oracle.model(oracle.CM, 32, 32, w.h, kappa=1.0, B=0.6)
    fl = oracle.Flow(m, w.dt, integrator="verlet")
    fl.set_fields(w.fields[0])
    inter = W.interior_mask(32, 32)
    E_prev, logged = fl.energy, []
    for n in range(1, 81):
        fl.step(1)
        phi, vel = fl.get_fields()
        s = fl.scalars()
        assert abs((phi * phi).sum(0)[inter] - 1.0).max() < 1e-14
        assert abs((phi * vel).sum(0)[inter]).max() < 1e-13
        if s["E"] > E_prev:                                  # eq. (4), strict
            logged.append(n)
            assert s["v_is_zero"] == 1 and np.abs(vel).max() == 0.0
        else:
            assert s["v_is_zero"] == 0
        E_prev = s["E"]
    assert fl.arrests() == logged and len(logged) >= 1
    assert np.array_equal(phi[:, ~inter], w.fields[0][:, ~inter])   # frozen halo


def test_converges_to_the_survey_minimum_of_config1():
    # independent anchor: SURVEY 8(c6) converged E, Q of config 1 (tests/golden)
    w = W.baseline_config(1)
    m = oracle.model(oracle.CM, w.Nx, w.Ny, w.h, kappa=w.kappa, B=w.B, K=w.K)
    fl = oracle.Flow(m, w.dt, integrator="verlet")
    fl.set_fields(w.fields[0])
    E0 = fl.energy
    fl.step(1500)
    E1 = fl.energy
    fl.step(1500)
    # without RK4's damping of the stiffest modes (omega dt = 1.6) the late flow arrests every
    # other step and creeps; it approaches the same minimum from above
    gold = _gold("E_converged")[0]
    assert gold < fl.energy < E1 < E0
    assert fl.energy - gold < 2e-5
    assert abs(fl.charge - _gold("Q_converged")[0]) < 1e-6
