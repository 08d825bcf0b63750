"""Pins for the oracle's general DMI term (eq. (5): D sum_i d_i.(n x d_i n); DESIGN
R16).  Exact derivative by brute force, agreement with the separately pinned Bloch special case,
and two analytic covariances of eq. (5): a proper spin rotation R about e3 maps (n, d) -> (Rn, Rd)
and an improper spin mirror M maps (n, d) -> (Mn, -Md), both leaving E unchanged (the triple
product d.(n x dn) is a pseudo-scalar; exchange, Zeeman and anisotropy only see n3 and |dn|)."""
import numpy as np
import pytest

import oracle
from paper_2603_24370_b200 import workloads as W
from tests.test_oracle_energy import INT, _fd_gradient

ROT90 = np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])     # about e3
MIRY = np.diag([1.0, -1.0, 1.0])


def _apply(A, f):
    return np.einsum("ab,bji->aji", A, f)


def _table(A, d, sign=1.0):
    return tuple(tuple(sign * (A @ np.array(v))) for v in d)


def test_gradient_is_exact_derivative_with_a_random_table():
    rng = np.random.default_rng(21)
    d = rng.standard_normal(6)
    m = oracle.model(oracle.CM, 9, 8, 0.25, kappa=0.8, B=0.4, K=0.2, dmi=d)
    f = rng.standard_normal((3, 8, 9))
    G, Gfd = oracle.gradient(m, f), _fd_gradient(m, f)
    assert np.abs(G - Gfd)[INT].max() <= 1e-8 * np.abs(Gfd).max()
    E, _, de, _ = oracle.energy_charge(m, f, densities=True)
    assert abs(E - oracle.energy_bond(m, f)) <= 1e-13 * m.h ** 2 * np.abs(de).sum()   # site = bond


def test_bloch_table_reproduces_the_default_path():
    rng = np.random.default_rng(22)
    f = rng.standard_normal((3, 12, 10))
    a = oracle.model(oracle.CM, 10, 12, 0.2, kappa=1.0, B=0.6, K=0.3)
    b = oracle.model(oracle.CM, 10, 12, 0.2, kappa=1.0, B=0.6, K=0.3, dmi=W.DMI_BLOCH)
    assert abs(oracle.energy_bond(a, f) - oracle.energy_bond(b, f)) < 1e-11
    assert abs(oracle.energy_charge(a, f)[0] - oracle.energy_charge(b, f)[0]) < 1e-11
    assert np.abs(oracle.gradient(a, f) - oracle.gradient(b, f)).max() < 1e-11


def test_named_tables_are_the_rotation_and_the_mirror_of_bloch():
    assert np.allclose(_table(ROT90, W.DMI_BLOCH), W.DMI_NEEL)
    assert np.allclose(_table(MIRY, W.DMI_BLOCH, -1.0), W.DMI_D2D)


@pytest.mark.parametrize("A,sign,name", [(ROT90, 1.0, "neel"), (MIRY, -1.0, "d2d")])
def test_spin_covariance_of_energy_gradient_and_flow(A, sign, name):
    w = W.cm_single(N=32)
    f = w.fields[0]
    d2 = _table(A, W.DMI_BLOCH, sign)
    a = oracle.model(oracle.CM, 32, 32, w.h, kappa=1.0, B=0.6, K=0.2)
    b = oracle.model(oracle.CM, 32, 32, w.h, kappa=1.0, B=0.6, K=0.2, dmi=d2)
    Af = _apply(A, f)
    Ea, Qa = oracle.energy_charge(a, f)
    Eb, Qb = oracle.energy_charge(b, Af)
    assert abs(Ea - Eb) < 1e-11 and abs(Qb - np.linalg.det(A) * Qa) < 1e-12
    assert np.abs(_apply(A, oracle.gradient(a, f)) - oracle.gradient(b, Af)).max() < 1e-11
    fa, fb = oracle.Flow(a, w.dt), oracle.Flow(b, w.dt)
    fa.set_fields(f)
    fb.set_fields(Af)
    fa.step(40)
    fb.step(40)
    assert fa.arrests() == fb.arrests() and len(fa.arrests()) >= 1
    assert np.abs(_apply(A, fa.get_fields()[0]) - fb.get_fields()[0]).max() < 1e-11
    if name == "d2d":                      # the mirrored hedgehog is an antiskyrmion: Q = +1
        assert abs(fb.charge - 1.0) < 5e-3
