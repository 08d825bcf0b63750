"""Pins for the oracle's stencils (PAPER.md:104 eq. 1, :109 eq. 2) and tree reduction."""
import math

import numpy as np
import pytest

import oracle


def _grid(Nx, Ny, h):
    x = (np.arange(Nx) - 3.0) * h
    y = (np.arange(Ny) - 5.0) * h
    return np.meshgrid(x, y)


INT = (slice(2, -2), slice(2, -2))


@pytest.mark.parametrize("deg", range(0, 6))
def test_polynomial_exactness(deg):
    # eq. (1) is exact for degree <= 4, eq. (2) for degree <= 5; one degree higher must fail.
    h = 0.37
    X, Y = _grid(13, 11, h)
    f = (0.3 + X) ** deg + 2.0 * (Y - 0.1) ** deg + (X * Y if deg >= 2 else 0.0)
    dfx = deg * (0.3 + X) ** max(deg - 1, 0) + (Y if deg >= 2 else 0.0)
    dfy = 2.0 * deg * (Y - 0.1) ** max(deg - 1, 0) + (X if deg >= 2 else 0.0)
    d2x = deg * (deg - 1) * (0.3 + X) ** max(deg - 2, 0)
    d2y = 2.0 * deg * (deg - 1) * (Y - 0.1) ** max(deg - 2, 0)
    dxy = np.ones_like(X) if deg >= 2 else np.zeros_like(X)
    scale = np.abs(f).max() / h ** 2
    if deg <= 4:
        assert np.abs(oracle.stencil("Dx", f, h) - dfx)[INT].max() <= 1e-13 * scale
        assert np.abs(oracle.stencil("Dy", f, h) - dfy)[INT].max() <= 1e-13 * scale
        assert np.abs(oracle.stencil("DxDy", f, h) - dxy)[INT].max() <= 1e-12 * scale
    assert np.abs(oracle.stencil("Lx", f, h) - d2x)[INT].max() <= 1e-12 * scale
    assert np.abs(oracle.stencil("Ly", f, h) - d2y)[INT].max() <= 1e-12 * scale


def test_first_failing_degree():
    h = 0.5
    X, Y = _grid(12, 12, h)
    # x^5: eq. (1) error = -(h^4/30) f^(5) = -4 h^4 ; x^6: eq. (2) error = -(h^4/90) f^(6) = -8 h^4
    e1 = (oracle.stencil("Dx", X ** 5, h) - 5 * X ** 4)[INT]
    assert np.allclose(e1, -4.0 * h ** 4, rtol=0, atol=1e-9)
    e2 = (oracle.stencil("Lx", X ** 6, h) - 30 * X ** 4)[INT]
    assert np.allclose(e2, -8.0 * h ** 4, rtol=0, atol=1e-8)


@pytest.mark.parametrize("q", [0.3, 1.1, 2.9])
def test_plane_wave_symbols(q):
    h = 0.2
    X, Y = _grid(16, 14, h)
    s = (8 * math.sin(q * h) - math.sin(2 * q * h)) / (6 * h)
    t2 = (30 - 32 * math.cos(q * h) + 2 * math.cos(2 * q * h)) / (12 * h * h)
    assert np.abs(oracle.stencil("Dx", np.sin(q * X), h) - s * np.cos(q * X))[INT].max() < 1e-12
    assert np.abs(oracle.stencil("Dy", np.cos(q * Y), h) + s * np.sin(q * Y))[INT].max() < 1e-12
    assert np.abs(oracle.stencil("Lx", np.sin(q * X), h) + t2 * np.sin(q * X))[INT].max() < 1e-11
    assert np.abs(oracle.stencil("Ly", np.cos(q * Y), h) + t2 * np.cos(q * Y))[INT].max() < 1e-11
    f = np.sin(q * X) * np.cos(0.7 * q * Y)
    s2 = (8 * math.sin(0.7 * q * h) - math.sin(1.4 * q * h)) / (6 * h)
    ref = -s * s2 * np.cos(q * X) * np.sin(0.7 * q * Y)
    assert np.abs(oracle.stencil("DxDy", f, h) - ref)[INT].max() < 1e-11


def test_halo_is_zero_and_transposition():
    rng = np.random.default_rng(1)
    f = rng.standard_normal((9, 12))
    for op in ("Dx", "Dy", "Lx", "Ly", "DxDy"):
        out = oracle.stencil(op, f, 0.3)
        m = np.ones_like(out, dtype=bool)
        m[INT] = False
        assert np.all(out[m] == 0.0)
    # x <-> y: a transposed operand must fail here
    assert np.array_equal(oracle.stencil("Dx", f, 0.3), oracle.stencil("Dy", f.T.copy(), 0.3).T)
    assert np.array_equal(oracle.stencil("Lx", f, 0.3), oracle.stencil("Ly", f.T.copy(), 0.3).T)


def test_tree_sum_order():
    # The aligned pairwise tree is NOT left-to-right: (1e16 + 1) + (-1e16 + 1) pairs differ.
    v = np.array([1e16, 1.0, -1e16, 1.0])
    assert oracle.tree_sum(v) == (1e16 + 1.0) + (-1e16 + 1.0)
    v = np.array([1.0, 1e16, -1e16, 1.0, 3.0])          # padded to 8
    assert oracle.tree_sum(v) == ((1.0 + 1e16) + (-1e16 + 1.0)) + ((3.0 + 0.0) + 0.0)
    rng = np.random.default_rng(7)
    for n in (1, 2, 3, 31, 32, 33, 100):
        x = rng.standard_normal(n)
        ref = np.zeros(1 << max(0, (n - 1).bit_length()))
        ref[:n] = x
        while ref.size > 1:
            ref = ref[0::2] + ref[1::2]
        assert oracle.tree_sum(x) == ref[0]
        assert abs(oracle.tree_sum(x) - math.fsum(x)) < 1e-13 * n


def test_tree_sum2d_rows_then_columns():
    rng = np.random.default_rng(3)
    a = rng.standard_normal((5, 7)) * 10.0 ** rng.integers(-8, 8, size=(5, 7))
    rows = np.array([oracle.tree_sum(r) for r in a])
    assert oracle.tree_sum2d(a) == oracle.tree_sum(rows)
