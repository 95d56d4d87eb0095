"""Pins for oracle/inflate_oracle.py: the identities of PAPER.md:L229 and the
right-invertibility requirement of L345-347 (Prop. 1)."""
import numpy as np

from oracle import inflate_oracle as Z


def test_identities_and_containment():
    rng = np.random.default_rng(0)
    lo = rng.standard_normal((3, 4, 7))
    hi = lo + rng.uniform(0, 1, lo.shape)
    c, R = Z.inflate(lo, hi, pad=0.0)
    assert np.allclose(c - R, lo, atol=1e-15) and np.allclose(c + R, hi, atol=1e-15)
    c, R = Z.inflate(lo, hi, pad=1e-6)
    assert np.all(c - R <= lo) and np.all(c + R >= hi) and np.all(R > 0)
    assert np.allclose(R - 0.5 * (hi - lo), 1e-6, atol=1e-15)


def test_dense_generator_is_right_invertible_even_for_zero_width():
    lo = np.zeros((2, 5))
    hi = np.zeros((2, 5))
    hi[0, 2] = 0.3
    E = np.array([0.0, 0.0, 0.02, 0.02, 0.0])
    c, R, Ebar = Z.inflate(lo, hi, pad=1e-6, E_diag=E, dense=True)
    assert Ebar.shape == (2, 5, 10)
    for t in range(2):
        assert np.linalg.matrix_rank(Ebar[t]) == 5
        assert np.allclose(Ebar[t] @ np.linalg.pinv(Ebar[t]), np.eye(5), atol=1e-9)
        assert np.allclose(Ebar[t][:, :5], np.diag(E)) and np.allclose(Ebar[t][:, 5:], np.diag(R[t]))


def test_vjp_is_the_transpose_of_the_linear_map():
    rng = np.random.default_rng(1)
    lo, hi = rng.standard_normal(6), rng.standard_normal(6)
    gc, gR = rng.standard_normal(6), rng.standard_normal(6)
    c, R = Z.inflate(lo, hi, pad=0.0)
    glo, ghi = Z.inflate_vjp(gc, gR)
    assert np.isclose(gc @ c + gR @ R, glo @ lo + ghi @ hi)
