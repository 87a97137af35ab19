"""Pins for oracle O1 (Chebyshev modal derivative; Eqs. 14-18) and the GL rule.

Each pin is something the mathematics fixes independently of the oracle's own formula:
exactness on monomials, the textbook collocation matrix, quadrature exactness.
"""
import numpy as np
import pytest


@pytest.mark.parametrize("N", [2, 3, 5, 8, 16, 24, 33])
def test_monomials_exact(oracle, N):
    x = oracle.cheb_nodes(N)
    assert np.all(np.diff(x) > 0) and x[0] == -1.0 and x[-1] == 1.0
    for p in range(N):  # S7: N points => exact to degree N-1
        du = oracle.cheb_derivative_line(x**p)
        ex = p * x ** (p - 1) if p > 0 else np.zeros(N)
        assert np.abs(du - ex).max() <= 2e-13 * max(1.0, p * p), (N, p)


def textbook_cgl_matrix(x):
    """D_ij = (c_i/c_j) (-1)^(i+j) / (x_i - x_j), i != j; closed-form diagonal (Canuto et al.;
    Trefethen, Spectral Methods in MATLAB, ch. 6) for ascending nodes x_j = -cos(pi j/(N-1))."""
    N = len(x)
    c = np.ones(N)
    c[0] = c[-1] = 2.0
    D = np.zeros((N, N))
    for i in range(N):
        for j in range(N):
            if i != j:
                D[i, j] = (c[i] / c[j]) * (-1.0) ** (i + j) / (x[i] - x[j])
    for j in range(1, N - 1):
        D[j, j] = -x[j] / (2.0 * (1.0 - x[j] ** 2))
    D[0, 0] = -(2.0 * (N - 1) ** 2 + 1.0) / 6.0
    D[-1, -1] = (2.0 * (N - 1) ** 2 + 1.0) / 6.0
    return D


@pytest.mark.parametrize("N", [4, 9, 16, 24])
def test_traced_matrix_is_textbook(oracle, N):
    """delta-function tracing: feeding e_k returns column k of D."""
    x = -np.cos(np.pi * np.arange(N) / (N - 1))
    D = np.stack([oracle.cheb_derivative_line(np.eye(N)[k]) for k in range(N)], axis=1)
    ref = textbook_cgl_matrix(x)
    assert np.abs(D - ref).max() <= 1e-12 * np.abs(ref).max()
    assert np.abs(D.sum(axis=1)).max() <= 1e-12 * np.abs(ref).max()  # derivative of a constant


def test_degree_N_aliases(oracle):
    """x^N on N points is NOT differentiated exactly: the error is that of the interpolant,
    d/dx of (x^N - 2^(1-N) * (x^2-1) U_{N-2}(x) ...) — just check it is O(1), not rounding."""
    N = 8
    x = oracle.cheb_nodes(N)
    du = oracle.cheb_derivative_line(x**N)
    assert np.abs(du - N * x ** (N - 1)).max() > 1e-3


def test_tiny_by_hand(oracle):
    # N=2: linear interpolant through (-1,u0),(1,u1): slope (u1-u0)/2
    assert np.allclose(oracle.cheb_derivative_line(np.array([3.0, 7.0])), [2.0, 2.0], atol=1e-15)
    # N=3: nodes -1,0,1, parabola through (u0,u1,u2): u' = (u2-u0)/2 + x (u0 - 2u1 + u2)
    u = np.array([1.0, -2.0, 5.0])
    ex = (u[2] - u[0]) / 2 + np.array([-1.0, 0.0, 1.0]) * (u[0] - 2 * u[1] + u[2])
    assert np.allclose(oracle.cheb_derivative_line(u), ex, atol=1e-14)


@pytest.mark.parametrize("L", [1, 4, 8, 16, 33])
def test_gauss_legendre(oracle, L):
    th, w = oracle.gl_nodes(L)
    x = np.cos(th)
    assert np.all(np.diff(th) > 0)
    assert abs(w.sum() - 2.0) < 1e-14
    assert np.abs(x + x[::-1]).max() < 1e-15 and np.abs(w - w[::-1]).max() < 1e-15
    for p in range(2 * L + 2):  # exact to degree 2(L+1)-1
        ex = 0.0 if p % 2 else 2.0 / (p + 1)
        assert abs((w * x**p).sum() - ex) < 1e-14, p
    # library cross-check
    xr, wr = np.polynomial.legendre.leggauss(L + 1)
    assert np.abs(np.sort(x) - xr).max() < 1e-14 and np.abs(w[::-1] - wr).max() < 1e-14


def test_double_build_rounding_floor(oracle, oracle_double):
    """SURVEY §7 hard part 1: the FP64 build of the same recurrence is measurably worse than
    long double at N=32 — the reason parity uses long double."""
    N = 32
    x = oracle.cheb_nodes(N)
    u = np.sin(2.0 * x) * np.exp(0.5 * x)
    ex = (2.0 * np.cos(2.0 * x) + 0.5 * np.sin(2.0 * x)) * np.exp(0.5 * x)
    e_ld = np.abs(oracle.cheb_derivative_line(u) - ex).max()
    e_d = np.abs(oracle_double.cheb_derivative_line(u) - ex).max()
    assert e_ld < 2e-13 and e_d > e_ld
