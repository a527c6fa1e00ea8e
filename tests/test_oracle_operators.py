"""Pins for O1 (LGL nodes, weights, derivative matrix) and O9 (LSRK54 coefficients) of the oracle.

What fixes the values, other than the oracle itself: textbook closed forms of the LGL rule, exactness of
the quadrature / derivative on polynomials, the summation-by-parts identity that
makes eq. (26) and eq. (32) equal, and the order conditions of a 4th-order Runge-Kutta scheme.
"""
import math

import numpy as np
import pytest


def closed_form(N):
    s = math.sqrt
    if N == 3:
        x = [1.0, s(1 / 5)]; w = [1 / 6, 5 / 6]
    elif N == 4:
        x = [1.0, s(3 / 7), 0.0]; w = [1 / 10, 49 / 90, 32 / 45]
    elif N == 5:
        x = [1.0, s((7 + 2 * s(7)) / 21), s((7 - 2 * s(7)) / 21)]
        w = [1 / 15, (14 - s(7)) / 30, (14 + s(7)) / 30]
    elif N == 6:
        x = [1.0, s(5 / 11 + 2 / 11 * s(5 / 3)), s(5 / 11 - 2 / 11 * s(5 / 3)), 0.0]
        w = [1 / 21, (124 - 7 * s(15)) / 350, (124 + 7 * s(15)) / 350, 256 / 525]
    nodes = np.zeros(N + 1); wts = np.zeros(N + 1)
    for i, (a, b) in enumerate(zip(x, w)):
        nodes[i] = -a; nodes[N - i] = a; wts[i] = b; wts[N - i] = b
    if N % 2 == 0:
        nodes[N // 2] = 0.0
    return nodes, wts


@pytest.mark.parametrize("N", [3, 4, 5, 6])
def test_lgl_closed_forms(oracle_mod, N):
    xi, w = oracle_mod.lgl(N)
    x0, w0 = closed_form(N)
    assert np.max(np.abs(xi - x0)) < 2e-16
    assert np.max(np.abs(w - w0)) < 4e-16


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7])
def test_lgl_quadrature_exactness(oracle_mod, N):
    xi, w = oracle_mod.lgl(N)
    assert abs(w.sum() - 2.0) < 1e-15
    assert np.all(np.diff(xi) > 0) and xi[0] == -1.0 and xi[-1] == 1.0
    assert np.max(np.abs(xi + xi[::-1])) == 0.0
    for p in range(0, 2 * N):                       # exact to degree 2N-1
        exact = 0.0 if p % 2 else 2.0 / (p + 1)
        assert abs(np.dot(w, xi ** p) - exact) < 1e-14
    if N >= 2:                                      # and NOT exact at degree 2N (inexact LGL quadrature)
        assert abs(np.dot(w, xi ** (2 * N)) - 2.0 / (2 * N + 1)) > 1e-6


@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 6, 7])
def test_derivative_matrix(oracle_mod, N):
    xi, w = oracle_mod.lgl(N)
    D = oracle_mod.dmat(N)
    # exact on polynomials of degree <= N (BASELINE invariant, 1e-13)
    for p in range(0, N + 1):
        d = D @ xi ** p
        exact = p * xi ** (p - 1) if p > 0 else np.zeros(N + 1)
        assert np.max(np.abs(d - exact)) < 1e-13, (N, p)
    assert np.max(np.abs(D.sum(axis=1))) < 1e-14
    # closed-form corner entries
    assert abs(D[0, 0] + N * (N + 1) / 4.0) < 1e-13
    assert abs(D[N, N] - N * (N + 1) / 4.0) < 1e-13
    # summation by parts: W D + (W D)^T = diag(-1, 0, ..., 0, 1)
    W = np.diag(w)
    B = np.zeros((N + 1, N + 1)); B[0, 0] = -1.0; B[N, N] = 1.0
    assert np.max(np.abs(W @ D + (W @ D).T - B)) < 1e-14
    # independent construction: differentiate the Lagrange polynomials with numpy.poly1d
    for j in range(N + 1):
        others = np.delete(xi, j)
        Lj = np.poly1d(others, r=True) / np.prod(xi[j] - others)
        assert np.max(np.abs(Lj.deriv()(xi) - D[:, j])) < 1e-12


def test_lsrk54_order_conditions(oracle_mod):
    A, B, Cc = oracle_mod.lsrk54_coeffs()
    s = 5
    # Butcher tableau of a 2N-storage scheme (Williamson): b_j and a_ij from A, B
    a = np.zeros((s, s)); b = np.zeros(s)
    # dU_j = sum_{i<=j} (prod_{m=i+1..j} A_m) dt f_i ; U_after_j = U0 + sum_{l<=j} B_l dU_l
    coef = np.zeros((s, s))  # coef[j, i]: weight of f_i in dU_j
    for j in range(s):
        for i in range(j + 1):
            coef[j, i] = np.prod(A[i + 1:j + 1])
    for stage in range(1, s):
        a[stage, :] = (B[:stage, None] * coef[:stage, :]).sum(axis=0)
    b = (B[:, None] * coef).sum(axis=0)
    c = a.sum(axis=1)
    assert np.max(np.abs(c - Cc)) < 1e-14
    one = np.ones(s)
    conds = [
        (b @ one, 1.0), (b @ c, 1 / 2), (b @ c ** 2, 1 / 3), (b @ (a @ c), 1 / 6),
        (b @ c ** 3, 1 / 4), (b @ (c * (a @ c)), 1 / 8), (b @ (a @ c ** 2), 1 / 12), (b @ (a @ (a @ c)), 1 / 24),
    ]
    for got, want in conds:
        assert abs(got - want) < 1e-14
    # stability polynomial of y' = lambda y: 1 + z + z^2/2 + z^3/6 + z^4/24 + z^5/200
    poly = [b @ one, b @ c, b @ (a @ c), b @ (a @ (a @ c)), b @ (a @ (a @ (a @ c)))]
    for got, want in zip(poly, [1.0, 1 / 2, 1 / 6, 1 / 24, 1 / 200]):
        assert abs(got - want) < 1e-14


def test_table1_fixture_matches_workload_defaults():
    """The constants used by the synthetic workloads are the ones the paper prints in Table 1."""
    import os
    import workloads as W
    vals = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "table1_constants.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split(); vals[k] = float(v)
    p = W.base_params()
    for k in ("R_d", "R_v", "c_vd", "c_vv", "T_0"):
        assert p[k] == vals[k]
    assert p["I_v0"] == vals["L_v0"] - vals["R_v"] * vals["T_0"]     # eq. (9)
