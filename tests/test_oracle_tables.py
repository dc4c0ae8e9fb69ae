"""Pins P1-P3, P12, P15 of the CPU oracle: tables, RK3, DOF counting.

None of these retypes the oracle's formula: they check closed forms, exactness properties
and identities that the mathematics fixes (Eq. 5, Eq. 8; L88, L103-L109).
"""
import math
import os

import numpy as np
import pytest

from oracle import oracle as orc

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _closed_forms():
    out = []
    with open(os.path.join(GOLD, "lgl_closed_forms.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            n, nodes, weights = line.split("|")
            ev = lambda s: [eval(t, {"sqrt": math.sqrt}) for t in s.split(",")]
            out.append((int(n), ev(nodes), ev(weights)))
    return out


@pytest.mark.parametrize("N,nodes,weights", _closed_forms())
def test_P1_lgl_closed_forms(N, nodes, weights):
    xi, w = orc.lgl(N)
    assert np.allclose(xi, nodes, rtol=0, atol=2e-15)
    assert np.allclose(w, weights, rtol=0, atol=2e-15)


@pytest.mark.parametrize("N", range(2, 9))
def test_P2_quadrature_exactness(N):
    """LGL quadrature with N+1 points integrates x^p exactly for p <= 2N-1 and NOT p = 2N."""
    xi, w = orc.lgl(N)
    assert abs(w.sum() - 2.0) < 4e-15
    assert np.all(np.diff(xi) > 0)
    for p in range(0, 2 * N):
        exact = 0.0 if p % 2 else 2.0 / (p + 1)
        assert abs(np.dot(w, xi ** p) - exact) < 5e-15, p
    p = 2 * N
    assert abs(np.dot(w, xi ** p) - 2.0 / (p + 1)) > 1e-6


@pytest.mark.parametrize("N", range(2, 9))
def test_P3_derivative_matrix(N):
    xi, _ = orc.lgl(N)
    D = orc.dmat(N)
    # exact on monomials of degree <= N
    for p in range(0, N + 1):
        d_exact = p * xi ** (p - 1) if p > 0 else np.zeros_like(xi)
        assert np.allclose(D @ xi ** p, d_exact, rtol=0, atol=2e-13), p
    # NOT exact on degree N+1 (so the test would notice a too-good-to-be-true table)
    assert np.max(np.abs(D @ xi ** (N + 1) - (N + 1) * xi ** N)) > 1e-3
    # corner entry and centro-antisymmetry (closed forms)
    assert abs(D[0, 0] + N * (N + 1) / 4.0) < 1e-13
    assert abs(D[N, N] - N * (N + 1) / 4.0) < 1e-13
    assert np.allclose(D, -D[::-1, ::-1], rtol=0, atol=1e-13)
    # index order (Q5): D[i][l] = h_l'(xi_i), so column l differentiates the
    # l-th cardinal function; check against a direct polynomial derivative of h_l.
    for l in range(N + 1):
        others = np.delete(xi, l)
        coef = np.poly(others) / np.prod(xi[l] - others)
        assert np.allclose(D[:, l], np.polyval(np.polyder(coef), xi), rtol=0, atol=1e-11)


def test_P12_rk3_amplification_polynomial():
    """With rhs := lambda q, one SSP-RK3 step multiplies q by 1 + z + z^2/2 + z^3/6."""
    dt = 0.3
    for lam in (-0.7, 0.45, -2.0):
        q0 = np.array([1.3, -0.2, 4.0])
        qs = q0
        for (a0, a1, b) in orc.SSP_RK3:
            qs = orc.rk_stage(a0, a1, b * dt, q0, qs, lam * qs)
        z = lam * dt
        assert np.allclose(qs, q0 * (1 + z + z * z / 2 + z ** 3 / 6), rtol=2e-15, atol=0)


def test_P12_rk3_third_order():
    """y' = -y^2, y(0)=1 -> y(1) = 1/2; the error of SSP-RK3 falls as dt^3."""
    errs = []
    for n in (20, 40, 80):
        dt = 1.0 / n
        y = np.array([1.0])
        for _ in range(n):
            y0 = y
            for (a0, a1, b) in orc.SSP_RK3:
                y = orc.rk_stage(a0, a1, b * dt, y0, y, -y * y)
        errs.append(abs(y[0] - 0.5))
    s1 = math.log2(errs[0] / errs[1]); s2 = math.log2(errs[1] / errs[2])
    assert 2.8 < s1 < 3.2 and 2.8 < s2 < 3.2


def test_rk_stage_aliasing():
    q0 = np.linspace(0, 1, 7); qs = q0 * 2; r = q0 - 1
    want = 0.75 * q0 + 0.25 * qs + 0.1 * r
    got = orc.rk_stage(0.75, 0.25, 0.1, q0, qs, r, out=qs)
    assert got is qs and np.array_equal(got, want)


def test_P15_paper_dof_counts():
    """DOF = Ne (N+1)^3 5 reproduces the three figures the paper prints."""
    with open(os.path.join(GOLD, "paper_dof_counts.txt")) as f:
        rows = [l.split("#")[0].split() for l in f if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for nx, ny, nz, N, dof in rows:
        nx, ny, nz, N, dof = map(int, (nx, ny, nz, N, dof))
        assert nx * ny * nz * (N + 1) ** 3 * 5 == dof
