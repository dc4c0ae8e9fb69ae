"""Pins of the oracle's IMEX path (NEXT-3; Section 2.3, Eq. 13):

P32  the linear operator is the Jacobian of S at the reference state: L(v) = lim S(eps v)/eps, checked
     against the oracle's own nonlinear tendency (element-local and assembled with walls);
P33  ARK2 tableau: row sums equal the abscissae of both tableaux, b is shared, sums to 1, and
     b.c = 1/2 for every coupling (the four second-order conditions of an additive RK scheme);
P34  GMRES on small dense systems reproduces numpy.linalg.solve, reaches the exact solution in
     at most n iterations, and the restarted form converges too;
P35  the ARK2 step is second order in dt: on linear acoustics (where S = L, so the step is the
     implicit part alone) against a fine-step reference, and on the nonlinear bubble workload
     against SSP-RK3 at a small dt; with dt -> 0 the two integrators agree;
P36  the implicit step is stable where explicit RK3 is not: config 3's mesh at the paper's
     dt = 0.5 s (acoustic |lambda dt| ~ 4) stays bounded over 20 steps.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2504_08157_b200 import inputs


def test_p32_linear_operator_is_the_jacobian_of_S_at_rest():
    wl = inputs.make_workload(3, N=4, scale=0.04)
    o = orc.Oracle.from_workload(wl)
    v = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=9)
    Lloc = orc.linear_tendency(o.N, o.par, v, o.ref, o.met)
    for eps, tol in ((1e-4, 2e-3), (1e-6, 2e-5)):
        S = orc.tendency(o.N, o.par, eps * v, o.ref, o.met) / eps
        for m in range(5):
            assert np.linalg.norm(S[m] - Lloc[m]) <= tol * np.linalg.norm(Lloc[m]), (eps, m)
    # assembled, with walls; the sources (Coriolis, sponge) are not part of L
    o2 = orc.Oracle(o.N, wl.mesh.xyz, wl.mesh.intma_cg, wl.mesh.n_global, wl.mesh.face_bc, wl.ref, wl.constants)
    eps = 1e-6
    S = o2.rhs(eps * v) / eps
    Lh = o2.linear(v)
    for m in range(5):
        assert np.linalg.norm(S[m] - Lh[m]) <= 2e-5 * np.linalg.norm(Lh[m])
    assert np.abs(o2.linear(np.zeros_like(v))).max() == 0.0


def test_p33_ark2_order_conditions():
    A, At, b = np.array(orc.ARK2_A), np.array(orc.ARK2_AT), np.array(orc.ARK2_B)
    c, ct = A.sum(axis=1), At.sum(axis=1)
    assert np.allclose(c, ct, atol=1e-15) and abs(c[2] - 1.0) < 1e-15
    assert abs(b.sum() - 1.0) < 1e-15
    assert abs(b @ c - 0.5) < 1e-15 and abs(b @ ct - 0.5) < 1e-15
    assert np.all(np.triu(A) == 0.0) and np.all(np.triu(At, 1) == 0.0)
    g = 1.0 - 1.0 / np.sqrt(2.0)
    assert At[0, 0] == 0.0 and abs(At[1, 1] - g) < 1e-16 and abs(At[2, 2] - g) < 1e-16   # SDIRK, explicit first stage
    # stiffly accurate (last row of At equals b): the implicit part damps the stiff limit, R(inf) = 0
    assert np.allclose(At[2], b, atol=1e-16)


def test_p34_gmres_against_dense_solve():
    rng = np.random.default_rng(4)
    n = 30
    A = np.eye(n) + 0.3 * rng.standard_normal((n, n)) / np.sqrt(n)
    b = rng.standard_normal(n)
    dot = lambda x, y: float(x @ y)
    x, its, rel = orc.gmres(lambda v: A @ v, b, np.zeros(n), dot, 1e-13, n, 0)
    assert its <= n and np.linalg.norm(x - np.linalg.solve(A, b)) <= 1e-11 * np.linalg.norm(x)
    xr, its_r, rel_r = orc.gmres(lambda v: A @ v, b, np.zeros(n), dot, 1e-12, 5, 50)
    assert rel_r <= 1e-12 and np.linalg.norm(xr - x) <= 1e-10 * np.linalg.norm(x)
    # the residual estimate from the rotated right-hand side is the true residual
    assert abs(np.linalg.norm(b - A @ xr) / np.linalg.norm(b) - rel_r) <= 1e-13


def _acoustic_oracle(N=4, n=4):
    L = 1000.0
    mesh = inputs.box_mesh(N, n, n, n, (L, L, L), periodic=(True, True, True))
    rho0, th0 = inputs.reference_uniform(mesh.xyz[2])
    const = dict(inputs.CONSTANTS); const["g"] = 0.0
    o = orc.Oracle(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, np.stack([rho0, th0]), const)
    x = mesh.xyz[0]
    q = np.zeros((5,) + x.shape)
    q[0] = 1e-6 * np.sin(2 * np.pi * x / L)        # tiny amplitude: the nonlinear terms are ~1e-12
    return o, q


def test_p35_ark2_is_second_order():
    o, q0 = _acoustic_oracle()
    T = 0.4                                         # c ~ 347 m/s: the wave travels ~140 m
    def run(nsteps):
        q = q0
        for _ in range(nsteps):
            q = o.step_ark2(q, T / nsteps, tol=1e-13)
        return q
    ref = run(64)
    e = [np.linalg.norm(run(n)[0] - ref[0]) for n in (4, 8, 16)]
    assert 3.3 < e[0] / e[1] < 4.7 and 3.3 < e[1] / e[2] < 4.9, e
    # nonlinear workload: ARK2 and SSP-RK3 converge to the same solution
    wl = inputs.make_workload(1)
    ob = orc.Oracle.from_workload(wl)
    qa = qb = wl.q
    for _ in range(4):
        qa = ob.step_ark2(qa, 0.0025, tol=1e-13)
        qb = ob.step_rk3(qb, 0.0025)
    for m in (0, 3, 4):
        assert np.linalg.norm(qa[m] - qb[m]) <= 1e-5 * max(np.linalg.norm(qb[m]), 1e-30), m


def test_p36_imex_is_stable_at_the_papers_time_step():
    wl = inputs.make_workload(3, N=4, scale=0.04)
    o = orc.Oracle.from_workload(wl)
    q = wl.q
    stats = []
    for _ in range(10):
        q = o.step_ark2(q, 0.5, wl.heating, tol=1e-8, m=20, max_restarts=20, stats=stats)   # PAPER.md:L296 dt = 0.5 s
    assert np.isfinite(q).all()
    assert np.abs(q[1:3]).max() < 30.0 and np.abs(q[3]).max() < 5.0      # a 20 m/s vortex stays a 20 m/s vortex
    assert max(r for _, r in stats) <= 1e-8
    # explicit SSP-RK3 at the same dt blows up within the same 10 steps
    qe = wl.q
    with np.errstate(all="ignore"):
        for _ in range(10):
            qe = o.step_rk3(qe, 0.5, wl.heating)
    assert (not np.isfinite(qe).all()) or np.abs(qe[3]).max() > 1e3
