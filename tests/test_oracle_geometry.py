"""Pins P4, P5, P6, P10, P14 of the CPU oracle: geometry, gradient/divergence exactness on
deformed meshes, free stream, DSS algebra, wall projection.

The expected values are analytic (volumes, exact polynomial derivatives, zero) or come from
an explicit boolean scatter matrix built here -- none re-calls the oracle's own routine.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2504_08157_b200 import inputs

UNIFORM = dict(inputs.CONSTANTS, g=0.0)


def _oracle(mesh, ref, constants=inputs.CONSTANTS, **kw):
    return orc.Oracle(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref,
                      constants, **kw)


@pytest.mark.parametrize("N", [2, 3, 4, 7])
def test_P4_volume_identity_on_perturbed_mesh(N):
    """sum(w J) = |Omega| exactly for trilinear elements and N >= 2 (J has degree <= 2 per
    direction, LGL is exact to degree 2N-1 >= 3)."""
    mesh = inputs.box_mesh(N, 3, 2, 3, (30.0, 20.0, 12.0), perturb=0.05, seed=11, z_ratio=1.1)
    met, jac, bad = orc.metrics(N, mesh.xyz)
    assert bad == 0
    wJ, M, om = orc.mass(N, mesh.intma_cg, mesh.n_global, jac)
    assert abs(wJ.sum() - 30.0 * 20.0 * 12.0) < 1e-12 * 7200.0
    assert abs(M.sum() - 7200.0) < 1e-12 * 7200.0


def test_P4_volume_identity_fails_for_N1():
    """N = 1 under-integrates J: the identity must visibly fail (guards against a vacuous pin)."""
    mesh = inputs.box_mesh(1, 3, 3, 3, (3.0, 3.0, 3.0), perturb=0.2, seed=5)
    met, jac, bad = orc.metrics(1, mesh.xyz)
    wJ, _, _ = orc.mass(1, mesh.intma_cg, mesh.n_global, jac)
    assert abs(wJ.sum() - 27.0) > 1e-9


def test_P4_affine_element_has_constant_analytic_metrics():
    """x = A xi + b  =>  grad xi_a = rows of A^-1 and J = det A at every node."""
    N = 3
    Nq = N + 1
    xi = inputs.lgl_points(N)
    A = np.array([[2.0, 0.3, -0.1], [0.2, 1.5, 0.4], [-0.3, 0.1, 0.8]])
    b = np.array([5.0, -2.0, 1.0])
    K, J, I = np.meshgrid(xi, xi, xi, indexing="ij")  # n = i + Nq (j + Nq k)
    ref = np.stack((I.ravel(), J.ravel(), K.ravel()))
    xyz = (A @ ref + b[:, None]).reshape(3, 1, Nq ** 3)
    met, jac, bad = orc.metrics(N, xyz)
    Ainv = np.linalg.inv(A)
    assert bad == 0
    assert np.allclose(jac, np.linalg.det(A), rtol=1e-13)
    for a in range(3):
        for c in range(3):
            assert np.allclose(met[3 * a + c], Ainv[a, c], rtol=0, atol=1e-13)


def test_negative_jacobian_is_reported():
    mesh = inputs.box_mesh(2, 1, 1, 1, (1.0, 1.0, 1.0))
    xyz = mesh.xyz.copy()
    xyz[0] = -xyz[0]  # mirror: left-handed element
    _, _, bad = orc.metrics(2, xyz)
    assert bad == 27


def _poly_fields(xyz, N, rng):
    """Random polynomial of total degree <= N in (x,y,z) (scaled coordinates) and its gradient."""
    x, y, z = xyz
    terms = [(a, b, c) for a in range(N + 1) for b in range(N + 1 - a) for c in range(N + 1 - a - b)]
    coef = rng.uniform(-1, 1, len(terms))
    f = np.zeros_like(x); fx = np.zeros_like(x); fy = np.zeros_like(x); fz = np.zeros_like(x)
    for cf, (a, b, c) in zip(coef, terms):
        f += cf * x ** a * y ** b * z ** c
        if a: fx += cf * a * x ** (a - 1) * y ** b * z ** c
        if b: fy += cf * b * x ** a * y ** (b - 1) * z ** c
        if c: fz += cf * c * x ** a * y ** b * z ** (c - 1)
    return f, (fx, fy, fz)


@pytest.mark.parametrize("N", [2, 3, 4, 5, 7])
def test_P5_polynomial_gradient_and_divergence_on_deformed_mesh(N):
    """A polynomial of total degree <= N composed with a trilinear map has degree <= N per
    direction, so D differentiates it exactly: with u = e_c constant, S_theta = -d theta'/dx_c;
    with rho = const, S_rho = -rho0 div(u_poly); with theta0 polynomial, -u.grad theta0."""
    rng = np.random.default_rng(100 + N)
    mesh = inputs.box_mesh(N, 2, 2, 2, (2.0, 2.0, 2.0), origin=(-1.0, -1.0, -1.0), perturb=0.08,
                           seed=N)
    rho0 = np.full(mesh.xyz[0].shape, 1.2)
    theta0, gth0 = _poly_fields(mesh.xyz, N, rng)
    theta0 = theta0 + 300.0
    met, jac, bad = orc.metrics(N, mesh.xyz)
    par = np.array([0.0, 1e5, 287.17, 1004.67, 717.5])
    tol = 2e-12 * (N + 1) ** 2
    f, grad = _poly_fields(mesh.xyz, N, rng)
    for c in range(3):
        q = np.zeros((5,) + rho0.shape)
        q[1 + c] = 1.0
        q[4] = f
        S = orc.tendency(N, par, q, np.stack((rho0, theta0)), met)
        assert np.max(np.abs(S[4] + grad[c] + gth0[c])) < tol, c
    # divergence: rho' = 0, theta' = 0 (p' = 0), u polynomial
    q = np.zeros((5,) + rho0.shape)
    div = np.zeros_like(rho0)
    grads = []
    for c in range(3):
        q[1 + c], g_ = _poly_fields(mesh.xyz, N, rng)
        grads.append(g_)
        div += g_[c]
    S = orc.tendency(N, par, q, np.stack((rho0, np.full_like(rho0, 300.0))), met)
    assert np.max(np.abs(S[0] + 1.2 * div)) < 5 * tol
    # momentum advection: S_u = -(u.grad) u exactly when p' = 0 (products evaluated pointwise)
    for c in range(3):
        adv = sum(q[1 + d] * grads[c][d] for d in range(3))
        assert np.max(np.abs(S[1 + c] + adv)) < 20 * tol


def test_P5_transposed_D_would_fail():
    """Sanity of the pin itself: differentiate along each axis separately so that a swapped
    (xi,eta,zeta) index or a transposed D cannot cancel."""
    N = 4
    mesh = inputs.box_mesh(N, 1, 1, 1, (2.0, 3.0, 5.0))
    x, y, z = mesh.xyz
    met, _, _ = orc.metrics(N, mesh.xyz)
    par = np.array([0.0, 1e5, 287.17, 1004.67, 717.5])
    ref = np.stack((np.full_like(x, 1.0), np.full_like(x, 300.0)))
    for c, (coord, expect) in enumerate(((x, 3 * x ** 2), (y, 3 * y ** 2), (z, 3 * z ** 2))):
        q = np.zeros((5,) + x.shape)
        q[1 + c] = 1.0
        q[4] = coord ** 3
        S = orc.tendency(N, par, q, ref, met)
        assert np.allclose(S[4], -expect, rtol=0, atol=1e-11)
        for d in range(3):
            if d != c:
                q2 = np.zeros_like(q); q2[1 + d] = 1.0; q2[4] = coord ** 3
                assert np.max(np.abs(orc.tendency(N, par, q2, ref, met)[4])) < 1e-11


@pytest.mark.parametrize("N", [2, 4, 7])
def test_P6_free_stream(N):
    """Constant state, uniform background, g = 0, perturbed periodic mesh => L(q) = 0."""
    mesh = inputs.box_mesh(N, 3, 3, 2, (3.0, 3.0, 2.0), perturb=0.05, seed=3,
                           periodic=(True, True, True))
    rho0, theta0 = inputs.reference_uniform(mesh.xyz[2])
    o = _oracle(mesh, np.stack((rho0, theta0)), UNIFORM)
    q = np.empty((5,) + rho0.shape)
    for m, v in enumerate((0.01, 3.0, -2.0, 1.0, 0.7)):
        q[m] = v
    r = o.rhs(q)
    assert o.wall_node.size == 0
    scale = 3.0 * 1.21 * 10.0  # |F| * |grad xi| bound
    assert np.max(np.abs(r)) < 1e-13 * scale * (N + 1) ** 2


def _scatter_matrix(intma_cg, n_global):
    NL = intma_cg.size
    Q = np.zeros((NL, n_global))
    Q[np.arange(NL), intma_cg.ravel()] = 1.0
    return Q


@pytest.mark.parametrize("periodic", [(False, False, False), (True, False, True)])
def test_P10_dss_equals_explicit_QQt(periodic):
    """DSS = Q Q^T with Q the boolean local<-global scatter matrix (Eq. 10-11's DSS operator,
    PAPER.md:L115-L121); omega sums to one over the copies of a node; DSS.omega is a
    projection that leaves continuous fields unchanged."""
    N = 2
    mesh = inputs.box_mesh(N, 2, 2, 2, (2.0, 2.0, 2.0), perturb=0.1, seed=9, periodic=periodic)
    Q = _scatter_matrix(mesh.intma_cg, mesh.n_global)
    assert np.all(Q.sum(axis=0) >= 1)  # every global node has a copy
    rng = np.random.default_rng(0)
    r = rng.standard_normal((5,) + mesh.intma_cg.shape)
    want = (Q @ (Q.T @ r.reshape(5, -1).T)).T.reshape(r.shape)
    got = orc.dss(mesh.intma_cg, mesh.n_global, r.copy())
    assert np.allclose(got, want, rtol=0, atol=1e-14)
    # mass and weights
    _, jac, _ = orc.metrics(N, mesh.xyz)
    wJ, M, om = orc.mass(N, mesh.intma_cg, mesh.n_global, jac)
    assert np.allclose(M, Q.T @ wJ.ravel(), rtol=1e-15)
    assert np.allclose(Q.T @ om.ravel(), 1.0, rtol=0, atol=4e-16)
    # projection: continuous field unchanged, and idempotent on arbitrary data
    cont = (Q @ rng.standard_normal(mesh.n_global)).reshape(1, *mesh.intma_cg.shape)
    P = lambda a: orc.dss(mesh.intma_cg, mesh.n_global, orc.weight(om, a))
    assert np.allclose(P(cont), cont, rtol=0, atol=1e-15)
    once = P(r)
    assert np.allclose(P(once), once, rtol=0, atol=1e-14)


def test_P10_dss_multiplicities():
    """Interior / face / edge / vertex nodes of a conforming box have 1/2/4/8 copies."""
    N = 3
    mesh = inputs.box_mesh(N, 3, 3, 3, (1.0, 1.0, 1.0))
    ones = np.ones((1,) + mesh.intma_cg.shape)
    mult = orc.dss(mesh.intma_cg, mesh.n_global, ones)[0]
    assert set(np.unique(mult)) == {1.0, 2.0, 4.0, 8.0}
    assert mult.sum() == sum(c * c for c in np.bincount(mesh.intma_cg.ravel()))
    assert mesh.n_global == (3 * N + 1) ** 3


def test_P14_wall_projection():
    """After A9 the velocity tendency has no normal component at any wall entry and its
    tangential part is untouched; rho' and theta' tendencies are not modified."""
    N = 3
    mesh = inputs.box_mesh(N, 2, 2, 2, (2.0, 2.0, 2.0), perturb=0.07, seed=4)
    met, _, _ = orc.metrics(N, mesh.xyz)
    node, nrm = orc.wall_list(N, mesh.face_bc, met)
    Nq = N + 1
    assert node.size == 6 * 4 * Nq * Nq  # 6 box sides x 4 element faces x Nq^2 nodes
    assert np.allclose(np.linalg.norm(nrm, axis=1), 1.0, rtol=0, atol=2e-16)
    # planar axis-aligned walls: outward normals are +-e_c, pointing away from the centre
    x = mesh.xyz.reshape(3, -1)[:, node]
    outward = np.sign(x - 1.0) * (np.abs(x - 1.0) > 1.0 - 1e-12)
    assert np.allclose(np.abs(nrm), np.abs(nrm).round(), atol=1e-14)
    assert np.all(np.einsum("tc,ct->t", nrm, outward) > 0.999)
    rng = np.random.default_rng(1)
    r = rng.standard_normal((5,) + mesh.intma_cg.shape)
    before = r.copy()
    orc.walls(node, nrm, r)
    rv = r.reshape(5, -1)[1:4][:, node]
    assert np.max(np.abs(np.einsum("ct,tc->t", rv, nrm))) < 2e-14
    assert np.array_equal(r[0], before[0]) and np.array_equal(r[4], before[4])
    # tangential part untouched: difference is parallel to the (sum of) normals
    d = (r - before).reshape(5, -1)[1:4]
    touched = np.zeros(d.shape[1], bool); touched[node] = True
    assert np.all(d[:, ~touched] == 0.0)
    nsum = np.zeros((d.shape[1], 3)); np.add.at(nsum, node, np.abs(nrm))
    assert np.all(np.abs(d.T)[nsum < 0.5] < 1e-14)  # components along non-normal axes unchanged
