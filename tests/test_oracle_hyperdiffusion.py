"""Pins of the oracle's tensor hyper-diffusion (NEXT-1; Eq. 14-16) against
what the mathematics fixes:

P26  tau on axis-aligned bricks: Eq. 15-16 collapse to tau = diag(sqrt(c_a/dt) h_a^2), the
     coefficient c_i going to the principal axis with the i-th LARGEST element length;
P27  tau with equal coefficients: tau = 4 sqrt(c/dt) J J^T on any (deformed) element, because
     E E^T = I and nu_i/lambda_i = 4 sqrt(c/dt) -- J rebuilt here from the coordinates by a
     separate NumPy route (Kronecker derivative operators);
P28  L f = div(tau grad f) is exact for a polynomial of degree <= N on an affine mesh (tau
     constant), including the mixed terms of a full tensor;
P29  a Fourier mode on a uniform periodic mesh is an eigenfunction: L f = -(k.tau k) f and
     H f = -(k.tau k)^2 f to discretisation error (spectral decay in N) -- sign (dissipative) and
     the power alpha = 2;
     one explicit Euler step of the oracle's full RHS damps the mode by 1 - dt (k.tau k)^2;
P30  rho' is untouched; H of a constant field is zero to round-off;
P31  H is single-valued on the copies of a global node (assembly after each application).
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2504_08157_b200 import inputs


def test_p26_tau_on_axis_aligned_bricks():
    mesh = inputs.box_mesh(3, 4, 2, 3, (400.0, 300.0, 60.0))          # hx = 100, hy = 150, hz = 20
    met, _, _ = orc.metrics(3, mesh.xyz)
    c, dt = (0.02, 0.005, 0.3), 0.25
    tau = orc.hd_tau(met, c, dt)
    # lambda_1 > lambda_2 > lambda_3 (L149): c_1 -> the longest edge (y, 150 m), c_2 -> x, c_3 -> z
    want = {3: np.sqrt(c[0] / dt) * 150.0 ** 2, 0: np.sqrt(c[1] / dt) * 100.0 ** 2,
            5: np.sqrt(c[2] / dt) * 20.0 ** 2}
    for comp in range(6):
        assert np.abs(tau[comp] - want.get(comp, 0.0)).max() <= 1e-10 * max(want.values())


def _jacobian_numpy(mesh):
    """dx_c/dxi_a at every node from Kronecker derivative operators (NumPy route)."""
    N, Nq = mesh.N, mesh.N + 1
    D = orc.dmat(N)
    I = np.eye(Nq)
    ops = [np.kron(I, np.kron(I, D)), np.kron(I, np.kron(D, I)), np.kron(D, np.kron(I, I))]
    J = np.empty((mesh.n_elem, mesh.Mn, 3, 3))
    for c in range(3):
        for a in range(3):
            J[:, :, c, a] = mesh.xyz[c] @ ops[a].T
    return J


def test_p27_equal_coefficients_give_J_Jt_on_deformed_elements():
    mesh = inputs.box_mesh(4, 2, 2, 2, (200.0, 200.0, 80.0), perturb=0.05, seed=5)
    met, _, _ = orc.metrics(4, mesh.xyz)
    c, dt = 0.013, 0.4
    tau = orc.hd_tau(met, (c, c, c), dt)
    J = _jacobian_numpy(mesh)
    T = 4.0 * np.sqrt(c / dt) * (J @ np.swapaxes(J, 2, 3))
    ref = np.stack([T[..., 0, 0], T[..., 0, 1], T[..., 0, 2], T[..., 1, 1], T[..., 1, 2], T[..., 2, 2]])
    assert np.abs(tau - ref).max() <= 1e-11 * np.abs(ref).max()


@pytest.mark.parametrize("N", [3, 5])
def test_p28_laplacian_of_a_polynomial_on_an_affine_mesh(N):
    mesh = inputs.box_mesh(N, 2, 2, 2, (2.0, 3.0, 1.0), origin=(-1.0, 0.5, 0.0))
    met, _, _ = orc.metrics(N, mesh.xyz)
    x, y, z = mesh.xyz
    # a full constant tensor (not the one Eq. 15 would give: orc_hd_laplacian takes any tau)
    t = dict(xx=1.3, xy=0.2, xz=-0.4, yy=0.7, yz=0.1, zz=2.1)
    tau = np.stack([np.full_like(x, t[k]) for k in ("xx", "xy", "xz", "yy", "yz", "zz")])
    f = x ** 3 + 2.0 * x * y * z - y ** 2 * z + 0.5 * z ** 3 + x * y
    # hand-derived second derivatives of f
    fxx, fyy, fzz = 6.0 * x, -2.0 * z, 3.0 * z
    fxy, fxz, fyz = 2.0 * z + 1.0, 2.0 * y, 2.0 * x - 2.0 * y
    want = (t["xx"] * fxx + t["yy"] * fyy + t["zz"] * fzz
            + 2.0 * (t["xy"] * fxy + t["xz"] * fxz + t["yz"] * fyz))
    got = orc.hd_laplacian(N, met, tau, f[None])[0]
    assert np.abs(got - want).max() <= 1e-11 * np.abs(want).max()


def _periodic_oracle(N, n, L, c, dt_hd):
    mesh = inputs.box_mesh(N, n, n, n, (L, L, L), periodic=(True, True, True))
    z = mesh.xyz[2]
    rho0, th0 = inputs.reference_uniform(z)
    ref = np.stack([rho0, th0])
    const = dict(inputs.CONSTANTS); const["g"] = 0.0
    o = orc.Oracle(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, const,
                   hd_c=c, hd_dt=dt_hd)
    return mesh, o


def test_p29_fourier_mode_is_an_eigenfunction_with_rate_nu2_k4():
    N, n, L = 8, 4, 400.0
    c, dt_hd = (0.004, 0.004, 0.004), 0.5
    mesh, o = _periodic_oracle(N, n, L, c, dt_hd)
    h = L / n
    nu = np.sqrt(c[0] / dt_hd) * h ** 2                      # tau = nu I on this mesh (P26)
    kx, ky, kz = 2 * np.pi / L * np.array([1.0, 1.0, 1.0])
    x, y, z = mesh.xyz
    mode = np.sin(kx * x) * np.cos(ky * y) * np.sin(kz * z)
    lam = nu * (kx ** 2 + ky ** 2 + kz ** 2)                 # k . tau k
    q = np.zeros((5,) + x.shape)
    q[4] = 0.3 * mode                                        # theta' only; u = 0 so Eq. 1 adds nothing
    H = o.hyperdiffusion(q)
    # measured: max error 1.6e-1, 1.3e-2, 2.3e-4 of lam^2 |f| at N = 4, 6, 8 (spectral decay; the
    # largest errors sit on element faces, where the strong form of Q30 averages one-sided values)
    err8 = np.abs(H[3] + lam ** 2 * q[4]).max() / (lam ** 2 * 0.3)
    assert err8 <= 1e-3
    mesh6, o6 = _periodic_oracle(6, n, L, c, dt_hd)
    q6 = np.zeros((5,) + mesh6.xyz[0].shape)
    q6[4] = 0.3 * np.sin(kx * mesh6.xyz[0]) * np.cos(ky * mesh6.xyz[1]) * np.sin(kz * mesh6.xyz[2])
    err6 = np.abs(o6.hyperdiffusion(q6)[3] + lam ** 2 * q6[4]).max() / (lam ** 2 * 0.3)
    assert 10.0 * err8 < err6 <= 5e-2
    assert np.abs(H[:3]).max() == 0.0
    # sign: dissipative.  sum M f H < 0
    assert (o.M[mesh.intma_cg] * o.omega * q[4] * H[3]).sum() < 0.0
    # through the full RHS and one explicit Euler stage (a0, a1, b) = (1, 0, 1)
    dt = 0.1 / lam ** 2
    r = o.rhs(q)
    q1 = orc.rk_stage(1.0, 0.0, dt, q, q, r)
    assert np.abs(q1[4] - (1.0 - dt * lam ** 2) * q[4]).max() <= 1e-4 * 0.3
    assert np.abs(r[0]).max() == 0.0                         # P30: rho' gets no hyper-diffusion


def test_p30_rest_state_and_rho_untouched():
    wl = inputs.make_workload(1)
    o0 = orc.Oracle.from_workload(wl)
    o1 = orc.Oracle.from_workload(wl, hd_c=(0.01, 0.01, 0.02), hd_dt=wl.dt)
    q = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=2)
    r0, r1 = o0.rhs(q), o1.rhs(q)
    assert np.array_equal(r0[0], r1[0])                      # rho' equation has no H (Eq. 1a)
    assert np.abs(r1[1:] - r0[1:]).max() > 0.0
    qc = np.zeros_like(q); qc[1], qc[2], qc[3], qc[4] = 1.5, -2.0, 0.25, 0.7
    # D annihilates constants to rounding (row sums): nothing but round-off of the operator's scale
    assert np.abs(o1.hyperdiffusion(qc)).max() <= 1e-12 * np.abs(o1.hyperdiffusion(q)).max()


def test_p31_hyperdiffusion_is_single_valued_on_shared_nodes():
    wl = inputs.make_workload(1, N=3)
    o = orc.Oracle.from_workload(wl, hd_c=(0.01, 0.01, 0.02), hd_dt=wl.dt)
    q = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=4)
    H = o.hyperdiffusion(q)
    cg = wl.mesh.intma_cg.reshape(-1)
    for m in range(4):
        glob = np.full(wl.mesh.n_global, np.nan)
        glob[cg] = H[m].reshape(-1)
        assert np.array_equal(glob[cg], H[m].reshape(-1))
