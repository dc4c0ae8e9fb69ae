"""Pins of the oracle's RI-velocity diagnostic (NEXT-4; Eq. 18-22) against
what the mathematics fixes -- none of them re-types orc_ri_velocity's formulas:

P20  area weight: sum of a over a level = the horizontal area of the box, exactly, also on the
     vertex-perturbed mesh (the integrand is of degree <= 2 per direction);
P21  uniform wind: the "weighted center" of a constant |u| is the area centroid of the box;
P22  solid-body rotation about the box centre: centroid = the centre; u_theta = Omega r at
     every point, so every strip mean lies in [Omega s eps, Omega (s+1) eps) and equals
     Omega times the mean radius of the strip's points (NumPy brute force over unique nodes);
     adding a radial and a vertical wind changes nothing (Eq. 21 projects them out);
P23  purely radial flow about the centre: u_theta = 0 in every strip, u_RI = 0;
P24  counting: with r_max beyond the box diagonal the counts of a level add up to its unique
     nodes (shared nodes once, Q28); a smaller r_max drops the far points (Q29);
P25  a compact vortex centred OFF the box centre (mesh-symmetric about its own centre): the
     centroid finds it, and u_RI is the peak of its tangential wind to discretisation error.
"""
import numpy as np
import pytest

from oracle import oracle as orc
from paper_2504_08157_b200 import inputs


def _mesh(N=4, nx=6, ny=6, nz=2, perturb=0.0, L=(600.0, 600.0, 100.0), origin=(-100.0, 50.0, 0.0)):
    return inputs.box_mesh(N, nx, ny, nz, L, origin=origin, perturb=perturb, seed=11)


def _q(mesh, u, v, w):
    q = np.zeros((5, mesh.n_elem, mesh.Mn))
    q[1], q[2], q[3] = u, v, w
    return q


def _centre(mesh):
    return (mesh.origin[0] + 0.5 * mesh.extent[0], mesh.origin[1] + 0.5 * mesh.extent[1])


@pytest.mark.parametrize("N,perturb", [(2, 0.0), (4, 0.05), (7, 0.05)])
def test_p20_area_weight_sums_to_the_level_area(N, perturb):
    mesh = _mesh(N=N, perturb=perturb)
    lev, n_lev = inputs.node_levels(mesh)
    a = orc.ri_area(N, mesh.xyz)
    area = mesh.extent[0] * mesh.extent[1]
    for l in (0, N // 2 + 1, n_lev - 1):
        s = a[lev == l].sum()
        # an element-interface level holds the nodes of the elements above AND below it
        mult = 2.0 if (l % N == 0 and 0 < l < n_lev - 1) else 1.0
        # perturbed interior level surfaces are not planar, but their horizontal projection still
        # tiles the box and x_xi y_eta - x_eta y_xi integrates to the projected area
        assert abs(s - mult * area) <= 1e-12 * area


@pytest.mark.parametrize("perturb", [0.0, 0.05])
def test_p21_uniform_wind_centroid_is_the_area_centroid(perturb):
    mesh = _mesh(perturb=perturb)
    lev, n_lev = inputs.node_levels(mesh)
    one = np.ones((mesh.n_elem, mesh.Mn))
    out = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                          _q(mesh, 3.0 * one, -4.0 * one, 0.5 * one), r_max=500.0)
    cx, cy = _centre(mesh)
    assert out["valid"].all()
    # boundary vertices stay on the walls (Q13), so the box and its centroid are unchanged
    assert np.abs(out["centroid"][[0, -1]] - [cx, cy]).max() <= 1e-10
    if perturb == 0.0:
        assert np.abs(out["centroid"] - [cx, cy]).max() <= 1e-10
    assert abs(out["umax_h"] - 5.0) <= 1e-14


def _unique_points(mesh, lev):
    """first local copy of every global node (NumPy route, independent of the C loop)."""
    flat = mesh.intma_cg.reshape(-1)
    _, first = np.unique(flat, return_index=True)
    return first, mesh.xyz[0].reshape(-1)[first], mesh.xyz[1].reshape(-1)[first], lev.reshape(-1)[first]


def test_p22_solid_body_rotation_and_projection():
    mesh = _mesh(N=4, nx=6, ny=6)
    lev, n_lev = inputs.node_levels(mesh)
    cx, cy = _centre(mesh)
    x, y = mesh.xyz[0], mesh.xyz[1]
    Om = 0.013
    u, v = -Om * (y - cy), Om * (x - cx)
    r_max, ns = 287.3, 50          # not commensurate with the node spacing
    base = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                           _q(mesh, u, v, 0 * u), r_max=r_max, n_strip=ns)
    assert np.abs(base["centroid"] - [cx, cy]).max() <= 1e-10
    eps = r_max / ns
    first, px, py, pl = _unique_points(mesh, lev)
    for l in (0, 3, n_lev - 1):
        # radii about the level's computed centroid (pinned above to 1e-10 of the centre): the
        # node AT the centre has r ~ 1e-13, not 0, and lands in strip 0 with u_theta = Om r
        r = np.hypot(px - base["centroid"][l, 0], py - base["centroid"][l, 1])
        for s in range(ns):
            sel = (pl == l) & (r >= s * eps) & (r < (s + 1) * eps) & (r > 0)
            assert base["count"][l, s] == sel.sum()
            if sel.sum():
                assert Om * s * eps - 1e-9 <= base["ubar"][l, s] < Om * (s + 1) * eps + 1e-9
                assert abs(base["ubar"][l, s] - Om * r[sel].mean()) <= 1e-12 * Om * r_max
    assert abs(base["u_ri"] - base["ubar"][base["count"] > 0].max()) == 0.0
    # clockwise rotation has the same tangential speed (Eq. 20 is a norm)
    cw = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                         _q(mesh, -u, -v, 0 * u), r_max=r_max, n_strip=ns)
    assert np.abs(cw["ubar"] - base["ubar"]).max() <= 1e-13
    # a radial wind c r and a vertical wind are projected out (centroid unchanged by symmetry)
    rr = np.hypot(x - cx, y - cy)
    mixed = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                            _q(mesh, u + 0.004 * (x - cx), v + 0.004 * (y - cy), 0.3 + 0 * rr),
                            r_max=r_max, n_strip=ns)
    assert np.abs(mixed["centroid"] - [cx, cy]).max() <= 1e-9
    assert np.abs(mixed["ubar"] - base["ubar"]).max() <= 1e-11
    assert (mixed["count"] == base["count"]).all()


def test_p23_radial_flow_has_no_tangential_wind():
    mesh = _mesh(N=3, nx=5, ny=5)
    lev, n_lev = inputs.node_levels(mesh)
    cx, cy = _centre(mesh)
    x, y = mesh.xyz[0], mesh.xyz[1]
    out = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                          _q(mesh, 0.02 * (x - cx), 0.02 * (y - cy), 0 * x), r_max=411.7)
    assert out["count"].sum() > 0
    assert out["u_ri"] <= 1e-12
    assert out["umax_h"] > 1.0


@pytest.mark.parametrize("N", [3, 5])
def test_p24_counts_cover_every_unique_node_once(N):
    # 3 x 5 elements and odd N: the box centre is an element centre and no node sits on it
    mesh = _mesh(N=N, nx=3, ny=5, nz=2)
    lev, n_lev = inputs.node_levels(mesh)
    cx, cy = _centre(mesh)
    x, y = mesh.xyz[0], mesh.xyz[1]
    out = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                          _q(mesh, -(y - cy), (x - cx), 0 * x), r_max=1.0e4)
    per_level = (3 * N + 1) * (5 * N + 1)
    assert n_lev == 2 * N + 1
    assert (out["count"].sum(axis=1) == per_level).all()   # shared nodes once (Q28)
    assert out["count"].sum() == mesh.n_global
    # a small r_max leaves the far points out (Q29)
    near = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                           _q(mesh, -(y - cy), (x - cx), 0 * x), r_max=150.0)
    first, px, py, pl = _unique_points(mesh, lev)
    assert near["count"].sum() == (np.hypot(px - cx, py - cy) < 150.0 - 1e-6).sum()


def test_p25_compact_off_centre_vortex_is_found():
    # 12 x 12 elements of 50 m; vortex centred on an element corner away from the box centre
    mesh = _mesh(N=5, nx=12, ny=12, nz=1, L=(600.0, 600.0, 50.0))
    lev, n_lev = inputs.node_levels(mesh)
    x0, y0 = mesh.origin[0] + 200.0, mesh.origin[1] + 350.0
    x, y = mesh.xyz[0], mesh.xyz[1]
    r = np.hypot(x - x0, y - y0)
    R, V = 150.0, 18.0
    s = np.clip(r / R, 0.0, 1.0)
    vt = V * 4.0 * s * (1.0 - s)               # peak V at r = R/2, zero beyond R (inside the box)
    with np.errstate(invalid="ignore", divide="ignore"):
        u = np.where(r > 0, -vt * (y - y0) / r, 0.0)
        v = np.where(r > 0, vt * (x - x0) / r, 0.0)
    out = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev,
                          _q(mesh, u, v, 0 * u), r_max=200.0, n_strip=50)
    assert np.abs(out["centroid"] - [x0, y0]).max() <= 1e-9    # mesh and field symmetric about it
    # strip width 4 m: the best strip mean is within the variation of vt across one strip of V
    assert V * (1.0 - 4.0 * (4.0 / R) ** 2) - 1e-9 <= out["u_ri"] <= V + 1e-12
    assert abs(out["umax_h"] - vt.max()) <= 1e-12
