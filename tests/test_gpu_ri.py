"""GPU parity of the RI-velocity diagnostic (numa_ri_*, Eq. 18-22) against the CPU
oracle on the same seeded inputs.  Index and bin work (point lists, strip counts) is compared
bit-exactly; centroids and strip means at 1e-12 (relative to the level / velocity scale)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2504_08157_b200 import binding, inputs

pytestmark = pytest.mark.gpu

TOL = 1e-12


def _compare(wl, q, r_max, n_strips=50, g=None):
    mesh = wl.mesh
    lev, n_lev = inputs.node_levels(mesh)
    o = orc.ri_velocity(mesh.N, mesh.xyz, mesh.intma_cg, mesh.n_global, lev, n_lev, q, r_max, n_strips)
    g = g or binding.Numa.from_workload(wl)
    g.ri_init(mesh.xyz, lev, n_lev, r_max, n_strips)
    ubar, count, cen, sc = g.ri_velocity(g.state(q))
    ubar2, count2, cen2, sc2 = g.ri_velocity(g.state(q))
    # bitwise reproducible run to run
    assert torch.equal(ubar, ubar2) and torch.equal(count, count2) and torch.equal(cen, cen2) and torch.equal(sc, sc2)
    ubar = ubar.cpu().numpy(); count = count.cpu().numpy(); cen = cen.cpu().numpy(); sc = sc.cpu().numpy()
    assert sc[2] == 0.0
    valid = cen[2 * n_lev:] != 0.0
    assert (valid == (o["valid"] != 0)).all()
    L = max(mesh.extent[0], mesh.extent[1])
    cg = cen[:2 * n_lev].reshape(n_lev, 2)
    assert np.abs(cg - o["centroid"])[valid].max(initial=0.0) <= TOL * L
    assert (count == o["count"]).all()                      # bin decisions: bit-exact
    scale = max(o["umax_h"], 1e-300)
    # Eq. 21 is ill-conditioned at the centroid itself: a point with r ~ 1e-16 L has an e_r that is
    # pure rounding, and its u_theta may be anything in [0, |u_h|].  Such a point (at most one per
    # level, in strip 0) widens the bound of its strip mean by |u_h| / count.
    flat = mesh.intma_cg.reshape(-1)
    _, first = np.unique(flat, return_index=True)
    px, py = mesh.xyz[0].reshape(-1)[first], mesh.xyz[1].reshape(-1)[first]
    pl = lev.reshape(-1)[first]
    uh = np.hypot(q[1].reshape(-1)[first], q[2].reshape(-1)[first])
    r = np.hypot(px - o["centroid"][pl, 0], py - o["centroid"][pl, 1])
    slack = np.zeros_like(ubar)
    for t in np.nonzero(r < 1e-6 * L)[0]:
        slack[pl[t], 0] += uh[t] / max(o["count"][pl[t], 0], 1)
    assert (np.abs(ubar - o["ubar"]) <= TOL * scale + slack).all()
    assert slack.max() <= 1e-6 * scale          # ... and it is a tiny correction, not a loophole
    assert abs(sc[0] - o["u_ri"]) <= TOL * scale + slack.max()
    assert abs(sc[1] - o["umax_h"]) <= 4e-16 * scale          # the GPU may contract u*u + v*v into an FMA
    return o, g


@pytest.mark.parametrize("cfg,N,scale", [(3, 4, 0.08), (4, 3, 0.05), (5, 7, 0.04), (4, 6, 0.06)])
def test_ri_velocity_matches_oracle_on_the_tc_workloads(cfg, N, scale):
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    r_max = 0.4873 * wl.mesh.extent[0]     # not commensurate with the node spacing
    o, g = _compare(wl, wl.q, r_max)
    assert o["u_ri"] > 5.0                 # the initial vortex (20 m/s at r_m) is seen
    # after a few steps (asymmetric heating acts) the diagnostic still matches
    qd = g.state(wl.q)
    g.step_rk3(qd, wl.dt, g.state(wl.heating), 5)
    oq = wl.q
    oo = orc.Oracle.from_workload(wl)
    for _ in range(5):
        oq = oo.step_rk3(oq, wl.dt, wl.heating)
    _compare(wl, oq, r_max, g=g)


def test_ri_velocity_on_perturbed_mesh_and_generic_state():
    wl = inputs.make_workload(2, N=4, scale=0.3)
    q = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=3)
    _compare(wl, q, 0.613 * wl.mesh.extent[0], n_strips=37)


def test_ri_level_at_rest_has_no_centroid_and_bad_levels_are_rejected():
    wl = inputs.make_workload(1)
    mesh = wl.mesh
    lev, n_lev = inputs.node_levels(mesh)
    q = inputs.smooth_random_state(mesh, wl.ref[0], wl.ref[1], seed=5)
    q[1:4][:, lev == 0] = 0.0           # bottom level at rest
    q[1:4][:, lev == 7] = 0.0
    o, g = _compare(wl, q, 700.0)
    assert o["valid"][0] == 0 and o["valid"][7] == 0 and o["count"][0].sum() == 0
    bad = lev.copy(); bad[3, 5] = n_lev
    with pytest.raises(binding.NumaError):
        g.ri_init(mesh.xyz, bad, n_lev, 700.0)
    with pytest.raises(binding.NumaError):
        g.ri_init(mesh.xyz, lev, n_lev, 700.0, n_strips=2000)
