"""GPU parity tests (-m gpu): the CUDA path, called through the C ABI, against the CPU
oracle on the same seeded inputs, element by element.

Tolerances (BASELINE.json north_star): relative L2 <= 1e-12 per field per RHS call and
<= 1e-10 per field after 100 RK3 steps.  DESIGN.md "Tolerance" (reading Q19): when a field
of the oracle is (nearly) zero by cancellation, the error is measured against the norm of
T = sum of |terms| of that equation instead (both are reported in the assertion message).
Index work (DSS gather/scatter order) is compared bit-exactly.
"""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2504_08157_b200 import binding, inputs

pytestmark = pytest.mark.gpu

TOL_RHS = 1e-12   # north_star: relative L2 per field per RHS call
TOL_100 = 1e-10   # north_star: relative L2 per field after 100 RK3 steps
TOL_T = 1e-14     # ~ 90 eps: rounding bound of the tendency relative to ||T|| (Q19)


def rel_l2(g, o, T=None):
    """Per-field parity error.  err/||o|| where the field is well conditioned; where the field
    is small by cancellation (hydrostatic / geostrophic / non-divergent balance) the bound
    that any two correctly rounded evaluations can meet is c*eps*||T|| with T the same
    expression evaluated with absolute values (the oracle computes it), so the error is
    reported as  err / max(||o||, (TOL_T/TOL_RHS) ||T||)  and compared with TOL_RHS, i.e.
    err <= max(1e-12 ||o||, 1e-14 ||T||)   (reading Q19)."""
    out = []
    for m in range(o.shape[0]):
        den = np.linalg.norm(o[m])
        if T is not None:
            den = max(den, (TOL_T / TOL_RHS) * np.linalg.norm(T[m]))
        err = np.linalg.norm(g[m] - o[m])
        out.append(err / den if den > 0 else err)
    return np.array(out)


def describe(g, o, T):
    """Diagnostic string: err/||o||, err/||T|| and kappa = ||T||/||o|| per field."""
    rows = []
    for m in range(o.shape[0]):
        err = np.linalg.norm(g[m] - o[m]); no = np.linalg.norm(o[m]); nT = np.linalg.norm(T[m])
        rows.append("f%d err/|o|=%.2e err/|T|=%.2e kappa=%.1e" % (m, err / max(no, 1e-300),
                                                                 err / max(nT, 1e-300), nT / max(no, 1e-300)))
    return "; ".join(rows)


def _pair(wl):
    o = orc.Oracle.from_workload(wl)
    g = binding.Numa.from_workload(wl)
    return o, g


def _np(t):
    return t.detach().cpu().numpy()


def _assembled_T(o, q):
    """Assembled sum-of-|terms| used to scale ill-conditioned fields."""
    r, T = o.rhs_local(q, want_T=True)
    o.dss(T)
    return T


CASES = [
    # (config, N, scale)
    (1, 4, 1.0), (1, 2, 1.0), (1, 3, 1.0), (1, 5, 1.0), (1, 6, 1.0), (1, 7, 1.0), (1, 8, 1.0),
    (2, 4, 0.35), (2, 7, 0.25),
    (3, 4, 0.07), (4, 3, 0.05), (4, 5, 0.06), (4, 6, 0.06), (4, 8, 0.07), (5, 7, 0.03),
]


@pytest.mark.parametrize("cfg,N,scale", CASES)
def test_setup_tables_match_oracle(cfg, N, scale):
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o, g = _pair(wl)
    D = _np(g.table(3)).reshape(N + 1, N + 1)
    w = _np(g.table(4))
    xi_o, w_o = orc.lgl(N)
    assert np.max(np.abs(D - orc.dmat(N))) < 2e-13
    assert np.max(np.abs(w - w_o)) < 1e-15
    met = _np(g.table(0)).reshape(o.met.shape)
    # error of an inverse scales with its largest entry (anisotropic elements: the tiny
    # cross terms carry round-off of the large ones)
    scale_m = np.max(np.abs(o.met))
    for c in range(9):
        assert np.max(np.abs(met[c] - o.met[c])) < 1e-12 * scale_m, c
    om = _np(g.table(1)).reshape(o.omega.shape)
    assert np.max(np.abs(om - o.omega)) < 1e-12
    p0 = _np(g.table(2)).reshape(o.omega.shape)
    c = wl.constants
    p0_o = c["p_a"] * (wl.ref[0] * c["R_gas"] * wl.ref[1] / c["p_a"]) ** (c["c_p"] / c["c_v"])
    assert np.max(np.abs(p0 / p0_o - 1.0)) < 1e-14


@pytest.mark.parametrize("cfg,N,scale", CASES)
def test_rhs_call_by_call_parity_on_generic_state(cfg, N, scale):
    """numa_rhs, numa_dss_or_flux, numa_apply_sources each against the oracle, on a seeded
    smooth state with all five fields non-zero (parity protocol)."""
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o, g = _pair(wl)
    q = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=1234 + cfg)
    qd = g.state(q)
    hd = None if wl.heating is None else g.state(wl.heating)
    # A2-A6
    r_o, T = o.rhs_local(q, want_T=True)
    r_g = g.rhs(qd)
    e = rel_l2(_np(r_g), r_o, T)
    assert np.all(e <= TOL_RHS), ("numa_rhs", describe(_np(r_g), r_o, T))
    # A7 on the GPU's own local result: bit-exact against the oracle's DSS of the same data
    r_in = _np(r_g).copy()
    g.dss_or_flux(r_g)
    want = o.dss(r_in.copy())
    assert np.array_equal(_np(r_g), want), "numa_dss_or_flux is not bit-exact"
    # full chain
    o.dss(r_o); o.dss(T)
    e = rel_l2(_np(r_g), r_o, T)
    assert np.all(e <= TOL_RHS), ("after DSS", describe(_np(r_g), r_o, T))
    g.apply_sources(qd, hd, r_g)
    o.apply_sources(q, wl.heating, r_o)
    e = rel_l2(_np(r_g), r_o, T)
    assert np.all(e <= TOL_RHS), ("after sources", describe(_np(r_g), r_o, T))
    # walls: no normal component left (normals from the GPU's own metric table, which the
    # setup test compares with the oracle's)
    if o.wall_node.size:
        rv = _np(r_g).reshape(5, -1)[1:4][:, o.wall_node]
        _, nrm_g = orc.wall_list(N, wl.mesh.face_bc, _np(g.table(0)).reshape(o.met.shape))
        scale_v = np.max(np.abs(rv)) + 1e-300
        # (sequential projections at edges leave ~ n1.n2 of the first normal: sanity bound)
        assert np.max(np.abs(np.einsum("ct,tc->t", rv, nrm_g))) < 1e-10 * scale_v
        assert np.max(np.abs(nrm_g - o.wall_normal)) < 1e-12


@pytest.mark.parametrize("cfg,N,scale", [(1, 4, 1.0), (2, 4, 0.35), (3, 4, 0.07), (5, 7, 0.03)])
def test_rhs_parity_on_workload_state_after_10_steps(cfg, N, scale):
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o, g = _pair(wl)
    q = wl.q
    for _ in range(10):
        q = o.step_rk3(q, wl.dt, wl.heating)
    r_o = o.rhs(q, wl.heating)
    T = _assembled_T(o, q)
    hd = None if wl.heating is None else g.state(wl.heating)
    r_g = g.full_rhs(g.state(q), hd)
    e = rel_l2(_np(r_g), r_o, T)
    print(describe(_np(r_g), r_o, T))
    assert np.all(e <= TOL_RHS), describe(_np(r_g), r_o, T)


def test_sources_and_rk_stage_pointwise():
    wl = inputs.make_workload(3, scale=0.05)
    o, g = _pair(wl)
    rng = np.random.default_rng(3)
    q = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=9)
    r = rng.standard_normal(q.shape)
    r_g = g.state(r)
    g.apply_sources(g.state(q), g.state(wl.heating), r_g)
    r_o = o.apply_sources(q, wl.heating, r.copy())
    # wall normals come from the metric terms of 700:1 anisotropic elements: allow 1e-12
    assert np.max(np.abs(_np(r_g) - r_o)) < 1e-12 * np.max(np.abs(r_o))
    q0 = rng.standard_normal(q.shape)
    out = torch.empty_like(r_g)
    g.rk_stage(0.75, 0.25, 0.25 * 0.1, g.state(q0), g.state(q), g.state(r), out)
    want = orc.rk_stage(0.75, 0.25, 0.25 * 0.1, q0, q, r)
    assert np.max(np.abs(_np(out) - want)) <= 4e-16 * np.max(np.abs(want))
    # aliasing q_out = qs
    qs_d = g.state(q)
    g.rk_stage(0.75, 0.25, 0.025, g.state(q0), qs_d, g.state(r), qs_d)
    assert np.array_equal(_np(qs_d), _np(out))


@pytest.mark.parametrize("cfg,N,scale,steps", [(1, 4, 1.0, 100), (2, 4, 0.25, 100), (2, 7, 0.2, 100),
                                               (3, 4, 0.06, 100), (5, 7, 0.025, 50)])
def test_100_rk3_steps_parity(cfg, N, scale, steps):
    """numa_step_rk3 (fused route) and the four-call route against the oracle after `steps`
    SSP-RK3 steps (config 5 states 50 steps)."""
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o, g = _pair(wl)
    q = wl.q
    refresh = wl.heating_refresh_steps
    heat = wl.heating
    qd = g.state(wl.q)
    hd = None if heat is None else g.state(heat)
    for s in range(steps):
        if refresh and s > 0 and s % refresh == 0:
            heat = wl.heating_at(s // refresh)
            hd = g.state(heat)
        q = o.step_rk3(q, wl.dt, heat)
        g.step_rk3(qd, wl.dt, hd, 1)
    assert np.all(np.isfinite(q))
    e = rel_l2(_np(qd), q)
    # fields that are still zero to round-off in the oracle are compared absolutely
    nz = np.array([np.linalg.norm(q[m]) > 0 for m in range(5)])
    assert np.all(e[nz] <= TOL_100), e
    # four separate calls give the same answer as the fused route after 3 steps
    qa = g.state(wl.q); qb = g.state(wl.q)
    hd0 = None if wl.heating is None else g.state(wl.heating)
    g.step_rk3(qa, wl.dt, hd0, 3)
    q1 = torch.empty_like(qb)
    (s1, s2, s3), dt = orc.SSP_RK3, wl.dt
    for _ in range(3):
        g.rk_stage(s1[0], s1[1], s1[2] * dt, qb, qb, g.full_rhs(qb, hd0), q1)
        g.rk_stage(s2[0], s2[1], s2[2] * dt, qb, q1, g.full_rhs(q1, hd0), q1)
        g.rk_stage(s3[0], s3[1], s3[2] * dt, qb, q1, g.full_rhs(q1, hd0), qb)
    # (velocity components that are small by symmetry carry the rounding of the large one:
    # they are scaled by the norm of the whole velocity)
    a, b = _np(qa), _np(qb)
    vel = np.sqrt(sum(np.linalg.norm(b[m]) ** 2 for m in (1, 2, 3)))
    den = [np.linalg.norm(b[0]), vel, vel, vel, np.linalg.norm(b[4])]
    e2 = np.array([np.linalg.norm(a[m] - b[m]) / (den[m] if den[m] > 0 else 1.0) for m in range(5)])
    assert np.all(e2 <= 1e-13), e2


def test_bitwise_reproducible_run_to_run():
    wl = inputs.make_workload(2, scale=0.3)
    g = binding.Numa.from_workload(wl)
    a = g.state(wl.q); b = g.state(wl.q)
    g.step_rk3(a, wl.dt, None, 5)
    g.step_rk3(b, wl.dt, None, 5)
    assert torch.equal(a, b)
    g2 = binding.Numa.from_workload(wl)
    c = g2.state(wl.q)
    g2.step_rk3(c, wl.dt, None, 5)
    assert torch.equal(a, c)


def test_copies_of_a_global_node_stay_bitwise_equal():
    wl = inputs.make_workload(1)
    g = binding.Numa.from_workload(wl)
    q = g.state(wl.q)
    g.step_rk3(q, wl.dt, None, 4)
    qh = _np(q).reshape(5, -1)
    cg = wl.mesh.intma_cg.ravel()
    for m in (0, 4):  # fields without wall projection
        glob = np.zeros(wl.mesh.n_global); glob[cg] = qh[m]
        assert np.array_equal(glob[cg], qh[m])


def test_atmosphere_at_rest_stays_bitwise_at_rest_on_gpu():
    for cfg, scale in ((1, 1.0), (3, 0.05)):
        wl = inputs.make_workload(cfg, scale=scale)
        g = binding.Numa.from_workload(wl)
        q = torch.zeros(wl.q.shape, dtype=torch.float64, device="cuda")
        r = g.full_rhs(q, None)
        assert torch.all(r == 0)
        g.step_rk3(q, wl.dt, None, 3)
        assert torch.all(q == 0)


# ---------------------------------------------------------------------------------------
# edge cases
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [2, 3, 4])
def test_single_element_and_ragged_element_counts(N):
    """One element (no shared nodes at all) and element counts that are not a multiple of
    the elements-per-block of the kernels."""
    for dims in ((1, 1, 1), (3, 1, 1), (5, 3, 1), (7, 1, 3)):
        mesh = inputs.box_mesh(N, *dims, (100.0 * dims[0], 100.0 * dims[1], 100.0 * dims[2]),
                               perturb=0.05, seed=N)
        rho0, theta0 = inputs.reference_neutral(mesh.xyz[2])
        ref = np.stack((rho0, theta0))
        q = inputs.smooth_random_state(mesh, rho0, theta0, seed=2)
        o = orc.Oracle(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
        g = binding.Numa(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
        r_o, T = o.rhs_local(q, want_T=True)
        o.dss(r_o); o.dss(T); o.apply_sources(q, None, r_o)
        r_g = g.full_rhs(g.state(q), None)
        e = rel_l2(_np(r_g), r_o, T)
        assert np.all(e <= TOL_RHS), (dims, e)
        qd = g.state(q)
        g.step_rk3(qd, 0.01, None, 2)
        qo = o.step_rk3(o.step_rk3(q, 0.01), 0.01)
        assert np.all(rel_l2(_np(qd), qo) <= 1e-13)


def test_periodic_mesh_parity():
    N = 4
    mesh = inputs.box_mesh(N, 4, 3, 3, (400.0, 300.0, 300.0), perturb=0.05, seed=8,
                           periodic=(True, True, False))
    rho0, theta0 = inputs.reference_neutral(mesh.xyz[2])
    ref = np.stack((rho0, theta0))
    q = inputs.smooth_random_state(mesh, rho0, theta0, seed=2)
    o = orc.Oracle(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
    g = binding.Numa(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
    r_o, T = o.rhs_local(q, want_T=True)
    o.dss(r_o); o.dss(T); o.apply_sources(q, None, r_o)
    e = rel_l2(_np(g.full_rhs(g.state(q), None)), r_o, T)
    assert np.all(e <= TOL_RHS), e


def test_scrambled_global_numbering_and_unused_ids():
    """The library must not rely on any structure of intma_cg: random relabelling of the
    global ids with gaps (unused ids) gives the same assembled result."""
    N = 3
    mesh = inputs.box_mesh(N, 3, 3, 2, (300.0, 300.0, 200.0), perturb=0.05, seed=8)
    rho0, theta0 = inputs.reference_neutral(mesh.xyz[2])
    ref = np.stack((rho0, theta0))
    q = inputs.smooth_random_state(mesh, rho0, theta0, seed=2)
    rng = np.random.default_rng(0)
    perm = rng.permutation(2 * mesh.n_global)[:mesh.n_global].astype(np.int32)
    cg2 = perm[mesh.intma_cg]
    g1 = binding.Numa(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
    g2 = binding.Numa(N, mesh.xyz, cg2, 2 * mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
    r1 = g1.full_rhs(g1.state(q), None)
    r2 = g2.full_rhs(g2.state(q), None)
    assert torch.equal(r1, r2)


def test_init_errors_on_device():
    mesh = inputs.box_mesh(2, 2, 1, 1, (2.0, 1.0, 1.0))
    rho0, theta0 = inputs.reference_neutral(mesh.xyz[2])
    ref = np.stack((rho0, theta0))
    xyz = mesh.xyz.copy(); xyz[0] = -xyz[0]
    with pytest.raises(binding.NumaError) as ei:
        binding.Numa(2, xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
    assert ei.value.status == 4
    with pytest.raises(binding.NumaError) as ei:
        binding.Numa(2, mesh.xyz, mesh.intma_cg, mesh.n_global - 1, mesh.face_bc, ref, inputs.CONSTANTS)
    assert ei.value.status == 1
    with pytest.raises(binding.NumaError) as ei:
        binding.Numa(2, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS,
                     method=1)
    assert ei.value.status == 2
    g = binding.Numa(2, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, ref, inputs.CONSTANTS)
    q = g.state(np.zeros((5,) + rho0.shape))
    with pytest.raises(binding.NumaError):
        g.rhs(q, out=q)  # rhs must not alias q


def test_host_buffer_entry_point_matches_device_path():
    wl = inputs.make_workload(3, scale=0.05)
    g = binding.Numa.from_workload(wl)
    qd = g.state(wl.q); hd = g.state(wl.heating)
    g.step_rk3(qd, wl.dt, hd, 2)
    qh = torch.from_numpy(wl.q.copy()).pin_memory()
    hh = torch.from_numpy(wl.heating.copy()).pin_memory()
    g.step_rk3_host(qh, wl.dt, hh, 2)
    assert torch.equal(qh, qd.cpu())


def test_full_size_cfg3_in_the_bench_configuration():
    """The workload and launch configuration bench.py times by default (config 3: 100x100x20
    elements, N=4, 25 M local nodes, heating + sponge + Coriolis + walls): one full RHS through
    the four C-ABI calls and two fused SSP-RK3 steps, against the oracle element by element at
    full size (the oracle needs ~1 min and ~10 GB of host memory for this)."""
    wl = inputs.make_workload(3)
    assert wl.mesh.n_local == 25_000_000
    o, g = _pair(wl)
    hd = g.state(wl.heating)
    # one RHS evaluation (four-call route) on the workload's initial state
    r_o = o.rhs(wl.q, wl.heating)
    T = _assembled_T(o, wl.q)
    r_g = _np(g.full_rhs(g.state(wl.q), hd))
    e = rel_l2(r_g, r_o, T)
    assert np.all(e <= TOL_RHS), describe(r_g, r_o, T)
    del r_g, r_o, T
    # two steps of the fused route (six stages)
    qd = g.state(wl.q)
    g.step_rk3(qd, wl.dt, hd, 2)
    q = wl.q
    for _ in range(2):
        q = o.step_rk3(q, wl.dt, wl.heating)
    qg = _np(qd)
    e = rel_l2(qg, q)
    assert np.all(e <= TOL_RHS * 6), e      # six stages, each within the per-call tolerance
    # copies of a global node are bitwise equal after the in-place DSS, at full size
    cg = wl.mesh.intma_cg.reshape(-1)
    first = np.full(wl.mesh.n_global, -1, dtype=np.int64)
    first[cg[::-1]] = np.arange(cg.size - 1, -1, -1)
    for m in range(5):
        f = qg[m].reshape(-1)
        assert np.array_equal(f, f[first[cg]])


def test_full_size_cfg4_N7_sweep_point():
    """Config 4 at N=7 in full (56x56x20 elements, 32.1 M local nodes: the element size of
    config 5 and the launch configuration of the high-order kernels): one fused SSP-RK3 step
    against the oracle, element by element."""
    wl = inputs.make_workload(4, N=7)
    assert wl.mesh.n_local == 32_112_640
    o, g = _pair(wl)
    hd = g.state(wl.heating)
    qd = g.state(wl.q)
    g.step_rk3(qd, wl.dt, hd, 1)
    q = o.step_rk3(wl.q, wl.dt, wl.heating)
    qg = _np(qd)
    # w starts at zero and after one step is dt times a tendency that is small by hydrostatic
    # cancellation (reading Q19): the velocity components are measured against the norm of the
    # whole velocity, as in test_100_rk3_steps_parity
    vel = np.sqrt(sum(np.linalg.norm(q[m]) ** 2 for m in (1, 2, 3)))
    den = [np.linalg.norm(q[0]), vel, vel, vel, np.linalg.norm(q[4])]
    e = np.array([np.linalg.norm(qg[m] - q[m]) / den[m] for m in range(5)])
    assert np.all(e <= TOL_RHS * 3), e      # three stages, each within the per-call tolerance
    assert np.all(rel_l2(qg, q) <= TOL_100)  # and plainly per field within the 100-step bound
