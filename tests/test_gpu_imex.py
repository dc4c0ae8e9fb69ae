"""GPU parity of the IMEX path (numa_linear_operator, numa_step_ark2; Eq. 13) against
the CPU oracle: the linear operator per call at 1e-12; ARK2 steps, whose implicit stages both
sides solve with the same GMRES(m) to a relative residual tol, at 100 tol (the two Krylov
iterations differ by rounding, their solutions by at most the residual tolerance times the
conditioning of I - dt gamma L, which is < 10 here)."""
import numpy as np
import pytest
import torch

from oracle import oracle as orc
from paper_2504_08157_b200 import binding, inputs

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("cfg,N,scale", [(1, 4, 1.0), (1, 2, 1.0), (2, 7, 0.2), (3, 4, 0.06), (4, 5, 0.05), (5, 7, 0.03), (4, 8, 0.05)])
def test_linear_operator_matches_oracle(cfg, N, scale):
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o = orc.Oracle.from_workload(wl)
    g = binding.Numa.from_workload(wl)
    q = inputs.smooth_random_state(wl.mesh, wl.ref[0], wl.ref[1], seed=21)
    Lo = o.linear(q)
    Lg = g.linear_operator(g.state(q)).cpu().numpy()
    for m in range(5):
        den = np.linalg.norm(Lo[m])
        if den == 0.0:      # neutral background (configs 1-2): L_theta = -u . grad theta0 vanishes identically
            assert np.abs(Lg[m]).max() == 0.0
            continue
        err = np.linalg.norm(Lg[m] - Lo[m]) / den
        assert err <= 1e-12, (m, err)


@pytest.mark.parametrize("cfg,N,scale,dt,steps", [(1, 4, 1.0, 0.05, 3), (3, 4, 0.05, 0.5, 3), (2, 5, 0.2, 0.04, 2),
                                                   (5, 7, 0.025, 0.5, 2)])
def test_ark2_steps_match_oracle(cfg, N, scale, dt, steps):
    """dt is several times the explicit limit of each mesh (config 3 / 5: the paper's 0.5 s, L296)."""
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o = orc.Oracle.from_workload(wl)
    g = binding.Numa.from_workload(wl)
    g.imex_init(20)
    tol = 1e-11
    stats = []
    qo = wl.q
    for _ in range(steps):
        qo = o.step_ark2(qo, dt, wl.heating, tol=tol, m=20, max_restarts=20, stats=stats)
    qd = g.state(wl.q)
    heat = None if wl.heating is None else g.state(wl.heating)
    its, rel = g.step_ark2(qd, dt, heat, steps, tol=tol, max_restarts=20)
    qg = qd.cpu().numpy()
    assert np.isfinite(qg).all() and rel <= tol
    its_o = sum(i for i, _ in stats)
    assert abs(its - its_o) <= max(2, its_o // 10), (its, its_o)     # same algorithm, same iteration counts
    vel = np.sqrt(sum(np.linalg.norm(qo[m]) ** 2 for m in (1, 2, 3)))
    den = [np.linalg.norm(qo[0]), vel, vel, vel, np.linalg.norm(qo[4])]
    for m in range(5):
        err = np.linalg.norm(qg[m] - qo[m]) / den[m]
        assert err <= 100 * tol, (m, err)
    # bitwise reproducible run to run
    qd2 = g.state(wl.q)
    g.step_ark2(qd2, dt, heat, steps, tol=tol, max_restarts=20)
    assert torch.equal(qd, qd2)


# ARK2 keeps H in the explicit part; dt * rho(H) is proportional to c dt / dt_ref and sits near 1 for the
# coefficients of test_rk3_steps_with_hyperdiffusion_fused_route at dt = dt_ref, so they are scaled by
# dt_ref / (2 dt) here (dt * rho(H) about 0.5)
@pytest.mark.parametrize("cfg,N,scale,dt,steps,c3", [(1, 4, 1.0, 0.05, 3, (2e-6, 2e-6, 4e-6)),
                                                      (3, 4, 0.05, 0.5, 2, (1.5e-6, 1.5e-6, 4.5e-6))])
def test_ark2_steps_with_hyperdiffusion_match_oracle(cfg, N, scale, dt, steps, c3):
    """The paper's tropical-cyclone set-up is IMEX plus hyper-diffusion (Eq. 13 with the H_q of
    Eq. 1, 14): numa_step_ark2 after numa_hd_init must include H in its explicit tendency, as the
    oracle's step_ark2 does through Oracle.rhs."""
    wl = inputs.make_workload(cfg, N=N, scale=scale)
    o = orc.Oracle.from_workload(wl, hd_c=c3, hd_dt=wl.dt)
    g = binding.Numa.from_workload(wl)
    g.hd_init(c3, wl.dt)
    g.imex_init(20)
    tol = 1e-11
    qo = wl.q
    for _ in range(steps):
        qo = o.step_ark2(qo, dt, wl.heating, tol=tol, m=20, max_restarts=20)
    heat = None if wl.heating is None else g.state(wl.heating)
    qd = g.state(wl.q)
    its, rel = g.step_ark2(qd, dt, heat, steps, tol=tol, max_restarts=20)
    qg = qd.cpu().numpy()
    assert np.isfinite(qg).all() and np.isfinite(qo).all() and rel <= tol
    vel = np.sqrt(sum(np.linalg.norm(qo[m]) ** 2 for m in (1, 2, 3)))
    den = [np.linalg.norm(qo[0]), vel, vel, vel, np.linalg.norm(qo[4])]
    for m in range(5):
        err = np.linalg.norm(qg[m] - qo[m]) / den[m]
        assert err <= 100 * tol, (m, err)
    # H is really inside the step: the same steps without hyper-diffusion differ by far more than the tolerance
    g0 = binding.Numa.from_workload(wl)
    g0.imex_init(20)
    q0 = g0.state(wl.q)
    g0.step_ark2(q0, dt, None if wl.heating is None else g0.state(wl.heating), steps, tol=tol, max_restarts=20)
    diff = np.linalg.norm(q0.cpu().numpy()[1:4] - qg[1:4]) / vel
    assert diff > 1e4 * tol, diff


def test_imex_errors_are_status_codes():
    wl = inputs.make_workload(1)
    g = binding.Numa.from_workload(wl)
    q = g.state(wl.q)
    with pytest.raises(binding.NumaError):
        g.step_ark2(q, 0.01)                       # before numa_imex_init
    with pytest.raises(binding.NumaError):
        g.imex_init(0)
    g.imex_init(5)
    with pytest.raises(binding.NumaError):
        g.step_ark2(q, 0.01, tol=0.0)
    # a solve that cannot reach tol (five Krylov vectors, no restart) is reported, not passed over:
    # the step is still taken (q finite and changed) and the residual read back is the true one
    import ctypes as C
    q1 = g.state(wl.q)
    its = C.c_int64(0); rel = C.c_double(0.0)
    st = g.lib.numa_step_ark2(g.ctx, C.c_void_p(q1.data_ptr()), None, 0.05, 1, 1e-14, 0, C.byref(its), C.byref(rel), None)
    torch.cuda.synchronize()
    assert st == 6 and b"GMRES" in g.lib.numa_last_error(g.ctx)     # NUMA_ERR_NOT_CONVERGED
    assert rel.value > 1e-14 and its.value > 0
    assert bool(torch.isfinite(q1).all()) and not torch.equal(q1, q)
