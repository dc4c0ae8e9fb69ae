"""Pins P17-P19 of the CPU oracle's pointwise sources (orc_sources: heating, Coriolis, sponge;
DESIGN.md readings Q9, Q10, Q15).  None of them re-types the three lines of orc_sources: each
drives the whole oracle (tendency -> weight -> DSS -> sources -> walls -> SSP-RK3) on a state
for which Eq. 1 reduces to an ordinary differential equation with a closed-form solution, so
that a flipped sign, a source added to the wrong field, a sponge that also damps rho', or a
coefficient read at the wrong node fails one of them.

All cases: g = 0, uniform background (rho0, theta0 constant), triply periodic VERTEX-PERTURBED
or uniform mesh, so that the Euler tendency of a spatially uniform state vanishes (every
D . const = 0) and only the source under test acts.
"""
import math

import numpy as np
import pytest

from oracle import oracle as orc
from paper_2504_08157_b200 import inputs

C0 = dict(inputs.CONSTANTS, g=0.0)


def _periodic_oracle(N=3, perturb=0.05, f_cor=0.0, sponge=None, ne=(3, 3, 2), seed=5):
    mesh = inputs.box_mesh(N, *ne, (300.0, 300.0, 200.0), perturb=perturb, seed=seed,
                           periodic=(True, True, True))
    rho0, theta0 = inputs.reference_uniform(mesh.xyz[2], 1.2, 300.0)
    sp = None if sponge is None else sponge(mesh)
    o = orc.Oracle(N, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc,
                   np.stack((rho0, theta0)), C0, f_cor=f_cor, sponge=sp)
    return mesh, o, sp


def _rk3_poly(z):
    """Amplification factor of SSP-RK3 on dq/dt = lambda q (pinned separately by P12)."""
    return 1.0 + z + z * z / 2.0 + z ** 3 / 6.0


# ---------------------------------------------------------------------------------------
# P17  Coriolis (reading Q10; f-plane, "background wind is not considered"):
# a spatially uniform horizontal wind on an f-plane performs an inertial oscillation,
#   du/dt = f v,  dv/dt = -f u   =>   (u + i v)(t) = (u0 + i v0) exp(-i f t):
# the wind vector turns CLOCKWISE (f > 0) at the rate f and keeps its speed.
# ---------------------------------------------------------------------------------------
def test_P17_coriolis_inertial_oscillation_turns_clockwise_and_keeps_speed():
    # dt is bound by the acoustic limit of explicit RK3 on 100 m elements (|lambda| dt < 1.73), so
    # the rotation rate is taken large: f dt = 0.01, RK3 error per step (f dt)^4/24 ~ 4e-10
    f, dt, steps = 0.2, 0.05, 100
    mesh, o, _ = _periodic_oracle(f_cor=f)
    u0, v0, w0 = 7.0, -3.0, 0.4
    q = np.zeros((5,) + mesh.xyz[0].shape)
    q[1] = u0; q[2] = v0; q[3] = w0
    for _ in range(steps):
        q = o.step_rk3(q, dt)
    t = steps * dt
    ue = u0 * math.cos(f * t) + v0 * math.sin(f * t)    # real part of (u0 + i v0) e^{-ift}
    ve = v0 * math.cos(f * t) - u0 * math.sin(f * t)
    speed = math.hypot(u0, v0)
    assert np.max(np.abs(q[1] - ue)) < 1e-7 * speed
    assert np.max(np.abs(q[2] - ve)) < 1e-7 * speed
    # the angle DEcreased by f t = 1 rad (clockwise); an anticlockwise turn is 2 rad away
    ang0 = math.atan2(v0, u0)
    ang = np.arctan2(q[2], q[1])
    dphi = (ang - ang0 + np.pi) % (2 * np.pi) - np.pi
    assert np.max(np.abs(dphi + f * t)) < 1e-7
    # speed conserved to the RK3 amplitude error  1 - |P(i f dt)|^steps ~ steps (f dt)^4 / 8
    assert np.max(np.abs(np.hypot(q[1], q[2]) / speed - 1.0)) < 2.0 * steps * (f * dt) ** 4 / 8
    # nothing else moves: w is not touched by the f-plane term, rho' and theta' stay zero
    assert np.max(np.abs(q[3] - w0)) < 1e-12
    assert np.max(np.abs(q[0])) < 1e-13 and np.max(np.abs(q[4])) < 1e-11


def test_P17_coriolis_single_rhs_is_orthogonal_to_the_wind():
    """(r_u, r_v) . (u, v) = 0 and (u, v) x (r_u, r_v) = -f |u|^2 < 0 node by node."""
    f = 5.0e-5
    mesh, o, _ = _periodic_oracle(f_cor=f, N=4)
    q = np.zeros((5,) + mesh.xyz[0].shape)
    q[1] = 11.0; q[2] = 4.0
    r = o.rhs(q)
    dot = r[1] * q[1] + r[2] * q[2]
    cross = q[1] * r[2] - q[2] * r[1]
    # (the advection of the uniform wind leaves ~1e-14 of round-off in r on the deformed mesh)
    assert np.max(np.abs(dot)) < 1e-9 * f * 137.0
    assert np.max(np.abs(cross + f * 137.0)) < 1e-9 * f * 137.0


# ---------------------------------------------------------------------------------------
# P18  Rayleigh sponge (reading Q9): dq_m/dt = -beta q_m for m = u, v, w, theta' and NOT
# for rho'.  (a) uniform beta, uniform state: every damped field decays by the RK3 factor
# P(-beta dt)^n -> exp(-beta t), rho' keeps its value.  (b) beta(y, z) and a shear flow
# u(y, z) x-hat (a steady solution of Eq. 1: u.grad u = u du/dx = 0, div(rho u) = 0): every
# node decays with ITS OWN coefficient, which pins the per-node indexing of the array.
# ---------------------------------------------------------------------------------------
def test_P18_sponge_uniform_decay_of_u_v_w_theta_and_not_of_rho():
    beta, dt, steps = 0.5, 0.05, 40
    mesh, o, _ = _periodic_oracle(sponge=lambda m: np.full(m.xyz[0].shape, beta))
    q = np.zeros((5,) + mesh.xyz[0].shape)
    start = (0.01, 3.0, -2.0, 0.7, 1.5)   # rho' uniform and non-zero: p' uniform, grad p' = 0
    for m in range(5):
        q[m] = start[m]
    for _ in range(steps):
        q = o.step_rk3(q, dt)
    amp = _rk3_poly(-beta * dt) ** steps
    assert abs(amp - math.exp(-beta * dt * steps)) < 1e-5      # it IS exponential decay
    for m in (1, 2, 3, 4):
        assert np.max(np.abs(q[m] - start[m] * amp)) < 1e-12 * abs(start[m]), m
    assert np.max(np.abs(q[0] - start[0])) < 1e-13 * start[0]


def test_P18_sponge_acts_node_by_node_on_a_shear_flow():
    dt, steps = 0.02, 25    # N = 4 on 67 m elements: acoustic RK3 limit ~0.04 s

    def beta_field(m):
        x, y, z = m.xyz
        return 1.5 * (0.5 + 0.5 * np.sin(2 * np.pi * y / 300.0) * np.cos(2 * np.pi * z / 200.0)) + 0.1

    mesh, o, beta = _periodic_oracle(N=4, perturb=0.0, sponge=beta_field, ne=(2, 3, 3))
    x, y, z = mesh.xyz
    u0 = 4.0 + 2.0 * np.cos(2 * np.pi * y / 300.0) + np.sin(4 * np.pi * z / 200.0)
    q = np.zeros((5,) + x.shape)
    q[1] = u0
    for _ in range(steps):
        q = o.step_rk3(q, dt)
    want = u0 * _rk3_poly(-beta * dt) ** steps
    assert np.max(np.abs(beta)) > 3 * np.min(np.abs(beta))      # the coefficient does vary
    assert np.max(np.abs(q[1] - want)) < 1e-12 * np.max(np.abs(u0))
    for m in (0, 2, 3, 4):
        assert np.max(np.abs(q[m])) < 1e-12, m


# ---------------------------------------------------------------------------------------
# P19  Heating (Eq. 1c; reading Q15): at rest, d theta'/dt = S_theta and
# nothing else has a tendency.  (a) one RHS of the atmosphere at rest with a node-varying
# heating field: r = (0, 0, 0, 0, S_theta) exactly.  (b) uniform heating over RK3 steps:
# theta' = S_theta t (RK3 integrates a constant exactly), p' stays uniform so no wind starts.
# ---------------------------------------------------------------------------------------
def test_P19_heating_enters_only_the_theta_equation():
    for cfg, scale in ((1, 1.0), (3, 0.04)):
        wl = inputs.make_workload(cfg, scale=scale)
        o = orc.Oracle.from_workload(wl)
        heat = inputs.heating_field(wl.mesh, 99) if wl.heating is None else wl.heating
        if cfg == 1:   # the generator's cells sit around the domain centre of a 1000 km box
            x, y, z = wl.mesh.xyz
            heat = 5e-3 * np.exp(-((x - 400.0) ** 2 + (y - 600.0) ** 2) / 200.0 ** 2) * np.sin(np.pi * z / 1000.0)
        assert np.max(np.abs(heat)) > 1e-3
        r = o.rhs(np.zeros_like(wl.q), heat)
        assert np.array_equal(r[4], heat)
        for m in range(4):
            assert np.all(r[m] == 0.0), m


def test_P19_uniform_heating_warms_linearly_and_starts_no_wind():
    h, dt, steps = 20.0 / 3600.0, 0.05, 30
    mesh, o, _ = _periodic_oracle()
    heat = np.full(mesh.xyz[0].shape, h)
    q = np.zeros((5,) + mesh.xyz[0].shape)
    for _ in range(steps):
        q = o.step_rk3(q, dt, heat)
    assert np.max(np.abs(q[4] - h * dt * steps)) < 1e-13
    for m in range(4):
        assert np.max(np.abs(q[m])) < 1e-10, m


@pytest.mark.parametrize("mutation", ["coriolis_sign", "sponge_on_rho", "heat_on_w"])
def test_the_pins_would_catch_a_mutated_source_term(mutation):
    """Meta-check: replace orc.sources by a plausibly wrong variant and confirm that the pin
    written for it fails (so the pins are not vacuous)."""
    real = orc.sources

    def wrong(q, heat, beta, f_cor, r):
        if mutation == "coriolis_sign":
            return real(q, heat, beta, -f_cor, r)
        if mutation == "sponge_on_rho":
            real(q, heat, beta, f_cor, r)
            if beta is not None:
                r[0] -= beta * q[0]
            return r
        real(q, None, beta, f_cor, r)
        if heat is not None:
            r[3] += heat
        return r

    orc.sources = wrong
    try:
        target = {"coriolis_sign": test_P17_coriolis_inertial_oscillation_turns_clockwise_and_keeps_speed,
                  "sponge_on_rho": test_P18_sponge_uniform_decay_of_u_v_w_theta_and_not_of_rho,
                  "heat_on_w": test_P19_heating_enters_only_the_theta_equation}[mutation]
        with pytest.raises(AssertionError):
            target()
    finally:
        orc.sources = real
