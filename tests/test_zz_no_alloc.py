"""numa_step_rk3_static: the SSP-RK3 step for callers that cannot allocate device memory.

Who that is: code coupled into a host model whose device memory all belongs to another runtime
(OpenACC data regions, a framework pool that claimed the whole GPU, so that a plain cudaMalloc
fails), or a time loop where cudaMalloc / cudaFree are forbidden because they synchronise the
device.  numa_step_rk3 asks such a caller for scratch it cannot get; the _static variant works in
a 64 MiB array compiled into the library instead (include/numa_b200.h).

What is checked: the variant runs the same kernels as numa_step_rk3, so its output must equal the
existing path's bit for bit (the repo's own bar for "same kernels, other plumbing", as for the
CUDA-graph route) -- on two calls in a row that share the built-in array, the second with another
state, another step count and no heating, after the array was deliberately filled with NaN by a
throw-away call on a mesh of another order (the array keeps the last call's contents and nothing
clears it).  Meshes beyond the limit must be refused with both sizes in the message.

This file sorts after every other test file on purpose: `pytest -x` stops at the first failure,
and a failure here must not hide the parity tests.  It passes alone in a fresh process (the first
call then also does the per-device address look-up) and after the rest of the suite.
"""
import ctypes as C

import numpy as np
import pytest
import torch

from paper_2504_08157_b200 import binding, inputs

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def test_static_scratch_step_equals_the_caller_scratch_step_on_two_calls_in_a_row():
    lib = binding.load_library()
    limit = lib.numa_static_scratch_bytes()
    assert limit == 64 << 20

    # leave NaN everywhere a larger-order mesh reaches in the shared array, padding included
    wl7 = inputs.make_workload(1, N=7)
    g7 = binding.Numa.from_workload(wl7)
    assert lib.numa_step_scratch_bytes(C.byref(g7.params)) <= limit
    poison = torch.full(wl7.q.shape, float("nan"), dtype=torch.float64, device=g7.device)
    g7.step_rk3_static(poison, wl7.dt, None, 1)
    torch.cuda.synchronize()
    assert bool(torch.isnan(poison).all())
    g7.close()

    # config-3 physics (heating, Coriolis, sponge, walls, stretched layers) on a 7 x 7 x 20 mesh
    wl = inputs.make_workload(3, scale=0.07)
    g = binding.Numa.from_workload(wl)
    assert lib.numa_step_scratch_bytes(C.byref(g.params)) <= limit
    heat = g.state(wl.heating)

    # call 1: three steps with heating
    a = g.state(wl.q); b = g.state(wl.q)
    g.step_rk3(a, wl.dt, heat, 3)              # existing path, torch-allocated scratch
    g.step_rk3_static(b, wl.dt, heat, 3)       # built-in array
    torch.cuda.synchronize()
    assert np.isfinite(_np(a)).all()
    assert np.array_equal(_np(a), _np(b))
    assert not np.array_equal(_np(a), wl.q)    # the steps did something

    # call 2, straight after: other state (call 1's result), other step count, no heating
    c = a.clone(); d = a.clone()
    g.step_rk3(c, 0.5 * wl.dt, None, 2)
    g.step_rk3_static(d, 0.5 * wl.dt, None, 2)
    torch.cuda.synchronize()
    assert np.isfinite(_np(c)).all()
    assert np.array_equal(_np(c), _np(d))
    assert not np.array_equal(_np(c), _np(a))

    # n_steps = 0 leaves q alone, NULL q is an argument error
    e = d.clone()
    g.step_rk3_static(e, wl.dt, None, 0)
    assert np.array_equal(_np(e), _np(d))
    st = lib.numa_step_rk3_static(g.ctx, None, None, wl.dt, 1, None)
    assert st == 1
    g.close()


def test_static_scratch_refuses_a_mesh_beyond_its_limit():
    """6400 elements at N = 4 need 11 x 800,000 x 8 B = 70.4 MB (+ record padding) > 64 MiB."""
    lib = binding.load_library()
    mesh = inputs.box_mesh(4, 20, 20, 16, (2000.0, 2000.0, 1600.0))
    rho0, theta0 = inputs.reference_neutral(mesh.xyz[2])
    g = binding.Numa(4, mesh.xyz, mesh.intma_cg, mesh.n_global, mesh.face_bc, np.stack((rho0, theta0)),
                     inputs.CONSTANTS)
    need = lib.numa_step_scratch_bytes(C.byref(g.params))
    assert need > lib.numa_static_scratch_bytes()
    q = torch.zeros((5,) + mesh.xyz.shape[1:], dtype=torch.float64, device=g.device)
    q[4] = 1.0
    with pytest.raises(binding.NumaError) as ei:
        g.step_rk3_static(q, 0.01, None, 1)
    assert ei.value.status == 5                                   # NUMA_ERR_WORKSPACE
    msg = str(ei.value)
    assert str(need) in msg and str(64 << 20) in msg and "numa_step_rk3" in msg
    torch.cuda.synchronize()
    assert float(q[4].min()) == 1.0 and float(q[:4].abs().max()) == 0.0   # nothing ran
    g.step_rk3(q, 0.01, None, 1)                                   # the caller-scratch path still serves it
    torch.cuda.synchronize()
    assert bool(torch.isfinite(q).all())
    g.close()
