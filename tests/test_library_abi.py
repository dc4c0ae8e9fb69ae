"""Host-side checks of the C-ABI library (no GPU compute): it loads, exports every symbol
that include/numa_b200.h declares, sizes its workspace sensibly and fails loudly (status
codes, no CPU fallback) when misused or when no CUDA device is present."""
import ctypes as C
import os
import re

import pytest

from paper_2504_08157_b200 import binding, inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols(header="numa_b200.h"):
    text = open(os.path.join(ROOT, "include", header)).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(numa_[a-z0-9_]+)\s*\(", text)))


def test_library_loads_and_exports_every_declared_symbol():
    lib = binding.load_library()
    declared = _declared_symbols()
    assert "numa_init_geometry" in declared and "numa_rk_stage" in declared
    for name in declared:
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == declared
    # the measurement entry points live in their own header, not in the product ABI
    measure = _declared_symbols("numa_b200_measure.h")
    assert sorted(binding.MEASURE_EXPORTS) == measure
    for name in measure:
        assert hasattr(lib, name), name
    assert not set(measure) & set(declared)


def test_north_star_entry_points_present():
    lib = binding.load_library()
    for name in ("numa_init_geometry", "numa_rhs", "numa_dss_or_flux", "numa_rk_stage",
                 "numa_apply_sources"):
        assert hasattr(lib, name)


def test_workspace_bytes_scales_with_problem():
    lib = binding.load_library()
    c = inputs.CONSTANTS
    p1 = binding.make_params(4, 64, 4913, c)
    p2 = binding.make_params(4, 128, 9537, c)
    b1 = lib.numa_workspace_bytes(C.byref(p1))
    b2 = lib.numa_workspace_bytes(C.byref(p2))
    NL = 64 * 125
    # 14 doubles of tables per local node (met[9], omega, rho0, theta0, p0, beta) plus two sets of
    # DSS index lists (natural and block-shell order: <= 5 int32 per node and set), one fixed
    # 6 MB of CUB + list-building scratch for meshes whose own tables are too small to alias it, the
    # padding of the block-shell records (<= 3 %) and alignment
    assert b1 >= NL * 8 * (9 + 1 + 3 + 1) and b1 < NL * (8 * 14 + 2 * 5 * 4) * 1.03 + (6 << 20) + (64 << 10)
    assert b2 > b1
    assert lib.numa_step_scratch_bytes(C.byref(p1)) >= 11 * NL * 8   # two block-shell states + heating
    for bad in (binding.make_params(1, 64, 100, c), binding.make_params(9, 64, 100, c),
                binding.make_params(4, 0, 100, c), binding.make_params(4, 64, 0, c)):
        assert lib.numa_workspace_bytes(C.byref(bad)) == 0


def test_argument_errors_are_status_codes():
    lib = binding.load_library()
    c = inputs.CONSTANTS
    p = binding.make_params(4, 64, 4913, c)
    ctx = C.c_void_p()
    st = lib.numa_init_geometry(C.byref(p), None, None, None, None, None, None, 0, None, C.byref(ctx))
    assert st == 1 and b"NULL" in lib.numa_last_error(None)
    dummy = C.c_void_p(256)
    pdg = binding.make_params(4, 64, 4913, c, method=1)
    st = lib.numa_init_geometry(C.byref(pdg), dummy, dummy, dummy, dummy, None, dummy, 1 << 30,
                                None, C.byref(ctx))
    assert st == 2  # NUMA_ERR_UNSUPPORTED: DG face flux is not built
    pcons = binding.make_params(4, 64, 4913, c, eqn_set=1)
    st = lib.numa_init_geometry(C.byref(pcons), dummy, dummy, dummy, dummy, None, dummy, 1 << 30,
                                None, C.byref(ctx))
    assert st == 2
    st = lib.numa_init_geometry(C.byref(p), dummy, dummy, dummy, dummy, None, dummy, 16, None,
                                C.byref(ctx))
    assert st == 5  # NUMA_ERR_WORKSPACE
    assert lib.numa_rhs(None, None, None, None) == 1
    assert lib.numa_dss_or_flux(None, None, None) == 1
    assert lib.numa_rk_stage(None, 1.0, 0.0, 1.0, None, None, None, None, None) == 1


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    wl = inputs.make_workload(1)
    with pytest.raises(RuntimeError, match="no CPU fallback"):
        binding.Numa.from_workload(wl)
    # the C entry point itself reports NUMA_ERR_CUDA rather than computing on the host
    lib = binding.load_library()
    p = binding.make_params(4, 64, 4913, inputs.CONSTANTS)
    nbytes = lib.numa_workspace_bytes(C.byref(p))
    ctx = C.c_void_p()
    dummy = C.c_void_p(256)
    st = lib.numa_init_geometry(C.byref(p), dummy, dummy, dummy, dummy, None, dummy, nbytes, None,
                                C.byref(ctx))
    assert st == 3 and not ctx.value
