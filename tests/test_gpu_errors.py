"""Error behaviour of the C-ABI on a GPU box (include/necsim.h: negative codes, message, no abort)."""
import ctypes as C

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ns():
    from paper_2108_05815_b200 import necsim
    necsim.lib()
    return necsim


def test_workspace_and_capacity_errors(ns):
    import torch
    L = ns.lib()
    sc = ns.Scenario(ns.EXPLICIT_GAUSSIAN, width=40, height=40, uniform_deme=2, sigma=1.0)
    p = ns.make_params()
    nbytes = C.c_size_t()
    assert L.necsim_simulate_workspace_size(sc._h, 0, C.byref(p), C.byref(nbytes)) == -1            # n_sampled = 0
    assert L.necsim_simulate_workspace_size(sc._h, sc.n_individuals + 1, C.byref(p), C.byref(nbytes)) == -1
    assert L.necsim_simulate_workspace_size(sc._h, 100, C.byref(p), C.byref(nbytes)) == 0 and nbytes.value > 0
    small = torch.empty(nbytes.value, dtype=torch.uint8, device="cuda")
    res = ns.Result()
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    # workspace too small for the capacity asked
    rc = L.necsim_simulate(sc._h, 1, 0.1, None, sc.n_individuals, C.byref(p), C.c_void_p(small.data_ptr()), small.numel(), stream, C.byref(res))
    assert rc == -2 and b"workspace" in L.necsim_last_error()
    # a mask selecting more individuals than the capacity the workspace was sized for
    mask = torch.ones(sc.n_individuals, dtype=torch.uint8, device="cuda")
    rc = L.necsim_simulate(sc._h, 1, 0.1, C.c_void_p(mask.data_ptr()), 100, C.byref(p), C.c_void_p(small.data_ptr()), small.numel(), stream, C.byref(res))
    assert rc == -2
    # misaligned workspace, bad params
    rc = L.necsim_simulate(sc._h, 1, 0.1, None, 100, C.byref(p), C.c_void_p(small.data_ptr() + 8), small.numel() - 8, stream, C.byref(res))
    assert rc in (-1, -2)
    bad = ns.make_params(block_threads=48)
    assert L.necsim_simulate_workspace_size(sc._h, 100, C.byref(bad), C.byref(nbytes)) == -1
    bad = ns.make_params(dedup_probe=9)
    assert L.necsim_simulate_workspace_size(sc._h, 100, C.byref(bad), C.byref(nbytes)) == -1
    # the handle still works after errors
    m = np.zeros(sc.n_individuals, np.uint8); m[:100] = 1
    out = sc.simulate(1, 0.1, m)
    assert out["richness"] >= 1 and int(out["events"]["abundance"].sum()) == 100
    sc.close()


def test_scenario_validation(ns):
    with pytest.raises(ns.NecsimError):
        ns.Scenario(ns.EXPLICIT_MATRIX, width=3, height=3, uniform_deme=1)                            # matrix missing
    with pytest.raises(ns.NecsimError):
        ns.Scenario(ns.EXPLICIT_MATRIX, width=2, height=1, deme=np.array([1, 0], np.uint32), matrix=np.ones((2, 2)))   # mass into non-habitat
    with pytest.raises(ns.NecsimError):
        ns.Scenario(ns.NONSPATIAL, uniform_deme=10, uniform_turnover=1000.0)                           # lambda * dt out of range
    with pytest.raises(ns.NecsimError):
        ns.Scenario(ns.SPATIALLY_IMPLICIT, local_size=10, meta_size=2**32, migration=0.1)
    with pytest.raises(ns.NecsimError):
        ns.Scenario(ns.NONSPATIAL, uniform_deme=10, sampler=7)
    with pytest.raises(ns.NecsimError):
        ns.Scenario(ns.EXPLICIT_GAUSSIAN, width=30, height=30, uniform_deme=1, sigma=float("nan"))
