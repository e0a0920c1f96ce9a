"""The C-ABI library builds, loads, and exports every symbol include/necsim.h declares (no compute calls)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "necsim.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(necsim_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    from paper_2108_05815_b200 import build, necsim
    path = build.build()
    L = ctypes.CDLL(path)
    names = _declared()
    assert "necsim_create_scenario" in names and "necsim_simulate" in names and "necsim_destroy" in names
    for n in names:
        assert hasattr(L, n), n
    assert set(names) == set(necsim.EXPORTS)


def test_struct_sizes_match_header(tmp_path):
    """The ctypes mirrors have the sizes a C compiler gives the structs of include/necsim.h (gcc compiles a probe)."""
    import subprocess
    from paper_2108_05815_b200 import necsim
    src = tmp_path / "probe.c"
    src.write_text('#include <stdio.h>\n#include "necsim.h"\nint main(void) { printf("%zu %zu %zu %zu\\n", sizeof(necsim_scenario_desc), '
                   'sizeof(necsim_sim_params), sizeof(necsim_event), sizeof(necsim_result)); return 0; }\n')
    exe = tmp_path / "probe"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    sizes = [int(v) for v in subprocess.check_output([str(exe)], text=True).split()]
    assert sizes == [ctypes.sizeof(necsim.ScenarioDesc), ctypes.sizeof(necsim.SimParams), necsim.EVENT_DTYPE.itemsize, ctypes.sizeof(necsim.Result)]
    assert sizes[2] == 32


def test_error_paths_without_gpu():
    """Argument validation that happens before any CUDA call works on a CPU-only box."""
    from paper_2108_05815_b200 import build, necsim
    L = necsim.lib()
    d = necsim.ScenarioDesc()
    d.kind = 7
    n = ctypes.c_size_t()
    assert L.necsim_scenario_workspace_size(ctypes.byref(d), ctypes.byref(n)) == -1
    assert b"kind" in L.necsim_last_error()
    d.kind, d.width, d.height, d.uniform_deme, d.uniform_turnover, d.delta_t = 0, 1, 1, 100, 1.0, 2.0
    assert L.necsim_scenario_workspace_size(ctypes.byref(d), ctypes.byref(n)) == 0
    assert L.necsim_destroy(None) == 0


def test_binding_fails_loudly_without_gpu():
    import pytest
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    from paper_2108_05815_b200 import necsim
    with pytest.raises(RuntimeError):
        necsim.Scenario(0, uniform_deme=10)
