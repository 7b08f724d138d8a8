"""The C-ABI library loads here (no GPU) and exports every symbol include/sw.h declares; without a
device the compute entry points fail loudly instead of falling back to anything (-m "not gpu")."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "sw.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(sw_[a-z_A-Z0-9]+)\s*\(", txt)))


@pytest.fixture(scope="module")
def binding():
    from paper_2302_14720_b200 import build, binding
    build.build()
    binding.lib()
    return binding


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for need in ("sw_create", "sw_sweep", "sw_labels", "sw_observables", "sw_create_batch", "sw_destroy",
                 "sw_spins", "sw_bonds", "sw_set_spins", "sw_series", "sw_stage_ms", "sw_last_error"):
        assert need in names


def test_library_exports_every_declared_symbol(binding):
    so = ctypes.CDLL(os.path.join(ROOT, "paper_2302_14720_b200", "libsw_b200.so"))
    for name in _declared():
        assert hasattr(so, name), f"{name} declared in sw.h but not exported"
    # and the binding marshals exactly that set
    assert sorted(binding.PROTOTYPES) == _declared()


def _declared4():
    txt = open(os.path.join(ROOT, "include", "phi4.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(phi4_[a-z_A-Z0-9]+)\s*\(", txt)))


def test_phi4_header_exports_and_binding_agree(binding):
    """include/phi4.h (the second workload): every declared call is exported and marshalled."""
    from paper_2302_14720_b200 import phi4
    so = ctypes.CDLL(os.path.join(ROOT, "paper_2302_14720_b200", "libsw_b200.so"))
    names = _declared4()
    assert "phi4_create" in names and "phi4_sweep" in names and "phi4_observables" in names
    for name in names:
        assert hasattr(so, name), f"{name} declared in phi4.h but not exported"
    assert sorted(phi4.PROTOTYPES) == names
    assert ctypes.sizeof(phi4.phi4_obs) == 88
    phi4.lib()
    import torch
    if not torch.cuda.is_available():
        assert not phi4.lib().phi4_create(4, 0.3, 1)
        assert b"no CPU path" in phi4.lib().phi4_last_error()
        assert not phi4.lib().phi4_create(1, 0.3, 1) and not phi4.lib().phi4_create(4, -1.0, 1)


def test_struct_layout_matches_header(binding):
    assert ctypes.sizeof(binding.sw_obs) == 56
    assert [f[0] for f in binding.sw_obs._fields_] == ["energy", "magnetisation", "n_clusters", "largest_cluster",
                                                      "sweep", "e_per_site", "abs_m_per_site"]


def test_host_only_entry_points(binding):
    assert binding.sw_version().startswith("sw-b200")
    assert binding.sw_workspace_bytes(1, 1) == 0
    assert binding.sw_workspace_bytes(32769, 1) == 0
    n = binding.sw_workspace_bytes(16384, 1)
    # int8 spins + bit-packed spins + 2 bond bit-planes + flip bit-plane + 16-bit tile-local roots + node arrays / border
    # slots of the open tile roots (the flat int32 labels and the generic paths' size array, 4 B/site each, are
    # allocated by the library the first time they are asked for)
    N = 16384 * 16384
    assert N * (1 + 4 / 8 + 2) <= n <= N * 4.6
    binding.sw_destroy(None)


def test_no_cpu_fallback(binding):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(binding.SwError) as e:
        binding.sw_create(64, 2.0, 1)
    assert "no usable CUDA device" in str(e.value) and "no CPU path" in str(e.value)
    with pytest.raises(RuntimeError):
        binding.SwendsenWang(64, 2.0, 1)


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_2302_14720_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(import|from)\s+oracle\b", txt, flags=re.M), f
                assert "sw_oracle" not in txt and "liboracle" not in txt, f
    o = open(os.path.join(ROOT, "oracle", "__init__.py")).read() + open(os.path.join(ROOT, "oracle", "sw_oracle.c")).read()
    assert "paper_2302_14720_b200 import" not in o and "libsw_b200" not in o and '#include "sw' not in o
