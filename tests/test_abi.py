"""CPU-only checks of the boundary: the C-ABI library builds (nvcc cross-compiles without a
GPU), loads, and exports every symbol include/aev.h declares.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_functions():
    src = open(os.path.join(ROOT, "include", "aev.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b((?:aev|ani)_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


def test_header_lists_the_north_star_entry_points():
    names = _declared_functions()
    for want in ("aev_create", "aev_neighbors", "aev_forward", "aev_backward", "ani_energy_forces"):
        assert want in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    import paper_2310_03121_b200 as pkg
    L = pkg.lib()
    assert os.path.exists(pkg.LIB_PATH)
    raw = ctypes.CDLL(pkg.LIB_PATH)
    for name in _declared_functions():
        assert hasattr(raw, name), "libaev_b200.so does not export %s" % name
    assert sorted(pkg.EXPORTS) == _declared_functions()
    assert L.aev_error_string(0) == b"ok"
    assert L.aev_error_string(-3).startswith(b"neighbour")


def test_binding_never_imports_the_oracle():
    src = open(os.path.join(ROOT, "paper_2310_03121_b200", "__init__.py")).read()
    assert not re.search(r"^\s*(import|from)\s+oracle", src, flags=re.M)
    for f in os.listdir(os.path.join(ROOT, "paper_2310_03121_b200", "csrc")):
        body = open(os.path.join(ROOT, "paper_2310_03121_b200", "csrc", f)).read()
        assert "aev_oracle" not in body
        assert not re.search(r'#include\s+"[^"]*oracle', body)


def test_create_without_gpu_fails_loudly():
    """There is no CPU fallback: without a CUDA device aev_create must return an error."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    import paper_2310_03121_b200 as pkg
    from gen import ani1x_style_params
    with pytest.raises(pkg.AevError):
        pkg.Context(ani1x_style_params(), max_atoms=8)


def test_sass_has_no_local_memory_spill_in_hot_kernels():
    """ptxas -v log of the build: the specialised hot kernels (the instantiations bench.py's C4 / C5 steps launch)
    and the tensor-core MLP must compile without register spills, all for sm_100a."""
    log = os.path.join(ROOT, "paper_2310_03121_b200", "build_ptxas.log")
    if not os.path.exists(log):
        import paper_2310_03121_b200.build as b
        b.build(force=True)
    txt = open(log).read()
    entries = re.findall(r"Compiling entry function '([^']+)' for '([^']+)'\s*\n[^\n]*\n\s*(\d+) bytes stack frame, "
                         r"(\d+) bytes spill stores, (\d+) bytes spill loads", txt)
    assert entries, "no ptxas -v records in build_ptxas.log"
    assert all(arch == "sm_100a" for _, arch, _, _, _ in entries)
    hot = {"k_aevILi5ELi4": 0, "k_backwardILi5ELi4ELb0": 0, "k_backwardILi5ELi4ELb1": 0, "k_nbrILi4ELi27": 0,
           "k_refreshILi4": 0, "k_mlp_tc": 0}
    for name, _, _, st, ld in entries:
        for key in hot:
            if key in name:
                hot[key] += 1
                assert int(st) == 0 and int(ld) == 0, "%s spills: %s B stores / %s B loads" % (key, st, ld)
    missing = [k for k, n in hot.items() if n == 0]
    assert not missing, "hot kernels not found in the ptxas log: %s" % missing


def test_a_failed_build_is_not_hidden_by_an_older_library(monkeypatch):
    """If the sources changed and nvcc fails, loading must raise instead of silently using the previous binary."""
    import paper_2310_03121_b200 as pkg
    import paper_2310_03121_b200.build as b
    assert b.compiler_present()
    assert os.path.exists(pkg.LIB_PATH)
    monkeypatch.setattr(pkg, "_lib", None)
    monkeypatch.setattr(b, "_stale", lambda: True)
    monkeypatch.setattr(b, "NVCC_FLAGS", b.NVCC_FLAGS + ["--no-such-nvcc-flag"])
    with pytest.raises(RuntimeError):
        pkg.lib()
    assert os.path.exists(pkg.LIB_PATH)      # the old library is left alone, just not loaded
