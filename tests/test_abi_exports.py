"""The C-ABI library builds, loads and exports every symbol include/mpm.h declares (no compute call: runs without a GPU)."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "mpm.h")).read()
    return sorted(set(re.findall(r"MPM_API\s+[\w\s\*]+?\b(mpm_\w+)\s*\(", text)))


def test_header_declares_the_boundary_calls():
    names = _declared()
    for need in ("mpm_create", "mpm_load_particles", "mpm_step", "mpm_read_particles", "mpm_read_grid",
                 "mpm_get_stats", "mpm_last_error", "mpm_destroy"):
        assert need in names


def test_library_builds_and_exports_every_declared_symbol():
    from paper_2404_17057_b200 import build, binding
    path = build.build()
    lib = ctypes.CDLL(path)
    for name in _declared():
        assert hasattr(lib, name), name
    assert sorted(binding.EXPORTS) == _declared()
    lib.mpm_abi_version.restype = ctypes.c_int
    assert lib.mpm_abi_version() == 3          # pure host function, no CUDA involved


def test_struct_layouts_match_the_header():
    """ctypes mirrors of mpm_config / mpm_stats have the size the C compiler gives the header's structs."""
    import subprocess
    import tempfile
    from paper_2404_17057_b200 import binding
    src = '#include "mpm.h"\n#include <stdio.h>\nint main(){printf("%zu %zu\\n", sizeof(mpm_config), sizeof(mpm_stats));return 0;}\n'
    with tempfile.TemporaryDirectory() as d:
        c = os.path.join(d, "s.c"); exe = os.path.join(d, "s")
        open(c, "w").write(src)
        subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), "-o", exe, c])
        a, b = map(int, subprocess.check_output([exe]).split())
    assert ctypes.sizeof(binding.Config) == a
    assert ctypes.sizeof(binding.Stats) == b


def test_no_cpu_fallback_without_cuda():
    """Without a CUDA device the product path fails loudly instead of routing anywhere else."""
    import pytest
    import torch
    from paper_2404_17057_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    with pytest.raises(RuntimeError):
        binding.load()
    with pytest.raises(RuntimeError):
        binding.Solver(dict(dim=2, n=[4, 4], dx=0.25))


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2404_17057_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "pyoracle" not in text and "mpm_oracle" not in text and "from oracle" not in text, f
    for f in ("mpm_oracle.c", "mpm_oracle.h", "pyoracle.py"):
        text = open(os.path.join(ROOT, "oracle", f)).read()
        assert "paper_2404_17057_b200" not in text.replace("paper_2404_17057_b200/)", "") or f != "mpm_oracle.c"
        assert "binding" not in text and "mpm.h" not in text, f
