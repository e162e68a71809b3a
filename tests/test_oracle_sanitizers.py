"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: oracle/mpm_oracle.c is compiled
once with -fsanitize=address,undefined and the brute-force pins, the boundary / recycling pins and a short run of every
workload generator are repeated against that build in a child process (the sanitizer runtime must be the first
library of the process, hence LD_PRELOAD).  Any report (heap overflow on a halo node, signed overflow in an index,
misaligned access) aborts the child and fails the test.  CPU only."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _gcc_file(name):
    out = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
    return out if os.path.isabs(out) and os.path.exists(out) else None


def test_oracle_pins_under_asan_ubsan(tmp_path):
    asan = _gcc_file("libasan.so")
    if asan is None:
        pytest.skip("gcc has no libasan.so on this machine")
    lib = str(tmp_path / "libmpm_oracle_san.so")
    subprocess.check_call(["gcc", "-std=c99", "-O1", "-g", "-ffp-contract=off", "-fno-omit-frame-pointer",
                           "-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fPIC", "-shared",
                           "-o", lib, os.path.join(ROOT, "oracle", "mpm_oracle.c"), "-lm"])
    env = dict(os.environ, MPM_ORACLE_LIB=lib, LD_PRELOAD=asan,
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1")
    sel = "brute_force or outflow_recycling or obstacle_rule or wall_inflow or derived_normals or mirror_symmetry"
    r = subprocess.run([sys.executable, "-m", "pytest", os.path.join(ROOT, "tests", "test_oracle_pins.py"), "-x", "-q",
                        "-p", "no:cacheprovider", "-k", sel], env=env, capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    assert "passed" in r.stdout and "ERROR: AddressSanitizer" not in r.stderr and "runtime error" not in r.stderr
    # every workload generator, a few full steps each (all boundary types, obstacle with derived normals, recycling)
    code = (
        "import sys; sys.path.insert(0, %r)\n"
        "from oracle import pyoracle as po\n"
        "from paper_2404_17057_b200 import inputs\n"
        "for w in (inputs.sod(nx=32, ny=4), inputs.periodic_box(n=24), inputs.cylinder(nx=64, ny=32), inputs.sedov(n=10),\n"
        "          inputs.clumps(n=8, num_particles=4000), inputs.sphere_tunnel()):\n"
        "    o = po.Oracle(w['cfg']); o.load_particles(w['x'], w['v'], w['mass'], w['rho'], w['e'])\n"
        "    o.step(0.0, w['cfl'], 6); assert o.stats().step == 6\n"
        "print('ok')\n" % ROOT)
    r = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, cwd=ROOT)
    assert r.returncode == 0 and "ok" in r.stdout, r.stdout[-2000:] + r.stderr[-3000:]
