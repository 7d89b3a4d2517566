"""The tracer checking itself: libarc_b200_checked.so is the library built with -DARC_CHECKED=1, in which the kernel
verifies every index it forms (cells, sources, levels, ring / queue slots, staging addresses) before using it
(csrc/arc_internal.cuh ARC_CHECK) and raises a device error otherwise.  A selection of the parity tests - every deposit
route, every bin count, donation through the queue, sources on faces, masks, the geometric correction, the thin region -
is run through that build in a subprocess: they must pass unchanged.  (compute-sanitizer is closed on the pool this was
developed on: profiles/r02_sanitizers.md.)"""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_parity_suite_through_the_checked_build():
    from paper_1807_07094_b200 import build as b
    lib = b.build(force=b.needs_build(checked=True), checked=True)
    env = dict(os.environ, ARC_B200_LIB=lib)
    probe = subprocess.run([sys.executable, "-c", "from paper_1807_07094_b200 import arc; print(arc.arc_version())"],
                           capture_output=True, text=True, cwd=ROOT, env=env)
    assert "checked build" in probe.stdout, probe.stdout + probe.stderr
    sel = ("tiny_random or four_bin_f32 or small_persistent or many_sources or faces_edges or parameter_variants or "
           "repeatable or tiny_workloads or masked_sources or config1_per_ray or two_traces_radii or injected_radii or config1_steps")
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "-p", "no:cacheprovider", "tests/test_gpu_parity.py",
                        "tests/test_gpu_geom.py", "tests/test_gpu_mask.py", "tests/test_gpu_thin.py", "-k", sel],
                       capture_output=True, text=True, cwd=ROOT, env=env, timeout=1800)
    tail = (r.stdout + r.stderr)[-3000:]
    assert r.returncode == 0, tail
    assert " passed" in tail and "failed" not in tail, tail
