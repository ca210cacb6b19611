"""The self-checking build of the library (-DMUCA_CHECKED, csrc/muca_device.cuh "Self-checks").

compute-sanitizer is closed on the GPU pool this library is developed on (profiles/r02_sanitizer.txt), so what its
racecheck / memcheck tools would watch in the sweep kernels -- the hand-over of deviates between paired warps through the
double-buffered shared ring, and the shared-memory address that is the walker's state -- is checked by the kernels
themselves in a second build of the same sources.  Here: every small parity case of tests/test_sanitizer_cases.py
passes under that build (no check fires, results identical to the oracle's), and the checks DO fire when a hand-over
is tagged wrongly on purpose.  The library is chosen when it is loaded, hence the subprocesses.
"""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(code, **env):
    e = dict(os.environ, MUCA_CHECKED="1", **env)
    return subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=e, capture_output=True, text=True, timeout=1200)


def test_parity_cases_pass_under_the_checked_build():
    r = subprocess.run([sys.executable, "-m", "pytest", "tests/test_sanitizer_cases.py", "-q", "-m", "gpu", "-x", "-p", "no:cacheprovider"],
                       cwd=ROOT, env=dict(os.environ, MUCA_CHECKED="1"), capture_output=True, text=True, timeout=1800)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-2000:]
    assert " passed" in r.stdout and "failed" not in r.stdout


PROBE = """
import sys
sys.path.insert(0, 'oracle')
import paper_1707_00919_b200 as mb
assert b'+checked' in mb.lib().muca_version()
g = mb.Muca({L}, {W}, 7)
try:
    g.run_iteration(1, 2)
    print('CLEAN')
except mb.MucaError as e:
    print('FIRED', e)
"""


@pytest.mark.parametrize("L,W", [(32, 70), (64, 40), (128, 33)])
def test_a_wrongly_tagged_hand_over_is_caught(L, W):
    clean = run(PROBE.format(L=L, W=W))
    assert "CLEAN" in clean.stdout, clean.stdout + clean.stderr
    bad = run(PROBE.format(L=L, W=W), MUCA_CHECKED_FAULT="3")
    assert "FIRED" in bad.stdout and "self-check failed" in bad.stdout, bad.stdout + bad.stderr


# The paired kernels address their delta table by an immediate and therefore check where the dynamic shared memory
# starts.  A mismatch (another driver's reserved area, a static __shared__ added later) must come back as an ordinary
# MUCA_ECUDA from muca_run_iteration, with the CUDA context still usable afterwards -- not as a trap that poisons the
# whole process.  MUCA_CHECKED_FAULT=-1 makes the kernels of the checked build pretend the mismatch.
BASE_PROBE = """
import sys
sys.path.insert(0, 'oracle')
import numpy as np, torch
import paper_1707_00919_b200 as mb
from paper_1707_00919_b200 import binding as B
g = mb.Muca({L}, {W}, 7)
E0, n0 = g.get_energies(), g.iteration
try:
    g.run_iteration(1, 2)
    print('CLEAN')
    assert g.iteration == n0 + 1
except mb.MucaError as e:
    print('FIRED', e)
    assert np.array_equal(g.get_energies(), E0) and g.iteration == n0  # the refused iteration touched nothing
torch.cuda.synchronize()                                   # no sticky error: the context still works
ctr, key = np.arange(32, dtype=np.uint32).reshape(8, 4), np.arange(16, dtype=np.uint32).reshape(8, 2)
assert mb.debug_philox(ctr, key).shape == (8, 4)
g.set_option(B.MUCA_OPT_KERNEL, B.MUCA_KERNEL_STREAMED)    # the plain kernel does not depend on the base (L >= 32)
if {L} >= 32:
    assert int(g.run_iteration(1, 2).sum()) == {W} * 2 * {L} * {L}
print('ALIVE')
"""


@pytest.mark.parametrize("L,W", [(16, 40), (32, 70), (64, 40)])
def test_a_shared_memory_base_mismatch_is_an_error_not_a_trap(L, W):
    clean = run(BASE_PROBE.format(L=L, W=W))
    assert "CLEAN" in clean.stdout and "ALIVE" in clean.stdout, clean.stdout + clean.stderr
    bad = run(BASE_PROBE.format(L=L, W=W), MUCA_CHECKED_FAULT="-1")
    assert "FIRED" in bad.stdout and "dynamic shared memory" in bad.stdout and "ALIVE" in bad.stdout, bad.stdout + bad.stderr
