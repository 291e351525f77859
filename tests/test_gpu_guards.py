"""Guard-band run of the sanitizer scenarios (tests/sanitize_scenarios.py): compute-sanitizer is closed on this GPU pool,
so out-of-bounds WRITES are looked for with 4 KB guard bands around every device buffer of the library
(pvg_guard_bands / pvg_check_guards), over every list builder, round structure and render target. In a subprocess:
the hook is process-wide."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_scenarios_leave_every_guard_band_intact():
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitize_scenarios.py")], capture_output=True, text=True,
                       timeout=900, cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert "none damaged" in r.stdout and "sanitize scenarios ok" in r.stdout


def test_a_damaged_band_is_reported():
    """The check must bite: a write 16 bytes in front of a workspace buffer is found."""
    code = r'''
import sys
sys.path.insert(0, %r)
import numpy as np, torch
import paper_2311_18561_b200 as pvg
from workloads import make_config
from cuda import cudart
pvg.use_torch_allocator(False)
pvg.guard_bands(True)
wl = make_config(0)
s = wl.scene
sc = pvg.Scene(s.mu, s.quat, s.scale, s.opacity, s.sh, s.tau, s.beta, s.vel, torch_allocator=False)
sc.render(wl.cameras[0], 0.37)
torch.cuda.synchronize()
assert pvg.check_guards()[0] == 0
d = sc.debug_info()
err, = cudart.cudaMemset(int(d.record) - 16, 0, 8)
assert int(err) == 0
bad, n = pvg.check_guards()
assert bad == 1 and n > 10, (bad, n)
print("damage detected")
''' % ROOT
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0 and "damage detected" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
