"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: the tiny scene of configs[0] is
projected, key-listed, rendered (brute force and Gaussian-major) and differentiated (O-8, O-9) in a child process
that preloads libasan; any
out-of-bounds access, use of uninitialised stack, signed overflow or misaligned access aborts the child."""
import os
import subprocess
import sys
from pathlib import Path

ROOT = Path(__file__).resolve().parent.parent

CHILD = r"""
import numpy as np
from paper_2606_17212_b200 import synth
from oracle import oracle as O
O.build()
wl = synth.workload_cfg0()
cam, t = wl.frames[0]
sc = O.OracleScene(wl.scene)
lv = wl.levels[0][::52]
a, sa = sc.render_batch(cam, t, lv, brute_force=True)
b, sb = sc.render_batch(cam, t, lv, brute_force=False)
assert np.array_equal(a, b) and np.array_equal(sa, sb)
p = sc.project(cam, t, np.array([3, 1, -1, 0], np.int8))
tile, dbits, idx = sc.keys(p, cam)
assert len(tile) == p["count"][p["valid"] == 1].sum()
ref, _ = sc.render(cam, t, np.full(4, 3, np.int8))
mse, psnr = O.distortion(a, ref)
assert mse.shape == (lv.shape[0],)
# the backward oracles (O-8, O-9): one state, random dL/d(image)
d3 = np.array([3, 1, -1, 0], np.int8)
g = np.random.default_rng(0).standard_normal((cam.H, cam.W, 3))
g9, gabs = sc.backward(cam, t, d3, g, want_abs=True)
gp = sc.project_backward(cam, t, d3, g9)
assert np.isfinite(gp["mean"]).all() and np.isfinite(gp["sh_base"]).all() and np.any(gp["quat"] != 0.0)
assert O.sh_basis_grad(16, (0.1, 0.2, 0.97)).shape == (3, 16)
print("sanitized oracle ok", len(tile))
"""


def test_oracle_runs_clean_under_asan_ubsan():
    asan = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    assert os.path.isabs(asan) and os.path.exists(asan), "libasan.so not found next to gcc"
    env = dict(os.environ, GSR_ORACLE_SANITIZE="1", LD_PRELOAD=asan, PYTHONPATH=str(ROOT),
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", CHILD], capture_output=True, text=True, env=env, cwd=str(ROOT), timeout=600)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "sanitized oracle ok" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr
