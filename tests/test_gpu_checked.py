"""The bounds-checked build of libbh (-DBH_CHECKED: device-side asserts on the walk's stack and list fills, on every
slot, node id and sort position the kernels compute) run over the small irregular cases in a subprocess.
compute-sanitizer is closed on this GPU pool; this is the repo's own substitute: a failed check traps the kernel,
the call returns BH_ERR_CUDA and the subprocess exits non-zero.  Results must equal the normal build's bit for bit."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import sys, hashlib
import numpy as np, torch
import bh_workloads as wl
import paper_1509_07370_b200 as bh
assert ("checked" in bh.lib_path()) == (sys.argv[1] == "checked"), bh.lib_path()
cases = [wl.uniform_sphere(16), wl.random_points(4099, seed=2, cube=(-1.0, 2.0, 0.5, 3.0)), wl.clustered_points(3000, seed=3),
         wl.with_duplicates(wl.random_points(500, seed=4), 40, seed=4), wl.with_duplicates(wl.random_points(500, seed=5), 40, seed=5, near=3e-7),
         wl.amr_collapsing_core(nroot=2, max_level=3), wl.random_points(33, seed=8), wl.random_points(2, seed=7)]
h = hashlib.sha256()
ctx = bh.Context(0)                       # one context across all inputs: speculated sort plans, aux clearing
for w in cases:
    d = [torch.from_numpy(np.ascontiguousarray(a)).cuda() for a in (w.x, w.y, w.z, w.m)]
    for periodic in (False, True):
        ctx.set_periodic(periodic, N=18, nref=2)
        ctx.build(*d, w.cube)
        for theta in (0.5, 1.0, 0.0) if w.n < 5000 else (0.5,):
            for mac in (0, 1):
                ctx.set_mac(mac)
                h.update(ctx.potential(theta, w.G).cpu().numpy().tobytes())
                h.update(ctx.last_group_counts().cpu().numpy().tobytes())
        if not periodic:
            phi, acc = ctx.field(0.5, w.G)
            h.update(acc.cpu().numpy().tobytes())
            h.update(ctx.essential_nodes((1.0, 0.0, 0.0), (2.0, 1.0, 1.0), 0.5).cpu().numpy().tobytes())
            ctx.set_group(1); h.update(ctx.potential(0.5, w.G).cpu().numpy().tobytes()); ctx.set_group(32)
            ctx.update_masses(d[3] * 2.0); h.update(ctx.potential(0.5, w.G).cpu().numpy().tobytes())
    ctx.set_periodic(False)
torch.cuda.synchronize()
print("DIGEST", h.hexdigest())
"""


def _run(mode):
    env = dict(os.environ, PYTHONPATH=ROOT)
    env["BH_CHECKED"] = "1" if mode == "checked" else "0"
    p = subprocess.run([sys.executable, "-c", SCRIPT, mode], cwd=ROOT, env=env, capture_output=True, text=True, timeout=900)
    assert p.returncode == 0, p.stdout[-2000:] + p.stderr[-4000:]
    return [ln for ln in p.stdout.splitlines() if ln.startswith("DIGEST")][0]


def test_checked_build_passes_and_agrees_with_the_product_build():
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    assert _run("checked") == _run("normal")
