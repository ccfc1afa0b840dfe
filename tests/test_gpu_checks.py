"""-m gpu: the -DMCRT_CHECKS build of the library (every storage-slot index is range-checked on
the device before use) runs small cases of every kernel path and must count zero violations.
Stands in for compute-sanitizer, which the GPU pool does not offer."""
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
from paper_1201_3588_b200 import mcrt, workloads as W
assert mcrt.debug_violations() == 0, "library was not built with -DMCRT_CHECKS"
cases = [W.c0(n_packets=20000, batch=10000),
         W.tiny_random(n_root=3, seed=4, external=True, n_packets=20000, batch=5000),
         W.tiny_random(n_root=2, sub=4, n_refined=8, seed=2, external=True, n_packets=20000, batch=5000),
         W.tiny_random(n_root=3, sub=3, n_refined=7, seed=8, external=True, n_packets=20000, batch=5000),
         W.tiny_random(n_root=2, sub=8, n_refined=3, seed=9, external=True, n_packets=20000, batch=5000),
         W.c2(n_root=16, n_packets=20000, batch=10000),
         W.c3(n_root=32, n_packets=20000, batch=10000),
         W.c4(n_root=24, n_packets=20000, batch=10000, corr_cells=3.0)]
for wl in cases:
    for layout in (1, 2):
        ctx = mcrt.from_workload(wl, layout=layout)
        ctx.set_observer(n_mu=4, n_pix=8, half_angle_deg=30.0, half_width_cm=wl.n_root * wl.root_size / 2)
        for f, c in wl.batches():
            ctx.run_batch(wl.seed, f, c)
        cn = ctx.get_counters()
        assert cn["emitted"] == cn["escaped"] == 20000 and cn["lost"] == 0, cn
        ctx.get_cell_temperature(); ctx.get_cell_energy(); ctx.get_sed_mu(); ctx.get_image()
        ctx.destroy()
print("VIOLATIONS", mcrt.debug_violations())
"""


def test_checked_build_counts_no_out_of_range_index():
    import torch
    assert torch.cuda.is_available()
    from paper_1201_3588_b200 import build
    lib = build.build_library(checks=True)
    env = dict(os.environ, MCRT_LIBRARY=lib, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
    r = subprocess.run([sys.executable, "-c", SCRIPT], env=env, cwd=ROOT, capture_output=True,
                       text=True, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "VIOLATIONS 0" in r.stdout, r.stdout


def test_production_build_has_no_checks():
    from paper_1201_3588_b200 import build, mcrt
    build.build_library()
    assert mcrt.debug_violations() == -1


DIGEST = r"""
import hashlib
import numpy as np
from paper_1201_3588_b200 import mcrt, workloads as W
h = hashlib.sha256()
for wl, layout, sweeps in [(W.c1(tau_v=3.0, n_packets=200000, batch=100000), 1, 0),
                           (W.tiny_random(n_root=13, seed=5, external=True, tau_cell=0.2, n_packets=60000, batch=20000), 2, 0),
                           (W.c2(n_root=32, n_packets=300000, batch=100000), 0, 0),
                           (W.c3(n_root=32, n_packets=200000, batch=100000), 2, 0),
                           (W.tiny_random(n_root=3, sub=3, n_refined=7, seed=8, external=True, n_packets=40000, batch=10000), 0, 0),
                           (W.c1(tau_v=3.0, n_packets=200000, batch=100000), 3, 0),
                           (W.c4(n_root=256, n_packets=400000, batch=200000), 0, 3)]:
    ctx = mcrt.from_workload(wl, layout=layout)
    if sweeps:
        ctx.set_region_sweeps(sweeps, (64, 128, 64))
    for f, c in wl.batches():
        ctx.run_batch(wl.seed, f, c)
    cn = ctx.get_counters()
    for a in (ctx.get_cell_energy()[0], ctx.get_sed(), ctx.get_cell_temperature(), cn["emitted_per_bin"]):
        h.update(np.ascontiguousarray(a).tobytes())
    h.update(repr(sorted((k, int(v)) for k, v in cn.items() if np.ndim(v) == 0)).encode())
    ctx.destroy()
print("DIGEST", h.hexdigest())
"""


def test_ptx_walk_equals_the_checked_build():
    """The production build walks through PTX blocks (transport_u.cuh walk_pair_ptx, walk_step_tl_ptx), the checked
    build through the C++ step: same operations in the same order, so tallies, SEDs, temperatures and counters
    must be identical bit for bit (plain walk, brick layout, cubes and subcubes with S = 3 and 4, bricked root,
    macro cubes, swept regions)."""
    from paper_1201_3588_b200 import build
    out = []
    for lib in (build.build_library(), build.build_library(checks=True)):
        env = dict(os.environ, MCRT_LIBRARY=lib, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
        r = subprocess.run([sys.executable, "-c", DIGEST], env=env, cwd=ROOT, capture_output=True, text=True,
                           timeout=600)
        assert r.returncode == 0, r.stdout + r.stderr
        out.append([l for l in r.stdout.splitlines() if l.startswith("DIGEST")][-1])
    assert out[0] == out[1], out
