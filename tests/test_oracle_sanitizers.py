"""The oracle under -fsanitize=address,undefined:
a second build of oracle/mcrt_oracle.cpp runs every code path the pins and the parity tests use
(single- and two-level walks, brute-force walker, external field, observer, split batch halves,
the serial Bjorkman-Wood scheme, traces) in a subprocess with libasan preloaded; any report
fails the test.  CPU only."""
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

SCRIPT = r"""
import numpy as np
from oracle import oracle as O
from paper_1201_3588_b200 import workloads as W
O.lib()
for wl in (W.c0(n_packets=3000, batch=1000),
           W.tiny_random(n_root=2, sub=4, n_refined=3, seed=5, external=True, n_packets=3000, batch=1000),
           W.tiny_random(n_root=3, sub=2, n_refined=9, seed=6, external=True, n_packets=3000, batch=1000),
           W.c2(n_root=16, n_packets=3000, batch=1000),
           W.c4(n_root=16, n_packets=3000, batch=1000, corr_cells=2.0)):
    o = O.Oracle(wl)
    o.set_observer(n_mu=5, n_pix=7, direction=(0.02, 0.01, 1.0), half_angle_deg=40.0,
                   half_width_cm=wl.n_root * wl.root_size)
    o.run(threads=2)
    c = o.counters()
    assert c["emitted"] == c["escaped"] == 3000 and c["lost"] == 0
    n, eps = o.cell_energy()
    assert int(n.sum()) == c["absorptions"]
    o.cell_temperature(); o.sed(); o.sed_mu(); o.image(); o.tables()
    o.update_temperature(n, 3000)
    o.transport_batch(wl.seed, 3000, 500, 1)
    for p in range(20):
        o.trace_packet(wl.seed, p)
        x, d, b, s = o.emit(wl.seed, p)
        o.walk(x, d, b, 1.3, walker=0)
    o.reset_tallies(3)
wl = W.tiny_random(n_root=2, sub=4, n_refined=8, seed=2, n_packets=400, batch=200)
b = O.Oracle(wl); b.set_walker(1); b.run()
wl = W.c0(n_packets=2000, batch=2000)
o = O.Oracle(wl); o.run_bw(wl.seed, 0, 2000, 2000)
print("sanitized oracle ok")
"""


def test_oracle_clean_under_asan_ubsan():
    from oracle import oracle as O
    lib = O.build(sanitize=True)
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    env = dict(os.environ, LD_PRELOAD=asan, MCRT_ORACLE_LIBRARY=lib, PYTHONPATH=ROOT,
               ASAN_OPTIONS="detect_leaks=0:halt_on_error=1", UBSAN_OPTIONS="halt_on_error=1:print_stacktrace=1",
               OMP_NUM_THREADS="2")
    r = subprocess.run([sys.executable, "-c", SCRIPT], env=env, cwd=ROOT, capture_output=True,
                       text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-3000:]
    assert "sanitized oracle ok" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-3000:]
