"""The oracle under AddressSanitizer and UndefinedBehaviorSanitizer ('build the oracle with
-fsanitize=address,undefined'): every collision variant, boundary condition and reorder setting the oracle has is stepped on
a small box in a child process that loads the instrumented build; any out-of-bounds access, use of freed memory, signed
overflow, bad shift or misaligned access aborts the child. The values the oracle computes are checked elsewhere."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

CHILD = r"""
import sys
import numpy as np
sys.path.insert(0, %(root)r)
import oracle.build as build
import oracle.binding as ob
ob._lib_path = build.build(sanitize=True)
from oracle.binding import Oracle
from paper_2406_15236_b200.inputs import uniform_maxwell

cases = [
    dict(thermostat=1, rebin_every=3, brick=(4, 2, 1)),
    dict(thermostat=1, bc=(0, 0, 1), g=(0.01, 0, 0)),
    dict(bc=(0, 2, 0)),
    dict(thermostat=1, bc=(0, 1, 0), wall_velocity=0.2),
    dict(conserve_L=1),
    dict(collision=1),
    dict(collision=1, conserve_L=1),
    dict(thermostat=1, shear_rate=0.05, dt=0.3),
    dict(conserve_L=1, bc=(0, 0, 1), phantoms=1),
    dict(collision=1, bc=(0, 0, 1), phantoms=1, wall_velocity=0.1),
    dict(thermostat=1, solute_id0=1000, solute_mass=5.0),
    dict(thermostat=1, grid_shift=0, brick=2),
]
cells = (6, 5, 7)
box = tuple(float(c) for c in cells)
n = int(np.prod(cells)) * 6 + 3
st = uniform_maxwell(box, n, 3)
for kw in cases:
    o = Oracle(box, cells, 6, 11, **kw)
    o.set_state(*st)
    o.step(7)
    o.get_state(); o.get_cells(); o.observables(cells[2] if kw.get("bc", (0, 0, 0))[1] == 0 else cells[1])
    o.grid_shift(3); o.srd_axis(5, 2)
# edge cases: no particles, one particle, every particle in one cell
o = Oracle(box, cells, 6, 11, thermostat=1)
z = np.zeros(0, np.float32)
o.set_state(z, z, z, z, z, z); o.step(2); o.observables()
one = [np.full(1, 0.5, np.float32)] * 6
o.set_state(*one); o.step(2)
crowd = [np.full(300, 2.5, np.float32)] * 3 + list(st[3:6][i][:300] for i in range(3))
o.set_state(*crowd); o.step(2); o.observables()
print("SANITIZED_OK")
"""


def test_oracle_runs_clean_under_asan_and_ubsan():
    def runtime(name):
        p = subprocess.run(["gcc", "-print-file-name=" + name], capture_output=True, text=True).stdout.strip()
        return p if os.path.isabs(p) and os.path.exists(p) else None

    asan, ubsan = runtime("libasan.so"), runtime("libubsan.so")
    if not asan or not ubsan:
        pytest.skip("sanitizer runtimes not installed")
    env = dict(os.environ)
    env["LD_PRELOAD"] = asan + ":" + ubsan
    env["ASAN_OPTIONS"] = "detect_leaks=0:halt_on_error=1:abort_on_error=0"      # (the interpreter itself leaks by design)
    env["UBSAN_OPTIONS"] = "halt_on_error=1:print_stacktrace=1"
    r = subprocess.run([sys.executable, "-c", CHILD % dict(root=ROOT)], env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0 and "SANITIZED_OK" in r.stdout, (r.stdout[-2000:], r.stderr[-4000:])
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr[-4000:]
