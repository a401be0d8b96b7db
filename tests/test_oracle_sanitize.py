"""The oracle under AddressSanitizer + UndefinedBehaviorSanitizer: the pin suite (without the
hour-scale box runs, which get a shortened stand-in here) is re-run in a child process against
``oracle/liboracle_san.so`` = the same source built with ``-fsanitize=address,undefined -fno-sanitize-recover``.
Any out-of-bounds access, use after free, signed overflow, bad shift or misaligned access in ``oracle/`` aborts the
child and fails this test."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _asan_runtime():
    try:
        p = subprocess.run(["gcc", "-print-file-name=libasan.so"], capture_output=True, text=True).stdout.strip()
    except OSError:
        return None
    return p if os.path.isabs(p) and os.path.exists(p) else None


@pytest.mark.skipif(_asan_runtime() is None, reason="gcc's libasan.so not found")
def test_oracle_pins_pass_under_asan_and_ubsan():
    env = dict(os.environ, ORACLE_SANITIZE="1", LD_PRELOAD=_asan_runtime(), OMP_NUM_THREADS="4",
               ASAN_OPTIONS="detect_leaks=0:abort_on_error=1", UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1")
    code = r"""
import sys, numpy as np
sys.path.insert(0, %r)
import oracle
assert oracle._SO.endswith("liboracle_san.so")
import pytest
# every pin except the two 16-seed / 4-seed x 3600-step box runs and the 40000-trial statistics
rc = pytest.main(["-q", "-x", "-p", "no:cacheprovider", "tests/test_oracle_pins.py", "-k",
                  "not box_golovin and not bruteforce and not pairings_of_four"])
assert rc == 0, rc
# shortened stand-ins for what was skipped: a box run with recycling, substepped coalescence in a full 3D step
o = oracle.Oracle(dx=100, dy=100, dz=100, dt=1.0, kernel="golovin", golovin_b=1500.0, seed=42)
o.set_recycle(True)
N = 2048
v = np.random.default_rng(1).exponential(4 / 3 * np.pi * 30.531e-6**3, N)
o.set_state(np.full(N, 2**23 * 10**6 // N, np.uint64), (v / (4 / 3 * np.pi)) ** (2 / 3), np.full(N, 1e-27), np.full(N, 0.5))
for _ in range(400):
    o.step(oracle.make_opts(adve=False, sedi=False, cond=False, coal=True, sstp_coal=2))
assert o.counters()["collisions"] > 1000
rng = np.random.default_rng(2)
o = oracle.Oracle(nx=4, ny=3, nz=5, dx=20.0, dy=20.0, dz=20.0, dt=1.0, kernel="geometric", seed=3)
o.set_threads(4)
nc, M = 60, 3000
o.set_fields(th=np.full(nc, 289.0), rv=np.full(nc, 9e-3), rhod=np.full(nc, 1.1), cx=rng.uniform(-.2, .2, 5 * 3 * 5),
             cy=rng.uniform(-.2, .2, 4 * 4 * 5), cz=rng.uniform(-.2, .2, 4 * 3 * 6))
rd = np.exp(rng.uniform(np.log(1e-8), np.log(3e-7), M))
o.set_state(rng.integers(1, 10**9, M).astype(np.uint64), (rd * rng.uniform(1.5, 400, M)) ** 2, rd**3, np.full(M, 0.61),
            x=rng.uniform(0, 80, M), y=rng.uniform(0, 60, M), z=rng.uniform(0, 100, M))
for _ in range(12):
    o.step(oracle.make_opts(RH_max=1.05, sstp_coal=3))
o.diag_mom(1, 1e-6, 1e-4, 3); o.diag_sd_conc()
assert o.n_live() < M          # SDs left through the bottom / top and were compacted away
print("sanitized oracle ok")
""" % ROOT
    r = subprocess.run([sys.executable, "-c", code], cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    assert r.returncode == 0 and "sanitized oracle ok" in r.stdout, (r.stdout[-3000:], r.stderr[-3000:])
