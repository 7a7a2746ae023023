"""The plain-C caller tests/harness/blip_harness.c (no Python between the caller and the C ABI):
it builds against include/blipgpu.h as a C11 translation unit, its self-test of every kernel
passes, and its per-call latency rows (BASELINE.json configs[3], PAPER.md:268 kernel (1)) are
well-formed."""
import json
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, os.path.join(ROOT, "tests", "harness"))
import build as harness_build  # noqa: E402


def test_harness_builds_as_plain_c():
    exe = harness_build.build(force=True)
    assert os.access(exe, os.X_OK)
    r = subprocess.run([exe], capture_output=True, text=True)
    assert r.returncode == 64 and "usage" in r.stderr


def oracle_library():
    """oracle/libblip_oracle.so, built if need be: handed to the self-test as an argument (it loads it
    with dlopen; the harness is never linked against the oracle, bench.py's latency mode never sees it)."""
    from oracle import build as oracle_build
    return oracle_build.build()


@pytest.mark.gpu
def test_harness_selftest():
    """Every kernel through the plain-C caller, each checked against the CPU fp64 oracle with
    north_star's tolerances (the tensor-core kernel too: against the oracle, not only against the
    FP32-pipe kernel)."""
    import re
    r = subprocess.run([harness_build.build(), "selftest", oracle_library()], capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "selftest: 0 failure(s)" in r.stdout
    assert "kernel=2" in r.stdout and "kernel=1" in r.stdout and "kernel=3" in r.stdout and "kernel=5" in r.stdout
    fracs = [float(x) for x in re.findall(r"worst error ([0-9.]+) of the tolerance against the oracle", r.stdout)]
    assert len(fracs) == 8 and 0.0 < max(fracs) < 0.5, r.stdout        # 4 kernels x 2 modes, a few % expected


@pytest.mark.gpu
def test_harness_selftest_on_the_checked_build():
    """The same self-test against the library compiled with -DBLIP_CHECKED: every table row, sorted
    slot, unit, staged plane and output index is compared with its bound inside the kernels and a
    violation traps (the stand-in for compute-sanitizer memcheck, which is closed on this pool)."""
    exe = harness_build.build(checked=True)
    r = subprocess.run([exe, "selftest", oracle_library()], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "selftest: 0 failure(s)" in r.stdout and "BLIP_ASSERT" not in r.stdout + r.stderr
    r = subprocess.run([exe, "fullsize"], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "fullsize: 0 failure(s)" in r.stdout and "BLIP_ASSERT" not in r.stdout + r.stderr


@pytest.mark.gpu
def test_harness_latency_rows():
    r = subprocess.run([harness_build.build(), "latency", "60"], capture_output=True, text=True, timeout=900)
    assert r.returncode == 0, r.stdout + r.stderr
    line = json.loads(r.stdout.strip().splitlines()[-1])
    rows = line["rows"]
    assert [x["M"] for x in rows if x["mode"] == "vgl"] == [1, 8, 32, 128, 512, 1536]
    for x in rows:
        assert x["kernel"] == 3 and 0.5 < x["us_back_to_back"] < 5e3 and x["us_call_and_wait_median"] >= x["us_p10"]
