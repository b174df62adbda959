"""The bounds-checked build of the library (-DWOLFF_CHECKED: every queue, list, tile and bit-plane index the growth
kernels compute is compared with its bound before use, device_common.cuh) on the small, knob-stressed cases of
tests/sanitizer_cases.py -- tiny tiles on few CTAs, 32-entry ring and inbox, bond tables on and off, every tier, the batch,
in-kernel measurement -- each compared with the oracle.  SURVEY.md section 4 tier 4 / section 5 "Race detection":
compute-sanitizer is closed on the development pool, this is the memory check that runs there."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
def test_checked_build_runs_clean_on_the_stress_cases():
    from paper_1110_0899_b200 import build
    lib = build.build(checked=True)
    env = dict(os.environ, WOLFF_B200_LIB=lib)
    out = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_cases.py")], env=env, capture_output=True, text=True,
                         timeout=900)
    assert out.returncode == 0, out.stdout[-2000:] + out.stderr[-4000:]
    assert "sanitizer cases passed: 21" in out.stdout


@pytest.mark.gpu
def test_schedule_perturbing_build_runs_clean_on_the_stress_cases():
    # -DWOLFF_JITTER: random sleeps of up to 2 us between the steps of every lock-free protocol of the growth kernels
    # (ring reserve / put / take, inbox slot / message, pending counts, publishing, stealing, termination), so that
    # interleavings the hardware rarely produces become common; every case is compared with the oracle, three rounds
    from paper_1110_0899_b200 import build
    lib = build.build(jitter=True)
    env = dict(os.environ, WOLFF_B200_LIB=lib)
    for which in ("tiles", "cluster", "tiles", "cluster", "tiles", "cluster"):
        out = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_cases.py"), which], env=env, capture_output=True, text=True,
                             timeout=900)
        assert out.returncode == 0, out.stdout[-2000:] + out.stderr[-4000:]
        assert "sanitizer cases passed" in out.stdout


@pytest.mark.gpu
def test_checked_build_reports_a_violation():
    # the check itself must be alive: the checked build honours a test hook that feeds it an index past its bound
    from paper_1110_0899_b200 import build
    lib = build.build(checked=True)
    code = (
        "import sys; sys.path.insert(0, %r)\n"
        "from paper_1110_0899_b200 import binding\n"
        "g = binding.Wolff(2, 16, 1.0, 2.0, 1)\n"
        "g.set_option('mode', 4); g.set_option('check_selftest', 1)\n"
        "g.run(3)\n"
        "try:\n"
        "    g.observables(); g.stats()\n"
        "except binding.WolffError as e:\n"
        "    print('caught', e.code, e)\n"
    ) % ROOT
    out = subprocess.run([sys.executable, "-c", code], env=dict(os.environ, WOLFF_B200_LIB=lib), capture_output=True, text=True, timeout=300)
    assert "caught -4" in out.stdout and "checked build" in out.stdout, out.stdout + out.stderr[-2000:]
