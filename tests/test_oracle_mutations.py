"""Mutation check of the oracle's pins (CPU only): every plausible one-line mistake in oracle/amp_oracle.cpp listed in
tests/oracle_mutants.py must make at least one pin of tests/test_oracle_pins.py fail.

For each mutant the oracle package is copied to a temporary directory, the one line is changed in the copy, and the named pins
run in a fresh interpreter whose import path finds the copy first (the copy builds its own liboracle.so).  The oracle's own
regression file (tests/golden/oracle_regression.json) is written BY the oracle and pins nothing: it is never among the killers.
An unmutated copy must pass the same pins (control).  The oracle under oracle/ is never touched.
"""
import os
import shutil
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

import pytest

from oracle_mutants import MUTANTS

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
PINS = os.path.join(ROOT, "tests", "test_oracle_pins.py")


def run_pins(mutation, select):
    """(return code, output tail) of `pytest test_oracle_pins.py -k select` against a copy of oracle/ with `mutation` applied"""
    tmp = tempfile.mkdtemp(prefix="oracle_mutant_")
    try:
        shutil.copytree(os.path.join(ROOT, "oracle"), os.path.join(tmp, "oracle"), ignore=shutil.ignore_patterns("*.so", "__pycache__"))
        if mutation is not None:
            old, new = mutation
            src = os.path.join(tmp, "oracle", "amp_oracle.cpp")
            text = open(src).read()
            assert text.count(old) == 1, f"mutation target occurs {text.count(old)} times: {old!r}"
            open(src, "w").write(text.replace(old, new))
        # `python -m pytest` puts the working directory first on sys.path: the copy shadows ROOT/oracle
        env = dict(os.environ, PYTHONPATH=tmp + os.pathsep + ROOT, OMP_NUM_THREADS="2")
        probe = subprocess.run([sys.executable, "-c", "import oracle.oracle as o; print(o._lib._name)"], cwd=tmp, env=env, capture_output=True, text=True)
        assert probe.returncode == 0 and probe.stdout.strip().startswith(tmp), (probe.stdout, probe.stderr[-2000:])
        r = subprocess.run([sys.executable, "-m", "pytest", PINS, "-x", "-q", "-p", "no:cacheprovider", "--rootdir", ROOT,
                            "-k", f"({select}) and not golden_oracle_regression"], cwd=tmp, env=env, capture_output=True, text=True)
        return r.returncode, (r.stdout + r.stderr)[-1500:]
    finally:
        shutil.rmtree(tmp, ignore_errors=True)


def test_mutant_list_is_well_formed():
    names = [m[0] for m in MUTANTS]
    assert len(set(names)) == len(names) and len(MUTANTS) >= 40
    text = open(os.path.join(ROOT, "oracle", "amp_oracle.cpp")).read()
    for name, old, new, select in MUTANTS:
        assert text.count(old) == 1 and old != new and select, name


def test_unmutated_copy_passes_the_pins_used_as_killers():
    rc, tail = run_pins(None, "P3c or P4b or P7 or P10 or P12_")
    assert rc == 0, tail


def test_every_mutant_is_killed_by_a_pin():
    with ThreadPoolExecutor(max(2, min(8, (os.cpu_count() or 2)))) as pool:
        results = list(pool.map(lambda m: (m[0],) + run_pins((m[1], m[2]), m[3]), MUTANTS))
    survivors = [(name, tail[-300:]) for name, rc, tail in results if rc != 1 or " failed" not in tail]
    assert not survivors, survivors
