"""The oracle reproduces its committed regression anchors (tests/golden/oracle_residuals.txt,
written by tests/golden/make_golden.py from oracle/ only).

This compares the oracle with its own earlier output: it guards against an unnoticed change of the oracle's
arithmetic between commits, and pins nothing.  What pins the oracle is in tests/test_oracle_pins*.py."""
import os

import pytest

from tests.golden import make_golden


def test_oracle_matches_committed_anchors():
    path = os.path.join(os.path.dirname(make_golden.__file__), "oracle_residuals.txt")
    want = [ln.split() for ln in open(path) if not ln.startswith("#")]
    got = list(make_golden.rows())
    assert len(want) == len(got)
    for w, g in zip(want, got):
        assert w[0] == g[0] and int(w[1]) == g[1]
        for a, b in zip(w[2:], g[2:]):
            assert b == pytest.approx(float(a), rel=1e-9, abs=1e-300)
