"""The oracle against its frozen output on config 1 (tests/golden/tiny_oracle.txt, written by
tests/golden/make_golden.py from oracle/ alone): integer lines exactly, floats to 1e-9 relative."""
import os
import re
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.join(HERE, "golden"))


def _split(line):
    return [(tok, None) if not re.fullmatch(r"[-+]?\d\.\d+e[-+]\d+", tok) else (None, float(tok)) for tok in line.split()]


def test_oracle_matches_frozen_values():
    import make_golden
    with open(os.path.join(HERE, "golden", "tiny_oracle.txt")) as fh:
        stored = fh.read().splitlines()
    now = make_golden.golden_lines()
    assert len(stored) == len(now)
    for a, b in zip(stored, now):
        ta, tb = _split(a), _split(b)
        assert len(ta) == len(tb), (a, b)
        for (sa, fa), (sb, fb) in zip(ta, tb):
            if fa is None:
                assert sa == sb, (a, b)
            else:
                assert abs(fa - fb) <= 1e-9 * max(abs(fa), 1e-12) + 1e-300, (a, b)
