"""Regression pin of the oracle's 3D cubic-cell path: the digests in
tests/golden/oracle_3d_digest.txt were written by the round-1 oracle (the version pinned by
P1-P12) before it was extended to 1D / 2D runs and non-cubic cells; the oracle as it stands must
reproduce them bit for bit."""
import os
import sys

sys.path.insert(0, os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden"))

import make_oracle_digest as mk  # noqa: E402


def test_oracle_3d_cubic_path_reproduces_round1_digests():
    want = {}
    for ln in open(os.path.join(os.path.dirname(mk.__file__), "oracle_3d_digest.txt")):
        if ln.startswith("#") or not ln.strip():
            continue
        name, digest, t, n = ln.split()
        want[name] = (digest, t, int(n))
    assert len(want) == len(mk.CASES)
    for c in mk.CASES:
        assert mk.run(c) == want[c[0]], c[0]
