"""Locality score (Eq. 3, 8, 9, 10): the oracle against a hand-worked example (tests/golden/locality_score.txt) and
simple invariants; the C library (host-only entry points of libfcg.so, no GPU needed) against the oracle on random
traces, value by value and in ranking order."""
import os

import numpy as np
import pytest

from oracle import fcg_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "locality_score.txt")
TRACES = [[0, 1, 2], [0, 1], [1, 3]]
PPL = {0: 10.0, 1: 20.0, 2: 40.0, 3: 5.0}


def _golden_rows():
    for line in open(GOLDEN):
        if line.strip() and not line.startswith("#"):
            a, b, g, fid, exp = line.split()
            yield float(a), float(b), float(g), int(fid), float(exp)


def _feed(obj):
    for t in TRACES:
        obj.record(t)
    for f, p in PPL.items():
        obj.set_ppl(f, p)


def test_oracle_matches_hand_worked_example():
    s = O.LocalityScore()
    _feed(s)
    rows = list(_golden_rows())
    assert len(rows) >= 8
    for a, b, g, fid, exp in rows:
        assert s.score(fid, a, b, g) == pytest.approx(exp, abs=1e-12), (a, b, g, fid)
    assert s.rank([0, 1, 2, 3], 0.5, 0.3, 0.2) == [2, 0, 1, 3]


def test_oracle_invariants():
    rng = np.random.default_rng(7)
    s = O.LocalityScore()
    for _ in range(30):
        s.record(rng.integers(0, 12, size=rng.integers(1, 9)).tolist())
    for f in range(12):
        s.set_ppl(f, float(rng.uniform(1, 50)))
    last = s.last
    for f in range(12):
        for w in ((1, 0, 0), (0, 1, 0), (0, 0, 1), (0.2, 0.5, 0.3)):
            v = s.score(f, *w)
            assert 0.0 <= v <= 1.0                      # every component is normalised to [0, 1]
            if f in last:
                assert v == 1.0                         # l_curr enforces immediate retention
    assert max(s.score(f, 1, 0, 0) for f in range(12) if f not in last) <= 1.0
    most = max(s.count, key=s.count.get)
    if most not in last:
        assert s.score(most, 1, 0, 0) == 1.0            # Eq. 8: the most invoked function has l_freq = 1
    s.forget(most)
    assert s.score(most, 0.5, 0.3, 0.2) == 0.0 and all(most not in kj for kj in s.follow)


def test_c_library_matches_oracle():
    from paper_2606_13097_b200.binding import FcgScorer
    c, o = FcgScorer(), O.LocalityScore()
    _feed(c), _feed(o)
    for a, b, g, fid, exp in _golden_rows():
        assert c.score(fid, a, b, g) == pytest.approx(exp, abs=1e-12)
    rng = np.random.default_rng(11)
    c, o = FcgScorer(), O.LocalityScore()
    for step in range(60):
        tr = rng.integers(0, 20, size=rng.integers(0, 10)).tolist()
        c.record(tr), o.record(tr)
        if step % 5 == 0:
            f, p = int(rng.integers(0, 20)), float(rng.uniform(0, 80))
            c.set_ppl(f, p), o.set_ppl(f, p)
        if step % 17 == 16:
            f = int(rng.integers(0, 20))
            c.forget(f), o.forget(f)
        w = rng.dirichlet([1, 1, 1])
        for f in range(21):
            assert c.score(f, *w) == pytest.approx(o.score(f, *w), abs=1e-12)
        ids = rng.permutation(21).tolist()
        ranked, scores = c.rank(ids, *w)
        ref = o.rank(ids, *w)
        assert ranked == ref or all(abs(o.score(x, *w) - o.score(y, *w)) < 1e-12 for x, y in zip(ranked, ref))
        assert scores == sorted(scores)
    c.close()
