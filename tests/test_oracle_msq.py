"""Pins for SURVEY.md 8c step 4-5: Table I values, textbook limits, crossing relations, channel table."""
import os
from collections import Counter

import numpy as np
import pytest

from oracle import bzo

PTS = [(2.0, -0.5, -1.5), (1.0, -0.5, -0.5), (3.7, -3.1, -0.6), (0.9, -0.05, -0.85)]


def test_table1_worked_point(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "table1_worked_point.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 7
    for kind, val in rows:
        assert bzo.msq(kind, 2.0, -0.5, -1.5, 0.5, 1.0) == pytest.approx(float(val), rel=1e-14)


def test_textbook_spin_colour_averaged_limits():
    # Unregulated (m^2 = 0) Table I divided by the number of initial colour x helicity states must be the textbook
    # averaged |M|^2/g^4 of massless QCD (Combridge, Kripfganz, Ranft 1977; Peskin & Schroeder Eq. 17.64-17.71):
    for s, t, u in PTS:
        book = {
            "A": (4 / 9) * (s * s + u * u) / t ** 2,
            "11": (4 / 9) * ((s * s + u * u) / t ** 2 + (s * s + t * t) / u ** 2) - (8 / 27) * s * s / (t * u),
            "1B": (4 / 9) * ((s * s + u * u) / t ** 2 + (t * t + u * u) / s ** 2) - (8 / 27) * u * u / (s * t),
            "ANN": (4 / 9) * (t * t + u * u) / s ** 2,
            "QQGG": (32 / 27) * (t * t + u * u) / (t * u) - (8 / 3) * (t * t + u * u) / s ** 2,
            "QG": -(4 / 9) * (s * s + u * u) / (s * u) + (s * s + u * u) / t ** 2,
            "GG": (9 / 2) * (3 - t * u / s ** 2 - s * u / t ** 2 - s * t / u ** 2),
        }
        states = {"A": 36, "11": 36, "1B": 36, "ANN": 36, "QQGG": 36, "QG": 96, "GG": 256}
        for kind, val in book.items():
            assert bzo.msq(kind, s, t, u, 0.0, 1.0) / states[kind] == pytest.approx(val, rel=1e-13)
        # g g -> q qbar is the time reverse of q qbar -> g g: averaged over 256 gluon states
        gg_qq = (1 / 6) * (t * t + u * u) / (t * u) - (3 / 8) * (t * t + u * u) / s ** 2
        assert bzo.msq("QQGG", s, t, u, 0.0, 1.0) / 256 == pytest.approx(gg_qq, rel=1e-13)


def test_crossing_relations_and_symmetries():
    for s, t, u in PTS:
        M = lambda k, a, b, c: bzo.msq(k, a, b, c, 0.0, 1.0)
        assert M("ANN", s, t, u) == pytest.approx(M("A", t, s, u), rel=1e-13)          # s <-> t
        assert M("1B", s, t, u) == pytest.approx(M("11", u, t, s), rel=1e-13)          # s <-> u
        assert M("QG", s, t, u) == pytest.approx(-M("QQGG", t, s, u), rel=1e-13)       # one fermion line crossed
        assert M("GG", s, t, u) == pytest.approx(M("GG", t, s, u), rel=1e-13)          # fully crossing symmetric
        assert M("GG", s, t, u) == pytest.approx(M("GG", u, t, s), rel=1e-13)
        for k in ("11", "ANN", "QQGG", "GG"):                                          # t <-> u symmetric rows
            assert bzo.msq(k, s, t, u, 0.3, 1.0) == pytest.approx(bzo.msq(k, s, u, t, 0.3, 1.0), rel=1e-13)
    # g^4 scaling and the regulator only enter through (t - m^2), (u - m^2)
    assert bzo.msq("GG", 2.0, -0.5, -1.5, 0.5, 3.0) == pytest.approx(3.0 * bzo.msq("GG", 2.0, -0.5, -1.5, 0.5, 1.0))
    assert bzo.msq("A", 2.0, -0.5, -1.5, 0.5, 1.0) == pytest.approx(16 * (4 + 2.25) / (-1.0) ** 2)
    assert bzo.msq("ANN", 2.0, -0.5, -1.5, 0.5, 1.0) == bzo.msq("ANN", 2.0, -0.5, -1.5, 0.0, 1.0)


def _kind(name):
    return bzo.KINDS[name]


def test_channel_counts_per_config():
    assert len(bzo.Oracle(np_=2, species=(0,)).channels()) == 1
    assert len(bzo.Oracle(np_=2, species=(1, 2, 3, 4, 5, 6)).channels()) == 90
    assert len(bzo.Oracle(np_=2, species=(0, 1, 2, 3, 4, 5, 6)).channels()) == 127
    assert len(bzo.Oracle(np_=2, species=(0, 1, 2)).channels()) == 1 + 2 + 4 * 2 + 2 + 2 * (2 + 1)


def test_channel_table_matches_eq3_eq4():
    # Eq. 3 for a quark at slot 1 and Eq. 4 for a gluon at slot 1; the paper's 1/2 for identical
    # pairs and 1 otherwise are (1/2) x (number of orderings of the final pair), so the ORDERED table must hold:
    sp = (0, 1, 2, 3, 4, 5, 6)
    ch = bzo.Oracle(np_=2, species=sp).channels()
    assert len(set(ch)) == len(ch)
    for a in range(7):
        mine = [c for c in ch if c[0] == a]
        kinds = Counter(c[4] for c in mine)
        if a == 0:
            assert kinds == {_kind("GG"): 1, _kind("QQGG"): 6, _kind("QG"): 12}
        else:
            assert kinds == {_kind("11"): 1, _kind("1B"): 2, _kind("QQGG"): 1, _kind("QG"): 2,
                             _kind("A"): 8, _kind("ANN"): 4}
    anti = lambda i: i + 1 if i % 2 else i - 1
    for (a, b, c, d, kind, crossed) in ch:
        # species content is conserved or converted exactly as the process says
        if kind in (_kind("A"), _kind("QG"), _kind("1B")):
            assert (c, d) == ((a, b) if not crossed else (b, a))
            if kind == _kind("1B"):
                assert b == anti(a)
            if kind == _kind("QG"):
                assert (a == 0) != (b == 0)
            if kind == _kind("A"):
                assert a != 0 and b != 0 and b != a and b != anti(a)
        elif kind == _kind("11"):
            assert a == b == c == d and a != 0 and not crossed
        elif kind == _kind("GG"):
            assert a == b == c == d == 0 and not crossed
        elif kind == _kind("ANN"):
            assert b == anti(a) and d == anti(c) and (c - 1) // 2 != (a - 1) // 2 and not crossed
        elif kind == _kind("QQGG"):
            assert not crossed
            assert (a == b == 0 and c != 0 and d == anti(c)) or (c == d == 0 and a != 0 and b == anti(a))
    # the table is closed under time reversal (needed for Eq. 22) and under exchanging the two incoming legs
    keys = {(a, b, c, d): (k, x) for (a, b, c, d, k, x) in ch}
    for (a, b, c, d), (k, x) in keys.items():
        assert keys[(c, d, a, b)] == (k, x)
        assert keys[(b, a, d, c)] == (k, x)
