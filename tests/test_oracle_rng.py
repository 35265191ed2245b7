"""Pins for SURVEY.md 8c step 1 (Philox4x32-10, uniforms) and pin P2 (isotropy, Marsaglia acceptance)."""
import math
import os

import numpy as np
from scipy import stats

from oracle import bzo


def test_philox_known_answers(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "philox4x32_10_kat.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        assert bzo.philox4x32_10(v[0:4], v[4:6]) == tuple(v[6:10])


def test_philox_counter_and_key_sensitivity():
    base = bzo.philox4x32_10((1, 2, 3, 4), (5, 6))
    seen = {base}
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        seen.add(bzo.philox4x32_10(c, (5, 6)))
    seen.add(bzo.philox4x32_10((1, 2, 3, 4), (6, 6)))
    seen.add(bzo.philox4x32_10((1, 2, 3, 4), (5, 7)))
    assert len(seen) == 7


def test_uniform_is_exact_and_open():
    # 52-bit integer + 1/2, times 2^-52: endpoints and one interior value, in exact rational arithmetic
    assert bzo.uniform(0, 0) == 2.0 ** -53
    assert bzo.uniform(0xFFFFFFFF, 0xFFFFFFFF) == 1.0 - 2.0 ** -53
    a, b = 0x9E3779B9, 0x12345678
    m = ((a >> 6) << 26) | (b >> 6)
    assert bzo.uniform(a, b) == (2 * m + 1) / 2.0 ** 53        # exact: numerator < 2^53
    # the low 6 bits of each word are dropped
    assert bzo.uniform(a | 0x3F, b | 0x3F) == bzo.uniform(a & ~0x3F, b & ~0x3F)


def _samples(n_cells=40, Ns=2000):
    o = bzo.Oracle(np_=8, pmin=-3.0, pmax=3.0, species=(0,), samples=Ns, seed=11)
    out = []
    for pc in range(100, 100 + n_cells):
        for smp in range(Ns):
            s = o.sample_one(3, 0, pc, smp)
            if s.attempts > 0:
                out.append((s.nhat[0], s.nhat[1], s.nhat[2], s.t / s.s, s.attempts))
    return np.array(out)


def test_P2_isotropy_and_acceptance():
    a = _samples()
    N = len(a)
    assert N > 70000
    n = a[:, :3]
    assert np.allclose(np.sum(n * n, axis=1), 1.0, atol=1e-14)
    # <n_c> = 0, <n_c n_d> = delta_cd / 3, each within 4 sigma
    for c in range(3):
        assert abs(n[:, c].mean()) < 4.0 * math.sqrt(1.0 / 3.0 / N)
        for d in range(3):
            m = (n[:, c] * n[:, d]).mean()
            target = 1.0 / 3.0 if c == d else 0.0
            var = (1.0 / 5.0 - 1.0 / 9.0) if c == d else 1.0 / 15.0
            assert abs(m - target) < 4.0 * math.sqrt(var / N)
    # each component of a uniform unit vector is uniform on [-1, 1] (Archimedes)
    for c in range(3):
        assert stats.kstest(0.5 * (n[:, c] + 1.0), "uniform").pvalue > 1e-4
    # t/s = -(1 - cos theta*)/2 is uniform on [-1, 0] for an isotropic CM direction
    ts = a[:, 3]
    assert abs(ts.mean() + 0.5) < 4.0 * math.sqrt(1.0 / 12.0 / N)
    assert stats.kstest(-ts, "uniform").pvalue > 1e-4
    # Marsaglia acceptance pi/4 per attempt -> mean number of attempts 4/pi
    att = a[:, 4]
    p = math.pi / 4.0
    assert abs(att.mean() - 1.0 / p) < 4.0 * math.sqrt((1.0 - p) / p ** 2 / N)


def test_samples_differ_between_steps_cells_and_seeds():
    o = bzo.Oracle(np_=6, species=(0,), samples=8, seed=0)
    c0, _ = o.debug_samples(0, 0, 0, o.Np)
    c1, _ = o.debug_samples(1, 0, 0, o.Np)
    assert (c0[..., 0] != c1[..., 0]).mean() > 0.9
    o.set_seed(1)
    c2, _ = o.debug_samples(0, 0, 0, o.Np)
    assert (c0[..., 0] != c2[..., 0]).mean() > 0.9
    # p2 cells are uniform over the box: chi^2 over the cells
    o2 = bzo.Oracle(np_=4, species=(0,), samples=4000, seed=5)
    cj, _ = o2.debug_samples(0, 0, 0, 8)
    counts = np.bincount(cj[..., 0].reshape(-1), minlength=64)
    assert stats.chisquare(counts).pvalue > 1e-4
