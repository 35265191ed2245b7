"""Pins of the oracle's NEXT-rank-3 functions: importance sampling of the t/u-channel peaks of Table I.
  I1  every sample conserves energy and momentum with massless legs, and the momentum transfer of the constructed
      momenta is the t that was drawn: the weight equals (1/s)/p(t) evaluated at the t of the four-vectors;
  I2  the weighted sample reproduces the isotropic measure of the hot path: <w> = 1, <w n> = 0, <w n_c n_d> = delta/3,
      <w t/s> = -1/2, and without a regulator the weights are 1;
  I3  Eq. 22-23: exact particle-number conservation;
  I4  same expectation as the uniform estimator (shell averages, g g -> g g) with a smaller spread when m^2 << s.
"""
import math

import numpy as np
import pytest

from oracle import bzo


def _centres(n, pmin, pmax):
    dp = (pmax - pmin) / n
    c = pmin + (np.arange(n) + 0.5) * dp
    pz, py, px = np.meshgrid(c, c, c, indexing="ij")
    return px.reshape(-1), py.reshape(-1), pz.reshape(-1)


def test_I1_kinematics_and_weight():
    o = bzo.Oracle(np_=8, pmin=-3.0, pmax=3.0, species=(0,), samples=8)
    m2 = 0.09
    n_ok = 0
    for pcell in (3, 77, 300, 511):
        for smp in range(500):
            sm, w = o.sample_one_is(2, 0, pcell, smp, m2)
            if not (sm.s > 0):
                continue
            p1, p2, p3, p4 = (np.array(v[:]) for v in (sm.p1, sm.p2, sm.p3, sm.p4))
            E3, E4 = np.linalg.norm(p3), np.linalg.norm(p4)
            assert np.abs(p1 + p2 - p3 - p4).max() <= 1e-14 * 12
            assert abs(sm.E1 + sm.E2 - E3 - E4) <= 1e-13 * (sm.E1 + sm.E2)        # massless outgoing legs on shell
            assert sm.E3 == pytest.approx(E3, rel=1e-12)
            assert -sm.s * (1 + 1e-12) <= sm.t <= sm.s * 1e-12
            assert sm.s + sm.t + sm.u == pytest.approx(0.0, abs=1e-12 * sm.s)
            t4 = -2 * (sm.E1 * E3 - p1 @ p3)
            assert sm.t == pytest.approx(t4, rel=1e-9, abs=1e-13)
            # the weight is (1/s) / p(t) at the t of the four-vectors: the construction realises the drawn t
            norm = 1 / m2 - 1 / (sm.s + m2)
            pt = 0.5 * (1 / ((m2 - sm.t) ** 2 * norm) + 1 / ((m2 - sm.u) ** 2 * norm))
            assert w == pytest.approx((1 / sm.s) / pt, rel=1e-7)
            assert np.linalg.norm(np.array(sm.nhat[:])) == pytest.approx(1.0, rel=1e-12)
            n_ok += 1
    assert n_ok > 1500


def test_I2_weighted_sample_is_isotropic():
    o = bzo.Oracle(np_=8, pmin=-3.0, pmax=3.0, species=(0,), samples=8)
    for m2 in (0.04, 1.0):
        W, N1, N2, TS = [], [], [], []
        for pcell in (77, 300):
            for smp in range(40000):
                sm, w = o.sample_one_is(5, 0, pcell, smp, m2)
                if not (sm.s > 0):
                    continue
                nh = np.array(sm.nhat[:])
                W.append(w)
                N1.append(w * nh)
                N2.append(w * np.outer(nh, nh).reshape(-1))
                TS.append(w * sm.t / sm.s)
        W, N1, N2, TS = np.array(W), np.array(N1), np.array(N2), np.array(TS)
        n = len(W)
        assert abs(W.mean() - 1) < 4 * W.std() / math.sqrt(n)
        assert np.all(np.abs(N1.mean(0)) < 4 * N1.std(0) / math.sqrt(n))
        assert np.all(np.abs(N2.mean(0) - np.eye(3).reshape(-1) / 3) < 4 * N2.std(0) / math.sqrt(n))
        assert abs(TS.mean() + 0.5) < 4 * TS.std() / math.sqrt(n)
        # the proposal does what it is for: most samples sit at small |t| or small |u|
    sm, w = o.sample_one_is(5, 0, 77, 0, 0.0)
    assert w == 1.0                                           # no regulator: uniform t, weight 1


def test_I3_exact_conservation():
    o = bzo.Oracle(np_=6, pmin=-3.0, pmax=3.0, species=(0, 1, 2, 3, 4, 5, 6), samples=12, seed=3)
    rng = np.random.default_rng(1)
    o.set_f(rng.uniform(0.02, 0.6, size=o.shape))
    dF = o.collision_is(0.01, 0)
    gross = o.gross()
    deg = np.array([16.0] + [6.0] * 6)[None, :, None]
    assert np.abs(dF).max() > 0
    assert abs((deg * dF).sum()) <= 1e-13 * (deg * gross).sum()


@pytest.mark.slow
def test_I4_same_expectation_smaller_variance():
    n, pmin, pmax, dt = 5, -2.0, 2.0, 0.01
    px, py, pz = _centres(n, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    f = np.where(r <= 0.85, 0.5, 0.05)[None, None, :]
    shells = [np.nonzero(np.abs(r - rr) < 1e-9)[0] for rr in (0.8, 0.8 * math.sqrt(2), 0.8 * math.sqrt(3))]
    ratios = {}
    for mD in (0.25, 0.8):
        kw = dict(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=3000, m_D=mD, threads=8)
        a_, b_ = bzo.Oracle(seed=8, **kw), bzo.Oracle(seed=9, **kw)
        a_.set_f(f)
        b_.set_f(f)
        A = np.array([a_.collision_is(dt, b)[0, 0] for b in range(10)])
        B = np.array([b_.collision(dt, b)[0, 0] for b in range(10)])
        for sh in shells:
            am, bm = A[:, sh].mean(axis=1), B[:, sh].mean(axis=1)
            ea, eb = am.std(ddof=1) / math.sqrt(len(am)), bm.std(ddof=1) / math.sqrt(len(bm))
            print("I4 m_D=%.2f shell r=%.3f: IS %.5e +- %.1e   uniform %.5e +- %.1e" % (mD, r[sh[0]], am.mean(), ea, bm.mean(), eb))
            assert abs(am.mean() - bm.mean()) < 4 * math.hypot(ea, eb)
        ratios[mD] = A.std(axis=0, ddof=1).mean() / B.std(axis=0, ddof=1).mean()
    print("I4 spread ratio IS/uniform:", ratios)
    assert ratios[0.25] < 0.8                                  # peaked regime: importance sampling pays
