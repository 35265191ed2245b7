"""Pins of the oracle's in-box sampler ("sample p2 and n so that p3, p4 stay in the box"):
bzo_sample_one_box / bzo_collision_box.  The CM direction is drawn uniformly from the tightest of the three zones
|a_c . n| <= beta_c of the sphere outside which p3 or p4 leaves the momentum box, and the deposit carries the zone's
area fraction beta as its weight (Archimedes' hat-box theorem), so that Eq. 20's expectation is unchanged.
  B1  every sample conserves energy and momentum with massless legs (as P1), its direction is a unit vector inside the
      zone, and the weight is the closed form min_c min(1, (L/2 - |P_c/2 - centre|) / (sqrt(s + P_c^2)/2)) recomputed here
      from the sample's p1, p2 alone;
  B2  the zone contains EVERY accepted direction: uniform directions on the whole sphere that keep p3 and p4 in the box
      all satisfy |a . n| <= beta for the zone the sampler chose (brute force, also on an off-centre box);
  B3  the weighted in-box sample reproduces the accepted part of the isotropic measure: for fixed (p1, p2),
      beta <1_acc h(n)>_zone = <1_acc h(n)>_sphere for h = 1, n_c, n_c n_d, t/s (the oracle's own uniform sampler on
      the right-hand side, 4 sigma);
  B4  Eq. 22-23: exact particle-number conservation;
  B5  same expectation as bzo_collision (shell averages of g g -> g g and the number-changing channels of the mixture,
      4 sigma); at equal numbers of generated samples its variance is 0.91 of the uniform sampler's (acceptance 0.78
      against 0.46: the rejected samples of the uniform sampler are zeros, which cost little variance).
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


def _zone(p1, p2, pmin, pmax):
    """The three zones from p1, p2 alone: unit vectors a_c, half-widths beta_c (numpy, independent of the oracle)."""
    E1, E2 = np.linalg.norm(p1), np.linalg.norm(p2)
    s = 2 * (E1 * E2 - p1 @ p2)
    P, E, M = p1 + p2, E1 + E2, math.sqrt(s)
    B, c0 = 0.5 * (pmax - pmin), 0.5 * (pmax + pmin)
    A = 0.5 * (M * np.eye(3) + np.outer(P, P) / (E + M))          # p3 = P/2 + A n  (S8c step 2)
    An = np.linalg.norm(A, axis=1)
    assert np.allclose(An, 0.5 * np.sqrt(s + P * P), rtol=1e-12)   # |A_c| = sqrt(s + P_c^2)/2
    beta = np.minimum(1.0, (B - np.abs(0.5 * P - c0)) / An)
    return A / An[:, None], beta, (P, E, M, s)


@pytest.mark.parametrize("box", [(-3.0, 3.0), (-1.0, 4.0)], ids=["centred", "off_centre"])
def test_B1_kinematics_zone_and_weight(box):
    pmin, pmax = box
    n = 8
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=8)
    n_ok, n_acc, n_tight = 0, 0, 0
    for pcell in (3, 77, 300, 511, 219):
        for smp in range(600):
            sm, w = o.sample_one_box(2, 0, pcell, smp)
            if not (sm.s > 0):
                assert w == 0.0 and sm.flag == 0
                continue
            p1, p2, p3, p4 = (np.array(v[:]) for v in (sm.p1, sm.p2, sm.p3, sm.p4))
            E3, E4 = np.linalg.norm(p3), np.linalg.norm(p4)
            assert np.abs(p1 + p2 - p3 - p4).max() <= 1e-14 * 16
            assert abs(sm.E1 + sm.E2 - E3 - E4) <= 1e-13 * (sm.E1 + sm.E2)
            assert sm.E3 == pytest.approx(E3, rel=1e-12)
            assert sm.s + sm.t + sm.u == pytest.approx(0.0, abs=1e-12 * sm.s)
            assert sm.t == pytest.approx(-2 * (sm.E1 * E3 - p1 @ p3), rel=1e-9, abs=1e-13)
            nh = np.array(sm.nhat[:])
            assert np.linalg.norm(nh) == pytest.approx(1.0, rel=1e-12)
            a, beta, _ = _zone(p1, p2, pmin, pmax)
            c = int(np.argmin(beta))
            assert w == pytest.approx(beta[c], rel=1e-12)
            assert abs(a[c] @ nh) <= beta[c] * (1 + 1e-12)                          # the direction lies in the zone
            inside = bool(np.all((p3 >= pmin) & (p3 < pmax) & (p4 >= pmin) & (p4 < pmax)))
            assert bool(sm.flag) == inside
            if beta[c] < 1.0:
                # the zone's own axis can never reject: that is the point of sampling it exactly
                assert pmin - 1e-12 <= p3[c] <= pmax + 1e-12 and pmin - 1e-12 <= p4[c] <= pmax + 1e-12
                n_tight += 1
            n_ok += 1
            n_acc += sm.flag
    assert n_ok > 2500 and n_tight > 1000
    assert n_acc / n_ok > 0.7                                                       # 0.46 with the uniform direction


@pytest.mark.parametrize("box", [(-3.0, 3.0), (-1.0, 4.0)], ids=["centred", "off_centre"])
def test_B2_zone_contains_every_accepted_direction(box):
    pmin, pmax = box
    rng = np.random.default_rng(5)
    px, py, pz = _centres(8, pmin, pmax)
    checked = 0
    for trial in range(300):
        pc = int(rng.integers(0, 512))
        p1 = np.array([px[pc], py[pc], pz[pc]])
        p2 = rng.uniform(pmin, pmax, 3)
        a, beta, (P, E, M, s) = _zone(p1, p2, pmin, pmax)
        if not s > 0:
            continue
        c = int(np.argmin(beta))
        v = rng.normal(size=(4000, 3))
        nh = v / np.linalg.norm(v, axis=1)[:, None]
        cc = nh @ P
        p3 = 0.5 * (M * nh + P[None, :] * (1 + cc / (E + M))[:, None])
        p4 = P[None, :] - p3
        acc = np.all((p3 >= pmin) & (p3 < pmax) & (p4 >= pmin) & (p4 < pmax), axis=1)
        assert np.all(np.abs(nh[acc] @ a[c]) <= beta[c] + 1e-12)
        # and the zone is exactly the per-axis condition: inside the zone <=> axis c keeps both legs in
        inz = np.abs(nh @ a[c]) <= beta[c]
        ok_c = (p3[:, c] >= pmin) & (p3[:, c] < pmax) & (p4[:, c] >= pmin) & (p4[:, c] < pmax)
        assert np.mean(inz == ok_c) > 0.999
        checked += int(acc.sum())
    assert checked > 100000


def test_B3_weighted_sample_reproduces_the_accepted_isotropic_measure():
    """For fixed (p1, p2) the two samplers differ only in how they use the Marsaglia draws.  Compared over MANY (p1, p2) at
    once: the sums of w 1_acc h(n) (in-box) and of 1_acc h(n) (uniform) over the same set of (cell, sample) pairs with
    different seeds agree within 4 sigma for h = 1, n_x, n_y, n_z, n_x n_y, n_z^2, t/s."""
    n = 8
    kw = dict(np_=n, pmin=-3.0, pmax=3.0, species=(0,), samples=8)

    def stats(seed, box):
        o = bzo.Oracle(seed=seed, **kw)
        rows = []
        for pcell in (0, 7, 77, 219, 300, 448, 511):                  # corners and faces: tight zones
            for smp in range(6000):
                if box:
                    sm, w = o.sample_one_box(1, 0, pcell, smp)
                else:
                    sm, w = o.sample_one(1, 0, pcell, smp), 1.0
                if not sm.flag:
                    rows.append(np.zeros(7))
                    continue
                nh = np.array(sm.nhat[:])
                rows.append(w * np.array([1.0, nh[0], nh[1], nh[2], nh[0] * nh[1], nh[2] ** 2, sm.t / sm.s]))
        r = np.array(rows)
        return r.mean(0), r.std(0, ddof=1) / math.sqrt(len(r)), float((r[:, 0] > 0).mean())

    mb, eb, acc_b = stats(11, True)
    mu, eu, acc_u = stats(12, False)
    print("B3 in-box ", mb, "+-", eb, "acceptance", acc_b, "\n   uniform", mu, "+-", eu, "acceptance", acc_u)
    assert np.all(np.abs(mb - mu) <= 4 * np.hypot(eb, eu))
    assert acc_b > 1.4 * acc_u                                         # corner cells: far more samples survive
    assert np.all(eb[[0, 5, 6]] < eu[[0, 5, 6]])                       # and the weighted estimate is the sharper one


def test_B4_exact_particle_number_conservation():
    sp = (0, 1, 2, 3, 4, 5, 6)
    o = bzo.Oracle(np_=6, pmin=-3.0, pmax=3.0, species=sp, samples=30, seed=4, threads=4)
    rng = np.random.Generator(np.random.Philox(key=3))
    o.set_f(0.02 + 0.5 * rng.random(o.shape))
    dF = o.collision_box(0.01, 7)
    gross = o.gross()
    deg = np.array([16.0] + [6.0] * 6)[None, :, None]
    assert np.abs(dF).max() > 0
    assert abs((deg * dF).sum()) <= 1e-13 * (deg * gross).sum()
    # through bzo_step with bzo_set_collision(3)
    o.set_collision(3)
    N0 = o.moments()["tot"][:, 0].sum()
    for _ in range(2):
        o.step(0.01)
    assert o.moments()["tot"][:, 0].sum() == pytest.approx(N0, rel=1e-13)


@pytest.mark.slow
def test_B5_same_expectation_as_the_uniform_sampler_and_smaller_spread():
    n = 6
    px, py, pz = _centres(n, -3.0, 3.0)
    pabs = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    shells = [pabs < 1.0, (pabs >= 1.0) & (pabs < 2.0), (pabs >= 2.0) & (pabs < 3.0), pabs >= 3.0]
    # glue, broad f: a large part of the phase space sits near the faces of the box
    f = (0.6 * np.exp(-(pabs / 2.2) ** 2))[None, None, :]
    kw = dict(np_=n, pmin=-3.0, pmax=3.0, species=(0,), m_D=0.6, threads=8, samples=400)
    batches = 40
    res = {}
    for name, seed in (("box", 21), ("uni", 22)):
        o = bzo.Oracle(seed=seed, **kw)
        o.set_f(f)
        res[name] = np.array([(o.collision_box if name == "box" else o.collision)(0.01, b)[0, 0] for b in range(batches)])
    sh = {k: np.array([[d[m].sum() for m in shells] for d in r]) for k, r in res.items()}
    mb, mu = sh["box"].mean(0), sh["uni"].mean(0)
    eb, eu = sh["box"].std(0, ddof=1) / math.sqrt(batches), sh["uni"].std(0, ddof=1) / math.sqrt(batches)
    print("B5 in-box ", mb, "+-", eb, "\n   uniform", mu, "+-", eu)
    assert np.all(np.abs(mb - mu) <= 4 * np.hypot(eb, eu))
    assert np.all(np.abs(mu) > 3 * eu)                                  # the comparison resolves the signal
    # Equal number of GENERATED samples: per-cell variances over the batches, summed over the cells.  The ratio is the
    # "samples to equal variance" of the in-box sampler.  Measured 0.91 (0.78 on the cells with |p| >= 3 GeV): the samples
    # the uniform direction throws away are zeros, and zeros are not where the variance comes from -- the in-box sampler
    # turns them into deposits with small weights beta.  It must not be WORSE than the uniform sampler, and it is not a
    # large gain either (DESIGN.md 10 draws the consequence for the GPU path).
    vb, vu = res["box"].var(0, ddof=1), res["uni"].var(0, ddof=1)
    ratio, ratio_hi = vb.sum() / vu.sum(), vb[shells[3]].sum() / vu[shells[3]].sum()
    print("B5 variance ratio in-box / uniform: all cells %.3f, |p| >= 3 GeV %.3f" % (ratio, ratio_hi))
    assert 0.7 < ratio < 1.0 and ratio_hi < 0.9
    # number-changing channels of the mixture: species numbers agree
    sp = (0, 1, 2, 3, 4, 5, 6)
    r2 = px ** 2 + py ** 2 + pz ** 2
    widths, amps = [3.0, 1.9, 2.1, 1.7, 2.3, 2.0, 1.8], [0.5, 0.30, 0.12, 0.25, 0.2, 0.15, 0.35]
    fm = np.stack([A * np.exp(-r2 / w) for A, w in zip(amps, widths)])[None]
    kwm = dict(np_=n, pmin=-3.0, pmax=3.0, species=sp, m_D=0.5, threads=8, samples=300)
    deg = np.array([16.0] + [6.0] * 6)
    out = {}
    for name, seed in (("box", 31), ("uni", 32)):
        o = bzo.Oracle(seed=seed, **kwm)
        o.set_f(fm)
        for k in ("A", "11", "1B", "QG", "GG"):
            o.set_msq_override(k, 0.0)
        a = np.array([((o.collision_box if name == "box" else o.collision)(0.01, b)[0].sum(axis=1) * deg) for b in range(8)])
        out[name] = (a.mean(0), a.std(0, ddof=1) / math.sqrt(8))
    (ab, eab), (au, eau) = out["box"], out["uni"]
    print("B5 mixture in-box", ab, "+-", eab, "\n           uniform", au, "+-", eau)
    assert np.all(np.abs(ab - au) <= 4 * np.hypot(eab, eau) + 0.01 * np.abs(au))
