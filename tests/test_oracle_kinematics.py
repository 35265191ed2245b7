"""Pin P1: invariants of the kinematic sample and of the binning (step 3)."""
import numpy as np

from oracle import bzo


def _norm(v):
    return float(np.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2))


def test_P1_energy_momentum_and_mandelstam():
    n = 9                                           # odd: has the p = 0 cell
    o = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=(0,), samples=40, seed=3)
    dp = 6.0 / n
    seen_flag = seen_rej = 0
    for pc in range(0, o.Np, 7):
        for smp in range(40):
            s = o.sample_one(2, 0, pc, smp)
            p1, p2, p3, p4 = (np.array(x[:]) for x in (s.p1, s.p2, s.p3, s.p4))
            # p1 is the cell centre, p2 lies in the box and in its cell
            idx = np.array([pc % n, (pc // n) % n, pc // (n * n)])
            assert np.allclose(p1, -3.0 + (idx + 0.5) * dp, atol=1e-15)
            assert np.all(p2 > -3.0) and np.all(p2 < 3.0)
            j = np.floor((p2 + 3.0) / dp).astype(int)
            assert s.j == j[0] + n * (j[1] + n * j[2])
            assert abs(s.E1 - _norm(p1)) <= 1e-15 * 6 and abs(s.E2 - _norm(p2)) <= 1e-15 * 6
            if s.attempts == 0:                    # !(s > 0): only the p = 0 cell in practice
                assert s.flag == 0 and s.k == -1 and s.l == -1
                assert _norm(p1) == 0.0
                continue
            E = s.E1 + s.E2
            scale = E
            assert np.allclose(p1 + p2, p3 + p4, atol=1e-13 * scale)           # momentum conservation
            E4 = E - s.E3
            assert abs(_norm(p3) - s.E3) <= 1e-13 * scale                        # massless outgoing legs
            assert abs(_norm(p4) - E4) <= 1e-13 * scale
            assert abs(s.s + s.t + s.u) <= 1e-13 * s.s                           # s + t + u = 0
            assert -s.s * (1 + 1e-13) <= s.t <= 1e-13 * s.s                      # -s <= t <= 0
            # s, t, u from the four-vectors
            assert abs(s.s - (E ** 2 - _norm(p1 + p2) ** 2)) <= 1e-12 * scale ** 2
            assert abs(s.t - ((s.E1 - s.E3) ** 2 - _norm(p1 - p3) ** 2)) <= 1e-12 * scale ** 2
            assert abs(s.u - ((s.E1 - E4) ** 2 - _norm(p1 - p4) ** 2)) <= 1e-12 * scale ** 2
            # binning and rejection (S9)
            for p, cell in ((p3, s.k), (p4, s.l)):
                inside = np.all(p >= -3.0) and np.all(p < 3.0)
                if inside:
                    q = np.floor((p + 3.0) / dp).astype(int)
                    assert cell == q[0] + n * (q[1] + n * q[2])
                else:
                    assert cell == -1
            assert s.flag == int(s.k >= 0 and s.l >= 0)
            seen_flag += s.flag
            seen_rej += 1 - s.flag
    assert seen_flag > 500 and seen_rej > 500


def test_debug_samples_agree_with_sample_one():
    o = bzo.Oracle(np_=6, species=(0, 1, 2), samples=16, seed=9)
    cells, stu = o.debug_samples(5, 0, 10, 20)
    for a, pc in enumerate(range(10, 20)):
        for smp in range(16):
            s = o.sample_one(5, 0, pc, smp)
            assert tuple(cells[a, smp]) == (s.j, s.k, s.l, s.flag)
            assert tuple(stu[a, smp]) == (s.s, s.t, s.u)


def test_kinematics_do_not_depend_on_species_or_f():
    a = bzo.Oracle(np_=6, species=(0,), samples=16, seed=9)
    b = bzo.Oracle(np_=6, species=(1, 2, 5), samples=16, seed=9)
    b.set_f(np.full(b.shape, 0.3))
    ca, sa = a.debug_samples(1, 0, 0, a.Np)
    cb, sb = b.debug_samples(1, 0, 0, b.Np)
    assert np.array_equal(ca, cb) and np.array_equal(sa, sb)


def test_acceptance_fraction_uniform_box():
    # S9 / probe chk3: for p1, p2 uniform over the box about 46 % of the samples keep both outgoing legs inside
    o = bzo.Oracle(np_=12, species=(0,), samples=32, seed=2)
    cells, _ = o.debug_samples(0, 0, 0, o.Np)
    frac = cells[..., 3].mean()
    assert 0.40 < frac < 0.52


def test_sample_one_honours_the_slab_offset_like_debug_samples():
    """bzo_set_slab: local cell x draws the samples of global cell x + offset in every entry point that samples (S8e: the Philox
    spatial counter is the cell's index in the undecomposed domain) -- bzo_sample_one included."""
    kw = dict(np_=8, pmin=-3.0, pmax=3.0, species=(0,), seed=5, samples=6)
    whole = bzo.Oracle(nx=1, ny=1, nz=4, **kw)
    part = bzo.Oracle(nx=1, ny=1, nz=2, **kw)
    part.set_slab(2, 0, 2)                                   # local cells 0, 1 = global cells 2, 3
    cells_w, stu_w = whole.debug_samples(3, 3, 100, 104)
    cells_p, stu_p = part.debug_samples(3, 1, 100, 104)
    assert np.array_equal(cells_w, cells_p) and np.array_equal(stu_w.view(np.uint64), stu_p.view(np.uint64))
    for k, pc in enumerate(range(100, 104)):
        for smp in range(6):
            a, b = whole.sample_one(3, 3, pc, smp), part.sample_one(3, 1, pc, smp)
            assert (a.j, a.k, a.l, a.flag) == (b.j, b.k, b.l, b.flag) == tuple(cells_w[k, smp])
            assert (a.s, a.t, a.u) == (b.s, b.t, b.u)
    c = whole.sample_one(3, 1, 100, 0)
    assert (c.s, c.t, c.u) != (part.sample_one(3, 1, 100, 0).s, part.sample_one(3, 1, 100, 0).t, part.sample_one(3, 1, 100, 0).u)
