"""Pins of the oracle's NEXT-rank-1 functions: the paper's own collision path -- integration variables
(k1x, k1y, k3x, k3y, k3z), k1z from the roots of E1 + E2 = E3 + Ep, weight 1/|J| (Eq. 17-21), massive
dispersion E^a = sqrt(p^2 + m_a^2) -- against what the paper and the mathematics fix:
  R1  every root conserves energy and momentum, is on shell, has the Jacobian of Eq. 19 (checked against a numerical
      derivative) and Mandelstam variables equal to the four-vector definitions, s + t + u = sum of the masses^2;
  R2  the roots are ALL the roots: a brute-force scan of E1(z) + E2(z) - Et over z finds the same ones;
  R3  Eq. 22-23: the four deposits cancel, total particle number is conserved to rounding, massive or not;
  R4  massless limit: the paper's sampler and the centre-of-mass sampler of the hot path are two parametrisations of
      the same integral (Eq. 5) and agree within Monte Carlo error (g g -> g g shell averages; species numbers of the
      number-changing channels of the 7-species mixture).
"""
import math

import numpy as np
import pytest

from oracle import bzo

SP7 = (0, 1, 2, 3, 4, 5, 6)
TUPLES = [(0.0, 0.0, 0.0, 0.0), (0.5, 0.5, 0.5, 0.5), (0.3, 0.9, 0.3, 0.9), (0.9, 0.3, 0.3, 0.9), (0.6, 0.6, 0.2, 0.2),
          (0.0, 0.7, 0.0, 0.7)]


def _centres(n, pmin, pmax):
    dp = (pmax - pmin) / n
    c = pmin + (np.arange(n) + 0.5) * dp
    pz, py, px = np.meshgrid(c, c, c, indexing="ij")
    return px.reshape(-1), py.reshape(-1), pz.reshape(-1)


def test_R1_roots_are_on_shell_conserve_energy_and_have_eq19_jacobian():
    n, pmin, pmax = 6, -3.0, 3.0
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=8)
    px, py, pz = _centres(n, pmin, pmax)
    dp = (pmax - pmin) / n
    seen = 0
    for msq in TUPLES:
        for pcell in (0, 37, 100, 215):
            p = np.array([px[pcell], py[pcell], pz[pcell]])
            for smp in range(400):
                k3, i3, roots = o.paper_sample(3, 0, pcell, smp, msq)
                k3 = np.array(k3)
                assert np.all((k3 >= pmin) & (k3 < pmax)) and i3 >= 0
                for R in roots:
                    seen += 1
                    k1, k2 = np.array(R.k1[:]), np.array(R.k2[:])
                    assert np.abs(k1 + k2 - k3 - p).max() <= 1e-14 * 6                    # k2 = k3 + p - k1 (Eq. 17)
                    E1, E2 = math.sqrt(k1 @ k1 + msq[0]), math.sqrt(k2 @ k2 + msq[1])
                    E3, Ep = math.sqrt(k3 @ k3 + msq[2]), math.sqrt(p @ p + msq[3])
                    for got, want in ((R.E1, E1), (R.E2, E2), (R.E3, E3), (R.Ep, Ep)):
                        assert got == pytest.approx(want, rel=1e-14)
                    assert abs((E1 + E2) - (E3 + Ep)) <= 1e-11 * (E3 + Ep)                # the root solves Eq. 18
                    # Eq. 19 against a central difference of E1(z) + E2(z) at fixed k1x, k1y, k3, p
                    h = 1e-6
                    def esum(z):
                        a = math.sqrt(k1[0] ** 2 + k1[1] ** 2 + z * z + msq[0])
                        q = k3 + p - np.array([k1[0], k1[1], z])
                        return a + math.sqrt(q @ q + msq[1])
                    assert R.J == pytest.approx((esum(k1[2] + h) - esum(k1[2] - h)) / (2 * h), rel=1e-6, abs=1e-8)
                    # massive Mandelstam variables from the four-vectors
                    s = (E1 + E2) ** 2 - (k1 + k2) @ (k1 + k2)
                    t = (E1 - E3) ** 2 - (k1 - k3) @ (k1 - k3)
                    u = (E1 - Ep) ** 2 - (k1 - p) @ (k1 - p)
                    assert R.s == pytest.approx(s, rel=1e-11, abs=1e-12)
                    assert R.t == pytest.approx(t, rel=1e-10, abs=1e-11)
                    assert R.u == pytest.approx(u, rel=1e-10, abs=1e-11)
                    assert R.s + R.t + R.u == pytest.approx(sum(msq), abs=1e-10 * max(1.0, R.s))
                    # cells
                    for k, cell in ((k1, R.i1), (k2, R.i2)):
                        q = np.floor((k - pmin) / dp).astype(int)
                        assert np.all((q >= 0) & (q < n)) and cell == q[0] + n * (q[1] + n * q[2])
    assert seen > 1500


def test_R2_brute_force_scan_finds_the_same_roots():
    n, pmin, pmax = 6, -3.0, 3.0
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=8)
    px, py, pz = _centres(n, pmin, pmax)
    zs = np.linspace(pmin, pmax, 60001)
    compared = 0
    for msq in TUPLES:
        for pcell in (5, 111, 190):
            p = np.array([px[pcell], py[pcell], pz[pcell]])
            for smp in range(60):
                k3, _, roots = o.paper_sample(1, 0, pcell, smp, msq)
                k3 = np.array(k3)
                if not roots:                                          # (k1x, k1y) come back with a root only
                    continue
                k1x, k1y = roots[0].k1[0], roots[0].k1[1]
                Et = math.sqrt(k3 @ k3 + msq[2]) + math.sqrt(p @ p + msq[3])
                P = k3 + p
                g = (np.sqrt(k1x ** 2 + k1y ** 2 + zs ** 2 + msq[0]) +
                     np.sqrt((P[0] - k1x) ** 2 + (P[1] - k1y) ** 2 + (P[2] - zs) ** 2 + msq[1]) - Et)
                sign_change = np.nonzero(np.sign(g[:-1]) * np.sign(g[1:]) < 0)[0]
                scan = []
                for i in sign_change:                                  # linear interpolation of the crossing
                    z = zs[i] - g[i] * (zs[i + 1] - zs[i]) / (g[i + 1] - g[i])
                    k2 = P - np.array([k1x, k1y, z])
                    if np.all((k2 >= pmin) & (k2 < pmax)):
                        scan.append(z)
                mine = sorted(R.k1[2] for R in roots)
                # a root within one scan step of the box edge may be counted on either side: skip those samples
                if any(min(abs(z - pmin), abs(z - pmax)) < 2e-4 for z in mine + scan):
                    continue
                assert len(mine) == len(scan), (msq, pcell, smp, mine, scan)
                assert np.allclose(mine, sorted(scan), atol=1e-6)
                compared += len(mine)
    assert compared > 300


@pytest.mark.parametrize("massive", [False, True])
def test_R3_symmetric_deposits_conserve_particle_number(massive):
    n = 5
    o = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=SP7, samples=6, seed=2, m_D=0.0 if massive else 0.6)
    rng = np.random.default_rng(4)
    f = rng.uniform(0.02, 0.6, size=o.shape)
    o.set_f(f)
    if massive:
        o.thermal_masses()
        assert (o.get_masses() > 0).all()
    dF = o.collision_paper(0.01, 0)
    gross = o.gross()
    deg = np.array([16.0] + [6.0] * 6)[None, :, None]
    assert np.abs(dF).max() > 0
    assert abs((deg * dF).sum()) <= 1e-13 * (deg * gross).sum()
    # individual species are not conserved (g <-> q qbar)
    assert abs((deg * dF)[:, 0].sum()) > 1e-6 * (deg * gross)[:, 0].sum()


@pytest.mark.slow
def test_R4a_massless_limit_agrees_with_cm_sampler_gg():
    # the setting of pin P4: over-occupied core in a thin bath, shell averages by the cubic symmetry
    n, pmin, pmax, mD, dt = 5, -2.0, 2.0, 0.8, 0.01
    px, py, pz = _centres(n, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    f = np.where(r <= 0.85, 0.5, 0.05)[None, None, :]
    shells = [np.nonzero(np.abs(r - rr) < 1e-9)[0] for rr in (0.8, 0.8 * math.sqrt(2), 0.8 * math.sqrt(3))]
    pap = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=40000, seed=8, m_D=mD, threads=8)
    cm = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=4000, seed=9, m_D=mD, threads=8)
    pap.set_f(f)
    cm.set_f(f)
    a = np.array([pap.collision_paper(dt, b)[0, 0] for b in range(6)])
    c = np.array([cm.collision(dt, b)[0, 0] for b in range(6)])
    for sh in shells:
        am, cmn = a[:, sh].mean(axis=1), c[:, sh].mean(axis=1)
        ea, ec = am.std(ddof=1) / math.sqrt(len(am)), cmn.std(ddof=1) / math.sqrt(len(cmn))
        print("R4a shell r=%.3f: paper sampler %.5e +- %.1e   CM sampler %.5e +- %.1e" % (r[sh[0]], am.mean(), ea, cmn.mean(), ec))
        assert ea < 0.05 * abs(cmn.mean())
        # both deposit on four cells; they differ by the binning of the labelled leg (slot 4 vs slot 1 on the cell
        # centre), O(dp^2): allow 3 % beside the statistical error
        assert abs(am.mean() - cmn.mean()) < 4 * math.hypot(ea, ec) + 0.03 * abs(cmn.mean())


@pytest.mark.slow
def test_R4b_massless_limit_agrees_with_cm_sampler_number_changing_channels():
    n = 6
    px, py, pz = _centres(n, -3.0, 3.0)
    r2 = px ** 2 + py ** 2 + pz ** 2
    widths, amps = [1.6, 0.9, 1.1, 0.7, 1.3, 1.0, 0.8], [0.5, 0.30, 0.12, 0.25, 0.2, 0.15, 0.35]
    f = np.stack([A * np.exp(-r2 / w) for A, w in zip(amps, widths)])[None]
    kw = dict(np_=n, pmin=-3.0, pmax=3.0, species=SP7, m_D=0.5, threads=8)
    pap, cm = bzo.Oracle(samples=6000, seed=3, **kw), bzo.Oracle(samples=1500, seed=5, **kw)
    for o in (pap, cm):
        o.set_f(f)
        for k in ("A", "11", "1B", "QG", "GG"):
            o.set_msq_override(k, 0.0)
    deg = np.array([16.0] + [6.0] * 6)
    a = np.array([(pap.collision_paper(0.01, b)[0].sum(axis=1) * deg) for b in range(6)])
    c = np.array([(cm.collision(0.01, b)[0].sum(axis=1) * deg) for b in range(6)])
    ea, ec = a.std(0, ddof=1) / math.sqrt(6), c.std(0, ddof=1) / math.sqrt(6)
    print("R4b paper", a.mean(0), "+-", ea, "\n    CM   ", c.mean(0), "+-", ec)
    assert c.mean(0)[0] < 0 and np.all(c.mean(0)[1:] > 0)
    assert np.all(ea < 0.03 * np.abs(c.mean(0)))
    assert np.all(np.abs(a.mean(0) - c.mean(0)) < 4 * np.hypot(ea, ec) + 0.03 * np.abs(c.mean(0)))


def test_R5_full_program_step_conserves_particle_number():
    """The paper's program as a whole (bzo_set_collision(1) + bzo_set_transport(1)): masses from the old f, Eq. 17-21,
    Eq. 15, Euler.  Total particle number is conserved step after step (Eq. 13 + Eq. 22-23); the masses move with f."""
    o = bzo.Oracle(nx=2, ny=2, nz=1, dx=0.3, np_=5, pmin=-3.0, pmax=3.0, species=(0, 1, 2), samples=20, seed=6)
    rng = np.random.default_rng(8)
    o.set_f(rng.uniform(0.05, 0.5, size=o.shape))
    o.set_collision(1)
    o.set_transport(1)
    N0 = o.moments()["tot"][:, 0].sum()
    masses = []
    for _ in range(3):
        o.step(0.01)
        masses.append(o.get_masses().copy())
        assert o.moments()["tot"][:, 0].sum() == pytest.approx(N0, rel=1e-13)
    assert (masses[0] > 0).all() and not np.array_equal(masses[0], masses[2])


@pytest.mark.parametrize("masses", [None, (0.41, 0.13, 0.13, 0.13), (0.5, 0.2, 0.25, 0.3)], ids=["massless", "equal_quarks", "four_masses"])
def test_R6_grouping_by_mass_tuple_equals_the_channel_by_channel_sum(masses):
    """bzo_collision_paper solves the roots once per distinct tuple of mass classes; bzo_collision_paper_plain walks
    Eq. 3-4 as printed (sample -> channel -> that channel's own root solve -> deposit).  Same roots, same terms, another
    summation order: they agree to rounding on the scale of the gross deposit (S16), massless, with degenerate quark
    masses and with four distinct masses, on two spatial cells with different masses."""
    o = bzo.Oracle(nx=2, ny=1, nz=1, dx=0.3, np_=5, pmin=-3.0, pmax=3.0, species=SP7, samples=12, seed=9, threads=2)
    rng = np.random.Generator(np.random.Philox(key=19))
    o.set_f(0.02 + 0.5 * rng.random(o.shape))
    if masses is not None:
        o.set_masses(np.array([masses, [1.3 * m for m in masses]]))
    a = o.collision_paper(0.01, 4)
    ga = o.gross()
    b = o.collision_paper_plain(0.01, 4)
    gb = o.gross()
    assert np.abs(a).max() > 0 and np.count_nonzero(a) > 0.5 * a.size
    assert np.all(np.abs(a - b) <= 1e-13 * np.maximum(ga, np.abs(a)))
    assert np.all(np.abs(ga - gb) <= 1e-13 * ga)
