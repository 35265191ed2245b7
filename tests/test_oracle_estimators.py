"""Pins P4, P5, P6, P9, P10, P3b of SURVEY.md 8c: the normalisation, channel bookkeeping and conservation of the
Monte Carlo estimator (Eq. 3-5, 20-23 of the paper), checked against things the oracle does not contain:
  P10  the closed-form loss rate that Eq. 4-5 give for a constant matrix element;
  P4   an independent numpy Monte Carlo of Eq. 5 in the PAPER'S OWN parametrisation (Eq. 17-21: k2 eliminated,
       k1z from the two roots of energy conservation, weight 1/|J|), with Table I's gg->gg typed here;
  P5   the labelled estimator (only the grid point itself, weight 1/2 x orderings) against the symmetric one (1/8);
  P6   exact particle-number conservation; P9 the direction of g -> q qbar conversion; P3b binned equilibrium.
"""
import math

import numpy as np
import pytest

from oracle import bzo

HBARC = 0.1973269804
SP7 = (0, 1, 2, 3, 4, 5, 6)
NDEG = np.array([16.0] + [6.0] * 6)


def _centres(n, pmin, pmax):
    dp = (pmax - pmin) / n
    c = pmin + (np.arange(n) + 0.5) * dp
    pz, py, px = np.meshgrid(c, c, c, indexing="ij")
    return px.reshape(-1), py.reshape(-1), pz.reshape(-1)


def _inv_r_over_cube(cx, cy, cz, h, m=24):
    """integral of 1/|p| over the cube of half-width h centred at (cx,cy,cz): Gauss-Legendre on 8 sub-cubes split at
    the centre (so a cube containing the origin has its singular point on sub-cube corners)."""
    x, w = np.polynomial.legendre.leggauss(m)

    def nodes(c):
        lo = c - h + 0.5 * h * (x + 1)
        hi = c + 0.5 * h * (x + 1)
        return np.concatenate([lo, hi]), np.concatenate([w, w]) * 0.5 * h

    X, WX = nodes(cx)
    Y, WY = nodes(cy)
    Z, WZ = nodes(cz)
    R = np.sqrt(X[:, None, None] ** 2 + Y[None, :, None] ** 2 + Z[None, None, :] ** 2)
    return float(np.sum(WX[:, None, None] * WY[None, :, None] * WZ[None, None, :] / R))


def test_inv_r_quadrature_helper():
    # closed form: integral of 1/r over the unit cube [0,1]^3 = -pi/4 + (3/2) ln(2 + sqrt 3); [-1,1]^3 is 8 octants
    unit = -math.pi / 4 + 1.5 * math.log(2 + math.sqrt(3))
    assert _inv_r_over_cube(0.0, 0.0, 0.0, 1.0) == pytest.approx(8 * unit, rel=2e-3)
    assert _inv_r_over_cube(3.0, 0.0, 0.0, 0.5) == pytest.approx(1.0 / 3.0, rel=2e-2)


def test_P10_constant_matrix_element_closed_form():
    # |M|^2 == 1 for g g <-> q qbar only, quarks empty: Eq. 4-5 give for the gluon at the grid point p1
    #   N_g df_g/dt = - (1/2E1) Int d^3p2/((2pi)^3 2E2) (1/8pi) f_g(p1) f_g(p2) = - f1 Int d^3p2 f2/|p2| / (256 pi^4 E1)
    # (final state q qbar: two distinct particles, factor 1; nothing is rejected because E1 + E2 < pmax).
    n, pmin, pmax, Q, c0, dt, Ns = 9, -3.0, 3.0, 1.0, 0.2, 0.01, 40000
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0, 1, 2), samples=Ns, seed=4, m_D=0.7)
    for kind in bzo.KINDS:
        o.set_msq_override(kind, 1.0 if kind == "QQGG" else 0.0)
    px, py, pz = _centres(n, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    inside = r <= Q
    assert inside.sum() == 19
    f = np.zeros((3, n ** 3))
    f[0, inside] = c0
    h = 0.5 * (pmax - pmin) / n
    integral = sum(c0 * _inv_r_over_cube(px[j], py[j], pz[j], h) for j in np.nonzero(inside)[0])
    cells = [i for i in np.nonzero(inside)[0] if r[i] > 0]
    expect = -(dt / HBARC) * c0 * integral / (256 * math.pi ** 4)         # x 1/E1, in number units N_g df
    est = []
    for batch in range(8):                                                  # independent evaluations: other step index
        tot = 0.0
        for i in cells:
            dN, _, _ = o.collision_tile(dt, batch, 0, f, i, i + 1, mode=1)
            assert np.count_nonzero(dN[0]) == 1 and dN[0, i] < 0            # labelled: only the grid point itself
            tot += dN[0, i] * r[i]
        est.append(tot / len(cells))
    est = np.array(est)
    err = est.std(ddof=1) / math.sqrt(len(est))
    assert err < 0.01 * abs(expect)
    assert abs(est.mean() - expect) < 4 * err


# --------------------------------------------------------------------------------------------------------------
# P4: Eq. 5 for g g -> g g in the paper's own parametrisation (Eq. 17-21), independent of the oracle's sampling.
def _paper_parametrisation_gg(f_cells, cells, n, pmin, pmax, alpha_s, m2, dt, n_per_cell, rng):
    """N_g dt C_g(p) for the cell centres p in `cells`, p labelled as the OUTGOING particle d of Eq. 5.
    Integration variables (k1x, k1y, k3x, k3y, k3z) uniform in the box (Eq. 20, V_domain = L^5); k1z from the two
    roots of E1 + E2 = E3 + Ep (Eq. 18-19) in the massless closed form; k2 = k3 + p - k1 (Eq. 17); integrand Eq. 21
    with sym = 1/2.  All four momenta must lie in the box (S9) and f is the binned f."""
    L = pmax - pmin
    dp = L / n
    g4 = (4 * math.pi * alpha_s) ** 2
    px, py, pz = _centres(n, pmin, pmax)

    def cell(k):
        q = np.floor((k - pmin) / dp).astype(np.int64)
        ok = np.all((q >= 0) & (q < n), axis=1)
        q = np.clip(q, 0, n - 1)
        return q[:, 0] + n * (q[:, 1] + n * q[:, 2]), ok

    def Mgg(s, t, u):
        return 16 * 8 * 9 * g4 * (3 - s * u / (t - m2) ** 2 - s * t / (u - m2) ** 2 - t * u / s ** 2)   # Table I

    out = []
    for ip in cells:
        p = np.array([px[ip], py[ip], pz[ip]])
        Ep = np.linalg.norm(p)
        N = n_per_cell
        k3 = rng.uniform(pmin, pmax, (N, 3))
        k1xy = rng.uniform(pmin, pmax, (N, 2))
        E3 = np.linalg.norm(k3, axis=1)
        P = k3 + p
        Et = E3 + Ep
        S_ = Et ** 2 - np.sum(P * P, axis=1)
        a = S_ + 2 * (P[:, 0] * k1xy[:, 0] + P[:, 1] * k1xy[:, 1])
        kp2 = np.sum(k1xy ** 2, axis=1)
        D = Et ** 2 - P[:, 2] ** 2
        H = a * a - 4 * kp2 * D
        ok = H >= 0
        sq = np.sqrt(np.where(ok, H, 0.0))
        c3, ok3 = cell(k3)
        acc = np.zeros(N)
        for sg in (+1.0, -1.0):
            z = (a * P[:, 2] + sg * Et * sq) / (2 * D)
            k1 = np.column_stack([k1xy, z])
            E1 = np.linalg.norm(k1, axis=1)
            k2 = P - k1
            E2 = np.linalg.norm(k2, axis=1)
            valid = ok & (np.abs(E1 + E2 - Et) < 1e-9 * Et)                 # spurious root of the squared equation
            J = z / E1 - (P[:, 2] - z) / E2                                  # Eq. 19
            c1, ok1 = cell(k1)
            c2, ok2 = cell(k2)
            s_ = 2 * (E1 * E2 - np.sum(k1 * k2, axis=1))
            t_ = -2 * (E1 * E3 - np.sum(k1 * k3, axis=1))
            u_ = -s_ - t_
            f1, f2, f3, fp = f_cells[c1], f_cells[c2], f_cells[c3], f_cells[ip]
            stat = f1 * f2 * (1 + f3) * (1 + fp) - (1 + f1) * (1 + f2) * f3 * fp
            good = valid & ok1 & ok2 & ok3 & (s_ > 0)
            with np.errstate(all="ignore"):
                w = stat * 0.5 * Mgg(s_, t_, u_) / np.abs(J) / ((2 * math.pi) ** 5 * 16 * E1 * E2 * E3 * Ep)
            acc += np.where(good, w, 0.0)
        out.append((dt / HBARC) * L ** 5 * acc.mean())
    return np.array(out)


@pytest.mark.slow
def test_P4_paper_parametrisation_agrees():
    # over-occupied core (7 cells) in a thin bath: the core scatters out, the shells around it fill up; cells of one
    # shell are equivalent by the cubic symmetry, so shell averages are compared
    n, pmin, pmax, alpha_s, mD, dt = 5, -2.0, 2.0, 0.3, 0.8, 0.01
    px, py, pz = _centres(n, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    f = np.where(r <= 0.85, 0.5, 0.05)
    shells = [np.nonzero(np.abs(r - rr) < 1e-9)[0] for rr in (0.8, 0.8 * math.sqrt(2), 0.8 * math.sqrt(3))]
    assert [len(s) for s in shells] == [6, 12, 8]
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), samples=60000, seed=8, m_D=mD)
    rng = np.random.default_rng(12345)
    for sh in shells:
        cells = sh[:6]
        orc, pap = [], []
        for b in range(5):
            orc.append(np.mean([o.collision_tile(dt, b, 0, f[None, :], int(i), int(i) + 1, mode=1)[0][0, i] for i in cells]))
            pap.append(_paper_parametrisation_gg(f, cells, n, pmin, pmax, alpha_s, mD * mD, dt, 250000, rng).mean())
        orc, pap = np.array(orc), np.array(pap)
        ea, eb = orc.std(ddof=1) / math.sqrt(len(orc)), pap.std(ddof=1) / math.sqrt(len(pap))
        print("P4 shell r=%.3f: oracle %.5e +- %.1e   paper-parametrisation %.5e +- %.1e" % (r[sh[0]], orc.mean(), ea, pap.mean(), eb))
        assert ea < 0.02 * abs(orc.mean())
        assert eb < 0.05 * abs(orc.mean())
        assert abs(orc.mean() - pap.mean()) < 4 * math.hypot(ea, eb)


# --------------------------------------------------------------------------------------------------------------
def _smooth_mixture(n, pmin, pmax):
    px, py, pz = _centres(n, pmin, pmax)
    r2 = px ** 2 + py ** 2 + pz ** 2
    widths = [1.6, 0.9, 1.1, 0.7, 1.3, 1.0, 0.8]
    amps = [0.5, 0.30, 0.12, 0.25, 0.2, 0.15, 0.35]
    f = np.stack([A * np.exp(-r2 / w) * (1 + 0.2 * px * (1 if a % 2 else -1)) for a, (A, w) in enumerate(zip(amps, widths))])
    return f, (px, py, pz, np.sqrt(r2))


def _labelled_vs_symmetric(n, Ns, m_D, elastic_off, batches=6):
    f, (px, py, pz, r) = _smooth_mixture(n, -3.0, 3.0)
    o = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=SP7, samples=Ns, seed=17, m_D=m_D)
    if elastic_off:
        for k in ("A", "11", "1B", "QG", "GG"):
            o.set_msq_override(k, 0.0)
    lab, sym = [], []
    for b in range(batches):
        dl, _, _ = o.collision_tile(0.01, b, 0, f, mode=1)
        ds, _, _ = o.collision_tile(0.01, b, 0, f, mode=0)
        assert abs(ds.sum()) < 1e-13 * np.abs(ds).sum()                     # P6 on the way
        lab.append(dl.sum(axis=1))
        sym.append(ds.sum(axis=1))
    lab, sym = np.array(lab), np.array(sym)
    d = lab - sym
    return lab.mean(0), sym.mean(0), d.mean(0), d.std(0, ddof=1) / math.sqrt(batches)


@pytest.mark.slow
def test_P5_symmetric_estimator_agrees_with_labelled():
    # Eq. 3-4 (labelled: only the grid point itself, weight 1/2 per ordered channel) against the symmetric reuse
    # (1/8 on four cells, S2), same f, same samples.  Both converge to the same integral; at finite cell size they
    # differ by the binning (slot 1 sits on the cell centre, slots 2-4 anywhere in their cells), O(dp^2).
    # (a) number-changing channels only (g g <-> q qbar, q qbar -> q' qbar'): species numbers, sharp to 0.1 %
    lab, sym, d, ed = _labelled_vs_symmetric(8, 800, 0.4, elastic_off=True)
    print("P5a lab", lab, "sym", sym, "rel", d / sym, "+-", ed / np.abs(sym))
    assert sym[0] < 0 and np.all(sym[1:] > 0)
    assert np.all(ed < 0.005 * np.abs(sym))
    assert np.all(np.abs(d) < 4 * ed + 0.015 * np.abs(sym))
    # pairs are created together: q and qbar of one flavour gain exactly the same number in the symmetric estimator
    assert np.allclose(sym[1::2], sym[2::2], rtol=1e-12)
    # (b) all 127 channels, smooth kernel (large regulator): quark numbers agree to a few per cent and the gluon
    # number gap (elastic g g -> g g does not conserve the labelled sum at finite dp) closes like dp^2
    lab8, sym8, d8, ed8 = _labelled_vs_symmetric(8, 1000, 1.5, elastic_off=False)
    lab12, sym12, d12, ed12 = _labelled_vs_symmetric(12, 300, 1.5, elastic_off=False)
    print("P5b n=8  rel", d8 / sym8, "+-", ed8 / np.abs(sym8))
    print("P5b n=12 rel", d12 / sym12, "+-", ed12 / np.abs(sym12))
    assert np.all(np.abs(d12[1:]) < 4 * ed12[1:] + 0.04 * np.abs(sym12[1:]))
    assert np.all(np.abs(d8[1:]) < 4 * ed8[1:] + 0.09 * np.abs(sym8[1:]))
    gap8, gap12 = abs(d8[0]) / 8 ** 3, abs(d12[0]) / 12 ** 3
    assert gap12 < gap8 / 1.5


def test_P6_exact_number_conservation_and_P9_direction():
    # CFG-0-like glue, quark species present but empty: g g -> q qbar must move number from g to q (Fig. 4a)
    n = 10
    o = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=SP7, samples=48, seed=0)
    px, py, pz = _centres(n, -3.0, 3.0)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    f = np.zeros((1, 7, n ** 3))
    f[0, 0] = 0.4 * (r <= 1.5)
    o.set_f(f)
    mom0 = o.moments()
    dF = o.collision(0.01, 0)
    G = o.gross()
    num = (NDEG[None, :, None] * dF).sum()
    den = (NDEG[None, :, None] * np.abs(dF)).sum()
    assert den > 0 and abs(num) <= 1e-13 * den                              # Eq. 23, NS: 1e-13
    assert (NDEG[None, :, None] * G).sum() >= den
    per_species = (NDEG[None, :, None] * dF).sum(axis=(0, 2))
    assert per_species[0] < 0 and np.all(per_species[1:] > 0)
    assert np.allclose(per_species[1:], per_species[1], rtol=0.2)           # flavour blind
    o.step(0.01)
    mom1 = o.moments()
    N0, N1 = mom0["tot"][:, 0], mom1["tot"][:, 0]
    assert abs(N1.sum() - N0.sum()) <= 1e-13 * N0.sum()                     # total conserved through bzo_step
    assert N1[0] < N0[0] and np.all(N1[1:] > 0)
    # over-occupied step: the soft cells gain first -- gluon dF at the smallest |p| is positive
    soft = np.argsort(r)[:8]
    o2 = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=(0,), samples=400, seed=0)
    o2.set_f(f[:, :1])
    dF2 = o2.collision(0.01, 0)
    assert dF2[0, 0, soft].sum() > 0
    # random dense f, all 127 channels: conservation again, and also for a second step index
    rng = np.random.default_rng(5)
    o.set_f(rng.uniform(0.02, 0.6, size=(1, 7, n ** 3)))
    for step in (0, 7):
        dF = o.collision(0.01, step)
        num = (NDEG[None, :, None] * dF).sum()
        den = (NDEG[None, :, None] * np.abs(dF)).sum()
        assert abs(num) <= 1e-13 * den


def test_threads_only_reorder_sums():
    n = 8
    rng = np.random.default_rng(6)
    f = rng.uniform(0.02, 0.6, size=(1, 3, n ** 3))
    a = bzo.Oracle(np_=n, species=(0, 1, 2), samples=16, seed=2, threads=1)
    b = bzo.Oracle(np_=n, species=(0, 1, 2), samples=16, seed=2, threads=3)
    a.set_f(f); b.set_f(f)
    da, db = a.collision(0.01, 3), b.collision(0.01, 3)
    assert np.all(np.abs(da - db) <= 1e-13 * np.maximum(a.gross(), 1e-300))
    # several spatial cells: identical bits for any thread count
    f2 = rng.uniform(0.02, 0.6, size=(8, 3, n ** 3))
    a2 = bzo.Oracle(nx=2, ny=2, nz=2, dx=0.2, np_=n, species=(0, 1, 2), samples=4, seed=2, threads=1)
    b2 = bzo.Oracle(nx=2, ny=2, nz=2, dx=0.2, np_=n, species=(0, 1, 2), samples=4, seed=2, threads=4)
    a2.set_f(f2); b2.set_f(f2)
    assert np.array_equal(a2.collision(0.01, 1), b2.collision(0.01, 1))
    assert np.array_equal(a2.stream(0.01), b2.stream(0.01))


def test_P3b_binned_equilibrium_relaxes_slowly():
    # Bose-Einstein at the cell centres (T = 0.5 GeV, mu = -0.2 GeV), gg -> gg: C[f] vanishes up to sampling noise and
    # a binning floor that falls with the cell size; a step function of similar content relaxes >= 5 x faster.
    T, mu, mD = 0.5, -0.2, 0.8
    ratio = {}
    for n, Ns in ((10, 1000), (16, 250)):
        o = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=(0,), samples=Ns, seed=3, m_D=mD, threads=4)
        px, py, pz = _centres(n, -3.0, 3.0)
        r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
        feq = 1.0 / (np.exp((r - mu) / T) - 1.0)
        step = 0.3 * (r <= 1.5)
        o.set_f(feq[None, None, :])
        rate_eq = np.linalg.norm(o.collision(0.01, 0)) / np.linalg.norm(feq)
        o.set_f(step[None, None, :])
        rate_step = np.linalg.norm(o.collision(0.01, 0)) / np.linalg.norm(step)
        ratio[n] = rate_eq / rate_step
    print("P3b equilibrium/step relaxation ratio", ratio)
    assert ratio[10] < 0.2
    assert ratio[16] < 0.75 * ratio[10]


def _entropy(f, species):
    """- sum_a N_a sum_p [ f ln f -+ (1 +- f) ln(1 +- f) ] of the binned distribution (Bose: upper signs, Fermi: lower)"""
    tot = 0.0
    for a, sid in enumerate(species):
        x = np.clip(f[:, a, :], 1e-300, None)
        if sid == 0:
            s = -(x * np.log(x) - (1.0 + x) * np.log1p(x))
        else:
            y = np.clip(1.0 - f[:, a, :], 1e-300, None)
            s = -(x * np.log(x) + y * np.log(y))
        tot += NDEG[sid] * s.sum()
    return tot


@pytest.mark.parametrize("species", [(0,), (1, 2, 3, 4)], ids=["glue", "two_flavours"])
def test_P11_h_theorem(species):
    """P11 (an invariant the oracle does not contain): with detailed balance built into Eq. 5's gain - loss bracket the
    entropy of the distribution cannot fall (H theorem).  Each deposit moves one weight A from two cells to two others; to first
    order dS = -A [ln(f_k f_l / (F_k F_l)) - ln(f_i f_j / (F_i F_j))] has the sign of -A ln(gain/loss) >= 0 whatever the matrix
    element, so the entropy of the binned f grows step by step up to O(A^2) and the Monte Carlo noise.  A wrong sign of the
    bracket, of a deposit or of F = 1 +- f makes it fall."""
    n = 8
    o = bzo.Oracle(np_=n, pmin=-3.0, pmax=3.0, species=species, alpha_s=0.3, m_D=0.5, seed=4, samples=48, threads=4)
    px, py, pz = _centres(n, -3.0, 3.0)
    pabs = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    f = np.zeros(o.shape)
    for a, sid in enumerate(species):
        f[0, a] = (0.4 if sid == 0 else 0.6) * (pabs <= 1.6)            # far from equilibrium: a step function
    o.set_f(f)
    s = [_entropy(o.get_f(), species)]
    n0 = (NDEG[list(species)][None, :, None] * o.get_f()).sum()
    for _ in range(12):
        o.step(0.05)
        s.append(_entropy(o.get_f(), species))
    s = np.array(s)
    assert np.all(np.diff(s) > 0.0), np.diff(s)
    assert s[-1] > 1.02 * s[0]
    n1 = (NDEG[list(species)][None, :, None] * o.get_f()).sum()
    assert abs(n1 - n0) <= 1e-12 * n0
    # negative control on a smooth, strictly positive non-equilibrium f (so that f stays positive either way): dt -> -dt flips
    # every deposit, and the entropy falls
    g = np.zeros(o.shape)
    for a, sid in enumerate(species):
        g[0, a] = 0.02 + 0.3 * np.exp(-(pabs - 1.5) ** 2 / 0.5)
    for sign in (+1.0, -1.0):
        o.set_f(g)
        o.step(sign * 0.01)
        h = o.get_f()
        assert h.min() > 0.0
        assert sign * (_entropy(h, species) - _entropy(g, species)) > 0.0
