"""Pin P3 (equilibrium kills the bracket of Eq. 5) and Eq. 22 (one weight, signs - - + +), SURVEY.md 8c step 6."""
import math

import numpy as np

from oracle import bzo

SP = (0, 1, 2, 3, 4, 5, 6)


def _feq(sp, E, T, mu):
    """Eq. 6-7 with chemical potential mu[sp]."""
    x = (E - mu[sp]) / T
    return 1.0 / (math.exp(x) - 1.0) if sp == 0 else 1.0 / (math.exp(x) + 1.0)


def _equilibrium_case(mu, T=0.45, n_samples=300):
    o = bzo.Oracle(np_=8, pmin=-3.0, pmax=3.0, species=SP, samples=8, seed=21)
    ch = o.channels()
    worst = 0.0
    count = 0
    for pc in range(0, o.Np, 5):
        for smp in range(8):
            s = o.sample_one(0, 0, pc, smp)
            if s.attempts == 0:
                continue
            E = (s.E1, s.E2, s.E3, s.E1 + s.E2 - s.E3)
            fv = np.array([[_feq(sp, E[slot], T, mu) for sp in SP] for slot in range(4)])
            dN, fwd, gross = o.sample_channels(fv, s.s, s.t, s.u, s.E1, s.E2, 0.4, 0.01)
            for q, (a, b, c, d, kind, crossed) in enumerate(ch):
                F = lambda sp_, f: 1 + f if sp_ == 0 else 1 - f
                gain = fv[0, a] * fv[1, b] * F(SP[c], fv[2, c]) * F(SP[d], fv[3, d])
                worst = max(worst, abs(fwd[q]) / gain)
            count += 1
            if count >= n_samples:
                return worst
    return worst


def test_P3_common_negative_chemical_potential():
    # 2->2 only: any common mu conserves mu_a + mu_b = mu_c + mu_d (P:342 reports negative mu for both)
    mu = {sp: -0.2 for sp in SP}
    assert _equilibrium_case(mu) < 1e-13


def test_P3_quark_antiquark_opposite_mu():
    # Eq. 7: quarks E - mu_q, antiquarks E + mu_q, gluons mu = 0; one mu per flavour
    mu = {0: 0.0, 1: 0.3, 2: -0.3, 3: -0.1, 4: 0.1, 5: 0.25, 6: -0.25}
    assert _equilibrium_case(mu) < 1e-13


def test_P3_wrong_statistics_would_not_vanish():
    # sanity of the test itself: gluons with a quark-like mu split break g g <-> q qbar detailed balance
    mu = {0: 0.0, 1: 0.3, 2: 0.3, 3: 0.0, 4: 0.0, 5: 0.0, 6: 0.0}
    assert _equilibrium_case(mu, n_samples=50) > 1e-3


def test_eq22_single_channel_deposit_pattern():
    o = bzo.Oracle(np_=8, species=(0,), samples=4, seed=1)
    rng = np.random.default_rng(0)
    for smp in range(4):
        s = o.sample_one(0, 0, 77, smp)
        fv = rng.uniform(0.05, 0.9, size=(4, 1))
        dN, fwd, gross = o.sample_channels(fv, s.s, s.t, s.u, s.E1, s.E2, 0.3, 0.01)
        A = dN[2, 0]
        assert A != 0.0 and gross == abs(A)
        assert dN[0, 0] == -A and dN[1, 0] == -A and dN[3, 0] == A             # Eq. 22
        # Bose bracket of Eq. 5 with F = 1 + f
        f1, f2, f3, f4 = fv[:, 0]
        assert math.isclose(fwd[0], f1 * f2 * (1 + f3) * (1 + f4) - (1 + f1) * (1 + f2) * f3 * f4, rel_tol=1e-13)
        # weight: A = K/(E1 E2) |M_gg|^2 fwd with K = (dt/hbarc) Vp / (2048 pi^4 Ns)
        K = (0.01 / 0.1973269804) * 6.0 ** 3 / (2048 * math.pi ** 4 * 4)
        g4 = (4 * math.pi * 0.3) ** 2
        assert math.isclose(A, K / (s.E1 * s.E2) * bzo.msq("GG", s.s, s.t, s.u, 0.3, g4) * fwd[0], rel_tol=1e-12)


def test_fermi_blocking_and_bose_enhancement_signs():
    # q q -> q q with the final states full (f = 1) has no gain; a full initial state has no loss (F_q = 1 - f)
    o = bzo.Oracle(np_=8, species=(1,), samples=4, seed=1)
    s = o.sample_one(0, 0, 77, 0)
    fv = np.array([[0.3], [0.4], [1.0], [0.2]])
    _, fwd, _ = o.sample_channels(fv, s.s, s.t, s.u, s.E1, s.E2, 0.3, 0.01)
    assert math.isclose(fwd[0], -(0.7 * 0.6 * 1.0 * 0.2), rel_tol=1e-14)       # only the loss of the reverse reaction
    fv = np.array([[1.0], [0.4], [0.1], [0.2]])
    _, fwd, _ = o.sample_channels(fv, s.s, s.t, s.u, s.E1, s.E2, 0.3, 0.01)
    assert math.isclose(fwd[0], 1.0 * 0.4 * 0.9 * 0.8, rel_tol=1e-14)
    # every per-sample deposit sums to zero in number units over the four slots and all species (Eq. 23)
    o7 = bzo.Oracle(np_=8, species=SP, samples=4, seed=1)
    fv = np.random.default_rng(3).uniform(0.05, 0.9, size=(4, 7))
    dN, _, gross = o7.sample_channels(fv, s.s, s.t, s.u, s.E1, s.E2, 0.3, 0.01)
    assert abs(dN.sum()) <= 1e-14 * gross
    assert abs(dN[:2].sum() + dN[2:].sum()) <= 1e-14 * gross
