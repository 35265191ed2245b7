"""Pins of the oracle's NEXT-rank-2 functions: thermal masses (Eq. 8-9) and the paper's own
central-difference drift + force operator (Eq. 15), against what the paper and the mathematics fix:
  V1  Eq. 8-9 on Bose-Einstein / Fermi-Dirac: m_g^2 = g^2 T^2 (1/2 + N_f/12), m_q^2 = g^2 T^2 / 3 (first step, E = |p|);
  V2  the iteration of P:107: the second evaluation uses E = sqrt(p^2 + m_a^2) of the right species (one-cell closed form);
  V3  Eq. 13's property: the operator sums to zero over the periodic phase space, per species;
  V4  constant mass: no force, and a Fourier mode in x is advected with the velocity p_i / E_p (massive);
  V5  Vlasov equilibrium f = F(E_p(x)): drift and force cancel in the continuum, so the discrete residual is O(h^2);
      a wrong sign or factor between the two terms leaves an O(1) residual;
  V6  momentum balance of the force term alone (summation by parts): sum_p p_x dF = -dt sum_p f dE/dx.
"""
import math

import numpy as np
import pytest

from oracle import bzo

SP7 = (0, 1, 2, 3, 4, 5, 6)


def _centres(n, pmin, pmax):
    dp = (pmax - pmin) / n
    c = pmin + (np.arange(n) + 0.5) * dp
    pz, py, px = np.meshgrid(c, c, c, indexing="ij")
    return px.reshape(-1), py.reshape(-1), pz.reshape(-1)


def test_V1_thermal_masses_closed_forms():
    T, pmin, pmax, alpha_s = 0.5, -6.0, 6.0, 0.3
    g2 = 4 * math.pi * alpha_s
    got = {}
    for n in (48, 96):
        px, py, pz = _centres(n, pmin, pmax)
        r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
        be, fd = 1.0 / np.expm1(r / T), 1.0 / (np.exp(r / T) + 1.0)
        o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=SP7, alpha_s=alpha_s)
        o.set_f(np.stack([be] + [fd] * 6)[None])
        got[n] = o.thermal_masses()[0]
        assert np.array_equal(o.get_masses()[0], got[n])
    # the Bose integrand goes like T/p^2 at the origin: linear convergence, Richardson-extrapolate (as pin P7)
    ext = 2 * got[96] - got[48]
    assert ext[0] == pytest.approx(g2 * T * T * (0.5 + 3 / 12), rel=1e-2)            # Eq. 8
    for fl in range(3):
        assert ext[1 + fl] == pytest.approx(g2 * T * T / 3, rel=1e-2)                # Eq. 9
    # Eq. 8 with E = |p| is the regulator of the collision path (S8a.1): same number through bzo_moments
    o = bzo.Oracle(np_=48, pmin=pmin, pmax=pmax, species=SP7, alpha_s=alpha_s)
    px, py, pz = _centres(48, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    o.set_f(np.stack([1.0 / np.expm1(r / T)] + [1.0 / (np.exp(r / T) + 1.0)] * 6)[None])
    assert o.moments()["m2"][0] == pytest.approx(o.thermal_masses()[0, 0], rel=1e-13)


def test_V2_mass_iteration_uses_massive_energy_of_the_right_species():
    n, pmin, pmax, alpha_s = 6, -3.0, 3.0, 0.3
    g2 = 4 * math.pi * alpha_s
    dp = (pmax - pmin) / n
    w = dp ** 3 / (2 * math.pi) ** 3
    px, py, pz = _centres(n, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    cg, cu, cg_f, cu_f = 17, 100, 0.8, 0.3                       # one gluon cell, one u-quark cell
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0, 1, 2), alpha_s=alpha_s)
    f = np.zeros((1, 3, n ** 3))
    f[0, 0, cg], f[0, 1, cu] = cg_f, cu_f
    o.set_f(f)
    m1 = o.thermal_masses()[0]
    Ig, Iu = w * cg_f / r[cg], w * cu_f / r[cu]
    assert m1[0] == pytest.approx(g2 * (6 * Ig + Iu), rel=1e-13)
    assert m1[1] == pytest.approx((4 / 3) * g2 * (2 * Ig + Iu), rel=1e-13)
    assert m1[2] == pytest.approx((4 / 3) * g2 * (2 * Ig), rel=1e-13)   # d: absent species, only the gluon term
    m2 = o.thermal_masses()[0]                                   # second step: E = sqrt(p^2 + m_a^2), a's own mass
    Ig2, Iu2 = w * cg_f / math.sqrt(r[cg] ** 2 + m1[0]), w * cu_f / math.sqrt(r[cu] ** 2 + m1[1])
    assert m2[0] == pytest.approx(g2 * (6 * Ig2 + Iu2), rel=1e-13)
    assert m2[1] == pytest.approx((4 / 3) * g2 * (2 * Ig2 + Iu2), rel=1e-13)
    assert m2[0] < m1[0]                                         # a mass under the integral lowers it


def test_V3_operator_sums_to_zero_over_periodic_phase_space():
    rng = np.random.default_rng(3)
    o = bzo.Oracle(nx=3, ny=2, nz=4, dx=0.3, np_=5, pmin=-2.0, pmax=2.0, species=(0, 1, 2, 5))
    f = rng.uniform(0.0, 1.0, size=o.shape)
    o.set_f(f)
    o.set_masses(rng.uniform(0.05, 0.9, size=(o.Nx, 4)))
    dF = o.vlasov(0.01)
    assert np.abs(dF).max() > 0
    for a in range(4):
        assert abs(dF[:, a].sum()) <= 1e-13 * np.abs(dF[:, a]).sum()


def test_V4_constant_mass_advects_with_massive_velocity():
    nx, n, dx, dt, m2 = 8, 4, 0.25, 0.01, 0.36
    o = bzo.Oracle(nx=nx, ny=1, nz=1, dx=dx, np_=n, pmin=-2.0, pmax=2.0, species=(0, 3))
    o.set_masses(np.tile([m2, 9.0, 0.81, 9.0], (nx, 1)))        # gluon 0.36, d quark 0.81; unused classes differ
    px, py, pz = _centres(n, -2.0, 2.0)
    k = 2 * math.pi * 2 / (nx * dx)
    x = (np.arange(nx) + 0.5) * dx
    A, B = 0.7, 0.2
    f = np.empty((nx, 2, n ** 3))
    f[:] = (A + B * np.cos(k * x))[:, None, None]
    o.set_f(f)
    dF = o.vlasov(dt)
    for a, mm in ((0, m2), (1, 0.81)):
        v = px / np.sqrt(px ** 2 + py ** 2 + pz ** 2 + mm)
        # -dt v (f(x+) - f(x-))/(2 dx) with f = A + B cos(kx):  +dt v B sin(kx) sin(k dx)/dx ; f does not depend on p: no force
        expect = dt * v[None, :] * (B * np.sin(k * x) * math.sin(k * dx) / dx)[:, None]
        assert np.abs(dF[:, a] - expect).max() <= 1e-13 * np.abs(expect).max()


def _equilibrium_residual(nx, n):
    Lx, pmax, sig2, dt = 2.0, 7.0, 4.0, 1.0               # F(E) = exp(-E^2/sigma^2): any function of E_p(x) is stationary
    dx = Lx / nx
    o = bzo.Oracle(nx=nx, ny=1, nz=1, dx=dx, np_=n, pmin=-pmax, pmax=pmax, species=(0,), threads=8)
    x = (np.arange(nx) + 0.5) * dx
    m2 = 4.0 + 1.5 * np.cos(2 * math.pi * x / Lx)
    o.set_masses(np.stack([m2] * 4, axis=1))
    px, py, pz = _centres(n, -pmax, pmax)
    E = np.sqrt((px ** 2 + py ** 2 + pz ** 2)[None, :] + m2[:, None])
    f = np.exp(-E * E / sig2)
    o.set_f(f[:, None, :])
    dF = o.vlasov(dt)[:, 0]
    # scale: the drift term alone, |p_x/E df/dx| = |p_x/E F'(E) dE/dx|, F' = -2 E F / sigma^2
    dEdx = (-1.5 * 2 * math.pi / Lx * np.sin(2 * math.pi * x / Lx))[:, None] / (2 * E)
    scale = np.abs(px[None, :] / E * (2 * E * f / sig2) * dEdx).max()
    return np.abs(dF).max() / scale


def test_V5_vlasov_equilibrium_residual_is_second_order():
    # masses (1.6 .. 2.3 GeV) and sigma = 2 GeV are resolved by dp = 0.44 and 0.22 GeV: the asymptotic regime
    r1, r2 = _equilibrium_residual(16, 32), _equilibrium_residual(32, 64)
    assert r1 < 0.12                      # the two terms cancel to truncation error (a sign error leaves ~2)
    assert 3.2 < r1 / r2 < 4.8, (r1, r2)  # O(dx^2 + dp^2)


def test_V6_force_term_momentum_balance():
    nx, n, dx, dt, pmax = 4, 12, 0.5, 0.02, 3.0
    o = bzo.Oracle(nx=nx, ny=1, nz=1, dx=dx, np_=n, pmin=-pmax, pmax=pmax, species=(0, 1))
    masses = np.array([[0.2, 0.3, 0, 0], [0.9, 0.5, 0, 0], [0.4, 1.1, 0, 0], [0.1, 0.2, 0, 0]], dtype=float)
    o.set_masses(masses)
    px, py, pz = _centres(n, -pmax, pmax)
    p2 = px ** 2 + py ** 2 + pz ** 2
    x0 = 2
    f = np.zeros((nx, 2, n ** 3))
    f[x0, 0] = np.exp(-((px - 0.4) ** 2 + py ** 2 + pz ** 2) / 0.18)      # vanishes (1e-16) at the box faces
    f[x0, 1] = 0.5 * np.exp(-(px ** 2 + (py + 0.3) ** 2 + pz ** 2) / 0.2)
    o.set_f(f)
    dF = o.vlasov(dt)
    for a in (0, 1):
        # at x0 the drift reads f(x0 +- 1) = 0; summation by parts of the force term of Eq. 15 in p_x:
        #   sum_p p_x dF(x0, p) = -dt sum_p f_p (E_p(x0+1) - E_p(x0-1)) / (2 dx)
        G = (np.sqrt(p2 + masses[x0 + 1, a]) - np.sqrt(p2 + masses[x0 - 1, a])) / (2 * dx)
        assert (px * dF[x0, a]).sum() == pytest.approx(-dt * (f[x0, a] * G).sum(), rel=1e-10)
        # and the force term moves no particles
        assert abs(dF[x0, a].sum()) <= 1e-13 * np.abs(dF[x0, a]).sum()
        # the neighbours see only the drift of f(x0): -dt (+-)(p_x/E(x0)) f(x0) / (2 dx)
        E0 = np.sqrt(p2 + masses[x0, a])
        assert np.abs(dF[x0 + 1, a] - dt * px / E0 * f[x0, a] / (2 * dx)).max() <= 1e-14
        assert np.abs(dF[x0 - 1, a] + dt * px / E0 * f[x0, a] / (2 * dx)).max() <= 1e-14


def test_V7_energy_balance_moments():
    """Eq. 11-12, 26: T^00_kin and the integrals Q_c of the source term S_ex = (1/2) sum_c (d m_c^2) Q_c.
    (a) one-cell closed forms with the degeneracies and the mass class of each species; (b) massless: T^00 is the energy
    density of bz_moments and Q reproduces Eq. 8; (c) Eq. 26 as an identity between the two outputs: at fixed f,
    d T^00 / d m_c^2 = Q_c / 2."""
    n, pmin, pmax, alpha_s = 6, -3.0, 3.0, 0.3
    g2 = 4 * math.pi * alpha_s
    w = ((pmax - pmin) / n) ** 3 / (2 * math.pi) ** 3
    px, py, pz = _centres(n, pmin, pmax)
    p2 = px ** 2 + py ** 2 + pz ** 2
    o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0, 1, 2, 5), alpha_s=alpha_s)
    # (a) one cell per species
    f = np.zeros((1, 4, n ** 3))
    cells, vals = (17, 100, 101, 200), (0.8, 0.3, 0.2, 0.4)
    for a, (cc, v) in enumerate(zip(cells, vals)):
        f[0, a, cc] = v
    o.set_f(f)
    masses = np.array([[0.4, 0.25, 0.7, 0.09]])
    o.set_masses(masses)
    d = o.energy_diag()[0]
    E = [math.sqrt(p2[cells[0]] + 0.4), math.sqrt(p2[cells[1]] + 0.25), math.sqrt(p2[cells[2]] + 0.25), math.sqrt(p2[cells[3]] + 0.09)]
    N = [16.0, 6.0, 6.0, 6.0]
    assert d[0] == pytest.approx(w * sum(Na * v * e for Na, v, e in zip(N, vals, E)), rel=1e-13)
    assert d[1] == pytest.approx(w * 16 * 0.8 / E[0], rel=1e-13)
    assert d[2] == pytest.approx(w * 6 * (0.3 / E[1] + 0.2 / E[2]), rel=1e-13)          # u and ubar share m_u
    assert d[3] == 0.0                                                                  # no d quarks
    assert d[4] == pytest.approx(w * 6 * 0.4 / E[3], rel=1e-13)
    # (b) massless
    rng = np.random.default_rng(5)
    f = rng.uniform(0.0, 1.0, size=(1, 4, n ** 3))
    o.set_f(f)
    o.set_masses(np.zeros((1, 4)))
    d = o.energy_diag()[0]
    mom = o.moments()
    assert d[0] == pytest.approx(mom["ne"][0, :, 1].sum(), rel=1e-13)
    assert g2 * (6 * d[1] / 16 + (d[2] + d[3] + d[4]) / 6) == pytest.approx(mom["m2"][0], rel=1e-13)       # Eq. 8
    # (c) d T00 / d m_c^2 = Q_c / 2 at fixed f (central difference, O(delta^2))
    base = np.array([0.5, 0.3, 0.2, 0.4])
    o.set_masses(base[None])
    Q = o.energy_diag()[0, 1:]
    for c in (0, 1, 3):
        delta = 1e-4
        up, dn = base.copy(), base.copy()
        up[c] += delta
        dn[c] -= delta
        o.set_masses(up[None])
        Tp = o.energy_diag()[0, 0]
        o.set_masses(dn[None])
        Tm = o.energy_diag()[0, 0]
        assert (Tp - Tm) / (2 * delta) == pytest.approx(0.5 * Q[c], rel=1e-6)
