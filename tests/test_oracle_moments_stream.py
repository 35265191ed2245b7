"""Pins P7 (Eq. 8, 10, 11 on Bose-Einstein / Fermi-Dirac closed forms) and P8 (upwind free streaming)."""
import math

import numpy as np
import pytest

from oracle import bzo

HBARC = 0.1973269804
ZETA3 = 1.2020569031595942


def _centres(n, pmin, pmax):
    dp = (pmax - pmin) / n
    c = pmin + (np.arange(n) + 0.5) * dp
    pz, py, px = np.meshgrid(c, c, c, indexing="ij")
    return px.reshape(-1), py.reshape(-1), pz.reshape(-1)


def _thermal(n, T, pmin, pmax):
    px, py, pz = _centres(n, pmin, pmax)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    return 1.0 / np.expm1(r / T), 1.0 / (np.exp(r / T) + 1.0)


def test_P7_thermal_closed_forms():
    # midpoint rule on a wide grid: T = 0.5 GeV, box [-6, 6] (12 T), mu = 0.  The Bose integrand of Eq. 8 goes like
    # T/p^2 at the origin, so its midpoint sum converges only linearly in dp: Richardson-extrapolate two grids.
    T, pmin, pmax, alpha_s = 0.5, -6.0, 6.0, 0.3
    g2 = 4 * math.pi * alpha_s
    m2_g, m2_all = {}, {}
    for n in (48, 96):
        be, fd = _thermal(n, T, pmin, pmax)
        o = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0,), alpha_s=alpha_s, dx=2.0)
        o.set_f(be[None, None, :])
        m = o.moments()
        m2_g[n] = m["m2"][0]
        o7 = bzo.Oracle(np_=n, pmin=pmin, pmax=pmax, species=(0, 1, 2, 3, 4, 5, 6), alpha_s=alpha_s)
        o7.set_f(np.stack([be] + [fd] * 6)[None])
        m7 = o7.moments()
        m2_all[n] = m7["m2"][0]
    # gluons only: n_g = 16 zeta(3) T^3/pi^2, e_g = 16 pi^2 T^4/30 (Eq. 10-11), Eq. 8 -> g^2 T^2/2
    assert m["ne"][0, 0, 0] == pytest.approx(16 * ZETA3 * T ** 3 / math.pi ** 2, rel=5e-3)
    assert m["ne"][0, 0, 1] == pytest.approx(16 * math.pi ** 2 * T ** 4 / 30, rel=2e-3)
    assert 2 * m2_g[96] - m2_g[48] == pytest.approx(g2 * T * T / 2, rel=1e-2)
    assert abs(m2_g[96] / (g2 * T * T / 2) - 1) < 0.55 * abs(m2_g[48] / (g2 * T * T / 2) - 1)   # linear convergence
    # totals: density x volume / hbarc^3 (number), GeV (energy)
    vol = 2.0 ** 3 / HBARC ** 3
    assert m["tot"][0, 0] == pytest.approx(m["ne"][0, 0, 0] * vol, rel=1e-14)
    assert m["tot"][0, 1] == pytest.approx(m["ne"][0, 0, 1] * vol, rel=1e-14)
    # all 7 species: quark densities 6 x (3/4) zeta(3) T^3/pi^2 and 6 x (7/8) pi^2 T^4/30,
    # Eq. 8 -> g^2 T^2 (1/2 + N_f/12) with N_f = 3 (the value SURVEY.md S7 notes: half the textbook Debye mass^2)
    for a in range(1, 7):
        assert m7["ne"][0, a, 0] == pytest.approx(6 * 0.75 * ZETA3 * T ** 3 / math.pi ** 2, rel=2e-3)
        assert m7["ne"][0, a, 1] == pytest.approx(6 * (7 / 8) * math.pi ** 2 * T ** 4 / 30, rel=2e-3)
    assert m7["ne"][0, 0, 0] == pytest.approx(m["ne"][0, 0, 0], rel=1e-14)
    assert 2 * m2_all[96] - m2_all[48] == pytest.approx(g2 * T * T * (0.5 + 3 / 12), rel=1e-2)
    # quarks only (one flavour pair): Eq. 8 -> g^2 T^2 / 12; the Fermi integrand is regular, no extrapolation needed
    be, fd = _thermal(96, T, pmin, pmax)
    oq = bzo.Oracle(np_=96, pmin=pmin, pmax=pmax, species=(3, 4), alpha_s=alpha_s)
    oq.set_f(np.stack([fd, fd])[None])
    assert oq.moments()["m2"][0] == pytest.approx(g2 * T * T / 12, rel=1e-2)
    # fixed regulator: m_D is returned squared, whatever f is
    of = bzo.Oracle(np_=8, species=(0,), m_D=0.7)
    assert of.moments()["m2"][0] == pytest.approx(0.49, rel=1e-15)


def test_m2_skips_the_zero_momentum_cell_and_is_linear():
    n = 5
    o = bzo.Oracle(np_=n, pmin=-2.5, pmax=2.5, species=(0, 1), alpha_s=0.3)
    f = np.zeros((1, 2, n ** 3))
    f[0, 0, (n ** 3) // 2] = 1e6                      # the p = 0 cell
    o.set_f(f)
    assert o.moments()["m2"][0] == 0.0
    f[0, 0, 0] = 0.2                                  # corner cell, |p| = 2 sqrt 3
    o.set_f(f)
    m_g = o.moments()["m2"][0]
    expect = 4 * math.pi * 0.3 * 1.0 / ((2 * math.pi) ** 3 * 2 * math.sqrt(3)) * 6 * 0.2
    assert m_g == pytest.approx(expect, rel=1e-13)
    f[0, 0, 0] = 0.0
    f[0, 1, 0] = 0.2                                  # the same occupation in a quark species weighs 1/6
    o.set_f(f)
    assert o.moments()["m2"][0] == pytest.approx(expect / 6, rel=1e-13)


def _stream_oracle(nx, ny, nz, n, dx):
    return bzo.Oracle(nx=nx, ny=ny, nz=nz, dx=dx, np_=n, pmin=-2.5, pmax=2.5, species=(0, 3), samples=2)


def test_P8_conservation_and_exact_shift():
    nx, ny, nz, n, dx = 6, 4, 3, 5, 0.25
    o = _stream_oracle(nx, ny, nz, n, dx)
    rng = np.random.default_rng(1)
    f = rng.uniform(0.0, 1.0, size=o.shape)
    o.set_f(f)
    dF = o.stream(0.1)
    # (i) flux form: sum over x of every (species, p) column is conserved (Eq. 13)
    assert np.all(np.abs(dF.sum(axis=0)) <= 1e-13 * np.abs(f).sum(axis=0))
    # the p = 0 cell does not move (v = 0)
    assert np.all(dF[:, :, (n ** 3) // 2] == 0.0)
    # (iii) a cell on the +x momentum axis has v = (1,0,0): with dt = dx one step is an exact shift by one cell
    pc = (n // 2 + 1) + n * ((n // 2) + n * (n // 2))
    dF1 = o.stream(dx)
    f4 = f.reshape(nz, ny, nx, 2, n ** 3)
    new = (f + dF1).reshape(nz, ny, nx, 2, n ** 3)[..., pc]
    assert np.allclose(new, np.roll(f4[..., pc], 1, axis=2), rtol=0, atol=1e-15)
    # and on the -y axis: shift by one cell towards smaller y
    pc = (n // 2) + n * ((n // 2 - 1) + n * (n // 2))
    new = (f + dF1).reshape(nz, ny, nx, 2, n ** 3)[..., pc]
    assert np.allclose(new, np.roll(f4[..., pc], -1, axis=1), rtol=0, atol=1e-15)
    # -z axis
    pc = (n // 2) + n * ((n // 2) + n * (n // 2 - 2))
    new = (f + dF1).reshape(nz, ny, nx, 2, n ** 3)[..., pc]
    assert np.allclose(new, np.roll(f4[..., pc], -1, axis=0), rtol=0, atol=1e-15)


def test_P8_fourier_mode_amplification():
    # (ii) one Fourier mode: amplitude x g per step, g = 1 - sum_d |c_d| (1 - exp(-i sign(c_d) k_d dx))
    nx, ny, nz, n, dx, dt = 8, 4, 2, 5, 0.2, 0.05
    o = _stream_oracle(nx, ny, nz, n, dx)
    kx, ky, kz = 2 * math.pi * 1 / (nx * dx), 2 * math.pi * 1 / (ny * dx), 2 * math.pi * 1 / (nz * dx)
    X = (np.arange(nx)) * dx
    Y = (np.arange(ny)) * dx
    Z = (np.arange(nz)) * dx
    phase = kx * X[None, None, :] + ky * Y[None, :, None] + kz * Z[:, None, None]
    px, py, pz = _centres(n, -2.5, 2.5)
    r = np.sqrt(px ** 2 + py ** 2 + pz ** 2)
    for part in (np.cos, np.sin):
        f = np.repeat(part(phase).reshape(-1)[:, None, None], 2, axis=1) * np.ones((1, 1, n ** 3))
        o.set_f(f)
        dF = o.stream(dt)
        res = (f + dF).reshape(nz, ny, nx, 2, n ** 3)
        for pc in (0, 7, 31, 63, 88, 124):
            v = np.array([px[pc], py[pc], pz[pc]]) / r[pc]
            c = v * dt / dx
            g = 1.0 - sum(abs(cd) * (1 - np.exp(-1j * np.sign(cd) * kd * dx)) for cd, kd in zip(c, (kx, ky, kz)))
            full = g * np.exp(1j * phase)
            expect = full.real if part is np.cos else full.imag
            assert np.allclose(res[..., 0, pc], expect, rtol=0, atol=1e-13)
            assert np.allclose(res[..., 1, pc], expect, rtol=0, atol=1e-13)


def test_homogeneous_grid_does_not_stream_and_step_is_unsplit():
    o = bzo.Oracle(np_=6, species=(0,), samples=8, seed=1)
    rng = np.random.default_rng(2)
    f = rng.uniform(0.05, 0.5, size=o.shape)
    o.set_f(f)
    assert np.all(o.stream(0.01) == 0.0)               # single periodic cell: neighbour = itself
    dFc = o.collision(0.01, 0)
    o.step(0.01)
    assert np.array_equal(o.get_f(), (f + 0.0) + dFc)   # Eq. 15: f + dF_stream + dF_coll from the old f
    # the step counter advances: the next step uses step index 1
    f1 = o.get_f()
    dFc1 = o.collision(0.01, 1)
    o.step(0.01)
    assert np.array_equal(o.get_f(), f1 + dFc1)
    # inhomogeneous: both increments are taken from the old f (S13)
    o2 = bzo.Oracle(nx=3, ny=2, nz=2, dx=0.3, np_=4, species=(0, 1, 2), samples=4, seed=5)
    f = rng.uniform(0.05, 0.5, size=o2.shape)
    o2.set_f(f)
    dFs, dFc = o2.stream(0.02), o2.collision(0.02, 0)
    o2.step(0.02)
    assert np.array_equal(o2.get_f(), (f + dFs) + dFc)
