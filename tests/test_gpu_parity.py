"""GPU parity: the CUDA path (through the C ABI of include/bz.h) against the CPU oracle, element by element, on the
same seeded inputs (workloads.py).  Targets (BASELINE.json north_star):
  - sampled cell indices and (s, t, u): bit exact;
  - dF and f after N steps: |gpu - cpu| <= 1e-11 * max(|cpu|, G) per value, G = the gross sum of |A| deposited into
    that value (reading S16 of SURVEY.md 8c: a net dF that cancels to ~0 is compared on the scale of what was
    summed);
  - moments within 1e-12 relative; particle number conserved to 1e-13 of the gross deposit per step.
"""
import numpy as np
import pytest
import torch

import workloads as wl
from oracle import bzo
from paper_1912_04457_b200 import bz

pytestmark = pytest.mark.gpu

TOL_DF = 1e-11
NDEG = {0: 16.0, 1: 6.0, 2: 6.0, 3: 6.0, 4: 6.0, 5: 6.0, 6: 6.0}


def _pair(cfg, threads=0):
    kw = dict(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species,
              alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples)
    import os
    o = bzo.Oracle(threads=threads or min(16, os.cpu_count() or 1), **kw)
    g = bz.Boltzmann(**kw)
    return o, g


def _deg(cfg):
    return np.array([NDEG[s] for s in cfg.species])[None, :, None]


def _assert_dF(dF_g, dF_o, gross, what):
    scale = np.maximum(np.abs(dF_o), gross)
    err = np.abs(dF_g - dF_o)
    bad = err > TOL_DF * scale
    assert not bad.any(), "%s: %d values off, worst %.3e of scale" % (what, bad.sum(), (err / np.maximum(scale, 1e-300)).max())
    nz = np.abs(dF_o).max()
    assert err.max() <= TOL_DF * nz


def _assert_conserved(cfg, dF, gross):
    num = (_deg(cfg) * dF).sum()
    den = (_deg(cfg) * gross).sum()
    assert abs(num) <= 1e-13 * den


SMALL = [
    wl.CONFIGS[0],                                                     # config 0 at full size: 216 k samples/step
    wl.scaled(wl.CONFIGS[1], np_=12, samples=40),
    wl.scaled(wl.CONFIGS[2], np_=13, samples=50),                      # odd grid, ragged sample count
    wl.scaled(wl.CONFIGS[3], nx=3, np_=10, samples=24),
    wl.scaled(wl.CONFIGS[4], nx=2, np_=11, samples=33),
]


@pytest.mark.parametrize("cfg", SMALL, ids=lambda c: c.name)
def test_sampled_indices_bit_exact(cfg):
    o, g = _pair(cfg)
    for step in (0, 3):
        for xcell in sorted({0, cfg.Nx - 1, cfg.Nx // 2}):
            co, so = o.debug_samples(step, xcell, 0, cfg.Np)
            cg, sg = g.debug_samples(step, xcell, 0, cfg.Np)
            assert np.array_equal(cg.cpu().numpy(), co)
            assert np.array_equal(sg.cpu().numpy().view(np.uint64), so.view(np.uint64))
    assert 0.05 < co[..., 3].mean() < 0.95


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_sampled_indices_bit_exact_full_size(k):
    # the five configs at their BASELINE.json sizes; the oracle checks whole spatial cells one by one
    cfg = wl.CONFIGS[k]
    o = bzo.Oracle(np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=(0,), seed=cfg.seed, samples=cfg.samples,
                   nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx)            # kinematics do not depend on species
    g = bz.Boltzmann(np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=(0,), seed=cfg.seed, samples=cfg.samples,
                     nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx)
    xcells = sorted({0, cfg.Nx - 1, (cfg.Nx * 5) // 7})
    half = cfg.Np // 2
    for xcell in xcells:
        for (b, e) in ((0, half), (half, cfg.Np)):
            co, so = o.debug_samples(cfg.steps - 1, xcell, b, e)
            cg, sg = g.debug_samples(cfg.steps - 1, xcell, b, e)
            assert np.array_equal(cg.cpu().numpy(), co)
            assert np.array_equal(sg.cpu().numpy().view(np.uint64), so.view(np.uint64))


@pytest.mark.parametrize("cfg", SMALL, ids=lambda c: c.name)
def test_collision_dF_parity_and_conservation(cfg):
    o, g = _pair(cfg)
    f = wl.initial_f(cfg)
    o.set_f(f)
    g.set_f(f)
    for step in (0, 5):
        dF_o = o.collision(cfg.dt, step)
        gross = o.gross()
        dF_g = g.collision(cfg.dt, step).cpu().numpy()
        assert np.abs(dF_o).max() > 0
        _assert_dF(dF_g, dF_o, gross, "%s step %d" % (cfg.name, step))
        _assert_conserved(cfg, dF_g, gross)
    # dense random f: every channel and every cell active (shape of the paper's Fig. 2 test)
    fr = wl.random_f(cfg, seed=7)
    o.set_f(fr)
    g.set_f(torch.from_numpy(fr).cuda())                                  # device-to-device path of bz_set_f
    dF_o = o.collision(cfg.dt, 1)
    gross = o.gross()
    dF_g = g.collision(cfg.dt, 1).cpu().numpy()
    _assert_dF(dF_g, dF_o, gross, cfg.name + " random f")
    _assert_conserved(cfg, dF_g, gross)
    assert np.count_nonzero(dF_g) > 0.9 * dF_g.size


@pytest.mark.parametrize("k", [1, 2])
def test_collision_dF_parity_full_size_homogeneous(k):
    # configs 1 and 2 at full size, one step (1.0 M and 6.9 M samples)
    cfg = wl.CONFIGS[k]
    o, g = _pair(cfg)
    f = wl.initial_f(cfg)
    o.set_f(f)
    g.set_f(f)
    dF_o = o.collision(cfg.dt, 0)
    gross = o.gross()
    dF_g = g.collision(cfg.dt, 0).cpu().numpy()
    _assert_dF(dF_g, dF_o, gross, cfg.name)
    _assert_conserved(cfg, dF_g, gross)


@pytest.mark.parametrize("cfg,steps", [(SMALL[0], 10), (SMALL[1], 4), (SMALL[2], 3), (SMALL[3], 5), (SMALL[4], 4)],
                         ids=lambda c: getattr(c, "name", str(c)))
def test_f_after_n_steps_and_moments(cfg, steps):
    o, g = _pair(cfg)
    f = wl.initial_f(cfg)
    o.set_f(f)
    g.set_f(f)
    m0 = g.moments()
    N0 = float(m0["tot"][:, 0].sum())
    for _ in range(steps):
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o = o.get_f()
    f_g = g.get_f().cpu().numpy()
    # per-value scale: the value itself or the gross deposit of the last step, whichever is larger
    _f_after_steps_check(f_g, f_o, o.gross(), cfg.name)
    # host-buffer path of bz_get_f
    host = torch.empty(g.shape, dtype=torch.float64)
    g.get_f(host)
    assert np.array_equal(host.numpy(), f_g)
    mo, mg = o.moments(), g.moments()
    for key in ("ne", "tot", "m2"):
        a, b = np.asarray(mo[key]), mg[key].numpy()
        assert np.all(np.abs(a - b) <= 1e-12 * np.maximum(np.abs(a), np.abs(a).max() * 1e-6)), key
    N1 = float(mg["tot"][:, 0].sum())
    assert abs(N1 - N0) <= 1e-12 * N0                                      # total particle number


@pytest.mark.parametrize("cfg", [SMALL[3], SMALL[4], wl.scaled(wl.CONFIGS[3], nx=4, np_=6, samples=4)],
                         ids=lambda c: c.name)
def test_stream_parity(cfg):
    o, g = _pair(cfg)
    f = wl.random_f(cfg, seed=3)
    o.set_f(f)
    g.set_f(f)
    for dt in (cfg.dt, cfg.dx):                                            # Courant number 1 on the axes: exact shift
        d_o = o.stream(dt)
        d_g = g.stream(dt).cpu().numpy()
        assert np.all(np.abs(d_g - d_o) <= 1e-13 * np.abs(f).max())
        assert np.all(np.abs(d_g.sum(axis=0)) <= 1e-12 * np.abs(f).sum(axis=0))   # Eq. 13: flux form conserves


def _f_after_steps_check(f_g, f_o, gross, what):
    """f after N steps (NS: 1e-11 relative per cell, reading S16): per value against max(|f|, gross deposit of the last
    step, 1e-3 max|f|) -- below 0.1 % of the peak the comparison is absolute, DESIGN.md 7 -- and 1e-11 max|f| overall."""
    scale = np.maximum(np.abs(f_o), gross)
    err = np.abs(f_g - f_o)
    assert (err <= TOL_DF * np.maximum(scale, np.abs(f_o).max() * 1e-3)).all(), (what, (err / np.maximum(scale, 1e-300)).max())
    assert err.max() <= TOL_DF * np.abs(f_o).max(), what


@pytest.mark.parametrize("k", [1, 2])
def test_f_after_all_steps_full_size_homogeneous(k):
    """Configs 1 and 2 at their BASELINE.json size for their own step count (20 and 50 Euler steps: 2.0e7 and 3.5e8
    kinematic samples): f after the last step and the moments against the oracle."""
    cfg = wl.CONFIGS[k]
    o, g = _pair(cfg)
    f = wl.initial_f(cfg)
    o.set_f(f)
    g.set_f(f)
    N0 = float(g.moments()["tot"][:, 0].sum())
    for _ in range(cfg.steps):
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o, f_g = o.get_f(), g.get_f().cpu().numpy()
    assert np.abs(f_o - f).max() > 1e-6 * np.abs(f).max()
    _f_after_steps_check(f_g, f_o, o.gross(), cfg.name)
    mo, mg = o.moments(), g.moments()
    for key in ("ne", "tot", "m2"):
        a, b = np.asarray(mo[key]), mg[key].numpy()
        assert np.all(np.abs(a - b) <= 1e-12 * np.maximum(np.abs(a), np.abs(a).max() * 1e-6)), key
    assert abs(float(mg["tot"][:, 0].sum()) - N0) <= 1e-12 * N0


def _config3_run(steps, dF_steps):
    cfg = wl.CONFIGS[3]
    o, g = _pair(cfg)
    f = wl.initial_f(cfg)
    o.set_f(f)
    g.set_f(f)
    N0 = float(g.moments()["tot"][:, 0].sum())
    for step in range(steps):
        if step in dF_steps:                                              # dF = dt C[f] on the current f, all 512 cells
            dF_o = o.collision(cfg.dt, step)
            gross = o.gross()
            dF_g = g.collision(cfg.dt, step).cpu().numpy()
            assert np.abs(dF_o).max() > 0
            _assert_dF(dF_g, dF_o, gross, "cfg3 full size, step %d" % step)
            _assert_conserved(cfg, dF_g, gross)
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o, f_g = o.get_f(), g.get_f().cpu().numpy()
    _f_after_steps_check(f_g, f_o, o.gross(), "cfg3 full size after %d steps" % steps)
    mo, mg = o.moments(), g.moments()
    for key in ("ne", "tot", "m2"):
        a, b = np.asarray(mo[key]), mg[key].numpy()
        assert np.all(np.abs(a - b) <= 1e-12 * np.maximum(np.abs(a), np.abs(a).max() * 1e-6)), key
    assert abs(float(mg["tot"][:, 0].sum()) - N0) <= 1e-12 * N0


def test_config3_full_size_dF_and_f_after_steps():
    """Config 3 at its BASELINE.json size (8^3 x 20^3 cells, 7 species, 2.6e8 samples per step): dF of steps 0 and 1 on
    every value, then f and the moments after 3 whole steps (collision + upwind streaming + Euler)."""
    _config3_run(3, (0, 1))


def test_config3_full_size_all_20_steps():
    """Config 3 for its own 20 steps (5.2e9 samples; the oracle needs ~3-5 min on 16 cores): f after the last step on every
    value, dF of the first and the last step."""
    _config3_run(wl.CONFIGS[3].steps, (0, 19))


# config 4's subset protocol: a fixed 64-cell subset -- the 4 x 4 x 4 block around the hot centre of the
# Gaussian -- and every 64th spatial cell
CFG4_BLOCK = [ix + 16 * (iy + 16 * iz) for iz in range(6, 10) for iy in range(6, 10) for ix in range(6, 10)]
CFG4_STRIDED = list(range(0, 4096, 64))


def _threaded(fn, items):
    import os
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=min(32, os.cpu_count() or 1)) as ex:   # ctypes releases the GIL; the calls only read the context
        return list(ex.map(fn, items))


def test_config4_full_size_subset_protocol():
    """Config 4 at full size (3.2 GB per copy, 3.6e9 samples per step), SURVEY.md 8d's protocol: the GPU runs whole
    steps; (1) sampled indices and (s, t, u) of EVERY sample of the 64-cell block and of every 64th cell are bit-exact;
    (2) on every step of a 3-step run the oracle is fed the GPU's f of the 64 block cells at the start of the step
    ("teacher forcing": the collision term is local in x) and its dF for those cells is compared value by value,
    with exact conservation per cell at 1e-13 of the gross deposit.  (The whole grid, streaming included, against the oracle:
    test_config4_full_size_whole_grid_one_step.)"""
    cfg = wl.CONFIGS[4]
    g = bz.Boltzmann(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax,
                     species=cfg.species, alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples)
    f0 = torch.from_numpy(wl.initial_f(cfg))
    g.set_f(f0)
    o = bzo.Oracle(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax,
                   species=cfg.species, alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples)
    deg = _deg(cfg)[0]
    degd = torch.from_numpy(_deg(cfg)).cuda()
    mom0 = g.moments()
    # (1) indices: kinematics do not depend on f; step = the last one of the config
    xs = sorted(set(CFG4_BLOCK) | set(CFG4_STRIDED))
    assert len(xs) == 128
    ref = _threaded(lambda x: o.debug_samples(cfg.steps - 1, x, 0, cfg.Np), xs)
    acc = 0.0
    for x, (co, so) in zip(xs, ref):
        cg, sg = g.debug_samples(cfg.steps - 1, x, 0, cfg.Np)
        assert np.array_equal(cg.cpu().numpy(), co), x
        assert np.array_equal(sg.cpu().numpy().view(np.uint64), so.view(np.uint64)), x
        acc += co[..., 3].mean()
    assert 0.3 < acc / len(xs) < 0.6                                       # S9: about 46 % of the samples deposit
    del ref
    # (2) dF with teacher forcing, every step
    for step in range(3):
        f_dev = g.get_f()
        dF_dev = g.collision(cfg.dt, step)
        tiles = [f_dev[x].cpu().numpy() for x in CFG4_BLOCK]
        res = _threaded(lambda q: o.collision_tile(cfg.dt, step, CFG4_BLOCK[q], tiles[q], want_gross=True), range(64))
        dF_host = dF_dev[CFG4_BLOCK].cpu().numpy()
        for q, x in enumerate(CFG4_BLOCK):
            dN, gross, m2 = res[q]
            dF_o, G = dN / deg, gross / deg
            assert np.abs(dF_o).max() > 0
            _assert_dF(dF_host[q], dF_o, G, "cfg4 xcell %d step %d" % (x, step))
            assert abs((deg * dF_host[q]).sum()) <= 1e-13 * gross.sum()      # Eq. 22-23 per spatial cell
        # the whole grid on the device: |sum N_a dF_a| against sum N_a |dF_a| <= the gross deposit
        num = float((dF_dev * degd).sum())
        den = float((dF_dev.abs() * degd).sum())
        assert abs(num) <= 1e-13 * den
        del f_dev, dF_dev
        g.step(cfg.dt)
    mom = g.moments()
    assert abs(float(mom["tot"][:, 0].sum()) - float(mom0["tot"][:, 0].sum())) <= 1e-12 * float(mom0["tot"][:, 0].sum())


def test_config4_full_size_whole_grid_one_step():
    """Config 4 at full size, ALL 4096 spatial cells (NS "f after N steps ... within 1e-11"): the
    streaming increment of the whole grid against bzo_stream, then one whole step (3.6e9 kinematic samples, upwind streaming,
    Euler) against bzo_step: every value of f at 1e-11 (S16), the moments at 1e-12.  The oracle's step takes 3-4 minutes on
    16 host cores."""
    cfg = wl.CONFIGS[4]
    o, g = _pair(cfg)
    f = wl.initial_f(cfg)
    o.set_f(f)
    g.set_f(torch.from_numpy(f))
    fmax = np.abs(f).max()
    d_o = o.stream(cfg.dt)
    d_g = g.stream(cfg.dt).cpu().numpy()
    assert np.abs(d_o).max() > 1e-6 * fmax
    d_g -= d_o
    assert np.abs(d_g).max() <= 1e-13 * fmax
    del d_o, d_g
    N0 = float(g.moments()["tot"][:, 0].sum())
    o.step(cfg.dt)
    g.step(cfg.dt)
    f_o, f_g = o.get_f(), g.get_f().cpu().numpy()
    assert np.abs(f_o - f).max() > 1e-6 * fmax
    del f
    _f_after_steps_check(f_g, f_o, o.gross(), "cfg4 whole grid, one step")
    del f_o, f_g
    mo, mg = o.moments(), g.moments()
    for key in ("ne", "tot", "m2"):
        a, b = np.asarray(mo[key]), mg[key].numpy()
        assert np.all(np.abs(a - b) <= 1e-12 * np.maximum(np.abs(a), np.abs(a).max() * 1e-6)), key
    assert abs(float(mg["tot"][:, 0].sum()) - N0) <= 1e-12 * N0
    g.close()
    o.close()


def test_edge_cases():
    # empty f: nothing is deposited, m^2 = 0 is never divided by because every bracket vanishes first
    cfg = wl.scaled(wl.CONFIGS[2], np_=6, samples=5)
    o, g = _pair(cfg)
    dF = g.collision(cfg.dt, 0).cpu().numpy()
    assert np.all(dF == 0.0)
    # ragged sample counts around the warp width, smallest grid, single quark species, generic species subset
    for species, np_, Ns in (((0,), 2, 1), ((3,), 5, 31), ((0, 1, 2), 7, 33), ((0, 2, 3, 6), 6, 65), ((1, 2, 5), 6, 64)):
        c = wl.scaled(wl.CONFIGS[2], np_=np_, samples=Ns, species=species)
        o, g = _pair(c)
        f = wl.random_f(c, seed=11)
        o.set_f(f)
        g.set_f(f)
        dF_o = o.collision(c.dt, 2)
        gross = o.gross()
        dF_g = g.collision(c.dt, 2).cpu().numpy()
        _assert_dF(dF_g, dF_o, gross, "species %s np %d Ns %d" % (species, np_, Ns))
        _assert_conserved(c, dF_g, gross)
    # fixed regulator mass and another seed
    c = wl.scaled(wl.CONFIGS[1], np_=8, samples=16, m_D=0.6, seed=12345)
    o, g = _pair(c)
    f = wl.random_f(c, seed=5)
    o.set_f(f)
    g.set_f(f)
    assert float(g.moments()["m2"][0]) == pytest.approx(0.36, rel=1e-15)
    _assert_dF(g.collision(c.dt, 0).cpu().numpy(), o.collision(c.dt, 0), o.gross(), "fixed m_D")
    # non-cubic spatial grid, two streams of calls on a user stream
    o = bzo.Oracle(nx=4, ny=2, nz=3, dx=0.3, np_=6, species=(0, 1, 2), samples=8, seed=1)
    g = bz.Boltzmann(nx=4, ny=2, nz=3, dx=0.3, np_=6, species=(0, 1, 2), samples=8, seed=1)
    s = torch.cuda.Stream()
    g.set_stream(s)
    f = np.random.default_rng(0).uniform(0.05, 0.5, size=o.shape)
    o.set_f(f)
    g.set_f(f)
    for _ in range(3):
        o.step(0.05)
        g.step(0.05)
    f_dev = g.get_f()                       # device copy enqueued on the context's stream s, not on torch's current one
    s.synchronize()                         # ... so s is synchronised AFTER get_f, before the tensor is read elsewhere
    f_o, f_g = o.get_f(), f_dev.cpu().numpy()
    assert np.abs(f_g - f_o).max() <= TOL_DF * np.abs(f_o).max()


# ---------------------------------------------------------------------------------------------- slabs
def _slab_kw(cfg, nz):
    return dict(nx=cfg.nx, ny=cfg.nx, nz=nz, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species,
                alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples)


@pytest.mark.parametrize("n_slabs", [1, 2, 3])
def test_slab_decomposition_matches_undecomposed_domain(n_slabs):
    """bz_set_slab + bz_copy_layers: the domain cut into z slabs with halo layers (several slabs run back to back on
    this one GPU, halo refresh in process) reproduces the undecomposed oracle: same sampled cells (the Philox spatial
    counter is the global cell index), f within the NS tolerance, totals within 1e-12."""
    from paper_1912_04457_b200 import slab
    cfg = wl.scaled(wl.CONFIGS[3], nx=4, np_=8, samples=16)
    nl = cfg.nx * cfg.nx
    o = bzo.Oracle(threads=8, **_slab_kw(cfg, cfg.nx))
    f0 = wl.random_f(cfg, seed=5)
    o.set_f(f0)
    doms = [slab.SlabDomain(lambda nz: bz.Boltzmann(**_slab_kw(cfg, nz)), cfg.nx, cfg.nx, cfg.nx, r, n_slabs)
            for r in range(n_slabs)]
    for d in doms:
        d.set_own(torch.from_numpy(f0[d.z0 * nl:d.z1 * nl].copy()).cuda())
    # sampled cells of a cell inside the last slab: local index differs from the global one, the samples must not
    d = doms[-1]
    xg = cfg.Nx - 2
    xl = xg - (d.z0 - 1) * nl
    co, so = o.debug_samples(2, xg, 0, cfg.Np)
    cg, sg = d.engine.debug_samples(2, xl, 0, cfg.Np)
    assert np.array_equal(cg.cpu().numpy(), co)
    assert np.array_equal(sg.cpu().numpy().view(np.uint64), so.view(np.uint64))
    steps = 3
    for _ in range(steps):
        o.step(cfg.dt)
        slab.exchange_in_process(doms)
        for d in doms:
            d.engine.step(cfg.dt)
    f_o = o.get_f()
    f_g = np.concatenate([d.get_own().cpu().numpy() for d in doms]).reshape(f_o.shape)
    assert np.abs(f_g - f_o).max() <= TOL_DF * np.abs(f_o).max()
    tot = sum(d.engine.moments()["tot"].numpy() for d in doms)
    assert np.allclose(tot, o.moments()["tot"], rtol=1e-12, atol=0)


def test_slab_halo_layers_do_not_collide():
    """dF_coll is exactly 0 in the halo layers and unchanged in the own layers."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=3, np_=8, samples=8)
    kw = _slab_kw(cfg, cfg.nx)
    a, b = bz.Boltzmann(**kw), bz.Boltzmann(**kw)
    f0 = wl.random_f(cfg, seed=9)
    a.set_f(f0)
    b.set_f(f0)
    b.set_slab(0, 1, 2)
    dA, dB = a.collision(cfg.dt, 0).cpu().numpy(), b.collision(cfg.dt, 0).cpu().numpy()
    nl = cfg.nx * cfg.nx
    assert not dB[:nl].any() and not dB[2 * nl:].any()
    assert np.abs(dB[nl:2 * nl] - dA[nl:2 * nl]).max() <= 1e-13 * np.abs(dA).max()
    with pytest.raises(bz.BzError):
        b.set_slab(0, 2, 1)


# ------------------------------------------------------------------------- user-defined matrix elements
@pytest.mark.parametrize("species,ovr", [
    ((0, 1, 2), {"QQGG": 1.0, "A": 0.0, "11": 0.0, "1B": 0.0, "ANN": 0.0, "QG": 0.0, "GG": 0.0}),   # the setting of pin P10
    ((0, 1, 2, 3, 4, 5, 6), {"GG": 40.0, "QG": 7.5, "ANN": 0.0}),                                  # some kinds, rest Table I
    ((1, 2, 3, 4, 5, 6), {"A": 3.0, "11": 5.0, "1B": 2.0}),
    ((0,), {"GG": 9.0}),                                                                           # pure-glue kernel
], ids=["p10", "mixture", "quarks", "glue"])
def test_msq_override_parity(species, ovr):
    """bz_set_msq_override: constant |M|^2 per kind of Table I on the GPU against the oracle's override hook (whose
    normalisation pin P10 checks against the closed form)."""
    cfg = wl.scaled(wl.CONFIGS[2], np_=9, samples=20)
    kw = dict(nx=1, ny=1, nz=1, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=species,
              alpha_s=cfg.alpha_s, m_D=0.7, seed=3, samples=cfg.samples)
    o, g = bzo.Oracle(threads=8, **kw), bz.Boltzmann(**kw)
    rng = np.random.Generator(np.random.Philox(key=11))
    f = 0.02 + 0.5 * rng.random((1, len(species), cfg.Np))
    o.set_f(f)
    g.set_f(f)
    for kind, v in ovr.items():
        o.set_msq_override(kind, v)
        g.set_msq_override(kind, v)
    dF_o = o.collision(cfg.dt, 1)
    dF_g = g.collision(cfg.dt, 1).cpu().numpy()
    _assert_dF(dF_g, dF_o, o.gross(), "override")
    assert np.abs(dF_o).max() > 0
    # restoring Table I gives the plain result again
    for kind in ovr:
        o.set_msq_override(kind, -1.0)
        g.set_msq_override(kind, -1.0)
    _assert_dF(g.collision(cfg.dt, 1).cpu().numpy(), o.collision(cfg.dt, 1), o.gross(), "restored")


def test_msq_sign_counts_against_the_oracle_channel_by_channel():
    """bz_msq_sign_counts (reading S8: the regulated Table I is evaluated literally and can be negative): the counters of
    every (kind, ordering) against the oracle, which evaluates bzo_msq for every depositing sample of the cells, and the
    (sample, channel) pair fraction that bench.py reports against a plain loop over the oracle's 127 ordered channels."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=2, np_=8, samples=12)
    o, g = _pair(cfg)
    f = wl.initial_f(cfg) + 0.05 * wl.random_f(cfg, seed=59)
    o.set_f(f)
    g.set_f(f)
    m2 = np.asarray(o.moments()["m2"])
    g4 = (4.0 * np.pi * cfg.alpha_s) ** 2
    step, xb, xe = 4, 1, 7
    acc_o, neg_o = 0, np.zeros((7, 2), dtype=np.int64)
    for x in range(xb, xe):
        cells, stu = o.debug_samples(step, x, 0, cfg.Np)
        for (s_, t_, u_) in stu[cells[..., 3] == 1]:
            acc_o += 1
            for kind in range(7):
                neg_o[kind, 0] += bzo.msq(kind, s_, t_, u_, m2[x], g4) < 0.0
                neg_o[kind, 1] += bzo.msq(kind, s_, u_, t_, m2[x], g4) < 0.0
    acc_g, neg_g = g.msq_sign_counts(step, xb, xe)
    assert acc_g == acc_o and acc_o > 1000
    assert np.array_equal(np.asarray(neg_g), neg_o)
    assert neg_o[4].min() > 0                                             # q qbar <-> g g does go negative (S8's example)
    # pair fraction: channel multiplicities from the product's table against the oracle's channel list, one by one
    mult = np.zeros((7, 2), dtype=np.int64)
    for row in bz.debug_paper_channels(cfg.species):
        mult[row[4], row[5]] += 1
    pairs_o = sum(neg_o[ch[4], ch[5]] for ch in o.channels())
    assert len(o.channels()) == mult.sum() == 127
    assert int((mult * np.asarray(neg_g)).sum()) == int(pairs_o)


# ------------------------------------------------- NEXT rank 2: thermal masses (Eq. 8-9) and Eq. 15 (drift + force)
VLASOV_CASES = [
    wl.scaled(wl.CONFIGS[3], nx=3, np_=10, samples=8),                 # 7 species, 27 spatial cells
    wl.scaled(wl.CONFIGS[4], nx=4, np_=7, samples=4),                  # odd momentum grid: the p = 0 cell
    wl.scaled(wl.CONFIGS[1], np_=6, samples=4),                        # quarks only, one spatial cell (own neighbour)
]


@pytest.mark.parametrize("cfg", VLASOV_CASES, ids=lambda c: c.name)
def test_thermal_masses_and_vlasov_parity(cfg):
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=21)
    o.set_f(f0)
    g.set_f(f0)
    # first evaluation: E = |p|; second: massive energies of the first
    for _ in range(3):
        mo, mg = o.thermal_masses(), g.thermal_masses().numpy()
        assert np.allclose(mg, mo, rtol=1e-12, atol=0)
    assert (mo[:, 0] > 0).all()
    # Eq. 15 with spatially varying masses
    rng = np.random.Generator(np.random.Philox(key=5))
    masses = 0.05 + rng.random((cfg.Nx, 4))
    if cfg.np_ % 2 == 1:
        masses[::3] = 0.0                                           # m = 0 cells: E = 0 at p = 0 (S10)
    o.set_masses(masses)
    g.set_masses(masses)
    dF_o, dF_g = o.vlasov(cfg.dt), g.vlasov(cfg.dt).cpu().numpy()
    if cfg.Nx == 1:
        assert not dF_o.any() and np.abs(dF_g).max() <= 1e-15        # homogeneous: a cell is its own neighbour
        return
    assert np.abs(dF_o).max() > 0
    assert np.abs(dF_g - dF_o).max() <= 1e-13 * np.abs(dF_o).max()
    for a in range(cfg.S):                                           # Eq. 13: nothing is created
        assert abs(dF_g[:, a].sum()) <= 1e-12 * np.abs(dF_g[:, a]).sum()


@pytest.mark.parametrize("scheme", [1, 2])
def test_step_with_eq15_transport(scheme):
    cfg = wl.scaled(wl.CONFIGS[3], nx=3, np_=8, samples=16)
    o, g = _pair(cfg)
    f0 = wl.initial_f(cfg) + 0.01
    for e in (o, g):
        e.set_f(f0)
        e.set_transport(scheme)
        if scheme == 2:
            e.set_masses(np.full((cfg.Nx, 4), 0.5))                  # constant m^2 = 0.5 GeV^2 as in Fig. 5
    for _ in range(4):
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o, f_g = o.get_f(), g.get_f().cpu().numpy()
    assert np.abs(f_g - f_o).max() <= 1e-11 * np.abs(f_o).max()
    mo, mg = o.moments(), g.moments()
    assert np.allclose(mg["tot"].numpy(), mo["tot"], rtol=1e-12, atol=0)
    if scheme == 1:
        assert np.allclose(g.thermal_masses().numpy(), o.thermal_masses(), rtol=1e-11, atol=0)
    # total particle number: conserved by the collision term (Eq. 22) and by Eq. 13's flux form
    N0 = None
    o2 = bzo.Oracle(threads=1, nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax,
                    species=cfg.species)
    o2.set_f(f0)
    N0 = o2.moments()["tot"][:, 0].sum()
    assert mg["tot"][:, 0].sum().item() == pytest.approx(N0, rel=1e-12)


# ------------------------------------------------------------------------------- bz_step_host (pipelined end to end)
@pytest.mark.parametrize("cfg", [wl.scaled(wl.CONFIGS[3], nx=5, np_=8, samples=16),      # 5 z layers: 5 chunks
                                 wl.scaled(wl.CONFIGS[4], nx=3, np_=7, samples=9),       # 3 chunks, odd grid
                                 wl.scaled(wl.CONFIGS[2], np_=8, samples=16)],           # 1 layer: the plain sequence
                         ids=lambda c: c.name)
def test_step_host_matches_oracle(cfg):
    """bz_step_host (host f in, one step, host f out, chunks of z layers pipelined over three streams) against the oracle,
    and the context is left as after bz_set_f + bz_step: a following bz_step continues from it."""
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=13)
    o.set_f(f0)
    hin = torch.from_numpy(f0.copy()).pin_memory()
    hout = torch.empty_like(hin).pin_memory()
    for _ in range(2):
        o.step(cfg.dt)
        g.step_host(cfg.dt, hin, hout)
        f_o = o.get_f()
        assert np.abs(hout.numpy() - f_o).max() <= TOL_DF * np.abs(f_o).max()
        hin.copy_(hout)
    assert np.array_equal(g.get_f().cpu().numpy(), hout.numpy())
    o.step(cfg.dt)
    g.step(cfg.dt)
    f_o = o.get_f()
    assert np.abs(g.get_f().cpu().numpy() - f_o).max() <= TOL_DF * np.abs(f_o).max()
    assert np.allclose(g.moments()["tot"].numpy(), o.moments()["tot"], rtol=1e-12, atol=0)


# ------------------------------------------------------------------ NEXT rank 1: the paper's own sampler (Eq. 17-21)
PAPER_TUPLES = [(0.0, 0.0, 0.0, 0.0), (0.5, 0.5, 0.5, 0.5), (0.3, 0.9, 0.3, 0.9), (0.9, 0.3, 0.3, 0.9), (0.0, 0.7, 0.0, 0.7)]


@pytest.mark.parametrize("cfg", [wl.scaled(wl.CONFIGS[2], np_=9, samples=40), wl.scaled(wl.CONFIGS[3], nx=2, np_=8, samples=33)],
                         ids=lambda c: c.name)
def test_paper_sampler_roots_bit_exact(cfg):
    """Cells of k1, k2, k3, the number of roots kept and (s, t, u) of every root: bit-exact against the oracle."""
    o, g = _pair(cfg)
    xcell = cfg.Nx - 1
    for msq in PAPER_TUPLES:
        cells, stu = g.debug_paper_samples(5, xcell, 0, cfg.Np, msq)
        cells, stu = cells.cpu().numpy(), stu.cpu().numpy()
        n_roots = 0
        for pc in range(0, cfg.Np, 7):
            for smp in range(cfg.samples):
                _, i3, roots = o.paper_sample(5, xcell, pc, smp, msq)
                row, srow = cells[pc, smp], stu[pc, smp]
                assert row[0] == i3 and row[1] == len(roots), (msq, pc, smp)
                for r, R in enumerate(roots):
                    assert (row[2 + 2 * r], row[3 + 2 * r]) == (R.i1, R.i2)
                    assert np.array_equal(srow[3 * r:3 * r + 3].view(np.uint64), np.array([R.s, R.t, R.u]).view(np.uint64))
                    n_roots += 1
        assert n_roots > 200


@pytest.mark.parametrize("cfg,massive", [(wl.scaled(wl.CONFIGS[0], np_=9, samples=24), False),
                                         (wl.scaled(wl.CONFIGS[1], np_=8, samples=12), True),
                                         (wl.scaled(wl.CONFIGS[2], np_=7, samples=10), True),
                                         (wl.scaled(wl.CONFIGS[3], nx=2, np_=6, samples=6), True)],
                         ids=["glue_massless", "quarks_massive", "mixture_massive", "inhom_massive"])
def test_paper_sampler_dF_parity_and_conservation(cfg, massive):
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=31)
    o.set_f(f0)
    g.set_f(f0)
    if massive:
        mo, mg = o.thermal_masses(), g.thermal_masses().numpy()
        assert np.allclose(mg, mo, rtol=1e-12, atol=0)
        g.set_masses(mo)                      # identical bits on both sides: the roots depend on them
    dF_o = o.collision_paper(cfg.dt, 2)
    dF_g = g.collision_paper(cfg.dt, 2).cpu().numpy()
    gross = o.gross()
    assert np.abs(dF_o).max() > 0
    _assert_dF(dF_g, dF_o, gross, "paper sampler")
    _assert_conserved(cfg, dF_g, gross)


def test_eq15_and_thermal_masses_full_size_config3():
    """NEXT rank 2 at the full size of config 3 (8^3 x 20^3 cells, 7 species: 28.7 M values), the launch configuration
    bench.py probes: thermal masses over two iterations and the Eq. 15 increment, every value against the oracle."""
    cfg = wl.CONFIGS[3]
    o, g = _pair(cfg, threads=16)
    f0 = wl.initial_f(cfg) + 1e-3 * wl.random_f(cfg, seed=2)
    o.set_f(f0)
    g.set_f(f0)
    for _ in range(2):
        mo, mg = o.thermal_masses(), g.thermal_masses().numpy()
        assert np.allclose(mg, mo, rtol=1e-12, atol=0)
    g.set_masses(mo)
    dF_o, dF_g = o.vlasov(cfg.dt), g.vlasov(cfg.dt).cpu().numpy()
    assert np.abs(dF_g - dF_o).max() <= 1e-13 * np.abs(dF_o).max()


def test_paper_sampler_roots_bit_exact_on_the_config4_momentum_grid():
    """NEXT rank 1 on config 4's momentum grid (24^3 over [-4, 4] GeV, 64 samples per cell), sampled grid points of a
    spatial cell with a non-zero Philox offset: cells and (s, t, u) of every root bit-exact."""
    cfg = wl.scaled(wl.CONFIGS[4], nx=2)
    o, g = _pair(cfg)
    o.set_slab(4090, 0, 2)
    g.set_slab(4090, 0, 2)
    msq = (0.21, 0.093, 0.21, 0.093)
    for pb in (0, 6911, 13800):
        cells, stu = g.debug_paper_samples(9, 5, pb, pb + 8, msq)
        cells, stu = cells.cpu().numpy(), stu.cpu().numpy()
        for k in range(8):
            for smp in range(cfg.samples):
                _, i3, roots = o.paper_sample(9, 5, pb + k, smp, msq)
                assert cells[k, smp, 0] == i3 and cells[k, smp, 1] == len(roots)
                for r, R in enumerate(roots):
                    assert (cells[k, smp, 2 + 2 * r], cells[k, smp, 3 + 2 * r]) == (R.i1, R.i2)
                    assert np.array_equal(stu[k, smp, 3 * r:3 * r + 3].view(np.uint64), np.array([R.s, R.t, R.u]).view(np.uint64))


@pytest.mark.parametrize("which", ["paper", "is", "box"])
def test_next_kernels_dF_parity_on_the_config4_momentum_grid(which):
    """The NEXT-row collision kernels in the launch geometry bench.py probes -- config 4's momentum grid (24^3 cells over
    [-4, 4] GeV, 64 samples per cell) and 64 spatial cells in one launch, so that the paper kernel runs its 8 CTA groups with
    rings that wrap thousands of times and the weighted samplers their full persistent grid: dF of four spatial cells against
    the oracle, value by value at 1e-11 (S16), with conservation per cell at 1e-13 of the gross deposit (Eq. 22).  The oracle
    runs one spatial cell at a time with that cell's f, global index and, for the paper's sampler (Eq. 17-21), its four
    distinct thermal masses: the collision term is local in x."""
    import os
    cfg = wl.scaled(wl.CONFIGS[4], nx=4)
    kw = dict(dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species, alpha_s=cfg.alpha_s, m_D=cfg.m_D,
              seed=cfg.seed, samples=cfg.samples)
    g = bz.Boltzmann(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, **kw)
    o = bzo.Oracle(nx=1, ny=1, nz=1, threads=min(16, os.cpu_count() or 1), **kw)
    f0 = wl.initial_f(cfg) + 0.05 * wl.random_f(cfg, seed=47)
    g.set_f(f0)
    rng = np.random.Generator(np.random.Philox(key=53))
    masses = 0.05 + 0.5 * rng.random((cfg.Nx, 4))                          # m_g^2, m_u^2, m_d^2, m_s^2: all different, per cell
    step = 2
    if which == "paper":
        g.set_masses(masses)
        dF = g.collision_paper(cfg.dt, step)
    else:
        dF = (g.collision_is if which == "is" else g.collision_box)(cfg.dt, step)
    deg = _deg(cfg)[0]
    for x in (0, 21, 42, 63):
        o.set_slab(x, 0, 1)                                               # the cell draws the samples of its global index
        o.set_f(f0[x][None])
        if which == "paper":
            o.set_masses(masses[x:x + 1])
        dF_o = {"paper": o.collision_paper, "is": o.collision_is, "box": o.collision_box}[which](cfg.dt, step)[0]
        G = o.gross()[0]
        dF_g = dF[x].cpu().numpy()
        assert np.abs(dF_o).max() > 0
        _assert_dF(dF_g, dF_o, G, "%s, xcell %d" % (which, x))
        assert abs((deg * dF_g).sum()) <= 1e-13 * (deg * G).sum()
    degd = torch.from_numpy(_deg(cfg)).cuda()
    assert abs(float((dF * degd).sum())) <= 1e-13 * float((dF.abs() * degd).sum())      # the whole launch


def test_step_with_the_importance_sampled_collision_term():
    """bz_set_collision(2): bz_step with bz_collision_is; f after 3 steps against the oracle."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=2, np_=7, samples=12)
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=43) * 0.5
    for e in (o, g):
        e.set_f(f0)
        e.set_collision(2)
    for _ in range(3):
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o = o.get_f()
    assert np.abs(g.get_f().cpu().numpy() - f_o).max() <= 1e-11 * np.abs(f_o).max()
    assert np.allclose(g.moments()["tot"].numpy(), o.moments()["tot"], rtol=1e-12, atol=0)


@pytest.mark.parametrize("scheme", [0, 1, 2])
def test_step_with_the_papers_collision_term(scheme):
    """bz_set_collision(1): bz_step with the paper's sampler; with transport scheme 1 this is the paper's program as a
    whole (masses from the old f, Eq. 17-21, Eq. 15, forward Euler).  f after 3 steps against the oracle."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=2, np_=6, samples=6)
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=41) * 0.5
    for e in (o, g):
        e.set_f(f0)
        e.set_collision(1)
        e.set_transport(scheme)
        if scheme == 2:
            e.set_masses(np.tile([0.5, 0.2, 0.25, 0.3], (cfg.Nx, 1)))
    for _ in range(3):
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o, f_g = o.get_f(), g.get_f().cpu().numpy()
    assert np.abs(f_o - f0).max() > 0
    assert np.abs(f_g - f_o).max() <= 1e-11 * np.abs(f_o).max()
    mo, mg = o.moments(), g.moments()
    assert np.allclose(mg["tot"].numpy(), mo["tot"], rtol=1e-12, atol=0)
    # back to the hot path: the cell-major copy is rebuilt and the next step is the CM sampler's again
    for e in (o, g):
        e.set_collision(0)
        e.set_transport(0)
    o.step(cfg.dt)
    g.step(cfg.dt)
    f_o = o.get_f()
    assert np.abs(g.get_f().cpu().numpy() - f_o).max() <= 1e-11 * np.abs(f_o).max()


def test_energy_balance_diagnostic_parity():
    """bz_energy_diag (Eq. 11-12, 26) against the oracle, massless and with spatially varying masses, odd grid."""
    cfg = wl.scaled(wl.CONFIGS[4], nx=3, np_=9, samples=4)
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=3)
    o.set_f(f0)
    g.set_f(f0)
    assert np.allclose(g.energy_diag().numpy(), o.energy_diag(), rtol=1e-12, atol=0)
    rng = np.random.Generator(np.random.Philox(key=2))
    masses = rng.random((cfg.Nx, 4))
    masses[::4] = 0.0
    o.set_masses(masses)
    g.set_masses(masses)
    d_o, d_g = o.energy_diag(), g.energy_diag().numpy()
    assert np.allclose(d_g, d_o, rtol=1e-12, atol=0) and (d_o > 0).all()


# ------------------------------------------------------------ NEXT rank 3: importance sampling of the t/u-channel peaks
@pytest.mark.parametrize("cfg", [wl.scaled(wl.CONFIGS[2], np_=9, samples=40), wl.scaled(wl.CONFIGS[4], nx=2, np_=24, samples=33)],
                         ids=lambda c: c.name)
def test_importance_sampler_cells_bit_exact(cfg):
    """Cells of p2, p3, p4, the flag, (s, t, u) and the weight of every importance-sampled sample: bit-exact."""
    o, g = _pair(cfg)
    xcell = cfg.Nx - 1
    for m2 in (0.04, 0.7, 0.0):
        pb, pe = (0, cfg.Np) if cfg.Np < 1000 else (6900, 6930)
        cells, stu, w = (t.cpu().numpy() for t in g.debug_samples_is(7, xcell, pb, pe, m2))
        for pc in range(pb, pe, 5):
            for smp in range(cfg.samples):
                sm, wt = o.sample_one_is(7, xcell, pc, smp, m2)
                row = cells[pc - pb, smp]
                assert tuple(row) == (sm.j, sm.k, sm.l, sm.flag), (m2, pc, smp)
                if sm.s > 0:
                    assert np.array_equal(stu[pc - pb, smp].view(np.uint64), np.array([sm.s, sm.t, sm.u]).view(np.uint64))
                    assert np.array([w[pc - pb, smp]]).view(np.uint64)[0] == np.array([wt]).view(np.uint64)[0]


@pytest.mark.parametrize("cfg,m_D", [(wl.scaled(wl.CONFIGS[0], np_=9, samples=40), 0.3),
                                     (wl.scaled(wl.CONFIGS[2], np_=8, samples=33), 0.0),
                                     (wl.scaled(wl.CONFIGS[3], nx=2, np_=7, samples=24), 0.5)],
                         ids=["glue_fixed", "mixture_from_f", "inhom_fixed"])
def test_importance_sampler_dF_parity_and_conservation(cfg, m_D):
    import dataclasses
    cfg = dataclasses.replace(cfg, m_D=m_D)
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=17)
    o.set_f(f0)
    g.set_f(f0)
    dF_o = o.collision_is(cfg.dt, 3)
    dF_g = g.collision_is(cfg.dt, 3).cpu().numpy()
    gross = o.gross()
    assert np.abs(dF_o).max() > 0
    _assert_dF(dF_g, dF_o, gross, "importance sampler")
    _assert_conserved(cfg, dF_g, gross)


# ------------------------------------------------------------ NEXT rank 3, other half: in-box sampling of the CM direction
@pytest.mark.parametrize("cfg", [wl.scaled(wl.CONFIGS[2], np_=9, samples=40), wl.scaled(wl.CONFIGS[4], nx=2, np_=24, samples=33),
                                 wl.scaled(wl.CONFIGS[0], np_=15, samples=64, pmin=-1.0, pmax=4.0)],
                         ids=["mix9", "cfg4_grid", "off_centre_box"])
def test_inbox_sampler_cells_bit_exact(cfg):
    """Cells of p2, p3, p4, the flag, (s, t, u) and the weight beta of every in-box sample: bit-exact."""
    o, g = _pair(cfg)
    xcell = cfg.Nx - 1
    pb, pe = (0, cfg.Np) if cfg.Np < 1000 else (cfg.Np // 2 - 12, cfg.Np // 2 + 48)
    cells, stu, w = (t.cpu().numpy() for t in g.debug_samples_box(7, xcell, pb, pe))
    n_acc = n_all = 0
    for pc in range(pb, pe, 3):
        for smp in range(cfg.samples):
            sm, wt = o.sample_one_box(7, xcell, pc, smp)
            row = cells[pc - pb, smp]
            assert tuple(row) == (sm.j, sm.k, sm.l, sm.flag), (pc, smp)
            assert np.array_equal(stu[pc - pb, smp].view(np.uint64), np.array([sm.s, sm.t, sm.u]).view(np.uint64))
            assert np.array([w[pc - pb, smp]]).view(np.uint64)[0] == np.array([wt]).view(np.uint64)[0]
            n_acc += sm.flag
            n_all += 1
    assert n_all > 600 and n_acc > 0.6 * n_all


@pytest.mark.parametrize("cfg", [wl.scaled(wl.CONFIGS[0], np_=9, samples=40),
                                 wl.scaled(wl.CONFIGS[2], np_=8, samples=33),
                                 wl.scaled(wl.CONFIGS[3], nx=2, np_=7, samples=24),
                                 wl.scaled(wl.CONFIGS[1], np_=8, samples=20)],
                         ids=["glue", "mixture", "inhom", "quarks"])
def test_inbox_sampler_dF_parity_and_conservation(cfg):
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=19)
    o.set_f(f0)
    g.set_f(f0)
    dF_o = o.collision_box(cfg.dt, 3)
    dF_g = g.collision_box(cfg.dt, 3).cpu().numpy()
    gross = o.gross()
    assert np.abs(dF_o).max() > 0
    _assert_dF(dF_g, dF_o, gross, "in-box sampler")
    _assert_conserved(cfg, dF_g, gross)
    # the hot path right after it: the sampler is a per-call choice, nothing sticks to the context
    _assert_dF(g.collision(cfg.dt, 3).cpu().numpy(), o.collision(cfg.dt, 3), o.gross(), "hot path after in-box")


def test_step_with_the_inbox_collision_term():
    """bz_set_collision(3): bz_step with the in-box estimator; f after 3 steps against the oracle."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=2, np_=7, samples=12)
    o, g = _pair(cfg)
    f0 = wl.random_f(cfg, seed=47) * 0.5
    for e in (o, g):
        e.set_f(f0)
        e.set_collision(3)
    for _ in range(3):
        o.step(cfg.dt)
        g.step(cfg.dt)
    f_o = o.get_f()
    assert np.abs(g.get_f().cpu().numpy() - f_o).max() <= 1e-11 * np.abs(f_o).max()
    assert np.allclose(g.moments()["tot"].numpy(), o.moments()["tot"], rtol=1e-12, atol=0)


# --------------------------------------------------------------------------------- bz_step_n (captured CUDA graph)
@pytest.mark.parametrize("cfg,n", [(wl.CONFIGS[0], 10), (wl.scaled(wl.CONFIGS[2], np_=12, samples=40), 7),
                                   (wl.scaled(wl.CONFIGS[3], nx=3, np_=8, samples=16), 6), (wl.scaled(wl.CONFIGS[1], np_=10, samples=33), 1)],
                         ids=["cfg0_full", "mix12", "inhom3", "quarks_one_step"])
def test_step_n_matches_oracle_and_step_loop(cfg, n):
    """bz_step_n(n): n Euler steps replayed from a captured CUDA graph (device-resident Philox step word) against the
    oracle's n steps; then bz_step continues from the same state and step counter, and a second bz_step_n reuses the graph."""
    o, g = _pair(cfg)
    f = wl.initial_f(cfg) + 0.01 * wl.random_f(cfg, seed=23)
    o.set_f(f)
    g.set_f(f)
    g.step_n(cfg.dt, n)
    for _ in range(n):
        o.step(cfg.dt)
    _f_after_steps_check(g.get_f().cpu().numpy(), o.get_f(), o.gross(), "step_n(%d)" % n)
    o.step(cfg.dt)
    g.step(cfg.dt)                                                         # the host step counter moved with the device's
    _f_after_steps_check(g.get_f().cpu().numpy(), o.get_f(), o.gross(), "step after step_n")
    g.step_n(cfg.dt, 4)
    for _ in range(4):
        o.step(cfg.dt)
    f_o, f_g = o.get_f(), g.get_f().cpu().numpy()
    _f_after_steps_check(f_g, f_o, o.gross(), "second step_n")
    mo, mg = o.moments(), g.moments()
    for key in ("ne", "tot", "m2"):
        a, b = np.asarray(mo[key]), mg[key].numpy()
        assert np.all(np.abs(a - b) <= 1e-12 * np.maximum(np.abs(a), np.abs(a).max() * 1e-6)), key


def test_step_n_with_odd_n_keeps_one_graph_per_buffer_parity():
    """Calls of bz_step_n with an odd n start from alternating buffers (the single ordinary step in front swaps f and f_new):
    each parity has its own instantiated graph, so the third and fourth call replay what the first two captured.  The launch
    counter sees 3 kernels for the ordinary step and 6 per replayed pair -- a capture enqueues nothing and counts nothing --
    and the state after 4 x 5 steps is the oracle's after 20."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=2, np_=8, samples=16)
    o, g = _pair(cfg)
    f = wl.initial_f(cfg) + 0.01 * wl.random_f(cfg, seed=31)
    o.set_f(f)
    g.set_f(f)
    g.step(cfg.dt)                                                         # the cell-major copy exists from here on (no pack launch below)
    o.step(cfg.dt)
    for call in range(4):
        before = bz.launch_count()
        g.step_n(cfg.dt, 5)
        assert bz.launch_count() - before == 3 + 2 * 6, call
        for _ in range(5):
            o.step(cfg.dt)
    _f_after_steps_check(g.get_f().cpu().numpy(), o.get_f(), o.gross(), "4 x step_n(5)")
    assert np.allclose(g.moments()["tot"].numpy(), o.moments()["tot"], rtol=1e-12, atol=0)


def test_checkpoint_restart_continues_the_run():
    """bz_get_f + (seed, step) is a complete checkpoint.  A run of 6 steps against one that is stopped after 3,
    read out to the host, and continued in a NEW context from bz_set_f + bz_set_step: same f (the two differ only in the
    order of the deposits' sums), same moments, and both equal to the oracle's uninterrupted 6 steps."""
    cfg = wl.scaled(wl.CONFIGS[3], nx=3, np_=8, samples=16)
    o, a = _pair(cfg)
    f = wl.initial_f(cfg) + 0.01 * wl.random_f(cfg, seed=37)
    o.set_f(f)
    a.set_f(f)
    for _ in range(6):
        o.step(cfg.dt)
        a.step(cfg.dt)
    _, b = _pair(cfg, threads=1)
    b.set_f(f)
    for _ in range(3):
        b.step(cfg.dt)
    saved = torch.empty(b.shape, dtype=torch.float64)
    b.get_f(saved)                                                         # the checkpoint: f on the host; seed and step are the caller's
    b.close()
    _, c = _pair(cfg, threads=1)                                           # a fresh context: seed from the config, step counter 0
    c.set_f(saved)
    c.set_step(3)
    for _ in range(3):
        c.step(cfg.dt)
    f_a, f_c, f_o = a.get_f().cpu().numpy(), c.get_f().cpu().numpy(), o.get_f()
    _f_after_steps_check(f_c, f_o, o.gross(), "restarted run")
    assert np.abs(f_c - f_a).max() <= TOL_DF * np.abs(f_a).max()
    assert np.allclose(c.moments()["tot"].numpy(), a.moments()["tot"].numpy(), rtol=1e-12, atol=0)
    c.set_step(0)                                                          # the wrong step word draws other samples: the checkpoint needs it
    c.set_f(saved)
    for _ in range(3):
        c.step(cfg.dt)
    assert np.abs(c.get_f().cpu().numpy() - f_a).max() > 1e3 * TOL_DF * np.abs(f_a).max()


def test_slab_step_host_on_one_gpu():
    """SlabDomain.step_host (the end-to-end leg of the slab path: boundary layers up, halo exchange, bz_step_host over the
    own layers of a slab context) with world = 1 against the oracle on the undecomposed periodic domain."""
    from paper_1912_04457_b200 import slab
    cfg = wl.scaled(wl.CONFIGS[3], nx=4, np_=8, samples=16)
    nl = cfg.nx * cfg.nx
    o = bzo.Oracle(threads=8, **_slab_kw(cfg, cfg.nx))
    f0 = wl.random_f(cfg, seed=29)
    o.set_f(f0)
    dom = slab.SlabDomain(lambda nz: bz.Boltzmann(**_slab_kw(cfg, nz)), cfg.nx, cfg.nx, cfg.nx, 0, 1)
    f_local = np.zeros(((cfg.nx + 2) * nl, cfg.S, cfg.Np))
    f_local[nl:-nl] = f0
    hin = torch.from_numpy(f_local).pin_memory()
    hout = torch.zeros_like(hin).pin_memory()
    for _ in range(3):
        o.step(cfg.dt)
        dom.step_host(cfg.dt, hin, hout)
        f_o = o.get_f()
        got = hout.numpy()[nl:-nl]
        assert np.abs(got - f_o).max() <= TOL_DF * np.abs(f_o).max()
        assert not hout.numpy()[:nl].any() and not hout.numpy()[-nl:].any()      # halo layers of the host buffer are not written
        hin.copy_(hout)
    assert np.allclose(dom.moments_totals().numpy(), o.moments()["tot"], rtol=1e-12, atol=0)


# --------------------------------------------------------------------------------- long runs: properties at full size
def _entropy(f, cfg):
    """s = - sum_a N_a sum_p [ f ln f -+ (1 +- f) ln(1 +- f) ]  (Bose: upper signs, Fermi: lower), in units of d3p/(2 pi)^3"""
    tot = 0.0
    for a, sid in enumerate(cfg.species):
        x = f[:, a, :].clamp(min=1e-300)
        if sid == 0:
            s = -(x * x.log() - (1.0 + x) * (1.0 + x).log())
        else:
            y = (1.0 - f[:, a, :]).clamp(min=1e-300)
            s = -(x * x.log() + y * y.log())
        tot += NDEG[sid] * float(s.sum())
    return tot


@pytest.mark.parametrize("k,steps", [(0, 1000), (1, 2000)], ids=["cfg0_1000_steps", "cfg1_2000_steps"])
def test_long_run_properties_full_size(k, steps):
    """The regime of the paper's own runs (10^4-10^6 steps of one spatial cell): config 0 and config 1 at full size
    for 1000 / 2000 steps through bz_step_n (captured graph, no host round trip per step).  What holds at any length: total
    particle number (Eq. 22-23) and, for quarks, the net number of every flavour are conserved to rounding; f stays finite
    and inside the Pauli bound; the entropy of the binned distribution grows (H theorem of Eq. 5's gain - loss bracket).
    Energy is not asserted: deposits at cell centres conserve it only up to the cell size (the paper's Fig. 5, P:262-275:
    1.5 % at 30^3 after 1 fm/c; on config 0's 15^3 grid it doubles within 10 fm/c -- a property of the method: the first
    10 of these steps agree with the oracle value by value, test_f_after_all_steps_full_size_homogeneous)."""
    cfg = wl.CONFIGS[k]
    _, g = _pair(cfg, threads=1)
    f0 = torch.from_numpy(wl.initial_f(cfg))
    g.set_f(f0)
    m0 = g.moments()
    s_prev = _entropy(g.get_f(), cfg)
    s_first = s_prev
    for _ in range(5):
        g.step_n(cfg.dt, steps // 5)
        f = g.get_f()
        assert bool(torch.isfinite(f).all())
        s_now = _entropy(f, cfg)
        assert s_now > s_prev * (1.0 - 1e-4), (s_prev, s_now)
        s_prev = s_now
    assert s_prev > s_first * 1.01                                   # the step function has relaxed
    m1 = g.moments()
    n0, n1 = m0["tot"][:, 0].numpy(), m1["tot"][:, 0].numpy()
    assert abs(n1.sum() - n0.sum()) <= 1e-11 * n0.sum()
    if k == 1:
        for fl in range(3):                                          # N_q - N_qbar per flavour (species order u, ubar, d, dbar, s, sbar)
            assert abs((n1[2 * fl] - n1[2 * fl + 1]) - (n0[2 * fl] - n0[2 * fl + 1])) <= 1e-11 * n0.sum()
        assert float(f.max()) <= 1.0 + 1e-9 and float(f.min()) >= -1e-3
    e0, e1 = m0["tot"][:, 1].numpy().sum(), m1["tot"][:, 1].numpy().sum()
    print("long run %s: N %.12g -> %.12g, E %.6g -> %.6g, entropy %.6g -> %.6g" % (cfg.name, n0.sum(), n1.sum(), e0, e1, s_first, s_prev))


# --------------------------------------------------------------------------------- maximum size
def test_papers_largest_grid_on_one_gpu():
    """The largest grid the paper's program handles "on GPU clusters" (20^3 spatial x 40^3 momentum cells) with all
    seven species on ONE B200: 3.58e9 values, 123 GB of context (f, f_new, the two cell-major copies), 3.3e10 samples per step.
    Dense seeded random f generated on the device (the host never holds a copy).  Checked: sampled cells and (s, t, u) bit
    exact and dF within 1e-11 (S16) with conservation at 1e-13 of the gross deposit on the first, a middle and the last
    spatial cell -- the oracle runs one spatial cell at a time with that cell's f and global index (the collision term is
    local in x) -- conservation on the whole grid, and total particle number through a full step."""
    cfg = wl.PAPER_LARGEST
    import gc
    gc.collect()                                                      # contexts and tensors of the tests before this one
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 165e9:
        pytest.skip("needs 165 GB of free device memory, found %.0f GB" % (free / 1e9))
    kw = dict(dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species, alpha_s=cfg.alpha_s, m_D=cfg.m_D,
              seed=cfg.seed, samples=cfg.samples)
    g = bz.Boltzmann(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, **kw)
    gen = torch.Generator(device="cuda")
    gen.manual_seed(7)
    f = torch.empty(g.shape, dtype=torch.float64, device="cuda")
    for x0 in range(0, g.Nx, 250):
        f[x0:x0 + 250] = 0.02 + 0.58 * torch.rand((250,) + g.shape[1:], dtype=torch.float64, device="cuda", generator=gen)
    g.set_f(f)
    torch.cuda.synchronize()
    xs = (0, g.Nx // 2 + 3, g.Nx - 1)
    tiles = {x: f[x].cpu().numpy() for x in xs}
    del f
    torch.cuda.empty_cache()
    n0 = float(g.moments()["tot"][:, 0].sum())
    dF = torch.empty(g.shape, dtype=torch.float64, device="cuda")
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    g.collision(cfg.dt, 0, out=dF)
    e1.record()
    torch.cuda.synchronize()
    print("largest grid: bz_collision %.0f ms, %.3e samples/s" % (e0.elapsed_time(e1), cfg.samples_per_step / e0.elapsed_time(e1) * 1e3))
    deg = _deg(cfg)[0]
    o = bzo.Oracle(nx=1, ny=1, nz=1, threads=min(16, __import__("os").cpu_count() or 1), **kw)
    for x in xs:
        o.set_slab(x, 0, 1)                                           # the cell draws the samples of its global index
        o.set_f(tiles[x][None])
        dF_o, G = o.collision(cfg.dt, 0)[0], o.gross()[0]
        dF_g = dF[x].cpu().numpy()
        _assert_dF(dF_g, dF_o, G, "largest grid, xcell %d" % x)
        assert abs((deg * dF_g).sum()) <= 1e-13 * (deg * G).sum()
        co, so = o.debug_samples(3, 0, 31000, 31064)
        cg, sg = g.debug_samples(3, x, 31000, 31064)
        assert np.array_equal(cg.cpu().numpy(), co) and np.array_equal(sg.cpu().numpy().view(np.uint64), so.view(np.uint64)), x
    degd = torch.from_numpy(_deg(cfg)).cuda()
    num = sum(float((dF[x0:x0 + 250] * degd).sum()) for x0 in range(0, g.Nx, 250))
    den = sum(float((dF[x0:x0 + 250].abs() * degd).sum()) for x0 in range(0, g.Nx, 250))
    assert abs(num) <= 1e-13 * den
    del dF
    torch.cuda.empty_cache()
    g.step(cfg.dt)
    n1 = float(g.moments()["tot"][:, 0].sum())
    assert abs(n1 - n0) <= 1e-12 * n0
    g.close()


def test_step_host_pieces_full_size_config4():
    """bz_step_host at config 4's full size, where its pipeline cuts the first and the last z chunk into quarters (22 pieces):
    the end-to-end step from pinned host memory against the resident bz_step of a second context on the same input (itself
    checked against the oracle by the subset protocol above).  The two differ only in the order of the deposits' sums."""
    cfg = wl.CONFIGS[4]
    kw = dict(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species,
              alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples)
    f0 = torch.from_numpy(wl.initial_f(cfg))
    hin = f0.pin_memory()
    hout = torch.empty_like(f0).pin_memory()
    a, b = bz.Boltzmann(**kw), bz.Boltzmann(**kw)
    a.set_f(hin)
    for _ in range(2):
        a.step(cfg.dt)
        b.step_host(cfg.dt, hin, hout)
        fa = a.get_f()
        fb = hout.cuda()
        scale = float(fa.abs().max())
        assert float((fa - fb).abs().max()) <= TOL_DF * scale
        assert float((b.get_f() - fb).abs().max()) == 0.0                      # the context keeps what it wrote to the host
        hin.copy_(hout)
        del fa, fb
    ma, mb = a.moments(), b.moments()
    assert np.allclose(ma["tot"].numpy(), mb["tot"].numpy(), rtol=1e-12, atol=0)
    a.close()
    b.close()
