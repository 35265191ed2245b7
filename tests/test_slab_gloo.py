"""Slab decomposition: the host logic of paper_1912_04457_b200/slab.py -- who owns which z layers,
which layer goes to which neighbour, the Philox spatial-counter offset, the all-reduced totals -- covered on CPU with
world_size-2 (and 3) gloo process groups.  The compute engine plugged in here is the ORACLE (tests may use it); on a
GPU the engine is bz.Boltzmann (tests/test_gpu_parity.py::test_slab_*).  A decomposed run must reproduce the
undecomposed oracle bit for bit: the oracle's per-cell arithmetic does not depend on where the cell lives."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads as wl
from oracle import bzo
from paper_1912_04457_b200 import slab


class OracleEngine:
    """Adapter: the oracle behind the engine interface SlabDomain drives (layers as CPU tensors)."""

    device = torch.device("cpu")

    def __init__(self, **kw):
        self.o = bzo.Oracle(**kw)
        self.nz = kw["nz"]

    def set_slab(self, off, zb, ze):
        self.o.set_slab(off, zb, ze)

    def layer_values(self):
        return int(np.prod(self.o.shape)) // self.nz

    def get_layers(self, z0, n):
        lv = self.layer_values()
        return torch.from_numpy(self.o.get_f().reshape(-1)[z0 * lv:(z0 + n) * lv].copy())

    def set_layers(self, z0, n, buf):
        lv = self.layer_values()
        f = self.o.get_f().reshape(-1)
        f[z0 * lv:(z0 + n) * lv] = buf.numpy()
        self.o.set_f(f.reshape(self.o.shape))

    def step(self, dt):
        self.o.step(dt)

    def step_host(self, dt, f_in, f_out):
        """bz_step_host for a slab context: only the OWN layers are read from f_in and written to f_out; the halo layers
        are whatever the caller refreshed in the engine before the call."""
        lv = self.layer_values()
        own = slice(lv, (self.nz - 1) * lv)
        f = self.o.get_f().reshape(-1)
        f[own] = f_in.reshape(-1).numpy()[own]
        self.o.set_f(f.reshape(self.o.shape))
        self.o.step(dt)
        f_out.reshape(-1).numpy()[own] = self.o.get_f().reshape(-1)[own]

    def moments(self):
        m = self.o.moments()
        return {"tot": torch.from_numpy(np.array(m["tot"]))}


def _cfg():
    # 7 species, streaming + collision, 2 x 2 x 5 spatial cells (5 layers: ragged over 2 and 3 ranks), odd momentum grid
    return wl.scaled(wl.CONFIGS[3], nx=2, np_=5, samples=3)


def _kw(cfg, nz):
    return dict(nx=2, ny=2, nz=nz, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species,
                alpha_s=cfg.alpha_s, m_D=cfg.m_D, seed=cfg.seed, samples=cfg.samples)


NZ, STEPS = 5, 3


def _global_f(cfg):
    rng = np.random.default_rng(7)
    return rng.uniform(0.02, 0.6, size=(2 * 2 * NZ, cfg.S, cfg.Np))


def _reference(cfg):
    o = bzo.Oracle(**_kw(cfg, NZ))
    o.set_f(_global_f(cfg))
    for _ in range(STEPS):
        o.step(cfg.dt)
    return o.get_f(), np.array(o.moments()["tot"])


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = _cfg()
        dom = slab.SlabDomain(lambda nz: OracleEngine(**_kw(cfg, nz)), 2, 2, NZ, rank, world)
        f = _global_f(cfg)
        dom.set_own(torch.from_numpy(f[dom.z0 * 4:dom.z1 * 4].copy()))
        for _ in range(STEPS):
            dom.step(cfg.dt)
        tot = dom.moments_totals().numpy()
        np.save(os.path.join(out_dir, "own%d.npy" % rank), dom.get_own().numpy())
        np.save(os.path.join(out_dir, "tot%d.npy" % rank), tot)
        np.save(os.path.join(out_dir, "z%d.npy" % rank), np.array([dom.z0, dom.z1]))
    finally:
        dist.destroy_process_group()


def _worker_host(rank, world, port, out_dir):
    """The end-to-end leg: every step starts from host buffers (own layers only) and ends in host buffers."""
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = _cfg()
        dom = slab.SlabDomain(lambda nz: OracleEngine(**_kw(cfg, nz)), 2, 2, NZ, rank, world)
        f = _global_f(cfg)
        nl = 4
        hin = torch.zeros(((dom.nz_local + 2) * nl, cfg.S, cfg.Np), dtype=torch.float64)
        hin[nl:-nl] = torch.from_numpy(f[dom.z0 * nl:dom.z1 * nl].copy())
        hout = torch.full_like(hin, -7.0)
        for _ in range(STEPS):
            dom.step_host(cfg.dt, hin, hout)
            assert float(hout[:nl].min()) == -7.0 and float(hout[-nl:].max()) == -7.0      # halo layers of the host buffer untouched
            hin[nl:-nl] = hout[nl:-nl]
        np.save(os.path.join(out_dir, "own%d.npy" % rank), hout[nl:-nl].numpy())
    finally:
        dist.destroy_process_group()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_slab_range_is_a_partition():
    for nz in (1, 2, 5, 16, 17):
        for world in range(1, min(nz, 8) + 1):
            r = [slab.slab_range(nz, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nz
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1
    with pytest.raises(ValueError):
        slab.slab_range(2, 0, 3)


def test_single_rank_slab_with_self_halo_equals_plain_domain():
    cfg = _cfg()
    dom = slab.SlabDomain(lambda nz: OracleEngine(**_kw(cfg, nz)), 2, 2, NZ, 0, 1)
    dom.set_own(torch.from_numpy(_global_f(cfg)))
    for _ in range(STEPS):
        dom.step(cfg.dt)
    f_ref, tot_ref = _reference(cfg)
    assert np.array_equal(dom.get_own().numpy().reshape(f_ref.shape), f_ref)
    assert np.allclose(dom.moments_totals().numpy(), tot_ref, rtol=1e-14, atol=0)


def test_in_process_exchange_of_two_slabs():
    cfg = _cfg()
    doms = [slab.SlabDomain(lambda nz: OracleEngine(**_kw(cfg, nz)), 2, 2, NZ, r, 2) for r in range(2)]
    f = _global_f(cfg)
    for d in doms:
        d.set_own(torch.from_numpy(f[d.z0 * 4:d.z1 * 4].copy()))
    for _ in range(STEPS):
        slab.exchange_in_process(doms)
        for d in doms:
            d.engine.step(cfg.dt)
    f_ref, _ = _reference(cfg)
    got = np.concatenate([d.get_own().numpy() for d in doms]).reshape(f_ref.shape)
    assert np.array_equal(got, f_ref)


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_slabs_reproduce_the_undecomposed_domain(world, tmp_path):
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = _cfg()
    f_ref, tot_ref = _reference(cfg)
    parts, zs = [], []
    for r in range(world):
        parts.append(np.load(tmp_path / ("own%d.npy" % r)))
        zs.append(tuple(np.load(tmp_path / ("z%d.npy" % r))))
        # every rank holds the all-reduced totals of the whole domain
        assert np.allclose(np.load(tmp_path / ("tot%d.npy" % r)), tot_ref, rtol=1e-14, atol=0)
    assert zs == [slab.slab_range(NZ, r, world) for r in range(world)]
    got = np.concatenate(parts).reshape(f_ref.shape)
    assert np.array_equal(got, f_ref), "decomposed run differs from the undecomposed oracle"


@pytest.mark.parametrize("world", [2, 3])
def test_gloo_slabs_step_host_reproduces_the_undecomposed_domain(world, tmp_path):
    """SlabDomain.step_host over gloo: boundary layers staged, exchanged, then the engine's step_host on the own layers."""
    mp.spawn(_worker_host, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    cfg = _cfg()
    f_ref, _ = _reference(cfg)
    got = np.concatenate([np.load(tmp_path / ("own%d.npy" % r)) for r in range(world)]).reshape(f_ref.shape)
    assert np.array_equal(got, f_ref), "decomposed end-to-end run differs from the undecomposed oracle"
