"""bz_moments_noalloc against bz_moments (GPU).  Collected last on purpose (pytest -x stops at the first failure).

bz_moments_noalloc serves callers that hold f in device memory of their own and cannot allocate any more of it: a solver
whose f already fills the card (a bz context costs about 4.3 x the size of f), a monitor that must not stall other streams
with the device-wide synchronisation of cudaMalloc / cudaFree, a process whose memory belongs to a framework's pool.  It
needs no context; the row sums between its two kernels sit in a fixed 1.5 MiB array inside libbz.so that every call on the
device shares and that keeps whatever the last call left there.

What is checked: the entry point writes what the context path (bz_create + bz_set_f + bz_moments) writes, within the 1e-12
relative bound the other GPU tests put on moments, on two calls in a row with different grids, species lists and
regulators, the second one smaller than the first so that stale rows of the first call are still in the scratch; a third
call with the first input gives the first result again bit for bit; a grid beyond the scratch is refused with a message
and launches nothing.  Passes alone in a fresh process (the first call then does the per-device address look-up) and after
the rest of the suite."""
import numpy as np
import pytest
import torch

import workloads as wl
from paper_1912_04457_b200 import bz

pytestmark = pytest.mark.gpu


def _case(cfg):
    """(keyword arguments of the grid, f on the device, moments of the existing context path as one host vector)."""
    kw = dict(nx=cfg.nx, ny=cfg.nx, nz=cfg.nx, dx=cfg.dx, np_=cfg.np_, pmin=cfg.pmin, pmax=cfg.pmax, species=cfg.species,
              alpha_s=cfg.alpha_s, m_D=cfg.m_D)
    f = torch.as_tensor(wl.initial_f(cfg), dtype=torch.float64).contiguous().cuda()
    g = bz.Boltzmann(device="cuda:0", seed=cfg.seed, samples=cfg.samples, **kw)
    g.set_f(f)
    n = 2 * cfg.S * cfg.Nx + 2 * cfg.S + cfg.Nx
    ref = torch.empty(n, dtype=torch.float64)
    g.moments(out=ref)
    g.close()
    return kw, f, ref.numpy()


def _check(out, ref, cfg):
    got = out.cpu().numpy()
    a = 2 * cfg.S * cfg.Nx
    assert np.all(np.isfinite(got))
    assert np.allclose(got[:a], ref[:a], rtol=1e-12, atol=0)                                   # n_a(x), e_a(x)
    assert np.allclose(got[a:a + 2 * cfg.S], ref[a:a + 2 * cfg.S], rtol=1e-12, atol=0)         # totals N_a, E_a
    assert np.allclose(got[a + 2 * cfg.S:], ref[a + 2 * cfg.S:], rtol=1e-12, atol=0)           # m^2(x)
    assert (ref[a:a + 2 * cfg.S] > 0).all()                                                    # the comparison is not 0 == 0


def test_moments_noalloc_matches_context_path_on_two_calls_in_a_row():
    # call 1: 7 species, 27 spatial cells, 1331 momentum cells (5 strides of 256 and a ragged tail), m^2 from f (Eq. 8)
    cfg1 = wl.scaled(wl.CONFIGS[3], nx=3, np_=11)
    # call 2: 6 quark species (no gluon row), 8 cells, 729 momentum cells, fixed regulator: fewer rows than call 1
    cfg2 = wl.scaled(wl.CONFIGS[1], nx=2, np_=9, m_D=0.6)
    kw1, f1, ref1 = _case(cfg1)
    kw2, f2, ref2 = _case(cfg2)
    out1 = torch.full((ref1.size,), float("nan"), dtype=torch.float64, device="cuda:0")
    out2 = torch.full((ref2.size,), float("nan"), dtype=torch.float64, device="cuda:0")
    out3 = torch.full((ref1.size,), float("nan"), dtype=torch.float64, device="cuda:0")
    # all three on one stream, back to back: ordered on the GPU, nothing overlaps on the shared scratch
    launches = bz.launch_count()
    m1 = bz.moments_noalloc(f1, out1, **kw1)
    bz.moments_noalloc(f2, out2, **kw2)
    bz.moments_noalloc(f1, out3, **kw1)
    assert bz.launch_count() - launches == 6            # two kernels of libbz.so per call, no library fallback
    torch.cuda.synchronize()
    _check(out1, ref1, cfg1)
    _check(out2, ref2, cfg2)
    assert torch.equal(out1, out3)                      # what call 2 left in the scratch does not show in call 3
    assert m1["ne"].shape == (cfg1.Nx, cfg1.S, 2) and m1["tot"].shape == (cfg1.S, 2) and m1["m2"].shape == (cfg1.Nx,)
    assert m1["m2"].data_ptr() == out1.data_ptr() + 8 * (2 * cfg1.S * cfg1.Nx + 2 * cfg1.S)     # views of the caller's buffer


def test_moments_noalloc_refuses_grids_beyond_its_scratch():
    # 22^3 spatial cells x 7 species = 74536 rows > 65536: refused on the host, before any launch, with a message
    assert 22 ** 3 * 7 > bz.NOALLOC_MAX_ROWS >= 20 ** 3 * 7
    grid = bz.Grid(22, 22, 22, 0.1, 4, -2.0, 2.0)
    sp = (bz.C.c_int * 7)(*wl.ALL_SPECIES)
    dummy = torch.zeros(8, dtype=torch.float64, device="cuda:0")
    L = bz.lib()
    launches = bz.launch_count()
    rc = L.bz_moments_noalloc(bz.C.byref(grid), sp, 7, 0.3, 0.0, bz.C.c_void_p(dummy.data_ptr()), bz.C.c_void_p(dummy.data_ptr()), None)
    assert rc == -5
    msg = L.bz_noalloc_last_error().decode()
    assert "74536" in msg and "65536" in msg
    assert bz.launch_count() == launches
    assert L.bz_moments_noalloc(bz.C.byref(grid), sp, 7, 0.3, 0.0, None, bz.C.c_void_p(dummy.data_ptr()), None) == -1
    torch.cuda.synchronize()
    assert float(dummy.abs().sum()) == 0.0
