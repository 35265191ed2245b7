"""CPU-side checks of the product: the C-ABI library loads, exports what include/bz.h declares, refuses to run
without a device, and its factorised channel algebra equals the oracle's channel-by-channel definition."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest
import torch

from oracle import bzo
from paper_1912_04457_b200 import bz

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def debug_deposit_host(species, alpha_s, fv, s, t, u, m2, w, variant=1):
    """bz_debug_deposit_host of the TEST-ONLY libbz_testhooks.so (csrc/bz_testhooks.cu): the kernels' channel algebra
    compiled for the host.  libbz.so does not contain it."""
    from paper_1912_04457_b200 import build
    L = C.CDLL(build.build_testhooks())
    dp = C.POINTER(C.c_double)
    L.bz_debug_deposit_host.argtypes = [C.POINTER(C.c_int), C.c_int, C.c_double, dp] + [C.c_double] * 5 + [C.c_int, dp]
    fv = np.ascontiguousarray(fv, dtype=np.float64).reshape(4, 7)
    out = np.empty((4, 7), dtype=np.float64)
    sp = (C.c_int * len(species))(*species)
    rc = L.bz_debug_deposit_host(sp, len(species), alpha_s, fv.ctypes.data_as(dp), s, t, u, m2, w, variant, out.ctypes.data_as(dp))
    assert rc == 0
    return out


def test_library_exports_every_declared_symbol():
    header = open(os.path.join(ROOT, "include", "bz.h")).read()
    declared = set(re.findall(r"\b(bz_[a-z_0-9]+)\s*\(", header))
    declared -= {"bz_ctx", "bz_grid"}
    assert declared == set(bz.EXPORTS)
    L = bz.lib()
    for name in declared:
        assert hasattr(L, name), name
    assert not hasattr(L, "bz_debug_deposit_host")      # the host evaluation of the channel algebra is a test-only object


def test_moments_noalloc_checks_its_arguments_before_touching_the_device():
    """bz_moments_noalloc (include/bz.h): bad arguments (-1) and grids beyond the fixed scratch (-5, with a message that names
    both numbers) are refused on the host, before any CUDA call -- so this runs without a GPU."""
    L = bz.lib()
    buf = (C.c_double * 8)()
    ptr = C.cast(buf, C.c_void_p)
    sp7 = (C.c_int * 7)(0, 1, 2, 3, 4, 5, 6)
    big = bz.Grid(22, 22, 22, 0.1, 4, -2.0, 2.0)                      # 10648 cells x 7 species = 74536 rows > 65536
    assert L.bz_moments_noalloc(C.byref(big), sp7, 7, 0.3, 0.0, ptr, ptr, None) == -5
    msg = L.bz_noalloc_last_error().decode()
    assert "74536" in msg and str(bz.NOALLOC_MAX_ROWS) in msg
    ok = bz.Grid(2, 2, 2, 0.1, 4, -2.0, 2.0)
    assert L.bz_moments_noalloc(C.byref(ok), sp7, 7, 0.3, 0.0, None, ptr, None) == -1          # no input
    assert L.bz_moments_noalloc(C.byref(ok), sp7, 7, 0.3, 0.0, ptr, None, None) == -1          # no output
    assert L.bz_moments_noalloc(C.byref(ok), sp7, 7, -0.3, 0.0, ptr, ptr, None) == -1          # alpha_s <= 0
    assert L.bz_moments_noalloc(C.byref(ok), (C.c_int * 2)(3, 3), 2, 0.3, 0.0, ptr, ptr, None) == -1   # not ascending
    assert L.bz_moments_noalloc(C.byref(bz.Grid(2, 2, 2, 0.1, 1, -2.0, 2.0)), sp7, 7, 0.3, 0.0, ptr, ptr, None) == -1   # np < 2
    assert L.bz_noalloc_last_error().decode() != ""


def test_bad_arguments_are_rejected_without_a_device():
    L = bz.lib()
    h = C.c_void_p()
    g = bz.Grid(1, 1, 1, 1.0, 8, -3.0, 3.0)
    sp = (C.c_int * 2)(1, 1)                         # not strictly ascending
    assert L.bz_create(C.byref(g), sp, 2, 0.3, 0.0, C.byref(h)) == -1
    sp = (C.c_int * 1)(9)
    assert L.bz_create(C.byref(g), sp, 1, 0.3, 0.0, C.byref(h)) == -1
    g2 = bz.Grid(1, 1, 1, 1.0, 8, 3.0, -3.0)         # empty box
    sp = (C.c_int * 1)(0)
    assert L.bz_create(C.byref(g2), sp, 1, 0.3, 0.0, C.byref(h)) == -1
    assert L.bz_set_samples(None, 4) == -1
    assert L.bz_step(None, 0.1) == -1


@pytest.mark.skipif(torch.cuda.is_available(), reason="only meaningful on a box without a GPU")
def test_no_cpu_fallback():
    with pytest.raises(bz.BzError, match="no CUDA device"):
        bz.Boltzmann(np_=4, species=(0,))
    # and the library itself refuses: -2 with a message, no context usable
    L = bz.lib()
    h = C.c_void_p()
    g = bz.Grid(1, 1, 1, 1.0, 4, -3.0, 3.0)
    assert L.bz_create(C.byref(g), (C.c_int * 1)(0), 1, 0.3, 0.0, C.byref(h)) == -2
    assert b"no CUDA device" in L.bz_last_error(h)
    assert L.bz_step(h, 0.01) == -4
    L.bz_destroy(h)


@pytest.mark.parametrize("species", [(0,), (1, 2, 3, 4, 5, 6), (0, 1, 2, 3, 4, 5, 6), (0, 1, 2), (0, 1), (1, 2, 5),
                                     (0, 3, 4, 5), (2,), (0, 2, 3, 6)])
def test_factorised_channel_algebra_equals_channel_loop(species):
    # the kernels never loop over the 127 channels (csrc/bz_channels.cuh); their algebra, run on the host through
    # the test-only libbz_testhooks.so, must reproduce the oracle's channel-by-channel deposits up to summation order
    rng = np.random.default_rng(len(species) * 17 + species[0])
    o = bzo.Oracle(np_=8, species=species, samples=8, seed=3)
    S = len(species)
    K = (0.01 / 0.1973269804) * 6.0 ** 3 / (2048 * math.pi ** 4 * 8)
    done = 0
    for trial in range(150):
        sm = o.sample_one(0, 0, int(rng.integers(0, 512)), int(rng.integers(0, 8)))
        if sm.attempts == 0:
            continue
        fvS = rng.uniform(0.0, 0.9, size=(4, S))
        if trial % 5 == 0:
            fvS[rng.integers(0, 4), rng.integers(0, S)] = 0.0
        if trial % 7 == 0:
            fvS[:, :] = 0.0                                     # empty cells: nothing may be deposited
        dN, _, gross = o.sample_channels(fvS, sm.s, sm.t, sm.u, sm.E1, sm.E2, 0.37, 0.01)
        fv = rng.uniform(0.0, 1.0, size=(4, 7))                 # values of inactive species must be ignored
        fv[:, list(species)] = fvS
        for variant in (0, 1):                                  # whole bracket / gain + loss halves (collide_kernel)
            out = debug_deposit_host(species, 0.3, fv, sm.s, sm.t, sm.u, 0.37, K / (sm.E1 * sm.E2), variant)
            assert np.all(out[:, [i for i in range(7) if i not in species]] == 0.0)
            got = out[:, list(species)]
            if gross == 0.0:
                assert np.all(got == 0.0)
            else:
                # the halves are formed separately, so the comparison scale is the sum of |gain| + |loss| terms; for these
                # f in [0, 0.9) it is within a small factor of the oracle's gross sum of |A|
                assert np.abs(got - dN).max() <= (1e-12 if variant == 0 else 4e-12) * gross
                assert abs(got.sum()) <= 1e-12 * gross          # Eq. 23: number units sum to zero
        done += 1
    assert done > 100


@pytest.mark.parametrize("species", [(0,), (1, 2, 3, 4, 5, 6), (0, 1, 2, 3, 4, 5, 6), (0, 1, 2), (0, 1), (1, 2, 5), (0, 3, 4, 6)])
def test_paper_sampler_channel_table_matches_oracle(species):
    """The channel table of the paper sampler (bz_paper.cu, generated on the host) is the oracle's, as a set; channels of
    one mass-class tuple are contiguous."""
    from oracle import bzo
    rows = bz.debug_paper_channels(species)
    o = bzo.Oracle(np_=4, species=species)
    want = sorted(tuple(int(v) for v in c) for c in o.channels())
    got = sorted(tuple(int(v) for v in r[:6]) for r in rows)
    assert got == want
    cls = [0 if s == 0 else 1 + (s - 1) // 2 for s in species]
    keys = [int(r[6]) for r in rows]
    for r in rows:
        assert int(r[6]) == cls[r[0]] | cls[r[1]] << 2 | cls[r[2]] << 4 | cls[r[3]] << 6
    seen, last = set(), None
    for k in keys:
        if k != last:
            assert k not in seen
            seen.add(k)
            last = k


def test_bench_reference_arm_prints_the_contract_line():
    """bench.py --impl reference (the oracle arm) runs without a GPU and prints one JSON line with the contract's keys."""
    import json
    import subprocess
    import sys
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "0", "--steps", "1",
                          "--warmup", "3"], capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert out.returncode == 0, out.stderr[-2000:]
    line = json.loads(out.stdout.strip().splitlines()[-1])
    for key in ("impl", "metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling",
                "vs_baseline", "dtype", "data", "config", "cpu_baseline", "e2e"):
        assert key in line, key
    assert line["impl"] == "reference" and line["value"] > 0 and line["dtype"] == "f64"
    assert line["cpu_baseline"]["kind"] == "oracle" and line["cpu_baseline"]["cores"] >= 1
    assert line["e2e"]["h2d_bytes_per_step"] == 0 and line["e2e"]["d2h_bytes_per_step"] == 0
