"""ctypes binding of the CPU oracle (oracle/bzo.c).  TEST INFRASTRUCTURE ONLY.

Argument marshalling only; every number comes from libbzo.so.  See oracle/bzo.h for the
citations of each call.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_lib = None

KINDS = {"A": 0, "11": 1, "1B": 2, "ANN": 3, "QQGG": 4, "QG": 5, "GG": 6}


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("dx", C.c_double),
                ("np", C.c_int), ("pmin", C.c_double), ("pmax", C.c_double)]


class Channel(C.Structure):
    _fields_ = [("a", C.c_int), ("b", C.c_int), ("c", C.c_int), ("d", C.c_int), ("kind", C.c_int), ("crossed", C.c_int)]


class PRoot(C.Structure):
    _fields_ = [("k1", C.c_double * 3), ("k2", C.c_double * 3), ("i1", C.c_int), ("i2", C.c_int), ("E1", C.c_double),
                ("E2", C.c_double), ("E3", C.c_double), ("Ep", C.c_double), ("J", C.c_double), ("s", C.c_double),
                ("t", C.c_double), ("u", C.c_double)]


class Sample(C.Structure):
    _fields_ = [("flag", C.c_int), ("j", C.c_int), ("k", C.c_int), ("l", C.c_int), ("attempts", C.c_int),
                ("s", C.c_double), ("t", C.c_double), ("u", C.c_double),
                ("E1", C.c_double), ("E2", C.c_double), ("E3", C.c_double),
                ("p1", C.c_double * 3), ("p2", C.c_double * 3), ("p3", C.c_double * 3), ("p4", C.c_double * 3),
                ("nhat", C.c_double * 3)]


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(_build.build())
        dp, ip, vp = C.POINTER(C.c_double), C.POINTER(C.c_int), C.c_void_p
        L.bzo_create.argtypes = [C.POINTER(Grid), ip, C.c_int, C.c_double, C.c_double, C.POINTER(vp)]
        L.bzo_destroy.argtypes = [vp]
        L.bzo_set_seed.argtypes = [vp, C.c_ulonglong]
        L.bzo_set_samples.argtypes = [vp, C.c_int]
        L.bzo_set_threads.argtypes = [vp, C.c_int]
        L.bzo_get_threads.argtypes = [vp]
        L.bzo_set_step.argtypes = [vp, C.c_uint]
        L.bzo_set_slab.argtypes = [vp, C.c_uint, C.c_int, C.c_int]
        L.bzo_set_f.argtypes = [vp, dp]
        L.bzo_get_f.argtypes = [vp, dp]
        L.bzo_collision.argtypes = [vp, C.c_double, C.c_uint, dp]
        L.bzo_get_gross.argtypes = [vp, dp]
        L.bzo_stream.argtypes = [vp, C.c_double, dp]
        L.bzo_step.argtypes = [vp, C.c_double]
        L.bzo_set_masses.argtypes = [vp, dp]
        L.bzo_get_masses.argtypes = [vp, dp]
        L.bzo_thermal_masses.argtypes = [vp, dp]
        L.bzo_vlasov.argtypes = [vp, C.c_double, dp]
        L.bzo_set_transport.argtypes = [vp, C.c_int]
        L.bzo_set_collision.argtypes = [vp, C.c_int]
        L.bzo_energy_diag.argtypes = [vp, dp]
        L.bzo_collision_is.argtypes = [vp, C.c_double, C.c_uint, dp]
        L.bzo_sample_one_is.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, C.c_double, C.POINTER(Sample), dp]
        L.bzo_collision_box.argtypes = [vp, C.c_double, C.c_uint, dp]
        L.bzo_sample_one_box.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, C.POINTER(Sample), dp]
        L.bzo_paper_sample.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, dp, dp, ip, C.POINTER(PRoot)]
        L.bzo_collision_paper.argtypes = [vp, C.c_double, C.c_uint, dp]
        L.bzo_collision_paper_plain.argtypes = [vp, C.c_double, C.c_uint, dp]
        L.bzo_moments.argtypes = [vp, dp]
        L.bzo_debug_samples.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, ip, dp]
        L.bzo_sample_one.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, C.POINTER(Sample)]
        L.bzo_philox4x32_10.argtypes = [C.POINTER(C.c_uint), C.POINTER(C.c_uint), C.POINTER(C.c_uint)]
        L.bzo_philox4x32_10.restype = None
        L.bzo_uniform.argtypes = [C.c_uint, C.c_uint]
        L.bzo_uniform.restype = C.c_double
        L.bzo_msq.argtypes = [C.c_int] + [C.c_double] * 5
        L.bzo_msq.restype = C.c_double
        L.bzo_n_channels.argtypes = [vp]
        L.bzo_get_channels.argtypes = [vp, C.POINTER(Channel)]
        L.bzo_set_msq_override.argtypes = [vp, C.c_int, C.c_double]
        L.bzo_sample_channels.argtypes = [vp, dp] + [C.c_double] * 7 + [dp, dp]
        L.bzo_sample_channels.restype = C.c_double
        L.bzo_collision_tile.argtypes = [vp, C.c_double, C.c_uint, C.c_int, dp, C.c_int, C.c_int, C.c_int, dp, dp, dp]
        L.bzo_regulator_m2.argtypes = [vp, dp]
        L.bzo_regulator_m2.restype = C.c_double
        _lib = L
    return _lib


def _dptr(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _chk(rc, what):
    if rc != 0:
        raise RuntimeError("%s failed with code %d" % (what, rc))


def philox4x32_10(ctr, key):
    c = (C.c_uint * 4)(*ctr)
    k = (C.c_uint * 2)(*key)
    o = (C.c_uint * 4)()
    lib().bzo_philox4x32_10(c, k, o)
    return tuple(int(x) for x in o)


def uniform(a, b):
    return float(lib().bzo_uniform(a, b))


def msq(kind, s, t, u, m2, g4):
    return float(lib().bzo_msq(KINDS[kind] if isinstance(kind, str) else kind, s, t, u, m2, g4))


class Oracle:
    """Host-only context with the same call surface as the CUDA library (prefix bzo_)."""

    def __init__(self, nx=1, ny=1, nz=1, dx=1.0, np_=15, pmin=-3.0, pmax=3.0, species=(0,), alpha_s=0.3, m_D=0.0,
                 seed=0, samples=64, threads=1):
        self.grid = Grid(nx, ny, nz, dx, np_, pmin, pmax)
        self.species = tuple(species)
        self.S = len(self.species)
        self.Nx = nx * ny * nz
        self.Np = np_ ** 3
        self.n = np_
        self.Ns = samples
        self.shape = (self.Nx, self.S, self.Np)
        sp = (C.c_int * self.S)(*self.species)
        h = C.c_void_p()
        _chk(lib().bzo_create(C.byref(self.grid), sp, self.S, alpha_s, m_D, C.byref(h)), "bzo_create")
        self._h = h
        _chk(lib().bzo_set_seed(h, seed), "bzo_set_seed")
        _chk(lib().bzo_set_samples(h, samples), "bzo_set_samples")
        _chk(lib().bzo_set_threads(h, threads), "bzo_set_threads")

    def close(self):
        if self._h:
            lib().bzo_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- state
    def set_samples(self, n):
        _chk(lib().bzo_set_samples(self._h, n), "bzo_set_samples")
        self.Ns = n

    def set_seed(self, seed):
        _chk(lib().bzo_set_seed(self._h, seed), "bzo_set_seed")

    def set_threads(self, n):
        _chk(lib().bzo_set_threads(self._h, n), "bzo_set_threads")

    def set_step(self, step):
        _chk(lib().bzo_set_step(self._h, step), "bzo_set_step")

    def set_slab(self, xcell_offset, z_begin, z_end):
        _chk(lib().bzo_set_slab(self._h, xcell_offset & 0xFFFFFFFF, z_begin, z_end), "bzo_set_slab")

    def set_f(self, f):
        f = np.ascontiguousarray(f, dtype=np.float64).reshape(self.shape)
        _chk(lib().bzo_set_f(self._h, _dptr(f)), "bzo_set_f")

    def get_f(self):
        f = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_get_f(self._h, _dptr(f)), "bzo_get_f")
        return f

    # ---- the path
    def collision(self, dt, step):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_collision(self._h, dt, step, _dptr(dF)), "bzo_collision")
        return dF

    def gross(self):
        g = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_get_gross(self._h, _dptr(g)), "bzo_get_gross")
        return g

    def stream(self, dt):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_stream(self._h, dt, _dptr(dF)), "bzo_stream")
        return dF

    def step(self, dt):
        _chk(lib().bzo_step(self._h, dt), "bzo_step")

    # ---- NEXT rank 2: thermal masses (Eq. 8-9) and the central-difference drift + force of Eq. 15
    def set_masses(self, mass2):
        m = np.ascontiguousarray(mass2, dtype=np.float64).reshape(self.Nx, 4)
        _chk(lib().bzo_set_masses(self._h, _dptr(m)), "bzo_set_masses")

    def get_masses(self):
        m = np.empty((self.Nx, 4), dtype=np.float64)
        _chk(lib().bzo_get_masses(self._h, _dptr(m)), "bzo_get_masses")
        return m

    def thermal_masses(self):
        m = np.empty((self.Nx, 4), dtype=np.float64)
        _chk(lib().bzo_thermal_masses(self._h, _dptr(m)), "bzo_thermal_masses")
        return m

    # ---- NEXT rank 1: the paper's sampler (Eq. 17-21) with massive dispersion
    def paper_sample(self, step, xcell, pcell, sample, msq):
        m = (C.c_double * 4)(*msq)
        k3 = (C.c_double * 3)()
        i3 = C.c_int()
        roots = (PRoot * 2)()
        n = lib().bzo_paper_sample(self._h, step, xcell, pcell, sample, m, k3, C.byref(i3), roots)
        if n < 0:
            raise RuntimeError("bzo_paper_sample failed")
        return list(k3), i3.value, [roots[r] for r in range(n)]

    def collision_paper(self, dt, step):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_collision_paper(self._h, dt, step, _dptr(dF)), "bzo_collision_paper")
        return dF

    def collision_paper_plain(self, dt, step):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_collision_paper_plain(self._h, dt, step, _dptr(dF)), "bzo_collision_paper_plain")
        return dF

    # ---- NEXT rank 3: importance-sampled estimator
    def collision_is(self, dt, step):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_collision_is(self._h, dt, step, _dptr(dF)), "bzo_collision_is")
        return dF

    def sample_one_is(self, step, xcell, pcell, sample, m2):
        s = Sample()
        w = C.c_double()
        _chk(lib().bzo_sample_one_is(self._h, step, xcell, pcell, sample, m2, C.byref(s), C.byref(w)), "bzo_sample_one_is")
        return s, w.value

    # ---- NEXT rank 3, other half: in-box sampling of the CM direction
    def collision_box(self, dt, step):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_collision_box(self._h, dt, step, _dptr(dF)), "bzo_collision_box")
        return dF

    def sample_one_box(self, step, xcell, pcell, sample):
        s = Sample()
        w = C.c_double()
        _chk(lib().bzo_sample_one_box(self._h, step, xcell, pcell, sample, C.byref(s), C.byref(w)), "bzo_sample_one_box")
        return s, w.value

    def set_collision(self, mode):
        _chk(lib().bzo_set_collision(self._h, mode), "bzo_set_collision")

    def set_transport(self, scheme):
        _chk(lib().bzo_set_transport(self._h, scheme), "bzo_set_transport")

    def energy_diag(self):
        out = np.empty((self.Nx, 5), dtype=np.float64)
        _chk(lib().bzo_energy_diag(self._h, _dptr(out)), "bzo_energy_diag")
        return out

    def vlasov(self, dt):
        dF = np.empty(self.shape, dtype=np.float64)
        _chk(lib().bzo_vlasov(self._h, dt, _dptr(dF)), "bzo_vlasov")
        return dF

    def moments(self):
        out = np.empty(self.Nx * self.S * 2 + self.S * 2 + self.Nx, dtype=np.float64)
        _chk(lib().bzo_moments(self._h, _dptr(out)), "bzo_moments")
        a = self.Nx * self.S * 2
        return {"ne": out[:a].reshape(self.Nx, self.S, 2).copy(),
                "tot": out[a:a + 2 * self.S].reshape(self.S, 2).copy(),
                "m2": out[a + 2 * self.S:].copy()}

    def debug_samples(self, step, xcell, pbegin, pend, want_stu=True):
        n = pend - pbegin
        cells = np.empty((n, self.Ns, 4), dtype=np.int32)
        stu = np.empty((n, self.Ns, 3), dtype=np.float64) if want_stu else None
        _chk(lib().bzo_debug_samples(self._h, step, xcell, pbegin, pend, cells.ctypes.data_as(C.POINTER(C.c_int)),
                                     _dptr(stu) if want_stu else None), "bzo_debug_samples")
        return cells, stu

    # ---- hooks for the pins
    def sample_one(self, step, xcell, pcell, sample):
        s = Sample()
        _chk(lib().bzo_sample_one(self._h, step, xcell, pcell, sample, C.byref(s)), "bzo_sample_one")
        return s

    def channels(self):
        n = lib().bzo_n_channels(self._h)
        arr = (Channel * n)()
        _chk(lib().bzo_get_channels(self._h, arr), "bzo_get_channels")
        return [(c.a, c.b, c.c, c.d, c.kind, c.crossed) for c in arr]

    def set_msq_override(self, kind, value):
        _chk(lib().bzo_set_msq_override(self._h, KINDS[kind] if isinstance(kind, str) else kind, value), "override")

    def sample_channels(self, fv, s, t, u, E1, E2, m2, dt):
        fv = np.ascontiguousarray(fv, dtype=np.float64).reshape(4, self.S)
        dN = np.empty((4, self.S), dtype=np.float64)
        fwd = np.empty(lib().bzo_n_channels(self._h), dtype=np.float64)
        gross = lib().bzo_sample_channels(self._h, _dptr(fv), s, t, u, E1, E2, m2, dt, _dptr(dN), _dptr(fwd))
        return dN, fwd, float(gross)

    def collision_tile(self, dt, step, xcell, f_tile, pbegin=0, pend=None, mode=0, want_gross=False):
        pend = self.Np if pend is None else pend
        ft = np.ascontiguousarray(f_tile, dtype=np.float64).reshape(self.S, self.Np)
        dN = np.zeros((self.S, self.Np), dtype=np.float64)
        gross = np.zeros((self.S, self.Np), dtype=np.float64) if want_gross else None
        m2 = C.c_double()
        _chk(lib().bzo_collision_tile(self._h, dt, step, xcell, _dptr(ft), pbegin, pend, mode, _dptr(dN),
                                      _dptr(gross) if want_gross else None, C.byref(m2)), "bzo_collision_tile")
        return dN, gross, m2.value

    def regulator_m2(self, f_tile):
        ft = np.ascontiguousarray(f_tile, dtype=np.float64).reshape(self.S, self.Np)
        return float(lib().bzo_regulator_m2(self._h, _dptr(ft)))
