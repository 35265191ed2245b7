"""ctypes binding of libbz.so with the same names as include/bz.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of csrc/; there is no Python or CPU fallback: if the library
cannot be loaded, or no CUDA device is present, the calls raise.
"""
import ctypes as C
import os

import torch

from . import build as _build

LIB_PATH = _build.LIB
_lib = None


class Grid(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("dx", C.c_double),
                ("np", C.c_int), ("pmin", C.c_double), ("pmax", C.c_double)]


EXPORTS = ("bz_create", "bz_destroy", "bz_set_stream", "bz_set_seed", "bz_set_samples", "bz_set_step", "bz_set_slab",
           "bz_copy_layers", "bz_set_msq_override", "bz_thermal_masses", "bz_set_masses", "bz_vlasov",
           "bz_set_transport", "bz_step_host", "bz_collision_paper", "bz_set_collision", "bz_energy_diag", "bz_collision_is", "bz_debug_samples_is", "bz_collision_box", "bz_debug_samples_box", "bz_debug_paper_samples", "bz_debug_paper_channels", "bz_set_f",
           "bz_get_f", "bz_collision", "bz_stream", "bz_step", "bz_step_n", "bz_moments", "bz_last_error", "bz_set_profile",
           "bz_get_profile", "bz_measure_fp64_peak", "bz_launch_count", "bz_get_sample_counts",
           "bz_debug_samples", "bz_moments_noalloc", "bz_noalloc_last_error", "bz_msq_sign_counts")

KINDS = ("A", "11", "1B", "ANN", "QQGG", "QG", "GG")      # kinds of Table I in the order of bz_set_msq_override


def lib():
    """Load libbz.so (building it with nvcc first if it is missing or stale).  Raises if that fails."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        vp, dp, ip = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_int)
        L.bz_create.argtypes = [C.POINTER(Grid), ip, C.c_int, C.c_double, C.c_double, C.POINTER(vp)]
        L.bz_destroy.argtypes = [vp]
        L.bz_set_stream.argtypes = [vp, vp]
        L.bz_set_seed.argtypes = [vp, C.c_ulonglong]
        L.bz_set_samples.argtypes = [vp, C.c_int]
        L.bz_set_step.argtypes = [vp, C.c_uint]
        L.bz_set_slab.argtypes = [vp, C.c_uint, C.c_int, C.c_int]
        L.bz_set_msq_override.argtypes = [vp, C.c_int, C.c_double]
        L.bz_thermal_masses.argtypes = [vp, vp]
        L.bz_set_masses.argtypes = [vp, vp]
        L.bz_vlasov.argtypes = [vp, C.c_double, vp]
        L.bz_set_transport.argtypes = [vp, C.c_int]
        L.bz_step_host.argtypes = [vp, C.c_double, vp, vp]
        L.bz_collision_paper.argtypes = [vp, C.c_double, C.c_uint, vp]
        L.bz_set_collision.argtypes = [vp, C.c_int]
        L.bz_energy_diag.argtypes = [vp, vp]
        L.bz_collision_is.argtypes = [vp, C.c_double, C.c_uint, vp]
        L.bz_debug_samples_is.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, C.c_double, vp, vp, vp]
        L.bz_collision_box.argtypes = [vp, C.c_double, C.c_uint, vp]
        L.bz_debug_samples_box.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, vp, vp, vp]
        L.bz_debug_paper_samples.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, dp, vp, vp]
        L.bz_debug_paper_channels.argtypes = [ip, C.c_int, ip, C.c_int]
        L.bz_copy_layers.argtypes = [vp, C.c_int, C.c_int, vp, C.c_int]
        L.bz_set_f.argtypes = [vp, vp, C.c_int]
        L.bz_get_f.argtypes = [vp, vp, C.c_int]
        L.bz_collision.argtypes = [vp, C.c_double, C.c_uint, vp]
        L.bz_stream.argtypes = [vp, C.c_double, vp]
        L.bz_step.argtypes = [vp, C.c_double]
        L.bz_step_n.argtypes = [vp, C.c_double, C.c_int]
        L.bz_moments.argtypes = [vp, vp]
        L.bz_last_error.argtypes = [vp]
        L.bz_last_error.restype = C.c_char_p
        L.bz_set_profile.argtypes = [vp, C.c_int]
        L.bz_get_profile.argtypes = [vp, C.c_int, dp, ip]
        L.bz_measure_fp64_peak.argtypes = [dp]
        L.bz_get_sample_counts.argtypes = [vp, C.POINTER(C.c_ulonglong), C.POINTER(C.c_ulonglong), C.c_int]
        L.bz_launch_count.argtypes = []
        L.bz_launch_count.restype = C.c_ulonglong
        L.bz_debug_samples.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.c_int, vp, vp]
        L.bz_msq_sign_counts.argtypes = [vp, C.c_uint, C.c_int, C.c_int, C.POINTER(C.c_ulonglong)]
        L.bz_moments_noalloc.argtypes = [C.POINTER(Grid), ip, C.c_int, C.c_double, C.c_double, vp, vp, vp]
        L.bz_noalloc_last_error.argtypes = []
        L.bz_noalloc_last_error.restype = C.c_char_p
        _lib = L
    return _lib


class BzError(RuntimeError):
    pass


class Boltzmann:
    """One bz_ctx.  Methods carry the names of the C entry points without the prefix.

    Stream semantics: every call enqueues its work on the context's stream (the torch stream that was current when the
    object was made, or the one given to set_stream).  CUDA tensors returned by get_f / collision / stream / vlasov /
    get_layers are therefore ordered on THAT stream only: a consumer on another stream (torch streams are non-blocking
    with respect to each other) must synchronise it or wait on it first, e.g.
    torch.cuda.current_stream().wait_stream(s).  Calls that copy to host memory synchronise the stream themselves."""

    def __init__(self, nx=1, ny=1, nz=1, dx=1.0, np_=15, pmin=-3.0, pmax=3.0, species=(0,), alpha_s=0.3, m_D=0.0,
                 seed=0, samples=64, device="cuda:0"):
        self._h = None
        self.device = torch.device(device)
        self.species = tuple(species)
        self.S, self.Nx, self.Np, self.Ns = len(self.species), nx * ny * nz, np_ ** 3, samples
        self.shape = (self.Nx, self.S, self.Np)
        self.n_values = self.Nx * self.S * self.Np
        self._grid = Grid(nx, ny, nz, dx, np_, pmin, pmax)
        L = lib()
        if not torch.cuda.is_available():
            raise BzError("no CUDA device: libbz.so has no CPU path")
        h = C.c_void_p()
        with torch.cuda.device(self.device):
            rc = L.bz_create(C.byref(self._grid), (C.c_int * self.S)(*self.species), self.S, alpha_s, m_D, C.byref(h))
        if rc != 0:
            msg = L.bz_last_error(h).decode() if h else "bad argument"
            if h:
                L.bz_destroy(h)
            raise BzError("bz_create failed (%d): %s" % (rc, msg))
        self._h = h
        self._chk(L.bz_set_seed(h, seed), "bz_set_seed")
        self._chk(L.bz_set_samples(h, samples), "bz_set_samples")
        self.set_stream(torch.cuda.current_stream(self.device))

    # ---- plumbing
    def _chk(self, rc, what):
        if rc != 0:
            raise BzError("%s failed (%d): %s" % (what, rc, lib().bz_last_error(self._h).decode()))

    def close(self):
        if self._h:
            lib().bz_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _dev_ptr(self, t, n, dtype=torch.float64):
        if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == n):
            raise ValueError("expected a contiguous CUDA %s tensor with %d elements" % (dtype, n))
        return C.c_void_p(t.data_ptr())

    def set_stream(self, stream):
        self.torch_stream = stream
        self._chk(lib().bz_set_stream(self._h, C.c_void_p(stream.cuda_stream)), "bz_set_stream")

    def set_seed(self, seed):
        self._chk(lib().bz_set_seed(self._h, seed), "bz_set_seed")

    def set_samples(self, n):
        self._chk(lib().bz_set_samples(self._h, n), "bz_set_samples")
        self.Ns = n

    def set_step(self, step):
        self._chk(lib().bz_set_step(self._h, step), "bz_set_step")

    def set_msq_override(self, kind, value):
        """kind: 0..6 or one of KINDS; value >= 0 replaces that kind of Table I by a constant, < 0 restores it."""
        k = KINDS.index(kind) if isinstance(kind, str) else int(kind)
        self._chk(lib().bz_set_msq_override(self._h, k, float(value)), "bz_set_msq_override")

    def set_slab(self, xcell_offset, z_begin, z_end):
        self._chk(lib().bz_set_slab(self._h, xcell_offset & 0xFFFFFFFF, z_begin, z_end), "bz_set_slab")

    def layer_values(self):
        return self.n_values // self._grid.nz

    def get_layers(self, z0, n_layers, out=None):
        """n_layers z layers of f starting at z0 as a CUDA tensor (asynchronous device copy)."""
        n = n_layers * self.layer_values()
        if out is None:
            out = torch.empty(n, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_copy_layers(self._h, z0, n_layers, self._dev_ptr(out, n), 0), "bz_copy_layers")
        return out

    def set_layers(self, z0, n_layers, buf):
        n = n_layers * self.layer_values()
        self._chk(lib().bz_copy_layers(self._h, z0, n_layers, self._dev_ptr(buf, n), 1), "bz_copy_layers")

    # ---- state
    def set_f(self, f):
        """f: CUDA tensor (device copy) or CPU tensor / numpy array (host copy, synchronises)."""
        if isinstance(f, torch.Tensor) and f.is_cuda:
            self._chk(lib().bz_set_f(self._h, self._dev_ptr(f, self.n_values), 1), "bz_set_f")
        else:
            t = torch.as_tensor(f, dtype=torch.float64).contiguous()
            if t.numel() != self.n_values:
                raise ValueError("f has %d values, expected %d" % (t.numel(), self.n_values))
            self._chk(lib().bz_set_f(self._h, C.c_void_p(t.data_ptr()), 0), "bz_set_f")

    def get_f(self, out=None):
        """Returns a CUDA tensor (device copy); pass a CPU tensor as `out` for a host copy (synchronises)."""
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        if out.is_cuda:
            self._chk(lib().bz_get_f(self._h, self._dev_ptr(out, self.n_values), 1), "bz_get_f")
        else:
            if not (out.dtype == torch.float64 and out.is_contiguous() and out.numel() == self.n_values):
                raise ValueError("bad host buffer")
            self._chk(lib().bz_get_f(self._h, C.c_void_p(out.data_ptr()), 0), "bz_get_f")
        return out

    # ---- the path
    def collision(self, dt, step, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_collision(self._h, dt, step, self._dev_ptr(out, self.n_values)), "bz_collision")
        return out

    def stream(self, dt, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_stream(self._h, dt, self._dev_ptr(out, self.n_values)), "bz_stream")
        return out

    # ---- NEXT rank 2: thermal masses (Eq. 8-9) and the central-difference drift + force of Eq. 15
    def thermal_masses(self):
        out = torch.empty((self.Nx, 4), dtype=torch.float64)
        self._chk(lib().bz_thermal_masses(self._h, C.c_void_p(out.data_ptr())), "bz_thermal_masses")
        return out

    def set_masses(self, mass2):
        t = torch.as_tensor(mass2, dtype=torch.float64).contiguous()
        if t.numel() != self.Nx * 4 or t.is_cuda:
            raise ValueError("mass2: host array of Nx*4 doubles")
        self._chk(lib().bz_set_masses(self._h, C.c_void_p(t.data_ptr())), "bz_set_masses")

    def energy_diag(self):
        out = torch.empty((self.Nx, 5), dtype=torch.float64)
        self._chk(lib().bz_energy_diag(self._h, C.c_void_p(out.data_ptr())), "bz_energy_diag")
        return out

    def vlasov(self, dt, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_vlasov(self._h, dt, self._dev_ptr(out, self.n_values)), "bz_vlasov")
        return out

    # ---- NEXT rank 1: the paper's own sampler (Eq. 17-21) with massive dispersion
    def collision_paper(self, dt, step, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_collision_paper(self._h, dt, step, self._dev_ptr(out, self.n_values)), "bz_collision_paper")
        return out

    # ---- NEXT rank 3: importance-sampled estimator
    def collision_is(self, dt, step, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_collision_is(self._h, dt, step, self._dev_ptr(out, self.n_values)), "bz_collision_is")
        return out

    def debug_samples_is(self, step, xcell, pbegin, pend, m2):
        n = pend - pbegin
        cells = torch.empty((n, self.Ns, 4), dtype=torch.int32, device=self.device)
        stu = torch.empty((n, self.Ns, 3), dtype=torch.float64, device=self.device)
        w = torch.empty((n, self.Ns), dtype=torch.float64, device=self.device)
        self._chk(lib().bz_debug_samples_is(self._h, step, xcell, pbegin, pend, m2, C.c_void_p(cells.data_ptr()),
                                            C.c_void_p(stu.data_ptr()), C.c_void_p(w.data_ptr())), "bz_debug_samples_is")
        return cells, stu, w

    # ---- NEXT rank 3, other half: in-box sampling of the CM direction
    def collision_box(self, dt, step, out=None):
        if out is None:
            out = torch.empty(self.shape, dtype=torch.float64, device=self.device)
        self._chk(lib().bz_collision_box(self._h, dt, step, self._dev_ptr(out, self.n_values)), "bz_collision_box")
        return out

    def debug_samples_box(self, step, xcell, pbegin, pend):
        n = pend - pbegin
        cells = torch.empty((n, self.Ns, 4), dtype=torch.int32, device=self.device)
        stu = torch.empty((n, self.Ns, 3), dtype=torch.float64, device=self.device)
        w = torch.empty((n, self.Ns), dtype=torch.float64, device=self.device)
        self._chk(lib().bz_debug_samples_box(self._h, step, xcell, pbegin, pend, C.c_void_p(cells.data_ptr()),
                                             C.c_void_p(stu.data_ptr()), C.c_void_p(w.data_ptr())), "bz_debug_samples_box")
        return cells, stu, w

    def set_collision(self, mode):
        self._chk(lib().bz_set_collision(self._h, mode), "bz_set_collision")

    def debug_paper_samples(self, step, xcell, pbegin, pend, msq):
        n = pend - pbegin
        cells = torch.empty((n, self.Ns, 6), dtype=torch.int32, device=self.device)
        stu = torch.empty((n, self.Ns, 6), dtype=torch.float64, device=self.device)
        m = (C.c_double * 4)(*msq)
        self._chk(lib().bz_debug_paper_samples(self._h, step, xcell, pbegin, pend, m, C.c_void_p(cells.data_ptr()),
                                               C.c_void_p(stu.data_ptr())), "bz_debug_paper_samples")
        return cells, stu

    def set_transport(self, scheme):
        self._chk(lib().bz_set_transport(self._h, scheme), "bz_set_transport")

    def step(self, dt):
        self._chk(lib().bz_step(self._h, dt), "bz_step")

    def step_n(self, dt, n):
        """bz_step_n: n steps without returning to the host in between (two steps per replay of a captured CUDA graph)."""
        self._chk(lib().bz_step_n(self._h, dt, int(n)), "bz_step_n")

    def step_host(self, dt, f_in, f_out):
        """bz_step_host: f_in, f_out are CPU float64 tensors (pinned for full copy speed) of n_values elements."""
        for t in (f_in, f_out):
            if t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or t.numel() != self.n_values:
                raise ValueError("expected contiguous CPU float64 tensors with %d elements" % self.n_values)
        self._chk(lib().bz_step_host(self._h, dt, C.c_void_p(f_in.data_ptr()), C.c_void_p(f_out.data_ptr())), "bz_step_host")
        return f_out

    def moments(self, out=None):
        n = 2 * self.S * self.Nx + 2 * self.S + self.Nx
        if out is None:
            out = torch.empty(n, dtype=torch.float64)
        self._chk(lib().bz_moments(self._h, C.c_void_p(out.data_ptr())), "bz_moments")
        a = self.Nx * self.S * 2
        return {"ne": out[:a].view(self.Nx, self.S, 2), "tot": out[a:a + 2 * self.S].view(self.S, 2),
                "m2": out[a + 2 * self.S:]}

    def set_profile(self, on):
        self._chk(lib().bz_set_profile(self._h, int(bool(on))), "bz_set_profile")

    def get_profile(self, group=0):
        """(milliseconds, regions) of group 0 = collision kernel, 1 = stream + Euler kernel since the last call."""
        ms, n = C.c_double(), C.c_int()
        self._chk(lib().bz_get_profile(self._h, group, C.byref(ms), C.byref(n)), "bz_get_profile")
        return ms.value, n.value

    def sample_counts(self, reset=False):
        """(generated, accepted) kinematic samples of the hot path's collision kernel since the last reset."""
        g, a = C.c_ulonglong(), C.c_ulonglong()
        self._chk(lib().bz_get_sample_counts(self._h, C.byref(g), C.byref(a), int(bool(reset))), "bz_get_sample_counts")
        return g.value, a.value

    def msq_sign_counts(self, step, xbegin, xend):
        """bz_msq_sign_counts (reading S8): (accepted samples, counts[kind][crossed] of negative |M|^2 among them) for the
        samples bz_collision draws at `step` in spatial cells [xbegin, xend)."""
        out = (C.c_ulonglong * 15)()
        self._chk(lib().bz_msq_sign_counts(self._h, step, xbegin, xend, out), "bz_msq_sign_counts")
        return int(out[0]), [[int(out[1 + 2 * k]), int(out[2 + 2 * k])] for k in range(7)]

    def debug_samples(self, step, xcell, pbegin, pend, want_stu=True):
        n = pend - pbegin
        cells = torch.empty((n, self.Ns, 4), dtype=torch.int32, device=self.device)
        stu = torch.empty((n, self.Ns, 3), dtype=torch.float64, device=self.device) if want_stu else None
        self._chk(lib().bz_debug_samples(self._h, step, xcell, pbegin, pend, C.c_void_p(cells.data_ptr()),
                                         C.c_void_p(stu.data_ptr()) if want_stu else None), "bz_debug_samples")
        return cells, stu


def debug_paper_channels(species):
    """Host only: the paper sampler's ordered channel table as rows (a, b, c, d, kind, crossed, key)."""
    import numpy as np
    sp = (C.c_int * len(species))(*species)
    out = np.zeros((256, 7), dtype=np.int32)
    n = lib().bz_debug_paper_channels(sp, len(species), out.ctypes.data_as(C.POINTER(C.c_int)), 256)
    if n < 0:
        raise BzError("bz_debug_paper_channels: bad species list")
    return out[:n]


NOALLOC_MAX_ROWS = 65536      # bz_moments_noalloc: spatial cells x species its fixed scratch holds (include/bz.h)


def moments_noalloc(f, out, nx=1, ny=1, nz=1, dx=1.0, np_=15, pmin=-3.0, pmax=3.0, species=(0,), alpha_s=0.3, m_D=0.0,
                    stream=None):
    """bz_moments_noalloc: the moments of Boltzmann.moments() for a caller that holds f itself and cannot allocate device
    memory (its f fills the card, it must not stall other streams with cudaMalloc, or a framework pool owns the memory).

    f: contiguous CUDA float64 tensor, Nx*S*Np values in the library's layout (read only).  out: contiguous CUDA float64
    tensor of 2*S*Nx + 2*S + Nx values, overwritten.  BOTH come from the caller: nothing is allocated here or in the
    library, the scratch between the two kernels is a fixed 1.5 MiB array inside libbz.so, which limits the call to
    Nx*S <= NOALLOC_MAX_ROWS (BzError otherwise) and is shared by all calls: do not let two of them overlap on the GPU.
    Enqueued on `stream` (default: torch's current stream of f's device); returns views of `out` like moments().
    The first call on a device also resolves the scratch's address: make it before any stream capture."""
    S, Nx, Np = len(species), nx * ny * nz, np_ ** 3
    n_out = 2 * S * Nx + 2 * S + Nx
    for t, n in ((f, Nx * S * Np), (out, n_out)):
        if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n):
            raise ValueError("expected a contiguous CUDA float64 tensor with %d elements" % n)
    if out.device != f.device:
        raise ValueError("f and out must be on the same device")
    if stream is None:
        stream = torch.cuda.current_stream(f.device)
    grid = Grid(nx, ny, nz, dx, np_, pmin, pmax)
    L = lib()
    with torch.cuda.device(f.device):
        rc = L.bz_moments_noalloc(C.byref(grid), (C.c_int * S)(*species), S, alpha_s, m_D, C.c_void_p(f.data_ptr()),
                                  C.c_void_p(out.data_ptr()), C.c_void_p(stream.cuda_stream))
    if rc != 0:
        raise BzError("bz_moments_noalloc failed (%d): %s" % (rc, L.bz_noalloc_last_error().decode()))
    a = Nx * S * 2
    return {"ne": out[:a].view(Nx, S, 2), "tot": out[a:a + 2 * S].view(S, 2), "m2": out[a + 2 * S:]}


def measure_fp64_peak():
    """bz_measure_fp64_peak: measured FP64 FMA peak of the current device, TFLOP/s."""
    v = C.c_double()
    rc = lib().bz_measure_fp64_peak(C.byref(v))
    if rc != 0:
        raise BzError("bz_measure_fp64_peak failed (%d)" % rc)
    return v.value


def launch_count():
    """bz_launch_count: CUDA kernels launched by libbz.so in this process so far."""
    return int(lib().bz_launch_count())
