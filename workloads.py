"""Seeded synthetic inputs: the five BASELINE.json configs and their initial distributions.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the
method's arithmetic (no sampling, no matrix elements, no deposits): only grid geometry
(cell-centre coordinates) and the analytic initial conditions of BASELINE.json `configs`
(shape of the paper's own runs: step function Eq. 30-31; 30^3 mixture P:348;
spatial run P:308).  Readings S17-S19 of SURVEY.md 8c are applied here and listed in DESIGN.md.

The paper measures on no public benchmark or dataset; every input is an analytic function
of the cell centre plus, for config 4, a seeded 1 % multiplicative noise.
"""
from dataclasses import dataclass, replace

import numpy as np

ALL_SPECIES = (0, 1, 2, 3, 4, 5, 6)   # g, u, ubar, d, dbar, s, sbar


@dataclass(frozen=True)
class Config:
    name: str
    nx: int            # spatial cells per axis (nx = ny = nz)
    dx: float          # fm
    np_: int           # momentum cells per axis
    pmin: float        # GeV
    pmax: float
    species: tuple
    samples: int       # kinematic samples per (spatial cell, momentum cell)   (S3)
    steps: int
    dt: float          # fm/c
    alpha_s: float = 0.3
    m_D: float = 0.0   # <= 0: regulator mass^2 from the instantaneous f (S7)
    seed: int = 0      # Philox seed of the sampling (only config 0 states it; 0 everywhere)
    init: str = ""
    Qs: float = 1.0
    sigma: float = 0.5
    noise_seed: int = -1

    @property
    def Nx(self):
        return self.nx ** 3

    @property
    def Np(self):
        return self.np_ ** 3

    @property
    def S(self):
        return len(self.species)

    @property
    def n_values(self):
        return self.Nx * self.S * self.Np

    @property
    def samples_per_step(self):
        return self.Nx * self.Np * self.samples


CONFIGS = (
    Config("cfg0_glue15", 1, 1.0, 15, -3.0, 3.0, (0,), 64, 10, 0.01, init="glue_step", Qs=1.0),
    Config("cfg1_quarks20", 1, 1.0, 20, -3.0, 3.0, (1, 2, 3, 4, 5, 6), 128, 20, 0.01, init="quark_step", Qs=1.0),
    Config("cfg2_mix30", 1, 1.0, 30, -4.0, 4.0, ALL_SPECIES, 256, 50, 0.005, init="mix_homog", Qs=1.5),
    Config("cfg3_inhom8x20", 8, 0.2, 20, -3.0, 3.0, ALL_SPECIES, 64, 20, 0.005, init="mix_gauss", Qs=1.0, sigma=0.5),
    Config("cfg4_inhom16x24", 16, 0.1, 24, -4.0, 4.0, ALL_SPECIES, 64, 10, 0.0025, init="mix_gauss", Qs=2.0, sigma=0.6,
           noise_seed=1),
)

# The largest grid the paper's program handles, "on GPU clusters" (n_x,y,z = 20, n_px,py,pz = 40), with the momentum box
# of its 40^3 runs and all seven species: 3.58e9 phase-space values, 28.7 GB per copy.  Not one of BASELINE.json's
# configs: the maximum-size case of the parity tests (it fits one B200: f, f_new and the two cell-major copies are 123 GB).
PAPER_LARGEST = Config("paper_largest_20x40", 20, 0.1, 40, -2.0, 2.0, ALL_SPECIES, 64, 1, 0.0025, init="mix_gauss", Qs=1.0, sigma=0.6)


def scaled(cfg, **kw):
    """Same physics, smaller grid / fewer samples: the parity-test cases the oracle finishes in seconds."""
    return replace(cfg, **kw)


def momentum_centres(cfg):
    """|p| at the cell centres, shape (Np,), pcell = ipx + n*(ipy + n*ipz)."""
    n = cfg.np_
    dp = (cfg.pmax - cfg.pmin) / n
    c = cfg.pmin + (np.arange(n) + 0.5) * dp
    pz, py, px = np.meshgrid(c, c, c, indexing="ij")
    return np.sqrt(px ** 2 + py ** 2 + pz ** 2).reshape(-1), (px.reshape(-1), py.reshape(-1), pz.reshape(-1))


def spatial_profile(cfg):
    """Gaussian exp(-r^2/(2 sigma^2)) at the spatial cell centres, r from the box centre (S17), shape (Nx,)."""
    n = cfg.nx
    c = (np.arange(n) + 0.5) * cfg.dx - 0.5 * n * cfg.dx
    z, y, x = np.meshgrid(c, c, c, indexing="ij")
    r2 = (x ** 2 + y ** 2 + z ** 2).reshape(-1)
    return np.exp(-r2 / (2.0 * cfg.sigma ** 2))


def initial_f(cfg):
    """Initial occupation numbers, shape (Nx, S, Np) float64, C-contiguous (layout of SURVEY.md 8a)."""
    pabs, _ = momentum_centres(cfg)
    theta = (pabs <= cfg.Qs).astype(np.float64)            # theta at the cell centre, theta(0) = 1 (S19)
    f = np.zeros((cfg.Nx, cfg.S, cfg.Np), dtype=np.float64)
    for a, sp in enumerate(cfg.species):
        glue = sp == 0
        if cfg.init == "glue_step":
            f[:, a, :] = 0.1 * theta
        elif cfg.init == "quark_step":
            f[:, a, :] = 0.5 * theta
        elif cfg.init == "mix_homog":
            f[:, a, :] = (0.1 / cfg.alpha_s) * theta if glue else 0.05 * np.exp(-pabs / 0.5)
        elif cfg.init == "mix_gauss":
            amp = 0.1 if glue else 0.1 * 0.02
            f[:, a, :] = amp * spatial_profile(cfg)[:, None] * theta[None, :]
        else:
            raise ValueError("unknown init %r" % cfg.init)
    if cfg.noise_seed >= 0:
        # uniform 1 % multiplicative perturbation (config 4), numpy's own Philox bit generator
        rng = np.random.Generator(np.random.Philox(key=cfg.noise_seed))
        for x in range(cfg.Nx):
            f[x] *= 1.0 + 0.01 * (2.0 * rng.random((cfg.S, cfg.Np)) - 1.0)
    return f


def random_f(cfg, seed, lo=0.02, hi=0.6):
    """Dense random occupation numbers in [lo, hi) (the shape of the paper's Fig. 2 test)."""
    rng = np.random.Generator(np.random.Philox(key=seed))
    return lo + (hi - lo) * rng.random((cfg.Nx, cfg.S, cfg.Np))
