"""Seeded synthetic workloads for the LinMin hot path (inputs only -- no solver arithmetic).

This module is the ONE piece shared by the CUDA path's tests/bench and the CPU oracle's
tests: it draws libraries, abundances, noise levels and noisy spectra, and holds none of
the method's arithmetic (no Gram matrix, no projection, no solve).  The inputs stand in
for the paper's workloads, none of which is available offline:

  * PAPER.md:128-137 (section 3.1): 1000 sparse mixtures of 32 reference spectra plus
    additional flat/slope spectra, additive zero-mean Gaussian noise with a known
    per-channel standard deviation.
  * PAPER.md:175 (section 3.2), 250, 256, 274 (section 4): cubes of 1e5..3e5 spectra,
    56..110 channels, 36 endmembers.

Shapes, sizes and value ranges follow BASELINE.json `configs[0..4]`; every reading of
its wording is listed in DESIGN.md ("Input recipe").  All draws come from
numpy.random.Generator(PCG64(seed)) in the fixed order
    library -> support sizes -> supports -> weights -> sigma -> noise,
are made in float64, and `A`, `Y`, `sigma` are rounded ONCE to float32; the oracle and
the CUDA path consume these byte-identical float32 arrays.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

__all__ = ["Workload", "CONFIGS", "make_library", "make_workload", "make_cube", "config_names"]


@dataclass
class Workload:
    """One batch of synthetic spectra.  Layouts follow include/linmin.h."""
    name: str
    A: np.ndarray            # (L, R) float32, row-major: A[l, r]; the endmember library
    Y: np.ndarray            # (N, L) float32: one spectrum per row
    sigma: np.ndarray        # (N, L) float32 per-pixel per-channel noise std
    a0: np.ndarray           # (N, R) float64 ground-truth abundances (rows on the simplex)
    wavelength: np.ndarray   # (L,) float64, micrometres
    face: np.ndarray         # (N,) bool: pixel drawn "on a simplex face" (config 2 only)
    seed_key: tuple = field(default_factory=tuple)

    @property
    def N(self) -> int:
        return int(self.Y.shape[0])

    @property
    def L(self) -> int:
        return int(self.A.shape[0])

    @property
    def R(self) -> int:
        return int(self.A.shape[1])


# name -> recipe.  kmin/kmax: number of non-zero abundances per pixel (inclusive).
CONFIGS = {
    "tiny": dict(index=0, L=64, R=8, N=1000, lam=(1.0, 2.5), minerals=6, bands=(1, 3),
                 aerosols=0, pairs=0, k=(2, 3), sigma=(0.005, 0.005), face_frac=0.0, seed=0),
    "omega": dict(index=1, L=128, R=32, N=128 * 1024, lam=(0.95, 2.5), minerals=28, bands=(1, 4),
                  aerosols=2, pairs=0, k=(1, 5), sigma=(0.002, 0.01), face_frac=0.0, seed=1),
    "crism": dict(index=2, L=240, R=64, N=640 * 480, lam=(1.0, 2.6), minerals=60, bands=(1, 4),
                  aerosols=2, pairs=0, k=(1, 6), sigma=(0.002, 0.01), face_frac=0.05, seed=2),
    "stress": dict(index=3, L=240, R=256, N=65536, lam=(1.0, 2.6), minerals=126, bands=(1, 4),
                   aerosols=2, pairs=126, k=(2, 8), sigma=(0.002, 0.01), face_frac=0.0, seed=3),
    # config 4 = a stack of 128 OMEGA-like cubes; library from seed 4, cube c from
    # SeedSequence([4, c]).  make_workload("throughput", n_cubes=...) builds a prefix.
    "throughput": dict(index=4, L=128, R=32, N=128 * 1024, lam=(0.95, 2.5), minerals=28,
                       bands=(1, 4), aerosols=2, pairs=0, k=(1, 5), sigma=(0.002, 0.01),
                       face_frac=0.0, seed=4, cubes=128),
}


def config_names():
    return list(CONFIGS.keys())


def _mineral(rng: np.random.Generator, lam: np.ndarray, bands: tuple) -> np.ndarray:
    """Linear continuum (endpoint reflectances U(0.2,0.6)) times 1..n Gaussian absorption bands
    (depth U(0.05,0.4), FWHM U(20,150) nm, centre uniform on the grid)."""
    lo, hi = lam[0], lam[-1]
    r0, r1 = rng.uniform(0.2, 0.6, size=2)
    spec = r0 + (r1 - r0) * (lam - lo) / (hi - lo)
    nb = int(rng.integers(bands[0], bands[1] + 1))
    for _ in range(nb):
        depth = rng.uniform(0.05, 0.4)
        fwhm_um = rng.uniform(20.0, 150.0) * 1e-3
        centre = rng.uniform(lo, hi)
        s = fwhm_um / 2.3548200450309493
        spec = spec * (1.0 - depth * np.exp(-0.5 * ((lam - centre) / s) ** 2))
    return spec


def make_library(cfg: dict, rng: np.random.Generator):
    """Returns (A64 (L,R) float64, wavelength (L,))."""
    L, R = cfg["L"], cfg["R"]
    lam = np.linspace(cfg["lam"][0], cfg["lam"][1], L)
    cols = [_mineral(rng, lam, cfg["bands"]) for _ in range(cfg["minerals"])]
    # near-collinear partners (config 3): (1-eps)*base_i + eps*new mineral, eps = 0.1
    eps = 0.1
    for i in range(cfg["pairs"]):
        cols.append((1.0 - eps) * cols[i] + eps * _mineral(rng, lam, cfg["bands"]))
    cols.append(np.ones(L))                                   # flat
    cols.append((lam - lam[0]) / (lam[-1] - lam[0]))          # slope, 0..1
    for _ in range(cfg["aerosols"]):                          # smooth extinction shapes
        gamma = rng.uniform(0.5, 2.0)
        cols.append(np.exp(-gamma * (lam - lam[0]) / 1.0))
    A = np.stack(cols, axis=1)
    assert A.shape == (L, R), (A.shape, L, R)
    return A, lam


def _abundances(cfg: dict, rng: np.random.Generator, N: int):
    """Sparse Dirichlet(0.3) abundances.  Returns (a0 (N,R) float64, face (N,) bool)."""
    R = cfg["R"]
    kmin, kmax = cfg["k"]
    k = rng.integers(kmin, kmax + 1, size=N)
    face = np.zeros(N, dtype=bool)
    if cfg["face_frac"] > 0.0:
        face = rng.uniform(size=N) < cfg["face_frac"]
    kk = k + face.astype(k.dtype)            # face pixels draw one extra member, later zeroed
    kcap = int(kk.max())
    # support = first kk entries of a uniformly random permutation of 0..R-1
    order = np.argsort(rng.uniform(size=(N, R)), axis=1)[:, :kcap]
    w = rng.standard_gamma(0.3, size=(N, kcap))
    slot = np.arange(kcap)[None, :]
    w = np.where(slot < kk[:, None], w, 0.0)
    # simplex face: the LAST drawn member gets weight exactly 0 before normalisation
    w = np.where(face[:, None] & (slot == (kk[:, None] - 1)), 0.0, w)
    tot = w.sum(axis=1, keepdims=True)
    bad = tot[:, 0] <= 0.0                    # (all-underflow; practically never) -> pure pixel
    if bad.any():
        w[bad, 0] = 1.0
        tot = w.sum(axis=1, keepdims=True)
    w = w / tot
    a0 = np.zeros((N, R))
    np.put_along_axis(a0, order, w, axis=1)
    return a0, face


def make_cube(cfg: dict, A64: np.ndarray, rng: np.random.Generator, N: int):
    """Draw supports -> weights -> sigma -> noise for N pixels against library A64."""
    L = cfg["L"]
    a0, face = _abundances(cfg, rng, N)
    lo, hi = cfg["sigma"]
    if lo == hi:
        sigma = np.full((N, L), lo)
    else:
        sigma = rng.uniform(lo, hi, size=(N, L))
    noise = rng.standard_normal(size=(N, L))
    Y = a0 @ A64.T + sigma * noise
    return Y.astype(np.float32), sigma.astype(np.float32), a0, face


def make_workload(name: str, N: Optional[int] = None, n_cubes: Optional[int] = None,
                  first_cube: int = 0) -> Workload:
    """Build config `name`.  `N` truncates the number of pixels drawn for configs 0-3 (the
    stream order library -> supports -> ... means a truncated workload is NOT a prefix of the
    full one; tests that need the full config ask for it).  For "throughput", `n_cubes`
    cubes starting at `first_cube` are built, each exactly as in the full config."""
    cfg = CONFIGS[name]
    seed = cfg["seed"]
    if name == "throughput":
        rng_lib = np.random.Generator(np.random.PCG64(seed))
        A64, lam = make_library(cfg, rng_lib)
        n_cubes = cfg["cubes"] if n_cubes is None else n_cubes
        per = cfg["N"] if N is None else N
        Ys, Ss, As, Fs = [], [], [], []
        for c in range(first_cube, first_cube + n_cubes):
            rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, c])))
            Y, s, a0, face = make_cube(cfg, A64, rng, per)
            Ys.append(Y); Ss.append(s); As.append(a0); Fs.append(face)
        return Workload(name, A64.astype(np.float32), np.concatenate(Ys), np.concatenate(Ss),
                        np.concatenate(As), lam, np.concatenate(Fs), (seed, first_cube, n_cubes))
    rng = np.random.Generator(np.random.PCG64(seed))
    A64, lam = make_library(cfg, rng)
    n = cfg["N"] if N is None else N
    Y, s, a0, face = make_cube(cfg, A64, rng, n)
    return Workload(name, A64.astype(np.float32), Y, s, a0, lam, face, (seed,))
