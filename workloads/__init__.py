"""Seeded synthetic inputs for the ray-march hot path (configs C0..C4 of BASELINE.json).

This top-level module is the ONE piece shared by the CUDA path's tests/bench and the oracle's tests: it only
builds input arrays (j, kappa, sources) and the scalar call arguments.  It holds none of the
method's arithmetic (no marching, no interpolation, no direction lattice) and imports neither the
CUDA binding nor ``oracle/``.

The inputs stand in for data the paper used but that is not available here: the jf1uids turbulent
hydro snapshots with kappa ∝ rho and sources on the top-0.1 % density peaks (§3
"Turbulent snapshots from hydro"), the 128³ / 4,096 rays / 2,097 sources timing set-up
 and the uniform-medium point-source benchmark.  The recipe
(restated in DESIGN.md §5) keeps the shapes, the kappa ∝ rho prescription and the
source-placement rule.

Layout of every field: ``[nx][ny][nz][n_bins]`` float32, C order, bin innermost.  Source positions
are ``[n_src][3]`` float32 grid coordinates; voxel (a, b, c) is sampled at coordinate (a, b, c).
All arrays are generated in float64 and cast to float32 ONCE, so the oracle and the CUDA path read
bit-identical inputs.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = ["Workload", "lognormal_density", "bin_scalings", "make_config", "CONFIG_NAMES",
           "uniform_medium", "gaussian_blob"]

CONFIG_NAMES = ("C0", "C1", "C2", "C3", "C4")


@dataclass
class Workload:
    """One call's worth of inputs.  ``j``/``kappa``: [nx,ny,nz,n_bins] f32; ``sources``: [n_src,3] f32."""
    name: str
    j: np.ndarray
    kappa: np.ndarray
    sources: np.ndarray
    n_rays: int          # N_Omega
    step_size: float     # Delta s, cells
    c: float             # radiation velocity
    dt: float            # time step
    n_steps: int
    substeps_per_step: int   # N_s the recipe intends (integer ratio in all five configs)
    meta: dict = field(default_factory=dict)

    @property
    def shape(self):
        return self.j.shape[:3]

    @property
    def n_bins(self) -> int:
        return int(self.j.shape[3])

    @property
    def n_src(self) -> int:
        return int(self.sources.shape[0])

    @property
    def ray_substeps(self) -> int:
        return self.n_src * self.n_rays * self.n_steps * self.substeps_per_step

    @property
    def updates(self) -> int:
        """ray-substep-bin updates: the unit of BASELINE.json's metric."""
        return self.ray_substeps * self.n_bins

    def subset_sources(self, idx) -> "Workload":
        """Same medium, a subset of the sources (the field is additive over sources)."""
        idx = np.asarray(idx)
        return Workload(self.name + f"[{len(idx)}src]", self.j, self.kappa,
                        np.ascontiguousarray(self.sources[idx]), self.n_rays, self.step_size, self.c,
                        self.dt, self.n_steps, self.substeps_per_step, dict(self.meta))


def lognormal_density(n: int, seed: int, sigma_ln: float) -> np.ndarray:
    """rho = exp(sigma_ln * g), g a unit-variance Gaussian random field with P(k) ∝ k^(-11/3).

    Stand-in for the turbulent density of PAPER.md:54.  float64, shape (n, n, n), median 1.
    """
    rng = np.random.default_rng(seed)
    w = rng.standard_normal((n, n, n))
    W = np.fft.rfftn(w, axes=(0, 1, 2))
    k0 = np.fft.fftfreq(n) * n
    k2 = np.fft.rfftfreq(n) * n
    kk = np.sqrt(k0[:, None, None] ** 2 + k0[None, :, None] ** 2 + k2[None, None, :] ** 2)
    kk[0, 0, 0] = 1.0
    W *= kk ** (-11.0 / 6.0)          # amplitude ∝ k^(-11/6)  =>  P(k) ∝ k^(-11/3)
    W[0, 0, 0] = 0.0
    g = np.fft.irfftn(W, s=(n, n, n), axes=(0, 1, 2))
    g -= g.mean()
    g /= g.std()
    return np.exp(sigma_ln * g)


def bin_scalings(n_bins: int):
    """nu_b log-spaced from 1 to 4; kappa_b = kappa * nu_b^-3, j_b = j * exp(-nu_b) (BASELINE.json configs[3])."""
    if n_bins == 1:
        return np.ones(1), np.ones(1)
    nu = 4.0 ** (np.arange(n_bins) / (n_bins - 1))
    return nu ** -3.0, np.exp(-nu)


def _with_bins(base: np.ndarray, scale: np.ndarray) -> np.ndarray:
    out = base[..., None] * scale[None, None, None, :]
    return np.ascontiguousarray(out.astype(np.float32))


def _top_density_cells(rho: np.ndarray, n: int) -> np.ndarray:
    """Integer coordinates of the n highest-density cells; ties -> lower linear index."""
    order = np.argsort(-rho.ravel(), kind="stable")[:n]
    return np.stack(np.unravel_index(order, rho.shape), axis=1).astype(np.float32)


def uniform_medium(n: int, j0: float, kappa0: float, n_bins: int = 1):
    """Uniform j ≡ j0, kappa ≡ kappa0 (the medium of the closed-form pins)."""
    j = np.full((n, n, n, n_bins), j0, dtype=np.float32)
    k = np.full((n, n, n, n_bins), kappa0, dtype=np.float32)
    return j, k


def gaussian_blob(shape, centre, sigma: float, amplitude: float = 1.0) -> np.ndarray:
    """amplitude * exp(-r²/(2 sigma²)), r measured from ``centre`` (grid coordinates); float64 [nx,ny,nz]."""
    ax = [np.arange(s, dtype=np.float64) - c for s, c in zip(shape, centre)]
    r2 = ax[0][:, None, None] ** 2 + ax[1][None, :, None] ** 2 + ax[2][None, None, :] ** 2
    return amplitude * np.exp(-r2 / (2.0 * sigma * sigma))


def make_config(name: str) -> Workload:
    """Build config ``C0``..``C4`` (BASELINE.json configs[0..4]); seeds as in SURVEY.md §8(d)."""
    if name == "C0":
        n = 16
        ctr = (n - 1) / 2.0
        j = gaussian_blob((n, n, n), (ctr, ctr, ctr), 2.0)[..., None].astype(np.float32)
        kappa = np.full((n, n, n, 1), 0.1, dtype=np.float32)
        src = np.array([[ctr, ctr, ctr]], dtype=np.float32)
        return Workload("C0", np.ascontiguousarray(j), kappa, src, 64, 0.5, 1.0, 12.0, 1, 24,
                        {"grid": "16^3", "medium": "uniform kappa=0.1, Gaussian j sigma=2"})
    if name == "C1":
        n = 64
        rho = lognormal_density(n, 938901, 1.0)
        one = np.ones(1)
        src = np.random.default_rng(939901).uniform(0.0, n - 1.0, (16, 3)).astype(np.float32)
        return Workload("C1", _with_bins(1e-3 * rho ** 2, one), _with_bins(0.05 * rho, one), src,
                        1024, 0.5, 1.0, 16.0, 4, 32,
                        {"grid": "64^3", "medium": "lognormal sigma_ln=1, seed 938901"})
    if name in ("C2", "C3"):
        n = 128
        rho = lognormal_density(n, 938902, 1.5)
        if name == "C2":
            one = np.ones(1)
            return Workload("C2", _with_bins(1e-4 * rho ** 2, one), _with_bins(0.02 * rho, one),
                            _top_density_cells(rho, 2097), 4096, 0.5, 1.0, 222.0, 1, 444,
                            {"grid": "128^3", "medium": "lognormal sigma_ln=1.5, seed 938902",
                             "sources": "2,097 highest-density cells"})
        ks, js = bin_scalings(8)
        return Workload("C3", _with_bins(1e-4 * rho ** 2, js), _with_bins(0.02 * rho, ks),
                        _top_density_cells(rho, 256), 4096, 0.5, 1.0, 64.0, 2, 128,
                        {"grid": "128^3 x 8 bins", "medium": "lognormal sigma_ln=1.5, seed 938902",
                         "sources": "256 highest-density cells"})
    if name == "C4":
        n = 256
        rho = lognormal_density(n, 938904, 2.0)
        ks, js = bin_scalings(4)
        src = np.random.default_rng(939904).uniform(0.0, n - 1.0, (64, 3)).astype(np.float32)
        return Workload("C4", _with_bins(1e-4 * rho ** 2, js), _with_bins(0.02 * rho, ks), src,
                        16384, 0.5, 1.0, 32.0, 8, 64,
                        {"grid": "256^3 x 4 bins", "medium": "lognormal sigma_ln=2, seed 938904"})
    raise ValueError(f"unknown config {name!r}; expected one of {CONFIG_NAMES}")
