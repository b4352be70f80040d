"""Seeded synthetic inputs.

This module holds NONE of the method's arithmetic: it only draws particle positions and
normalised momenta with numpy's PCG64 generator.  It is the one module that serves both the
CPU oracle (``oracle/``) and the CUDA path: the tests and ``bench.py`` generate inputs here
and hand the same host arrays to both sides.  It imports neither of them.

The paper's own workloads are synthetic (particles uniform in a cube with
identical momenta); BASELINE.json's configs describe relativistic electron bunches.  Units:
metres for positions, dimensionless gamma*beta for momenta, Coulomb for charges.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

ELECTRON_CHARGE = -1.602176634e-19  # C, exact SI value


@dataclass
class Workload:
    """One synthetic bunch plus the FMM parameters BASELINE.json quotes for it."""
    name: str
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    px: np.ndarray
    py: np.ndarray
    pz: np.ndarray
    q: float = ELECTRON_CHARGE
    order_n: int = 4
    leaf_size: int = 64
    theta: float = 0.5
    seed: int = 0
    note: str = ""
    extra: dict = field(default_factory=dict)

    @property
    def N(self) -> int:
        return int(self.x.shape[0])

    def arrays(self):
        return self.x, self.y, self.z, self.px, self.py, self.pz


def momenta(rng: np.random.Generator, N: int, gamma0: float, sigma_delta: float,
            sigma_perp: float = 1e-3):
    """gamma_j = gamma0 (1 + sigma_delta N(0,1)); px, py ~ N(0, sigma_perp);
    pz = +sqrt(gamma_j^2 - 1 - px^2 - py^2)."""
    gam = gamma0 * (1.0 + sigma_delta * rng.standard_normal(N))
    px = sigma_perp * rng.standard_normal(N)
    py = sigma_perp * rng.standard_normal(N)
    pz = np.sqrt(np.maximum(gam * gam - 1.0 - px * px - py * py, 0.0))
    return px, py, pz


def gaussian_positions(rng: np.random.Generator, N: int, sigma=(1e-3, 1e-3, 1e-4)):
    return (sigma[0] * rng.standard_normal(N), sigma[1] * rng.standard_normal(N),
            sigma[2] * rng.standard_normal(N))


def ellipsoid_positions(rng: np.random.Generator, N: int, semi=(1e-3, 1e-3, 2e-4)):
    """Uniform in the ellipsoid: direction = normalised 3-D normal, radius = U^(1/3)."""
    v = rng.standard_normal((N, 3))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    r = rng.random(N) ** (1.0 / 3.0)
    return semi[0] * r * v[:, 0], semi[1] * r * v[:, 1], semi[2] * r * v[:, 2]


def gaussian_bunch(N: int, gamma0: float, sigma_delta: float, seed: int, *, order_n: int,
                   leaf_size: int, theta: float, name: str = "gaussian") -> Workload:
    rng = np.random.default_rng(seed)
    x, y, z = gaussian_positions(rng, N)
    px, py, pz = momenta(rng, N, gamma0, sigma_delta)
    return Workload(name, x, y, z, px, py, pz, order_n=order_n, leaf_size=leaf_size,
                    theta=theta, seed=seed)


def ellipsoid_bunch(N: int, gamma0: float, sigma_delta: float, seed: int, *, order_n: int,
                    leaf_size: int, theta: float, name: str = "ellipsoid") -> Workload:
    rng = np.random.default_rng(seed)
    x, y, z = ellipsoid_positions(rng, N)
    px, py, pz = momenta(rng, N, gamma0, sigma_delta)
    return Workload(name, x, y, z, px, py, pz, order_n=order_n, leaf_size=leaf_size,
                    theta=theta, seed=seed)


def paper_cube(N: int = 1_280_000, gamma0: float = 50.0, seed: int = 1007, *, order_n: int = 4,
               leaf_size: int | None = None, theta: float = 0.5) -> Workload:
    """Stand-in for the paper's own workload: uniform in [0,1]^3 m, every
    particle with p = (0, 0, sqrt(gamma^2 - 1)); N0 = (n+1)^3."""
    rng = np.random.default_rng(seed)
    x, y, z = rng.random(N), rng.random(N), rng.random(N)
    pz = np.full(N, np.sqrt(gamma0 * gamma0 - 1.0))
    return Workload("paper_cube", x, y, z, np.zeros(N), np.zeros(N), pz, order_n=order_n,
                    leaf_size=(order_n + 1) ** 3 if leaf_size is None else leaf_size,
                    theta=theta, seed=seed)


def config(i: int, N: int | None = None) -> Workload:
    """BASELINE.json ``configs[i-1]`` (1-based, as SURVEY.md 8(d) numbers them).
    ``N`` overrides the particle count (used for down-sized parity cases)."""
    if i == 1:
        w = gaussian_bunch(N or 4096, 10.0, 0.01, 1001, order_n=4, leaf_size=64, theta=0.5,
                           name="config1_gaussian_4k")
    elif i == 2:
        w = gaussian_bunch(N or 65536, 10.0, 0.01, 1002, order_n=5, leaf_size=128, theta=0.5,
                           name="config2_gaussian_64k")
    elif i == 3:
        w = ellipsoid_bunch(N or 1_048_576, 30.0, 0.005, 1003, order_n=6, leaf_size=256,
                            theta=0.5, name="config3_ellipsoid_1m")
    elif i == 4:
        w = gaussian_bunch(N or 4_194_304, 100.0, 0.02, 1004, order_n=6, leaf_size=256,
                           theta=0.4, name="config4_gaussian_4m_gamma100")
    elif i == 5:
        w = gaussian_bunch(N or 1_048_576, 10.0, 0.01, 1005, order_n=6, leaf_size=256,
                           theta=0.5, name="config5_gaussian_1m_sweep")
    elif i == 6:  # "5b": all-pairs ceiling
        w = gaussian_bunch(N or 262_144, 10.0, 0.01, 1006, order_n=4, leaf_size=256, theta=0.5,
                           name="config5b_allpairs_256k")
    elif i == 7:  # stand-in for the paper's Fig. 2-4 workload
        w = paper_cube(N or 1_280_000, order_n=4, theta=0.5)
        w.name = "paperP_cube_1p28m"
    elif i == 8:  # the paper's CPU-vs-GPU run: N = 2.56e7, n = 4, N0 = 125, eta = 0.5
        w = paper_cube(N or 25_600_000, order_n=4, theta=0.5)
        w.name = "paperP_cube_25p6m"
    else:
        raise ValueError(f"no such config: {i}")
    return w
