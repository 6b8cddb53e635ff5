"""Synthetic workloads: the five BASELINE.json configs and seeded input generators.

This module holds NO arithmetic of the method (no RPY, no Cholesky, no update,
no Philox): only workload shapes/parameters and numpy-seeded random chains.  It
is the one module both the oracle-side tests and the CUDA-side harness may
import (it imports neither of them).

The paper uses no public dataset: its workloads are random initial chain
configurations of BR-100 (:262, :301), BR-500 (:309-313)
and the N = 199..6399 timing sweep (:297).  The chains below are that workload.
"""
from __future__ import annotations

import math
from dataclasses import dataclass

import numpy as np


def rouse_lambda(n_beads: int) -> float:
    """Stand-in longest relaxation time (reading A12): the paper's lambda values live only in
    Fig. 8 (an image).  Textbook Rouse value in the paper's units."""
    return 1.0 / (12.0 * math.sin(math.pi / (2.0 * n_beads)) ** 2)


@dataclass(frozen=True)
class Workload:
    name: str
    n_chains: int        # C
    n_rods: int          # N
    dt: float
    flow: str            # "none" | "extension" | "shear"
    Wi: float
    steps: int           # steps BASELINE.json quotes for the config
    hstar: float = 0.25
    b: float = 1.0
    noise_seed: int = 0
    init_seed: int = 1000

    @property
    def n_beads(self) -> int:
        return self.n_rods + 1

    @property
    def M(self) -> int:
        return 3 * (self.n_rods + 1)

    @property
    def K(self) -> float:
        return 1.0 / self.dt          # reading A6: K* dt = 1 (PAPER.md:305 pairings)

    @property
    def rate(self) -> float:
        return 0.0 if self.flow == "none" else self.Wi / rouse_lambda(self.n_beads)

    def kappa(self) -> np.ndarray:
        """row-major kappa, v = kappa . r (extension matrix per BASELINE.json, reading A4)."""
        k = np.zeros((3, 3), dtype=np.float64)
        if self.flow == "extension":
            e = self.rate
            k[0, 0], k[1, 1], k[2, 2] = e, -0.5 * e, -0.5 * e
        elif self.flow == "shear":
            k[0, 1] = self.rate
        return k

    def cholesky_flops(self) -> float:
        M = float(self.M)
        return M ** 3 / 3.0 + M ** 2 / 2.0 + M / 6.0


CONFIGS = {
    "c1": Workload("c1", 1, 20, 1e-4, "none", 0.0, 1000, init_seed=1001),
    "c2": Workload("c2", 1024, 100, 1e-4, "extension", 10.0, 10000, init_seed=1002),
    "c3": Workload("c3", 256, 500, 5e-5, "shear", 100.0, 2000, init_seed=1003),
    "c4": Workload("c4", 16, 2000, 1e-4, "none", 0.0, 500, init_seed=1004),
    "c5": Workload("c5", 1, 10000, 5e-5, "extension", 10.0, 50, init_seed=1005),
}


def random_chains(n_chains: int, n_rods: int, b: float = 1.0, seed: int = 0,
                  rod_jitter: float = 0.0) -> np.ndarray:
    """Seeded freely-jointed random walks r[C][N_b][3] (numpy Generator, NOT the method's Philox):
    isotropic rod directions, rod lengths b*(1 + rod_jitter*normal), centre of mass at 0.
    rod_jitter ~ sqrt(dt/2) reproduces the stationary Fraenkel-rod length spread, so that spring
    tensions (and hence the D.F drift) are non-zero in one-step parity tests."""
    rng = np.random.default_rng(seed)
    z = rng.uniform(-1.0, 1.0, size=(n_chains, n_rods))
    phi = rng.uniform(0.0, 2.0 * np.pi, size=(n_chains, n_rods))
    s = np.sqrt(1.0 - z * z)
    q = np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=-1)
    length = b * (1.0 + rod_jitter * rng.standard_normal(size=(n_chains, n_rods, 1)))
    q = q * length
    r = np.zeros((n_chains, n_rods + 1, 3), dtype=np.float64)
    r[:, 1:, :] = np.cumsum(q, axis=1)
    r -= r.mean(axis=1, keepdims=True)
    return np.ascontiguousarray(r)


def random_spring_chains(n_chains: int, n_springs: int, nu: float, b: float = 1.0, seed: int = 0,
                         max_extension: float = 0.9) -> np.ndarray:
    """Seeded bead-spring starts r[C][N_b][3] for the Cohen-Pade comparison model: Gaussian link
    vectors with <Q^2> = nu b^2 (nu Kuhn steps per spring), clipped to max_extension of the full length nu b,
    centre of mass at 0.  numpy Generator only; none of the method's arithmetic."""
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((n_chains, n_springs, 3)) * math.sqrt(nu / 3.0) * b
    length = np.linalg.norm(q, axis=-1, keepdims=True)
    q *= np.minimum(1.0, max_extension * nu * b / length)
    r = np.zeros((n_chains, n_springs + 1, 3), dtype=np.float64)
    r[:, 1:, :] = np.cumsum(q, axis=1)
    r -= r.mean(axis=1, keepdims=True)
    return np.ascontiguousarray(r)
