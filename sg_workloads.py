"""Seeded synthetic inputs and the BASELINE.json workload table.

This module serves both the oracle (oracle/) and the CUDA path (paper_1309_1599_b200/) and holds none
of the method's arithmetic: no local field, no update rule, no Philox.  It only names the five
workloads of BASELINE.json (`configs`) and draws generic test inputs (arbitrary coupling matrices,
unit vectors, rotations) with numpy's own generator.  The recipe is stated in DESIGN.md section 5.
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class Workload:
    name: str
    L: int
    n_samples: int
    n_replicas: int
    n_temps: int
    beta_min: float
    beta_max: float
    n_or: int          # overrelaxation sweeps per unit (1 HB + n_or OR + 1 PT)
    sigma_D: float     # std of the off-diagonal anisotropy entries
    measure_every: int  # units between measurements
    units: int         # run length BASELINE.json quotes
    seed: int = 1

    @property
    def n_sites(self):
        return self.L ** 3

    @property
    def n_copies(self):
        return self.n_replicas * self.n_temps

    @property
    def betas(self):
        """beta linearly spaced between beta_min and beta_max (BASELINE.json configs)."""
        return np.linspace(self.beta_min, self.beta_max, self.n_temps)

    @property
    def updates_per_unit(self):
        """single-spin updates in one unit: (1 HB + n_or OR) sweeps of S*C*N sites."""
        return (1 + self.n_or) * self.n_samples * self.n_copies * self.n_sites


# BASELINE.json `configs`, in order.  "variance raised to 2" => sigma_D = sqrt(2) for config 3.
CONFIGS = [
    Workload("cfg0_L4", 4, 1, 2, 4, 0.6, 1.6, 4, 1.0, 1, 1000),
    Workload("cfg1_L8", 8, 8, 4, 16, 0.5, 2.0, 8, 1.0, 1, 10000),
    Workload("cfg2_L16", 16, 32, 4, 24, 0.5, 2.2, 16, 1.0, 10, 10000),
    Workload("cfg3_L32", 32, 16, 4, 32, 0.5, 2.4, 16, 2.0 ** 0.5, 1, 5000),
    Workload("cfg4_L64", 64, 4, 4, 48, 0.5, 2.6, 32, 1.0, 10, 1000),
]


def random_unit_vectors(rng, shape):
    """Array [..., 3] of unit vectors, isotropic."""
    v = rng.standard_normal(tuple(shape) + (3,))
    return v / np.linalg.norm(v, axis=-1, keepdims=True)


def random_spins(rng, n_copies, n_sites, fp32=True):
    """[n_copies][3][N] unit spins; fp32=True rounds the components to fp32-representable doubles."""
    s = np.moveaxis(random_unit_vectors(rng, (n_copies, n_sites)), -1, 1)
    s = np.ascontiguousarray(s)
    return s.astype(np.float32).astype(np.float64) if fp32 else s


def random_couplings(rng, n_sites, kind="general", sigma_D=1.0, fp32=True):
    """[3][N][3][3] coupling matrices drawn with numpy: 'general' (9 independent normals),
    'offdiag_sym' (a*1 + symmetric off-diagonal), 'isotropic' (a*1)."""
    if kind == "general":
        M = rng.standard_normal((3, n_sites, 3, 3))
    else:
        a = rng.standard_normal((3, n_sites))
        M = a[..., None, None] * np.eye(3)
        if kind == "offdiag_sym":
            d = sigma_D * rng.standard_normal((3, n_sites, 3))
            for k, (p, q) in enumerate([(0, 1), (0, 2), (1, 2)]):
                M[..., p, q] += d[..., k]
                M[..., q, p] += d[..., k]
        elif kind != "isotropic":
            raise ValueError(kind)
    M = np.ascontiguousarray(M)
    return M.astype(np.float32).astype(np.float64) if fp32 else M


def random_rotations(rng, n, proper=True):
    """n random orthogonal 3x3 matrices (QR of a Gaussian matrix); proper=True forces det = +1."""
    A = rng.standard_normal((n, 3, 3))
    Q, Rm = np.linalg.qr(A)
    Q = Q * np.sign(np.diagonal(Rm, axis1=1, axis2=2))[:, None, :]
    if proper:
        Q[:, :, 0] *= np.linalg.det(Q)[:, None]
    return Q


def shard_samples(n_samples_per_rank, rank):
    """Weak-scaling shard: rank r owns the global samples
    [r*n, (r+1)*n); returns first_sample.  Samples are independent, no collective."""
    return rank * n_samples_per_rank
