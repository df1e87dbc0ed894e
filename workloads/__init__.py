"""Seeded synthetic inputs for the Hermitian PSD-projection path.

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench.
It holds none of the method's arithmetic: it only draws random Hermitian
matrices (as full complex128 arrays) with the spectra BASELINE.json's
`configs` describe.  It never packs, projects, clamps or eigendecomposes.
Packing into the svec layout is done by whichever side consumes the matrix
(oracle.pack in the tests, the library's own pack kernel in bench.py).

Recipe (also stated in DESIGN.md §Inputs):
  * rng = numpy.random.default_rng(20519 + config_number)
  * Haar unitary: QR of an i.i.d. complex Gaussian, then Q <- Q diag(r_ii/|r_ii|)
  * X = Q diag(lam) Q^H, symmetrised once as (X + X^H)/2
  * "N(0, 1e-3)" / "N(0, 1e-2)" are standard deviations
  * config 4's G has Re, Im i.i.d. N(0,1), scaled by 1/sqrt(n)
  * config 5: among the 4080 noise values, 8 draws are each repeated 32 times
    (4 forced positive, 4 forced negative); the 16 large values stay distinct.

There is no public dataset behind the paper's workloads: "a randomly generated
feasible pair of instruments defines a GYNI objective", so
these stand in for ADMM iterates u~ - v (Eq. D33).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional

import numpy as np

BASE_SEED = 20519


@dataclass
class Block:
    """One Hermitian block. `Q`/`lam` are set when the block was built as
    Q diag(lam) Q^H (so tests can form a closed-form reference from them)."""
    X: np.ndarray
    Q: Optional[np.ndarray] = None
    lam: Optional[np.ndarray] = None

    @property
    def n(self) -> int:
        return int(self.X.shape[0])


@dataclass
class Workload:
    name: str
    blocks: List[Block] = field(default_factory=list)

    @property
    def sizes(self) -> List[int]:
        return [b.n for b in self.blocks]

    @property
    def svec_len(self) -> int:
        return int(sum(n * n for n in self.sizes))


def _cgauss(rng: np.random.Generator, *shape: int) -> np.ndarray:
    return rng.standard_normal(shape) + 1j * rng.standard_normal(shape)


def haar_unitary(rng: np.random.Generator, n: int) -> np.ndarray:
    """Haar-distributed unitary: QR of a complex Gaussian with R's diagonal
    phases folded back into Q ("phases fixed", BASELINE.json config 1)."""
    if n == 0:
        return np.zeros((0, 0), dtype=np.complex128)
    q, r = np.linalg.qr(_cgauss(rng, n, n))
    dr = np.diagonal(r)
    ph = np.where(np.abs(dr) > 0, dr / np.where(np.abs(dr) > 0, np.abs(dr), 1.0), 1.0)
    return q * ph[None, :]


def from_spectrum(rng: np.random.Generator, lam: np.ndarray) -> Block:
    lam = np.asarray(lam, dtype=np.float64)
    q = haar_unitary(rng, lam.shape[0])
    x = (q * lam[None, :]) @ q.conj().T
    x = 0.5 * (x + x.conj().T)
    return Block(X=x, Q=q, lam=lam)


def gue_like(rng: np.random.Generator, n: int, scale: float = 1.0) -> Block:
    """(G + G^H)/2 with Re, Im of G i.i.d. N(0,1), times `scale`."""
    g = _cgauss(rng, n, n) * scale
    return Block(X=0.5 * (g + g.conj().T))


def spectrum_gauss(rng, n):
    return rng.standard_normal(n)


def spectrum_admm_lowrank(rng, n, n_big=8, lo=0.5, hi=2.0, sd=1e-3):
    n_big = min(n_big, n)
    big = rng.uniform(lo, hi, size=n_big)
    noise = rng.standard_normal(n - n_big) * sd
    return np.concatenate([big, noise])


def spectrum_clustered(rng, n, n_big=16, lo=0.1, hi=1.0, sd=1e-2, n_clusters=8, mult=32):
    """n_big distinct large values, then noise values of which `n_clusters`
    draws are each repeated `mult` times exactly (half forced > 0, half < 0)."""
    n_big = min(n_big, n)
    rest = n - n_big
    n_clusters = min(n_clusters, rest // mult) if mult > 0 else 0
    singles = rest - n_clusters * mult
    big = rng.uniform(lo, hi, size=n_big)
    cvals = np.abs(rng.standard_normal(n_clusters)) * sd
    cvals[n_clusters // 2:] *= -1.0
    noise = rng.standard_normal(singles) * sd
    lam = np.concatenate([big, np.repeat(cvals, mult), noise])
    return lam[rng.permutation(n)]


# --------------------------------------------------------------------------
# BASELINE.json configs, 1-based as in SURVEY §8(d)
# --------------------------------------------------------------------------

def config1() -> Workload:
    rng = np.random.default_rng(BASE_SEED + 1)
    return Workload("cfg1_n16_haar_gauss", [from_spectrum(rng, spectrum_gauss(rng, 16))])


def config2(n_mats: int = 256, n: int = 81) -> Workload:
    rng = np.random.default_rng(BASE_SEED + 2)
    return Workload(f"cfg2_{n_mats}x_n{n}_gue", [gue_like(rng, n) for _ in range(n_mats)])


def config3(n: int = 625) -> Workload:
    rng = np.random.default_rng(BASE_SEED + 3)
    return Workload(f"cfg3_n{n}_admm_lowrank", [from_spectrum(rng, spectrum_admm_lowrank(rng, n))])


def config4(big=(1296, 2401), n_small: int = 64, small: int = 36) -> Workload:
    rng = np.random.default_rng(BASE_SEED + 4)
    blocks = [gue_like(rng, n, 1.0 / np.sqrt(n)) for n in big]
    blocks += [gue_like(rng, small, 1.0 / np.sqrt(small)) for _ in range(n_small)]
    return Workload("cfg4_mixed_" + "_".join(str(b) for b in big) + f"_{n_small}x{small}", blocks)


def config5(n: int = 4096, n_big: int = 16, n_clusters: int = 8, mult: int = 32) -> Workload:
    rng = np.random.default_rng(BASE_SEED + 5)
    lam = spectrum_clustered(rng, n, n_big=n_big, n_clusters=n_clusters, mult=mult)
    return Workload(f"cfg5_n{n}_clustered", [from_spectrum(rng, lam)])


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make(config: int, **kw) -> Workload:
    return CONFIGS[config](**kw)
