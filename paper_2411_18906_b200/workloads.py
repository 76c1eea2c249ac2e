"""Seeded synthetic workloads (BASELINE.json:configs) -- INPUT GENERATORS ONLY.

This module serves both the CUDA path and the CPU oracle with identical inputs and holds none of the
method's arithmetic (no SRO, no objective, no proposal logic).  It imports neither `oracle/` nor the CUDA
binding.  The workloads stand in for the paper's: lattice supercells S = A*L^3, a random start
 and a user-given target alpha.  The paper uses no dataset; nothing here is taken from one.

The target draw follows DESIGN.md reading A21: for the off-diagonal pairs (i<j) in row-major order with
idx = 0, 1, ...: u = Philox4x32-10(ctr=(idx, 0, 0xFFFFFFFE, 0), key=(seed lo, seed hi))[0] / 2^32,
alpha_ij = alpha_ji = lo + (hi - lo) * u; the diagonal follows from the sum rule sum_j c_j alpha_ij = 0.
(The tiny Philox below only generates inputs; the method's RNG lives in the kernels and, separately, in the oracle.)
"""
from dataclasses import dataclass, field
from typing import List, Optional, Tuple

import numpy as np

_M0, _M1, _W0, _W1 = 0xD2511F53, 0xCD9E8D57, 0x9E3779B9, 0xBB67AE85
_MASK = 0xFFFFFFFF


def _philox_word0(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for r in range(10):
        if r:
            k0 = (k0 + _W0) & _MASK
            k1 = (k1 + _W1) & _MASK
        p0, p1 = _M0 * c0, _M1 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & _MASK, p1 & _MASK, ((p0 >> 32) ^ c3 ^ k1) & _MASK, p0 & _MASK
    return c0


def target_alpha(n_species, n_shells, conc, seed=None, lo=0.0, hi=0.0):
    """alpha_target[S][M][M]: shell 1 drawn (if seed is not None), all other shells zero."""
    t = np.zeros((n_shells, n_species, n_species), dtype=np.float64)
    if seed is None:
        return t
    key = (seed & _MASK, (seed >> 32) & _MASK)
    idx = 0
    for i in range(n_species):
        for j in range(i + 1, n_species):
            u = _philox_word0((idx, 0, 0xFFFFFFFE, 0), key) / 4294967296.0
            t[0, i, j] = t[0, j, i] = lo + (hi - lo) * u
            idx += 1
    for i in range(n_species):
        acc = 0.0
        for j in range(n_species):
            if j != i:
                acc += conc[j] * t[0, i, j]
        t[0, i, i] = -acc / conc[i]
    return t


@dataclass
class Workload:
    name: str
    lattice: str                      # "fcc" | "bcc"
    dims: Tuple[int, int, int]        # conventional cells
    conc: List[float]
    n_shells: int
    shell_w: List[float]
    n_chains: int
    n_steps: int
    K: int
    seed: int                         # Philox key for init + proposals
    target_seed: Optional[int] = None
    target_range: Tuple[float, float] = (0.0, 0.0)
    target: np.ndarray = field(default=None, repr=False)

    def __post_init__(self):
        if self.target is None:
            self.target = target_alpha(len(self.conc), self.n_shells, self.conc, self.target_seed,
                                       self.target_range[0], self.target_range[1])

    @property
    def n_sites(self):
        return (4 if self.lattice == "fcc" else 2) * self.dims[0] * self.dims[1] * self.dims[2]

    @property
    def n_species(self):
        return len(self.conc)

    def create_args(self):
        """Positional arguments shared by hea_create and the oracle constructor."""
        return (self.lattice, self.dims, np.asarray(self.conc, dtype=np.float64),
                np.asarray(self.shell_w, dtype=np.float64), self.target)


def config(i, **override):
    """BASELINE.json:configs[i-1] (c1..c4); gaps filled per DESIGN.md A19/A21."""
    if i == 1:
        w = dict(name="c1", lattice="fcc", dims=(5, 5, 5), conc=[0.2] * 5, n_shells=2, shell_w=[1.0, 0.5],
                 n_chains=64, n_steps=10_000, K=32, seed=1)
    elif i == 2:
        w = dict(name="c2", lattice="bcc", dims=(10, 10, 10), conc=[0.25] * 4, n_shells=3,
                 shell_w=[1.0, 0.5, 0.25], n_chains=1024, n_steps=100_000, K=32, seed=2)
    elif i == 3:
        w = dict(name="c3", lattice="fcc", dims=(20, 20, 20), conc=[0.2] * 5, n_shells=3,
                 shell_w=[1.0, 0.5, 0.25], n_chains=256, n_steps=1_000_000, K=64, seed=3,
                 target_seed=7, target_range=(-0.15, 0.15))
    elif i == 4:
        w = dict(name="c4", lattice="fcc", dims=(40, 40, 40), conc=[0.25] * 4, n_shells=2, shell_w=[1.0, 0.5],
                 n_chains=16, n_steps=10_000_000, K=128, seed=4, target_seed=11, target_range=(-0.2, 0.2))
    else:
        raise ValueError("configs 1..4 are fixed workloads; config 5 is the sweep (recount_sweep / chain_sweep)")
    w.update(override)
    return Workload(**w)


def recount_sweep_workload(L, batch):
    """configs[4], recount leg: fcc L^3, 5 species equiatomic, 3 shells, `batch` random configurations, seed 5."""
    return Workload(name=f"c5-recount-L{L}-B{batch}", lattice="fcc", dims=(L, L, L), conc=[0.2] * 5, n_shells=3,
                    shell_w=[1.0, 0.5, 0.25], n_chains=batch, n_steps=0, K=32, seed=5)


def chain_sweep_workload(n_chains, n_steps=10_000):
    """configs[4], MC leg: the 2,000-atom bcc cell of c2 with 1..65,536 chains, seed 5."""
    return Workload(name=f"c5-mc-C{n_chains}", lattice="bcc", dims=(10, 10, 10), conc=[0.25] * 4, n_shells=3,
                    shell_w=[1.0, 0.5, 0.25], n_chains=n_chains, n_steps=n_steps, K=32, seed=5)


def large_m_workload(n_chains=16, n_steps=100_000):
    """A cell the shared-memory (halo) MC engine cannot hold: fcc 40^3 with FIVE species (a byte per padded site does not
    fit, nibbles hold at most four species) -- hea_mc_run falls back to the table-driven window engine with the
    occupancy read through L2.  Shape of the paper's 5-species fcc rows (Table 1) at the c4 cell size."""
    return Workload(name="x1-fcc40-M5", lattice="fcc", dims=(40, 40, 40), conc=[0.2] * 5, n_shells=2, shell_w=[1.0, 0.5],
                    n_chains=n_chains, n_steps=n_steps, K=128, seed=8, target_seed=11, target_range=(-0.2, 0.2))


RECOUNT_SWEEP_L = (10, 20, 40, 60, 80, 100)
RECOUNT_SWEEP_B = (1, 4, 16, 64, 256, 1024)
CHAIN_SWEEP_C = (1, 4, 16, 64, 256, 1024, 4096, 16384, 65536)


# ---- second workload (Fig. 3): non-equiatomic Fe40Mn40Cr10Co10.  The paper takes the
# target SRO of the 256,000-atom model from a 500-atom cell equilibrated by MC-MD (LAMMPS: out of scope); here the
# 500-atom cell is driven by this library's own MC toward a seeded target and its MEASURED alpha (hea_sro_full) becomes
# the target of the large cell -- the same data flow (small cell -> alpha -> large cell), synthetic values.
FIG3_CONC = [0.4, 0.4, 0.1, 0.1]


def fig3_small_workload(n_steps=2000):
    """fcc 5^3 (500 atoms), Fe40Mn40Cr10Co10, shells 1-2, seeded first-shell target; one chain."""
    return Workload(name="fig3-small", lattice="fcc", dims=(5, 5, 5), conc=list(FIG3_CONC), n_shells=2,
                    shell_w=[1.0, 0.5], n_chains=1, n_steps=n_steps, K=32, seed=6, target_seed=13,
                    target_range=(-0.1, 0.1))


def fig3_large_workload(alpha_small, n_chains=16, n_steps=10_000_000):
    """fcc 40^3 (256,000 atoms), same composition; target = alpha measured on the small cell, [S][M][M]."""
    t = np.ascontiguousarray(alpha_small, dtype=np.float64).reshape(2, 4, 4)
    return Workload(name="fig3-large", lattice="fcc", dims=(40, 40, 40), conc=list(FIG3_CONC), n_shells=2,
                    shell_w=[1.0, 0.5], n_chains=n_chains, n_steps=n_steps, K=128, seed=6, target=t)
