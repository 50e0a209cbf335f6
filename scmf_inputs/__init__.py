"""Seeded synthetic inputs for the SCMF Monte-Carlo step (shared by oracle, CUDA path, bench).

This module holds NONE of the method's arithmetic (no Philox move stream, no cell index, no
energy, no omega).  It only builds the problem statement (chains, bead types, b, chiN, kappaN,
grid, box) and a seeded initial state, as BASELINE.json `configs[0..4]` describe them:

* first bead of every chain uniform in the periodic box [0, L)^3,
* every further bead = previous bead + N(0, b^2/3)^3 ("Gaussian random walk"), accumulated in
  double and rounded once to fp32; positions are NOT wrapped (reading R7),
* AB diblocks: first half of the beads type 0 (A), second half type 1 (B),
* binary blend: exactly n/2 all-A chains and n/2 all-B chains, order shuffled.

The paper's own workloads (the JUPITER-suite SOMA case, and the NIPS membrane
sub-domains) are not available; these synthetic melts stand in for them
(SURVEY.md section 8(d)).  Random numbers come from numpy's Philox bit generator keyed by the
config seed; they never collide with the move stream because that one is produced inside the
oracle / the CUDA kernels from (seed, step, half-sweep, chain, bead).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional, Tuple

import numpy as np

__all__ = ["Workload", "System", "CONFIGS", "config", "make_system", "scaled", "custom_system", "species_system"]


@dataclass(frozen=True)
class Workload:
    """Problem statement of one BASELINE.json config (no state)."""

    name: str
    n_chains: int
    N: int                                   # beads per chain
    n_types: int
    architecture: str                        # "diblock" | "homopolymer" | "blend" | "custom"
    grid: Tuple[int, int, int]
    box: Tuple[float, float, float]          # in units of b
    chiN: float                              # off-diagonal chi*N (all pairs s != t)
    kappaN: float
    seed: int
    steps: int
    b: float = 1.0
    move_halfwidth: float = 0.5
    f_A: float = 0.5

    @property
    def n_beads(self) -> int:
        return self.n_chains * self.N

    @property
    def n_cells(self) -> int:
        return self.grid[0] * self.grid[1] * self.grid[2]


@dataclass
class System:
    """A workload plus its seeded initial state, ready to hand to either implementation."""

    workload: Workload
    type_patterns: np.ndarray                # uint8 [n_patterns][N]
    chain_pattern: Optional[np.ndarray]      # uint8 [n_chains] or None (= all pattern 0)
    chiN: np.ndarray                         # float32 [T][T], symmetric, zero diagonal
    x: np.ndarray                            # float32 [n_chains*N], index c*N+i
    y: np.ndarray
    z: np.ndarray
    extra: dict = field(default_factory=dict)
    n_single: Optional[np.ndarray] = None    # uint64 [T]: single-bead molecules per type, stored after the chains
    species: Optional[list] = None           # [(n_chains_s, N_s), ...]: polymer species of different chain lengths, stored
                                             # species by species; workload.N is then the reference length, pattern rows max N_s long

    @property
    def n_patterns(self) -> int:
        return int(self.type_patterns.shape[0])

    def bead_types(self) -> np.ndarray:
        """uint8 [n_chains*N] type of every bead (harness-side bookkeeping only)."""
        w = self.workload
        if self.species is not None:
            cp = np.zeros(w.n_chains, dtype=np.int64) if self.chain_pattern is None else self.chain_pattern.astype(np.int64)
            parts, c0 = [], 0
            for n_s, N_s in self.species:
                parts.append(self.type_patterns[cp[c0:c0 + n_s], :N_s].reshape(-1))
                c0 += n_s
            t = np.concatenate(parts)
        elif self.chain_pattern is None:
            t = np.tile(self.type_patterns[0], w.n_chains)
        else:
            t = self.type_patterns[self.chain_pattern].reshape(-1)
        if self.n_single is not None:
            t = np.concatenate([t, np.repeat(np.arange(w.n_types, dtype=np.uint8), self.n_single.astype(np.int64))])
        return t


# BASELINE.json configs[0..4]; cell size b/2 everywhere, so box = grid / 2.
CONFIGS = (
    Workload("cfg0_diblock_small", 256, 32, 2, "diblock", (16, 16, 16), (8.0, 8.0, 8.0),
             20.0, 50.0, seed=1, steps=10),
    Workload("cfg1_ideal_homopolymer", 65536, 64, 1, "homopolymer", (64, 64, 64),
             (32.0, 32.0, 32.0), 0.0, 0.0, seed=2, steps=1000),
    Workload("cfg2_diblock_medium", 524288, 32, 2, "diblock", (64, 64, 64),
             (32.0, 32.0, 32.0), 20.0, 50.0, seed=3, steps=100),
    Workload("cfg3_blend", 1048576, 64, 2, "blend", (128, 128, 128), (64.0, 64.0, 64.0),
             2.5, 50.0, seed=4, steps=100),
    Workload("cfg4_diblock_large", 4194304, 32, 2, "diblock", (256, 256, 128),
             (128.0, 128.0, 64.0), 30.0, 50.0, seed=5, steps=50),
)


def config(i: int) -> Workload:
    return CONFIGS[i]


def scaled(w: Workload, n_chains: int, grid: Tuple[int, int, int]) -> Workload:
    """Same melt (density per cell, cell size, fields) at a smaller size; parity-test helper.

    Keeps cell size b/2 (box = grid/2); the caller picks n_chains so that beads per cell stay
    near the original if that matters for the test.
    """
    box = tuple(g * 0.5 * w.b for g in grid)
    return replace(w, name=f"{w.name}_scaled_{n_chains}", n_chains=n_chains, grid=tuple(grid),
                   box=box)


def _patterns(w: Workload, rng: np.random.Generator):
    N = w.N
    if w.architecture == "homopolymer":
        return np.zeros((1, N), dtype=np.uint8), None
    if w.architecture == "diblock":
        nA = int(round(w.f_A * N))
        pat = np.zeros((1, N), dtype=np.uint8)
        pat[0, nA:] = 1
        return pat, None
    if w.architecture == "blend":
        pat = np.zeros((2, N), dtype=np.uint8)
        pat[1, :] = 1
        ids = np.zeros(w.n_chains, dtype=np.uint8)
        ids[w.n_chains // 2:] = 1
        rng.shuffle(ids)                      # "types assigned by a random shuffle" (configs[3])
        return pat, ids
    raise ValueError(f"unknown architecture {w.architecture!r}")


def make_system(w: Workload, chunk_chains: int = 1 << 20) -> System:
    """Seeded initial state for workload `w` (deterministic for a given numpy version)."""
    rng = np.random.Generator(np.random.Philox(key=[w.seed, 0x5C3F_1217]))
    pats, chain_pattern = _patterns(w, rng)
    T = w.n_types
    chiN = np.full((T, T), w.chiN, dtype=np.float32)
    np.fill_diagonal(chiN, 0.0)

    n, N = w.n_chains, w.N
    sigma = w.b / np.sqrt(3.0)
    out = [np.empty(n * N, dtype=np.float32) for _ in range(3)]
    for c0 in range(0, n, chunk_chains):
        c1 = min(n, c0 + chunk_chains)
        for d in range(3):
            steps = rng.standard_normal((c1 - c0, N))          # float64
            steps *= sigma
            steps[:, 0] = rng.random(c1 - c0) * w.box[d]       # first bead uniform in [0, L)
            np.cumsum(steps, axis=1, out=steps)
            out[d][c0 * N:c1 * N] = steps.reshape(-1)          # one rounding to fp32
    return System(w, pats, chain_pattern, chiN, out[0], out[1], out[2])


def custom_system(n_chains: int, N: int, n_types: int, type_patterns, chain_pattern, chiN,
                  kappaN: float, grid, box, seed: int, b: float = 1.0,
                  move_halfwidth: float = 0.5, name: str = "custom", n_single=None) -> System:
    """Arbitrary architecture (edge-case tests): explicit patterns and a full chiN matrix."""
    w = Workload(name, n_chains, N, n_types, "custom", tuple(int(g) for g in grid),
                 tuple(float(v) for v in box), 0.0, float(kappaN), seed=seed, steps=1, b=b,
                 move_halfwidth=move_halfwidth)
    rng = np.random.Generator(np.random.Philox(key=[seed, 0x5C3F_1217]))
    sigma = b / np.sqrt(3.0)
    out = []
    for d in range(3):
        steps = rng.standard_normal((n_chains, N)) * sigma
        steps[:, 0] = rng.random(n_chains) * box[d]
        out.append(np.cumsum(steps, axis=1).reshape(-1).astype(np.float32))
    ns = None
    if n_single is not None:                     # single-bead molecules: uniform in the box, appended after the chains
        ns = np.ascontiguousarray(n_single, dtype=np.uint64).reshape(n_types)
        for d in range(3):
            out[d] = np.concatenate([out[d], (rng.random(int(ns.sum())) * box[d]).astype(np.float32)])
    pats = np.ascontiguousarray(np.asarray(type_patterns, dtype=np.uint8).reshape(-1, N))
    cp = None if chain_pattern is None else np.ascontiguousarray(chain_pattern, dtype=np.uint8)
    chi = np.ascontiguousarray(np.asarray(chiN, dtype=np.float32).reshape(n_types, n_types))
    return System(w, pats, cp, chi, out[0], out[1], out[2], n_single=ns)


def species_system(species, N_ref: int, n_types: int, type_patterns, chain_pattern, chiN, kappaN: float, grid, box,
                   seed: int, b: float = 1.0, move_halfwidth: float = 0.5, name: str = "species", n_single=None) -> System:
    """Several polymer species of different chain lengths in one box (the paper's polymer / solvent / non-solvent
    systems): species = [(n_chains_s, N_s), ...], chains stored species by species; N_ref is the
    reference chain length (the N of chiN, kappaN and of 1/N); type_patterns rows have max N_s entries, a chain
    uses the first N_s of its row.  Gaussian random-walk start like the configs'."""
    species = [(int(a), int(c)) for a, c in species]
    n_chains = sum(a for a, _ in species)
    n_max = max(c for _, c in species)
    w = Workload(name, n_chains, int(N_ref), n_types, "custom", tuple(int(g) for g in grid), tuple(float(v) for v in box),
                 0.0, float(kappaN), seed=seed, steps=1, b=b, move_halfwidth=move_halfwidth)
    rng = np.random.Generator(np.random.Philox(key=[seed, 0x5C3F_1218]))
    sigma = b / np.sqrt(3.0)
    out = [[], [], []]
    for n_s, N_s in species:
        for d in range(3):
            steps = rng.standard_normal((n_s, N_s)) * sigma
            steps[:, 0] = rng.random(n_s) * box[d]
            out[d].append(np.cumsum(steps, axis=1).reshape(-1).astype(np.float32))
    ns = None
    if n_single is not None:
        ns = np.ascontiguousarray(n_single, dtype=np.uint64).reshape(n_types)
        for d in range(3):
            out[d].append((rng.random(int(ns.sum())) * box[d]).astype(np.float32))
    pats = np.ascontiguousarray(np.asarray(type_patterns, dtype=np.uint8).reshape(-1, n_max))
    cp = None if chain_pattern is None else np.ascontiguousarray(chain_pattern, dtype=np.uint8)
    chi = np.ascontiguousarray(np.asarray(chiN, dtype=np.float32).reshape(n_types, n_types))
    return System(w, pats, cp, chi, np.concatenate(out[0]), np.concatenate(out[1]), np.concatenate(out[2]), n_single=ns, species=species)
