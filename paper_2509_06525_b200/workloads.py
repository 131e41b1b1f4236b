"""Seeded synthetic inputs shaped like the paper's workloads (numpy only).

This module holds NONE of the method's arithmetic: it only lays out atoms on a
honeycomb lattice, displaces them with numpy's seeded Gaussian generator and
names the parameters of each BASELINE.json config.  Both the CUDA path and the
CPU oracle receive exactly these arrays.

Geometry (reading A6): rectangular 4-atom graphene cell,
a_CC = 1.42 A, L_x = sqrt(3) a (zigzag period), L_y = 3 a (armchair period),
basis s0 = (0,0) [A], s1 = (0,a) [B], s2 = (L_x/2, 3a/2) [A], s3 = (L_x/2, 5a/2) [B],
z0 = 10 A in a 20 A box, pbc = (1,1,0); atom index i = (c_y*n_x + c_x)*4 + s.

The paper measures on its own MD/ML-generated structures (PAPER.md:33, :106,
:192), which are not available; these lattices stand in for them: 100 M-atom
graphene (Fig. 4a), ~10^6-10^7-atom thermally disordered graphene (Fig. 4b), and
a 1 M-atom h-BN/graphene heterojunction (Fig. 4c-d).
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import Optional

import numpy as np

A_CC = 1.42
LX = np.sqrt(3.0) * A_CC
LY = 3.0 * A_CC
LZ = 20.0
Z0 = 10.0
SEED_LATTICE = 20250906
SEED_VECTORS = 6525


@dataclass(frozen=True)
class Workload:
    name: str
    nx: int
    ny: int
    cutoff: float
    onsite: tuple                 # [n_species] eV
    t0: tuple                     # [n_species][n_species] eV (row-major, symmetric)
    r0: float = A_CC
    beta: float = 0.0
    sigma_xy: float = 0.0         # in-plane Gaussian displacement, A
    sigma_z: float = 0.0          # out-of-plane Gaussian displacement, A
    sigma_onsite: float = 0.0     # per-atom onsite disorder (std dev, A10), eV
    stripe: int = 0               # h-BN/graphene stripe width in cells along x (0 = none)
    a: Optional[float] = None     # energy half-width; None -> Gershgorin helper (A8)
    b: Optional[float] = None
    M: int = 256
    R: int = 4
    seed: int = SEED_VECTORS
    n_energies: int = 4001
    e_min: Optional[float] = None  # None -> b - a
    e_max: Optional[float] = None
    use_diag: bool = True
    note: str = ""

    @property
    def n_atoms(self) -> int:
        return 4 * self.nx * self.ny

    @property
    def n_species(self) -> int:
        return len(self.onsite)

    def scaled(self, nx: int, ny: int, **kw) -> "Workload":
        """Same construction on a smaller supercell (parity-test sizes)."""
        return replace(self, nx=nx, ny=ny, name=f"{self.name}@{nx}x{ny}", **kw)


_C = (0.0,)
_T_C = (-2.7,)
# species 0 = C, 1 = B, 2 = N (A9); undefined pairs (B-B, N-N) get 0
_HBN_ONSITE = (0.0, 2.3, -2.3)
_HBN_T0 = (-2.7, -2.5, -2.8,
           -2.5, 0.0, -2.6,
           -2.8, -2.6, 0.0)

CONFIGS = {
    # BASELINE.json:configs[0]
    "c1": Workload("c1-pristine-24x24", 24, 24, 1.95, _C, _T_C, a=8.5, b=0.0, M=256, R=4,
                   use_diag=False, note="NN graphene, random trace R=4 and exact trace"),
    # configs[1], literal cutoff 4.0 A (A7: 18 neighbours, K=20) and variant b (2.65 A, K~10)
    "c2": Workload("c2-disordered-500x500-rc4.0", 500, 500, 4.0, _C, _T_C, beta=3.37,
                   sigma_xy=0.05, sigma_z=0.10, sigma_onsite=0.05, M=3000, R=8),
    "c2b": Workload("c2b-disordered-500x500-rc2.65", 500, 500, 2.65, _C, _T_C, beta=3.37,
                    sigma_xy=0.05, sigma_z=0.10, sigma_onsite=0.05, M=3000, R=8),
    # configs[2]
    "c3": Workload("c3-disordered-1600x1600-rc4.0", 1600, 1600, 4.0, _C, _T_C, beta=3.37,
                   sigma_xy=0.05, sigma_z=0.10, sigma_onsite=0.05, M=5000, R=4),
    "c3b": Workload("c3b-disordered-1600x1600-rc2.65", 1600, 1600, 2.65, _C, _T_C, beta=3.37,
                    sigma_xy=0.05, sigma_z=0.10, sigma_onsite=0.05, M=5000, R=4),
    # configs[3]
    "c4": Workload("c4-hbn-graphene-1000x250", 1000, 250, 1.95, _HBN_ONSITE, _HBN_T0,
                   sigma_xy=0.05, sigma_z=0.10, stripe=125, a=10.0, b=0.0, M=3000, R=8),
    # configs[4]
    "c5": Workload("c5-pristine-5000x5000", 5000, 5000, 1.95, _C, _T_C, a=8.5, b=0.0,
                   M=3000, R=2, use_diag=False, e_min=-8.5, e_max=8.5,
                   note="the memory-bound scaling case; the metric is quoted on this one"),
}


@dataclass
class Inputs:
    pos: np.ndarray                       # float64 [N,3]
    species: np.ndarray                   # int32 [N]
    box: np.ndarray                       # float64 [3]
    pbc: np.ndarray                       # int32 [3]
    onsite_shift: Optional[np.ndarray]    # float64 [N] or None
    workload: Workload = field(repr=False, default=None)


def make_inputs(w: Workload, seed: int = SEED_LATTICE, tile: Optional[tuple] = None) -> Inputs:
    """The lattice of workload `w`.  Atoms are numbered row-major (cell row, cell, basis atom).  tile = (tx, ty)
    renumbers the SAME atoms tile-major: blocks of tx x ty cells one after the other (row-major inside a block
    and over the blocks) -- the same structure, another order of its rows, for measuring what the numbering of
    the input costs the gathers (bench.py --tile-numbering)."""
    nx, ny = w.nx, w.ny
    n = 4 * nx * ny
    basis = np.array([[0.0, 0.0], [0.0, A_CC], [LX / 2, 1.5 * A_CC], [LX / 2, 2.5 * A_CC]])
    pos = np.empty((ny, nx, 4, 3), dtype=np.float64)
    cx = np.arange(nx, dtype=np.float64) * LX
    cy = np.arange(ny, dtype=np.float64) * LY
    pos[..., 0] = cx[None, :, None] + basis[None, None, :, 0]
    pos[..., 1] = cy[:, None, None] + basis[None, None, :, 1]
    pos[..., 2] = Z0
    pos = pos.reshape(n, 3)
    rng = np.random.Generator(np.random.PCG64(seed))
    if w.sigma_xy > 0.0 or w.sigma_z > 0.0:
        # drawn in a fixed order: x, y, z for all atoms
        for axis, sig in ((0, w.sigma_xy), (1, w.sigma_xy), (2, w.sigma_z)):
            d = rng.standard_normal(n)
            if sig > 0.0:
                pos[:, axis] += sig * d
    shift = None
    if w.sigma_onsite > 0.0:
        shift = w.sigma_onsite * rng.standard_normal(n)
    species = np.zeros((ny, nx, 4), dtype=np.int32)
    if w.stripe > 0:
        hbn = ((np.arange(nx) // w.stripe) % 2) == 1      # odd stripes are h-BN
        sub = np.array([1, 2, 1, 2], dtype=np.int32)      # A sites boron, B sites nitrogen
        species[:, hbn, :] = sub[None, None, :]
    species = species.reshape(n)
    box = np.array([nx * LX, ny * LY, LZ])
    pbc = np.array([1, 1, 0], dtype=np.int32)
    if tile is not None:
        tx, ty = int(tile[0]), int(tile[1])
        if tx < 1 or ty < 1:
            raise ValueError("tile = (tx, ty) cells, both >= 1")
        cy, cx, bs = np.meshgrid(np.arange(ny), np.arange(nx), np.arange(4), indexing="ij")
        cy, cx, bs = cy.ravel(), cx.ravel(), bs.ravel()
        order = np.lexsort((bs, cx % tx, cy % ty, cx // tx, cy // ty))   # last key is the primary one
        pos = np.ascontiguousarray(pos[order])
        species = np.ascontiguousarray(species[order])
        if shift is not None:
            shift = np.ascontiguousarray(shift[order])
    return Inputs(pos, species, box, pbc, shift, w)


def inputs_digest(inp: Inputs) -> str:
    """SHA-256 of the generated arrays: stored in the full-size goldens (tests/golden/) so that a test
    notices if the generators ever produce a different lattice."""
    import hashlib
    h = hashlib.sha256()
    h.update(np.ascontiguousarray(inp.pos).tobytes())
    h.update(np.ascontiguousarray(inp.species).tobytes())
    if inp.onsite_shift is not None:
        h.update(np.ascontiguousarray(inp.onsite_shift).tobytes())
    return h.hexdigest()


def energy_grid(w: Workload, a: float, b: float) -> np.ndarray:
    """E_j = E_min + j (E_max - E_min)/(G-1), endpoints included (C6)."""
    lo = w.e_min if w.e_min is not None else b - a
    hi = w.e_max if w.e_max is not None else b + a
    return np.linspace(lo, hi, w.n_energies)


def algorithmic_bytes_per_atom_pass(width: int, has_diag: bool, R: int) -> int:
    """B = 12 K + 8 [diag] + 48 R bytes per atom per recursion pass."""
    return 12 * width + (8 if has_diag else 0) + 48 * R


# ---- synthetic Slater-Koster s,p parameters for the multi-orbital runs (bench.py --orbitals sp) ----
# graphene-like two-centre integrals (eV): ss_sigma, sp_sigma, pp_sigma, pp_pi, scaled per species pair
# (species 0 = C, 1 = B, 2 = N as in config 4); inputs only, no method arithmetic.
SK_CC = (-6.769, 5.580, 5.037, -3.033)
SK_ONSITE_S = (-8.868, -6.0, -11.0)
SK_ONSITE_P = (0.0, 2.3, -2.3)
_SK_PAIR_SCALE = {(0, 0): 1.0, (1, 2): 0.96, (0, 1): 0.93, (0, 2): 1.04, (1, 1): 0.5, (2, 2): 0.5}


SK_D = (-2.1, -1.7, 0.9, -1.3, 0.8, -0.15)      # sd_sigma, pd_sigma, pd_pi, dd_sigma, dd_pi, dd_delta
SK_ONSITE_D = (6.5, 7.0, 5.5)


def spd_table(n_species: int) -> np.ndarray:
    """[ns][ns][10]: ss_sigma, sp_sigma, pp_sigma, pp_pi, sd_sigma, pd_sigma, pd_pi, dd_sigma, dd_pi, dd_delta."""
    t = np.zeros((n_species, n_species, 10))
    for (a, b), f in _SK_PAIR_SCALE.items():
        if a < n_species and b < n_species:
            t[a, b] = t[b, a] = f * np.array(SK_CC + SK_D)
    return t


def sk_table(n_species: int) -> np.ndarray:
    t = np.zeros((n_species, n_species, 4))
    for (a, b), f in _SK_PAIR_SCALE.items():
        if a < n_species and b < n_species:
            t[a, b] = t[b, a] = f * np.array(SK_CC)
    return t


# ---- synthetic weights for the descriptor + MLP Hamiltonian (Eq. 2; bench.py / tests, NEXT-3) ----
# Blob layout (doubles), shared by both implementations as an INPUT format:
#   c [ns][ns][F][Nb] | MLP_e: W1 [Hd][F], b1 [Hd], W2 [F][Hd], b2 [F] |
#   MLP_lambda: W1 [Hd][F], b1 [Hd], W2 [Hd], b2 [1] | per species: W1 [Hd][F], b1 [Hd], W2 [Hd], b2 [1]
MLP_DIMS = (3, 8, 8, 16)       # species, features F, basis functions Nb, hidden width Hd


def mlp_pack(c, env, hop, ons) -> np.ndarray:
    """c [ns,ns,F,Nb]; env = (W1, b1, W2, b2); hop = (W1, b1, W2, b2); ons = list of the same per species."""
    parts = [np.asarray(c, dtype=np.float64).ravel()]
    for group in [env, hop, *ons]:
        parts += [np.asarray(x, dtype=np.float64).ravel() for x in group]
    return np.ascontiguousarray(np.concatenate(parts))


def mlp_weights(dims=MLP_DIMS, seed: int = 65250, hop_out: int = 1, onsite_out: int = 1) -> np.ndarray:
    """Seeded random weights of moderate size (|t| of a few eV at bond length); c symmetric in the pair.
    hop_out / onsite_out: outputs of MLP_lambda / the onsite MLPs (1, 1: one orbital; 4, 2: s,p blocks)."""
    ns, F, Nb, Hd = dims
    rng = np.random.Generator(np.random.PCG64(seed))
    c = rng.normal(0.0, 1.0, (ns, ns, F, Nb)) / np.sqrt(Nb)
    c = 0.5 * (c + c.transpose(1, 0, 2, 3))
    def layer(out_dim, scale):
        return (rng.normal(0.0, 1.0, (Hd, F)) / np.sqrt(F), rng.normal(0.0, 0.3, Hd),
                rng.normal(0.0, scale, (out_dim, Hd)) / np.sqrt(Hd), rng.normal(0.0, 0.1, out_dim))
    env = layer(F, 1.0)
    hop = layer(hop_out, 4.0)
    ons = [layer(onsite_out, 1.0) for _ in range(ns)]
    return mlp_pack(c, env, hop, ons)
