"""CPU oracle for the KPM/LSQT DOS path -- TEST INFRASTRUCTURE ONLY.

ctypes wrapper around oracle/libgtbo.so (built from oracle/*.cpp by
oracle/build.py).  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this package; the product
(paper_2509_06525_b200) never does and shares no code with it.
See oracle/gtbo.h for the cited definition of every function.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass
from typing import Optional

import numpy as np

from . import build as _build

OK, ERR_INVALID_ARG, ERR_BOX_TOO_SMALL, ERR_ELL_OVERFLOW = 0, -1, -2, -3


class OracleError(RuntimeError):
    def __init__(self, status: int, where: str):
        super().__init__(f"oracle {where} failed with status {status}")
        self.status = status


class _Model(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("onsite", C.c_void_p), ("t0", C.c_void_p),
                ("r0", C.c_double), ("beta", C.c_double), ("onsite_shift", C.c_void_p)]


class _Ell(C.Structure):
    _fields_ = [("n", C.c_int64), ("width", C.c_int32), ("cols", C.c_void_p),
                ("vals", C.c_void_p), ("diag", C.c_void_p)]


@dataclass
class Ell:
    """Host ELL matrix in the canonical export layout (slot-major [width][n])."""
    n: int
    width: int
    cols: np.ndarray            # int32 [width, n]
    vals: np.ndarray            # float64 [width, n]
    diag: Optional[np.ndarray]  # float64 [n] or None

    def _c(self) -> _Ell:
        return _Ell(self.n, self.width, self.cols.ctypes.data, self.vals.ctypes.data,
                    self.diag.ctypes.data if self.diag is not None else None)

    def to_dense(self) -> np.ndarray:
        h = np.zeros((self.n, self.n))
        rows = np.arange(self.n)
        for k in range(self.width):
            np.add.at(h, (rows, self.cols[k]), self.vals[k])
        if self.diag is not None:
            h[rows, rows] += self.diag
        return h


_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.gtbo_mix64.restype = C.c_uint64
        _lib.gtbo_mix64.argtypes = [C.c_uint64]
        _lib.gtbo_hash.restype = C.c_uint64
        _lib.gtbo_hash.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64]
        _lib.gtbo_uniform.restype = C.c_double
        _lib.gtbo_uniform.argtypes = [C.c_uint64, C.c_uint32, C.c_uint64]
    return _lib


def _f64(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.float64)


def _i32(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.int32)


def _check(st: int, where: str) -> None:
    if st != OK:
        raise OracleError(st, where)


def mix64(z: int) -> int:
    return lib().gtbo_mix64(C.c_uint64(z & (2**64 - 1)))


def hash64(seed: int, r: int, i: int) -> int:
    return lib().gtbo_hash(C.c_uint64(seed & (2**64 - 1)), C.c_uint32(r), C.c_uint64(i))


def uniform(seed: int, r: int, i: int) -> float:
    return lib().gtbo_uniform(C.c_uint64(seed & (2**64 - 1)), C.c_uint32(r), C.c_uint64(i))


def neighbor_counts(pos, box, pbc, cutoff: float, method: int = 1):
    pos = _f64(pos)
    n = pos.shape[0]
    box, pbc = _f64(box), _i32(pbc)
    counts = np.zeros(n, dtype=np.int32)
    width = C.c_int32(0)
    st = lib().gtbo_neighbor_counts(C.c_void_p(pos.ctypes.data), C.c_int64(n),
                                    C.c_void_p(box.ctypes.data), C.c_void_p(pbc.ctypes.data),
                                    C.c_double(cutoff), C.c_int32(method),
                                    C.c_void_p(counts.ctypes.data), C.byref(width))
    _check(st, "neighbor_counts")
    return counts, int(width.value)


def build_hamiltonian(pos, species, box, pbc, cutoff: float, onsite, t0, r0: float = 1.0,
                      beta: float = 0.0, onsite_shift=None, width: Optional[int] = None,
                      method: int = 1, with_diag: bool = True) -> Ell:
    pos, species = _f64(pos), _i32(species)
    n = pos.shape[0]
    box, pbc = _f64(box), _i32(pbc)
    onsite, t0 = _f64(onsite), _f64(t0)
    shift = _f64(onsite_shift) if onsite_shift is not None else None
    if width is None:
        _, width = neighbor_counts(pos, box, pbc, cutoff, method)
    H = Ell(n, width, np.zeros((width, n), dtype=np.int32), np.zeros((width, n)),
            np.zeros(n) if with_diag else None)
    model = _Model(onsite.shape[0], onsite.ctypes.data, t0.ctypes.data, r0, beta,
                   shift.ctypes.data if shift is not None else None)
    hc = H._c()
    st = lib().gtbo_build_hamiltonian(C.c_void_p(pos.ctypes.data), C.c_void_p(species.ctypes.data),
                                      C.c_int64(n), C.c_void_p(box.ctypes.data),
                                      C.c_void_p(pbc.ctypes.data), C.c_double(cutoff),
                                      C.byref(model), C.c_int32(method), C.byref(hc))
    _check(st, "build_hamiltonian")
    return H


def spectral_bounds(H: Ell):
    out = np.zeros(2)
    hc = H._c()
    _check(lib().gtbo_spectral_bounds(C.byref(hc), C.c_void_p(out.ctypes.data)), "spectral_bounds")
    return float(out[0]), float(out[1])


def random_phase_fill(seed: int, r0: int, R: int, n: int) -> np.ndarray:
    phi = np.zeros((n, R, 2))
    st = lib().gtbo_random_phase_fill(C.c_uint64(seed & (2**64 - 1)), C.c_int32(r0), C.c_int32(R),
                                      C.c_int64(n), C.c_void_p(phi.ctypes.data))
    _check(st, "random_phase_fill")
    return phi


def random_phase_rows(seed: int, r0: int, R: int, rows) -> np.ndarray:
    """Rows `rows` of random_phase_fill(seed, r0, R, n): [len(rows)][R][2]."""
    rows = np.ascontiguousarray(rows, dtype=np.int64).reshape(-1)
    phi = np.zeros((rows.shape[0], R, 2))
    st = lib().gtbo_random_phase_rows(C.c_uint64(seed & (2**64 - 1)), C.c_int32(r0), C.c_int32(R),
                                      C.c_void_p(rows.ctypes.data), C.c_int64(rows.shape[0]),
                                      C.c_void_p(phi.ctypes.data))
    _check(st, "random_phase_rows")
    return phi


def kpm_moments(H: Ell, a: float, b: float, M: int, R: int = 1, seed: int = 0, mode: int = 0,
                algo: int = 0, return_im: bool = False):
    mu = np.zeros(M)
    im = C.c_double(0.0)
    hc = H._c()
    st = lib().gtbo_kpm_moments(C.byref(hc), C.c_double(a), C.c_double(b), C.c_int32(M),
                                C.c_int32(R), C.c_uint64(seed & (2**64 - 1)), C.c_int32(mode),
                                C.c_int32(algo), C.c_void_p(mu.ctypes.data), C.byref(im))
    _check(st, "kpm_moments")
    return (mu, float(im.value)) if return_im else mu


def kpm_step_rows(H: Ell, a: float, b: float, first: bool, phi_prev, phi_cur, rows) -> np.ndarray:
    phi_cur = _f64(phi_cur)
    R = phi_cur.shape[1]
    phi_prev = _f64(phi_prev) if phi_prev is not None else None
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    out = np.zeros((rows.shape[0], R, 2))
    hc = H._c()
    st = lib().gtbo_kpm_step_rows(C.byref(hc), C.c_double(a), C.c_double(b), C.c_int32(int(first)),
                                  C.c_int32(R),
                                  C.c_void_p(phi_prev.ctypes.data if phi_prev is not None else None),
                                  C.c_void_p(phi_cur.ctypes.data), C.c_void_p(rows.ctypes.data),
                                  C.c_int64(rows.shape[0]), C.c_void_p(out.ctypes.data))
    _check(st, "kpm_step_rows")
    return out


def jackson(M: int) -> np.ndarray:
    g = np.zeros(M)
    _check(lib().gtbo_jackson(C.c_int32(M), C.c_void_p(g.ctypes.data)), "jackson")
    return g


def dos(mu, a: float, b: float, energies, kernel: int = 1, scale: float = 1.0) -> np.ndarray:
    mu, energies = _f64(mu), _f64(energies)
    rho = np.zeros(energies.shape[0])
    st = lib().gtbo_dos(C.c_void_p(mu.ctypes.data), C.c_int32(mu.shape[0]), C.c_double(a),
                        C.c_double(b), C.c_int32(kernel), C.c_void_p(energies.ctypes.data),
                        C.c_int32(energies.shape[0]), C.c_double(scale),
                        C.c_void_p(rho.ctypes.data))
    _check(st, "dos")
    return rho


# ---------------------------------------------------------------- VAC conductivity (Eq. 3)
def _p(x: np.ndarray) -> C.c_void_p:
    return C.c_void_p(x.ctypes.data)


def velocity_ell(H: Ell, pos, box, pbc, axis: int = 0) -> np.ndarray:
    """vvals[k][i] = vals[k][i] * (x_j - x_i)_axis, minimum image (reading V1); V = i * vvals."""
    pos, box, pbc = _f64(pos), _f64(box), _i32(pbc)
    out = np.zeros((H.width, H.n))
    hc = H._c()
    _check(lib().gtbo_velocity_ell(C.byref(hc), _p(pos), _p(box), _p(pbc), C.c_int32(axis), _p(out)),
           "velocity_ell")
    return out


def velocity_apply(H: Ell, vvals, x) -> np.ndarray:
    """y = V x;  x is [n][R][2]."""
    x, vvals = _f64(x), _f64(vvals)
    y = np.zeros_like(x)
    hc = H._c()
    _check(lib().gtbo_velocity_apply(C.byref(hc), _p(vvals), C.c_int32(x.shape[1]), _p(x), _p(y)),
           "velocity_apply")
    return y


def evolve(H: Ell, a: float, b: float, dt: float, x, return_terms: bool = False):
    """y = exp(-i H dt) x (Chebyshev-Bessel expansion, reading V4);  x is [n][R][2]."""
    x = _f64(x)
    y = np.zeros_like(x)
    terms = C.c_int32(0)
    hc = H._c()
    _check(lib().gtbo_evolve(C.byref(hc), C.c_double(a), C.c_double(b), C.c_double(dt),
                             C.c_int32(x.shape[1]), _p(x), _p(y), C.byref(terms)), "evolve")
    return (y, int(terms.value)) if return_terms else y


def vac_moments(H: Ell, vvals, a: float, b: float, M: int, n_steps: int, dt: float, R: int = 1,
                seed: int = 0, mode: int = 0) -> np.ndarray:
    """C[j][n] (readings V2, V3)."""
    vvals = _f64(vvals)
    out = np.zeros((n_steps, M))
    hc = H._c()
    _check(lib().gtbo_vac_moments(C.byref(hc), _p(vvals), C.c_double(a), C.c_double(b), C.c_int32(M),
                                  C.c_int32(n_steps), C.c_double(dt), C.c_int32(R),
                                  C.c_uint64(seed & (2**64 - 1)), C.c_int32(mode), _p(out)),
           "vac_moments")
    return out


def vac_conductivity(Cm, a: float, b: float, energies, dt: float, kernel: int = 1,
                     scale: float = 1.0):
    """(rho_vv[j][g], sigma[j][g]) from C[j][n] (readings V5, V6)."""
    Cm, energies = _f64(Cm), _f64(energies)
    n_steps, M = Cm.shape
    G = energies.shape[0]
    rv, sg = np.zeros((n_steps, G)), np.zeros((n_steps, G))
    _check(lib().gtbo_vac_conductivity(_p(Cm), C.c_int32(M), C.c_int32(n_steps), C.c_double(a),
                                       C.c_double(b), C.c_int32(kernel), _p(energies), C.c_int32(G),
                                       C.c_double(dt), C.c_double(scale), _p(rv), _p(sg)),
           "vac_conductivity")
    return rv, sg


# ---------------------------------------------------------------- Slater-Koster s,p blocks (NEXT-2)
class _SkModel(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("onsite_s", C.c_void_p), ("onsite_p", C.c_void_p),
                ("sk", C.c_void_p), ("r0", C.c_double), ("beta", C.c_double),
                ("onsite_shift", C.c_void_p)]


def sk_hamiltonian(nbr: Ell, pos, species, box, pbc, onsite_s, onsite_p, sk, r0: float = 1.0,
                   beta: float = 0.0, onsite_shift=None, with_diag: bool = True) -> Ell:
    """Scalar ELL over the 4n orbitals (s, px, py, pz per atom) from the neighbour lists of `nbr`."""
    pos, species, box, pbc = _f64(pos), _i32(species), _f64(box), _i32(pbc)
    es, ep, sk = _f64(onsite_s).reshape(-1), _f64(onsite_p).reshape(-1), _f64(sk).reshape(-1)
    ns = es.shape[0]
    assert sk.shape[0] == ns * ns * 4
    shift = _f64(onsite_shift) if onsite_shift is not None else None
    n, K = nbr.n, nbr.width
    H = Ell(4 * n, 4 * K, np.zeros((4 * K, 4 * n), dtype=np.int32), np.zeros((4 * K, 4 * n)),
            np.zeros(4 * n) if with_diag else None)
    model = _SkModel(ns, es.ctypes.data, ep.ctypes.data, sk.ctypes.data, r0, beta,
                     shift.ctypes.data if shift is not None else None)
    nc, hc = nbr._c(), H._c()
    _check(lib().gtbo_sk_hamiltonian(C.byref(nc), _p(pos), _p(species), _p(box), _p(pbc),
                                     C.byref(model), C.byref(hc)), "sk_hamiltonian")
    return H


# ---------------------------------------------------------------- descriptor + MLP hopping (Eq. 2, NEXT-3)
class _MlpModel(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_features", C.c_int32), ("n_basis", C.c_int32),
                ("n_hidden", C.c_int32), ("r_cut", C.c_double), ("weights", C.c_void_p)]


def mlp_descriptor(dims, r_cut: float, weights, si: int, sj: int, r: float) -> np.ndarray:
    ns, F, Nb, Hd = dims
    w = _f64(weights)
    m = _MlpModel(ns, F, Nb, Hd, r_cut, w.ctypes.data)
    out = np.zeros(F)
    _check(lib().gtbo_mlp_descriptor(C.byref(m), C.c_int32(si), C.c_int32(sj), C.c_double(r), _p(out)),
           "mlp_descriptor")
    return out


def mlp_hamiltonian(nbr: Ell, pos, species, box, pbc, dims, r_cut: float, weights,
                    with_diag: bool = True, return_v: bool = False):
    """H on the pattern of `nbr` with t_ij, eps_i from the descriptor + MLPs (weight blob: gtbo_mlp.cpp)."""
    ns, F, Nb, Hd = dims
    pos, species, box, pbc, w = _f64(pos), _i32(species), _f64(box), _i32(pbc), _f64(weights)
    H = Ell(nbr.n, nbr.width, nbr.cols.copy(), np.zeros((nbr.width, nbr.n)),
            np.zeros(nbr.n) if with_diag else None)
    v = np.zeros((nbr.n, F))
    m = _MlpModel(ns, F, Nb, Hd, r_cut, w.ctypes.data)
    hc = H._c()
    _check(lib().gtbo_mlp_hamiltonian(C.byref(m), _p(pos), _p(species), _p(box), _p(pbc), C.byref(hc),
                                      _p(v)), "mlp_hamiltonian")
    return (H, v) if return_v else H


# ---------------------------------------------------------------- Slater-Koster s,p,d blocks (NEXT-2)
class _SpdModel(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("onsite_s", C.c_void_p), ("onsite_p", C.c_void_p),
                ("onsite_d", C.c_void_p), ("sk", C.c_void_p), ("r0", C.c_double), ("beta", C.c_double),
                ("onsite_shift", C.c_void_p)]


def spd_hamiltonian(nbr: Ell, pos, species, box, pbc, onsite_s, onsite_p, onsite_d, sk, r0: float = 1.0,
                    beta: float = 0.0, onsite_shift=None, with_diag: bool = True) -> Ell:
    """Scalar ELL over the 9n orbitals (s, p, d per atom) from the neighbour lists of `nbr`."""
    pos, species, box, pbc = _f64(pos), _i32(species), _f64(box), _i32(pbc)
    es, ep, ed = (_f64(x).reshape(-1) for x in (onsite_s, onsite_p, onsite_d))
    sk = _f64(sk).reshape(-1)
    ns = es.shape[0]
    assert sk.shape[0] == ns * ns * 10
    shift = _f64(onsite_shift) if onsite_shift is not None else None
    n, K = nbr.n, nbr.width
    H = Ell(9 * n, 9 * K, np.zeros((9 * K, 9 * n), dtype=np.int32), np.zeros((9 * K, 9 * n)),
            np.zeros(9 * n) if with_diag else None)
    model = _SpdModel(ns, es.ctypes.data, ep.ctypes.data, ed.ctypes.data, sk.ctypes.data, r0, beta,
                      shift.ctypes.data if shift is not None else None)
    nc, hc = nbr._c(), H._c()
    _check(lib().gtbo_spd_hamiltonian(C.byref(nc), _p(pos), _p(species), _p(box), _p(pbc),
                                      C.byref(model), C.byref(hc)), "spd_hamiltonian")
    return H


def spd_step_atoms(nbr: Ell, pos, species, box, pbc, onsite_s, onsite_p, onsite_d, sk, a: float, b: float,
                   first: bool, atoms, x_own, x_nbr, prev=None, r0: float = 1.0, beta: float = 0.0,
                   onsite_shift=None) -> np.ndarray:
    """One Chebyshev step of the s,p,d orbital matrix on the listed atoms without materialising H:
    x_own [q][9][R][2], x_nbr [q][K][9][R][2], prev like x_own -> out [q][9][R][2]."""
    pos, species, box, pbc = _f64(pos), _i32(species), _f64(box), _i32(pbc)
    es, ep, ed = (_f64(x).reshape(-1) for x in (onsite_s, onsite_p, onsite_d))
    sk = _f64(sk).reshape(-1)
    ns = es.shape[0]
    assert sk.shape[0] == ns * ns * 10
    shift = _f64(onsite_shift) if onsite_shift is not None else None
    atoms = np.ascontiguousarray(atoms, dtype=np.int64).reshape(-1)
    x_own, x_nbr = _f64(x_own), _f64(x_nbr)
    q, R = atoms.shape[0], x_own.shape[2]
    assert x_own.shape == (q, 9, R, 2) and x_nbr.shape == (q, nbr.width, 9, R, 2)
    prev = _f64(prev) if prev is not None else None
    out = np.zeros((q, 9, R, 2))
    model = _SpdModel(ns, es.ctypes.data, ep.ctypes.data, ed.ctypes.data, sk.ctypes.data, r0, beta,
                      shift.ctypes.data if shift is not None else None)
    nc = nbr._c()
    _check(lib().gtbo_spd_step_atoms(C.byref(nc), _p(pos), _p(species), _p(box), _p(pbc), C.byref(model),
                                     C.c_double(a), C.c_double(b), C.c_int32(int(first)), C.c_int32(R),
                                     _p(atoms), C.c_int64(q), _p(x_own), _p(x_nbr),
                                     C.c_void_p(prev.ctypes.data if prev is not None else None), _p(out)),
           "spd_step_atoms")
    return out


def mlp_sk_hamiltonian(nbr: Ell, pos, species, box, pbc, dims, r_cut: float, weights,
                       with_diag: bool = True) -> Ell:
    """Eq. 2 feeding the s,p Slater-Koster blocks: scalar ELL over 4n orbitals (blob with 4 / 2 outputs)."""
    ns, F, Nb, Hd = dims
    pos, species, box, pbc, w = _f64(pos), _i32(species), _f64(box), _i32(pbc), _f64(weights)
    n, K = nbr.n, nbr.width
    H = Ell(4 * n, 4 * K, np.zeros((4 * K, 4 * n), dtype=np.int32), np.zeros((4 * K, 4 * n)),
            np.zeros(4 * n) if with_diag else None)
    m = _MlpModel(ns, F, Nb, Hd, r_cut, w.ctypes.data)
    nc, hc = nbr._c(), H._c()
    _check(lib().gtbo_mlp_sk_hamiltonian(C.byref(m), C.byref(nc), _p(pos), _p(species), _p(box), _p(pbc),
                                         C.byref(hc)), "mlp_sk_hamiltonian")
    return H


def spd_block_from_integrals(u, V, Vt=None) -> np.ndarray:
    """E [9][9] of a pair from its bond direction and ten (scaled) integrals; Vt: those of the reversed pair."""
    u, V = _f64(u), _f64(V)
    Vt = V if Vt is None else _f64(Vt)
    E = np.zeros((9, 9))
    _check(lib().gtbo_spd_block_from_integrals(_p(u), _p(V), _p(Vt), _p(E)), "spd_block_from_integrals")
    return E


def mlp_spd_hamiltonian(nbr: Ell, pos, species, box, pbc, dims, r_cut: float, weights,
                        with_diag: bool = True) -> Ell:
    """Eq. 2 feeding the s,p,d Slater-Koster blocks: scalar ELL over 9n orbitals (blob with 10 / 3 outputs)."""
    ns, F, Nb, Hd = dims
    pos, species, box, pbc, w = _f64(pos), _i32(species), _f64(box), _i32(pbc), _f64(weights)
    n, K = nbr.n, nbr.width
    H = Ell(9 * n, 9 * K, np.zeros((9 * K, 9 * n), dtype=np.int32), np.zeros((9 * K, 9 * n)),
            np.zeros(9 * n) if with_diag else None)
    m = _MlpModel(ns, F, Nb, Hd, r_cut, w.ctypes.data)
    nc, hc = nbr._c(), H._c()
    _check(lib().gtbo_mlp_spd_hamiltonian(C.byref(m), C.byref(nc), _p(pos), _p(species), _p(box), _p(pbc),
                                          C.byref(hc)), "mlp_spd_hamiltonian")
    return H


def carrier_density(rho, energies, e_ref: float) -> np.ndarray:
    """n(E_j) = int_{e_ref}^{E_j} rho dE by the trapezoid rule (reading V7)."""
    rho, energies = _f64(rho), _f64(energies)
    out = np.zeros_like(rho)
    _check(lib().gtbo_carrier_density(_p(rho), _p(energies), C.c_int32(rho.shape[0]), C.c_double(e_ref),
                                      _p(out)), "carrier_density")
    return out


def mobility(sigma, n, scale: float = 1.0, n_min: float = 0.0) -> np.ndarray:
    """mu = scale * sigma / |n| where |n| > n_min, else 0 (reading V8)."""
    sigma, n = _f64(sigma), _f64(n)
    out = np.zeros_like(sigma)
    _check(lib().gtbo_mobility(_p(sigma), _p(n), C.c_int32(sigma.shape[0]), C.c_double(scale),
                               C.c_double(n_min), _p(out)), "mobility")
    return out
