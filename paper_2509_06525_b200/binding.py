"""Thin Python binding of libgtb_kpm.so (include/gtb.h): argument marshalling only.

Every function has the name of the C call it wraps (without the gtb_ prefix), takes torch CUDA
tensors (or allocates the outputs / workspace as torch tensors), passes raw device pointers and
the current CUDA stream, and raises GtbError on a non-zero status.  All arithmetic of the path
runs in the library's CUDA kernels.  There is no CPU fallback: without the built library, or
without a CUDA device, the calls fail.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import Optional

import numpy as np
import torch

from . import build as _build

OK = 0
ERR_INVALID_ARG, ERR_BOX_TOO_SMALL, ERR_ELL_OVERFLOW, ERR_WORKSPACE = -1, -2, -3, -4
ERR_DIVERGED, ERR_CUDA, ERR_INDEX_RANGE, ERR_NOT_PACKABLE, ERR_STATIC_LIMIT = -5, -6, -7, -8, -9
MAX_WIDTH = 64

# every symbol include/gtb.h declares (tests check that the library exports each of them)
EXPORTS = (
    "gtb_status_string", "gtb_last_cuda_error", "gtb_version", "gtb_launch_count",
    "gtb_build_workspace_bytes", "gtb_neighbor_width", "gtb_build_hamiltonian",
    "gtb_bounds_workspace_bytes", "gtb_spectral_bounds", "gtb_random_phase_fill",
    "gtb_kpm_workspace_bytes", "gtb_kpm_moments", "gtb_kpm_status", "gtb_kpm_step", "gtb_kpm_moments_static",
    "gtb_dos", "gtb_jackson",
    "gtb_velocity_ell", "gtb_velocity_apply", "gtb_evolve_workspace_bytes", "gtb_evolve",
    "gtb_vac_workspace_bytes", "gtb_vac_moments", "gtb_vac_conductivity",
    "gtb_sk_hamiltonian", "gtb_mlp_weight_count", "gtb_mlp_hamiltonian",
    "gtb_spd_workspace_bytes", "gtb_spd_hamiltonian", "gtb_spd_bonds_bytes", "gtb_spd_bonds",
    "gtb_spd_blocks", "gtb_spd_bounds_workspace_bytes", "gtb_spd_bounds",
    "gtb_pack_workspace_bytes", "gtb_packed_rows_bytes", "gtb_packed_dict_bytes", "gtb_pack_ell",
    "gtb_window_bytes", "gtb_window_ell", "gtb_pair_slots", "gtb_mlp_spd_weight_count", "gtb_mlp_spd_blocks",
    "gtb_strip_plan", "gtb_ring_halo", "gtb_strips_workspace_bytes", "gtb_kpm_moments_strips",
    "gtb_mlp_sk_weight_count", "gtb_mlp_sk_hamiltonian", "gtb_carrier_density", "gtb_mobility",
)

KERNEL_AUTO, KERNEL_ROW, KERNEL_ROW_X2, KERNEL_TILE = 0, 1, 2, 3      # gtb_kpm_options.kernel
OPT_PER_PASS_LAUNCH, OPT_SCALAR_BLOCKS, OPT_BLOCK_DIRECT, OPT_SEPARATE_AXPY = 1, 2, 4, 8   # gtb_kpm_options.flags
OPT_GRID_SYNC = 16
MODE_ORB9 = 32              # ... gtb_spd_hamiltonian's (9 orbitals per atom)
MODE_BLOCK9 = 64            # ... the block form written by spd_blocks (H.n = atoms)
MODE_BOND9 = 128            # ... the bond form written by spd_bonds (matrix-free)
MODE_WINDOW = 512           # ... the windowed tiles written by window_ell (wide rows, for one R)
MODE_PACKED = 256           # ... the packed rows + value dictionary written by pack_ell (K <= 4)
MODE_ORB4 = 16              # kpm_moments mode flag: H is gtb_sk_hamiltonian's orbital-blocked matrix
HBAR_EV_FS = 0.6582119569   # hbar in eV*fs: a time of t fs is t / HBAR_EV_FS in the library's hbar/eV


class GtbError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        msg = f"gtb_{where} failed: {status_string(status)} (status {status})"
        if detail:
            msg += f": {detail}"
        super().__init__(msg)
        self.status = status


class _Model(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("onsite", C.c_void_p), ("t0", C.c_void_p),
                ("r0", C.c_double), ("beta", C.c_double), ("onsite_shift", C.c_void_p)]


class _Ell(C.Structure):
    _fields_ = [("n", C.c_int64), ("width", C.c_int32), ("cols", C.c_void_p),
                ("vals", C.c_void_p), ("diag", C.c_void_p)]


class _Options(C.Structure):
    _fields_ = [("kernel", C.c_int32), ("tile_stages", C.c_int32), ("flags", C.c_int32),
                ("loop_begin", C.c_void_p), ("loop_end", C.c_void_p),
                ("loop_passes", C.POINTER(C.c_int32)), ("alt", C.c_void_p), ("alt_mode", C.c_int32)]


class LoopTimer:
    """Caller-owned CUDA events for the timing hooks of gtb_kpm_options (the library records them
    around its recursion loop; it keeps no timing state of its own)."""

    def __init__(self):
        self.begin = torch.cuda.Event(enable_timing=True)
        self.end = torch.cuda.Event(enable_timing=True)
        self.begin.record()      # torch creates the cudaEvent_t at the first record
        self.end.record()
        self.passes = C.c_int32(0)

    def ms(self):
        """(device milliseconds between the two events, fused passes between them); waits for `end`."""
        self.end.synchronize()
        return float(self.begin.elapsed_time(self.end)), int(self.passes.value)


def options(kernel: int = KERNEL_AUTO, tile_stages: int = 0, flags: int = 0,
            timer: Optional[LoopTimer] = None, alt=None, alt_mode: int = 0) -> _Options:
    """A gtb_kpm_options value (argument marshalling only).  alt: an Ell from pack_ell / window_ell of the same
    matrix for vac_moments' fused passes (alt_mode MODE_PACKED / MODE_WINDOW)."""
    o = _Options(kernel, tile_stages, flags, None, None, None, None, 0)
    if alt is not None:
        o._alt_c = alt._c()              # keep the struct (and through `alt` the tensors) alive
        o._alt = alt
        o.alt = C.addressof(o._alt_c)
        o.alt_mode = alt_mode
    if timer is not None:
        o.loop_begin = timer.begin.cuda_event
        o.loop_end = timer.end.cuda_event
        o.loop_passes = C.pointer(timer.passes)
        o._timer = timer         # keep the events alive as long as the struct
    return o


def _opt(o: Optional[_Options]):
    return C.byref(o) if o is not None else None


_lib: Optional[C.CDLL] = None


def lib() -> C.CDLL:
    """Loads libgtb_kpm.so, building it with nvcc first if it is missing or stale."""
    global _lib
    if _lib is None:
        path = _build.LIB
        if _build.needs_build():
            path = _build.build()
        if not os.path.exists(path):
            raise ImportError(f"{path} is missing and could not be built; no fallback exists")
        L = C.CDLL(path)
        L.gtb_status_string.restype = C.c_char_p
        L.gtb_status_string.argtypes = [C.c_int]
        L.gtb_last_cuda_error.restype = C.c_char_p
        L.gtb_launch_count.restype = C.c_int64
        for name in ("gtb_build_workspace_bytes", "gtb_bounds_workspace_bytes"):
            getattr(L, name).restype = C.c_size_t
            getattr(L, name).argtypes = [C.c_int64]
        L.gtb_kpm_workspace_bytes.restype = C.c_size_t
        L.gtb_kpm_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32]
        L.gtb_evolve_workspace_bytes.restype = C.c_size_t
        L.gtb_evolve_workspace_bytes.argtypes = [C.c_int64, C.c_int32]
        L.gtb_vac_workspace_bytes.restype = C.c_size_t
        L.gtb_vac_workspace_bytes.argtypes = [C.c_int64, C.c_int32, C.c_int32, C.c_int32]
        _lib = L
    return _lib


def status_string(status: int) -> str:
    return lib().gtb_status_string(int(status)).decode()


def last_cuda_error() -> str:
    return lib().gtb_last_cuda_error().decode()


def version() -> int:
    return lib().gtb_version()


def launch_count() -> int:
    return int(lib().gtb_launch_count())


def _check(st: int, where: str) -> None:
    if st != OK:
        raise GtbError(st, where, last_cuda_error() if st == ERR_CUDA else "")


def _stream() -> C.c_void_p:
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _ptr(t: Optional[torch.Tensor]) -> C.c_void_p:
    return C.c_void_p(t.data_ptr() if t is not None else None)


def _dev(t: torch.Tensor, dtype: torch.dtype, name: str) -> torch.Tensor:
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA tensor")
    if t.dtype != dtype or not t.is_contiguous():
        raise TypeError(f"{name} must be contiguous {dtype}")
    return t


def _host_f64(x, n: int) -> np.ndarray:
    a = np.ascontiguousarray(x, dtype=np.float64).reshape(-1)
    if a.shape[0] != n:
        raise ValueError(f"expected {n} doubles, got {a.shape[0]}")
    return a


def workspace(nbytes: int, device=None) -> torch.Tensor:
    """A caller-owned device workspace (torch allocations are 512-byte aligned)."""
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device or "cuda")


@dataclass
class Ell:
    """ELL matrix on the device in the layout of include/gtb.h (slot-major [width][n])."""
    n: int
    width: int
    cols: torch.Tensor            # int32 [width, n]
    vals: torch.Tensor            # float64 [width, n]
    diag: Optional[torch.Tensor]  # float64 [n] or None

    def _c(self) -> _Ell:
        return _Ell(self.n, self.width, self.cols.data_ptr() if self.width else None,
                    self.vals.data_ptr() if self.width else None,
                    self.diag.data_ptr() if self.diag is not None else None)

    @staticmethod
    def from_host(cols, vals, diag=None, device="cuda") -> "Ell":
        cols = torch.as_tensor(np.ascontiguousarray(cols, dtype=np.int32)).to(device)
        vals = torch.as_tensor(np.ascontiguousarray(vals, dtype=np.float64)).to(device)
        d = None if diag is None else torch.as_tensor(np.ascontiguousarray(diag, dtype=np.float64)).to(device)
        return Ell(int(cols.shape[1]), int(cols.shape[0]), cols, vals, d)

    def nbytes(self) -> int:
        return self.n * (12 * self.width + (8 if self.diag is not None else 0))


def build_workspace_bytes(n: int) -> int:
    return int(lib().gtb_build_workspace_bytes(n))


def bounds_workspace_bytes(n: int) -> int:
    return int(lib().gtb_bounds_workspace_bytes(n))


def kpm_workspace_bytes(n: int, M: int, R_batch: int) -> int:
    return int(lib().gtb_kpm_workspace_bytes(n, M, R_batch))


def neighbor_width(pos: torch.Tensor, box, pbc, cutoff: float, want_counts: bool = False,
                   ws: Optional[torch.Tensor] = None):
    pos = _dev(pos, torch.float64, "pos")
    n = pos.shape[0]
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    counts = torch.empty(n, dtype=torch.int32, device=pos.device) if want_counts else None
    if ws is None:
        ws = workspace(build_workspace_bytes(n), pos.device)
    width = C.c_int32(0)
    st = lib().gtb_neighbor_width(_ptr(pos), C.c_int64(n), C.c_void_p(box_h.ctypes.data),
                                  C.c_void_p(pbc_h.ctypes.data), C.c_double(cutoff), _ptr(counts),
                                  _ptr(ws), C.c_size_t(ws.numel()), _stream(), C.byref(width))
    _check(st, "neighbor_width")
    return (int(width.value), counts) if want_counts else int(width.value)


def build_hamiltonian(pos: torch.Tensor, species: torch.Tensor, box, pbc, cutoff: float, onsite,
                      t0, r0: float = 1.0, beta: float = 0.0,
                      onsite_shift: Optional[torch.Tensor] = None, width: Optional[int] = None,
                      with_diag: bool = True, ws: Optional[torch.Tensor] = None) -> Ell:
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    n = pos.shape[0]
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    onsite_h = np.ascontiguousarray(onsite, dtype=np.float64).reshape(-1)
    ns = onsite_h.shape[0]
    t0_h = _host_f64(t0, ns * ns)
    if onsite_shift is not None:
        onsite_shift = _dev(onsite_shift, torch.float64, "onsite_shift")
    if ws is None:
        ws = workspace(build_workspace_bytes(n), pos.device)
    if width is None:
        width = neighbor_width(pos, box_h, pbc_h, cutoff, ws=ws)
    H = Ell(n, width, torch.empty((width, n), dtype=torch.int32, device=pos.device),
            torch.empty((width, n), dtype=torch.float64, device=pos.device),
            torch.empty(n, dtype=torch.float64, device=pos.device) if with_diag else None)
    model = _Model(ns, onsite_h.ctypes.data, t0_h.ctypes.data, r0, beta,
                   onsite_shift.data_ptr() if onsite_shift is not None else None)
    hc = H._c()
    need = C.c_int32(0)
    st = lib().gtb_build_hamiltonian(_ptr(pos), _ptr(species), C.c_int64(n),
                                     C.c_void_p(box_h.ctypes.data), C.c_void_p(pbc_h.ctypes.data),
                                     C.c_double(cutoff), C.byref(model), C.byref(hc), _ptr(ws),
                                     C.c_size_t(ws.numel()), _stream(), C.byref(need))
    if st == ERR_ELL_OVERFLOW:
        raise GtbError(st, "build_hamiltonian", f"width {width} given, {need.value} needed")
    _check(st, "build_hamiltonian")
    return H


def spectral_bounds(H: Ell, ws: Optional[torch.Tensor] = None) -> torch.Tensor:
    out = torch.empty(2, dtype=torch.float64, device=H.vals.device)
    if ws is None:
        ws = workspace(bounds_workspace_bytes(H.n), out.device)
    hc = H._c()
    st = lib().gtb_spectral_bounds(C.byref(hc), _ptr(out), _ptr(ws), C.c_size_t(ws.numel()),
                                   _stream())
    _check(st, "spectral_bounds")
    return out


def random_phase_fill(seed: int, r0: int, R: int, n: int, device="cuda") -> torch.Tensor:
    phi = torch.empty((n, R, 2), dtype=torch.float64, device=device)
    st = lib().gtb_random_phase_fill(C.c_uint64(seed & (2**64 - 1)), C.c_int32(r0), C.c_int32(R),
                                     C.c_int64(n), _ptr(phi), _stream())
    _check(st, "random_phase_fill")
    return phi


def kpm_moments(H: Ell, a: float, b: float, M: int, R_total: int = 1,
                R_batch: Optional[int] = None, seed: int = 0, mode: int = 0,
                ws: Optional[torch.Tensor] = None, mu: Optional[torch.Tensor] = None,
                check: bool = False, opt: Optional[_Options] = None) -> torch.Tensor:
    dev = H.vals.device if H.width else H.diag.device
    if R_batch is None:
        R_batch = R_total if (mode & 1) == 0 else 8
    if mu is None:
        mu = torch.empty(M, dtype=torch.float64, device=dev)
    if ws is None:
        rows = 9 * H.n if mode & (MODE_BLOCK9 | MODE_BOND9) else H.n
        ws = workspace(kpm_workspace_bytes(rows, M, R_batch), dev)
    hc = H._c()
    st = lib().gtb_kpm_moments(C.byref(hc), C.c_double(a), C.c_double(b), C.c_int32(M),
                               C.c_int32(R_total), C.c_int32(R_batch),
                               C.c_uint64(seed & (2**64 - 1)), C.c_int32(mode), _ptr(mu), _ptr(ws),
                               C.c_size_t(ws.numel()), _stream(), _opt(opt))
    _check(st, "kpm_moments")
    if check:
        kpm_status(ws)
    return mu


STATIC_WS_BYTES = 4 << 20          # GTB_STATIC_WS_BYTES


def kpm_moments_static(H: Ell, a: float, b: float, M: int, R_total: int = 1, R_batch: Optional[int] = None,
                       seed: int = 0, mode: int = 0, mu: Optional[torch.Tensor] = None,
                       opt: Optional[_Options] = None) -> torch.Tensor:
    """gtb_kpm_moments_static: the moments with the scratch in the library's static device array (no
    allocation inside the call; pass `mu` to allocate nothing here either).  GtbError(ERR_STATIC_LIMIT)
    when the run needs more than STATIC_WS_BYTES."""
    dev = H.vals.device if H.width else H.diag.device
    if R_batch is None:
        R_batch = R_total if (mode & 1) == 0 else 8
    if mu is None:
        mu = torch.empty(M, dtype=torch.float64, device=dev)
    hc = H._c()
    st = lib().gtb_kpm_moments_static(C.byref(hc), C.c_double(a), C.c_double(b), C.c_int32(M),
                                      C.c_int32(R_total), C.c_int32(R_batch), C.c_uint64(seed & (2**64 - 1)),
                                      C.c_int32(mode), _ptr(mu), _stream(), _opt(opt))
    _check(st, "kpm_moments_static")
    return mu


def kpm_status(ws: torch.Tensor) -> None:
    _check(lib().gtb_kpm_status(_ptr(ws), _stream()), "kpm_status")


def kpm_step(H: Ell, a: float, b: float, first: bool, phi_cur: torch.Tensor, phi_io: torch.Tensor,
             ws: Optional[torch.Tensor] = None, opt: Optional[_Options] = None,
             mode: int = 0) -> torch.Tensor:
    """One fused pass; phi_io is overwritten with phi_{n+1}.  Returns the two sums (device [2])."""
    phi_cur = _dev(phi_cur, torch.float64, "phi_cur")
    phi_io = _dev(phi_io, torch.float64, "phi_io")
    R = phi_cur.shape[1]
    sums = torch.empty(2, dtype=torch.float64, device=phi_cur.device)
    if ws is None:
        ws = workspace(kpm_workspace_bytes(phi_cur.shape[0], 2, R), phi_cur.device)
    hc = H._c()
    st = lib().gtb_kpm_step(C.byref(hc), C.c_double(a), C.c_double(b), C.c_int32(int(first)),
                            C.c_int32(R), _ptr(phi_cur), _ptr(phi_io), _ptr(sums), C.c_int32(mode),
                            _ptr(ws), C.c_size_t(ws.numel()), _stream(), _opt(opt))
    _check(st, "kpm_step")
    return sums


def dos(mu: torch.Tensor, a: float, b: float, energies: torch.Tensor, kernel: int = 1,
        scale: float = 1.0, rho: Optional[torch.Tensor] = None) -> torch.Tensor:
    mu = _dev(mu, torch.float64, "mu")
    energies = _dev(energies, torch.float64, "energies")
    if rho is None:
        rho = torch.empty_like(energies)
    st = lib().gtb_dos(_ptr(mu), C.c_int32(mu.shape[0]), C.c_double(a), C.c_double(b),
                       C.c_int32(kernel), _ptr(energies), C.c_int32(energies.shape[0]),
                       C.c_double(scale), _ptr(rho), _stream())
    _check(st, "dos")
    return rho


def jackson(M: int, device="cuda") -> torch.Tensor:
    g = torch.empty(M, dtype=torch.float64, device=device)
    _check(lib().gtb_jackson(C.c_int32(M), _ptr(g), _stream()), "jackson")
    return g


# ---------------------------------------------------------------- VAC conductivity (Eq. 3)
def evolve_workspace_bytes(n: int, R: int) -> int:
    return int(lib().gtb_evolve_workspace_bytes(n, R))


def vac_workspace_bytes(n: int, M: int, n_steps: int, R_batch: int) -> int:
    return int(lib().gtb_vac_workspace_bytes(n, M, n_steps, R_batch))


def velocity_ell(H: Ell, pos: torch.Tensor, box, pbc, axis: int = 0) -> torch.Tensor:
    """vvals [width][n] with V = i * vvals on the pattern of H (reading V1)."""
    pos = _dev(pos, torch.float64, "pos")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    out = torch.empty_like(H.vals)
    hc = H._c()
    st = lib().gtb_velocity_ell(C.byref(hc), _ptr(pos), C.c_void_p(box_h.ctypes.data),
                                C.c_void_p(pbc_h.ctypes.data), C.c_int32(axis), _ptr(out), _stream())
    _check(st, "velocity_ell")
    return out


def velocity_apply(H: Ell, vvals: torch.Tensor, x: torch.Tensor) -> torch.Tensor:
    x = _dev(x, torch.float64, "x")
    y = torch.empty_like(x)
    hc = H._c()
    st = lib().gtb_velocity_apply(C.byref(hc), _ptr(vvals), C.c_int32(x.shape[1]), _ptr(x), _ptr(y),
                                  _stream())
    _check(st, "velocity_apply")
    return y


def evolve(H: Ell, a: float, b: float, dt: float, phi: torch.Tensor,
           ws: Optional[torch.Tensor] = None) -> int:
    """phi <- exp(-i H dt) phi in place; returns the number of Chebyshev terms used."""
    phi = _dev(phi, torch.float64, "phi")
    R = phi.shape[1]
    if ws is None:
        ws = workspace(evolve_workspace_bytes(H.n, R), phi.device)
    terms = C.c_int32(0)
    hc = H._c()
    st = lib().gtb_evolve(C.byref(hc), C.c_double(a), C.c_double(b), C.c_double(dt), C.c_int32(R),
                          _ptr(phi), C.byref(terms), _ptr(ws), C.c_size_t(ws.numel()), _stream())
    _check(st, "evolve")
    return int(terms.value)


def vac_moments(H: Ell, vvals: torch.Tensor, a: float, b: float, M: int, n_steps: int, dt: float,
                R_total: int = 1, R_batch: Optional[int] = None, seed: int = 0, mode: int = 0,
                ws: Optional[torch.Tensor] = None, out: Optional[torch.Tensor] = None,
                check: bool = False, opt: Optional[_Options] = None) -> torch.Tensor:
    """C[j][n], j < n_steps, n < M (readings V2, V3)."""
    dev = H.vals.device
    if R_batch is None:
        R_batch = R_total if (mode & 1) == 0 else 8
    if out is None:
        out = torch.empty((n_steps, M), dtype=torch.float64, device=dev)
    if ws is None:
        ws = workspace(vac_workspace_bytes(H.n, M, n_steps, R_batch), dev)
    hc = H._c()
    st = lib().gtb_vac_moments(C.byref(hc), _ptr(vvals), C.c_double(a), C.c_double(b), C.c_int32(M),
                               C.c_int32(n_steps), C.c_double(dt), C.c_int32(R_total),
                               C.c_int32(R_batch), C.c_uint64(seed & (2**64 - 1)), C.c_int32(mode),
                               _ptr(out), _ptr(ws), C.c_size_t(ws.numel()), _stream(), _opt(opt))
    _check(st, "vac_moments")
    if check:
        kpm_status(ws)
    return out


def vac_conductivity(Cm: torch.Tensor, a: float, b: float, energies: torch.Tensor, dt: float,
                     kernel: int = 1, scale: float = 1.0):
    """(rho_vv[j][g], sigma[j][g]) from C[j][n] (readings V5, V6)."""
    Cm = _dev(Cm, torch.float64, "C")
    energies = _dev(energies, torch.float64, "energies")
    n_steps, M = Cm.shape
    G = energies.shape[0]
    rv = torch.empty((n_steps, G), dtype=torch.float64, device=Cm.device)
    sg = torch.empty_like(rv)
    st = lib().gtb_vac_conductivity(_ptr(Cm), C.c_int32(M), C.c_int32(n_steps), C.c_double(a),
                                    C.c_double(b), C.c_int32(kernel), _ptr(energies), C.c_int32(G),
                                    C.c_double(dt), C.c_double(scale), _ptr(rv), _ptr(sg), _stream())
    _check(st, "vac_conductivity")
    return rv, sg


# ---------------------------------------------------------------- Slater-Koster s,p blocks (NEXT-2)
class _SkModel(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("onsite_s", C.c_void_p), ("onsite_p", C.c_void_p),
                ("sk", C.c_void_p), ("r0", C.c_double), ("beta", C.c_double),
                ("onsite_shift", C.c_void_p)]


def sk_hamiltonian(nbr: Ell, pos: torch.Tensor, species: torch.Tensor, box, pbc, onsite_s, onsite_p,
                   sk, r0: float = 1.0, beta: float = 0.0, onsite_shift: Optional[torch.Tensor] = None,
                   with_diag: bool = True) -> Ell:
    """Scalar ELL over the 4n orbitals (s, px, py, pz per atom) from the neighbour lists of `nbr`."""
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    es = np.ascontiguousarray(onsite_s, dtype=np.float64).reshape(-1)
    ep = np.ascontiguousarray(onsite_p, dtype=np.float64).reshape(-1)
    ns = es.shape[0]
    sk_h = _host_f64(sk, ns * ns * 4)
    if onsite_shift is not None:
        onsite_shift = _dev(onsite_shift, torch.float64, "onsite_shift")
    n, K, dev = nbr.n, nbr.width, pos.device
    H = Ell(4 * n, 4 * K, torch.empty((4 * K, 4 * n), dtype=torch.int32, device=dev),
            torch.empty((4 * K, 4 * n), dtype=torch.float64, device=dev),
            torch.empty(4 * n, dtype=torch.float64, device=dev) if with_diag else None)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    model = _SkModel(ns, es.ctypes.data, ep.ctypes.data, sk_h.ctypes.data, r0, beta,
                     onsite_shift.data_ptr() if onsite_shift is not None else None)
    nc, hc = nbr._c(), H._c()
    st = lib().gtb_sk_hamiltonian(C.byref(nc), _ptr(pos), _ptr(species), C.c_void_p(box_h.ctypes.data),
                                  C.c_void_p(pbc_h.ctypes.data), C.byref(model), C.byref(hc),
                                  _ptr(status), _stream())
    _check(st, "sk_hamiltonian")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "sk_hamiltonian", "species index out of range")
    return H


# ---------------------------------------------------------------- descriptor + MLP Hamiltonian (Eq. 2, NEXT-3)
class _MlpModel(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("n_features", C.c_int32), ("n_basis", C.c_int32),
                ("n_hidden", C.c_int32), ("r_cut", C.c_double), ("weights", C.c_void_p)]


def mlp_hamiltonian(nbr: Ell, pos: torch.Tensor, species: torch.Tensor, box, pbc, dims, r_cut: float,
                    weights: torch.Tensor, with_diag: bool = True, return_v: bool = False):
    """H on the neighbour lists of `nbr` (its cols are shared, not copied) with t_ij, eps_i from Eq. 2."""
    ns, F, Nb, Hd = dims
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    weights = _dev(weights, torch.float64, "weights")
    lib().gtb_mlp_weight_count.restype = C.c_size_t
    need = int(lib().gtb_mlp_weight_count(C.c_int32(ns), C.c_int32(F), C.c_int32(Nb), C.c_int32(Hd)))
    if weights.numel() != need:
        raise GtbError(ERR_INVALID_ARG, "mlp_hamiltonian", f"weight blob has {weights.numel()} doubles, {need} expected")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    dev = pos.device
    H = Ell(nbr.n, nbr.width, nbr.cols, torch.empty((nbr.width, nbr.n), dtype=torch.float64, device=dev),
            torch.empty(nbr.n, dtype=torch.float64, device=dev) if with_diag else None)
    v = torch.empty((nbr.n, F), dtype=torch.float64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    model = _MlpModel(ns, F, Nb, Hd, r_cut, weights.data_ptr())
    hc = H._c()
    st = lib().gtb_mlp_hamiltonian(C.byref(model), _ptr(pos), _ptr(species), C.c_void_p(box_h.ctypes.data),
                                   C.c_void_p(pbc_h.ctypes.data), C.byref(hc), _ptr(v), _ptr(status), _stream())
    _check(st, "mlp_hamiltonian")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "mlp_hamiltonian", "species index out of range")
    return (H, v) if return_v else H


# ---------------------------------------------------------------- Slater-Koster s,p,d blocks (NEXT-2)
class _SpdModel(C.Structure):
    _fields_ = [("n_species", C.c_int32), ("onsite_s", C.c_void_p), ("onsite_p", C.c_void_p),
                ("onsite_d", C.c_void_p), ("sk", C.c_void_p), ("r0", C.c_double), ("beta", C.c_double),
                ("onsite_shift", C.c_void_p)]


def spd_hamiltonian(nbr: Ell, pos: torch.Tensor, species: torch.Tensor, box, pbc, onsite_s, onsite_p,
                    onsite_d, sk, r0: float = 1.0, beta: float = 0.0,
                    onsite_shift: Optional[torch.Tensor] = None, with_diag: bool = True) -> Ell:
    """Scalar ELL over the 9n orbitals (s, p, d per atom) from the neighbour lists of `nbr`."""
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    es, ep, ed = (np.ascontiguousarray(x, dtype=np.float64).reshape(-1) for x in (onsite_s, onsite_p, onsite_d))
    ns = es.shape[0]
    sk_h = _host_f64(sk, ns * ns * 10)
    if onsite_shift is not None:
        onsite_shift = _dev(onsite_shift, torch.float64, "onsite_shift")
    n, K, dev = nbr.n, nbr.width, pos.device
    H = Ell(9 * n, 9 * K, torch.empty((9 * K, 9 * n), dtype=torch.int32, device=dev),
            torch.empty((9 * K, 9 * n), dtype=torch.float64, device=dev),
            torch.empty(9 * n, dtype=torch.float64, device=dev) if with_diag else None)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    lib().gtb_spd_workspace_bytes.restype = C.c_size_t
    ws = workspace(int(lib().gtb_spd_workspace_bytes()), dev)
    model = _SpdModel(ns, es.ctypes.data, ep.ctypes.data, ed.ctypes.data, sk_h.ctypes.data, r0, beta,
                      onsite_shift.data_ptr() if onsite_shift is not None else None)
    nc, hc = nbr._c(), H._c()
    st = lib().gtb_spd_hamiltonian(C.byref(nc), _ptr(pos), _ptr(species), C.c_void_p(box_h.ctypes.data),
                                   C.c_void_p(pbc_h.ctypes.data), C.byref(model), C.byref(hc), _ptr(status),
                                   _ptr(ws), C.c_size_t(ws.numel()), _stream())
    _check(st, "spd_hamiltonian")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "spd_hamiltonian", "species index out of range")
    return H


def mlp_sk_hamiltonian(nbr: Ell, pos: torch.Tensor, species: torch.Tensor, box, pbc, dims, r_cut: float,
                       weights: torch.Tensor, with_diag: bool = True) -> Ell:
    """Eq. 2 feeding the s,p Slater-Koster blocks: scalar ELL over the 4n orbitals (use mode=MODE_ORB4)."""
    ns, F, Nb, Hd = dims
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    weights = _dev(weights, torch.float64, "weights")
    lib().gtb_mlp_sk_weight_count.restype = C.c_size_t
    need = int(lib().gtb_mlp_sk_weight_count(C.c_int32(ns), C.c_int32(F), C.c_int32(Nb), C.c_int32(Hd)))
    if weights.numel() != need:
        raise GtbError(ERR_INVALID_ARG, "mlp_sk_hamiltonian", f"weight blob has {weights.numel()} doubles, {need} expected")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    n, K, dev = nbr.n, nbr.width, pos.device
    H = Ell(4 * n, 4 * K, torch.empty((4 * K, 4 * n), dtype=torch.int32, device=dev),
            torch.empty((4 * K, 4 * n), dtype=torch.float64, device=dev),
            torch.empty(4 * n, dtype=torch.float64, device=dev) if with_diag else None)
    v = torch.empty((n, F), dtype=torch.float64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    model = _MlpModel(ns, F, Nb, Hd, r_cut, weights.data_ptr())
    nc, hc = nbr._c(), H._c()
    st = lib().gtb_mlp_sk_hamiltonian(C.byref(model), C.byref(nc), _ptr(pos), _ptr(species),
                                      C.c_void_p(box_h.ctypes.data), C.c_void_p(pbc_h.ctypes.data),
                                      C.byref(hc), _ptr(v), _ptr(status), _stream())
    _check(st, "mlp_sk_hamiltonian")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "mlp_sk_hamiltonian", "species index out of range")
    return H


def spd_bonds(nbr: Ell, pos: torch.Tensor, species: torch.Tensor, box, pbc, onsite_s, onsite_p, onsite_d, sk,
              r0: float = 1.0, beta: float = 0.0, onsite_shift: Optional[torch.Tensor] = None) -> Ell:
    """The bond (matrix-free) form of the s,p,d Hamiltonian for kpm_moments(..., mode=MODE_BOND9): the
    neighbour lists of `nbr` (shared) and a device block of parameter tables + atom records in `vals`."""
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    es, ep, ed = (np.ascontiguousarray(x, dtype=np.float64).reshape(-1) for x in (onsite_s, onsite_p, onsite_d))
    ns = es.shape[0]
    sk_h = _host_f64(sk, ns * ns * 10)
    if onsite_shift is not None:
        onsite_shift = _dev(onsite_shift, torch.float64, "onsite_shift")
    dev = pos.device
    lib().gtb_spd_bonds_bytes.restype = C.c_size_t
    nbytes = int(lib().gtb_spd_bonds_bytes(C.c_int64(nbr.n)))
    blob = torch.empty(nbytes // 8, dtype=torch.float64, device=dev)
    Hm = Ell(nbr.n, nbr.width, nbr.cols, blob, None)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    model = _SpdModel(ns, es.ctypes.data, ep.ctypes.data, ed.ctypes.data, sk_h.ctypes.data, r0, beta,
                      onsite_shift.data_ptr() if onsite_shift is not None else None)
    nc, hc = nbr._c(), Hm._c()
    st = lib().gtb_spd_bonds(C.byref(nc), _ptr(pos), _ptr(species), C.c_void_p(box_h.ctypes.data),
                             C.c_void_p(pbc_h.ctypes.data), C.byref(model), C.byref(hc), _ptr(status), _stream())
    _check(st, "spd_bonds")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "spd_bonds", "species index out of range")
    return Hm


def spd_blocks(Hm: Ell, with_diag: bool = True) -> Ell:
    """The block form (cols [K][n] shared, blocks [K][81][n], onsite [9][n]) for mode=MODE_BLOCK9."""
    dev = Hm.vals.device
    Hb = Ell(Hm.n, Hm.width, Hm.cols, torch.empty((max(Hm.width, 1), 81, Hm.n), dtype=torch.float64, device=dev),
             torch.empty((9, Hm.n), dtype=torch.float64, device=dev) if with_diag else None)
    mc, bc = Hm._c(), Hb._c()
    _check(lib().gtb_spd_blocks(C.byref(mc), C.byref(bc), _stream()), "spd_blocks")
    return Hb


def spd_bounds(H: Ell, mode: int) -> torch.Tensor:
    """Gershgorin interval (device [2]) of the orbital matrix held in block or bond form."""
    out = torch.empty(2, dtype=torch.float64, device=H.vals.device)
    lib().gtb_spd_bounds_workspace_bytes.restype = C.c_size_t
    ws = workspace(int(lib().gtb_spd_bounds_workspace_bytes()), out.device)
    hc = H._c()
    _check(lib().gtb_spd_bounds(C.byref(hc), C.c_int32(mode), _ptr(out), _ptr(ws), C.c_size_t(ws.numel()),
                                _stream()), "spd_bounds")
    return out


def mlp_spd_blocks(nbr: Ell, pos: torch.Tensor, species: torch.Tensor, box, pbc, dims, r_cut: float,
                   weights: torch.Tensor, with_diag: bool = True) -> Ell:
    """Eq. 2 feeding the s,p,d blocks (ten-output MLP_lambda): the block form for mode=MODE_BLOCK9."""
    ns, F, Nb, Hd = dims
    pos = _dev(pos, torch.float64, "pos")
    species = _dev(species, torch.int32, "species")
    weights = _dev(weights, torch.float64, "weights")
    lib().gtb_mlp_spd_weight_count.restype = C.c_size_t
    need = int(lib().gtb_mlp_spd_weight_count(C.c_int32(ns), C.c_int32(F), C.c_int32(Nb), C.c_int32(Hd)))
    if weights.numel() != need:
        raise GtbError(ERR_INVALID_ARG, "mlp_spd_blocks", f"weight blob has {weights.numel()} doubles, {need} expected")
    box_h = _host_f64(box, 3)
    pbc_h = np.ascontiguousarray(pbc, dtype=np.int32)
    n, K, dev = nbr.n, nbr.width, pos.device
    Hb = Ell(n, K, nbr.cols, torch.empty((max(K, 1), 81, n), dtype=torch.float64, device=dev),
             torch.empty((9, n), dtype=torch.float64, device=dev) if with_diag else None)
    v = torch.empty((n, F), dtype=torch.float64, device=dev)
    status = torch.zeros(1, dtype=torch.int32, device=dev)
    model = _MlpModel(ns, F, Nb, Hd, r_cut, weights.data_ptr())
    nc, hc = nbr._c(), Hb._c()
    st = lib().gtb_mlp_spd_blocks(C.byref(model), C.byref(nc), _ptr(pos), _ptr(species),
                                  C.c_void_p(box_h.ctypes.data), C.c_void_p(pbc_h.ctypes.data),
                                  C.byref(hc), _ptr(v), _ptr(status), _stream())
    _check(st, "mlp_spd_blocks")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "mlp_spd_blocks", "species index out of range")
    return Hb


def strip_plan(n: int, n_strips: int, halo: int, p: int) -> dict:
    """Host-only: the rows strip p owns and where its two halos come from (include/gtb.h)."""
    out = (C.c_int64 * 6)()
    _check(lib().gtb_strip_plan(C.c_int64(n), C.c_int32(n_strips), C.c_int64(halo), C.c_int32(p), out), "strip_plan")
    return dict(zip(("row0", "rows", "lo_first", "hi_first", "lo_owner", "hi_owner"), (int(x) for x in out)))


def ring_halo(H: Ell) -> int:
    scratch = torch.zeros(1, dtype=torch.int32, device=H.vals.device)
    h = C.c_int64(0)
    hc = H._c()
    _check(lib().gtb_ring_halo(C.byref(hc), _ptr(scratch), _stream(), C.byref(h)), "ring_halo")
    return int(h.value)


def kpm_moments_strips(H: Ell, n_strips: int, a: float, b: float, M: int, R_total: int = 1,
                       R_batch: Optional[int] = None, seed: int = 0, mode: int = 0, halo: Optional[int] = None,
                       want_phi: bool = False, check: bool = False, opt: Optional[_Options] = None):
    """gtb_kpm_moments on n_strips row strips with one halo exchange per pass; (mu, phi_last or None)."""
    dev = H.vals.device
    if R_batch is None:
        R_batch = R_total if mode == 0 else 8
    if halo is None:
        halo = ring_halo(H)
    L = lib()
    L.gtb_strips_workspace_bytes.restype = C.c_size_t
    need = int(L.gtb_strips_workspace_bytes(C.c_int64(H.n), C.c_int32(H.width), C.c_int32(int(H.diag is not None)),
                                            C.c_int32(n_strips), C.c_int64(halo), C.c_int32(M), C.c_int32(R_batch)))
    if need == 0:
        raise GtbError(ERR_INVALID_ARG, "kpm_moments_strips", "a strip is narrower than the halo")
    ws = workspace(need, dev)
    mu = torch.empty(M, dtype=torch.float64, device=dev)
    phi = torch.empty((H.n, R_batch, 2), dtype=torch.float64, device=dev) if want_phi else None
    hc = H._c()
    st = L.gtb_kpm_moments_strips(C.byref(hc), C.c_int32(n_strips), C.c_int64(halo), C.c_double(a), C.c_double(b),
                                  C.c_int32(M), C.c_int32(R_total), C.c_int32(R_batch),
                                  C.c_uint64(seed & (2**64 - 1)), C.c_int32(mode), _ptr(mu), _ptr(phi), _ptr(ws),
                                  C.c_size_t(ws.numel()), _stream(), _opt(opt))
    _check(st, "kpm_moments_strips")
    if check:
        kpm_status(ws)
    return mu, phi


def pack_ell(H: Ell, ws: Optional[torch.Tensor] = None) -> Optional[Ell]:
    """The packed form of a narrow matrix (K <= 4) for mode=MODE_PACKED: `cols` holds the 16-byte packed rows
    (int32 [n][4]; `short_rows`: 8-byte rows in its first half), `vals` the header + value dictionary.  None when the matrix does not fit the format
    (GTB_ERR_NOT_PACKABLE): stay on the plain path."""
    L = lib()
    for name in ("gtb_pack_workspace_bytes", "gtb_packed_dict_bytes"):
        getattr(L, name).restype = C.c_size_t
    L.gtb_packed_rows_bytes.restype = C.c_size_t
    L.gtb_packed_rows_bytes.argtypes = [C.c_int64]
    dev = H.vals.device
    if ws is None:
        ws = workspace(int(L.gtb_pack_workspace_bytes()), dev)
    rows = torch.empty((int(L.gtb_packed_rows_bytes(H.n)) // 16, 4), dtype=torch.int32, device=dev)
    blob = torch.empty(int(L.gtb_packed_dict_bytes()) // 8, dtype=torch.float64, device=dev)
    P = Ell(H.n, H.width, rows, blob, None)
    hc, pc = H._c(), P._c()
    nv = C.c_int32(0)
    st = L.gtb_pack_ell(C.byref(hc), C.byref(pc), _ptr(ws), C.c_size_t(ws.numel()), _stream(), C.byref(nv))
    if st == ERR_NOT_PACKABLE:
        return None
    _check(st, "pack_ell")
    if pc.diag:                      # K = 4 with a diagonal: the array is still read
        P.diag = H.diag
    P.n_values = int(nv.value)
    P.width = int(pc.width)          # K | 0x100: 8-byte rows (K <= 3 and at most 16 distinct values)
    P.short_rows = bool(P.width & 0x100)
    return P


def pair_slots(H: Ell, R: int) -> Ell:
    """gtb_pair_slots: the same matrix as a plain ELL with the slots of neighbouring rows ordered for the gathers
    of an R-vector pass (R = 4: rows 2q, 2q + 1 alternate in column parity); a copy for any other R."""
    Hp = Ell(H.n, H.width, torch.empty_like(H.cols), torch.empty_like(H.vals), H.diag)
    hc, pc = H._c(), Hp._c()
    _check(lib().gtb_pair_slots(C.byref(hc), C.c_int32(R), C.byref(pc), _stream()), "pair_slots")
    return Hp


def window_ell(H: Ell, R: int) -> Optional[Ell]:
    """The windowed-tile form of a wide matrix for mode=MODE_WINDOW with R_batch = R (2, 4 or 8).  None when a
    tile's neighbours are too scattered (GTB_ERR_NOT_PACKABLE): stay on the plain path."""
    L = lib()
    L.gtb_window_bytes.restype = C.c_size_t
    dev = H.vals.device
    nbytes = int(L.gtb_window_bytes(C.c_int64(H.n), C.c_int32(H.width), C.c_int32(R),
                                    C.c_int32(int(H.diag is not None))))
    if nbytes == 0:
        raise GtbError(ERR_INVALID_ARG, "window_ell", "R must be 2, 4 or 8 and the width at least 1")
    blob = torch.empty(nbytes // 8, dtype=torch.float64, device=dev)
    scratch = torch.zeros(1, dtype=torch.int32, device=dev)
    Wd = Ell(H.n, H.width, H.cols, blob, H.diag)
    hc, wc = H._c(), Wd._c()
    need = C.c_int32(0)
    st = L.gtb_window_ell(C.byref(hc), C.c_int32(R), C.byref(wc), _ptr(scratch), _stream(), C.byref(need))
    if st == ERR_NOT_PACKABLE:
        return None
    _check(st, "window_ell")
    Wd.width = int(wc.width)         # K + 65536 x blocks of the largest window
    Wd.R = R
    Wd.blocks = int(need.value)
    return Wd


# ---------------------------------------------------------------- Fig. 4b post-processing
def carrier_density(rho: torch.Tensor, energies: torch.Tensor, e_ref: float) -> torch.Tensor:
    """n(E_j) = int_{e_ref}^{E_j} rho dE by the trapezoid rule (reading V7)."""
    rho = _dev(rho, torch.float64, "rho")
    energies = _dev(energies, torch.float64, "energies")
    out = torch.empty_like(rho)
    status = torch.zeros(1, dtype=torch.int32, device=rho.device)
    st = lib().gtb_carrier_density(_ptr(rho), _ptr(energies), C.c_int32(rho.shape[0]), C.c_double(e_ref),
                                   _ptr(out), _ptr(status), _stream())
    _check(st, "carrier_density")
    if int(status.item()) != 0:
        raise GtbError(ERR_INVALID_ARG, "carrier_density", "grid not ascending or e_ref outside it")
    return out


def mobility(sigma: torch.Tensor, n: torch.Tensor, scale: float = 1.0, n_min: float = 0.0) -> torch.Tensor:
    """mu = scale * sigma / |n| where |n| > n_min, else 0 (reading V8)."""
    sigma = _dev(sigma, torch.float64, "sigma")
    n = _dev(n, torch.float64, "n")
    out = torch.empty_like(sigma)
    _check(lib().gtb_mobility(_ptr(sigma), _ptr(n), C.c_int32(sigma.shape[0]), C.c_double(scale),
                              C.c_double(n_min), _ptr(out), _stream()), "mobility")
    return out
