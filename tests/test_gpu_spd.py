"""GPU parity of the s,p,d Slater-Koster path (9 orbitals per atom):
block assembly against oracle/gtbo_spd.cpp, then the scalar kernels and the 9x9 blocked pass (K7b9,
GTB_MODE_ORB9) on the 9n-orbital matrix.  Tolerances: columns and onsite bit-exact; values 1e-13 of the
largest (frame construction, sqrt, divisions, exp, FMA contraction); moments 1e-9 (north_star)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu

V1 = np.array([-6.769, 5.580, 5.037, -3.033, -2.1, -1.7, 0.9, -1.3, 0.8, -0.15])
V3 = np.zeros((3, 3, 10))
for (a, b), f in {(0, 0): 1.0, (1, 2): 0.96, (0, 1): 0.93, (0, 2): 1.04, (1, 1): 0.5, (2, 2): 0.5}.items():
    V3[a, b] = V3[b, a] = f * V1
ES, EP, ED = [-8.868, -6.0, -11.0], [0.0, 2.3, -2.3], [6.5, 7.0, 5.5]


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _both(key, nx, ny, cutoff, beta, **kw):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    ns = int(inp.species.max()) + 1
    sk = V1.reshape(1, 1, 10) if ns == 1 else V3
    ones = np.ones((ns, ns))
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                     with_diag=False, method=1)
    Ho = oracle.spd_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, ES[:ns], EP[:ns], ED[:ns],
                                sk, r0=1.42, beta=beta, onsite_shift=inp.onsite_shift)
    nbr_g = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, cutoff, [0.0] * ns,
                                  ones, with_diag=False)
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    Hg = gtb.spd_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, ES[:ns], EP[:ns],
                             ED[:ns], sk, r0=1.42, beta=beta, onsite_shift=shift)
    return w, inp, Ho, Hg


CASES = [("c1", 12, 12, 1.95, 0.0, {}), ("c2b", 13, 9, 2.65, 3.37, {}), ("c2", 15, 11, 1.95, 2.0, {}),
         ("c4", 24, 9, 1.95, 1.5, {"stripe": 3})]


@pytest.mark.parametrize("key,nx,ny,cutoff,beta,kw", CASES)
def test_blocks_match_oracle(key, nx, ny, cutoff, beta, kw):
    w, inp, Ho, Hg = _both(key, nx, ny, cutoff, beta, **kw)
    assert Hg.n == Ho.n == 9 * w.n_atoms and Hg.width == Ho.width
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()
    assert np.abs(Hg.vals.cpu().numpy() - Ho.vals).max() <= 1e-13 * np.abs(Ho.vals).max()
    assert (Hg.diag.cpu().numpy() == Ho.diag).all()


@pytest.mark.parametrize("key,nx,ny,cutoff,beta,kw", CASES)
@pytest.mark.parametrize("R_total,R_batch", [(2, 2), (4, 4), (8, 8), (3, 3)])
def test_moments_scalar_and_blocked(key, nx, ny, cutoff, beta, kw, R_total, R_batch):
    w, inp, Ho, Hg = _both(key, nx, ny, cutoff, beta, **kw)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    M = 49
    ref = oracle.kpm_moments(Ho, a, b, M, R_total, 31, mode=0, algo=0)
    plain = gtb.kpm_moments(Hg, a, b, M, R_total, R_batch, 31, check=True).cpu().numpy()
    assert np.abs(plain - ref).max() <= 1e-9 and np.abs(plain - ref).max() <= 1e-12
    got = gtb.kpm_moments(Hg, a, b, M, R_total, R_batch, 31, mode=gtb.MODE_ORB9, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12
    assert np.abs(got - plain).max() <= 1e-13
    Hn, Hon = gtb.Ell(Hg.n, Hg.width, Hg.cols, Hg.vals, None), oracle.Ell(Ho.n, Ho.width, Ho.cols, Ho.vals, None)
    ref = oracle.kpm_moments(Hon, a, b, 20, R_total, 32, mode=0, algo=0)
    got = gtb.kpm_moments(Hn, a, b, 20, R_total, R_batch, 32, mode=gtb.MODE_ORB9).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12


def test_exact_trace_dos_and_vac_on_the_spd_matrix():
    w, inp, Ho, Hg = _both("c2b", 4, 3, 2.65, 3.37)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    got = gtb.kpm_moments(Hg, a, b, 32, mode=1 | gtb.MODE_ORB9, R_batch=8).cpu().numpy()
    th = np.arccos((np.linalg.eigvalsh(Ho.to_dense()) - b) / a)
    assert np.abs(got - np.array([np.cos(k * th).mean() for k in range(32)])).max() <= 1e-12
    E = np.linspace(b - a, b + a, 201)[1:-1]
    rho_ref = oracle.dos(got, a, b, E)
    assert np.abs(gtb.dos(_dev(got), a, b, _dev(E)).cpu().numpy() - rho_ref).max() <= 1e-8 * rho_ref.max()
    pos9 = np.repeat(inp.pos, 9, axis=0)
    vo = oracle.velocity_ell(Ho, pos9, inp.box, inp.pbc, 0)
    vg = gtb.velocity_ell(Hg, _dev(pos9), inp.box, inp.pbc, 0)
    dt = 0.1 / gtb.HBAR_EV_FS
    ref = oracle.vac_moments(Ho, vo, a, b, 12, 3, dt, R=2, seed=4, mode=0)
    for mode in (0, gtb.MODE_ORB9):
        c = gtb.vac_moments(Hg, vg, a, b, 12, 3, dt, 2, 2, 4, mode=mode, check=True).cpu().numpy()
        assert np.abs(c - ref).max() <= 1e-11 * ref[0, 0]


def test_bad_flags_and_species():
    w, inp, Ho, Hg = _both("c1", 6, 6, 1.95, 0.0)
    with pytest.raises(gtb.GtbError):
        gtb.kpm_moments(Hg, 30.0, 0.0, 8, 2, 2, 0, mode=gtb.MODE_ORB4 | gtb.MODE_ORB9)
    nbr = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, 1.95, [0.0], [1.0],
                                with_diag=False)
    bad = inp.species.copy()
    bad[5] = 2
    with pytest.raises(gtb.GtbError):
        gtb.spd_hamiltonian(nbr, _dev(inp.pos), _dev(bad), inp.box, inp.pbc, [0.0], [0.0], [0.0], V1)
