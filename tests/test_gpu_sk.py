"""GPU parity of the multi-orbital Slater-Koster path (NEXT-2): block assembly
against oracle/gtbo_sk.cpp, then the unchanged KPM / DOS / VAC kernels on the 4n-orbital matrix.
Tolerances: columns bit-exact; values 8 ulp of the largest parameter (a square root, three divisions
and one exp of another libm, FMA contraction); moments 1e-9 (north_star), DOS 1e-8 of its peak."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu

SK1 = np.array([-6.769, 5.580, 5.037, -3.033])
SK3 = np.zeros((3, 3, 4))                       # C, B, N (config 4's species), symmetric table
for (a, b), scale in {(0, 0): 1.0, (1, 2): 0.96, (0, 1): 0.93, (0, 2): 1.04, (1, 1): 0.5, (2, 2): 0.5}.items():
    SK3[a, b] = SK3[b, a] = scale * SK1


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _both(key, nx, ny, cutoff, beta, **kw):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    ns = int(inp.species.max()) + 1
    sk = SK1.reshape(1, 1, 4) if ns == 1 else SK3
    es, ep = [-8.868, -6.0, -11.0][:ns], [0.0, 2.3, -2.3][:ns]
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns,
                                     np.ones((ns, ns)), with_diag=False, method=1)
    Ho = oracle.sk_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, es, ep, sk, r0=1.42,
                               beta=beta, onsite_shift=inp.onsite_shift)
    nbr_g = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, cutoff,
                                  [0.0] * ns, np.ones((ns, ns)), with_diag=False)
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    Hg = gtb.sk_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, es, ep, sk,
                            r0=1.42, beta=beta, onsite_shift=shift)
    return w, inp, Ho, Hg


CASES = [("c1", 24, 24, 1.95, 0.0, {}), ("c2b", 21, 13, 2.65, 3.37, {}), ("c2", 19, 11, 1.95, 2.0, {}),
         ("c4", 24, 9, 1.95, 1.5, {"stripe": 3})]


@pytest.mark.parametrize("key,nx,ny,cutoff,beta,kw", CASES)
def test_blocks_match_oracle(key, nx, ny, cutoff, beta, kw):
    w, inp, Ho, Hg = _both(key, nx, ny, cutoff, beta, **kw)
    assert Hg.n == Ho.n == 4 * w.n_atoms and Hg.width == Ho.width
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()
    assert np.abs(Hg.vals.cpu().numpy() - Ho.vals).max() <= 8 * 2.0**-52 * np.abs(Ho.vals).max()
    assert (Hg.diag.cpu().numpy() == Ho.diag).all()
    dense = Ho.to_dense() if Ho.n <= 2400 else None
    if dense is not None:
        assert np.abs(dense - dense.T).max() <= 1e-14      # the assembled matrix is symmetric


@pytest.mark.parametrize("key,nx,ny,cutoff,beta,kw", CASES)
@pytest.mark.parametrize("R", [2, 8])
def test_moments_and_dos_on_the_orbital_matrix(key, nx, ny, cutoff, beta, kw, R):
    w, inp, Ho, Hg = _both(key, nx, ny, cutoff, beta, **kw)
    lo, hi = oracle.spectral_bounds(Ho)
    lo_hi = gtb.spectral_bounds(Hg).cpu().numpy()
    assert np.abs(lo_hi - [lo, hi]).max() <= 1e-12 * max(abs(lo), abs(hi))
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    M = 96
    ref = oracle.kpm_moments(Ho, a, b, M, R, 11, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, M, R, R, 11, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-9
    assert np.abs(got - ref).max() <= 1e-12
    E = np.linspace(b - a, b + a, 301)[1:-1]
    rho_ref = oracle.dos(ref, a, b, E)
    rho = gtb.dos(_dev(got), a, b, _dev(E)).cpu().numpy()
    assert np.abs(rho - rho_ref).max() <= 1e-8 * rho_ref.max()


@pytest.mark.parametrize("key,nx,ny,cutoff,beta,kw", CASES)
@pytest.mark.parametrize("R_total,R_batch", [(2, 2), (4, 4), (8, 8), (6, 4), (3, 3)])
def test_blocked_pass_matches_oracle_and_scalar_path(key, nx, ny, cutoff, beta, kw, R_total, R_batch):
    """K7b (mode | MODE_ORB4): whole 4x4 blocks per thread.  R_batch = 3 falls back to the scalar path."""
    w, inp, Ho, Hg = _both(key, nx, ny, cutoff, beta, **kw)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    M = 65
    ref = oracle.kpm_moments(Ho, a, b, M, R_total, 21, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, M, R_total, R_batch, 21, mode=gtb.MODE_ORB4, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12
    plain = gtb.kpm_moments(Hg, a, b, M, R_total, R_batch, 21, mode=0).cpu().numpy()
    assert np.abs(got - plain).max() <= 1e-13         # same vectors, another summation order
    # without the diagonal array as well
    Hn = gtb.Ell(Hg.n, Hg.width, Hg.cols, Hg.vals, None)
    Hon = oracle.Ell(Ho.n, Ho.width, Ho.cols, Ho.vals, None)
    ref = oracle.kpm_moments(Hon, a, b, 33, R_total, 22, mode=0, algo=0)
    got = gtb.kpm_moments(Hn, a, b, 33, R_total, R_batch, 22, mode=gtb.MODE_ORB4).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12


def test_blocked_exact_trace_against_eigvalsh():
    w, inp, Ho, Hg = _both("c2b", 5, 4, 2.65, 3.37)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    got = gtb.kpm_moments(Hg, a, b, 40, mode=1 | gtb.MODE_ORB4, R_batch=8).cpu().numpy()
    th = np.arccos((np.linalg.eigvalsh(Ho.to_dense()) - b) / a)
    assert np.abs(got - np.array([np.cos(k * th).mean() for k in range(40)])).max() <= 1e-12


def test_exact_trace_against_eigvalsh():
    w, inp, Ho, Hg = _both("c2b", 5, 4, 2.65, 3.37)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    M = 40
    got = gtb.kpm_moments(Hg, a, b, M, mode=1, R_batch=8).cpu().numpy()
    th = np.arccos((np.linalg.eigvalsh(Ho.to_dense()) - b) / a)
    exact = np.array([np.cos(k * th).mean() for k in range(M)])
    assert np.abs(got - exact).max() <= 1e-12


def test_vac_moments_with_per_orbital_positions():
    w, inp, Ho, Hg = _both("c2", 19, 11, 1.95, 2.0)
    pos4 = np.repeat(inp.pos, 4, axis=0)                    # X acts on the atom of each orbital
    vo = oracle.velocity_ell(Ho, pos4, inp.box, inp.pbc, 0)
    vg = gtb.velocity_ell(Hg, _dev(pos4), inp.box, inp.pbc, 0)
    assert np.abs(vg.cpu().numpy() - vo).max() <= 8 * 2.0**-52 * np.abs(vo).max()
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    dt = 0.1 / gtb.HBAR_EV_FS
    ref = oracle.vac_moments(Ho, vo, a, b, 24, 3, dt, R=2, seed=4, mode=0)
    got = gtb.vac_moments(Hg, vg, a, b, 24, 3, dt, 2, 2, 4, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-11 * ref[0, 0]
    # and with the blocked pass (propagation and bra-dot moments on 4x4 blocks)
    for R in (2, 4, 8):
        ref = oracle.vac_moments(Ho, vo, a, b, 17, 3, dt, R=R, seed=4, mode=0)
        got = gtb.vac_moments(Hg, vg, a, b, 17, 3, dt, R, R, 4, mode=gtb.MODE_ORB4, check=True).cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-11 * ref[0, 0]


def test_bad_species_and_shapes_are_reported():
    w = W.CONFIGS["c1"].scaled(6, 6)
    inp = W.make_inputs(w)
    nbr = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, 1.95, [0.0], [1.0],
                                with_diag=False)
    bad = inp.species.copy()
    bad[7] = 3
    with pytest.raises(gtb.GtbError):
        gtb.sk_hamiltonian(nbr, _dev(inp.pos), _dev(bad), inp.box, inp.pbc, [0.0], [0.0], SK1)
