"""GPU parity of the block and bond (matrix-free) forms of the s,p,d Hamiltonian (csrc/spd9.cu,
GTB_MODE_BLOCK9 / GTB_MODE_BOND9; Fig. 4a) against the oracle's scalar matrix
(oracle.spd_hamiltonian, pins P31-P35, P39) and, at 10^8 atoms x 9 orbitals, against the oracle's
sampled-atom step (oracle.spd_step_atoms, pin P40)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _asym_table(ns, seed=3):
    rng = np.random.default_rng(seed)
    t = rng.uniform(-3.0, 3.0, (ns, ns, 10))
    for q in (0, 2, 3, 7, 8, 9):                       # same-l integrals: symmetric in the pair
        t[..., q] = 0.5 * (t[..., q] + t[..., q].T)
    return t


CASES = [("c2b", 9, 7, {}, 2.65, 3.37, False), ("c4", 12, 5, {"stripe": 3}, 1.95, 0.0, True),
         ("c4", 8, 6, {"stripe": 2}, 2.65, 1.5, True), ("c5", 11, 9, {}, 3.0, 0.0, False)]


def _setup(key, nx, ny, kw, cutoff, beta, asym):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    ns = len(w.onsite)
    sk = _asym_table(ns) if asym else W.spd_table(ns)
    es, ep, ed = W.SK_ONSITE_S[:ns], W.SK_ONSITE_P[:ns], W.SK_ONSITE_D[:ns]
    ones = np.ones((ns, ns))
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                     with_diag=False)
    Ho = oracle.spd_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, es, ep, ed, sk, r0=1.42,
                                beta=beta, onsite_shift=inp.onsite_shift)
    nbr_g = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                  with_diag=False)
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    Hm = gtb.spd_bonds(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, es, ep, ed, sk, r0=1.42,
                       beta=beta, onsite_shift=shift)
    return w, inp, nbr_o, Ho, Hm


@pytest.mark.parametrize("key,nx,ny,kw,cutoff,beta,asym", CASES)
def test_blocks_onsite_and_bounds_match_the_oracle_matrix(key, nx, ny, kw, cutoff, beta, asym):
    w, inp, nbr_o, Ho, Hm = _setup(key, nx, ny, kw, cutoff, beta, asym)
    n, K = nbr_o.n, nbr_o.width
    Hb = gtb.spd_blocks(Hm)
    assert (Hb.cols.cpu().numpy() == nbr_o.cols).all()
    got = Hb.vals.cpu().numpy().reshape(K, 9, 9, n)                      # [k][nu][mu][i]
    want = Ho.vals.reshape(K, 9, n, 9).transpose(0, 1, 3, 2)             # scalar slot 9k+nu, row 9i+mu
    assert np.abs(got - want).max() <= 1e-13 * max(np.abs(want).max(), 1.0)
    assert np.abs(Hb.diag.cpu().numpy() - Ho.diag.reshape(n, 9).T).max() <= 1e-15
    lo, hi = oracle.spectral_bounds(Ho)
    for H, mode in ((Hb, gtb.MODE_BLOCK9), (Hm, gtb.MODE_BOND9)):
        b = gtb.spd_bounds(H, mode).cpu().numpy()
        assert b[0] == pytest.approx(lo, rel=1e-12) and b[1] == pytest.approx(hi, rel=1e-12)


@pytest.mark.parametrize("key,nx,ny,kw,cutoff,beta,asym", CASES)
@pytest.mark.parametrize("R", [2, 4, 8])
def test_block_and_bond_passes_match_oracle_rows_and_moments(key, nx, ny, kw, cutoff, beta, asym, R):
    w, inp, nbr_o, Ho, Hm = _setup(key, nx, ny, kw, cutoff, beta, asym)
    Hb = gtb.spd_blocks(Hm)
    N = Ho.n
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    phi0 = oracle.random_phase_fill(11, 0, R, N)
    rows = np.arange(N)
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, rows)
    phi2 = oracle.kpm_step_rows(Ho, a, b, False, phi0, phi1, rows)
    M = 33
    ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
    for H, mode in ((Hb, gtb.MODE_BLOCK9), (Hm, gtb.MODE_BOND9)):
        g0 = _dev(phi0)
        g1 = torch.empty_like(g0)
        s = gtb.kpm_step(H, a, b, True, g0, g1, mode=mode).cpu().numpy()
        assert np.abs(g1.cpu().numpy() - phi1).max() <= 1e-13
        assert s[0] == pytest.approx(N * R, rel=1e-13)
        s = gtb.kpm_step(H, a, b, False, g1, g0, mode=mode).cpu().numpy()         # g0 <- phi_2
        assert np.abs(g0.cpu().numpy() - phi2).max() <= 1e-13
        assert s[0] == pytest.approx((phi1 * phi1).sum(), rel=1e-13)
        assert s[1] == pytest.approx((phi2 * phi1).sum(), rel=1e-11, abs=1e-9)
        got = gtb.kpm_moments(H, a, b, M, R, R, 5, mode=mode, check=True).cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-9            # north_star
        assert np.abs(got - ref).max() <= 1e-12
    exact = gtb.kpm_moments(Hm, a, b, 12, mode=1 | gtb.MODE_BOND9, R_batch=8).cpu().numpy()
    ev = np.linalg.eigvalsh(Ho.to_dense()) if N <= 4000 else None
    if ev is not None:
        x = (ev - b) / a
        want = np.array([np.cos(k * np.arccos(x)).mean() for k in range(12)])
        assert np.abs(exact - want).max() <= 1e-12


def test_rejected_inputs():
    w, inp, nbr_o, Ho, Hm = _setup("c4", 8, 6, {"stripe": 2}, 1.95, 0.0, False)
    with pytest.raises(gtb.GtbError):                       # R_batch must be 2, 4 or 8
        gtb.kpm_moments(Hm, 30.0, 0.0, 8, 3, 3, 5, mode=gtb.MODE_BOND9)
    with pytest.raises(gtb.GtbError):                       # one representation at a time
        gtb.kpm_moments(Hm, 30.0, 0.0, 8, 2, 2, 5, mode=gtb.MODE_BOND9 | gtb.MODE_BLOCK9)
    ns = 3
    bad = W.spd_table(ns).copy()
    bad[0, 1, 2] += 0.1                                     # pp_sigma(C, B) != pp_sigma(B, C): no symmetric H
    nbr_g = gtb.Ell(Hm.n, Hm.width, Hm.cols, Hm.vals, None)
    with pytest.raises(gtb.GtbError):
        gtb.spd_bonds(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, W.SK_ONSITE_S[:ns],
                      W.SK_ONSITE_P[:ns], W.SK_ONSITE_D[:ns], bad, r0=1.42)


def test_hundred_million_atoms_times_nine_orbitals_sampled_against_the_oracle():
    """The paper's own headline workload (Fig. 4a: 10^8 graphene atoms, s,p,d orbitals,
    third-nearest-neighbour cutoff), matrix-free on one GPU: neighbour lists in full (bit-exact), the
    first pass and one recursion pass on sampled atoms (both ends of the index range, across the periodic
    seam, random atoms) against oracle.spd_step_atoms, and the properties of the moments that hold at
    any size."""
    w = W.CONFIGS["c5"]
    cutoff = 3.0                                            # shells at 1.42, 2.46, 2.84 A: 3 + 6 + 3 = 12
    inp = W.make_inputs(w)
    n, R = w.n_atoms, 2
    es, ep, ed, sk = W.SK_ONSITE_S[:1], W.SK_ONSITE_P[:1], W.SK_ONSITE_D[:1], W.spd_table(1)
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0], [1.0],
                                     with_diag=False)
    d_pos, d_spec = _dev(inp.pos), _dev(inp.species)
    nbr_g = gtb.build_hamiltonian(d_pos, d_spec, inp.box, inp.pbc, cutoff, [0.0], [1.0], with_diag=False)
    assert nbr_g.width == 12 == nbr_o.width
    for k in range(12):
        assert (nbr_g.cols[k].cpu().numpy() == nbr_o.cols[k]).all()
    Hm = gtb.spd_bonds(nbr_g, d_pos, d_spec, inp.box, inp.pbc, es, ep, ed, sk, r0=1.42)
    del nbr_g                                               # Hm shares the columns; the unit hoppings go
    torch.cuda.empty_cache()
    lo, hi = gtb.spd_bounds(Hm, gtb.MODE_BOND9).tolist()
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    rng = np.random.default_rng(7)
    edge = 4 * w.nx
    atoms = np.unique(np.concatenate([np.arange(0, 64), np.arange(edge - 32, edge + 32),
                                      np.arange(n - 64, n), rng.integers(0, n, 1500)])).astype(np.int64)
    nb = nbr_o.cols[:, atoms].T                                           # [q][K]
    orb = lambda at: (9 * at[..., None] + np.arange(9)).astype(np.int64)   # orbital rows of atoms
    own_rows, nbr_rows = orb(atoms), orb(nb)
    seed = w.seed
    phi0_own = oracle.random_phase_rows(seed, 0, R, own_rows.ravel()).reshape(len(atoms), 9, R, 2)
    phi0_nbr = oracle.random_phase_rows(seed, 0, R, nbr_rows.ravel()).reshape(len(atoms), 12, 9, R, 2)
    g0 = gtb.random_phase_fill(seed, 0, R, 9 * n)
    t_own = torch.as_tensor(own_rows.ravel()).cuda()
    assert np.abs(g0[t_own].cpu().numpy().reshape(phi0_own.shape) - phi0_own).max() <= 4 * 2.0**-52
    g1 = torch.empty_like(g0)
    ws = gtb.workspace(gtb.kpm_workspace_bytes(9 * n, 2, R))
    s = gtb.kpm_step(Hm, a, b, True, g0, g1, ws=ws, mode=gtb.MODE_BOND9).cpu().numpy()
    assert s[0] == pytest.approx(9.0 * n * R, rel=1e-13)
    args = (nbr_o, inp.pos, inp.species, inp.box, inp.pbc, es, ep, ed, sk, a, b)
    # the oracle steps from the DEVICE's phi_0 rows, so that one libm's sincos does not enter
    t_nbr = torch.as_tensor(nbr_rows.ravel()).cuda()
    x_own = g0[t_own].cpu().numpy().reshape(phi0_own.shape)
    x_nbr = g0[t_nbr].cpu().numpy().reshape(phi0_nbr.shape)
    want1 = oracle.spd_step_atoms(*args, True, atoms, x_own, x_nbr, r0=1.42)
    got1 = g1[t_own].cpu().numpy().reshape(want1.shape)
    assert np.abs(got1 - want1).max() <= 1e-13
    y_own = got1
    y_nbr = g1[t_nbr].cpu().numpy().reshape(phi0_nbr.shape)
    want2 = oracle.spd_step_atoms(*args, False, atoms, y_own, y_nbr, prev=x_own, r0=1.42)
    s = gtb.kpm_step(Hm, a, b, False, g1, g0, ws=ws, mode=gtb.MODE_BOND9).cpu().numpy()   # g0 <- phi_2
    assert np.abs(g0[t_own].cpu().numpy().reshape(want2.shape) - want2).max() <= 1e-13
    assert s[0] > 0.0 and np.isfinite(s).all()
    del g0, g1, ws
    torch.cuda.empty_cache()
    # moments at full size: mu_0 = 1 exactly, mu_1 = Tr H~ / N within the stochastic bound, |mu_n| <= 1
    M = 8
    mu = gtb.kpm_moments(Hm, a, b, M, R, R, seed, mode=gtb.MODE_BOND9, check=True).cpu().numpy()
    tr1 = ((es[0] + 3 * ep[0] + 5 * ed[0]) / 9.0 - b) / a
    bound = 5.0 / np.sqrt(9.0 * n * R)
    assert mu[0] == pytest.approx(1.0, abs=1e-13) and np.abs(mu).max() <= 1.0 + 1e-13
    assert abs(mu[1] - tr1) <= bound
