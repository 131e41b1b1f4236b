"""Pins of the s,p,d Slater-Koster oracle (oracle/gtbo_spd.cpp) against things
other than itself: entries of the printed Slater-Koster table, the diatomic molecule by m-sectors, the
s,p oracle, rotational invariance and the paper's block symmetry.  P31-P35."""
import numpy as np
import pytest

import oracle
from paper_2509_06525_b200 import workloads as W

# ss_s, sp_s, pp_s, pp_p, sd_s, pd_s, pd_p, dd_s, dd_p, dd_d (eV), synthetic
V = np.array([-6.769, 5.580, 5.037, -3.033, -2.1, -1.7, 0.9, -1.3, 0.8, -0.15])
ES, EP, ED = -8.868, 0.0, 6.5
S, X, Y, Z, XY, YZ, ZX, X2Y2, Z2 = range(9)
ELL = np.array([0, 1, 1, 1, 2, 2, 2, 2, 2])


def _spd(pos, box, pbc, cutoff, sk=V, beta=0.0, species=None):
    species = np.zeros(len(pos), dtype=np.int32) if species is None else species
    nbr = oracle.build_hamiltonian(pos, species, box, pbc, cutoff, [0.0], [1.0], with_diag=False, method=0)
    return nbr, oracle.spd_hamiltonian(nbr, pos, species, box, pbc, [ES], [EP], [ED], sk, r0=1.42, beta=beta)


def _dimer_block(u):
    u = np.asarray(u, dtype=float)
    u = u / np.linalg.norm(u)
    pos = np.array([[5.0, 5.0, 5.0], 5.0 + 1.3 * u])
    nbr, H = _spd(pos, [30.0] * 3, [0, 0, 0], 2.0)
    return u, H.to_dense()[:9, 9:], H


# ---------------------------------------------------------------------------------- P31
@pytest.mark.parametrize("u", [(1, 2, -2), (0.3, -0.5, 0.81), (0, 0, 1), (1, 0, 0), (1, 1, 0)])
def test_entries_of_the_slater_koster_table(u):
    (l, m, n), E, _ = _dimer_block(u)
    ss, sp, pps, ppp, sd, pds, pdp, dds, ddp, ddd = V
    r3 = np.sqrt(3.0)
    want = {
        (S, XY): r3 * l * m * sd,
        (S, X2Y2): r3 / 2 * (l * l - m * m) * sd,
        (S, Z2): (n * n - (l * l + m * m) / 2) * sd,
        (X, XY): r3 * l * l * m * pds + m * (1 - 2 * l * l) * pdp,
        (Z, Z2): n * (n * n - (l * l + m * m) / 2) * pds + r3 * n * (l * l + m * m) * pdp,
        (XY, XY): 3 * l * l * m * m * dds + (l * l + m * m - 4 * l * l * m * m) * ddp + (n * n + l * l * m * m) * ddd,
        (Z2, Z2): (n * n - (l * l + m * m) / 2) ** 2 * dds + 3 * n * n * (l * l + m * m) * ddp
                  + 0.75 * (l * l + m * m) ** 2 * ddd,
        (S, S): ss, (S, X): l * sp, (X, S): -l * sp,
        (X, Y): l * m * (pps - ppp), (Z, Z): n * n * pps + (1 - n * n) * ppp,
    }
    for (a, b), val in want.items():
        assert E[a, b] == pytest.approx(val, abs=1e-14), (a, b)


# ---------------------------------------------------------------------------------- P32
@pytest.mark.parametrize("u", [(0, 0, 1), (1, 2, -2), (-3, 1, 0.5)])
def test_diatomic_molecule_by_m_sectors(u):
    """Two-centre integrals are diagonal in the bond frame: the 18 levels are those of the sigma sector
    (s, p_sigma, d_sigma on both atoms), twice the pi sector (p_pi, d_pi) and twice the delta sector."""
    _, _, H = _dimer_block(u)
    got = np.linalg.eigvalsh(H.to_dense())
    ss, sp, pps, ppp, sd, pds, pdp, dds, ddp, ddd = V
    def sector(onsite, T):
        D = np.diag(onsite)
        return np.linalg.eigvalsh(np.block([[D, T], [T.T, D]]))
    sig = sector([ES, EP, ED], np.array([[ss, sp, sd], [-sp, pps, pds], [sd, -pds, dds]]))
    pi = sector([EP, ED], np.array([[ppp, pdp], [-pdp, ddp]]))
    dl = sector([ED], np.array([[ddd]]))
    want = np.sort(np.concatenate([sig, pi, pi, dl, dl]))
    assert np.abs(got - want).max() <= 1e-13


# ---------------------------------------------------------------------------------- P33
def test_sp_sub_blocks_equal_the_sp_oracle():
    w = W.CONFIGS["c2"].scaled(5, 3)
    inp = W.make_inputs(w)
    nbr, H9 = _spd(inp.pos, inp.box, inp.pbc, 2.65, beta=3.37)
    H4 = oracle.sk_hamiltonian(nbr, inp.pos, np.zeros(nbr.n, dtype=np.int32), inp.box, inp.pbc, [ES], [EP],
                               V[:4], r0=1.42, beta=3.37)
    D9 = H9.to_dense().reshape(nbr.n, 9, nbr.n, 9)
    D4 = H4.to_dense().reshape(nbr.n, 4, nbr.n, 4)
    assert np.abs(D9[:, :4, :, :4] - D4).max() <= 1e-14      # two roundings apart: u u^T + e e^T vs 1 - u u^T


# ---------------------------------------------------------------------------------- P34
def test_rotation_invariance_symmetry_and_block_parity():
    w = W.CONFIGS["c2b"].scaled(4, 3)
    inp = W.make_inputs(w)
    free, box = [0, 0, 0], [200.0] * 3
    nbr, H = _spd(inp.pos + 50.0, box, free, 2.65, beta=2.0)
    D = H.to_dense()
    assert np.abs(D - D.T).max() <= 1e-14
    B = D.reshape(nbr.n, 9, nbr.n, 9)
    sign = (-1.0) ** (ELL[:, None] + ELL[None, :])
    assert np.abs(B - sign[None, :, None, :] * B.transpose(2, 1, 0, 3)).max() <= 1e-14
    e0 = np.linalg.eigvalsh(D)
    for seed in (1, 2):
        q, _ = np.linalg.qr(np.random.default_rng(seed).standard_normal((3, 3)))
        pos = (inp.pos - inp.pos.mean(0)) @ q.T + 100.0
        e1 = np.linalg.eigvalsh(_spd(pos, box, free, 2.65, beta=2.0)[1].to_dense())
        assert np.abs(e1 - e0).max() <= 1e-11


# ---------------------------------------------------------------------------------- P35
def test_layout_padding_and_onsite():
    w = W.CONFIGS["c2b"].scaled(5, 4)
    inp = W.make_inputs(w)
    nbr, H = _spd(inp.pos, inp.box, inp.pbc, 2.65, beta=3.37)
    assert H.n == 9 * nbr.n and H.width == 9 * nbr.width
    rows = np.arange(H.n)
    for k in range(nbr.width):
        j = np.repeat(nbr.cols[k], 9)
        pad = j == rows // 9
        for nu in range(9):
            c = H.cols[9 * k + nu]
            assert (c[~pad] == 9 * j[~pad] + nu).all() and (c[pad] == rows[pad]).all()
            assert (H.vals[9 * k + nu][pad] == 0).all()
    assert (H.diag.reshape(-1, 9) == np.array([ES, EP, EP, EP, ED, ED, ED, ED, ED])).all()


# ---------------------------------------------------------------------------------- P39
def _asym_table(seed=3):
    """[2][2][10], same-l integrals (ss, pp, dd) symmetric in the species pair, mixed-l ones
    (sp_sigma, sd_sigma, pd_sigma, pd_pi) different for (A, B) and (B, A) -- the normal heteronuclear case."""
    rng = np.random.default_rng(seed)
    t = rng.uniform(-3.0, 3.0, (2, 2, 10))
    for q in (0, 2, 3, 7, 8, 9):
        t[1, 0, q] = t[0, 1, q]
    return t


@pytest.mark.parametrize("u", [(0, 0, 1), (1, 2, -2), (-3, 1, 0.5)])
def test_heteronuclear_diatomic_with_a_species_asymmetric_table(u):
    """PAPER.md:88, H_ij^{l l'} = (-1)^{l+l'} H_ji^{l' l}: the (l_a > l_b) element of the (A, B) block is made
    of the (B, A) integral.  Closed form by m-sectors with orbitals of both atoms quantised along the bond
    A -> B: <l_A|H|l'_B> = V_{l l'}(AB) for l <= l', (-1)^{l+l'} V_{l' l}(BA) for l > l'.  A wrong species
    order in any mixed-l element changes the spectrum (the (A,B) and (B,A) entries differ by O(1))."""
    t = _asym_table()
    es, ep, ed = [-8.0, -5.5], [0.3, -1.1], [6.5, 4.0]
    u = np.asarray(u, dtype=float) / np.linalg.norm(u)
    pos = np.array([[5.0, 5.0, 5.0], 5.0 + 1.3 * u])
    species = np.array([0, 1], dtype=np.int32)
    nbr = oracle.build_hamiltonian(pos, species, [30.0] * 3, [0, 0, 0], 2.0, [0.0, 0.0], np.ones((2, 2)),
                                   with_diag=False, method=0)
    H = oracle.spd_hamiltonian(nbr, pos, species, [30.0] * 3, [0, 0, 0], es, ep, ed, t, r0=1.42).to_dense()
    assert np.abs(H - H.T).max() <= 1e-14
    ab, ba = t[0, 1], t[1, 0]
    def sector(on_a, on_b, T):
        return np.linalg.eigvalsh(np.block([[np.diag(on_a), T], [T.T, np.diag(on_b)]]))
    sig = sector([es[0], ep[0], ed[0]], [es[1], ep[1], ed[1]],
                 np.array([[ab[0], ab[1], ab[4]], [-ba[1], ab[2], ab[5]], [ba[4], -ba[5], ab[7]]]))
    pi = sector([ep[0], ed[0]], [ep[1], ed[1]], np.array([[ab[3], ab[6]], [-ba[6], ab[8]]]))
    dl = sector([ed[0]], [ed[1]], np.array([[ab[9]]]))
    want = np.sort(np.concatenate([sig, pi, pi, dl, dl]))
    assert np.abs(np.linalg.eigvalsh(H) - want).max() <= 1e-13


def test_asymmetric_table_keeps_h_symmetric_and_the_doubling_identities_valid():
    """On a two-species disordered lattice: H = H^T, and the direct and the doubling moments agree (the
    identities need a symmetric H)."""
    w = W.CONFIGS["c4"].scaled(6, 3, stripe=3)
    inp = W.make_inputs(w)
    species = (inp.species > 0).astype(np.int32)
    nbr = oracle.build_hamiltonian(inp.pos, species, inp.box, inp.pbc, 2.65, [0.0, 0.0], np.ones((2, 2)),
                                   with_diag=False)
    H = oracle.spd_hamiltonian(nbr, inp.pos, species, inp.box, inp.pbc, [-8.0, -5.5], [0.3, -1.1], [6.5, 4.0],
                               _asym_table(), r0=1.42, beta=1.5)
    D = H.to_dense()
    assert np.abs(D - D.T).max() <= 1e-13
    lo, hi = oracle.spectral_bounds(H)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    m0 = oracle.kpm_moments(H, a, b, 24, 2, 7, mode=0, algo=0)
    m1 = oracle.kpm_moments(H, a, b, 24, 2, 7, mode=0, algo=1)
    assert np.abs(m0 - m1).max() <= 1e-12


# ---------------------------------------------------------------------------------- P40
def test_sampled_atom_step_equals_the_step_on_the_assembled_matrix():
    """spd_step_atoms (H never materialised, vectors given sparsely; used at 10^8 atoms) against two
    separately pinned functions: spd_hamiltonian (P31-P35, P39) + kpm_step_rows (dense product pin), on a
    two-species disordered lattice, first and later steps, every atom; and random_phase_rows against
    random_phase_fill."""
    w = W.CONFIGS["c4"].scaled(6, 4, stripe=3)
    inp = W.make_inputs(w)
    species = (inp.species > 0).astype(np.int32)
    shift = 0.01 * np.arange(len(species), dtype=float)
    es, ep, ed, sk = [-8.0, -5.5], [0.3, -1.1], [6.5, 4.0], _asym_table()
    nbr = oracle.build_hamiltonian(inp.pos, species, inp.box, inp.pbc, 2.65, [0.0, 0.0], np.ones((2, 2)),
                                   with_diag=False)
    H = oracle.spd_hamiltonian(nbr, inp.pos, species, inp.box, inp.pbc, es, ep, ed, sk, r0=1.42, beta=1.5,
                               onsite_shift=shift)
    n, K, R = nbr.n, nbr.width, 2
    a, b = 31.0, -0.7
    phi0 = oracle.random_phase_fill(5, 0, R, 9 * n)
    rows = np.array([0, 7, 9 * n - 1, 40])
    assert np.array_equal(oracle.random_phase_rows(5, 0, R, rows), phi0[rows])
    all_rows = np.arange(9 * n)
    phi1 = oracle.kpm_step_rows(H, a, b, True, None, phi0, all_rows)
    phi2 = oracle.kpm_step_rows(H, a, b, False, phi0, phi1, all_rows)
    atoms = np.arange(n)
    def sparse(x):
        xo = x.reshape(n, 9, R, 2)
        return xo[atoms], xo[nbr.cols[:, atoms].T]          # [q][9][R][2], [q][K][9][R][2]
    o0, n0 = sparse(phi0)
    args = (nbr, inp.pos, species, inp.box, inp.pbc, es, ep, ed, sk, a, b)
    got1 = oracle.spd_step_atoms(*args, True, atoms, o0, n0, r0=1.42, beta=1.5, onsite_shift=shift)
    assert np.abs(got1.reshape(-1, R, 2) - phi1).max() <= 1e-15
    o1, n1 = sparse(phi1)
    got2 = oracle.spd_step_atoms(*args, False, atoms, o1, n1, prev=o0, r0=1.42, beta=1.5, onsite_shift=shift)
    assert np.abs(got2.reshape(-1, R, 2) - phi2).max() <= 1e-15
