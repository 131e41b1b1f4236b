"""Pins of the Slater-Koster s,p oracle (oracle/gtbo_sk.cpp) against things
other than itself: the textbook diatomic molecule in closed form, rotational invariance, the paper's
block symmetry, and reductions to the single-orbital path.  P20-P25."""
import numpy as np
import pytest

import oracle
from paper_2509_06525_b200 import workloads as W

# graphene-like s,p parameters (eV): ss_sigma, sp_sigma, pp_sigma, pp_pi; onsite s, p
SK = np.array([-6.769, 5.580, 5.037, -3.033])
ES, EP = -8.868, 0.0


def _nbr(pos, species, box, pbc, cutoff):
    return oracle.build_hamiltonian(pos, species, box, pbc, cutoff, [0.0], [1.0], with_diag=False,
                                    method=0)


def _sk(pos, box, pbc, cutoff, sk=SK, es=ES, ep=EP, beta=0.0, r0=1.42):
    species = np.zeros(len(pos), dtype=np.int32)
    nbr = _nbr(pos, species, box, pbc, cutoff)
    return oracle.sk_hamiltonian(nbr, pos, species, box, pbc, [es], [ep], sk, r0=r0, beta=beta)


def _rotation(seed):
    q, _ = np.linalg.qr(np.random.default_rng(seed).standard_normal((3, 3)))
    return q * np.sign(np.linalg.det(q))


# ---------------------------------------------------------------------------------- P20
@pytest.mark.parametrize("direction", [(0, 0, 1), (1, 0, 0), (0, 1, 0), (1, 2, -2), (-3, 1, 0.5)])
def test_diatomic_molecule_closed_form(direction):
    """Two atoms r apart: pi levels eps_p +- V_pp_pi (twice each); sigma levels = the roots of
    [[eps_s + V_ss, -V_sp], [-V_sp, eps_p - V_pp_sigma]] and [[eps_s - V_ss, V_sp], [V_sp, eps_p + V_pp_sigma]]
    (the textbook homonuclear diatomic), whatever the bond direction."""
    u = np.array(direction, dtype=float)
    u /= np.linalg.norm(u)
    pos = np.array([[5.0, 5.0, 5.0], [5.0, 5.0, 5.0] + 1.3 * u])
    H = _sk(pos, [20.0, 20.0, 20.0], [0, 0, 0], 2.0)
    got = np.linalg.eigvalsh(H.to_dense())
    vss, vsp, vpps, vppp = SK
    even = np.linalg.eigvalsh(np.array([[ES + vss, -vsp], [-vsp, EP - vpps]]))
    odd = np.linalg.eigvalsh(np.array([[ES - vss, vsp], [vsp, EP + vpps]]))
    want = np.sort(np.concatenate([even, odd, [EP + vppp] * 2, [EP - vppp] * 2]))
    assert np.abs(got - want).max() <= 1e-13


# ---------------------------------------------------------------------------------- P21
def test_spectrum_is_invariant_under_rigid_rotation():
    w = W.CONFIGS["c2b"].scaled(4, 3)
    inp = W.make_inputs(w)
    free = [0, 0, 0]
    box = [100.0, 100.0, 100.0]
    e0 = np.linalg.eigvalsh(_sk(inp.pos, box, free, 2.65, beta=2.0).to_dense())
    for seed in (1, 2):
        Rm = _rotation(seed)
        pos = (inp.pos - inp.pos.mean(0)) @ Rm.T + 50.0
        e1 = np.linalg.eigvalsh(_sk(pos, box, free, 2.65, beta=2.0).to_dense())
        assert np.abs(e1 - e0).max() <= 1e-12


# ---------------------------------------------------------------------------------- P22
def test_block_symmetry_of_the_paper():
    """H_ij^{l l'} = (-1)^{l + l'} H_ji^{l' l}; with real orbitals H is symmetric and the
    s-p blocks are odd under exchange of the two atoms."""
    w = W.CONFIGS["c2"].scaled(5, 3)
    inp = W.make_inputs(w)
    H = _sk(inp.pos, inp.box, inp.pbc, 2.65, beta=3.37)
    D = H.to_dense().reshape(H.n // 4, 4, H.n // 4, 4)
    assert np.abs(H.to_dense() - H.to_dense().T).max() <= 1e-15
    ell = np.array([0, 1, 1, 1])
    sign = (-1.0) ** (ell[:, None] + ell[None, :])
    # block (i, j) with orbital indices (mu, nu) against the "same bond seen from j": (nu, mu) swapped
    assert np.abs(D - sign[None, :, None, :] * D.transpose(2, 1, 0, 3)).max() <= 1e-15


# ---------------------------------------------------------------------------------- P23
def test_s_only_limit_is_the_single_orbital_hamiltonian():
    w = W.CONFIGS["c2b"].scaled(5, 4)
    inp = W.make_inputs(w)
    species = np.zeros(len(inp.pos), dtype=np.int32)
    H1 = oracle.build_hamiltonian(inp.pos, species, inp.box, inp.pbc, 2.65, [0.7], [-2.7], r0=1.42,
                                  beta=3.37, method=0)
    H4 = _sk(inp.pos, inp.box, inp.pbc, 2.65, sk=np.array([-2.7, 0.0, 0.0, 0.0]), es=0.7, ep=9.0,
             beta=3.37)
    D = H4.to_dense().reshape(H1.n, 4, H1.n, 4)
    assert np.abs(D[:, 0, :, 0] - H1.to_dense()).max() <= 1e-15
    assert np.abs(D[:, 1:, :, 1:] - 9.0 * np.eye(3 * H1.n).reshape(H1.n, 3, H1.n, 3)).max() == 0.0


# ---------------------------------------------------------------------------------- P24
def test_flat_graphene_decouples_into_sigma_and_pi():
    """In a flat sheet n = 0 for every bond: p_z couples only to p_z with V_pp_pi, i.e. the p_z block
    is the single-orbital nearest-neighbour model with t = V_pp_pi (config 1's Hamiltonian)."""
    w = W.CONFIGS["c1"].scaled(6, 5)
    inp = W.make_inputs(w)
    H1 = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, 1.95, [EP], [SK[3]],
                                  method=0)
    H4 = _sk(inp.pos, inp.box, inp.pbc, 1.95)
    D = H4.to_dense().reshape(H1.n, 4, H1.n, 4)
    assert np.abs(D[:, 3, :, 3] - H1.to_dense()).max() <= 1e-15
    assert np.abs(D[:, :3, :, 3]).max() == 0.0 and np.abs(D[:, 3, :, :3]).max() == 0.0
    # and the moments add up: Tr T_n(H~) over 4N orbitals = sigma part + pi part
    a, b = 25.0, -6.0
    mu4 = oracle.kpm_moments(H4, a, b, 24, 1, 0, mode=1)
    mu_pi = oracle.kpm_moments(H1, a, b, 24, 1, 0, mode=1)
    E = np.linalg.eigvalsh(D[:, :3, :, :3].reshape(3 * H1.n, 3 * H1.n))
    th = np.arccos((E - b) / a)
    mu_sigma = np.array([np.cos(k * th).mean() for k in range(24)])
    assert np.abs(mu4 - (3 * mu_sigma + mu_pi) / 4).max() <= 1e-12


# ---------------------------------------------------------------------------------- P25
def test_layout_padding_and_onsite():
    w = W.CONFIGS["c2b"].scaled(5, 4)          # disordered: neighbour counts vary, rows are padded
    inp = W.make_inputs(w)
    species = np.zeros(len(inp.pos), dtype=np.int32)
    nbr = _nbr(inp.pos, species, inp.box, inp.pbc, 2.65)
    shift = np.linspace(-0.1, 0.1, nbr.n)
    H = oracle.sk_hamiltonian(nbr, inp.pos, species, inp.box, inp.pbc, [ES], [EP], SK, r0=1.42,
                              beta=3.37, onsite_shift=shift)
    assert H.n == 4 * nbr.n and H.width == 4 * nbr.width
    rows = np.arange(H.n)
    for k in range(nbr.width):
        for nu in range(4):
            j = np.repeat(nbr.cols[k], 4)
            pad = j == rows // 4
            c = H.cols[4 * k + nu]
            assert (c[~pad] == 4 * j[~pad] + nu).all() and (c[pad] == rows[pad]).all()
            assert (H.vals[4 * k + nu][pad] == 0).all()
    assert np.allclose(H.diag.reshape(-1, 4), np.stack([ES + shift, EP + shift, EP + shift, EP + shift], 1),
                       rtol=0, atol=1e-15)


# ---------------------------------------------------------------------------------- P38
@pytest.mark.parametrize("direction", [(0, 0, 1), (1, 2, -2), (-3, 1, 0.5)])
def test_heteronuclear_diatomic_with_a_species_asymmetric_table(direction):
    """H_ij^{p,s} = -H_ji^{s,p}, and H_ji^{s,p} carries the integral of (s on j, p on i), i.e.
    the table entry of the species pair (s_j, s_i).  With V_sp(A s, B p) != V_sp(B s, A p) the sigma sector
    in the basis (s_A, p_sigma_A, s_B, p_sigma_B), p_sigma pointing from A to B, is
    [[es_A, 0, V_ss, V_sp(AB)], [0, ep_A, -V_sp(BA), V_pp_sigma], [., ., es_B, 0], [., ., 0, ep_B]]."""
    sk = np.array([[[0.0] * 4, [-5.1, 4.2, 3.9, -2.2]], [[-5.1, 6.3, 3.9, -2.2], [0.0] * 4]])
    es, ep = [-8.0, -5.5], [0.3, -1.1]
    u = np.array(direction, dtype=float)
    u /= np.linalg.norm(u)
    pos = np.array([[5.0, 5.0, 5.0], [5.0, 5.0, 5.0] + 1.3 * u])
    species = np.array([0, 1], dtype=np.int32)
    nbr = oracle.build_hamiltonian(pos, species, [20.0] * 3, [0, 0, 0], 2.0, [0.0, 0.0], np.ones((2, 2)),
                                   with_diag=False, method=0)
    H = oracle.sk_hamiltonian(nbr, pos, species, [20.0] * 3, [0, 0, 0], es, ep, sk, r0=1.42).to_dense()
    assert np.abs(H - H.T).max() <= 1e-14
    vss, vsp_ab, vpps, vppp = sk[0, 1]
    vsp_ba = sk[1, 0, 1]
    sig = np.linalg.eigvalsh(np.array([[es[0], 0.0, vss, vsp_ab], [0.0, ep[0], -vsp_ba, vpps],
                                       [vss, -vsp_ba, es[1], 0.0], [vsp_ab, vpps, 0.0, ep[1]]]))
    pi = np.linalg.eigvalsh(np.array([[ep[0], vppp], [vppp, ep[1]]]))
    want = np.sort(np.concatenate([sig, pi, pi]))
    assert np.abs(np.linalg.eigvalsh(H) - want).max() <= 1e-13
