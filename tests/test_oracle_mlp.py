"""Pins of the descriptor + MLP Hamiltonian oracle (oracle/gtbo_mlp.cpp; Eq. 2) against
things other than itself: numpy's Chebyshev routines, closed forms on the pristine lattice, a hand-made
weight set that collapses the networks to a polynomial in r, a numpy forward pass, and invariants. P26-P30."""
import numpy as np
import pytest
from numpy.polynomial import chebyshev as cheb

import oracle
from paper_2509_06525_b200 import workloads as W

DIMS = W.MLP_DIMS
NS, F, NB, HD = DIMS
RC = 2.0


def _nbr(w, inp, cutoff):
    ns = len(w.onsite)
    return oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns,
                                    np.ones((ns, ns)), with_diag=False, method=0)


def _unpack(blob):
    c = blob[:NS * NS * F * NB].reshape(NS, NS, F, NB)
    off = NS * NS * F * NB
    def take(shape):
        nonlocal off
        size = int(np.prod(shape))
        out = blob[off:off + size].reshape(shape)
        off += size
        return out
    env = (take((HD, F)), take((HD,)), take((F, HD)), take((F,)))
    hop = (take((HD, F)), take((HD,)), take((1, HD)), take((1,)))
    ons = [(take((HD, F)), take((HD,)), take((1, HD)), take((1,))) for _ in range(NS)]
    assert off == blob.size
    return c, env, hop, ons


def _np_mlp(p, x):
    W1, b1, W2, b2 = p
    z = W1 @ x + b1
    return W2 @ (z / (1.0 + np.exp(-z))) + b2


# ---------------------------------------------------------------------------------- P26
@pytest.mark.parametrize("r", [0.0, 0.31, 1.0, 1.42, RC * (1 - 1 / np.sqrt(2)), 1.99, RC, 2.5])
def test_descriptor_against_numpy_chebyshev(r):
    blob = W.mlp_weights()
    c = _unpack(blob)[0]
    got = oracle.mlp_descriptor(DIMS, RC, blob, 1, 2, r)
    x = 2 * (r / RC - 1) ** 2 - 1
    fc = 0.5 * (1 + np.cos(np.pi * r / RC)) if r < RC else 0.0
    fk = np.array([0.5 * (cheb.chebval(x, [0] * k + [1]) + 1) * fc for k in range(NB)])
    assert np.abs(got - c[1, 2] @ fk).max() <= 1e-14
    if r == 0.0:                                   # x = 1: every T_k = 1, f_c = 1, so f_k = 1
        assert np.abs(got - c[1, 2].sum(1)).max() <= 1e-14
    if r >= RC:
        assert (got == 0).all()
    assert np.abs(got - oracle.mlp_descriptor(DIMS, RC, blob, 2, 1, r)).max() == 0.0   # c symmetric


# ---------------------------------------------------------------------------------- P27
def test_pristine_lattice_closed_form():
    """Every atom of the pristine sheet has three neighbours at a_cc: v_i = 3 C(a_cc), all hoppings equal
    MLP_lambda(C(a_cc) * MLP_e(6 C(a_cc))), all onsite energies equal."""
    w = W.CONFIGS["c1"].scaled(6, 5)
    inp = W.make_inputs(w)
    blob = W.mlp_weights()
    c, env, hop, ons = _unpack(blob)
    H, v = oracle.mlp_hamiltonian(_nbr(w, inp, 1.95), inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC,
                                  blob, return_v=True)
    C0 = oracle.mlp_descriptor(DIMS, RC, blob, 0, 0, 1.42)
    assert np.abs(v - 3 * C0).max() <= 1e-13
    t = _np_mlp(hop, C0 * _np_mlp(env, 6 * C0))[0]
    assert np.abs(H.vals - t).max() <= 1e-12 and abs(t) > 1e-3
    assert np.abs(H.diag - _np_mlp(ons[0], 3 * C0)[0]).max() <= 1e-12


# ---------------------------------------------------------------------------------- P28
def test_collapsed_networks_give_a_polynomial_hopping():
    """MLP_e = constant 1 (zero weights, unit output bias) and MLP_lambda linearised (tiny first-layer
    weights: silu(z) = z/2 + O(z^2)) turn t_ij into sum_n w_n C_n(r_ij): a closed form in r alone."""
    w = W.CONFIGS["c2b"].scaled(5, 4)
    inp = W.make_inputs(w)
    rng = np.random.default_rng(0)
    c = rng.normal(size=(NS, NS, F, NB))
    c = 0.5 * (c + c.transpose(1, 0, 2, 3))
    eps = 1e-6
    env = (np.zeros((HD, F)), np.zeros(HD), np.zeros((F, HD)), np.ones(F))
    W1 = np.zeros((HD, F))
    W1[:F, :F] = eps * np.eye(F)
    wn = rng.normal(size=F)
    W2 = np.zeros((1, HD))
    W2[0, :F] = 2.0 * wn / eps
    hop = (W1, np.zeros(HD), W2, np.zeros(1))
    ons = [(np.zeros((HD, F)), np.zeros(HD), np.zeros((1, HD)), np.array([0.25 * (s + 1)])) for s in range(NS)]
    blob = W.mlp_pack(c, env, hop, ons)
    nbr = _nbr(w, inp, 1.95)
    H = oracle.mlp_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC, blob)
    i = np.arange(nbr.n)[None, :].repeat(nbr.width, 0)
    d = inp.pos[nbr.cols] - inp.pos[i]
    d -= inp.box * np.rint(d / inp.box) * inp.pbc
    r = np.linalg.norm(d, axis=-1)
    x = 2 * (r / RC - 1) ** 2 - 1
    fk = np.stack([0.5 * (cheb.chebval(x, [0] * k + [1]) + 1) for k in range(NB)], -1)
    fk *= (0.5 * (1 + np.cos(np.pi * r / RC)))[..., None]
    want = np.einsum("n,nk,srk->sr", wn, c[0, 0], fk)
    want[nbr.cols == i] = 0.0
    assert np.abs(H.vals - want).max() <= 1e-5 * np.abs(want).max()      # O(eps) linearisation error
    assert np.abs(H.diag - 0.25).max() == 0.0


# ---------------------------------------------------------------------------------- P29
def test_full_forward_pass_against_numpy_on_a_disordered_heterostructure():
    w = W.CONFIGS["c4"].scaled(8, 3, stripe=2)
    inp = W.make_inputs(w)
    blob = W.mlp_weights()
    c, env, hop, ons = _unpack(blob)
    nbr = _nbr(w, inp, 1.95)
    H, v = oracle.mlp_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC, blob, return_v=True)
    n = nbr.n
    def C(i, j):
        d = inp.pos[j] - inp.pos[i]
        d -= inp.box * np.rint(d / inp.box) * inp.pbc
        return oracle.mlp_descriptor(DIMS, RC, blob, int(inp.species[i]), int(inp.species[j]),
                                     float(np.linalg.norm(d)))
    vv = np.zeros((n, F))
    for i in range(n):
        for k in range(nbr.width):
            j = nbr.cols[k, i]
            if j != i:
                vv[i] += C(i, j)
    assert np.abs(v - vv).max() <= 1e-13
    for i in range(0, n, 7):
        for k in range(nbr.width):
            j = nbr.cols[k, i]
            t = 0.0 if j == i else _np_mlp(hop, C(i, j) * _np_mlp(env, vv[i] + vv[j]))[0]
            assert abs(H.vals[k, i] - t) <= 1e-12
        assert abs(H.diag[i] - _np_mlp(ons[inp.species[i]], vv[i])[0]) <= 1e-12


# ---------------------------------------------------------------------------------- P30
def test_symmetry_and_rigid_motion_invariance():
    w = W.CONFIGS["c2b"].scaled(5, 4)
    inp = W.make_inputs(w)
    blob = W.mlp_weights()
    free, box = [0, 0, 0], [200.0, 200.0, 200.0]
    def spectrum(pos):
        nbr = oracle.build_hamiltonian(pos, inp.species, box, free, 1.95, [0.0], [1.0], with_diag=False,
                                       method=0)
        H = oracle.mlp_hamiltonian(nbr, pos, inp.species, box, free, DIMS, RC, blob)
        D = H.to_dense()
        assert np.abs(D - D.T).max() <= 1e-14              # t_ij = t_ji (PAPER.md:88 for l = l')
        return np.linalg.eigvalsh(D)
    e0 = spectrum(inp.pos + 50.0)
    q, _ = np.linalg.qr(np.random.default_rng(3).standard_normal((3, 3)))
    e1 = spectrum((inp.pos - inp.pos.mean(0)) @ q.T + 100.0)
    assert np.abs(e1 - e0).max() <= 1e-11


# ---------------------------------------------------------------------------------- P36
def _blob_sk(c, env, hop4, ons2):
    return W.mlp_pack(c, env, hop4, ons2)


def test_mlp_sk_with_constant_networks_is_the_slater_koster_oracle():
    """MLP_lambda with zero weights and the four integrals as output bias, onsite MLPs with (eps_s, eps_p)
    as bias: the result must be gtbo_sk_hamiltonian's with those constants (beta = 0)."""
    w = W.CONFIGS["c4"].scaled(8, 3, stripe=2)
    inp = W.make_inputs(w)
    ns = 3
    nbr = _nbr(w, inp, 1.95)
    V = np.array([-6.769, 5.580, 5.037, -3.033])
    es, ep = [-8.9, -6.0, -11.0], [0.0, 2.3, -2.3]
    c = np.random.default_rng(0).normal(size=(NS, NS, F, NB))
    c = 0.5 * (c + c.transpose(1, 0, 2, 3))
    env = (np.zeros((HD, F)), np.zeros(HD), np.zeros((F, HD)), np.ones(F))
    hop4 = (np.zeros((HD, F)), np.zeros(HD), np.zeros((4, HD)), V)
    ons2 = [(np.zeros((HD, F)), np.zeros(HD), np.zeros((2, HD)), np.array([es[s], ep[s]])) for s in range(NS)]
    H = oracle.mlp_sk_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC,
                                  _blob_sk(c, env, hop4, ons2))
    table = np.broadcast_to(V, (ns, ns, 4))
    Hs = oracle.sk_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, es, ep, table, beta=0.0)
    assert (H.cols == Hs.cols).all()
    assert np.abs(H.vals - Hs.vals).max() <= 1e-15 and np.abs(H.diag - Hs.diag).max() == 0.0


def test_mlp_sk_parameters_are_the_mlp_outputs_and_the_matrix_is_symmetric():
    w = W.CONFIGS["c2b"].scaled(5, 4)
    inp = W.make_inputs(w)
    blob = W.mlp_weights(DIMS, 11, hop_out=4, onsite_out=2)
    nbr = _nbr(w, inp, 1.95)
    H = oracle.mlp_sk_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC, blob)
    D = H.to_dense()
    assert np.abs(D - D.T).max() <= 1e-14
    # the s-s entry of every block is MLP_lambda's first output: redo it in numpy for a few pairs
    c = blob[:NS * NS * F * NB].reshape(NS, NS, F, NB)
    off = NS * NS * F * NB
    def take(shape):
        nonlocal off
        size = int(np.prod(shape))
        out = blob[off:off + size].reshape(shape)
        off += size
        return out
    envp = (take((HD, F)), take((HD,)), take((F, HD)), take((F,)))
    hopp = (take((HD, F)), take((HD,)), take((4, HD)), take((4,)))
    def Cn(i, j):
        d = inp.pos[j] - inp.pos[i]
        d -= inp.box * np.rint(d / inp.box) * inp.pbc
        return oracle.mlp_descriptor(DIMS, RC, blob, 0, 0, float(np.linalg.norm(d))), d / np.linalg.norm(d)
    v = np.zeros((nbr.n, F))
    for i in range(nbr.n):
        for k in range(nbr.width):
            j = nbr.cols[k, i]
            if j != i:
                v[i] += Cn(i, j)[0]
    B = D.reshape(nbr.n, 4, nbr.n, 4)
    for i in range(0, nbr.n, 9):
        for k in range(nbr.width):
            j = nbr.cols[k, i]
            if j == i:
                continue
            Cij, u = Cn(i, j)
            Vp = _np_mlp(hopp, Cij * _np_mlp(envp, v[i] + v[j]))
            assert abs(B[i, 0, j, 0] - Vp[0]) <= 1e-12
            assert np.abs(B[i, 0, j, 1:] - u * Vp[1]).max() <= 1e-12
            assert abs(np.trace(B[i, 1:, j, 1:]) - (Vp[2] + 2 * Vp[3])) <= 1e-12   # tr of the p-p block


# ---------------------------------------------------------------------------------- P41
def test_mlp_spd_with_constant_networks_is_the_spd_oracle():
    """Eq. 2 feeding the s,p,d blocks (reading E7): MLP_lambda with zero weights and the ten integrals as output
    bias, onsite MLPs with (eps_s, eps_p, eps_d) as bias, must give gtbo_spd_hamiltonian's matrix (beta = 0)."""
    w = W.CONFIGS["c4"].scaled(8, 3, stripe=2)
    inp = W.make_inputs(w)
    ns = 3
    nbr = _nbr(w, inp, 2.65)
    V = np.array([-6.769, 5.580, 5.037, -3.033, -2.1, -1.7, 0.9, -1.3, 0.8, -0.15])
    es, ep, ed = [-8.9, -6.0, -11.0], [0.0, 2.3, -2.3], [6.5, 7.0, 5.5]
    c = np.random.default_rng(0).normal(size=(NS, NS, F, NB))
    c = 0.5 * (c + c.transpose(1, 0, 2, 3))
    env = (np.zeros((HD, F)), np.zeros(HD), np.zeros((F, HD)), np.ones(F))
    hop = (np.zeros((HD, F)), np.zeros(HD), np.zeros((10, HD)), V)
    ons = [(np.zeros((HD, F)), np.zeros(HD), np.zeros((3, HD)), np.array([es[s], ep[s], ed[s]])) for s in range(NS)]
    H = oracle.mlp_spd_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, DIMS, 3.0,
                                   W.mlp_pack(c, env, hop, ons))
    Hs = oracle.spd_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, es, ep, ed,
                                np.broadcast_to(V, (ns, ns, 10)), beta=0.0)
    assert (H.cols == Hs.cols).all()
    assert np.abs(H.vals - Hs.vals).max() <= 1e-15 and np.abs(H.diag - Hs.diag).max() == 0.0


def test_mlp_spd_blocks_are_built_from_the_mlp_outputs_and_the_matrix_is_symmetric():
    """A numpy forward pass gives the ten integrals of sampled pairs; the block must be the spd construction
    (pinned by P31-P35) of those integrals and the bond direction; H = H^T."""
    w = W.CONFIGS["c2b"].scaled(5, 4)
    inp = W.make_inputs(w)
    blob = W.mlp_weights(DIMS, 11, hop_out=10, onsite_out=3)
    nbr = _nbr(w, inp, 1.95)
    H = oracle.mlp_spd_hamiltonian(nbr, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC, blob)
    D = H.to_dense()
    assert np.abs(D - D.T).max() <= 1e-14
    off = NS * NS * F * NB
    def take(shape):
        nonlocal off
        size = int(np.prod(shape))
        out = blob[off:off + size].reshape(shape)
        off += size
        return out
    envp = (take((HD, F)), take((HD,)), take((F, HD)), take((F,)))
    hopp = (take((HD, F)), take((HD,)), take((10, HD)), take((10,)))
    onsp = [(take((HD, F)), take((HD,)), take((3, HD)), take((3,))) for _ in range(NS)]
    assert off == blob.size
    def Cn(i, j):
        d = inp.pos[j] - inp.pos[i]
        d -= inp.box * np.rint(d / inp.box) * inp.pbc
        return oracle.mlp_descriptor(DIMS, RC, blob, 0, 0, float(np.linalg.norm(d))), d / np.linalg.norm(d)
    v = np.zeros((nbr.n, F))
    for i in range(nbr.n):
        for k in range(nbr.width):
            j = nbr.cols[k, i]
            if j != i:
                v[i] += Cn(i, j)[0]
    B = D.reshape(nbr.n, 9, nbr.n, 9)
    for i in range(0, nbr.n, 9):
        eps = _np_mlp(onsp[0], v[i])
        assert np.abs(np.diag(B[i, :, i, :]) - np.repeat(eps, [1, 3, 5])).max() <= 1e-12
        for k in range(nbr.width):
            j = nbr.cols[k, i]
            if j == i:
                continue
            Cij, u = Cn(i, j)
            Vp = _np_mlp(hopp, Cij * _np_mlp(envp, v[i] + v[j]))
            assert np.abs(B[i, :, j, :] - oracle.spd_block_from_integrals(u, Vp)).max() <= 1e-12
