"""Pins for the oracle's random phases and Chebyshev moments (north_star).

Pins used: closed-form zone-folded eigenvalues of the
periodic honeycomb supercell, printed moments, closed-walk counts, numpy eigvalsh on tiny
disordered lattices, direct-vs-doubling, invariants and the published splitmix64 output.
"""
import math

import numpy as np
import pytest
from numpy.polynomial import chebyshev as npcheb

import oracle
from paper_2509_06525_b200 import workloads as W


def _build(w, inp, with_diag=True):
    return oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite,
                                    w.t0, w.r0, w.beta, inp.onsite_shift, method=1,
                                    with_diag=with_diag)


def _closed_form_eigs(nx, ny, t):
    # P1: E = +-|t| sqrt(1 + 4 cos(pi m/nx) cos(pi n/ny) + 4 cos^2(pi m/nx)),
    #     m = 0..nx-1, n = 0..2ny-1  (zone folding of the 2-atom honeycomb bands)
    m = np.arange(nx)[:, None]
    n = np.arange(2 * ny)[None, :]
    cx = np.cos(np.pi * m / nx)
    f2 = 1.0 + 4.0 * cx * np.cos(np.pi * n / ny) + 4.0 * cx**2
    e = abs(t) * np.sqrt(np.clip(f2, 0.0, None)).ravel()
    return np.concatenate([e, -e])


def _moments_from_eigs(ev, a, b, M):
    th = np.arccos(np.clip((ev - b) / a, -1.0, 1.0))
    return np.array([np.cos(k * th).mean() for k in range(M)])


# ---------------------------------------------------------------- RNG (C3, P10)
def test_splitmix64_published_first_output():
    assert oracle.mix64(0x9E3779B97F4A7C15) == 0xE220A8397B1DCDAF


def test_hash_vectors(golden):
    for seed, r, i, h, u in golden("splitmix64_vectors.txt"):
        assert oracle.hash64(int(seed), int(r), int(i)) == int(h, 16)
        assert oracle.uniform(int(seed), int(r), int(i)) == float(u)


def test_random_phase_fill_is_unit_modulus_at_the_hashed_angle():
    n, R, seed, r0 = 500, 3, 77, 2
    phi = oracle.random_phase_fill(seed, r0, R, n)
    assert phi.shape == (n, R, 2)
    assert np.abs(np.hypot(phi[..., 0], phi[..., 1]) - 1.0).max() < 4e-16
    u = np.array([[oracle.uniform(seed, r0 + k, i) for k in range(R)] for i in range(n)])
    ang = np.mod(np.arctan2(phi[..., 1], phi[..., 0]), 2 * np.pi) / (2 * np.pi)
    assert np.abs(ang - u).max() < 1e-15
    assert 0.0 <= u.min() and u.max() < 1.0 and abs(u.mean() - 0.5) < 0.03


# --------------------------------------------- exact trace vs closed forms (P1-P3)
@pytest.mark.parametrize("algo", [0, 1])
def test_exact_trace_matches_closed_form_eigenvalues_24x24(algo, golden):
    w = W.CONFIGS["c1"]
    H = _build(w, W.make_inputs(w), with_diag=False)
    mu = oracle.kpm_moments(H, w.a, w.b, w.M, mode=1, algo=algo)
    ref = _moments_from_eigs(_closed_form_eigs(w.nx, w.ny, -2.7), w.a, w.b, w.M)
    assert np.abs(mu - ref).max() < 1e-12                      # north_star: 1e-12
    assert np.abs(mu[1::2]).max() < 1e-13                      # bipartite: odd moments vanish
    assert mu[0] == pytest.approx(1.0, abs=1e-15)
    for n, val in golden("graphene_24x24_exact_moments.txt"):  # P2 printed values
        assert mu[int(n)] == pytest.approx(float(val), abs=1e-12)


def test_closed_form_eigenvalues_are_the_dense_spectrum():
    # the pin itself, checked against a library routine on a smaller supercell
    w = W.CONFIGS["c1"].scaled(6, 5)
    H = _build(w, W.make_inputs(w), with_diag=False)
    ev = np.linalg.eigvalsh(H.to_dense())
    assert np.abs(np.sort(_closed_form_eigs(6, 5, -2.7)) - ev).max() < 1e-12


def test_low_moments_from_closed_walk_counts(golden):
    # P3: mu_2k = sum_j c_j W_j h^j with T_2k(x) = sum_j c_j x^j, h = t/a, W_0 = 1
    walks = {0: 1.0}
    walks.update({int(k): float(v) for k, v in golden("honeycomb_closed_walks.txt")})
    w = W.CONFIGS["c1"].scaled(14, 12)
    H = _build(w, W.make_inputs(w), with_diag=False)
    a = 8.5
    mu = oracle.kpm_moments(H, a, 0.0, 11, mode=1, algo=0)
    h = -2.7 / a
    for n in (2, 4, 6, 8, 10):
        c = npcheb.cheb2poly([0.0] * n + [1.0])
        expect = sum(c[j] * walks[j] * h**j for j in range(0, n + 1, 2))
        assert mu[n] == pytest.approx(expect, abs=1e-13)


# ------------------------------ disordered / h-BN tiny lattices vs eigvalsh (P4, P6)
@pytest.mark.parametrize("key,nx,ny,stripe", [("c2", 7, 5, 0), ("c2b", 9, 6, 0), ("c4", 8, 4, 2)])
def test_exact_trace_matches_dense_diagonalisation(key, nx, ny, stripe):
    w = W.CONFIGS[key].scaled(nx, ny, stripe=stripe)
    inp = W.make_inputs(w)
    H = _build(w, inp)
    lo, hi = oracle.spectral_bounds(H)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2 + 0.3      # b != 0 on purpose
    M = 40
    ev = np.linalg.eigvalsh(H.to_dense())
    ref = _moments_from_eigs(ev, a, b, M)
    for algo in (0, 1):
        mu = oracle.kpm_moments(H, a, b, M, mode=1, algo=algo)
        assert np.abs(mu - ref).max() < 1e-12
        # P6: mu_1 = (sum_i diag_i - N b) / (N a)
        assert mu[1] == pytest.approx((H.diag.sum() - H.n * b) / (H.n * a), abs=1e-13)


# ------------------------------------------------ random-phase mode (P5, P6, P7)
def test_direct_equals_doubling_on_the_same_vectors():
    w = W.CONFIGS["c2"].scaled(20, 14)
    H = _build(w, W.make_inputs(w))
    lo, hi = oracle.spectral_bounds(H)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    for M in (1, 2, 7, 64):
        mu0, im = oracle.kpm_moments(H, a, b, M, R=3, seed=11, mode=0, algo=0, return_im=True)
        mu1 = oracle.kpm_moments(H, a, b, M, R=3, seed=11, mode=0, algo=1)
        assert np.abs(mu0 - mu1).max() < 1e-13
        assert im < 1e-12                                    # A12: Im parts are a diagnostic
        assert mu0[0] == pytest.approx(1.0, abs=1e-14)       # |exp(i theta)| = 1
        assert np.abs(mu0).max() <= 1.0 + 1e-12


def test_random_moments_follow_the_definition_with_dense_algebra():
    # m_n = Re <phi_0| T_n(H~) |phi_0> evaluated with numpy's dense eigendecomposition
    w = W.CONFIGS["c2b"].scaled(6, 5)
    inp = W.make_inputs(w)
    H = _build(w, inp)
    a, b, M, R, seed = 14.0, 0.05, 24, 2, 99
    ev, U = np.linalg.eigh(H.to_dense())
    phi = oracle.random_phase_fill(seed, 0, R, H.n)
    z = phi[..., 0] + 1j * phi[..., 1]                      # [n, R]
    c = U.T @ z                                             # eigen-components
    th = np.arccos((ev - b) / a)
    ref = np.array([(np.abs(c) ** 2 * np.cos(k * th)[:, None]).sum() for k in range(M)])
    ref /= H.n * R
    mu = oracle.kpm_moments(H, a, b, M, R=R, seed=seed, mode=0, algo=0)
    assert np.abs(mu - ref).max() < 1e-12


def test_stochastic_trace_converges_to_exact_trace():
    # P7: |mu^R - mu^exact| <~ 5/sqrt(N R), shrinking with R
    w = W.CONFIGS["c1"]
    H = _build(w, W.make_inputs(w), with_diag=False)
    M = 32
    exact = _moments_from_eigs(_closed_form_eigs(w.nx, w.ny, -2.7), w.a, w.b, M)
    err = {}
    for R in (4, 64):
        mu = oracle.kpm_moments(H, w.a, w.b, M, R=R, seed=W.SEED_VECTORS, mode=0, algo=1)
        err[R] = np.abs(mu - exact).max()
        assert err[R] < 5.0 / math.sqrt(H.n * R)
    assert err[64] < err[4]


def test_step_rows_matches_dense_matrix_product():
    w = W.CONFIGS["c2b"].scaled(7, 5)
    H = _build(w, W.make_inputs(w))
    a, b, R = 13.0, -0.2, 3
    rng = np.random.default_rng(5)
    prev = rng.standard_normal((H.n, R, 2))
    cur = rng.standard_normal((H.n, R, 2))
    rows = np.array([0, 3, H.n - 1, 17])
    Ht = (H.to_dense() - b * np.eye(H.n)) / a
    zc = cur[..., 0] + 1j * cur[..., 1]
    zp = prev[..., 0] + 1j * prev[..., 1]
    first = oracle.kpm_step_rows(H, a, b, True, None, cur, rows)
    nxt = oracle.kpm_step_rows(H, a, b, False, prev, cur, rows)
    r1 = (Ht @ zc)[rows]
    r2 = (2 * Ht @ zc - zp)[rows]
    assert np.abs(first[..., 0] + 1j * first[..., 1] - r1).max() < 1e-13
    assert np.abs(nxt[..., 0] + 1j * nxt[..., 1] - r2).max() < 1e-13
