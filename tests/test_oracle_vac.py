"""Pins of the VAC-conductivity oracle (oracle/gtbo_vac.cpp; Eq. 3) against things
other than itself: dense commutators, exact diagonalisation (numpy eigh), closed forms, invariants.
P14 velocity operator, P15 propagator, P16 exact-trace moments, P17 closed-form Tr V^2,
P18 stochastic vs exact trace, P19 reconstruction and time integral."""
import numpy as np
import pytest

import oracle
from paper_2509_06525_b200 import workloads as W


def _lattice(key, nx, ny, pbc=None, **kw):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    pbc = inp.pbc if pbc is None else np.asarray(pbc, dtype=np.int32)
    H = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, pbc, w.cutoff, w.onsite, w.t0, w.r0,
                                 w.beta, inp.onsite_shift, method=0)
    return w, inp, pbc, H


def _dense(H, vals):
    m = np.zeros((H.n, H.n))
    rows = np.arange(H.n)
    for k in range(H.width):
        np.add.at(m, (rows, H.cols[k]), vals[k])
    return m


def _cplx(x):          # [n][R][2] -> complex [n][R]
    return x[..., 0] + 1j * x[..., 1]


def _scale(H):
    lo, hi = oracle.spectral_bounds(H)
    return 1.01 * (hi - lo) / 2.0, (hi + lo) / 2.0


# ---------------------------------------------------------------------------------- P14
@pytest.mark.parametrize("axis", [0, 1, 2])
def test_velocity_is_the_commutator_on_an_open_cluster(axis):
    # no periodic image: X is a well-defined diagonal operator and V = i [H, X] exactly
    w, inp, pbc, H = _lattice("c2b", 6, 5, pbc=(0, 0, 0))
    vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, axis)
    Hd = H.to_dense()
    X = np.diag(inp.pos[:, axis])
    V = 1j * (Hd @ X - X @ Hd)
    assert np.abs(1j * _dense(H, vv) - V).max() <= 1e-14
    assert np.abs(V - V.conj().T).max() == 0.0        # Hermitian


def test_velocity_uses_the_minimum_image_and_is_antisymmetric():
    w, inp, pbc, H = _lattice("c2", 6, 4)
    vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, 0)
    A = _dense(H, vv)
    assert np.abs(A + A.T).max() <= 1e-15
    i = np.arange(H.n)[None, :].repeat(H.width, 0)
    d = inp.pos[H.cols, 0] - inp.pos[i, 0]
    d -= inp.box[0] * np.rint(d / inp.box[0])
    assert np.abs(d).max() <= w.cutoff                 # a bond is never longer than the cutoff
    assert np.abs(vv - H.vals * d).max() <= 1e-15
    assert (vv[H.cols == i] == 0).all()                # padding slots (col = i) carry zero


def test_velocity_apply_matches_dense_product():
    w, inp, pbc, H = _lattice("c4", 8, 3, stripe=2)
    vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, 0)
    rng = np.random.default_rng(1)
    x = rng.standard_normal((H.n, 3, 2))
    y = _cplx(oracle.velocity_apply(H, vv, x))
    assert np.abs(y - (1j * _dense(H, vv)) @ _cplx(x)).max() <= 1e-13


# ---------------------------------------------------------------------------------- P15
@pytest.mark.parametrize("dt", [0.05, 0.1519, 1.3])   # 0.1519 hbar/eV = the paper's 0.1 fs
def test_propagator_matches_exact_diagonalisation(dt):
    w, inp, pbc, H = _lattice("c2b", 5, 4)
    a, b = _scale(H)
    E, Q = np.linalg.eigh(H.to_dense())
    rng = np.random.default_rng(2)
    x = rng.standard_normal((H.n, 2, 2))
    y, terms = oracle.evolve(H, a, b, dt, x, return_terms=True)
    exact = Q @ (np.exp(-1j * E * dt)[:, None] * (Q.T @ _cplx(x)))
    assert np.abs(_cplx(y) - exact).max() <= 2e-13
    assert a * dt < terms < a * dt + 40                # a few terms past the turning point m = a dt
    # unitary, and two steps equal one step of twice the length
    assert np.abs((np.abs(_cplx(y))**2).sum(0) - (np.abs(_cplx(x))**2).sum(0)).max() <= 1e-12
    y2 = oracle.evolve(H, a, b, dt, y)
    assert np.abs(_cplx(y2) - _cplx(oracle.evolve(H, a, b, 2 * dt, x))).max() <= 4e-13


def test_propagator_of_zero_time_is_the_identity():
    w, inp, pbc, H = _lattice("c1", 4, 4)
    x = np.random.default_rng(3).standard_normal((H.n, 1, 2))
    assert np.abs(oracle.evolve(H, 8.5, 0.0, 0.0, x) - x).max() <= 1e-15


# ---------------------------------------------------------------------------------- P16
def _exact_vac_moments(H, vv, a, b, M, n_steps, dt):
    """(1/N) sum_kl T_n(E~_k) |V_kl|^2 cos((E_k - E_l) tau_j) from numpy eigh (Eq. 3 in the eigenbasis)."""
    E, Q = np.linalg.eigh(H.to_dense())
    Vkl = Q.T @ (1j * _dense(H, vv)) @ Q
    w2 = np.abs(Vkl)**2
    th = np.arccos(np.clip((E - b) / a, -1, 1))
    out = np.zeros((n_steps, M))
    for j in range(n_steps):
        s = (w2 * np.cos((E[:, None] - E[None, :]) * j * dt)).sum(1)       # per eigenstate k
        for n in range(M):
            out[j, n] = (np.cos(n * th) * s).sum() / H.n
    return out


@pytest.mark.parametrize("key,nx,ny,kw", [("c1", 5, 4, {}), ("c2b", 5, 4, {}), ("c4", 8, 3, {"stripe": 2})])
def test_exact_trace_vac_moments_match_exact_diagonalisation(key, nx, ny, kw):
    w, inp, pbc, H = _lattice(key, nx, ny, **kw)
    a, b = (w.a, w.b) if w.a is not None else _scale(H)
    vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, 0)
    M, T, dt = 24, 6, 0.1519
    got = oracle.vac_moments(H, vv, a, b, M, T, dt, mode=1)
    ref = _exact_vac_moments(H, vv, a, b, M, T, dt)
    assert np.abs(got - ref).max() <= 1e-11 * max(1.0, np.abs(ref).max())
    assert got[1:, 0].max() < got[0, 0]                # the autocorrelation decays from tau = 0


# ---------------------------------------------------------------------------------- P17
def test_trace_of_v_squared_of_pristine_graphene_is_closed_form():
    # per atom: sum over the 3 bonds of t^2 dx^2 = t^2 * 2 * (sqrt(3)/2 * a_cc)^2 = 1.5 t^2 a_cc^2
    w, inp, pbc, H = _lattice("c1", 6, 5)
    for axis, want in ((0, 1.5), (1, 1.5)):            # isotropic: y gives a^2 + 2 (a/2)^2 = 1.5 a^2 too
        vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, axis)
        c = oracle.vac_moments(H, vv, w.a, w.b, 1, 1, 0.1, mode=1)
        assert c[0, 0] == pytest.approx(want * 2.7**2 * 1.42**2, rel=1e-13)


# ---------------------------------------------------------------------------------- P18
def test_random_phase_estimate_converges_to_the_exact_trace():
    w, inp, pbc, H = _lattice("c2b", 8, 6)
    a, b = _scale(H)
    vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, 0)
    M, T, dt = 8, 3, 0.1519
    exact = oracle.vac_moments(H, vv, a, b, M, T, dt, mode=1)
    est = oracle.vac_moments(H, vv, a, b, M, T, dt, R=64, seed=5, mode=0)
    assert np.abs(est - exact).max() <= 6 * exact[0, 0] / np.sqrt(H.n * 64)
    est2 = oracle.vac_moments(H, vv, a, b, M, T, dt, R=64, seed=6, mode=0)
    assert np.abs(est - est2).max() > 0                # the seed matters


# ---------------------------------------------------------------------------------- P19
def test_reconstruction_is_the_dos_kernel_and_the_integral_is_the_trapezoid_rule():
    rng = np.random.default_rng(4)
    M, T, G, dt, a, b = 40, 7, 33, 0.3, 9.0, 0.4
    mu = rng.standard_normal(M) / (1 + np.arange(M))
    f = rng.standard_normal(T)
    Cm = f[:, None] * mu[None, :]
    E = np.linspace(b - 0.95 * a, b + 0.95 * a, G)
    rv, sg = oracle.vac_conductivity(Cm, a, b, E, dt, kernel=1, scale=2.5)
    rho = oracle.dos(mu, a, b, E)
    assert np.abs(rv - f[:, None] * rho[None, :]).max() <= 1e-13 * np.abs(rv).max()
    cum = np.concatenate([[0.0], np.cumsum((f[1:] + f[:-1]) / 2) * dt])
    assert np.abs(sg - 2.5 * cum[:, None] * rho[None, :]).max() <= 1e-12 * np.abs(sg).max()
    assert (sg[0] == 0).all()


def test_vac_density_at_time_zero_is_non_negative_and_particle_hole_symmetric():
    w, inp, pbc, H = _lattice("c1", 8, 6)
    vv = oracle.velocity_ell(H, inp.pos, inp.box, pbc, 0)
    Cm = oracle.vac_moments(H, vv, w.a, w.b, 64, 2, 0.1519, mode=1)
    E = np.linspace(-8.0, 8.0, 81)
    rv, sg = oracle.vac_conductivity(Cm, w.a, w.b, E, 0.1519)
    assert rv[0].min() >= -1e-12                        # Tr[delta(E-H) V^2] >= 0 with a positive kernel
    assert np.abs(rv[0] - rv[0][::-1]).max() <= 1e-10   # bipartite lattice, zero onsite
    assert np.abs(Cm[0, 1::2]).max() <= 1e-12           # odd moments vanish for the same reason


# ---------------------------------------------------------------------------------- P37 (Fig. 4b post-processing)
def test_carrier_density_closed_forms_and_mobility():
    E = np.linspace(-2.0, 3.0, 501)
    # graphene-like DOS rho = |E|: n(E) = E|E|/2 relative to the neutrality point E = 0 (trapezoid is exact
    # on the linear pieces; the grid contains 0)
    n = oracle.carrier_density(np.abs(E), E, 0.0)
    assert np.abs(n - E * np.abs(E) / 2).max() <= 1e-13
    # constant DOS, reference off the grid points: n = rho0 (E - e_ref)
    n = oracle.carrier_density(np.full_like(E, 0.7), E, 0.123456)
    assert np.abs(n - 0.7 * (E - 0.123456)).max() <= 1e-13
    # against numpy's trapezoid on a non-uniform grid, reference at a grid point
    rng = np.random.default_rng(0)
    Eg = np.sort(rng.uniform(-1, 1, 64))
    rho = rng.uniform(0.1, 1.0, 64)
    n = oracle.carrier_density(rho, Eg, Eg[20])
    want = np.array([np.trapezoid(rho[20:j + 1], Eg[20:j + 1]) if j >= 20 else -np.trapezoid(rho[j:21], Eg[j:21])
                     for j in range(64)])
    assert np.abs(n - want).max() <= 1e-13
    sigma = rng.uniform(0.0, 2.0, 64)
    mu = oracle.mobility(sigma, n, scale=3.0, n_min=1e-6)
    live = np.abs(n) > 1e-6
    assert (mu[~live] == 0).all() and np.abs(mu[live] - 3.0 * sigma[live] / np.abs(n[live])).max() <= 1e-12
    assert mu[20] == 0.0                                    # no carriers at the reference energy
    with pytest.raises(oracle.OracleError):
        oracle.carrier_density(rho, Eg, 2.0)                # reference outside the grid
