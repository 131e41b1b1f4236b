"""GPU parity of the VAC-conductivity path (Eq. 3):
velocity operator, Chebyshev-Bessel propagator, VAC moments, conductivity -- the CUDA path through the
C ABI against oracle/gtbo_vac.cpp on the same seeded inputs.  Tolerances: velocity values bit-exact
(one product of the same operands); vectors 1e-13 absolute per propagation step (fp64 reordering
plus two Bessel routines); moments 1e-9 absolute relative to C_0(0) (north_star's moment tolerance,
the VAC moments being un-normalised: C_0(0) = Tr V^2 / N); sigma 1e-8 of its peak."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu

DT = 0.1 / gtb.HBAR_EV_FS     # the paper's 0.1 fs


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _setup(key, nx, ny, **kw):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                                  w.r0, w.beta, inp.onsite_shift, method=1, with_diag=w.use_diag)
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite,
                               w.t0, w.r0, w.beta, shift, with_diag=w.use_diag)
    if w.a is not None:
        a, b = w.a, w.b
    else:
        lo, hi = oracle.spectral_bounds(Ho)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    return w, inp, Ho, Hg, a, b


CASES = [("c1", 24, 24, {}), ("c2", 37, 23, {}), ("c2b", 41, 29, {}), ("c3", 33, 31, {}),
         ("c4", 48, 21, {"stripe": 6}), ("c5", 57, 43, {})]


@pytest.mark.parametrize("key,nx,ny,kw", CASES)
@pytest.mark.parametrize("axis", [0, 1])
def test_velocity_values_bit_exact(key, nx, ny, kw, axis):
    w, inp, Ho, Hg, a, b = _setup(key, nx, ny, **kw)
    ref = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, axis)
    got = gtb.velocity_ell(Hg, _dev(inp.pos), inp.box, inp.pbc, axis).cpu().numpy()
    if w.beta == 0.0:
        assert (got == ref).all()                       # same operands, one rounding each
    else:                                               # hoppings differ by <= 4 ulp (another exp)
        assert np.abs(got - ref).max() <= 4 * 2.0**-52 * np.abs(ref).max()
    assert (got[Ho.cols == np.arange(Ho.n)[None, :]] == 0).all()


@pytest.mark.parametrize("R", [1, 2, 3, 8])
def test_velocity_apply_matches_oracle(R):
    w, inp, Ho, Hg, a, b = _setup("c2b", 23, 17)
    vo = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, 0)
    x = oracle.random_phase_fill(3, 0, R, Ho.n)
    ref = oracle.velocity_apply(Ho, vo, x)
    got = gtb.velocity_apply(Hg, _dev(vo), _dev(x)).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("key,nx,ny,kw,R", [("c1", 24, 24, {}, 4), ("c2", 37, 23, {}, 8),
                                             ("c3", 33, 31, {}, 4), ("c5", 57, 43, {}, 2),
                                             ("c2b", 23, 17, {}, 3)])
@pytest.mark.parametrize("dt", [DT, 1.3, 0.0])
def test_propagator_matches_oracle(key, nx, ny, kw, R, dt):
    w, inp, Ho, Hg, a, b = _setup(key, nx, ny, **kw)
    x = oracle.random_phase_fill(9, 0, R, Ho.n)
    ref, terms_ref = oracle.evolve(Ho, a, b, dt, x, return_terms=True)
    g = _dev(x)
    terms = gtb.evolve(Hg, a, b, dt, g)
    assert abs(terms - terms_ref) <= 1                  # two Bessel routines at a 1e-18 threshold
    assert np.abs(g.cpu().numpy() - ref).max() <= 1e-13
    # ten steps in a row stay on the oracle's trajectory and on the unit circle norm
    ref10 = x
    g = _dev(x)
    for _ in range(10):
        ref10 = oracle.evolve(Ho, a, b, dt, ref10)
        gtb.evolve(Hg, a, b, dt, g)
    got = g.cpu().numpy()
    assert np.abs(got - ref10).max() <= 1e-12
    assert abs((got**2).sum() / (Ho.n * R) - 1.0) <= 1e-12


@pytest.mark.parametrize("key,nx,ny,kw", CASES)
def test_vac_moments_match_oracle(key, nx, ny, kw):
    w, inp, Ho, Hg, a, b = _setup(key, nx, ny, **kw)
    vo = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, 0)
    vg = gtb.velocity_ell(Hg, _dev(inp.pos), inp.box, inp.pbc, 0)
    M, T = 33, 4
    ref = oracle.vac_moments(Ho, vo, a, b, M, T, DT, R=w.R, seed=w.seed, mode=0)
    got = gtb.vac_moments(Hg, vg, a, b, M, T, DT, w.R, w.R, w.seed, check=True).cpu().numpy()
    scale = ref[0, 0]
    assert scale > 0
    assert np.abs(got - ref).max() <= 1e-9 * scale      # north_star's moment tolerance
    assert np.abs(got - ref).max() <= 1e-11 * scale     # what reordering actually costs


@pytest.mark.parametrize("R_total,R_batch", [(1, 1), (2, 2), (3, 3), (5, 2), (8, 8), (6, 4)])
def test_vac_moments_for_every_vector_batching(R_total, R_batch):
    w, inp, Ho, Hg, a, b = _setup("c2b", 23, 17)
    vo = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, 1)
    M, T = 16 + (R_total & 1), 3
    ref = oracle.vac_moments(Ho, vo, a, b, M, T, DT, R=R_total, seed=77, mode=0)
    got = gtb.vac_moments(Hg, _dev(vo), a, b, M, T, DT, R_total, R_batch, 77).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-11 * ref[0, 0]


def test_exact_trace_vac_moments_vs_oracle_and_eigh():
    w, inp, Ho, Hg, a, b = _setup("c4", 8, 3, stripe=2)
    vo = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, 0)
    M, T = 24, 5
    ref = oracle.vac_moments(Ho, vo, a, b, M, T, DT, mode=1)
    got = gtb.vac_moments(Hg, _dev(vo), a, b, M, T, DT, mode=1, R_batch=8).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-11 * ref[0, 0]
    # and against Eq. 3 in the eigenbasis (numpy eigh), independent of both implementations
    Hd = Ho.to_dense()
    A = np.zeros_like(Hd)
    for k in range(Ho.width):
        np.add.at(A, (np.arange(Ho.n), Ho.cols[k]), vo[k])
    E, Q = np.linalg.eigh(Hd)
    w2 = np.abs(Q.T @ (1j * A) @ Q)**2
    th = np.arccos(np.clip((E - b) / a, -1, 1))
    for j in range(T):
        s = (w2 * np.cos((E[:, None] - E[None, :]) * j * DT)).sum(1)
        exact = np.array([(np.cos(n * th) * s).sum() / Ho.n for n in range(M)])
        assert np.abs(got[j] - exact).max() <= 1e-10 * ref[0, 0]


def test_conductivity_reconstruction_and_time_integral():
    w, inp, Ho, Hg, a, b = _setup("c2", 21, 13)
    vo = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, 0)
    M, T = 64, 6
    Cm = oracle.vac_moments(Ho, vo, a, b, M, T, DT, R=2, seed=1, mode=0)
    E = np.linspace(b - a, b + a, 401)
    rv_ref, sg_ref = oracle.vac_conductivity(Cm, a, b, E, DT, scale=3.0)
    rv, sg = gtb.vac_conductivity(_dev(Cm), a, b, _dev(E), DT, scale=3.0)
    assert np.abs(rv.cpu().numpy() - rv_ref).max() <= 1e-11 * np.abs(rv_ref).max()
    assert np.abs(sg.cpu().numpy() - sg_ref).max() <= 1e-11 * np.abs(sg_ref).max()
    # end to end: GPU moments -> GPU conductivity against the oracle chain
    Cg = gtb.vac_moments(Hg, gtb.velocity_ell(Hg, _dev(inp.pos), inp.box, inp.pbc, 0), a, b, M, T, DT,
                         2, 2, 1)
    rv2, sg2 = gtb.vac_conductivity(Cg, a, b, _dev(E), DT, scale=3.0)
    assert np.abs(sg2.cpu().numpy() - sg_ref).max() <= 1e-8 * np.abs(sg_ref).max()
    assert (sg2[0] == 0).all()


def test_vac_argument_validation():
    w, inp, Ho, Hg, a, b = _setup("c1", 6, 6)
    vg = gtb.velocity_ell(Hg, _dev(inp.pos), inp.box, inp.pbc, 0)
    with pytest.raises(gtb.GtbError):
        gtb.velocity_ell(Hg, _dev(inp.pos), inp.box, inp.pbc, 3)
    with pytest.raises(gtb.GtbError):
        gtb.vac_moments(Hg, vg, -1.0, 0.0, 8, 2, DT, 2, 2, 0)
    with pytest.raises(gtb.GtbError):
        gtb.vac_moments(Hg, vg, a, b, 8, 0, DT, 2, 2, 0)
    with pytest.raises(gtb.GtbError):
        gtb.vac_moments(Hg, vg, a, b, 8, 2, DT, 2, 2, 0, ws=gtb.workspace(1024))


def test_carrier_density_and_mobility_match_oracle():
    rng = np.random.default_rng(0)
    for E in (np.linspace(-8.5, 8.5, 4001), np.sort(rng.uniform(-3, 3, 257))):
        rho = rng.uniform(0.0, 1.0, E.shape[0])
        sigma = rng.uniform(0.0, 5.0, E.shape[0])
        for e_ref in (float(E[len(E) // 3]), 0.01234, float(E[0]), float(E[-1])):
            ref = oracle.carrier_density(rho, E, e_ref)
            got = gtb.carrier_density(_dev(rho), _dev(E), e_ref)
            assert np.abs(got.cpu().numpy() - ref).max() <= 1e-13 * max(1.0, np.abs(ref).max())
            mu_ref = oracle.mobility(sigma, ref, scale=2.0, n_min=1e-9)
            mu = gtb.mobility(_dev(sigma), _dev(ref), 2.0, 1e-9).cpu().numpy()
            assert np.abs(mu - mu_ref).max() <= 1e-12 * np.abs(mu_ref).max()
    with pytest.raises(gtb.GtbError):
        gtb.carrier_density(_dev(rho), _dev(E), 99.0)


# ---- the fused passes of the VAC path on a compressed form of the same matrix (gtb_kpm_options.alt) ----------
@pytest.mark.parametrize("key,nx,ny,kw,R,form", [("c5", 57, 43, {}, 2, "packed"), ("c4", 48, 21, {"stripe": 6}, 4, "packed"),
                                                 ("c2", 61, 47, {}, 8, "window"), ("c3", 53, 41, {}, 4, "window")])  # noqa: E501
def test_vac_moments_on_packed_rows_and_windowed_tiles(key, nx, ny, kw, R, form):
    w, inp, Ho, Hg, a, b = _setup(key, nx, ny, **kw)
    vo = oracle.velocity_ell(Ho, inp.pos, inp.box, inp.pbc, 0)
    vg = gtb.velocity_ell(Hg, _dev(inp.pos), inp.box, inp.pbc, 0)
    M, T = 20, 4
    ref = oracle.vac_moments(Ho, vo, a, b, M, T, DT, R=R, seed=7, mode=0)
    plain = gtb.vac_moments(Hg, vg, a, b, M, T, DT, R, R, 7, check=True).cpu().numpy()
    if form == "packed":
        alt, mode = gtb.pack_ell(Hg), gtb.MODE_PACKED
    else:
        alt, mode = gtb.window_ell(Hg, R), gtb.MODE_WINDOW
    assert alt is not None
    got = gtb.vac_moments(Hg, vg, a, b, M, T, DT, R, R, 7, check=True,
                          opt=gtb.options(alt=alt, alt_mode=mode)).cpu().numpy()
    c00 = abs(ref[0, 0])
    assert np.abs(got - plain).max() <= 1e-13 * c00          # same vectors bit for bit, other block sums
    assert np.abs(got - ref).max() <= 1e-11 * c00
    if form == "window":
        with pytest.raises(gtb.GtbError):                     # built for R vectors per pass
            gtb.vac_moments(Hg, vg, a, b, M, T, DT, 2, 2, 7, opt=gtb.options(alt=alt, alt_mode=mode))
