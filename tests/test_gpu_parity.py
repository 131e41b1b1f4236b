"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances (BASELINE.json:north_star):
neighbour lists / ELL columns bit-exact; |d mu_n| <= 1e-9; DOS <= 1e-8 of its peak."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu

MU_TOL = 1e-9          # north_star
DOS_TOL = 1e-8         # of the peak value, north_star
ULP4 = 4 * 2.0**-52    # relative: values that pass through exp / sincos of another libm


def _dev(x, dtype=None):
    t = torch.as_tensor(np.ascontiguousarray(x))
    if dtype is not None:
        t = t.to(dtype)
    return t.cuda()


def _oracle_H(w, inp, width=None, with_diag=True):
    return oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite,
                                    w.t0, w.r0, w.beta, inp.onsite_shift, width=width, method=1,
                                    with_diag=with_diag)


def _gpu_H(w, inp, width=None, with_diag=True, pbc=None):
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    return gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box,
                                 inp.pbc if pbc is None else pbc, w.cutoff, w.onsite, w.t0, w.r0,
                                 w.beta, shift, width=width, with_diag=with_diag)


def _scale(Ho):
    lo, hi = oracle.spectral_bounds(Ho)
    return 1.01 * (hi - lo) / 2.0, (hi + lo) / 2.0


# sizes span several 256-row tiles with a ragged tail; stripe shrunk with the lattice for c4
SMALL = [("c1", 24, 24, {}), ("c2", 37, 23, {}), ("c2b", 41, 29, {}), ("c3", 33, 31, {}),
         ("c4", 48, 21, {"stripe": 6}), ("c5", 57, 43, {})]


def _small(key, nx, ny, kw):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    return w, W.make_inputs(w)


# ------------------------------------------------------------------ a4: random phases (C3)
@pytest.mark.parametrize("seed,r0,R,n", [(0, 0, 1, 7), (6525, 0, 8, 1000), (2**64 - 1, 5, 3, 4099),
                                         (12345, 2, 2, 0)])
def test_random_phase_fill_matches_oracle(seed, r0, R, n):
    got = gtb.random_phase_fill(seed, r0, R, n).cpu().numpy()
    ref = oracle.random_phase_fill(seed, r0, R, n)
    assert got.shape == ref.shape
    if n:
        # |cos|,|sin| <= 1 and both libms are within 2 ulp of the exact value of the same theta
        assert np.abs(got - ref).max() <= ULP4


# ------------------------------------------------------------------ a1/a2: neighbours and ELL
@pytest.mark.parametrize("key,nx,ny,kw", SMALL)
def test_ell_columns_bit_exact_and_values_match(key, nx, ny, kw):
    w, inp = _small(key, nx, ny, kw)
    Ho = _oracle_H(w, inp)
    width, counts = gtb.neighbor_width(_dev(inp.pos), inp.box, inp.pbc, w.cutoff, want_counts=True)
    oc, ow = oracle.neighbor_counts(inp.pos, inp.box, inp.pbc, w.cutoff, 1)
    assert width == ow == Ho.width
    assert (counts.cpu().numpy() == oc).all()
    Hg = _gpu_H(w, inp)
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()                      # bit-exact
    vg, vo = Hg.vals.cpu().numpy(), Ho.vals
    if w.beta == 0.0:
        assert (vg.view(np.uint64) == vo.view(np.uint64)).all()          # table lookups: exact
    else:
        assert np.abs(vg - vo).max() <= ULP4 * np.abs(vo).max()          # one exp apart
        assert ((vg == 0.0) == (vo == 0.0)).all()
    assert (Hg.diag.cpu().numpy().view(np.uint64) == Ho.diag.view(np.uint64)).all()
    # Gershgorin bounds (C7)
    lo, hi = oracle.spectral_bounds(Ho)
    got = gtb.spectral_bounds(Hg).cpu().numpy()
    assert got[0] == pytest.approx(lo, rel=1e-14) and got[1] == pytest.approx(hi, rel=1e-14)


def test_wider_ell_is_padded_with_own_column_and_zero():
    w, inp = _small("c2b", 19, 13, {})
    Ho = _oracle_H(w, inp, width=14)
    Hg = _gpu_H(w, inp, width=14)
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()
    pad = Ho.vals == 0.0
    assert (Hg.vals.cpu().numpy()[pad] == 0.0).all()
    assert (Hg.cols.cpu().numpy()[pad] == np.broadcast_to(np.arange(Ho.n), Ho.cols.shape)[pad]).all()


@pytest.mark.parametrize("pbc", [(0, 1, 0), (1, 0, 0), (0, 0, 0), (1, 1, 1)])
def test_free_boundaries_and_tiny_periodic_grids(pbc):
    # 9 x 2 cells: the periodic y axis has fewer than three search cells at r_c = 4.0
    w = W.CONFIGS["c2"].scaled(9, 2)
    inp = W.make_inputs(w)
    pbc = np.array(pbc, dtype=np.int32)
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, pbc, w.cutoff, w.onsite, w.t0,
                                  w.r0, w.beta, inp.onsite_shift, method=0)   # brute force
    Hg = _gpu_H(w, inp, pbc=pbc)
    assert Hg.width == Ho.width
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()
    assert np.abs(Hg.vals.cpu().numpy() - Ho.vals).max() <= ULP4 * np.abs(Ho.vals).max()


def test_build_errors():
    w, inp = _small("c2", 12, 8, {})
    with pytest.raises(gtb.GtbError) as e:
        _gpu_H(w, inp, width=5)
    assert e.value.status == gtb.ERR_ELL_OVERFLOW and "needed" in str(e.value)
    small = W.CONFIGS["c2"].scaled(2, 1)          # 4.9 x 4.3 A box < 2 * 4.0 A
    with pytest.raises(gtb.GtbError) as e:
        _gpu_H(small, W.make_inputs(small))
    assert e.value.status == gtb.ERR_BOX_TOO_SMALL
    bad = inp.species.copy()
    bad[5] = 3
    with pytest.raises(gtb.GtbError) as e:
        gtb.build_hamiltonian(_dev(inp.pos), _dev(bad), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                              w.r0, w.beta)
    assert e.value.status == gtb.ERR_INVALID_ARG


# ------------------------------------------------------------------ a5-a7: moments (C4, C5)
@pytest.mark.parametrize("key,nx,ny,kw", SMALL)
def test_moments_match_oracle_direct_definition(key, nx, ny, kw):
    w, inp = _small(key, nx, ny, kw)
    Ho = _oracle_H(w, inp, with_diag=w.use_diag)
    Hg = _gpu_H(w, inp, with_diag=w.use_diag)
    a, b = (w.a, w.b) if w.a is not None else _scale(Ho)
    M = 256 if key == "c1" else 301
    ref, im = oracle.kpm_moments(Ho, a, b, M, w.R, w.seed, mode=0, algo=0, return_im=True)
    ws = gtb.workspace(gtb.kpm_workspace_bytes(Ho.n, M, w.R))
    got = gtb.kpm_moments(Hg, a, b, M, w.R, w.R, w.seed, ws=ws, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= MU_TOL
    assert np.abs(got - ref).max() <= 1e-12          # what fp64 reordering actually costs
    assert got[0] == pytest.approx(1.0, abs=1e-14) and im < 1e-12


@pytest.mark.parametrize("R_total,R_batch", [(1, 1), (2, 2), (3, 3), (4, 4), (5, 5), (7, 2), (8, 8),
                                             (9, 4), (16, 8)])
def test_moments_for_every_vector_batching(R_total, R_batch):
    w, inp = _small("c2b", 23, 17, {})
    Ho, Hg = _oracle_H(w, inp), _gpu_H(w, inp)
    a, b = _scale(Ho)
    M = 64 + (R_total & 1)                              # odd and even M
    ref = oracle.kpm_moments(Ho, a, b, M, R_total, 99, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, M, R_total, R_batch, 99).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12


def test_exact_trace_config1_against_oracle_and_closed_form_eigenvalues():
    w, inp = _small("c1", 24, 24, {})
    Ho, Hg = _oracle_H(w, inp, with_diag=False), _gpu_H(w, inp, with_diag=False)
    ref = oracle.kpm_moments(Ho, w.a, w.b, w.M, mode=1, algo=0)
    got = gtb.kpm_moments(Hg, w.a, w.b, w.M, mode=1, R_batch=8).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12
    # pin P1: zone-folded honeycomb bands, E = +-|t| sqrt(1 + 4 cx cy + 4 cx^2)
    m = np.arange(w.nx)[:, None]
    n = np.arange(2 * w.ny)[None, :]
    cx = np.cos(np.pi * m / w.nx)
    e = 2.7 * np.sqrt(np.clip(1 + 4 * cx * np.cos(np.pi * n / w.ny) + 4 * cx**2, 0, None)).ravel()
    th = np.arccos(np.concatenate([e, -e]) / w.a)
    exact = np.array([np.cos(k * th).mean() for k in range(w.M)])
    assert np.abs(got - exact).max() <= 1e-12                     # north_star: 1e-12
    assert np.abs(got[1::2]).max() <= 1e-13                       # particle-hole symmetry
    # ragged last batch of basis vectors (2304 = 7 * 329 + 1)
    got7 = gtb.kpm_moments(Hg, w.a, w.b, 40, mode=1, R_batch=7).cpu().numpy()
    assert np.abs(got7 - exact[:40]).max() <= 1e-12


def test_exact_trace_on_a_disordered_hbn_lattice_vs_eigvalsh():
    w, inp = _small("c4", 12, 5, {"stripe": 3})
    Ho, Hg = _oracle_H(w, inp), _gpu_H(w, inp)
    ev = np.linalg.eigvalsh(Ho.to_dense())
    th = np.arccos((ev - w.b) / w.a)
    exact = np.array([np.cos(k * th).mean() for k in range(48)])
    got = gtb.kpm_moments(Hg, w.a, w.b, 48, mode=1, R_batch=4).cpu().numpy()
    assert np.abs(got - exact).max() <= 1e-12


def test_single_step_and_sums_match_oracle_rows():
    w, inp = _small("c3", 33, 31, {})
    Ho, Hg = _oracle_H(w, inp), _gpu_H(w, inp)
    a, b = _scale(Ho)
    n, R = Ho.n, 4
    phi0 = oracle.random_phase_fill(7, 0, R, n)
    rows = np.arange(n)
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, rows)
    phi2 = oracle.kpm_step_rows(Ho, a, b, False, phi0, phi1, rows)
    g0 = _dev(phi0)
    g1 = torch.empty_like(g0)
    s = gtb.kpm_step(Hg, a, b, True, g0, g1).cpu().numpy()
    assert np.abs(g1.cpu().numpy() - phi1).max() <= 1e-14
    assert s[0] == pytest.approx(n * R, rel=1e-14)
    assert s[1] == pytest.approx((phi1 * phi0).sum(), rel=1e-12, abs=1e-9)
    s = gtb.kpm_step(Hg, a, b, False, g1, g0).cpu().numpy()       # g0 <- phi_2
    assert np.abs(g0.cpu().numpy() - phi2).max() <= 1e-14
    assert s[0] == pytest.approx((phi1 * phi1).sum(), rel=1e-13)
    assert s[1] == pytest.approx((phi2 * phi1).sum(), rel=1e-12, abs=1e-9)


# K7 has two implementations: the register path and the TMA-staged tile path.
# gtb_kpm_options.kernel pins one or the other, tile_stages the depth of the shared-memory ring.
@pytest.mark.parametrize("key,nx,ny,kw,R", [("c2", 37, 23, {}, 8), ("c3", 33, 31, {}, 4),
                                             ("c2b", 41, 29, {}, 2), ("c4", 48, 21, {"stripe": 6}, 8),
                                             ("c5", 57, 43, {}, 2), ("c5", 57, 43, {}, 4)])
@pytest.mark.parametrize("kernel,stages", [(gtb.KERNEL_AUTO, 0), (gtb.KERNEL_ROW, 0), (gtb.KERNEL_TILE, 1),
                                           (gtb.KERNEL_TILE, 2), (gtb.KERNEL_TILE, 3), (gtb.KERNEL_TILE, 5)])
def test_both_k7_paths_match_oracle_rows(key, nx, ny, kw, R, kernel, stages):
    opt = gtb.options(kernel=kernel, tile_stages=stages)
    w, inp = _small(key, nx, ny, kw)
    Ho = _oracle_H(w, inp, with_diag=w.use_diag)
    Hg = _gpu_H(w, inp, with_diag=w.use_diag)
    a, b = (w.a, w.b) if w.a is not None else _scale(Ho)
    n = Ho.n
    phi0 = oracle.random_phase_fill(11, 0, R, n)
    rows = np.arange(n)
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, rows)
    phi2 = oracle.kpm_step_rows(Ho, a, b, False, phi0, phi1, rows)
    g0 = _dev(phi0)
    g1 = torch.empty_like(g0)
    s = gtb.kpm_step(Hg, a, b, True, g0, g1, opt=opt).cpu().numpy()
    assert np.abs(g1.cpu().numpy() - phi1).max() <= 1e-14
    assert s[0] == pytest.approx(n * R, rel=1e-14)
    s = gtb.kpm_step(Hg, a, b, False, g1, g0, opt=opt).cpu().numpy()
    assert np.abs(g0.cpu().numpy() - phi2).max() <= 1e-14
    assert s[0] == pytest.approx((phi1 * phi1).sum(), rel=1e-13)
    assert s[1] == pytest.approx((phi2 * phi1).sum(), rel=1e-12, abs=1e-9)
    M = 65
    ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, M, R, R, 5, opt=opt).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12


def test_a_pinned_kernel_that_cannot_take_the_matrix_is_an_error():
    """gtb_kpm_options: no silent detour (include/gtb.h)."""
    w, inp = _small("c2", 37, 23, {})
    Hg = _gpu_H(w, inp, with_diag=True)                       # K = 20
    with pytest.raises(gtb.GtbError):
        gtb.kpm_moments(Hg, 20.0, 0.0, 8, 2, 2, 5, opt=gtb.options(kernel=gtb.KERNEL_ROW_X2))
    with pytest.raises(gtb.GtbError):
        gtb.kpm_moments(Hg, 20.0, 0.0, 8, 3, 3, 5, opt=gtb.options(kernel=gtb.KERNEL_TILE))   # R = 3
    with pytest.raises(gtb.GtbError):
        gtb.kpm_moments(Hg, 20.0, 0.0, 8, 2, 2, 5, opt=gtb.options(kernel=7))


# K7p: small systems run all passes in one cooperative launch (default); GTB_OPT_PER_PASS_LAUNCH takes
# the per-pass launches.  Both must agree with the oracle and with each other.
@pytest.mark.parametrize("key,nx,ny,kw,R", [("c1", 24, 24, {}, 4), ("c2", 37, 23, {}, 8), ("c3", 33, 31, {}, 2),
                                             ("c4", 48, 21, {"stripe": 6}, 8), ("c5", 57, 43, {}, 2)])
@pytest.mark.parametrize("M", [2, 3, 64, 257])
def test_single_launch_path_matches_oracle_and_per_pass_path(key, nx, ny, kw, R, M):
    w, inp = _small(key, nx, ny, kw)
    Ho = _oracle_H(w, inp, with_diag=w.use_diag)
    Hg = _gpu_H(w, inp, with_diag=w.use_diag)
    a, b = (w.a, w.b) if w.a is not None else _scale(Ho)
    ref = oracle.kpm_moments(Ho, a, b, M, R, 9, mode=0, algo=0)
    l0 = gtb.launch_count()
    got = gtb.kpm_moments(Hg, a, b, M, R, R, 9, check=True).cpu().numpy()
    used = gtb.launch_count() - l0
    assert np.abs(got - ref).max() <= 1e-12
    l0 = gtb.launch_count()
    per_pass = gtb.kpm_moments(Hg, a, b, M, R, R, 9, check=True,
                               opt=gtb.options(flags=gtb.OPT_PER_PASS_LAUNCH)).cpu().numpy()
    assert np.abs(got - per_pass).max() <= 1e-13
    if M >= 64:
        assert used < (gtb.launch_count() - l0) // 4      # the single-launch path really was taken
    grid = gtb.kpm_moments(Hg, a, b, M, R, R, 9, check=True, opt=gtb.options(flags=gtb.OPT_GRID_SYNC)).cpu().numpy()
    assert np.abs(got - grid).max() <= 1e-13              # K7c (one cluster) vs K7p (grid barrier), where both apply


# K7c: tiny systems (n T <= 8192 elements, K <= 4) run inside one thread-block cluster with phi in distributed
# shared memory; sizes around the limits: one element per CTA slot, ragged last CTA, exactly full, one too many
@pytest.mark.parametrize("nx,ny,R,width", [(24, 24, 4, None), (24, 24, 4, 4), (32, 32, 4, None), (45, 45, 2, None),
                                           (16, 16, 8, None), (3, 3, 2, None), (32, 33, 4, None), (23, 19, 2, None)])
def test_cluster_path_matches_oracle(nx, ny, R, width):
    w, inp = _small("c1", nx, ny, {})
    Ho = _oracle_H(w, inp, width=width, with_diag=False)
    Hg = _gpu_H(w, inp, width=width, with_diag=False)
    M = 96
    ref = oracle.kpm_moments(Ho, w.a, w.b, M, R, 9, mode=0, algo=0)
    l0 = gtb.launch_count()
    got = gtb.kpm_moments(Hg, w.a, w.b, M, R, R, 9, check=True).cpu().numpy()
    used = gtb.launch_count() - l0
    assert np.abs(got - ref).max() <= 1e-12
    if Ho.n * (R // 2) <= 8192:
        assert used <= 6                                   # fill, one cluster launch, reduce, finish
    exact = gtb.kpm_moments(Hg, w.a, w.b, 32, mode=1, R_batch=8).cpu().numpy()
    want = oracle.kpm_moments(Ho, w.a, w.b, 32, mode=1, algo=0) if Ho.n <= 2400 else None
    if want is not None:
        assert np.abs(exact - want).max() <= 1e-12
    w4, inp4 = _small("c4", 12, 8, {"stripe": 3})          # with a diagonal and three species
    Ho4, Hg4 = _oracle_H(w4, inp4, with_diag=True), _gpu_H(w4, inp4, with_diag=True)
    ref4 = oracle.kpm_moments(Ho4, w4.a, w4.b, 40, R, 3, mode=0, algo=0)
    got4 = gtb.kpm_moments(Hg4, w4.a, w4.b, 40, R, R, 3, check=True).cpu().numpy()
    assert np.abs(got4 - ref4).max() <= 1e-12


# K7x2 (narrow rows: two elements in flight per thread) against the oracle's rows and against K7, on sizes
# whose element count is odd in units of the grid stride, with width 3 and a padded width 4.
@pytest.mark.parametrize("key,nx,ny,kw,R,width", [("c5", 57, 43, {}, 2, None), ("c5", 57, 43, {}, 8, 4),
                                                   ("c4", 48, 21, {"stripe": 6}, 8, None),
                                                   ("c1", 24, 24, {}, 4, 4), ("c5", 301, 127, {}, 2, None)])
def test_two_elements_in_flight_path(key, nx, ny, kw, R, width):
    opts = {"1": gtb.options(kernel=gtb.KERNEL_ROW_X2), "0": gtb.options(kernel=gtb.KERNEL_ROW)}
    w, inp = _small(key, nx, ny, kw)
    Ho = _oracle_H(w, inp, width=width, with_diag=w.use_diag)
    Hg = _gpu_H(w, inp, width=width, with_diag=w.use_diag)
    a, b = (w.a, w.b) if w.a is not None else _scale(Ho)
    n = Ho.n
    phi0 = oracle.random_phase_fill(11, 0, R, n)
    rows = np.arange(n) if n < 20000 else np.unique(np.r_[0:300, n - 300:n, np.arange(0, n, 97)])
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, np.arange(n))
    phi2 = oracle.kpm_step_rows(Ho, a, b, False, phi0, phi1, rows)
    out = {}
    for x2 in ("1", "0"):
        g1, g0 = _dev(phi1), _dev(phi0)
        s = gtb.kpm_step(Hg, a, b, False, g1, g0, opt=opts[x2]).cpu().numpy()       # g0 <- phi_2
        out[x2] = g0.cpu().numpy()
        assert np.abs(out[x2][rows] - phi2).max() <= 1e-14
        assert s[0] == pytest.approx((phi1 * phi1).sum(), rel=1e-13)
    assert (out["1"] == out["0"]).all()                               # same arithmetic per element
    M = 33
    ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0) if n < 20000 else None
    got = gtb.kpm_moments(Hg, a, b, M, R, R, 5, opt=opts["1"]).cpu().numpy()
    old = gtb.kpm_moments(Hg, a, b, M, R, R, 5, opt=opts["0"]).cpu().numpy()
    assert np.abs(got - old).max() <= 1e-13
    if ref is not None:
        assert np.abs(got - ref).max() <= 1e-12


@pytest.mark.parametrize("drop", [1, 2, 3])
def test_atom_count_not_a_multiple_of_four_takes_the_register_path(drop):
    # bulk copies need 16-byte aligned slot rows (n % 4 == 0); any other n must still be exact
    w, inp = _small("c2b", 23, 17, {})
    n = inp.pos.shape[0] - drop
    args = (inp.box, (0, 0, 0), w.cutoff, w.onsite, w.t0, w.r0, w.beta)
    shift = inp.onsite_shift[:n]
    Ho = oracle.build_hamiltonian(inp.pos[:n], inp.species[:n], *args, shift, method=1)
    Hg = gtb.build_hamiltonian(_dev(inp.pos[:n]), _dev(inp.species[:n]), *args, _dev(shift))
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()
    a, b = _scale(Ho)
    for R in (2, 4, 8):
        ref = oracle.kpm_moments(Ho, a, b, 48, R, 3, mode=0, algo=0)
        got = gtb.kpm_moments(Hg, a, b, 48, R, R, 3).cpu().numpy()
        assert np.abs(got - ref).max() <= 1e-12


def test_divergence_is_reported():
    w, inp = _small("c5", 20, 20, {})
    Hg = _gpu_H(w, inp, with_diag=False)
    ws = gtb.workspace(gtb.kpm_workspace_bytes(Hg.n, 4000, 2))
    with pytest.raises(gtb.GtbError) as e:
        gtb.kpm_moments(Hg, 2.0, 0.0, 4000, 2, 2, 1, ws=ws, check=True)   # spectrum is +-8.1 eV
    assert e.value.status == gtb.ERR_DIVERGED


# ------------------------------------------------------------------ a8: DOS (C6)
@pytest.mark.parametrize("M,kernel", [(1, 1), (2, 1), (256, 1), (256, 0), (3000, 1), (5000, 1)])
def test_dos_from_oracle_moments(M, kernel):
    rng = np.random.default_rng(M)
    th = rng.uniform(0, np.pi, 4000)
    mu = np.array([np.cos(k * th).mean() for k in range(M)])      # moments of a real spectrum
    a, b = 8.5, 0.3
    E = np.linspace(b - a, b + a, 4001)                           # endpoints sit on |x| = 1 (A13)
    ref = oracle.dos(mu, a, b, E, kernel=kernel, scale=2.0)
    got = gtb.dos(_dev(mu), a, b, _dev(E), kernel=kernel, scale=2.0).cpu().numpy()
    assert got[0] == 0.0 and got[-1] == 0.0
    assert np.abs(got - ref).max() <= DOS_TOL * np.abs(ref).max()
    assert np.abs(got - ref).max() <= 1e-11 * np.abs(ref).max()
    E2 = np.array([b - 2 * a, b + a * (1 + 1e-15), b, b + 0.999999 * a])
    got2 = gtb.dos(_dev(mu), a, b, _dev(E2), kernel=kernel).cpu().numpy()
    ref2 = oracle.dos(mu, a, b, E2, kernel=kernel)
    assert got2[0] == 0.0 and got2[1] == 0.0
    assert np.abs(got2 - ref2).max() <= DOS_TOL * max(np.abs(ref).max(), np.abs(ref2).max())


def test_jackson_coefficients():
    for M in (1, 2, 257, 3000):
        assert np.abs(gtb.jackson(M).cpu().numpy() - oracle.jackson(M)).max() <= 1e-15


@pytest.mark.parametrize("key,nx,ny,kw", SMALL)
def test_end_to_end_dos(key, nx, ny, kw):
    w, inp = _small(key, nx, ny, kw)
    Ho = _oracle_H(w, inp, with_diag=w.use_diag)
    Hg = _gpu_H(w, inp, with_diag=w.use_diag)
    a, b = (w.a, w.b) if w.a is not None else _scale(Ho)
    M = 400
    E = W.energy_grid(w, a, b)
    ref = oracle.dos(oracle.kpm_moments(Ho, a, b, M, w.R, w.seed), a, b, E)
    mu = gtb.kpm_moments(Hg, a, b, M, w.R, w.R, w.seed)
    got = gtb.dos(mu, a, b, _dev(E)).cpu().numpy()
    assert np.abs(got - ref).max() <= DOS_TOL * ref.max()
    # interior points only: when fl((E_max - b)/a) lands one ulp inside |x| < 1 the end point
    # carries the 1/sqrt(1 - x^2) weight (both sides agree on it above; it is not part of the integral)
    assert abs(np.trapezoid(got[1:-1], E[1:-1]) - 1.0) < 1e-3 and got.min() > -1e-12
