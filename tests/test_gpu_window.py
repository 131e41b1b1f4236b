"""GPU parity of the windowed-tile pass K7w (csrc/window.cu, gtb_window_ell + GTB_MODE_WINDOW; SURVEY.md
sec. 8(f) NEXT-4: sliced ELL, 16-bit window-relative columns, phi_n gathered from shared memory) against the
oracle's rows and moments and against the TMA-staged pass K7t, which it must reproduce bit for bit (R = 4: to
rounding -- the builder re-orders the slots of row pairs there)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _both(w, inp, with_diag=True, perm=None):
    pos, spec, shift = inp.pos, inp.species, inp.onsite_shift
    if perm is not None:
        pos, spec = pos[perm], spec[perm]
        shift = shift[perm] if shift is not None else None
    Ho = oracle.build_hamiltonian(pos, spec, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta, shift,
                                  with_diag=with_diag)
    Hg = gtb.build_hamiltonian(_dev(pos), _dev(spec), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta,
                               _dev(shift) if shift is not None else None, with_diag=with_diag)
    return Ho, Hg


# sizes: several tiles per CTA and a ragged last tile (n not a multiple of the tile), n % 4 == 0 for K7t
CASES = [("c2", 61, 47, 8, True), ("c2", 61, 47, 4, True), ("c3", 53, 41, 4, False), ("c2b", 67, 45, 2, True),
         ("c2b", 41, 29, 8, True), ("c4", 48, 21, 8, True), ("c5", 57, 43, 2, False), ("c2", 250, 64, 8, True)]


@pytest.mark.parametrize("key,nx,ny,R,diag", CASES)
def test_windowed_pass_matches_the_oracle_and_the_tile_pass(key, nx, ny, R, diag):
    kw = {"stripe": 6} if key == "c4" else {}
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    Ho, Hg = _both(w, inp, with_diag=diag)
    Wd = gtb.window_ell(Hg, R)
    assert Wd is not None and 1 <= Wd.blocks <= 40 and Wd.width == Ho.width + 65536 * Wd.blocks + (R << 24)
    n = Ho.n
    if w.a is not None:
        a, b = w.a, w.b
    else:
        lo, hi = oracle.spectral_bounds(Ho)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    phi0 = oracle.random_phase_fill(11, 0, R, n)
    rows = np.arange(n) if n < 30000 else np.unique(np.r_[0:600, n - 600:n, np.arange(0, n, 61)])
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, np.arange(n))
    phi2 = oracle.kpm_step_rows(Ho, a, b, False, phi0, phi1, rows)
    tile = gtb.options(kernel=gtb.KERNEL_TILE)
    g0 = _dev(phi0)
    g1, q1 = torch.empty_like(g0), torch.empty_like(g0)
    s = gtb.kpm_step(Wd, a, b, True, g0, g1, mode=gtb.MODE_WINDOW).cpu().numpy()
    gtb.kpm_step(Hg, a, b, True, g0, q1, opt=tile)
    assert np.abs(g1.cpu().numpy() - phi1).max() <= 1e-14
    # R = 4: gtb_window_ell re-orders the slots of row pairs (bank conflicts), so the sums run in another order
    same = (lambda x, y: torch.equal(x, y)) if R != 4 else (lambda x, y: (x - y).abs().max().item() <= 4e-15)
    assert same(g1, q1)
    assert s[0] == pytest.approx(n * R, rel=1e-13)
    g1, g0w, g0t = _dev(phi1), _dev(phi0), _dev(phi0)
    s = gtb.kpm_step(Wd, a, b, False, g1, g0w, mode=gtb.MODE_WINDOW).cpu().numpy()      # <- phi_2
    gtb.kpm_step(Hg, a, b, False, g1, g0t, opt=tile)
    assert same(g0w, g0t)
    assert np.abs(g0w.cpu().numpy()[rows] - phi2).max() <= 1e-14
    assert s[0] == pytest.approx((phi1 * phi1).sum(), rel=1e-13)
    M = 65
    got = gtb.kpm_moments(Wd, a, b, M, 2 * R, R, 5, mode=gtb.MODE_WINDOW, check=True).cpu().numpy()   # two batches
    old = gtb.kpm_moments(Hg, a, b, M, 2 * R, R, 5, opt=tile, check=True).cpu().numpy()
    assert np.abs(got - old).max() <= 1e-13
    if n < 30000:
        ref = oracle.kpm_moments(Ho, a, b, M, 2 * R, 5, mode=0, algo=0)
        assert np.abs(got - ref).max() <= 1e-12
    with pytest.raises(gtb.GtbError):           # built for R vectors per pass: another batch size is refused
        gtb.kpm_moments(Wd, a, b, 8, 3 * R // 2, R, 5, mode=gtb.MODE_WINDOW)


def test_tile_major_numbering_shrinks_the_window_and_keeps_parity():
    """The same lattice with its atoms numbered tile-major (workloads.make_inputs(tile=...), bench.py
    --tile-numbering): smaller windows, and moments equal to the oracle's on the same renumbered input."""
    w = W.CONFIGS["c2"].scaled(128, 96)
    R, M = 8, 33
    blocks = []
    for tile in (None, (4, 4)):
        inp = W.make_inputs(w, tile=tile)
        Ho, Hg = _both(w, inp)
        Wd = gtb.window_ell(Hg, R)
        assert Wd is not None
        blocks.append(Wd.blocks)
        lo, hi = oracle.spectral_bounds(Ho)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
        got = gtb.kpm_moments(Wd, a, b, M, R, R, 5, mode=gtb.MODE_WINDOW, check=True).cpu().numpy()
        ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
        assert np.abs(got - ref).max() <= 1e-12
    assert blocks[1] < blocks[0]


def test_a_numbering_without_locality_stays_on_the_plain_path():
    w = W.CONFIGS["c2"].scaled(61, 47)
    inp = W.make_inputs(w)
    perm = np.random.default_rng(3).permutation(inp.pos.shape[0])
    Ho, Hg = _both(w, inp, perm=perm)
    assert gtb.window_ell(Hg, 8) is None
    M, R = 33, 8
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, M, R, R, 5, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12
