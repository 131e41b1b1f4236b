"""Pins for the oracle's neighbour search / Hamiltonian assembly (Eq. 1).

Each test pins oracle/gtbo_hamiltonian.cpp to something other than itself:
honeycomb shell counts, brute force vs cell buckets, symmetry, a bond census
 and hand-placed atoms.
"""
import math

import numpy as np
import pytest

import oracle
from paper_2509_06525_b200 import workloads as W


def _build(w, inp, method=1, width=None):
    return oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite,
                                    w.t0, w.r0, w.beta, inp.onsite_shift, width=width,
                                    method=method, with_diag=True)


@pytest.mark.parametrize("cutoff,expected", [(1.95, 3), (2.65, 9), (3.3, 12), (4.0, 18), (4.5, 24)])
def test_pristine_shell_counts(cutoff, expected):
    # honeycomb shells: 3 at a, 6 at sqrt(3)a, 3 at 2a, 6 at sqrt(7)a, 6 at 3a (C1)
    w = W.CONFIGS["c1"].scaled(8, 6)
    inp = W.make_inputs(w)
    for method in (0, 1):
        counts, width = oracle.neighbor_counts(inp.pos, inp.box, inp.pbc, cutoff, method)
        assert width == expected
        assert (counts == expected).all()


def test_displaced_third_shell_is_exactly_12():
    # P8: with the config-2 displacements and r_c = 3.3 A every atom keeps 12 neighbours
    w = W.CONFIGS["c2"].scaled(30, 20)
    inp = W.make_inputs(w)
    counts, width = oracle.neighbor_counts(inp.pos, inp.box, inp.pbc, 3.3, 1)
    assert width == 12 and (counts == 12).all()


@pytest.mark.parametrize("key,nx,ny", [("c2", 14, 9), ("c2b", 20, 12), ("c4", 16, 7)])
def test_brute_force_equals_cell_buckets_bit_exact(key, nx, ny):
    w = W.CONFIGS[key].scaled(nx, ny, stripe=4 if key == "c4" else 0)
    inp = W.make_inputs(w)
    c0, w0 = oracle.neighbor_counts(inp.pos, inp.box, inp.pbc, w.cutoff, 0)
    c1, w1 = oracle.neighbor_counts(inp.pos, inp.box, inp.pbc, w.cutoff, 1)
    assert w0 == w1 and (c0 == c1).all()
    H0 = _build(w, inp, 0, w0)
    H1 = _build(w, inp, 1, w1)
    assert (H0.cols == H1.cols).all()
    assert (H0.vals.view(np.uint64) == H1.vals.view(np.uint64)).all()
    assert (H0.diag.view(np.uint64) == H1.diag.view(np.uint64)).all()


def test_free_boundaries_and_small_periodic_grid():
    # non-periodic x, tiny periodic y (2 cells of the bucket grid), displaced atoms
    w = W.CONFIGS["c2"].scaled(9, 2)
    inp = W.make_inputs(w)
    pbc = np.array([0, 1, 0], dtype=np.int32)
    c0, w0 = oracle.neighbor_counts(inp.pos, inp.box, pbc, 4.0, 0)
    c1, w1 = oracle.neighbor_counts(inp.pos, inp.box, pbc, 4.0, 1)
    assert w0 == w1 and (c0 == c1).all()
    assert c0.min() < 18  # edge atoms lose neighbours


def test_sorted_symmetric_padded():
    w = W.CONFIGS["c2"].scaled(12, 10)
    inp = W.make_inputs(w)
    H = _build(w, inp)
    n, K = H.n, H.width
    rows = np.arange(n)
    counts, _ = oracle.neighbor_counts(inp.pos, inp.box, inp.pbc, w.cutoff, 1)
    for i in range(n):
        c = H.cols[:counts[i], i]
        assert (np.diff(c) > 0).all() and (c != i).all()       # ascending, no self, no repeats
        assert (H.cols[counts[i]:, i] == i).all()              # padding: col = i
        assert (H.vals[counts[i]:, i] == 0.0).all() and not np.signbit(H.vals[counts[i]:, i]).any()
    dense = H.to_dense()
    assert (dense == dense.T).all()                            # H = H^T bit-exact (P8)
    assert K == counts.max()
    assert np.allclose(np.diag(dense), inp.onsite_shift)       # eps_i = onsite[s_i] + shift_i
    assert (H.diag == w.onsite[0] + inp.onsite_shift).all()
    del rows


def test_hopping_law_on_hand_placed_atoms(golden):
    # t(r) = t0 exp(-beta (r/r0 - 1)) (BASELINE.json:configs[1]); t(r0) = t0 exactly, and
    # the 2nd/3rd/4th-shell values printed in SURVEY.md A8.
    feats = {r[0]: (float(r[1]), float(r[2])) for r in golden("graphene_dos_features.txt")}
    a = W.A_CC
    box = np.array([50.0, 50.0, 50.0])
    pbc = np.zeros(3, dtype=np.int32)
    for r, key in ((a, None), (math.sqrt(3) * a, "t_shell2"), (2 * a, "t_shell3"),
                   (math.sqrt(7) * a, "t_shell4")):
        pos = np.array([[10.0, 10.0, 10.0], [10.0 + r, 10.0, 10.0]])
        H = oracle.build_hamiltonian(pos, [0, 0], box, pbc, 4.0, [0.0], [-2.7], r0=a, beta=3.37,
                                     method=0)
        assert H.width == 1 and H.cols[0, 0] == 1 and H.cols[0, 1] == 0
        assert H.vals[0, 0] == H.vals[0, 1]
        if key is None:
            assert H.vals[0, 0] == pytest.approx(-2.7, abs=1e-15)
        else:
            assert abs(H.vals[0, 0] - feats[key][0]) < feats[key][1]
    # beta = 0 -> constant
    H = oracle.build_hamiltonian(pos, [0, 0], box, pbc, 4.0, [0.0], [-2.7], beta=0.0, method=0)
    assert H.vals[0, 0] == -2.7


def test_min_image_and_strict_cutoff():
    box = np.array([10.0, 10.0, 10.0])
    pbc = np.array([1, 1, 1], dtype=np.int32)
    # two atoms 1.0 apart through the periodic boundary (unwrapped coordinates, one outside the box)
    pos = np.array([[0.25, 5.0, 5.0], [9.25, 5.0, 5.0], [-10.5, 5.0, 5.0]])
    counts, _ = oracle.neighbor_counts(pos, box, pbc, 1.5, 0)
    assert counts.tolist() == [2, 2, 2]            # 0-1: 1.0, 0-2: 0.75 (image), 1-2: 0.25 (image)
    counts1, _ = oracle.neighbor_counts(pos, box, pbc, 1.5, 1)
    assert counts1.tolist() == [2, 2, 2]
    # strict '<': a pair at exactly the cutoff is not a neighbour
    pos = np.array([[1.0, 1.0, 1.0], [3.0, 1.0, 1.0]])
    for method in (0, 1):
        c, _ = oracle.neighbor_counts(pos, box, pbc, 2.0, method)
        assert c.tolist() == [0, 0]
        c, _ = oracle.neighbor_counts(pos, box, pbc, 2.0000001, method)
        assert c.tolist() == [1, 1]
    # periodic length below 2 r_c is refused (A20)
    with pytest.raises(oracle.OracleError) as e:
        oracle.neighbor_counts(pos, box, pbc, 5.5, 0)
    assert e.value.status == oracle.ERR_BOX_TOO_SMALL


def test_ell_overflow_reported():
    w = W.CONFIGS["c1"].scaled(6, 4)
    inp = W.make_inputs(w)
    with pytest.raises(oracle.OracleError) as e:
        _build(w, inp, width=2)
    assert e.value.status == oracle.ERR_ELL_OVERFLOW


def test_hbn_graphene_bond_census():
    # P9 scaled down: n_stripes interfaces, each with one C-B and one C-N bond per cell row;
    # C-C and B-N share the rest equally; total bonds = 3N/2.
    stripe, n_stripes, ny = 5, 4, 6
    w = W.CONFIGS["c4"].scaled(stripe * n_stripes, ny, stripe=stripe)
    inp = W.make_inputs(w)
    H = _build(w, inp)
    assert H.width == 3
    n = H.n
    bonds = {t: int((H.vals == t).sum()) // 2 for t in (-2.7, -2.6, -2.5, -2.8)}
    assert bonds[-2.5] == n_stripes * ny and bonds[-2.8] == n_stripes * ny
    assert bonds[-2.7] == bonds[-2.6] == (3 * n // 2 - 2 * n_stripes * ny) // 2
    assert sum(bonds.values()) == 3 * n // 2
    assert H.diag.sum() == 0.0 and set(np.unique(H.diag)) == {-2.3, 0.0, 2.3}
    # full-size checksum of P9 follows from the same census: 23.72016 at 1000x250, stripe 125
    full = (748000 * 2 * 2.7**2 + 748000 * 2 * 2.6**2 + 2000 * 2 * 2.5**2 + 2000 * 2 * 2.8**2
            + 500000 * 2.3**2) / 1e6
    assert full == pytest.approx(23.72016, abs=1e-9)


def test_gershgorin_bounds_contain_spectrum():
    w = W.CONFIGS["c2b"].scaled(8, 6)
    inp = W.make_inputs(w)
    H = _build(w, inp)
    lo, hi = oracle.spectral_bounds(H)
    ev = np.linalg.eigvalsh(H.to_dense())
    assert lo <= ev[0] and ev[-1] <= hi
    # and they are the row-sum bounds of the dense matrix (library re-computation)
    dense = H.to_dense()
    off = np.abs(dense).sum(1) - np.abs(np.diag(dense))
    assert lo == pytest.approx((np.diag(dense) - off).min(), rel=1e-14)
    assert hi == pytest.approx((np.diag(dense) + off).max(), rel=1e-14)


def test_tile_major_numbering_is_the_same_structure():
    """workloads.make_inputs(tile=...) renumbers the atoms and nothing else: the same set of atoms (positions,
    species, onsite shifts), every block of tx x ty cells contiguous, and the exact-trace moments -- which do not
    depend on the order of the rows -- unchanged."""
    w = W.CONFIGS["c4"].scaled(16, 12, stripe=4, M=24)
    a, t = W.make_inputs(w), W.make_inputs(w, tile=(4, 3))
    ka, kt = np.lexsort(a.pos.T), np.lexsort(t.pos.T)
    assert np.array_equal(a.pos[ka], t.pos[kt]) and np.array_equal(a.species[ka], t.species[kt])
    assert not np.array_equal(a.pos, t.pos)
    # the first 4 x 3 x 4 atoms are the first block of cells (disorder << cell size)
    first = t.pos[: 4 * 3 * 4]
    assert first[:, 0].max() < 4 * W.LX and first[:, 1].max() < 3 * W.LY
    mus = []
    for inp in (a, t):
        H = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0,
                                     w.beta, inp.onsite_shift)
        mus.append(oracle.kpm_moments(H, w.a, w.b, w.M, mode=1))
    np.testing.assert_allclose(mus[0], mus[1], rtol=0, atol=1e-13)
