"""gtb_pair_slots (csrc/pairslots.cu): the same matrix as a plain ELL whose rows keep their entries in a slot order
that suits the 64-byte gathers of an R = 4 pass (rows 2q, 2q + 1 alternate in column parity).  It must be the same
matrix -- every row a permutation of the original row, padding slots unchanged in kind -- and every pass must
reproduce the oracle on it."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _both(w, inp):
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta,
                                  inp.onsite_shift)
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0,
                               w.beta, _dev(inp.onsite_shift) if inp.onsite_shift is not None else None)
    return Ho, Hg


def _same_parity(cols):
    a, b = cols[:, 0:-1:2], cols[:, 1::2]
    return float(((a & 1) == (b & 1)).mean())


@pytest.mark.parametrize("key,nx,ny", [("c3b", 53, 41), ("c3", 37, 29), ("c4", 48, 21)])
def test_paired_slots_are_the_same_matrix_and_run_to_the_oracle(key, nx, ny):
    kw = {"stripe": 6} if key == "c4" else {}
    w = W.CONFIGS[key].scaled(nx, ny, R=4, **kw)
    inp = W.make_inputs(w)
    Ho, Hg = _both(w, inp)
    Hp = gtb.pair_slots(Hg, 4)
    n, K = Ho.n, Ho.width
    c0, v0 = Hg.cols.cpu().numpy(), Hg.vals.cpu().numpy()
    c1, v1 = Hp.cols.cpu().numpy(), Hp.vals.cpu().numpy()
    assert c1.shape == (K, n) and Hp.diag is Hg.diag
    # every row: the same multiset of (column, value) pairs; padding stays (column = row, value 0)
    o0, o1 = np.lexsort((v0, c0), axis=0), np.lexsort((v1, c1), axis=0)
    assert np.array_equal(np.take_along_axis(c0, o0, 0), np.take_along_axis(c1, o1, 0))
    assert np.array_equal(np.take_along_axis(v0, o0, 0), np.take_along_axis(v1, o1, 0))
    pad = c1 == np.arange(n)[None, :]
    assert (v1[pad] == 0.0).all()
    assert _same_parity(c1) <= 0.5 * _same_parity(c0) + 0.02       # what the re-ordering is for
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    R = 4
    phi0 = oracle.random_phase_fill(11, 0, R, n)
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, np.arange(n))
    for opt in (gtb.options(kernel=gtb.KERNEL_TILE), gtb.options(kernel=gtb.KERNEL_ROW), None):
        g0, g1 = _dev(phi0), torch.empty((n, R, 2), dtype=torch.float64, device="cuda")
        gtb.kpm_step(Hp, a, b, True, g0, g1, opt=opt)
        assert np.abs(g1.cpu().numpy() - phi1).max() <= 1e-14
    M = 65
    got = gtb.kpm_moments(Hp, a, b, M, 2 * R, R, 5, check=True).cpu().numpy()
    ref = oracle.kpm_moments(Ho, a, b, M, 2 * R, 5, mode=0, algo=0)
    assert np.abs(got - ref).max() <= 1e-12
    # the windowed and the bounds paths take it like any other ELL
    lo2, hi2 = gtb.spectral_bounds(Hp).tolist()
    assert lo2 == pytest.approx(lo, rel=1e-14) and hi2 == pytest.approx(hi, rel=1e-14)


@pytest.mark.parametrize("key,nx,ny,diag", [("c5", 57, 43, False), ("c4", 48, 21, True), ("c1", 24, 24, False)])
def test_quads_of_rows_at_two_vectors_per_pass(key, nx, ny, diag):
    """R = 2: the slots of rows 4q .. 4q + 3 are permuted so that the four gathered columns differ in their two low
    bits; same matrix, same results through the plain and the packed pass."""
    kw = {"stripe": 6} if key == "c4" else {}
    w = W.CONFIGS[key].scaled(nx, ny, R=2, **kw)
    inp = W.make_inputs(w)
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta,
                                  inp.onsite_shift, with_diag=diag)
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0,
                               w.beta, _dev(inp.onsite_shift) if inp.onsite_shift is not None else None,
                               with_diag=diag)
    Hq = gtb.pair_slots(Hg, 2)
    n, K = Ho.n, Ho.width
    assert K <= 4 and n % 4 == 0
    c0, v0 = Hg.cols.cpu().numpy(), Hg.vals.cpu().numpy()
    c1, v1 = Hq.cols.cpu().numpy(), Hq.vals.cpu().numpy()
    o0, o1 = np.lexsort((v0, c0), axis=0), np.lexsort((v1, c1), axis=0)
    assert np.array_equal(np.take_along_axis(c0, o0, 0), np.take_along_axis(c1, o1, 0))
    assert np.array_equal(np.take_along_axis(v0, o0, 0), np.take_along_axis(v1, o1, 0))

    def distinct(c):
        s = np.sort((c & 3).reshape(K, n // 4, 4), axis=2)
        return float((np.diff(s, axis=2) != 0).all(axis=2).mean())
    assert distinct(c1) >= 0.95 and distinct(c0) <= 0.2
    if w.a is not None:
        a, b = w.a, w.b
    else:
        lo, hi = oracle.spectral_bounds(Ho)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    M, R = 65, 2
    ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
    got = gtb.kpm_moments(Hq, a, b, M, R, R, 5, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12
    P = gtb.pack_ell(Hq)
    assert P is not None
    got = gtb.kpm_moments(P, a, b, M, R, R, 5, mode=gtb.MODE_PACKED, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12


def test_wide_rows_at_two_vectors_per_pass_are_arranged_position_by_position():
    """R = 2, K > 4 (the neighbour lists of the s,p,d bond form): same rows, four distinct residues per quad and
    position nearly everywhere, and the moments of the oracle."""
    w = W.CONFIGS["c2b"].scaled(41, 29, R=2)
    inp = W.make_inputs(w)
    Ho, Hg = _both(w, inp)
    Hq = gtb.pair_slots(Hg, 2)
    n, K = Ho.n, Ho.width
    assert K > 4 and n % 4 == 0
    c0, v0 = Hg.cols.cpu().numpy(), Hg.vals.cpu().numpy()
    c1, v1 = Hq.cols.cpu().numpy(), Hq.vals.cpu().numpy()
    o0, o1 = np.lexsort((v0, c0), axis=0), np.lexsort((v1, c1), axis=0)
    assert np.array_equal(np.take_along_axis(c0, o0, 0), np.take_along_axis(c1, o1, 0))
    assert np.array_equal(np.take_along_axis(v0, o0, 0), np.take_along_axis(v1, o1, 0))

    def distinct(c):
        s = np.sort((c & 3).reshape(K, n // 4, 4), axis=2)
        return float((np.diff(s, axis=2) != 0).all(axis=2).mean())
    assert distinct(c1) >= 0.8 and distinct(c1) >= 4 * distinct(c0)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    ref = oracle.kpm_moments(Ho, a, b, 65, 2, 5, mode=0, algo=0)
    got = gtb.kpm_moments(Hq, a, b, 65, 2, 2, 5, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-12


@pytest.mark.parametrize("n", [1, 2, 3, 5, 6, 7, 1023])
@pytest.mark.parametrize("K,R", [(3, 2), (4, 2), (9, 2), (7, 4), (1, 4)])
def test_ragged_sizes_keep_every_row(n, K, R):
    """Row counts that are not a multiple of the group (2 or 4 rows): the last group is short; every row still
    comes out as a permutation of itself."""
    rng = np.random.default_rng(100 * n + 10 * K + R)
    cols = rng.integers(0, n, size=(K, n)).astype(np.int32)
    vals = rng.standard_normal((K, n))
    pad = rng.random((K, n)) < 0.2
    cols[pad] = np.broadcast_to(np.arange(n, dtype=np.int32), (K, n))[pad]
    vals[pad] = 0.0
    vals[cols == np.arange(n)[None, :]] = 0.0            # a slot on the diagonal is a padding slot
    H = gtb.Ell.from_host(cols, vals)
    Hp = gtb.pair_slots(H, R)
    c1, v1 = Hp.cols.cpu().numpy(), Hp.vals.cpu().numpy()
    o0, o1 = np.lexsort((vals, cols), axis=0), np.lexsort((v1, c1), axis=0)
    assert np.array_equal(np.take_along_axis(cols, o0, 0), np.take_along_axis(c1, o1, 0))
    assert np.array_equal(np.take_along_axis(vals, o0, 0), np.take_along_axis(v1, o1, 0))


def test_other_vector_counts_get_a_copy_and_bad_arguments_are_refused():
    w = W.CONFIGS["c2b"].scaled(21, 17)
    inp = W.make_inputs(w)
    _, Hg = _both(w, inp)
    Hp = gtb.pair_slots(Hg, 8)
    assert torch.equal(Hp.cols, Hg.cols) and torch.equal(Hp.vals, Hg.vals)
    hc = Hg._c()
    import ctypes as C
    assert gtb.lib().gtb_pair_slots(C.byref(hc), C.c_int32(4), C.byref(hc), None) == gtb.ERR_INVALID_ARG   # in place
    assert gtb.lib().gtb_pair_slots(C.byref(hc), C.c_int32(0), C.byref(Hp._c()), None) == gtb.ERR_INVALID_ARG
