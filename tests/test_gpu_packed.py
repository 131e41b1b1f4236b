"""GPU parity of the packed narrow-row format (csrc/packed.cu, gtb_pack_ell + GTB_MODE_PACKED; SURVEY.md
sec. 8(f) NEXT-4): 16-bit ring-relative columns and a dictionary of the distinct fp64 hoppings, decoded in
the fused pass K7x2p.  Lossless, so the pass must reproduce the plain path's vectors bit for bit and the
oracle's rows / moments to the usual tolerances."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _both(w, inp, width=None, with_diag=True):
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta,
                                  inp.onsite_shift, width=width, with_diag=with_diag)
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                               w.r0, w.beta, shift, width=width, with_diag=with_diag)
    return Ho, Hg


# (config, nx, ny, extra, width, diagonal, R): K = 3 without / with a folded diagonal, padded K = 4 with a
# separate diagonal array, a dictionary too large for shared memory (beta != 0: every hopping distinct)
CASES = [("c5", 57, 43, {}, None, False, 2), ("c5", 301, 127, {}, None, False, 2),
         ("c4", 48, 21, {"stripe": 6}, None, True, 8), ("c4", 48, 21, {"stripe": 6}, 4, True, 4),
         ("c1", 24, 24, {}, 4, False, 4), ("c4", 30, 17, {"stripe": 5, "beta": 1.3}, None, True, 2)]


@pytest.mark.parametrize("key,nx,ny,kw,width,diag,R", CASES)
def test_packed_pass_is_bit_identical_to_the_plain_pass_and_matches_the_oracle(key, nx, ny, kw, width, diag, R):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    Ho, Hg = _both(w, inp, width=width, with_diag=diag)
    P = gtb.pack_ell(Hg)
    assert P is not None and (P.width & 0xff) == Ho.width
    # 8-byte rows when K <= 3 and the dictionary has at most 16 entries, else 16-byte rows
    assert P.short_rows == (Ho.width <= 3 and P.n_values <= 16) and P.short_rows == bool(P.width & 0x100)
    assert (P.diag is None) == (not diag or Ho.width <= 3)
    if kw.get("beta"):
        assert P.n_values > 1024                       # dictionary read from global memory
    else:
        assert P.n_values <= 8
    n = Ho.n
    if w.a is not None and not kw.get("beta"):
        a, b = w.a, w.b
    else:
        lo, hi = oracle.spectral_bounds(Ho)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    phi0 = oracle.random_phase_fill(11, 0, R, n)
    rows = np.arange(n) if n < 20000 else np.unique(np.r_[0:300, n - 300:n, np.arange(0, n, 97)])
    phi1 = oracle.kpm_step_rows(Ho, a, b, True, None, phi0, np.arange(n))
    phi2 = oracle.kpm_step_rows(Ho, a, b, False, phi0, phi1, rows)
    plain = gtb.options(kernel=gtb.KERNEL_ROW_X2)
    g0, g1 = _dev(phi0), torch.empty((n, R, 2), dtype=torch.float64, device="cuda")
    gtb.kpm_step(P, a, b, True, g0, g1, mode=gtb.MODE_PACKED)
    assert np.abs(g1.cpu().numpy() - phi1).max() <= 1e-14
    q1 = torch.empty_like(g1)
    gtb.kpm_step(Hg, a, b, True, g0, q1, opt=plain)
    assert torch.equal(g1, q1)
    g1, g0p, g0q = _dev(phi1), _dev(phi0), _dev(phi0)
    s = gtb.kpm_step(P, a, b, False, g1, g0p, mode=gtb.MODE_PACKED).cpu().numpy()          # g0p <- phi_2
    gtb.kpm_step(Hg, a, b, False, g1, g0q, opt=plain)
    assert torch.equal(g0p, g0q)                                                          # lossless
    assert np.abs(g0p.cpu().numpy()[rows] - phi2).max() <= 1e-14
    assert s[0] == pytest.approx((phi1 * phi1).sum(), rel=1e-13)
    M = 65
    got = gtb.kpm_moments(P, a, b, M, R, R, 5, mode=gtb.MODE_PACKED, check=True).cpu().numpy()
    old = gtb.kpm_moments(Hg, a, b, M, R, R, 5, opt=plain, check=True).cpu().numpy()
    assert np.abs(got - old).max() <= 1e-13
    if n < 20000:
        ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
        assert np.abs(got - ref).max() <= 1e-12
    exact = gtb.kpm_moments(P, a, b, 16, mode=1 | gtb.MODE_PACKED, R_batch=8).cpu().numpy()
    plain_exact = gtb.kpm_moments(Hg, a, b, 16, mode=1, R_batch=8).cpu().numpy()
    assert np.abs(exact - plain_exact).max() <= 1e-13


def test_matrices_that_do_not_fit_stay_on_the_plain_path():
    # wide rows
    w = W.CONFIGS["c2b"].scaled(9, 7)
    _, Hg = _both(w, W.make_inputs(w))
    assert Hg.width > 4 and gtb.pack_ell(Hg) is None
    # more than 65535 distinct hoppings
    w = W.CONFIGS["c4"].scaled(150, 100, stripe=25, beta=1.3)
    _, Hg = _both(w, W.make_inputs(w))
    assert Hg.width <= 4 and gtb.pack_ell(Hg) is None
    # a neighbour more than 32767 rows away on the ring (4 nx = 36000 rows between cell rows, n/2 with ny = 2)
    w = W.CONFIGS["c5"].scaled(9000, 2)
    _, Hg = _both(w, W.make_inputs(w), with_diag=False)
    assert gtb.pack_ell(Hg) is None
    # ... and just inside the range
    w = W.CONFIGS["c5"].scaled(8000, 3)
    _, Hg = _both(w, W.make_inputs(w), with_diag=False)
    assert gtb.pack_ell(Hg) is not None
    with pytest.raises(gtb.GtbError):                        # R_batch must be 2, 4 or 8
        gtb.kpm_moments(gtb.pack_ell(Hg), 8.5, 0.0, 8, 3, 3, 5, mode=gtb.MODE_PACKED)
