"""GPU check of the 1-D strip decomposition (csrc/strips.cu) on one device: the
partitioned run must reproduce the unpartitioned one -- last Chebyshev vector bit for bit, moments to the order
of the block sums -- and the oracle's moments."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


@pytest.mark.parametrize("key,nx,ny,R,P", [("c5", 57, 43, 2, 2), ("c5", 57, 43, 2, 5), ("c4", 48, 21, 8, 3),
                                           ("c2", 37, 29, 8, 2), ("c2b", 41, 31, 4, 4), ("c1", 24, 24, 3, 2),
                                           ("c5", 300, 9, 2, 1)])
def test_strips_reproduce_the_unpartitioned_run(key, nx, ny, R, P):
    kw = {"stripe": 6} if key == "c4" else {}
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta,
                                  inp.onsite_shift, with_diag=w.use_diag)
    shift = _dev(inp.onsite_shift) if inp.onsite_shift is not None else None
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                               w.r0, w.beta, shift, with_diag=w.use_diag)
    if w.a is not None:
        a, b = w.a, w.b
    else:
        lo, hi = oracle.spectral_bounds(Ho)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    n = Ho.n
    halo = gtb.ring_halo(Hg)
    d = np.abs(Ho.cols - np.arange(n)[None, :])
    assert halo == int(np.minimum(d, n - d).max())
    M = 33
    S = (M + 1) // 2
    mu, phi = gtb.kpm_moments_strips(Hg, P, a, b, M, R, R, 5, want_phi=True, check=True)
    ref = oracle.kpm_moments(Ho, a, b, M, R, 5, mode=0, algo=0)
    one = gtb.kpm_moments(Hg, a, b, M, R, R, 5, check=True).cpu().numpy()
    assert np.abs(mu.cpu().numpy() - ref).max() <= 1e-12
    assert np.abs(mu.cpu().numpy() - one).max() <= 1e-13
    # phi_S of the unpartitioned recursion, pass by pass through gtb_kpm_step
    cur = gtb.random_phase_fill(5, 0, R, n)
    io = torch.empty_like(cur)
    for k in range(S):
        gtb.kpm_step(Hg, a, b, k == 0, cur, io)
        cur, io = io, cur
    assert torch.equal(phi, cur)
    exact, _ = gtb.kpm_moments_strips(Hg, P, a, b, 12, mode=1, R_batch=8)
    plain = gtb.kpm_moments(Hg, a, b, 12, mode=1, R_batch=8).cpu().numpy()
    assert np.abs(exact.cpu().numpy() - plain).max() <= 1e-13


def test_strips_narrower_than_the_halo_are_refused():
    w = W.CONFIGS["c5"].scaled(57, 43)
    inp = W.make_inputs(w)
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                               with_diag=False)
    with pytest.raises(gtb.GtbError):
        gtb.kpm_moments_strips(Hg, 64, 8.5, 0.0, 8, 2, 2, 5)      # 9804 rows / 64 = 152 < halo 228
