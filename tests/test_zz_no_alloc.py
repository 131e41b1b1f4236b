"""gtb_kpm_moments_static (include/gtb.h): the Chebyshev moments with the scratch in the library's static device
array, for callers that cannot allocate.  Its output must equal the existing path's (gtb_kpm_moments with a
caller-owned workspace) -- same kernels on the same inputs -- on two calls in a row, although the second call
finds the first call's contents in the shared array; and it must equal the oracle's moments within the tolerance
of tests/test_gpu_parity.py.  A run that needs more than GTB_STATIC_WS_BYTES is refused before anything is
launched.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = 1e-12     # the moment tolerance of tests/test_gpu_parity.py


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _pair(w):
    inp = W.make_inputs(w)
    Ho = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0, w.beta,
                                  inp.onsite_shift, with_diag=w.use_diag)
    Hg = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0,
                               w.beta, _dev(inp.onsite_shift) if inp.onsite_shift is not None else None,
                               with_diag=w.use_diag)
    return Ho, Hg


def test_static_scratch_equals_the_workspace_path_twice_in_a_row():
    w1 = W.CONFIGS["c1"]                                  # 2304 atoms, M = 256, R = 4: 2.7 MiB of scratch
    w2 = W.CONFIGS["c2b"].scaled(23, 17, M=96, R=8)       # another size, width, R and kernel right behind it
    for w, seed in ((w1, 7), (w2, 11), (w1, 7)):
        Ho, Hg = _pair(w)
        if w.a is not None:
            a, b = w.a, w.b
        else:
            lo, hi = oracle.spectral_bounds(Ho)
            a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
        assert gtb.kpm_workspace_bytes(Ho.n, w.M, w.R) <= gtb.STATIC_WS_BYTES
        want = gtb.kpm_moments(Hg, a, b, w.M, w.R, w.R, seed, check=True)
        mu = torch.full((w.M,), float("nan"), dtype=torch.float64, device="cuda")
        got1 = gtb.kpm_moments_static(Hg, a, b, w.M, w.R, w.R, seed, mu=mu).clone()
        got2 = gtb.kpm_moments_static(Hg, a, b, w.M, w.R, w.R, seed, mu=mu).clone()
        torch.cuda.synchronize()
        assert torch.isfinite(got1).all()
        assert (got1 - want).abs().max().item() <= TOL and (got2 - want).abs().max().item() <= TOL
        assert torch.equal(got1, want) and torch.equal(got2, want)      # same kernels, same inputs: same bits
        ref = oracle.kpm_moments(Ho, a, b, w.M, w.R, seed, mode=0, algo=0)
        assert np.abs(got2.cpu().numpy() - ref).max() <= TOL
    # exact-trace mode through the same array (basis vectors in batches of 8, the last one ragged)
    wt = W.CONFIGS["c1"].scaled(5, 3, M=40)
    Ho, Hg = _pair(wt)
    want = gtb.kpm_moments(Hg, wt.a, wt.b, wt.M, 1, 8, 0, mode=1, check=True)
    got = gtb.kpm_moments_static(Hg, wt.a, wt.b, wt.M, 1, 8, 0, mode=1)
    assert torch.equal(got, want)
    assert np.abs(got.cpu().numpy() - oracle.kpm_moments(Ho, wt.a, wt.b, wt.M, mode=1)).max() <= TOL


def test_static_scratch_refuses_what_does_not_fit():
    w = W.CONFIGS["c1"].scaled(64, 64)                    # 16384 atoms x R = 8: the vectors alone are 4 MiB
    _, Hg = _pair(w)
    assert gtb.kpm_workspace_bytes(Hg.n, 64, 8) > gtb.STATIC_WS_BYTES
    mu = torch.full((64,), 3.0, dtype=torch.float64, device="cuda")
    before = gtb.launch_count()
    with pytest.raises(gtb.GtbError) as err:
        gtb.kpm_moments_static(Hg, w.a, w.b, 64, 8, 8, 1, mu=mu)
    assert err.value.status == gtb.ERR_STATIC_LIMIT and "GTB_STATIC_WS_BYTES" in str(err.value)
    assert gtb.launch_count() == before and bool((mu == 3.0).all())     # nothing ran, nothing was written
    w1 = W.CONFIGS["c1"]
    _, H1 = _pair(w1)
    with pytest.raises(gtb.GtbError) as err:              # fits in atoms, not in moments (the per-pass partial sums)
        gtb.kpm_moments_static(H1, w1.a, w1.b, 4096, 4, 4, 1)
    assert err.value.status == gtb.ERR_STATIC_LIMIT
