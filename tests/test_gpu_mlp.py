"""GPU parity of the descriptor + MLP Hamiltonian (Eq. 2; NEXT-3) against
oracle/gtbo_mlp.cpp, then the unchanged KPM path on the result.  Tolerance: 1e-12 relative to the largest
|t| (a cos, a sqrt, 2 Hd exps of another libm, FMA contraction over ~500 terms); moments 1e-9."""
import numpy as np
import pytest
import torch

import oracle
from paper_2509_06525_b200 import binding as gtb
from paper_2509_06525_b200 import workloads as W

pytestmark = pytest.mark.gpu
DIMS, RC = W.MLP_DIMS, 2.0


def _dev(x):
    return torch.as_tensor(np.ascontiguousarray(x)).cuda()


def _both(key, nx, ny, cutoff, seed=65250, **kw):
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    ns = len(w.onsite)
    blob = W.mlp_weights(DIMS, seed)
    ones = np.ones((ns, ns))
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                     with_diag=False, method=1)
    Ho, vo = oracle.mlp_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC, blob,
                                    return_v=True)
    nbr_g = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, cutoff, [0.0] * ns,
                                  ones, with_diag=False)
    Hg, vg = gtb.mlp_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, DIMS, RC,
                                 _dev(blob), return_v=True)
    return w, inp, Ho, vo, Hg, vg


CASES = [("c1", 24, 24, 1.95, {}), ("c2", 37, 23, 1.95, {}), ("c2b", 21, 13, 1.99, {}),
         ("c4", 48, 21, 1.95, {"stripe": 6})]


@pytest.mark.parametrize("key,nx,ny,cutoff,kw", CASES)
def test_features_hoppings_and_onsite_match_oracle(key, nx, ny, cutoff, kw):
    w, inp, Ho, vo, Hg, vg = _both(key, nx, ny, cutoff, **kw)
    assert np.abs(vg.cpu().numpy() - vo).max() <= 1e-13 * max(1.0, np.abs(vo).max())
    scale = np.abs(Ho.vals).max()
    assert scale > 1e-2
    assert np.abs(Hg.vals.cpu().numpy() - Ho.vals).max() <= 1e-12 * scale
    assert np.abs(Hg.diag.cpu().numpy() - Ho.diag).max() <= 1e-12 * max(1.0, np.abs(Ho.diag).max())
    pad = Ho.cols == np.arange(Ho.n)[None, :]
    assert (Hg.vals.cpu().numpy()[pad] == 0).all()


@pytest.mark.parametrize("key,nx,ny,cutoff,kw", CASES[1:])
def test_moments_on_the_mlp_hamiltonian(key, nx, ny, cutoff, kw):
    w, inp, Ho, vo, Hg, vg = _both(key, nx, ny, cutoff, seed=7, **kw)
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    ref = oracle.kpm_moments(Ho, a, b, 96, 4, 13, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, 96, 4, 4, 13, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-9
    assert np.abs(got - ref).max() <= 1e-11


def test_other_instantiated_sizes_and_rejections():
    w = W.CONFIGS["c2"].scaled(9, 7)
    inp = W.make_inputs(w)
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, 1.95, [0.0], [1.0],
                                     with_diag=False, method=1)
    nbr_g = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, 1.95, [0.0], [1.0],
                                  with_diag=False)
    for dims in [(1, 4, 4, 8), (2, 16, 8, 32)]:
        blob = W.mlp_weights(dims, 3)
        Ho = oracle.mlp_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, dims, RC, blob)
        Hg = gtb.mlp_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, dims, RC, _dev(blob))
        assert np.abs(Hg.vals.cpu().numpy() - Ho.vals).max() <= 1e-12 * np.abs(Ho.vals).max()
        assert np.abs(Hg.diag.cpu().numpy() - Ho.diag).max() <= 1e-12 * max(1.0, np.abs(Ho.diag).max())
    with pytest.raises(gtb.GtbError):            # sizes that are not instantiated
        gtb.mlp_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, (1, 5, 5, 7), RC,
                            _dev(W.mlp_weights((1, 5, 5, 7), 3)))
    with pytest.raises(gtb.GtbError):            # wrong blob length
        gtb.mlp_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, (1, 8, 8, 16), RC,
                            _dev(np.zeros(10)))
    bad = inp.species.copy()
    bad[3] = 5
    with pytest.raises(gtb.GtbError):            # species out of range is reported, not dereferenced
        gtb.mlp_hamiltonian(nbr_g, _dev(inp.pos), _dev(bad), inp.box, inp.pbc, (1, 8, 8, 16), RC,
                            _dev(W.mlp_weights((1, 8, 8, 16), 3)))


@pytest.mark.parametrize("key,nx,ny,cutoff,kw", CASES)
def test_mlp_feeding_the_slater_koster_blocks(key, nx, ny, cutoff, kw):
    """Eq. 2 -> four bond integrals per pair -> s,p blocks; then moments with the blocked pass."""
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    ns = len(w.onsite)
    blob = W.mlp_weights(DIMS, 21, hop_out=4, onsite_out=2)
    ones = np.ones((ns, ns))
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                     with_diag=False, method=1)
    Ho = oracle.mlp_sk_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, DIMS, RC, blob)
    nbr_g = gtb.build_hamiltonian(_dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, cutoff, [0.0] * ns,
                                  ones, with_diag=False)
    Hg = gtb.mlp_sk_hamiltonian(nbr_g, _dev(inp.pos), _dev(inp.species), inp.box, inp.pbc, DIMS, RC, _dev(blob))
    assert (Hg.cols.cpu().numpy() == Ho.cols).all()
    scale = np.abs(Ho.vals).max()
    assert np.abs(Hg.vals.cpu().numpy() - Ho.vals).max() <= 1e-12 * scale
    assert np.abs(Hg.diag.cpu().numpy() - Ho.diag).max() <= 1e-12 * max(1.0, np.abs(Ho.diag).max())
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    ref = oracle.kpm_moments(Ho, a, b, 48, 4, 3, mode=0, algo=0)
    got = gtb.kpm_moments(Hg, a, b, 48, 4, 4, 3, mode=gtb.MODE_ORB4, check=True).cpu().numpy()
    assert np.abs(got - ref).max() <= 1e-9 and np.abs(got - ref).max() <= 1e-11


# ---- Eq. 2 feeding the s,p,d blocks (ten-output MLP_lambda, reading E7): blocks and blocked moments ----------
@pytest.mark.parametrize("key,nx,ny,kw,cutoff", [("c2b", 9, 7, {}, 2.65), ("c4", 12, 5, {"stripe": 3}, 1.95),
                                                 ("c5", 11, 9, {}, 3.0)])
def test_mlp_spd_blocks_and_moments_match_the_oracle(key, nx, ny, kw, cutoff):
    import numpy as np, torch
    w = W.CONFIGS[key].scaled(nx, ny, **kw)
    inp = W.make_inputs(w)
    ns = len(w.onsite)
    dims = (3, 8, 8, 16)
    blob = W.mlp_weights(dims, 23, hop_out=10, onsite_out=3)
    r_cut = max(2.0, 1.05 * cutoff)
    ones = np.ones((ns, ns))
    nbr_o = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                     with_diag=False)
    Ho = oracle.mlp_spd_hamiltonian(nbr_o, inp.pos, inp.species, inp.box, inp.pbc, dims, r_cut, blob)
    dev = lambda x: torch.as_tensor(np.ascontiguousarray(x)).cuda()
    nbr_g = gtb.build_hamiltonian(dev(inp.pos), dev(inp.species), inp.box, inp.pbc, cutoff, [0.0] * ns, ones,
                                  with_diag=False)
    Hb = gtb.mlp_spd_blocks(nbr_g, dev(inp.pos), dev(inp.species), inp.box, inp.pbc, dims, r_cut, dev(blob))
    n, K = nbr_o.n, nbr_o.width
    got = Hb.vals.cpu().numpy().reshape(K, 9, 9, n)                      # [k][nu][mu][i]
    want = Ho.vals.reshape(K, 9, n, 9).transpose(0, 1, 3, 2)
    scale = max(np.abs(want).max(), 1.0)
    assert np.abs(got - want).max() <= 1e-12 * scale
    assert np.abs(Hb.diag.cpu().numpy() - Ho.diag.reshape(n, 9).T).max() <= 1e-12 * scale
    lo, hi = oracle.spectral_bounds(Ho)
    a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    bounds = gtb.spd_bounds(Hb, gtb.MODE_BLOCK9).cpu().numpy()
    assert bounds[0] == pytest.approx(lo, rel=1e-11) and bounds[1] == pytest.approx(hi, rel=1e-11)
    for R in (2, 8):
        ref = oracle.kpm_moments(Ho, a, b, 33, R, 5, mode=0, algo=0)
        mu = gtb.kpm_moments(Hb, a, b, 33, R, R, 5, mode=gtb.MODE_BLOCK9, check=True).cpu().numpy()
        assert np.abs(mu - ref).max() <= 1e-9
        assert np.abs(mu - ref).max() <= 1e-11
