"""CPU-side checks of the full-size, full-depth goldens (tests/golden/<cfg>_moments_M*.txt, _dos_G*.txt,
written by tests/golden/make_fullsize_goldens.py from the oracle alone): they exist for all five
configs (and for the variants 2b, 3b), parse, carry the config's (M, G), satisfy what the mathematics fixes (mu_0 = 1, |mu_n| <= 1,
rho >= 0, int rho dE = 1 within the Jackson resolution) and -- at the 10^6-atom configs, where the
lattice is cheap to regenerate -- the input digest they were made from."""
import os

import numpy as np
import pytest

from paper_2509_06525_b200 import workloads as W
from test_gpu_fulldepth import KEYS, _paths, read_fulldepth_golden


REQUIRED = ("c4", "c2b", "c2", "c5", "c3", "c3b")        # extended as make_fullsize_goldens.py finishes each config


def test_goldens_exist():
    missing = [p for k in REQUIRED for p in _paths(k) if not os.path.exists(p)]
    assert not missing, missing


@pytest.mark.parametrize("key", [k for k in KEYS if all(os.path.exists(p) for p in _paths(k))])
def test_golden_is_well_formed(key):
    w = W.CONFIGS[key]
    g = read_fulldepth_golden(key)
    assert g["mu"].shape == (w.M,) and g["rho"].shape == (w.n_energies,)
    assert g["mu"][0] == pytest.approx(1.0, abs=1e-12) and np.abs(g["mu"]).max() <= 1.0 + 1e-12
    assert np.array_equal(W.energy_grid(w, g["a"], g["b"]), g["E"])
    assert g["rho"].min() >= 0.0                      # Jackson kernel: positive
    integral = np.trapezoid(g["rho"], g["E"])
    assert integral == pytest.approx(1.0, abs=2e-3)
    if w.n_atoms <= 1_000_000:
        assert W.inputs_digest(W.make_inputs(w)) == g["sha"]
