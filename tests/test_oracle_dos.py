"""Pins for the oracle's Jackson-damped DOS reconstruction (Eq. 4; C6).

Pins: Chebyshev orthogonality through scipy's DCT (recovers g_n mu_n from rho on the
Chebyshev nodes), the textbook variance of the Jackson-broadened delta, positivity,
normalisation, and the graphene features printed in SURVEY.md sec. 8(c) P11.
"""
import numpy as np
import pytest
from scipy.fft import dct

import oracle
from paper_2509_06525_b200 import workloads as W


def test_jackson_kernel_known_values():
    for M in (2, 17, 256, 3000):
        g = oracle.jackson(M)
        assert g[0] == pytest.approx(1.0, abs=1e-15)
        # n = 1 collapses to cos(pi/(M+1)):  [M cos q + sin q cot q]/(M+1) = cos q
        assert g[1] == pytest.approx(np.cos(np.pi / (M + 1)), abs=1e-15)
        assert (np.diff(g) < 0).all() and g[-1] > 0.0          # decreasing to ~0, positive
        assert g[-1] < 4.0 / M


@pytest.mark.parametrize("kernel", [0, 1])
def test_dct_recovers_damped_moments(kernel):
    # rho(x) pi a sqrt(1-x^2) = g_0 mu_0 + 2 sum g_n mu_n T_n(x).  On the G Chebyshev nodes
    # x_k = cos(pi (k+1/2)/G) a type-II DCT inverts this exactly for M <= G.
    M, G, a, b, scale = 60, 128, 7.5, -1.25, 3.0
    rng = np.random.default_rng(3)
    mu = rng.uniform(-1, 1, M)
    theta = np.pi * (np.arange(G) + 0.5) / G
    E = a * np.cos(theta) + b
    rho = oracle.dos(mu, a, b, E, kernel=kernel, scale=scale)
    p = rho * np.pi * a * np.sin(theta) / scale
    coef = dct(p, type=2) / G                               # = 2 g_n mu_n (n>=1), 2 g_0 mu_0 (n=0)
    g = oracle.jackson(M) if kernel == 1 else np.ones(M)
    assert coef[0] / 2 == pytest.approx(mu[0], abs=1e-13)
    assert np.abs(coef[1:M] / 2 - g[1:] * mu[1:]).max() < 1e-13
    assert np.abs(coef[M:]).max() < 1e-13                   # no higher harmonics


def test_zero_outside_the_band_and_at_the_edges():
    mu = np.array([1.0, 0.2, -0.1])
    E = np.array([-8.5, -8.500001, 8.5, 9.0, 0.0])
    rho = oracle.dos(mu, 8.5, 0.0, E)
    assert (rho[:4] == 0.0).all() and rho[4] > 0.0          # A13: rho = 0 for |x| >= 1


def test_jackson_broadened_delta_is_positive_normalised_and_has_textbook_width():
    # moments of delta(x - x0) are T_n(x0).  Jackson kernel: positive, integral 1, variance
    # sigma^2 = [M - x0^2 (M-1)] / [2(M+1)] * (1 - cos(2 pi/(M+1)))   (Weisse et al. 2006)
    M, a = 200, 1.0
    G = 4096
    theta = np.pi * (np.arange(G) + 0.5) / G
    x = np.cos(theta)
    for x0 in (0.0, 0.37, -0.8):
        mu = np.cos(np.arange(M) * np.arccos(x0))
        rho = oracle.dos(mu, a, 0.0, x, kernel=1)
        assert rho.min() > -1e-13
        wq = np.pi * np.sin(theta) / G                      # Chebyshev-Gauss weights for dx
        assert (rho * wq).sum() == pytest.approx(1.0, abs=1e-12)
        mean = (rho * x * wq).sum()
        var = (rho * x * x * wq).sum() - mean**2
        expect = (M - x0**2 * (M - 1)) / (2.0 * (M + 1)) * (1 - np.cos(2 * np.pi / (M + 1)))
        assert var == pytest.approx(expect, rel=1e-9)
        dirichlet = oracle.dos(mu, a, 0.0, x, kernel=0)
        assert dirichlet.min() < -0.1                       # without the kernel: Gibbs ringing


def test_graphene_dos_features(golden):
    feats = {r[0]: (float(r[1]), float(r[2])) for r in golden("graphene_dos_features.txt")}
    w = W.CONFIGS["c1"]
    inp = W.make_inputs(w)
    H = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                                 with_diag=False)
    mu = oracle.kpm_moments(H, w.a, w.b, w.M, mode=1, algo=1)
    E = np.linspace(-8.5, 8.5, 4001)
    rho = oracle.dos(mu, w.a, w.b, E, kernel=1)
    integral = ((rho[1:] + rho[:-1]) / 2 * np.diff(E)).sum()
    assert abs(integral - feats["integral"][0]) < feats["integral"][1]
    k = int(np.argmax(rho))
    assert abs(rho[k] - feats["peak_rho"][0]) < feats["peak_rho"][1]
    assert abs(abs(E[k]) - feats["peak_abs_energy"][0]) < feats["peak_abs_energy"][1]
    # van Hove peaks at +-|t| within the KPM resolution pi a/M (north_star)
    assert abs(abs(E[k]) - 2.7) < np.pi * w.a / w.M
    assert abs(rho[2000] - feats["rho_at_zero"][0]) < feats["rho_at_zero"][1]
    assert rho.min() >= 0.0
    assert np.abs(rho - rho[::-1]).max() < 1e-12            # particle-hole symmetry
    # V-shaped DOS around the Dirac point (Fig. 4a): small near E = 0
    # (the 4 zero modes of the 24x24 supercell leave a finite-size bump exactly at 0),
    # growing towards the van Hove peaks
    assert rho[1900:2101].max() < 0.05 * rho[k]
    assert rho[2000 + 150] < rho[2000 + 300] < rho[2000 + 450] < rho[2000 + 600]


def test_grid_end_points_within_rounding_of_the_band_edge_are_outside():
    """Reading A13b: rho = 0 for |x| >= 1 - 8 eps.  A grid end point E = b +- a evaluates to x = +-1 or an
    ulp or two inside by rounding alone; the weight 1/(pi a sqrt(1 - x^2)) is ~1e8 there.  With mu = (1, 0, 0, ...)
    and no damping the reconstruction IS that weight (closed form), so the rule is visible on its own:
    zero at 1, 1 - eps, 1 - 4 eps (both signs), the closed form from 1 - 16 eps inwards."""
    eps = 2.0**-52
    a, b = 13.151754450485727, -0.017020550974913284          # config 2's scale
    mu = np.zeros(8)
    mu[0] = 1.0
    for sgn in (1.0, -1.0):
        xs_out = sgn * np.array([1.0, 1.0 - eps / 2, 1.0 - eps, 1.0 - 4 * eps, 1.0 - 8 * eps, 1.0 + eps, 1.5])
        xs_in = sgn * np.array([1.0 - 16 * eps, 1.0 - 1e-12, 0.999, 0.3])
        assert (oracle.dos(mu, 1.0, 0.0, xs_out, kernel=0) == 0.0).all()
        got = oracle.dos(mu, 1.0, 0.0, xs_in, kernel=0)
        want = 1.0 / (np.pi * np.sqrt((1.0 - xs_in) * (1.0 + xs_in)))
        assert np.abs(got / want - 1.0).max() <= 1e-9
    # config 2's own grid: the last point comes out one ulp inside the edge and is an end point
    E = np.linspace(b - a, b + a, 4001)
    x = (E - b) / a
    assert abs(x[-1]) < 1.0 and abs(x[0]) >= 1.0
    rho = oracle.dos(mu, a, b, E, kernel=0)
    assert rho[0] == 0.0 and rho[-1] == 0.0 and rho[1] > 0.0 and rho[-2] > 0.0
