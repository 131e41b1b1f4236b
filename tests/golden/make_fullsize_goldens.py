"""Writes the full-size, full-depth expected values of tests/test_gpu_fulldepth.py.

    python tests/golden/make_fullsize_goldens.py c2 c2b c4 c3 c5

Calls ONLY the CPU oracle (oracle/) and the seeded input generators
(paper_2509_06525_b200/workloads.py, which hold none of the method's arithmetic); nothing here
touches the CUDA path.  For every named config it runs the oracle at the config's own
(N, M, R, seed) -- BASELINE.json:configs, DESIGN.md sec. 4 -- and stores

    tests/golden/<cfg>_moments_M<M>.txt     mu_0 .. mu_{M-1}          (north_star: |dmu_n| <= 1e-9)
    tests/golden/<cfg>_dos_G<G>.txt         Jackson DOS on the config's grid (<= 1e-8 of the peak)

c2, c2b, c4 (10^6 atoms) use the oracle's primary mode, the plain definition m_n = Re<phi_0|phi_n>
with M SpMVs (algo 0).  c3 (1.024e7 atoms, M = 5000) and c5 (10^8 atoms, M = 3000) use the
oracle's own doubling mode (algo 1; SURVEY.md sec. 8(d) "Oracle timing" allows it on a small
host) AFTER this script has checked it against the direct mode on the same lattice, scale and
seed at reduced depth (M = 48) to 1e-12; the check is recorded in the header.

Each file's header carries the scale (a, b) as hex floats -- the numbers the GPU run must be
given (reading A8: computed once and passed to both sides) -- and a SHA-256 of the input arrays
so that the test notices if the generators ever produce different lattices.
"""
from __future__ import annotations

import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_2509_06525_b200 import workloads as W  # noqa: E402

DOUBLING = {"c3", "c3b", "c5"}      # configs whose full-depth run uses the oracle's doubling mode
M_CHECK = 48


def remake_dos(key: str) -> None:
    """--dos-only: rewrite <cfg>_dos_G<G>.txt from the stored moments (oracle.dos alone; used after reading
    A13b changed the value at grid points within 8 eps of |x| = 1, which leaves the moments untouched)."""
    w = W.CONFIGS[key]
    head, mu = [], []
    with open(os.path.join(HERE, f"{key}_moments_M{w.M}.txt")) as f:
        for line in f:
            t = line.split()
            if line.startswith("#") and not line.startswith("# n "):
                head.append(line.rstrip("\n"))
            elif t and t[0] in ("a", "b", "inputs_sha256"):
                head.append(line.rstrip("\n"))
            elif t and t[0] == "mu":
                mu.append(float.fromhex(t[2]))
    vals = {l.split()[0]: l.split()[1] for l in head if not l.startswith("#")}
    a, b = float.fromhex(vals["a"]), float.fromhex(vals["b"])
    mu = np.array(mu)
    assert mu.shape == (w.M,)
    E = W.energy_grid(w, a, b)
    rho = oracle.dos(mu, a, b, E)
    with open(os.path.join(HERE, f"{key}_dos_G{E.shape[0]}.txt"), "w") as f:
        f.write("\n".join(head) + "\n# j  E_j  rho(E_j)   (oracle.dos of the stored moments, Jackson kernel, scale 1;"
                " reading A13b)\n")
        for j, (e, r) in enumerate(zip(E, rho)):
            f.write(f"rho {j} {float(e).hex()} {float(r).hex()}\n")
    print(f"[{key}] DOS rewritten from the stored moments", flush=True)


def make(key: str) -> None:
    w = W.CONFIGS[key]
    t0 = time.time()
    inp = W.make_inputs(w)
    H = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                                 w.r0, w.beta, inp.onsite_shift, method=1, with_diag=w.use_diag)
    if w.a is not None:
        a, b = float(w.a), float(w.b)
    else:                                   # reading A8
        lo, hi = oracle.spectral_bounds(H)
        a, b = 1.01 * (hi - lo) / 2.0, (hi + lo) / 2.0
    digest = W.inputs_digest(inp)
    print(f"[{key}] N={H.n} K={H.width} a={a!r} b={b!r} built in {time.time() - t0:.0f} s", flush=True)
    algo = 1 if key in DOUBLING else 0
    check = ""
    if algo == 1:
        m0 = oracle.kpm_moments(H, a, b, M_CHECK, w.R, w.seed, mode=0, algo=0)
        m1 = oracle.kpm_moments(H, a, b, M_CHECK, w.R, w.seed, mode=0, algo=1)
        d = float(np.abs(m0 - m1).max())
        assert d <= 1e-12, d
        check = f"doubling vs direct at M={M_CHECK}, same lattice/scale/seed: max|dmu| = {d:.3e}"
        print(f"[{key}] {check}", flush=True)
    t1 = time.time()
    mu = oracle.kpm_moments(H, a, b, w.M, w.R, w.seed, mode=0, algo=algo)
    secs = time.time() - t1
    print(f"[{key}] M={w.M} R={w.R} algo={algo}: {secs:.0f} s", flush=True)
    E = W.energy_grid(w, a, b)
    rho = oracle.dos(mu, a, b, E)
    head = [
        f"# {w.name}: N={H.n} K={H.width} diag={int(H.diag is not None)} M={w.M} R={w.R} seed={w.seed}",
        f"# written by tests/golden/make_fullsize_goldens.py from oracle.kpm_moments(mode=0, algo={algo})"
        f" [{'doubling identities' if algo else 'plain definition, M SpMVs'}] in {secs:.0f} s"
        f" with OMP_NUM_THREADS={os.environ.get('OMP_NUM_THREADS', 'default')}",
        "# cites: BASELINE.json:configs / north_star (recursion, moments, tolerances 1e-9 / 1e-8 of the peak);"
        " DESIGN.md sec. 3 (A1, A8, A13, A17), sec. 4 (input recipe)",
    ]
    if check:
        head.append(f"# {check}")
    head += [f"a {a.hex()}", f"b {b.hex()}", f"inputs_sha256 {digest}"]
    with open(os.path.join(HERE, f"{key}_moments_M{w.M}.txt"), "w") as f:
        f.write("\n".join(head) + "\n# n  mu_n\n")
        for n, v in enumerate(mu):
            f.write(f"mu {n} {float(v).hex()}\n")
    with open(os.path.join(HERE, f"{key}_dos_G{E.shape[0]}.txt"), "w") as f:
        f.write("\n".join(head) + "\n# j  E_j  rho(E_j)   (oracle.dos, Jackson kernel, scale 1)\n")
        for j, (e, r) in enumerate(zip(E, rho)):
            f.write(f"rho {j} {float(e).hex()} {float(r).hex()}\n")
    print(f"[{key}] done in {time.time() - t0:.0f} s", flush=True)


if __name__ == "__main__":
    args = sys.argv[1:]
    dos_only = "--dos-only" in args
    keys = [k for k in args if not k.startswith("--")] or ["c4", "c2b", "c2", "c3", "c5"]
    for k in keys:
        (remake_dos if dos_only else make)(k)
