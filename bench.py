#!/usr/bin/env python
"""Benchmark of the KPM/LSQT density-of-states hot path (BASELINE.json metric).

    python bench.py --gpus N --steps K --warmup W [--workload c5] [--impl reference]

A "step" is one pass of the whole hot path over one batch of synthetic input:
build_hamiltonian (cell list + ELL assembly) -> kpm_moments (random phases, ceil(M/2) fused
Chebyshev passes, doubling identities) -> dos (Jackson kernel, 4001 energies).  The N=1 workload
is BASELINE.json:configs[4] ("c5": pristine graphene, 5000x5000 cells = 10^8 atoms, ELL width 3,
M=3000, R=2, complex128), the configuration the metric is quoted on.  `value` is
atoms*moments*vectors per second of the whole step with inputs resident in HBM; `e2e` is the same
through the same calls with HOST (pinned) inputs, host<->device copies inside the timed region.
With N>1 (torchrun) every rank runs an independent replica on its own seed (the path has no
exchange step: "replicas only") and value = all ranks' units / max time.
`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2509_06525_b200 import workloads as W  # noqa: E402

METRIC = "atom-Chebyshev-moment updates/sec (fp64 complex)"
UNIT = "atom*moment*vector updates/s"
KERNEL = "auto"                 # set by --kernel: pins the fused-pass kernel through gtb_kpm_options
STAGES = 0                      # set by --stages: ring depth of the staged passes (0 = the library's default)
WINDOW = True                   # cleared by --no-window: windowed tiles (gtb_window_ell, K7w) for wide rows
TILE_NUMBERING = None           # --tile-numbering TXxTY: the same lattice with its atoms numbered tile-major (input order study)
PACK = True                     # cleared by --no-pack: packed narrow rows (gtb_pack_ell, K7x2p) when the matrix fits
REP = "scalar"                  # set by --rep (spd only): scalar ELL expansion, stored 9x9 blocks, or bonds (matrix-free)
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # 148 SMs x 64 FP64 FMA lanes x 2 flop x clocks.max.sm
HOPPING = "analytic"            # set by --hopping: "analytic" t(r) or "mlp" (descriptor + MLPs of Eq. 2)
ORBITALS = "pz"                 # set by --orbitals: "pz" (one orbital per atom), "sp" (4) or "spd" (9)
ORB_COUNT = {"pz": 1, "sp": 4, "spd": 9}
VAC_DT = 0.1 / 0.6582119569     # the paper's 0.1 fs time step in hbar/eV

def _ncu_traffic(quantity: str, key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from
    profiles/traffic.json (written from `ncu --set full` captures by
    `python -m paper_2509_06525_b200.ncu_traffic`; the .md next to it names the commands).
    None when no capture of this configuration exists."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        with open(path) as f:
            entry = json.load(f).get(quantity, {}).get(key)
    except (OSError, ValueError):
        return None
    return float(entry["dram_bytes_per_launch"]) if entry else None


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """Samples SM clocks and throttle reasons with nvidia-smi while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self._stop, self._t = index, [], threading.Event(), None

    def _run(self):
        while not self._stop.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([x.strip() for x in out.strip().split(",")])
            except Exception:
                pass
            self._stop.wait(0.2)

    def __enter__(self):
        self._t = threading.Thread(target=self._run, daemon=True)
        self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        self._t.join(timeout=6)

    def summary(self):
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
            except ValueError:
                continue
            for name, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _workload(args) -> W.Workload:
    w = W.CONFIGS[args.workload]
    if args.cutoff:
        w = W.replace(w, cutoff=args.cutoff, name=f"{w.name}-rc{args.cutoff:g}")
    if args.nx or args.ny:
        w = w.scaled(args.nx or w.nx, args.ny or w.ny)
    if args.moments:
        w = W.replace(w, M=args.moments)
    return w


# ----------------------------------------------------------------------------- CPU oracle arm
def _oracle_step(w, inp, energies_of):
    import oracle
    t0 = time.perf_counter()
    H = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                                 w.r0, w.beta, inp.onsite_shift, method=1, with_diag=w.use_diag)
    if HOPPING == "mlp":
        H = oracle.mlp_hamiltonian(H, inp.pos, inp.species, inp.box, inp.pbc, W.MLP_DIMS,
                                   max(2.0, 1.05 * w.cutoff), W.mlp_weights(), with_diag=True)
    if ORBITALS == "sp":
        ns = len(w.onsite)
        H = oracle.sk_hamiltonian(H, inp.pos, inp.species, inp.box, inp.pbc, W.SK_ONSITE_S[:ns],
                                  W.SK_ONSITE_P[:ns], W.sk_table(ns), r0=1.42, beta=w.beta,
                                  onsite_shift=inp.onsite_shift)
    elif ORBITALS == "spd":
        ns = len(w.onsite)
        H = oracle.spd_hamiltonian(H, inp.pos, inp.species, inp.box, inp.pbc, W.SK_ONSITE_S[:ns],
                                   W.SK_ONSITE_P[:ns], W.SK_ONSITE_D[:ns], W.spd_table(ns), r0=1.42,
                                   beta=w.beta, onsite_shift=inp.onsite_shift)
    if w.a is None or ORBITALS != "pz" or HOPPING == "mlp":
        lo, hi = oracle.spectral_bounds(H)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    else:
        a, b = w.a, w.b
    mu = oracle.kpm_moments(H, a, b, w.M, w.R, w.seed, mode=0, algo=0)   # the plain definition
    rho = oracle.dos(mu, a, b, energies_of(w, a, b))
    return time.perf_counter() - t0, rho


def _oracle_vac_step(w, inp, n_steps, dt):
    import oracle
    t0 = time.perf_counter()
    H = oracle.build_hamiltonian(inp.pos, inp.species, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0,
                                 w.r0, w.beta, inp.onsite_shift, method=1, with_diag=w.use_diag)
    if w.a is None:
        lo, hi = oracle.spectral_bounds(H)
        a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
    else:
        a, b = w.a, w.b
    vv = oracle.velocity_ell(H, inp.pos, inp.box, inp.pbc, 0)
    Cm = oracle.vac_moments(H, vv, a, b, w.M, n_steps, dt, R=w.R, seed=w.seed, mode=0)
    _, sigma = oracle.vac_conductivity(Cm, a, b, W.energy_grid(w, a, b), dt)
    return time.perf_counter() - t0, sigma


def _cpu_sample_vac(w: W.Workload, n_steps: int):
    """Bounded VAC sample for the oracle: <= 160 000 atoms, M and the step count cut so that one
    run is roughly 10-30 s (the oracle's VAC loop is serial over vectors)."""
    nx, ny = min(w.nx, 200), min(w.ny, 200)
    return w.scaled(nx, ny, M=min(w.M, 64)), min(n_steps, 4)


def _cpu_sample(w: W.Workload) -> W.Workload:
    """Bounded sample of the workload for the oracle: same construction, 10^6 atoms at most,
    moments cut so that one pass is roughly 10-30 s of CPU work."""
    nx, ny = min(w.nx, 500), min(w.ny, 500)
    n = 4 * nx * ny
    width_guess = {1.95: 3, 2.65: 10, 4.0: 20}.get(w.cutoff, 10)
    budget = 4e9 * 8 / (width_guess + 5)     # updates that take ~20 s at ~2e8 upd/s for width 3
    if ORBITALS != "pz":
        budget /= ORB_COUNT[ORBITALS] ** 2   # B x the rows, B x the width
    M = int(max(16, min(w.M, budget / (n * w.R))))
    return w.scaled(nx, ny, M=M)


def _cores():
    try:
        import oracle  # noqa: F401
        return int(os.environ.get("OMP_NUM_THREADS", os.cpu_count() or 1))
    except Exception:
        return os.cpu_count() or 1


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = _workload(args)
    if args.quantity == "vac":
        s, ns = _cpu_sample_vac(w, args.time_steps)
        inp = W.make_inputs(s)
        times = [_oracle_vac_step(s, inp, ns, VAC_DT)[0] for _ in range(args.steps)]
        t = float(np.mean(times))
        value = s.n_atoms * s.M * s.R * ns / t
        sample = f"{s.name}: N={s.n_atoms}, M={s.M}, R={s.R}, time steps={ns}, build+velocity+vac_moments+conductivity"
    else:
        s = _cpu_sample(w)
        inp = W.make_inputs(s)
        times = [_oracle_step(s, inp, W.energy_grid)[0] for _ in range(args.steps)]
        t = float(np.mean(times))
        orb = ORB_COUNT[ORBITALS]
        value = orb * s.n_atoms * s.M * s.R / t
        sample = f"{s.name}: N={s.n_atoms} x {orb} orbitals, M={s.M}, R={s.R}, build+moments(direct)+dos"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": w.name, "quantity": args.quantity, "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": _cores(), "kind": "oracle",
                             "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- CUDA arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2509_06525_b200 import binding as gtb
    from paper_2509_06525_b200 import replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    gtb.lib()

    w = _workload(args)
    inp = W.make_inputs(w, tile=TILE_NUMBERING)
    n = w.n_atoms
    seed = replicas.replica_seed(w.seed, rank)      # independent replica per rank
    # host inputs in pinned memory (e2e arm) and resident copies (device arm)
    h_pos = torch.from_numpy(inp.pos).pin_memory()
    h_spec = torch.from_numpy(inp.species).pin_memory()
    h_shift = torch.from_numpy(inp.onsite_shift).pin_memory() if inp.onsite_shift is not None else None
    d_pos, d_spec = h_pos.to(dev), h_spec.to(dev)
    d_shift = h_shift.to(dev) if h_shift is not None else None
    h2d = h_pos.numel() * 8 + h_spec.numel() * 4 + (h_shift.numel() * 8 if h_shift is not None else 0)

    ws_build = gtb.workspace(gtb.build_workspace_bytes(n), dev)
    width = gtb.neighbor_width(d_pos, inp.box, inp.pbc, w.cutoff, ws=ws_build)
    n_orb = ORB_COUNT[ORBITALS] * n                   # rows of H: the unit of the metric
    ws_kpm = gtb.workspace(gtb.kpm_workspace_bytes(n_orb, w.M, w.R), dev)
    ws_bounds = gtb.workspace(gtb.bounds_workspace_bytes(n_orb), dev)
    gtb.lib().gtb_pack_workspace_bytes.restype = __import__("ctypes").c_size_t
    ws_pack = gtb.workspace(int(gtb.lib().gtb_pack_workspace_bytes()), dev)
    mu = torch.empty(w.M, dtype=torch.float64, device=dev)
    h_rho = torch.empty(w.n_energies, dtype=torch.float64).pin_memory()
    state = {}
    if HOPPING == "mlp":
        state["mlp_w"] = torch.from_numpy(W.mlp_weights()).to(dev)

    timer = gtb.LoopTimer()
    opt = gtb.options(kernel={"auto": gtb.KERNEL_AUTO, "row": gtb.KERNEL_ROW, "row_x2": gtb.KERNEL_ROW_X2,
                              "tile": gtb.KERNEL_TILE}[KERNEL], tile_stages=STAGES, timer=timer)

    def step(pos, spec, shift):
        # the width is a property of (lattice, cutoff) found once above (gtb_neighbor_width): the
        # assembly checks it (GTB_ERR_ELL_OVERFLOW), so the neighbour search runs once per step
        H = gtb.build_hamiltonian(pos, spec, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0,
                                  w.beta, shift, width=width, with_diag=w.use_diag, ws=ws_build)
        if HOPPING == "mlp":   # Eq. 2: descriptor + MLPs on the neighbour lists just built
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            H = gtb.mlp_hamiltonian(H, pos, spec, inp.box, inp.pbc, W.MLP_DIMS, max(2.0, 1.05 * w.cutoff),
                                    state["mlp_w"], with_diag=True)
            e1.record()
            state["mlp_events"] = (e0, e1)
        if ORBITALS == "sp":   # Slater-Koster s,p blocks on the neighbour lists just built
            ns = len(w.onsite)
            H = gtb.sk_hamiltonian(H, pos, spec, inp.box, inp.pbc, W.SK_ONSITE_S[:ns],
                                   W.SK_ONSITE_P[:ns], W.sk_table(ns), r0=1.42, beta=w.beta,
                                   onsite_shift=shift)
        elif ORBITALS == "spd" and REP == "scalar":
            ns = len(w.onsite)
            H = gtb.spd_hamiltonian(H, pos, spec, inp.box, inp.pbc, W.SK_ONSITE_S[:ns], W.SK_ONSITE_P[:ns],
                                    W.SK_ONSITE_D[:ns], W.spd_table(ns), r0=1.42, beta=w.beta,
                                    onsite_shift=shift)
        elif ORBITALS == "spd":      # bond form (matrix-free) or stored 9x9 blocks on the same neighbour lists
            ns = len(w.onsite)
            if w.R in (2, 4):         # neighbour slots arranged so that the gathers of adjacent atoms share L1 wavefronts
                H = gtb.pair_slots(H, w.R)
            Hm = gtb.spd_bonds(H, pos, spec, inp.box, inp.pbc, W.SK_ONSITE_S[:ns], W.SK_ONSITE_P[:ns],
                               W.SK_ONSITE_D[:ns], W.spd_table(ns), r0=1.42, beta=w.beta, onsite_shift=shift)
            H = Hm if REP == "bonds" else gtb.spd_blocks(Hm)
            rmode = gtb.MODE_BOND9 if REP == "bonds" else gtb.MODE_BLOCK9
            lo, hi = gtb.spd_bounds(H, rmode).tolist()
            a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
            gtb.kpm_moments(H, a, b, w.M, w.R, w.R, seed, mode=rmode, ws=ws_kpm, mu=mu, opt=opt)
            if "E" not in state:
                state["E"] = torch.from_numpy(W.energy_grid(w, a, b)).to(dev)
            rho = gtb.dos(mu, a, b, state["E"])
            state["H"], state["a"], state["b"], state["rho"] = H, a, b, rho
            return rho
        if w.a is None or ORBITALS != "pz" or HOPPING == "mlp":
            lo, hi = gtb.spectral_bounds(H, ws=ws_bounds).tolist()
            a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
        else:
            a, b = w.a, w.b
        kmode = {"sp": gtb.MODE_ORB4, "spd": gtb.MODE_ORB9}.get(ORBITALS, 0)
        Hk = H
        state["packed"] = None
        # (R = 8 narrow rows run K7t faster than the packed pass: c4 0.0703 against 0.0748 ms)
        if PACK and KERNEL == "auto" and ORBITALS == "pz" and H.width <= 4 and w.R in (2, 4) and n * (w.R // 2) > 148 * 8 * 256:
            # R = 2: first the slots of rows 4q .. 4q + 3 permuted so that the four 32-byte gathers share an L1 wavefront
            Hs = gtb.pair_slots(H, w.R) if w.R == 2 else H
            P = gtb.pack_ell(Hs, ws=ws_pack)         # part of the timed step; None: does not fit, plain path
            if P is not None:
                Hk, kmode, state["packed"] = P, gtb.MODE_PACKED, P
        state["windowed"] = None
        if WINDOW and KERNEL == "auto" and ORBITALS == "pz" and H.width >= 16 and w.R in (2, 4, 8):   # K = 11: K7t is as fast
            Wd = gtb.window_ell(H, w.R)              # part of the timed step; None: no locality, K7t stays
            if Wd is not None:
                Hk, kmode, state["windowed"] = Wd, gtb.MODE_WINDOW, Wd
        state["paired"] = False
        if Hk is H and ORBITALS == "pz" and w.R == 4 and H.width <= 48:
            # plain ELL at R = 4: the same matrix with the slots of rows 2q, 2q + 1 alternating in column parity
            # (gtb_pair_slots: their 64-byte gathers then share an L1 wavefront); part of the timed step
            Hk, state["paired"] = gtb.pair_slots(H, w.R), True
        gtb.kpm_moments(Hk, a, b, w.M, w.R, w.R, seed, mode=kmode, ws=ws_kpm, mu=mu, opt=opt)
        if "E" not in state:
            state["E"] = torch.from_numpy(W.energy_grid(w, a, b)).to(dev)
        rho = gtb.dos(mu, a, b, state["E"])
        state["H"], state["a"], state["b"], state["rho"] = H, a, b, rho
        return rho

    def barrier():
        replicas.barrier(dev)

    def timed(fn, steps):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = gtb.launch_count()
        loop_ms, loop_passes = 0.0, 0
        e0.record()
        for _ in range(steps):
            fn()
            ms, passes = timer.ms()                 # CUDA events on the launching stream
            loop_ms += ms
            loop_passes += passes
        e1.record()
        barrier()
        t = replicas.max_over_ranks(e0.elapsed_time(e1), dev)
        return t, gtb.launch_count() - l0, loop_ms, loop_passes

    def device_step():
        step(d_pos, d_spec, d_shift)

    def e2e_step():
        pos = h_pos.to(dev, non_blocking=True)
        spec = h_spec.to(dev, non_blocking=True)
        shift = h_shift.to(dev, non_blocking=True) if h_shift is not None else None
        rho = step(pos, spec, shift)
        h_rho.copy_(rho, non_blocking=True)
        torch.cuda.current_stream().synchronize()

    for _ in range(args.warmup):
        device_step()
    with ClockSampler(local) as clk:
        ms, launches, loop_ms, loop_passes = timed(device_step, args.steps)
    H = state["H"]
    for _ in range(min(args.warmup, 1)):
        e2e_step()
    ms_e2e, _, _, _ = timed(e2e_step, args.steps)
    # a diverged or non-finite run must not print a throughput
    gtb.kpm_status(ws_kpm)
    rho_h = state["rho"].cpu().numpy()
    if not (np.isfinite(rho_h).all() and rho_h.max() > 0.0):
        raise SystemExit("bench.py: the density of states is not finite / not positive; no number is reported")

    units = float(n_orb) * w.M * w.R * args.steps        # per rank
    value = replicas.whole_job_value(units, ms)
    e2e = replicas.whole_job_value(units, ms_e2e)
    # roofline of the dominant kernel (the fused pass K7): algorithmic bytes per launch
    # = N * (12 K + 8 [diag] + 48 R), over its mean launch duration
    orb4 = ORBITALS != "pz" and w.R in (2, 4, 8) and not (ORBITALS == "spd" and REP != "scalar")
    B = ORB_COUNT[ORBITALS]
    per_atom = W.algorithmic_bytes_per_atom_pass(H.width, H.diag is not None, w.R)
    flops_per_launch = None
    plain_per_atom = per_atom
    packed = state.get("packed")
    if packed is not None:   # one 16-byte (short rows: 8-byte) word per row (+ the diagonal array when K = 4), + the vectors
        per_atom = (8 if packed.short_rows else 16) + (8 if packed.diag is not None else 0) + 48 * w.R
    rep9 = ORBITALS == "spd" and REP != "scalar"
    if rep9 and REP == "blocks":   # per ATOM: K x (column + 81 values) + 9 onsite + 9 orbital rows of vectors; / 9 per row
        per_atom = (H.width * (4 + 648) + 72 + 9 * 48 * w.R) / 9.0
    elif rep9:                     # per ATOM: K columns + own record + shift + vectors (each neighbour record once: in the 32)
        per_atom = (4 * H.width + 32 + 8 + 9 * 48 * w.R) / 9.0
        # closed-form action: 64 FMA per real component and pair + ~50 FMA-equivalents of geometry, + the epilogue
        flops_per_launch = float(n) * (H.width * (2 * 64 * 2 * w.R + 100) + 9 * 2 * w.R * 8)
    elif orb4:   # per orbital row: K blocks of (4 B column + 8 B^2 B values) shared by B rows, + diag + vectors
        per_atom = (H.width // B) * (4 + 8 * B * B) // B + (8 if H.diag is not None else 0) + 48 * w.R
    bytes_per_launch = float(n_orb) * per_atom
    k7_ms = loop_ms / max(loop_passes, 1)
    peak, peak_src = _peaks()
    achieved = bytes_per_launch / (k7_ms * 1e-3) / 1e9
    small = not orb4 and KERNEL == "auto" and w.R in (2, 4, 8) and n_orb * (w.R // 2) <= 148 * 4 * 256
    vec = w.R in (2, 4, 8)
    tile = KERNEL == "tile" or (KERNEL == "auto" and (H.width > 4 or w.R == 8) and n % 4 == 0 and vec)
    x2 = KERNEL == "row_x2" or (KERNEL == "auto" and H.width <= 4 and vec and not tile)
    windowed = state.get("windowed")
    if rep9 or packed is not None or windowed is not None:
        small = False
    k7_name = ("cheb_packed_kernel (K7x2p: fused Chebyshev pass on packed rows of %d bytes, 16-bit relative columns + value "
               "dictionary of %d entries, two elements in flight per thread)" % (8 if packed.short_rows else 16, packed.n_values)
               if packed is not None else
               "cheb_window_kernel (K7w: fused Chebyshev pass on windowed tiles, phi_n gathered from shared memory; "
               "largest window %d blocks)" % windowed.blocks if windowed is not None else
               "cheb_bond9_kernel (K7m: fused Chebyshev pass, 9x9 pair action rebuilt from the bond vector)"
               if rep9 and REP == "bonds" else
               "cheb_block9_kernel (K7bb: fused Chebyshev pass on stored 9x9 blocks [K][81][n])" if rep9 else
               "cheb_cluster_kernel (K7c: all passes in one 8-CTA cluster, phi in distributed shared memory; "
               "ms_per_launch is per PASS)" if small and H.width <= 4 and n_orb * (w.R // 2) <= 8192 else
               "cheb_small_kernel (K7p: all passes in one cooperative launch; ms_per_launch is per PASS)" if small else
               ("cheb_orb%d_kernel (K7b: fused Chebyshev pass on %dx%d orbital blocks)" % (B, B, B)) if orb4 else
               "cheb_tile_kernel (K7t: fused Chebyshev pass, ELL slots staged by TMA)" if tile else
               "cheb_step_x2_kernel (K7x2: fused Chebyshev pass, two elements in flight per thread)" if x2 else
               "cheb_step_kernel (K7: fused Chebyshev pass, register path)")
    roofline = {"bound": "hbm", "kernel": k7_name,
                "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "peak_source": peak_src, "frac_of_8TBs_nominal": achieved / 8000.0,
                "traffic": _ncu_traffic("dos-packed", w.name) if packed is not None else
                _ncu_traffic("dos-window", w.name) if windowed is not None else
                _ncu_traffic("dos" if ORBITALS == "pz" else "dos-" + ORBITALS +
                                        ("" if REP == "scalar" else "-" + REP), w.name)
                if KERNEL == "auto" else None,
                "algorithmic_bytes_per_launch": bytes_per_launch, "bytes_per_atom_pass": per_atom,
                "ms_per_launch": k7_ms, "launches_timed": loop_passes,
                "share_of_step": loop_ms / ms}
    if packed is not None:   # NEXT-4: fewer bytes than the sec. 8(d) bound; both figures side by side
        roofline["uncompressed_bytes_per_atom_pass"] = plain_per_atom
        roofline["frac_on_uncompressed_bytes"] = float(n_orb) * plain_per_atom / (k7_ms * 1e-3) / 1e9 / peak
    if flops_per_launch is not None:   # the matrix-free pass has two roofs: report against the lower one
        t_hbm = bytes_per_launch / (peak * 1e9)
        t_alu = flops_per_launch / (FP64_PEAK_TFLOPS * 1e12)
        tf = flops_per_launch / (k7_ms * 1e-3) / 1e12
        roofline["hbm_frac"] = achieved / peak
        roofline["alu"] = {"achieved": tf, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": tf / FP64_PEAK_TFLOPS,
                           "algorithmic_flops_per_launch": flops_per_launch,
                           "peak_source": "derived: 148 SMs x 64 FP64 FMA lanes x 2 flop x 1.965 GHz"}
        if t_alu > t_hbm:
            roofline.update(bound="alu", achieved=tf, peak=FP64_PEAK_TFLOPS, unit="TFLOP/s",
                            frac=tf / FP64_PEAK_TFLOPS, peak_source=roofline["alu"]["peak_source"])
            roofline.pop("frac_of_8TBs_nominal", None)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64 (complex128 vectors)",
            "data": "synthetic",
            "config": {"workload": w.name, "atoms": n, "orbitals_per_atom": n_orb // n,
                       "ell_width": H.width,
                       "representation": REP if ORBITALS == "spd" else "packed rows" if packed is not None else
                                         "ell, slots paired for R = 4" if state.get("paired") else "ell",
                       "cutoff_A": w.cutoff, "numbering": ("tile-major %dx%d cells" % TILE_NUMBERING) if TILE_NUMBERING else "row-major",
                       "moments": w.M,
                       "vectors": w.R, "energies": w.n_energies, "passes_per_step": (w.M + 1) // 2,
                       "l2": "inputs larger than L2 (working set %.1f GB)" % (
                           (2 * n_orb * w.R * 16 + (H.nbytes() if not rep9 else H.cols.numel() * 4 + H.vals.numel() * 8)) / 1e9),
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "seconds_per_full_dos": ms / args.steps * 1e-3,
            "recursion_updates_per_s": float(n_orb) * w.M * w.R / ((loop_ms / args.steps + k7_ms) * 1e-3),
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": h_rho.numel() * 8, "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": launches, "roofline": roofline, "clocks": clk.summary()}
    if HOPPING == "mlp":
        torch.cuda.synchronize()
        line["config"]["hopping"] = "descriptor + MLPs of Eq. 2, F, Nb, Hd = %d, %d, %d (synthetic weights)" % W.MLP_DIMS[1:]
        line["mlp_hamiltonian_ms"] = state["mlp_events"][0].elapsed_time(state["mlp_events"][1])
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline:
            s = _cpu_sample(w)
            t, _ = _oracle_step(s, W.make_inputs(s), W.energy_grid)
            orb = ORB_COUNT[ORBITALS]
            line["cpu_baseline"] = {
                "value": orb * s.n_atoms * s.M * s.R / t, "unit": UNIT, "cores": _cores(), "kind": "oracle",
                "sample": f"{s.name}: N={s.n_atoms} x {orb} orbitals, M={s.M}, R={s.R}, build+moments(direct)+dos, {t:.1f} s"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def run_vac(args):
    """Same contract as run_ours for the VAC conductivity (Eq. 3): a step = build_hamiltonian ->
    velocity_ell -> vac_moments (n_steps time points, M moments each: M-1 fused passes per point
    plus two Chebyshev-Bessel propagations) -> vac_conductivity.  units = N*M*R*n_steps."""
    import torch
    import torch.distributed as dist
    from paper_2509_06525_b200 import binding as gtb
    from paper_2509_06525_b200 import replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback")
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    gtb.lib()
    w = _workload(args)
    T = args.time_steps
    inp = W.make_inputs(w)
    n = w.n_atoms
    seed = replicas.replica_seed(w.seed, rank)
    h_pos = torch.from_numpy(inp.pos).pin_memory()
    h_spec = torch.from_numpy(inp.species).pin_memory()
    h_shift = torch.from_numpy(inp.onsite_shift).pin_memory() if inp.onsite_shift is not None else None
    d_pos, d_spec = h_pos.to(dev), h_spec.to(dev)
    d_shift = h_shift.to(dev) if h_shift is not None else None
    h2d = h_pos.numel() * 8 + h_spec.numel() * 4 + (h_shift.numel() * 8 if h_shift is not None else 0)
    B = ORB_COUNT[ORBITALS]
    n_rows = B * n                                    # rows of H: orbitals
    ws_build = gtb.workspace(gtb.build_workspace_bytes(n), dev)
    ws_vac = gtb.workspace(gtb.vac_workspace_bytes(n_rows, w.M, T, w.R), dev)
    ws_bounds = gtb.workspace(gtb.bounds_workspace_bytes(n_rows), dev)
    vmode = {"sp": gtb.MODE_ORB4, "spd": gtb.MODE_ORB9}.get(ORBITALS, 0)
    Cm = torch.empty((T, w.M), dtype=torch.float64, device=dev)
    h_sigma = torch.empty((T, w.n_energies), dtype=torch.float64).pin_memory()
    state = {}
    width = gtb.neighbor_width(d_pos, inp.box, inp.pbc, w.cutoff, ws=ws_build)
    timer = gtb.LoopTimer()
    opt = gtb.options(timer=timer)

    def step(pos, spec, shift):
        H = gtb.build_hamiltonian(pos, spec, inp.box, inp.pbc, w.cutoff, w.onsite, w.t0, w.r0,
                                  w.beta, shift, width=width, with_diag=w.use_diag, ws=ws_build)
        vpos = pos
        if ORBITALS != "pz":     # Slater-Koster blocks on the neighbour lists; every orbital sits at its atom
            ns = len(w.onsite)
            if ORBITALS == "sp":
                H = gtb.sk_hamiltonian(H, pos, spec, inp.box, inp.pbc, W.SK_ONSITE_S[:ns], W.SK_ONSITE_P[:ns],
                                       W.sk_table(ns), r0=1.42, beta=w.beta, onsite_shift=shift)
            else:
                H = gtb.spd_hamiltonian(H, pos, spec, inp.box, inp.pbc, W.SK_ONSITE_S[:ns], W.SK_ONSITE_P[:ns],
                                        W.SK_ONSITE_D[:ns], W.spd_table(ns), r0=1.42, beta=w.beta,
                                        onsite_shift=shift)
            vpos = pos.repeat_interleave(B, dim=0)
        if w.a is None or ORBITALS != "pz":
            lo, hi = gtb.spectral_bounds(H, ws=ws_bounds).tolist()
            a, b = 1.01 * (hi - lo) / 2, (hi + lo) / 2
        else:
            a, b = w.a, w.b
        if ORBITALS == "pz" and w.R in (2, 4) and H.width <= 48:
            H = gtb.pair_slots(H, w.R)    # the same matrix with its slots arranged for the gathers of an R-vector pass
        vv = gtb.velocity_ell(H, vpos, inp.box, inp.pbc, 0)
        vopt, state["alt"] = opt, None
        if ORBITALS == "pz" and w.R in (2, 4, 8):   # the fused passes on the compressed form, as the DOS path
            alt = None
            if PACK and H.width <= 4 and w.R in (2, 4):
                alt, amode, aname = gtb.pack_ell(H), gtb.MODE_PACKED, "packed rows (K7x2p)"
            elif WINDOW and H.width >= 16:
                alt, amode, aname = gtb.window_ell(H, w.R), gtb.MODE_WINDOW, "windowed tiles (K7w)"
            if alt is not None:
                vopt = gtb.options(timer=timer, alt=alt, alt_mode=amode)
                state["alt"] = aname
        gtb.vac_moments(H, vv, a, b, w.M, T, VAC_DT, w.R, w.R, seed, mode=vmode, ws=ws_vac, out=Cm, opt=vopt)
        if "E" not in state:
            state["E"] = torch.from_numpy(W.energy_grid(w, a, b)).to(dev)
        _, sigma = gtb.vac_conductivity(Cm, a, b, state["E"], VAC_DT)
        state["H"], state["a"], state["b"], state["vv"] = H, a, b, vv
        return sigma

    def timed(fn, steps):
        replicas.barrier(dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = gtb.launch_count()
        loop_ms, loop_passes = 0.0, 0
        e0.record()
        for _ in range(steps):
            fn()
            ms, passes = timer.ms()
            loop_ms += ms
            loop_passes += passes
        e1.record()
        replicas.barrier(dev)
        return replicas.max_over_ranks(e0.elapsed_time(e1), dev), gtb.launch_count() - l0, loop_ms, loop_passes

    def device_step():
        step(d_pos, d_spec, d_shift)

    def e2e_step():
        pos = h_pos.to(dev, non_blocking=True)
        spec = h_spec.to(dev, non_blocking=True)
        shift = h_shift.to(dev, non_blocking=True) if h_shift is not None else None
        h_sigma.copy_(step(pos, spec, shift), non_blocking=True)
        torch.cuda.current_stream().synchronize()

    for _ in range(args.warmup):
        device_step()
    with ClockSampler(local) as clk:
        ms, launches, loop_ms, loop_passes = timed(device_step, args.steps)
    H = state["H"]
    e2e_step()
    ms_e2e, _, _, _ = timed(e2e_step, args.steps)
    gtb.kpm_status(ws_vac)
    units = float(n_rows) * w.M * w.R * T * args.steps
    plain = W.algorithmic_bytes_per_atom_pass(H.width, H.diag is not None, w.R)
    if vmode:    # blocked passes: K/B blocks of (4 B column + 8 B^2 B values) shared by B rows
        plain = (H.width // B) * (4 + 8 * B * B) // B + (8 if H.diag is not None else 0) + 48 * w.R
    per_atom = plain + 16 * w.R
    bytes_per_launch = float(n_rows) * per_atom
    k_ms = loop_ms / max(loop_passes, 1)
    peak, peak_src = _peaks()
    achieved = bytes_per_launch / (k_ms * 1e-3) / 1e9
    # the other kernels of a time point, timed on their own with CUDA events on the same stream: one
    # propagation (gtb_evolve: terms - 1 passes with the Chebyshev-Bessel accumulation fused in, + the
    # first term's accumulation launch + two vector copies of the stand-alone call) and one velocity_apply
    a_, b_ = state["a"], state["b"]
    phi = gtb.random_phase_fill(seed, 0, w.R, n_rows, device=dev)
    ws_ev = gtb.workspace(gtb.evolve_workspace_bytes(n_rows, w.R), dev)
    terms = gtb.evolve(H, a_, b_, VAC_DT, phi, ws=ws_ev)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reps = 5
    e0.record()
    for _ in range(reps):
        gtb.evolve(H, a_, b_, VAC_DT, phi, ws=ws_ev)
    e1.record()
    e1.synchronize()
    ev_ms = e0.elapsed_time(e1) / reps
    y = gtb.velocity_apply(H, state["vv"], phi)      # warm-up: the output allocation
    e0.record()
    for _ in range(reps):
        y = gtb.velocity_apply(H, state["vv"], phi)
    e1.record()
    e1.synchronize()
    va_ms = e0.elapsed_time(e1) / reps
    step_ms = ms / args.steps
    prop_bytes = float(n_rows) * (plain + 32 * w.R)          # + the accumulator read and written
    va_bytes = float(n_rows) * (12 * H.width + 48 * w.R)     # columns, velocity values, x gathered once, y, bra
    kernels = [
        {"kernel": "moment pass (fused Chebyshev pass, dot products against the evolved bra)",
         "ms_per_launch": k_ms, "launches_per_step": T * (w.M - 1), "GB/s": achieved, "frac": achieved / peak,
         "share_of_step": k_ms * T * (w.M - 1) / step_ms},
        {"kernel": "propagation pass (fused Chebyshev pass + Chebyshev-Bessel accumulation; %d terms per U(dt); "
                   "timed as gtb_evolve / (terms - 1))" % terms,
         "ms_per_launch": ev_ms / (terms - 1), "launches_per_step": 2 * (T - 1) * (terms - 1),
         "GB/s": prop_bytes / (ev_ms / (terms - 1) * 1e-3) / 1e9,
         "frac": prop_bytes / (ev_ms / (terms - 1) * 1e-3) / 1e9 / peak,
         "share_of_step": 2 * (T - 1) * ev_ms / step_ms},
        {"kernel": "velocity_apply_kernel (chi_0 = V psi_R with the C_0 dot product)",
         "ms_per_launch": va_ms, "launches_per_step": T + 1, "GB/s": va_bytes / (va_ms * 1e-3) / 1e9,
         "frac": va_bytes / (va_ms * 1e-3) / 1e9 / peak, "share_of_step": (T + 1) * va_ms / step_ms},
    ]
    accounted = sum(k["share_of_step"] for k in kernels)
    line = {"metric": METRIC, "value": replicas.whole_job_value(units, ms), "unit": UNIT,
            "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64 (complex128 vectors)", "data": "synthetic",
            "config": {"workload": w.name, "quantity": "vac (Eq. 3)", "atoms": n, "orbitals_per_atom": B,
                       "ell_width": H.width,
                       "fused_passes_on": state.get("alt") or "plain ELL",
                       "moments": w.M, "vectors": w.R, "time_steps": T, "dt_fs": 0.1,
                       "energies": w.n_energies, "passes_per_step": T * (w.M - 1),
                       "l2": "inputs larger than L2 (working set %.1f GB)" % (
                           (4 * n_rows * w.R * 16 + 1.67 * H.nbytes()) / 1e9),
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "seconds_per_conductivity": ms / args.steps * 1e-3,
            "e2e": {"value": replicas.whole_job_value(units, ms_e2e), "unit": UNIT,
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": h_sigma.numel() * 8,
                    "ms_per_step": ms_e2e / args.steps},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "kernel": "fused Chebyshev pass, dot products against the evolved bra "
                                                   "(cheb_tile_kernel / cheb_step_kernel, kDotL variant)",
                         "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                         "peak_source": peak_src, "traffic": _ncu_traffic("vac", w.name),
                         "algorithmic_bytes_per_launch": bytes_per_launch,
                         "bytes_per_atom_pass": per_atom, "ms_per_launch": k_ms,
                         "launches_timed": loop_passes,
                         "share_of_step": k_ms * T * (w.M - 1) * args.steps / ms,
                         "kernels": kernels, "share_accounted": accounted},
            "clocks": clk.summary()}
    if rank == 0:
        if world == 1 and not args.no_cpu_baseline and ORBITALS == "pz":
            s, ns = _cpu_sample_vac(w, T)
            t, _ = _oracle_vac_step(s, W.make_inputs(s), ns, VAC_DT)
            line["cpu_baseline"] = {
                "value": s.n_atoms * s.M * s.R * ns / t, "unit": UNIT, "cores": _cores(), "kind": "oracle",
                "sample": f"{s.name}: N={s.n_atoms}, M={s.M}, R={s.R}, time steps={ns}, {t:.1f} s"}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    p = argparse.ArgumentParser()
    p.add_argument("--gpus", type=int, default=1)
    p.add_argument("--steps", type=int, default=3)
    p.add_argument("--warmup", type=int, default=3)
    p.add_argument("--impl", default="ours", choices=["ours", "reference"])
    p.add_argument("--workload", default="c5", choices=sorted(W.CONFIGS))
    p.add_argument("--nx", type=int, default=0, help="override the supercell (debugging)")
    p.add_argument("--ny", type=int, default=0)
    p.add_argument("--moments", type=int, default=0, help="override M (debugging)")
    p.add_argument("--no-cpu-baseline", action="store_true")
    p.add_argument("--quantity", default="dos", choices=["dos", "vac"],
                   help="dos: the headline path (Eq. 4); vac: the VAC conductivity (Eq. 3, NEXT-1)")
    p.add_argument("--time-steps", type=int, default=24, help="vac: points of the time grid (dt = 0.1 fs)")
    p.add_argument("--hopping", default="analytic", choices=["analytic", "mlp"],
                   help="analytic: t(r) of the configs; mlp: descriptor + MLPs of Eq. 2 with synthetic weights (NEXT-3)")
    p.add_argument("--kernel", default="auto", choices=["auto", "row", "row_x2", "tile"],
                   help="pin the fused-pass kernel (gtb_kpm_options.kernel); auto: picked from the matrix shape")
    p.add_argument("--rep", default="bonds", choices=["scalar", "blocks", "bonds"],
                   help="--orbitals spd: scalar ELL expansion (K7b9), stored 9x9 blocks (K7bb) or bonds = matrix-free (K7m)")
    p.add_argument("--stages", type=int, default=0, help="gtb_kpm_options.tile_stages (K7t, K7w); 0 = default")
    p.add_argument("--no-window", action="store_true", help="keep wide matrices on the plain ELL path (K7t)")
    p.add_argument("--no-pack", action="store_true", help="keep narrow matrices on the plain ELL path (K7x2)")
    p.add_argument("--tile-numbering", default="", help="TXxTY: number the input atoms tile-major in blocks of TX x TY "
                   "cells instead of row-major (same lattice; shows what the input order costs the gathers)")
    p.add_argument("--cutoff", type=float, default=0.0, help="override the neighbour cutoff in Angstrom "
                   "(3.0 on the pristine lattice = third-nearest neighbours, K = 12: Fig. 4a)")
    p.add_argument("--orbitals", default="pz", choices=["pz", "sp", "spd"],
                   help="pz: one orbital per atom (the headline); sp: Slater-Koster s,px,py,pz blocks (NEXT-2, dos only)")
    args = p.parse_args()
    global ORBITALS, HOPPING, KERNEL, REP, PACK, WINDOW, STAGES, TILE_NUMBERING
    STAGES = args.stages
    if args.tile_numbering:
        tx, _, ty = args.tile_numbering.lower().partition("x")
        TILE_NUMBERING = (int(tx), int(ty))
    WINDOW = not args.no_window
    PACK = not args.no_pack
    KERNEL = args.kernel
    REP = args.rep
    ORBITALS = args.orbitals
    HOPPING = args.hopping
    if args.hopping == "mlp" and (args.orbitals != "pz" or args.quantity == "vac"):
        raise SystemExit("bench.py: --hopping mlp is wired for --orbitals pz --quantity dos")
    if args.quantity == "vac" and not args.moments:
        args.moments = 512
    if args.impl == "reference":
        run_reference(args)
    elif args.quantity == "vac":
        run_vac(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
