"""bench.py's reference arm on CPU: the JSON line of the contract (keys, units, the oracle as
cpu_baseline), and the N > 1 rule that only rank 0 runs and prints it."""
import json
import os
import subprocess
import sys

from conftest import ROOT


def _run(extra_env, *args):
    env = dict(os.environ, **extra_env)
    return subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", *args],
                          capture_output=True, text=True, env=env, timeout=600)


def test_reference_arm_prints_one_contract_line():
    res = _run({}, "--workload", "c1", "--steps", "1", "--warmup", "0")
    assert res.returncode == 0, res.stderr
    lines = [x for x in res.stdout.splitlines() if x.strip()]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["higher_is_better"] is True and d["vs_baseline"] is None
    assert d["unit"] == "atom*moment*vector updates/s" and d["value"] > 0 and d["n_gpus"] == 1
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["value"] == d["value"]
    assert d["cpu_baseline"]["cores"] >= 1 and "N=2304" in d["cpu_baseline"]["sample"]
    assert d["e2e"] == {"value": d["value"], "unit": d["unit"], "h2d_bytes_per_step": 0,
                        "d2h_bytes_per_step": 0}
    assert d["config"]["workload"].startswith("c1") and d["data"] == "synthetic" and d["dtype"] == "f64"


def test_reference_arm_other_ranks_exit_quietly():
    res = _run({"RANK": "1", "WORLD_SIZE": "2", "LOCAL_RANK": "1"}, "--gpus", "2", "--workload", "c1",
               "--steps", "1", "--warmup", "0")
    assert res.returncode == 0 and res.stdout.strip() == ""


def test_reference_arm_covers_the_vac_and_sp_variants():
    for extra in (["--quantity", "vac", "--time-steps", "2", "--moments", "8"], ["--orbitals", "sp", "--moments", "8"],
                  ["--hopping", "mlp", "--moments", "8"]):
        res = _run({}, "--workload", "c1", "--steps", "1", "--warmup", "0", *extra)
        assert res.returncode == 0, res.stderr
        d = json.loads(res.stdout.strip().splitlines()[-1])
        assert d["impl"] == "reference" and d["value"] > 0
