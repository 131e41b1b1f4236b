"""Host protocol of the strip decomposition (gtb_strip_plan, include/gtb.h) on CPU with two gloo ranks: each
rank owns a strip of a vector, sends the rows its neighbour's halos name and receives its own; afterwards its
local [own | lo halo | hi halo] array must hold exactly the global rows the plan says, wrap-around included."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2509_06525_b200 import binding as gtb


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, halo, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    plan = gtb.strip_plan(n, world, halo, rank)
    glob = torch.arange(n, dtype=torch.float64) * 1.5 + 0.25            # "phi": every rank can check any row
    own = glob[plan["row0"]:plan["row0"] + plan["rows"]].clone()
    local = torch.full((plan["rows"] + 2 * halo,), -1.0, dtype=torch.float64)
    local[:plan["rows"]] = own
    # exchange: my LAST halo rows are my hi neighbour's lo halo; my FIRST halo rows are my lo neighbour's hi halo
    send_hi, send_lo = own[plan["rows"] - halo:].contiguous(), own[:halo].contiguous()
    recv_lo, recv_hi = torch.empty(halo, dtype=torch.float64), torch.empty(halo, dtype=torch.float64)
    ops = [dist.P2POp(dist.isend, send_hi, plan["hi_owner"], tag=1), dist.P2POp(dist.isend, send_lo, plan["lo_owner"], tag=2),
           dist.P2POp(dist.irecv, recv_lo, plan["lo_owner"], tag=1), dist.P2POp(dist.irecv, recv_hi, plan["hi_owner"], tag=2)]
    for r in dist.batch_isend_irecv(ops):
        r.wait()
    local[plan["rows"]:plan["rows"] + halo] = recv_lo
    local[plan["rows"] + halo:] = recv_hi
    want_lo = glob[(plan["lo_first"] + torch.arange(halo)) % n]
    want_hi = glob[(plan["hi_first"] + torch.arange(halo)) % n]
    ok = bool(torch.equal(local[plan["rows"]:plan["rows"] + halo], want_lo) and torch.equal(local[plan["rows"] + halo:], want_hi))
    with open(os.path.join(out, f"r{rank}.txt"), "w") as f:
        f.write("ok" if ok else "bad")
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("n,halo", [(1000, 37), (9804, 228), (64, 16)])
def test_two_rank_halo_exchange_follows_the_plan(tmp_path, n, halo):
    mp.spawn(_worker, args=(2, _free_port(), n, halo, str(tmp_path)), nprocs=2, join=True)
    assert [open(tmp_path / f"r{r}.txt").read() for r in range(2)] == ["ok", "ok"]


def test_plan_covers_the_rows_once_and_names_ring_neighbours():
    for n, P, halo in ((1000, 3, 40), (9804, 5, 228), (100_000_000, 8, 20_004), (17, 1, 3)):
        plans = [gtb.strip_plan(n, P, halo, p) for p in range(P)]
        assert plans[0]["row0"] == 0 and sum(q["rows"] for q in plans) == n
        for p, q in enumerate(plans):
            assert q["row0"] % 4 == 0 and (p == P - 1 or q["rows"] % 4 == 0)
            assert q["lo_owner"] == (p - 1) % P and q["hi_owner"] == (p + 1) % P
            assert q["lo_first"] == (q["row0"] - halo) % n and q["hi_first"] == (q["row0"] + q["rows"]) % n
            if P > 1:
                assert q["rows"] >= halo
    with pytest.raises(gtb.GtbError):
        gtb.strip_plan(1000, 8, 200, 0)          # 124-row strips, 200-row halo
