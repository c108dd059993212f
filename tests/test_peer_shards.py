"""Ranks on several GPUs (include/optcc.h "ranks on several GPUs"; paper_2606_01680_b200/peers.py).

CPU part (gloo, world size 2): who owns which rank, the handle exchange, and that the shards of the column executor's
work items tile every region exactly once.  GPU part: two processes share the one GPU this pool gives a call; each owns
half of the ranks' buffers, opens the other half across the process boundary, runs its shard of the work items over all
p buffers, and after the barrier every process's own ranks hold the oracle's bits.  The kernels of different processes
never wait for one another (the only joins are host barriers), so sharing a GPU is safe; what is NOT exercised is the
NVLink path itself (peer accesses go to the same HBM here).
"""
import json
import os
import socket
import subprocess
import sys
import textwrap

import numpy as np
import pytest

from paper_2606_01680_b200 import binding as B
from paper_2606_01680_b200 import peers as P
from paper_2606_01680_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _spawn(script_text, tmp_path, world, env_extra, timeout=600):
    script = tmp_path / "worker.py"
    script.write_text(script_text)
    port = _free_port()
    procs = []
    for r in range(world):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(world), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), **env_extra)
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for pr in procs:
        so, se = pr.communicate(timeout=timeout)
        assert pr.returncode == 0, (so[-1500:], se[-3000:])
        outs.append(json.loads([l for l in so.splitlines() if l.startswith("RESULT ")][0][7:]))
    return sorted(outs, key=lambda o: o["rank"])


@pytest.mark.parametrize("p,world", [(16, 2), (16, 8), (5, 2), (7, 3), (128, 8), (4, 4)])
def test_every_rank_has_one_owner_in_contiguous_blocks(p, world):
    owners = [P.owner_of(r, p, world) for r in range(p)]
    assert owners == sorted(owners) and set(owners) == set(range(world))        # contiguous blocks, nobody idle
    sizes = [len(P.local_ranks(s, p, world)) for s in range(world)]
    assert sum(sizes) == p and max(sizes) - min(sizes) <= 1
    assert sorted(r for s in range(world) for r in P.local_ranks(s, p, world)) == list(range(p))


def test_handle_table_rejects_gaps_duplicates_and_short_handles():
    h = lambda r: bytes([r]) * 64
    assert P.handle_table([[(0, h(0)), (1, h(1))], [(2, h(2))]], 3) == [h(0), h(1), h(2)]
    with pytest.raises(ValueError):
        P.handle_table([[(0, h(0))], [(0, h(1)), (1, h(1))]], 2)          # announced twice
    with pytest.raises(ValueError):
        P.handle_table([[(0, h(0))], []], 2)                             # rank 1 missing
    with pytest.raises(ValueError):
        P.handle_table([[(0, b"short"), (1, h(1))]], 2)


@pytest.mark.parametrize("n_shards", [1, 2, 3, 8])
def test_shards_of_the_work_items_tile_every_region_exactly_once(n_shards):
    """What optcc_execute_shard(..., s, S) runs for s = 0 .. S-1 is a partition of the column executor's work items, and
    the items of all shards together cover every 16-byte unit of every region once (host tables, no GPU needed)."""
    p, n = 16, 2 ** 18 + 6
    ell = [8.0 / 7.0] + [1.0] * (p - 1)
    plan = B.optcc_plan(p, 1, ell, n, W.F32, k=4, exec_mode=B.OPTCC_EXEC_COLUMN)
    rec, items = B.optcc_column_tables(plan)
    taken = np.zeros(len(items), dtype=np.int32)
    for s in range(n_shards):
        taken[list(P.shard_items(len(items), s, n_shards))] += 1
    assert (taken == 1).all()
    A = plan.info["unit_elems"]
    covered = np.zeros(-(-n // A), dtype=np.int32)
    lists = {}
    for it in items:
        off, ln = int(rec[int(it["first"])]["off"]), int(rec[int(it["first"])]["len"])
        lists.setdefault((off, ln), []).append(it)
    tu = max(int(it["units"]) for it in items)
    for (off, ln), its in lists.items():
        for it in its:
            u0 = off // A + int(it["tile"]) * tu
            covered[u0:u0 + int(it["units"])] += 1
    assert (covered == 1).all()


GLOO_WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import torch.distributed as dist
    from paper_2606_01680_b200 import peers as P
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    p = 6
    mine = P.local_ranks(rank, p, world)
    fake = [(r, bytes([16 * rank + r]) * 64) for r in mine]          # stands in for optcc_peer_alloc's handles
    table = P.handle_table(P.gather_objects(fake), p)
    dist.barrier()
    print("RESULT " + json.dumps({"rank": rank, "mine": mine, "table": [t[0] for t in table]}), flush=True)
    dist.destroy_process_group()
""") % ROOT


def test_handle_exchange_over_gloo(tmp_path):
    outs = _spawn(GLOO_WORKER, tmp_path, 2, {"CUDA_VISIBLE_DEVICES": ""}, timeout=240)
    assert outs[0]["mine"] == [0, 1, 2] and outs[1]["mine"] == [3, 4, 5]
    want = [0, 1, 2, 16 + 3, 16 + 4, 16 + 5]                           # every rank's handle from the process that owns it
    assert outs[0]["table"] == want and outs[1]["table"] == want      # the same table, in rank order, on every process


GPU_WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np
    import torch, torch.distributed as dist
    from paper_2606_01680_b200 import binding as B, workloads as W, peers as P
    from oracle import planner as OP, interpreter as OI
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    results = []
    for (p, st, n, dtype, k) in [(8, {3: 1.5}, 300007, W.F32, 4), (16, {0: 8.0 / 7.0}, 2 ** 20 + 6, W.F32, 4),
                                 (5, {2: 1.5}, 50003, W.BF16, 4)]:
        ell = tuple(float(st.get(i, 1.0)) for i in range(p))
        w = W.Workload("peers", p, 1, ell, n, dtype, "normal", 1.0, 77 + p)
        x = W.all_inputs(w)                                            # (every process draws the same seeded inputs)
        plan = B.optcc_plan(p, 1, ell, n, dtype, k=k)
        s = P.PeerSession(plan, rank, world, device="cuda:0", verify=True)
        s.upload_local(x)
        s.execute()
        y = s.download_local()
        oplan = OP.build_plan(p, 1, list(ell), n, dtype, k=k)
        y_or = OI.run_f32(oplan, x) if dtype == W.F32 else OI.run_bf16(oplan, x)
        ok = all(y[r].tobytes() == y_or[r].tobytes() for r in s.mine)
        v = s.verify()
        results.append({"p": p, "mine": s.mine, "ok": bool(ok), "bad": v["bad_elements"], "overlap": v["overlap_elements"],
                        "checked": v["checked"], "remote": len(s.opened)})
        s.close()
    print("RESULT " + json.dumps({"rank": rank, "results": results}), flush=True)
    dist.destroy_process_group()
""") % ROOT


@pytest.mark.gpu
def test_two_processes_each_own_half_of_the_ranks_and_run_half_of_the_tiles(tmp_path):
    outs = _spawn(GPU_WORKER, tmp_path, 2, {}, timeout=900)
    cases = [(8, 300007), (16, 2 ** 20 + 6), (5, 50003)]
    for c, (p, n) in enumerate(cases):
        r0, r1 = outs[0]["results"][c], outs[1]["results"][c]
        assert r0["ok"] and r1["ok"]                                   # every process's own ranks hold the oracle's bits
        assert sorted(r0["mine"] + r1["mine"]) == list(range(p))
        assert r0["remote"] == p - len(r0["mine"]) and r1["remote"] == p - len(r1["mine"])   # the rest came from the peer
        assert r0["bad"] == r0["overlap"] == r1["bad"] == r1["overlap"] == 0
        assert r0["checked"] + r1["checked"] == p * n                  # the two shards' tiles cover every element once
