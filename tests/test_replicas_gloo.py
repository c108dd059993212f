"""World-size-2 test of the multi-GPU plumbing on CPU (gloo): shards, barrier, max-over-ranks, aggregate."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import json, os, sys
    sys.path.insert(0, %r)
    import numpy as np
    from paper_2606_01680_b200 import workloads as W
    from paper_2606_01680_b200.replicas import Replicas
    rep = Replicas(backend="gloo")
    w = rep.shard(W.config(0).scaled(4096))
    x = W.all_inputs(w)
    rep.barrier()
    t = rep.max_over_ranks([1.0 + rep.rank, 5.0 - rep.rank])
    ok_all = rep.all_true(True)
    ok_mixed = rep.all_true(rep.rank == 0)
    out = {"rank": rep.rank, "world": rep.world, "seed": w.seed, "first": float(x[1, 7]), "t": t,
           "ok_all": ok_all, "ok_mixed": ok_mixed, "agg": rep.aggregate(100.0, t[0])}
    rep.barrier()
    print("RESULT " + json.dumps(out), flush=True)
    rep.close()
""") % ROOT


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_two_rank_replicas_over_gloo(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        so, se = p.communicate(timeout=240)
        assert p.returncode == 0, se[-2000:]
        outs.append(json.loads([l for l in so.splitlines() if l.startswith("RESULT ")][0][7:]))
    outs.sort(key=lambda o: o["rank"])
    assert [o["world"] for o in outs] == [2, 2]
    assert outs[0]["seed"] != outs[1]["seed"] and outs[0]["first"] != outs[1]["first"]   # every rank has its own shard
    for o in outs:
        assert o["t"] == [2.0, 5.0]                 # max over ranks, the same on every rank
        assert o["ok_all"] is True and o["ok_mixed"] is False
        assert o["agg"] == 2 * 100.0 / 2.0          # whole-job units / slowest rank's time


def test_single_process_is_a_noop():
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK")}
    code = ("import sys; sys.path.insert(0, %r)\n"
            "from paper_2606_01680_b200.replicas import Replicas\n"
            "from paper_2606_01680_b200 import workloads as W\n"
            "r = Replicas(); w = W.config(0)\n"
            "assert not r.active and r.shard(w) is w and r.max_over_ranks([3.0]) == [3.0] and r.all_true(True)\n"
            "assert r.aggregate(10.0, 2.0) == 5.0; r.barrier(); r.close(); print('ok')\n") % ROOT
    res = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=240)
    assert res.returncode == 0 and "ok" in res.stdout, res.stderr[-2000:]


def test_launcher_starts_the_replicas_itself(tmp_path):
    """`bench.py --gpus N` without torchrun goes through replicas.launch: N workers on 127.0.0.1, the same barrier and
    max-over-ranks; here two CPU workers over gloo."""
    import json
    from paper_2606_01680_b200.replicas import launch
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    out = tmp_path / "out.txt"
    wrapper = tmp_path / "wrap.py"
    wrapper.write_text(textwrap.dedent("""
        import os, runpy, sys, io, contextlib
        buf = io.StringIO()
        with contextlib.redirect_stdout(buf):
            runpy.run_path(%r, run_name="__main__")
        with open(%r + "." + os.environ["RANK"], "w") as f:
            f.write(buf.getvalue())
    """) % (str(script), str(out)))
    rc = launch(2, str(wrapper), [], extra_env={"CUDA_VISIBLE_DEVICES": ""}, timeout=300)
    assert rc == 0
    outs = []
    for r in range(2):
        text = open(str(out) + "." + str(r)).read()
        outs.append(json.loads([l for l in text.splitlines() if l.startswith("RESULT ")][0][7:]))
    assert sorted(o["rank"] for o in outs) == [0, 1] and all(o["world"] == 2 and o["t"] == [2.0, 5.0] for o in outs)
