"""Multi-GPU plumbing: "replicas only".

The OPTCC executor never mixes two element indices, so N GPUs shard a job along the element axis: every rank holds
all p virtual ranks' slice and runs the same plan on it.  There is no data-path collective; torch.distributed is
used only for the barrier around the timed region and the max-over-ranks of the device times.  Backend "nccl" on
GPUs, "gloo" in the CPU tests.
"""
import os
import socket
import subprocess
import sys

import torch
import torch.distributed as dist

from . import workloads as W


class Replicas:
    def __init__(self, backend=None, device=None):
        self.rank = int(os.environ.get("RANK", "0"))
        self.world = int(os.environ.get("WORLD_SIZE", "1"))
        self.local_rank = int(os.environ.get("LOCAL_RANK", "0"))
        self.device = device
        self.active = self.world > 1
        if self.active and not dist.is_initialized():
            backend = backend or ("nccl" if torch.cuda.is_available() else "gloo")
            kw = {"device_id": device} if (backend == "nccl" and device is not None) else {}
            dist.init_process_group(backend, **kw)

    def barrier(self):
        if self.active:
            dist.barrier()

    def max_over_ranks(self, values):
        """Element-wise maximum of a list of floats over all ranks (the timing rule: a step takes as long as the
        slowest rank)."""
        if not self.active:
            return [float(v) for v in values]
        t = torch.tensor(list(values), dtype=torch.float64, device=self.device if dist.get_backend() == "nccl" else "cpu")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return [float(v) for v in t.cpu()]

    def all_true(self, flag):
        """Logical AND of a boolean over all ranks (verification / parity flags)."""
        return self.max_over_ranks([0.0 if flag else 1.0])[0] == 0.0

    def shard(self, w):
        """This rank's shard of a weak-scaled job: the same shape (p, ell, n per rank) with its own input stream --
        the world x n element job is cut along the element axis, rank r takes elements [r n, (r+1) n)."""
        if not self.active:
            return w
        return W.Workload(w.name, w.p, w.g, w.ell, w.n, w.dtype, w.dist, w.sigma, w.seed + 1000 * self.rank, w.note)

    def aggregate(self, per_rank_units, seconds_max):
        """Whole-job throughput: units all ranks processed / the slowest rank's time."""
        return self.world * per_rank_units / seconds_max

    def close(self):
        if self.active and dist.is_initialized():
            dist.destroy_process_group()


def launch(nproc, script, argv, extra_env=None, timeout=None):
    """Start `nproc` replicas of `script argv` on this node, one process per GPU, through torch.distributed.run
    (rendezvous on 127.0.0.1, a free port): what `bench.py --gpus N` does when it is not already running under
    torchrun.  The workers' output is handed through; returns the launcher's exit code."""
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    env = dict(os.environ)
    env.setdefault("NCCL_DEBUG", "WARN")
    if extra_env:
        env.update(extra_env)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={int(nproc)}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), script] + list(argv)
    return subprocess.run(cmd, env=env, timeout=timeout).returncode
