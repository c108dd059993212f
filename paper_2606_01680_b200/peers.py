"""Ranks on several GPUs of one NVLink / NVSwitch domain (include/optcc.h "ranks on several GPUs").

Plumbing only: which process owns which rank, the exchange of the 64-byte buffer handles, views of raw device pointers
as torch tensors for the copies in and out.  Every step of the AllReduce itself runs in liboptcc's kernels
(optcc_execute_shard): process s of S takes the column executor's work items i = s (mod S) through their flow lists over
the p rank buffers, of which its own live in local HBM and the others are mapped from the peers.

Launch one process per GPU (torch.distributed: any backend serves for the exchange and the barriers; the data path
has no collective).  On a box with ONE GPU several processes may share it -- handles open across processes whatever the
device -- which is how tests/test_peer_shards.py exercises this file.
"""
import numpy as np

from . import binding as B


def owner_of(rank, p, world):
    """The process that owns `rank`: contiguous blocks of ranks (the GPUs of one server sit next to each other,
    PAPER.md:847), sizes differing by at most one."""
    return (rank * world) // p


def local_ranks(proc, p, world):
    return [r for r in range(p) if owner_of(r, p, world) == proc]


def shard_items(n_items, shard, n_shards):
    """The work items optcc_execute_shard(..., shard, n_shards) runs (include/optcc.h): i = shard (mod n_shards)."""
    return range(shard, n_items, n_shards)


def gather_objects(obj, group=None):
    """[obj of process 0, obj of process 1, ...] on every process."""
    import torch.distributed as dist
    out = [None] * dist.get_world_size(group)
    dist.all_gather_object(out, obj, group=group)
    return out


def handle_table(gathered, p):
    """gathered: per process a list of (rank, handle) -> list of p handles indexed by rank; every rank exactly once."""
    table = [None] * p
    for per_proc in gathered:
        for rank, handle in per_proc:
            if not (0 <= rank < p) or table[rank] is not None:
                raise ValueError(f"rank {rank} announced twice or out of range")
            if len(handle) != 64:
                raise ValueError("a buffer handle is 64 bytes")
            table[rank] = bytes(handle)
    missing = [r for r in range(p) if table[r] is None]
    if missing:
        raise ValueError(f"no process announced ranks {missing}")
    return table


class _DevView:
    """A raw device pointer as something torch.as_tensor understands."""

    def __init__(self, ptr, n, typestr):
        self.__cuda_array_interface__ = {"shape": (int(n),), "typestr": typestr, "data": (int(ptr), False), "version": 2}


class PeerSession:
    """One process's side: buffers of its own ranks (peer-shareable), the peers' buffers opened, a local workspace."""

    def __init__(self, plan, proc, world, device="cuda:0", group=None, verify=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("liboptcc executes on a CUDA device; there is no CPU fallback")
        self.torch = torch
        self.plan, self.proc, self.world, self.group = plan, int(proc), int(world), group
        self.device = torch.device(device)
        i = plan.info
        self.p, self.n = i["p"], i["n"]
        self.bf16 = i["dtype"] == B.OPTCC_BF16
        self.esize = 2 if self.bf16 else 4
        self.mine = local_ranks(self.proc, self.p, self.world)
        self.opened = []
        with torch.cuda.device(self.device):
            torch.cuda.init()
            torch.empty(1, device=self.device)           # the context exists before the library's first call
            own = {}
            for r in self.mine:
                ptr, handle = B.optcc_peer_alloc(max(16, self.n * self.esize))
                own[r] = (ptr, handle)
            self.own = own
            table = handle_table(gather_objects([(r, h) for r, (_, h) in own.items()], group), self.p)
            self.bufs = []
            for r in range(self.p):
                if r in own:
                    self.bufs.append(own[r][0])
                else:
                    q = B.optcc_peer_open(table[r])
                    self.opened.append(q)
                    self.bufs.append(q)
            nbytes = i["verify_workspace_bytes"] if verify else i["workspace_bytes"]
            self.workspace = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=self.device)
            self.ws_ptr = self.workspace.data_ptr() + (-self.workspace.data_ptr()) % 256

    def _view(self, r):
        t = self.torch.as_tensor(_DevView(self.own[r][0], self.n, "<i2" if self.bf16 else "<f4"), device=self.device)
        return t

    def upload_local(self, x):
        """x[r]: numpy array of rank r's n elements (float32, or uint16 bf16 bit patterns) for every own rank r."""
        for r in self.mine:
            a = np.ascontiguousarray(x[r])
            src = self.torch.from_numpy(a.view(np.int16) if self.bf16 else a)
            self._view(r).copy_(src)
        self.torch.cuda.synchronize(self.device)

    def download_local(self):
        out = {}
        for r in self.mine:
            a = self._view(r).cpu().numpy()
            out[r] = a.view(np.uint16) if self.bf16 else a
        return out

    def barrier(self):
        import torch.distributed as dist
        self.torch.cuda.synchronize(self.device)
        dist.barrier(group=self.group)

    def execute(self, stream=None):
        """Inputs of every process in place (barrier), this process's shard, everybody's shard done (barrier)."""
        s = (self.torch.cuda.current_stream(self.device) if stream is None else stream).cuda_stream
        self.barrier()
        with self.torch.cuda.device(self.device):
            B.optcc_execute_shard(self.plan, self.bufs, self.ws_ptr, self.proc, self.world, s)
        self.barrier()

    def verify(self, stream=None, raise_on_fail=True):
        s = (self.torch.cuda.current_stream(self.device) if stream is None else stream).cuda_stream
        with self.torch.cuda.device(self.device):
            return B.optcc_verify_shard(self.plan, self.ws_ptr, self.proc, self.world, s, raise_on_fail)

    def close(self):
        """Peers close what they opened, then (after a barrier) owners free."""
        with self.torch.cuda.device(self.device):
            for q in self.opened:
                B.optcc_peer_close(q)
            self.opened = []
            self.barrier()
            B.optcc_workspace_forget(self.ws_ptr)
            for r, (ptr, _) in self.own.items():
                B.optcc_peer_free(ptr)
            self.own = {}
