"""PyTorch plumbing for liboptcc: device memory and streams only (no arithmetic of the method lives here).

`Session` owns the device buffers a plan needs (p rank buffers + the workspace) and forwards to the C-ABI calls
of `binding`.  It fails loudly without CUDA: there is no CPU path.
"""
import numpy as np
import torch

from . import binding as B


def _require_cuda():
    if not torch.cuda.is_available():
        raise RuntimeError("liboptcc executes on a CUDA device (B200, sm_100a); no GPU is visible and there is no CPU fallback")


class Session:
    """Device state for one plan: rank buffers (separate allocations, so any n keeps 16-byte alignment),
    workspace sized for execute (and verify, if asked).  shards > 1: the rank buffers hold `shards` element shards
    of the plan's n each (optcc_execute_host_sharded)."""

    def __init__(self, plan, device="cuda:0", verify=False, alloc_bufs=True, shards=1):
        _require_cuda()
        self.plan = plan
        self.device = torch.device(device)
        i = plan.info
        self.p, self.n = i["p"], i["n"]
        self.torch_dtype = torch.float32 if i["dtype"] == B.OPTCC_F32 else torch.bfloat16
        self.np_dtype = np.float32 if i["dtype"] == B.OPTCC_F32 else np.uint16
        nbytes = i["verify_workspace_bytes"] if verify else i["workspace_bytes"]
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(int(nbytes) + 256, dtype=torch.uint8, device=self.device)
            off = (-self.workspace.data_ptr()) % 256
            self.ws_ptr = self.workspace.data_ptr() + off
            self._ws_off = off
            self.shards = int(shards)
            self.bufs = [torch.empty(self.n * self.shards, dtype=self.torch_dtype, device=self.device) for _ in range(self.p)] if alloc_bufs else None

    # -- data movement (plumbing) --
    def upload(self, x):
        """x: [p, n] numpy array (float32, or uint16 bf16 bit patterns) or list of p arrays."""
        for r in range(self.p):
            a = np.ascontiguousarray(x[r])
            if self.torch_dtype == torch.bfloat16:
                t = torch.from_numpy(a.view(np.int16)).view(torch.bfloat16)   # bit patterns, no conversion
            else:
                t = torch.from_numpy(a)
            self.bufs[r].copy_(t, non_blocking=False)

    def download(self, ranks=None):
        """-> numpy [len(ranks), n] (float32, or uint16 bf16 bit patterns)."""
        ranks = range(self.p) if ranks is None else ranks
        out = np.empty((len(ranks), self.n), dtype=self.np_dtype)
        for j, r in enumerate(ranks):
            t = self.bufs[r]
            if self.torch_dtype == torch.bfloat16:
                t = t.view(torch.int16)
            out[j] = t.cpu().numpy().view(self.np_dtype)
        return out

    def masks(self):
        """After verify(): contributor masks as numpy uint64 [p, n, W] (W = mask_words), widened from the
        workspace's mask_bytes-wide little-endian storage."""
        i = self.plan.info
        eb, W, pn = i["mask_bytes"], i["mask_words"], i["padded_n"]
        start = self._ws_off + i["mask_offset_bytes"]
        raw = self.workspace[start:start + self.p * pn * eb].cpu().numpy()
        if eb == 2:
            m = raw.view("<u2").reshape(self.p, pn)[:, :self.n].astype(np.uint64)[:, :, None]
        elif eb == 4:
            m = raw.view("<u4").reshape(self.p, pn)[:, :self.n].astype(np.uint64)[:, :, None]
        else:
            m = raw.view("<u8").reshape(self.p, pn, W)[:, :self.n, :]
        return np.ascontiguousarray(m)

    # -- the C-ABI calls --
    def _stream(self, stream):
        s = torch.cuda.current_stream(self.device) if stream is None else stream
        return s.cuda_stream

    def prepare(self, stream=None):
        with torch.cuda.device(self.device):
            B.optcc_prepare(self.plan, self.ws_ptr, self._stream(stream))

    def execute(self, stream=None):
        with torch.cuda.device(self.device):
            B.optcc_execute(self.plan, self.bufs, self.ws_ptr, self._stream(stream))

    def execute_host(self, host_in, host_out, stream=None):
        with torch.cuda.device(self.device):
            B.optcc_execute_host(self.plan, host_in, host_out, self.bufs, self.ws_ptr, self._stream(stream))

    def execute_host_sharded(self, host_in, host_out, stream=None):
        with torch.cuda.device(self.device):
            B.optcc_execute_host_sharded(self.plan, self.n * self.shards, host_in, host_out, self.bufs, self.ws_ptr,
                                         self._stream(stream))

    def check(self, stream=None):
        with torch.cuda.device(self.device):
            B.optcc_workspace_check(self.plan, self.ws_ptr, self._stream(stream))

    def __del__(self):
        try:
            B.optcc_workspace_forget(self.ws_ptr)     # the address may come back from the allocator for something else
        except Exception:
            pass

    def verify(self, stream=None, raise_on_fail=True):
        with torch.cuda.device(self.device):
            return B.optcc_verify(self.plan, self.ws_ptr, self._stream(stream), raise_on_fail=raise_on_fail)
