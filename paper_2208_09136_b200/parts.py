"""Split of ONE call over several parts (rqa_options.part_index, part_count, reduce).

Each part visits its share of the tiles of the triangle (diagonal blocks dealt round robin) and hands every exact
integer counter that must be summed over the parts to a `reduce` callback; afterwards every part holds the complete,
identical outputs.  This module only builds such callbacks (plumbing, no arithmetic of the method):

  dist_reduce()    one process per GPU: torch.distributed.all_reduce(SUM) on a tensor that wraps the counters in place
                   (NCCL over NVLink for device counters; gloo for the host-memory stand-in the CPU tests use)
  LocalParts       the parts as threads of ONE process on ONE GPU, summed between host barriers: no kernel ever waits
                   on another kernel, the parts simply take turns on the device.  This is how the split is tested where
                   only one GPU is available.
"""
from __future__ import annotations

import ctypes
import threading

import numpy as np


class _CudaArray:
    """Minimal __cuda_array_interface__ holder: n int64 words at a raw device pointer."""

    def __init__(self, ptr: int, n: int):
        self.__cuda_array_interface__ = {"shape": (n,), "typestr": "<i8", "data": (ptr, False), "version": 2}


def counters_tensor(ptr: int, n: int, device: str = "cuda"):
    """A torch int64 tensor that aliases the n uint64 counters at `ptr` (int64 addition is uint64 addition mod 2^64)."""
    import torch
    if device == "cpu":
        buf = (ctypes.c_int64 * n).from_address(ptr)
        return torch.from_numpy(np.frombuffer(buf, dtype=np.int64))
    return torch.as_tensor(_CudaArray(ptr, n), device="cuda")


def dist_reduce(device: str = "cuda", group=None):
    """reduce callback for binding.make_options: all-reduce (sum) over the ranks of `group`, in place, ordered on the
    current torch stream (the stream the library call was given)."""
    import torch.distributed as dist

    def reduce(ptr: int, n: int, stream: int) -> None:
        dist.all_reduce(counters_tensor(ptr, n, device), op=dist.ReduceOp.SUM, group=group)
    return reduce


class LocalParts:
    """Run a call split into `parts` parts inside one process on one GPU: thread p runs fn(p, reduce_p, stream_p) with
    its own stream, buffers and workspace; reduce_p sums the parts' counters between host barriers."""

    def __init__(self, parts: int):
        self.parts = parts
        self.barrier = threading.Barrier(parts)
        self.slots = [None] * parts
        self.reduce_calls = 0

    def _reduce_for(self, p: int):
        import torch

        def reduce(ptr: int, n: int, stream: int) -> None:
            torch.cuda.synchronize()                       # this part's kernels up to here are done
            self.slots[p] = counters_tensor(ptr, n)
            self.barrier.wait()
            if p == 0:
                total = self.slots[0].clone()
                for q in range(1, self.parts):
                    assert self.slots[q].numel() == n, "every part makes the same sequence of reduce calls"
                    total += self.slots[q]
                for q in range(self.parts):
                    self.slots[q].copy_(total)
                torch.cuda.synchronize()
                self.reduce_calls += 1
            self.barrier.wait()
        return reduce

    def run(self, fn):
        import torch
        device = torch.cuda.current_device()
        results, errors = [None] * self.parts, []

        def work(p):
            try:
                torch.cuda.set_device(device)
                stream = torch.cuda.Stream()
                with torch.cuda.stream(stream):
                    results[p] = fn(p, self._reduce_for(p), stream)
                    stream.synchronize()
            except BaseException as e:                      # noqa: BLE001 - reported to the caller below
                errors.append(e)
                self.barrier.abort()
        threads = [threading.Thread(target=work, args=(p,)) for p in range(self.parts)]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        if errors:
            raise errors[0]
        return results
