"""Host-side multi-GPU plumbing (paper_2208_09136_b200/shard.py) under gloo on CPU, world size 2: the path shards by
independent series with no data-path collective; the only communication is the timing reduction bench.py uses
(barrier, max-over-ranks time, summed units)."""
import os
import socket

import pytest

from paper_2208_09136_b200 import shard, workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import torch.distributed as dist
    r, w = shard.init_process_group("gloo")
    assert (r, w) == (rank, world)
    real = shard.realisations_for_rank(r, w)
    shard.barrier(w)
    # rank r "processed" (r+1)*1000 units in (r+1)*10 ms: the job's time is the slowest rank's, units add up
    value, ms = shard.whole_job_throughput((r + 1) * 1000.0, (r + 1) * 10.0, w)
    mx = shard.max_over_ranks(float(r), w)
    out.put((r, real, value, ms, mx))
    shard.barrier(w)
    dist.destroy_process_group()


def test_world_size_2_gloo():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [[0], [1]]                  # disjoint realisations: weak scaling, no exchange
    for _, _, value, ms, mx in res:
        assert ms == 20.0 and mx == 1.0
        assert value == pytest.approx(3000.0 / 20e-3)


def test_ranks_get_distinct_series():
    """Different realisations give different noise, same shape: per-GPU work is fixed as the job grows."""
    a = wl.config4(N=500, which=[4], realisation=shard.realisations_for_rank(0, 2)[0])
    b = wl.config4(N=500, which=[4], realisation=shard.realisations_for_rank(1, 2)[0])
    assert a.series.shape == b.series.shape and a.units == b.units
    assert not (a.series == b.series).all()
    with pytest.raises(ValueError):
        shard.realisations_for_rank(2, 2)


def test_single_process_is_a_no_op():
    assert shard.max_over_ranks(3.5, 1) == 3.5 and shard.sum_over_ranks(2.0, 1) == 2.0
    assert shard.whole_job_throughput(100.0, 50.0, 1) == (2000.0, 50.0)
    shard.barrier(1)


# ------------------------------------------------------ the reduce callback of a split call, under gloo on CPU
def _reduce_worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1",
                      MASTER_PORT=str(port))
    import numpy as np
    import torch.distributed as dist
    from paper_2208_09136_b200 import binding as B, parts
    shard.init_process_group("gloo")
    # the counters a part would hand over: uint64 values, including ones above 2^63 (int64 addition wraps like uint64)
    a = np.array([rank + 1, 10 * (rank + 1), (1 << 63) + rank, 0], dtype=np.uint64)
    opt = B.make_options(part_index=rank, part_count=world, reduce=parts.dist_reduce("cpu"))
    # call the callback exactly as librqa.so does: through the C function pointer stored in rqa_options
    rc = opt.reduce(None, a.ctypes.data, a.size, None)
    out.put((rank, rc, [int(x) for x in a]))
    shard.barrier(world)
    dist.destroy_process_group()


def test_split_call_reduce_callback_world_size_2_gloo():
    """rqa_options.reduce for one process per GPU (parts.dist_reduce): an in-place all-reduce(sum) of exact uint64
    counters.  gloo on host memory stands in for NCCL on device memory; the callback is invoked through the same C
    function pointer the library calls."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_reduce_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    expect = [3, 30, ((1 << 63) + (1 << 63) + 1) % (1 << 64), 0]
    for _, rc, vals in res:
        assert rc == 0 and vals == expect


def test_split_call_options_are_validated_without_a_gpu():
    """part_index / part_count change the tiling and hence the workspace size; sizes are computable on a CPU-only box
    and the parts of one call agree on every shared buffer's size (same sequence of reduce calls with the same n)."""
    from paper_2208_09136_b200 import binding as B
    B.load_library()
    v = B.RqaPoints()
    v.data, v.n_points, v.m, v.batch, v.point_stride, v.coord_stride, v.batch_stride, v.theiler = None, 50000, 3, 2, 1, 1, 50002, 0
    noop = lambda ptr, n, stream: None                      # noqa: E731
    whole = B.rqa_workspace_bytes(v, 20)
    sizes = [B.rqa_workspace_bytes(v, 20, B.make_options(part_index=p, part_count=4, reduce=noop)) for p in range(4)]
    assert all(s > 0 for s in sizes) and max(sizes) <= whole
    with pytest.raises(B.RqaError):
        B.rqa_workspace_bytes(v, 20, B.make_options(part_index=4, part_count=4, reduce=noop))
    with pytest.raises(B.RqaError):
        B.rqa_workspace_bytes(v, 20, B.make_options(part_index=0, part_count=2))       # a split needs a reduce callback
