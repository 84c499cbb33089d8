"""World-size-2 `gloo` test of the multi-GPU plumbing:
step ranges tile the run, the long-exposure all-reduce sums the per-rank PSFs, timing is max over ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1608_00386_b200 import sharding


def test_step_ranges_tile_the_run():
    for world in (1, 2, 3, 8):
        for total in (0, 1, 7, 1000):
            got = [sharding.split_steps(r, world, total, step0=5) for r in range(world)]
            assert sum(c for _, c in got) == total
            nxt = 5
            for first, count in got:
                assert first == nxt
                nxt += count
        weak = [sharding.step_range(r, world, 50, step0=3) for r in range(world)]
        assert weak == [(3 + 50 * r, 50) for r in range(world)]


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    r, lr, w = sharding.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    first, count = sharding.split_steps(r, w, 7)
    # stand-in for the per-rank long exposure: step k contributes k+1 to every pixel
    psf = torch.zeros(4, 4, dtype=torch.float32)
    for k in range(first, first + count):
        psf += float(k + 1)
    # every rank loads the C-ABI library itself (one process per GPU); without a CUDA device the library must refuse
    # loudly instead of falling back to anything (the compute calls are covered on the GPU by tests/test_gpu_*.py)
    from paper_1608_00386_b200 import binding, inputs
    lib = binding.load_library()
    version = lib.ao_version().decode()
    refused = None
    if not torch.cuda.is_available():
        try:
            binding.Geometry(inputs.make_config(0), device="cuda:0")
        except Exception as ex:          # RuntimeError from the binding or AoError(AO_ERR_CUDA) from ao_geometry_create
            refused = type(ex).__name__
    sharding.barrier()
    sharding.sum_over_ranks_(psf)
    t = sharding.max_over_ranks(0.5 + rank)
    out.put((rank, psf.numpy().copy(), t, first, count, version, refused))
    dist.destroy_process_group()


def test_two_rank_gloo_psf_allreduce_and_max_time():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=120) for _ in procs), key=lambda x: x[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, psf, t, first, count, version, refused in res:
        assert np.all(psf == float(sum(range(1, 8))))     # 1+...+7 over both ranks
        assert t == 1.5                                    # max over ranks
        assert "sm_100a" in version and "normal build" in version
        assert torch.cuda.is_available() or refused in ("RuntimeError", "AoError")
    assert [(r[3], r[4]) for r in res] == [(0, 4), (4, 3)]
