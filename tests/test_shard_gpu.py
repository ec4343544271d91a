"""N > 1 through the real pipeline: two ranks score one stack with the CUDA library, images sharded
(shard.run_sharded) and orientations sharded (shard.run_orientation_sharded), and must reproduce one rank's bits.
  * backend gloo: both ranks use cuda:0 and exchange host tensors -- runs on a one-GPU box.  The ranks' kernels never wait on
    one another (every exchange sits between kernel launches and goes through the host), so sharing the GPU is safe.
  * backend nccl: one GPU per rank, device tensors -- skipped below two devices."""
import os
import socket

import numpy as np
import pytest

import bioem_workloads as W

pytestmark = pytest.mark.gpu
CHUNK = 5


def _worker(rank, world, port, backend, q):
    import torch
    import torch.distributed as dist
    from paper_1609_06634_b200 import BioEM
    from paper_1609_06634_b200.shard import run_orientation_sharded, run_sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dev = rank if backend == "nccl" else 0
    torch.cuda.set_device(dev)
    if backend == "nccl":
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", dev))
    else:
        dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = W.build_workload("small_mid")

        def make_ctx():
            b = BioEM(device=dev)
            b.load_workload(wl, images=False)
            b.set_orientation_chunk(CHUNK)
            return b
        by_img = run_sharded(make_ctx, wl["images"])
        with make_ctx() as b:
            b.push_images(wl["images"])
            by_ori = run_orientation_sharded(b, CHUNK, orientation_posterior=True)
        q.put((rank, {k: np.asarray(v).tolist() for k, v in by_img.items()}, {k: np.asarray(v).tolist() for k, v in by_ori.items()}))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("backend", ["gloo", "nccl"])
def test_two_ranks_reproduce_one_rank(backend):
    import torch
    import torch.multiprocessing as mp
    from paper_1609_06634_b200 import BioEM
    if backend == "nccl" and torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, backend, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = {}
    for _ in procs:
        r, a, b = q.get(timeout=600)
        got[r] = (a, b)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    wl = W.build_workload("small_mid")
    with BioEM() as b:
        b.load_workload(wl)
        b.set_orientation_chunk(CHUNK)
        b.run()
        want = dict(logp=b.get_log_posterior(), **b.get_best())
        b.set_orientation_posterior(True)                                    # the orientation-sharded run asks for P:225 too
        b.run()
        want_po = dict(logp=b.get_log_posterior(), logp_orient=b.get_orientation_log_posterior(), **b.get_best())
    for r in range(2):
        for which, ref in ((0, want), (1, want_po)):                         # images sharded, orientations sharded
            assert set(got[r][which]) == set(ref)
            for k, v in ref.items():
                assert np.array_equal(np.asarray(got[r][which][k], dtype=v.dtype), v), (r, which, k)
