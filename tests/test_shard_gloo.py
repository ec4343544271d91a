"""N > 1 host logic on CPU: world_size-2 gloo run of paper_1609_06634_b200.shard (images shard, no data-path
collective, results concatenated in image order).  The scoring call is a stand-in (a per-image function of the pixels):
what is under test is the partition, the ragged gather and the ordering, not the kernels."""
import os
import socket

import numpy as np
import pytest

from paper_1609_06634_b200.shard import image_shard


def test_image_shard_partitions_exactly():
    for n in (0, 1, 2, 5, 16, 255, 256, 1023):
        for world in (1, 2, 3, 4, 8):
            blocks = [image_shard(n, r, world) for r in range(world)]
            assert blocks[0][0] == 0 and blocks[-1][1] == n
            assert all(blocks[i][1] == blocks[i + 1][0] for i in range(world - 1))
            sizes = [e - b for b, e in blocks]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        image_shard(4, 2, 2)


def _score(ctx, block):
    # stand-in for push_images + run + get_*: any per-image function; int and float outputs, 2-D like [I][M]
    s = block.reshape(len(block), -1).astype(np.float64)
    return dict(logp=np.stack([s.sum(1), (s * s).sum(1)], axis=1), orient=np.argmax(s, axis=1).astype(np.int32)[:, None])


def _worker(rank, world, port, n_img, q):
    import torch.distributed as dist
    from paper_1609_06634_b200.shard import run_sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        imgs = np.random.default_rng(7).normal(size=(n_img, 6, 6)).astype(np.float32)     # same stack on every rank
        out = run_sharded(lambda: None, imgs, score=_score)
        q.put((rank, {k: v.tolist() for k, v in out.items()}))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_img", [7, 1])
def test_two_ranks_equal_one_rank(n_img):
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n_img, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    imgs = np.random.default_rng(7).normal(size=(n_img, 6, 6)).astype(np.float32)
    want = _score(None, imgs)
    for r in range(2):
        assert np.array_equal(np.array(got[r]["logp"]), want["logp"])                   # bit-identical, image order kept
        assert np.array_equal(np.array(got[r]["orient"], dtype=np.int32), want["orient"])
