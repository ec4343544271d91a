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


def test_run_in_subsets_concatenates_in_image_order():
    # a stack processed in subsets; ragged last subset, a subset larger than the stack, an empty stack
    from paper_1609_06634_b200.shard import run_in_subsets
    rng = np.random.default_rng(3)
    images = rng.normal(size=(11, 4, 4)).astype(np.float32)
    want = _score(None, images)
    for subset in (1, 3, 4, 11, 50):
        got = run_in_subsets(None, images, subset, score=_score)
        assert set(got) == set(want) and all(np.array_equal(got[k], want[k]) and got[k].dtype == want[k].dtype for k in want)
    assert run_in_subsets(None, images[:0], 4, score=_score) == {}
    with pytest.raises(ValueError):
        run_in_subsets(None, images, 0, score=_score)


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


# ------------------------------------------------------------------ orientation sharding
def test_orientation_shard_cuts_whole_chunks():
    from paper_1609_06634_b200.shard import orientation_shard
    for n_orient, chunk in ((40, 5), (41, 5), (4096, 32), (7, 32), (64, 1)):
        for world in (1, 2, 3, 8):
            sl = [orientation_shard(n_orient, chunk, r, world) for r in range(world)]
            assert sl[0][0] == 0 and sl[-1][1] == n_orient
            assert all(sl[i][1] == sl[i + 1][0] for i in range(world - 1))
            assert all(b % chunk == 0 for b, e in sl if e > b)


class _FakeCtx:
    """Stand-in for BioEM with the phased calls of include/bioem.h and the same buffer contracts (a byte blob of per-chunk
    partials, an [I][M][K] re-score array), computing on the host from a seeded score table: what is under test is the exchange in
    shard.run_orientation_sharded (ragged blobs, chunk order, all_reduce of owner-or-zero values), not the kernels."""
    K = 8

    def __init__(self, n_img, n_models, n_orient):
        self.n_img, self.n_models, self.n_orient = n_img, n_models, n_orient
        rng = np.random.default_rng(11)
        self.score = rng.normal(size=(n_img, n_models, n_orient)).astype(np.float32)      # "log-term" of (image, model, orientation)
        self.fine = self.score.astype(np.float64) + rng.normal(size=self.score.shape) * 1e-3   # its "FP64 re-scored" value
        self.chunk, self.sl = 0, (0, n_orient)

    def set_orientation_chunk(self, c):
        self.chunk = c

    def set_orientation_slice(self, b, e):
        self.sl = (b, e) if e >= 0 else (0, self.n_orient)

    def run_partial(self):
        b, e = self.sl
        assert b % self.chunk == 0
        self.nch = -(-(e - b) // self.chunk)
        # blob: float32 sum per (model, chunk, image) then int32 argmax orientation (global index) per (model, chunk, image)
        sums = np.zeros((self.n_models, self.nch, self.n_img), np.float32)
        arg = np.zeros((self.n_models, self.nch, self.n_img), np.int32)
        for ch in range(self.nch):
            o0, o1 = b + ch * self.chunk, min(b + (ch + 1) * self.chunk, e)
            for o in range(o0, o1):                               # float32 accumulation in grid order inside a chunk
                sums[:, ch, :] = sums[:, ch, :] + self.score[:, :, o].T
            arg[:, ch, :] = (np.argmax(self.score[:, :, o0:o1], axis=2) + o0).T
        self.blob = np.concatenate([sums.ravel().view(np.uint8), arg.ravel().view(np.uint8)])

    def get_partials_size(self):
        return self.blob.size, self.nch

    def export_partials(self, dst):
        dst.numpy()[: self.blob.size] = self.blob

    def merge_partials(self, blobs=None, stride_bytes=0, chunks_of_blob=None):
        if blobs is None:
            blobs, stride_bytes, chunks_of_blob = self.blob, self.blob.size, [self.nch]
        else:
            blobs = blobs.numpy()
        tot = np.zeros((self.n_img, self.n_models), np.float32)
        cand = []
        for r, nch in enumerate(chunks_of_blob):
            raw = blobs[r * stride_bytes: r * stride_bytes + nch * self.n_models * self.n_img * 8]
            n = nch * self.n_models * self.n_img
            sums = raw[: 4 * n].view(np.float32).reshape(self.n_models, nch, self.n_img)
            arg = raw[4 * n: 8 * n].view(np.int32).reshape(self.n_models, nch, self.n_img)
            for ch in range(nch):                                 # blobs in rank order, chunks in order: the 1-rank order
                tot = tot + sums[:, ch, :].T
                cand.append(arg[:, ch, :].T)
        self.tot = tot
        cand = np.stack(cand, axis=2)                             # [I][M][all chunks]: candidate orientations
        sc = np.take_along_axis(self.score, cand, axis=2)
        order = np.argsort(-sc, axis=2, kind="stable")[:, :, : self.K]
        self.cand = np.take_along_axis(cand, order, axis=2)
        if self.cand.shape[2] < self.K:
            self.cand = np.concatenate([self.cand, -np.ones((self.n_img, self.n_models, self.K - self.cand.shape[2]), np.int32)], axis=2)

    def rescore_local(self):
        b, e = self.sl
        own = (self.cand >= b) & (self.cand < e)
        self.g = np.where(own, np.take_along_axis(self.fine, np.clip(self.cand, 0, None), axis=2), 0.0)

    def rescore_shape(self):
        return (self.n_img, self.n_models, self.K)

    def export_rescore(self, dst):
        dst.numpy()[...] = self.g

    def import_rescore(self, src):
        self.g = src.numpy().copy()

    def finish(self):
        pass

    def set_orientation_posterior(self, on):
        self.want_po = bool(on)

    def get_orientation_log_posterior(self):
        """This rank's orientations only, [I][M][e - b]: the FP32 score, with the re-scored candidates that fall on the
        orientation (known on every rank after the all_reduce) added -- so a wrong gather AND a stale g both show."""
        assert self.want_po
        b, e = self.sl
        out = self.score[:, :, b:e].astype(np.float64)
        for k in range(self.K):
            c = self.cand[:, :, k]
            own = (c >= b) & (c < e)
            i, m = np.nonzero(own)
            out[i, m, c[i, m] - b] += self.g[i, m, k]
        return out

    def get_log_posterior(self):
        return self.tot.astype(np.float64) + self.g.max(axis=2)

    def get_best(self):
        k = np.argmax(np.where(self.cand >= 0, self.g, -np.inf), axis=2)
        return dict(orient=np.take_along_axis(self.cand, k[:, :, None], axis=2)[:, :, 0].astype(np.int32))


def _orient_worker(rank, world, port, q):
    import torch.distributed as dist
    from paper_1609_06634_b200.shard import run_orientation_sharded
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        out = run_orientation_sharded(_FakeCtx(5, 2, 43), chunk=4, orientation_posterior=True)   # 11 chunks, the last one ragged: 6 + 5 over two ranks
        q.put((rank, {k: v.tolist() for k, v in out.items()}))
    finally:
        dist.destroy_process_group()


def test_orientation_sharding_two_ranks_equal_one_rank():
    import torch.multiprocessing as mp
    from paper_1609_06634_b200.shard import run_orientation_sharded
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_orient_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    want = run_orientation_sharded(_FakeCtx(5, 2, 43), chunk=4, orientation_posterior=True)    # no process group: one rank, the whole grid
    assert want["logp_orient"].shape == (5, 2, 43)
    for r in range(2):
        assert np.array_equal(np.array(got[r]["logp"]), want["logp"])                   # bit-identical on every rank
        assert np.array_equal(np.array(got[r]["logp_orient"]), want["logp_orient"])     # each rank's part, side by side
        assert np.array_equal(np.array(got[r]["orient"], dtype=np.int32), want["orient"])
