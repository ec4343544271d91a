"""Multi-GPU host logic: the path shards over IMAGES with no data-path collective (paper: MPI over independent work,
"absence of both communication and load-imbalances").  One process per GPU; every rank
holds the models and grids, scores its contiguous block of the image stack, and the per-image results are
concatenated in image order with one all_gather at the end (results only: a few bytes per image, not on the data path).
Because an image's result never depends on another image, the gathered output is bit-identical to a 1-GPU run.

Nothing here computes anything of the method: `score` is BioEM.push_images + run + get_* on the rank's block.
"""
from __future__ import annotations

import numpy as np


def image_shard(n_images: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous block [begin, end) of rank `rank`: sizes differ by at most one, earlier ranks take the remainder."""
    if world < 1 or not 0 <= rank < world or n_images < 0:
        raise ValueError("image_shard: need world >= 1, 0 <= rank < world, n_images >= 0")
    q, r = divmod(n_images, world)
    begin = rank * q + min(rank, r)
    return begin, begin + q + (1 if rank < r else 0)


def gather_by_image(local: dict, n_images: int, group=None) -> dict:
    """all_gather the per-image result arrays (first axis = this rank's images) into full arrays in image order.
    Works with any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests); ragged blocks are padded."""
    import torch
    import torch.distributed as dist

    if not dist.is_available() or not dist.is_initialized():
        return {k: np.asarray(v) for k, v in local.items()}
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    cap = max(image_shard(n_images, r, world)[1] - image_shard(n_images, r, world)[0] for r in range(world))
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    out = {}
    for k in sorted(local):
        a = np.ascontiguousarray(local[k])
        b, e = image_shard(n_images, rank, world)
        if a.shape[0] != e - b:
            raise ValueError(f"gather_by_image: '{k}' has {a.shape[0]} rows, this rank owns {e - b} images")
        pad = np.zeros((cap,) + a.shape[1:], dtype=a.dtype)
        pad[: a.shape[0]] = a
        t = torch.from_numpy(pad).to(dev)
        parts = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(parts, t, group=group)
        rows = []
        for r, p in enumerate(parts):
            rb, re_ = image_shard(n_images, r, world)
            rows.append(p[: re_ - rb].cpu().numpy())
        out[k] = np.concatenate(rows, axis=0)
    return out


def default_score(ctx, block) -> dict:
    """The library calls on one block of images: a0 (push_images), a1-a7 (run), results."""
    ctx.push_images(block)
    ctx.run()
    return dict(logp=ctx.get_log_posterior(), **ctx.get_best())


def score_block_and_gather(ctx, block, n_images: int, score=None, group=None) -> dict:
    """This rank already holds ITS block of a stack of `n_images` images (block r = image_shard(n_images, r, world); e.g. each
    rank read its own part of the stack): score it and all_gather the per-image results in image order."""
    import torch.distributed as dist

    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    b, e = image_shard(n_images, rank, world)
    if len(block) != e - b:
        raise ValueError(f"score_block_and_gather: rank {rank} owns images [{b}, {e}) but was handed {len(block)}")
    return gather_by_image((score or default_score)(ctx, block), n_images, group)


def run_sharded(make_ctx, images, score=None, group=None) -> dict:
    """Score `images` ([I][N][N]) across the ranks of `group`.  `make_ctx()` returns a configured context (models and
    grids set, no images); `score(ctx, block)` returns a dict of per-image arrays and defaults to the library calls."""
    import torch.distributed as dist

    world = dist.get_world_size(group) if dist.is_initialized() else 1
    rank = dist.get_rank(group) if dist.is_initialized() else 0
    b, e = image_shard(len(images), rank, world)

    ctx = make_ctx()
    local = (score or default_score)(ctx, images[b:e]) if e > b else None
    if local is None:                                         # more ranks than images: contribute empty blocks
        probe = (score or default_score)(ctx, images[:1]) if len(images) else {}
        local = {k: np.asarray(v)[:0] for k, v in probe.items()}
    return gather_by_image(local, len(images), group)
