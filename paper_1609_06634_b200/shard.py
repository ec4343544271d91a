"""Multi-GPU host logic.  Two ways to shard, both from the paper:
  * IMAGES (default; run_sharded, score_block_and_gather): no data-path collective at all;
  * ORIENTATIONS (run_orientation_sharded): the paper's MPI axis -- every rank holds all images and a slice of the grid, one
    all_gather of the per-chunk partials {m, s, top-8} and one all_reduce of the re-scored candidates; bit-identical to one GPU.

Image sharding: the path shards over IMAGES with no data-path collective (paper: MPI over independent work,
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


def run_in_subsets(ctx, images, subset: int, score=None) -> dict:
    """An image stack that does not fit device memory ("processed in subsets"): `subset` images at a time through one
    configured context, results concatenated in image order.  The calculated images (a1-a3) are built by the first subset and
    reused by the others (the context's cache), so the cost over the whole-stack run is one a0 per subset.  The bits are those of
    the whole-stack run when the orientation chunk is set explicitly (the automatic one depends on the image count)."""
    if subset < 1:
        raise ValueError("run_in_subsets: subset must be >= 1")
    parts = [(score or default_score)(ctx, images[i:i + subset]) for i in range(0, len(images), subset)]
    if not parts:
        return {}
    return {k: np.concatenate([np.asarray(p[k]) for p in parts], axis=0) for k in parts[0]}


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


def orientation_shard(n_orient: int, chunk: int, rank: int, world: int) -> tuple[int, int]:
    """Slice [begin, end) of the orientation grid for rank `rank`: whole chunks of `chunk` orientations (every rank cuts the grid
    at the same places as one GPU with that chunk size would), chunk counts differing by at most one, in grid order."""
    if chunk < 1 or world < 1 or not 0 <= rank < world:
        raise ValueError("orientation_shard: need chunk >= 1, world >= 1, 0 <= rank < world")
    n_chunks = -(-n_orient // chunk)
    b, e = image_shard(n_chunks, rank, world)
    return min(b * chunk, n_orient), min(e * chunk, n_orient)


def run_orientation_sharded(ctx, chunk: int, group=None, orientation_posterior: bool = False) -> dict:
    """Score the images pushed into `ctx` against the whole grid with the orientation grid sharded over the ranks of `group`
    ("MPI over orientations").  `ctx` is a configured BioEM context (models, grids, images; the same on every rank).
    Exchange steps ("absence of communication" but for the final gather): one all_gather of the per-chunk partials, one
    all_reduce of the FP64 re-scored candidates.  Every rank returns the full results, bit-identical to one GPU with
    set_orientation_chunk(chunk) (include/bioem.h).  orientation_posterior=True adds "logp_orient" [I][M][O]: every rank
    computes the entries of its own orientations, one more all_gather puts the parts side by side."""
    import torch
    import torch.distributed as dist

    on = dist.is_available() and dist.is_initialized()
    world = dist.get_world_size(group) if on else 1
    rank = dist.get_rank(group) if on else 0
    if orientation_posterior:
        chunk = min(chunk, 32)                                               # the library's cap with that option (include/bioem.h)
    ob, oe = orientation_shard(ctx.n_orient, chunk, rank, world)
    ctx.set_orientation_chunk(chunk)
    ctx.set_orientation_slice(ob, oe)
    if orientation_posterior:
        ctx.set_orientation_posterior(True)
    try:
        ctx.run_partial()
        if world == 1:
            ctx.merge_partials()
            ctx.rescore_local()
        else:
            dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
            nbytes, nchunks = ctx.get_partials_size()
            meta = torch.tensor([nbytes, nchunks], dtype=torch.int64, device=dev)
            metas = [torch.empty_like(meta) for _ in range(world)]
            dist.all_gather(metas, meta, group=group)
            sizes = [int(m[0]) for m in metas]
            chunks = [int(m[1]) for m in metas]
            stride = max(max(sizes), 4)
            mine = torch.zeros(stride, dtype=torch.uint8, device=dev)
            ctx.export_partials(mine)
            allb = torch.empty(world * stride, dtype=torch.uint8, device=dev)
            dist.all_gather_into_tensor(allb, mine, group=group) if dev.type == "cuda" else \
                dist.all_gather(list(allb.view(world, stride).unbind(0)), mine, group=group)
            ctx.merge_partials(allb, stride, chunks)
            ctx.rescore_local()
            g = torch.empty(ctx.rescore_shape(), dtype=torch.float64, device=dev)
            ctx.export_rescore(g)
            dist.all_reduce(g, op=dist.ReduceOp.SUM, group=group)            # owner's value + exact zeros
            ctx.import_rescore(g)
        ctx.finish()
        out = dict(logp=ctx.get_log_posterior(), **ctx.get_best())
        if orientation_posterior:
            part = ctx.get_orientation_log_posterior()                       # [I][M][oe - ob]
            if world == 1:
                out["logp_orient"] = part
            else:
                spans = [orientation_shard(ctx.n_orient, chunk, r, world) for r in range(world)]
                width = max(max(e - b for b, e in spans), 1)
                mine = torch.zeros(part.shape[:2] + (width,), dtype=torch.float64, device=dev)
                mine[:, :, : oe - ob] = torch.from_numpy(part).to(dev)
                parts = [torch.empty_like(mine) for _ in range(world)]
                dist.all_gather(parts, mine, group=group)
                out["logp_orient"] = np.concatenate([p[:, :, : e - b].cpu().numpy() for p, (b, e) in zip(parts, spans)], axis=2)
        return out
    finally:
        ctx.set_orientation_slice(0, -1)
        if orientation_posterior:
            ctx.set_orientation_posterior(False)
