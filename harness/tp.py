"""Tensor-parallel view of stage 4 (PAPER.md 6.1 L271: TP=2 on the paper's testbed).

Decisions (stages 1-3) are replicated on every TP rank: same inputs, same deterministic kernels, same victim list,
no collective.  Stage 4 shards by KV head: a chunk is [kv_head][token][dim], so rank t of `tp` owns bytes
[t*cb/tp, (t+1)*cb/tp) of every chunk of every block, in its OWN pool on its OWN GPU behind its OWN PCIe link.
Swap-out / swap-in of a rank therefore touch nothing another rank touches: independent units, no exchange.

This module holds the slicing arithmetic and the per-rank driver that `bench.py --gpus N` runs (one process per GPU,
launched by torch.distributed.run).  It is harness code: byte ranges only, none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np


def head_slice(chunk_bytes: int, tp: int, rank: int):
    """(byte offset inside a chunk, bytes) of rank `rank`'s KV-head slice.  chunk_bytes must split evenly into
    16-byte-aligned slices (kv_heads % tp == 0 in every model the paper names)."""
    if tp < 1 or not 0 <= rank < tp:
        raise ValueError("rank outside the TP group")
    if chunk_bytes % tp or (chunk_bytes // tp) % 16:
        raise ValueError("chunk does not split into 16-byte aligned head slices")
    sb = chunk_bytes // tp
    return rank * sb, sb


def shard_pool(full: np.ndarray, tp: int, rank: int, layout: str) -> np.ndarray:
    """Rank `rank`'s pool bytes cut out of an unsharded pool given as uint8[chunk][block][byte]."""
    off, sb = head_slice(full.shape[2], tp, rank)
    shard = full[:, :, off:off + sb]
    if layout == "layer":
        return np.ascontiguousarray(shard).reshape(-1)
    return np.ascontiguousarray(shard.transpose(1, 0, 2)).reshape(-1)   # block-major


def interleave_pages(rank_pages, n: int, n_chunks: int) -> np.ndarray:
    """The unsharded staged pages uint8[n][chunk][byte] rebuilt from the ranks' staged pages (rank order)."""
    parts = [np.asarray(p, np.uint8).reshape(n, n_chunks, -1) for p in rank_pages]
    return np.concatenate(parts, axis=2)


def tp_swap_sweep(torch, cw, gen, hdist, stream, rank: int, world: int, ns=(64, 512), n_chunks: int = 160,
                  chunk_bytes: int = 32768, M: int = 12288):
    """BASELINE.json configs[3] sharded over `world` TP ranks (one GPU and one PCIe link each): every rank swaps the
    SAME victims of its own head slice out and back in; time = the slowest rank's device time, bytes = all ranks'."""
    off, sb = head_slice(chunk_bytes, world, rank)
    page = n_chunks * sb
    rows = []
    with torch.cuda.stream(stream):
        pool = torch.empty(M * page, dtype=torch.uint8, device="cuda")
        pv = pool.view(torch.int64)
        for o in range(0, pv.numel(), 1 << 27):                 # distinct content per rank, filled in 1 GiB pieces
            e = min(pv.numel(), o + (1 << 27))
            torch.arange(o, e, dtype=torch.int64, device="cuda", out=pv[o:e])
            pv[o:e].mul_(2 * rank + 1)
        ctx = cw.Context(num_blocks=M, table_log2_slots=15, max_requests=1, max_hashed_blocks=1, n_chunks=n_chunks,
                         chunk_bytes=sb, chunk_stride=M * sb, block_stride=sb, pool=pool,
                         staging_bytes=2 * (320 << 20), stream_main=stream)
        nmax = max(ns)
        h = torch.empty(nmax * page, dtype=torch.uint8).pin_memory()
        p3 = pool.view(n_chunks, M, sb)
        for n in ns:
            vic = torch.from_numpy(gen.swap_victims(4, M, n).astype(np.int32)).cuda()   # replicated decision
            t = {}
            for name, fn in (("out", lambda: (ctx.swap_out(vic, None, n, None, h), ctx.join_copy())),
                             ("in", lambda: ctx.swap_in(None, h, vic, n))):
                best = 1e30
                for i in range(4):
                    hdist.barrier()
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    fn()
                    e1.record(stream)
                    ctx.sync()
                    if i:
                        best = min(best, e0.elapsed_time(e1))
                t[name] = best
            sample = vic[: min(n, 4)].long()
            ok = bool(torch.equal(p3[:, sample, :].permute(1, 0, 2).reshape(sample.numel(), page).cpu(),
                                  h.view(nmax, page)[: sample.numel()]))
            row = {"n_blocks": n, "rank_page_bytes": page, "pages_ok": ok}
            for name in ("out", "in"):
                bytes_all, ms = hdist.aggregate(float(n * page), t[name], "cuda")
                row[f"swap_{name}_gbs_all_links"] = round(bytes_all / ms / 1e6, 2)
            ok_all, _ = hdist.aggregate(1.0 if ok else 0.0, 1.0, "cuda")
            row["pages_ok"] = bool(ok_all == world)
            rows.append(row)
        ctx.close()
        del pool, h, p3, pv
    torch.cuda.empty_cache()
    return {"tp": world, "head_slice_bytes_per_chunk": sb, "rows": rows,
            "note": "every rank swaps the same victims of its own KV-head slice over its own PCIe link; no collective"}
