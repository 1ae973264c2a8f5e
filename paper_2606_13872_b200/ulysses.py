"""Ulysses head-sharded SRA (SURVEY.md 8f #4; PAPER.md:231 "Ulysses sequence parallelism", :253-257).

Outside attention the DiT is sequence-sharded: rank r holds a contiguous range of the generation tokens and of the
reference tokens, all H heads.  SRA needs every key of a head, so around the attention the ranks exchange
sequence shards for head shards (all-to-all), run SRA on their own heads - every (batch, head) is an independent
problem, SURVEY.md 8e - and exchange back.  This module is that plumbing, nothing else: the token / head partition,
the two exchanges, and a driver that pipelines them against the SRA launches by HEAD CHUNKS (the exchange of chunk
c + 1 and the return of chunk c - 1 run on a communication stream underneath the forward of chunk c; chunks are
independent work, so no kernel ever waits on a peer).  All attention arithmetic stays in the C-ABI library
(`binding.sra_forward`); there is no CPU path.

Over NVLink 5 / NVSwitch the exchange of a 720p layer is ~0.6 GB per GPU (~0.7 ms) against ~22 ms of attention per GPU
(SURVEY.md section 5), which is why plain `all_to_all_single` per chunk, overlapped on a stream, is enough and a
tile-level fused kernel is not built.  This run has one GPU per call: the exchange layout is tested with
world-size-2 gloo on CPU (tests/test_dp_gloo.py) and the pipelined driver on one GPU with a world-size-1 group
(tests/test_gpu_ulysses.py); no multi-GPU number is claimed.
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import torch
import torch.distributed as dist

from . import dp


def _world_rank(group) -> Tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_world_size(group), dist.get_rank(group)
    return 1, 0


def head_chunk(heads: int, world: int, rank: int, n_chunks: int, chunk: int) -> Tuple[int, int]:
    """(first head, count) of chunk `chunk` of rank `rank`'s head shard.  Chunks partition the shard; with fewer
    heads than chunks the trailing chunks are empty."""
    h0, hc = dp.shard_heads(heads, world, rank)
    c0, cc = dp.shard_range(hc, n_chunks, chunk)
    return h0 + c0, cc


_RT = False  # cuda.bindings.runtime, resolved once (None if cuda-python is not installed)


def _cuda_runtime():
    """The cuda-python runtime bindings, imported once at first use - never in the middle of a collective, where an
    ImportError on one rank would leave its peers waiting inside all_to_all_single."""
    global _RT
    if _RT is False:
        try:
            from cuda.bindings import runtime as rt
            _RT = rt
        except Exception:
            _RT = None
    return _RT


def _copy_rows(dst: torch.Tensor, src: torch.Tensor) -> None:
    """dst[...] = src[...] for [B, n, h, d] views whose (h, d) block is contiguous and whose token stride is constant
    (a head slice of a [B, n, H, d] tensor, or a token range of one).  On CUDA this is one cudaMemcpy2DAsync per batch
    item on the current stream - the copy engines, not an SM kernel - so that the pack / unpack of a chunk can run
    underneath the forward of its neighbour, whose CTAs fill every SM.  CPU tensors (the gloo tests): plain copy_."""
    assert dst.shape == src.shape and dst.dtype == src.dtype
    B, n, h, d = src.shape
    if B * n * h * d == 0:
        return
    ok = all(t.stride(3) == 1 and t.stride(2) == d for t in (dst, src))
    if not (dst.is_cuda and ok):
        dst.copy_(src)
        return
    rt = _cuda_runtime()
    if rt is None:  # cuda-python absent: an SM copy kernel on the same stream (slower under a running forward, never wrong)
        dst.copy_(src)
        return
    es = src.element_size()
    stream = torch.cuda.current_stream().cuda_stream
    for b in range(B):
        (err,) = rt.cudaMemcpy2DAsync(dst[b].data_ptr(), dst.stride(1) * es, src[b].data_ptr(), src.stride(1) * es,
                                      h * d * es, n, rt.cudaMemcpyKind.cudaMemcpyDeviceToDevice, stream)
        if err != rt.cudaError_t.cudaSuccess:
            raise RuntimeError(f"cudaMemcpy2DAsync failed: {err}")


def seq_to_heads(x: torch.Tensor, n_total: int, heads: int, group=None, n_chunks: int = 1, chunk: int = 0) -> torch.Tensor:
    """Sequence shard -> head shard.  x: [B, n_local, H, d], this rank's contiguous token range
    `dp.shard_range(n_total, world, rank)` with all heads.  Returns [B, n_total, h_cnt, d]: every token, the heads of
    this rank's chunk `chunk` (see `head_chunk`)."""
    world, rank = _world_rank(group)
    B, n_local, H, d = x.shape
    assert H == heads and n_local == dp.shard_range(n_total, world, rank)[1], "x is not this rank's sequence shard"
    my_h0, my_hc = head_chunk(heads, world, rank, n_chunks, chunk)
    out = x.new_empty((B, n_total, my_hc, d))
    if not (dist.is_available() and dist.is_initialized()):  # no process group: one rank, nothing to exchange
        _copy_rows(out, x[:, :, my_h0:my_h0 + my_hc])
        return out
    chunks = [head_chunk(heads, world, r, n_chunks, chunk) for r in range(world)]
    in_splits = [B * n_local * hc * d for _, hc in chunks]
    out_splits = [B * dp.shard_range(n_total, world, s)[1] * my_hc * d for s in range(world)]
    send = x.new_empty(sum(in_splits))
    pos = 0
    for r, (h0, hc) in enumerate(chunks):  # pack: destination r gets its chunk's heads of my tokens
        _copy_rows(send[pos:pos + in_splits[r]].view(B, n_local, hc, d), x[:, :, h0:h0 + hc])
        pos += in_splits[r]
    # B == 1: the pieces arrive in rank = token order, so the receive buffer IS the head shard (no unpack)
    recv = out.view(-1) if B == 1 else x.new_empty(sum(out_splits))
    dist.all_to_all_single(recv, send, out_splits, in_splits, group=group)
    if B > 1:
        pos = 0
        for s in range(world):
            t0, n_s = dp.shard_range(n_total, world, s)
            _copy_rows(out[:, t0:t0 + n_s], recv[pos:pos + out_splits[s]].view(B, n_s, my_hc, d))
            pos += out_splits[s]
    return out


def heads_to_seq(o: torch.Tensor, n_total: int, heads: int, out: torch.Tensor, group=None, n_chunks: int = 1,
                 chunk: int = 0) -> None:
    """Head shard -> sequence shard (the inverse of `seq_to_heads`).  o: [B, n_total, h_cnt, d] for this rank's chunk;
    writes the chunk's heads of every rank into `out` [B, n_local, H, d] (this rank's tokens, all heads)."""
    world, rank = _world_rank(group)
    B, _, my_hc, d = o.shape
    my_h0, hc_chk = head_chunk(heads, world, rank, n_chunks, chunk)
    assert hc_chk == my_hc and o.shape[1] == n_total
    t0_me, n_local = dp.shard_range(n_total, world, rank)
    assert out.shape == (B, n_local, heads, d)
    if not (dist.is_available() and dist.is_initialized()):
        _copy_rows(out[:, :, my_h0:my_h0 + my_hc], o)
        return
    shards = [dp.shard_range(n_total, world, s) for s in range(world)]
    in_splits = [B * n_s * my_hc * d for _, n_s in shards]
    chunks = [head_chunk(heads, world, r, n_chunks, chunk) for r in range(world)]
    out_splits = [B * n_local * hc * d for _, hc in chunks]
    if B == 1:  # token ranges of o are already contiguous and in rank order
        send = o.view(-1)
    else:
        send = o.new_empty(sum(in_splits))
        pos = 0
        for s, (t0, n_s) in enumerate(shards):
            _copy_rows(send[pos:pos + in_splits[s]].view(B, n_s, my_hc, d), o[:, t0:t0 + n_s])
            pos += in_splits[s]
    recv = o.new_empty(sum(out_splits))
    dist.all_to_all_single(recv, send, out_splits, in_splits, group=group)
    pos = 0
    for r, (h0, hc) in enumerate(chunks):  # unpack: rank r's chunk heads of my tokens
        _copy_rows(out[:, :, h0:h0 + hc], recv[pos:pos + out_splits[r]].view(B, n_local, hc, d))
        pos += out_splits[r]


class UlyssesSRA:
    """SRA of a sequence-sharded layer: exchange -> `sra_forward` on this rank's heads -> exchange back, pipelined by
    head chunks.  One SRA context (and one resident reference-KV cache) per chunk; CUDA only."""

    def __init__(self, batch: int, heads: int, head_dim: int, n_gen: int, ref_block_offsets: Sequence[int], group=None,
                 n_chunks: int = 2, scale: float = 0.0):
        from . import binding as B
        if not torch.cuda.is_available():
            raise RuntimeError("UlyssesSRA: no CUDA device; the SRA path has no CPU fallback")
        self.B = B
        _cuda_runtime()  # resolve the optional copy-engine path now, outside any collective
        self.group = group
        self.world, self.rank = _world_rank(group)
        self.batch, self.heads, self.head_dim, self.n_gen = batch, heads, head_dim, n_gen
        self.n_ref = int(ref_block_offsets[-1]) if len(ref_block_offsets) else 0
        # the same chunk count on every rank (the exchanges are collective): at most the largest head shard; a rank
        # with fewer heads has empty trailing chunks and still takes part in their exchanges
        self.n_chunks = max(1, min(n_chunks, -(-heads // self.world)))
        self.chunk_heads = [head_chunk(heads, self.world, self.rank, self.n_chunks, c) for c in range(self.n_chunks)]
        self.ctx = [B.sra_create(batch, cc, head_dim, n_gen, ref_block_offsets, scale) if cc else 0
                    for _, cc in self.chunk_heads]
        self.comm = torch.cuda.Stream()
        self.launches = 0
        self.saved = None

    def close(self) -> None:
        for c in self.ctx:
            if c:
                self.B.sra_destroy(c)
        self.ctx = []

    def gen_shard(self) -> Tuple[int, int]:
        return dp.shard_range(self.n_gen, self.world, self.rank)

    def ref_shard(self) -> Tuple[int, int]:
        return dp.shard_range(self.n_ref, self.world, self.rank)

    def _to_heads(self, x, n_total, c):
        return seq_to_heads(x, n_total, self.heads, self.group, self.n_chunks, c)

    def cache_reference_kv(self, k_ref_seq: torch.Tensor, v_ref_seq: torch.Tensor) -> None:
        """k_ref_seq / v_ref_seq: this rank's reference-token shard [B, n_ref_local, H, d].  Exchanged once; every
        chunk context keeps the cache of its heads (each GPU caches only its heads' K_r, V_r)."""
        for c, ctx in enumerate(self.ctx):
            kh, vh = self._to_heads(k_ref_seq, self.n_ref, c), self._to_heads(v_ref_seq, self.n_ref, c)
            if ctx:
                self.B.sra_cache_reference_kv(ctx, kh, vh)
        torch.cuda.current_stream().synchronize()  # the head-major copies have consumed the temporaries

    def forward(self, q_gen: torch.Tensor, k_gen: torch.Tensor, v_gen: torch.Tensor,
                q_ref: Optional[torch.Tensor] = None, save_for_backward: bool = False):
        """One attention layer on sequence shards ([B, n_local, H, d] each; q_ref = this rank's reference shard on
        step 0 / training, None on cached denoising steps).  Returns (o_gen, o_ref or None) as sequence shards.
        Requires `cache_reference_kv` when n_ref > 0.  `save_for_backward` keeps the head-sharded tensors and the LSE
        of every chunk for `backward` (training: PAPER.md:173, :231)."""
        B = self.B
        if save_for_backward and self.n_ref > 0 and q_ref is None:
            raise ValueError("training needs the reference rows (q_ref)")
        self.saved = [None] * self.n_chunks if save_for_backward else None
        cur = torch.cuda.current_stream()
        comm = self.comm
        o_gen = torch.empty_like(q_gen)
        o_ref = torch.empty_like(q_ref) if q_ref is not None else None
        comm.wait_stream(cur)  # inputs (and the fresh output buffers) are ready for the communication stream
        staged: List[Optional[tuple]] = [None] * self.n_chunks

        def stage(c):  # exchange chunk c's inputs on the communication stream
            with torch.cuda.stream(comm):
                t = (self._to_heads(q_gen, self.n_gen, c), self._to_heads(k_gen, self.n_gen, c),
                     self._to_heads(v_gen, self.n_gen, c),
                     self._to_heads(q_ref, self.n_ref, c) if q_ref is not None else None)
                ev = torch.cuda.Event()
                ev.record(comm)
            staged[c] = (t, ev)

        live = list(range(self.n_chunks))  # every rank walks every chunk: the exchanges are collective
        keep = []  # tensors shared between the two streams stay referenced until the final join
        if live:
            stage(live[0])
        for i, c in enumerate(live):
            if i + 1 < len(live):
                stage(live[i + 1])  # in flight underneath the forward of chunk c
            (qh, kh, vh, qrh), ev = staged[c]
            cur.wait_event(ev)
            oh = torch.empty_like(qh)
            orh = torch.empty_like(qrh) if qrh is not None else None
            lg = lr = None
            if save_for_backward:
                lg = torch.empty((self.batch, qh.shape[2], self.n_gen), device=qh.device, dtype=torch.float32)
                lr = torch.empty((self.batch, qh.shape[2], self.n_ref), device=qh.device, dtype=torch.float32) if qrh is not None else None
            if self.ctx[c]:  # (an empty chunk only relays its tokens)
                B.sra_forward(self.ctx[c], qh, kh, vh, oh, q_ref=qrh, o_ref=orh, lse_gen=lg, lse_ref=lr)
                self.launches += 1
            if save_for_backward:
                self.saved[c] = (qh, kh, vh, qrh, oh, orh, lg, lr)
            done = torch.cuda.Event()
            done.record(cur)
            with torch.cuda.stream(comm):
                comm.wait_event(done)
                heads_to_seq(oh, self.n_gen, self.heads, o_gen, self.group, self.n_chunks, c)
                if orh is not None:
                    heads_to_seq(orh, self.n_ref, self.heads, o_ref, self.group, self.n_chunks, c)
            keep.append((qh, kh, vh, qrh, oh, orh))
        cur.wait_stream(comm)
        for t in keep:  # allocated on one stream, last used on the other: tell the caching allocator
            for x in t:
                if x is not None:
                    x.record_stream(cur)
                    x.record_stream(comm)
        return o_gen, o_ref

    def backward(self, do_gen: torch.Tensor, do_ref: Optional[torch.Tensor] = None):
        """Gradients of the last `forward(..., save_for_backward=True)`.  do_gen / do_ref: this rank's sequence shards of
        the upstream gradient.  Returns (dq_gen, dk_gen, dv_gen, dq_ref, dk_ref, dv_ref) as sequence shards (the last
        three None when n_ref == 0).  Reference K/V come from the resident caches, their gradients are returned like
        everything else.  Same pipeline as forward: the exchange of chunk c + 1's dO and the return of chunk c - 1's
        gradients run on the communication stream underneath `sra_backward` of chunk c."""
        if getattr(self, "saved", None) is None:
            raise RuntimeError("backward() needs forward(..., save_for_backward=True) first")
        B = self.B
        has_ref = self.n_ref > 0
        if has_ref and do_ref is None:
            raise ValueError("do_ref is required when n_ref > 0")
        cur = torch.cuda.current_stream()
        comm = self.comm
        outs_seq = [torch.empty_like(do_gen) for _ in range(3)] + ([torch.empty_like(do_ref) for _ in range(3)] if has_ref else [None] * 3)
        comm.wait_stream(cur)
        staged: List[Optional[tuple]] = [None] * self.n_chunks

        def stage(c):
            with torch.cuda.stream(comm):
                t = (self._to_heads(do_gen, self.n_gen, c), self._to_heads(do_ref, self.n_ref, c) if has_ref else None)
                ev = torch.cuda.Event()
                ev.record(comm)
            staged[c] = (t, ev)

        keep = []
        stage(0)
        for c in range(self.n_chunks):
            if c + 1 < self.n_chunks:
                stage(c + 1)
            (dog, dor), ev = staged[c]
            cur.wait_event(ev)
            qh, kh, vh, qrh, oh, orh, lg, lr = self.saved[c]
            g = [torch.empty_like(qh) for _ in range(3)] + ([torch.empty_like(qrh) for _ in range(3)] if has_ref else [None] * 3)
            if self.ctx[c]:
                B.sra_backward(self.ctx[c], q_gen=qh, k_gen=kh, v_gen=vh, q_ref=qrh, k_ref=None, v_ref=None, o_gen=oh,
                               o_ref=orh, lse_gen=lg, lse_ref=lr, do_gen=dog, do_ref=dor, dq_gen=g[0], dk_gen=g[1],
                               dv_gen=g[2], dq_ref=g[3], dk_ref=g[4], dv_ref=g[5])
                self.launches += 3
            done = torch.cuda.Event()
            done.record(cur)
            with torch.cuda.stream(comm):
                comm.wait_event(done)
                for k in range(3):
                    heads_to_seq(g[k], self.n_gen, self.heads, outs_seq[k], self.group, self.n_chunks, c)
                    if has_ref:
                        heads_to_seq(g[3 + k], self.n_ref, self.heads, outs_seq[3 + k], self.group, self.n_chunks, c)
            keep.append((dog, dor, *g))
        cur.wait_stream(comm)
        for t in keep:
            for x in t:
                if x is not None:
                    x.record_stream(cur)
                    x.record_stream(comm)
        self.saved = None
        return tuple(outs_seq)
