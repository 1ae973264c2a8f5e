#!/usr/bin/env python
"""bench.py - SRA forward throughput on B200 (BASELINE.json metric: "SRA fwd useful TFLOP/s and %
of B200 dense BF16 peak; ms per DiT attention layer").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 720p] [--impl ours|reference]

One "step" = one full SRA forward pass of one DiT attention layer on the workload (SURVEY.md 8a rows
a1 + a3 + a4 + a5): `sra_cache_reference_kv` (re-lay the reference K/V into the resident cache) +
`sra_forward` over generation AND reference query rows.  a2 (the tile schedule) is built once at
`sra_create`.  Useful FLOPs = 4 * d * pairs * H * B with pairs counted from the mask
(N_g (N_g + N_r) + sum_j b_j^2); padded / masked tile work earns nothing.

Output: ONE JSON line on stdout (rank 0).  Everything else goes to stderr.
  value      useful TFLOP/s, inputs resident in HBM, CUDA-event timed, max over ranks
  e2e        the same step through `sra_forward_host` (HOST pinned buffers in and out; H2D + D2H copies
             inside the timed region)
  roofline   the forward kernel against the measured dense-bf16 tensor peak (MEASURED_PEAKS.json)
  cpu_baseline  the fp64 oracle (oracle/, as it stands) timed on this box's host cores on a bounded sample
  parity     CUDA path vs oracle on that sample; contract tolerance max-abs <= 2e-2, mean-abs <= 2e-3
             (bf16 I/O, fp32 accumulation) plus the self-imposed relative gate rel_l2 <= 1e-2

`--impl reference` times the oracle alone (no GPU), same metric/unit/config.
Multi-GPU (torchrun, one process per GPU): every (batch item, head) is independent, so ranks own whole
batch items, no data-path collective; weak scaling (the global batch is N x the per-GPU batch).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sra_fwd_useful_tflops"
UNIT = "TFLOP/s"
MAX_ABS_TOL, MEAN_ABS_TOL, REL_L2_TOL = 2e-2, 2e-3, 1e-2
NOMINAL_BF16_TFLOPS = 2250.0
FALLBACK_PEAKS = {"bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "hbm_gbs": 6650.0}


def log(*a):
    print(*a, file=sys.stderr, flush=True)


_RESULT_FD = None


def claim_stdout():
    """The contract is ONE JSON line on stdout.  Native libraries print there too (NCCL's version banner at the first
    communicator), so the real stdout is set aside for the result line and fd 1 is pointed at stderr for everything
    else."""
    global _RESULT_FD
    if _RESULT_FD is None:
        sys.stdout.flush()
        _RESULT_FD = os.dup(1)
        os.dup2(2, 1)


def emit(out):
    line = (json.dumps(out) + "\n").encode()
    if _RESULT_FD is None:
        sys.stdout.write(line.decode())
        sys.stdout.flush()
    else:
        os.write(_RESULT_FD, line)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            d = json.load(f)
        return {"bf16_tflops": float(d["bf16_tflops"]), "bf16_tflops_sustained": float(d["bf16_tflops_sustained"]),
                "hbm_gbs": float(d["hbm_gbs"])}, "measured"
    except Exception:
        return dict(FALLBACK_PEAKS), "fallback"


def load_traffic(workload):
    """DRAM bytes per forward launch from the committed ncu --set full capture (profiles/traffic.json)."""
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f).get(workload, {}).get("sra_fwd_kernel_dram_bytes")
    except Exception:
        return None


def useful_flops(w, include_ref_rows=True, backward=False):
    pairs = w.n_gen * (w.n_gen + w.n_ref)
    if include_ref_rows:
        pairs += sum(b * b for b in w.ref_block_sizes)
    return 4.0 * w.head_dim * pairs * w.heads * w.batch * (2.5 if backward else 1.0)


# --------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------------------------- oracle legs
def oracle_sample_rows(w, n_gen_rows, n_ref_rows, seed=0):
    import numpy as np
    rng = np.random.default_rng(seed)
    g = set(int(x) for x in (0, 127, 128, w.n_gen - 1) if x < w.n_gen)
    while len(g) < min(n_gen_rows, w.n_gen):
        g.add(int(rng.integers(0, w.n_gen)))
    r = set()
    off = w.ref_block_offsets
    if w.n_ref and n_ref_rows:
        for x in (off[0], off[1] - 1, off[-2], off[-1] - 1):
            r.add(int(x))
        while len(r) < min(n_ref_rows, w.n_ref):
            r.add(int(rng.integers(0, w.n_ref)))
    rows = sorted(g)[:n_gen_rows] + [w.n_gen + x for x in sorted(r)[:n_ref_rows]]
    return np.asarray(rows, dtype=np.int32)


def sample_flops(w, rows, n_heads, valid=None, frames=None, window=-1):
    """Useful FLOPs of the sampled rows: 4 d per visible (query, key) pair under the same mask options the oracle gets."""
    import bisect
    fl = 0.0
    off = w.ref_block_offsets
    n_valid = w.n_ref if valid is None else int(sum(1 for v in valid if v))
    for r in rows:
        if r < w.n_gen:
            vis = w.n_gen
            if frames is not None and window >= 0:
                f = bisect.bisect_right(frames, int(r)) - 1
                n_fr = len(frames) - 1
                vis = frames[min(n_fr, f + window + 1)] - frames[max(0, f - window)]
            vis += n_valid
        else:
            t = r - w.n_gen
            j = max(k for k in range(len(off) - 1) if off[k] <= t)
            if valid is None:
                vis = off[j + 1] - off[j]
            else:
                vis = int(sum(1 for v in valid[off[j]:off[j + 1]] if v)) if valid[t] else 0
        fl += 4.0 * w.head_dim * vis
    return fl * n_heads * w.batch


def run_oracle_sample(w, bits_h, heads, rows, valid=None, frames=None, window=-1):
    """Times oracle/ (plain C fp64, OpenMP over rows) on `rows` x `heads`.  bits_h: uint16 arrays already
    restricted to `heads`.  valid / frames + window: the optional mask restrictions, which the
    oracle materialises in its visibility predicate.  Returns (seconds, o [B, n_rows, len(heads), d], lse)."""
    from oracle import c_oracle
    t0 = time.perf_counter()
    o, lse = c_oracle.forward_rows(bits_h["q_gen"], bits_h["k_gen"], bits_h["v_gen"], bits_h.get("q_ref"),
                                   bits_h.get("k_ref"), bits_h.get("v_ref"), w.ref_block_offsets,
                                   1.0 / math.sqrt(w.head_dim), rows, valid=valid, gen_frame_offsets=frames,
                                   window=window if frames is not None else -1)
    return time.perf_counter() - t0, o, lse


def parity_record(got, ref, got_lse=None, ref_lse=None):
    """GPU vs oracle on the same sampled outputs: the contract gates + rel_l2; empty rows (invalid reference tokens:
    O = 0, LSE = -inf on both sides) are compared as such."""
    import numpy as np
    diff = np.abs(got - ref)
    rel_l2 = float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300))
    rec = {"max_abs": float(diff.max()), "mean_abs": float(diff.mean()), "rel_l2": rel_l2,
           "tolerance": {"max_abs": MAX_ABS_TOL, "mean_abs": MEAN_ABS_TOL, "rel_l2": REL_L2_TOL}}
    ok = bool(diff.max() <= MAX_ABS_TOL and diff.mean() <= MEAN_ABS_TOL and rel_l2 <= REL_L2_TOL and np.isfinite(got).all())
    if got_lse is not None:
        empty = np.isneginf(ref_lse)
        same_empty = bool(np.array_equal(np.isneginf(got_lse), empty))
        rec["lse_max_abs"] = float(np.abs(got_lse[~empty] - ref_lse[~empty]).max()) if (~empty).any() else 0.0
        rec["empty_rows"] = int(empty.sum())
        ok = ok and same_empty and rec["lse_max_abs"] <= 2e-3
    rec["ok"] = ok
    return rec


def bench_reference(args, w):
    """--impl reference: the oracle as it stands on the host cores, each step a bounded sample."""
    import numpy as np
    from oracle import c_oracle
    from paper_2606_13872_b200 import inputs as I
    c_oracle.build()
    cores = c_oracle.num_threads()
    heads = [0]
    wh = w.replace(heads=len(heads))
    t = I.make_inputs(wh)  # the CPU recipe (heads are i.i.d.: a 1-head workload is a sample of the 40-head one)
    bits = {k: I.bf16_bits(v) for k, v in t.items()}
    # calibrate: a few rows, then size a step so the whole run stays ~<= 90 s
    probe = oracle_sample_rows(w, 8, 2)
    dt, _, _ = run_oracle_sample(wh, bits, heads, probe)
    rate = sample_flops(w, probe, 1) / dt
    budget_s = 90.0 / max(1, args.steps + args.warmup)
    per_row = 4.0 * w.head_dim * (w.n_gen + w.n_ref)
    n_rows = int(max(8, min(4096, rate * budget_s / per_row)))
    rows = oracle_sample_rows(w, n_rows, max(2, n_rows // 8))
    fl = sample_flops(w, rows, 1)
    for _ in range(args.warmup):
        run_oracle_sample(wh, bits, heads, rows)
    times = []
    for _ in range(args.steps):
        dt, _, _ = run_oracle_sample(wh, bits, heads, rows)
        times.append(dt)
    total = sum(times)
    val = fl * args.steps / total / 1e12
    sample = f"{len(rows)} query rows x 1 head of {w.name} against all visible keys, per step"
    out = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_of(w, args, extra={"sample": sample}),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    emit(out)


def config_of(w, args, extra=None):
    c = {"workload": f"{w.name}: B{w.batch} H{w.heads} d{w.head_dim}, gen {w.n_gen} tokens + ref {w.n_ref} tokens in "
                     f"{len(w.ref_block_sizes)} blocks of {w.ref_block_sizes[0] if w.ref_block_sizes else 0}",
         "step": "sra_cache_reference_kv + sra_forward (G and R query rows) = one DiT attention layer forward",
         "dist": w.dist, "global_batch": w.batch * args.gpus, "parallelism": f"dp{args.gpus} (whole batch items per rank, no collective)",
         "l2": "inputs per step (>= 3 GB at 720p) exceed the 126 MB L2; no explicit flush"}
    if extra:
        c.update(extra)
    return c


# --------------------------------------------------------------------------------------------- ours
def bench_ours(args, w):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import dp
    from paper_2606_13872_b200 import inputs as I

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SRA path has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks, peaks_kind = load_peaks()

    # weak scaling (default): this rank owns global batch items [b0, b0 + w.batch).
    # --shard heads (strong scaling of a B = 1 config; what Ulysses SP leaves each GPU with,
    # PAPER.md:231): the job is ONE item, rank r owns a contiguous slice of its heads - still no data-path collective.
    b0, _ = dp.shard_batch(w.batch, world, rank)
    seed_off = dp.unit_seed(0, b0)
    scaling = "weak"
    if args.shard == "heads":
        h0, hn = dp.shard_heads(w.heads, world, rank)
        if hn == 0:
            raise SystemExit(f"bench.py --shard heads: rank {rank} of {world} owns no head of {w.heads}")
        w = w.replace(heads=hn)
        seed_off = 7919 * h0  # (synthetic data: each head slice is drawn on its own)
        scaling = "strong"
    names = ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref") if w.n_ref else ("q_gen", "k_gen", "v_gen")
    t = {n: I.make_tensor_device(w, n, dev, seed_offset=seed_off) for n in names}
    o_gen = torch.empty_like(t["q_gen"])
    o_ref = torch.empty_like(t["q_ref"]) if w.n_ref else None
    lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev, dtype=torch.float32)
    lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev, dtype=torch.float32) if w.n_ref else None
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    fl = useful_flops(w)
    assert abs(B.sra_useful_flops(ctx, True) - fl) <= 1e-6 * fl
    valid = frames = None
    if args.window >= 0:
        # refiner-style sparse temporal attention: 21 latent frames, generation keys of frames within
        # the window only; the C oracle applies the same frame rule in its visibility predicate
        n_frames = 21 if w.n_gen % 21 == 0 else 1
        frames = [i * (w.n_gen // n_frames) for i in range(n_frames + 1)]
        B.sra_set_temporal_window(ctx, frames, args.window)
        fl = B.sra_useful_flops(ctx, True)
    if args.invalid_frac > 0 and w.n_ref:
        # sparse validity masking: a seeded per-token mask; useful FLOPs follow the valid tokens only
        valid = np.random.default_rng(w.seed).random(w.n_ref) >= args.invalid_frac
        B.sra_set_reference_validity(ctx, valid)
        fl = B.sra_useful_flops(ctx, True)

    def step():
        if w.n_ref:
            B.sra_cache_reference_kv(ctx, t["k_ref"], t["v_ref"])
        B.sra_forward(ctx, t["q_gen"], t["k_gen"], t["v_gen"], o_gen, q_ref=t.get("q_ref"), o_ref=o_ref,
                      lse_gen=lse_gen, lse_ref=lse_ref)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    launches0 = B.sra_launch_count(ctx)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    kev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    ev[0].record()
    for i in range(args.steps):
        if w.n_ref:
            B.sra_cache_reference_kv(ctx, t["k_ref"], t["v_ref"])
        kev[i][0].record()
        B.sra_forward(ctx, t["q_gen"], t["k_gen"], t["v_gen"], o_gen, q_ref=t.get("q_ref"), o_ref=o_ref,
                      lse_gen=lse_gen, lse_ref=lse_ref)
        kev[i][1].record()
        ev[i + 1].record()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    launches = B.sra_launch_count(ctx) - launches0
    elapsed_ms = ev[0].elapsed_time(ev[-1])
    kernel_ms = [a.elapsed_time(b) for a, b in kev]
    elapsed_ms = dp.max_over_ranks(elapsed_ms, dev)
    total_fl = dp.sum_over_ranks(fl * args.steps, dev)
    value = total_fl / (elapsed_ms * 1e-3) / 1e12

    # ---- e2e: HOST pinned buffers through sra_forward_host (H2D of q/k/v(+q_ref), D2H of o(+o_ref) timed)
    e2e = None
    e2e_out = None
    try:
        host = {n: torch.empty(t[n].shape, dtype=torch.bfloat16).pin_memory() for n in ("q_gen", "k_gen", "v_gen")}
        for n in host:
            host[n].copy_(t[n])
        h_o_gen = torch.empty(o_gen.shape, dtype=torch.bfloat16).pin_memory()
        h_q_ref = h_o_ref = None
        if w.n_ref:
            h_q_ref = torch.empty(t["q_ref"].shape, dtype=torch.bfloat16).pin_memory()
            h_q_ref.copy_(t["q_ref"])
            h_o_ref = torch.empty(o_ref.shape, dtype=torch.bfloat16).pin_memory()
        h2d = sum(x.numel() * 2 for x in host.values()) + (h_q_ref.numel() * 2 if h_q_ref is not None else 0)
        d2h = h_o_gen.numel() * 2 + (h_o_ref.numel() * 2 if h_o_ref is not None else 0)

        def e2e_step():
            if w.n_ref:
                B.sra_cache_reference_kv(ctx, t["k_ref"], t["v_ref"])  # the reference K/V are resident by design
            B.sra_forward_host(ctx, host["q_gen"], host["k_gen"], host["v_gen"], h_o_gen, q_ref=h_q_ref, o_ref=h_o_ref)

        n_e2e = max(1, min(args.steps, 5))
        e2e_step()
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n_e2e):
            e2e_step()
        e1.record()
        barrier()
        e2e_ms = dp.max_over_ranks(e0.elapsed_time(e1), dev)
        e2e_val = dp.sum_over_ranks(fl * n_e2e, dev) / (e2e_ms * 1e-3) / 1e12
        # the pipelined host path merges two fp32 partials for its reference-first slabs, so those rows may differ
        # from the single-pass device path in the last bf16 bit; both are checked against the oracle below
        o_dev = o_gen.cpu()
        same = bool(torch.equal(h_o_gen, o_dev))
        max_diff = float((h_o_gen.float() - o_dev.float()).abs().max())
        ulp_top = float(o_dev.float().abs().max()) * 2.0 ** -7
        del o_dev
        e2e = {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": e2e_ms / n_e2e, "steps": n_e2e, "api": "sra_forward_host (C ABI, host pointers)",
               "matches_device_path": bool(max_diff <= ulp_top), "bit_identical_to_device_path": same,
               "max_abs_diff_vs_device_path": max_diff}
        e2e_out = (h_o_gen, h_o_ref)
        del host, h_q_ref
    except Exception as ex:  # pinned allocation can fail on a small box: report, do not hide
        log(f"e2e leg failed: {ex!r}")
        e2e = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0, "error": repr(ex)}

    # ---- oracle legs (rank 0, N == 1): parity on a sample + cpu_baseline
    cpu_baseline = parity = None
    if rank == 0 and world == 1 and not args.no_oracle:
        from oracle import c_oracle
        c_oracle.build()
        heads = sorted(set(int(round(x)) for x in np.linspace(0, w.heads - 1, min(4, w.heads))))
        rows = oracle_sample_rows(w, args.oracle_rows, max(2, args.oracle_rows // 4))
        bits_h = {n: I.bf16_bits(t[n][:, :, heads].contiguous().cpu()) for n in names}
        wh = w.replace(heads=len(heads))
        dt, o_or, lse_or = run_oracle_sample(wh, bits_h, heads, rows, valid, frames, args.window)
        sfl = sample_flops(w, rows, len(heads), valid, frames, args.window)
        sample = (f"{len(rows)} query rows ({int((rows < w.n_gen).sum())} G + {int((rows >= w.n_gen).sum())} R) x heads {heads} "
                  f"of the same {w.name} inputs, all visible keys; {sfl / 1e9:.1f} GFLOP fp64 in {dt:.1f} s")
        cpu_baseline = {"value": sfl / dt / 1e12, "unit": UNIT, "cores": c_oracle.num_threads(), "kind": "oracle",
                        "sample": sample, "seconds": dt,
                        "extrapolated_s_per_layer": dt * fl / sfl}
        g_rows = rows[rows < w.n_gen]
        r_rows = rows[rows >= w.n_gen] - w.n_gen
        got = [o_gen[:, torch.as_tensor(g_rows, device=dev).long()][:, :, heads].float().cpu().numpy()]
        got_lse = [lse_gen[:, heads][:, :, torch.as_tensor(g_rows, device=dev).long()].cpu().numpy()]
        if len(r_rows):
            got.append(o_ref[:, torch.as_tensor(r_rows, device=dev).long()][:, :, heads].float().cpu().numpy())
            got_lse.append(lse_ref[:, heads][:, :, torch.as_tensor(r_rows, device=dev).long()].cpu().numpy())
        got = np.concatenate(got, axis=1).astype(np.float64)
        got_lse = np.concatenate(got_lse, axis=2).astype(np.float64)
        parity = parity_record(got, o_or, got_lse, lse_or)
        parity.update(rows=int(len(rows)), heads=heads)
        if e2e_out is not None and e2e is not None and e2e.get("value") is not None:
            # the same sampled rows of what sra_forward_host returned, against the same oracle values
            hg = [e2e_out[0][:, torch.as_tensor(g_rows).long()][:, :, heads].float().numpy()]
            if len(r_rows) and e2e_out[1] is not None:
                hg.append(e2e_out[1][:, torch.as_tensor(r_rows).long()][:, :, heads].float().numpy())
            hg = np.concatenate(hg, axis=1).astype(np.float64)
            e2e["parity"] = parity_record(hg, o_or)
    e2e_out = None

    B.sra_destroy(ctx)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- legs (N == 1, the default 720p line only): the rest of SURVEY.md 8 on the same line, same run
    legs = None
    if world == 1 and args.legs and w.name == "720p" and args.window < 0 and args.invalid_frac == 0:
        del t, o_gen, o_ref, lse_gen, lse_ref
        torch.cuda.empty_cache()
        legs = {}
        for name, fn in (("denoise8", lambda: leg_denoise8(args, w, dev, peaks, peaks_kind)),
                         ("train", lambda: leg_train(args)), ("short128", lambda: leg_short(args))):
            try:
                legs[name] = fn()
            except Exception as ex:  # a failed leg is reported, never hidden
                log(f"leg {name} failed: {ex!r}")
                legs[name] = {"error": repr(ex)}
            torch.cuda.empty_cache()
    k_ms = statistics.mean(kernel_ms)
    achieved = fl / (k_ms * 1e-3) / 1e12
    peak = peaks["bf16_tflops_sustained"]
    roofline = {
        "bound": "tensor", "kernel": "sra_fwd_kernel<128>" if w.head_dim == 128 else "sra_fwd_kernel<64>",
        "achieved": achieved, "peak": peak, "unit": UNIT, "frac": achieved / peak,
        "peak_kind": f"{peaks_kind} cuBLAS bf16, sustained (kernel timed back to back inside a seconds-long step loop)",
        "frac_of_burst": achieved / peaks["bf16_tflops"], "peak_burst": peaks["bf16_tflops"],
        "frac_of_nominal": achieved / NOMINAL_BF16_TFLOPS, "peak_nominal": NOMINAL_BF16_TFLOPS,
        "kernel_ms": k_ms, "kernel_ms_min": min(kernel_ms), "algorithmic_flops_per_launch": fl,
        "traffic": load_traffic(w.name),
    }
    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": scaling, "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": config_of(w, args, {**({"parallelism": f"heads{world} (one item, {w.heads} heads per rank, no collective)",
                                          "global_batch": w.batch} if scaling == "strong" else {}),
                                      **({"invalid_ref_frac": args.invalid_frac} if args.invalid_frac > 0 else {}),
                                      **({"temporal_window_frames": args.window} if args.window >= 0 else {})} or None),
        "pct_of_peak": {"measured_sustained": 100 * value / world / peaks["bf16_tflops_sustained"],
                        "measured_burst": 100 * value / world / peaks["bf16_tflops"],
                        "nominal_2250": 100 * value / world / NOMINAL_BF16_TFLOPS},
        "ms_per_layer": elapsed_ms / args.steps,
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
        "cpu_baseline": cpu_baseline, "parity": parity,
    }
    if legs is not None:
        out["legs"] = legs
    emit(out)
    if world > 1:
        dist.destroy_process_group()


def leg_denoise8(args, w, dev, peaks, peaks_kind):
    """BASELINE.json configs[2] as written ("reuse cached ref KV over 8 denoising steps") with the
    protocol of SURVEY.md 8d: step 0 = sra_cache_reference_kv + sra_forward over G and R rows; steps 1-7 = cached
    steps (q_ref = k_ref = v_ref = NULL: G rows only, reference K/V from the resident cache), FRESH generation
    tensors every step (seed + 1000 * step).  Every step is bracketed by CUDA events on the launching stream."""
    import numpy as np
    import torch
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import inputs as I
    n_steps = 8
    ref = {n: I.make_tensor_device(w, n, dev) for n in ("q_ref", "k_ref", "v_ref")}
    gens = [{n: I.make_tensor_device(w, n, dev, step=s) for n in ("q_gen", "k_gen", "v_gen")} for s in range(n_steps)]
    o_gen = torch.empty_like(gens[0]["q_gen"])
    o_ref = torch.empty_like(ref["q_ref"])
    lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev, dtype=torch.float32)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    fl0, flc = B.sra_useful_flops(ctx, True), B.sra_useful_flops(ctx, False)

    def run(s):
        g = gens[s]
        if s == 0:
            B.sra_cache_reference_kv(ctx, ref["k_ref"], ref["v_ref"])
            B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, q_ref=ref["q_ref"], o_ref=o_ref, lse_gen=lse_gen)
        else:
            B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, lse_gen=lse_gen)

    for s in (0, 1, 2):  # warm-up: a full step and two cached steps
        run(s)
    torch.cuda.synchronize()
    cache_bytes = B.sra_cache_bytes(ctx)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(n_steps + 1)]
    launches = []
    ev[0].record()
    for s in range(n_steps):
        l0 = B.sra_launch_count(ctx)
        run(s)
        ev[s + 1].record()
        launches.append(B.sra_launch_count(ctx) - l0)
    torch.cuda.synchronize()
    ms = [ev[s].elapsed_time(ev[s + 1]) for s in range(n_steps)]
    # parity of the LAST cached step (fresh tensors of step 7, resident cache) on sampled generation rows
    from oracle import c_oracle
    c_oracle.build()
    heads = [0, w.heads - 1]
    rows = oracle_sample_rows(w, 96, 0)
    g = gens[n_steps - 1]
    bits_h = {n: I.bf16_bits(x[:, :, heads].contiguous().cpu()) for n, x in {**g, **ref}.items()}
    _, o_or, lse_or = run_oracle_sample(w.replace(heads=len(heads)), bits_h, heads, rows)
    idx = torch.as_tensor(rows, device=dev).long()
    got = o_gen[:, idx][:, :, heads].float().cpu().numpy().astype(np.float64)
    got_lse = lse_gen[:, heads][:, :, idx].cpu().numpy().astype(np.float64)
    parity = parity_record(got, o_or, got_lse, lse_or)
    parity.update(rows=int(len(rows)), heads=heads, step=n_steps - 1)
    same_cache = B.sra_cache_bytes(ctx) == cache_bytes
    B.sra_destroy(ctx)
    cached = ms[1:]
    peak = peaks["bf16_tflops_sustained"]
    return {
        "workload": w.name, "protocol": "step 0 = cache build + G and R rows; steps 1-7 = cached (q_ref NULL), fresh G tensors per step",
        "step0_ms": ms[0], "cached_step_ms": cached, "cached_step_ms_mean": statistics.mean(cached),
        "mean_ms_over_8_steps": statistics.mean(ms), "launches_per_step": launches,
        "cache_bytes": int(cache_bytes), "cache_unchanged_over_cached_steps": bool(same_cache),
        "step0_useful_tflops": fl0 / (ms[0] * 1e-3) / 1e12,
        "cached_step_useful_tflops": flc / (statistics.mean(cached) * 1e-3) / 1e12,
        "cached_step_frac_of_sustained_peak": flc / (statistics.mean(cached) * 1e-3) / 1e12 / peak,
        "useful_tflops_over_8_steps": (fl0 + 7 * flc) / (sum(ms) * 1e-3) / 1e12,
        "peak": peak, "peak_kind": f"{peaks_kind} cuBLAS bf16, sustained", "parity": parity,
    }


def leg_train(args):
    """BASELINE.json configs[4] (rows a6-a8): the --mode train measurement, shortened, with its oracle check."""
    from paper_2606_13872_b200 import inputs as I
    a = argparse.Namespace(**{**vars(args), "steps": 4, "warmup": 3, "train_parity": not args.no_oracle})
    out = bench_train(a, I.WORKLOADS["train"], emit_line=False)
    keep = ("metric", "value", "unit", "ms_per_step", "steps", "warmup", "gpu_launches", "clocks", "roofline", "parity")
    leg = {k: out[k] for k in keep}
    leg["workload"] = out["config"]["workload"]
    return leg


def leg_short(args):
    """north_star's cache-bound short-query case (128 rows against the 40 s cache): the --mode short measurement."""
    from paper_2606_13872_b200 import inputs as I
    a = argparse.Namespace(**{**vars(args), "steps": 20, "warmup": 3})
    out = bench_short(a, I.WORKLOADS["short128"], emit_line=False)
    keep = ("metric", "value", "unit", "ms_per_step", "steps", "useful_tflops", "gpu_launches", "roofline", "cuda_graph", "parity")
    leg = {k: out[k] for k in keep}
    leg["workload"] = out["config"]["workload"]
    return leg


def bench_train(args, w, emit_line=True):
    """--mode train (BASELINE.json configs[4]): one step = sra_forward (fresh reference K/V, LSE written) +
    sra_backward (a6 + a7 + a8) on the workload; value = useful fwd+bwd TFLOP/s (3.5 x forward FLOPs)."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import dp
    from paper_2606_13872_b200 import inputs as I

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SRA path has no CPU fallback")
    if w.n_ref == 0:
        raise SystemExit("bench.py --mode train: needs a reference (configs[4] shape)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks, peaks_kind = load_peaks()
    b0, _ = dp.shard_batch(w.batch, world, rank)
    seed_off = dp.unit_seed(0, b0)
    t = {n: I.make_tensor_device(w, n, dev, seed_offset=seed_off) for n in I.TENSOR_ORDER}
    o_gen, o_ref = torch.empty_like(t["q_gen"]), torch.empty_like(t["q_ref"])
    lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev, dtype=torch.float32)
    lse_ref = torch.empty((w.batch, w.heads, w.n_ref), device=dev, dtype=torch.float32)
    grads = {n: torch.empty_like(t["q_gen" if n.endswith("_gen") else "q_ref"])
             for n in ("dq_gen", "dk_gen", "dv_gen", "dq_ref", "dk_ref", "dv_ref")}
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    B.sra_set_kernel_timing(ctx, True)
    fl_f, fl_b = useful_flops(w), useful_flops(w, backward=True)
    assert abs(B.sra_useful_flops(ctx, True, True) - fl_b) <= 1e-6 * fl_b

    def fwd():
        B.sra_forward(ctx, t["q_gen"], t["k_gen"], t["v_gen"], o_gen, q_ref=t["q_ref"], k_ref=t["k_ref"],
                      v_ref=t["v_ref"], o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref)

    def bwd():
        B.sra_backward(ctx, q_gen=t["q_gen"], k_gen=t["k_gen"], v_gen=t["v_gen"], q_ref=t["q_ref"], k_ref=t["k_ref"],
                       v_ref=t["v_ref"], o_gen=o_gen, o_ref=o_ref, lse_gen=lse_gen, lse_ref=lse_ref,
                       do_gen=t["do_gen"], do_ref=t["do_ref"], **grads)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        fwd(); bwd()
    barrier()
    launches0 = B.sra_launch_count(ctx)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k_ms = {k: [] for k in ("fwd", "bwd_pre", "bwd_main", "bwd_fin")}
    barrier()
    e0.record()
    for _ in range(args.steps):
        fwd(); bwd()
    e1.record()
    barrier()
    # per-kernel device times of the LAST timed step (the library brackets each launch with CUDA events on the
    # launching stream; reading them earlier would synchronise inside the timed loop)
    for k, which in (("fwd", B.KERNEL_FWD), ("bwd_pre", B.KERNEL_BWD_PREPROCESS), ("bwd_main", B.KERNEL_BWD_MAIN),
                     ("bwd_fin", B.KERNEL_BWD_DQ_FINALIZE)):
        k_ms[k].append(B.sra_kernel_time_ms(ctx, which))
    clocks = sampler.stop() if rank == 0 else None
    launches = B.sra_launch_count(ctx) - launches0
    elapsed_ms = dp.max_over_ranks(e0.elapsed_time(e1), dev)
    total_fl = dp.sum_over_ranks((fl_f + fl_b) * args.steps, dev)
    value = total_fl / (elapsed_ms * 1e-3) / 1e12

    parity = None
    if rank == 0 and world == 1 and args.train_parity:
        parity = train_parity(w, t, grads, dev)
    B.sra_destroy(ctx)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    km = {k: statistics.mean(v) for k, v in k_ms.items()}
    achieved = fl_b / (km["bwd_main"] * 1e-3) / 1e12
    peak = peaks["bf16_tflops_sustained"]
    roofline = {
        "bound": "tensor", "kernel": "sra_bwd_kernel<128>", "achieved": achieved, "peak": peak, "unit": UNIT,
        "frac": achieved / peak,
        "peak_kind": f"{peaks_kind} cuBLAS bf16, sustained (kernel timed inside a seconds-long step loop)",
        "frac_of_burst": achieved / peaks["bf16_tflops"], "peak_burst": peaks["bf16_tflops"],
        "frac_of_nominal": achieved / NOMINAL_BF16_TFLOPS, "peak_nominal": NOMINAL_BF16_TFLOPS,
        "kernel_ms": km["bwd_main"], "algorithmic_flops_per_launch": fl_b,
        "traffic": (load_traffic_all().get(w.name, {}) or {}).get("sra_bwd_kernel_dram_bytes"),
        "kernel_ms_all": km,
        "fwd_kernel": {"achieved": fl_f / (km["fwd"] * 1e-3) / 1e12, "frac": fl_f / (km["fwd"] * 1e-3) / 1e12 / peak,
                       "kernel_ms": km["fwd"], "algorithmic_flops_per_launch": fl_f},
    }
    cfg = config_of(w, args)
    cfg["step"] = "sra_forward (fresh reference K/V, LSE) + sra_backward (preprocess + main + dQ finalise): one DiT attention layer fwd+bwd"
    out = {
        "metric": "sra_train_useful_tflops", "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "bf16", "data": "synthetic", "config": cfg,
        "pct_of_peak": {"measured_sustained": 100 * value / world / peaks["bf16_tflops_sustained"],
                        "measured_burst": 100 * value / world / peaks["bf16_tflops"],
                        "nominal_2250": 100 * value / world / NOMINAL_BF16_TFLOPS},
        "e2e": None, "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline, "cpu_baseline": None,
        "parity": parity,
    }
    if emit_line:
        emit(out)
    if world > 1:
        dist.destroy_process_group()
    return out


def train_parity(w, t, grads, dev, b=0, h=0, n_rows=48, n_cols=48):
    """Backward parity at full size (slow: the oracle needs the forward of EVERY row of one (b, h) - ~1 TFLOP of
    fp64 - before it can give dK/dV of sampled keys): sampled query rows for dQ, sampled key columns for dK/dV."""
    import numpy as np
    from oracle import c_oracle
    from paper_2606_13872_b200 import inputs as I
    c_oracle.build()
    t0 = time.perf_counter()
    bits = {n: I.bf16_bits(t[n][b:b + 1, :, h:h + 1].contiguous().cpu()) for n in I.TENSOR_ORDER}
    args6 = [bits[k] for k in ("q_gen", "k_gen", "v_gen", "q_ref", "k_ref", "v_ref")]
    scale = 1.0 / math.sqrt(w.head_dim)
    o, lse = c_oracle.forward_head(*args6, w.ref_block_offsets, scale, 0, 0)
    rng = np.random.default_rng(1)
    n = w.n_gen + w.n_ref
    off = w.ref_block_offsets
    edge = [0, 63, 64, 127, 128, w.n_gen - 1, w.n_gen, w.n_gen + off[1] - 1, w.n_gen + off[1], n - 1]
    rows = np.asarray(sorted(set(edge) | set(int(x) for x in rng.integers(0, n, n_rows))), dtype=np.int32)
    cols = np.asarray(sorted(set(edge) | set(int(x) for x in rng.integers(0, n, n_cols))), dtype=np.int32)
    dq, dk, dv = c_oracle.backward_head(*args6, bits["do_gen"], bits["do_ref"], off, scale, 0, 0, o, lse, rows=rows,
                                        cols=cols)
    res = {"b": b, "h": h, "rows": int(len(rows)), "cols": int(len(cols)), "oracle_seconds": time.perf_counter() - t0,
           "tolerance": {"max_abs": MAX_ABS_TOL, "mean_abs": MEAN_ABS_TOL, "rel_l2": REL_L2_TOL}}
    ok = True
    for name, ref, idx in (("dq", dq, rows), ("dk", dk, cols), ("dv", dv, cols)):
        gi = idx[idx < w.n_gen]
        ri = idx[idx >= w.n_gen] - w.n_gen
        got = np.concatenate([grads[name + "_gen"][b, :, h][torch_index(gi, dev)].float().cpu().numpy(),
                              grads[name + "_ref"][b, :, h][torch_index(ri, dev)].float().cpu().numpy()], axis=0)
        diff = np.abs(got - ref)
        rel = float(np.linalg.norm(got - ref) / max(np.linalg.norm(ref), 1e-300))
        res[name] = {"max_abs": float(diff.max()), "mean_abs": float(diff.mean()), "rel_l2": rel}
        ok = ok and bool(np.isfinite(got).all() and diff.max() <= MAX_ABS_TOL and diff.mean() <= MEAN_ABS_TOL
                         and rel <= REL_L2_TOL)
    res["ok"] = ok
    return res


def torch_index(idx, dev):
    import torch
    return torch.as_tensor(idx, device=dev).long()


def load_traffic_all():
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            return json.load(f)
    except Exception:
        return {}


def bench_short(args, w, emit_line=True):
    """--mode short (north_star "cache-bound short-query cases", SURVEY.md 8d auxiliary sweep): cached denoising
    steps of a few generation rows against the resident reference cache.  Arithmetic intensity ~ N_g FLOP/B is
    below the ridge (~250 FLOP/B) for N_g <= 256, so the step is judged on HBM GB/s: algorithmic bytes = the
    resident K/V cache + the step's q/k/v in + o out (+ LSE), over the device time of sra_fwd_kernel + the merge of
    the key-split partials.  Four rotating sets of generation tensors; the cache alone (>= 0.4 GB) exceeds L2."""
    import torch
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import inputs as I
    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("bench.py --mode short is a single-GPU diagnostic")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SRA path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peaks, peaks_kind = load_peaks()
    ref = {n: I.make_tensor_device(w, n, dev) for n in ("k_ref", "v_ref")}
    sets = [{n: I.make_tensor_device(w, n, dev, step=s) for n in ("q_gen", "k_gen", "v_gen")} for s in range(4)]
    o_gen = torch.empty_like(sets[0]["q_gen"])
    lse_gen = torch.empty((w.batch, w.heads, w.n_gen), device=dev, dtype=torch.float32)
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    B.sra_set_kernel_timing(ctx, True)
    B.sra_cache_reference_kv(ctx, ref["k_ref"], ref["v_ref"])
    n_split, _ = B.sra_split_schedule_copy(ctx)
    fl = useful_flops(w, include_ref_rows=False)
    row = w.heads * w.head_dim * 2
    alg_bytes = B.sra_cache_bytes(ctx) + 4 * w.batch * w.n_gen * row + w.batch * w.heads * w.n_gen * 4

    def step(i):
        g = sets[i % 4]
        B.sra_forward(ctx, g["q_gen"], g["k_gen"], g["v_gen"], o_gen, lse_gen=lse_gen)

    for i in range(max(args.warmup, 3)):
        step(i)
    torch.cuda.synchronize()
    launches0 = B.sra_launch_count(ctx)
    sampler = ClockSampler(0)
    sampler.start()
    k_ms = []
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for i in range(args.steps):
        step(i)
    e1.record()
    torch.cuda.synchronize()
    elapsed_ms = e0.elapsed_time(e1)
    for i in range(min(args.steps, 8)):  # per-kernel device times, one step at a time (reading them synchronises)
        step(i)
        ms = B.sra_kernel_time_ms(ctx, B.KERNEL_FWD)
        if n_split > 1:
            ms += B.sra_kernel_time_ms(ctx, B.KERNEL_FWD_MERGE)
        k_ms.append(ms)
    clocks = sampler.stop()
    launches = B.sra_launch_count(ctx) - launches0
    # the same loop replayed from ONE CUDA graph (a steady-state call neither allocates nor synchronises, so it can be
    # captured): what the launch overhead of two sub-millisecond kernels per step is worth
    graph_rec = None
    try:
        B.sra_set_kernel_timing(ctx, False)
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            for i in range(args.steps):
                step(i)
        graph.replay()
        torch.cuda.synchronize()
        g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        g0.record()
        graph.replay()
        g1.record()
        torch.cuda.synchronize()
        g_ms = g0.elapsed_time(g1) / args.steps
        graph_rec = {"ms_per_step": g_ms, "steps_per_graph": args.steps, "eager_ms_per_step": elapsed_ms / args.steps,
                     "gbs": alg_bytes / (g_ms * 1e-3) / 1e9, "frac_of_copy_peak": alg_bytes / (g_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]}
        del graph
    except Exception as ex:
        log(f"graph replay leg failed: {ex!r}")
        graph_rec = {"error": repr(ex)}
    parity = None
    if not args.no_oracle:
        # the last step's output (set (steps - 1) % 4 ... the per-kernel loop above ran sets 0 .. min(steps, 8) - 1)
        import numpy as np
        from oracle import c_oracle
        c_oracle.build()
        last = (min(args.steps, 8) - 1) % 4
        step(last)
        torch.cuda.synchronize()
        heads = [0, w.heads - 1]
        rows = oracle_sample_rows(w, 48, 0)
        gs = sets[last]
        bits_h = {n: I.bf16_bits(x[:, :, heads].contiguous().cpu()) for n, x in {**gs, **ref}.items()}
        bits_h["q_ref"] = None
        _, o_or, lse_or = run_oracle_sample(w.replace(heads=len(heads)), bits_h, heads, rows)
        idx = torch.as_tensor(rows, device=dev).long()
        parity = parity_record(o_gen[:, idx][:, :, heads].float().cpu().numpy().astype(np.float64), o_or,
                               lse_gen[:, heads][:, :, idx].cpu().numpy().astype(np.float64), lse_or)
        parity.update(rows=int(len(rows)), heads=heads)
    B.sra_destroy(ctx)
    kernel_ms = statistics.median(k_ms)
    achieved = alg_bytes / (kernel_ms * 1e-3) / 1e9
    # which roofline: arithmetic intensity of the step against the ridge of the two measured peaks
    intensity = fl / alg_bytes
    ridge = peaks["bf16_tflops_sustained"] * 1e12 / (peaks["hbm_gbs"] * 1e9)
    tensor_bound = intensity > ridge
    achieved_tf = fl / (kernel_ms * 1e-3) / 1e12
    cfg = config_of(w, args)
    cfg["step"] = "sra_forward, cached denoising step (q_ref = k_ref = v_ref = NULL): G rows against gen K/V + resident reference cache"
    cfg["n_split"] = n_split
    out = {
        "metric": "sra_short_query_cache_gbs", "value": alg_bytes * args.steps / (elapsed_ms * 1e-3) / 1e9, "unit": "GB/s",
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": elapsed_ms / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "bf16", "data": "synthetic",
        "config": cfg, "useful_tflops": fl * args.steps / (elapsed_ms * 1e-3) / 1e12, "e2e": None, "cuda_graph": graph_rec,
        "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "tensor" if tensor_bound else "hbm",
                     "kernel": "sra_fwd_kernel<128>" + (" + sra_fwd_merge_kernel<128>" if n_split > 1 else ""),
                     "achieved": achieved_tf if tensor_bound else achieved,
                     "peak": peaks["bf16_tflops_sustained"] if tensor_bound else peaks["hbm_gbs"],
                     "unit": UNIT if tensor_bound else "GB/s",
                     "frac": achieved_tf / peaks["bf16_tflops_sustained"] if tensor_bound else achieved / peaks["hbm_gbs"],
                     "peak_kind": f"{peaks_kind} cuBLAS bf16, sustained" if tensor_bound else f"{peaks_kind} copy bandwidth",
                     "intensity_flop_per_byte": intensity, "ridge_flop_per_byte": ridge,
                     "hbm_gbs": achieved, "hbm_frac": achieved / peaks["hbm_gbs"], "kernel_ms": kernel_ms,
                     "algorithmic_bytes_per_launch": alg_bytes, "algorithmic_flops_per_launch": fl,
                     "traffic": (lambda t: (t.get("sra_fwd_kernel_dram_bytes", 0) + t.get("sra_fwd_merge_kernel_dram_bytes", 0)) or None)(
                         load_traffic_all().get(w.name, {}) or {})},
        "cpu_baseline": None, "parity": parity,
    }
    if emit_line:
        emit(out)
    return out


def bench_rope(args, w):
    """--mode rope: the producer side of the reference-KV cache.  Pure data movement
    with 6 FLOP per pair, so it is judged on HBM GB/s.  Times, per launch with the library's own CUDA events,
      fused   : sra_cache_reference_kv_rope - rotate K_r inside the head-major cache write
                (algorithmic bytes = read K_r, V_r + write both caches + the fp32 table once),
      unfused : sra_apply_rope on K_r in place, then sra_cache_reference_kv (one more read + write of K_r),
      step    : sra_apply_rope on the fresh Q_g, K_g of a denoising step (read + write of both + the table).
    The headline value is the fused producer; the tensors (>= 0.8 GB) exceed L2, so nothing is flushed."""
    import torch
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import inputs as I
    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("bench.py --mode rope is a single-GPU diagnostic")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SRA path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peaks, peaks_kind = load_peaks()
    t = {n: I.make_tensor_device(w, n, dev) for n in ("k_ref", "v_ref", "q_gen", "k_gen")}
    cr, sr = (x.to(dev) for x in I.rope_tables(w, "ref"))
    cg, sg = (x.to(dev) for x in I.rope_tables(w, "gen"))
    ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
    B.sra_set_kernel_timing(ctx, True)
    row = w.heads * w.head_dim * 2
    kv_bytes = w.batch * w.n_ref * row
    g_bytes = w.batch * w.n_gen * row
    tab_ref, tab_gen = w.n_ref * w.head_dim * 4, w.n_gen * w.head_dim * 4   # cos + sin, [n, d/2] fp32 each
    alg = {"fused": 4 * kv_bytes + tab_ref, "unfused": 6 * kv_bytes + tab_ref, "step": 4 * g_bytes + tab_gen}
    ms = {"fused": [], "unfused": [], "step": []}
    n_warm = max(args.warmup, 3)
    launches0 = 0
    sampler = ClockSampler(0)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for i in range(n_warm + args.steps):
        if i == n_warm:
            torch.cuda.synchronize()
            launches0 = B.sra_launch_count(ctx)
            sampler.start()
            e0.record()
        B.sra_cache_reference_kv_rope(ctx, t["k_ref"], t["v_ref"], cr, sr)
        a = B.sra_kernel_time_ms(ctx, B.KERNEL_CACHE_RELAYOUT)
        B.sra_apply_rope(ctx, t["k_ref"], None, cr, sr, w.n_ref)     # (values keep rotating; the timing does not care)
        b = B.sra_kernel_time_ms(ctx, B.KERNEL_ROPE)
        B.sra_cache_reference_kv(ctx, t["k_ref"], t["v_ref"])
        b += B.sra_kernel_time_ms(ctx, B.KERNEL_CACHE_RELAYOUT)
        B.sra_apply_rope(ctx, t["q_gen"], t["k_gen"], cg, sg, w.n_gen)
        c = B.sra_kernel_time_ms(ctx, B.KERNEL_ROPE)
        if i >= n_warm:
            ms["fused"].append(a); ms["unfused"].append(b); ms["step"].append(c)
    e1.record()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    launches = B.sra_launch_count(ctx) - launches0
    B.sra_destroy(ctx)
    med = {k: statistics.median(v) for k, v in ms.items()}
    gbs = {k: alg[k] / (med[k] * 1e-3) / 1e9 for k in med}
    cfg = config_of(w, args)
    cfg["step"] = "sra_cache_reference_kv_rope (fused RoPE + head-major cache write); also the unfused route and the per-step Q_g/K_g rotation"
    cfg["l2"] = "tensors larger than L2, no flush"
    out = {
        "metric": "sra_rope_cache_producer_gbs", "value": gbs["fused"], "unit": "GB/s", "n_gpus": 1, "steps": args.steps,
        "warmup": n_warm, "ms_per_step": med["fused"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic", "config": cfg, "e2e": None, "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": "relayout_rope_head_major_kernel", "achieved": gbs["fused"],
                     "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": gbs["fused"] / peaks["hbm_gbs"],
                     "peak_kind": f"{peaks_kind} copy bandwidth", "kernel_ms": med["fused"],
                     "algorithmic_bytes_per_launch": alg["fused"],
                     "traffic": (load_traffic_all().get(w.name, {}) or {}).get("relayout_rope_head_major_kernel_dram_bytes")},
        "rope": {k: {"ms": med[k], "algorithmic_bytes": alg[k], "gbs": gbs[k]} for k in med},
        "fused_over_unfused_time": med["fused"] / med["unfused"],
        "cpu_baseline": None, "parity": None,
    }
    emit(out)


def bench_ulysses(args, w):
    """--mode ulysses: one cached denoising step of a SEQUENCE-SHARDED layer -
    all-to-all to head shards, sra_forward per head chunk, all-to-all back, pipelined on a communication stream
    (paper_2606_13872_b200/ulysses.py).  Strong scaling over heads: total work is fixed, rank r owns H / N heads.
    With N = 1 (all this run can measure) the exchange is a self-exchange through NCCL plus the pack / unpack copies;
    the line also reports the un-pipelined pieces (`direct_ms` = sra_forward alone on this rank's heads,
    `exchange_ms` = the exchanges alone) so that the overlap is visible: pipelined ~ direct, not direct + exchange."""
    import torch
    import torch.distributed as dist
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import dp, ulysses
    from paper_2606_13872_b200 import inputs as I
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SRA path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    else:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29577")
        dist.init_process_group("nccl", rank=0, world_size=1, device_id=dev)
    n_chunks = args.chunks
    u = ulysses.UlyssesSRA(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets, n_chunks=n_chunks)
    g0, gn = u.gen_shard()
    r0, rn = u.ref_shard()
    # every rank draws the whole tensor with the same seed and keeps its token shard (synthetic; no file, no exchange)
    def shard(name, t0, n):
        return I.make_tensor_device(w, name, dev)[:, t0:t0 + n].contiguous()
    kr, vr = shard("k_ref", r0, rn), shard("v_ref", r0, rn)
    u.cache_reference_kv(kr, vr)
    del kr, vr
    q, k, v = shard("q_gen", g0, gn), shard("k_gen", g0, gn), shard("v_gen", g0, gn)
    torch.cuda.empty_cache()
    fl = useful_flops(w, include_ref_rows=False)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    def timed(fn, n):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(n):
            fn()
        e1.record()
        barrier()
        return dp.max_over_ranks(e0.elapsed_time(e1), dev) / n

    for _ in range(max(args.warmup, 3)):
        u.forward(q, k, v)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    launches0 = u.launches
    ms = timed(lambda: u.forward(q, k, v), args.steps)
    launches = u.launches - launches0
    clocks = sampler.stop() if rank == 0 else None

    # the pieces, un-pipelined, for comparison: the forwards alone first (same thermal / power state as the loop
    # above), then the exchanges alone
    staged = [(u._to_heads(q, w.n_gen, c), u._to_heads(k, w.n_gen, c), u._to_heads(v, w.n_gen, c)) for c in range(u.n_chunks)]
    outs = [torch.empty_like(t[0]) for t in staged]

    def direct():
        for c in range(u.n_chunks):
            if u.ctx[c]:
                B.sra_forward(u.ctx[c], staged[c][0], staged[c][1], staged[c][2], outs[c])
    direct()
    direct_ms = timed(direct, args.steps)

    def exchange_only():
        o = torch.empty_like(q)
        for c in range(u.n_chunks):
            qh = u._to_heads(q, w.n_gen, c); u._to_heads(k, w.n_gen, c); u._to_heads(v, w.n_gen, c)
            ulysses.heads_to_seq(qh, w.n_gen, w.heads, o, None, u.n_chunks, c)
    exchange_only()
    exchange_ms = timed(exchange_only, 5)
    u.close()
    dist.destroy_process_group()
    if rank != 0:
        return
    peaks, peaks_kind = load_peaks()
    value = fl / (ms * 1e-3) / 1e12
    cfg = config_of(w, args)
    cfg["parallelism"] = f"ulysses: {world} rank(s) x {w.heads // world if w.heads % world == 0 else w.heads / world} heads, {u.n_chunks} head chunks per rank"
    cfg["step"] = "cached denoising step on sequence shards: all-to-all -> sra_forward per head chunk -> all-to-all, stream-pipelined"
    cfg["l2"] = "tensors larger than L2, no flush"
    out = {
        "metric": "sra_ulysses_useful_tflops", "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic", "config": cfg, "e2e": None, "gpu_launches": int(launches), "clocks": clocks,
        "pieces": {"pipelined_ms": ms, "direct_ms": direct_ms, "exchange_ms": exchange_ms,
                   "hidden_fraction_of_exchange": max(0.0, min(1.0, (direct_ms + exchange_ms - ms) / exchange_ms)) if exchange_ms > 0 else None},
        "roofline": {"bound": "tensor", "kernel": "sra_fwd_kernel<128>", "achieved": fl / world / (direct_ms * 1e-3) / 1e12,
                     "peak": peaks["bf16_tflops_sustained"], "unit": UNIT,
                     "frac": fl / world / (direct_ms * 1e-3) / 1e12 / peaks["bf16_tflops_sustained"],
                     "peak_kind": f"{peaks_kind} cuBLAS bf16, sustained", "kernel_ms": direct_ms,
                     "algorithmic_flops_per_launch": fl / world / u.n_chunks, "traffic": None},
        "cpu_baseline": None, "parity": None,
    }
    emit(out)


def bench_sweep(args):
    """--mode sweep (BASELINE.json configs[3]; "linear in reference length"): one full forward
    layer (cache build + G and R rows) at 5 / 10 / 20 / 40 s of reference; fits t(N_r) = a + c N_r to the
    forward-kernel times and reports R^2 and t(40 s) / t(5 s) (useful-FLOP ratio 3.88; dense concat: 14.4)."""
    import numpy as np
    import torch
    from paper_2606_13872_b200 import binding as B
    from paper_2606_13872_b200 import inputs as I
    if int(os.environ.get("WORLD_SIZE", "1")) != 1:
        raise SystemExit("bench.py --mode sweep is a single-GPU diagnostic")
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the SRA path has no CPU fallback")
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    peaks, peaks_kind = load_peaks()
    pts = []
    for name in ("sweep5s", "sweep10s", "sweep20s", "sweep40s"):
        w = I.WORKLOADS[name]
        t = {n: I.make_tensor_device(w, n, dev) for n in I.TENSOR_ORDER[:6]}
        o_gen, o_ref = torch.empty_like(t["q_gen"]), torch.empty_like(t["q_ref"])
        ctx = B.sra_create(w.batch, w.heads, w.head_dim, w.n_gen, w.ref_block_offsets)
        B.sra_cache_reference_kv(ctx, t["k_ref"], t["v_ref"])
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        for i in range(max(args.warmup, 3) + args.steps):
            j = i - max(args.warmup, 3)
            if j >= 0:
                ev[j][0].record()
            B.sra_forward(ctx, t["q_gen"], t["k_gen"], t["v_gen"], o_gen, q_ref=t["q_ref"], o_ref=o_ref)
            if j >= 0:
                ev[j][1].record()
        torch.cuda.synchronize()
        ms = statistics.median(a.elapsed_time(b) for a, b in ev)
        fl = useful_flops(w)
        pts.append({"workload": name, "n_ref": w.n_ref, "ms": ms, "useful_tflop": fl / 1e12, "tflops": fl / (ms * 1e-3) / 1e12})
        B.sra_destroy(ctx)
        del t, o_gen, o_ref
        torch.cuda.empty_cache()
    x = np.array([p["n_ref"] for p in pts], dtype=np.float64)
    y = np.array([p["ms"] for p in pts], dtype=np.float64)
    c, a = np.polyfit(x, y, 1)
    r2 = 1.0 - float(((a + c * x - y) ** 2).sum() / ((y - y.mean()) ** 2).sum())
    out = {"metric": "sra_fwd_sweep_linearity", "value": r2, "unit": "R^2 of t(N_r) = a + c N_r", "n_gpus": 1,
           "steps": args.steps, "warmup": max(args.warmup, 3), "higher_is_better": True, "dtype": "bf16", "data": "synthetic",
           "config": {"workload": "long-reference sweep: 480p gen (32,760) + 5/10/20/40 s reference in 1560-token blocks"},
           "fit": {"a_ms": float(a), "c_ms_per_ref_token": float(c), "r2": r2, "t40_over_t5": float(y[-1] / y[0]),
                   "useful_flop_ratio_40_over_5": pts[-1]["useful_tflop"] / pts[0]["useful_tflop"],
                   "dense_concat_ratio_40_over_5": float(((32760 + x[-1]) / (32760 + x[0])) ** 2)},
           "points": pts, "peak_sustained_tflops": peaks["bf16_tflops_sustained"], "peak_kind": peaks_kind}
    emit(out)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=None, help="default: 720p (--mode fwd), train (--mode train)")
    ap.add_argument("--mode", default="fwd", choices=["fwd", "train", "short", "sweep", "rope", "ulysses"],
                    help="fwd: the BASELINE metric (forward layer); train: configs[4] forward + backward; "
                         "short: cache-bound short-query cached steps (--workload short128|short512|short2048), HBM roofline; "
                         "sweep: configs[3] long-reference sweep, linear fit of time vs reference length")
    ap.add_argument("--train-parity", action="store_true",
                    help="--mode train: also check dQ/dK/dV of one (batch, head) against the oracle (minutes of CPU)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-oracle", action="store_true", help="skip the cpu_baseline / parity legs")
    ap.add_argument("--shard", default="batch", choices=["batch", "heads"],
                    help="--mode fwd, N > 1: batch = weak scaling (one item per rank), heads = strong scaling (one item, H / N heads per rank)")
    ap.add_argument("--no-legs", dest="legs", action="store_false",
                    help="--mode fwd on 720p: skip the extra legs (8-step cached protocol, training step, short-query step)")
    ap.add_argument("--oracle-rows", type=int, default=768, help="generation rows in the oracle sample")
    ap.add_argument("--chunks", type=int, default=4, help="--mode ulysses: head chunks per rank (pipeline depth)")
    ap.add_argument("--window", type=int, default=-1,
                    help="--mode fwd: sparse temporal attention window in latent frames (PAPER.md:143); -1 = off")
    ap.add_argument("--invalid-frac", type=float, default=0.0,
                    help="--mode fwd: fraction of reference tokens marked invalid (sparse validity masking, PAPER.md:225)")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # `python bench.py --gpus N` without a launcher: start the N ranks ourselves, exactly as the driver's
        # torchrun line would (one process per GPU, rendezvous on 127.0.0.1); rank 0 of that job prints the line
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.stdout.flush()
        os.execv(sys.executable, cmd)
    claim_stdout()
    if args.warmup < 3 and args.impl == "ours":
        log("note: W < 3 warm-up steps breaks the timing rules; use --warmup >= 3 for a reportable number")
    from paper_2606_13872_b200 import inputs as I
    w = I.WORKLOADS[args.workload or {"train": "train", "short": "short128"}.get(args.mode, "720p")]
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus:
        log(f"note: --gpus {args.gpus} but WORLD_SIZE={world}; the job has WORLD_SIZE ranks and reports that")
        args.gpus = world
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) != 0:
            return
        bench_reference(args, w)
    elif args.mode == "train":
        bench_train(args, w)
    elif args.mode == "short":
        bench_short(args, w)
    elif args.mode == "sweep":
        bench_sweep(args)
    elif args.mode == "rope":
        bench_rope(args, w)
    elif args.mode == "ulysses":
        bench_ulysses(args, w)
    else:
        bench_ours(args, w)


if __name__ == "__main__":
    main()
