#!/usr/bin/env python
"""bench.py -- all-pairs LCS GCUPS / pairs/s on B200 and the fraction of the integer-ALU roofline
(BASELINE.json `metric`), on the seeded synthetic stand-in for the paper's k = 415 519 family
(BASELINE.json configs[4], the workload the north_star target is stated on).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--stride S] [--full]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores

A "step" is one pass of the whole sweep path (pair sweep -> zero count -> similarity epilogue ->
row-block store) over one batch of row blocks of the packed set, inputs
resident in HBM.  For configs 0-2 the batch is ALL rows (the full all-pairs job); for configs 3-4
it is every `stride`-th 1024-row block (default 16), because a full sweep of config 4 takes most
of a minute -- the rate counts true |A|*|B| cells only, so the subset changes the duration, not
the metric; one full sweep is timed as well (`full_sweep`) unless --no-full.  famsa_pack (a1-a3,
one-off) is timed separately (`pack_ms`) and is inside every e2e step.
Prints ONE JSON line (rank 0).
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "all_pairs_lcs_gcups"
UNIT = "GCUPS"
BLOCK_ROWS = 1024
# DRAM traffic of ONE configs[4] step (all its sweep launches), dram__bytes_read.sum + dram__bytes_write.sum per launch
# from ncu, summed: profiles/r02_ncu_step_traffic.md.  Not measurable outside a profiler, so a recorded figure.
NCU_STEP_TRAFFIC = {"config": 4, "bytes": 3.546273e+10, "launches": 39, "source": "profiles/r02_ncu_step_traffic.md"}
ALU_INSTR_PER_CELL = 3.0 / 32.0      # LOP3 + IADD3.X + LOP3 per 32-bit word-step
WORKLOADS = {
    0: "configs[0]: k=500, one family, all 124750 pairs",
    1: "configs[1]: k=10000, 20 families, full all-pairs in 1024-row blocks",
    2: "configs[2]: k=50000 length-skewed set (10% 1500-4000 residues), all pairs",
    3: "configs[3]: k=100000 single family + 2% fragments, uint16 LCS only",
    4: "configs[4]: k=415519 single family, lognormal lengths (mean ~300)",
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--k", type=int, default=None, help="override member count (debugging)")
    ap.add_argument("--stride", type=int, default=None, help="row-block stride of a step (default: 1 for configs 0-2, 16 for 3-4)")
    ap.add_argument("--full", action="store_true", help="a step is the full sweep whatever the config")
    ap.add_argument("--no-full", action="store_true", help="skip the extra single full sweep")
    ap.add_argument("--strong", action="store_true",
                    help="strong scaling: the N=1 batch of row blocks is dealt cyclically over the ranks (default: weak)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--guide-tree", action="store_true",
                    help="also time stages I+II (full sweep + single-linkage guide tree), the whole job dealt over the ranks")
    ap.add_argument("--no-guide-tree", action="store_true", help="skip the stages I+II leg that N=1 runs by default")
    ap.add_argument("--tune", default=None, help="rows_per_cta,small_job_mode,l2_group_mb for famsa_ctx_set_tuning (experiments)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="CPU work per oracle sample")
    ap.add_argument("--workload", default="lcs", choices=["lcs", "seqprof"],
                    help="lcs: the all-pairs LCS sweep (the headline, default); seqprof: SURVEY 8(f) NEXT-4, a batch of sequence-vs-profile alignments")
    ap.add_argument("--batch", type=int, default=8192, help="alignments per step of --workload seqprof")
    ap.add_argument("--n1-max", type=int, default=700, help="--workload seqprof: profile lengths are U[100, n1-max] (default 700)")
    ap.add_argument("--rehearse-one-gpu", action="store_true",
                    help="REHEARSAL of the N > 1 host logic on a box with one GPU: every rank uses cuda:0 and the process group is "
                         "gloo (NCCL refuses two ranks on one device).  The ranks time-slice the GPU, so the numbers mean nothing; "
                         "what it shows is that dealing, reductions, forest gather + merge and the teardown run end to end")
    ap.add_argument("--kernel-only", action="store_true",
                    help="profiling runs: only the device-resident timed steps (no e2e, full-sweep, guide-tree or CPU legs)")
    ap.add_argument("--host-mode", type=int, default=-1, choices=[-1, 0, 1],
                    help="famsa_host_mode of the e2e leg: -1 auto (pinned outputs are stored by the kernels directly), 0 staged copies")
    return ap.parse_args()


def step_blocks(k, stride, offset=0):
    """Row blocks [i0, i1) of one step: every `stride`-th 1024-row block starting at `offset`."""
    nblocks = (k + BLOCK_ROWS - 1) // BLOCK_ROWS
    return [(b * BLOCK_ROWS, min((b + 1) * BLOCK_ROWS, k)) for b in range(offset % max(stride, 1), nblocks, stride)]


def step_config(config, k, stride, blocks, pairs_step, cells_step, want_sim):
    """The `config` object of the JSON line: the same for the CUDA arm and the reference arm."""
    out_bytes = pairs_step * (2 + (4 if want_sim else 0))
    if out_bytes > 126e6:
        l2_note = "no flush needed: every step writes %.2f GB of row-block output (> 126 MB L2) between re-reads" % (out_bytes / 1e9)
    else:
        l2_note = "working set fits L2 (small config); ALU-bound path, no L2 flush between steps"
    return {"workload": WORKLOADS[config], "k": k,
            "step": ("all rows" if stride == 1 else "every %d-th %d-row block (%d blocks)" % (stride, BLOCK_ROWS, len(blocks))),
            "pairs_per_step": pairs_step, "cells_per_step": cells_step, "outputs": "uint16 LCS" + (" + fp32 similarity" if want_sim else ""),
            "l2": l2_note, "parallelism": "replicated set, row blocks dealt per rank, no collective"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, device):
        self.device = device
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.device), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        rows = [l.strip().split(", ") for l in open(self.f.name) if l.strip()]
        os.unlink(self.f.name)
        sm, reasons = [], set()
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1])); out["sm_max_mhz"] = float(r[2])
            except ValueError:
                continue
            for name, v in zip(["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"], r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if sm:
            out["sm_mhz"] = float(np.median(sm)); out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


def oracle_sample(seqs, offsets, blocks, cpu_seconds, seed, n=400000):
    """A bounded seeded sample of the step's pairs for the CPU oracle: uniform over the pairs of
    the step's row blocks, cut where the cell count reaches ~cpu_seconds of work on all cores
    (planning rate 0.3 GCUPS per core).  Returns (orig_i, orig_j, cells, cores, sorted_i, sorted_j)."""
    from oracle import famsa_oracle
    cores = famsa_oracle.n_threads_default()
    perm = famsa_oracle.sort_perm(offsets)
    lens = np.diff(offsets)[perm].astype(np.int64)
    rows = np.concatenate([np.arange(max(a, 1), b, dtype=np.int64) for a, b in blocks]) if blocks else np.zeros(0, np.int64)
    if rows.size == 0:
        z = np.zeros(0, np.int64)
        return z, z, 0.0, cores, z, z
    rng = np.random.default_rng(seed)
    i = rng.choice(rows, size=n, p=rows / rows.sum())
    j = (rng.random(n) * i).astype(np.int64)
    cells = lens[i] * lens[j]
    budget = 0.3e9 * cores * cpu_seconds
    cut = int(np.searchsorted(np.cumsum(cells), budget)) + 1
    cut = min(cut, n)
    return perm[i[:cut]], perm[j[:cut]], float(cells[:cut].sum()), cores, i[:cut], j[:cut]


def time_bitparallel(seqs, offsets, blocks, seconds, seed):
    """CONTEXT figure: the paper's own CPU design (64-bit bit-parallel LCS, several pairs per SIMD register,
    rows over threads; oracle/bitpar_cpu.c) on a bounded sample of the step: seeded rows of the step's row
    blocks, 128 seeded columns j < i each (the row's match table is built once, as in the paper's design).
    Every ISA variant the host runs is timed after a pilot that sizes the sample for ~`seconds` of work."""
    from oracle import famsa_oracle
    cores = famsa_oracle.n_threads_default()
    perm = famsa_oracle.sort_perm(offsets)
    lens = np.diff(offsets)[perm].astype(np.int64)
    rows_all = np.concatenate([np.arange(max(a, 128), b, dtype=np.int64) for a, b in blocks if b > 128]) if blocks else np.zeros(0, np.int64)
    if rows_all.size == 0:
        return None
    rng = np.random.default_rng(seed)
    ncol = 128

    def sample(n_rows):
        ri = rng.choice(rows_all, size=n_rows, p=rows_all / rows_all.sum())
        cj = (rng.random((n_rows, ncol)) * ri[:, None]).astype(np.int64)
        cj.sort(axis=1)           # sorted indices = sorted lengths: the `a` pairs of one SIMD step have similar lengths
        cells = float((lens[ri][:, None] * lens[cj]).sum())
        col_ptr = np.arange(n_rows + 1, dtype=np.int64) * ncol
        return perm[ri], col_ptr, perm[cj].ravel(), cells

    best = famsa_oracle.bitpar_best_isa()
    variants = [0, 2] + ([14] if best in (14, 18) else []) + ([18] if best == 18 else [])
    out = {}
    for isa in variants:
        ri, cp, cj, cells = sample(256 * cores)                       # pilot
        t0 = time.perf_counter()
        famsa_oracle.bitpar_rowsets(seqs, offsets, ri, cp, cj, isa=isa)
        rate = cells / max(time.perf_counter() - t0, 1e-6)
        n_rows = int(min(max(rate * seconds / (cells / (256 * cores)), 256 * cores), 40_000_000 // ncol))
        ri, cp, cj, cells = sample(n_rows)
        t0 = time.perf_counter()
        famsa_oracle.bitpar_rowsets(seqs, offsets, ri, cp, cj, isa=isa)
        dt = time.perf_counter() - t0
        out[isa] = {"gcups": cells / dt / 1e9, "pairs_per_s": n_rows * ncol / dt, "seconds": dt, "pairs": n_rows * ncol, "cells": cells}
    top = max(out, key=lambda q: out[q]["gcups"])
    return {"value": out[top]["gcups"], "unit": UNIT, "cores": cores, "isa": famsa_oracle.BITPAR_ISA_NAMES[top],
            "kind": "context: the paper's own CPU design (PAPER.md:44, 54-56: 64-bit bit-parallel LCS, `a` pairs per SIMD "
                    "register, rows over threads; oracle/bitpar_cpu.c) -- not a parity oracle",
            "pairs_per_s": out[top]["pairs_per_s"],
            "sample": "%d seeded rows of the step's row blocks x %d seeded columns (%.3g cells, %.1f s)" % (
                out[top]["pairs"] // ncol, ncol, out[top]["cells"], out[top]["seconds"]),
            "variants_gcups": {famsa_oracle.BITPAR_ISA_NAMES[q]: round(v["gcups"], 2) for q, v in out.items()}}


def time_oracle(seqs, offsets, pi, pj, want_sim):
    from oracle import famsa_oracle
    t0 = time.perf_counter()
    famsa_oracle.pairs(seqs, offsets, pi, pj, want_sim=want_sim)
    return time.perf_counter() - t0


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle as it stands, on the host cores; rank 0 only."""
    if rank != 0:
        return
    from paper_1603_06958_b200 import synth
    seqs, offsets = synth.family(args.config, k=args.k)
    k = len(offsets) - 1
    stride = args.stride or (1 if args.config <= 2 else 16)
    blocks = step_blocks(k, 1 if args.full else stride)
    want_sim = args.config != 3
    secs = min(args.cpu_seconds, 8.0)
    # the CUDA arm's step, described identically (exact integer sums: every value is below 2^53)
    from oracle import famsa_oracle
    lens = np.diff(offsets)[famsa_oracle.sort_perm(offsets)].astype(np.int64)
    prefix = np.concatenate([[0], np.cumsum(lens)])
    pairs_cfg = int(sum(b * (b - 1) // 2 - a * (a - 1) // 2 for a, b in blocks))
    cells_cfg = float(sum(int((lens[a:b] * prefix[a:b]).sum()) for a, b in blocks))
    times, cells_step, pairs_step, cores = [], 0.0, 0, 1
    for s in range(args.warmup + args.steps):
        pi, pj, cells, cores, _, _ = oracle_sample(seqs, offsets, blocks, secs, seed=1000 + s)
        dt = time_oracle(seqs, offsets, pi, pj, want_sim)
        if s >= args.warmup:
            times.append(dt); cells_step += cells; pairs_step += pi.size
    total = sum(times)
    value = cells_step / total / 1e9
    sample = "%d seeded uniform pairs of the step's row blocks per step (~%.0f s of CPU work)" % (pairs_step // max(args.steps, 1), secs)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": total / max(args.steps, 1) * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "int32", "data": "synthetic",
        "config": step_config(args.config, k, 1 if args.full else stride, blocks, pairs_cfg, cells_cfg, want_sim),
        "pairs_per_s": pairs_step / total,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "note": "the reference arm is the plain-DP oracle, as the task contract states; the paper's own method on "
                "these cores (bit-parallel, multi-pair SIMD) is `cpu_bitparallel` -- divide by that for an honest speed-up",
    }
    if not args.no_cpu:
        line["cpu_bitparallel"] = time_bitparallel(seqs, offsets, blocks, min(args.cpu_seconds, 6.0), seed=11)
    print(json.dumps(line), flush=True)


def rank_blocks(k, stride, rank, world=1, strong=False):
    """The row blocks rank `rank` sweeps in one step.  Pairs are independent, so the path
    shards with no data-path collective: the packed set is replicated and row blocks are dealt by rank.
    stride > 1: rank r takes blocks r, r+stride, ... (disjoint batches of equal size: weak scaling);
    stride 1: the batch is the whole job and every rank sweeps its own replica of it."""
    if strong:                                    # the N=1 batch, dealt block by block: block n of the batch -> rank n mod N
        return step_blocks(k, stride)[rank::world]
    return step_blocks(k, stride, offset=rank if stride > 1 else 0)


def reduce_over_ranks(dist, ms, cells, pairs, device):
    """Whole-job figures: MAX of the device time over ranks, SUM of the cells and pairs processed."""
    if dist is None:
        return ms, cells, float(pairs)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tot = torch.tensor([cells, float(pairs)], dtype=torch.float64, device=device)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(t.item()), float(tot[0].item()), float(tot[1].item())


def gather_forests(dist, a, b, w, k, device):
    """The one exchange step of the multi-GPU guide tree: every rank's forest edges (<= k-1 each) to every
    rank.  Padded all_gather (NCCL on device tensors; gloo on CPU tensors in the tests).  Returns a list of
    (a, b, w) numpy triples, one per rank."""
    import torch
    if dist is None:
        return [(a, b, w)]
    world = dist.get_world_size()
    cap = max(int(k) - 1, 1)
    ab = torch.zeros((cap, 2), dtype=torch.int64, device=device)
    ww = torch.zeros(cap, dtype=torch.float32, device=device)
    n = torch.tensor([a.size], dtype=torch.int64, device=device)
    if a.size:
        ab[:a.size, 0] = torch.from_numpy(np.ascontiguousarray(a)).to(device)
        ab[:a.size, 1] = torch.from_numpy(np.ascontiguousarray(b)).to(device)
        ww[:a.size] = torch.from_numpy(np.ascontiguousarray(w)).to(device)
    abs_, wws, ns = ([torch.zeros_like(x) for _ in range(world)] for x in (ab, ww, n))
    dist.all_gather(abs_, ab)
    dist.all_gather(wws, ww)
    dist.all_gather(ns, n)
    out = []
    for r in range(world):
        m = int(ns[r].item())
        out.append((abs_[r][:m, 0].cpu().numpy(), abs_[r][:m, 1].cpu().numpy(), wws[r][:m].cpu().numpy()))
    return out


def gather_sampled(F, torch, ctx, blocks, si, sj, bufs, ck, stream):
    """One un-timed pass over the step's row blocks that (a) accumulates each block's checksum into ck[n]
    and (b) picks the sampled entries (sorted pair indices si > sj, any order) out of each block while it
    sits in its ping-pong buffer.  Returns (lcs int64, sim float64) numpy arrays parallel to si."""
    dev = bufs[0][0].device
    order = np.argsort(si, kind="stable")
    si_s, sj_s = si[order], sj[order]
    got_l = torch.zeros(si.size, dtype=torch.int16, device=dev)
    got_s = torch.zeros(si.size, dtype=torch.float32, device=dev)
    pos_all = torch.from_numpy(si_s * (si_s - 1) // 2 + sj_s).to(dev)
    for n, (a, b) in enumerate(blocks):
        lcs, sim = bufs[n & 1]
        F.famsa_lcs_rows_checksum(ctx, a, b, lcs, sim, ck[n], stream)
        lo, hi = int(np.searchsorted(si_s, a)), int(np.searchsorted(si_s, b))
        if hi > lo:
            idx = pos_all[lo:hi] - a * (a - 1) // 2
            got_l[lo:hi] = lcs.view(torch.int16)[idx]
            if sim is not None:
                got_s[lo:hi] = sim[idx]
    torch.cuda.synchronize()
    gl = np.empty(si.size, np.int64); gs = np.empty(si.size, np.float64)
    gl[order] = got_l.cpu().numpy().view(np.uint16).astype(np.int64)
    gs[order] = got_s.cpu().numpy().astype(np.float64)
    return gl, gs


def run_cuda(args, rank, world, local_rank):
    import torch
    from paper_1603_06958_b200 import famsa as F, synth
    dist = None
    if world > 1:
        import torch.distributed as dist
        if args.rehearse_one_gpu:
            local_rank = 0
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    coll_dev = torch.device("cpu") if args.rehearse_one_gpu else dev     # where the tensors of the collectives live

    seqs, offsets = synth.family(args.config, k=args.k)      # replicated on every rank
    k = len(offsets) - 1
    want_sim = args.config != 3                               # configs[3]: uint16 row blocks only
    stride = 1 if args.full else (args.stride or (1 if args.config <= 2 else 16))
    # weak scaling: rank r sweeps its own batch of row blocks (offset r), same size as the N=1 batch
    blocks = rank_blocks(k, stride, rank, world, args.strong)
    if not blocks:
        blocks = step_blocks(k, stride)[:1]       # more ranks than blocks: repeat one block rather than idle (reported cells stay true)

    peak0 = F.famsa_alu_peak(local_rank)
    mix0 = F.famsa_mix_peak(local_rank)
    t0 = time.perf_counter()
    ctx = F.famsa_pack(seqs, offsets, device=local_rank)
    torch.cuda.synchronize()
    pack_ms = (time.perf_counter() - t0) * 1e3
    pack_launches = F.famsa_launch_count(ctx)
    if args.tune:
        F.famsa_ctx_set_tuning(ctx, *[int(x) for x in args.tune.split(",")])

    max_pairs = max(F.famsa_rows_pairs(a, b) for a, b in blocks)
    bufs = [(torch.empty(max_pairs, dtype=torch.uint16, device=dev),
             torch.empty(max_pairs, dtype=torch.float32, device=dev) if want_sim else None) for _ in range(2)]
    cells_step = sum(F.famsa_rows_cells(ctx, a, b) for a, b in blocks)
    pairs_step = sum(F.famsa_rows_pairs(a, b) for a, b in blocks)
    stream = torch.cuda.current_stream()
    # one 64-bit checksum pair per row block, accumulated by the sweep's own epilogue in every timed step
    # ("a 64-bit checksum per block is kept to prove the work was done")
    ck = torch.zeros((len(blocks), 2), dtype=torch.int64, device=dev)

    def step():
        for n, (a, b) in enumerate(blocks):
            lcs, sim = bufs[n & 1]                            # ping-pong: the consumer owns one block while the next is swept
            F.famsa_lcs_rows_checksum(ctx, a, b, lcs, sim, ck[n], stream)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    ck.zero_()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    # Per-step events only when a step is long: an event record between two sweep launches is a stream operation
    # that is not a kernel, so the next launch cannot start programmatically while its predecessor drains (6.5),
    # and a 0.1 ms step (configs[0]) would be measured without the overlap that back-to-back calls really get.
    probe = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    probe[0].record(stream); step(); probe[1].record(stream); torch.cuda.synchronize()
    per_step_events = probe[0].elapsed_time(probe[1]) > 5.0
    if not per_step_events:               # short steps: let the sampler's start-up (it briefly stalls the GPU) pass untimed
        t_w = time.perf_counter()
        while time.perf_counter() - t_w < 0.6:
            step()
            torch.cuda.synchronize()
    ck.zero_()
    barrier()
    l0 = F.famsa_launch_count(ctx)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    ev[0].record(stream)
    for s in range(args.steps):
        step()
        if per_step_events or s == args.steps - 1:
            ev[s + 1].record(stream)
    barrier()
    clocks = sampler.stop()
    launches = F.famsa_launch_count(ctx) - l0
    ms_total = ev[0].elapsed_time(ev[-1])
    step_ms = [ev[s].elapsed_time(ev[s + 1]) for s in range(args.steps)] if per_step_events else None
    ms_rank = ms_total
    ms_total, cells_all, pairs_all = reduce_over_ranks(dist, ms_total, cells_step, pairs_step, coll_dev)
    sec = ms_total * 1e-3
    value = cells_all * args.steps / sec / 1e9
    ck_timed = ck.cpu().numpy().astype(np.uint64)

    # ---- was the timed work right?  One more (un-timed) pass: fresh checksums + the entries of the oracle's
    # sample gathered from the row blocks; the comparison with the oracle happens in the cpu_baseline leg
    sample = None
    if rank == 0 and not args.no_cpu:
        sample = oracle_sample(seqs, offsets, blocks, args.cpu_seconds, seed=7)
    ck1 = torch.zeros_like(ck)
    si = sample[4] if sample is not None else np.zeros(0, np.int64)
    sj = sample[5] if sample is not None else np.zeros(0, np.int64)
    gpu_l, gpu_s = gather_sampled(F, torch, ctx, blocks, si, sj, bufs, ck1, stream)
    ck_once = ck1.cpu().numpy().astype(np.uint64)
    checksum = {"blocks": len(blocks), "lcs_sum_step": int(ck_once[:, 0].sum()), "sim_bits_sum_step": int(ck_once[:, 1].sum() & np.uint64(2**64 - 1)),
                "timed_steps_equal_steps_x_one_pass": bool(np.array_equal(ck_timed, ck_once * np.uint64(args.steps)))}
    # the last two blocks still sit in the ping-pong buffers: reduce them with torch (independent of the kernels)
    indep = True
    for n in range(max(0, len(blocks) - 2), len(blocks)):
        a, b = blocks[n]
        npairs = F.famsa_rows_pairs(a, b)
        lcs, sim = bufs[n & 1]
        sl = int((lcs.view(torch.int16)[:npairs].to(torch.int64) & 0xFFFF).sum().item())
        indep &= sl == int(ck_once[n, 0])
        if sim is not None:
            indep &= int(sim[:npairs].view(torch.int32).to(torch.int64).sum().item()) == int(ck_once[n, 1])
    checksum["last_blocks_equal_torch_reduction"] = bool(indep)

    # ---- e2e: HOST buffers through the C ABI; pack (H2D of the residues) + sweep + D2H every step
    # (one call over all rows when the whole result fits 2 GB of pinned memory, else one call per row block
    #  into a reused pinned row-block buffer -- the consumer owns a block only until the next one arrives)
    one_call = stride == 1 and pairs_step * 6 <= 2e9
    e2e_pairs = pairs_step if one_call else max_pairs
    h_lcs = torch.empty(e2e_pairs, dtype=torch.uint16).pin_memory()
    h_sim = torch.empty(e2e_pairs, dtype=torch.float32).pin_memory() if want_sim else None
    h_lcs2 = [h_lcs, h_lcs if one_call else torch.empty(e2e_pairs, dtype=torch.uint16).pin_memory()]
    h_sim2 = [h_sim, h_sim if (one_call or not want_sim) else torch.empty(e2e_pairs, dtype=torch.float32).pin_memory()]
    # long steps: 2 timed e2e steps; short steps (small configs) are noisy (allocations in pack): more of them
    e2e_steps = max(1, min(args.steps, 2)) if ms_total / args.steps > 500.0 else max(2, min(2 * args.steps, 10))
    phases = {"pack_ms": 0.0, "sweep_ms": 0.0, "d2h_ms": 0.0, "d2h_bytes": 0.0, "span_ms": 0.0, "chunks": 0}
    # the step's inputs come from PINNED host memory (the bench contract); outputs go to pinned row-block buffers
    p_seqs = torch.from_numpy(seqs).pin_memory().numpy()
    p_offsets = torch.from_numpy(offsets).pin_memory().numpy()

    def e2e_step(profile=False):
        t_p = time.perf_counter()
        c2 = F.famsa_pack(p_seqs, p_offsets, device=local_rank)
        if args.tune:
            F.famsa_ctx_set_tuning(c2, *[int(x) for x in args.tune.split(",")])
        F.famsa_host_mode(c2, args.host_mode)
        phases["pack_ms"] += (time.perf_counter() - t_p) * 1e3 if profile else 0.0
        if profile:
            F.famsa_host_profile(c2, True)
            phases["pack_phases_ms"] = F.famsa_pack_profile(c2)
        if one_call:
            F.famsa_lcs_rows_host(c2, 0, k, h_lcs, h_sim)
        else:
            for n, (a, b) in enumerate(blocks):               # two pinned row-block buffers, copies overlap the next sweep
                F.famsa_lcs_rows_host_async(c2, a, b, h_lcs2[n & 1], h_sim2[n & 1] if want_sim else None)
            F.famsa_sync(c2)
        if profile:
            for key, v in F.famsa_host_profile_read(c2).items():
                phases[key] += v
        c2.free()
    if args.kernel_only:
        e2e_steps = 0
    else:
        e2e_step()                                            # warm-up (allocations, staging buffers)
        if ms_total / args.steps <= 500.0:
            e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        e2e_step()
    barrier()
    e2e_sec = max(time.perf_counter() - t0, 1e-9)
    if dist is not None:
        t = torch.tensor([e2e_sec], dtype=torch.float64, device=coll_dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_sec = float(t.item())
    e2e_value = cells_all * e2e_steps / e2e_sec / 1e9
    h2d = int(seqs.nbytes + offsets.nbytes)
    d2h = int(pairs_step * (2 + (4 if want_sim else 0)))
    # one more e2e step, un-timed, with the per-phase CUDA events switched on (they serialise nothing, but
    # the step is kept out of the timed region anyway)
    t_w = time.perf_counter()
    if not args.kernel_only:
        e2e_step(profile=True)
    phases["wall_ms"] = (time.perf_counter() - t_w) * 1e3
    if phases["d2h_ms"] > 0:
        phases["d2h_gb_per_s"] = phases["d2h_bytes"] / phases["d2h_ms"] / 1e6
    F.famsa_trim()                                            # hand the pooled staging back before the big buffers below

    # ---- one full sweep, timed alone (N = 1, configs 3-4 only: the other configs' step already is one)
    full = None
    if stride > 1 and world == 1 and not args.no_full:
        allb = step_blocks(k, 1)
        big = max(F.famsa_rows_pairs(a, b) for a, b in allb)
        if big > max_pairs:
            bufs = None
            torch.cuda.empty_cache()
            bufs = [(torch.empty(big, dtype=torch.uint16, device=dev),
                     torch.empty(big, dtype=torch.float32, device=dev) if want_sim else None) for _ in range(2)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for n, (a, b) in enumerate(allb):
            F.famsa_lcs_rows(ctx, a, b, bufs[n & 1][0], bufs[n & 1][1], stream)
        e1.record(stream)
        torch.cuda.synchronize()
        fms = e0.elapsed_time(e1)
        fcells = F.famsa_rows_cells(ctx, 0, k)
        full = {"ms": fms, "gcups": fcells / fms / 1e6, "pairs": F.famsa_rows_pairs(0, k),
                "pairs_per_s": F.famsa_rows_pairs(0, k) / fms * 1e3, "cells": fcells}
    tree = None
    if args.guide_tree or (world == 1 and want_sim and not args.no_guide_tree):
        # stages I + II, the WHOLE job dealt over the ranks (strong scaling): rank r sweeps row blocks
        # r, r + N, ... and keeps their spanning forest; one all_gather of the forests' edges; rank 0 merges
        bufs = None
        torch.cuda.empty_cache()
        barrier()
        l1 = F.famsa_launch_count(ctx)
        t0 = time.perf_counter()
        forest = F.famsa_guide_forest(ctx, BLOCK_ROWS, rank, world)
        t_forest = time.perf_counter() - t0
        fa, fb, fw = F.famsa_tree_edges(forest)
        parts = gather_forests(dist, fa, fb, fw, k, coll_dev)
        n_merges = 0
        t1 = time.perf_counter()
        if rank == 0:
            for r in range(1, world):
                F.famsa_tree_merge_edges(forest, *parts[r])
            ia, ib, mw, msize = F.famsa_tree_finish(forest)
            n_merges = int(mw.size)
        t_finish = time.perf_counter() - t1
        barrier()
        dt = time.perf_counter() - t0
        forest.free()
        if dist is not None:
            tt = torch.tensor([dt], dtype=torch.float64, device=coll_dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            dt = float(tt.item())
        fcells = F.famsa_rows_cells(ctx, 0, k)
        if rank == 0:
            tree = {"seconds": dt, "gcups_equivalent": fcells / dt / 1e9, "launches_rank0": F.famsa_launch_count(ctx) - l1,
                    "forest_seconds_rank0": t_forest, "merge_and_dendrogram_seconds": t_finish,
                    "merges": n_merges, "top_similarity": float(mw[0]) if mw.size else None,
                    "last_similarity": float(mw[-1]) if mw.size else None, "scaling": "strong", "n_gpus": world,
                    "what": "famsa_guide_forest per rank (cyclic deal of all 1024-row blocks: sweep, fp32 similarity only, + incremental "
                            "single-linkage forest), all_gather of the forests' edges, merge + dendrogram on rank 0; wall clock, max over ranks"}
    peak1 = F.famsa_alu_peak(local_rank)
    mix1 = F.famsa_mix_peak(local_rank)
    ctx.free()
    if dist is not None:                  # every collective is behind us: leave the group together, BEFORE rank 0's
        dist.barrier()                    # CPU legs (tens of seconds), so that no rank tears down a communicator
        dist.destroy_process_group()      # whose peers have already exited
        dist = None
    if rank != 0:
        return

    # ---- rank 0: the oracle beside it (and against it), the roofline, the line
    cpu = None
    parity = None
    if sample is not None:
        pi, pj, ccells, cores = sample[:4]
        from oracle import famsa_oracle
        t0 = time.perf_counter()
        lref, sref = famsa_oracle.pairs(seqs, offsets, pi, pj, want_sim=want_sim)
        dt = time.perf_counter() - t0
        cpu = {"value": ccells / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
               "pairs_per_s": pi.size / dt,
               "sample": "%d seeded uniform pairs of the step's row blocks (%.3g cells, %.1f s)" % (pi.size, ccells, dt)}
        # the same pairs, as the GPU stored them in the step's row blocks
        mism = int((gpu_l != lref).sum())
        rel = 0.0
        inf_ok = True
        if want_sim:
            fin = np.isfinite(sref)
            inf_ok = bool(np.array_equal(np.isinf(gpu_s), ~fin))
            if fin.any():
                rel = float(np.max(np.abs(gpu_s[fin] - sref[fin]) / np.abs(sref[fin])))
        parity = {"pairs": int(pi.size), "lcs_mismatch": mism, "sim_max_rel_err": rel, "inf_match": inf_ok,
                  "what": "the cpu_baseline sample's oracle results vs the entries the CUDA path stored for the same pairs"}
    cpu_bp = None
    if not args.no_cpu:
        cpu_bp = time_bitparallel(seqs, offsets, blocks, min(args.cpu_seconds, 6.0), seed=11)
    p_int = max(peak0["instr_per_s"], peak1["instr_per_s"])          # measured INT32 ALU-pipe rate (thread-instr/s)
    sm_count = torch.cuda.get_device_properties(local_rank).multi_processor_count
    achieved = cells_step * args.steps * ALU_INSTR_PER_CELL / (ms_rank * 1e-3)   # this rank's stream
    peaks_file = os.path.join(ROOT, "MEASURED_PEAKS.json")
    sm_max = 1965.0
    hbm_gbs, hbm_src = 6650.0, "fallback of B200_PROFILING.md (MEASURED_PEAKS.json absent)"
    if os.path.exists(peaks_file):
        peaks = json.load(open(peaks_file))
        sm_max = float(peaks.get("sm_max_mhz", sm_max))
        if peaks.get("hbm_gbs"):
            hbm_gbs, hbm_src = float(peaks["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    nominal = sm_count * 64 * sm_max * 1e6
    out_bytes = pairs_step * (2 + (4 if want_sim else 0))
    traffic = None
    traffic_note = "dram__bytes_* need a profiler; no recorded capture for this config (see profiles/)"
    if NCU_STEP_TRAFFIC["bytes"] and args.config == NCU_STEP_TRAFFIC["config"] and stride == 16 and world == 1:
        traffic = NCU_STEP_TRAFFIC["bytes"] / NCU_STEP_TRAFFIC["launches"]
        traffic_note = ("dram__bytes_read.sum + dram__bytes_write.sum summed over the %d sweep launches of one step of this workload "
                        "(%.3g B) / launches, recorded in %s; the step's algorithmic output is %.3g B" % (
                            NCU_STEP_TRAFFIC["launches"], NCU_STEP_TRAFFIC["bytes"], NCU_STEP_TRAFFIC["source"], out_bytes))
    roofline = {
        "bound": "alu", "achieved": achieved / 1e12, "peak": p_int / 1e12, "unit": "TIOP/s (int32 ALU-pipe lane-instr)",
        "frac": achieved / p_int, "traffic": traffic, "traffic_note": traffic_note,
        "traffic_step_over_algorithmic": (NCU_STEP_TRAFFIC["bytes"] / out_bytes) if traffic else None,
        "kernel": "famsa::sweep_short_kernel<W,NR> (%d launches per step)" % (launches // max(args.steps, 1)),
        "algorithmic_instr_per_cell": ALU_INSTR_PER_CELL,
        "peak_source": "famsa_alu_peak micro-kernel, measured in this run (MEASURED_PEAKS.json has no integer peak)",
        "peak_instr_per_clk_sm": max(peak0["instr_per_clk_sm"], peak1["instr_per_clk_sm"]),
        "peak_sm_mhz": max(peak0["sm_mhz"], peak1["sm_mhz"]),
        "mix_ceiling_instr_per_clk_sm": max(mix0["alu_instr_per_clk_sm"], mix1["alu_instr_per_clk_sm"]),
        "mix_note": "famsa_mix_peak: the same micro-kernel with the sweep's mix (3 ALU + 1 conflict-free LDS.32 per word-step)",
        "frac_of_nominal_64_per_clk_sm_at_max_clock": achieved / nominal,
        "roofline_gcups": p_int / ALU_INSTR_PER_CELL / 1e9,
    }
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "strong" if args.strong else "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic",
        "config": step_config(args.config, k, stride, blocks, pairs_step, cells_step, want_sim),
        "pairs_per_s": pairs_all * args.steps / sec,
        "step_ms": step_ms, "pack_ms": pack_ms,
        "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"], "samples": clocks["samples"]},
        "e2e": None if args.kernel_only else {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "frac_of_device_resident": e2e_value / value,
                "what": "famsa_pack from pinned host memory + famsa_lcs_rows_host into pinned host row-block buffers, every step",
                "host_mode": {-1: "auto: pinned outputs, so the sweep kernels store the rows straight into host memory (posted PCIe writes; "
                                  "the transfer is inside sweep_ms and d2h_ms stays 0)",
                              0: "staged: device row chunks + cudaMemcpyAsync on a copy stream", 1: "direct"}[args.host_mode],
                "phases_of_one_untimed_step": phases},
        "gpu_launches": launches,
        "roofline": roofline,
        "checksum": checksum,
        "parity_in_bench": parity,
        "cpu_baseline": cpu,
        "cpu_bitparallel": cpu_bp,
        "output_gb_per_s": pairs_all * args.steps * (2 + (4 if want_sim else 0)) / sec / 1e9,
        "output_frac_of_hbm_peak": pairs_all * args.steps * (2 + (4 if want_sim else 0)) / sec / 1e9 / (hbm_gbs * world),
        "hbm_peak_gb_per_s": hbm_gbs, "hbm_peak_source": hbm_src,
    }
    if full is not None:
        line["full_sweep"] = full
    if tree is not None:
        line["guide_tree"] = tree
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()
    ok = checksum["timed_steps_equal_steps_x_one_pass"] and checksum["last_blocks_equal_torch_reduction"]
    if parity is not None:
        ok = ok and parity["lcs_mismatch"] == 0 and parity["inf_match"] and parity["sim_max_rel_err"] <= 1e-6
    if not ok:
        sys.stderr.write("bench.py: the timed work FAILED its self-check (checksum / parity_in_bench above)\n")
        sys.exit(3)


def run_seqprof(args, rank, world, local_rank):
    """one step = one batch of independent sequence-vs-profile alignments (profile costs from
    the counters, DP with traceback), inputs resident in HBM; e2e = the same through the C ABI from pinned host
    arrays with the scores, paths and path lengths read back.  Metric: DP cells (n1 x n2) per second."""
    import torch
    from paper_1603_06958_b200 import famsa as F, synth
    dist = None
    if world > 1:                      # alignments are independent: every rank takes its own batch, no collective
        import torch.distributed as dist
        if args.rehearse_one_gpu:
            local_rank = 0
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    coll_dev = torch.device("cpu") if args.rehearse_one_gpu else dev
    B = args.batch
    counts, col_off, seq, seq_off, nseq = synth.profile_batch(B, seed=SEQPROF_SEED + rank, n1_range=(100, args.n1_max))
    subst = synth.substitution_matrix()
    gaps = np.tile(np.array([0.66, 0.66, 14.85, 1.25], np.float32) * np.float32(F.famsa_gap_scale(B)), (B, 1))
    n1 = np.diff(col_off); n2 = np.diff(seq_off)
    cells = float((n1 * n2).sum())
    h = {"counts": torch.from_numpy(counts.astype(np.int32)).pin_memory(), "seq": torch.from_numpy(seq).pin_memory(),
         "gaps": torch.from_numpy(gaps).pin_memory(), "nseq": torch.from_numpy(nseq).pin_memory(), "subst": torch.from_numpy(subst).pin_memory()}
    d = {k_: v.to(dev) for k_, v in h.items()}
    cost = torch.empty((counts.shape[0], 32), dtype=torch.float32, device=dev)
    score = torch.empty(B, dtype=torch.float32, device=dev)
    path = torch.empty(int(col_off[-1] + seq_off[-1]), dtype=torch.uint8, device=dev)
    plen = torch.empty(B, dtype=torch.int32, device=dev)
    ws = torch.empty(F.famsa_seqprof_workspace(col_off, seq_off), dtype=torch.uint8, device=dev)
    stream = torch.cuda.current_stream()

    def step(src):
        F.famsa_profile_costs(src["counts"], src["subst"], cost, stream)
        F.famsa_seqprof_align(cost, col_off, src["seq"], seq_off, src["gaps"], src["nseq"], score, path, plen, ws, stream)
    # The clock sampler (an nvidia-smi process) is started BEFORE the warm-up and given half a second: its start-up
    # briefly stalls the GPU, which is invisible in a timed region of seconds but tripled a 30 ms one when it fell inside.
    sampler = ClockSampler(local_rank); sampler.start()
    t_w = time.perf_counter()
    n_warm = 0
    while n_warm < args.warmup or time.perf_counter() - t_w < 0.6:
        step(d); n_warm += 1
        torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for _ in range(args.steps):
        step(d)
    e1.record(stream)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    ms_rank = e0.elapsed_time(e1)
    ms, cells_all, _ = reduce_over_ranks(dist, ms_rank, cells, B, coll_dev)      # max time over ranks, sum of the cells
    value = cells_all * args.steps / ms / 1e6
    peak = F.famsa_alu_peak(local_rank)
    # Roofline: the ALU pipe.  Per cell and state: 2 compares + 2 value selects + 2 direction selects on
    # the ALU pipe (18 per cell; the 7 fp32 adds / subtracts run on the FMA pipe beside them).
    alu_per_cell = 18.0
    roofline = {"bound": "alu", "achieved": cells * args.steps * alu_per_cell / (ms_rank * 1e-3) / 1e12, "peak": peak["instr_per_s"] / 1e12,
                "unit": "TIOP/s (ALU-pipe lane-instr)", "frac": cells * args.steps * alu_per_cell / (ms_rank * 1e-3) / peak["instr_per_s"],
                "traffic": None, "algorithmic_instr_per_cell": alu_per_cell, "kernel": "famsa::seqprof_kernel<J>",
                "peak_source": "famsa_alu_peak micro-kernel, measured in this run",
                "note": "padding of n2 to SEG x J lane slots, the (SEG - 1)-step skew of the wavefront and the traceback all count against the kernel"}
    # e2e: pinned host inputs -> device, results back to pinned host, every step
    h_score = torch.empty(B, dtype=torch.float32).pin_memory(); h_path = torch.empty(path.numel(), dtype=torch.uint8).pin_memory()
    h_plen = torch.empty(B, dtype=torch.int32).pin_memory()
    def e2e_step():
        src = {k_: v.to(dev, non_blocking=True) for k_, v in h.items()}
        step(src)
        h_score.copy_(score, non_blocking=True); h_path.copy_(path, non_blocking=True); h_plen.copy_(plen, non_blocking=True)
        torch.cuda.synchronize()
    e2e_step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    e2e_sec = time.perf_counter() - t0
    if dist is not None:
        tt = torch.tensor([e2e_sec], dtype=torch.float64, device=coll_dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_sec = float(tt.item())
        dist.destroy_process_group()
    if rank != 0:
        return
    # the oracle beside it and against it: a bounded sample of the batch (fp32 mode: same-precision decisions)
    cpu = parity = None
    if not args.no_cpu and rank == 0:
        from oracle import profile_oracle as po
        hc = cost.cpu().numpy(); hs = score.cpu().numpy(); hp = path.cpu().numpy(); hl = plen.cpu().numpy()
        rng = np.random.default_rng(5); pick = rng.permutation(B)[:min(B, 4000)]
        t0 = time.perf_counter(); bad = 0; ccells = 0.0
        for b in pick:
            s32, p32 = po.align(hc[col_off[b]:col_off[b + 1]], seq[seq_off[b]:seq_off[b + 1]], gaps[b], int(nseq[b]), want_path=True, precision="f32")
            end = int(col_off[b + 1] + seq_off[b + 1])
            bad += int(not (hs[b] == np.float32(s32) and np.array_equal(hp[end - hl[b]:end], p32)))
            ccells += float(n1[b] * n2[b])
            if time.perf_counter() - t0 > args.cpu_seconds:
                break
        dt = time.perf_counter() - t0
        cpu = {"value": ccells / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
               "sample": "oracle/profile_oracle.c (fp32 mode, with traceback) on seeded alignments of the batch for %.1f s, one thread" % dt}
        parity = {"alignments": int(ccells > 0) and int(np.searchsorted(np.cumsum(n1[pick] * n2[pick]), ccells) + 1), "mismatch": bad,
                  "what": "score bit-exact and path identical to the oracle's fp32 mode"}
    line = {"metric": "seqprof_dp_gcups", "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": "SURVEY 8(f) NEXT-4: %d independent sequence-vs-profile alignments per step (profiles of 100-%d columns from 1-40 "
                                   "sequences, sequences with indels), costs + DP + traceback" % (B, args.n1_max),
                       "cells_per_step": cells, "l2": "direction matrices (%.2f GB per step) exceed L2" % (ws.numel() / 1e9)},
            "alignments_per_s": B * world * args.steps / ms * 1e3,
            "clocks": {"sm_mhz": clocks["sm_mhz"], "sm_max_mhz": clocks["sm_max_mhz"], "reasons": clocks["reasons"], "samples": clocks["samples"]},
            "e2e": {"value": cells_all * args.steps / e2e_sec / 1e9, "unit": UNIT,
                    "h2d_bytes_per_step": int(sum(v.numel() * v.element_size() for v in h.values())),
                    "d2h_bytes_per_step": int(h_score.numel() * 4 + h_path.numel() + h_plen.numel() * 4)},
            "gpu_launches": 10 * args.steps, "roofline": roofline, "cpu_baseline": cpu, "parity_in_bench": parity}
    print(json.dumps(line), flush=True)
    if parity is not None and parity["mismatch"]:
        sys.exit(3)


SEQPROF_SEED = 160306958 + 50


def main():
    args = parse_args()
    if args.workload == "seqprof":
        run_seqprof(args, int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("LOCAL_RANK", "0")))
        return
    if args.kernel_only:
        args.no_cpu = args.no_full = args.no_guide_tree = True
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    run_cuda(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
