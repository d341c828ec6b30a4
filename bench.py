#!/usr/bin/env python
"""bench.py -- throughput of the SubQuad candidate-pair affinity path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload configX] [--impl reference]

A step = one pass of the whole hot path over one synthetic repertoire:
    sq_pack -> sq_minhash -> sq_lsh_candidates (sorted) -> sq_edit_distance
with the inputs resident in HBM (`value`), and the same through sq_pipeline_host with pinned
HOST buffers, copies inside the timed region (`e2e`).  Prints ONE JSON line (rank 0).
Multi-GPU: the path partitions into independent repertoires (donors), one per rank, no
data-path collective ("scaling": "weak").  `--impl reference` times the CPU oracle.
"""
import argparse
import hashlib
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
TRAFFIC_JSON = os.path.join(ROOT, "profiles", "traffic.json")

from paper_2602_17330_b200 import datagen as dg  # noqa: E402
from paper_2602_17330_b200 import shard  # noqa: E402

METRIC = "candidate_pairs_verified_per_s"
UNIT = "pairs/s"
ALU_OPS_PER_COLUMN_WORD = 7         # ALU-pipe logic ops of one Myers/Hyyro column step
SAD_OPS_PER_FILTER_CELL = 5         # byte-wise SAD instructions per cell of the bag filter (20 residues)
# dram bytes per launch of the dominant kernel come from the committed `ncu --set full` summary
# profiles/traffic.json, which names the sha256 of the kernel sources it was captured on: a build
# from other sources reports "traffic": null instead of a stale number
# bounded oracle samples: whole clonal families (so that candidates per sequence stay those of the full
# workload), about this many sequences
ORACLE_SAMPLE = {"config1": 2000, "config2": 100_000, "config3": 150_000, "config4": 60_000, "config5": 2000}
CAP_PER_SEQ = {"config2": 40, "config3": 60, "config4": 200}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default=os.environ.get("SQ_BENCH_WORKLOAD", "config4"),
                    choices=["config1", "config2", "config3", "config4", "config5"])
    ap.add_argument("--n", type=int, default=0, help="override the number of sequences")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def kernel_source_sha():
    """sha256 over the CUDA sources of libsubquad.so (what an ncu capture is valid for)"""
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2602_17330_b200", "csrc")
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            with open(os.path.join(d, name), "rb") as f:
                h.update(name.encode() + b"\0" + f.read())
    return h.hexdigest()


def captured_traffic(workload, n, kernel_class):
    """(bytes per launch, source) from profiles/traffic.json if it was captured on these very
    kernel sources for this workload and kernel class, else (None, why)."""
    try:
        with open(TRAFFIC_JSON) as f:
            t = json.load(f)
    except Exception:
        return None, "no profiles/traffic.json"
    if t.get("kernel_source_sha256") != kernel_source_sha():
        return None, "profiles/traffic.json was captured on other kernel sources"
    for e in t.get("entries", []):
        if e.get("workload") == workload and e.get("n") == n and e.get("kernel_class") == kernel_class:
            return float(e["dram_bytes_per_launch"]), e.get("capture", "profiles/traffic.json")
    return None, "no entry for this workload / kernel in profiles/traffic.json"


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except Exception:
        pass
    return "unknown"


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start the N ranks ourselves (one process per
    GPU, torch.distributed.run on this node) and hand their output through."""
    import socket
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms.  The process is started BEFORE
    the warm-up (its start-up stalls the GPU for a while) and only the samples stamped inside
    the timed region [mark(), stop()] are kept."""
    Q = ("timestamp,clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.t_mark = None

    def mark(self):
        import datetime
        self.t_mark = datetime.datetime.now()

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        import datetime
        t_end = datetime.datetime.now()
        time.sleep(0.15)
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            out = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        margin = datetime.timedelta(milliseconds=120)
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                ts = datetime.datetime.strptime(f[0], "%Y/%m/%d %H:%M:%S.%f")
                if self.t_mark is not None and not (self.t_mark - margin <= ts <= t_end + margin):
                    continue
                f = f[1:]
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def make_repertoire(workload, n, rank):
    gen = dg.GENERATORS[workload]
    rep = gen(n, seed=rank) if n else gen(seed=rank)
    return rep


# ---------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------
def oracle_step(rep_sample, P, threads=None):
    """one pass of the oracle over a repertoire: (pairs, seconds per stage, cells)"""
    import oracle
    if threads is not None:
        oracle.set_num_threads(threads)
    t0 = time.perf_counter()
    sig = oracle.minhash(rep_sample.seqs, rep_sample.offsets, P["k"], P["H"], dg.DEFAULT_SEED64)
    t1 = time.perf_counter()
    pairs, raw, _ = oracle.lsh_sorted(sig, P["bands"], P["rows"], P["cap"])
    t2 = time.perf_counter()
    dist = oracle.edit_distance_pairs(rep_sample.seqs, rep_sample.offsets, pairs, P["max_d"])
    t3 = time.perf_counter()
    L = rep_sample.lengths
    cells = float((L[pairs[:, 0]].astype(np.float64) * L[pairs[:, 1]]).sum()) if pairs.size else 0.0
    return {"pairs": int(pairs.shape[0]), "raw": int(raw), "t": t3 - t0, "t_minhash": t1 - t0, "t_lsh": t2 - t1,
            "t_edit": t3 - t2, "cells": cells, "hits": int((dist <= P["max_d"]).sum()), "pair_list": pairs}


def subset(rep, idx):
    """the sequences `idx` (ascending) of a repertoire, as a repertoire of their own"""
    lens = rep.lengths[idx]
    offs = np.zeros(idx.size + 1, np.int64)
    np.cumsum(lens, out=offs[1:])
    src = np.repeat(rep.offsets[idx] - offs[:-1], lens) + np.arange(int(offs[-1]), dtype=np.int64)
    return dg.Repertoire(rep.seqs[src], offs, rep.family[idx], rep.n_edits[idx], rep.name)


def sample_of(rep, n_s):
    """About n_s sequences: WHOLE clonal families (family ids 0, 1, ... in the generator's order, every
    member wherever the final permutation put it), so that the sample has the candidate density of
    the full workload; a plain prefix when the repertoire has no families."""
    n_s = min(n_s, rep.n)
    if rep.n == n_s or rep.family.size == 0 or int(rep.family.min()) < 0:
        return subset(rep, np.arange(n_s)), f"first {n_s} sequences"
    sizes = np.bincount(rep.family)
    nf = int(np.searchsorted(np.cumsum(sizes), n_s)) + 1
    idx = np.nonzero(rep.family < nf)[0]
    return subset(rep, idx), f"all {idx.size} members of the first {nf} clonal families"


def cpu_baseline(rep, workload, P):
    """The oracle as it stands on this box's host cores, on a bounded sample of the same workload:
    all cores (OpenMP over independent items; the sort of the LSH stage is single-threaded) and one
    core.  A reported baseline, not a target."""
    import oracle
    cores = oracle.num_threads()
    s, what = sample_of(rep, ORACLE_SAMPLE[workload])
    r = oracle_step(s, P)
    pl = r.pop("pair_list")
    # one thread: the two parallel stages again (the LSH stage is single-threaded anyway)
    oracle.set_num_threads(1)
    t0 = time.perf_counter()
    oracle.minhash(s.seqs, s.offsets, P["k"], P["H"], dg.DEFAULT_SEED64)
    t1 = time.perf_counter()
    oracle.edit_distance_pairs(s.seqs, s.offsets, pl, P["max_d"])
    t2 = time.perf_counter()
    oracle.set_num_threads(cores)
    t_single = (t1 - t0) + r["t_lsh"] + (t2 - t1)
    return {"value": r["pairs"] / r["t"], "unit": UNIT, "cores": cores, "kind": "oracle",
            "cpu_model": cpu_model(),
            "sample": f"{what} of {workload} (of {rep.n}); {r['pairs']} candidate pairs "
                      f"({r['pairs'] / max(s.n, 1):.1f} per sequence, {r['raw']} before dedupe) in {r['t']:.2f} s "
                      f"(minhash {r['t_minhash']:.2f} s, lsh {r['t_lsh']:.2f} s single-thread qsort, "
                      f"edit {r['t_edit']:.2f} s)",
            "minhash_seqs_per_s": s.n / max(r["t_minhash"], 1e-9),
            "lsh_candidate_pairs_per_s": r["pairs"] / max(r["t_lsh"], 1e-9),
            "edit_gcups": r["cells"] / max(r["t_edit"], 1e-9) / 1e9,
            "single_thread": {"value": r["pairs"] / t_single, "unit": UNIT,
                              "minhash_seqs_per_s": s.n / max(t1 - t0, 1e-9),
                              "edit_gcups": r["cells"] / max(t2 - t1, 1e-9) / 1e9}}


def all_pairs_oracle(rep, P):
    """oracle on the all-pairs block of the first 2,000 sequences: seconds, pairs, cells"""
    import oracle
    s, what = sample_of(rep, ORACLE_SAMPLE["config1"])
    L = s.lengths.astype(np.float64)
    cells = (L.sum() ** 2 - (L ** 2).sum()) / 2
    npairs = s.n * (s.n - 1) // 2
    t0 = time.perf_counter()
    if P["max_d"] < 0:
        oracle.all_pairs_full(s.seqs, s.offsets)
    else:
        oracle.all_pairs_threshold(s.seqs, s.offsets, P["max_d"], use_cutoff=False)
    return time.perf_counter() - t0, npairs, cells, s, what


def cpu_baseline_all_pairs(rep, workload, P):
    import oracle
    cores = oracle.num_threads()
    t, npairs, cells, s, what = all_pairs_oracle(rep, P)
    oracle.set_num_threads(1)
    sub1 = subset(s, np.arange(min(s.n, 500)))
    t1, np1, cells1, _, _ = all_pairs_oracle(sub1, P)
    oracle.set_num_threads(cores)
    return {"value": npairs / t, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
            "sample": f"all-pairs block of the {what} of {workload} (of {rep.n}): {npairs} pairs, plain "
                      f"Wagner-Fischer, in {t:.2f} s",
            "gcups": cells / t / 1e9,
            "single_thread": {"value": np1 / t1, "unit": UNIT, "gcups": cells1 / t1 / 1e9,
                              "sample": f"first {sub1.n} sequences"}}


def run_reference(args):
    """--impl reference: there is no reference implementation (PAPER.md only); the base contract's
    reference arm is the oracle, as it stands, on the host cores, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    world = int(os.environ.get("WORLD_SIZE", "1"))
    workload = args.workload
    P = dg.PARAMS[workload]
    cores = oracle.num_threads()
    if workload in ("config1", "config5"):
        rep = dg.GENERATORS[workload](ORACLE_SAMPLE[workload], seed=0)
        for _ in range(min(args.warmup, 1)):
            all_pairs_oracle(rep, P)
        ts = []
        for _ in range(args.steps):
            t, npairs, cells, s, what = all_pairs_oracle(rep, P)
            ts.append(t)
        t = sum(ts)
        value = npairs * args.steps / t
        metric = "all_pairs_evaluated_per_s"
        sample = f"{workload} generator at n={rep.n}: {npairs} pairs per step, plain Wagner-Fischer"
        cfg = {"workload": f"{workload} generator at n={rep.n} (bounded oracle sample)", "max_d": P["max_d"]}
    else:
        n_s = min(ORACLE_SAMPLE[workload], 60_000)
        rep = dg.GENERATORS[workload](n_s, seed=0)
        for _ in range(min(args.warmup, 1)):
            oracle_step(rep, P)
        ts, pairs = [], 0
        for _ in range(args.steps):
            r = oracle_step(rep, P)
            ts.append(r["t"]); pairs = r["pairs"]
        t = sum(ts)
        value = pairs * args.steps / t
        metric = METRIC
        sample = f"{workload} generator at n={n_s}, {pairs} pairs per step"
        cfg = {"workload": f"{workload} generator at n={n_s} (bounded oracle sample)",
               **{k: P[k] for k in ("k", "H", "bands", "rows", "cap", "max_d")}}
    line = {
        "impl": "reference", "metric": metric, "value": value, "unit": UNIT, "n_gpus": world,
        "ranks_that_computed": 1, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32/u64 integer",
        "data": "synthetic", "gpu_launches": 0, "config": cfg,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "cpu_model": cpu_model(),
                         "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


# ---------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------
def time_cross_join(binding, dev, flush):
    """sq_join (device output) and sq_join_host (blocks streamed to pinned host memory) on two
    synthetic repertoires; outside the timed step, reported beside it."""
    import torch
    a, b = dg.split(dg.config3(1_000_000, seed=0), 100_000)
    max_len = int(max(a.lengths.max(), b.lengths.max()))
    cap, block_cap, max_d = 60_000_000, 8_000_000, 2
    ctx = []
    for rep, other in ((a, b), (b, a)):
        sq = binding.SubQuad(dev.index or 0)
        sq.set_workspace(sq.workspace_bytes(binding.OP_JOIN, rep.n, int(rep.offsets[-1]), max_len,
                                            pair_capacity=cap if rep is a else 1, n_other=other.n))
        sq.pack(torch.from_numpy(rep.seqs).to(dev), torch.from_numpy(rep.offsets).to(dev), alphabet=20,
                max_len=max_len)
        ctx.append(sq)
    sa, sb = ctx
    pairs = torch.empty((cap, 2), dtype=torch.int32, device=dev)
    dist = torch.empty(cap, dtype=torch.int16, device=dev)
    hits = sa.join(sb, max_d, pairs, dist)
    ph = torch.empty((hits + 16, 2), dtype=torch.int32).pin_memory()
    dh = torch.empty(hits + 16, dtype=torch.int16).pin_memory()
    batch_rows = 16384
    sa.join_host(sb, max_d, ph, dh, block_capacity=block_cap, batch_rows=batch_rows)
    t_dev, t_host = [], []
    for _ in range(3):
        flush.fill_(1); torch.cuda.synchronize()
        t0 = time.perf_counter(); sa.join(sb, max_d, pairs, dist); t_dev.append(time.perf_counter() - t0)
        flush.fill_(1); torch.cuda.synchronize()
        t0 = time.perf_counter()
        h2 = sa.join_host(sb, max_d, ph, dh, block_capacity=block_cap, batch_rows=batch_rows)
        t_host.append(time.perf_counter() - t0)
    assert h2 == hits
    sa.profile_enable(True); sa.profile_reset()
    sa.join(sb, max_d, pairs, dist)
    prof = {k: round(v[0], 3) for k, v in sa.profile_read().items() if v[1]}
    sa.profile_enable(False)
    cells = a.n * b.n
    td, th = sum(t_dev) / 3, sum(t_host) / 3
    out = {"workload": "config3 recipe split 100,000 x 900,000, max_d=2", "cells": cells, "hits": int(hits),
           "join_ms": td * 1e3, "cells_per_s": cells / td,
           "join_host_ms": th * 1e3, "join_host_cells_per_s": cells / th,
           "block_capacity": block_cap, "batch_rows": batch_rows, "d2h_bytes": int(hits) * 10, "kernel_ms": prof,
           "timing": "host clock around the synchronising call (sq_join / sq_join_host), 3 runs"}
    sa.close(); sb.close()
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2602_17330_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    workload = args.workload
    P = dg.PARAMS[workload]
    rep = make_repertoire(workload, args.n, shard.rank_seed(rank))   # one independent repertoire per rank
    n = rep.n
    total_len = int(rep.offsets[-1])
    max_len = int(rep.lengths.max())
    sq = binding.SubQuad(local_rank)
    stride = (max_len + 1 + 15) // 16 * 16

    seqs_h = torch.from_numpy(rep.seqs).pin_memory()
    offs_h = torch.from_numpy(rep.offsets).pin_memory()
    seqs_d = seqs_h.to(dev, non_blocking=True)
    offs_d = offs_h.to(dev, non_blocking=True)
    sig = torch.empty((n, P["H"]), dtype=torch.int32, device=dev)

    # capacity: start from an estimate, grow on SQ_ERR_CAPACITY (untimed)
    capacity = int(CAP_PER_SEQ[workload] * n)
    pairs = dist_out = None

    def alloc(cap):
        nonlocal pairs, dist_out
        pairs = dist_out = None
        torch.cuda.empty_cache()
        ws = max(sq.workspace_bytes(binding.OP_LSH, n, total_len, max_len, P["H"], P["bands"],
                                    P["cap"], cap),
                 0 if args.no_e2e else sq.workspace_bytes(binding.OP_PIPELINE_HOST, n, total_len,
                                                          max_len, P["H"], P["bands"], P["cap"], cap))
        ws += 4 * cap + 8 * n + (1 << 20)      # room for the graph step's scratch above the LSH scratch
        sq.workspace = None
        sq.set_workspace(ws)
        pairs = torch.empty((cap, 2), dtype=torch.int32, device=dev)
        dist_out = torch.empty(cap, dtype=torch.int16, device=dev)

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step(timed):
        """one pass of the whole path; returns (count, [t_pack, t_minhash, t_lsh, t_edit] ms)"""
        e = [ev() for _ in range(5)]
        e[0].record()
        sq.pack(seqs_d, offs_d, 20, max_len)
        e[1].record()
        sq.minhash(P["k"], P["H"], dg.DEFAULT_SEED64, sig)
        e[2].record()
        cnt = sq.lsh_candidates(sig, P["bands"], P["rows"], P["cap"], pairs)
        e[3].record()
        sq.edit_distance(pairs, cnt, P["max_d"], dist_out)
        e[4].record()
        e[4].synchronize()
        return cnt, [e[i].elapsed_time(e[i + 1]) for i in range(4)]

    alloc(capacity)
    while True:
        try:
            cnt, _ = step(False)
            break
        except binding.SubQuadError as ex:
            if ex.code != binding.SQ_ERR_CAPACITY:
                raise
            capacity = int(ex.required * 1.02) + 1024
            alloc(capacity)
    raw = sq.last_raw_pairs()

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(1.0)                        # let nvidia-smi finish its start-up outside the timing
    for _ in range(max(0, args.warmup - 1)):
        step(False)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler.mark()
    sq.profile_enable(True)
    sq.profile_reset()
    launches0 = sq.kernel_launches()
    t_steps, stages = [], []
    wall0 = time.perf_counter()
    for _ in range(args.steps):
        flush.fill_(1)                     # L2 flush between timed iterations (outside the events)
        torch.cuda.synchronize()
        c2, st = step(True)
        assert c2 == cnt
        t_steps.append(sum(st)); stages.append(st)
    torch.cuda.synchronize()
    wall = time.perf_counter() - wall0
    prof = sq.profile_read()
    sq.profile_enable(False)
    launches = sq.kernel_launches() - launches0
    clocks = sampler.stop()
    if world > 1:
        dist.barrier()

    step_ms = sum(t_steps) / args.steps
    st_ms = [sum(s[i] for s in stages) / args.steps for i in range(4)]
    # work units of this rank
    lens = torch.from_numpy(rep.lengths.astype(np.int32)).to(dev)
    pi = pairs[:cnt, 0].long(); pj = pairs[:cnt, 1].long()
    cells = float((lens[pi].double() * lens[pj].double()).sum().item())
    text_cols = float(lens[pj].double().sum().item())
    hits = int((dist_out[:cnt] <= P["max_d"]).sum().item())
    del pi, pj

    # aggregate over ranks: units summed, time = max over ranks (paper_2602_17330_b200/shard.py)
    step_ms_all, tot = shard.aggregate(step_ms, {"pairs": cnt, "seqs": n, "cells": cells}, dev)
    cnt_all, n_all, cells_all = tot["pairs"], tot["seqs"], tot["cells"]

    # ---- next-1: weighted edit distance on the same candidates, timed beside the path
    weighted = None
    try:
        sub_d = torch.from_numpy(dg.class_substitution_costs()).to(dev)
        wd = torch.empty_like(dist_out)
        sq.edit_distance_weighted(pairs, cnt, sub_d, 1, 2 * P["max_d"], wd)
        torch.cuda.synchronize()
        tw_ms = []
        for _ in range(3):
            flush.fill_(1); torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record(); sq.edit_distance_weighted(pairs, cnt, sub_d, 1, 2 * P["max_d"], wd); b.record()
            b.synchronize(); tw_ms.append(a.elapsed_time(b))
        tw = sum(tw_ms) / len(tw_ms)
        weighted = {"ms": tw, "pairs_per_s": cnt / (tw * 1e-3), "gcups": cells / (tw * 1e-3) / 1e9,
                    "table": "class costs 0/1/2, indel 1, max_d %d" % (2 * P["max_d"]),
                    "hits": int((wd[:cnt] <= 2 * P["max_d"]).sum().item())}
        del wd
    except Exception as ex:
        weighted = {"error": repr(ex)[:200]}

    # ---- next-2: sparse similarity graph from the verified candidates, tau = 0.7
    graph = None
    try:
        mm = int(np.ceil(0.7 * P["H"]))
        row_ptr = torch.empty(n + 1, dtype=torch.int64, device=dev)
        col = torch.empty(cnt, dtype=torch.int32, device=dev)
        wgt = torch.empty(cnt, dtype=torch.float32, device=dev)
        edges = sq.affinity_graph(pairs, dist_out, cnt, P["max_d"], sig, mm, row_ptr, col, wgt)
        tg_ms = []
        for _ in range(2):
            flush.fill_(1); torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record(); sq.affinity_graph(pairs, dist_out, cnt, P["max_d"], sig, mm, row_ptr, col, wgt); b.record()
            b.synchronize(); tg_ms.append(a.elapsed_time(b))
        tg = sum(tg_ms) / len(tg_ms)
        graph = {"ms": tg, "edges": int(edges), "min_matches": mm, "pairs_per_s": cnt / (tg * 1e-3),
                 "GBs_algorithmic": (cnt * (10 + 8 * P["H"]) + edges * 8 + 8 * n) / (tg * 1e-3) / 1e9}
        del row_ptr, col, wgt
    except Exception as ex:
        graph = {"error": repr(ex)[:200]}

    # ---- next-3/4: cross-repertoire join, 100,000 x 900,000 CDR3s (config-3 recipe
    # split in two, the 1 M multi-donor pool shape of PAPER.md L647), max_d = 2
    join = None
    if rank == 0 and not args.no_e2e and workload == "config4":
        try:
            join = time_cross_join(binding, dev, flush)
        except Exception as ex:
            join = {"error": repr(ex)[:200]}

    # ---- e2e: through the C ABI with HOST buffers -------------------------------------------
    # headline: sq_pipeline_host_csr (row offsets + partner + byte distance: 5 B per candidate over
    # PCIe); beside it the pair-list form sq_pipeline_host (10 B per candidate)
    e2e, e2e_pairs = None, None
    if not args.no_e2e:
        e2e_steps = max(1, min(args.steps, 3))

        def time_host_api(call):
            call()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                c3 = call()
            torch.cuda.synchronize()
            t = (time.perf_counter() - t0) / e2e_steps
            assert c3 == cnt
            t_ms, _ = shard.aggregate(1e3 * t, {}, dev)
            return t_ms * 1e-3
        try:
            row_ptr_h = torch.empty(n + 1, dtype=torch.int64).pin_memory()
            col_h = torch.empty(capacity, dtype=torch.int32).pin_memory()
            d8_h = torch.empty(capacity, dtype=torch.uint8).pin_memory()
            te = time_host_api(lambda: sq.pipeline_host_csr(
                seqs_h, offs_h, 20, max_len, P["k"], P["H"], dg.DEFAULT_SEED64, P["bands"], P["rows"],
                P["cap"], P["max_d"], row_ptr_h, col_h, d8_h))
            e2e = {"value": cnt_all / te, "unit": UNIT,
                   "h2d_bytes_per_step": total_len + 8 * (n + 1),
                   "d2h_bytes_per_step": 5 * cnt + 8 * (n + 1), "ms_per_step": 1e3 * te,
                   "steps": e2e_steps,
                   "api": "sq_pipeline_host_csr (pinned host buffers; row_ptr int64, col uint32, dist uint8)"}
            del row_ptr_h, col_h, d8_h
        except Exception as ex:               # e.g. not enough pinned host memory
            e2e = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}
        try:
            pairs_h = torch.empty((capacity, 2), dtype=torch.int32).pin_memory()
            dist_h = torch.empty(capacity, dtype=torch.int16).pin_memory()
            te = time_host_api(lambda: sq.pipeline_host(
                seqs_h, offs_h, 20, max_len, P["k"], P["H"], dg.DEFAULT_SEED64, P["bands"], P["rows"],
                P["cap"], P["max_d"], pairs_h, dist_h))
            e2e_pairs = {"value": cnt_all / te, "unit": UNIT,
                         "h2d_bytes_per_step": total_len + 8 * (n + 1),
                         "d2h_bytes_per_step": 10 * cnt, "ms_per_step": 1e3 * te, "steps": e2e_steps,
                         "api": "sq_pipeline_host (pinned host buffers; pairs uint32[.][2], dist uint16)"}
            del pairs_h, dist_h
        except Exception as ex:
            e2e_pairs = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}

    if rank != 0:
        return
    # ---- rooflines ---------------------------------------------------------------------------
    hbm_peak, peak_src = measured_peaks()
    int_peak = {name: sq.int_peak(kind, 2048) for kind, name in
                ((0, "lop3"), (1, "iadd"), (3, "imad"), (4, "umin"), (5, "lop3+imad"),
                 (8, "lop3+imad_fresh_operands"), (9, "dp_column_mix_7lop3_4imad"))}
    # LOP3 share of the DP column's own instruction mix: the ceiling the register file sets
    int_peak["lop3_inside_dp_column_mix"] = int_peak["dp_column_mix_7lop3_4imad"] * 7.0 / 11.0
    # the product's own column chain alone (shared-memory resident, no global memory), as LOP3 per second
    int_peak["lop3_dp_chain_alone"] = sq.dp_chain_peak(20, 2000) * ALU_OPS_PER_COLUMN_WORD
    B = P["bands"]
    K = args.steps
    rec = n * B                                    # (sequence, band) records
    sw = 4 * (1 if B <= 4 else 2 if B <= 8 else 4 if B <= 16 else 8)   # S row width (words)
    alg_bytes = {   # algorithmic bytes per STEP of each kernel class
        "pack": total_len + 8 * (n + 1) + n * stride + 12 * n,
        "minhash": n * (stride + 4 + 4 * P["H"]),
        "band_key": n * (4 * P["H"] + 12 * B + 4),
        "sort_hist": 8 * (rec + n),                # keys read once for all digit histograms
        "sort_scatter": 24 * (4 * rec + n),        # read + write (key 8 B, id 4 B) per pass, 4 passes
        "scan": 12 * (rec + 4 * n),                # counts -> offsets; per-sequence scans
        "bucket_scan": rec * (8 + 4 + 4) + rec * 12 + 8 * n + 8 * rec,   # keys + ids in, S out; id -> internal row; mixed-run detection
        "emit": rec * (4 + 4 * sw) + 8 * rec + 4 * cnt,        # ids + S rows; counts out, offsets in; partners out
        "row_sort": 4 * cnt + 4 * rec + 8 * cnt + 16 * (cnt // 32) + 12 * n,   # partners + offsets in, pairs out,
                                                                              # chunk schedule of the DP stage out
    }
    kernels = {}
    tot_prof = sum(ms for ms, _ in prof.values()) or 1.0
    for name, (ms, ln) in prof.items():
        if ln == 0:
            continue
        k = {"ms_per_step": ms / K, "launches_per_step": ln / K, "share": ms / tot_prof}
        if name in alg_bytes:
            k["bound"] = "hbm"
            k["achieved_GBs"] = alg_bytes[name] / (ms / K * 1e-3) / 1e9
            k["frac"] = k["achieved_GBs"] / hbm_peak
        if name == "edit_distance":
            ops = ALU_OPS_PER_COLUMN_WORD * text_cols * ((max_len + 31) // 32)
            k["bound"] = "alu"
            k["achieved_Gops"] = ops / (ms / K * 1e-3) / 1e9
            k["frac"] = k["achieved_Gops"] * 1e9 / int_peak["lop3"]
            k["frac_of_lop3_inside_dp_column_mix"] = k["achieved_Gops"] * 1e9 / int_peak["lop3_inside_dp_column_mix"]
            k["frac_of_dp_chain_alone"] = k["achieved_Gops"] * 1e9 / int_peak["lop3_dp_chain_alone"]
        if name == "minhash":
            L = rep.lengths
            upd = float(np.maximum(L - P["k"] + 1, 0).sum()) * P["H"]
            k["alu_Gupdates_per_s"] = upd / (ms / K * 1e-3) / 1e9
            k["alu_frac_of_imad_peak"] = upd / (ms / K * 1e-3) / int_peak["imad"]
        kernels[name] = k
    dom = max(kernels, key=lambda q: kernels[q]["ms_per_step"])
    kd = kernels[dom]
    if kd.get("bound") == "alu":
        roof = {"kernel": dom, "bound": "alu", "achieved": kd["achieved_Gops"],
                "peak": int_peak["lop3"] / 1e9, "unit": "Gop/s", "frac": kd["frac"], "traffic": None,
                "peak_source": "sq_int_peak LOP3 stream measured in this run"}
    else:
        roof = {"kernel": dom, "bound": "hbm", "achieved": kd.get("achieved_GBs"), "peak": hbm_peak,
                "unit": "GB/s", "frac": kd.get("frac"), "traffic": None, "peak_source": peak_src}
    roof["avg_launch_ms"] = kd["ms_per_step"] / max(kd["launches_per_step"], 1)
    roof["traffic"], roof["traffic_source"] = captured_traffic(workload, n, dom)

    cpu = None if args.no_cpu_baseline else cpu_baseline(rep, workload, P)
    line = {
        "metric": METRIC, "value": cnt_all / (step_ms_all * 1e-3), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms_all,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32/u64 integer", "data": "synthetic",
        "config": {"workload": f"{workload}: N={n} CDR3-like sequences per GPU "
                               f"(BASELINE.json configs[{int(workload[-1]) - 1}])",
                   **{k: P[k] for k in ("k", "H", "bands", "rows", "cap", "max_d")},
                   "candidate_pairs": cnt, "raw_pairs_before_dedupe": raw, "hits": hits,
                   "timing": "CUDA events per step on the library's stream; 256 MB L2 flush "
                             "between timed steps (outside the events); parallelism: one "
                             "independent repertoire per GPU, no collective"},
        "stages": {"pack_ms": st_ms[0], "minhash_ms": st_ms[1], "lsh_ms": st_ms[2],
                   "edit_ms": st_ms[3],
                   "minhash_seqs_per_s": n / (st_ms[1] * 1e-3),
                   "lsh_candidate_pairs_per_s": cnt / (st_ms[2] * 1e-3),
                   "lsh_raw_pairs_per_s": raw / (st_ms[2] * 1e-3),
                   "edit_pairs_per_s": cnt / (st_ms[3] * 1e-3),
                   "edit_gcups": cells / (st_ms[3] * 1e-3) / 1e9,
                   "wall_s_timed_region": wall},
        "weighted_edit_distance": weighted, "affinity_graph": graph, "cross_join": join,
        "roofline": roof, "kernels": kernels, "int_peak_ops_per_s": int_peak,
        "cpu_baseline": cpu, "e2e": e2e, "e2e_pair_list": e2e_pairs, "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line))


def run_all_pairs(args):
    """configs 1 and 5: the exhaustive tile path (sq_pack + sq_all_pairs), one line, same contract.
    value = pairs i<j evaluated per second; stages carry GCUPS (full-matrix-equivalent cells)."""
    import torch
    from paper_2602_17330_b200 import binding
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    workload = args.workload
    P = dg.PARAMS[workload]
    rep = make_repertoire(workload, args.n, shard.rank_seed(rank))
    n, max_len, total_len = rep.n, int(rep.lengths.max()), int(rep.offsets[-1])
    npairs = n * (n - 1) // 2
    cap = npairs if P["max_d"] < 0 else 8_000_000
    sq = binding.SubQuad(local_rank)
    sq.set_workspace(sq.workspace_bytes(binding.OP_ALL_PAIRS, n, total_len, max_len, 0, 1, 0, cap))
    seqs_d = torch.from_numpy(rep.seqs).to(dev)
    offs_d = torch.from_numpy(rep.offsets).to(dev)
    pairs = torch.empty((cap, 2), dtype=torch.int32, device=dev) if P["max_d"] >= 0 else None
    dist_out = torch.empty(cap, dtype=torch.int16, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def step():
        e0, e1 = ev(), ev()
        e0.record()
        sq.pack(seqs_d, offs_d, 20, max_len)
        c = sq.all_pairs(P["max_d"], pairs, dist_out)
        e1.record(); e1.synchronize()
        return c, e0.elapsed_time(e1)

    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(1.0)
    for _ in range(args.warmup):
        cnt, _ = step()
    torch.cuda.synchronize()
    sampler.mark()
    sq.profile_enable(True); sq.profile_reset()
    l0 = sq.kernel_launches()
    ts = []
    for _ in range(args.steps):
        flush.fill_(1); torch.cuda.synchronize()
        c2, t = step()
        assert c2 == cnt
        ts.append(t)
    prof = sq.profile_read(); sq.profile_enable(False)
    launches = sq.kernel_launches() - l0
    clocks = sampler.stop()
    step_ms = sum(ts) / len(ts)
    L = rep.lengths.astype(np.float64)
    cells = (L.sum() ** 2 - (L ** 2).sum()) / 2
    step_ms_all, tot = shard.aggregate(step_ms, {"pairs": npairs, "cells": cells}, dev)
    survivors = sq.last_raw_pairs() if P["max_d"] >= 0 else npairs

    # ---- e2e: the same through HOST buffers (pinned): H2D of sequences + offsets, pack, all pairs,
    # D2H of the results, all inside the timed region
    e2e = None
    if not args.no_e2e:
        seqs_h = torch.from_numpy(rep.seqs).pin_memory()
        offs_h = torch.from_numpy(rep.offsets).pin_memory()
        n_out = int(cnt)
        dist_h = torch.empty(max(n_out, 1), dtype=torch.int16).pin_memory()
        pairs_h = torch.empty((max(n_out, 1), 2), dtype=torch.int32).pin_memory() if pairs is not None else None

        def host_step():
            sd = seqs_h.to(dev, non_blocking=True)
            od = offs_h.to(dev, non_blocking=True)
            sq.pack(sd, od, 20, max_len)
            c = sq.all_pairs(P["max_d"], pairs, dist_out)
            dist_h[:c].copy_(dist_out[:c], non_blocking=True)
            if pairs_h is not None:
                pairs_h[:c].copy_(pairs[:c], non_blocking=True)
            torch.cuda.synchronize()
            return c
        host_step()
        e2e_steps = max(1, min(args.steps, 5))
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            c3 = host_step()
        te = (time.perf_counter() - t0) / e2e_steps
        assert c3 == cnt
        te_ms, _ = shard.aggregate(1e3 * te, {}, dev)
        e2e = {"value": tot["pairs"] / (te_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": total_len + 8 * (n + 1),
               "d2h_bytes_per_step": n_out * (2 if pairs_h is None else 10), "ms_per_step": te_ms,
               "steps": e2e_steps,
               "api": "pinned host tensors -> sq_pack -> sq_all_pairs -> pinned host tensors (copies timed)"}
    if rank != 0:
        return
    K = args.steps
    words = (max_len + 31) // 32
    lop3 = sq.int_peak(0, 2048)
    sad = sq.int_peak(7, 2048)
    kernels = {k: {"ms_per_step": ms / K, "launches_per_step": ln / K} for k, (ms, ln) in prof.items() if ln}
    Ls = rep.lengths.astype(np.float64)
    if P["max_d"] < 0:
        # fused tile kernel: every pair i < j runs every column of its text j (the row i is the pattern)
        text_cols = float((Ls * np.arange(n)).sum())            # sequence j is the text of j pairs
        k = kernels["all_pairs"]
        ops = ALU_OPS_PER_COLUMN_WORD * text_cols * words
        k.update(bound="alu", achieved_Gops=ops / (k["ms_per_step"] * 1e-3) / 1e9)
        k["frac"] = k["achieved_Gops"] * 1e9 / lop3
        roof = {"kernel": "all_pairs", "bound": "alu", "achieved": k["achieved_Gops"], "peak": lop3 / 1e9,
                "unit": "Gop/s", "frac": k["frac"], "peak_source": "sq_int_peak LOP3 stream measured in this run",
                "ops": f"{ALU_OPS_PER_COLUMN_WORD} logic ops x text columns x {words} word(s) per pair (DESIGN.md 5)"}
        cells_computed = cells
    else:
        # two kernels: the bag-distance filter over all cells (SAD instructions) and the banded DP on
        # its survivors (window of NWIN words per column)
        nwin = 2 if P["max_d"] <= 16 else 3
        kf = kernels["all_pairs"]
        f_ops = SAD_OPS_PER_FILTER_CELL * float(npairs)
        kf.update(bound="alu", achieved_Gops=f_ops / (kf["ms_per_step"] * 1e-3) / 1e9)
        kf["frac"] = kf["achieved_Gops"] * 1e9 / sad
        kf["peak"] = "sq_int_peak vabsdiff4 stream (%.0f Gop/s)" % (sad / 1e9)
        mean_len = float(Ls.mean())
        cells_computed = survivors * mean_len * 32.0 * nwin        # band cells of the survivors' DP
        if "edit_distance" in kernels:
            kd = kernels["edit_distance"]
            d_ops = ALU_OPS_PER_COLUMN_WORD * survivors * mean_len * nwin
            kd.update(bound="alu", achieved_Gops=d_ops / (kd["ms_per_step"] * 1e-3) / 1e9,
                      columns="survivors x mean text length (the survivor list is not returned)")
            kd["frac"] = kd["achieved_Gops"] * 1e9 / lop3
        roof = {"kernel": "all_pairs (bag-distance filter)", "bound": "alu", "achieved": kf["achieved_Gops"],
                "peak": sad / 1e9, "unit": "Gop/s", "frac": kf["frac"],
                "peak_source": "sq_int_peak vabsdiff4 stream measured in this run",
                "ops": f"{SAD_OPS_PER_FILTER_CELL} byte-wise SAD instructions per cell i<j (DESIGN.md 5)"}
    dom = max(kernels, key=lambda q: kernels[q]["ms_per_step"])
    roof["avg_launch_ms"] = kernels["all_pairs"]["ms_per_step"] / max(kernels["all_pairs"]["launches_per_step"], 1)
    roof["traffic"], roof["traffic_source"] = captured_traffic(workload, n, "all_pairs")
    cpu = None if args.no_cpu_baseline else cpu_baseline_all_pairs(rep, workload, P)
    line = {
        "metric": "all_pairs_evaluated_per_s", "value": tot["pairs"] / (step_ms_all * 1e-3), "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": step_ms_all,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32 integer",
        "data": "synthetic",
        "config": {"workload": f"{workload}: exhaustive tile path over N={n} sequences "
                               f"(BASELINE.json configs[{int(workload[-1]) - 1}])",
                   "max_d": P["max_d"], "max_len": max_len, "outputs": int(cnt),
                   "filter_survivors": int(survivors),
                   "timing": "CUDA events per step; 256 MB L2 flush between timed steps"},
        "stages": {"gcups_full_matrix_equivalent": tot["cells"] / (step_ms_all * 1e-3) / 1e9,
                   "gcups_cells_actually_computed": cells_computed / (step_ms * 1e-3) / 1e9,
                   "cells_full_matrix": cells, "cells_actually_computed": cells_computed},
        "roofline": roof, "dominant_class": dom, "kernels": kernels,
        "int_peak_ops_per_s": {"lop3": lop3, "vabsdiff4": sad},
        "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line))


def main():
    args = parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        sys.exit(spawn_ranks(args))          # no launcher: start one rank per GPU ourselves
    if args.impl == "reference":
        run_reference(args)
    elif args.workload in ("config1", "config5"):
        run_all_pairs(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
