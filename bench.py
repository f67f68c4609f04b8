#!/usr/bin/env python
"""bench.py -- SPH step throughput of the B200 path (BASELINE.json metric), one JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference]

A "step" is one pass of the whole hot path (sph_step: hash -> onesweep sort -> reorder -> cell
ranges -> comm hash + compaction -> interaction loops with the integration in their epilogue) over the particles of
BASELINE.json configs[k] (default k = 4: 64 M particles, the largest single-GPU configuration, the one
the roofline bars of BASELINE.json's north_star are about; k = 0..3 are parity-test sizes).  N > 1 (torchrun) runs N
independent replicas (the one-GPU path does not shard; "weak" scaling).

`value`     particles/s, inputs resident in HBM, CUDA-event time of the K steps (L2 flushed
            between steps, outside the timed intervals), max over ranks.
`e2e`       the same metric through sph_step_host with pinned HOST buffers: H2D of the state,
            the step, D2H of the state + boundary list, inside the timed region.
`roofline`  the dominant kernel (interaction loop): algorithmic flops 8*Cand + 66*Pairs
             / its CUDA-event time, against the FP32 ALU peak.
`cpu_baseline` / --impl reference: the oracle as it stands on the host cores, bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "sph_step_particles_per_s"
UNIT = "particles/s"
FLOP_PER_CAND = 8.0      # 3 FADD + 1 FMUL + 2 FFMA
FLOP_PER_PAIR = 66.0     # kernel factor 7 + density rate 10 + velocity gradient 22 + momentum 27
BYTES_PER_PARTICLE = {   # algorithmic HBM bytes per particle per stage;
                         # reorder = 124 + the 48 B of packed interaction records it writes inside sph_step
    "hash": 20.0, "sort": None, "reorder": 172.0, "cell_ranges": None, "comm_hash": None,
    "interact": 96.0, "integrate": 156.0,
}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the interaction kernel from the
# committed `ncu --set full` capture (profiles/), keyed by config; None until captured.
NCU_TRAFFIC_BYTES = {
    1: 93.69e6,    # profiles/r01d_interact_v6_ncu_full.md (68.6 MB read + 25.1 MB written)
    4: 12.302e9,   # profiles/r02a_interact_cfg4_ncu_full.md (8.636 GB read + 3.666 GB written; 6.14 GB algorithmic)
}


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "sm_max_mhz": float(d.get("sm_max_mhz", 1965.0)),
                "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "source": "fallback (B200_PROFILING.md)"}


def fp32_peak_tflops(sm_count, sm_mhz):
    # 128 FP32 lanes per SM, 1 FMA (2 flop) per lane per cycle
    return sm_count * 128 * 2 * sm_mhz * 1e6 / 1e12


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 50 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                 "--format=csv,noheader,nounits", "-lms", "50"],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm, mx, reasons = [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(mx)) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def candidates_and_counts(cell_start, cell_end, dims):
    """Cand = sum_i (#particles in the 27-bucket stencil of i's bucket), from the cell tables."""
    nx, ny, nz = (int(d) for d in dims)
    cnt = (cell_end.astype(np.int64) - cell_start.astype(np.int64)).reshape(nz, ny, nx)
    pad = np.pad(cnt, 1)
    box = np.zeros_like(cnt)
    for dz in range(3):
        for dy in range(3):
            for dx in range(3):
                box += pad[dz:dz + nz, dy:dy + ny, dx:dx + nx]
    return int((cnt * box).sum())


def max_over_ranks(x, world, device):
    """Device-timed quantities are reported as the MAX over ranks (all-reduce on `device`:
    NCCL on the GPU box, gloo in the CPU tests)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n_per_rank, steps, world, total_ms):
    """Replicas only: every rank steps its own copy of the workload, so the
    job processed world * n * steps particles in the slowest rank's time."""
    return world * n_per_rank * steps / (total_ms * 1e-3)


def oracle_sample(w, n_sample):
    """Bounded sample of the workload for the CPU legs: the first n_sample particles in id order
    (whole lattice planes from z = 0), on the workload's own grid."""
    n = min(w.n, n_sample)
    return (w.posm[:n].copy(), w.velr[:n].copy(), np.ascontiguousarray(w.sig[:, :n]),
            w.owner[:n].copy(), n)


def time_oracle(w, n_sample, steps, warmup):
    import oracle
    posm, velr, sig, owner, n = oracle_sample(w, n_sample)
    times, pairs = [], 0
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        r = oracle.step(posm, velr, sig, owner, w.origin, w.dims, w.h, w.K, w.G, w.n_owners, w.dt)
        t1 = time.perf_counter()
        if it >= warmup:
            times.append(t1 - t0)
            pairs += r.rates.pair_count
        posm, velr, sig = (r.posm.astype(np.float32), r.velr.astype(np.float32),
                           r.sig.astype(np.float32))
    tot = sum(times)
    return {"value": n * steps / tot, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"first {n} of {w.n} particles in id order (z-planes from 0), whole oracle "
                      f"step, {steps} steps after {warmup} warm-up",
            "pair_interactions_per_s": pairs / tot, "s_per_step": tot / steps}


def workload_name(w, k):
    scaled = f" (lengths x {w.meta['scale']})" if w.meta.get("scale", 1.0) != 1.0 else ""
    return f"configs[{k}] {w.name}{scaled}: {w.n} particles, grid {tuple(int(d) for d in w.dims)}, " \
           f"{w.n_owners} owners"


def run_reference(args, rank, world):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if rank != 0:
        return
    from paper_2310_03596_b200 import workloads
    w = workloads.config(args.config, scale=args.scale if args.config == 3 else None)
    cb = time_oracle(w, args.ref_sample, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": cb["value"], "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": cb["s_per_step"] * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": workload_name(w, args.config), "sample": cb["sample"]},
        "cpu_baseline": {"value": cb["value"], "unit": UNIT, "cores": 1, "kind": "oracle",
                         "sample": cb["sample"]},
        "e2e": {"value": cb["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "pair_interactions_per_s": cb["pair_interactions_per_s"], "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2310_03596_b200 import sph, workloads

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the SPH path has no CPU fallback")
    dev = torch.device(f"cuda:{local_rank}")
    torch.cuda.set_device(dev)
    w = workloads.config(args.config, scale=args.scale if args.config == 3 else None)
    n, K, W = w.n, args.steps, max(args.warmup, 3)
    ctx = sph.Context.for_workload(w, device=str(dev), flags=args.flags)
    state0 = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner, device=str(dev))
    state = state0.clone()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # 2x the 126 MB L2
    pair_acc = torch.zeros(1, dtype=torch.int64, device=dev)
    ctx.enable_timing(True)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(W):
        ctx.sph_step(state, w.dt)
    torch.cuda.synchronize(dev)
    # counters for the roofline (state after warm-up, not timed)
    out = ctx.alloc_outputs(n)
    probe = state.clone()
    ctx.sph_step(probe, w.dt, out)
    torch.cuda.synchronize(dev)
    pairs_step = int(out.pair_count.cpu()[0])
    cand_step = candidates_and_counts(sph.as_u32(out.cell_start), sph.as_u32(out.cell_end), w.dims)
    boundary = int(sph.as_u32(out.boundary_count)[0])
    del out, probe

    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    launches0 = ctx.launch_count()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    stage_ms, stage_w = {}, 0
    ctx.enable_timing(True)                             # resets the library's ring of stage events
    barrier()
    for it in range(K):
        flush.zero_()                                   # L2 flush, outside the timed interval
        evs[it][0].record()
        ctx.sph_step(state, w.dt)                       # pair_count = NULL: the count is optional (include/sph.h)
        evs[it][1].record()
        if (it + 1) % sph.TIMING_SLOTS == 0 or it == K - 1:
            # the stage events live in a ring of TIMING_SLOTS steps inside the library: drain it
            # (one host sync per ring, between steps) so that EVERY timed step enters the average
            m_ = (it % sph.TIMING_SLOTS) + 1
            for k_, v in ctx.get_timing().items():
                stage_ms[k_] = stage_ms.get(k_, 0.0) + v * m_
            stage_w += m_
    barrier()
    launches = ctx.launch_count() - launches0
    total_ms = sum(a.elapsed_time(b) for a, b in evs)
    stage_ms = {k_: v / stage_w for k_, v in stage_ms.items()}
    total_ms = max_over_ranks(total_ms, world, dev)

    # ---- NEXT-1 (not part of the step metric): per-owner send buffers of the last boundary list ----
    pack = None
    if boundary > 0:
        bids_dev = torch.empty(n, dtype=torch.int32, device=dev)
        bcnt = torch.zeros(1, dtype=torch.int32, device=dev)
        o2 = ctx.alloc_outputs(n)
        ctx.sph_step(state.clone(), w.dt, o2)
        torch.cuda.synchronize(dev)
        m_b = int(sph.as_u32(o2.boundary_count)[0])
        pk_ms = []
        pk_out = (torch.empty(w.n_owners + 1, dtype=torch.int32, device=dev),
                  torch.empty(max(m_b, 1), dtype=torch.int32, device=dev), sph.State.empty(max(m_b, 1), dev))
        for _ in range(5):
            flush.zero_()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record()
            ctx.sph_pack_boundary(state, o2.boundary_ids, m_b, out=pk_out)
            b_.record()
            torch.cuda.synchronize(dev)
            pk_ms.append(a_.elapsed_time(b_))
        pk = float(np.median(pk_ms[1:]))
        pk_gbs = 156.0 * m_b / (pk * 1e-3) / 1e9 if pk > 0 else 0.0
        pack = {"ms": round(pk, 4), "boundary_particles": m_b, "bytes_per_boundary_particle": 156,
                "gbs": round(pk_gbs, 1), "hbm_frac": round(pk_gbs / load_peaks()["hbm_gbs"], 3),
                "note": "outputs pre-allocated (no allocation inside the timed interval)"}
        del o2, bids_dev, bcnt, pk_out

    # ---- NEXT-1, second half (not part of the step metric): per-destination send lists ----
    dests = None
    if w.n_owners > 1 and n * (w.n_owners - 1) < (1 << 30):
        hh = ctx.sph_hash(state.posm)
        sh_, pm_ = ctx.sph_sort(hh)
        so_ = state.owner[pm_.long()].contiguous()
        cs_, ce_ = ctx.sph_cell_ranges(sh_)
        _ch, _bi, cnt_, _oc = ctx.sph_comm_hash(sh_, so_, pm_, cs_, ce_)
        offs_, ids_ = ctx.sph_pack_destinations(sh_, so_, pm_)          # sizes the buffer (one host sync)
        torch.cuda.synchronize(dev)
        m_b2 = int(sph.as_u32(cnt_)[0])
        total_d = int(sph.as_u32(offs_)[-1])
        ts = []
        for _ in range(5):
            flush.zero_()
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record()
            ctx.sph_pack_destinations(sh_, so_, pm_, dest_ids=ids_, dest_offsets=offs_)
            b_.record()
            torch.cuda.synchronize(dev)
            ts.append(a_.elapsed_time(b_))
        bcast = m_b2 * (w.n_owners - 1)
        dests = {"ms": round(float(np.median(ts[1:])), 4), "entries": total_d, "broadcast_entries": bcast,
                 "entries_over_broadcast": round(total_d / bcast, 4) if bcast else None,
                 "record_bytes_saved": 156 * (bcast - total_d),
                 "note": "entries = sum over destinations g of the boundary particles g really needs (reading D1); "
                         "broadcast = every boundary particle to every other owner (PAPER.md:23)"}
        del hh, sh_, pm_, so_, cs_, ce_, _ch, _bi, cnt_, _oc, offs_, ids_

    # ---- NEXT-3 (not part of the step metric): steps e / f as separate interaction passes ----
    split = None
    if w.n_owners > 1:
        hh = ctx.sph_hash(state.posm)
        sh_, pm_ = ctx.sph_sort(hh)
        st_ = ctx.sph_reorder(pm_, state)
        cs_, ce_ = ctx.sph_cell_ranges(sh_)

        def _t(fn):
            ts = []
            for _ in range(4):
                flush.zero_()
                a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a_.record()
                r_ = fn()
                b_.record()
                torch.cuda.synchronize(dev)
                ts.append(a_.elapsed_time(b_))
            return float(np.median(ts[1:])), r_

        t_all, r_all = _t(lambda: ctx.sph_interact(st_, sh_, cs_, ce_))
        t_e, r_e = _t(lambda: ctx.sph_interact_split(st_, sh_, cs_, ce_, 1))
        t_f, r_f = _t(lambda: ctx.sph_interact_split(st_, sh_, cs_, ce_, 2))
        t_ef, r_ef = _t(lambda: ctx.sph_interact_ef(st_, sh_, cs_, ce_))
        split = {"single_pass_ms": round(t_all, 4), "pass_e_ms": round(t_e, 4), "pass_f_ms": round(t_f, 4),
                 "e_and_f_one_search_ms": round(t_ef, 4), "e_and_f_over_single": round(t_ef / t_all, 3),
                 "pairs_single": int(r_all[3].cpu()[0]), "pairs_e": int(r_e[3].cpu()[0]),
                 "pairs_f": int(r_f[3].cpu()[0]),
                 "note": "stand-alone sph_interact calls (pack pass and output allocation included)"}
        del hh, sh_, pm_, st_, cs_, ce_, r_all, r_e, r_f, r_ef

    # ---- NEXT-2 (not part of the step metric): one balancing sweep and what it does to the exchange set ----
    bal = None
    if 1 < w.n_owners and args.balance_sweeps > 0:
        st_b = state.clone()
        o_b = ctx.alloc_outputs(n)
        ctx.sph_step(st_b.clone(), w.dt, o_b)
        torch.cuda.synchronize(dev)
        frac = [int(sph.as_u32(o_b.boundary_count)[0]) / n]
        ms_b, swaps = [], []
        for _ in range(args.balance_sweeps):
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record()
            _bh, sw_ = ctx.sph_balance(st_b.posm, st_b.owner, want_hash=False)
            b_.record()
            torch.cuda.synchronize(dev)
            ms_b.append(a_.elapsed_time(b_))
            del _bh
            swaps.append(int(sw_.cpu()[0]))
            ctx.sph_step(st_b.clone(), w.dt, o_b)
            torch.cuda.synchronize(dev)
            frac.append(int(sph.as_u32(o_b.boundary_count)[0]) / n)
        # the same sweep with the optional bal_hash output stored (the parity tests' form), on a copy
        own_h = st_b.owner.clone()
        a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a_.record()
        _bh, _sw = ctx.sph_balance(st_b.posm, own_h, want_hash=True)
        b_.record()
        torch.cuda.synchronize(dev)
        ms_with_hash = a_.elapsed_time(b_)
        del own_h, _bh, _sw
        bal = {"sweep_ms": [round(x, 3) for x in ms_b], "sweep_ms_note": "bal_hash not stored (optional output NULL)",
               "sweep_ms_hashes_stored": round(ms_with_hash, 3), "swapped_pairs": swaps,
               "boundary_fraction": [round(x, 4) for x in frac], "owner_pairs": w.n_owners * (w.n_owners - 1) // 2}
        del st_b, o_b

    # ---- end to end through the C-ABI with pinned host buffers ----
    host = sph.State.from_numpy(w.posm, w.velr, w.sig, w.owner, device="cpu", pin=True)
    bids = torch.empty(n, dtype=torch.int32).pin_memory().numpy().view(np.uint32)
    ctx.sph_step_host(host, w.dt, 1, bids)               # warm-up (allocates staging)
    e2e_steps = min(K, 5)
    barrier()
    t0 = time.perf_counter()
    m_last = 0
    for _ in range(e2e_steps):
        m_last, _pc = ctx.sph_step_host(host, w.dt, 1, bids)   # synchronises before returning
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world, dev)
    clocks = sampler.stop() if rank == 0 else None
    if rank != 0:
        return

    peaks = load_peaks()
    props = torch.cuda.get_device_properties(dev)
    ms_per_step = total_ms / K
    value = whole_job_value(n, K, world, total_ms)
    flops = FLOP_PER_CAND * cand_step + FLOP_PER_PAIR * pairs_step
    t_int = stage_ms["interact"] * 1e-3
    fp32_peak = fp32_peak_tflops(props.multi_processor_count, peaks["sm_max_mhz"])
    achieved_tf = flops / t_int / 1e12
    stages = {}
    n_sort_passes = (max(1, int(np.ceil(np.log2(max(2, w.n_cells))))) + 7) // 8
    for k_, v in stage_ms.items():
        e = {"ms": round(v, 4)}
        b = BYTES_PER_PARTICLE.get(k_)
        if k_ == "sort":
            # inside sph_step the digit histograms are counted by the fused hash kernel, so this
            # stage is the onesweep passes alone: 16 B per particle and pass (keys + values in and
            # out).  The 4 B histogram read of SURVEY.md's 52 B/p belongs to stand-alone sph_sort.
            b = 16.0 * n_sort_passes
            e["note"] = f"{n_sort_passes} onesweep passes only (16 B/p each); histograms are in the hash stage"
        if k_ == "cell_ranges":
            b = 4.0 + 8.0 * w.n_cells / n
        if k_ == "comm_hash":
            b = 12.0 + 0.5 + 4.0 + 8.0 * boundary / n
        if k_ == "integrate":
            # inside sph_step the interaction epilogue integrates and scatters:
            # no separate pass runs, the stage boundary is kept only for the report
            e["fused_into"] = "interact"
            b = None
        if k_ == "hash":
            e["note"] = "fused with the digit histograms of the sort inside sph_step (the sort reads its keys once less)"
        if b and k_ != "interact" and v > 0:
            e["gbs"] = round(b * n / (v * 1e-3) / 1e9, 1)
            e["hbm_frac"] = round(e["gbs"] / peaks["hbm_gbs"], 3)
        stages[k_] = e
    # hash + sort as ONE fused stage on SURVEY.md 8(a)'s bytes (20 B/p hash + 4 B/p histogram read
    # + 16 B/p per pass): the fusion moved the histogram's bytes AND time into the hash kernel, so
    # only the sum can be compared with the survey's per-stage table
    hs_ms = stage_ms["hash"] + stage_ms["sort"]
    if hs_ms > 0:
        hs_b = 20.0 + 4.0 + 16.0 * n_sort_passes
        hs_gbs = hs_b * n / (hs_ms * 1e-3) / 1e9
        stages["hash_plus_sort"] = {"ms": round(hs_ms, 4), "bytes_per_particle": hs_b, "gbs": round(hs_gbs, 1),
                                    "hbm_frac": round(hs_gbs / peaks["hbm_gbs"], 3)}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(w, args.config), "l2": "flushed between steps (256 MB memset, untimed)",
                   "replicas": world, "boundary_particles": boundary, "interact_kernel": "direct" if args.flags & 1 else "tiled"},
        "pair_interactions_per_s": world * pairs_step / (ms_per_step * 1e-3),
        "pairs_per_step": pairs_step, "candidates_per_step": cand_step,
        "clocks": clocks,
        "e2e": {"value": world * n * e2e_steps / e2e_s, "unit": UNIT,
                "h2d_bytes_per_step": 60 * n, "d2h_bytes_per_step": 56 * n + 4 * m_last + 12,
                "steps": e2e_steps, "api": "sph_step_host (pinned host buffers)"},
        "gpu_launches": int(launches),
        "roofline": {"kernel": "interact", "bound": "alu", "achieved": achieved_tf, "peak": fp32_peak,
                     "unit": "TFLOP/s", "frac": achieved_tf / fp32_peak,
                     "traffic": NCU_TRAFFIC_BYTES.get(args.config),
                     "traffic_source": ("constant from the committed ncu --set full capture under profiles/ "
                                        "(dram__bytes_read.sum + dram__bytes_write.sum per launch); not measured by this run"
                                        if NCU_TRAFFIC_BYTES.get(args.config) else None),
                     "algorithmic_bytes": BYTES_PER_PARTICLE["interact"] * n,
                     "peak_source": f"{props.multi_processor_count} SMs x 128 lanes x 2 x "
                                    f"{peaks['sm_max_mhz']:.0f} MHz (DESIGN.md section 7)",
                     "hbm_peak_gbs": peaks["hbm_gbs"], "hbm_peak_source": peaks["source"],
                     "interact_hbm_gbs": BYTES_PER_PARTICLE["interact"] * n / t_int / 1e9},
        "stages": stages,
    }
    if pack:
        pack["gbs"] = round(pack["bytes_per_boundary_particle"] * pack["boundary_particles"] / (pack["ms"] * 1e-3) / 1e9, 1)
        pack["hbm_frac"] = round(pack["gbs"] / peaks["hbm_gbs"], 3)
        line["next1_pack_boundary"] = pack
    if dests:
        line["next1_pack_destinations"] = dests
    if split:
        line["next3_split_passes"] = split
    if bal:
        line["next2_balance"] = bal
    if world == 1 and not args.no_cpu_baseline:
        cb = time_oracle(w, args.cpu_sample, 3, 1)
        line["cpu_baseline"] = {k_: cb[k_] for k_ in ("value", "unit", "cores", "kind", "sample")}
        line["cpu_baseline"]["host_cores"] = os.cpu_count()
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=4, help="BASELINE.json configs[k] (default: the 64 M-particle headline)")
    ap.add_argument("--scale", type=float, default=None,
                    help="configs[3] only: scale every length of the geometry (1.13 gives the ~32 M particles "
                         "BASELINE.json quotes; the dimensions as stated give 22.0 M)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--flags", type=int, default=0, help="sph_params.flags (1 = direct interaction kernel)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--balance-sweeps", type=int, default=2, help="NEXT-2 report: balancing sweeps to time (0 = skip)")
    ap.add_argument("--cpu-sample", type=int, default=300000)
    ap.add_argument("--ref-sample", type=int, default=100000)
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    try:
        run_ours(args, rank, world, local_rank)
    finally:
        if world > 1:
            import torch.distributed as dist
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
