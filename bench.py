#!/usr/bin/env python
"""Benchmark of the composition hot path (pack -> compose) on BASELINE.json's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload large|medium|skewed|nlp|tiny|dups]
                    [--impl ours|reference] [--no-e2e] [--no-cpu-baseline]

One "step" = one pass of the whole hot path over one pair of synthetic transducers: pack(M1),
pack(M2), compose_packed (count, scan, match, emit, target resolve — visited table or partitioned —, merge,
assembly).  Inputs are resident in HBM when the timed region of `value` starts; `e2e` repeats the step
through the C ABI with HOST buffers (H2D of the inputs and D2H of the whole result inside the timed region).

`roofline` is SURVEY §8(d)'s number: the algorithmic bytes of the whole composition (exact device-side counts) divided by
the device time of fstc_compose_packed, against the measured HBM peak; `roofline.stage_groups` splits the same terms over
the stage groups that serve them (CUDA events on the compose stream, library `profile` mode) and names the dominant one;
`roofline.achieved_vs_own_traffic` keeps the achieved bandwidth of the resolve kernels on the bytes their design moves
(not a fraction of the method's bytes); `traffic` = DRAM bytes of one composition from the committed ncu capture.
`ms_steps` carries every timed step.

N > 1 (torchrun): the path shards by independent problems — every rank composes its own seeded pair of
the same shape, no data-path collective ("scaling": "weak"); time = max over ranks, value = Σ arcs / time.

`--impl reference` times the CPU oracle (oracle/, as it stands, 1 core) on a bounded sample of the same
workload; it is a deliberately slow baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "composed_raw_arcs_per_sec"
UNIT = "arcs/s"
# bounded oracle samples (raw-arc budget) sized for roughly 10-30 s of one host core
ORACLE_SAMPLE_BUDGET = {"large": 20_000_000, "medium": 60_000_000, "skewed": 60_000_000, "nlp": 0, "tiny": 0, "dups": 40_000_000}
WORKLOAD_DESC = {
    "large": "large random (BASELINE.json configs[3]): |Q1|=|Q2|=1e5, |Σ|=|Δ|=2e4, |Γ|=5e3 Zipf 1.1, 5e6 arcs each, "
             "max_raw_arcs=1e9 (rule T)",
    "medium": "medium random (configs[1]): |Q1|=|Q2|=1e4, |Σ|=|Δ|=1e3, |Γ|=1e3 Zipf 1.0, 2e5 arcs each, complete",
    "skewed": "skewed/high-merge (configs[4]): |Q|=2e3, |Σ|=|Δ|=10, |Γ|=50 Zipf 1.5, 1e6 arcs each, power-law degree, "
              "max_raw_arcs=1e9",
    "nlp": "NLP-shaped (configs[2]): 50x8 lattice ∘ 30k-state bigram (3e6 arcs), complete",
    "tiny": "tiny random (configs[0])",
    "dups": "medium random + 10 % parallel duplicate arcs (NOT a BASELINE config: the workload of the merge on chip, SURVEY §8(f)1): "
            "|Q1|=|Q2|=1e4, |Γ|=1e3 Zipf 1.0, 2.2e5 arcs each, every source duplicate-prone, complete",
}


def _peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clocks and throttle reasons during the timed region: NVML in a thread of this process (no subprocess
    polling the driver beside the timed work), nvidia-smi only as a fallback."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc, self.stop_flag, self.nvml = index, [], None, False, None

    def start(self):
        try:
            import pynvml
            pynvml.nvmlInit()
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            idx = int(vis.split(",")[self.index]) if vis and vis.split(",")[self.index].isdigit() else self.index
            self.nvml = (pynvml, pynvml.nvmlDeviceGetHandleByIndex(idx))
            self.t = threading.Thread(target=self._poll_nvml, daemon=True)
            self.t.start()
            return
        except Exception:
            self.nvml = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "250"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _poll_nvml(self):
        nv, h = self.nvml
        R = {"hw_slowdown": nv.nvmlClocksThrottleReasonHwSlowdown,
             "hw_thermal_slowdown": nv.nvmlClocksThrottleReasonHwThermalSlowdown,
             "sw_thermal_slowdown": nv.nvmlClocksThrottleReasonSwThermalSlowdown,
             "sw_power_cap": nv.nvmlClocksThrottleReasonSwPowerCap}
        while not self.stop_flag:
            try:
                sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
                mx = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
                bits = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                self.rows.append([str(sm), str(mx), "0"] + ["Active" if bits & R[n] else "Not Active" for n in
                                                           ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")])
            except Exception:
                pass
            time.sleep(0.05)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self) -> dict:
        if self.nvml:
            self.stop_flag = True
            self.t.join(timeout=1)
        elif self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            try:
                self.proc.wait(timeout=2)
            except Exception:
                self.proc.kill()
        else:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no NVML, no nvidia-smi"]}
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); mx = float(r[1])
            except ValueError:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        # clocks under load: the upper half of the samples (idle gaps between steps pull the median down)
        load = sm[len(sm) // 2:] if sm else []
        return {"sm_mhz": load[len(load) // 2] if load else None, "sm_max_mhz": mx, "samples": len(sm),
                "reasons": sorted(reasons), "source": "nvml" if self.nvml else "nvidia-smi"}


# Stage groups of the library's `profile` times, and the SURVEY §8(d) terms each one serves.
STAGE_GROUPS = {
    "index": ("count", "scan", "match"),                       # 16·E + 8·Σ_E(s1+s2)
    "expand": ("emit", "sort", "reduce"),                      # 12·Σ_matches(n1+n2) + 20·M + 40·R_m (+ table-level probes, fused)
    "visited": ("table", "rs_scatter", "rs_dedupe", "rs_gather"),   # 12·R + 12·S of the levels resolved outside the emit kernel
    "assemble": ("assemble",),                                 # 9·S
}


def alg_bytes(st: dict) -> dict:
    """SURVEY §8(d) algorithmic bytes from exact device-side counts: of the whole composition, and split over the
    stage groups that serve each term.  The visited-set term (12 per raw arc + 12 per state) of the levels whose targets
    are resolved inside the emit kernel (visited table) is charged to `expand`; the rest to `visited`."""
    E, R, S, M = st["n_expanded"], st["n_raw_arcs"], st["n_states"], st["n_arcs"]
    Rm = st["n_raw_sorted"]
    Rp, Sp = st["n_resolved_arcs"], st["rs_dedupe_new"]        # arcs / new states of the partitioned-resolve levels
    groups = {
        "index": 16 * E + 8 * st["n_seg_visited"],
        "expand": 12 * st["n_match_arcs"] + 20 * M + 40 * Rm + 12 * (R - Rp) + 12 * (S - Sp),
        "visited": 12 * Rp + 12 * Sp,
        "assemble": 9 * S,
    }
    return {"path": sum(groups.values()), "groups": groups}


def own_traffic(st: dict) -> dict:
    """Bytes each hot kernel of the partitioned resolve moves BY DESIGN (not SURVEY's model): what its
    achieved bandwidth is measured on (`achieved_vs_own_traffic`)."""
    rec = st.get("rs_rec_bytes", 8)
    return {
        "rs_scatter": (2 * rec) * (st["rs_scatter_recs"] + st["rs_scatter_dest_recs"]) + 6 * st["rs_scatter_dest_recs"],
        "rs_dedupe": 8 * st["rs_dedupe_states"] + (rec + 4) * st["rs_dedupe_arcs"] + 8 * st["rs_dedupe_new"],
        "rs_gather": 14 * st["rs_gather_recs"],
    }


def rank_seeds(workload: str, rank: int):
    """Every rank composes its own pair of the same shape: independent problems, no data-path collective."""
    from paper_1805_06383_b200 import workloads
    s1, s2 = workloads.CONFIGS[workload]["seeds"]
    return s1 + 1000 * rank, s2 + 1000 * rank


def reduce_over_ranks(dist, world: int, time_like, sum_like, device):
    """(max over ranks of each time-like value, sum over ranks of each additive value)."""
    import torch
    tm = torch.tensor([float(x) for x in time_like], dtype=torch.float64, device=device)
    ts = torch.tensor([float(x) for x in sum_like], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(tm, op=dist.ReduceOp.MAX)
        dist.all_reduce(ts, op=dist.ReduceOp.SUM)
    return [float(x) for x in tm], [float(x) for x in ts]


def run_reference(args, rank, world):
    """The CPU oracle, as it stands, on a bounded sample of the workload (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    from paper_1805_06383_b200 import workloads
    m1, m2 = workloads.make_config(args.workload)
    full_budget = int(workloads.CONFIGS[args.workload]["max_raw_arcs"])
    sample = ORACLE_SAMPLE_BUDGET[args.workload] or full_budget
    if full_budget:
        sample = min(sample, full_budget) if sample else full_budget
    secs, arcs = [], 0
    for i in range(args.warmup + args.steps):
        r = oracle.compose(m1, m2, max_raw_arcs=sample, keep_arcs=False)
        if i >= args.warmup:
            secs.append(r.seconds)
            arcs = r.n_raw_arcs
        if sum(secs) > 240:      # keep the whole run within a few minutes
            break
    steps = len(secs)
    t = sum(secs)
    value = arcs * steps / t
    desc = f"oracle.compose on the same inputs with max_raw_arcs={sample} ({arcs} raw arcs per step), 1 thread"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * t / steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD_DESC[args.workload], "sample": desc},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="large", choices=sorted(WORKLOAD_DESC))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--merge-mode", type=int, default=0)
    ap.add_argument("--resolve-mode", type=int, default=0, help="0 auto, 1 visited table only, 2 partitioned resolve only")
    ap.add_argument("--deterministic", action="store_true", help="fstc_opts_t.deterministic: ids in key order inside every level")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--batch", type=int, default=0, help="workload nlp only: also time B seeded lattices against the one packed "
                    "language model, fstc_compose_batch against B calls of fstc_compose_packed (adds a \"batch\" object)")
    ap.add_argument("--fixed-warmup", action="store_true", help="exactly --warmup untimed steps (profiler runs), no settling loop")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    import torch.distributed as dist
    from paper_1805_06383_b200 import fstc, workloads
    fstc.lib()                                   # no CUDA library, no benchmark (there is no fallback)
    assert torch.cuda.is_available(), "bench.py needs a CUDA device"
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # every rank composes its own seeded pair of the same shape (independent problems, no collective)
    s1, s2 = workloads.CONFIGS[args.workload]["seeds"]
    m1, m2 = workloads.make_config(args.workload, seeds=rank_seeds(args.workload, rank))
    budget = int(workloads.CONFIGS[args.workload]["max_raw_arcs"])
    d1, d2 = fstc.DeviceFst.from_host(m1), fstc.DeviceFst.from_host(m2)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2

    def step(profile=True):
        """pack + compose on device-resident inputs; returns (ms, stats, pack_launches)."""
        flush.fill_(1)                                                   # L2 flush, outside the timed region
        e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        e0.record()
        p1 = fstc.fstc_pack(d1, 1)
        t1 = time.perf_counter()
        p2 = fstc.fstc_pack(d2, 2)
        t2 = time.perf_counter()
        e1.record()
        r = fstc.fstc_compose_packed(p1, p2, merge_mode=args.merge_mode, max_raw_arcs=budget, profile=profile,
                                     resolve_mode=args.resolve_mode, deterministic=args.deterministic)
        t3 = time.perf_counter()
        e2.record()
        torch.cuda.synchronize()
        st = r.stats
        host_ms = [round(1e3 * (b - a), 2) for a, b in ((t0, t1), (t1, t2), (t2, t3))]      # pack, pack, compose on the host clock
        st["pack_ms"], st["compose_ms"] = e0.elapsed_time(e1), e1.elapsed_time(e2)
        launches = st["n_kernel_launches"] + p1.info().get("n_kernel_launches", 0) + p2.info().get("n_kernel_launches", 0)
        del r
        p1.free(); p2.free()
        if os.environ.get("FSTC_ALLOC_TRACE") or os.environ.get("FSTC_RS_TRACE"):   # debug knobs of the library: mark the steps
            print(f"[bench] step done: {e0.elapsed_time(e2):.2f} ms, stages {sum(st['ms'].values()):.2f} ms, host {host_ms}, "
                  f"lib total {st['ms_total']:.2f}", file=sys.stderr, flush=True)
        return e0.elapsed_time(e2), st, launches

    # warm-up: at least W (>= 3) untimed steps; then, while the machine is still settling (memory pools filling, clocks
    # ramping), up to 30 more until three steps in a row agree within 2 % of the fastest step seen
    n_warm, recent, best = 0, [], float("inf")
    while n_warm < (max(args.warmup, 3) + 30 if not args.fixed_warmup else args.warmup):
        ms, st, _ = step()
        n_warm += 1
        best = min(best, ms)
        recent = (recent + [ms])[-3:]
        if not args.fixed_warmup and n_warm >= max(args.warmup, 3) and len(recent) == 3 and max(recent) <= 1.02 * best:
            break
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    ms_steps, stats, launches = [], [], 0
    for _ in range(args.steps):
        ms, st, nl = step()
        ms_steps.append(ms); stats.append(st); launches += nl
    barrier()
    clocks = sampler.stop()

    t_ms = sum(ms_steps)
    arcs = sum(s["n_raw_arcs"] for s in stats)
    (t_ms,), (arcs, launches) = reduce_over_ranks(dist, world, [t_ms], [arcs, launches], "cuda")
    value = arcs / (t_ms * 1e-3)

    st = stats[-1]
    peak, peak_src = _peaks()
    ab = alg_bytes(st)
    compose_ms = sum(s["compose_ms"] for s in stats) / len(stats)
    pack_ms = sum(s["pack_ms"] for s in stats) / len(stats)
    stage_ms = {k: sum(s["ms"][k] for s in stats) / len(stats) for k in fstc.STAGES}
    # the headline fraction is B_alg / t_compose_packed / peak; per stage group the same terms over the
    # group's device time (CUDA events on the compose stream, library `profile` mode)
    path_gbs = ab["path"] / (compose_ms * 1e-3) / 1e9
    groups = {}
    for gname, members in STAGE_GROUPS.items():
        ms = sum(stage_ms[m] for m in members)
        gb = ab["groups"][gname]
        groups[gname] = {"stages": list(members), "ms_per_step": ms, "alg_bytes_per_step": gb,
                         "achieved_GBs": gb / (ms * 1e-3) / 1e9 if ms > 0 else 0.0,
                         "frac": gb / (ms * 1e-3) / 1e9 / peak if ms > 0 else 0.0,
                         "share_of_compose": ms / compose_ms if compose_ms > 0 else 0.0}
    dom = max(groups, key=lambda g: groups[g]["ms_per_step"])
    own = own_traffic(st)
    own_k = {}
    for k, (stage, nl) in {"rs_scatter": ("rs_scatter", "rs_scatter_launches"), "rs_dedupe": ("rs_dedupe", "rs_dedupe_launches"),
                           "rs_gather": ("rs_gather", "rs_gather_launches")}.items():
        if stage_ms[stage] > 0:
            own_k[k] = {"ms_per_step": stage_ms[stage], "launches_per_step": st[nl], "own_bytes_per_step": own[k],
                        "achieved_GBs": own[k] / (stage_ms[stage] * 1e-3) / 1e9}
    traffic = None
    tpath = os.path.join(ROOT, "profiles", f"kernel_traffic_{args.workload}.json")
    if os.path.exists(tpath):
        try:
            # measured DRAM bytes of one whole composition (ncu --set full, summed over the kernels of one step)
            traffic = json.load(open(tpath)).get("dram_bytes_per_step")
        except Exception:
            traffic = None
    latency_bound = st["n_raw_arcs"] < 10_000_000

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": n_warm, "ms_per_step": t_ms / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD_DESC[args.workload], "name": args.workload, "seeds": [s1, s2],
                   "max_raw_arcs": budget, "merge_mode": args.merge_mode, "resolve_mode": args.resolve_mode, "deterministic": bool(args.deterministic), "parallelism": f"replicas x{world}",
                   "cache": "L2 flushed (256 MiB write) before every step; working set >> L2"},
        "result": {"small_path": st["small_path"], "n_states": st["n_states"], "n_arcs": st["n_arcs"], "n_raw_arcs": st["n_raw_arcs"],
                   "n_levels": st["n_levels"], "truncated": st["truncated"], "n_expanded": st["n_expanded"],
                   "merged_arcs_per_sec": st["n_arcs"] * world / (t_ms / args.steps * 1e-3)},
        "timing_ms": {"pack": pack_ms, "compose_packed": compose_ms, "stages": stage_ms,
                      "compose_raw_arcs_per_sec": st["n_raw_arcs"] / (compose_ms * 1e-3)},
        # algorithmic bytes of the whole composition / compose time, against the measured HBM peak
        "roofline": {"bound": "hbm", "kernel": "path: every kernel of fstc_compose_packed", "achieved": path_gbs, "peak": peak,
                     "unit": "GB/s", "frac": path_gbs / peak, "peak_source": peak_src, "traffic": traffic,
                     "alg_bytes_per_step": ab["path"], "alg_bytes_per_raw_arc": ab["path"] / max(1, st["n_raw_arcs"]),
                     "ms_per_step": compose_ms, "frac_of_8TBs_nominal": path_gbs / 8000.0,
                     "meaningful": not latency_bound,
                     "note": ("latency-bound workload (< 1e7 arcs): report ms, the HBM fraction says nothing" if latency_bound else
                              "B_alg = 16E + 8Σ(s1+s2) + 12Σ(n1+n2) + 12R + 12S + 20M + 9S + 40R_m (SURVEY §8(d))"),
                     "dominant_stage_group": dom, "stage_groups": groups,
                     "achieved_vs_own_traffic": own_k},
        "ms_steps": [round(x, 3) for x in ms_steps], "compose_ms_steps": [round(s_["compose_ms"], 3) for s_ in stats],
        "clocks": clocks, "gpu_launches": int(launches),
        "host": {"nproc": os.cpu_count()},
    }

    # ---- end to end through the C ABI with host buffers (rank-local, then max over ranks)
    if not args.no_e2e:
        pin = lambda a: torch.from_numpy(a).pin_memory()     # noqa: E731
        class HostFst:                                        # pinned host tensors: mem = FSTC_MEM_HOST
            pass
        hs = []
        for m in (m1, m2):
            h = HostFst()
            h.n_states, h.n_isyms, h.n_osyms, h.start = m.n_states, m.n_isyms, m.n_osyms, m.start
            for n in ("src", "ilabel", "olabel", "tgt", "weight", "accept"):
                setattr(h, n, pin(getattr(m, n)))
            hs.append(h)
        na, ns = st["n_arcs"], st["n_states"]
        out = {"pair": torch.empty(2 * ns, dtype=torch.int32).pin_memory(),
               "expanded": torch.empty(ns, dtype=torch.uint8).pin_memory(),
               "accept": torch.empty(max(1, ns), dtype=torch.int32).pin_memory()}
        for n in ("src", "ilabel", "olabel", "tgt"):
            out[n] = torch.empty(na, dtype=torch.int32).pin_memory()
        out["weight"] = torch.empty(na, dtype=torch.float32).pin_memory()
        h2d = sum(int(getattr(h, n).numel()) * 4 for h in hs for n in ("src", "ilabel", "olabel", "tgt", "weight", "accept"))
        n_e2e = max(1, min(args.e2e_steps, args.steps))

        def e2e_run(spill):
            """fstc_compose on pinned host arrays; the result reaches `out` through fstc_result_to_host after the call, or
            (spill) through fstc_spill_t while the search runs: finished levels cross PCIe on a second stream and the arcs
            are never held on the device beyond their level."""
            tot_ms, tot_arcs, d2h, saved = 0.0, 0, 0, 0
            for i in range(1 + n_e2e):
                flush.fill_(1)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                barrier()
                a.record()
                if spill:
                    r = fstc.fstc_compose(hs[0], hs[1], merge_mode=args.merge_mode, max_raw_arcs=budget,
                                          resolve_mode=args.resolve_mode, spill=out, spill_keep_device=False)
                else:
                    r = fstc.fstc_compose(hs[0], hs[1], merge_mode=args.merge_mode, max_raw_arcs=budget, resolve_mode=args.resolve_mode)
                    r.to_host(out)
                b.record()
                torch.cuda.synchronize()
                if i > 0:
                    tot_ms += a.elapsed_time(b)
                    tot_arcs += r.n_raw_arcs
                d2h = 8 * r.n_states + r.n_states + 4 * r.n_accept + 20 * r.n_arcs
                saved = r.stats["spill_bytes_saved"]
                del r
            (tot_ms,), (tot_arcs,) = reduce_over_ranks(dist, world, [tot_ms], [tot_arcs], "cuda")
            return tot_ms, tot_arcs, d2h, saved

        e2e_ms, e2e_arcs, d2h, _ = e2e_run(False)
        sp_ms, sp_arcs, _, spill_saved = e2e_run(True)
        line["e2e"] = {"value": e2e_arcs / (e2e_ms * 1e-3), "unit": UNIT, "h2d_bytes_per_step": h2d,
                       "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / n_e2e, "steps": n_e2e,
                       "api": "fstc_compose(pinned host arrays) + fstc_result_to_host(pinned host arrays)",
                       "pcie_floor_ms": (h2d + d2h) / 52e9 * 1e3,
                       "with_host_spill": {"value": sp_arcs / (sp_ms * 1e-3), "ms_per_step": sp_ms / n_e2e,
                                           "api": "fstc_compose(pinned host arrays in, fstc_spill_t pinned host arrays out, keep_device = 0)",
                                           "device_bytes_never_held": int(spill_saved)}}
        del out

    # ---- many lattices against one language model: the operands packed and resident, one call for all
    if args.batch > 0 and args.workload == "nlp" and rank == 0:
        lm = fstc.fstc_pack(d2, 2)
        lats = [fstc.fstc_pack(fstc.DeviceFst.from_host(l), 1) for l in workloads.make_lattices(args.batch, seed0=s1)]

        def timed(fn, reps=5):
            best, out = float("inf"), None
            for i in range(2 + reps):
                flush.fill_(1)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize()
                a.record()
                out = fn()
                b.record()
                torch.cuda.synchronize()
                if i >= 2:
                    best = min(best, a.elapsed_time(b))
            return best, out

        t_batch, res = timed(lambda: fstc.fstc_compose_batch(lats, lm))
        t_loop, res1 = timed(lambda: [fstc.fstc_compose_packed(l, lm) for l in lats])
        assert [r.n_arcs for r in res] == [r.n_arcs for r in res1] and [r.n_states for r in res] == [r.n_states for r in res1]
        raw = sum(r.n_raw_arcs for r in res)
        # the same call without the binding's result objects: the C ABI as a C caller sees it (host clock around the call,
        # which ends with its own stream synchronisation)
        import ctypes
        ptrs = (ctypes.c_void_p * args.batch)(*[p.ptr for p in lats])
        o_c = fstc._opts()
        t_c = float("inf")
        for i in range(7):
            outs = (ctypes.c_void_p * args.batch)()
            flush.fill_(1)
            torch.cuda.synchronize()
            c0 = time.perf_counter()
            rc = fstc.lib().fstc_compose_batch(ctypes.addressof(ptrs), args.batch, lm.ptr, ctypes.addressof(o_c), fstc._stream_ptr(None),
                                               ctypes.addressof(outs), None)
            c1 = time.perf_counter()
            assert rc == 0
            for a in outs:
                fstc.lib().fstc_result_free(a)
            if i >= 2:
                t_c = min(t_c, (c1 - c0) * 1e3)
        line["batch"] = {"lattices": args.batch, "api": "fstc_compose_batch(B packed lattices, one packed language model)",
                         "ms": t_batch, "lattices_per_sec": args.batch / (t_batch * 1e-3), "raw_arcs_per_sec": raw / (t_batch * 1e-3),
                         "c_abi_ms": t_c, "c_abi_lattices_per_sec": args.batch / (t_c * 1e-3),
                         "raw_arcs": raw, "arcs": sum(r.n_arcs for r in res), "states": sum(r.n_states for r in res),
                         "launches": res[0].stats["n_kernel_launches"], "small_path": sum(r.stats["small_path"] for r in res),
                         "one_call_per_lattice_ms": t_loop, "speedup_vs_one_call_per_lattice": t_loop / t_batch,
                         "timing": "best of 5 after 2 untimed, CUDA events, L2 flushed before each"}
        del res, res1, lats, lm

    # ---- the oracle, as it stands, on this box's host cores (rank 0, N = 1 only)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        sample = ORACLE_SAMPLE_BUDGET[args.workload] or budget
        if budget:
            sample = min(sample, budget) if sample else budget
        r = oracle.compose(m1, m2, max_raw_arcs=sample, keep_arcs=False)
        line["cpu_baseline"] = {
            "value": r.n_raw_arcs / r.seconds, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"oracle.compose (serial C++, fp64, Algorithm 1) on the same inputs with max_raw_arcs={sample}: "
                      f"{r.n_raw_arcs} raw arcs in {r.seconds:.2f} s on 1 of {os.cpu_count()} cores"}

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
