#!/usr/bin/env python
"""bench.py -- throughput of the AND/OR-graph pathway traversal (arXiv 1804.02867) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload genome] [--cap 262144]

A *step* is one pass of the whole hot path (roots, classify, beam select, expand, support dedup, minimality filter,
canonical output: SURVEY.md 8(a) rows a-2..a-8) over one seeded synthetic network that is already resident in HBM
(the graph builder a-1 ran before; it is inside the `e2e` figure).  Metric = partial pathways expanded per second,
whole job; EFMs/s and children/s ride along in `extra`.  Prints ONE JSON line on rank 0.

N > 1 (torchrun): the path shards by independent problems -- rank r traverses the network of generator seed r with
the same parameters, no data-path collective, scaling = weak.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores, on bounded samples of the same
workload (same network and parameters, smaller beam), as the tier's reference arm.
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

DEFAULT_CAP = 1 << 24         # frontier_cap of the timed workload: the largest power of two whose workspace fits the 180 GB of
                              # one B200 (153 GB).  If the allocation fails the next smaller power is timed.
PARITY_CAP = 1 << 18          # sweep point at which tests/ compares every output with the oracle (the oracle needs minutes there)
PROPERTY_CAP = 1 << 20        # sweep point at which tests/ checks Def 2 / Def 3 / order on every output
DEFAULT_SWEEP = "262144,1048576,4194304"
DEFAULT_MAX_CANDIDATES = 1 << 22


def sized_params(params, cap, max_candidates=None):
    """Workspace sizing of the genome workload at beam `cap` (the library defaults are worst-case bounds: largest possible
    entry x cap, largest fan-out x cap; measured needs are far smaller and an overflow is a loud EFM_E_CAPACITY)."""
    p = dict(params)
    p["frontier_cap"] = cap
    # balanced pathways found per step: 2.4 x cap at 2^18, 1.9 x at 2^20, 1.4 x at 2^22, 0.93 x at 2^24 (plus duplicates)
    p["max_candidates"] = max(max_candidates or DEFAULT_MAX_CANDIDATES, (4 if cap <= (1 << 22) else 2) * cap)
    if cap >= (1 << 20):
        p["max_frontier_bytes"] = 1792 * cap      # packed entries average about 1 KB
        p["max_child_keys"] = 48 * cap            # about 17 children are evaluated per parent on average, 25 on the widest levels
    return p
WORKLOAD_TEXT = ("{name}-seed{{rank}} (BASELINE.json configs[4]: 1000+150 metabolites, 2000 reactions, 30% reversible, depth cap 60, "
                 "8 target exchange reactions)")
METRIC = "partial_pathways_expanded_per_sec"
UNIT = "expanded/s"


def _peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "100", "-i", str(index)], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for r in self.rows if t0 <= r[0] <= t1 + 0.2] or self.rows
        for _, line in rows:
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                for nm, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                pass
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _workload(name: str, seed: int, cap: int):
    from netgen import make_network
    net = make_network(name, seed)
    params = dict(net.params)
    if cap:
        params["frontier_cap"] = cap
    return net, params


def _oracle_threads():
    import oracle
    return max(1, min(oracle.max_threads(), os.cpu_count() or 1))


def run_oracle_sample(name: str, cap: int):
    """One oracle run on the bounded sample; returns (expanded, seconds, outputs, threads)."""
    import oracle
    oracle.build()
    net, params = _workload(name, 0, cap)
    th = _oracle_threads()
    t = time.time()
    res = oracle.enumerate_pathways(net.S, net.reversible, net.internal, params, net.seed_sets, threads=th,
                                    self_check=False)
    dt = time.time() - t
    return res.stats["expanded"], dt, res.stats["output"], th


def oracle_sample_cap(workload: str, cap: int, steps: int, warmup: int, cores: int) -> int:
    """The bounded sample BOTH oracle legs run (the `cpu_baseline` of the repo arm and every step of `--impl reference`): same
    network and parameters, the largest power-of-two beam with which steps + warmup whole oracle runs end in about 150 s.
    The oracle costs ~2 ms per unit of frontier_cap per 8 threads on the genome network (measured)."""
    budget = 150.0 / max(1, steps + warmup)
    per_cap = {"genome": 2.0e-3, "mid": 1.3e-4, "core": 2.5e-6, "small": 1e-7, "toy": 1e-8}.get(workload, 2e-3) * 8.0 / max(1, cores)
    c = 256
    while c * 2 <= cap and c * 2 * per_cap <= budget:
        c *= 2
    return c


def main_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cores = _oracle_threads()
    cap = oracle_sample_cap(args.workload, args.cap, args.steps, max(args.warmup, 3), cores)   # as the repo arm's cpu_baseline
    for _ in range(args.warmup):
        run_oracle_sample(args.workload, cap)
    t_sum, exp_sum, outs = 0.0, 0, 0
    for _ in range(args.steps):
        e, dt, outs, _th = run_oracle_sample(args.workload, cap)
        t_sum += dt
        exp_sum += e
    value = exp_sum / t_sum
    sample = f"same network/parameters as config.workload, frontier_cap {cap} instead of {args.cap}; whole oracle run per step"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1000.0 * t_sum / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int64", "data": "synthetic",
            "config": {"workload": WORKLOAD_TEXT.format(name=args.workload), "frontier_cap": args.cap, "reference_sample_cap": cap},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "extra": {"efms_per_s": outs * args.steps / t_sum}}
    print(json.dumps(line))
    return 0


def reduce_over_ranks(times_ms, counts, dist, device):
    """Whole-job figures of a replica run: every time is the MAX over ranks, every count the SUM over ranks
    (rank r works on its own independent problem).  `dist` is torch.distributed or None."""
    import torch
    if dist is None:
        return list(times_ms) + list(counts)
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    c = torch.tensor(list(counts), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return t.tolist() + c.tolist()


def agreed_cap(cap_used: int, dist, device) -> int:
    """The beam every replica times: the smallest one any rank had to fall back to (MIN over ranks), so that the summed
    throughput describes ONE configuration.  `dist` is torch.distributed or None."""
    import torch
    if dist is None:
        return int(cap_used)
    t = torch.tensor([int(cap_used)], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return int(t.item())


def rank_problem(workload: str, rank: int, cap: int):
    """The independent problem rank `rank` owns: the synthetic network of generator seed `rank`."""
    return _workload(workload, rank, cap)


def main_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1804_02867_b200 import build
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    import paper_1804_02867_b200 as efm

    # rank r owns the independent problem of generator seed r (weak scaling, no collective on the data path)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")   # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def make_enumerator(cap):
        net_, params_ = rank_problem(args.workload, rank, cap)
        if args.workload == "genome":
            params_ = sized_params(params_, cap, args.max_candidates)
        else:
            params_["max_candidates"] = args.max_candidates
        return net_, params_, efm.Enumerator(net_.S, net_.reversible, net_.internal, params_, device=local, flags=efm.EFM_F_TIMING)

    # the largest beam whose workspace this GPU can hold right now: the requested one, else the next smaller powers of two
    cap_used, fallback_note = args.cap, None
    while True:
        net, params, en = make_enumerator(cap_used)
        try:
            en.enumerate(net.seed_sets, dense=False)
            break
        except (torch.cuda.OutOfMemoryError, efm.EfmError) as exc:
            if isinstance(exc, efm.EfmError) and exc.code not in (efm.EFM_E_NOMEM, efm.EFM_E_CUDA):
                raise
            en.close()
            del en
            torch.cuda.empty_cache()
            if cap_used <= (1 << 18):
                raise
            fallback_note = f"frontier_cap {args.cap} did not fit ({type(exc).__name__}); timed {cap_used // 2}"
            cap_used //= 2
    if world > 1:
        # replicas time ONE configuration: every rank takes the smallest beam any rank had to fall back to
        agreed = agreed_cap(cap_used, dist, torch.device("cuda"))
        if agreed != cap_used:
            en.close()
            del en
            torch.cuda.empty_cache()
            cap_used = agreed
            fallback_note = f"frontier_cap {args.cap} did not fit on every rank; all ranks timed {cap_used}"
            net, params, en = make_enumerator(cap_used)
            en.enumerate(net.seed_sets, dense=False)
    args.cap = cap_used
    for _ in range(max(args.warmup, 3) - 1):
        en.enumerate(net.seed_sets, dense=False)
    # ---- device-resident figure: K steps, each timed by the library with CUDA events on the launching stream
    sampler = ClockSampler(local) if rank == 0 else None
    barrier()
    t0 = time.time()
    ms = 0.0
    acc = {}
    for _ in range(args.steps):
        flush.fill_(1)   # evict L2 between timed iterations (not timed)
        torch.cuda.synchronize()
        st = en.enumerate(net.seed_sets, dense=False).stats
        ms += st["ms_total"]
        for k, v in st.items():
            acc[k] = acc.get(k, 0) + v
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    # ---- end to end through the public API with HOST buffers: graph build from S, upload, traversal, result D2H
    e2e_s = 0.0
    h2d = d2h = 0
    for it in range(args.steps + 1):   # iteration 0 is an untimed warm-up (pinned result buffers get allocated)
        flush.fill_(1)
        torch.cuda.synchronize()
        t = time.time()
        en2 = efm.Enumerator(net.S, net.reversible, net.internal, params, device=local)
        t_a = time.time()
        en2._workspace = en._workspace          # device memory is allocated once by torch, outside the step
        en2._lib.efm_workspace_invalidate(en2._h)
        r2 = en2.enumerate(net.seed_sets, dense=False)
        t_b = time.time()
        row_ptr, rxn, val = en2.result_csr(pinned=True)   # compressed rows into pinned host memory
        e2e_s += (time.time() - t) if it > 0 else 0.0
        e2e_parts = (t_a - t, t_b - t_a, time.time() - t_b)
        gi = en2.graph_info()
        h2d = int(r2.stats["h2d_bytes"]) + net.S.nbytes   # counted by the library from the copies it makes, plus S itself (host)
        d2h = (row_ptr.numel() * 8 + rxn.numel() * 4 + val.numel() * 8 + int(r2.stats["levels"]) * 256)
        del row_ptr, rxn, val   # back to torch's pinned-memory cache: the next step reuses the buffers
        en2.close()
        en2._workspace = None
    barrier()

    ms_max, e2e_ms_max, expanded_all, outputs_all, children_all = reduce_over_ranks(
        [ms, e2e_s * 1000.0], [float(acc["expanded"]), float(acc["output"]), float(acc["children"])],
        dist if world > 1 else None, torch.device("cuda", local))

    # ---- other beam sizes of the same workload (rank 0, one warm-up + two timed steps each): the curve the headline sits on
    sweep = []
    if rank == 0 and args.sweep:
        ws_bytes = en.workspace_bytes()
        en.close()
        en._workspace = None
        torch.cuda.empty_cache()
        for cap_s in [int(x) for x in args.sweep.split(",") if x]:
            if cap_s == args.cap:
                continue
            try:
                net_s, params_s, en_s = make_enumerator(cap_s)
                en_s.enumerate(net_s.seed_sets, dense=False)
                tot, acc_s = 0.0, {}
                for _ in range(2):
                    flush.fill_(1)
                    torch.cuda.synchronize()
                    st = en_s.enumerate(net_s.seed_sets, dense=False).stats
                    tot += st["ms_total"]
                    for k, v in st.items():
                        acc_s[k] = acc_s.get(k, 0) + v
                ms_e = acc_s["ms_order"] + acc_s["ms_expand_count"] + acc_s["ms_expand_write"]
                sweep.append({"frontier_cap": cap_s, "ms_per_step": tot / 2, "value": acc_s["expanded"] / (tot * 1e-3),
                              "outputs_per_step": acc_s["output"] / 2, "levels": acc_s["levels"] / 2,
                              "roofline_frac": acc_s["algo_bytes"] / (ms_e * 1e-3) / 1e9 / _peaks()[0],
                              "filter_share": acc_s["ms_filter"] / tot, "workspace_bytes": en_s.workspace_bytes()})
                en_s.close()
                del en_s
                torch.cuda.empty_cache()
            except Exception as exc:   # a sweep point never takes the headline down
                sweep.append({"frontier_cap": cap_s, "error": f"{type(exc).__name__}: {exc}"[:200]})
    else:
        ws_bytes = en.workspace_bytes()

    if rank == 0:
        peak, peak_src = _peaks()
        # one "launch" of the expansion = k_order + k_expand (evaluate) + k_compact + k_materialise of one level
        n_exp_launch = max(1.0, acc["levels"] - args.steps)   # the last level of a traversal has nothing to expand
        ms_expand = acc["ms_order"] + acc["ms_expand_count"] + acc["ms_expand_write"]
        achieved = acc["algo_bytes"] / (ms_expand * 1e-3) / 1e9 if ms_expand > 0 else 0.0
        # dram__bytes_read + write of the four kernels over one full level, from the committed ncu --set full capture of
        # this workload (profiles/r2_traffic.json names the summary it was read from); null for any other configuration
        traffic, traffic_src = args.traffic, "--traffic"
        if traffic is None:
            traffic_src = None
            try:
                with open(os.path.join(ROOT, "profiles", "r2_traffic.json")) as fh:
                    tj = json.load(fh)
                if args.workload == tj["workload"] and args.cap == tj["frontier_cap"]:
                    traffic, traffic_src = float(tj["dram_bytes_per_full_level"]), tj["source"]
            except Exception:
                pass
        roofline = {"bound": "hbm", "kernel": "expansion of one level: k_order + k_expand (evaluate) + k_compact + k_materialise", "achieved": achieved,
                    "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                    "peak_source": peak_src, "launches_per_step": n_exp_launch / args.steps,
                    "avg_launch_ms": ms_expand / max(1, n_exp_launch),
                    "algo_bytes_per_launch": acc["algo_bytes"] / max(1, n_exp_launch),
                    "share_of_step": ms_expand / ms if ms else None}
        # the oracle as it stands on this box's host cores, bounded sample of the same workload
        cpu = None
        if not args.no_cpu_baseline:
            # the same sample as a step of `--impl reference` under the same --steps / --warmup, repeated up to ~10 s of CPU work
            cap_s = oracle_sample_cap(args.workload, args.cap, args.steps, max(args.warmup, 3), _oracle_threads())
            e = dt = runs = 0
            while dt < 10.0 and runs < 8:
                e1, dt1, outs, th = run_oracle_sample(args.workload, cap_s)
                e, dt, runs = e + e1, dt + dt1, runs + 1
            cpu = {"value": e / dt, "unit": UNIT, "cores": th, "kind": "oracle",
                   "sample": f"same network/parameters, frontier_cap {cap_s} instead of {args.cap} (the sample of --impl reference); "
                             f"{runs} whole oracle runs ({dt:.1f} s, {e} expansions, {outs} outputs each)"}
        line = {"metric": METRIC, "value": expanded_all / (ms_max * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "int64", "data": "synthetic",
                "config": {"workload": WORKLOAD_TEXT.format(name=args.workload),
                           "frontier_cap": args.cap, "fallback": fallback_note, "workspace_bytes": int(ws_bytes),
                           "params": {k: int(v) for k, v in params.items()},
                           "l2": "flushed between timed iterations (256 MiB write)", "parallelism": f"replicas x{world}"},
                "clocks": clocks,
                "e2e": {"value": expanded_all / (e2e_ms_max * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                        "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_ms_max / args.steps,
                        "what": "efm_create (graph builder from host S) + efm_enumerate (graph upload + traversal) + "
                                "efm_result_copy_csr to pinned host memory, wall clock",
                        "parts_ms_last_step": {"efm_create": 1e3 * e2e_parts[0], "efm_enumerate": 1e3 * e2e_parts[1],
                                               "result_copy": 1e3 * e2e_parts[2]}},
                "gpu_launches": int(acc["launches"]),
                "roofline": roofline,
                "cpu_baseline": cpu,
                "extra": {"efms_per_s": outputs_all / (ms_max * 1e-3), "children_per_s": children_all / (ms_max * 1e-3),
                          "outputs_per_step": outputs_all / args.steps / world, "levels": acc["levels"] / args.steps,
                          "phase_ms_per_step": {k: acc[k] / args.steps for k in
                                                ("ms_order", "ms_expand_count", "ms_beam", "ms_expand_write", "ms_hash",
                                                 "ms_filter", "ms_output")},
                          "phase_names": {"ms_order": "k_order", "ms_expand_count": "k_expand", "ms_beam": "k_select_*", "ms_expand_write":
                                          "k_compact + k_materialise", "ms_hash": "k_dedup_*", "ms_filter": "k_filter_*",
                                          "ms_output": "k_out_* + k_bitonic_*"},
                          "work_profile_per_step": {k: acc[k] / args.steps for k in
                                                    ("expanded", "first_visits", "general_children", "materialised")},
                          "sweep": sweep, "host_syncs_per_step": acc["host_syncs"] / args.steps,
                          "filter_pairs_per_s": (acc["filter_pairs"] / (acc["ms_filter"] * 1e-3)) if acc["ms_filter"] else None}}
        print(json.dumps(line))
    if en._h:
        en.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="genome", choices=["toy", "small", "core", "mid", "genome"])
    ap.add_argument("--cap", type=int, default=DEFAULT_CAP, help="frontier_cap (beam) of the workload")
    ap.add_argument("--max-candidates", type=int, default=DEFAULT_MAX_CANDIDATES)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", default=DEFAULT_SWEEP, help="comma-separated frontier_cap values also timed (rank 0; '' = none)")
    ap.add_argument("--traffic", type=float, default=None,
                    help="ncu dram bytes per expansion of a level (default: the profiles/ capture of the default workload)")
    args = ap.parse_args()
    if args.impl == "reference":
        return main_reference(args)
    return main_ours(args)


if __name__ == "__main__":
    sys.exit(main())
