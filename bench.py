#!/usr/bin/env python
"""bench.py -- headline benchmark: 3pCF triangles/s on BASELINE.json configs[1] (1e6 Neyman-Scott
points, fp64 weights, + an equal-size uniform random catalogue; r<30, 15 bins) on B200.

A "step" is one pass of the whole hot path over the batch: for BOTH catalogues, graph build (cell
list, count, scan, fill) + 3pCF enumeration + fold, through the C ABI.  `value` = triangles counted
per second with the points already resident in HBM; `e2e` = the same through the ABI with pinned HOST
buffers (H2D of points/weights and D2H of the histograms inside the timed region).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2|cfg1|...]

N > 1 (torchrun): the path shards by independent catalogues -- every rank runs the same workload with a
different seed, no data-path collective ("weak" scaling); time = max over ranks.
--impl reference: times the CPU oracle (oracle/) on the host cores on a bounded sample of the workload.
"""
from __future__ import annotations

import argparse
import hashlib
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import catalogues as cat  # noqa: E402


# dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel on cfg2, from the committed
# ncu --set full capture (profiles/r1_c_table_3pcf_full.md)
DRAM_TRAFFIC_BYTES = {"k_3pcf_table<weighted>": 576.641024e6 + 5.040896e6,
                      "k_3pcf_table<counts>": 301.802240e6 + 3.864832e6}


L2_READ_GBS = 12000.0      # L2 -> SM read bandwidth, 16-byte loads over a 32-64 MB working set (same micro-benchmark)
RED_PEAK_GOPS = 193.0      # global RED.E.ADD.(U64|F64), spread addresses, all SMs: best line of the micro-benchmark,
                           # whose loop overhead makes it a slight under-estimate (kernels reach ~1.1 of it)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured", d
    return 6650.0, "fallback", {}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks/throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index = index
        self.rows = []
        self.proc = None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([x.strip() for x in line.split(",")])
        except Exception:
            pass

    def stop(self):
        if self.proc is not None:
            self.proc.terminate()
        self.join(timeout=2)
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = max(mx, float(r[1]))
                for k, nme in enumerate(names):
                    if r[3 + k].lower().startswith("active"):
                        reasons.add(nme)
            except Exception:
                continue
        busy = [x for x in sm if x > 0]
        return {"sm_mhz": float(np.median(busy)) if busy else None, "sm_max_mhz": mx or None,
                "reasons": sorted(reasons), "samples": len(sm)}


def rank_seed_shift(rank: int) -> int:
    """Sharding rule for N > 1: every rank runs the same workload shape on its own seeds (independent
    catalogues, no data-path collective)."""
    return 1000 * rank


def max_over_ranks(value: float, device=None) -> float:
    """Time of a multi-rank step = the slowest rank's device time (all-reduce MAX of one scalar; works on
    the gloo backend with CPU tensors, which is how tests/test_multirank_host.py exercises it)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(value: float, device=None) -> float:
    """Whole-job units processed = sum over ranks (all-reduce SUM of one scalar)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([value], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())


def allreduce_hist(arr, device=None):
    """Strong-scaling mode: every rank enumerates the hubs of its shard of ONE catalogue (shard_count = world,
    shard_index = rank); the histograms add up to the full result with one all-reduce (SUM) -- the only
    collective a multi-GPU run of this path needs."""
    import torch
    import torch.distributed as dist
    t = torch.from_numpy(np.ascontiguousarray(arr))
    if device is not None:
        t = t.to(device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()


def workload(name: str, seed_shift: int = 0):
    """List of catalogues (dicts from catalogues.py) making up one batch."""
    if name == "cfg2":
        return [cat.config2_data(seed=2001 + seed_shift), cat.config2_randoms(seed=2002 + seed_shift)]
    if name == "cfg2small":   # 1/8 replica (same densities) for quick checks
        return [cat.config2_data(seed=2001 + seed_shift, n=125_000, L=500.0, mean_parents=1250.0),
                cat.config2_randoms(seed=2002 + seed_shift, n=125_000, L=500.0)]
    if name == "cfg1":
        return [cat.config1(seed=1001 + seed_shift)]
    if name == "cfg5p":       # scaled replica of configs[4] (same density, L=425)
        return [cat.config5(seed=5001 + seed_shift, n=39_062, L=425.0)]
    if name == "cfg5":        # configs[4] in full: 2.5e6 points, 8.4e9 edges, 42 GB of CSR (use --steps 1 --warmup 0)
        return [cat.config5(seed=5001 + seed_shift)]
    if name == "cfg3":        # configs[2]: 4pCF (+ the 2pCF of the same graph for the disconnected term)
        return [cat.config3(seed=3001 + seed_shift)]
    if name == "cfg4":        # configs[3]: parity-decomposed 4pCF, weighted
        return [cat.config4(seed=4001 + seed_shift)]
    if name == "cfg4s":       # 1/8 replica of configs[3] (same density, 15 x 15 degree cap)
        return [cat.config4(seed=4001 + seed_shift, n=62_500, cap_deg=15.0)]
    raise SystemExit(f"unknown workload {name}")


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """The CPU oracle as it stands, on the host cores, on a bounded sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cats = workload(args.workload)
    stride = args.ref_stride
    tri = 0
    t_total = 0.0
    for _ in range(args.warmup):
        pass  # the oracle has no warm-up state; the build below is part of every step
    per_step = []
    for _ in range(args.steps):
        t0 = time.perf_counter()
        tri = 0
        for c in cats:
            g = oracle.Graph(c["points"], c["weights"], c["box"], c["r_min"], c["r_max"], c["nbins"])
            cnt, _ = g.pcf3(hubs=(0, g.n, stride))
            tri += int(cnt.sum())
            del g
        per_step.append(time.perf_counter() - t0)
    t_total = float(np.mean(per_step))
    value = tri / t_total
    sample = (f"full graph build + 3pCF walk on every {stride}-th hub of each catalogue "
              f"({tri} triangles per step)")
    line = {
        "impl": "reference", "metric": "3pCF triangles/s", "value": value, "unit": "triangles/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "note": "CPU oracle (plain C + OpenMP), not tuned"},
        "cpu_baseline": {"value": value, "unit": "triangles/s", "cores": oracle.threads(), "kind": "oracle",
                         "sample": sample},
        "e2e": {"value": value, "unit": "triangles/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line))


def cpu_baseline(cats, budget_s: float = 20.0):
    import oracle
    t0 = time.perf_counter()
    tri = 0
    # bounded sample (~20 s on 16 cores): the build of the full graph and every hub of each catalogue
    stride = 1
    for c in cats:
        g = oracle.Graph(c["points"], c["weights"], c["box"], c["r_min"], c["r_max"], c["nbins"])
        cnt, _ = g.pcf3(hubs=(0, g.n, stride))
        tri += int(cnt.sum())
        del g
    dt = time.perf_counter() - t0
    return {"value": tri / dt, "unit": "triangles/s", "cores": oracle.threads(), "kind": "oracle",
            "sample": f"oracle graph build + 3pCF walk on every {stride}-th hub of each catalogue: "
                      f"{tri} triangles in {dt:.1f} s"}


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2607_06604_b200 as gr

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the product path has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    gr.load_library()

    strong = args.scaling == "strong" and world > 1
    cats = workload(args.workload, seed_shift=0 if strong else rank_seed_shift(rank))
    dev = [(torch.from_numpy(c["points"]).cuda(), None if c["weights"] is None else torch.from_numpy(c["weights"]).cuda())
           for c in cats]
    pin = [(torch.from_numpy(c["points"]).pin_memory(), None if c["weights"] is None else torch.from_numpy(c["weights"]).pin_memory())
           for c in cats]
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")    # > 126 MB L2
    stats = {}

    def step(host: bool, count_work: bool = False):
        """one pass of the hot path over the batch; returns (triangles, per-step stats, per-catalogue stats)"""
        tri = 0
        st = {"enum_ms": 0.0, "build_ms": 0.0, "query_ms": 0.0, "launches": 0.0, "edges": 0}
        per = []
        digest = hashlib.sha1()
        for c, d, p in zip(cats, dev, pin):
            pts, w = (p if host else d)
            kind = c["kind"]
            g = gr.gramsci_build_graph(pts, w, c["box"], c["r_min"], c["r_max"], c["nbins"], algo=args.algo,
                                       want_pixels=(kind == "4pcf_parity"),
                                       device_mem_cap_bytes=int(args.cap_gib * 2 ** 30),
                                       shard_count=world if strong else 0, shard_index=rank if strong else 0)
            st["build_ms"] += g.timing(0)
            st["launches"] += g.timing(3)
            if kind == "3pcf":
                cnt, ws = g.pcf3(counts=True, weighted=(w is not None), host=host)
            elif kind == "4pcf":
                cnt, ws = g.pcf4(counts=True, weighted=(w is not None), host=host)
            else:
                cnt, _, ws, _ = g.pcf4_parity(counts=True, weighted=(w is not None), host=host)
            if strong:                     # partial histograms of the shards -> full result on every rank
                cnt = allreduce_hist(cnt, "cuda")
                if ws is not None:
                    ws = allreduce_hist(ws, "cuda")
            digest.update(np.ascontiguousarray(cnt).tobytes())
            pc = {"name": c["name"], "enum_ms": g.timing(2), "weighted": w is not None}
            st["enum_ms"] += g.timing(2)
            st["query_ms"] += g.timing(1)
            st["launches"] += g.timing(3)
            t = int(cnt.sum())
            tri += t
            e = g.info()["n_edges"]
            st["edges"] += e
            if count_work:
                sp, tl = g.work_counters() if kind == "3pcf" else (0, 0)
                # algorithmic bytes of the enumeration: spoke rows + hub tails (4 B per
                # element), b_ij per hub-spoke pair, two bin bytes per hit (+ two fp64 weights when weighted)
                pc.update(spoke=sp, tail=tl, edges=e, hits=t,
                          bytes=4.0 * sp + 4.0 * tl + e + 2.0 * t)
            pc["n_windows"] = g.info()["n_windows"]
            pc["staged_bytes"] = g.timing(4)
            per.append(pc)
            g.free()
        stats["sha1"] = digest.hexdigest()
        stats["windows"] = [p_["n_windows"] for p_ in per]
        stats["staged_bytes"] = sum(p_["staged_bytes"] for p_ in per)
        return tri, st, per

    def timed(host: bool, steps: int, warmup: int):
        for _ in range(warmup):
            step(host)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        total_ms, tri, agg, per_agg = 0.0, 0, None, None
        for _ in range(steps):
            flush.fill_(1)                      # flush L2 between timed iterations (not timed)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            tri, st, per = step(host)
            e1.record()
            torch.cuda.synchronize()
            total_ms += e0.elapsed_time(e1)
            agg = st if agg is None else {k: agg[k] + st[k] for k in st}
            per_agg = [p["enum_ms"] for p in per] if per_agg is None else [a + p["enum_ms"] for a, p in zip(per_agg, per)]
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        return (max_over_ranks(total_ms, "cuda") / steps, tri, {k: v / steps for k, v in agg.items()},
                [a / steps for a in per_agg])

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    _, _, work = step(False, count_work=True)       # untimed: exact work counters of this workload
    ms, tri, st, enum_ms = timed(False, args.steps, args.warmup)
    clocks = sampler.stop() if rank == 0 else None
    if args.skip_e2e:
        ms_e2e = None
    else:
        ms_e2e, tri2, _, _ = timed(True, max(1, args.steps // 2), 1)
        assert tri2 == tri
    tri_all = float(tri) if strong else sum_over_ranks(float(tri), "cuda")

    # second headline of BASELINE.json's metric: 4pCF quadruplets/s on configs[2] (query only, rank 0, untimed region)
    four = None
    if rank == 0 and not args.no_4pcf:
        c3 = cat.config3()
        g = gr.gramsci_build_graph(torch.from_numpy(c3["points"]).cuda(), None, c3["box"], c3["r_min"], c3["r_max"], c3["nbins"])
        best = None
        for _ in range(3):
            ec, _ = g.pcf4()
            best = g.timing(1) if best is None else min(best, g.timing(1))
        four = {"workload": "cfg3", "quadruplets": int(ec.sum()), "query_ms": best,
                "quadruplets_per_s": float(ec.sum()) / (best * 1e-3)}
        g.free()

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    peak, peak_kind, peaks = load_peaks()
    h2d = sum(c["points"].nbytes + (0 if c["weights"] is None else c["weights"].nbytes) for c in cats)
    d2h = sum(8 * c["nbins"] ** 3 * (1 if c["weights"] is None else 2) for c in cats)
    # roofline of the dominant kernel = the enumeration launch with the largest share of the step
    dom = max(range(len(cats)), key=lambda k: enum_ms[k])
    dw = work[dom]
    dom_s = enum_ms[dom] * 1e-3
    achieved = dw["bytes"] / dom_s / 1e9
    kind0 = cats[0]["kind"]
    unit = "triangles/s" if kind0 == "3pcf" else "quadruplets/s"
    metric = "3pCF triangles/s" if kind0 == "3pcf" else ("4pCF quadruplets/s" if kind0 == "4pcf" else "parity-4pCF quadruplets/s")
    if kind0 == "3pcf":
        kern = ("k_3pcf_table" if args.algo != 2 else "k_3pcf_bsearch") + ("<weighted>" if dw["weighted"] else "<counts>")
    else:
        kern = "k_4pcf"
    if kind0 == "3pcf":
        roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": DRAM_TRAFFIC_BYTES.get(kern) if args.workload == "cfg2" else None,
                "kernel": f"{kern} on {dw['name']}", "peak_kind": f"hbm copy, {peak_kind}",
                "launch_ms": enum_ms[dom], "algorithmic_bytes_per_launch": dw["bytes"],
                "units_per_launch": {"spoke_row_elements": dw["spoke"], "tail_elements": dw["tail"],
                                     "hub_spoke_pairs": dw["edges"], "hits": dw["hits"]},
                # t_roof = max(CSR once from HBM, spoke rows + hit bytes from L2); fraction = t_roof / t
                "l2_roofline": {"l2_peak_gbs": L2_READ_GBS,
                                "t_roof_ms": 1e3 * max(5.0 * dw["edges"] / (peak * 1e9),
                                                       (4.0 * dw["spoke"] + dw["hits"]) / (L2_READ_GBS * 1e9)),
                                "frac": max(5.0 * dw["edges"] / (peak * 1e9),
                                            (4.0 * dw["spoke"] + dw["hits"]) / (L2_READ_GBS * 1e9)) / dom_s},
                "per_launch": [{"catalogue": w_["name"], "launch_ms": enum_ms[k_], "achieved": w_["bytes"] / (enum_ms[k_] * 1e-3) / 1e9,
                                "frac": w_["bytes"] / (enum_ms[k_] * 1e-3) / 1e9 / peak} for k_, w_ in enumerate(work)],
                "note": "algorithmic bytes = 4*sum len(N+(j)) + 4*sum len(tail) + E + 2*hits (DESIGN.md "
                        "section 6); spoke rows are re-read from L2/L1, so this is an L2->SM figure and may "
                        "exceed the HBM peak; traffic = dram read+write of one ncu --set full launch "
                        "(profiles/)"}
    else:
        # 4pCF kernels are bound by the L2 atomic rate: one RED per hit and output channel;
        # peak = RED.E.ADD.64 rate measured on this pool's B200 by csrc/ubench_atomics.cu (profiles/r1_ubench_atomics.txt)
        # one RED per hit and kind of output (counts, weighted sums); the parity split costs no extra RED: a hit goes
        # to the raw histogram of its sign class and the fold forms even / odd
        ch = 1 if cats[dom]["weights"] is None else 2
        red_rate = dw["hits"] * ch / dom_s / 1e9
        roof = {"bound": "l2-atomics", "achieved": red_rate, "peak": RED_PEAK_GOPS, "unit": "Gatomic/s",
                "frac": red_rate / RED_PEAK_GOPS, "traffic": None, "kernel": f"{kern} on {dw['name']}",
                "launch_ms": enum_ms[dom], "units_per_launch": {"hits": dw["hits"], "channels": ch}}
    line = {
        "metric": metric, "value": tri_all / (ms * 1e-3), "unit": unit,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": args.workload, "catalogues": [c["name"] for c in cats],
                   "n_points": [int(c["points"].shape[0]) for c in cats], "tuples_per_step": tri,
                   "counts_sha1": stats.get("sha1"), "cap_gib": args.cap_gib, "n_windows": stats.get("windows"),
                   "staged_bytes_per_step": stats.get("staged_bytes"),
                   "edges_per_step": st["edges"], "hub_spoke_edges_per_s": st["edges"] / (ms * 1e-3),
                   "step": "graph build + enumeration (3pCF / 4pCF / parity-4pCF by workload) + fold for every "
                   "catalogue", "l2": "flushed between timed steps (256 MiB write); the CSR of the default workload "
                   "(>=0.3 GB per catalogue) exceeds the 126 MB L2",
                   "algo": args.algo, "build_ms": st["build_ms"], "query_ms": st["query_ms"],
                   "enum_kernel_ms": st["enum_ms"], "enum_kernel_ms_per_catalogue": enum_ms,
                   "query_only_tuples_per_s": tri / (st["query_ms"] * 1e-3), "four_pcf": four},
        "clocks": clocks,
        "e2e": None if ms_e2e is None else {"value": tri_all / (ms_e2e * 1e-3), "unit": unit,
                                            "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                                            "ms_per_step": ms_e2e},
        "gpu_launches": int(round(st["launches"] * args.steps)),
        "roofline": roof,
    }
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(cats)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--algo", type=int, default=0)
    ap.add_argument("--ref-stride", type=int, default=1)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-4pcf", action="store_true")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = every rank its own catalogues (default); strong = the hubs of ONE workload "
                         "sharded over the ranks (every rank builds the whole graph), histograms all-reduced")
    ap.add_argument("--skip-e2e", action="store_true", help="big workloads only: no host-buffer leg (e2e = null)")
    ap.add_argument("--cap-gib", type=float, default=0.0,
                    help="device_mem_cap_bytes in GiB (0 = whole CSR resident); forces the out-of-core tiler")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
