#!/usr/bin/env python
"""bench.py -- throughput of the phase-tracking hot path (DE fit of every block + Doppler products).

One "step" = one pass of the whole hot path over one synthetic track: pt_fit_blocks (the persistent
DE kernel) followed by pt_doppler_products.  Default workload = BASELINE.json config 2, the one-hour
track the target is quoted on (3600 blocks x 16000 samples, NP = 128, D = 5, 1000 generations).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload config2|config1|config3s]

Prints ONE JSON line (rank 0).  `value` = candidate-sample fitness evaluations per second (whole job, inputs
resident in HBM); `e2e` = the same metric through pt_track_host with pinned HOST buffers (copies inside the
timed region); `roofline` = the DE kernel against the XU (MUFU) issue roofline of the B200;
`cpu_baseline` = the fp64 oracle on the host cores on a bounded sample.
Under torchrun each rank fits its own track (weak scaling; no data-path collective).
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

METRIC = "candidate-sample fitness evals/sec"
UNIT = "sample-evals/s"
SM_COUNT = 148
XU_LANES_PER_SM = 16            # MUFU lanes per SM (4 per sub-partition): one cosine per sample-evaluation
SM_MAX_MHZ = 1965.0
XU_PEAK = SM_COUNT * XU_LANES_PER_SM * SM_MAX_MHZ * 1e6     # 4.65e12 sample-evaluations/s, DESIGN.md "Roofline"
# dram__bytes_read.sum + dram__bytes_write.sum of the DE-kernel launches of one step, from an `ncu --set full` capture of the
# same command (profile file named beside the number); reported as roofline.traffic_ncu, never as a live measurement
NCU_TRAFFIC = {"config2": {"bytes": 2.497e8, "source": "profiles/r2_bench_launches.md (the two DE-kernel launches of one step: 243.5 MB read + 6.1 MB written)"}}


def kernel_name(plan: dict, wl) -> str:
    """Which evaluation kernel the plan runs (include/pt.h, pt_fit_blocks_launches): told from its geometry."""
    obj = "cor" if wl.de["objective"] else "chi2"
    if plan["threads"] == 640:
        return "pt_tc_kernel<D=%d,fit,%s> (phase by tcgen05.mma kind::tf32)" % (wl.de["D"], obj)
    if plan["cands_per_thread"] == 1:
        return "pt_run_kernel<D=%d,fit,%s,%s> (thread = candidate, run-local Horner)" % (wl.de["D"], "resident" if plan["resident"] else "streamed", obj)
    return "pt_block_kernel<C=%d,D=%d,fit,%s>" % (plan["cands_per_thread"], wl.de["D"], obj)


def peak_probe(kind: int) -> float:
    """Measured ALU stream rate of the device (bench-only library libpt_probe.so): kind 0 FFMA, kind 1 MUFU.COS."""
    import ctypes as C
    from paper_1906_10598_b200 import build as _b
    lib = C.CDLL(_b.build_probe())
    lib.pt_bench_peak_probe.argtypes = [C.c_int32, C.c_void_p]
    lib.pt_bench_peak_probe.restype = C.c_int32
    v = C.c_double(0.0)
    rc = lib.pt_bench_peak_probe(int(kind), C.byref(v))
    if rc != 0:
        raise RuntimeError("pt_bench_peak_probe failed (%d)" % rc)
    return float(v.value)


def sm_clock_probe(with_mma: bool) -> float:
    """SM clock [MHz] a MUFU-bound kernel runs at, measured in-kernel (clock64 / globaltimer), without and with tcgen05.mma activity."""
    import ctypes as C
    from paper_1906_10598_b200 import build as _b
    lib = C.CDLL(_b.build_probe())
    lib.pt_bench_sm_clock.argtypes = [C.c_int32, C.c_void_p]
    lib.pt_bench_sm_clock.restype = C.c_int32
    v = C.c_double(0.0)
    rc = lib.pt_bench_sm_clock(1 if with_mma else 0, C.byref(v))
    if rc != 0:
        raise RuntimeError("pt_bench_sm_clock failed (%d)" % rc)
    return float(v.value)


def algorithmic_traffic(wl, quant_bits: int = 0) -> float:
    """Bytes one step must move through HBM: every sample once, the boxes, and the per-block outputs."""
    D = wl.de["D"]
    samples = wl.B * wl.N * (quant_bits / 8.0 if quant_bits else 4.0)
    return float(samples + wl.B * (2 * D * 8 + D * 8 + 4 + 4))


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


def make_workload(name: str, case: int):
    from paper_1906_10598_b200 import workloads as W
    if name == "config2":
        return W.config2(case=case)
    if name == "config1":
        return W.config1(case=case)
    if name == "config3s":       # a 3600-block slice of config 3 around the occultation (D = 6)
        return W.config3(blocks=range(16200, 19800), case=case)
    if name == "config2_ncu":    # one wave of config-2 blocks, 100 generations: short enough for `ncu --set full`
        return W.config2(blocks=range(148), case=case, generations=100)
    if name == "config3_ncu":    # one wave of config-3 blocks (D = 6) around the occultation, 100 generations
        return W.config3(blocks=range(17926, 18074), case=case, generations=100)
    if name == "paper_ncu":      # paper-shaped blocks (streamed, D = 6, NP = 400), 10 generations: short enough for `ncu --set full`
        wl = W.paper_blocks(B=148, case=case)
        wl.de["generations"] = 10
        return wl
    if name == "config1_ncu":    # config 1 (60 blocks: clusters of 2 CTAs per block), 100 generations
        return W.config1(case=case, generations=100)
    if name == "sweep1k_ncu":    # config-4 sweep point N = 1024, NP = 128 (8 CTAs of 128 threads per SM)
        return W.config4(1024, 128, B=1024, generations=200)
    if name == "config2_2w":     # two waves of config-2 blocks (the tensor-core kernel fits two blocks per CTA at a time)
        return W.config2(blocks=range(296), case=case, generations=100)
    if name == "config3_2w":
        return W.config3(blocks=range(17852, 18148), case=case, generations=100)
    if name == "config3":        # BASELINE config 3 at full size: 36000 blocks x 10000 samples, D = 6, 1500 generations
        return W.config3(case=case)
    if name == "paper":          # the paper's own block shape and Table 4 settings
        return W.paper_blocks(B=148, case=case)
    if name == "tiny":           # for CPU-side plumbing tests
        return W.config2(blocks=range(4), case=case, generations=3)
    raise SystemExit("unknown workload %s" % name)


def apply_variant(wl, strategy: int, objective: str, fix_a1: bool = False):
    """--strategy / --objective: the widened rows.  For the correlation objective the amplitude
    is fixed (Eq. 6): a0 = the profile's amplitude at the block centre, a1 = 0, zero-width boxes."""
    wl.de["strategy"] = int(strategy) if strategy else int(wl.de.get("strategy", 1))
    wl.de["objective"] = 1 if objective == "cor" else 0
    if fix_a1:          # amplitude slope fixed at zero: the kernel takes its constant-amplitude loop
        wl.lo = wl.lo.copy(); wl.hi = wl.hi.copy()
        wl.lo[:, 1] = wl.hi[:, 1] = 0.0
        wl.meta["fix_a1"] = True
    if objective == "cor":
        wl.lo = wl.lo.copy(); wl.hi = wl.hi.copy()
        wl.lo[:, 0] = wl.hi[:, 0] = wl.truth[:, 0]
        wl.lo[:, 1] = wl.hi[:, 1] = 0.0
    return wl


def sample_evals(wl) -> float:
    return float(wl.B) * wl.de["NP"] * (wl.de["generations"] + 1) * wl.N


class ClockSampler:
    """nvidia-smi clocks / throttle reasons while the timed region runs (B200_PROFILING.md recipe)."""

    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu_index = gpu_index
        self.proc = None
        self.lines = []
        self.thread = None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu_index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "200"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            tok = [t.strip() for t in ln.split(",")]
            if len(tok) < 9:
                continue
            try:
                sm.append(float(tok[1])); smax.append(float(tok[2])); power.append(float(tok[3]))
            except ValueError:
                continue
            for nm, v in zip(names, tok[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = [c for c, p in zip(sm, power) if p >= 0.5 * max(power)] or sm
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "power_w_max": float(max(power)), "samples": len(sm)}


def cpu_baseline(wl, budget_blocks=None, generations=200) -> dict:
    """The fp64 oracle, as it stands, on the host cores: DE on the first `cores` blocks of the workload for a
    reduced generation count (the metric is a rate, every generation costs the same)."""
    import oracle
    cores = oracle.num_threads()
    nb = min(wl.B, budget_blocks or cores)
    # bounded sample: about 2e10 sample-evaluations (10-30 s at the ~1e9/s the oracle reaches on 16 cores)
    G = int(max(2, min(generations, wl.de["generations"], 2e10 * cores / 16 / (float(nb) * wl.de["NP"] * wl.N) - 1)))
    t0 = time.perf_counter()
    oracle.fit_blocks(wl.x[:nb], wl.fs, wl.lo[:nb], wl.hi[:nb], NP=wl.de["NP"], generations=G, F=wl.de["F"],
                      CR=wl.de["CR"], seed=1, block_index=wl.block_index[:nb], strategy=wl.de.get("strategy", 1),
                      objective=wl.de.get("objective", 0))
    dt = time.perf_counter() - t0
    units = float(nb) * wl.de["NP"] * (G + 1) * wl.N
    return {"value": units / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "DE fit of blocks 0..%d of %s for %d of %d generations (fp64 C oracle, OpenMP over blocks), %.1f s"
                      % (nb - 1, wl.name, G, wl.de["generations"], dt)}


def run_reference(args, rank: int, world: int):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    if rank != 0:
        return
    import oracle
    from paper_1906_10598_b200 import workloads as W
    cores = oracle.num_threads()
    nb = max(1, min(cores, 64))
    if args.workload == "paper":
        wl = W.paper_blocks(B=nb)
    elif args.workload == "config1":
        wl = W.config1(blocks=range(min(nb, 60)))
    elif args.workload == "config3s":
        wl = W.config3(blocks=range(16200, 16200 + nb))
    elif args.workload == "tiny":
        wl = W.config2(blocks=range(2), generations=3)
    else:
        wl = W.config2(blocks=range(nb))
    wl = apply_variant(wl, args.strategy, args.objective, args.fix_a1)
    # bounded sample per step: about 2e10 sample-evaluations at most (10-30 s on 16 cores)
    G = int(max(2, min(wl.de["generations"], args.ref_generations, 2e10 * cores / 16 / (float(wl.B) * wl.de["NP"] * wl.N) - 1)))
    units = float(wl.B) * wl.de["NP"] * (G + 1) * wl.N
    times = []
    for it in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        res = oracle.fit_blocks(wl.x, wl.fs, wl.lo, wl.hi, NP=wl.de["NP"], generations=G, F=wl.de["F"], CR=wl.de["CR"],
                                seed=1, block_index=wl.block_index, strategy=wl.de["strategy"], objective=wl.de["objective"])
        oracle.doppler_products(res["best"], wl.T, 0.0, [1])
        dt = time.perf_counter() - t0
        if it >= args.warmup:
            times.append(dt)
    ms = 1e3 * float(np.mean(times))
    value = units / (ms * 1e-3)
    sample = ("each step = DE fit of %d blocks of %s for %d of %d generations (fp64 C oracle, OpenMP over blocks)"
              % (wl.B, wl.name, G, wl.de["generations"]))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(args.workload, wl, full=False),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_sweep(args, dev):
    """BASELINE.json config 4: block length x population sweep, 1024 blocks per launch, D = 5, 200 generations.
    One JSON line: `points` = fitness evals/s and XU-roofline fraction of every (N, NP); `value` = all points together."""
    import torch
    from paper_1906_10598_b200 import pt, workloads as W
    Ns = [int(v) for v in args.sweep_n.split(",")]
    NPs = [int(v) for v in args.sweep_np.split(",")]
    B, G = args.sweep_blocks, args.sweep_generations
    points, tot_units, tot_ms, n_launches = [], 0.0, 0.0, 0
    sampler = ClockSampler(dev.index or 0)
    sampler.start()
    for N in Ns:
        wl = W.config4(N, NPs[0], B=B, generations=G)
        x, lo, hi = (torch.from_numpy(a).to(dev) for a in (wl.x, wl.lo, wl.hi))
        for NP in NPs:
            cfg = pt.make_config(D=5, NP=NP, generations=G, F=0.5, CR=0.9, seed=1, t0=wl.t0)
            plan = pt.pt_fit_blocks_plan(B, N, cfg)
            launches = pt.pt_fit_blocks_launches(B, N, cfg)
            for _ in range(max(1, args.warmup if N * NP < 2 ** 22 else 1)):
                pt.pt_fit_blocks(x, wl.fs, lo, hi, cfg)
            torch.cuda.synchronize()
            steps = args.steps if N * NP < 2 ** 24 else 1
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(steps):
                r = pt.pt_fit_blocks(x, wl.fs, lo, hi, cfg)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / steps
            n_launches += steps * len(launches)
            units = float(B) * NP * (G + 1) * N
            rate = units / (ms * 1e-3)
            tot_units += units
            tot_ms += ms
            ok = float((r["best_rss"] > 0).float().mean().item())
            points.append({"N": N, "NP": NP, "ms": ms, "sample_evals_per_s": rate, "fitness_evals_per_s": rate / N,
                           "xu_frac": rate / XU_PEAK, "resident": plan["resident"], "threads": plan["threads"],
                           "ctas_per_sm": plan["ctas_per_sm"], "smem": plan["smem"], "launches": len(launches), "finite": ok})
        del x
    clocks = sampler.stop()
    line = {"metric": METRIC, "value": tot_units / (tot_ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tot_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": "BASELINE.json config 4 (throughput sweep)", "blocks": B, "generations": G, "D": 5,
                       "N": Ns, "NP": NPs, "l2": "block samples staged once (resident) or streamed from L2/HBM every generation"},
            "roofline": {"bound": "alu", "peak": XU_PEAK / 1e12, "unit": "T sample-evals/s (1 MUFU cosine each)",
                         "achieved": tot_units / (tot_ms * 1e-3) / 1e12, "frac": tot_units / (tot_ms * 1e-3) / XU_PEAK,
                         "traffic": None},
            "points": points, "clocks": clocks, "gpu_launches": n_launches}
    print(json.dumps(line), flush=True)


def run_strong(args, rank: int, local_rank: int, world: int, dev):
    """--scaling strong: one track (config2 / config3 / config3s) split over the ranks.  Each rank synthesises and fits only its
    contiguous range of blocks (the Philox counter carries the block's index in the full track, so the split draws the random
    numbers of the unsplit fit); the one exchange of the path is the all-gather of best[B][D] before the Doppler products."""
    import torch
    import torch.distributed as dist
    from paper_1906_10598_b200 import pt, shard, workloads as W
    if not dist.is_initialized():
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29541")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=dev)
    full = {"config2": (W.config2, range(3600)), "config3": (W.config3, range(36000)), "config3s": (W.config3, range(16200, 19800)),
            "tiny": (lambda **k: W.config2(generations=3, **k), range(8))}
    if args.workload not in full:
        raise SystemExit("--scaling strong takes --workload config2 | config3 | config3s")
    make, blocks = full[args.workload]
    blocks = list(blocks)
    B = len(blocks)
    mine = shard.block_range(B, rank, world)
    wl = apply_variant(make(blocks=[blocks[k] for k in mine]), args.strategy, args.objective, args.fix_a1)
    cfg = pt.make_config(D=wl.de["D"], NP=wl.de["NP"], generations=wl.de["generations"], F=wl.de["F"], CR=wl.de["CR"], seed=1,
                         t0=wl.t0, strategy=wl.de["strategy"], objective=wl.de["objective"])
    m_int = [max(1, int(round(tc / wl.T))) for tc in (1.0, 10.0, 60.0)]
    x_h, lo_h, hi_h = (torch.from_numpy(a).pin_memory() for a in (wl.x, wl.lo, wl.hi))
    x, lo, hi = x_h.to(dev), lo_h.to(dev), hi_h.to(dev)
    units = float(B) * wl.de["NP"] * (wl.de["generations"] + 1) * wl.N

    def step(xd, lod, hid):
        r = shard.fit_track_sharded(xd, wl.fs, lod, hid, cfg, B)          # block_index = position in the full track
        return r, pt.pt_doppler_products(r["best"], wl.T, 0.0, m_int)

    def barrier():
        dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step(x, lo, hi)
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        r, prod = step(x, lo, hi)
    e1.record()
    barrier()
    clocks = sampler.stop()
    tt = torch.tensor([e0.elapsed_time(e1)], dtype=torch.float64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    ms_per_step = float(tt.item()) / args.steps
    # end to end: this rank's samples from pinned host memory, sharded fit, products, results back on the host
    barrier()
    t0 = time.perf_counter()
    n_e2e = max(1, min(args.steps, 2))
    for _ in range(n_e2e):
        r, prod = step(x_h.to(dev, non_blocking=True), lo_h.to(dev, non_blocking=True), hi_h.to(dev, non_blocking=True))
        out = [r["best"].cpu(), r["best_rss"].cpu(), r["status"].cpu(), prod[0].cpu(), prod[1].cpu()] + [v.cpu() for v in prod[2]]
    barrier()
    tt = torch.tensor([(time.perf_counter() - t0) / n_e2e], dtype=torch.float64, device=dev)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    e2e_s = float(tt.item())
    if rank == 0:
        value = units / (ms_per_step * 1e-3)
        cfgd = workload_config(args.workload, wl)
        cfgd["blocks"] = B
        cfgd["parallelism"] = ("one track split into contiguous block ranges over %d rank(s); one all-gather of best[B][D] (%.2f MB, NCCL) "
                               "before the Doppler products" % (world, B * wl.de["D"] * 8 / 1e6))
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32",
                "data": "synthetic", "config": cfgd, "real_time_factor": B * wl.T / (ms_per_step * 1e-3),
                "roofline": {"bound": "alu", "achieved": value / 1e12, "peak": world * XU_PEAK / 1e12,
                             "unit": "T sample-evals/s (1 MUFU cosine each)", "frac": value / (world * XU_PEAK),
                             "traffic": algorithmic_traffic(wl) * B / max(1, wl.B)},
                "clocks": clocks,
                "e2e": {"value": units / e2e_s, "unit": UNIT, "ms_per_step": 1e3 * e2e_s,
                        "h2d_bytes_per_step": int(sum(t.numel() * t.element_size() for t in (x_h, lo_h, hi_h))),
                        "d2h_bytes_per_step": int(sum(t.numel() * t.element_size() for t in out))},
                # this rank's DE-kernel launches + 2 Doppler kernels + one kernel per integration interval, per step
                "gpu_launches": args.steps * (len(pt.pt_fit_blocks_launches(wl.B, wl.N, cfg)) + 2 + len([m for m in m_int if B // m > 0]))}
        print(json.dumps(line), flush=True)
    dist.destroy_process_group()


def workload_config(name: str, wl, full=True) -> dict:
    return {"workload": "BASELINE.json config 2 (one-hour track)" if name == "config2" else name,
            "strategy": wl.de.get("strategy", 1), "a1": "fixed at 0" if wl.meta.get("fix_a1") else "free", "objective": "cor (Eq. 5-6)" if wl.de.get("objective", 0) else "chi2 (Eq. 4)",
            "blocks": wl.B if full else "%d (sample)" % wl.B, "samples_per_block": wl.N, "fs_hz": wl.fs,
            "NP": wl.de["NP"], "D": wl.de["D"], "generations": wl.de["generations"], "F": wl.de["F"], "CR": wl.de["CR"],
            "box": "tracking ranges (PAPER.md:191-197) about the truth" if wl.meta.get("box") == "tracking" else
            "literal +-20% around the analytic profile", "l2": "inputs_exceed_l2" if wl.x.nbytes > 126e6 else
            "inputs_fit_l2 (block samples are staged once into shared memory; HBM traffic is negligible)",
            "parallelism": "one persistent CTA per data block; ranks fit independent tracks"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2")
    ap.add_argument("--ref-generations", type=int, default=100)
    ap.add_argument("--strategy", type=int, default=0, help="mutation strategy 1..6 (Table 4); 0 = the workload's own (DE/rand/1)")
    ap.add_argument("--quant", type=int, default=0, choices=[0, 1, 2, 4, 8, 16],
                    help="feed packed samples of this many bits (Table 3 formats, pt_fit_blocks_q / pt_track_host_q)")
    ap.add_argument("--fix-a1", action="store_true", help="fix the amplitude slope at zero (a1 box [0, 0], PAPER.md:139)")
    ap.add_argument("--objective", default="chi2", choices=["chi2", "cor"], help="Eq. 4 (default) or Eq. 5-6")
    ap.add_argument("--kernel", default="auto", choices=["auto", "run", "tc", "classic"],
                    help="force the forward-difference (pt_run_kernel), tensor-core (pt_tc_kernel) or FP32-pipe Horner (pt_block_kernel) "
                         "evaluation kernel (PT_KERNEL hook)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="weak: every rank fits its own track (default); strong: ONE track split into contiguous block ranges over "
                         "the ranks (shard.fit_track_sharded), all-gather of the fitted parameters before the Doppler products")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--sweep-n", default="1024,4096,16384,65536,262144")
    ap.add_argument("--sweep-np", default="32,64,128,256,512")
    ap.add_argument("--sweep-blocks", type=int, default=1024)
    ap.add_argument("--sweep-generations", type=int, default=200)
    args = ap.parse_args()

    if args.kernel != "auto":
        os.environ["PT_KERNEL"] = args.kernel
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))

    if args.impl == "reference":
        run_reference(args, rank, world)
        return

    import torch
    from paper_1906_10598_b200 import pt

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    pt.lib()                                              # fail loudly if the CUDA library is missing
    if args.workload == "sweep":
        if world > 1:
            raise SystemExit("--workload sweep is a 1-GPU report")
        run_sweep(args, dev)
        return
    if args.scaling == "strong":
        run_strong(args, rank, local_rank, world, dev)
        return
    wl = apply_variant(make_workload(args.workload, case=rank), args.strategy, args.objective, args.fix_a1)   # every rank fits its own track
    cfg = pt.make_config(D=wl.de["D"], NP=wl.de["NP"], generations=wl.de["generations"], F=wl.de["F"], CR=wl.de["CR"],
                         seed=1 + rank, t0=wl.t0, strategy=wl.de["strategy"], objective=wl.de["objective"])
    plan = pt.pt_fit_blocks_plan(wl.B, wl.N, cfg)
    launches = pt.pt_fit_blocks_launches(wl.B, wl.N, cfg)
    plan["launches"] = launches
    m_int = [max(1, int(round(tc / wl.T))) for tc in (1.0, 10.0, 60.0)]
    quant, qkw = None, {}
    if args.quant:      # the receiver's recording format (Table 3): packed samples, unpacked in-kernel while staging
        from paper_1906_10598_b200 import workloads as W
        xq, qd = W.quantise(wl.x, args.quant)
        quant = pt.make_quant(qd["bits"], qd["is_signed"], qd["scale"], qd["offset"])
        qkw = dict(quant=quant, N=wl.N)
        x_h = torch.from_numpy(xq).pin_memory()
    else:
        x_h = torch.from_numpy(wl.x).pin_memory()
    lo_h = torch.from_numpy(wl.lo).pin_memory()
    hi_h = torch.from_numpy(wl.hi).pin_memory()
    x, lo, hi = x_h.to(dev), lo_h.to(dev), hi_h.to(dev)
    torch.cuda.synchronize()
    units = sample_evals(wl)

    def step(ev=None):
        if ev:
            ev[0].record()
        r = pt.pt_fit_blocks(x, wl.fs, lo, hi, cfg, **qkw)
        if ev:
            ev[1].record()
        prod = pt.pt_doppler_products(r["best"], wl.T, 0.0, m_int)
        if ev:
            ev[2].record()
        return r, prod

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(args.steps)]
    t_start = torch.cuda.Event(enable_timing=True)
    t_end = torch.cuda.Event(enable_timing=True)
    barrier()
    t_start.record()
    for k in range(args.steps):
        r, prod = step(evs[k])
    t_end.record()
    barrier()
    clocks = sampler.stop()
    total_ms = t_start.elapsed_time(t_end)
    fit_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    prod_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    if dist is not None:
        tt = torch.tensor([total_ms], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        total_ms = float(tt.item())
    ms_per_step = total_ms / args.steps
    value = units * world / (ms_per_step * 1e-3)

    # ---- end to end through the C ABI with HOST buffers (H2D + fit + products + D2H inside the timed region) ----
    e2e = None
    if not args.no_e2e:
        pt.pt_track_host(x_h, wl.fs, lo_h, hi_h, cfg, 0.0, m_int, **qkw)          # warm-up
        barrier()
        t0 = time.perf_counter()
        n_e2e = max(1, min(args.steps, 2))
        for _ in range(n_e2e):
            out = pt.pt_track_host(x_h, wl.fs, lo_h, hi_h, cfg, 0.0, m_int, **qkw)
        barrier()
        e2e_s = (time.perf_counter() - t0) / n_e2e
        if dist is not None:
            tt = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e2e_s = float(tt.item())
        h2d = x_h.numel() * x_h.element_size() + lo_h.numel() * 8 + hi_h.numel() * 8
        d2h = sum(v.numel() * v.element_size() for k, v in out.items() if k != "intervals") + \
            sum(v.numel() * 8 for v in out["intervals"])
        e2e = {"value": units * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * e2e_s, "real_time_factor": wl.B * wl.T / e2e_s}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    achieved = units / (fit_ms * 1e-3)
    sm_mhz = clocks.get("sm_mhz") or SM_MAX_MHZ
    roofline = {"bound": "alu", "achieved": achieved / 1e12, "peak": XU_PEAK / 1e12, "unit": "T sample-evals/s (1 MUFU cosine each)",
                "frac": achieved / XU_PEAK,
                # algorithmic bytes of one step, computed from the workload; the ncu-measured DRAM bytes of the same command
                # (a committed profile, not this run) ride along as traffic_ncu
                "traffic": algorithmic_traffic(wl, args.quant),
                "traffic_ncu": NCU_TRAFFIC.get(args.workload) if not (wl.de["objective"] or args.quant or args.strategy) else None,
                "kernel": kernel_name(plan, wl),
                "kernel_ms": fit_ms, "peak_source": "derived: 148 SMs x 16 MUFU lanes x 1965 MHz (DESIGN.md); "
                "MEASURED_PEAKS.json holds no ALU peak",
                "frac_at_sampled_clock": achieved / (SM_COUNT * XU_LANES_PER_SM * sm_mhz * 1e6),
                # algorithmic flops per sample-evaluation: chi^2 5 (D=5) / 6 FMA; correlation 3 / 4 FMA
                "fp32_flops_achieved_tflops": achieved * ((10 if wl.de["D"] == 5 else 12) - (4 if wl.de["objective"] else
                                                            (2 if wl.meta.get("fix_a1") else 0))) / 1e12}
    try:
        roofline["measured_mufu_peak"] = peak_probe(1) / 1e12
        roofline["measured_ffma_peak_tflops"] = 2 * peak_probe(0) / 1e12
        # the clock a kernel really runs at (in-kernel clock64 / globaltimer): tensor-core activity lowers it, nvidia-smi does not show it
        roofline["sm_mhz_in_kernel"] = {"no_tensor_activity": sm_clock_probe(False), "with_tcgen05_mma": sm_clock_probe(True)}
        if plan["threads"] == 640:
            roofline["frac_at_in_kernel_clock"] = achieved / (SM_COUNT * XU_LANES_PER_SM * roofline["sm_mhz_in_kernel"]["with_tcgen05_mma"] * 1e6)
    except Exception as exc:  # diagnostics only
        roofline["probe_error"] = str(exc)

    # the steps around the hot path, timed on their own after the timed region: FFT acquisition of the
    # initial ranges of every block, and the continuity check of the fitted track (no block of a clean track is re-searched)
    extras = {}
    try:
        if quant is not None:
            raise RuntimeError("skipped: acquisition and continuity check take fp32 samples")
        M = 1 << int(np.floor(np.log2(max(8, min(4096, wl.N // 2)))))
        acq = pt.make_acq_config(M=M, spacing=(wl.N - M) // 2, f_rel=0.0, f_bins=2.0, fdot_bins=2.0, a_rel=0.2)
        retry = pt.make_retry_config(phi_tol=1.5, F_tol=2.0)
        pt.pt_acquire(x, wl.fs, wl.de["D"], acq)
        lo2, hi2 = lo.clone(), hi.clone()
        fit2 = {k: v.clone() for k, v in r.items()}
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        ev[0].record()
        for _ in range(5):
            pt.pt_acquire(x, wl.fs, wl.de["D"], acq)
        ev[1].record()
        is_track = wl.meta.get("box") != "tracking"            # paper_blocks are independent blocks, not one track
        att = pt.pt_refit_doubtful(x, wl.fs, lo2, hi2, cfg, retry, fit2) if is_track else None
        ev[2].record()
        torch.cuda.synchronize()
        extras = {"acquire_ms": ev[0].elapsed_time(ev[1]) / 5, "acquire_piece": M}
        if is_track:
            extras.update({"continuity_check_ms": ev[1].elapsed_time(ev[2]), "blocks_researched": int((att > 0).sum().item())})
    except Exception as exc:  # diagnostics only
        extras = {"extras_error": str(exc)}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic", "config": workload_config(args.workload, wl),
            "real_time_factor": wl.B * wl.T * world / (ms_per_step * 1e-3),
            "fitness_evals_per_s": value / wl.N, "fit_ms": fit_ms, "doppler_products_ms": prod_ms, "plan": plan,
            "roofline": roofline, "clocks": clocks,
            # per step: the DE-kernel launches (pt_fit_blocks_launches: segments of exactly full grids), 2 Doppler kernels
            # (per-block columns, prefix scan) and one kernel per integration interval
            "gpu_launches": args.steps * (len(launches) + 2 + len([m for m in m_int if wl.B // m > 0])),
            "peaks_file": _peaks().get("when")}
    if quant is not None:
        line["config"]["samples"] = "%d-bit packed (Table 3), unpacked in-kernel" % args.quant
    line.update(extras)
    if e2e is not None:
        line["e2e"] = e2e
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(wl)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
