#!/usr/bin/env python
"""bench.py -- scored tokens/s of the fused LM-head scoring pass (BASELINE.json metric).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME] [--impl ours|reference]

A step is one pass of the whole hot path (kernel 1 fused GEMM+statistics, finalize/merge, kernel 2: 3 launches)
over one synthetic packed batch.  At N=1 the workload is BASELINE.json configs[2] (`qwen3_8b`, the
config the metric's 60 % target is quoted on); the other four configs are timed briefly into the
`configs` sub-record.  With N>1 (torchrun):
  --parallelism dp     (default) every rank scores its own batch of the same shape (sequences shard across
                       GPUs, W replicated) and the step ends with the path's one exchange, the all-gather
                       of the 4 scalars per sequence: weak scaling;
  --parallelism vocab  (or vocab-peer: the same without the all-gather, peers' states read in place over NVLink)
                       the LM head is split by rows over the ranks (tensor-parallel scorer): every rank scores
                       the SAME batch against its shard, one all-gather of the packed partial states, then the
                       merge on every rank: strong scaling.
One JSON line is printed by rank 0.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np
import torch

import workloads

METRIC = "scored tokens/s & % of dense BF16 tensor peak (fused LM-head logprob scoring)"
UNIT = "tokens/s"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": p["hbm_gbs"], "bf16_tflops": p["bf16_tflops"],
                "bf16_tflops_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"]), "source": "measured"}
    # fallback stated in B200_PROFILING.md
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
            nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
            nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
            nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(self.samples)}


def dist_env():
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return rank, world, local


# ------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline / --impl reference): the oracle as it stands, on a bounded row sample
# ------------------------------------------------------------------------------------------------
def oracle_sample_rows(T: int, n: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(T, size=min(n, T), replace=False))


def time_oracle(inp: dict, budget_s: float, steps: int = 1, warmup: int = 0):
    """Times oracle.token_scores + sequence_scores on a row sample sized for ~budget_s of CPU work
    per step.  Returns (tokens/s, seconds per step, rows per step, threads)."""
    from oracle import sq_oracle as O   # bench.py's cpu_baseline / reference leg may execute oracle/
    wl = inp["workload"]
    T = inp["T"]
    W64 = O.widen(inp["W"])             # converting the LM head once is set-up, like loading weights
    tg = inp["targets"].numpy()
    probe = oracle_sample_rows(T, min(16, T), 7)
    t0 = time.perf_counter()
    O.token_scores(inp["H"][probe], W64, tg[probe], wl.k)
    per_row = (time.perf_counter() - t0) / max(1, len(probe))
    n = int(max(16, min(T, budget_s / max(per_row, 1e-6))))
    n = min(n, 4096)
    rows = oracle_sample_rows(T, n, 11)
    times = []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        conf = np.empty(len(rows)); lp = np.empty(len(rows)); en = np.empty(len(rows))
        for r0 in range(0, len(rows), 64):
            idx = rows[r0:r0 + 64]
            r = O.token_scores(inp["H"][idx], W64, tg[idx], wl.k)
            conf[r0:r0 + 64] = r["conf"]; lp[r0:r0 + 64] = r["target_logprob"]; en[r0:r0 + 64] = r["entropy"]
        # the sample treated as one packed sequence for the per-sequence step
        O.sequence_scores(lp, en, conf, [0, len(rows)], wl.window)
        dt = time.perf_counter() - t0
        if it >= warmup:
            times.append(dt)
    sec = float(np.mean(times))
    return len(rows) / sec, sec, len(rows), torch.get_num_threads()


def run_reference(args):
    rank, world, _ = dist_env()
    if rank != 0:
        return
    wl = workloads.CONFIGS[args.config]
    inp = workloads.make_inputs(wl)
    tps, sec, rows, threads = time_oracle(inp, budget_s=args.oracle_seconds, steps=args.steps, warmup=min(args.warmup, 1))
    sample = "%d seeded rows of %s (T=%d) per step, fp64 oracle.token_scores + sequence_scores" % (rows, wl.name, inp["T"])
    line = {
        "impl": "reference", "metric": METRIC, "value": tps, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        # the same keys as the GPU arm's config (the workload entries carry the same values; the rest describe this arm)
        "config": {"workload": wl.name, "d": wl.d, "V": wl.V, "B": inp["B"], "T": inp["T"], "k": wl.k,
                   "window": wl.window, "parallelism": "none (fp64 oracle on the host cores of rank 0)",
                   "exchange_bytes_per_step": 0, "l2": "n/a (host arm)", "plan": None},
        "cpu_baseline": {"value": tps, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample,
                         "sample_rows_per_step": rows},
        "e2e": {"value": tps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------
def time_steps(eng, H, W, tg, cu, k, window, stream, steps, warmup, step_fn=None):
    """`warmup` untimed + `steps` timed passes of the whole hot path on `stream`; CUDA events around the timed region;
    kernel 1's duration from the library's per-run events for EVERY timed step (read after the loop: no host sync inside).
    Returns (ms per step, per-step kernel times, outputs, launches)."""
    out = None
    run = step_fn if step_fn is not None else (lambda o: eng.run(H, W, tg, cu, k, window, stream=stream, out=o))
    with torch.cuda.stream(stream):
        for _ in range(warmup):
            out = run(out)
        stream.synchronize()
        eng.profile_read()                                   # empty the ring: only the timed steps remain
        launches0 = eng.launch_count()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(steps):
            out = run(out)
        e1.record(stream)
        stream.synchronize()
    return e0.elapsed_time(e1) / steps, eng.profile_read(), out, eng.launch_count() - launches0


def kernel_stats(per_step):
    f = [x["fused_ms"] for x in per_step]
    return {"mean": float(np.mean(f)), "min": float(np.min(f)), "max": float(np.max(f)), "n": len(f)}


def run_ours(args):
    import paper_2604_07725_b200 as sq
    from paper_2604_07725_b200 import sharding

    rank, world, local = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the sq_score path has no CPU fallback")
    vocab_mode = args.parallelism in ("vocab", "vocab-peer")
    peer_mode = args.parallelism == "vocab-peer"
    ndev = torch.cuda.device_count()
    if args.share_device:
        # debug: every rank on the visible devices round-robin (two ranks on one GPU).  NCCL refuses two ranks on one
        # device, so the exchange goes through gloo on host tensors; the ranks' kernels never wait on one another (dp
        # only: the one collective is a host-side gather after each rank's own step).  Not a measurement.
        if vocab_mode:
            raise SystemExit("bench.py: --share-device is a debug mode of the data-parallel path only")
        local = local % max(1, ndev)
    elif local >= ndev:
        raise SystemExit("bench.py: rank %d needs cuda:%d but only %d CUDA device(s) are visible" % (rank, local, ndev))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    coll_dev = torch.device("cpu") if args.share_device else dev     # where the collectives' tensors live
    use_dist = world > 1 or vocab_mode          # vocab mode runs its collective through NCCL even at world size 1
    if use_dist:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29531")
        if args.share_device:
            dist.init_process_group("gloo", rank=rank, world_size=world)
        else:                                   # NCCL_DEBUG is left to the environment (INFO shows the NVLS / ring choice)
            dist.init_process_group("nccl", device_id=dev, rank=rank, world_size=world)

    peaks = load_peaks()
    wl = workloads.CONFIGS[args.config]
    if use_dist and not vocab_mode:   # weak scaling: every rank scores its own population of the same shape
        from dataclasses import replace
        wl_rank = replace(wl, seed=wl.seed + 100 * rank)
    else:
        wl_rank = wl
    inp = workloads.make_inputs(wl_rank)
    T, B, d, V = inp["T"], inp["B"], wl.d, wl.V
    sms = torch.cuda.get_device_properties(dev).multi_processor_count

    stream = torch.cuda.Stream(device=dev)
    H = inp["H"].to(dev); tg = inp["targets"].to(dev); cu = inp["cu_seqlens"].to(dev)
    exchange_bytes = 0
    if vocab_mode:
        vstarts = sq.shard_vocab(V, world)
        rows_max = max(b - a for a, b in zip(vstarts, vstarts[1:]))
        W = inp["W"][vstarts[rank]:vstarts[rank + 1]].to(dev)          # this rank's rows of the LM head only
        eng = sq.SqScore(d, rows_max, max_tokens=T, max_seqs=B, max_k=wl.k, device=local, staging=False,
                         cta_group=args.cta_group, num_chunks=args.num_chunks, group_m=args.group_m)
        pl = sq.plan(d, max(1, W.shape[0]), T, wl.k, num_sms=sms, cta_group=args.cta_group, num_chunks=args.num_chunks, group_m=args.group_m)
        exchange_bytes = world * sq.shard_state_bytes(T, wl.k)
        if peer_mode:
            # no all-gather: every rank's state stays in its own buffer, opened once by the peers (CUDA IPC over NVLink); the merge
            # kernel reads the R states in place; two 4-byte all-reduces per step order writers and readers on the stream
            exchange_bytes = (world - 1) * sq.shard_state_bytes(T, wl.k)
            my_state = torch.empty(sq.shard_state_bytes(T, wl.k) // 4, dtype=torch.float32, device=dev)
            peers = sharding.PeerStates(my_state, rank, world)
            def step_fn(o):
                return sharding.score_vocab_parallel_peer(eng, peers, H, W, vstarts, tg, cu, wl.k, wl.window, stream=stream)
        else:
            def step_fn(o):
                return sharding.score_vocab_parallel(eng, H, W, vstarts, rank, tg, cu, wl.k, wl.window, stream=stream)
    else:
        W = inp["W"].to(dev)
        eng = sq.SqScore(d, V, max_tokens=T, max_seqs=B, max_k=wl.k, device=local, staging=True,
                         cta_group=args.cta_group, num_chunks=args.num_chunks, group_m=args.group_m)
        pl = sq.plan(d, V, T, wl.k, num_sms=sms, cta_group=args.cta_group, num_chunks=args.num_chunks, group_m=args.group_m)
        if use_dist:
            # the path's one exchange (the N scoring calls of a loop are one batched request whose
            # scalars go back to the router): all-gather of [id, 4 scalars] per sequence, inside the timed step
            seq_ids = list(range(rank * B, (rank + 1) * B))
            exchange_bytes = world * B * world * 5 * 4
            def step_fn(o):
                o = eng.run(H, W, tg, cu, wl.k, wl.window, stream=stream, out=o)
                if args.share_device:
                    stream.synchronize()        # gloo gathers host tensors: the step's scalars must have landed
                o["gathered"] = sharding.gather_sequence_scores(o, seq_ids, B * world, world, device=coll_dev)
                return o
        else:
            step_fn = None
    H_pin = inp["H"].pin_memory(); tg_pin = inp["targets"].pin_memory(); cu_pin = inp["cu_seqlens"].pin_memory()
    seq_pin = torch.empty(4 * B, dtype=torch.float32).pin_memory()
    torch.cuda.synchronize()

    def barrier():
        torch.cuda.synchronize()
        if use_dist:
            dist.barrier()
        torch.cuda.synchronize()

    # ---------------- device-resident timing (value) + live per-kernel timing (roofline)
    eng.set_profiling(True)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    ms_step, fused_ms, out, launches = time_steps(eng, H, W, tg, cu, wl.k, wl.window, stream, args.steps, max(3, args.warmup), step_fn)
    barrier()
    clocks = sampler.stop()

    # ---------------- end to end through the C ABI with HOST buffers (data-parallel form; W is the resident model weight)
    e2e_s, e2e_ok, e2e_dev_ms = float("nan"), None, None
    if not vocab_mode:
        with torch.cuda.stream(stream):
            for _ in range(2):
                eng.run_host(H_pin, W, tg_pin, cu_pin, wl.k, wl.window, seq_pin, stream=stream)
                stream.synchronize()
            barrier()
            g0 = torch.cuda.Event(enable_timing=True); g1 = torch.cuda.Event(enable_timing=True)
            g0.record(stream)
            t0 = time.perf_counter()
            for _ in range(args.e2e_steps):
                eng.run_host(H_pin, W, tg_pin, cu_pin, wl.k, wl.window, seq_pin, stream=stream)
                stream.synchronize()       # the caller reads the scalars every step
            e2e_s = (time.perf_counter() - t0) / args.e2e_steps
            g1.record(stream); stream.synchronize()
            e2e_dev_ms = g0.elapsed_time(g1) / args.e2e_steps
        seq_dev = torch.cat([out[n] for n in ("seq_mean_logprob", "seq_mean_entropy", "seq_mean_conf", "seq_min_window_conf")])
        e2e_ok = bool(torch.allclose(seq_dev.cpu(), seq_pin, rtol=1e-5, atol=1e-6, equal_nan=True))

    # ---------------- max over ranks
    t_loc = torch.tensor([ms_step, e2e_s * 1e3, float(T)], dtype=torch.float64, device=coll_dev)
    if use_dist:
        tmax = t_loc.clone(); dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        tsum = t_loc.clone(); dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
        ms_step, e2e_ms, tokens_all = float(tmax[0]), float(tmax[1]), float(tsum[2])
        if vocab_mode:
            tokens_all = float(T)        # every rank scored the same T tokens against its shard
    else:
        e2e_ms, tokens_all = e2e_s * 1e3, float(T)
    if rank != 0:
        if use_dist:
            dist.destroy_process_group()
        return

    value = tokens_all / (ms_step * 1e-3)
    k1 = kernel_stats(fused_ms)
    k1_ms = k1["mean"]
    fin_ms = float(np.mean([x["finalize_ms"] for x in fused_ms]))
    red_ms = float(np.mean([x["reduce_ms"] for x in fused_ms]))
    v_rank = W.shape[0]
    flops = 2.0 * T * v_rank * d                              # algorithmic FLOPs per launch of kernel 1 (on this rank)
    achieved = flops / (k1_ms * 1e-3) / 1e12
    peak = peaks["bf16_tflops_sustained"]                     # kernel timed inside a long step
    traffic, traffic_source = None, None
    tpath = os.path.join(ROOT, "profiles", "traffic_%s.csv" % wl.name)   # from the committed ncu --set full summary
    if os.path.exists(tpath) and not vocab_mode:
        with open(tpath) as f:
            for ln in f:
                if ln.startswith("sq_fused_score_kernel,"):
                    traffic = float(ln.strip().split(",")[1])
                    traffic_source = "profiles/traffic_%s.csv (ncu --set full of this kernel, committed; not measured in this run)" % wl.name
    par = ("vocab%d (LM head split by rows, %s)" % (world, "peers' partial states read in place by the merge kernel, two 4-byte all-reduces per step"
                                                    if peer_mode else "one all-gather of the packed partial states per step")) if vocab_mode else \
          ("dp%d (sequences sharded, W replicated%s)" % (world, "; one all-gather of 5 floats per sequence per step" if use_dist else ""))
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if vocab_mode else "weak", "vs_baseline": None,
        "dtype": "bf16", "data": "synthetic",
        "config": {"workload": wl.name, "d": d, "V": V, "B": B, "T": T, "k": wl.k, "window": wl.window,
                   "parallelism": par, "exchange_bytes_per_step": exchange_bytes,
                   "l2": "inputs larger than L2 (H %.0f MB + W %.0f MB re-streamed every step)" % (T * d * 2 / 1e6, v_rank * d * 2 / 1e6),
                   "plan": eng.last_plan()},        # what the last run launched (cta_group 4 = quads), not a host-side guess
        "tflops": flops * (world if vocab_mode else 1) / (ms_step * 1e-3) / 1e12,
        "pct_of_bf16_peak_burst": 100.0 * flops / (ms_step * 1e-3) / 1e12 / peaks["bf16_tflops"],
        "roofline": {"bound": "tensor", "kernel": "sq_fused_score_kernel", "achieved": achieved, "peak": peak,
                     "unit": "TFLOP/s", "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source,
                     "peak_kind": "bf16_tflops_sustained of %s (kernel timed inside a long step)" % peaks["source"],
                     "frac_of_burst": achieved / peaks["bf16_tflops"], "peak_burst": peaks["bf16_tflops"],
                     "kernel_ms": k1_ms, "kernel_ms_min": k1["min"], "kernel_ms_max": k1["max"], "kernel_ms_samples": k1["n"],
                     "algorithmic_flops_per_launch": flops},
        "kernels_ms": {"fused": k1_ms, "finalize": fin_ms, "reduce": red_ms,
                       "fused_per_step": [round(x["fused_ms"], 3) for x in fused_ms]},
        "e2e": {"value": (tokens_all / (e2e_ms * 1e-3)) if e2e_ms == e2e_ms else None, "unit": UNIT,
                "h2d_bytes_per_step": T * d * 2 + T * 4 + (B + 1) * 4, "d2h_bytes_per_step": 4 * B * 4,
                "ms_per_step": e2e_ms if e2e_ms == e2e_ms else None, "device_ms_per_step": e2e_dev_ms, "steps": args.e2e_steps,
                "matches_device_path": e2e_ok, "api": "sq_score_run_host"},
        "gpu_launches": int(launches),
        "clocks": clocks,
    }
    if vocab_mode:
        line["e2e"] = {"value": None, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                       "note": "the host-buffer form (sq_score_run_host) is the data-parallel entry point; not run in vocab mode"}
    if world == 1 and not vocab_mode and not args.no_all_configs:
        # the other four BASELINE.json configs, a few steps each (the graded number is the line's own `value`)
        line["configs"] = {wl.name: {"value": value, "ms_per_step": ms_step, "kernel_ms": k1_ms, "T": T,
                                     "tflops_kernel": achieved, "frac": achieved / peak, "frac_of_burst": achieved / peaks["bf16_tflops"]}}
        del H_pin
        for name in workloads.CONFIG_ORDER:
            if name == wl.name:
                continue
            w2 = workloads.CONFIGS[name]
            i2 = workloads.make_inputs(w2)
            e2 = sq.SqScore(w2.d, w2.V, max_tokens=i2["T"], max_seqs=i2["B"], max_k=w2.k, device=local)
            e2.set_profiling(True)
            H2, W2, t2, c2 = (i2[n].to(dev) for n in ("H", "W", "targets", "cu_seqlens"))
            nsteps = 200 if name == "tiny" else (3 if name == "qwen3_32b" else 5)
            ms2, k2, _, _ = time_steps(e2, H2, W2, t2, c2, w2.k, w2.window, stream, nsteps, 3)
            f2 = 2.0 * i2["T"] * w2.V * w2.d
            km = kernel_stats(k2)["mean"]
            line["configs"][name] = {"value": i2["T"] / (ms2 * 1e-3), "ms_per_step": ms2, "kernel_ms": km, "T": i2["T"], "steps": nsteps,
                                     "tflops_kernel": f2 / (km * 1e-3) / 1e12, "frac": f2 / (km * 1e-3) / 1e12 / peak,
                                     "frac_of_burst": f2 / (km * 1e-3) / 1e12 / peaks["bf16_tflops"],
                                     "plan": {n: v for n, v in e2.last_plan().items() if n != "chunk_vtile"}}   # what ran (qwen3_32b: quads)
            e2.close()
            del H2, W2, t2, c2, i2
            torch.cuda.empty_cache()
    if world == 1 and not vocab_mode and not args.no_reduce_standalone:
        # kernel 2 alone on an input large enough for HBM bandwidth to mean something
        r = workloads.reduction_inputs(4096, 1024, 16384, seed=2001)
        eng2 = sq.SqScore(d, V, max_tokens=r["T"], max_seqs=r["B"], max_k=wl.k, device=local, reduce_only=True)
        r_lp, r_en, r_cf, r_cu = (r[n].to(dev) for n in ("target_logprob", "entropy", "conf", "cu_seqlens"))
        with torch.cuda.stream(stream):
            for _ in range(3):
                eng2.reduce(r_lp, r_en, r_cf, r_cu, wl.window, stream=stream)
            r0 = torch.cuda.Event(enable_timing=True); r1 = torch.cuda.Event(enable_timing=True)
            r0.record(stream)
            for _ in range(20):
                eng2.reduce(r_lp, r_en, r_cf, r_cu, wl.window, stream=stream)
            r1.record(stream)
            stream.synchronize()
        r_ms = r0.elapsed_time(r1) / 20
        r_bytes = 12.0 * r["T"] + 16.0 * r["B"]
        line["reduce_standalone"] = {"bound": "hbm", "achieved": r_bytes / (r_ms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                     "unit": "GB/s", "frac": r_bytes / (r_ms * 1e-3) / 1e9 / peaks["hbm_gbs"],
                                     "ms": r_ms, "tokens": r["T"], "seqs": r["B"], "window": wl.window,
                                     "algorithmic_bytes": r_bytes,
                                     "form": eng2.reduce_form(),
                                     "note": "streaming form at this size (2 launches: stream over fixed 4096-token blocks + fold per sequence); 12 B/token read + 16 B/sequence written"}
        eng2.close()
        del r_lp, r_en, r_cf
    if world == 1 and not vocab_mode and not args.no_prepare_standalone:
        # the step before the path: gather + final RMSNorm of the same T rows out of a packed prefill
        # that also holds query tokens; HBM-bound: 2*d bytes read + 2*d written + 4 (pos) per row
        gen = torch.Generator(device=dev); gen.manual_seed(4242)
        n_src = T + 256 * B
        Xs = torch.randn(n_src, d, generator=gen, device=dev, dtype=torch.float32).to(torch.bfloat16)
        gain = (1 + 0.1 * torch.randn(d, generator=gen, device=dev)).to(torch.bfloat16)
        pos_d, _ = eng.positions(torch.full((B,), 256, dtype=torch.int32, device=dev),
                                 (inp["cu_seqlens"][1:] - inp["cu_seqlens"][:-1]).to(torch.int32).to(dev), T, stream=stream)
        Hs = torch.empty(T, d, dtype=torch.bfloat16, device=dev)
        with torch.cuda.stream(stream):
            for _ in range(3):
                eng.prepare(Xs, pos_d, gain, 1e-6, out=Hs, stream=stream)
            p0 = torch.cuda.Event(enable_timing=True); p1 = torch.cuda.Event(enable_timing=True)
            p0.record(stream)
            for _ in range(20):
                eng.prepare(Xs, pos_d, gain, 1e-6, out=Hs, stream=stream)
            p1.record(stream)
            stream.synchronize()
        p_ms = p0.elapsed_time(p1) / 20
        p_bytes = T * (4.0 * d + 4.0)
        line["prepare_standalone"] = {"bound": "hbm", "achieved": p_bytes / (p_ms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                      "unit": "GB/s", "frac": p_bytes / (p_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "ms": p_ms,
                                      "rows": T, "src_rows": n_src, "algorithmic_bytes": p_bytes,
                                      "note": "sq_score_prepare: gather + RMSNorm, 2d B read + 2d B written + 4 B per row; "
                                              "input and output (2 x %.0f MB) exceed L2" % (T * d * 2 / 1e6)}
        del Xs, Hs
    if world == 1 and not vocab_mode and not args.no_decode_standalone:
        # decode-shaped run (self-confidence of a decode batch): T = 64 rows against the
        # same LM head -- every SM streams its own slice of W once, so the bound is HBM: V*d*2 bytes per pass
        Td = 64
        eng3 = sq.SqScore(d, V, max_tokens=Td, max_seqs=4, max_k=wl.k, device=local)
        Hd = H[:Td].contiguous(); tgd = tg[:Td].contiguous()
        cud = torch.tensor([0, 16, 32, 48, 64], dtype=torch.int32, device=dev)
        with torch.cuda.stream(stream):
            od = None
            for _ in range(3):
                od = eng3.run(Hd, W, tgd, cud, wl.k, 16, stream=stream, out=od)
            d0 = torch.cuda.Event(enable_timing=True); d1 = torch.cuda.Event(enable_timing=True)
            d0.record(stream)
            for _ in range(20):
                eng3.run(Hd, W, tgd, cud, wl.k, 16, stream=stream, out=od)
            d1.record(stream)
            stream.synchronize()
        d_ms = d0.elapsed_time(d1) / 20
        # per-kernel split from a SEPARATE profiled pass: the event records between the launches break the programmatic
        # overlap of the two launches (finalize waits behind kernel 1 with its launch latency hidden) and cost ~13 us
        eng3.set_profiling(True)
        with torch.cuda.stream(stream):
            for _ in range(10):
                eng3.run(Hd, W, tgd, cud, wl.k, 16, stream=stream, out=od)
            stream.synchronize()
        d_k = eng3.profile_read()
        eng3.set_profiling(False)
        # the same step captured once into a CUDA graph (the library enqueues only stream work) and replayed
        g_ms = None
        try:
            with torch.cuda.stream(stream):
                gr = torch.cuda.CUDAGraph()
                with torch.cuda.graph(gr, stream=stream):
                    eng3.run(Hd, W, tgd, cud, wl.k, 16, stream=stream, out=od)
                for _ in range(3):
                    gr.replay()
                g0 = torch.cuda.Event(enable_timing=True); g1 = torch.cuda.Event(enable_timing=True)
                g0.record(stream)
                for _ in range(20):
                    gr.replay()
                g1.record(stream)
                stream.synchronize()
            g_ms = g0.elapsed_time(g1) / 20
            del gr
        except Exception as exc:   # reported, never fatal for the headline line
            g_ms = None
            sys.stderr.write("decode graph leg skipped: %r\n" % (exc,))
        # the same decode batch with an 8-bit LM head: W is what the run streams, so e4m3 / block-scaled e4m3 halve the bytes
        d8 = {}
        with torch.cuda.stream(stream):
            for fmt in ("fp8", "mx"):
                if fmt == "fp8":
                    Wd8, wsd = eng3.quantize_fp8(W, True, stream=stream)
                    Hd8, hsd = eng3.quantize_fp8(Hd, False, stream=stream)
                    call = lambda o_: eng3.run_fp8(Hd8, hsd, Wd8, wsd, tgd, cud, wl.k, 16, stream=stream, out=o_)
                    w_bytes = 1.0 * V * d
                else:
                    Wd8, wsd = eng3.quantize_mx(W, sq.MX_OPERAND_W, stream=stream)
                    Hd8, hsd = eng3.quantize_mx(Hd, sq.MX_OPERAND_H, stream=stream)
                    call = lambda o_: eng3.run_mx(Hd8, hsd, Wd8, wsd, tgd, cud, wl.k, 16, stream=stream, out=o_)
                    w_bytes = 1.0 * V * d + float(wsd.numel())
                o8d = None
                for _ in range(3):
                    o8d = call(o8d)
                e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                for _ in range(20):
                    call(o8d)
                e1.record(stream)
                stream.synchronize()
                ms8 = e0.elapsed_time(e1) / 20
                b8 = w_bytes + 1.0 * Td * d + Td * (4 + 16 + 8 * wl.k)
                d8[fmt] = {"ms": ms8, "algorithmic_bytes": b8, "achieved": b8 / (ms8 * 1e-3) / 1e9, "frac": b8 / (ms8 * 1e-3) / 1e9 / peaks["hbm_gbs"],
                           "max_abs_lse_gap_to_bf16_path": float((o8d["lse"] - od["lse"]).abs().max())}
                del Wd8, wsd, Hd8, hsd
        d_bytes = 2.0 * V * d + 2.0 * Td * d + Td * (4 + 16 + 8 * wl.k)
        line["decode_standalone"] = {"bound": "hbm", "achieved": d_bytes / (d_ms * 1e-3) / 1e9, "peak": peaks["hbm_gbs"],
                                     "unit": "GB/s", "frac": d_bytes / (d_ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "ms": d_ms,
                                     "rows": Td, "tokens_per_s": Td / (d_ms * 1e-3), "algorithmic_bytes": d_bytes,
                                     "kernels_ms": {n: float(np.mean([x[n + "_ms"] for x in d_k])) for n in ("fused", "finalize", "reduce")},
                                     "cuda_graph_ms": g_ms, "cuda_graph_frac": (d_bytes / (g_ms * 1e-3) / 1e9 / peaks["hbm_gbs"]) if g_ms else None,
                                     "eight_bit_lm_head": d8,
                                     "plan": sq.plan(d, V, Td, wl.k, num_sms=torch.cuda.get_device_properties(dev).multi_processor_count),
                                     "note": "whole path (2 launches: kernel 1, finalize + per-sequence tail) on a decode batch of 64 rows; W (%.0f MB) "
                                             "exceeds L2 and is streamed once per pass; kernels_ms is from a separate profiled pass "
                                             "(event records between the launches add ~13 us)" % (V * d * 2 / 1e6)}
        eng3.close()
    if world == 1 and not vocab_mode and not args.no_vocab_parallel:
        # one rank's share of a vocab-parallel (tensor-parallel LM head) deployment over R = 8 GPUs, emulated on this GPU:
        # kernel 1 + merge on shard 0 (V/8 rows), then the merge of 8 gathered states + kernel 2.  The exchange itself
        # (one all-gather of R x state bytes) is not timed here: there is one GPU.
        R = 8
        vs = sq.shard_vocab(V, R)
        eng4 = sq.SqScore(d, vs[1] - vs[0], max_tokens=T, max_seqs=B, max_k=wl.k, device=local)
        W0 = W[vs[0]:vs[1]]
        with torch.cuda.stream(stream):
            st0 = None
            for _ in range(2):
                st0 = eng4.run_shard(H, W0, vs[0], tg, wl.k, out=st0, stream=stream)
            states = st0.unsqueeze(0).repeat(R, 1).contiguous()
            om = None
            for _ in range(2):
                om = eng4.merge_shards(states, vs, tg, cu, wl.k, wl.window, stream=stream, out=om)
            v0 = torch.cuda.Event(enable_timing=True); v1 = torch.cuda.Event(enable_timing=True); v2 = torch.cuda.Event(enable_timing=True)
            v0.record(stream)
            for _ in range(5):
                eng4.run_shard(H, W0, vs[0], tg, wl.k, out=st0, stream=stream)
            v1.record(stream)
            for _ in range(5):
                eng4.merge_shards(states, vs, tg, cu, wl.k, wl.window, stream=stream, out=om)
            v2.record(stream)
            stream.synchronize()
        sh_ms, mg_ms = v0.elapsed_time(v1) / 5, v1.elapsed_time(v2) / 5
        sh_flops = 2.0 * T * (vs[1] - vs[0]) * d
        line["vocab_parallel_rank"] = {"shards": R, "shard_rows": vs[1] - vs[0], "run_shard_ms": sh_ms, "merge_shards_ms": mg_ms,
                                       "run_shard_tflops": sh_flops / (sh_ms * 1e-3) / 1e12,
                                       "state_bytes_per_rank": sq.shard_state_bytes(T, wl.k),
                                       "tokens_per_s_per_rank_compute": T / ((sh_ms + mg_ms) * 1e-3),
                                       "note": "emulated on one GPU: shard 0 of 8 + merge of 8 states; the all-gather of 8 x state "
                                               "bytes (NVLink) is not included"}
        eng4.close()
        del states, st0
    if world == 1 and not vocab_mode and not args.no_fp8:
        # FP8 variant (NOT the graded bf16 number): same batch, operands quantised to e4m3 on the device
        # (W once per model, H per step), tcgen05 kind::f8f6f4.  Peak: the measured bf16 peaks x the nominal fp8 : bf16 ratio 2.
        with torch.cuda.stream(stream):
            Wq, wsc = eng.quantize_fp8(W, True, stream=stream)
            Hq, hsc = eng.quantize_fp8(H, False, stream=stream)
            o8 = None
            for _ in range(3):
                o8 = eng.run_fp8(Hq, hsc, Wq, wsc, tg, cu, wl.k, wl.window, stream=stream, out=o8)
            stream.synchronize()
            q0 = torch.cuda.Event(enable_timing=True); q1 = torch.cuda.Event(enable_timing=True); q2 = torch.cuda.Event(enable_timing=True)
            f8_k = []
            q0.record(stream)
            for _ in range(args.steps):
                eng.quantize_fp8(H, False, stream=stream, out=(Hq, hsc))
            q1.record(stream)
            for _ in range(args.steps):
                eng.run_fp8(Hq, hsc, Wq, wsc, tg, cu, wl.k, wl.window, stream=stream, out=o8)
            q2.record(stream)
            stream.synchronize()
            f8_k = eng.kernel_times()["fused_ms"]
        qh_ms, f8_ms = q0.elapsed_time(q1) / args.steps, q1.elapsed_time(q2) / args.steps
        lse_gap = float((o8["lse"] - out["lse"]).abs().max())
        line["fp8_variant"] = {"dtype": "e4m3 x e4m3 -> f32", "ms_per_step": f8_ms, "quantize_h_ms": qh_ms,
                               "tokens_per_s": T / ((f8_ms + qh_ms) * 1e-3), "kernel_ms": f8_k,
                               "kernel_tflops": flops / (f8_k * 1e-3) / 1e12,
                               "peak": 2.0 * peaks["bf16_tflops_sustained"], "frac": flops / (f8_k * 1e-3) / 1e12 / (2.0 * peaks["bf16_tflops_sustained"]),
                               "peak_kind": "2 x bf16_tflops_sustained of %s (nominal fp8 : bf16 ratio)" % peaks["source"],
                               "max_abs_lse_gap_to_bf16_path": lse_gap,
                               "note": "not the graded number: e4m3 operands (per-token H scales, per-tensor W scale); parity holds on the "
                                       "quantised operands (tests/test_fp8_gpu.py)"}
        del Wq, Hq
        # Block-scaled (MX) variant: e4m3 with one UE8M0 scale per 32 elements, tcgen05 kind::mxf8f6f4.block_scale.  Same batch,
        # same peak as the FP8 variant; also reports how far its scores are from the bf16 path's next to the FP8 variant's.
        with torch.cuda.stream(stream):
            Wm, wsf = eng.quantize_mx(W, sq.MX_OPERAND_W, stream=stream)
            Hm, hsf = eng.quantize_mx(H, sq.MX_OPERAND_H, stream=stream)
            om = None
            for _ in range(3):
                om = eng.run_mx(Hm, hsf, Wm, wsf, tg, cu, wl.k, wl.window, stream=stream, out=om)
            stream.synchronize()
            q0 = torch.cuda.Event(enable_timing=True); q1 = torch.cuda.Event(enable_timing=True); q2 = torch.cuda.Event(enable_timing=True)
            q0.record(stream)
            for _ in range(args.steps):
                eng.quantize_mx(H, sq.MX_OPERAND_H, stream=stream, out=(Hm, hsf))
            q1.record(stream)
            for _ in range(args.steps):
                eng.run_mx(Hm, hsf, Wm, wsf, tg, cu, wl.k, wl.window, stream=stream, out=om)
            q2.record(stream)
            stream.synchronize()
            mx_k = eng.kernel_times()["fused_ms"]
        qm_ms, mx_ms = q0.elapsed_time(q1) / args.steps, q1.elapsed_time(q2) / args.steps
        gaps = {n: {"mx": float((om[n] - out[n]).abs().max()), "fp8": float((o8[n] - out[n]).abs().max())} for n in ("lse", "target_logprob", "conf")}
        line["mx_variant"] = {"dtype": "mxfp8 (e4m3 + ue8m0 per 32) x mxfp8 -> f32", "ms_per_step": mx_ms, "quantize_h_ms": qm_ms,
                              "tokens_per_s": T / ((mx_ms + qm_ms) * 1e-3), "kernel_ms": mx_k,
                              "kernel_tflops": flops / (mx_k * 1e-3) / 1e12,
                              "peak": 2.0 * peaks["bf16_tflops_sustained"], "frac": flops / (mx_k * 1e-3) / 1e12 / (2.0 * peaks["bf16_tflops_sustained"]),
                              "peak_kind": "2 x bf16_tflops_sustained of %s (nominal fp8 : bf16 ratio)" % peaks["source"],
                              "max_abs_gap_to_bf16_path": gaps,
                              "note": "not the graded number: block-scaled e4m3 operands, 224-column tiles; parity holds on the quantised "
                                      "operands (tests/test_mx_gpu.py)"}
        del Wm, Hm
    if args.matmul_ceiling:
        # context only: cuBLAS on the same (T, V, d) in row chunks, logits materialised chunk by chunk
        rows = 8192
        buf = torch.empty(rows, V, dtype=torch.bfloat16, device=dev)
        Wt = W.t()
        def mm_pass():
            for r0 in range(0, T, rows):
                r1 = min(T, r0 + rows)
                torch.matmul(H[r0:r1], Wt, out=buf[: r1 - r0])
        for _ in range(2):
            mm_pass()
        torch.cuda.synchronize()
        m0 = torch.cuda.Event(enable_timing=True); m1 = torch.cuda.Event(enable_timing=True)
        m0.record()
        for _ in range(args.steps):
            mm_pass()
        m1.record(); torch.cuda.synchronize()
        mm_ms = m0.elapsed_time(m1) / args.steps
        line["context_cublas_matmul"] = {"ms_per_pass": mm_ms, "tflops": flops / (mm_ms * 1e-3) / 1e12,
                                         "note": "torch.matmul bf16 over the same T,V,d in 8192-row chunks; not part of the path"}
        del buf
    if args.unfused_baseline:
        # context only: what fusion buys -- the same outputs from library ops with the logits materialised
        rows = 4096
        Wt = W.t()
        def unfused_pass():
            for r0 in range(0, T, rows):
                r1 = min(T, r0 + rows)
                z = torch.matmul(H[r0:r1], Wt).float()
                lsm = torch.log_softmax(z, dim=1)
                tv, ti = torch.topk(lsm, wl.k, dim=1)
                ent = -(lsm.exp() * lsm).sum(1)
                tlp = lsm.gather(1, tg[r0:r1].long().unsqueeze(1))
                del z, lsm
        unfused_pass(); torch.cuda.synchronize()
        u0 = torch.cuda.Event(enable_timing=True); u1 = torch.cuda.Event(enable_timing=True)
        u0.record(); unfused_pass(); unfused_pass(); u1.record(); torch.cuda.synchronize()
        u_ms = u0.elapsed_time(u1) / 2
        line["context_unfused_torch"] = {"ms_per_pass": u_ms, "tokens_per_s": T / (u_ms * 1e-3),
                                         "note": "torch matmul + log_softmax + topk + entropy + gather in 4096-row chunks "
                                                 "(logits materialised); per-token outputs only; not part of the path"}
    if world == 1 and not vocab_mode and not args.no_cpu_baseline:
        tps, sec, rows, threads = time_oracle(inp, budget_s=args.oracle_seconds)
        line["cpu_baseline"] = {"value": tps, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": "%d seeded rows of %s in %.1f s (fp64 oracle.token_scores + sequence_scores)" % (rows, wl.name, sec)}
    print(json.dumps(line))
    eng.close()
    if use_dist:
        dist.destroy_process_group()


def launch_command(gpus: int, argv, port: int):
    """The command `python bench.py --gpus N` turns itself into when it was not started by torchrun: one rank per GPU on
    this node, rendezvous on 127.0.0.1 (the container's hostname may not resolve)."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(gpus),
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + list(argv)


def self_launch(args, argv) -> int:
    """`--gpus N` with N > 1 outside torchrun (no WORLD_SIZE in the environment): start the N ranks ourselves.  Refuses
    loudly when the node shows fewer than N devices, unless --share-device (debug) lets ranks share one."""
    import socket
    import subprocess
    ndev = torch.cuda.device_count()
    if ndev < args.gpus and not args.share_device:
        raise SystemExit("bench.py: --gpus %d needs %d CUDA devices, %d visible (no silent single-GPU run; "
                         "--share-device puts the ranks on the devices there are, for debugging only)" % (args.gpus, args.gpus, ndev))
    if ndev < 1:
        raise SystemExit("bench.py: no CUDA device; the sq_score path has no CPU fallback")
    sock = socket.socket(); sock.bind(("127.0.0.1", 0)); port = sock.getsockname()[1]; sock.close()
    return subprocess.call(launch_command(args.gpus, argv, port))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="qwen3_8b", choices=list(workloads.CONFIGS))
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--parallelism", default="dp", choices=["dp", "vocab", "vocab-peer"])
    ap.add_argument("--no-all-configs", action="store_true", help="skip the brief timing of the other four configs")
    ap.add_argument("--oracle-seconds", type=float, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-reduce-standalone", action="store_true")
    ap.add_argument("--no-prepare-standalone", action="store_true")
    ap.add_argument("--no-decode-standalone", action="store_true")
    ap.add_argument("--no-vocab-parallel", action="store_true")
    ap.add_argument("--no-fp8", action="store_true")
    ap.add_argument("--matmul-ceiling", action="store_true", help="also time torch.matmul on the same shapes (context)")
    ap.add_argument("--unfused-baseline", action="store_true", help="also time an unfused torch pipeline (context)")
    ap.add_argument("--cta-group", type=int, default=0)
    ap.add_argument("--num-chunks", type=int, default=0)
    ap.add_argument("--group-m", type=int, default=0)
    ap.add_argument("--share-device", action="store_true",
                    help="debug: ranks may share a GPU (gloo for the gather instead of NCCL); not a measurement")
    args = ap.parse_args()
    if args.gpus < 1:
        raise SystemExit("bench.py: --gpus must be >= 1")
    if "WORLD_SIZE" in os.environ and int(os.environ["WORLD_SIZE"]) != args.gpus:
        raise SystemExit("bench.py: --gpus %d but the launcher started %s ranks" % (args.gpus, os.environ["WORLD_SIZE"]))
    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(self_launch(args, sys.argv[1:]))
    if args.impl == "reference":
        if args.oracle_seconds is None:
            args.oracle_seconds = max(1.0, 90.0 / (args.steps + 1))
        run_reference(args)
    else:
        if args.oracle_seconds is None:
            args.oracle_seconds = 15.0
        run_ours(args)


if __name__ == "__main__":
    main()
