#!/usr/bin/env python
"""bench.py -- param-updates/s and effective HBM GB/s of the LayUp update+gossip round.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config NAME|all] [--impl ours|reference]
                  [--optimizer sgd|adamw] [--mix pushsum|lossy|symmetric] [--mode round|layers|graph]
                  [--tuning key=value,...] [--no-per-config]

A "step" is one layup_round(): the whole hot path (straggler mask, peer choice, push-sum
weights, local step, push, peer mix, reverse-layer work list) over all K replicas of all
layers of one synthetic batch of gradients.  Default workload = BASELINE.json:configs[2]
(K=16 replicas of the GPT-2-medium parameter set, fp32 + momentum), the largest config
and the one north_star's bandwidth target is stated on.

Prints ONE JSON line; its "per_config" list carries the same measurement (ms per round,
param-updates/s, effective GB/s, launches) for all five BASELINE configs, the L2-resident ones
also replayed from a CUDA graph (layup_graph_*), and "cpu_baseline" times the oracle on all
host cores (the same source built with -fopenmp) beside the single-threaded figure.  N > 1 (torchrun): the path does not shard (north_star: "no
sharding across GPUs, no collectives"), so each rank runs an independent replica set
("replicas only") and value is the sum over ranks / max time.
--impl reference times the CPU oracle as it stands on a bounded sample of the workload.
"""
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

import numpy as np  # noqa: E402
import torch  # noqa: E402

import synth  # noqa: E402

METRIC = "param_updates_per_s"
UNIT = "param-updates/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="gpt2m_k16")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--optimizer", default="sgd", choices=["sgd", "adamw"],
                    help="local step: the config's SGD(+momentum) [default, BASELINE.json] or AdamW (NEXT-3)")
    ap.add_argument("--mix", default="pushsum", choices=["pushsum", "lossy", "symmetric"],
                    help="mixer: push-sum fold [default, BASELINE.json], contention-lossy or symmetric (NEXT-4)")
    ap.add_argument("--skip-prob", type=float, default=None,
                    help="override the workload's straggler probability (configs[3] semantics on any shape)")
    ap.add_argument("--mode", default="round", choices=["round", "layers", "graph"],
                    help="round: one layup_round per step (one reverse-layer work list); layers: L per-layer "
                         "launches on 4 streams; graph: all timed rounds recorded once with layup_graph_* and replayed")
    ap.add_argument("--tuning", default="", help="layup_tuning fields, e.g. launch_shape=2,stages=4 (include/layup.h)")
    ap.add_argument("--no-per-config", action="store_true", help="skip the per_config list (all five BASELINE configs)")
    ap.add_argument("--per-config-steps", type=int, default=0, help="timed rounds per config in per_config (0: the config's own round count, at most 20)")
    return ap.parse_args()


def tuning_dict(args):
    out = {}
    for kv in filter(None, args.tuning.split(",")):
        k, v = kv.split("=")
        out[k.strip()] = int(v)
    return out or None


def get_workload(name):
    try:
        return synth.workload(int(name))
    except ValueError:
        return synth.workload(name)


ADAMW = dict(weight_decay=0.0031235, beta1=0.9, beta2=0.95, eps=1e-8)   # PAPER.md:469-480 (GPT-2 medium row)
MIXES = {"pushsum": 0, "lossy": 1, "symmetric": 2}


def rule_kwargs(args):
    """Keyword arguments shared by LayUp(...) and oracle.Oracle(...): optimiser and mixer."""
    kw = dict(mix_mode=MIXES[args.mix])
    if args.optimizer == "adamw":
        kw.update(optimizer=1, **ADAMW)
    return kw


def bench_config(w, args):
    """The workload, identically for both arms (ours and --impl reference): what is computed, not how it is launched."""
    return {"workload": "%s (%s)" % (w.name, w.note), "K": w.K, "L": w.L, "params_per_replica": w.params_per_replica,
            "momentum": w.momentum, "lr": w.lr, "skip_prob": w.skip_prob, "optimizer": args.optimizer, "mix": args.mix}


def bytes_per_update(w, args=None):
    """read x, g; write x (+ read/write m (+ read/write v))."""
    if args is not None and args.optimizer == "adamw":
        return 28
    return 20 if w.momentum != 0.0 else 12


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def committed_traffic(name, optimizer="sgd"):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed ncu capture
    (profiles/traffic.csv, see profiles/traffic.md) and where it comes from (summary file, capture date, git
    hash of the kernels captured -- a COMMITTED figure, not a live one: a stale capture shows here);
    (None, None) if this (workload, optimizer) was not captured."""
    p = os.path.join(ROOT, "profiles", "traffic.csv")
    if os.path.exists(p):
        import csv
        with open(p) as f:
            for row in csv.DictReader(f):
                if row["workload"] == name and row["optimizer"] == optimizer:
                    return float(row["dram_bytes_per_launch"]), "%s, captured %s at %s" % (
                        row["source"], row.get("captured", "?"), row.get("git", "?"))
    return None, None


# ---- oracle sample (cpu_baseline and --impl reference) -------------------------------
def oracle_sample(w, seconds, steps=None, warmup=0, args=None, all_cores=False):
    """Times oracle/ as it stands on a bounded sample of the workload: the LAST layers of the
    layer list (output side first, as the path walks them) up to a budget of parameter updates
    per round.  all_cores: the same source built with -fopenmp (element loops on every host
    core, bit-identical results); else the default single-threaded build."""
    import oracle
    oracle.use_omp(all_cores)
    try:
        return _oracle_sample(oracle, w, seconds, steps, warmup, args, all_cores)
    finally:
        oracle.use_omp(False)            # never leave the OpenMP build as the process-wide default


def _oracle_sample(oracle, w, seconds, steps, warmup, args, all_cores):
    budget = 200e6                       # param-updates per round in the sample
    layers, tot = [], 0
    for l in reversed(range(w.L)):
        if layers and tot + w.K * w.numel[l] > budget:
            break
        layers.append(l)
        tot += w.K * w.numel[l]
    layers = sorted(layers)
    sub = synth.shrink(w, [w.numel[l] for l in layers])
    mom = 0.0 if (args is not None and args.optimizer == "adamw") else sub.momentum
    ref = oracle.Oracle(sub.numel, sub.K, sub.lr, mom, sub.seed, sub.peer_mode, sub.skip_prob,
                        **(rule_kwargs(args) if args is not None else {}))
    xs, grads_fn = synth.host_state(sub)
    for l in range(sub.L):
        ref.x[l][:] = xs[l]
    grads = grads_fn(0)
    for s in range(warmup):
        ref.round(s, grads)
    done, t_used, step = 0, 0.0, warmup
    per_step_updates = []
    while True:
        _, act = oracle.schedule(sub.seed, step, sub.L, sub.K, sub.peer_mode, sub.skip_prob)
        t0 = time.perf_counter()
        ref.round(step, grads)
        t_used += time.perf_counter() - t0
        per_step_updates.append(int(act.sum()) * sum(sub.numel))
        step += 1
        done += 1
        if steps is not None:
            if done >= steps:
                break
        elif t_used >= seconds or done >= 50:
            break
    ups = sum(per_step_updates) / t_used
    sample = "layers %d..%d of %d (%.1fM params/replica, K=%d), %d rounds, %s" % (
        layers[0], layers[-1], w.L, sum(sub.numel) / 1e6, sub.K, done,
        "OpenMP over elements, %d threads" % (os.cpu_count() or 1) if all_cores else "single thread")
    return ups, t_used / done, sample, sum(per_step_updates) / done


def cpu_baseline(w, args):
    """The oracle on the box's host cores: all cores (reported value) and one thread beside it."""
    half = args.cpu_seconds / 2
    a_ups, _, a_sample, _ = oracle_sample(w, half, args=args, all_cores=True)
    s_ups, _, s_sample, _ = oracle_sample(w, half, args=args, all_cores=False)
    return {"value": a_ups, "unit": UNIT, "cores": os.cpu_count() or 1, "kind": "oracle", "sample": a_sample,
            "single_thread": {"value": s_ups, "cores": 1, "sample": s_sample}}


def run_reference(args, w, rank, world):
    if rank != 0:
        return
    ups, s_per_step, sample, _ = oracle_sample(w, args.cpu_seconds, steps=args.steps, warmup=min(args.warmup, 1), args=args,
                                               all_cores=True)
    line = {
        "metric": METRIC, "value": ups, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": s_per_step * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic", "impl": "reference",
        "config": bench_config(w, args),
        "cpu_baseline": {"value": ups, "unit": UNIT, "cores": os.cpu_count() or 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": ups, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ---- clocks sampling ------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.perf_counter(), line.strip()))

    def summary(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        rows = [r for (t, r) in self.rows if t0 <= t <= t1] or [r for (_, r) in self.rows[-3:]]
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax = float(f[1])
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def algorithmic_bytes(w, lu, steps_range, args=None):
    """12/20/28 B per active param-update, 8 B for an idle replica that receives."""
    if w.skip_prob == 0.0:
        n = w.K * w.params_per_replica
        return [bytes_per_update(w, args) * n] * len(steps_range), [n] * len(steps_range)
    bts, ups = [], []
    numel = np.array(w.numel, dtype=np.float64)
    for s in steps_range:
        peer, active = lu.layup_schedule(s)
        b = u = 0.0
        for i in range(w.K):
            if active[i]:
                b += bytes_per_update(w, args) * numel.sum(); u += numel.sum()
            else:
                recv = np.array([(peer[l] == i).any() for l in range(w.L)])
                b += 8 * numel[recv].sum()
        bts.append(b); ups.append(u)
    return bts, ups


def reduce_over_ranks(dist, ms, updates, nbytes, device):
    """Replicas-only aggregation: time = MAX over ranks, work = SUM over ranks.
    dist is torch.distributed (any backend) or None for a single process."""
    if dist is None:
        return float(ms), float(updates), float(nbytes)
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    tot = torch.tensor([updates, nbytes], device=device, dtype=torch.float64)
    dist.all_reduce(tot, op=dist.ReduceOp.SUM)
    return float(t.item()), float(tot[0].item()), float(tot[1].item())


class Timed:
    """One timed run of `steps` rounds on a fresh ctx: CUDA events on the launching stream around the
    whole sequence (ms), the library's own event pairs around every launching call (kernel_ms)."""

    def __init__(self, args, w, rank, local_rank, mode, barrier):
        from paper_2410_05985_b200 import WHAT_G, WHAT_X, LayUp
        self.w, self.mode, self.args = w, mode, args
        mom = 0.0 if args.optimizer == "adamw" else w.momentum
        self.lu = lu = LayUp(w.K, w.numel, w.lr, mom, w.seed + 1000 * rank, w.peer_mode, w.skip_prob, device=local_rank,
                             tuning=tuning_dict(args), **rule_kwargs(args))
        for l in range(w.L):
            synth.fill_init_(w, l, lu.view(WHAT_X, l))
            synth.fill_grad_(w, 0, l, lu.view(WHAT_G, l), data_seed=w.seed + 1000 * rank)
        torch.cuda.synchronize()
        self.streams = [torch.cuda.Stream() for _ in range(4)] if mode == "layers" else None
        self.step = 0
        self.barrier = barrier

    def one_step(self):
        lu, w, s = self.lu, self.w, self.step
        if self.mode == "layers":
            for k, l in enumerate(reversed(range(w.L))):
                lu.layup_layer_update(s, l, self.streams[k % 4])
        else:
            lu.layup_round(s)
        self.step += 1

    def run(self, steps, warmup):
        lu, w = self.lu, self.w
        for _ in range(warmup):
            self.one_step()
        lu.layup_sync()
        graph = gstream = None
        if self.mode == "graph":
            # all timed rounds recorded once (the round counter is device state), then one replay to warm up
            gstream = torch.cuda.Stream()
            lu.layup_graph_begin(gstream)
            for r in range(steps):
                lu.layup_round(self.step + r, gstream)
            graph = lu.layup_graph_end()
            lu.layup_graph_launch(graph, gstream)
            self.step += steps
            lu.layup_sync()
        launches0 = lu.layup_launch_count()
        lu.layup_profile(self.mode != "graph")
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        self.barrier()
        self.t0 = time.perf_counter()
        self.first = self.step
        cur = torch.cuda.current_stream()
        for st in (self.streams or []) + ([gstream] if gstream else []):
            st.wait_stream(cur)
        tstream = gstream or cur
        ev0.record(tstream)
        if graph is not None:
            lu.layup_graph_launch(graph, gstream)
            self.step += steps
        else:
            for _ in range(steps):
                self.one_step()
        for st in (self.streams or []):
            cur.wait_stream(st)
        ev1.record(tstream)
        self.barrier()
        self.t1 = time.perf_counter()
        ms = ev0.elapsed_time(ev1)
        n_k, k_ms = lu.layup_profile_read()
        lu.layup_profile(False)
        launches = lu.layup_launch_count() - launches0
        if graph is not None:
            lu.layup_graph_destroy(graph)
        bts, ups = algorithmic_bytes(w, lu, range(self.first, self.first + steps), self.args)
        return dict(ms=ms, steps=steps, launches=launches, n_k=n_k, k_ms=k_ms, bytes=sum(bts), updates=sum(ups))

    def close(self):
        self.lu.close()
        del self.lu
        torch.cuda.empty_cache()


def per_config_report(args, rank, local_rank, barrier, main_name, main_entry):
    """north_star "Report per config": every BASELINE config under the same clock.  The L2-resident
    configs are also replayed from a CUDA graph (launch-latency path)."""
    out = []
    for w in synth.workloads():
        if w.name == main_name:
            out.append(main_entry)
            continue
        steps = args.per_config_steps or min(w.rounds, 20)
        small = w.K * w.params_per_replica * 12 < 126e6
        for mode in (["round", "graph"] if small else ["round"]):
            try:
                t = Timed(args, w, rank, local_rank, mode, barrier)
                r = t.run(steps, max(args.warmup, 3))
                t.close()
                out.append(config_entry(w, mode, r))
            except Exception as ex:                      # e.g. not enough HBM next to the main arena
                out.append({"workload": w.name, "mode": mode, "error": str(ex)[:200]})
    # straggler rounds at HBM size: configs[3]'s semantics (each replica idles with probability 0.25 per
    # round and still receives) on the shapes of configs[1], [4] and, if a second
    # arena fits beside the main one, configs[2]
    for name in ("gpt2s_k8", "manysmall_k64", "gpt2m_k16"):
        w = synth.shrink(synth.workload(name), synth.workload(name).numel, skip_prob=0.25)
        need = w.K * sum((n + 31) // 32 * 32 for n in w.numel) * 4 * 3 + (6 << 30)
        if torch.cuda.mem_get_info()[0] < need:
            out.append({"workload": "%s shapes, skip_prob 0.25" % name, "mode": "round", "error": "needs %.0f GB of free HBM" % (need / 2**30)})
            continue
        try:
            t = Timed(args, w, rank, local_rank, "round", barrier)
            r = t.run(10, max(args.warmup, 3))
            t.close()
            e = config_entry(w, "round", r)
            e["workload"] = "%s shapes, skip_prob 0.25" % name
            e["note"] = "effective bytes: 12/20 B per active param-update, 8 B per element of an idle replica that receives a push"
            out.append(e)
        except Exception as ex:
            out.append({"workload": "%s shapes, skip_prob 0.25" % name, "mode": "round", "error": str(ex)[:200]})
    return out


def config_entry(w, mode, r):
    ms = r["ms"] / r["steps"]
    gbs = r["bytes"] / r["steps"] / (ms * 1e-3) / 1e9
    e = {"workload": "%s (%s)" % (w.name, w.note), "K": w.K, "L": w.L, "mode": mode, "rounds_timed": r["steps"],
         "ms_per_round": ms, "param_updates_per_s": r["updates"] / (r["ms"] * 1e-3), "effective_hbm_gbs": gbs,
         "frac_of_8TBs_nominal": gbs / 8000.0, "launches_per_round": r["launches"] / r["steps"],
         "l2": "inputs larger than L2" if r["bytes"] / r["steps"] > 4 * 126e6 else "L2-resident (launch-latency bound)"}
    if r["n_k"]:
        e["kernel_ms_per_round"] = r["k_ms"] / r["steps"]
    return e


def run_ours(args, w, rank, world, local_rank):
    from paper_2410_05985_b200 import WHAT_G
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        if not dist.is_initialized():
            dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    timed = Timed(args, w, rank, local_rank, args.mode, barrier)
    lu = timed.lu
    sampler = ClockSampler(local_rank) if rank == 0 else None
    time.sleep(0.3)
    r = timed.run(args.steps, args.warmup)
    clocks = sampler.summary(timed.t0, timed.t1) if sampler else None
    step = timed.step
    n_k, k_ms, launches = r["n_k"], r["k_ms"], r["launches"]

    ms, job_updates, job_bytes = reduce_over_ranks(dist, r["ms"], r["updates"], r["bytes"], torch.device("cuda", local_rank))
    value = job_updates / (ms * 1e-3)
    eff_gbs = job_bytes / (ms * 1e-3) / 1e9

    # ---- roofline of the dominant kernel (the fused update kernel), this rank
    peak, peak_src = measured_peak()
    if n_k:
        k_avg_ms = k_ms / n_k
        bytes_per_launch = r["bytes"] / n_k
    else:                                                # graph replay: the whole sequence is one timed launch
        k_avg_ms, bytes_per_launch = r["ms"] / args.steps, r["bytes"] / args.steps
    achieved = bytes_per_launch / (k_avg_ms * 1e-3) / 1e9 if k_avg_ms > 0 else 0.0
    kernel = "layup_update_persist" if (tuning_dict(args) or {}).get("launch_shape") == 2 else "layup_update_tma"
    traffic, traffic_from = committed_traffic(w.name, args.optimizer) if args.mix == "pushsum" and kernel == "layup_update_tma" else (None, None)
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_from": traffic_from,
                "kernel": kernel,
                "kernel_ms_avg": k_avg_ms, "kernel_launches": n_k, "algorithmic_bytes_per_launch": bytes_per_launch,
                "peak_source": peak_src, "frac_of_8TBs_nominal": achieved / 8000.0}

    # ---- the read-only diagnostic kernel of the path (layup_disagreement), device time
    diag = None
    try:
        lu.layup_disagreement(False)
        d_ms = []
        for _ in range(3):
            lu.layup_disagreement(False)
            d_ms.append(lu.layup_disagreement_ms())
        d = float(np.median(d_ms))
        diag = {"kernel": "layup_disagreement_kernel", "ms": d, "read_gbs": 4.0 * w.K * w.params_per_replica / (d * 1e-3) / 1e9,
                "frac_of_measured_peak": 4.0 * w.K * w.params_per_replica / (d * 1e-3) / 1e9 / peak}
    except Exception as ex:
        diag = {"error": str(ex)[:200]}

    # ---- e2e: same metric through the C-ABI with HOST buffers (h2d grads + d2h params in the timed region)
    e2e = None
    if not args.no_e2e:
        try:
            total = w.K * w.params_per_replica
            g_host = torch.empty(total, dtype=torch.float32, pin_memory=True)
            x_host = torch.empty(total, dtype=torch.float32, pin_memory=True)
            off = 0
            for l, n in enumerate(w.numel):      # host gradients = the same synthetic batch, unpadded
                g_host[off:off + w.K * n].view(w.K, n).copy_(lu.view(WHAT_G, l))
                off += w.K * n
            torch.cuda.synchronize()
            lu.layup_round_host(step, g_host, x_host); step += 1       # warm-up (stream/event creation)
            barrier()
            te0 = time.perf_counter()
            e_first = step
            for _ in range(args.e2e_steps):
                lu.layup_round_host(step, g_host, x_host); step += 1
            barrier()
            e_s = time.perf_counter() - te0
            if dist is not None:
                t = torch.tensor([e_s], device="cuda", dtype=torch.float64)
                dist.all_reduce(t, op=dist.ReduceOp.MAX)
                e_s = float(t.item())
            _, e_ups = algorithmic_bytes(w, lu, range(e_first, e_first + args.e2e_steps), args)
            e2e = {"value": world * sum(e_ups) / e_s, "unit": UNIT, "h2d_bytes_per_step": 4 * total,
                   "d2h_bytes_per_step": 4 * total, "steps": args.e2e_steps, "ms_per_step": e_s / args.e2e_steps * 1e3,
                   "api": "layup_round_host (pinned host grads in, params out, layer-pipelined)"}
            # the same call when the step's result read back is a metric, not the parameters: gradients in,
            # the push-sum weights w[L][K] out -- what a training loop would do every step
            barrier()
            tm0 = time.perf_counter()
            m_first = step
            for _ in range(args.e2e_steps):
                lu.layup_round_host(step, g_host, None); step += 1
                lu.layup_weights()
            barrier()
            m_s = time.perf_counter() - tm0
            _, m_ups = algorithmic_bytes(w, lu, range(m_first, m_first + args.e2e_steps), args)
            e2e["metric_only"] = {"value": world * sum(m_ups) / m_s, "unit": UNIT, "h2d_bytes_per_step": 4 * total,
                                  "d2h_bytes_per_step": 8 * w.L * w.K, "ms_per_step": m_s / args.e2e_steps * 1e3,
                                  "api": "layup_round_host (pinned host grads in, no parameter read-back) + layup_weights"}
            del g_host, x_host
        except Exception as ex:                  # e.g. the box cannot pin 2 x K x N x 4 bytes
            e2e = {"value": None, "unit": UNIT, "error": str(ex)[:200]}
    lu.layup_sync()
    main_entry = config_entry(w, args.mode, r)
    timed.close()

    per_config = None
    if not args.no_per_config and world == 1 and args.config == "gpt2m_k16":
        per_config = per_config_report(args, rank, local_rank, barrier, w.name, main_entry)

    # the other kernels of the path, inside the object the driver's record keeps: the diagnostic's read
    # rate and the per_config row furthest below the peak (HBM-bound rows only)
    others = {}
    if diag and "read_gbs" in diag:
        others["layup_disagreement"] = {"read_gbs": diag["read_gbs"], "frac": diag["read_gbs"] / peak, "ms": diag["ms"]}
    hbm_rows = [e for e in (per_config or []) if "effective_hbm_gbs" in e and e.get("l2", "").startswith("inputs larger")]
    if hbm_rows:
        worst = min(hbm_rows, key=lambda e: e["effective_hbm_gbs"])
        others["worst_per_config_row"] = {"workload": worst["workload"], "mode": worst["mode"], "ms_per_round": worst["ms_per_round"],
                                          "effective_hbm_gbs": worst["effective_hbm_gbs"], "frac": worst["effective_hbm_gbs"] / peak}
    roofline["others"] = others or None

    if rank != 0:
        return
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        cpu = cpu_baseline(w, args)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": bench_config(w, args),
        # how this arm launches the workload (GPU-only settings; the reference arm has none)
        "launch": {"mode": args.mode, "tuning": tuning_dict(args), "parallelism": "replicas only x%d" % world,
                   "l2": "inputs larger than L2" if job_bytes / args.steps / world > 4 * 126e6 else
                         "L2-resident working set (launch-latency bound, see DESIGN.md)"},
        "effective_hbm_gbs": eff_gbs, "frac_of_8TBs_nominal": eff_gbs / world / 8000.0,
        "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches, "clocks": clocks,
        "diagnostic": diag, "per_config": per_config,
    }
    print(json.dumps(line), flush=True)


def main():
    args = parse()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    # --config all: the per-config report north_star asks for, one JSON line per BASELINE config
    # (the default invocation prints exactly one line, for configs[2])
    names = [w.name for w in synth.workloads()] if args.config == "all" else [args.config]
    for name in names:
        w = get_workload(name)
        if args.skip_prob is not None:
            w = synth.shrink(w, w.numel, skip_prob=args.skip_prob)
        if args.impl == "reference":
            run_reference(args, w, rank, world)
        else:
            run_ours(args, w, rank, world, local_rank)
    if world > 1 and args.impl != "reference":
        import torch.distributed as dist
        if dist.is_initialized():
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
