#!/usr/bin/env python
"""bench.py — committed tokens/s of the DEX expand-commit-collapse step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl dex|reference] [--workload c2]

Metric (BASELINE.json:metric): committed tokens/s at the Llama-2-7B shape, bf16, batch 1,
X = {8,16,24,32} (config c2), next to the library's own AR baseline (X = {L}, same kernels),
with the segment GEMM's achieved HBM GB/s against the measured copy peak.

A "step" is one whole run of the workload's hot path: rewind the sequence to its prefilled
prompt (dex_rewind: the prompt's committed K/V stays resident in HBM) and run DEX rounds
(dex_step: expand -> exit -> commit -> collapse) until `gen_len` tokens
are committed.  `value` = committed tokens of all ranks / device time of the K steps (CUDA
events on the library's stream, max over ranks).  `e2e` repeats the step through the C ABI with
HOST buffers: dex_prefill from a pinned host prompt, the rounds, dex_get_tokens to the host.

Multi-GPU: the path shards only across independent
sequences -> "replicas only": every rank runs its own replica of the workload, no collective on
the data path, scaling = weak.

`--impl reference` times the CPU oracle (oracle/, NumPy fp32, as it stands) on a bounded sample
of the same workload; rank 0 only.
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

import numpy as np

METRIC = "committed_tokens_per_s"
UNIT = "tokens/s"
NOMINAL_HBM_GBS = 8000.0          # the denominator BASELINE.json:metric names
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent


def measured_hbm_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic_ratio():
    """DRAM (read + write) bytes / algorithmic bytes of k_round from the committed `ncu --set full` capture
    (profiles/k_round_r*_traffic.csv, newest round); None if absent."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "k_round_r*_traffic.csv")))
    if not files:
        return None, None
    dram = alg = 0.0
    with open(files[-1]) as f:
        for row in csv.DictReader(f):
            dram += float(row["dram_read_bytes"]) + float(row["dram_write_bytes"])
            alg += float(row["algorithmic_bytes"])
    return (dram / alg if alg > 0 else None), os.path.relpath(files[-1], ROOT)


def ncu_tensor_pipe(workload):
    """sm__pipe_tensor_cycles_active of the dominant kernel from the committed ncu capture of this workload (SURVEY 8(d):
    to be reported where stages are wide); None if no capture exists for it."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "tensor_pipe_r2.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload:
                    return {"active_pct": float(row["sm__pipe_tensor_cycles_active_pct"]), "kernel": row["kernel"],
                            "source": "NOT a counter of this run: " + row["source"]}
    except Exception:
        pass
    return None


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln)

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.thread.join(timeout=2)
        sm, mx, pw, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def replica_prompt_seq(rank):
    """Multi-GPU = replicas only: rank r decodes its own independent sequence, drawn
    from the workload's prompt seed with sequence id r.  No data-path collective exists."""
    return int(rank)


def max_over_ranks(ms, world, device=None):
    """Device time of the slowest rank (the job's time); identity at world == 1."""
    if world == 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_tokens_per_s(world, steps, tokens_per_step, ms_max):
    """Whole-job throughput: tokens committed by ALL ranks / time of the slowest rank."""
    return world * steps * tokens_per_step / (ms_max * 1e-3)


def run_rounds(g, T, flags, S=1):
    """DEX rounds until every one of the S batched sequences has committed T tokens (a sequence that is done keeps
    stepping with the others, as in a serving batch; only its first T tokens count).  Returns (#rounds,
    layer_evals, critical_layers, k histogram)."""
    n = [0] * S
    rounds, evals, crit = 0, 0, 0
    hist = [0] * 8
    while min(n) < T:
        res = g.step(flags)
        rounds += 1
        alive = False
        for s in range(S):
            r = res[s]
            if n[s] < T:
                evals += r.layer_evals
                crit += r.critical_layers
            if r.committed and n[s] < T:
                n[s] += 1
                hist[r.match_k] += 1
            alive |= bool(r.active and not r.done)
        if not alive:
            break
    return rounds, evals, crit, hist


def time_steps(torch, g, n_prompt, T, K, flags, S=1):
    """K steps (rewind + T committed tokens per sequence each) between two CUDA events on the library's stream."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    stats = None
    e0.record(g.stream)
    for _ in range(K):
        for s_ in range(S):
            g.rewind(s_, n_prompt)
        stats = run_rounds(g, T, flags, S)
    e1.record(g.stream)
    torch.cuda.synchronize()
    return e0.elapsed_time(e1), stats


def bench_dex(args):
    import torch
    import dex_synth
    import paper_2606_29223_b200 as P
    from paper_2606_29223_b200 import build
    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the DEX library has no CPU fallback")
    build.build()
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    wl = dex_synth.workload(args.workload)
    T = args.gen_len or wl.gen_len
    n_prompt = args.prompt_len or wl.prompt_len
    shape, X = wl.shape, wl.depths
    if args.depths:                      # exploration-set sweep (resolution / single-exit ablation)
        X = tuple(int(x) for x in args.depths.split(","))
    N, L = len(X), shape.n_layers
    w_host = dex_synth.make_weights(shape, wl.weight_seed, threads=16)
    w_dev = {k: v.to(device=dev, dtype=(torch.float32 if k.startswith("norm") else torch.bfloat16)).contiguous()
             for k, v in w_host.items()}
    del w_host
    # the prompt lives in PINNED host memory: dex_prefill copies it to the device inside the e2e region
    S = wl.n_seqs                        # independent lattices batched into the same launches (c5: 4)
    prompt_pin = torch.empty((S, n_prompt), dtype=torch.int32).pin_memory()
    prompts = prompt_pin.numpy()
    for s_ in range(S):
        prompts[s_, :] = dex_synth.make_prompt(shape.vocab, n_prompt, wl.prompt_seed, seq=replica_prompt_seq(rank) * S + s_)
    max_ctx = n_prompt + T + 8
    FL = P.DEX_STEP_AUTOCOLLAPSE
    mode = dict(decs=args.decs, sample=1 if args.temperature > 0 else 0, temperature=max(args.temperature, 1e-6),
                sample_seed=args.sample_seed)
    adapters = None
    if args.adapters:                    # inducing-adapter exits: synthetic, untrained
        adapters = dex_synth.make_adapters(shape, N - 1, seed=wl.weight_seed + 1, alpha=1e-3, m=args.adapter_dim)
    g = P.Dex(shape, w_dev, X, max_seqs=S, max_ctx=max_ctx, device=dev, act_planes=args.act_planes, adapters=adapters,
              lookahead=args.lookahead, round_kernel=args.round_kernel, **mode)
    a = P.Dex(shape, w_dev, (L,), max_seqs=S, max_ctx=max_ctx, device=dev, act_planes=args.act_planes,
              round_kernel=args.round_kernel, **mode)
    for s_ in range(S):
        g.prefill(s_, prompts[s_])
        a.prefill(s_, prompts[s_])

    def rewind_all(d):
        for s_ in range(S):
            d.rewind(s_, n_prompt)

    def tokens_all(d):
        return np.stack([d.tokens(s_)[n_prompt:n_prompt + T] for s_ in range(S)])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    def max_ranks(ms):
        return max_over_ranks(ms, world, dev)

    # ---- warm-up (>= 3 steps), also captures the CUDA graphs ----
    W = max(3, args.warmup)
    for _ in range(W):
        rewind_all(g)
        run_rounds(g, T, FL, S)
    for _ in range(2):
        rewind_all(a)
        run_rounds(a, T, FL, S)

    # ---- timed region: K steps, device time, max over ranks ----
    g.profile(0)
    clocks = ClockSampler(local_rank)
    clocks.start()
    barrier()
    ms, (rounds, evals, crit, hist) = time_steps(torch, g, n_prompt, T, args.steps, FL, S)
    barrier()
    clk = clocks.stop()
    _, counters = g.profile(-1)
    ms = max_ranks(ms)
    dex_tokens = tokens_all(g)
    value = job_tokens_per_s(world, args.steps, S * T, ms)

    # ---- same-kernel AR baseline (X = {L}) ----
    a.profile(0)
    barrier()
    ms_ar, (rounds_ar, _, _, _) = time_steps(torch, a, n_prompt, T, args.steps, FL, S)
    barrier()
    _, counters_ar = a.profile(-1)
    ms_ar = max_ranks(ms_ar)
    ar_tokens = tokens_all(a)
    ar_value = job_tokens_per_s(world, args.steps, S * T, ms_ar)
    lossless = bool(np.array_equal(dex_tokens, ar_tokens))

    # ---- e2e: host prompt -> dex_prefill -> rounds -> dex_get_tokens (host), per step ----
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.perf_counter()
    e0.record(g.stream)
    e2e_rounds = 0
    for _ in range(args.steps):
        for s_ in range(S):
            g.prefill(s_, prompts[s_])
        e2e_rounds += run_rounds(g, T, FL, S)[0]
        out = np.stack([g.tokens(s_, n_prompt + T) for s_ in range(S)])
    e1.record(g.stream)
    barrier()
    wall_ms = (time.perf_counter() - t0) * 1e3
    ms_e2e = max_ranks(max(e0.elapsed_time(e1), 0.0))
    assert np.array_equal(out[:, n_prompt:], dex_tokens)
    res_bytes = __import__("ctypes").sizeof(P.DexStepResult)
    e2e = {"value": world * args.steps * S * T / (ms_e2e * 1e-3), "unit": UNIT,
           "h2d_bytes_per_step": int(S * (4 * n_prompt + 4 * g.cfg.max_ctx // g.cfg.page_size + 4)),
           "d2h_bytes_per_step": int(res_bytes * S * e2e_rounds // args.steps + 4 * S * (n_prompt + T)),
           "wall_ms_per_step": wall_ms / args.steps,
           "includes": "dex_prefill of the pinned host prompt, all rounds with per-round host results, dex_get_tokens"}

    # ---- roofline of the dominant kernel: k_round, the persistent round kernel (all layer-steps of all live
    #      stages + the exit head of one round in one launch).  One profiled pass of the same workload with a
    #      CUDA-event pair around every k_round launch on the library's stream (graph replay off);
    #      algorithmic bytes = bf16 weights of the live stages + LM head + committed K/V attended.
    peak, peak_src = measured_hbm_peak()
    roofline, phases = None, None
    if rank == 0:
        rewind_all(g)
        g.profile(1)
        run_rounds(g, T, FL, S)
        ph, ct = g.profile(0)
        k_us, k_launches, k_bytes = ph[1], ct[2], ct[3] + ct[4] + ct[5]
        ach = k_bytes / (k_us * 1e-6) / 1e9
        ratio, ratio_src = ncu_traffic_ratio()
        roofline = {"kernel": "k_round (persistent round kernel: segment GEMMs + glue + lattice attention + fused exit)",
                    "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "frac_of_8TBs": ach / NOMINAL_HBM_GBS, "peak_source": peak_src,
                    "traffic": (ratio * k_bytes / max(1, k_launches)) if (ratio and wl.key == "c2") else None,
                    "traffic_source": (f"NOT a counter of this run: dram read+write / algorithmic = {ratio:.4f} measured by the "
                                       f"committed ncu --set full capture {ratio_src} (c2), x this run's algorithmic bytes "
                                       "per launch") if ratio else None,
                    "lm_head_restream_bytes_per_launch": ct[6] / max(1, k_launches),
                    "tensor_pipe": ncu_tensor_pipe(wl.key),
                    "launches": int(k_launches), "avg_launch_us": k_us / max(1, k_launches),
                    "algorithmic_bytes_per_launch": k_bytes / max(1, k_launches),
                    "share_of_step": k_us / max(1e-9, ph[7] if ph[7] > 0 else sum(ph[:6])),
                    "how": "profiled pass after the timed region: cudaEvent pair around each k_round launch on the "
                           "library stream (graph replay off); bytes = bf16 weights of the live stages + LM head + "
                           "committed K/V attended (dex_profile counters)"}
        # the same rounds through the per-op kernels (round_kernel bypassed): where the time would go without k_round
        rewind_all(g)
        g.profile(2)
        run_rounds(g, T, FL, S)
        ph2, ct2 = g.profile(0)
        names = ("bookkeeping", "segment_gemm", "glue", "attention", "exit_gemm", "commit_collapse")
        phases = {n: ph2[i] / (S * T) for i, n in enumerate(names)}
        phases["unit"] = "us per committed token, per-op kernel path (profiled pass, kernels serialised)"
        phases["k_round_path"] = {"bookkeeping": ph[0] / (S * T), "k_round": ph[1] / (S * T), "commit_collapse": ph[5] / (S * T)}

    # whole-step roofline of the timed region (north_star: weight + KV bytes touched per step)
    step_bytes = (counters[3] + counters[4] + counters[5]) / args.steps
    step_ach = step_bytes * args.steps / (ms * 1e-3) / 1e9
    ar_bytes = (counters_ar[3] + counters_ar[4] + counters_ar[5]) / args.steps
    ar_ach = ar_bytes * args.steps / (ms_ar * 1e-3) / 1e9

    cpu = cpu_baseline(args, wl) if (rank == 0 and world == 1 and not args.no_cpu) else None

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": W,
            "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16", "data": "synthetic",
            "config": {"workload": f"{wl.key}: {shape.name} L={L} d={shape.d_model} X={list(X)} prompt={n_prompt} "
                                   f"gen={T} bs={S} {'greedy' if args.temperature <= 0 else 'sample T=%g' % args.temperature} decs={args.decs}"
                                   + (f" adapters m={adapters['w1'].shape[1]} (random init)" if adapters is not None else "")
                                   + (f" lookahead={args.lookahead}" if args.lookahead else ""),
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "act_planes": args.act_planes, "round_kernel": args.round_kernel,
                       "l2": "inputs larger than L2 (13.5 GB of weights streamed per pass vs 126 MB L2)",
                       "step": "dex_rewind to the prompt + DEX rounds until gen tokens are committed"},
            "clocks": clk, "e2e": e2e, "gpu_launches": int(counters[1]),
            "roofline": roofline, "cpu_baseline": cpu,
            "ar_baseline": {"value": ar_value, "unit": UNIT, "ms_per_token": ms_ar / (args.steps * S * T),
                            "hbm_GBs": ar_ach, "frac_of_measured_peak": ar_ach / peak, "frac_of_8TBs": ar_ach / NOMINAL_HBM_GBS,
                            "what": "same library and kernels, X = {L}"},
            "dex_over_ar": value / ar_value,
            "dex_equals_ar_tokens": lossless,
            "per_token": {"rounds_per_sequence_token": rounds / T, "layer_evals": evals / (S * T), "critical_layers": crit / (S * T),
                          "ms": ms / (args.steps * S * T), "match_k_hist": hist[:N]},
            "step_roofline": {"bytes_per_step": step_bytes, "achieved_GBs": step_ach, "frac_of_measured_peak": step_ach / peak,
                              "frac_of_8TBs": step_ach / NOMINAL_HBM_GBS,
                              "what": "weights of live stages + LM head per round + committed K/V attended, / timed region"},
            "phases": phases,
        }
        print(json.dumps(line))
    g.close()
    a.close()
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
def oracle_sample(wl, n_prompt, n_tokens, n_steps, ar_tokens=0):
    """The CPU oracle (NumPy, fp32 at the 7B-class shapes) on a bounded sample of the workload:
    the workload's model tensors and exploration set, a prompt shortened to `n_prompt` tokens
    (prefill untimed), `n_tokens` committed DEX tokens per step.  Returns (seconds per step list,
    threads)."""
    import copy
    import dex_synth
    import oracle
    shape, X = wl.shape, wl.depths
    w = dex_synth.make_weights(shape, wl.weight_seed, threads=16)
    dt = np.float64 if shape.d_model <= 512 else np.float32
    om = oracle.OracleModel(shape, w, dtype=dt, kv_round="bf16")
    del w
    p = dex_synth.make_prompt(shape.vocab, n_prompt, wl.prompt_seed)
    from oracle.ar import prefill
    state = prefill(om, [int(t) for t in p])
    times = []
    for _ in range(n_steps):
        st = ([list(x) for x in state[0]], [list(x) for x in state[1]])
        t0 = time.perf_counter()
        oracle.dex_decode(om, p, n_tokens, X, decs=True, state=st)
        times.append(time.perf_counter() - t0)
    ar_s = None
    if ar_tokens:                          # CPU AR leg: the oracle's own AR greedy, same tensors
        st = ([list(x) for x in state[0]], [list(x) for x in state[1]])
        t0 = time.perf_counter()
        oracle.ar_greedy(om, p, ar_tokens, state=st)
        ar_s = (ar_tokens, time.perf_counter() - t0)
    try:
        from threadpoolctl import threadpool_info
        threads = max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        threads = os.cpu_count()
    return (times, threads, ar_s) if ar_tokens else (times, threads)


def cpu_baseline(args, wl):
    n_prompt, n_tok = (wl.prompt_len, 16) if wl.key == "c1" else (8, args.cpu_tokens)
    times, threads, ar_s = oracle_sample(wl, n_prompt, n_tok, 1, ar_tokens=max(4, n_tok // 3))
    return {"value": n_tok / times[0], "unit": UNIT, "cores": int(threads), "kind": "oracle",
            "ar_value": ar_s[0] / ar_s[1], "ar_what": f"oracle AR greedy on the same tensors, {ar_s[0]} tokens, {ar_s[1]:.1f} s",
            "sample": f"{wl.key} tensors and X, prompt shortened to {n_prompt} tokens (prefill untimed), "
                      f"{n_tok} committed DEX tokens, NumPy {'fp64' if wl.key == 'c1' else 'fp32'}, {times[0]:.1f} s"}


def bench_reference(args):
    rank, _, world = dist_env()
    if rank != 0:
        return
    import dex_synth
    wl = dex_synth.workload(args.workload)
    n_prompt, n_tok = (wl.prompt_len, 16) if wl.key == "c1" else (8, 2)
    W = min(args.warmup, 1)
    times, threads = oracle_sample(wl, n_prompt, n_tok, W + args.steps)
    t = times[W:]
    value = n_tok * len(t) / sum(t)
    sample = (f"{wl.key} tensors and X, prompt shortened to {n_prompt} tokens (prefill untimed), "
              f"{n_tok} committed DEX tokens per step, NumPy {'fp64' if wl.key == 'c1' else 'fp32'}")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": W, "ms_per_step": 1e3 * sum(t) / len(t), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64" if wl.key == "c1" else "f32", "data": "synthetic",
        "config": {"workload": f"{wl.key}: {wl.shape.name} X={list(wl.depths)} (CPU oracle, bounded sample)", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": int(threads), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="dex", choices=["dex", "reference"])
    ap.add_argument("--workload", default="c2")
    ap.add_argument("--depths", default="", help="comma-separated exploration set X (last = L); default: the workload's")
    ap.add_argument("--decs", type=int, default=1, help="1: DECS masking (Alg. 2), 0: vanilla decoding of the exits")
    ap.add_argument("--temperature", type=float, default=0.0, help="> 0: sampling-mode DECS (Alg. 2 lines 10-15)")
    ap.add_argument("--sample-seed", type=int, default=2024)
    ap.add_argument("--lookahead", type=int, default=0, help="P > 0: sparse lattice, position look-ahead cap (PAPER.md:534)")
    ap.add_argument("--adapters", type=int, default=0, help="1: inducing-adapter exits at the non-final depths (random init)")
    ap.add_argument("--adapter-dim", type=int, default=0, help="adapter width m (0: 2 d_model, the paper's)")
    ap.add_argument("--gen-len", type=int, default=0)
    ap.add_argument("--prompt-len", type=int, default=0)
    ap.add_argument("--act-planes", type=int, default=2)
    ap.add_argument("--round-kernel", type=int, default=1, help="1: k_round (grid barriers), 2: k_flow (dataflow, experimental), 0: per-op kernels")
    ap.add_argument("--cpu-tokens", type=int, default=24, help="committed tokens of the oracle sample (c2: about 13 s of CPU work)")
    ap.add_argument("--no-cpu", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        bench_reference(args)
    else:
        bench_dex(args)


if __name__ == "__main__":
    main()
