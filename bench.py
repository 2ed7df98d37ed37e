#!/usr/bin/env python
"""bench.py -- throughput of the BA hot path (libba, include/ba.h) on B200.

A *step* is one full BA iteration (output sweep, input sweep, reductions, update: all SURVEY 8(a)
rows) at BASELINE.json configs[3]: n=24, d=0.70, uniform p0.  A *term* is a pair (x,y) with
emb(y,x)>0; one iteration visits every term once per sweep, i.e. 2 T(n) terms (T(24)=564842295746).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--n 24] [--d 0.70] [--mode enum|fast]
    python bench.py --impl reference ...     # the CPU oracle, as it stands, on the host cores

Prints ONE JSON line (rank 0).  N>1 (torchrun): independent replicas, one per GPU, each a different
d of configs[2]'s sweep around the headline d (replicas only, no collective);
value = terms all ranks processed / max-over-ranks device time.
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


def terms_per_sweep(n):
    """T(n) = sum_k 2^k sum_{i<=n-k} C(n,i)   (Lemma 6)."""
    from math import comb
    return sum((1 << k) * sum(comb(n, i) for i in range(n - k + 1)) for k in range(n + 1))


def config_name(n, d):
    if n == 24 and abs(d - 0.70) < 1e-12:
        return "BASELINE.json configs[3], the headline throughput config"
    if n == 28 and abs(d - 0.80) < 1e-12:
        return "BASELINE.json configs[4]"
    if n == 20:
        return "one d of BASELINE.json configs[2]"
    return "not a BASELINE.json config: parity / profiling size"


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thr = threading.Thread(target=self._read, daemon=True)
            self.thr.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [t.strip() for t in ln.split(",")]
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
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


# ---------------------------------------------------------------------------------------------
# Roofline of the dominant kernel.  The sweeps are bound by plain ALU issue,
# not by HBM (compulsory traffic is ~1e-3 of the term work) and not by tensor cores (no contraction).
#   algorithmic work  : C_MIN lane-instructions per (x,y) term -- integer emb combine (one IDP.2A / IMAD), int->FP64
#                       convert, FP64 FMA, fetch of the gathered operand -- times T(n) terms per launch
#   peak              : MEASURED in this run by libba's microbenchmarks (ba_measure_peaks): per pipe the warp-
#                       instructions per clock per SM, the clock the kernels saw, the SM count.  Per term the path needs
#                       at least 2 FP64-pipe instructions (convert + FMA), 1 integer-multiply-pipe instruction, 1 LDS.64
#                       unless operands are shared, and 4 issue slots; the binding pipe gives the terms/s ceiling, and
#                       peak = C_MIN x that ceiling.  The nominal formula (4 schedulers x 32 lanes x clock) is kept as a
#                       cross-check.
C_MIN = 4
NEED = {"dfma": 2.0, "idp2a": 1.0, "lds64": 1.0, "issue": 4.0}     # pipe instructions per term (c_min per pipe)


def measured_alu_peak(pk):
    """(terms/s ceiling, binding pipe, per-pipe ceilings) from ba_measure_peaks()."""
    rate = {"dfma": pk["dfma"], "idp2a": pk["idp2a"], "lds64": pk["lds64"], "issue": pk["ffma"]}
    per_pipe = {k: rate[k] * 32.0 / NEED[k] * pk["sms"] * pk["sm_mhz"] * 1e6 for k in rate}
    bind = min(per_pipe, key=per_pipe.get)
    return per_pipe[bind], bind, per_pipe


def read_traffic(kernel, n):
    """Per-launch DRAM bytes of `kernel` from the committed ncu --set full summary -- only if that capture was taken at
    this n -- else None."""
    path = os.path.join(ROOT, "profiles", "roofline_traffic.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return d.get(kernel) if int(d.get("n", -1)) == int(n) else None
    except (OSError, ValueError):
        return None


def oracle_sample(n_s, d, K):
    """Time the CPU oracle (as it stands) on a bounded sample: the dense n_s-bit channel, K iterations.
    Returns (terms/s, seconds of BA, seconds of matrix build, threads)."""
    import numpy as np
    from oracle import oracle as orc
    t0 = time.perf_counter()
    E = orc.emb_dense(n_s)
    W = orc.channel(n_s, d, E)
    t_build = time.perf_counter() - t0
    p0 = np.full(1 << n_s, 1.0 / (1 << n_s))
    t0 = time.perf_counter()
    orc.ba_run(W, p0, K)
    t_run = time.perf_counter() - t0
    return 2 * terms_per_sweep(n_s) * K / t_run, t_run, t_build, orc.num_threads()


def run_reference(args, rank, world):
    if rank != 0:
        return
    n_s = args.oracle_n
    import numpy as np
    from oracle import oracle as orc
    E = orc.emb_dense(n_s)
    W = orc.channel(n_s, args.d, E)
    p = np.full(1 << n_s, 1.0 / (1 << n_s))
    for _ in range(args.warmup):
        p = orc.ba_step(W, p)["p_next"]
    t0 = time.perf_counter()
    for _ in range(args.steps):
        p = orc.ba_step(W, p)["p_next"]
    dt = time.perf_counter() - t0
    T = terms_per_sweep(n_s)
    val = 2 * T * args.steps / dt
    sample = (f"dense oracle at its reach: n={n_s}, d={args.d}, uniform p0, one BA iteration per step "
              f"({2 * T} terms); the n={args.n} workload itself needs a 2^{args.n} x 2^{args.n + 1} matrix")
    out = {"impl": "reference", "metric": "xy_channel_terms_per_s", "value": val, "unit": "terms/s",
           "iterations_per_s": args.steps / dt, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic",
           "config": {"workload": f"BDC_d^n BA iteration, n={args.n}, d={args.d}, uniform p0 ({config_name(args.n, args.d)})",
                      "sample": sample},
           "cpu_baseline": {"value": val, "unit": "terms/s", "cores": orc.num_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": val, "unit": "terms/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out), flush=True)


def run_ours(args, rank, world, local_rank):
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2604_05867_b200 as ba
    from paper_2604_05867_b200 import replicas

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libba has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    n = args.n
    d = replicas.replica_d(rank, world, args.d)
    mode = ba.BA_MODE_ENUM if args.mode == "enum" else ba.BA_MODE_FAST
    T = terms_per_sweep(n)
    NX = 1 << n

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    pk = ba.ba_measure_peaks()               # pipe microbenchmarks on this device, before the timed region
    ctx = ba.ba_create(n, d, device=dev)
    ba.ba_set_mode(ctx, mode)
    if args.exact_k >= 0:
        ba.ba_set_exact(ctx, args.exact_k)
    if args.symmetry:
        ba.ba_set_symmetry(ctx, 1)

    # ---- device-resident arm: inputs (p) already in HBM when the timed region starts ---------------
    ba.ba_iterate(ctx, args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    ba.ba_iterate(ctx, args.steps)
    ev1.record()
    barrier()
    ms_total = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    tm = ba.ba_last_timing(ctx)
    setup_ms = ba.ba_setup_ms(ctx)           # the one-off Hc pass (ran inside the warm-up)
    I, U = ba.ba_bounds(ctx)
    hist = ba.ba_get_history(ctx, min(args.steps + args.warmup, 4096))      # {I_t, U_t, log2 Z_t} of every iteration so far
    ms_total = replicas.max_over_ranks(ms_total, world, dev)

    # ---- end-to-end arm: the C ABI with HOST buffers; H2D of p and D2H of p + bounds every step -----
    p_host = torch.empty(NX, dtype=torch.float64).pin_memory()
    p_np = p_host.numpy()
    ba.ba_get_p(ctx, out=p_np)
    e2e_steps = args.e2e_steps if args.e2e_steps > 0 else args.steps
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        ba.ba_set_p(ctx, p_np)            # H2D  8*2^n bytes (validated copy, no renormalisation)
        ba.ba_iterate(ctx, 1)
        ba.ba_bounds(ctx)                 # D2H  16 bytes (synchronises)
        ba.ba_get_p(ctx, out=p_np)        # D2H  8*2^n bytes
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = replicas.max_over_ranks(e2e_s, world, dev)
    ba.ba_destroy(ctx)

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks, peaks_src = load_peaks()
    ms_step = ms_total / args.steps
    value = 2.0 * T * world * args.steps / (ms_total * 1e-3)
    launches_per_iter = 6 if args.mode == "enum" else 2 * n + 4
    # Terms the sweep kernels enumerate one by one: all but the pairs (v, empty) -- 2^m per (high part, prefix) node, T(h)
    # nodes -- which both sweeps sum in factored form (P:181 at the tile boundary).  The roofline
    # counts the enumerated terms only; `value` counts all T(n) terms of the channel, whose contributions are all there.
    m_low = min(n, 8)
    T_enum = T - (1 << m_low) * terms_per_sweep(n - m_low)
    # dominant kernel: the slower sweep (per-kernel CUDA events recorded by libba on the launch stream)
    if args.mode == "enum":
        dom_name, dom_ms = ("k_enum_out", tm["out_ms"]) if tm["out_ms"] >= tm["in_ms"] else ("k_enum_in", tm["in_ms"])
        terms_peak, bind, per_pipe = measured_alu_peak(pk)
        peak = C_MIN * terms_peak / 1e12
        achieved = C_MIN * T_enum / (dom_ms * 1e-3) / 1e12
        oth_ms = min(tm["out_ms"], tm["in_ms"])
        roofline = {"bound": "alu", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "Tinstr/s",
                    "frac": achieved / peak, "traffic": read_traffic(dom_name, n),
                    "other_kernel": {"name": "k_enum_in" if dom_name == "k_enum_out" else "k_enum_out",
                                     "kernel_ms": oth_ms, "frac": C_MIN * T_enum / (oth_ms * 1e-3) / 1e12 / peak},
                    "measured_peaks": {"warp_instr_per_clk_per_sm": {"dfma": pk["dfma"], "idp2a": pk["idp2a"], "lds64": pk["lds64"],
                                                                     "ffma_issue": pk["ffma"]},
                                       "sm_mhz": pk["sm_mhz"], "sms": pk["sms"],
                                       "pipe_instr_per_term": NEED, "binding_pipe": bind,
                                       "terms_per_s_ceiling_by_pipe": per_pipe},
                    "nominal_peak_crosscheck": 148 * 4 * 32 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12,
                    "peak_source": "measured in this run: ba_measure_peaks (libba microbenchmarks), binding pipe x C_MIN",
                    "algorithmic": f"{C_MIN} lane-instructions per enumerated term x {T_enum} terms per launch "
                                   f"(T({n})={T} less the {T - T_enum} pairs (v, empty), summed in factored form)",
                    "kernel_ms": dom_ms, "kernel_terms_per_s": T_enum / (dom_ms * 1e-3),
                    "gather_equiv_GBps": 8.0 * T_enum / (dom_ms * 1e-3) / 1e9,
                    "hbm_peak_GBps": peaks.get("hbm_gbs"), "hbm_peak_source": peaks_src}
    else:
        # FAST mode: n streaming stages per sweep, each reads <= 3 and writes 1 double per element
        stage_bytes = sum(((4 << s) - 1) * (1 << (n - s - 1)) * 8 * 3 for s in range(n))
        dom_ms = max(tm["out_ms"], tm["in_ms"])
        achieved = stage_bytes / (dom_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "k_fast_fwd/k_fast_bwd (n stages)", "achieved": achieved,
                    "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"], "traffic": None,
                    "peak_source": peaks_src, "kernel_ms": dom_ms}

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        val, t_run, t_build, thr = oracle_sample(args.oracle_n, d, args.oracle_iters)
        cpu = {"value": val, "unit": "terms/s", "cores": thr, "kind": "oracle",
               "sample": f"dense oracle at its reach: n={args.oracle_n}, d={d}, uniform p0, {args.oracle_iters} BA iterations "
                         f"in {t_run:.2f} s (+{t_build:.1f} s to build the explicit matrix, not counted); "
                         f"it cannot run n={n} (2^{n} x 2^{n + 1} dense entries)"}

    out = {"metric": "xy_channel_terms_per_s", "value": value, "unit": "terms/s",
           "iterations_per_s": world * args.steps / (ms_total * 1e-3),
           "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms_step,
           "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": (f"BDC_d^n BA iteration, n={n}, d={d}, uniform p0 ({config_name(n, d)})" if args.exact_k < 0 else
                                   f"exact channel BDC_{{n,k}} BA iteration, n={n}, k={args.exact_k}, uniform p0 (not a BASELINE.json config; "
                                   f"the sweeps skip the nodes and prefixes that cannot reach length k)"),
                      "mode": args.mode, "terms_per_iteration": 2 * T,
                      "term_counting": ("effective (exact channel: nodes / prefixes that cannot reach length k are skipped; value counts 2 T(n))"
                                        if args.mode == "enum" and args.exact_k >= 0 else
                                        f"enumerated, except the pairs (v, empty) ({100.0 * (T - T_enum) / T:.1f} % of the terms), which "
                                        "both sweeps sum in factored form (P:181)" if args.mode == "enum" and not args.symmetry else
                                        "effective (complement symmetry: half the terms are enumerated, the rest mirrored)" if args.mode == "enum"
                                        else "effective (FAST mode does not enumerate terms)"),
                      "l2_policy": f"inputs_exceed_l2 (p {8 * NX / 1e6:.0f} MB, q and c {16 * NX / 1e6:.0f} MB each, "
                                   f"Apart {8 * ((2 << max(n - 8, 0)) - 1) * 511 / 1e6:.0f} MB vs 126 MB L2)" if n >= 24
                                   else "arrays fit L2 at this n (not the headline config)",
                      "parallelism": "single GPU" if world == 1 else f"{world} independent replicas (d sweep), no collective"},
           "kernels_ms": {"out_sweep": tm["out_ms"], "in_sweep": tm["in_ms"], "reduce_update": tm["update_ms"]},
           "setup_ms": setup_ms,
           "bounds_bits": {"I_lower": I, "maxD_upper": U, "upper_over_n": U / n,
                           "running_min_upper_over_n": float(hist[:, 1].min()) / n,
                           "upper_over_n_by_iteration": [round(float(v) / n, 9) for v in hist[:, 1]][-32:]},
           "roofline": roofline, "cpu_baseline": cpu, "clocks": clocks,
           "e2e": {"value": 2.0 * T * world * e2e_steps / e2e_s, "unit": "terms/s", "steps": e2e_steps,
                   "ms_per_step": e2e_s / e2e_steps * 1e3,
                   "h2d_bytes_per_step": 8 * NX, "d2h_bytes_per_step": 8 * NX + 16},
           "gpu_launches": launches_per_iter * args.steps}
    print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--n", type=int, default=24)
    ap.add_argument("--d", type=float, default=0.70)
    ap.add_argument("--mode", choices=["enum", "fast"], default="enum")
    ap.add_argument("--oracle-n", type=int, default=14)
    ap.add_argument("--oracle-iters", type=int, default=10)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=0, help="steps of the end-to-end arm (default: --steps)")
    ap.add_argument("--symmetry", action="store_true",
                    help="complement symmetry (ba_set_symmetry): half the terms are enumerated; terms/s is then 'effective'")
    ap.add_argument("--exact-k", type=int, default=-1,
                    help="run the paper's exact channel BDC_{n,k} (ba_set_exact) instead of BDC_d^n; not a BASELINE.json config")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
