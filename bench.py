#!/usr/bin/env python
"""bench.py — GKR prover gates/s (all layers, device-timed) on BASELINE.json's configs, one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config k] [--impl ours|reference] [--schedule s]

A "step" is one pass of the whole hot path (vc_evaluate + vc_prove_layer for every layer)
over one synthetic input that is already resident in HBM.  N=1 workload: BASELINE.json configs[1]
(F2 circuit, n = 2^20).  N>1: replicas only: every rank proves its own instance of the
same circuit (data seed + rank), no data-path collective; value = gates of all ranks / max-over-ranks time.
See DESIGN.md "Measurement" for the algorithmic byte / multiply counts used in the roofline objects.
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
sys.path.insert(0, ROOT)

import vc_workloads as W  # noqa: E402

METRIC = "GKR prover gates/sec (all layers, device-timed)"
UNIT = "gates/s"


# ---------------------------------------------------------------------------------------------- counts
def algorithmic_counts(c):
    """Algorithmic bytes and mod-p multiplies of one step, from SURVEY.md §8(d).

    per gate-round: 9 B record + 16 B weight read+write + 8 B fixed operand (phase 1 only) -> 33 B / 25 B;
    per layer: two shrinking fold tables (read 8*2^(s-j), write half: ~24*2^s B per phase), one 8*2^s B pass for
    the line restriction, 8*2^{s_i} B to write the beta weights; evaluation: 9 B record + 16 B operands + 8 B result.
    multiplies: 3 per gate-round, 2^{s_i} (beta), ~2*2^s (folds), (s-1)*2^s (line), 1 per MULT gate (evaluation).
    """
    per_layer = []
    for i, L in enumerate(c.layers):
        n, s = 1 << L.log_size, c.log_below(i)
        nb = 1 << s
        if i == 0 and c.sum_output:      # the sum gate: s rounds over the shrinking table, read 8*2^(s-j) and write half per round
            per_layer.append(dict(n=1, s=s, prove_bytes=24 * nb, round_bytes=[12 * (nb >> j) for j in range(s)],
                                  eval_bytes=8 * nb, modmul=nb, modmul_eval=0))
            continue
        rounds_bytes = n * s * (33 + 25)
        table_bytes = 2 * 24 * nb
        line_bytes = 8 * nb
        beta_bytes = 8 * n
        eval_bytes = n * 33
        mm = 3 * n * 2 * s + n + 2 * nb + max(s - 1, 0) * nb
        mm_eval = int(np.count_nonzero(L.type == W.MULT))
        per_layer.append(dict(n=n, s=s, prove_bytes=rounds_bytes + table_bytes + line_bytes + beta_bytes,
                              round_bytes=[n * (17 + (8 if ph == 1 else 0)) + 8 * (nb >> j) for ph in (1, 2) for j in range(s)],
                              eval_bytes=eval_bytes, modmul=mm, modmul_eval=mm_eval))
    return dict(layers=per_layer,
                bytes=sum(l["prove_bytes"] + l["eval_bytes"] for l in per_layer),
                modmul=sum(l["modmul"] + l["modmul_eval"] for l in per_layer))


FUSED_SOURCES = ("fp61.cuh", "vc_state.cuh", "vc_kernels.cuh", "vc_fused.cu", "vc_fused.cuh", "vc_fused_line.cuh", "vc_fused_small.cuh",
                 "vc_fused_thin.cuh", "vc_fused_wide.cuh", "vc_cluster.cuh")


def csrc_digest() -> str:
    """SHA-256 over the device sources the fused proof kernels (k_fused<*>, k_cluster, k_eval_all) are compiled from — the
    translation unit vc_fused.cu and every .cuh it includes: ties profiles/r02_traffic.json to the kernel it was captured on."""
    import hashlib
    h = hashlib.sha256()
    base = os.path.join(ROOT, "paper_1202_1350_b200", "csrc")
    for name in FUSED_SOURCES:
        with open(os.path.join(base, name), "rb") as f:
            h.update(name.encode()); h.update(f.read())
    return h.hexdigest()


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ---------------------------------------------------------------------------------------------- clocks
class ClockSampler(threading.Thread):
    """One `nvidia-smi --query-gpu=... -lms 20` process for the whole timed part (the recipe's clocks line in
    B200_PROFILING.md), started before and killed after: forking a fresh nvidia-smi per sample re-initialises the driver
    library every time (the interval itself does not matter: 20 to 200 ms measured the same)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.samples, self.stop_flag, self.proc = index, [], threading.Event(), None

    def run(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-i", str(self.index),
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                parts = [p.strip() for p in line.split(",")]
                if len(parts) >= 6:
                    self.samples.append(parts)
                if self.stop_flag.is_set():
                    break
        except Exception:
            pass

    def summary(self):
        self.stop_flag.set()
        if self.proc is not None:
            try:
                self.proc.terminate()
            except Exception:
                pass
        if self.ident is not None:
            self.join(timeout=6)
        sm = [float(s[0]) for s in self.samples if s and s[0].replace(".", "").isdigit()]
        mx = [float(s[1]) for s in self.samples if len(s) > 1 and s[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = sorted({n for s in self.samples for n, v in zip(names, s[2:6]) if v.lower().startswith("active")})
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------- oracle legs
def oracle_full_proof(k: int):
    """The oracle as it stands, one thread, whole proof of config k. Returns (seconds, gates)."""
    import oracle
    c = W.config(k)
    oc = oracle.OracleCircuit(c)
    t0 = time.perf_counter()
    oc.prove(c.input, W.challenge_seed(k))
    return time.perf_counter() - t0, c.gates


def oracle_sample_step(oc, c, V, seed, layers):
    """Oracle proves the sampled layers in isolation (entry state from the counter-based draws)."""
    import oracle  # noqa: F401
    gr = 0
    for i in layers:
        z, claim, ctr = oc.layer_entry(i, seed, V[i])
        oc.prove_layer(i, V[i + 1], seed, ctr, z, claim, debug=False)
        gr += (1 << c.layers[i].log_size) * 2 * c.log_below(i)
    return gr


def workload_config(c, k, world=1, schedule=0):
    """The `config` object of the bench line: the same keys for both arms."""
    return {"workload": f"BASELINE.json configs[{k - 1}]: {c.name}" if k else f"paper scale (not a BASELINE.json config): {c.name}",
            "gates": c.gates, "layers": c.d, "rounds": c.rounds, "gate_rounds": c.gate_rounds, "replicas": world,
            "schedule": schedule}


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only).

    There is no reference implementation to install (/root/reference holds PAPER.md only), so the reference arm is the
    oracle.  One whole oracle proof of config 2 takes ~6 s: a step is therefore a BOUNDED SAMPLE of the workload — evaluate
    the circuit, then prove a fixed set of its layers in isolation (their entry state comes from the counter-based
    draws) — and `value` is the throughput of that sample in the metric's unit: the sample's share of the circuit's gates
    (by gate-rounds, the oracle's cost driver) divided by the measured time of the step.  `ms_per_step` is the measured
    time of the sample, nothing is extrapolated.
    """
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    k = args.config
    c = W.config(k)
    seed = W.challenge_seed(k)
    oc = oracle.OracleCircuit(c)
    # sample: the layers whose gate-rounds sum to ~6 M (about half a second of oracle time), widest first that fits
    order = sorted(range(c.d), key=lambda i: -(1 << c.layers[i].log_size) * c.log_below(i))
    budget, layers, tot = 6_000_000, [], 0
    for i in order:
        gr = (1 << c.layers[i].log_size) * 2 * c.log_below(i)
        if tot + gr <= budget:
            layers.append(i)
            tot += gr
    layers = sorted(layers) or [c.d - 1 if c.gate_rounds < budget else 0]
    V = oc.evaluate(c.input)
    for _ in range(args.warmup):
        oracle_sample_step(oc, c, V, seed, layers)
    t0 = time.perf_counter()
    gr = 0
    for _ in range(args.steps):
        V = oc.evaluate(c.input)
        gr += oracle_sample_step(oc, c, V, seed, layers)
    dt = (time.perf_counter() - t0) / args.steps          # measured seconds per step (one sample)
    gr //= args.steps
    sample_gates = c.gates * gr / c.gate_rounds            # the sample's share of the circuit, in gates
    value = sample_gates / dt
    sample = (f"per step: evaluate + oracle proof of layers {layers[0]}..{layers[-1]} ({len(layers)} layers, {gr} of "
              f"{c.gate_rounds} gate-rounds = {sample_gates:.0f} gate-equivalents) in isolation, {dt:.3f} s measured; "
              f"value = gate-equivalents / measured time, no extrapolation")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u64 (F_p, p=2^61-1)", "data": "synthetic",
            "config": workload_config(c, k, 1, 0),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------- our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    import ctypes as C
    import paper_1202_1350_b200 as vc

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    k = args.config
    c = W.config(k)
    if args.f2_log_n and not args.paper_scale:
        args.paper_scale = f"f2:{args.f2_log_n}"
    if args.paper_scale:                         # paper-scale workloads: the constructions of configs 2-5 at Table 2's sizes
        from vc_workloads import circuits
        kind, n = args.paper_scale.split(":")
        n = int(n)
        c = {"f2": lambda: circuits.f2_circuit(n, W.data_seed(2)), "f0": lambda: circuits.f0_circuit(n, W.data_seed(3)),
             "matmul": lambda: circuits.matmul_circuit(n, W.data_seed(4)),
             "matmuleq": lambda: circuits.matmul_eq_circuit(n, W.data_seed(4)),
             "f2sum": lambda: circuits.f2_sum_circuit(n, W.data_seed(2)), "f0sum": lambda: circuits.f0_sum_circuit(n, W.data_seed(3)), "pm": lambda: circuits.pm_circuit(n, 3, W.data_seed(5))}[kind]()
        k = 0
    from paper_1202_1350_b200 import replicas
    c.input = replicas.replica_input(c.input, W.data_seed(k or 2), rank)   # replicas: same circuit, another seeded input
    seed = W.challenge_seed(k or 2)
    L = vc.lib()
    gc = vc.Circuit(c, hosted_chunk_log=args.hosted_chunk_log or None)
    if args.hosted_chunk_log:
        gc.set_hosted_weights(args.hosted_swap)
        args.schedule = 2                        # the one schedule of a hosted handle (copy-every-message)
    gc.set_schedule(args.schedule)
    gc.set_input(c.input)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")

    def step():
        gc.evaluate(stream)
        gc.prove(seed, stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    if args.round_trace:                         # -DVC_TRACE builds only: where the cycles of the wide (k_fused<4>) rounds go, as CTA 0 sees them
        from collections import defaultdict
        for _ in range(3):
            step()
            torch.cuda.synchronize()
        n = 60000
        h = np.zeros(n, dtype=np.uint64)
        assert L.vc_debug_trace(gc.handle, h.ctypes.data, n, None) == 0
        codes = (h >> np.uint64(48)).astype(np.int64)
        clk = (h & np.uint64((1 << 48) - 1)).astype(np.int64)
        if not codes.any():
            print("no trace words: build with VC_NVCC_EXTRA=-DVC_TRACE (paper_1202_1350_b200/build.py)")
            gc.close()
            return
        end = int(np.argmax(codes == 0)) if (codes == 0).any() else n
        names = {("L", 11): "set-up (beta, gate state, start claim)", (11, 12): "barrier", (12, 13): "level build / phase switch", (13, 14): "barrier: level j ready",
                 (14, 21): "gate loop (a4 + pending a6)", (21, 15): "commit", (15, 16): "barrier + rendezvous + barrier", (16, 13): "fold of level j (+ publish)",
                 (16, 12): "phase switch (eq tables, phase-2 state)", (16, 17): "after the last round", (17, 70): "line restriction: start",
                 (70, 71): "line: points l(t)", (71, 72): "line: 8 words -> cubic -> P points per thread", (72, 73): "line: barrier", (73, 74): "line: block fold tree",
                 (74, 75): "line: Lagrange continuation", (75, 76): "line: eq weight + accumulate", (76, 72): "line: next block", (76, 18): "line: grid all-reduce",
                 (18, 19): "line_finish (tau, z, claim)"}
        layer, prev, acc, out = -1, None, None, []
        for cd, t in zip(codes[:end], clk[:end]):
            if cd >= 100 + c.d:                  # not a mark: the end of what this launch wrote
                break
            if cd >= 100:                        # 100 + layer: a layer starts
                if layer >= 0:
                    out.append((layer, acc))
                layer, acc, prev = int(cd) - 100, defaultdict(lambda: [0, 0]), (int(cd), int(t))
                continue
            if prev is None:
                continue
            key = ("L" if prev[0] >= 100 else prev[0], int(cd))
            acc[key][0] += 1
            acc[key][1] += int(t) - prev[1]
            prev = (int(cd), int(t))
        if layer >= 0:
            out.append((layer, acc))
        print("SM-clock cycles between trace marks of CTA 0, last launch of the proof (the wide layers); codes: vc_fused_wide.cuh VC_TR(n), 70..76 = line restriction")
        for layer, d in out:
            tot = sum(v[1] for v in d.values())
            print(f"layer {layer}: {tot} cycles")
            for (a_, b_), (cnt, cyc) in sorted(d.items(), key=lambda kv: -kv[1][1]):
                print(f"   {str(a_):>3}->{b_:<3} n={cnt:3d} avg={cyc / cnt:8.0f} sum={cyc:8d} {100 * cyc / tot:5.1f}%  {names.get((a_, b_), '')}")
        gc.close()
        return
    if args.layer_times:                         # per-layer device time of warm proofs (%globaltimer stamps of the fused kernels): not a bench value
        best = None
        for _ in range(5):
            step()
            torch.cuda.synchronize()
            st = gc.layer_stamps().astype(np.int64)
            dt = np.diff(st) / 1e3
            best = dt if best is None else np.minimum(best, dt)
        tot = 0.0
        for i in range(c.d):
            n, s = c.layers[i].log_size, c.log_below(i)
            gr = (1 << n) * 2 * s
            print(f"layer {i:3d} n=2^{n:2d} s={s:2d} rounds={2 * s:3d} {best[i]:9.1f} us {best[i] / (2 * s):8.2f} us/round {gr / best[i] / 1e3:9.2f} Ggr/s")
            tot += best[i]
        print(f"total us {tot:.3f} (min over 5 warm proofs, per layer; includes the launch gap where a new kernel starts)")
        gc.close()
        return
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.3)
    # ---- device-timed steps, inputs resident; L2 flushed between steps outside the event pairs
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    l0 = L.vc_launch_count()
    barrier()
    for a, b in evs:
        flush.fill_(1)
        a.record(stream)
        step()
        b.record(stream)
    barrier()
    launches = int(L.vc_launch_count() - l0)
    ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = float(sum(ms))
    # ---- end to end through the C ABI with host buffers (pinned), copies inside the timed region
    h_in = torch.from_numpy(np.ascontiguousarray(c.input).view(np.int64)).pin_memory()
    h_out = torch.zeros(gc.n_out, dtype=torch.int64).pin_memory()
    h_tr = torch.zeros(gc.words, dtype=torch.int64).pin_memory()
    # untimed warm-up of the end-to-end path: at least W calls and at least 0.3 s of them — the first ~20 copies from a fresh
    # pinned buffer run at a quarter of the link's rate on this pool (H2D of 8.4 MB: 0.70 ms, then 0.16 ms), which is the host
    # link waking up, not the library
    e2e_warm, t_w = 0, time.perf_counter()
    while e2e_warm < max(args.warmup, 3) or time.perf_counter() - t_w < 0.3:
        vc.vc_run_host(gc.handle, h_in, seed, h_out, h_tr, stream)
        e2e_warm += 1
    barrier()
    e2e_ms, e2e_list = 0.0, []
    for _ in range(args.steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        vc.vc_run_host(gc.handle, h_in, seed, h_out, h_tr, stream)
        b.record(stream)
        torch.cuda.synchronize()
        e2e_ms += a.elapsed_time(b)
        e2e_list.append(a.elapsed_time(b))
    barrier()
    clocks = sampler.summary()
    total_ms, e2e_ms = replicas.max_over_ranks([total_ms, e2e_ms], device="cuda")
    ms_per_step = total_ms / args.steps
    value = replicas.whole_job_value(c.gates, world, ms_per_step)
    e2e_value = replicas.whole_job_value(c.gates, world, e2e_ms / args.steps)

    if rank == 0:
        # ---- per-kernel-kind timing (CUDA events inside the library, on the launching stream), three extra steps
        counts = algorithmic_counts(c)
        peak, peak_src = measured_peaks()
        nk = 10
        kinds = ["evaluate", "setup(beta,start)", "round", "update+fold", "line", "fused_narrow", "fused_wide", "misc", "fused_thin", "cluster"]
        acc_l, acc_ms, nprof = [0] * nk, [0.0] * nk, 3
        for _ in range(nprof):
            flush.fill_(1)
            L.vc_profile_enable(1)
            step()
            pl, pm = (C.c_uint64 * nk)(), (C.c_double * nk)()
            L.vc_profile_read(pl, pm)
            L.vc_profile_enable(0)
            for i in range(nk):
                acc_l[i] += int(pl[i]); acc_ms[i] += float(pm[i])
        prof = {kinds[i]: {"launches": acc_l[i] // nprof, "ms": round(acc_ms[i] / nprof, 4)} for i in range(nk) if acc_l[i]}
        prof_total = sum(v["ms"] for v in prof.values())
        # algorithmic bytes / multiplies of every kernel kind: the layers IT proves (the library says which), its own time
        kind_bytes, kind_mm = {kk: 0 for kk in kinds}, {kk: 0 for kk in kinds}
        try:
            lk = gc.layer_kinds() if args.schedule == 0 else None
        except Exception:
            lk = None
        for i, lay in enumerate(counts["layers"]):
            kind_bytes["evaluate"] += lay["eval_bytes"]; kind_mm["evaluate"] += lay["modmul_eval"]
            if lk is not None:
                kind_bytes[kinds[int(lk[i])]] += lay["prove_bytes"]; kind_mm[kinds[int(lk[i])]] += lay["modmul"]
            else:                                # streaming schedule: split by step as algorithmic_counts does
                kind_bytes["round"] += sum(lay["round_bytes"]); kind_mm["round"] += 2 * lay["n"] * 2 * lay["s"]
        # integer-multiply rate (fp61 multiplies/s) measured live: 8 independent chains per thread, one CTA set per SM
        sms = torch.cuda.get_device_properties(local).multi_processor_count
        outw = torch.empty(sms * 8 * 256, dtype=torch.int64, device="cuda")
        best = 0.0
        for _ in range(3):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            L.vc_bench_modmul(sms * 8, 256, 4096, 8, outw.data_ptr(), stream.cuda_stream)
            b.record(stream)
            torch.cuda.synchronize()
            best = max(best, sms * 8 * 256 * 4096 * 8 / (a.elapsed_time(b) * 1e-3))
        for kk, v in prof.items():
            if kind_bytes.get(kk):
                v["algorithmic_bytes"] = int(kind_bytes[kk]); v["algorithmic_modmul"] = int(kind_mm[kk])
                v["algorithmic_GBps"] = round(kind_bytes[kk] / (v["ms"] * 1e-3) / 1e9, 1)
                v["hbm_frac"] = round(kind_bytes[kk] / (peak * 1e9) / (v["ms"] * 1e-3), 4)
                v["alu_frac"] = round(kind_mm[kk] / best / (v["ms"] * 1e-3), 4)
        dom = max(prof, key=lambda n_: prof[n_]["ms"])
        dom_bytes, dom_mm, dom_ms = kind_bytes.get(dom, 0), kind_mm.get(dom, 0), prof[dom]["ms"]
        ach = dom_bytes / (dom_ms * 1e-3) / 1e9
        t_hbm = counts["bytes"] / (peak * 1e9)
        t_alu = counts["modmul"] / best
        roof_ms = max(t_hbm, t_alu) * 1e3
        # which bound is the slower one FOR THE DOMINANT KERNEL (BASELINE.json north_star: the roofline is the slower of the two)
        dom_hbm_ms, dom_alu_ms = dom_bytes / (peak * 1e9) * 1e3, dom_mm / best * 1e3
        traffic, traffic_src = None, None         # DRAM bytes of the dominant kernel from the committed ncu capture (not measured in this run)
        try:
            with open(os.path.join(ROOT, "profiles", "r02_traffic.json")) as f:
                tj = json.load(f)
            if k == 2 and args.schedule == 0 and tj.get("kernel_kind") == dom:
                if tj.get("csrc_sha256") == csrc_digest():    # the capture is of THIS kernel source: else no traffic figure
                    traffic = int(tj["dram_bytes_read"]) + int(tj["dram_bytes_write"])
                    traffic_src = f"profiles/r02_traffic.json (ncu --set full capture of commit {tj.get('commit', '?')}, same digest of the fused kernels' sources as this build, one launch)"
                else:
                    traffic_src = "profiles/r02_traffic.json is of another kernel source (digest of the fused kernels' sources differs): no traffic figure for this build"
        except Exception:
            pass
        roofline = {"bound": "hbm" if dom_hbm_ms >= dom_alu_ms else "alu", "kernel": dom,
                    "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                    "what": (f"{dom}: ALGORITHMIC bytes of the layers this kernel proves (SURVEY.md §8(d): 33/25 B per gate-round + tables + "
                             f"line pass + beta write) / its own CUDA-event time, averaged over {nprof} launches; not DRAM traffic "
                             f"(the working set is shared-memory/L2 resident: see `traffic`)"),
                    "kernel_ms": dom_ms, "kernel_algorithmic_bytes": int(dom_bytes), "kernel_algorithmic_modmul": int(dom_mm),
                    "kernel_hbm_bound_ms": dom_hbm_ms, "kernel_alu_bound_ms": dom_alu_ms,
                    "frac_at_8TBps": dom_bytes / 8e12 * 1e3 / dom_ms, "alu_frac": dom_alu_ms / dom_ms,
                    "kernel_share_of_step": dom_ms / prof_total, "per_kind": prof,
                    "step": {"algorithmic_bytes": counts["bytes"], "algorithmic_modmul": counts["modmul"],
                             "hbm_bound_ms": t_hbm * 1e3, "modmul_rate_per_s": best, "alu_bound_ms": t_alu * 1e3,
                             "roofline_ms": roof_ms, "frac": roof_ms / ms_per_step,
                             "frac_at_8TBps": counts["bytes"] / 8e12 * 1e3 / ms_per_step,
                             "alu_frac": t_alu * 1e3 / ms_per_step}}
        # ---- NEXT-1: the verifier with its O(S) sums on the GPU, beside the library's host verifier
        # (outside the timed region; wall clock around the synchronous calls)
        verifier = None
        try:
            vt = []
            for _ in range(5):
                t0 = time.perf_counter()
                verdict = gc.verify_device(seed, stream=stream)
                vt.append((time.perf_counter() - t0) * 1e3)
            h_out, h_tr = gc.outputs().copy(), gc.transcript().copy()
            t0 = time.perf_counter()
            verdict_host = gc.verify(c.input, h_out, seed, h_tr)
            host_ms = (time.perf_counter() - t0) * 1e3
            verifier = {"device_ms": float(np.median(vt)), "host_ms": host_ms, "accept": bool(verdict[0]),
                        "agree": verdict == verdict_host, "kernels": c.d + 2,
                        "what": "vc_verify_transcript_device (d+2 kernels + host round checks) vs vc_verify_transcript (1 host thread)"}
        except Exception as e:                       # never let the extra line break the bench contract
            verifier = {"error": str(e)}
        # ---- the oracle, timed beside it on the host cores (bounded: one whole proof of config 2 is ~15 s)
        cpu = None
        if not args.no_cpu_baseline and k:
            if c.gate_rounds <= 200_000_000:
                sec, gates = oracle_full_proof(k)
                cpu = {"value": gates / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
                       "sample": f"one whole proof of this workload (evaluate + all {c.d} layers), {sec:.1f} s, 1 thread"}
            else:
                import oracle
                oc = oracle.OracleCircuit(c)
                V = oc.evaluate(c.input)
                lay = [max(range(c.d), key=lambda i: (1 << c.layers[i].log_size) * c.log_below(i))]
                t0 = time.perf_counter()
                gr = oracle_sample_step(oc, c, V, seed, lay)
                sec = (time.perf_counter() - t0) * c.gate_rounds / gr
                cpu = {"value": c.gates / sec, "unit": UNIT, "cores": 1, "kind": "oracle",
                       "sample": f"layer {lay[0]} in isolation ({gr} of {c.gate_rounds} gate-rounds), extrapolated by gate-rounds"}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "u64 (F_p, p=2^61-1)", "data": "synthetic",
                "config": dict(workload_config(c, k, world, args.schedule),
                               l2="flushed between steps (256 MiB fill, outside the event pairs)",
                               ms_min=min(ms), ms_median=float(np.median(ms))),
                "clocks": clocks, "gpu_launches": launches,
                "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(c.input.nbytes),
                        "d2h_bytes_per_step": int(8 * (gc.n_out + gc.words)), "ms_per_step": e2e_ms / args.steps,
                        "ms_min": min(e2e_list), "ms_median": float(np.median(e2e_list)), "warmup_calls": e2e_warm},
                "roofline": roofline, "cpu_baseline": cpu, "verifier": verifier}
        if args.hosted_chunk_log:                # copy-every-message: the per-message traffic over the host link, inside the timed steps
            hb = gc.hosted_bytes()
            line["hosted"] = {"chunk_log": args.hosted_chunk_log, "weights": "swapped through host memory" if args.hosted_swap else "recomputed per message", "proof_h2d_bytes": hb[0], "proof_d2h_bytes": hb[1],
                              "note": "records (and, with --hosted-swap, weights) streamed from pinned host memory for every message (PAPER.md:165); counted on top of e2e's input/output copies"}
        print(json.dumps(line), flush=True)
    gc.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--schedule", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--hosted-swap", action="store_true", help="with --hosted-chunk-log: swap the weights through host memory per message (the paper's wording) instead of recomputing them on the device")
    ap.add_argument("--hosted-chunk-log", type=int, default=0, help="time the copy-every-message approach (SURVEY.md §8f NEXT-3): records and weights in pinned host memory, streamed per message in pieces of 2^N gates")
    ap.add_argument("--round-trace", action="store_true", help="with a -DVC_TRACE build: cycles between the trace marks of the wide layers' rounds (CTA 0), and exit")
    ap.add_argument("--layer-times", action="store_true", help="print the per-layer device times of a warm proof (fused schedule) and exit")
    ap.add_argument("--paper-scale", default="", help="f2:N | f0:N | matmul:LOG_M | matmuleq:LOG_M (the single-output circuit of PAPER.md:230) | f2sum:N | f0sum:N (the paper's circuits with ONE sum gate of fan-in n at the output, PAPER.md:220) | pm:LOG_T — time a construction at another size (e.g. f2:23, f0:21, matmul:8, pm:19) instead of a BASELINE.json config; no CPU baseline")
    ap.add_argument("--f2-log-n", type=int, default=0, help="time the F2 construction at n = 2^N instead of a BASELINE.json config (implies --no-cpu-baseline)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
