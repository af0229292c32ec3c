#!/usr/bin/env python
"""bench.py -- throughput of the sparse, truncated state-vector gate path on B200.

Workload (config.workload = "cfg5"): BASELINE.json configs[4] -- n=56, the 4000-gate
sparse-growth mix from seed 4, sv_truncate(K=2^28, 1-1e-4) after every gate.  The circuit
is first run (untimed) until the state reaches the cap; a "step" is then the next
`--gates-per-step` gates, each applied and truncated: one pass of the whole hot path
(SURVEY.md rows a-1..a-9).  value = amplitude-terms entering a gate, summed over the
timed gates, per second (whole job).  The state (6.4 GB at the cap) is far larger than L2,
so no L2 flush is needed between steps.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "amplitude_terms_per_sec_per_gate"
UNIT = "terms/s"


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--k-log2", type=int, default=28, help="log2 of the hard cap K (28 = the config's own)")
    ap.add_argument("--gates-per-step", type=int, default=32)
    ap.add_argument("--cap-mult", type=int, default=8, help="capacity = cap-mult * K (8 = worst case of an 8x8 gate)")
    ap.add_argument("--two-call", action="store_true",
                    help="time sv_apply_gate + sv_truncate instead of the fused sv_apply_gate_truncate")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=15.0)
    ap.add_argument("--jsonl", default="", help="optional per-gate JSONL log")
    ap.add_argument("--no-circuits", action="store_true", help="skip the circuit wall times of configs 1-5")
    return ap.parse_args()


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured"
        except Exception:
            pass
    return 6650.0, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                       "--format=csv,noheader,nounits", "-lms", "200"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        time.sleep(0.25)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [r.strip().split(",") for r in open(self.f.name) if r.strip()]
        os.unlink(self.f.name)
        sm, mx, reasons = [], [], set()
        for r in rows:
            try:
                sm.append(float(r[1])); mx.append(float(r[2]))
            except Exception:
                continue
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for nm, v in zip(names, r[5:9]):
                if v.strip().lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            out["sm_mhz"] = float(np.median(sm)); out["sm_max_mhz"] = float(max(mx)); out["samples"] = len(sm)
        out["reasons"] = sorted(reasons)
        return out


# ------------------------------------------------------------------------------------------
# CPU oracle arm (cpu_baseline of the default run, and the whole of --impl reference)
# ------------------------------------------------------------------------------------------
def oracle_sample(k_log2_sample, gates_per_step, steps, warmup, budget_s):
    """The oracle, as it stands, on the same cfg5 circuit at a scaled cap: run to the cap,
    then time steps of `gates_per_step` gates (apply + truncate), bounded by budget_s."""
    from oracle.sparse import SparseOracle
    from paper_2607_07816_b200 import workloads as W
    c = W.config5(max_terms=1 << k_log2_sample)
    o = SparseOracle(c.n)
    gi = 0
    while gi < len(c.gates) and o.num_terms() < 0.9 * c.max_terms:
        g = c.gates[gi]; gi += 1
        o.apply_gate(g.qubits, g.U); o.truncate(c.max_terms, c.min_mass)
    terms, secs, done = 0, 0.0, 0
    per_step = []
    t_budget = time.perf_counter()
    for s in range(warmup + steps):
        t0 = time.perf_counter(); nt = 0
        for _ in range(gates_per_step):
            g = c.gates[gi % len(c.gates)]; gi += 1
            nt += o.num_terms()
            o.apply_gate(g.qubits, g.U); o.truncate(c.max_terms, c.min_mass)
        dt = time.perf_counter() - t0
        if s >= warmup:
            terms += nt; secs += dt; done += 1; per_step.append(dt)
        if time.perf_counter() - t_budget > budget_s and done >= 1:
            break
    return {"value": terms / secs if secs > 0 else 0.0, "unit": UNIT, "cores": 1, "nproc": os.cpu_count(), "kind": "oracle",
            "sample": "cfg5 circuit at cap 2^%d (full config: 2^28), %d step(s) of %d gates after reaching the cap, apply+truncate"
                      % (k_log2_sample, done, gates_per_step),
            "steps_done": done, "ms_per_step": 1e3 * secs / max(done, 1)}


def run_reference(args):
    from paper_2607_07816_b200 import dist
    rank, _, world = dist.env_world()
    if rank != 0:
        return
    r = oracle_sample(14, args.gates_per_step, args.steps, min(args.warmup, 1), budget_s=150.0)
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": r["steps_done"], "warmup": min(args.warmup, 1), "ms_per_step": r["ms_per_step"],
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "cfg5", "n_qubits": 56, "K_log2": 28, "min_mass": 1 - 1e-4,
                       "gates_per_step": args.gates_per_step, "sampled_at_K_log2": 14},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": 1, "nproc": os.cpu_count(), "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_circuits(engine, W, dev, torch):
    """Wall time (CUDA events around the whole gate loop, after one untimed run for configs 1-4) of the five
    configs at the sizes BASELINE.json names; truncation after every gate where the config says so."""
    out = {}
    specs = [("cfg1", W.config1(), 1 << 13, 2), ("cfg2", W.config2(), 1 << 22, 2), ("cfg3", W.config3(), (1 << 26) + 1024, 2),
             ("cfg4", W.config4(), 1 << 30, 2), ("cfg5", W.config5(), 1 << 31, 1)]   # cfg5: all 4000 gates, once
    for name, c, cap, reps in specs:
        torch.cuda.empty_cache()      # the previous arena sits in torch's cache; hand it back before asking
        free_b, _ = torch.cuda.mem_get_info(dev)
        if engine.lib.sv_arena_bytes(cap) > 0.9 * free_b:
            out[name] = {"skipped": "arena does not fit"}
            continue
        res = None
        for rep in range(reps):
            sv = engine.SparseSV(c.n, cap, device=dev)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize(); a.record()
            log_kept, peak_terms = 0.0, 1
            try:
                if name in ("cfg1", "cfg2"):     # small / mid-size states: the whole list as ONE call (sv_apply_circuit, look-ahead)
                    kf = sv.apply_circuit([(g.qubits, g.U) for g in c.gates], c.max_terms if c.truncate_every_gate else 0,
                                          c.min_mass if c.truncate_every_gate else 1.0)
                    log_kept = float(np.sum(np.log(kf)))
                for g in (c.gates if name not in ("cfg1", "cfg2") else []):
                    if c.truncate_every_gate:
                        kept = sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)
                        peak_terms = max(peak_terms, sv.stats()["n_mid"])
                        log_kept += float(np.log(kept))
                    else:
                        sv.apply_gate(g.qubits, g.U)
                b.record(); torch.cuda.synchronize()
                k, _, p = sv.top(1)
                res = {"n_qubits": c.n, "gates": len(c.gates), "wall_ms": a.elapsed_time(b), "final_terms": sv.num_terms(),
                       "peak_terms_before_cut": int(peak_terms), "log_retained_mass": log_kept, "top_p": float(p[0]),
                       "norm": sv.norm(), "select_fallbacks": sv.stats()["fallbacks"], "small_path_gates": sv.stats()["small_gates"],
                       "top_is_secret": (int(k[0]) == c.secret) if c.secret is not None else None,
                       "variant": c.notes.get("variant")}
            except engine.SvError as ex:
                res = {"error": str(ex)}
            sv.close()
        out[name] = res
    out["ring44"] = run_ring_scaling(engine, W, dev, torch)
    return out


def run_ring_scaling(engine, W, dev, torch):
    """The paper's own experiment shape: the u3 + cz ring at n = 44 (synthetic
    angles), reordered (sv_reorder_gates) and fused into <= 4-qubit blocks (sv_fuse_gates), one fused call per block
    with top-k truncation, wall time against k (the paper's Fig. 2: time proportional to k).  Second of two runs."""
    c = W.ring_peaked()
    gates = [(list(g.qubits), g.U) for g in c.gates]
    order = engine.reorder_gates(gates, [W.is_diagonal(U) for _, U in gates])
    blocks = engine.fuse_gates([gates[i] for i in order], 4)
    res = {"n_qubits": c.n, "instructions": len(gates), "blocks": len(blocks), "by_K_log2": {}}
    for klog in (6, 12, 16, 20, 24, 26):
        K = 1 << klog
        torch.cuda.empty_cache()
        free_b, _ = torch.cuda.mem_get_info(dev)
        if engine.lib.sv_arena_bytes(16 * K) > 0.9 * free_b:
            res["by_K_log2"][str(klog)] = {"skipped": "arena does not fit"}
            continue
        try:
            for rep in range(2):
                sv = engine.SparseSV(c.n, 16 * K, device=dev)
                a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                torch.cuda.synchronize(); a.record()
                log_kept = float(np.sum(np.log(sv.apply_circuit(blocks, K, 1.0))))      # one call for the whole circuit
                b.record(); torch.cuda.synchronize()
                k, _, p = sv.top(1)
                r = {"wall_ms": a.elapsed_time(b), "final_terms": sv.num_terms(), "log_retained_mass": log_kept,
                     "top_p": float(p[0]), "top_is_secret": int(k[0]) == c.secret, "select_fallbacks": sv.stats()["fallbacks"],
                     "small_path_gates": sv.stats()["small_gates"]}
                sv.close()
            res["by_K_log2"][str(klog)] = r
        except engine.SvError as ex:
            res["by_K_log2"][str(klog)] = {"error": str(ex)}
    return res


# ------------------------------------------------------------------------------------------
# the CUDA engine arm
# ------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_2607_07816_b200 import dist, engine, workloads as W
    rank, local_rank, world = dist.init("nccl")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    K = 1 << args.k_log2
    c = W.config5(max_terms=K)
    free_b, _ = torch.cuda.mem_get_info(dev)
    cap_mult = args.cap_mult
    while cap_mult > 2 and engine.lib.sv_arena_bytes(cap_mult * K) > 0.92 * free_b:
        cap_mult -= 1
    sv = engine.SparseSV(c.n, cap_mult * K, device=dev)
    G = args.gates_per_step
    log = open(args.jsonl, "w") if (args.jsonl and rank == 0) else None

    def ev():
        return torch.cuda.Event(enable_timing=True)

    # ---- untimed ramp: run the circuit until the state sits at the cap ----
    gi = 0
    while gi < len(c.gates) and sv.num_terms() < 0.9 * K:
        g = c.gates[gi]; gi += 1
        sv.apply_gate(g.qubits, g.U); sv.truncate(c.max_terms, c.min_mass)
    ramp_gates = gi

    per_gate = []   # (klass, name, n_in, n_pre, n_kept, passes, e_a0, e_a1 (None: fused call), e_t1)
    fused_default = not args.two_call

    def one_step(record, fused=None, sink=None):
        nonlocal gi
        fused = fused_default if fused is None else fused
        sink = per_gate if sink is None else sink
        nt = 0
        for _ in range(G):
            g = c.gates[gi % len(c.gates)]; gi += 1
            n_in = sv.num_terms()
            if record:
                e0, e1, e2 = ev(), ev(), ev()
                e0.record()
            if fused:
                sv.apply_gate_truncate(g.qubits, g.U, c.max_terms, c.min_mass)
                if record:
                    e2.record()
                    st = sv.stats()
                    sink.append((g.klass, g.name, n_in, st["n_mid"], st["n_out"], st["passes"], e0, None, e2))
            else:
                sv.apply_gate(g.qubits, g.U)
                if record:
                    e1.record()              # (the apply step ends here; stats() is a host-side struct copy)
                    st = sv.stats()
                sv.truncate(c.max_terms, c.min_mass)
                if record:
                    e2.record()
                    sink.append((g.klass, g.name, n_in, st["n_out"], sv.stats()["n_out"], st["passes"], e0, e1, e2))
            nt += n_in
        return nt

    for _ in range(args.warmup):
        one_step(False)
    sv.profile(True)
    l0 = sv.stats()["launches"]
    clocks = ClockSampler(local_rank)
    dist.barrier(); torch.cuda.synchronize()
    clocks.start()
    t_start, t_end = ev(), ev()
    t_start.record()
    terms = 0
    for _ in range(args.steps):
        terms += one_step(True)
    t_end.record()
    torch.cuda.synchronize(); dist.barrier()
    clk = clocks.stop()
    ms = t_start.elapsed_time(t_end)
    launches = sv.stats()["launches"] - l0
    prof = sv.profile_get()
    sv.profile(False)
    tot_terms, max_ms = dist.aggregate(terms, ms, dev)

    # ---- per gate class summary (rank 0) ----
    hbm, peak_kind = peaks()

    def summarise(records, logf):
        classes = {}
        for (kl, name, n_in, n_pre, n_kept, passes, e0, e1, e2) in records:
            total = e0.elapsed_time(e2)
            ta, tt = (e0.elapsed_time(e1), e1.elapsed_time(e2)) if e1 is not None else (None, None)
            d = classes.setdefault(kl, {"gates": 0, "n_in": 0, "ms": 0.0, "apply_ms": 0.0, "trunc_ms": 0.0, "apply_bytes": 0.0,
                                        "trunc_bytes": 0.0, "passes": 0, "split": True})
            d["gates"] += 1; d["n_in"] += n_in; d["ms"] += total; d["passes"] += passes
            d["apply_bytes"] += 24.0 * (n_in + n_pre); d["trunc_bytes"] += 24.0 * (n_pre + n_kept)
            if ta is None:
                d["split"] = False
            else:
                d["apply_ms"] += ta; d["trunc_ms"] += tt
            if logf:
                logf.write(json.dumps({"class": kl, "gate": name, "n_in": n_in, "n_pre": n_pre, "n_kept": n_kept, "passes": passes,
                                       "ms": total, "apply_ms": ta, "trunc_ms": tt}) + "\n")
        out = {}
        for kl, d in classes.items():
            o = {"gates": d["gates"], "mean_passes": d["passes"] / d["gates"], "ms_mean": d["ms"] / d["gates"],
                 "terms_per_s": d["n_in"] / (d["ms"] * 1e-3) if d["ms"] > 0 else None}
            if d["split"] and d["apply_ms"] > 0:
                o.update({
                    "apply_terms_per_s": d["n_in"] / (d["apply_ms"] * 1e-3),
                    "apply_roofline_frac_of_8TBs": d["apply_bytes"] / (d["apply_ms"] * 1e-3) / 8.0e12,
                    "apply_roofline_frac_of_measured": d["apply_bytes"] / (d["apply_ms"] * 1e-3) / (hbm * 1e9),
                    "trunc_roofline_frac_of_measured": d["trunc_bytes"] / (d["trunc_ms"] * 1e-3) / (hbm * 1e9) if d["trunc_ms"] > 0 else None,
                    "apply_ms_mean": d["apply_ms"] / d["gates"], "trunc_ms_mean": d["trunc_ms"] / d["gates"]})
            out[kl] = o
        return out

    per_class = summarise(per_gate, log)
    # the same gates through the two separate calls, after the timed region: the apply / truncate split per class
    per_class_two_call = None
    if fused_default:
        two = []
        g_keep = gi
        for _ in range(min(args.steps, 3)):
            one_step(True, fused=False, sink=two)
        torch.cuda.synchronize()
        gi = g_keep
        per_class_two_call = summarise(two, None)

    dom = max(prof, key=lambda k: prof[k]["ms"])
    dk = prof[dom]
    ach = dk["alg_bytes"] / (dk["ms"] * 1e-3) / 1e9 if dk["ms"] > 0 else 0.0
    # dram__bytes_read + dram__bytes_write of one captured launch of that kernel at this workload, from the committed
    # ncu --set full summary of this round (profiles/r2_traffic.json names the capture); null if it has no entry
    traffic, traffic_note = None, None
    tp = os.path.join(ROOT, "profiles", "r2_traffic.json")
    if os.path.exists(tp):
        try:
            t = json.load(open(tp)).get(dom)
            if t:
                traffic, traffic_note = t["dram_bytes_per_launch"], t.get("note")
        except Exception:
            pass
    kern = {k: {"ms": v["ms"], "launches": v["launches"],
                "GBs": (v["alg_bytes"] / (v["ms"] * 1e-3) / 1e9) if v["ms"] > 0 else None,
                "frac_of_measured": (v["alg_bytes"] / (v["ms"] * 1e-3) / 1e9 / hbm) if v["ms"] > 0 else None} for k, v in prof.items()}
    timed = [k for k in kern if kern[k]["launches"] and k != "sel_hist"]       # (the select levels run on candidates: O(1 %) of the state)
    low = min(timed, key=lambda k: kern[k]["frac_of_measured"]) if timed else None
    # what north_star grades: per gate class, the apply step as a fraction of 24 B x (N_in + N_out) at 8 TB/s (and at the
    # measured copy peak), from the two-call diagnostic steps; the fused call's ms per gate beside it
    targets = {"diag": 0.60, "perm": 0.60, "gen1": 0.40, "gen2": 0.40, "gen3": 0.40}
    pc_roof = {}
    for kl, tgt in targets.items():
        two = (per_class_two_call or {}).get(kl) or (per_class.get(kl) if not fused_default else None)
        o = {"target_frac_of_8TBs": tgt, "fused_ms_per_gate": per_class.get(kl, {}).get("ms_mean") if fused_default else None}
        if two and "apply_roofline_frac_of_8TBs" in two:
            o.update({"apply_frac_of_8TBs": two["apply_roofline_frac_of_8TBs"], "apply_frac_of_measured": two["apply_roofline_frac_of_measured"],
                      "apply_ms_per_gate": two["apply_ms_mean"], "trunc_ms_per_gate": two["trunc_ms_mean"], "mean_passes": two["mean_passes"],
                      "gates": two["gates"], "meets_target": bool(two["apply_roofline_frac_of_8TBs"] >= tgt)})
        pc_roof[kl] = o
    # the whole path of the timed region: one read of every gate's input + one write of what it keeps, against the time
    path_bytes = sum(24.0 * (r[2] + r[4]) for r in per_gate)
    whole = {"alg_bytes": path_bytes, "frac_of_8TBs": path_bytes / (ms * 1e-3) / 8.0e12, "frac_of_measured": path_bytes / (ms * 1e-3) / (hbm * 1e9),
             "definition": "sum over timed gates of 24 B x (N_in + N_kept) / device time of the timed region"}
    roofline = {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": hbm, "unit": "GB/s", "frac": ach / hbm,
                "traffic": traffic, "traffic_note": traffic_note, "peak_kind": peak_kind, "launches": dk["launches"],
                "avg_launch_ms": dk["ms"] / max(dk["launches"], 1),
                "alg_bytes_per_launch": dk["alg_bytes"] / max(dk["launches"], 1),
                "share_of_timed_region": dk["ms"] / ms if ms > 0 else None,
                "lowest": {"kernel": low, "frac": kern[low]["frac_of_measured"], "GBs": kern[low]["GBs"]} if low else None,
                "kernels": kern, "per_class": pc_roof, "whole_path": whole}

    # ---- e2e: host state in, top-k out, through the same C ABI ----
    e2e = None
    if not args.no_e2e:
        n_state = sv.num_terms()
        hk, ha, _ = sv.export()                       # untimed: the step's input, on the host
        tk = torch.from_numpy(hk.view(np.int64)).pin_memory()
        ta = torch.from_numpy(ha).pin_memory()
        hk_p, ha_p = tk.numpy().view(np.uint64), ta.numpy()
        g_start = gi
        e_terms, e_ms, e_steps = 0, 0.0, max(1, min(args.steps, 3))
        d2h = 0
        for s in range(1 + e_steps):
            gi = g_start
            dist.barrier(); torch.cuda.synchronize()
            a, b = ev(), ev()
            a.record()
            sv.load(hk_p, ha_p)                       # H2D of this step's input state (pinned)
            nt = one_step(False)
            topk = sv.top(16)                         # D2H of the step's result
            b.record(); torch.cuda.synchronize()
            if s >= 1:
                e_ms += a.elapsed_time(b)
                e_terms += nt
            d2h = int(topk[0].nbytes + topk[1].nbytes + topk[2].nbytes)
        et, em = dist.aggregate(e_terms, e_ms, dev)
        e2e = {"value": et / (em * 1e-3), "unit": UNIT, "h2d_bytes_per_step": int(hk_p.nbytes + ha_p.nbytes + G * 16 * 64),
               "d2h_bytes_per_step": d2h, "steps": e_steps,
               "note": "sv_load(host pinned state) + %d x (the same call as the timed region) + sv_top(16); same gates every step" % G}

    # ---- circuit wall times of BASELINE.json configs[0..4] at their full sizes (reported, not the headline) ----
    circuits = None
    if rank == 0 and world == 1 and not args.no_circuits:
        sv.close()
        circuits = run_circuits(engine, W, dev, torch)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_sample(16, G, 2, 0, budget_s=args.cpu_seconds)
        for k in ("steps_done", "ms_per_step"):
            cpu.pop(k, None)

    if rank == 0:
        line = {"metric": METRIC, "value": tot_terms / (max_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": max_ms / args.steps, "higher_is_better": True, "scaling": "weak",
                "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": "cfg5", "n_qubits": c.n, "K_log2": args.k_log2, "min_mass": c.min_mass,
                           "gates_per_step": G, "call": "sv_apply_gate + sv_truncate" if args.two_call else "sv_apply_gate_truncate",
                           "capacity_terms": cap_mult * K, "ramp_gates": ramp_gates,
                           "l2": "inputs larger than L2 (state %.2f GB)" % (24.0 * K / 1e9),
                           "parallelism": "replicas x%d" % world},
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clk,
                "per_class": per_class, "per_class_two_call": per_class_two_call, "circuit_ms_per_gate": max_ms / (args.steps * G), "circuits": circuits}
        print(json.dumps(line), flush=True)
    if log:
        log.close()
    sv.close()
    dist.shutdown()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
