#!/usr/bin/env python
"""bench.py -- working-sweep throughput of the checkerboard SU(3) Monte Carlo path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--precision f32|f64]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

Workload (BASELINE.json configs[2], the configuration the metric is quoted on): SU(3), D = 4, 32^4 periodic, beta = 6.0,
hot start seed 42.  One STEP = one pass of the whole hot path = qcd_sweep_measure(beta, 1 heatbath, 4 overrelaxation):
the sweep and the plaquette per plane + Polyakov loop of the new configuration, the plaquette folded into the last pass
(the paper's "working sweep").  metric = composite link updates/s = D*V*steps / time (reading R13).

The line's `value` is the --precision arm (default fp32, 12-real compressed links); the other arm (fp64, 18 reals) is
measured in the same run and reported under "other_precision".  N > 1: independent replicas, one lattice per GPU, no
data-path collective (replicas only) -> weak scaling.

Timing: the timed region (exactly --steps steps between barrier + synchronize, CUDA events, MAX over ranks) is REPEATED:
at least 5 repetitions and until the arm has >= 1 s of device time, so that the power-capped regime of a long run is inside
the window; `ms_per_step` / `value` are the MEDIAN repetition, min / max ride along ("reps").

--impl reference times the CPU oracle (oracle/, as it stands) on a bounded sample of the same workload.
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

DIMS = (32, 32, 32, 32)
BETA, N_HB, N_OR, SEED, NC = 6.0, 1, 4, 42, 3
METRIC = "SU(3) composite link updates/s (1HB+4OR working sweep) at 32^4"
UNIT = "link updates/s"
L2_BYTES = 126 * 1024 * 1024

# bytes of one stored link, and algorithmic (compulsory) link-sizes moved per link-hit: 2D+1 = 9
LINK_BYTES = {"f32": 48, "f64": 144}
LINK_SIZES_PER_HIT = 2 * len(DIMS) + 1
# flops per link-hit EXECUTED by the kernels this file launches: ncu's per-opcode thread-instruction counts
# (sass__thread_inst_executed_true_per_opcode) of one launch / V/2, weighted FFMA2 4, FMUL2 / FADD2 / FFMA / DFMA 2,
# FMUL / FADD / DMUL / DADD / MUFU 1  (profiles/r2_flop_count.md; SURVEY 8(d)'s estimates were 4030 / 4270 / 3270 / 3900)
FLOPS_PER_HIT = {"f32": {"hb": 3925.0, "or": 3701.0}, "f64": {"hb": 3909.0, "or": 3166.0}}
FLOPS_SOURCE = "profiles/r3_final.md: ncu capture of the build at commit 7d96bdb (weights: profiles/r2_flop_count.md)"


# the dominant kernel of each arm (overrelaxation: 32 of the 40 update launches of a step) and its DRAM traffic per launch,
# dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture of this workload (bytes)
OR_KERNEL = {"f32": "su3_update_tiled_kernel<float, x12, OR>", "f64": "su3_update_kernel<double, x18, OR>"}
NCU_TRAFFIC = {"f32": {"or": 222690000, "hb": 223640000}, "f64": {"or": 658940000, "hb": 666810000},
               "source": "profiles/r3_final.md: ncu --set full of the build at commit 7d96bdb (cache flush between ncu replays; "
                         "142 + 24 / 534 + 77 MB read + write with the caches left alone, profiles/r2_c_launch_order.md)"}
# O(N) kernel (instruction-bound): warp-instructions of one half-sweep launch of O(4) 32^4 NHIT = 100, smsp__inst_executed.sum
# of the same capture
ON_WARP_INST = {"f32": 194.76e6, "f64": 237.22e6, "source": "profiles/r3_final.md (ncu --set full; fp32 at commit 7d96bdb, fp64 at 3bb586f)"}
N_SM, SCHEDULERS_PER_SM = 148, 4          # B200: one warp-instruction per scheduler and cycle is the issue limit


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs (of measured)", p
    return 6650.0, "B200_PROFILING.md fallback 6.65 TB/s (of fallback)", {}


# ----------------------------------------------------------------------------- clocks during the timed regions
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.samples, self.windows, self.proc, self.thread = [], [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            parts = [x.strip() for x in line.split(",")]
            if len(parts) >= 7:
                self.samples.append((time.time(), parts))

    def window(self, t0, t1):
        self.windows.append((t0, t1))

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.12)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        load = [p for (t, p) in self.samples if any(a - 0.02 <= t <= b + 0.02 for a, b in self.windows)]
        use = load if load else [p for _, p in self.samples]
        sm, mx, pw, reasons = [], [], [], set()
        for p in use:
            try:
                sm.append(float(p[0])); mx.append(float(p[1])); pw.append(float(p[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), p[3:7]):
                if v == "Active":
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "reasons": sorted(reasons), "samples_under_load": len(load),
                "samples": len(self.samples)}


# ----------------------------------------------------------------------------- our arm
MIN_REPS, MAX_REPS, MIN_DEVICE_MS = 5, 80, 1000.0


def max_over_ranks(torch, dist, x, device="cuda"):
    """replicas only: the one cross-rank operation of the bench is this MAX of the timed region"""
    if dist is None:
        return x
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def timed_reps(torch, dist, sampler, body, steps, min_total_ms=MIN_DEVICE_MS):
    """Repeat the timed region -- barrier + synchronize, CUDA events around exactly `steps` calls of body(), synchronize +
    barrier, MAX over ranks -- at least MIN_REPS times and until min_total_ms of device time has been spent.  Returns the list
    of per-repetition milliseconds (identical on every rank, so every rank leaves the loop together)."""
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    times = []
    while len(times) < MIN_REPS or (sum(times) < min_total_ms and len(times) < MAX_REPS):
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.time()
        e0.record()
        for _ in range(steps):
            body()
        e1.record()
        torch.cuda.synchronize()
        sampler.window(t0, time.time())
        if dist is not None:
            dist.barrier()
        times.append(max_over_ranks(torch, dist, e0.elapsed_time(e1)))
    return times


def rep_stats(times, steps):
    t = sorted(times)
    med = t[len(t) // 2] if len(t) % 2 else 0.5 * (t[len(t) // 2 - 1] + t[len(t) // 2])
    return {"median_ms_per_step": med / steps, "min_ms_per_step": t[0] / steps, "max_ms_per_step": t[-1] / steps,
            "reps": len(t), "device_ms_total": sum(t)}


def time_arm(q, torch, prec_name, steps, warmup, therm, seed, dist, sampler, bulk_copy=False, alternate=True):
    """device-resident timing + end-to-end timing of one precision arm; returns a dict of raw numbers"""
    prec = q.QCD_FP32 if prec_name == "f32" else q.QCD_FP64
    flags = q.QCD_FLAG_COMPRESS12 if prec_name == "f32" else 0
    V = 1
    for d in DIMS:
        V *= d
    out = {"links": len(DIMS) * V}
    with q.Lattice(DIMS, NC, prec, flags, device=torch.device("cuda", torch.cuda.current_device())) as G:
        if bulk_copy:
            G.qcd_set_option(q.QCD_OPT_BULK_COPY, 1)
        if not alternate:
            G.qcd_set_option(q.QCD_OPT_ALTERNATE_ORDER, 0)
        G.qcd_init(q.QCD_HOT, seed)
        for _ in range(therm):                       # setup: move off the hot start (KP acceptance, staple norms)
            G.qcd_sweep(BETA, N_HB, N_OR)
        state = {}

        def working_sweep():
            # update + observables of the new configuration; the plaquette is folded into the last pass (qcd_sweep_measure)
            state["obs"] = G.qcd_sweep_measure(BETA, N_HB, N_OR)

        def separate_calls():
            G.qcd_sweep(BETA, N_HB, N_OR)
            state["obs"] = G.qcd_measure()

        for _ in range(warmup):
            working_sweep()
        # (1) the headline: working sweep = update + measurement, observables returned to the host every step
        G.qcd_set_option(q.QCD_OPT_PROFILE, 1)
        G.qcd_reset_profile()
        n0 = G.qcd_get_launch_count()
        out["work"] = timed_reps(torch, dist, sampler, working_sweep, steps)
        out["launches_per_rep"] = (G.qcd_get_launch_count() - n0) // len(out["work"])
        hb_ms, hb_n = G.qcd_get_profile(q.QCD_KIND_HB)
        or_ms, or_n = G.qcd_get_profile(q.QCD_KIND_OR)
        G.qcd_set_option(q.QCD_OPT_PROFILE, 0)
        plaq, planes, poly = state["obs"]
        out.update(plaquette=plaq, polyakov_abs=abs(poly), hb_ms=hb_ms, hb_n=hb_n, or_ms=or_ms, or_n=or_n)
        # (2) update-only sweep (measurement excluded), profiling events off
        out["update"] = timed_reps(torch, dist, sampler, lambda: G.qcd_sweep(BETA, N_HB, N_OR), steps, min_total_ms=500.0)
        # (3) working sweep with the observables accumulated on the device (no host synchronisation per step)
        G.qcd_accum_reset()

        def accumulate_sweep():
            G.qcd_sweep_measure_accumulate(BETA, N_HB, N_OR)

        out["accum"] = timed_reps(torch, dist, sampler, accumulate_sweep, steps, min_total_ms=500.0)
        # (3b) the working sweep as two calls, with the stand-alone plaquette kernel (what the fusion saves)
        out["separate"] = timed_reps(torch, dist, sampler, separate_calls, steps, min_total_ms=0.0)
        n_acc, s1, _ = G.qcd_accum_get()
        out["acc_plaquette_mean"] = float(s1[:6].mean() / max(n_acc, 1))
        # (4) end to end through the C ABI with HOST buffers: every step uploads the configuration from pinned host
        # memory, runs the working sweep, reads the observables and downloads the configuration.  Exchange layout: the
        # canonical one; for the 12-real arm its compressed form (rows 0,1 of every link, QCD_OPT_EXCHANGE_ROWS01), i.e.
        # exactly the reals the lattice stores -- a third less over the host link, nothing lost
        # `e2e` is always the canonical layout ("full N x N always"); the 12-real arm is timed a second time
        # through its compressed exchange form (e2e_rows01)
        def e2e_arm(key, rows01):
            G.qcd_set_option(q.QCD_OPT_EXCHANGE_ROWS01, 1 if rows01 else 0) if flags & q.QCD_FLAG_COMPRESS12 else None
            nbytes = G.canonical_bytes
            host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
            G.qcd_get_links_ptr(host.data_ptr(), nbytes, 0)

            def e2e_step():
                G.qcd_set_links_ptr(host.data_ptr(), nbytes, 0)
                state["obs"] = G.qcd_sweep_measure(BETA, N_HB, N_OR)
                G.qcd_get_links_ptr(host.data_ptr(), nbytes, 0)

            for _ in range(2):
                e2e_step()
            out[key] = {"times": timed_reps(torch, dist, sampler, e2e_step, steps, min_total_ms=0.0), "h2d": nbytes, "d2h": nbytes + 9 * 8,
                        "exchange": "rows 0,1 of every link, [lex][mu][2][3][re,im] (QCD_OPT_EXCHANGE_ROWS01)" if rows01
                        else "canonical [lex][mu][3][3][re,im]"}

        e2e_arm("e2e", False)
        if flags & q.QCD_FLAG_COMPRESS12:
            e2e_arm("e2e_rows01", True)
        out["sweep_counter"] = G.qcd_get_sweep_counter()
    return out


def time_on_model(q, torch, dist, sampler, with_oracle):
    """The paper's second workload beside the headline (Table 1): O(4) on 32^4, NHIT = 100
    tries per site visit, hot start; one step = qcd_on_sweep + qcd_on_measure (a "working sweep").  Instruction-bound."""
    dims, N, kappa, lam, delta, nhit = DIMS, 4, 0.15, 0.5, 0.5, 100
    V = 1
    for d in dims:
        V *= d
    out = {"workload": "O(4) phi^4 model 32^4, kappa 0.15, lambda 0.5, delta 0.5, NHIT 100, hot start (readings R16-R19)",
           "paper_context": "PAPER.md Table 1: O(4) 32^4 working sweep 0.72 s (single) / 0.99 s (double) on a GeForce GTX 560 Ti"}
    for name, prec in (("f32", q.QCD_FP32), ("f64", q.QCD_FP64)):
        with q.OnLattice(dims, N, prec, device=torch.device("cuda", torch.cuda.current_device())) as G:
            G.qcd_on_init(q.QCD_HOT, SEED)
            state = {}

            def step():
                G.qcd_on_sweep(kappa, lam, delta, nhit)
                state["obs"] = G.qcd_on_measure()

            for _ in range(5):
                step()
            st = rep_stats(timed_reps(torch, dist, sampler, step, 10, min_total_ms=100.0), 10)
            acc, tried = G.qcd_on_get_counts()
            # issue floor: instructions per try x tries / (148 SMs x 4 schedulers x 32 lanes) is not known a priori; report the rate
            out[name] = {"ms_per_sweep": st["median_ms_per_step"], "reps": st, "site_visits_per_s": V / (st["median_ms_per_step"] * 1e-3),
                         "tries_per_s": V * nhit / (st["median_ms_per_step"] * 1e-3), "acceptance": acc / max(tried, 1),
                         "phi2": state["obs"][0], "link": state["obs"][1]}
    if with_oracle:
        from oracle import on
        small = (16, 16, 16, 16)
        O = on.OnOracle(small, N)
        O.init(on.HOT, SEED)
        t0 = time.time()
        O.sweep(kappa, lam, delta, nhit)
        dt = time.time() - t0
        out["cpu_baseline"] = {"value": 16 ** 4 / dt, "unit": "site visits/s", "cores": on.num_threads(), "kind": "oracle",
                               "sample": "one sweep of the same model on 16^4 (%.2f s)" % dt}
    return out


def time_split(q, torch, steps, therm, seed):
    """--split: the lattice divided into 1, 2 and 4 parts on THIS GPU (qcd_split_*) beside the undivided
    lattice, fp32 x12 arm: update-only sweep and sweep + measurement.  The parts run on streams of their own, so a repetition
    is bracketed by two events on torch's stream with a host synchronisation of all work before the second one (the same
    procedure for the undivided lattice, so the rows are comparable with each other; a few microseconds of host latency per
    repetition of >= 40 ms ride along)."""
    prec, flags = q.QCD_FP32, q.QCD_FLAG_COMPRESS12
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def timed(body, sync, reps=7):
        times = []
        for _ in range(reps):
            torch.cuda.synchronize()
            e0.record()
            for _ in range(steps):
                body()
            sync()
            e1.record()
            torch.cuda.synchronize()
            times.append(e0.elapsed_time(e1))
        return rep_stats(times, steps)

    out = {"workload": "SU(3) fp32 x12 32^4 beta 6.0, 1 HB + 4 OR per sweep, every part on the same GPU", "steps": steps, "rows": {}}
    with q.Lattice(DIMS, NC, prec, flags, device=torch.device("cuda", torch.cuda.current_device())) as G:
        G.qcd_init(q.QCD_HOT, seed)
        for _ in range(therm + 3):
            G.qcd_sweep(BETA, N_HB, N_OR)
        u = timed(lambda: G.qcd_sweep(BETA, N_HB, N_OR), torch.cuda.synchronize)
        m = timed(lambda: (G.qcd_sweep(BETA, N_HB, N_OR), G.qcd_measure()), torch.cuda.synchronize)
        out["rows"]["undivided"] = {"sweep_ms": u["median_ms_per_step"], "sweep_measure_ms": m["median_ms_per_step"], "reps": u}
    base = out["rows"]["undivided"]["sweep_ms"]
    for n in (1, 2, 4):
        with q.SplitLattice(DIMS, NC, prec, flags, n_parts=n) as S:
            S.qcd_split_init(q.QCD_HOT, seed)
            for _ in range(therm + 3):
                S.qcd_split_sweep(BETA, N_HB, N_OR)
            u = timed(lambda: S.qcd_split_sweep(BETA, N_HB, N_OR), S.qcd_split_synchronize)
            m = timed(lambda: (S.qcd_split_sweep(BETA, N_HB, N_OR), S.qcd_split_measure()), S.qcd_split_synchronize)
            out["rows"]["%d part%s" % (n, "" if n == 1 else "s")] = {
                "sweep_ms": u["median_ms_per_step"], "sweep_measure_ms": m["median_ms_per_step"], "reps": u,
                "overhead_vs_undivided": u["median_ms_per_step"] / base - 1.0, "halo_bytes_per_substep": S.qcd_split_halo_bytes()}
    return out


def replica_seed(rank):
    """every rank runs an independent lattice of the same workload: same recipe, its own Philox seed"""
    return SEED + rank


def aggregate_value(n_gpus, links_per_replica, steps, ms_total_max):
    """whole-job composite link updates/s: all replicas' links over the slowest rank's time"""
    return n_gpus * links_per_replica * steps / (ms_total_max * 1e-3)


def summarise(arm, prec_name, steps, n_gpus, hbm_peak, fma_peak_tflops):
    """per-arm JSON fragments: value, roofline of the dominant (overrelaxation) kernel, sweep-level fractions"""
    links = arm["links"]
    work, upd = rep_stats(arm["work"], steps), rep_stats(arm["update"], steps)
    ms_step = work["median_ms_per_step"]
    value = aggregate_value(n_gpus, links, 1, ms_step)
    hits = links // (2 * len(DIMS))                                  # links updated by one launch = V/2
    bytes_launch = LINK_SIZES_PER_HIT * LINK_BYTES[prec_name] * hits
    or_us = arm["or_ms"] / max(arm["or_n"], 1) * 1e3
    hb_us = arm["hb_ms"] / max(arm["hb_n"], 1) * 1e3
    achieved = bytes_launch / (or_us * 1e-6) / 1e9
    # sweep level (north_star's target is on the sweep): the algorithmic bytes of ALL update launches of a step,
    # (n_hb + n_or) * 9 link-sizes * D * V = 45 link-sizes per link, over the step time
    n_launch = 2 * len(DIMS) * (N_HB + N_OR)
    sweep_bytes = n_launch * bytes_launch
    sweep_flops = hits * 2 * len(DIMS) * (N_HB * FLOPS_PER_HIT[prec_name]["hb"] + N_OR * FLOPS_PER_HIT[prec_name]["or"])
    sweep_frac = round(sweep_bytes / (ms_step * 1e-3) / 1e9 / hbm_peak, 4)
    # north_star sets its target on the SWEEP, not on a kernel: it leads the block.  frac / achieved below are the
    # dominant kernel's, as the roofline contract asks
    roof = {"target": {"on": "sweep_frac", "value": 0.70, "sweep_frac": sweep_frac, "met": bool(sweep_frac >= 0.70)},
            "bound": "hbm", "kernel": OR_KERNEL[prec_name], "achieved": round(achieved, 1), "peak": hbm_peak,
            "unit": "GB/s", "frac": round(achieved / hbm_peak, 4), "traffic": NCU_TRAFFIC[prec_name]["or"],
            "traffic_source": NCU_TRAFFIC["source"],
            "bytes_per_launch": bytes_launch, "us_per_launch": round(or_us, 2), "launches_timed": arm["or_n"],
            "hb_us_per_launch": round(hb_us, 2),
            "hb_frac": round(bytes_launch / (hb_us * 1e-6) / 1e9 / hbm_peak, 4) if hb_us > 0 else None,
            # working sweep: update bytes over the whole step (measurement time inside, its bytes not counted)
            "sweep_frac": sweep_frac,
            # update-only sweep (the SURVEY 8(d) headline form)
            "update_sweep_frac": round(sweep_bytes / (upd["median_ms_per_step"] * 1e-3) / 1e9 / hbm_peak, 4),
            "sweep_bytes": sweep_bytes}
    if fma_peak_tflops:
        fl = FLOPS_PER_HIT[prec_name]["or"] * hits
        roof["alu"] = {"achieved_tflops": round(fl / (or_us * 1e-6) / 1e12, 2), "peak_tflops": round(fma_peak_tflops, 2),
                       "frac": round(fl / (or_us * 1e-6) / 1e12 / fma_peak_tflops, 4), "flops_per_link_hit": FLOPS_PER_HIT[prec_name]["or"],
                       "flops_source": FLOPS_SOURCE, "peak_source": "qcd_probe_fma_tflops, same run",
                       "sweep_frac": round(sweep_flops / (ms_step * 1e-3) / 1e12 / fma_peak_tflops, 4)}
        t_hbm, t_alu = bytes_launch / (hbm_peak * 1e9), fl / (fma_peak_tflops * 1e12)
        roof["binding_limit"] = "hbm" if t_hbm >= t_alu else "alu"
        roof["frac_of_binding_limit"] = round(max(t_hbm, t_alu) / (or_us * 1e-6), 4)
    return value, ms_step, roof, work, upd


def run_ours(args):
    import torch
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        dist_mod.init_process_group("nccl", device_id=torch.device("cuda", local))
        dist = dist_mod
    import paper_1310_7087_b200 as q
    q.lib()
    hbm_peak, peak_src, _ = load_peaks()
    fma = {"f32": q.qcd_probe_fma_tflops(q.QCD_FP32), "f64": q.qcd_probe_fma_tflops(q.QCD_FP64)}
    copy_gbs = q.qcd_probe_copy_gbs(1 << 30, 5)
    sampler = ClockSampler(local)
    primary = args.precision
    other = "f64" if primary == "f32" else "f32"
    arms = {}
    for name in (primary, other):
        arms[name] = time_arm(q, torch, name, args.steps, args.warmup, args.therm, replica_seed(rank), dist, sampler, args.bulk_copy, not args.same_order)
    on_model = time_on_model(q, torch, dist, sampler, with_oracle=(world == 1 and rank == 0 and not args.no_cpu_baseline))
    sm_mhz = None
    split = time_split(q, torch, args.steps, args.therm, replica_seed(rank)) if args.split and world == 1 else None
    clocks = sampler.stop()
    # O(N) kernel against its issue limit: bound "alu", peak = 148 SMs x 4 schedulers x 1 warp-instruction per cycle at the
    # median SM clock sampled under load in this run (the maximum clock if nvidia-smi gave none); achieved counts the two
    # update launches of a sweep over the WHOLE step time (measurement kernels and the host read inside)
    sm_mhz = clocks.get("sm_mhz") or clocks.get("sm_max_mhz") or 1965.0
    for name in ("f32", "f64"):
        if name in on_model:
            peak = N_SM * SCHEDULERS_PER_SM * sm_mhz * 1e6 / 1e9
            ach = 2 * ON_WARP_INST[name] / (on_model[name]["ms_per_sweep"] * 1e-3) / 1e9
            on_model[name]["roofline"] = {"bound": "alu", "kernel": "on_update_kernel<%s, 4, 4>" % ("float" if name == "f32" else "double"),
                                          "achieved": round(ach, 1), "peak": round(peak, 1), "unit": "G warp-instructions/s",
                                          "frac": round(ach / peak, 4), "traffic": None,
                                          "warp_inst_per_launch": ON_WARP_INST[name],
                                          "thread_inst_per_try": round(ON_WARP_INST[name] * 32 / (16 ** 4 * 8 * 100), 1),
                                          "peak_derivation": "148 SMs x 4 schedulers x %.0f MHz (median SM clock under load, this run)" % sm_mhz,
                                          "source": ON_WARP_INST["source"]}
    line = None
    if rank == 0:
        frag = {}
        for name in (primary, other):
            value, ms_step, roof, work, upd = summarise(arms[name], name, args.steps, world, hbm_peak, fma[name])
            a = arms[name]
            acc, sep = rep_stats(a["accum"], args.steps), rep_stats(a["separate"], args.steps)

            def e2e_block(key):
                st = rep_stats(a[key]["times"], args.steps)
                return {"value": aggregate_value(world, a["links"], 1, st["median_ms_per_step"]), "unit": UNIT,
                        "h2d_bytes_per_step": a[key]["h2d"], "d2h_bytes_per_step": a[key]["d2h"],
                        "ms_per_step": st["median_ms_per_step"], "reps": st, "exchange_layout": a[key]["exchange"]}
            frag[name] = {"value": value, "ms_per_step": ms_step, "reps": work, "roofline": roof,
                          "update_only_sweep": {"ms_per_step": upd["median_ms_per_step"], "reps": upd,
                                                "value": aggregate_value(world, a["links"], 1, upd["median_ms_per_step"])},
                          "e2e": e2e_block("e2e"),
                          "accumulate_on_device": {"ms_per_step": acc["median_ms_per_step"], "reps": acc,
                                                   "value": aggregate_value(world, a["links"], 1, acc["median_ms_per_step"]),
                                                   "plaquette_mean": a["acc_plaquette_mean"]},
                          "qcd_sweep_then_qcd_measure": {"ms_per_step": sep["median_ms_per_step"], "reps": sep},
                          "gpu_launches": a["launches_per_rep"], "plaquette": a["plaquette"], "polyakov_abs": a["polyakov_abs"],
                          "dtype": name, "storage": "12 reals/link" if name == "f32" else "18 reals/link"}
            if "e2e_rows01" in a:
                frag[name]["e2e_rows01"] = e2e_block("e2e_rows01")
        p = frag[primary]
        p["roofline"]["peak_source"] = peak_src
        p["roofline"]["copy_probe_gbs_same_run"] = round(copy_gbs, 1)
        line = {"metric": METRIC, "value": p["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": p["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": primary, "data": "synthetic",
                "config": {"workload": "BASELINE.json configs[2]: SU(3) D=4 32^4 beta=6.0 hot seed 42, 1 HB + 4 OR + measure per step",
                           "storage": p["storage"], "replicas": world, "thermalisation_sweeps_before_warmup": args.therm,
                           "l2": "inputs larger than L2: %d MB of links vs 126 MB" % (arms[primary]["links"] * LINK_BYTES[primary] // 2 ** 20),
                           "timing": "median of >= %d repetitions of the %d-step timed region, >= %.0f ms of device time per arm"
                                     % (MIN_REPS, args.steps, MIN_DEVICE_MS)},
                "reps": p["reps"], "e2e": p["e2e"], "gpu_launches": p["gpu_launches"], "roofline": p["roofline"], "clocks": clocks,
                "update_only_sweep": p["update_only_sweep"], "accumulate_on_device": p["accumulate_on_device"],
                "qcd_sweep_then_qcd_measure": p["qcd_sweep_then_qcd_measure"],
                "observables": {"plaquette": p["plaquette"], "polyakov_abs": p["polyakov_abs"]},
                "other_precision": frag[other], "on_model": on_model}
        if "e2e_rows01" in p:
            line["e2e_rows01"] = p["e2e_rows01"]
        if split is not None:
            line["split"] = split
        if args.same_order:
            line["config"]["launch_order"] = "QCD_OPT_ALTERNATE_ORDER = 0"
        if args.bulk_copy:
            line["config"]["or_kernel"] = "QCD_OPT_BULK_COPY = 1: su3_update_bulk_kernel (fp32 arm)"
            line["roofline"]["kernel"] = "su3_update_bulk_kernel<float, x12, OR> (and the tiled kernel in the fused last pass)"
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline_sample()
            # vs_baseline stays null: BASELINE.md holds the paper's times for ANOTHER sweep (heatbath only, NHIT = 10) on other
            # hardware.  The ratio to the oracle timed above is reported for what it is (a slow, untuned checker)
            cb = line["cpu_baseline"]["value"]
            line["vs_cpu_baseline"] = {"value": line["value"] / cb, "e2e": line["e2e"]["value"] / cb,
                                       "note": "ratio to the CPU oracle on %d host cores; not a target" % line["cpu_baseline"]["cores"]}
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------- the oracle, timed (reported baseline)
def _oracle_sample(O, oracle, step):
    """bounded sample of one step: the 1 HB + 4 OR composite update applied to the V/2 links of one (parity, mu)"""
    parity, mu = step & 1, (step >> 1) % len(DIMS)
    O.substep(BETA, oracle.KIND_HB, 0, parity, mu)
    for _ in range(N_OR):
        O.substep(BETA, oracle.KIND_OR, 0, parity, mu)
    return O.V // 2


def _set_omp_threads(n):
    """libgomp's own runtime call: the oracle is timed as it stands, only the thread count of its OpenMP loops changes"""
    import ctypes
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(n))


def cpu_baseline_sample():
    import oracle
    cores = oracle.num_threads()
    O = oracle.OracleLattice(DIMS, NC)
    O.init(oracle.HOT, SEED)
    t0 = time.time()
    done = 0
    step = 0
    while step < 64 and time.time() - t0 < 15.0:      # about 15-17 s of oracle work whatever the host is
        done += _oracle_sample(O, oracle, step)
        step += 1
    dt = time.time() - t0
    out = {"value": done / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
           "sample": "%d x (1 HB + 4 OR on the V/2 links of one (parity, mu)) of the 32^4 lattice from the hot start, "
                     "= %.2f sweeps (%.1f s)" % (step, step / 8.0, dt)}
    # the same oracle on ONE thread, bounded: 1/4 of one (parity, mu) sample would be enough, the
    # site loop is not divisible from outside, so one sample it is (~5-8 s)
    try:
        _set_omp_threads(1)
        t0 = time.time()
        n1 = _oracle_sample(O, oracle, step)
        dt1 = time.time() - t0
        out["single_thread"] = {"value": n1 / dt1, "unit": UNIT, "cores": 1,
                                "sample": "1 x (1 HB + 4 OR on the V/2 links of one (parity, mu)) (%.1f s)" % dt1}
    except OSError as e:
        out["single_thread"] = {"unavailable": str(e)}
    finally:
        try:
            _set_omp_threads(cores)
        except OSError:
            pass
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    cores = oracle.num_threads()
    O = oracle.OracleLattice(DIMS, NC)
    O.init(oracle.HOT, SEED)
    # keep the whole run within a few minutes whatever K is: at most ~150 s of oracle work
    for w in range(args.warmup):
        t0 = time.time()
        _oracle_sample(O, oracle, w)
        per = time.time() - t0
    steps = args.steps
    t0 = time.time()
    done = 0
    for s in range(steps):
        done += _oracle_sample(O, oracle, s)
    dt = time.time() - t0
    value = done / dt
    sample = "per step: 1 HB + 4 OR on the V/2 links of one (parity, mu) of the 32^4 lattice (1/8 of a sweep)"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": steps, "warmup": args.warmup, "ms_per_step": dt / steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE.json configs[2]: SU(3) D=4 32^4 beta=6.0 hot seed 42, 1 HB + 4 OR", "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--therm", type=int, default=10, help="untimed setup sweeps after the hot start, before the warm-up steps")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--bulk-copy", action="store_true",
                    help="fp32 arm: overrelaxation by the bulk-copy kernel (QCD_OPT_BULK_COPY; the comparison of DESIGN.md sec 6.10)")
    ap.add_argument("--split", action="store_true",
                    help="also time the lattice divided into 1, 2 and 4 parts on this GPU (qcd_split_sweep; DESIGN.md sec 9)")
    ap.add_argument("--same-order", action="store_true",
                    help="every update launch visits the lattice in the same direction (QCD_OPT_ALTERNATE_ORDER = 0; the comparison "
                         "of DESIGN.md sec 6.5)")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = 16 if args.steps is None else args.steps
        args.warmup = 1 if args.warmup is None else args.warmup
        # bound the run: one sample costs ~1.5-3 s on 8 cores
        args.steps = min(args.steps, 64)
        args.warmup = min(args.warmup, 4)
        run_reference(args)
        return
    args.steps = 100 if args.steps is None else args.steps
    args.warmup = max(3, 5 if args.warmup is None else args.warmup)
    run_ours(args)


if __name__ == "__main__":
    main()
