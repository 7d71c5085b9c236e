#!/usr/bin/env python
"""bench.py -- working-sweep throughput of the checkerboard SU(3) Monte Carlo path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--precision f32|f64]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P \
        bench.py --gpus N --steps K --warmup W

Workload (BASELINE.json configs[2], the configuration the metric is quoted on): SU(3), D = 4, 32^4 periodic, beta = 6.0,
hot start seed 42.  One STEP = one pass of the whole hot path = qcd_sweep(beta, 1 heatbath, 4 overrelaxation)
+ qcd_measure(plaquette per plane, Polyakov loop)  (the paper's "working sweep",
PAPER.md:134).  metric = composite link updates/s = D*V*steps / time (reading R13).

The line's `value` is the --precision arm (default fp32, 12-real compressed links); the other arm (fp64, 18 reals) is
measured in the same run and reported under "other_precision".  N > 1: independent replicas, one lattice per GPU, no
data-path collective (replicas only) -> weak scaling.

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
# algorithmic flops per link-hit (FP instructions of the kernels' SASS, FMA = 2)
FLOPS_PER_HIT = {"f32": {"hb": 4270.0, "or": 4030.0}, "f64": {"hb": 3900.0, "or": 3270.0}}


# the dominant kernel of each arm (overrelaxation: 32 of the 40 update launches of a step) and its DRAM traffic per launch,
# dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture of this workload (bytes)
OR_KERNEL = {"f32": "su3_update_tiled_kernel<float, x12, OR>", "f64": "su3_update_kernel<double, x18, OR>"}
NCU_TRAFFIC = {"f32": {"or": 221946880, "hb": 220709888}, "f64": {"or": 658459392, "hb": 656831232},
               "source": "profiles/r1_f_launches_and_ncu.md"}


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
def time_arm(q, torch, prec_name, steps, warmup, therm, seed, dist, sampler, do_e2e=True):
    """device-resident timing + end-to-end timing of one precision arm; returns a dict of raw numbers"""
    prec = q.QCD_FP32 if prec_name == "f32" else q.QCD_FP64
    flags = q.QCD_FLAG_COMPRESS12 if prec_name == "f32" else 0
    V = 1
    for d in DIMS:
        V *= d
    links = len(DIMS) * V
    out = {}
    with q.Lattice(DIMS, NC, prec, flags, device=torch.device("cuda", torch.cuda.current_device())) as G:
        G.qcd_init(q.QCD_HOT, seed)
        for _ in range(therm):                       # setup: move off the hot start (KP acceptance, staple norms)
            G.qcd_sweep(BETA, N_HB, N_OR)
        for _ in range(warmup):
            G.qcd_sweep(BETA, N_HB, N_OR)
            G.qcd_measure()
        G.qcd_set_option(q.QCD_OPT_PROFILE, 1)
        G.qcd_reset_profile()
        n0 = G.qcd_get_launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        t0 = time.time()
        e0.record()
        for _ in range(steps):
            G.qcd_sweep(BETA, N_HB, N_OR)
            plaq, planes, poly = G.qcd_measure()
        e1.record()
        torch.cuda.synchronize()
        sampler.window(t0, time.time())
        if dist is not None:
            dist.barrier()
        ms = e0.elapsed_time(e1)
        out["launches"] = G.qcd_get_launch_count() - n0
        hb_ms, hb_n = G.qcd_get_profile(q.QCD_KIND_HB)
        or_ms, or_n = G.qcd_get_profile(q.QCD_KIND_OR)
        G.qcd_set_option(q.QCD_OPT_PROFILE, 0)
        out.update(ms_total=ms, plaquette=plaq, polyakov_abs=abs(poly), hb_ms=hb_ms, hb_n=hb_n, or_ms=or_ms, or_n=or_n)
        out["sweep_counter"] = G.qcd_get_sweep_counter()
        # the same working sweep with the observables accumulated on the device (qcd_measure_accumulate: no host
        # synchronisation per step, one qcd_accum_get at the end) -- reported beside the headline, not instead of it
        G.qcd_accum_reset()
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            G.qcd_sweep(BETA, N_HB, N_OR)
            G.qcd_measure_accumulate()
        e1.record()
        n_acc, s1, _ = G.qcd_accum_get()
        torch.cuda.synchronize()
        out["acc_ms_total"] = e0.elapsed_time(e1)
        out["acc_plaquette_mean"] = float(s1[:6].mean() / max(n_acc, 1))

        if do_e2e:
            # end to end through the C ABI with HOST buffers: every step uploads the configuration from pinned host
            # memory (canonical layout), runs the working sweep, reads the observables and downloads the configuration
            nbytes = G.canonical_bytes
            host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
            G.qcd_get_links_ptr(host.data_ptr(), nbytes, 0)
            for _ in range(2):
                G.qcd_set_links_ptr(host.data_ptr(), nbytes, 0)
                G.qcd_sweep(BETA, N_HB, N_OR)
                G.qcd_measure()
                G.qcd_get_links_ptr(host.data_ptr(), nbytes, 0)
            if dist is not None:
                dist.barrier()
            torch.cuda.synchronize()
            t0 = time.time()
            e0.record()
            for _ in range(steps):
                G.qcd_set_links_ptr(host.data_ptr(), nbytes, 0)
                G.qcd_sweep(BETA, N_HB, N_OR)
                G.qcd_measure()
                G.qcd_get_links_ptr(host.data_ptr(), nbytes, 0)
            e1.record()
            torch.cuda.synchronize()
            sampler.window(t0, time.time())
            out["e2e_ms_total"] = e0.elapsed_time(e1)
            out["h2d"] = nbytes
            out["d2h"] = nbytes + 9 * 8
    out["links"] = links
    return out


def max_over_ranks(torch, dist, x, device="cuda"):
    """replicas only: the one cross-rank operation of the bench is this MAX of the timed region"""
    if dist is None:
        return x
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def replica_seed(rank):
    """every rank runs an independent lattice of the same workload: same recipe, its own Philox seed"""
    return SEED + rank


def aggregate_value(n_gpus, links_per_replica, steps, ms_total_max):
    """whole-job composite link updates/s: all replicas' links over the slowest rank's time"""
    return n_gpus * links_per_replica * steps / (ms_total_max * 1e-3)


def summarise(arm, prec_name, steps, n_gpus, hbm_peak, fma_peak_tflops):
    """per-arm JSON fragments: value, roofline of the dominant (overrelaxation) kernel, sweep breakdown"""
    links = arm["links"]
    ms_step = arm["ms_total"] / steps
    value = aggregate_value(n_gpus, links, steps, arm["ms_total"])
    hits = links // (2 * len(DIMS))                                  # links updated by one launch = V/2
    bytes_launch = LINK_SIZES_PER_HIT * LINK_BYTES[prec_name] * hits
    or_us = arm["or_ms"] / max(arm["or_n"], 1) * 1e3
    hb_us = arm["hb_ms"] / max(arm["hb_n"], 1) * 1e3
    achieved = bytes_launch / (or_us * 1e-6) / 1e9
    roof = {"bound": "hbm", "kernel": OR_KERNEL[prec_name], "achieved": round(achieved, 1), "peak": hbm_peak,
            "unit": "GB/s", "frac": round(achieved / hbm_peak, 4), "traffic": NCU_TRAFFIC[prec_name]["or"],
            "traffic_source": NCU_TRAFFIC["source"],
            "bytes_per_launch": bytes_launch, "us_per_launch": round(or_us, 2), "launches_timed": arm["or_n"],
            "hb_us_per_launch": round(hb_us, 2),
            "hb_frac": round(bytes_launch / (hb_us * 1e-6) / 1e9 / hbm_peak, 4) if hb_us > 0 else None}
    if fma_peak_tflops:
        fl = FLOPS_PER_HIT[prec_name]["or"] * hits
        roof["alu"] = {"achieved_tflops": round(fl / (or_us * 1e-6) / 1e12, 2), "peak_tflops": round(fma_peak_tflops, 2),
                       "frac": round(fl / (or_us * 1e-6) / 1e12 / fma_peak_tflops, 4), "flops_per_link_hit": FLOPS_PER_HIT[prec_name]["or"],
                       "peak_source": "qcd_probe_fma_tflops, same run"}
        t_hbm, t_alu = bytes_launch / (hbm_peak * 1e9), fl / (fma_peak_tflops * 1e12)
        roof["binding_limit"] = "hbm" if t_hbm >= t_alu else "alu"
        roof["frac_of_binding_limit"] = round(max(t_hbm, t_alu) / (or_us * 1e-6), 4)
    return value, ms_step, roof


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
        arms[name] = time_arm(q, torch, name, args.steps, args.warmup, args.therm, replica_seed(rank), dist, sampler)
        arms[name]["ms_total"] = max_over_ranks(torch, dist, arms[name]["ms_total"])
        arms[name]["e2e_ms_total"] = max_over_ranks(torch, dist, arms[name]["e2e_ms_total"])
    clocks = sampler.stop()
    line = None
    if rank == 0:
        frag = {}
        for name in (primary, other):
            value, ms_step, roof = summarise(arms[name], name, args.steps, world, hbm_peak, fma[name])
            a = arms[name]
            e2e_val = aggregate_value(world, a["links"], args.steps, a["e2e_ms_total"])
            frag[name] = {"value": value, "ms_per_step": ms_step, "roofline": roof,
                          "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": a["h2d"], "d2h_bytes_per_step": a["d2h"],
                                  "ms_per_step": a["e2e_ms_total"] / args.steps},
                          "accumulate_on_device": {"ms_per_step": a["acc_ms_total"] / args.steps,
                                                   "value": aggregate_value(world, a["links"], args.steps, a["acc_ms_total"]),
                                                   "plaquette_mean": a["acc_plaquette_mean"]},
                          "gpu_launches": a["launches"], "plaquette": a["plaquette"], "polyakov_abs": a["polyakov_abs"],
                          "dtype": name, "storage": "12 reals/link" if name == "f32" else "18 reals/link"}
        p = frag[primary]
        p["roofline"]["peak_source"] = peak_src
        p["roofline"]["copy_probe_gbs_same_run"] = round(copy_gbs, 1)
        line = {"metric": METRIC, "value": p["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                "ms_per_step": p["ms_per_step"], "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": primary, "data": "synthetic",
                "config": {"workload": "BASELINE.json configs[2]: SU(3) D=4 32^4 beta=6.0 hot seed 42, 1 HB + 4 OR + measure per step",
                           "storage": p["storage"], "replicas": world, "thermalisation_sweeps_before_warmup": args.therm,
                           "l2": "inputs larger than L2: %d MB of links vs 126 MB" % (arms[primary]["links"] * LINK_BYTES[primary] // 2 ** 20)},
                "e2e": p["e2e"], "gpu_launches": p["gpu_launches"], "roofline": p["roofline"], "clocks": clocks,
                "accumulate_on_device": p["accumulate_on_device"],
                "observables": {"plaquette": p["plaquette"], "polyakov_abs": p["polyakov_abs"]},
                "other_precision": frag[other]}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline_sample()
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
    return {"value": done / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d x (1 HB + 4 OR on the V/2 links of one (parity, mu)) of the 32^4 lattice from the hot start, "
                      "= %.2f sweeps (%.1f s)" % (step, step / 8.0, dt)}


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
