"""Per-kernel and per-sweep timing of one library build at the benchmark workload (SU(3) 32^4, beta 6.0, 1 HB + 4 OR).

    python -m paper_1310_7087_b200.timing [--lib PATH] [f32] [f64]

Prints one JSON line: mean device time per overrelaxation / heatbath launch (CUDA events around each run of same-kind
launches, QCD_OPT_PROFILE) and per sweep (CUDA events around 30 / 12 sweeps without profiling), after 11 setup sweeps.
Used to compare tuning builds (`python -m paper_1310_7087_b200.build -D NAME=VALUE --out other.so --objdir DIR`); the
numbers in profiles/*tiling experiments* and DESIGN.md sec 6.7 come from it.  `bench.py` is the benchmark; this is a probe.
"""
import json
import os
import sys


def main(argv):
    lib = None
    if "--lib" in argv:
        i = argv.index("--lib")
        lib = argv[i + 1]
        argv = argv[:i] + argv[i + 2:]
        os.environ["QCD_B200_LIB"] = os.path.abspath(lib)
    import torch
    from . import binding as q
    precs = [a for a in argv if a in ("f32", "f64")] or ["f32", "f64"]
    out = {"lib": os.path.basename(lib) if lib else "libqcd_b200.so"}
    for pr in precs:
        prec, flags = (q.QCD_FP32, q.QCD_FLAG_COMPRESS12) if pr == "f32" else (q.QCD_FP64, 0)
        with q.Lattice((32, 32, 32, 32), 3, prec, flags) as G:
            G.qcd_init(q.QCD_HOT, 42)
            for _ in range(8):
                G.qcd_sweep(6.0, 1, 4)
            G.qcd_set_option(q.QCD_OPT_PROFILE, 1)
            for _ in range(3):
                G.qcd_sweep(6.0, 1, 4)
            G.qcd_reset_profile()
            n = 30 if pr == "f32" else 12
            for _ in range(n):
                G.qcd_sweep(6.0, 1, 4)
            hb_ms, hb_n = G.qcd_get_profile(q.QCD_KIND_HB)
            or_ms, or_n = G.qcd_get_profile(q.QCD_KIND_OR)
            G.qcd_set_option(q.QCD_OPT_PROFILE, 0)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(n):
                G.qcd_sweep(6.0, 1, 4)
            e1.record()
            torch.cuda.synchronize()
            out[pr] = {"or_us": round(1e3 * or_ms / or_n, 2), "hb_us": round(1e3 * hb_ms / hb_n, 2),
                       "sweep_ms": round(e0.elapsed_time(e1) / n, 4), "plaquette": round(G.qcd_measure()[0], 6)}
    print(json.dumps(out))


if __name__ == "__main__":
    main(sys.argv[1:])
