"""Power and clocks of the hot path's pieces, each looped alone for a few seconds on the current GPU (B200):

    python -m paper_2006_07964_b200.power_probe [--workload sweep256] [--seconds 3] > profiles/r2_power.md

Rows: the register-resident DFMA probe (cfd_fp64_peak_probe), torch copies (HBM-resident and L2-resident), every hot
kernel class alone (cfd_profile_only; the results of those runs are garbage by construction, only time, clocks and power
are read), the three sweeps, the whole RHS, and the idle device.  nvidia-smi is sampled every 200 ms during each loop
(bench.ClockSampler).  Measurement aid: nothing here is on the product path.
"""
from __future__ import annotations

import argparse
import os
import sys
import time

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import torch

    import bench
    from paper_2006_07964_b200 import binding as B

    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="sweep256")
    ap.add_argument("--seconds", type=float, default=3.0)
    a = ap.parse_args()
    gpu = "GPU-" + str(torch.cuda.get_device_properties(0).uuid)
    rows = []

    def loop(name, fn, unit_per_call=None, unit=""):
        fn()
        torch.cuda.synchronize()
        s = bench.ClockSampler(gpu)
        s.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0, n = time.time(), 0
        e0.record()
        while time.time() - t0 < a.seconds:
            for _ in range(10):
                fn()
            n += 10
            torch.cuda.synchronize()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / n
        c = s.stop()
        rate = f"{unit_per_call / ms / 1e9:.2f} {unit}" if unit_per_call else ""
        rows.append((name, ms, rate, c.get("sm_mhz"), c.get("power_w_max"), ",".join(c.get("reasons", [])) or "-"))

    probe = []
    loop("DFMA probe (register-resident chains)", lambda: probe.append(B.device_peak_probe(8192)))
    rows[-1] = rows[-1][:2] + (f"{probe[-1]:.1f} TFLOP/s",) + rows[-1][3:]
    x = torch.empty(1 << 28, dtype=torch.float64, device="cuda")
    y = torch.empty_like(x)
    loop("torch copy 2 GiB -> 2 GiB (HBM)", lambda: y.copy_(x), 2 * x.numel() * 8 * 1e3, "GB/s")
    del x, y
    x = torch.empty(1 << 21, dtype=torch.float64, device="cuda")
    y = torch.empty_like(x)
    loop("torch copy 16 MiB -> 16 MiB (L2-resident)", lambda: y.copy_(x), 2 * x.numel() * 8 * 1e3, "GB/s")
    del x, y
    case = bench.make_case(a.workload)
    ctx = B.Context(case.dims, case.faces, case.params, device="cuda:0")
    ctx.load_case(case)
    pts = case.npoints
    for name, mask in (("k_visc_march alone", 1 << 3), ("xi sweep alone", 1 << 0), ("eta sweep alone", 1 << 1),
                       ("zeta sweep alone", 1 << 2), ("three sweeps", 0b0111), ("whole RHS (cfd_rhs)", 0b1111)):
        ctx.profile_only(mask)
        loop(f"{name} ({a.workload})", ctx.rhs, pts * 1e3, "Gpts/s")
    ctx.profile_only()
    ctx.close()
    time.sleep(2.0)
    s = bench.ClockSampler(gpu)
    s.start()
    time.sleep(2.0)
    c = s.stop()
    rows.append(("idle (after the loops)", 0.0, "", c.get("sm_mhz"), c.get("power_w_max"), "-"))
    print("# Power and clocks of the pieces of the hot path, each looped alone\n")
    print(f"Command: `python -m paper_2006_07964_b200.power_probe --workload {a.workload} --seconds {a.seconds:g}`"
          f" on {torch.cuda.get_device_name(0)}; nvidia-smi sampled every 200 ms during each loop (median SM clock, maximum power).\n")
    print("| loop | ms per call | rate | SM MHz (median) | power W (max) | throttle reasons |")
    print("|---|---|---|---|---|---|")
    for r in rows:
        print(f"| {r[0]} | {r[1]:.4f} | {r[2]} | {r[3]} | {r[4]} | {r[5]} |")


if __name__ == "__main__":
    main()
