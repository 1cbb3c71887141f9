"""Measure the roofline denominators of this device with krr_peak_probe (SURVEY 8(d) "Which roofline").

    python -m paper_2409_01712_b200.peaks [--seconds 2.5] [--out FILE.json]

For every kind (kind::f16, kind::f8f6f4, kind::mxf8f6f4.block_scale on CTA pairs with operands resident in shared
memory; the three-instruction FP32-class sequence; FFMA) it reports
  burst      the best of the first short launches (a kernel timed alone, the GPU cool), and
  sustained  total flops / total device time of back-to-back launches for `--seconds` (a kernel inside a long
             power-capped step),
with the SM clock and throttle reasons nvidia-smi reported meanwhile.  bench.py --peaks calls `measure()`.
"""
import argparse
import json
import statistics
import subprocess
import time

import torch

from . import binding as krr

WORK = {"f16": 4096, "f16x3": 2048, "f8": 4096, "mxf8": 4096, "ffma": 20000}      # ~1-3 ms per launch


class _Clocks:
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.sw_power_cap,clocks_event_reasons.hw_slowdown,clocks_event_reasons.sw_thermal_slowdown"

    def __init__(self, index):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                                       "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"samples": 0}
        self.p.terminate()
        try:
            out, _ = self.p.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
            out, _ = self.p.communicate()
        sm, pw, reasons = [], [], set()
        for line in out.strip().splitlines():
            f = [x.strip() for x in line.split(",")]
            try:
                sm.append(float(f[0])); pw.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for nm, v in zip(("sw_power_cap", "hw_slowdown", "sw_thermal_slowdown"), f[3:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"samples": 0}
        return {"samples": len(sm), "sm_mhz_median": statistics.median(sm), "sm_mhz_min": min(sm), "power_w_max": max(pw),
                "reasons": sorted(reasons)}


def measure_kind(kind, seconds, device_index=0):
    work = WORK[kind]
    for _ in range(3):
        krr.peak_probe(kind, work)
    time.sleep(0.5)                                   # let the part cool: the burst figure is a cold start
    burst = 0.0
    for _ in range(5):
        ms, fl = krr.peak_probe(kind, work)
        burst = max(burst, fl / (ms * 1e-3) / 1e12)
    clk = _Clocks(device_index)
    t0 = time.perf_counter()
    tot_ms, tot_fl, n = 0.0, 0.0, 0
    while time.perf_counter() - t0 < seconds:
        ms, fl = krr.peak_probe(kind, 4 * work)
        tot_ms += ms; tot_fl += fl; n += 1
    clocks = clk.stop()
    return {"burst_tflops": round(burst, 1), "sustained_tflops": round(tot_fl / (tot_ms * 1e-3) / 1e12, 1),
            "launches": n, "device_seconds": round(tot_ms * 1e-3, 3), "clocks": clocks}


def measure(seconds=2.5, kinds=("f16", "f16x3", "f8", "mxf8", "ffma"), device_index=0):
    torch.cuda.set_device(device_index)
    out = {"device": torch.cuda.get_device_name(device_index),
           "how": "krr_peak_probe: tcgen05 cta_group::2 M=N=256 MMAs on smem-resident pseudo-random operands, no global "
                  "traffic (f16x3 = the hi*hi + lo*hi + hi*lo sequence; its figure counts all three instructions); "
                  "FFMA: 8 chains per thread"}
    for k in kinds:
        out[k] = measure_kind(k, seconds, device_index)
    return out


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--seconds", type=float, default=2.5)
    ap.add_argument("--out", default=None)
    a = ap.parse_args()
    res = measure(a.seconds)
    txt = json.dumps(res, indent=1)
    print(txt)
    if a.out:
        with open(a.out, "w") as f:
            f.write(txt + "\n")
