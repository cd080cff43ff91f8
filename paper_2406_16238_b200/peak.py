"""FP64 peak record of the GPU this runs on, as one JSON object on stdout:

    python -m paper_2406_16238_b200.peak > profiles/fp64_peak_b200.json

The numbers come from afqmc_measure_fp64_peak (csrc/peak.cu): register-only issue loops of
mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) and of FP64 FMA on every SM, no memory traffic - the denominators of
every "tensor" roofline fraction bench.py reports (MEASURED_PEAKS.json has no FP64 entry).  Burst = 200 ms per
loop, sustained = 2 s per loop; SM clock and board power are sampled with nvidia-smi while the loops run."""
from __future__ import annotations

import json
import subprocess
import threading
import time


def _sample(stop, out):
    q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.sw_power_cap,clocks_event_reasons.hw_slowdown"
    while not stop.is_set():
        try:
            r = subprocess.run(["nvidia-smi", "-i", "0", f"--query-gpu={q}", "--format=csv,noheader,nounits"],
                               capture_output=True, text=True, timeout=5)
            f = [x.strip() for x in r.stdout.strip().split(",")]
            out.append((float(f[0]), float(f[1]), float(f[2]), f[3], f[4]))
        except Exception:
            pass
        time.sleep(0.1)


def main():
    import torch
    from . import afqmc
    torch.cuda.set_device(0)
    afqmc.measure_fp64_peak(50.0)                      # warm-up
    rec = {"gpu": torch.cuda.get_device_name(0), "sms": torch.cuda.get_device_properties(0).multi_processor_count,
           "how": "afqmc_measure_fp64_peak (csrc/peak.cu): register-only mma.sync.m8n8k4.f64 / DFMA issue loops on all SMs",
           "when": time.strftime("%Y-%m-%dT%H:%M:%SZ", time.gmtime())}
    for name, ms in (("burst_200ms", 200.0), ("sustained_2s", 2000.0)):
        stop, samples = threading.Event(), []
        t = threading.Thread(target=_sample, args=(stop, samples))
        t.start()
        dmma, dfma, mhz = afqmc.measure_fp64_peak(ms)
        stop.set()
        t.join()
        smi_mhz = sorted(s[0] for s in samples)[len(samples) // 2] if samples else None
        rec[name] = {"dmma_tflops": dmma, "dfma_tflops": dfma,
                     # per SM and clock at the SM clock nvidia-smi reports under this load (128 = one DMMA.8x8x4 per
                     # 4 clocks per SM)
                     "flop_per_clk_per_sm_dmma": dmma * 1e12 / (rec["sms"] * smi_mhz * 1e6) if smi_mhz else None,
                     "nvidia_smi": {"sm_mhz": smi_mhz,
                                    "sm_max_mhz": samples[0][1] if samples else None,
                                    "power_w_max": max((s[2] for s in samples), default=None),
                                    "sw_power_cap_seen": any(s[3] == "Active" for s in samples),
                                    "hw_slowdown_seen": any(s[4] == "Active" for s in samples)}}
    print(json.dumps(rec, indent=1))


if __name__ == "__main__":
    main()
