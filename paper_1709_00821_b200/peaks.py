"""Measured issue and shared-memory peaks of this GPU ("builder must microbenchmark DFMA and
shared-memory peaks and use the measured values") — the denominators of bench.py's "alu" roofline.

    python -m paper_1709_00821_b200.peaks [--iters N] [--json]

Calls rketd_measure_peak (include/rketd.h; kernels in csrc/rketd_peaks.cu) for every form and prints, per form, the
thread-instructions (bytes) per clock and SM, the SM clock the run held, and the board power sampled while it ran.
Marshalling and printing only; `alu_peaks()` is what bench.py imports.
"""
from __future__ import annotations

import json
import sys
import threading
import time

FP_INSTR_PER_CELL_STEP = 7        # kernel form (csrc/rketd_device.cuh): H 2, E 3, G 2


class _Power:
    """board power [W] and SM clock [MHz] sampled through NVML every 20 ms while a microbenchmark runs"""

    def __init__(self, index=0):
        self.w, self.mhz = [], []
        self._stop = threading.Event()
        self._h = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self._p = pynvml
            self._h = pynvml.nvmlDeviceGetHandleByIndex(index)
        except Exception:
            self._h = None

    def __enter__(self):
        def poll():
            while not self._stop.is_set():
                try:
                    self.w.append(self._p.nvmlDeviceGetPowerUsage(self._h) / 1000.0)
                    self.mhz.append(self._p.nvmlDeviceGetClockInfo(self._h, self._p.NVML_CLOCK_SM))
                except Exception:
                    pass
                self._stop.wait(0.02)
        if self._h is not None:
            self._t = threading.Thread(target=poll, daemon=True)
            self._t.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._h is not None:
            self._t.join(timeout=5)


def measure(what: int, iters: int = 4000, seconds: float = 0.0, stream: int = 0):
    """one form; with seconds > 0 the run is repeated for that long (so that NVML sees the load) and the last result kept"""
    from . import rketd
    with _Power() as pw:
        r = rketd.rketd_measure_peak(what, iters, stream)
        t0 = time.perf_counter()
        while time.perf_counter() - t0 < seconds:
            r = rketd.rketd_measure_peak(what, iters, stream)
    r["power_w_max"] = round(max(pw.w), 1) if pw.w else None
    r["nvml_sm_mhz_min"] = min(pw.mhz) if pw.mhz else None
    return r


def max_sm_mhz(index: int = 0) -> float:
    try:
        import pynvml
        pynvml.nvmlInit()
        return float(pynvml.nvmlDeviceGetMaxClockInfo(pynvml.nvmlDeviceGetHandleByIndex(index), pynvml.NVML_CLOCK_SM))
    except Exception:
        return 1965.0            # B200 (MEASURED_PEAKS.json sm_max_mhz)


def alu_peaks(dtype: str, stream: int = 0, iters: int = 4000, index: int = 0):
    """What bench.py divides by.  The microbenchmarks give lanes per clock and SM (clock-invariant: the run's own cycle
    counter) for the best FMA form of `dtype` and for the stencil's own 7-instruction mix; the ceilings in Gcell/s are
    lanes x SMs x the device's MAXIMUM SM clock / 7 — the clock the microbenchmark happened to hold (it may run right
    after a power-capped stretch) is reported beside them, not folded in."""
    from . import rketd
    base = 0 if dtype == "f64" else 4
    forms = {n: rketd.rketd_measure_peak(base + i, iters, stream) for i, n in enumerate(("1reg", "2reg", "3reg", "2reg_const"))}
    mix = rketd.rketd_measure_peak(8 if dtype == "f64" else 9, iters, stream)
    best = max(forms.values(), key=lambda r: r["per_clk_sm"])
    mhz = max_sm_mhz(index)
    to_gcells = lambda lanes: lanes * best["sms"] * mhz * 1e6 / FP_INSTR_PER_CELL_STEP / 1e9
    return {"fma_lanes_per_clk_sm": {k: round(v["per_clk_sm"], 2) for k, v in forms.items()},
            "fma_best_form": best["name"], "fma_best_lanes": round(best["per_clk_sm"], 2), "fma_sm_mhz_held": round(best["sm_mhz"], 1),
            "sms": best["sms"], "sm_max_mhz": mhz,
            "fma_peak_gcells": to_gcells(best["per_clk_sm"]),
            "mix_lanes_per_clk_sm": round(mix["per_clk_sm"], 2), "mix_sm_mhz_held": round(mix["sm_mhz"], 1),
            "mix_peak_gcells": to_gcells(mix["per_clk_sm"])}


def main(argv):
    from . import rketd
    iters = int(argv[argv.index("--iters") + 1]) if "--iters" in argv else 4000
    rows = [measure(i, iters, seconds=0.5) for i in range(len(rketd.PEAK_NAMES))]
    if "--json" in argv:
        print(json.dumps(rows))
        return
    print(f"{'form':18s} {'per clk and SM':>15s} {'device per ns':>15s} {'SM MHz held':>12s} {'NVML MHz min':>13s} {'power W max':>12s}")
    for r in rows:
        if r["name"].startswith("lat_"):
            print(f"{r['name']:28s} {r['per_clk_sm']:10.1f} cycles per operation ({r['per_ns']:.2f} ns at {r['sm_mhz']:.0f} MHz)")
            continue
        unit = "B" if r["name"] == "lds128" else "thread-instr"
        print(f"{r['name']:18s} {r['per_clk_sm']:15.2f} {r['per_ns']:15.1f} {r['sm_mhz']:12.1f} "
              f"{str(r['nvml_sm_mhz_min']):>13s} {str(r['power_w_max']):>12s}   ({unit}; {r['sms']} SMs)")
    for dt in ("f64", "f32"):
        p = alu_peaks(dt, iters=iters)
        print(f"{dt}: FMA peak {p['fma_peak_gcells']:.0f} Gcell/s ({p['fma_best_form']}: {p['fma_best_lanes']} lanes/clk/SM x {p['sms']} SMs x "
              f"{p['sm_max_mhz']:.0f} MHz / 7), stencil-mix issue ceiling {p['mix_peak_gcells']:.0f} Gcell/s ({p['mix_lanes_per_clk_sm']} lanes/clk/SM)")


if __name__ == "__main__":
    main(sys.argv[1:])
