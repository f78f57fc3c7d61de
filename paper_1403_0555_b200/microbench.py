"""Roofline denominators and cost-model probes of the relaxation kernels, measured on the device in use.

`python -m paper_1403_0555_b200.microbench` prints one table (markdown) of what DESIGN.md section 7.1 quotes: the
FP64 FMA issue rate for different operand patterns, the dependent-issue latency, the FP64 tensor-core rate, and the
cost of the shared-memory instructions of a site update.  Everything runs in libu1gf_measure.so (include/u1gf_measure.h); this module
only converts rates to cycles.  Needs a CUDA device; there is no CPU path.
"""
from __future__ import annotations

import subprocess
import sys


def sm_clock_mhz() -> float:
    """Current SM clock as nvidia-smi reports it right after a kernel ran (the probes hold the boost clock)."""
    try:
        out = subprocess.run(["nvidia-smi", "--query-gpu=clocks.sm,clocks.max.sm", "--format=csv,noheader,nounits", "-i", "0"],
                             capture_output=True, text=True, check=True).stdout.strip().split(",")
        return float(out[1])   # the probes run at the maximum SM clock on an otherwise idle B200 (bench.py samples it)
    except (OSError, subprocess.CalledProcessError, ValueError, IndexError):
        return 1965.0


def main() -> int:
    import torch
    from . import binding as b
    assert torch.cuda.is_available(), "microbench needs a CUDA device"
    props = torch.cuda.get_device_properties(0)
    sms, mhz = props.multi_processor_count, sm_clock_mhz()
    smsp_cycles_per_s = sms * 4 * mhz * 1e6      # scheduler-cycles per second on the whole GPU
    sm_cycles_per_s = sms * mhz * 1e6
    rows = []

    def fp64(pattern, label, per_instr=32.0):
        rate = b.measure_fp64_rate(pattern, 150.0)                 # thread-level FMAs per second
        cyc = smsp_cycles_per_s / (rate / per_instr)               # scheduler cycles per warp-level instruction
        rows.append((label, f"{cyc:.2f} cycles / warp-instr / scheduler", f"{2 * rate / 1e12:.1f} TFLOP/s"))
        return rate

    fp64(0, "DFMA, multiplicand and addend reusable (`x = x*a + b`): the roofline denominator")
    fp64(2, "complex multiply-accumulate of w_i, operands in registers")
    fp64(1, "DFMA, three fresh register operands")
    fp64(3, "reusable-operand DFMA stream + 2 integer instructions per DFMA (FMAs counted)")
    fp64(4, "three-fresh-operand DFMA stream + 2 integer instructions per DFMA (FMAs counted)")
    fp64(6, "DMMA m8n8k4 (FP64 tensor core), per 8-FMA instruction", per_instr=32.0 * 8.0)
    chain = b.measure_fp64_rate(5, 100.0)
    lat = (sms * 4 * 32) / chain * mhz * 1e6                        # one warp per scheduler, one chain per warp
    rows.append(("dependent DFMA -> DFMA issue latency", f"{lat:.1f} cycles", ""))
    for mix, label, n in ((1, "8 warp-uniform LDS.128 (the links of a site)", 8),
                          (0, "4 lane-strided LDS.128 + 1 STS.128 (out-of-block neighbours and the store)", 5),
                          (2, "all 13 shared-memory instructions of a 4^4 site update", 13)):
        rate = b.measure_smem_rate(mix, 100.0)                      # warp-level instructions per second
        rows.append((label, f"{sm_cycles_per_s / rate * n:.1f} cycles / site / SM",
                     f"{sm_cycles_per_s / rate:.2f} cycles / instr / SM"))
    for cs, remote in ((2, True), (8, True), (9, True), (16, True), (16, False)):
        rate, ncl = b.measure_dsmem_rate(cs, remote, 60.0)
        rows.append((f"distributed shared memory, cluster of {cs} CTAs x 512 threads x 200 KB, 128-bit loads from "
                     f"{'the neighbour CTA' if remote else 'the own CTA through the cluster window'}",
                     f"{rate / (mhz * 1e6):.1f} bytes / cycle / SM", f"{ncl} clusters resident ({ncl * cs} SMs)"))
    print(f"device: {props.name}, {sms} SMs, SM clock taken as {mhz:.0f} MHz\n")
    print("| probe | result | |")
    print("|---|---|---|")
    for r in rows:
        print("| " + " | ".join(r) + " |")
    return 0


if __name__ == "__main__":
    sys.exit(main())
