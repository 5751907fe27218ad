"""FP64-pipe probe of the device: what independent double-precision chains sustain (roofline denominator check).

    python -m paper_2401_04576_b200.probe

Prints, for each instruction mix of ia_probe_fp64 and for 1..16 resident warps per SM sub-partition, the
sustained FP64 thread-instructions per second and its fraction of SMs x 64 lanes x max SM clock.
DESIGN.md section 6 quotes this table (profiles/r01_pipe_probe.md).
"""
from __future__ import annotations

import json

import torch

from . import binding as b

MODES = {0: "DFMA rn, 8 chains", 1: "DADD.RM/DMUL.RP, 8 chains", 2: "DFMA.RM/RP, 8 chains",
         3: "DFMA.RM/RP, 1 chain", 4: "DFMA.RM/RP, 2 chains", 5: "DFMA.RM/RP, 4 chains",
         6: "DFMA.RM/RP + 1 LOP3 each", 7: "DFMA.RM/RP + 1 FFMA each",
         8: "DFMA.RM/RP, 3 register operands", 9: "DMUL.RM/DADD.RP, 2 register operands",
         10: "DFMA 3 reg, multiplier shared by 4", 11: "DFMA 3 reg, multiplier shared by 2"}


def main():
    assert torch.cuda.is_available(), "needs a CUDA device"
    props = torch.cuda.get_device_properties(0)
    n_sm = props.multi_processor_count
    mhz = 1965                                   # B200 maximum SM clock; read from NVML when it is there
    try:
        import pynvml
        pynvml.nvmlInit()
        mhz = pynvml.nvmlDeviceGetMaxClockInfo(pynvml.nvmlDeviceGetHandleByIndex(0), pynvml.NVML_CLOCK_SM)
    except Exception:
        pass
    peak = n_sm * 64 * mhz * 1e6
    ctx = b.Context(0)
    out = {"n_sm": n_sm, "sm_max_mhz": mhz, "peak_T_inst_per_s": peak / 1e12, "rows": []}
    # blocks of 256 threads = 8 warps = 2 warps per sub-partition; 1..8 blocks per SM
    for mode, name in MODES.items():
        for per_sm in (1, 2, 4, 8):
            rate = max(ctx.ia_probe_fp64(mode, 8192, n_sm * per_sm) for _ in range(3))
            out["rows"].append({"mode": mode, "mix": name, "warps_per_subpartition": 2 * per_sm,
                                "T_inst_per_s": rate / 1e12, "frac_of_peak": rate / peak})
            print(f"{name:28s} {2 * per_sm:3d} warps/SMSP  {rate / 1e12:7.3f} T inst/s  {rate / peak:6.3f}")
    print(json.dumps(out))
    ctx.close()


if __name__ == "__main__":
    main()
