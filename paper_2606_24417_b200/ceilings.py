"""Print the measured ceilings of the current device as one JSON line.

    python -m paper_2606_24417_b200.ceilings [--bytes 536870912] [--iters 24000]

Issue rates of one SM sub-partition by instruction mix (1e9 warp instructions per second, counted in SASS) and random
32-byte-sector access rates over an array of `--bytes` (1e9 accesses per second), through the C ABI
(sbf_ceiling_pipe_rate / sbf_ceiling_random_sector, include/sbf_bench.h, libsbf_bench_b200.so).  bench.py calls the same entry points in its own
run; this front end exists so that the micro-benchmarks can be profiled on their own (profiles/ceilings_ncu_r02.md).
"""
from __future__ import annotations

import argparse
import json
import sys


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--bytes", type=int, default=512 << 20)
    ap.add_argument("--iters", type=int, default=24000)
    ap.add_argument("--skip-pipes", action="store_true")
    args = ap.parse_args()
    import paper_2606_24417_b200 as sbf
    out = {"array_bytes": args.bytes, "pipe_g_warp_inst_per_s_per_smsp": {}, "random_sector_g_per_s": {}}
    if not args.skip_pipes:
        for mode in range(sbf.sbf_ceiling_pipe_modes()):
            out["pipe_g_warp_inst_per_s_per_smsp"][sbf.sbf_ceiling_pipe_mode_name(mode)] = sbf.sbf_ceiling_pipe_rate(mode, args.iters)[0]
    for mode, name in enumerate(["red_or_b64_x4", "red_or_b64_x1", "ld_nc_256", "cp_async_2x16", "tma_reduce_or_32B",
                                 "ld_nc_256_L2_64B", "cp_async_2x16_L2_64B", "st_256"]):
        out["random_sector_g_per_s"][name] = sbf.sbf_ceiling_random_sector(mode, args.bytes)
    print(json.dumps(out))
    return 0


if __name__ == "__main__":
    sys.exit(main())
