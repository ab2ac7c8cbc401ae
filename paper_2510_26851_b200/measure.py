"""python -m paper_2510_26851_b200.measure — the measured ceilings DESIGN.md and bench.py quote, on this device:
the non-FMA FP32 issue rate and the rate of scattered 16-byte stores / loads (fof.h "Measured ceilings")."""
from __future__ import annotations

import json
import sys


def main():
    import torch

    from . import binding as B

    assert torch.cuda.is_available(), "needs a CUDA device"
    out = {"device": torch.cuda.get_device_name(0), "fp32_nonfma_lane_ops_per_s": B.fof_measure_fp32_issue()}
    n = 1 << 24
    src = torch.empty(n * 4, dtype=torch.float32, device="cuda").normal_()
    dst = torch.empty_like(src)
    rows = []
    for k in (0, 5, 8, 12, 16, 20, 24):
        st = B.fof_measure_scatter(src, dst, k, True)
        ld = B.fof_measure_scatter(src, dst, k, False)
        rows.append({"log2_window_records": k, "scattered_stores_rec_per_s": st, "scattered_loads_rec_per_s": ld,
                     "stores_ms_per_2^24": 1e3 * n / st, "loads_ms_per_2^24": 1e3 * n / ld})
    out["copy_of_2^24_16B_records"] = rows
    json.dump(out, sys.stdout, indent=1)
    print()


if __name__ == "__main__":
    main()
