"""Throughput of cuhpx_reorder (NESTED <-> RING, paper section III-B) on one GPU, one JSON line per case.

    python -m paper_2510_01785_b200.reorder_bench

Device-timed with CUDA events (3 warm-ups, 20 calls); the roofline is HBM: algorithmic bytes = 2 x batch x npix x
element size (every element read once and written once); peak from MEASURED_PEAKS.json when present.
"""
from __future__ import annotations

import json
import os

import torch

from . import binding as B

CASES = [(1024, 8, torch.float32), (4096, 1, torch.float64), (4096, 4, torch.float32), (2048, 8, torch.float64)]


def main() -> None:
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    peak = 6650.0
    try:
        peak = json.load(open(os.path.join(root, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        pass
    for nside, batch, dt in CASES:
        npix = 12 * nside * nside
        a = torch.randn(batch, npix, dtype=dt, device="cuda")
        o = torch.empty_like(a)
        code = B._dtype_code(dt)
        for d, name in [(B.CUHPX_NEST2RING, "nest2ring"), (B.CUHPX_RING2NEST, "ring2nest")]:
            for _ in range(3):
                B.cuhpx_reorder(nside, batch, code, d, a, o)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(20):
                B.cuhpx_reorder(nside, batch, code, d, a, o)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1) / 20
            gbs = 2 * a.numel() * a.element_size() / ms / 1e6
            print(json.dumps({"op": name, "nside": nside, "batch": batch, "dtype": str(dt).split(".")[-1], "ms": ms,
                              "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak}}),
                  flush=True)


if __name__ == "__main__":
    main()
