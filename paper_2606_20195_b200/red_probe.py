"""L2 atomic-throughput probe: the second term of the roofline.

    python -m paper_2606_20195_b200.red_probe [--iters N]

Times `sketch_red_probe` (result-discarding REDs with the scatter kernels' address pattern, values from
registers, no A loads) with CUDA events for the operand widths the kernels use, on the sketch shapes of
BASELINE.json's configs, and prints one JSON line per case.  Needs a GPU; there is no CPU path.
"""
from __future__ import annotations

import argparse
import json

KINDS = [(0, "f16x2", 2, 2), (1, "v2.f16x2", 4, 2), (2, "v4.f16x2", 8, 2), (3, "f32", 1, 4), (4, "v2.f32", 2, 4), (5, "v4.f32", 4, 4),
         # candidates for sketches beyond tensor memory: plain L2 read-modify-write, TMA bulk reductions
         (6, "plain ld.cg/HADD2/st.cg 16 B", 8, 2), (7, "bulk-reduce f16", 8, 2), (8, "bulk-reduce f32", 4, 4)]
SHAPES = [("c2", 128, 64), ("c3/c5", 256, 128), ("c4", 1024, 256), ("e1", 2048, 1024), ("e1-d4096", 4096, 1024), ("grid d/n=32", 32768, 1024)]


def main() -> int:
    import torch

    from . import binding as ss

    ap = argparse.ArgumentParser()
    ap.add_argument("--iters", type=int, default=2000)
    ap.add_argument("--ctas-per-sm", type=int, default=8)
    args = ap.parse_args()
    if not torch.cuda.is_available():
        raise SystemExit("red_probe needs a CUDA device")
    dev = torch.device("cuda")
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    grid = sms * args.ctas_per_sm
    for name, d, n in SHAPES:
        for kind, kname, vec, eb in KINDS:
            for P in (1, 8, 64):
                if P * d * n * eb > (1 << 30):
                    continue
                buf = torch.zeros(P * d * n * eb, dtype=torch.uint8, device=dev)
                ss.sketch_red_probe(buf, d, n, kind, P, grid, 200)          # warm-up
                torch.cuda.synchronize()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                ops = ss.sketch_red_probe(buf, d, n, kind, P, grid, args.iters)
                e1.record()
                torch.cuda.synchronize()
                sec = e0.elapsed_time(e1) * 1e-3
                print(json.dumps({"shape": name, "d": d, "n": n, "op": kname, "replicas": P, "lane_red_per_s": ops / sec,
                                  "payload_TBps": ops * vec * eb / sec / 1e12, "grid": grid, "iters": args.iters}), flush=True)
    return 0


if __name__ == "__main__":
    raise SystemExit(main())
