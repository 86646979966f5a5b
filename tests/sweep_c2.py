"""configs[1] sweep at full size (N = 2^20): theta in {0.3, 0.5, 0.7, 1.0} x p in {2, 4, 6, 8}, one tree, moments per p,
lists per theta; RMS force error against the fp64 direct sum on the 4096-sink subsample and forces per second.

    python tests/sweep_c2.py            (needs a B200; prints the markdown table quoted in DESIGN.md section 7)

Not a test (the gates are in test_gpu_parity.py); it lives here because it uses the oracle, which only tests/,
smoke() and bench.py's cpu_baseline leg may do.
"""
import math
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import oracle  # noqa: E402
from paper_1407_2600_b200 import dsk, workloads  # noqa: E402


def main():
    cfg = workloads.CONFIGS[2]
    pos, mass = workloads.make(2)
    n = len(pos)
    sink = workloads.subsample(2, n, 4096)
    da, _ = oracle.direct_iso(pos, mass, cfg["eps"], sink)
    d = dsk.Dsk(n, 1.0, False, cfg["eps"], 0.5, 4, p_max=8)
    tp, tm = torch.from_numpy(pos).cuda(), torch.from_numpy(mass).cuda()
    acc = torch.empty((n, 3), dtype=torch.float32, device="cuda")
    stream = torch.cuda.current_stream()
    print("| theta | p | E_rms vs direct | ms per evaluation (tree + force) | particles/s | M2P per sink | P2P per sink |")
    print("|---|---|---|---|---|---|---|")
    for theta in (0.3, 0.5, 0.7, 1.0):
        for p in (2, 4, 6, 8):
            d.set_params(theta=theta, p=p)
            ms = []
            for it in range(3):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                d.build_tree(tp, tm)
                d.accel(tp, tm, acc, None)
                e1.record(stream)
                e1.synchronize()
                ms.append(e0.elapsed_time(e1))
            st = d.get_stats()
            a = acc.cpu().numpy().astype(np.float64)[sink]
            erms = math.sqrt(((a - da) ** 2).sum() / (da ** 2).sum())
            t = float(np.median(ms))
            print(f"| {theta} | {p} | {erms:.2e} | {t:.2f} | {n / t * 1e3:.3g} | {st['n_m2p'] / n:.0f} | {st['n_p2p'] / n:.0f} |")
    d.close()


if __name__ == "__main__":
    main()
