"""Measurement aid: print the in-context clock trace of the tcgen05 GEMM kernels (ROSA_DBG=64).

    ROSA_DBG=64 python -m paper_2607_01088_b200.clock_trace [config]

Runs three `rosa_denoise_batch_ex` calls of a seeded case (default BASELINE.json configs[2]: B=64 ragged) and
reads back `rosa_debug_gemm_trace`: for every GEMM class the clock64 values CTA 0 and CTA 64 of the LAST launch
of that class wrote at fixed points of the kernel (cycles relative to the CTA's first instruction).  No
arithmetic of the method happens here; the numbers go into profiles/ by hand.
"""
from __future__ import annotations

import os
import sys

from . import binding as rosa
from . import cases, runner

SLOTS = {1: "setup", 2: "pdl_wait", 10: "tma0", 3: "mma0", 13: "mma_kb8", 9: "tile0_last_kb", 11: "epi0_beg",
         12: "epi0_end", 4: "last_tile_last_kb", 5: "epiL_beg", 6: "epiL_end", 7: "cta_sync", 8: "cluster_sync"}
CLASSES = {2 * 2: "embed (BIAS_F32)", 3 * 2: "QKV (ROPE)", 4 * 2: "O (RESID, K<=2048)", 4 * 2 + 1: "down (RESID, K>2048)",
           5 * 2: "gate/up (GEGLU)", 6 * 2: "final (FINAL)"}


def main(argv):
    if not (int(os.environ.get("ROSA_DBG", "0")) & 64):
        raise SystemExit("set ROSA_DBG=64 (the trace stores are compiled in but switched off otherwise)")
    case = cases.make_case(int(argv[1]) if len(argv) > 1 else 2)
    lc = runner.LoadedCase(case)
    for _ in range(3):
        lc.run()
    tr = rosa.rosa_debug_gemm_trace()
    lc.close()
    for c, name in CLASSES.items():
        for cta in (0, 1):
            t = tr[c, cta]
            if t[0] == 0:
                continue
            print(f"{name:24s} CTA {cta * 64:3d}: " +
                  "  ".join(f"{n} {int(t[s] - t[0])}" for s, n in SLOTS.items() if t[s]))
    ch = tr.reshape(-1)[15 * 32:15 * 32 + 20]
    if ch[0]:  # builds with the chunk-level stamps in the residual epilogue (profiles/r1_gemm_epilogue_trace.md)
        print("residual epilogue, CTA 64 warp 2, per 32-column chunk [top, acc loaded, transposed, h added, stored]:",
              [int(x - ch[0]) for x in ch if x])


if __name__ == "__main__":
    main(sys.argv)
