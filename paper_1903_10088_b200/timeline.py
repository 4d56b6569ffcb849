"""Phase timeline of K1/K2 in the timed launch configuration (diagnostics, not part of the method).

    python -m paper_1903_10088_b200.timeline [--workload 3] [--slices 1] [--iters 60] [--no-overlap]

Builds the timeline variant of the library (the same sources with -DOSIV_TRACE: every block stamps its SM's cycle
counter at its phase boundaries, see include/osiv.h `osiv_debug_timeline`), runs one reconstruction of the workload and
prints, for the last two iterations, where the time of an iteration goes: block start -> dependent-launch wait ->
main loop -> block barrier -> epilogue -> exit for both kernels, and the gaps between a kernel's last exit and its
successor's release.  The stamps cost a few instructions per phase; the numbers are a breakdown, not a benchmark.
"""
from __future__ import annotations

import argparse
import ctypes as C
import os
import sys

import numpy as np

os.environ["OSIV_TRACE_BUILD"] = "1"          # before the binding loads the library

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TL_BLOCKS, TL_SLOTS = 256, 16
SLOTS = ("start", "before wait", "after wait", "loop end", "after barrier", "end")


def fetch():
    from . import binding
    buf = np.zeros((4, TL_BLOCKS, TL_SLOTS), dtype=np.uint64)
    st = binding.lib().osiv_debug_timeline(buf.ctypes.data_as(C.c_void_p), buf.size)
    if st != 0:
        raise RuntimeError("osiv_debug_timeline failed: not the timeline build?")
    return buf


def to_ns(t, sm_mhz):
    """slots 0-5 and 7 are SM cycle counts; slot 8 is the global nanosecond timer at slot 0: every stamp in global ns"""
    out = t.astype(np.float64).copy()
    for j in (0, 1, 2, 3, 4, 5, 7, 9, 10, 11, 12, 13, 14, 15):
        out[:, j] = t[:, 8] + (t[:, j] - t[:, 0]) * (1e3 / sm_mhz)
    return out


def summarise(buf, n_last, sm_mhz):
    """rows of (name, blocks, times) in microseconds relative to the earlier iteration's K1 release"""
    order = [((n_last - 1) & 1, 0), ((n_last - 1) & 1, 1), (n_last & 1, 0), (n_last & 1, 1)]
    names = [f"K1({n_last - 1})", f"K2({n_last - 1})", f"K1({n_last})", f"K2({n_last})"]
    tabs = []
    for par, k in order:
        t = buf[par * 2 + k].astype(np.int64)
        used = t[:, 0] > 0
        tabs.append(to_ns(t[used], sm_mhz))
    t0 = float(np.min(tabs[0][:, 2]))                    # first block of the first kernel released
    out = []
    for name, t in zip(names, tabs):
        rel = (t[:, :16] - t0) * 1e-3
        out.append((name, t.shape[0], rel))
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--workload", default="3")
    ap.add_argument("--slices", type=int, default=1)
    ap.add_argument("--iters", type=int, default=60)
    ap.add_argument("--no-overlap", action="store_true")
    ap.add_argument("--sm-mhz", type=float, default=1965.0, help="SM clock the cycle stamps are converted with (B200 boost clock)")
    args = ap.parse_args()
    import torch
    import synth_inputs as si
    import paper_1903_10088_b200 as osiv
    cfg = si.scan_config(args.workload)
    geom = osiv.Geometry(cfg.nx, cfg.ny, cfg.pixel_mm, cfg.n_views, cfg.n_channels, cfg.sad_mm, cfg.sdd_mm)
    counts = torch.from_numpy(np.stack([si.make_case(cfg, slice_index=s)[2] for s in range(args.slices)])).cuda()
    prm = osiv.Params(beta=cfg.betas[0], n_subsets=cfg.n_subsets, n_iters=args.iters)
    with osiv.Handle(geom, max_batch=args.slices) as h:
        if args.no_overlap:
            h.set_overlap(False)
        for _ in range(3):
            h.reconstruct(counts, cfg.i0, prm)
        torch.cuda.synchronize()
        buf = fetch()
        plan = h.plan(cfg.n_subsets, args.slices)
    rows = summarise(buf, args.iters - 1, args.sm_mhz)
    print(f"# phase timeline, workload {args.workload}, {args.slices} slice(s), iterations {args.iters - 2} and {args.iters - 1}"
          f" (us after the first release of {rows[0][0]}; median [min .. max] over the blocks of slice group 0)")
    print(f"plan: {plan}")
    print("| kernel | blocks | " + " | ".join(SLOTS) + " |")
    print("|---|---|" + "---|" * len(SLOTS))
    for name, nb, rel in rows:
        cells = [f"{np.median(rel[:, j]):.2f} [{rel[:, j].min():.2f} .. {rel[:, j].max():.2f}]" for j in range(6)]
        print(f"| {name} | {nb} | " + " | ".join(cells) + " |")
    print()
    print("| kernel | prologue (start->before wait) | wait | main loop (after wait->loop end) | barrier wait | epilogue (after barrier->end) | first release -> last end |")
    print("|---|---|---|---|---|---|---|")
    for name, nb, rel in rows:
        d = lambda a, b: np.median(rel[:, b] - rel[:, a])
        mx = lambda a, b: np.max(rel[:, b] - rel[:, a])
        print(f"| {name} | {d(0, 1):.2f} | {d(1, 2):.2f} | {d(2, 3):.2f} (max {mx(2, 3):.2f}) | {d(3, 4):.2f} | {d(4, 5):.2f} (max {mx(4, 5):.2f}) | "
              f"{rel[:, 5].max() - rel[:, 2].min():.2f} |")
    print()
    print("work balance over blocks, main loop (after wait -> loop end): mean / median / max / min us; mean = what a perfectly balanced grid would take")
    for name, nb, rel in rows:
        d = rel[:, 3] - rel[:, 2]
        print(f"  {name}: {d.mean():.2f} / {np.median(d):.2f} / {d.max():.2f} / {d.min():.2f}")
    print()
    print("prologue mark (slot 7: K1 own ray loaded and clipped; K2 tile origin known), us after block start, median [max]:")
    for name, nb, rel in rows:
        d = rel[:, 7] - rel[:, 0]
        print(f"  {name}: {np.median(d):.2f} [{d.max():.2f}]")
    print("staged K2 only, us after the dependent-launch wait returned, median [max] over blocks (latest warp of a block): "
          "TV gradients done / warp 0 has issued its loads / residual windows stored / block barrier passed / blob landed / first trip walked / loop end")
    for name, nb, rel in rows:
        if name.startswith("K2") and rel[:, 11].max() > rel[:, 0].min():
            d = [rel[:, j] - rel[:, 2] for j in (9, 10, 12, 11, 13, 14, 3)]
            print(f"  {name}: " + " / ".join(f"{np.median(x):.2f} [{x.max():.2f}]" for x in d))
    ends = [rel[:, 5].max() for _, _, rel in rows]
    rels = [rel[:, 2].min() for _, _, rel in rows]
    print()
    for i in range(1, 4):
        print(f"{rows[i - 1][0]} last end -> {rows[i][0]} first release: {rels[i] - ends[i - 1]:.2f} us; "
              f"{rows[i][0]} release spread over blocks: {rows[i][2][:, 2].max() - rows[i][2][:, 2].min():.2f} us")
    print(f"one iteration (K1 release -> next K1 release): {rels[2] - rels[0]:.2f} us")


if __name__ == "__main__":
    main()
