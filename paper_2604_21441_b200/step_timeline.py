"""Timeline of the kernels of ONE evaluation as they really run (the PDL chain; ncu and the stage events serialise them):

    NNP_EXTRA_NVCC_FLAGS=-DNNP_STEP_TIMELINE python -m paper_2604_21441_b200.build   # instrumented library (profiling only)
    python -m paper_2604_21441_b200.step_timeline [--config 2] [--steps 20] > profiles/rNN_step_timeline.md
    python -m paper_2604_21441_b200.build                                            # (touch a source first) product build again

Thread 0 of every block stamps %globaltimer into its kernel's slot (csrc/nnp_internal.h TL_SCOPE / TL_WAITED / TL_MARK);
this script runs evaluations with the L2 flushed in between, reads the slots after each, and prints the medians relative
to the first block of the first kernel.  Needs a GPU and a library built with the flag; the numbers carry the stamping
overhead (two to four atomics per block) and are for the picture, not for the bench line."""
import argparse
import ctypes as C
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

UNITS = [("nnp_debug_step_timeline_neighbor", ["k_bin_cells", "k_cell_sort", "k_neighbors"]),
         ("nnp_debug_step_timeline_aev", ["k_aev_forward"]),
         ("nnp_debug_step_timeline_mlp", ["k_tc_pack_w1", "k_mlp_tc"]),
         ("nnp_debug_step_timeline_force", ["k_aev_backward", "k_force_out"])]


def main():
    import torch
    import gen
    import paper_2604_21441_b200 as nnp
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--steps", type=int, default=20)
    args = ap.parse_args()
    L = nnp.lib()
    if not hasattr(L, UNITS[0][0]):
        sys.exit("library built without -DNNP_STEP_TIMELINE")
    cfg = gen.get_config(args.config)
    n = cfg["pos"].shape[0]
    P = gen.perturbed_positions(cfg["pos64"], cfg["perturb_seed"], 4)
    ws = nnp.Workspace(nnp.Model(cfg["aev"], cfg["nets"], cfg["celu_alpha"]), n, n)
    ws.set_small_path(0)
    dpos = [torch.from_numpy(P[t]).cuda() for t in range(4)]
    dZ = torch.from_numpy(cfg["Z"]).cuda()
    E = torch.zeros(1, dtype=torch.float64, device="cuda")
    F = torch.zeros((n, 3), dtype=torch.float32, device="cuda")
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    h = (C.c_ulonglong * 24)()
    rows = []
    for it in range(args.steps + 5):
        for name, _ in UNITS:
            getattr(L, name)(h)      # re-arm
        flush.zero_()
        torch.cuda.synchronize()
        ws.eval(dpos[it % 4], dZ, cfg["box"], 1, None, E, F)
        torch.cuda.synchronize()
        rec = []
        for name, kernels in UNITS:
            getattr(L, name)(h)
            a = np.array(list(h), dtype=np.uint64).reshape(4, 6)
            for k in range(len(kernels)):
                rec.append(a[k].astype(np.float64))
        if it >= 5:
            rec = np.array(rec)
            rows.append((rec - rec[0, 0]) / 1e3)     # us after the first block of the first kernel
    assert ws.status() == 0
    med = np.median(np.array(rows), axis=0)
    names = [k for _, ks in UNITS for k in ks]
    print(f"# Step timeline, cfg {args.config} ({n} atoms), median of {args.steps} evaluations, L2 flushed in between\n")
    print("Command: `NNP_EXTRA_NVCC_FLAGS=-DNNP_STEP_TIMELINE python -m paper_2604_21441_b200.build && "
          f"python -m paper_2604_21441_b200.step_timeline --config {args.config} --steps {args.steps}`\n")
    print("us after the first block of the first kernel (thread 0 of each block, %globaltimer):\n")
    print("| kernel | first block in | last block in | first block past its wait | last block out | mark first | mark last |")
    print("|---|---|---|---|---|---|---|")
    for nm, r in zip(names, med):
        f = lambda v: "" if (v > 1e9 or v < -1e9) else f"{v:.1f}"
        print(f"| {nm} | {f(r[0])} | {f(r[3])} | {f(r[1])} | {f(r[2])} | {f(r[4])} | {f(r[5])} |")
    print("\n(k_aev_backward: \"past its wait\" = the block's MLP tile flags are up; k_mlp_tc marks = end of a CTA's first tile.)")


if __name__ == "__main__":
    main()
