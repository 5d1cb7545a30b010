"""Phase timeline of the persistent solver (k_persistent) from globaltimer stamps of thread 0 of every CTA.

Needs the debug build of the library (clock stamps are compiled out of the shipped one):

    python paper_2605_13987_b200/build.py --debug && WTIDE_STAMPS=1 python -m paper_2605_13987_b200.stamps 1
    python paper_2605_13987_b200/build.py --force          # back to the shipped build

Prints, for Euler substep 1 of output step 2 of BASELINE.json config <n>, when the CTAs pass each phase boundary
(ns after the first CTA entered the launch; min / mean / max over the z-line CTAs and over the boundary CTAs) and the
stamps of thread 0 inside the two z-line passes.  A timing tool: the table it solves is not checked.
"""
import ctypes
import os
import sys

import numpy as np


def main():
    os.environ["WTIDE_STAMPS"] = "1"
    import torch

    import paper_2605_13987_b200 as wt
    from wtide_inputs import geometry_desc, reduced_desc
    cfg = int(sys.argv[1]) if len(sys.argv) > 1 else 1
    d = reduced_desc(geometry_desc(cfg), nt=8)
    g = wt.wt_make_geometry(d)
    plan = wt.wt_describe_plan(g)
    print(plan)
    if not hasattr(wt._lib, "wt_debug_stamps_offset"):
        sys.exit("this libwtide.so is not a debug build: python paper_2605_13987_b200/build.py --debug")
    nz_cta = int(plan.split(" z-line")[0].split()[-1])
    need = wt.wt_query(g, wt.WT_Q_SOLVE_WORKSPACE_BYTES)
    ws = torch.zeros(need + 256, dtype=torch.uint8, device="cuda")
    wt.wt_solve_H([g], workspace=ws)
    torch.cuda.synchronize()
    wt._lib.wt_debug_stamps_offset.restype = ctypes.c_int64
    wt._lib.wt_debug_stamps_offset.argtypes = [ctypes.c_void_p]
    off = wt._lib.wt_debug_stamps_offset(g.handle)
    a0 = (ws.data_ptr() + 255) // 256 * 256 - ws.data_ptr()
    raw = ws[a0 + off: a0 + off + 256 * 1024].cpu().numpy().view(np.uint64).reshape(-1, 64)
    n_cta = int((raw[:, 0] > 0).sum())
    st = raw[:n_cta].astype(np.int64)
    st = np.where(st > 0, st - st[:, 0].min(), -1)
    names = ["substep starts", "plane phase done", "grid barrier passed", "z pass A done | B: contributions in", "published | B: rhs formed",
             "charges arrived | B: charges published", "z pass B done"]
    for k in range(7):
        col = st[:, 7 + k]
        z, b = col[:nz_cta], col[nz_cta:]
        print("%-42s Z CTAs: min %7d mean %7.0f max %7d   B CTAs: min %7d mean %7.0f max %7d" % (names[k], z.min(), z.mean(), z.max(), b.min(), b.mean(), b.max()))
    print("next substep starts                        %7d .. %7d" % (st[:, 14].min(), st[:, 14].max()))
    fine = raw[:nz_cta, 32:48].astype(np.int64)
    lab = ["A start", "A loads returned", "A forward stage 1 + barrier", "A forward stage 2 + barrier", "A per-mode update + barrier", "A pad-layer sums + barrier",
           "A pad contributions", None, "B start", "B charge spectrum", "B source added + barrier", "B inverse stage 1 + barrier", "B stored", "B end"]
    for k, name in enumerate(lab):
        if name:
            v = fine[:, k] - fine[:, 0]
            print("  in-pass %-30s min %7d mean %7.0f max %7d" % (name, v.min(), v.mean(), v.max()))


if __name__ == "__main__":
    main()
