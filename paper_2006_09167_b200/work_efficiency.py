"""Algorithmic work efficiency of the cluster-pair list (Fig. 5):
"the fraction of interactions calculated that are within the actual cut-off, shown as function of
buffer size for three common cut-off distances", for this build's 8x8 cluster shape next to the
particle (1x1) Verlet list.  The figure's own values are an image; only its definition is used.

    python -m paper_2006_09167_b200.work_efficiency [--nside 20] [--rc 0.8 1.0 1.2] [--buffers 0 0.05 0.1 0.15 0.2]

For every (rc, buffer) the water box of config 1's recipe is searched with rlist = rc + buffer through
the C ABI; efficiency = atom pairs with r < rc (any exclusion status, counted by the library over the
list) / (64 x listed cluster pairs).  Two cluster numbers are printed: the searched list (bounding-box
predicate, what the paper's CPU search produces) and the list after a prune at the same rlist (atom
distances, the dual-list inner list).  The 1x1 reference is the ideal-gas ratio (rc / rlist)^3.
The tolerance-based Verlet-buffer estimate of L159-L161 is paper_2006_09167_b200/verlet_buffer.py.
"""
from __future__ import annotations

import argparse
import json


def efficiency_table(nside: int, rcs, buffers, device: int = 0):
    import torch

    from . import nb, workloads

    if not torch.cuda.is_available():
        raise RuntimeError("work_efficiency needs a CUDA device: the list is built by the library, there is no CPU fallback")
    w = workloads.water_box(nside)
    dev = torch.device("cuda", device)
    x = torch.from_numpy(w.x).to(dev)
    q = torch.from_numpy(w.q).to(dev)
    t = torch.from_numpy(w.type).to(dev)
    rows = []
    for rc in rcs:
        for b in buffers:
            rl = rc + b
            if rl > 0.5 * float(w.box.min()):
                continue
            ctx = nb.context_for(w, device=device, rc=rc)
            ctx.put_atoms(x, q, t, w.box)
            ctx.search(rl)
            n_int, n_exc = ctx.count_pairs()
            searched = ctx.list_count(0)
            ctx.prune(rl, 0, 1)
            pruned = ctx.list_count(1)
            n_int2, n_exc2 = ctx.count_pairs()
            assert (n_int2, n_exc2) == (n_int, n_exc), "pruning at rlist >= rc must not lose a pair within rc"
            slots = ctx.count_slots()
            rows.append({"rc": rc, "buffer": b, "pairs_within_rc": n_int + n_exc,
                         "cluster_pairs_searched": searched, "cluster_pairs_pruned": pruned,
                         "slots_streamed": slots,
                         "eff_searched": (n_int + n_exc) / (64.0 * searched), "eff_pruned": (n_int + n_exc) / (64.0 * pruned),
                         "eff_streamed": (n_int + n_exc) / float(slots),
                         "eff_1x1_ideal": (rc / rl) ** 3})
            ctx.close()
    return {"workload": w.name, "natoms": w.natoms, "cluster": "8x8", "rows": rows}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--nside", type=int, default=20)
    ap.add_argument("--rc", type=float, nargs="+", default=[0.8, 1.0, 1.2])
    ap.add_argument("--buffers", type=float, nargs="+", default=[0.0, 0.05, 0.1, 0.15, 0.2])
    a = ap.parse_args()
    tab = efficiency_table(a.nside, a.rc, a.buffers)
    print(json.dumps({k: v for k, v in tab.items() if k != "rows"}))
    print("rc      buffer  eff(8x8 searched)  eff(8x8 pruned)  eff(8x1 streamed)  eff(1x1 ideal)")
    for r in tab["rows"]:
        print(f"{r['rc']:<7g} {r['buffer']:<7g} {r['eff_searched']:<18.4f} {r['eff_pruned']:<16.4f} {r['eff_streamed']:<18.4f} {r['eff_1x1_ideal']:.4f}")


if __name__ == "__main__":
    main()
