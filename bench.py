#!/usr/bin/env python
"""bench.py -- the cluster-pair short-range non-bonded step on B200 (BASELINE.json metric:
"non-bonded pair interactions/s and force-step us at 1 B200; % FP32 peak").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--coulomb ewald|rf]
  python bench.py --impl reference ...      # the fp64 CPU oracle, as it stands, on the host cores

One "step" is one MD step of the whole hot path on the synthetic water box, in the paper's
schedule: every step stages new coordinates
(nb_put_atoms) and computes forces (nb_forces); every nstlist-th step first rebuilds the grid and
the outer pair list (nb_search) and prunes it fully; every other step prunes one rolling part of
the outer list, before the forces (nb_prune) or next to them on a second stream (nb_prune_overlapped,
PAPER.md L193; --prune auto benches the faster).  Whatever --steps is, BOTH kinds of step are timed in
the same run: K inner steps and S = max(3, ceil(K/nstlist)) search steps (the schedule is restarted
S times), and ms_per_step = (mean search step + (nstlist-1) * mean inner step) / nstlist is the cost
of a step in the proportions the method prescribes -- every row of SURVEY 8(a) is inside it.
`value` = effective pair interactions (non-excluded atom pairs with r < rc, the paper's "effective"
throughput, L167-L173) per second = mean pairs per step / ms_per_step.

N > 1 (torchrun): the path does not shard ("replicas only"): every rank runs an
independent replica on its own GPU, no data-path collective; value = sum over ranks / max time.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "effective non-bonded pair interactions/s (cluster-pair step: put_atoms+search/prune+forces)"
UNIT = "pairs/s"
# FP32 work of the force kernel per atom-pair slot: what the unmasked F-only
# step executes, counted in its SASS -- packed FFMA2 = 4 flop, FMUL2/FADD2 = 2, FFMA = 2,
# FADD/FMUL/MUFU/compare/select = 1 -- divided by the 256 slots of a warp step.  (SURVEY 8.4's estimate of the
# method's work was 62 / 40; the smaller executed count is the one used.)
FLOP_PER_SLOT = {"ewald": 54.75, "rf": 35.75, "none": 30.75}
N_SM, FP32_LANES_PER_SM = 148, 128   # B200_PROFILING.md: 148 SMs; 128 FP32 lanes/SM (4 SMSP x 32)
HBM_FALLBACK_GBS = 6650.0            # B200_PROFILING.md fallback when MEASURED_PEAKS.json is absent
PRUNE_FLOP_PER_CHECK = 8             # 3 sub + 1 mul + 2 fma (= 5 more flop) per atom-pair distance check
GRID_BYTES_PER_ATOM = 120            # algorithmic bytes of (a2) per atom


def measured_hbm_gbs():
    """(GB/s, source): the driver-measured copy bandwidth, else the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel, config, coulomb):
    """DRAM bytes per launch of `kernel` ("force" / "prune") from the NEWEST committed ncu --set full summary
    under profiles/ for this workload (dram__bytes_read.sum + dram__bytes_write.sum of its first captured
    launch), or (None, reason).  Nothing is hard-coded: a summary that is not there gives null."""
    import glob
    import re
    tag = f"cfg{config}" + ("_rf" if coulomb == "rf" else "")
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", f"r*_{kernel}_full_{tag}.md")))
    if not files:
        return None, f"no profiles/r*_{kernel}_full_{tag}.md committed for this workload"
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    total, found = 0.0, 0
    with open(files[-1]) as fh:
        for line in fh:
            m = re.match(r"\| `dram__bytes_(read|write)\.sum` \| (\w+) \| ([0-9.eE+-]+) \|", line)
            if m and m.group(2) in scale:
                total += float(m.group(3)) * scale[m.group(2)]
                found += 1
    if found < 2:
        return None, f"{os.path.basename(files[-1])} has no dram__bytes rows"
    return total, "profiles/" + os.path.basename(files[-1])


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json configs[k] (default 2: ~96k atoms)")
    ap.add_argument("--coulomb", default="ewald", choices=["ewald", "rf"], help="config 2 only")
    ap.add_argument("--water-nside", type=int, default=0,
                    help="instead of a BASELINE config: nside^3 water molecules, run parameters of config 1 (PAPER.md Fig. 7 size sweep)")
    ap.add_argument("--lj-rc", type=float, default=0.0,
                    help="instead of a BASELINE config: the LJ-only fluid of PAPER.md Fig. 6 (157 464 atoms) at this cut-off, nm")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-flush", action="store_true", help="do not flush L2 between timed steps")
    ap.add_argument("--prune", default="auto", choices=["auto", "plain", "overlapped"],
                    help="rolling prune on the caller's stream before the force kernel (plain), on the library's second "
                         "stream next to it (overlapped, PAPER.md L193: the part pruned on this step's coordinates is first "
                         "used by the next step), or whichever of the two is faster over a short untimed trial (auto)")
    ap.add_argument("--inner-step", default="nb_step", choices=["nb_step", "calls"],
                    help="inner steps of the device leg through nb_step (one call, one CUDA graph launch) or through the three "
                         "calls nb_put_atoms / nb_prune / nb_forces; the e2e leg and the stage-timing passes always use the calls")
    ap.add_argument("--e2e-prune", default="overlapped", choices=["overlapped", "plain"],
                    help="e2e leg: nb_step_host (rolling prune hidden behind the host<->device copies) or put/prune/forces in sequence")
    ap.add_argument("--first-prune", default="separate", choices=["separate", "fused"],
                    help="first use of a fresh list: nb_prune(.., 0, 1) then nb_forces (separate), or the one-kernel nb_forces_prune "
                         "(fused, PAPER.md L189)")
    ap.add_argument("--split-frac", type=float, default=0.0,
                    help="side measurement of the local / non-local kernel pair (SURVEY 8.1 f4, PAPER.md L101): the molecules with "
                         "x < frac * Lx are local, the rest non-local; prints its own JSON line instead of the bench line")
    return ap.parse_args()


def load_workload(args):
    from paper_2006_09167_b200 import workloads
    if args.lj_rc > 0:
        return workloads.lj_fluid(54, rc=args.lj_rc)
    if args.water_nside > 0:
        return workloads.water_box(args.water_nside)
    if args.config == 2:
        return workloads.config2(args.coulomb)
    return workloads.by_index(args.config)


def workload_config(w, args, extra=None):
    origin = ("PAPER.md Fig. 6 stand-in (SURVEY 8.1 f2)" if args.lj_rc > 0 else
              "PAPER.md Fig. 7 size sweep stand-in (SURVEY 8.1 f2)" if args.water_nside > 0 else
              f"BASELINE.json configs[{args.config}]")
    cfg = {"workload": f"{origin} {w.name}: {w.natoms} atoms, box "
                       f"{float(w.box[0]):.4f}x{float(w.box[1]):.4f}x{float(w.box[2]):.4f} nm, {w.coulomb} rc={w.rc}, "
                       f"rlist_outer={w.rlist_outer}, rlist_inner={w.rlist_inner}, nstlist={w.nstlist}, "
                       f"rolling prune in {w.nparts} parts",
           "natoms": w.natoms, "nstlist": w.nstlist, "nparts": w.nparts,
           "parallelism": "replicas only (one independent box per GPU)"}
    if extra:
        cfg.update(extra)
    return cfg


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.stop_flag = index, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:   # NVML missing: report no clocks rather than fail the bench
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                 nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                 nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap"}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.002)

    def result(self):
        self.stop_flag = True
        if self.nv is not None and not self.samples:   # (a region shorter than the thread's start-up: one reading now)
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
            except Exception:
                pass
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": []}
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons)}


class Replica:
    """One box on one GPU, driven through the Python binding of the C ABI."""

    def __init__(self, w, device_index, flush, overlapped=False, fused_first=False):
        import numpy as np
        import torch
        from paper_2006_09167_b200 import nb
        self.torch, self.np, self.w = torch, np, w
        self.dev = torch.device("cuda", device_index)
        torch.cuda.set_device(self.dev)
        self.ctx = nb.context_for(w, device=device_index)
        nframes = w.nstlist
        # coordinates of the motion recipe for one list lifetime, resident in HBM / pinned on the host
        frames = np.stack([w.positions_at(t) for t in range(nframes)])
        self.x_dev = torch.from_numpy(frames).to(self.dev)
        self.x_host = torch.from_numpy(frames).pin_memory()
        self.q_dev = torch.from_numpy(w.q).to(self.dev)
        self.t_dev = torch.from_numpy(w.type).to(self.dev)
        self.q_host = torch.from_numpy(w.q).pin_memory()
        self.t_host = torch.from_numpy(w.type).pin_memory()
        self.f_dev = torch.zeros((w.natoms, 3), dtype=torch.float32, device=self.dev)
        self.e_dev = torch.zeros(2, dtype=torch.float64, device=self.dev)
        self.v_dev = torch.zeros(9, dtype=torch.float64, device=self.dev)
        self.f_host = torch.zeros((w.natoms, 3), dtype=torch.float32).pin_memory()
        self.e_host = torch.zeros(2, dtype=torch.float64).pin_memory()
        self.v_host = torch.zeros(9, dtype=torch.float64).pin_memory()
        # L2 flush buffer: 256 MiB > 126 MB L2, written between timed steps (outside the events)
        self.flush_buf = torch.empty(256 << 20, dtype=torch.uint8, device=self.dev) if flush else None
        self.pairs_at_frame = None
        self.slots_at_frame = None
        self.overlapped = overlapped
        self.fused_first = fused_first
        self.e2e_overlap = True

    def _rolling_prune(self, fr):
        w, c = self.w, self.ctx
        if self.overlapped:
            c.prune_overlapped(w.rlist_inner, fr % w.nparts, w.nparts)   # next to the force kernel (L193)
        else:
            c.prune(w.rlist_inner, fr % w.nparts, w.nparts)              # rolling part (L193)

    def step_device(self, t):
        """Inputs already in HBM (the `value` leg)."""
        w, c = self.w, self.ctx
        fr = t % w.nstlist
        # charges and types are constant: handed over with the coordinates of a search step only
        c.put_atoms(self.x_dev[fr], self.q_dev if fr == 0 else None, self.t_dev if fr == 0 else None, w.box)
        if fr == 0:
            c.search(w.rlist_outer)
            if self.fused_first:                   # first use of a fresh list: prune inside the force kernel
                c.forces_prune(w.rlist_inner, self.f_dev, self.e_dev, self.v_dev)
            else:
                c.prune(w.rlist_inner, 0, 1)       # ... or a full prune (L187) followed by the force kernel
                c.forces(self.f_dev, self.e_dev, self.v_dev)   # energies + virial once per list lifetime
        else:
            self._rolling_prune(fr)
            c.forces(self.f_dev, None, None)

    def step_device_graph(self, t):
        """Same schedule, inner steps through nb_step (put + rolling prune + forces as one call / one CUDA graph launch)."""
        w, c = self.w, self.ctx
        fr = t % w.nstlist
        if fr == 0:
            self.step_device(t)
        else:
            c.step(self.x_dev[fr], w.rlist_inner, fr % w.nparts, w.nparts, self.f_dev)

    def step_host(self, t):
        """Host buffers in, host buffers out (the `e2e` leg): copies inside the timed region.  Inner steps go through
        nb_step_host: the rolling prune of the NEXT step's part runs on this step's coordinates, on the library's second
        stream, next to the device-to-host copy of the forces and the next host-to-device copy."""
        w, c = self.w, self.ctx
        fr = t % w.nstlist
        if fr == 0:
            c.put_atoms_host(self.x_host[fr].numpy(), self.q_host.numpy(), self.t_host.numpy(), w.box)
            c.search(w.rlist_outer)
            c.prune(w.rlist_inner, 0, 1)
            c.forces_host(self.f_host.numpy(), self.e_host.numpy(), self.v_host.numpy())
        elif self.e2e_overlap and w.nparts <= 32:
            c.step_host(self.x_host[fr].numpy(), self.f_host.numpy(), w.rlist_inner, (fr + 1) % w.nparts, w.nparts)
        else:
            c.put_atoms_host(self.x_host[fr].numpy(), None, None, w.box)
            c.prune(w.rlist_inner, fr % w.nparts, w.nparts)
            c.forces_host(self.f_host.numpy(), None, None)

    def flush(self):
        if self.flush_buf is not None:
            self.flush_buf.fill_(1)

    def count_pass(self):
        """Untimed pass over one list lifetime that records, per frame, the effective pair count and
        the atom-pair slots the force kernel evaluates (both counted by the library's own kernels)."""
        w = self.w
        self.pairs_at_frame, self.slots_at_frame = [], []
        for t in range(w.nstlist):
            self.step_device(t)
            n_int, _ = self.ctx.count_pairs()
            self.pairs_at_frame.append(n_int)
            self.slots_at_frame.append(self.ctx.count_slots())

    @staticmethod
    def schedule(nstlist, k_inner):
        """Schedule positions of the timed region: S = max(3, ceil(K/nstlist)) list lifetimes are started (a
        search step at position 0 each) and K inner steps follow them, spread evenly; every step is timed."""
        n_search = max(3, -(-k_inner // max(nstlist - 1, 1)))
        per = [k_inner // n_search + (1 if i < k_inner % n_search else 0) for i in range(n_search)]
        pos = []
        for n in per:
            pos.append(0)
            pos.extend(1 + (j % max(nstlist - 1, 1)) for j in range(n))
        return pos

    def timed(self, step_fn, positions):
        """Times the steps at the given schedule positions with one CUDA-event pair per step on the stream
        the library launches on.  Returns {"search"/"inner": (ms, steps, effective pairs, slots)}."""
        torch = self.torch
        stream = torch.cuda.current_stream(self.dev)
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in positions]
        for i, t in enumerate(positions):
            self.flush()
            ev[i][0].record(stream)
            step_fn(t)
            ev[i][1].record(stream)
        torch.cuda.synchronize(self.dev)
        out = {"search": [0.0, 0, 0, 0], "inner": [0.0, 0, 0, 0]}
        for (a, b), t in zip(ev, positions):
            fr = t % self.w.nstlist
            o = out["search" if fr == 0 else "inner"]
            o[0] += a.elapsed_time(b)
            o[1] += 1
            o[2] += self.pairs_at_frame[fr]
            o[3] += self.slots_at_frame[fr]
        return out


def schedule_mean(pop, nstlist):
    """(ms per step, pairs per step, slots per step) of the method's schedule -- one search step and
    nstlist-1 inner steps per list lifetime -- from the two timed populations."""
    s, i = pop["search"], pop["inner"]
    if i[1] == 0:
        return s[0] / s[1], s[2] / s[1], s[3] / s[1]
    wts, wti = 1.0 / nstlist, (nstlist - 1.0) / nstlist
    return (wts * s[0] / s[1] + wti * i[0] / i[1], wts * s[2] / s[1] + wti * i[2] / i[1],
            wts * s[3] / s[1] + wti * i[3] / i[1])


def cpu_baseline(w, budget_s=12.0):
    """The oracle as it stands (fp64, linked cells, OpenMP over the host cores), timed on the same
    workload: whole force+energy evaluations until ~budget_s of CPU work is spent."""
    from oracle import oracle as O
    beta = O.beta_from_rtol(w.rc, w.ewald_rtol) if w.coulomb == "ewald" else 0.0
    p = O.Params(rc=w.rc, ntypes=w.ntypes, coulomb=w.coulomb, beta=beta)
    reps, spent, npairs = 0, 0.0, 0
    method = "cells" if min(w.box) >= 3.0 * w.rc else "allpairs"   # (the linked-cell loop wants 3 cells per axis: config 0 is smaller)
    while reps < 2 or (spent < budget_s and reps < 50):
        t0 = time.perf_counter()
        r = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p, method=method)
        spent += time.perf_counter() - t0
        npairs += r.npairs
        reps += 1
    return {"value": npairs / spent, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle",
            "sample": f"{reps} full force+energy+virial evaluations of the same {w.natoms}-atom box by "
                      f"oracle_forces_{method} (fp64), {spent:.1f} s of wall time",
            "ms_per_eval": 1e3 * spent / reps}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/unit.  Each step is one oracle
    force+energy+virial evaluation of the BENCHED workload itself (same seeded box as the b200 arm);
    only when the whole --steps/--warmup run would not end within a few minutes is a smaller box of
    the same recipe/density/cut-offs evaluated instead, and the line says which."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import oracle as O
    from paper_2006_09167_b200 import workloads
    full = load_workload(args)
    nsteps = args.steps + args.warmup
    budget = 150.0
    run = dict(rc=full.rc, rlist_outer=full.rlist_outer, rlist_inner=full.rlist_inner, nstlist=full.nstlist,
               nparts=full.nparts, coulomb=full.coulomb)

    def make(nside):
        L = (nside ** 3 / workloads.MOLECULES_PER_NM3) ** (1.0 / 3.0)
        return workloads._lattice_water(f"sample_{nside}", workloads.SEED_BASE + 100 + nside, nside, 0, L, **run)

    def evaluate(w):
        beta = O.beta_from_rtol(w.rc, w.ewald_rtol) if w.coulomb == "ewald" else 0.0
        p = O.Params(rc=w.rc, ntypes=w.ntypes, coulomb=w.coulomb, beta=beta)
        t0 = time.perf_counter()
        r = O.forces(w.x, w.q, w.type, w.box, w.lj_c6c12, w.excl_off, w.excl_idx, p,
                     method="cells" if min(w.box) >= 3.0 * w.rc else "allpairs")
        return time.perf_counter() - t0, r.npairs

    evaluate(full)                       # (pages the library and the box in)
    dt_full, _ = evaluate(full)
    if dt_full * nsteps <= budget:
        w, which = full, "the benched workload itself"
    else:
        min_side = int(3.0 * full.rc * workloads.MOLECULES_PER_NM3 ** (1.0 / 3.0)) + 2   # >= 3 cells of rc per axis
        probe = make(min_side)
        evaluate(probe)
        dt, _ = evaluate(probe)
        per_mol = dt / min_side ** 3
        nside = min_side
        full_side = round((full.natoms / 3) ** (1.0 / 3.0))
        while nside + 1 <= full_side and per_mol * (nside + 1) ** 3 * nsteps <= budget:
            nside += 1
        w = probe if nside == min_side else make(nside)
        which = (f"a {w.natoms}-atom water box of the same recipe/density/cut-offs (the {full.natoms}-atom workload would "
                 f"take {dt_full * nsteps:.0f} s for {nsteps} evaluations, over the {budget:.0f} s budget)")
    for _ in range(args.warmup):
        evaluate(w)
    spent, npairs = 0.0, 0
    for _ in range(args.steps):
        dt, n = evaluate(w)
        spent += dt
        npairs += n
    value = npairs / spent
    sample = f"each step = one oracle_forces_cells evaluation (fp64, force+energy+virial) of {which}"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * spent / max(args.steps, 1),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(full, args, {"reference_sample_atoms": w.natoms,
                                                   "reference_sample": "full workload" if w is full else "sized sample"}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": O.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


class Ranks:
    """Barrier and max / sum over the ranks of a torchrun launch.  The path does not shard ("replicas
    only"): every rank runs an independent replica, so these are the ONLY
    inter-rank operations -- timing scalars, no data-path collective.  `device` is the CUDA device
    of the rank under NCCL, or "cpu" under gloo (tests/test_bench_dist.py)."""

    def __init__(self, world, device):
        self.world, self.device = world, device

    def _sync(self):
        import torch
        if str(self.device) != "cpu":
            torch.cuda.synchronize(self.device)

    def barrier(self):
        import torch.distributed as dist
        self._sync()
        if self.world > 1:
            dist.barrier()
        self._sync()

    def _reduce(self, v, op):
        if self.world == 1:
            return v
        import torch
        import torch.distributed as dist
        t = torch.tensor([v], dtype=torch.float64, device=self.device)
        dist.all_reduce(t, op=op)
        return float(t.item())

    def max(self, v):
        import torch.distributed as dist
        return self._reduce(v, dist.ReduceOp.MAX)

    def sum(self, v):
        import torch.distributed as dist
        return self._reduce(v, dist.ReduceOp.SUM)

    def job_value(self, units_local, ms_local):
        """Whole-job throughput: units all ranks processed / the slowest rank's device time."""
        ms_max = self.max(ms_local)
        return self.sum(float(units_local)) / (ms_max * 1e-3), ms_max


def run_b200(args):
    import torch
    import torch.distributed as dist
    from paper_2006_09167_b200 import nb
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the non-bonded path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)

    ranks = Ranks(world, dev)
    barrier, max_over_ranks, sum_over_ranks = ranks.barrier, ranks.max, ranks.sum

    w = load_workload(args)
    rep = Replica(w, local_rank, flush=not args.no_flush, overlapped=args.prune == "overlapped" and w.nparts <= 32,
                  fused_first=args.first_prune == "fused")
    rep.e2e_overlap = args.e2e_prune == "overlapped"
    ctx = rep.ctx
    fma_peak = ctx.measure_fp32_peak()          # lane-FMA/s of a register-resident FFMA chain, this GPU, now
    fp32_forms = ctx.measure_fp32_pipe()        # pipe occupancy of the FP32 / FP32x2 instruction forms, this GPU, now
    rep.count_pass()                            # untimed: per-frame pair and slot counts (also warms everything up)
    W = max(args.warmup, 3)
    K = args.steps
    positions = Replica.schedule(w.nstlist, K)  # K inner steps + S >= 3 search steps, all timed
    S = sum(1 for t in positions if t == 0)

    # ---------------- device-resident leg: `value` ----------------
    for i in range(W):
        rep.step_device(i)
    # The `value` pass carries no stage timing at all: an event pair around one kernel costs two event records per
    # launch, each a serialisation point of the stream (measured: +5 us on the 116 us inner step of config 2 with only
    # the force kernel timed, 13-26 % with every stage timed).  The force kernel (the roofline's kernel) is timed with
    # CUDA events in a second pass over the same schedule positions, the remaining stages in a third.
    ctx.timing_enable(False)
    prune_trial = None
    if args.prune == "auto" and w.nparts <= 32:
        # untimed trial: 24 inner steps of each mode (after their own warm-up), the faster one is benched
        trial_pos = [0] + list(range(1, 25))
        prune_trial = {}
        for mode in ("plain", "overlapped"):
            rep.overlapped = mode == "overlapped"
            fn = rep.step_device_graph if (args.inner_step == "nb_step" and not rep.overlapped) else rep.step_device
            for t in trial_pos[:9]:
                fn(t)
            pop_t = rep.timed(fn, trial_pos)
            prune_trial[mode] = pop_t["inner"][0] / pop_t["inner"][1]
        rep.overlapped = prune_trial["overlapped"] < prune_trial["plain"]
    use_step = args.inner_step == "nb_step" and not rep.overlapped
    step_value = rep.step_device_graph if use_step else rep.step_device
    for i in range(W):
        step_value(i)
    launches0 = ctx.get_stats()["kernel_launches"]
    barrier()
    sampler = ClockSampler(local_rank)
    sampler.start()
    pop = rep.timed(step_value, positions)
    barrier()
    st1 = ctx.get_stats()
    launches = st1["kernel_launches"] - launches0 - 3   # get_stats itself launches three counting kernels
    # second pass: the same steps with an event pair around the force kernel only
    force_bit = (1 << nb.NB_T_NAMES.index("force")) | (1 << nb.NB_T_NAMES.index("force_energy"))
    ctx.timing_stages(force_bit)
    ctx.timing_enable(True)
    ctx.timing_read(reset=True)
    # (plain prune in both stage passes: the stage timer brackets launches on the caller's stream, and the force kernel
    # is to be timed alone, not next to a prune on the second stream)
    was_overlapped, rep.overlapped = rep.overlapped, False
    pop_f = rep.timed(rep.step_device, positions)
    stages = ctx.timing_read(reset=True)
    # third pass: the other stages
    ctx.timing_stages(0xFFFFFFFF & ~force_bit)
    rep.timed(rep.step_device, positions)
    rep.overlapped = was_overlapped
    stages_other = ctx.timing_read(reset=True)
    clocks = sampler.result()   # sampled every 2 ms over the three timed passes (the value pass alone lasts a few ms at --steps 20)
    stages = {k: (stages[k] if k in ("force", "force_energy") else stages_other[k]) for k in stages}
    ctx.timing_stages(0xFFFFFFFF)
    ctx.timing_enable(False)
    ms_step, pairs_step, slots_step = schedule_mean(pop, w.nstlist)
    ms_step_f, _, _ = schedule_mean(pop_f, w.nstlist)
    ms_step_max = max_over_ranks(ms_step)
    value = sum_over_ranks(float(pairs_step)) / (ms_step_max * 1e-3)
    ms_search = max_over_ranks(pop["search"][0] / max(pop["search"][1], 1))
    ms_inner = max_over_ranks(pop["inner"][0] / max(pop["inner"][1], 1))

    # ---------------- host-buffer leg: `e2e` ----------------
    e2e = None
    if not args.no_e2e:
        for i in range(W):
            rep.step_host(i)
        barrier()
        pop_h = rep.timed(rep.step_host, positions)
        barrier()
        ms_h, pairs_h, _ = schedule_mean(pop_h, w.nstlist)
        ms_h_max = max_over_ranks(ms_h)
        n = w.natoms
        e2e = {"value": sum_over_ranks(float(pairs_h)) / (ms_h_max * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": n * 12 + n * 8 / w.nstlist,        # x every step; q, type on search steps
               "d2h_bytes_per_step": n * 12 + 11 * 8 / w.nstlist,       # f every step; energies + virial on search steps
               "prune": "nb_step_host: next step's part pruned next to the copies" if rep.e2e_overlap and w.nparts <= 32 else "plain",
               "ms_per_step": ms_h_max, "ms_search_step": pop_h["search"][0] / max(pop_h["search"][1], 1),
               "ms_inner_step": pop_h["inner"][0] / max(pop_h["inner"][1], 1)}

    # ---------------- rooflines ----------------
    sm_max = clocks["sm_max_mhz"] or 1965
    peak_tflops = N_SM * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    hbm_gbs, hbm_src = measured_hbm_gbs()
    per_stage_us = {k: (1e3 * v[0] / v[1] if v[1] else None) for k, v in stages.items()}
    # dominant kernel: the force kernel (FP32 ALU bound), F-only flavour of the inner steps
    f_ms, f_n = stages["force"]
    flop_slot = FLOP_PER_SLOT[w.coulomb]
    slots_per_launch = pop["inner"][3] / max(pop["inner"][1], 1)
    force_us = 1e3 * f_ms / max(f_n, 1)
    achieved = flop_slot * slots_per_launch / (force_us * 1e-6) / 1e12 if f_n else 0.0
    workload_is_config = args.lj_rc <= 0 and args.water_nside <= 0
    traffic, traffic_src = ncu_traffic("force", args.config, w.coulomb) if workload_is_config else (None, "not a BASELINE config")
    roofline = {"bound": "alu", "kernel": "k_force (a7)", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": achieved / peak_tflops, "traffic": traffic,
                "traffic_source": "dram__bytes_read.sum + dram__bytes_write.sum of one k_force launch, ncu --set full: " + traffic_src,
                "peak_source": f"derived: {N_SM} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x {sm_max} MHz (clocks.max.sm); "
                               "MEASURED_PEAKS.json has no FP32 entry",
                "measured_ffma_chain_tflops": 2 * fma_peak / 1e12,
                "frac_of_measured_ffma_chain": achieved / (2 * fma_peak / 1e12),
                "fp32_pipe_cycles_per_warp_instruction": fp32_forms,
                "fp32_pipe_note": "measured (nb_measure_fp32_pipe, 4 warps per sub-partition): an FFMA2 with three different register "
                                  "pairs holds the FP32 pipe ~4 cycles (register-file bandwidth), with a repeated or constant operand "
                                  "~2.3-2.5, a scalar FFMA ~1; the kernel's step is 124 packed instructions, see DESIGN.md section 6",
                "flop_per_slot": flop_slot, "slots_per_launch": slots_per_launch, "kernel_us": force_us,
                "kernel_us_is": "mean of the F-only launches (the inner steps), CUDA events on the launching stream, in a second timed "
                                "pass over the same schedule positions with the plain prune, i.e. the kernel alone (ms_per_step of that "
                                "pass: ms_per_step_with_force_events); "
                                "the F+E+virial launches of the search steps are stage_us.force_energy",
                "ms_per_step_with_force_events": ms_step_f}

    line = None
    if rank == 0:
        st = st1
        # prune kernel (a6): one rolling part per inner step; arithmetic = 64 distance checks per outer cluster pair
        n_outer, n_listed = st["n_pairs_outer"], slots_step / 8.0   # listed j atoms ~ slots / 8
        p_us = per_stage_us["prune"]
        prune_launch_pairs = n_outer * (S + (pop["inner"][1]) / w.nparts) / max(S + pop["inner"][1], 1)   # mean over full + rolling launches
        prune_flop = prune_launch_pairs * 64 * PRUNE_FLOP_PER_CHECK
        prune_bytes = prune_launch_pairs * 4 + st["nslots"] * 16 + (prune_launch_pairs / max(n_outer, 1)) * n_listed * 4
        ptraffic, ptraffic_src = ncu_traffic("prune", args.config, w.coulomb) if workload_is_config else (None, "not a BASELINE config")
        roofline_prune = None
        if p_us:
            roofline_prune = {"kernel": "k_prune (a6)", "kernel_us": p_us,
                              "kernel_us_is": "mean over the timed launches: S full prunes and K rolling parts (plain-prune pass)",
                              "bound": "alu", "achieved": prune_flop / (p_us * 1e-6) / 1e12, "peak": peak_tflops, "unit": "TFLOP/s",
                              "frac": prune_flop / (p_us * 1e-6) / 1e12 / peak_tflops,
                              "flop_per_check": PRUNE_FLOP_PER_CHECK, "checks_per_launch": prune_launch_pairs * 64,
                              "hbm": {"achieved": prune_bytes / (p_us * 1e-6) / 1e9, "peak": hbm_gbs, "unit": "GB/s",
                                      "frac": prune_bytes / (p_us * 1e-6) / 1e9 / hbm_gbs, "peak_source": hbm_src,
                                      "algorithmic_bytes_per_launch": prune_bytes,
                                      "bytes_are": "4 B per outer cluster pair read + xq once (16 B/slot) + 4 B per surviving j-atom entry written",
                                      "traffic": ptraffic, "traffic_source": ptraffic_src}}
        # gridding (a2): HBM-side algorithmic bytes, and what the launch count alone costs
        g_us = per_stage_us["grid"]
        roofline_grid = None
        if g_us:
            gbytes = GRID_BYTES_PER_ATOM * w.natoms
            roofline_grid = {"kernels": "k_bin, k_col_scan, k_col_scatter, k_col_layout, k_grid_tail (a2)", "stage_us": g_us,
                             "bound": "hbm", "bytes_per_atom": GRID_BYTES_PER_ATOM, "achieved": gbytes / (g_us * 1e-6) / 1e9,
                             "peak": hbm_gbs, "unit": "GB/s", "frac": gbytes / (g_us * 1e-6) / 1e9 / hbm_gbs, "peak_source": hbm_src,
                             "launches": 5, "launch_floor_us": 5 * 2.5,
                             "note": "latency- and sort-bound at these sizes: five dependent launches (~2.5 us each) and a "
                                     "per-column shared-memory sort; once per nstlist steps"}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": ms_step_max, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f32", "data": "synthetic",
                "config": workload_config(w, args, {"l2": "flushed between timed steps (256 MiB fill)" if not args.no_flush
                                                    else "not flushed", "prune": ("overlapped (second stream, next to the force kernel; the part pruned on this step's coordinates "
                                                              "is first used by the next step)" if rep.overlapped else "plain (before the force kernel)"),
                                                    "prune_trial_ms_inner_step": prune_trial,
                                                    "first_prune": args.first_prune,
                                                    "inner_step": "nb_step (CUDA graph)" if use_step else "three calls"}),
                "schedule": {"timed_inner_steps": pop["inner"][1], "timed_search_steps": S, "ms_inner_step": ms_inner,
                             "ms_search_step": ms_search,
                             "ms_per_step_is": "(ms_search_step + (nstlist-1) * ms_inner_step) / nstlist"},
                "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline,
                "roofline_prune": roofline_prune, "roofline_grid": roofline_grid,
                "raw_pairs_per_s_per_gpu": slots_step / (ms_step * 1e-3),
                "work_efficiency": pairs_step / max(slots_step, 1),
                "stage_us": per_stage_us,
                "stage_share_of_step": {k: ((v / w.nstlist if k in ("grid", "search", "masks") else v) / (1e3 * ms_step) if v else None)
                                        for k, v in per_stage_us.items()},
                "stage_timing": "the timed region of `value` carries no stage events; force: second pass over the same steps with an event "
                                "pair around the force kernel; other stages: third pass with the plain prune",
                "list": {k: st[k] for k in ("nsuper", "n_sci_entries", "n_joint_outer", "n_pairs_outer", "n_pairs_inner",
                                            "n_excl_masks", "n_work_units", "list_grow_retries")}}
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w)
        print(json.dumps(line))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_split(args):
    """Inner steps with the force work as the paper's two kernels: put + rolling prune, then
    nb_forces_nonlocal (high-priority stream) and nb_forces_local.  Reports when the halo forces are complete (host clock
    at the return of nb_sync_nonlocal) and when everything is, next to the same steps through nb_forces.  One GPU; not
    the bench line."""
    import time

    import numpy as np
    import torch
    from paper_2006_09167_b200 import nb, workloads
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the non-bonded path has no CPU fallback")
    w0 = load_workload(args)
    w, nlocal = workloads.local_first(w0, lambda x: x[:, 0] < args.split_frac * w0.box[0])
    dev = torch.device("cuda", 0)
    torch.cuda.set_device(dev)
    ctx = nb.context_for(w, device=0)
    ctx.set_local(nlocal)
    frames = torch.from_numpy(np.stack([w.positions_at(t) for t in range(w.nstlist)])).to(dev)
    q, typ = torch.from_numpy(w.q).to(dev), torch.from_numpy(w.type).to(dev)
    f = torch.zeros((w.natoms, 3), dtype=torch.float32, device=dev)
    flush = None if args.no_flush else torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    ctx.put_atoms(frames[0], q, typ, w.box)
    ctx.search(w.rlist_outer)
    ctx.prune(w.rlist_inner, 0, 1)
    info = ctx.split_info()

    def step(fr, split):
        ctx.put_atoms(frames[fr], None, None, w.box)
        ctx.prune(w.rlist_inner, fr % w.nparts, w.nparts)
        if split:
            ctx.forces_nonlocal(f)
            ctx.forces_local(f)
        else:
            ctx.forces(f, None, None)

    out = {}
    for split in (False, True):
        t_halo, t_all = [], []
        for k in range(args.warmup + args.steps):
            fr = 1 + k % (w.nstlist - 1)
            if flush is not None:
                flush.fill_(1)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            step(fr, split)
            if split:
                ctx.sync_nonlocal()
                t1 = time.perf_counter()
            torch.cuda.synchronize()
            t2 = time.perf_counter()
            if k >= args.warmup:
                t_all.append(t2 - t0)
                if split:
                    t_halo.append(t1 - t0)
        out["split" if split else "union"] = {"us_all_forces": 1e6 * float(np.median(t_all)),
                                              **({"us_halo_forces": 1e6 * float(np.median(t_halo))} if split else {})}
    print(json.dumps({"measurement": "local / non-local kernel pair (SURVEY 8.1 f4, PAPER.md L101), inner step = put + rolling "
                                     "prune + forces, host clock from the first call to completion, median",
                      "config": workload_config(w, args, {"nlocal": nlocal, "split_frac": args.split_frac,
                                                          "segments_local": info["nseg_local"],
                                                          "segments_nonlocal": info["nseg"] - info["nseg_local"]}),
                      "steps": args.steps, "warmup": args.warmup, **out}))
    return 0


def main():
    args = parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.split_frac > 0:
        return run_split(args)
    return run_b200(args)


if __name__ == "__main__":
    sys.exit(main())
