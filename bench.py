#!/usr/bin/env python
"""bench.py -- throughput of the all-pairs softened-gravity hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C1] [--impl reference]

One "step" = one pass of the whole hot path over one batch of synthetic input: one nb_force call
(j-pack + pair-interaction kernel + j-split reduce) on BASELINE.json configs[1] -- the N = 131072
equal-mass Plummer sphere, i-set = j-set, eps = 1/256, seed 1 (the paper's largest N).
Metric: interactions/s = n_i * n_j / t (the paper's N^2 of Eq. (4)), with Gflop/s at
20 and 38 flop per interaction alongside.

Prints ONE JSON line on rank 0.  Multi-GPU (N > 1, under torchrun): the path does not shard in this
build (BASELINE.json: "Everything runs on one GPU"), so N ranks run N independent replicas with no
data-path collective ("replicas only"); value = total interactions of all ranks / max time.
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

import numpy as np  # noqa: E402

METRIC = "interactions/s"
FP32_INST_PER_PAIR = 13          # FMA-pipe instructions per interaction (acc + phi), DESIGN.md "Roofline"
FP32_LANES_PER_SM_CLK = 128
CONFIG_INDEX = {"C0": 0, "C1": 1, "C2": 2, "C3": 3, "C4": 4}
L2_FLUSH_BYTES = 256 << 20       # > 126 MB L2


def modelled_traffic(args, prob, nb, sm_count):
    """DRAM bytes one launch of the dominant kernel moves, MODELLED from the live plan (not pasted from an old capture):
    first touch of the inputs it reads + its outputs + the j-split partials (written, then read by the second pass; they
    fit L2, so this is an upper bound for them).  The ncu measurements it is checked against are in profiles/."""
    if args.op != "force":
        return None, "not modelled for this op (ncu captures: profiles/)"
    w = prob.w
    base = 16.0 * w.n_j + 12.0 * w.n_i + 16.0 * w.n_i              # packed j (or x_j + m_j), x_i, a + phi
    sp = nb.plan_query_small(w.n_i, w.n_j, sm_count)
    if sp["default"]:
        groups = sp["S"] // sp["CS"]
        partial = 2.0 * 32.0 * w.n_i * groups if groups > 1 else 0.0
        return base + partial, f"modelled from the live plan (small-i-set kernel, {groups} partial group(s) of 32 B per i)"
    p = nb.plan_query(w.n_i, w.n_j, sm_count)
    partial = 2.0 * 32.0 * w.n_i * p["S"] if p["S"] > 1 else 0.0
    return base + partial, (f"modelled from the live plan (S = {p['S']} j-chunks x n_i x 32 B of FP64 partials, written and read "
                            "back; ncu on C1: 72.0 MB, profiles/r02_ncu_c1.md)")


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"sm_max_mhz": 1965.0, "hbm_gbs": 6650.0}, "fallback"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thread = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as exc:  # NVML missing: report that, never fake numbers
            self.nv, self.h, self.err = None, None, repr(exc)

    def _run(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.02)

    def start(self):
        if self.nv is not None:
            self._thread = threading.Thread(target=self._run, daemon=True)
            self._thread.start()

    def stop(self) -> dict:
        self._stop.set()
        if self._thread is not None:
            self._thread.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML unavailable"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


def physical_gpu_index(local_rank: int) -> int:
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


ORACLE_KEEP = {}     # the last oracle_rate run's (idx, acc, pot): --check compares the timed GPU output with it


def oracle_rate(w, target_seconds: float, rng_seed: int = 0):
    """Times the CPU oracle, as it stands, on a bounded i-sample of workload w.  Returns (pairs/s, cores, sample)."""
    import oracle
    cores = oracle.num_threads()
    rng = np.random.default_rng(rng_seed)

    def run(n_i):
        idx = np.sort(rng.choice(w.n_i, n_i, replace=False))
        xi = np.ascontiguousarray(w.xi[idx])
        t0 = time.perf_counter()
        ra, rp = oracle.force(xi, w.x_j, w.m_j, w.eps2)
        dt = time.perf_counter() - t0
        ORACLE_KEEP.update(idx=idx, acc=ra, pot=rp)
        return dt

    n_probe = min(w.n_i, max(64, 8 * cores))
    run(min(n_probe, 64))                                   # page in, spin up the OpenMP team
    t_probe = run(n_probe)
    rate = n_probe * w.n_j / t_probe
    n_i = int(min(w.n_i, max(n_probe, target_seconds * rate / w.n_j)))
    t = run(n_i)
    return n_i * w.n_j / t, cores, f"{n_i} of {w.n_i} i-particles (seeded, sorted) x all {w.n_j} j-particles, {t:.2f} s"


def reduce_max(values, world):
    """Max over ranks of a list of floats (device timings): NCCL on the GPU, gloo on the CPU tests."""
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor(list(values), dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def replica_throughput(pairs_per_rank_step, world, steps, total_ms):
    """Whole-job interactions/s of `world` independent replicas: all ranks' units / the slowest rank's time."""
    return world * pairs_per_rank_step * steps / (total_ms * 1e-3)


def reference_arm(args, wl):
    """--impl reference: the CPU oracle (this tier has no reference implementation), rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    if args.op == "force":
        w = wl.config(CONFIG_INDEX[args.config])
        name = workload_name(args.config, w)
    elif args.op == "jerk":
        w = wl.plummer_workload(131072, 1.0 / 256, seed=1, name="H1", with_velocities=True)
        name = "row f1 (H1): plummer N=131072 with velocities, one force+jerk+phi evaluation"
    elif args.op == "cunbody":
        w = wl.config(1)
        name = "row f3 (G1): configs[1]'s particles, Fig. A.3 pipeline (oracle force on a sample)"
    elif args.op == "cunbody4":
        w = wl.plummer_workload(131072, 1.0 / 256, seed=1, name="H1", with_velocities=True)
        name = "row f3 (G2): H1's particles, Fig. A.4 pipeline (oracle force_jerk on a sample)"
    elif args.op == "lj":
        w = LJ_ROWS(wl)
        name = "row f3 (L1): Lennard-Jones fluid, 131072 particles (oracle lennard_jones on a sample)"
    elif args.op == "hermite":
        w = wl.plummer_workload(65536, 1.0 / 128, seed=4, name="C4", with_velocities=True)
        name = "C4's particles, force+jerk evaluations of the Hermite integration (oracle force_jerk on a sample)"
    elif args.op == "block":
        w = wl.plummer_workload(65536, 1.0 / 128, seed=4, name="C4", with_velocities=True)
        name = "row f4 (B1): C4's particles, force+jerk evaluations of the block-step integration (oracle force_jerk on a sample)"
    elif args.op == "leapfrog":
        w = wl.config(4)
        name = "BASELINE.json configs[4] (C4): force evaluations of the KDK integration, N=65536 (oracle force on a sample)"
    else:
        w = wl.tree_list_workload(524288, 32, 256, 2000, 6000, 1.0 / 128, seed=7, name="T1")
        name = "row f2 (T1): tree lists, 524288 particles, groups 32..256, lists 2000..6000"
    per_step = max(0.5, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_rate_op(args.op, w, per_step / 4)
    rates, sample, cores = [], "", 0
    t0 = time.perf_counter()
    for s in range(args.steps):
        r, cores, sample = oracle_rate_op(args.op, w, per_step, rng_seed=s)
        rates.append(r)
    wall = time.perf_counter() - t0
    value = float(np.mean(rates))
    f_lo, f_hi = OPS[args.op]["flops"]
    out = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * wall / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": name, "op": args.op},
        f"gflops_{f_lo}": f_lo * 1e-9 * value, f"gflops_{f_hi}": f_hi * 1e-9 * value,
        "cpu_baseline": {"value": value, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": METRIC, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(out), flush=True)


def workload_name(cfg_name, w):
    return (f"BASELINE.json configs[{CONFIG_INDEX[cfg_name]}] ({cfg_name}): {w.meta.get('model', '')}, "
            f"n_i={w.n_i}, n_j={w.n_j}, eps2={w.eps2:.6g}, seed={w.seed}, one nb_force call with phi")


# ---------------------------------------------------------------------------------------------
# The ops bench.py can time.  "force" (default) is the contract line: BASELINE.json's metric on
# configs[1].  "jerk" (row f1) and "batched" (row f2) are the widened rows, each with its own
# instruction count per interaction for the roofline.
OPS = {
    "force": {"inst": 13, "kernel": "nb_force_kernel (pair interaction, rows a2-a7)", "flops": (20, 38)},
    "jerk": {"inst": 27, "kernel": "nb_hermite_kernel (force + jerk + potential, row f1)", "flops": (60, 60)},
    "batched": {"inst": 13, "kernel": "nb_force_kernel<BATCHED> (row f2)", "flops": (20, 38)},
    # BASELINE.json configs[4]: one bench "step" = one nb_leapfrog_kdk call of LEAPFROG_KDK_PER_CALL KDK steps that
    # continues the integration (the first call also pays the initial force evaluation)
    # (the integration needs phi only at the final time: 100 of the 101 evaluations of a call run the 12-instruction
    #  loop without it, so the algorithmic count for the roofline is 12 per interaction here)
    # row f3: the paper's cunbody_api call for its Fig. A.3 pipeline through the generalised kernel (scalar FP32;
    # the listing has no potential: 12 FP32-pipe instructions per interaction)
    "cunbody": {"inst": 12, "kernel": "pipeline_kernel2<PipelineForceA3> (generalised kernel, packed path, row f3)", "flops": (20, 38)},
    # Fig. A.4 through the generalised kernel: the listing's 27 FP32-pipe instructions per pair (28 in the packed form's SASS)
    "cunbody4": {"inst": 27, "kernel": "pipeline_kernel2<PipelineForceJerkPotA4> (generalised kernel, packed path, row f3)", "flops": (60, 60)},
    "leapfrog": {"inst": 12, "kernel": "nb_force_kernel<PHI=false> inside nb_leapfrog_kdk (row a8)", "flops": (20, 38)},
}
# row f3, a central force other than gravity (reading R19): 24 FP32-pipe instructions per pair in the SASS of
# pipeline_kernel<PipelineLennardJones> (12 FMUL + 7 FFMA + 5 FADD) + 1 MUFU.RSQ; Gflop/s printed at 24 and at 50 per pair
# row f2 with the lists as int32 indices into ONE packed particle array (nb_force_batched_indexed): same kernel arithmetic,
# the ring filled by gathered cp.async copies; 4 B per list entry + 16 B per distinct particle cross PCIe in the e2e leg
OPS["batched_indexed"] = {"inst": 13, "kernel": "nb_batched_kernel<INDEXED> (row f2, lists as indices)", "flops": (20, 38)}
OPS["lj"] = {"inst": 24, "kernel": "pipeline_kernel<PipelineLennardJones> (generalised kernel, row f3)", "flops": (24, 50)}
LEAPFROG_KDK_PER_CALL = 100


def LJ_ROWS(wl):
    """row f3 (L1): the Lennard-Jones bench workload -- a dense fluid of 131072 particles (jittered lattice, density 0.8)."""
    return wl.lj_fluid_rows(131072, 0.8, 0.1, seed=1)
# (phi is wanted only at the final time: 100 of the 101 evaluations of a call run the 26-instruction loop without it)
OPS["hermite"] = {"inst": 26, "kernel": "nb_hermite_kernel<PHI=false> inside nb_hermite4 (consumer of row f1)", "flops": (60, 60)}
# row f4, active-subset integration: one bench "step" = one cycle of BLOCK_SUB_STEPS nb_hermite4_block_step calls under a
# three-level block schedule (half of the particles due every sub-step, a quarter every 2nd, a quarter every 4th)
OPS["block"] = {"inst": 26, "kernel": "nb_hermite_kernel<PHI=false> inside nb_hermite4_block_step (row f4, n_act x n pairs)",
                "flops": (60, 60)}
BLOCK_SUB_STEPS = 4


class Problem:
    """One op on one workload: device call, end-to-end call from pinned host buffers, oracle sample."""

    def __init__(self, op, cfg_name, nb, torch, wl):
        self.op, self.nb, self.torch = op, nb, torch
        if op == "force":
            if isinstance(cfg_name, tuple):                                   # --n N --n-i M: an active subset (C2's recipe)
                w = wl.subset_workload(cfg_name[0], cfg_name[1], 1.0 / 256, seed=1, name=f"subset{cfg_name[1]}of{cfg_name[0]}")
                name = (f"shape scan: {w.meta.get('model', '')}, n_i={w.n_i}, n_j={w.n_j}, eps2={w.eps2:.6g}, seed=1, "
                        f"one nb_force call with phi")
            elif isinstance(cfg_name, int):
                w = wl.plummer_workload(cfg_name, 1.0 / 256, seed=1, name=f"plummer{cfg_name}")
                name = f"N-scan: {w.meta.get('model', '')}, n_i=n_j={cfg_name}, eps2={w.eps2:.6g}, seed=1, one nb_force call with phi"
            else:
                w = wl.config(CONFIG_INDEX[cfg_name])
                name = workload_name(cfg_name, w)
            self.w, self.pairs, self.name = w, float(w.pairs), name
            self.host = [w.x_j, w.m_j] + ([] if w.x_i is None else [w.x_i])
            self.n_out = w.n_i
        elif op == "leapfrog":
            w = self.integrator_workload(cfg_name, wl)
            self.w = w
            self.pairs = float(w.n_j) ** 2 * (LEAPFROG_KDK_PER_CALL + 1)     # force evaluations per call x N^2
            self.name = ((f"BASELINE.json configs[4] (C4)" if w.name == "C4" else "small system (C4's recipe at another N)") +
                         f": {w.meta.get('model', '')} with Aarseth velocities, N={w.n_j}, "
                         f"eps2={w.eps2:.6g}, dt=1/512, seed=4; one step = one nb_leapfrog_kdk call of "
                         f"{LEAPFROG_KDK_PER_CALL} KDK steps (the config's 1000 steps = 10 such calls)")
            self.host = [w.x_j, w.v, w.m_j]
            self.n_out = w.n_j
            self.kdk_done = 0
        elif op == "cunbody":
            w = wl.config(1)
            self.w, self.pairs = w, float(w.pairs)
            self.name = (f"row f3 (G1): configs[1]'s particles as the paper's rows p_xi[n][4] = (x,y,z,eps2), p_xj[n][4] = "
                         f"(x,y,z,m) (Fig. A.1), n={w.n_j}, eps2={w.eps2:.6g}; one nb_cunbody_force call (Fig. A.3 pipeline, no phi)")
            p_xi = np.concatenate([w.x_j, np.full((w.n_j, 1), w.eps2, np.float32)], axis=1).astype(np.float32)
            p_xj = np.concatenate([w.x_j, w.m_j[:, None]], axis=1).astype(np.float32)
            self.host = [np.ascontiguousarray(p_xj), np.ascontiguousarray(p_xi)]
            self.n_out = w.n_j
        elif op == "cunbody4":
            w = wl.plummer_workload(131072, 1.0 / 256, seed=1, name="H1", with_velocities=True)
            self.w, self.pairs = w, float(w.n_j) ** 2
            self.name = (f"row f3 (G2): H1's particles as the paper's rows p_xi[n][6] = (x, v), p_xj[n][7] = (x, v, m) (Fig. A.2), "
                         f"n={w.n_j}, eps2 = 1/256^2 (the listing's constant); one nb_cunbody_force_jerk_pot call (Fig. A.4 pipeline)")
            p_xi = np.concatenate([w.x_j, w.v], axis=1).astype(np.float32)
            p_xj = np.concatenate([w.x_j, w.v, w.m_j[:, None]], axis=1).astype(np.float32)
            self.host = [np.ascontiguousarray(p_xj), np.ascontiguousarray(p_xi)]
            self.n_out = w.n_j
        elif op == "lj":
            rows = LJ_ROWS(wl)
            self.w, self.pairs = rows, float(rows.shape[0]) ** 2
            self.name = (f"row f3 (L1): Lennard-Jones fluid on a jittered simple-cubic lattice, density 0.8, sigma in [0.9, 1.1], eps in "
                         f"[0.5, 1.5], rows (x,y,z,sigma/2,sqrt(eps)), n={rows.shape[0]}, seed=1; one nb_cunbody_lennard_jones call")
            self.host = [rows, rows]
            self.n_out = rows.shape[0]
        elif op == "hermite":
            w = self.integrator_workload(cfg_name, wl)
            self.w = w
            self.pairs = float(w.n_j) ** 2 * (LEAPFROG_KDK_PER_CALL + 1)
            self.name = (f"configs[4]'s particles (C4: N={w.n_j}, eps2={w.eps2:.6g}, dt=1/512, seed=4) under the 4th-order Hermite "
                         f"scheme: one step = one nb_hermite4 call of {LEAPFROG_KDK_PER_CALL} time steps (101 force+jerk evaluations)")
            self.host = [w.x_j, w.v, w.m_j]
            self.n_out = w.n_j
            self.kdk_done = 0
        elif op == "block":
            w = wl.config(4)
            self.w = w
            level = wl.block_levels(w.n_j, seed=4)
            self.active = [np.nonzero(s % (1 << level) == 0)[0].astype(np.int32) for s in range(1, BLOCK_SUB_STEPS + 1)]
            self.pairs = float(sum(a.size for a in self.active)) * float(w.n_j)
            self.sub_dt = w.dt / BLOCK_SUB_STEPS
            self.name = (f"row f4 (B1): configs[4]'s particles (C4: N={w.n_j}, eps2={w.eps2:.6g}, seed=4) under block time steps, "
                         f"three levels (seeded: 1/2 of the particles step with dt/4, 1/4 with dt/2, 1/4 with dt = 1/512); one "
                         f"step = one cycle of {BLOCK_SUB_STEPS} nb_hermite4_block_step calls, n_act = "
                         f"{[int(a.size) for a in self.active]} of {w.n_j} against all {w.n_j}")
            dx, dv, dm = (torch.from_numpy(a).cuda() for a in (w.x_j, w.v, w.m_j))
            a0, j0, _ = nb.force_jerk(dx, dv, dx, dv, dm, w.eps2, want_pot=False)      # a, j of the start state (set-up)
            torch.cuda.synchronize()
            self.host = [w.x_j, w.v, w.m_j, a0.cpu().numpy(), j0.cpu().numpy(), np.zeros(w.n_j, dtype=np.float64)] + self.active
            self.n_out = w.n_j
            self.cycles_done = 0
        elif op == "jerk":
            n_sub = cfg_name[1] if isinstance(cfg_name, tuple) else 0     # --n N --n-i M: an active subset (C2's recipe)
            n_h = cfg_name[0] if isinstance(cfg_name, tuple) else (cfg_name if isinstance(cfg_name, int) else 131072)   # --n N: the N-scan of row f1
            w = wl.plummer_workload(n_h, 1.0 / 256, seed=1, name="H1" if n_h == 131072 else f"plummer{n_h}", with_velocities=True)
            if n_sub:
                import dataclasses
                idx = np.sort(np.random.default_rng(1).choice(n_h, n_sub, replace=False))
                w = dataclasses.replace(w, x_i=np.ascontiguousarray(w.x_j[idx]), i_index=idx.astype(np.int64), name=f"subset{n_sub}of{n_h}")
            self.w, self.pairs = w, float(w.n_i) * float(w.n_j)
            self.name = (f"row f1 ({'H1' if n_h == 131072 and not n_sub else 'shape scan'}): {w.meta.get('model', '')} with Aarseth velocities, "
                         f"n_i={w.n_i}, n_j={w.n_j}, eps2={w.eps2:.6g}, seed=1, one nb_force_jerk call with phi"
                         + (" (configs[1]'s particles)" if n_h == 131072 and not n_sub else ""))
            self.host = [w.x_j, w.v, w.m_j] + ([w.x_i, np.ascontiguousarray(w.v[w.i_index])] if n_sub else [])
            self.n_out = w.n_i
        elif op == "batched_indexed":
            w = wl.tree_list_workload(524288, 32, 256, 2000, 6000, 1.0 / 128, seed=7, name="T1")
            self.w, self.pairs = w, float(w.pairs)
            # the distinct list records are the tree code's particle array (particles + cell pseudo-particles), the lists
            # become indices into it: pure re-indexing of the seeded workload, no arithmetic
            rec = np.ascontiguousarray(np.concatenate([w.x_j, w.m_j[:, None]], axis=1).astype(np.float32))
            key = rec.view(np.uint64).reshape(-1, 2)
            _, first, inv = np.unique(key[:, 0] ^ (key[:, 1] * np.uint64(0x9E3779B97F4A7C15)), return_index=True, return_inverse=True)
            xm_p = np.ascontiguousarray(rec[first])
            assert np.array_equal(xm_p[inv], rec)
            self.name = (f"row f2 (T1 indexed): {w.meta.get('model', '')}; 524288 particles in {w.n_batch} groups of 32..256, lists "
                         f"of 2000..6000 as int32 indices ({inv.size} entries) into {xm_p.shape[0]} distinct packed records, "
                         f"eps2={w.eps2:.6g}, seed=7, one nb_force_batched_indexed call with phi")
            self.host = [w.i_offsets, w.j_offsets, w.x_i, inv.astype(np.int32), xm_p]
            self.n_out = w.x_i.shape[0]
        else:
            w = wl.tree_list_workload(524288, 32, 256, 2000, 6000, 1.0 / 128, seed=7, name="T1")
            self.w, self.pairs = w, float(w.pairs)
            self.name = (f"row f2 (T1): {w.meta.get('model', '')}; 524288 particles in {w.n_batch} groups of 32..256, "
                         f"lists of 2000..6000, eps2={w.eps2:.6g}, seed=7, one nb_force_batched call with phi")
            self.host = [w.i_offsets, w.j_offsets, w.x_i, w.x_j, w.m_j]
            self.n_out = w.x_i.shape[0]
        self.dev = [torch.from_numpy(a).cuda() for a in self.host]
        self.pinned = [torch.from_numpy(a).pin_memory() for a in self.host]
        n = self.n_out
        self.outs = [torch.empty((n, 4 if op == "lj" else (7 if op == "cunbody4" else 3)), dtype=torch.float32, device="cuda")]
        if op == "block":
            self.outs = [self.dev[k] for k in (0, 1, 3, 4)]            # the state itself is the result: x, v, a, j
        if op in ("jerk", "hermite"):
            self.outs.append(torch.empty((n, 3), dtype=torch.float32, device="cuda"))
        if op not in ("cunbody", "cunbody4", "lj", "block"):
            self.outs.append(torch.empty((n,), dtype=torch.float32, device="cuda"))
        self.h_outs = [torch.empty(o.shape, dtype=torch.float32).pin_memory() for o in self.outs]
        self.h2d = int(sum(a.nbytes for a in self.host))
        self.d2h = int(sum(o.numel() * 4 for o in self.outs))

    @staticmethod
    def integrator_workload(cfg_name, wl):
        """C4, or -- with --n N -- C4's recipe (Plummer sphere with Aarseth velocities, eps = 1/128, dt = 1/512, seed 4) at another N."""
        if isinstance(cfg_name, int):
            return wl.plummer_workload(cfg_name, 1.0 / 128, seed=4, name=f"plummer{cfg_name}", with_velocities=True, dt=1.0 / 512, n_steps=1000)
        return wl.config(4)

    def call(self, t=None):
        t = self.dev if t is None else t
        nb, w = self.nb, self.w
        if self.op == "force":
            xj, mj = t[0], t[1]
            xi = xj if w.x_i is None else t[2]
            nb.force(xi, xj, mj, w.eps2, acc_out=self.outs[0], pot_out=self.outs[1])
        elif self.op == "cunbody":
            nb.cunbody_force(t[0], t[1], self.outs[0])
        elif self.op == "cunbody4":
            nb.cunbody_force_jerk_pot(t[0], t[1], self.outs[0])
        elif self.op == "lj":
            nb.cunbody_lennard_jones(t[0], t[1], self.outs[0])
        elif self.op == "leapfrog":
            nb.leapfrog_kdk(t[0], t[1], t[2], w.eps2, w.dt, LEAPFROG_KDK_PER_CALL, acc_io=self.outs[0], pot_out=self.outs[1])
            if t is self.dev:
                self.kdk_done += LEAPFROG_KDK_PER_CALL
        elif self.op == "hermite":
            nb.hermite4(t[0], t[1], t[2], w.eps2, w.dt, LEAPFROG_KDK_PER_CALL, acc_io=self.outs[0], jerk_io=self.outs[1],
                        pot_out=self.outs[2])
            if t is self.dev:
                self.kdk_done += LEAPFROG_KDK_PER_CALL
        elif self.op == "block":
            base = self.cycles_done * BLOCK_SUB_STEPS if t is self.dev else 0          # staged state starts at time 0
            launches = 0
            for s in range(1, BLOCK_SUB_STEPS + 1):
                nb.hermite4_block_step(t[0], t[1], t[2], t[3], t[4], t[5], t[5 + s], (base + s) * self.sub_dt, w.eps2)
                launches += nb.last_launch_count()
            self.launches = launches
            if t is self.dev:
                self.cycles_done += 1
        elif self.op == "batched_indexed":
            nb.force_batched_indexed(t[0], t[1], t[2], t[3], t[4], w.eps2, acc_out=self.outs[0], pot_out=self.outs[1])
        elif self.op == "jerk":
            xi, vi = (t[3], t[4]) if len(t) > 3 else (t[0], t[1])
            nb.force_jerk(xi, vi, t[0], t[1], t[2], w.eps2, acc_out=self.outs[0], jerk_out=self.outs[1], pot_out=self.outs[2])
        else:
            nb.force_batched(t[0], t[1], t[2], t[3], t[4], w.eps2, acc_out=self.outs[0], pot_out=self.outs[1])

    def call_e2e(self):
        """Inputs from pinned host memory, results back to pinned host memory, blocking."""
        nb, w = self.nb, self.w
        if self.op == "force":
            h = [p.numpy() for p in self.pinned]
            nb.force_host(h[0] if w.x_i is None else h[2], h[0], h[1], w.eps2,
                          acc_out=self.h_outs[0].numpy(), pot_out=self.h_outs[1].numpy())
            return
        if self.op == "jerk":
            h = [p.numpy() for p in self.pinned]
            nb.force_jerk_host(h[3] if len(h) > 3 else h[0], h[4] if len(h) > 3 else h[1], h[0], h[1], h[2], w.eps2, acc_out=self.h_outs[0].numpy(),
                               jerk_out=self.h_outs[1].numpy(), pot_out=self.h_outs[2].numpy())
            return
        staged = [p.cuda(non_blocking=True) for p in self.pinned]
        self.call(staged)
        outs = [staged[k] for k in (0, 1, 3, 4)] if self.op == "block" else self.outs
        for h, d in zip(self.h_outs, outs):
            h.copy_(d, non_blocking=True)
        self.torch.cuda.synchronize()

    @property
    def e2e_api(self):
        if self.op == "force":
            return "nb_force_host (pinned host buffers)"
        if self.op == "jerk":
            return "nb_force_jerk_host (pinned host buffers)"
        if self.op == "cunbody":
            return "pinned host rows -> cudaMemcpyAsync -> nb_cunbody_force -> cudaMemcpyAsync -> pinned host"
        if self.op == "cunbody4":
            return "pinned host rows -> cudaMemcpyAsync -> nb_cunbody_force_jerk_pot -> cudaMemcpyAsync -> pinned host"
        if self.op == "lj":
            return "pinned host rows -> cudaMemcpyAsync -> nb_cunbody_lennard_jones -> cudaMemcpyAsync -> pinned host"
        if self.op == "block":
            return ("pinned host (x, v, m, a, j, t, 4 active lists) -> cudaMemcpyAsync -> 4 x nb_hermite4_block_step -> "
                    "cudaMemcpyAsync of x, v, a, j -> pinned host")
        if self.op == "hermite":
            return "pinned host (x, v, m) -> cudaMemcpyAsync -> nb_hermite4 (100 steps) -> cudaMemcpyAsync of a, j, phi -> pinned host"
        if self.op == "leapfrog":
            return "pinned host (x, v, m) -> cudaMemcpyAsync -> nb_leapfrog_kdk (100 KDK steps) -> cudaMemcpyAsync of a, phi -> pinned host"
        name = {"jerk": "force_jerk", "batched_indexed": "force_batched_indexed"}.get(self.op, "force_batched")
        return f"pinned host tensors -> cudaMemcpyAsync -> nb_{name} -> cudaMemcpyAsync -> pinned host"

    def plan(self, sm_count):
        if self.op == "force":
            sp = self.nb.plan_query_small(self.w.n_i, self.w.n_j, sm_count)
            return dict(sp, kernel="nb_small_kernel") if sp["default"] else self.nb.plan_query(self.w.n_i, self.w.n_j, sm_count)
        if self.op in ("cunbody", "cunbody4", "lj"):
            return {"cta": "256 threads x 8 or 4 i-records as packed pairs, double-buffered 128-record j tiles, Bloom test per tile, "
                           "j-range split over S CTAs in whole waves + second pass"}
        if self.op == "hermite":
            return self.nb.plan_query_jerk(self.w.n_j, self.w.n_j, sm_count)
        if self.op == "leapfrog":
            return self.nb.plan_query(self.w.n_j, self.w.n_j, sm_count)
        if self.op == "jerk":
            sp = self.nb.plan_query_small_jerk(self.w.n_i, self.w.n_j, sm_count)
            return dict(sp, kernel="nb_small_hermite_kernel") if sp["default"] else self.nb.plan_query_jerk(self.w.n_i, self.w.n_j, sm_count)
        if self.op == "block":
            return {str(int(a.size)): self.nb.plan_query_jerk(int(a.size), self.w.n_j, sm_count) for a in self.active[:3]}
        return {"cta": "one row of CTAs, 8 warps split each list (WJ = 8), no split across CTAs"}


def oracle_rate_op(op, w, target_seconds, rng_seed=0):
    """CPU oracle, as it stands, on a bounded sample of the op's workload: (pairs/s, cores, sample)."""
    import oracle
    if op in ("force", "leapfrog", "cunbody"):
        return oracle_rate(w, target_seconds, rng_seed)
    if op in ("hermite", "block", "cunbody4"):
        op = "jerk"
    if op == "batched_indexed":
        op = "batched"
    cores = oracle.num_threads()
    rng = np.random.default_rng(rng_seed)
    if op == "lj":
        n = w.shape[0]

        def run_lj(n_i):
            idx = np.sort(rng.choice(n, n_i, replace=False))
            rows_i = np.ascontiguousarray(w[idx])
            t0 = time.perf_counter()
            oracle.lennard_jones(rows_i, w)
            return time.perf_counter() - t0
        run_lj(64)
        n_probe = max(64, 8 * cores)
        rate = n_probe * n / run_lj(n_probe)
        n_i = int(min(n, max(n_probe, target_seconds * rate / n)))
        t = run_lj(n_i)
        return n_i * n / t, cores, f"{n_i} of {n} i-particles (seeded) x all {n} j-particles, {t:.2f} s"
    if op == "jerk":
        def run(n_i):
            idx = np.sort(rng.choice(w.n_i, n_i, replace=False))
            v_all = w.v if w.i_index is None else w.v[w.i_index]
            xi, vi = np.ascontiguousarray(w.xi[idx]), np.ascontiguousarray(v_all[idx])
            t0 = time.perf_counter()
            oracle.force_jerk(xi, vi, w.x_j, w.v, w.m_j, w.eps2)
            return time.perf_counter() - t0
        run(64)
        n_probe = max(64, 8 * cores)
        rate = n_probe * w.n_j / run(n_probe)
        n_i = int(min(w.n_i, max(n_probe, target_seconds * rate / w.n_j)))
        t = run(n_i)
        return n_i * w.n_j / t, cores, f"{n_i} of {w.n_i} i-particles (seeded) x all {w.n_j} j-particles, {t:.2f} s"
    order = rng.permutation(w.n_batch)
    pairs, t0, used = 0, time.perf_counter(), 0
    for b in order:
        i0, i1, j0, j1 = (int(v) for v in (w.i_offsets[b], w.i_offsets[b + 1], w.j_offsets[b], w.j_offsets[b + 1]))
        oracle.force(w.x_i[i0:i1], w.x_j[j0:j1], w.m_j[j0:j1], w.eps2)
        pairs += (i1 - i0) * (j1 - j0)
        used += 1
        if time.perf_counter() - t0 > target_seconds:
            break
    t = time.perf_counter() - t0
    return pairs / t, cores, f"{used} of {w.n_batch} sub-problems (seeded order), one oracle.force call each, {t:.2f} s"


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", default="C1", choices=["C0", "C1", "C2", "C3"])
    ap.add_argument("--op", default="force", choices=sorted(OPS))
    ap.add_argument("--n", type=int, default=0, help="--op force / jerk (leapfrog / hermite: C4's recipe at this N): an equal-mass Plummer sphere of this N "
                    "(eps = 1/256, seed 1) instead of a BASELINE.json config; for the N-scan in profiles/")
    ap.add_argument("--n-i", type=int, default=0, help="with --n N (--op force / jerk): the i-set is a seeded random subset of this many of the "
                    "N particles (C2's recipe at another shape)")
    ap.add_argument("--shard", action="store_true", help="--op force only: i-shard ONE problem over the ranks (row f4: "
                    "all-gather of the packed j records over NCCL, then nb_force_packed on the local i-slice; strong "
                    "scaling) instead of N independent replicas")
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--check", action="store_true", help="--op force / jerk: add a 'parity' object -- the timed call's "
                    "output against the CPU oracle (Eq. (3), PAPER.md:278) on the i-particles the cpu_baseline leg evaluated "
                    "(all 131072 of C1 when the host finishes them in --cpu-seconds), else on 2048 sampled ones")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup

    from paper_astro_ph_0703100_b200 import workloads as wl

    if args.impl == "reference":
        reference_arm(args, wl)
        return

    import torch
    import torch.distributed as dist

    import paper_astro_ph_0703100_b200 as nb

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    nb.lib()
    peaks, peaks_kind = load_peaks()
    op = OPS[args.op]
    if args.op in ("leapfrog", "hermite") and args.n > 0:
        # small systems replay their steps from a CUDA graph inside the library, which needs a capturable stream: the whole
        # run (flushes, events, calls) goes to a side stream instead of the default one
        torch.cuda.set_stream(torch.cuda.Stream())

    # inputs resident in HBM before the timed region
    prob = Problem(args.op, ((args.n, args.n_i) if 0 < args.n_i < args.n else args.n) if (args.n > 0 and args.op in ("force", "jerk", "leapfrog", "hermite")) else args.config,
                   nb, torch, wl)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream()
    if args.shard:
        if args.op != "force" or prob.w.x_i is not None:
            raise SystemExit("--shard needs --op force on a config whose i-set is its j-set (C0, C1, C3, --n)")
        from paper_astro_ph_0703100_b200 import sharded
        n_all = prob.w.n_j
        lo, hi = sharded.shard_range(n_all, rank, world)
        x_loc, m_loc = prob.dev[0][lo:hi].contiguous(), prob.dev[1][lo:hi].contiguous()
        acc_loc, pot_loc = prob.outs[0][lo:hi], prob.outs[1][lo:hi]

        def sharded_call(t=None):
            xm_all = sharded.gather_packed(x_loc, m_loc, n_all)          # the one exchange step: 16 B x N over NCCL
            nb.force_packed(x_loc, xm_all, prob.w.eps2, acc_out=acc_loc, pot_out=pot_loc)
        prob.call = sharded_call
        prob.call_e2e = sharded_call                                     # no host leg in the sharded mode
        prob.pairs = float(n_all) * float(n_all) / world                 # per rank; replica_throughput multiplies by world

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        flush.fill_(1)
        prob.call()
    torch.cuda.synchronize()
    launches_per_step = prob.launches if args.op == "block" else nb.last_launch_count()

    sampler = ClockSampler(physical_gpu_index(local_rank))
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    # the library's per-kernel events make every launch of a launch-bound small-system run slower and switch its step graph
    # off: those lines (--op leapfrog / hermite --n N) are timed without them, their roofline comes from the whole call
    kernel_events = not (args.op in ("leapfrog", "hermite") and args.n > 0)
    nb.profile_enable(kernel_events)
    barrier()
    sampler.start()
    t_wall0 = time.perf_counter()
    for s in range(args.steps):
        flush.fill_(s & 0xff)                      # L2 flush between timed iterations (outside the events)
        ev[s][0].record(stream)
        prob.call()
        ev[s][1].record(stream)
    barrier()
    t_wall = time.perf_counter() - t_wall0
    clocks = sampler.stop()
    nb.profile_enable(False)
    n_k, k_ms = nb.profile_read()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = float(sum(step_ms))

    # small calls are launch-bound: also report the same call replayed from a CUDA graph (no L2 flush between replays).
    # GRAPH_CALLS calls are captured into ONE graph: a graph of a single 5-us kernel replayed in a Python loop measures the
    # host's cudaGraphLaunch rate (~8 us per replay), not the device
    graph_ms = None
    GRAPH_CALLS, GRAPH_REPLAYS = 50, 8
    if args.op in ("force", "jerk") and not args.shard and prob.pairs < 2.0 ** 30:
        gs = torch.cuda.Stream()
        with torch.cuda.stream(gs):
            for _ in range(3):
                prob.call()                                # warm this stream's workspace
            gs.synchronize()
            g = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g, stream=gs):
                for _ in range(GRAPH_CALLS):
                    prob.call()
            g.replay()
            gs.synchronize()
            g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            g0.record(gs)
            for _ in range(GRAPH_REPLAYS):
                g.replay()
            g1.record(gs)
            gs.synchronize()
        graph_ms = g0.elapsed_time(g1) / (GRAPH_CALLS * GRAPH_REPLAYS)

    # end to end with HOST buffers (pinned), copies inside the timed region
    e2e_steps = max(3, min(args.steps, 10))
    for _ in range(2):
        prob.call_e2e()
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        prob.call_e2e()
    torch.cuda.synchronize()
    e2e_ms = 1e3 * (time.perf_counter() - t0)

    # max over ranks
    total_ms, e2e_ms = reduce_max([total_ms, e2e_ms], world)

    if rank == 0:
        pairs = prob.pairs
        value = replica_throughput(pairs, world, args.steps, total_ms)
        e2e_value = replica_throughput(pairs, world, e2e_steps, e2e_ms)
        f_max = float(peaks.get("sm_max_mhz", 1965.0)) * 1e6
        sm_count = torch.cuda.get_device_properties(0).multi_processor_count
        peak_inst = sm_count * FP32_LANES_PER_SM_CLK * f_max                 # FP32-pipe lane-instructions / s
        # interactions per launch of the dominant kernel (a leapfrog call launches it once per force evaluation)
        pairs_k = float(prob.w.n_j) ** 2 if args.op in ("leapfrog", "hermite") else pairs   # (sharded: this rank's slice x all j)
        if args.op == "block":
            pairs_k = pairs / BLOCK_SUB_STEPS                                # mean over the cycle's launches (n_act varies)
        k_rate = pairs_k * n_k / (k_ms * 1e-3) if n_k else 0.0
        if not kernel_events:                                                # whole calls instead of kernels: evaluations / call time
            n_k, k_ms = args.steps * (LEAPFROG_KDK_PER_CALL + 1), total_ms
            k_rate = pairs_k * n_k / (k_ms * 1e-3)
        inst = op["inst"]
        achieved = inst * k_rate
        traffic, traffic_kind = modelled_traffic(args, prob, nb, sm_count)
        roofline = {
            "bound": "alu",
            "kernel": ("nb_small_kernel (small-i-set kernel: pair interaction packed over j, rows a1-a7 in one launch)"
                       if args.op == "force" and nb.plan_query_small(prob.w.n_i, prob.w.n_j, sm_count)["default"] else
                       "nb_small_hermite_kernel (small-i-set force + jerk kernel, packed over j, one launch)"
                       if args.op == "jerk" and nb.plan_query_small_jerk(prob.w.n_i, prob.w.n_j, sm_count)["default"] else op["kernel"]),
            "achieved": achieved / 1e12, "peak": peak_inst / 1e12, "unit": "FP32-pipe Tinst/s",
            "frac": achieved / peak_inst, "traffic": traffic,
            "traffic_unit": "DRAM bytes per launch of the dominant kernel",
            "traffic_kind": traffic_kind,
            "kernel_ms": k_ms / max(1, n_k), "kernel_launches_timed": n_k,
            "kernel_interactions_per_s": k_rate, "roofline_interactions_per_s": peak_inst / inst,
            "peak_source": f"{sm_count} SMs x {FP32_LANES_PER_SM_CLK} FP32 lanes x sm_max_mhz {f_max / 1e6:.0f} MHz "
                           f"({peaks_kind} MEASURED_PEAKS.json clock), {inst} FMA-pipe instr/interaction",
        }
        if clocks.get("sm_mhz"):
            roofline["frac_at_observed_clock"] = achieved / (sm_count * FP32_LANES_PER_SM_CLK * clocks["sm_mhz"] * 1e6)
        f_lo, f_hi = op["flops"]
        out = {
            "metric": METRIC, "value": value, "unit": METRIC, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": total_ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if args.shard else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": prob.name, "op": args.op,
                       "parallelism": (f"i-sharded over {world} rank(s): all-gather of packed j + nb_force_packed" if args.shard
                                       else ("replicas only" if world > 1 else "1 gpu")),
                       "l2": f"flushed between timed iterations ({L2_FLUSH_BYTES >> 20} MiB write, outside the events)",
                       "plan": prob.plan(sm_count)},
            f"gflops_{f_lo}": f_lo * 1e-9 * value, f"gflops_{f_hi}": f_hi * 1e-9 * value,
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": METRIC, "h2d_bytes_per_step": prob.h2d, "d2h_bytes_per_step": prob.d2h,
                    "steps": e2e_steps, "ms_per_step": e2e_ms / e2e_steps, "api": prob.e2e_api},
            "gpu_launches": int(launches_per_step * args.steps),
            "roofline": roofline,
            "wall_s_timed_region": t_wall,
            "paper_context": {"gflops_38_8800gtx_n131072": 256, "interactions_per_s_8800gtx_n131072": 6.74e9,
                              "gflops_force_jerk_8800gtx_n131072": 179,
                              "note": "PAPER.md:314 (includes PCIe copies) and PAPER.md:343; context, not target"},
        }
        if graph_ms is not None:
            out["graph_replay"] = {"ms_per_call": graph_ms, "value": pairs / (graph_ms * 1e-3), "unit": METRIC,
                                   "note": f"{GRAPH_CALLS} calls captured into one CUDA graph, replayed {GRAPH_REPLAYS}x back to "
                                           "back, per call; L2 warm (device time per call: a one-call graph replayed from Python "
                                           "measures the host's launch rate instead)"}
        if args.op == "block":
            out["block_steps_per_s"] = BLOCK_SUB_STEPS * args.steps / (total_ms * 1e-3)
            # the scheduler's share when the due sets are not precomputed: nb_block_schedule + the 4-byte read-back of n_act
            level = wl.block_levels(prob.w.n_j, seed=4)
            dt_k = torch.from_numpy(prob.sub_dt * 2.0 ** level.astype(np.float64)).cuda()
            for _ in range(3):
                _, _, n_act = nb.block_schedule(prob.dev[5], dt_k)
                n_act.item()
            reps = 50
            t0 = time.perf_counter()
            for _ in range(reps):
                _, _, n_act = nb.block_schedule(prob.dev[5], dt_k)
                n_due = int(n_act.item())
            out["scheduler"] = {"us_per_call": 1e6 * (time.perf_counter() - t0) / reps, "n_due": n_due,
                                "api": "nb_block_schedule (5 launches) + 4-byte read-back of n_act, host wall clock",
                                "share_of_a_block_step": (time.perf_counter() - t0) / reps / (total_ms * 1e-3 / (BLOCK_SUB_STEPS * args.steps))}
        if args.op == "block":
            # An ADAPTIVE run never repeats a shape: n_act differs at every block step, so every call plans a new
            # decomposition.  64 block steps with 64 distinct n_act on a copy of the state, timed on the HOST wall clock
            # (enqueue + planning + device), with the planner's cache misses counted (nb_debug_plans_computed).
            rng = np.random.default_rng(11)
            order = rng.permutation(prob.w.n_j)
            sizes = [int(v) for v in np.unique(rng.integers(8, 4096, 96))[:64]]
            acts = [torch.from_numpy(np.sort(order[:k]).astype(np.int32)).cuda() for k in sizes]
            st = [t.clone() for t in prob.dev[:6]]
            t_now = float(st[5].max().item())
            for a in acts[:4]:                                           # warm the workspace, not the plan cache (sizes differ)
                t_now += 1e-9
                nb.hermite4_block_step(st[0], st[1], st[2], st[3], st[4], st[5], a, t_now, prob.w.eps2)
            torch.cuda.synchronize()
            plans0 = nb.debug_plans_computed()
            t0 = time.perf_counter()
            for a in acts[4:]:
                t_now += 1e-9
                nb.hermite4_block_step(st[0], st[1], st[2], st[3], st[4], st[5], a, t_now, prob.w.eps2)
            t_enq = time.perf_counter() - t0
            torch.cuda.synchronize()
            t_all = time.perf_counter() - t0
            n_steps = len(acts) - 4
            out["adaptive"] = {"block_steps": n_steps, "n_act_range": [sizes[4], sizes[-1]], "distinct_shapes": n_steps,
                               "plans_computed": nb.debug_plans_computed() - plans0,
                               "host_enqueue_us_per_step": 1e6 * t_enq / n_steps, "wall_us_per_step": 1e6 * t_all / n_steps,
                               "block_steps_per_s": n_steps / t_all,
                               "note": "every step a new (n_act, n): no plan-cache hit; host wall clock including the planner"}
        if args.op == "hermite":
            out["hermite_steps_per_s"] = LEAPFROG_KDK_PER_CALL * args.steps / (total_ms * 1e-3)
        if args.op == "leapfrog":
            out["kdk_steps_per_s"] = LEAPFROG_KDK_PER_CALL * args.steps / (total_ms * 1e-3)
        if args.op in ("leapfrog", "hermite") and not args.no_cpu_baseline:
            import oracle
            w = prob.w
            _, _, e_start = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
            _, _, e_end = oracle.energy(prob.dev[0].cpu().numpy(), prob.dev[1].cpu().numpy(), w.m_j, w.eps2)
            out["energy"] = {"time_steps": prob.kdk_done, "kdk_steps": prob.kdk_done, "E_start": e_start, "E_end": e_end,
                             "rel_drift": abs(e_end - e_start) / abs(e_start), "by": "oracle.energy (FP64) on the GPU's FP32 (x, v)"}
        if args.op == "block" and not args.no_cpu_baseline:
            import oracle
            w = prob.w
            _, _, e_start = oracle.energy(w.x_j, w.v, w.m_j, w.eps2)
            _, _, e_end = oracle.energy(prob.dev[0].cpu().numpy(), prob.dev[1].cpu().numpy(), w.m_j, w.eps2)
            out["energy"] = {"cycles": prob.cycles_done, "block_steps": prob.cycles_done * BLOCK_SUB_STEPS,
                             "time": prob.cycles_done * w.dt, "E_start": e_start, "E_end": e_end,
                             "rel_drift": abs(e_end - e_start) / abs(e_start),
                             "by": "oracle.energy (FP64) on the GPU's FP32 (x, v), all clocks equal at the end of a cycle"}
        if args.op == "leapfrog":
            out["kdk_steps_per_s"] = LEAPFROG_KDK_PER_CALL * args.steps / (total_ms * 1e-3)
        if not args.no_cpu_baseline:
            v, cores, sample = oracle_rate_op(args.op, prob.w, args.cpu_seconds)
            out["cpu_baseline"] = {"value": v, "unit": METRIC, "cores": cores, "kind": "oracle", "sample": sample}
        if args.check and args.op in ("force", "jerk") and not args.shard:
            import oracle
            w = prob.w
            prob.call()
            torch.cuda.synchronize()
            if args.op == "force" and "idx" in ORACLE_KEEP and not args.no_cpu_baseline:
                # the cpu_baseline leg has just evaluated the oracle on its i-sample (all of C1 on the GPU box): use it
                idx, ra, rp = ORACLE_KEEP["idx"], ORACLE_KEEP["acc"], ORACLE_KEEP["pot"]
                got = [o.cpu().numpy()[idx] for o in prob.outs]
                par = oracle.error_metrics(got[0], ra, got[1], rp)
            else:
                idx = np.sort(np.random.default_rng(0).choice(w.n_i, min(2048, w.n_i), replace=False))
                got = [o.cpu().numpy()[idx] for o in prob.outs]
                if args.op == "force":
                    ra, rp = oracle.force(w.xi[idx], w.x_j, w.m_j, w.eps2)
                    par = oracle.error_metrics(got[0], ra, got[1], rp)
                else:
                    v_all = w.v if w.i_index is None else w.v[w.i_index]
                    ra, rj, rp = oracle.force_jerk(w.xi[idx], v_all[idx], w.x_j, w.v, w.m_j, w.eps2)
                    par = oracle.error_metrics(got[0], ra, got[2], rp)
                    ej = oracle.error_metrics(got[1], rj)
                    par["jerk_max"], par["jerk_rms"] = ej["acc_max"], ej["acc_rms"]
            par["sample"] = f"{len(idx)} of {w.n_i} i-particles (seeded) x all {w.n_j} j-particles, oracle in FP64"
            par["tolerance"] = "acc (jerk) RMS <= 1e-5, max <= 1e-4; phi RMS <= 1e-5 (BASELINE.json north_star)"
            out["parity"] = par
        print(json.dumps(out), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
