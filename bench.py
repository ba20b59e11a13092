#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200-native NeuralFluid pressure projection (forward + adjoint).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--n 256]

Metric (BASELINE.json): ms per forward + adjoint pressure projection at 256^3, both MGPCG solves to a relative
residual of 1e-6, plus achieved HBM GB/s vs the measured peak.  Workload: BASELINE.json configs[3], the 256^3
channel-gate (Dirichlet p = 1 / 0 on -x / +x, closed y/z walls, a 4-cell plate rotating about y, alpha rebuilt every
step), synthetic and seeded (paper_2405_14903_b200/workloads.py).

A "step" is one pass of the whole hot path (SURVEY.md 8a rows a-1 .. a-10):
  forward : nf_advect -> nf_set_solid(phi^{n+1}, u_s^{n+1}) -> nf_project
  backward: nf_project_adjoint (dJ/dUhat, dJ/dalpha, dJ/dU_s) -> nf_weights_adjoint -> nf_advect_adjoint
`value` is the metric's scope -- the device time of nf_project + nf_project_adjoint per step, taken with CUDA events
inside the K timed steps, every input resident in HBM; `ms_per_step` / `full_step_ms` is the whole step.  `e2e` is the
same two projections (plus the nf_set_solid they need) through the C ABI's host-buffer entry points with pinned host
arrays, copies inside the timed region.

Multi-GPU (torchrun): replicas only -- every rank runs its own simulation, no collective on
the data path; value = max-over-ranks time / (K * N).

--impl reference: the fp64 CPU oracle (oracle/nf_oracle.py, as it stands) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "ms per fwd+adjoint pressure projection at 256^3 (1e-6 resid)"
TOL, MAXIT = 1e-6, 400
# algorithmic bytes per FINE cell per launch of each kernel class of the PCG iteration
BYTES = {"apply_A": 25.0, "cg_update": 17.0, "cg_pupdate": 12.0, "down1_fine": 9.0, "down2_fine": 5.5,
         "up1_fine": 13.5, "up2_fine": 13.0, "vec_coarse": 41.0 / 7.0, "rbgs_fine": 24.0, "restrict_fine": 20.5,
         "prolong_fine": 8.5, "sweep_fine": 13.0}


def coarse_bytes_per_fine_cell(nu_l1, nu_deep):
    """Algorithmic bytes of the cooperative coarse kernel per FINE cell.  One level with nu sweeps
    before and after the coarse correction moves, per cell of that level: pre-smoother from zero 9 (r, code in; z
    out), every further half sweep 13 (z, r, code in; z out), residual + restriction 5.5 (+ 4 for r once nu > 1),
    prolongation + black half sweep 13.5, red half sweep 13 -> 41 for nu = 1, 41 + 52 (nu - 1) + 4 otherwise.
    Level 1 holds 1/8 of the fine cells, the deeper ones 1/64 + 1/512 + ... = 1/56."""
    per = lambda nu: 41.0 + (52.0 * (nu - 1) + 4.0 if nu > 1 else 0.0)
    return per(nu_l1) / 8.0 + per(nu_deep) / 56.0


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            pk = json.load(f)
        return float(pk["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1])
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# --------------------------------------------------------------------------------------------------------------
# workload: BASELINE.json configs[3]
# --------------------------------------------------------------------------------------------------------------
class GateWorkload:
    """Device-resident inputs of the channel-gate rollout.  Geometry of `nsteps` consecutive time levels is
    precomputed on the host (closed-form SDF and rigid velocity, workloads.config4_solid) and kept in HBM."""

    def __init__(self, n, nsteps, seed_shift=0, warm_start=False):
        import numpy as np
        import torch
        from paper_2405_14903_b200 import api, workloads as wl
        self.torch, self.np = torch, np
        P = wl.config4_params(n, seed=1004 + seed_shift)
        self.P, self.n = P, n
        self.g = api.Grid(n, n, n, P["dx"])
        self.g.set_dt_rho(P["dt_over_rho"])
        if warm_start:
            self.g.set_solver_options(1, 1, 8)  # nf_project starts from the pressure of the previous step
        for f in range(6):
            self.g.set_domain_bc(f, P["bc_types"][f], P["bc_values"][f])
        d = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
        self.U0 = [d(a) for a in wl.config4_initial_velocity(P)]
        self.geom = []
        for s in range(1, nsteps + 1):
            phi, us = wl.config4_solid(P, s)
            self.geom.append((d(phi), [d(a) for a in us]))
        rng = np.random.default_rng(77 + seed_shift)
        self.gin = [d(rng.standard_normal(a.shape).astype(np.float32)) for a in self.U0]  # dJ/dU^{n+1}
        self.U = [a.clone() for a in self.U0]
        self.Uprev = [torch.empty_like(a) for a in self.U0]
        self.Uhat = [torch.empty_like(a) for a in self.U0]
        self.G = [torch.empty_like(a) for a in self.U0]
        self.ga = [torch.empty_like(a) for a in self.U0]
        self.gs = [torch.empty_like(a) for a in self.U0]
        self.p = torch.zeros(self.g.shape_p, dtype=torch.float32, device="cuda")
        self.gphi = torch.empty(self.g.shape_sdf, dtype=torch.float32, device="cuda")
        self.iters = []
        self.ev = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
        self.proj_ms = 0.0
        self.step_no = 0
        self.proj_events = None   # list of (e0, e1, e2, e3) per step while the metric's scope is being timed

    def step(self, record=False):
        """One pass of the whole hot path (rows a-1 .. a-10)."""
        g, P = self.g, self.P
        phi, us = self.geom[self.step_no % len(self.geom)]
        self.step_no += 1
        for a, b in zip(self.Uprev, self.U):
            a.copy_(b)                                            # saved U^n (back-prop state)
        g.advect(*self.U, P["dt"])                                # a-8
        g.set_solid(phi, *us)                                     # a-1 (+ hierarchy)
        for a, b in zip(self.Uhat, self.U):
            a.copy_(b)                                            # saved Uhat
        pe = None
        if self.proj_events is not None:  # events only (no sync): the projections' share of the timed steps
            pe = [self.torch.cuda.Event(enable_timing=True) for _ in range(4)]
            self.proj_events.append(pe)
            pe[0].record()
        if record:
            self.ev[0].record()
        rc1 = g.project(*self.U, self.p, tol=TOL, maxit=MAXIT)    # a-2 .. a-6
        if record:
            self.ev[1].record()
        if pe:
            pe[1].record()
        it_f = g.last_solve_info()["iters"] if record else -1
        for a, b in zip(self.G, self.gin):
            a.copy_(b)
        if record:
            self.ev[2].record()
        if pe:
            pe[2].record()
        rc2 = g.project_adjoint(*self.G, p_saved=self.p, uhat=self.Uhat, galpha=self.ga, gus=self.gs, tol=TOL,
                                maxit=MAXIT)                      # a-7
        if record:
            self.ev[3].record()
        if pe:
            pe[3].record()
        it_a = g.last_solve_info()["iters"] if record else -1
        g.weights_adjoint(*self.ga, self.gphi)                    # a-10
        g.advect_adjoint(*self.Uprev, *self.G, P["dt"])           # a-9
        if record:
            self.torch.cuda.synchronize()
            self.proj_ms += self.ev[0].elapsed_time(self.ev[1]) + self.ev[2].elapsed_time(self.ev[3])
            self.iters.append((it_f, it_a))
        if rc1 != 0 or rc2 != 0:
            raise RuntimeError("solver did not converge (rc %d / %d)" % (rc1, rc2))


def run_ours(args):
    import numpy as np
    import torch
    import torch.distributed as dist
    from paper_2405_14903_b200 import api, replicas
    api.load_library()  # fail loudly if the CUDA extension is missing: there is no fallback
    rank, world, local = replicas.rank_world()
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    n, K, W = args.n, args.steps, max(args.warmup, 3)
    wlk = GateWorkload(n, min(K + W, 20), seed_shift=replicas.seed_shift(rank), warm_start=args.warm_start)
    g = wlk.g

    def barrier():
        replicas.barrier(dist)
        torch.cuda.synchronize()

    for _ in range(W):
        wlk.step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    wlk.proj_events = []
    e0.record()
    for _ in range(K):
        wlk.step()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    # the metric's literal scope: nf_project + nf_project_adjoint of every timed step (CUDA events, same stream)
    proj_total = sum(a.elapsed_time(b) + c.elapsed_time(d_) for a, b, c, d_ in wlk.proj_events)
    wlk.proj_events = None
    launches = g.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    ms_total = replicas.max_over_ranks(ms_total, dist, device="cuda")
    proj_total = replicas.max_over_ranks(proj_total, dist, device="cuda")
    ms_per_step = ms_total / K
    value = replicas.job_value_ms(proj_total, K, world)
    step_value = replicas.job_value_ms(ms_total, K, world)

    # ---- extra (untimed-for-the-headline) passes: projection share, iteration counts, per-kernel roofline ----
    nrec = min(K, 3)
    for _ in range(nrec):
        wlk.step(record=True)
    proj_ms = wlk.proj_ms / nrec
    g.profile_enable(True)
    wlk.step()
    prof = g.profile()
    g.profile_enable(False)
    ninfo = g.info()
    ncell = n ** 3
    peak, peak_src = _peaks()
    # algorithmic bytes per fine cell per launch (DESIGN.md section 8 / SURVEY.md 8d.2), fp32
    # fused p-update + A-apply + deferred x update: z, p, x, code in; p', q, x out = 25; fused r update + pre-smoother:
    # r, q, code in; r, z out = 17; the cooperative coarse kernel: every level below the finest one, 41 B per coarse cell
    # summed over the levels (1/8 + 1/64 + ...) = 41/7 B per FINE cell
    KNAME = {"apply_A": "k_papply4", "cg_update": "k_update_down1", "down1_fine": "k_down1", "down2_fine": "k_down2",
             "up1_fine": "k_up1", "up2_fine": "k_up2", "vec_coarse": "k_vcoarse"}
    kern = {}
    sweeps = g.sweeps()
    bytes_of = dict(BYTES)
    bytes_of["vec_coarse"] = coarse_bytes_per_fine_cell(sweeps[2], sweeps[3])
    for name, (ms, cnt) in prof.items():
        if cnt == 0:
            continue
        kk = {"ms_total": round(ms, 4), "launches": cnt, "us_per_launch": round(1e3 * ms / cnt, 2)}
        if name in bytes_of:
            kk["gbs"] = round(bytes_of[name] * ncell / (ms / cnt * 1e-3) / 1e9, 1)
            kk["frac_of_peak"] = round(kk["gbs"] / peak, 3)
        kern[name] = kk
    tot_ms = sum(v["ms_total"] for v in kern.values())
    # the dominant kernel = the largest share of the profiled step's device time, over ALL kernel classes
    dom = max(kern, key=lambda k: kern[k]["ms_total"])
    # dram bytes per launch from the committed ncu --set full capture of THIS build (profiles/, 256^3 only)
    traffic = None
    try:
        if n == 256:
            with open(os.path.join(ROOT, "profiles", "r2_traffic.json")) as f:
                traffic = json.load(f).get(KNAME.get(dom, ""))
    except Exception:
        traffic = None
    roof = {"bound": "hbm", "kernel": dom, "achieved": kern[dom].get("gbs"), "peak": peak, "unit": "GB/s",
            "frac": round(kern[dom]["gbs"] / peak, 4) if "gbs" in kern[dom] else None, "traffic": traffic,
            "peak_source": peak_src, "algorithmic_bytes_per_cell": round(bytes_of.get(dom, 0.0), 2),
            "cells_per_launch": ncell, "share_of_step": round(kern[dom]["ms_total"] / tot_ms, 3)}
    if "vec_coarse" in kern:
        # the cooperative coarse kernel works on L2-resident levels (ncu: ~25 MB of DRAM traffic per launch for 98 MB of
        # algorithmic bytes) behind 16 grid barriers: its HBM fraction measures latency, not bandwidth
        kern["vec_coarse"]["note"] = "latency-bound: grid barriers over L2-resident levels"
        if dom == "vec_coarse":
            roof["note"] = kern["vec_coarse"]["note"]
    # second-largest kernel, for context
    others = sorted((k for k in kern if k != dom), key=lambda k: -kern[k]["ms_total"])
    if others:
        o = others[0]
        roof["next_largest"] = {"kernel": o, "share_of_step": round(kern[o]["ms_total"] / tot_ms, 3),
                                "achieved": kern[o].get("gbs"), "frac": kern[o].get("frac_of_peak")}
    it_names = ["apply_A", "cg_update", "down2_fine", "vec_coarse", "up1_fine", "up2_fine"]
    if all(k_ in kern for k_ in it_names):
        it_us = sum(kern[k_]["us_per_launch"] for k_ in it_names)
        it_b = sum(bytes_of[k_] for k_ in it_names)
        roof["iteration"] = {"launches": len(it_names), "bytes_per_cell": round(it_b, 1), "us": round(it_us, 1),
                             "gbs": round(it_b * ncell / (it_us * 1e-6) / 1e9, 1),
                             "frac": round(it_b * ncell / (it_us * 1e-6) / 1e9 / peak, 3)}
    its = wlk.iters
    mcell_it = (ninfo["active_cells"] * sum(a + b for a, b in its) / len(its)) / (proj_ms * 1e-3) / 1e6

    # ---- e2e: host buffers through the C ABI, copies inside the timed region --------------------------------
    e2e = None
    if rank == 0 or world > 1:
        pin = lambda t_: t_.detach().cpu().pin_memory()
        hU = [pin(a) for a in wlk.U0]
        hG = [pin(a) for a in wlk.gin]
        hUw = [torch.empty_like(a).pin_memory() for a in hU]
        hGw = [torch.empty_like(a).pin_memory() for a in hG]
        hp = torch.empty(g.shape_p, dtype=torch.float32).pin_memory()
        hphi = pin(wlk.geom[0][0]); hus = [pin(a) for a in wlk.geom[0][1]]
        dphi = torch.empty_like(wlk.geom[0][0]); dus = [torch.empty_like(a) for a in wlk.geom[0][1]]

        def e2e_refresh():
            # harness work, NOT part of the user's step: nf_project_host / nf_project_adjoint_host work in place on
            # the host arrays, so the step's inputs are restored from a pristine copy before each timed step
            for a, b in zip(hUw, hU):
                a.copy_(b)
            for a, b in zip(hGw, hG):
                a.copy_(b)

        def e2e_step():
            dphi.copy_(hphi, non_blocking=True)
            for a, b in zip(dus, hus):
                a.copy_(b, non_blocking=True)
            g.set_solid(dphi, *dus)
            g.project_host(*hUw, hp, tol=TOL, maxit=MAXIT)
            g.project_adjoint_host(*hGw, tol=TOL, maxit=MAXIT)
            g.host_sync()                # (host-async mode: the D2H of the projection overlapped the adjoint)
            return float(hp[0, 0, 0])  # the step's result is read on the host

        ke = max(2, min(K, 5))
        g.set_host_async(True)
        e2e_refresh()
        e2e_step()
        dt_ms = 0.0
        for _ in range(ke):
            e2e_refresh()
            barrier()
            t0 = time.perf_counter()
            e2e_step()
            torch.cuda.synchronize()
            dt_ms += (time.perf_counter() - t0) * 1e3
        t = torch.tensor([dt_ms], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        h2d = sum(a.numel() for a in hU + hG + hus) * 4 + hphi.numel() * 4
        d2h = sum(a.numel() for a in hU + hG) * 4 + hp.numel() * 4
        e2e = {"value": round(float(t.item()) / (ke * world), 3), "unit": "ms", "h2d_bytes_per_step": h2d,
               "d2h_bytes_per_step": d2h, "steps": ke,
               "scope": "H2D(phi,u_s,Uhat,g) + nf_set_solid + nf_project_host + nf_project_adjoint_host + D2H(U,p,dJ/dUhat)"}

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(args.cpu_n)
    if rank == 0:
        line = {"metric": METRIC, "value": round(value, 3), "unit": "ms", "n_gpus": world, "steps": K, "warmup": W,
                "ms_per_step": round(ms_per_step, 3), "higher_is_better": False, "scaling": "weak",
                "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "value_scope": "nf_project + nf_project_adjoint (the metric's scope), summed over the K timed steps with "
                               "CUDA events and divided by K; ms_per_step / full_step_ms = the whole hot-path step",
                "full_step_ms": round(step_value, 3), "ns_per_cell": round(value * 1e6 / ncell, 4),
                "config": {"workload": "configs[3] channel-gate %d^3, 20-step geometry cycle; a step = advect, set_solid, "
                                       "project, project_adjoint, weights_adjoint, advect_adjoint" % n,
                           "grid": [n, n, n], "tol": TOL, "l2_policy": "inputs exceed L2 (>1 GB working set per step)",
                           "parallelism": "replicas x%d" % world, "levels": ninfo["levels"],
                           "sweeps_fine_l1_deeper": [sweeps[0], sweeps[2], sweeps[3]],
                           "x0": "previous pressure (forward solve)" if args.warm_start else "zero",
                           "active_cells": ninfo["active_cells"]},
                "projection_ms": round(proj_ms, 3), "iters_fwd_adj": its, "mcell_iters_per_s": round(mcell_it, 1),
                "gpu_launches": int(launches), "clocks": clocks, "e2e": e2e, "roofline": roof, "kernels": kern,
                "cpu_baseline": cpu,
                "paper_context": "RTX A6000 whole step (advect+viscosity+project) at 64^3: 0.105 s fwd / 0.117-0.301 s "
                                 "bwd (PAPER.md Tables 2-3); no projection-only number is published"}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# --------------------------------------------------------------------------------------------------------------
# the oracle, timed (cpu_baseline leg and --impl reference)
# --------------------------------------------------------------------------------------------------------------
def _oracle_case(n):
    """Inputs of the oracle legs: the channel-gate at n^3, face weights already built (the metric's scope is the two
    projections; nf_set_solid is outside `value` on the CUDA arm too)."""
    from oracle import nf_oracle as orc
    from paper_2405_14903_b200 import workloads as wl
    import numpy as np
    P = wl.config4_params(n)
    U = wl.config4_initial_velocity(P)
    phi, us = wl.config4_solid(P, 1)
    rng = np.random.default_rng(77)
    gin = [rng.standard_normal(a.shape).astype(np.float32) for a in U]
    bc = orc.BC(P["bc_types"], P["bc_values"])
    alpha = orc.face_weights(phi, bc)
    return P, U, alpha, us, gin, bc


def _oracle_step(case):
    """project + project_adjoint with the oracle as it stands, tol = 1e-6 (the metric's tolerance and scope)."""
    from oracle import nf_oracle as orc
    P, U, alpha, us, gin, bc = case
    Un, p = orc.project(U, alpha, us, P["dx"], P["dt_over_rho"], bc, tol=TOL)
    orc.project_adjoint(gin, alpha, p, U, us, P["dx"], P["dt_over_rho"], bc, tol=TOL)


def _threads_used():
    try:
        from threadpoolctl import threadpool_info
        return max([i.get("num_threads", 1) for i in threadpool_info()] + [1])
    except Exception:
        return 1


def _sample_text(n):
    return ("channel-gate shape at %d^3 (%.4f of the 256^3 cells of the metric's workload): fp64 NumPy Jacobi-PCG "
            "projection + adjoint projection, both to 1e-6 (the oracle as it stands)" % (n, (n / 256.0) ** 3))


def cpu_baseline(n):
    case = _oracle_case(n)
    t0 = time.perf_counter()
    _oracle_step(case)
    ms = (time.perf_counter() - t0) * 1e3
    return {"value": round(ms, 1), "unit": "ms", "cores": _threads_used(), "host_cores": os.cpu_count(),
            "kind": "oracle", "grid": [n, n, n], "ns_per_cell": round(ms * 1e6 / n ** 3, 2),
            "sample": _sample_text(n) + "; one pass; measured scaling of this oracle: time ~ n^4 (iterations ~ n), "
                      "BASELINE.md section 3"}


def run_reference(args):
    """The reference arm = the oracle (there is no reference code: /root/reference holds the paper only), same metric,
    unit and scope as the CUDA arm's `value`, on a bounded sample of the workload: the largest gate grid of
    {48, 64, 80, 96, 128} whose K + W steps fit ~4 minutes by the measured n^4 cost model (8 s at 64^3)."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return
    K, W = args.steps, args.warmup
    budget = 240.0 / max(K + W, 1)
    n = 48
    for cand in (64, 80, 96, 128):
        if 8.0 * (cand / 64.0) ** 4 <= budget:
            n = cand
    if args.cpu_n_forced:
        n = args.cpu_n
    case = _oracle_case(n)
    for _ in range(W):
        _oracle_step(case)
    t0 = time.perf_counter()
    for _ in range(K):
        _oracle_step(case)
    ms = (time.perf_counter() - t0) * 1e3 / K
    sample = _sample_text(n) + " per step"
    line = {"impl": "reference", "metric": METRIC, "value": round(ms, 1), "unit": "ms", "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": round(ms, 1), "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "value_scope": "oracle project + project_adjoint (the metric's scope) on a bounded sample: NOT the 256^3 "
                           "grid -- compare ns_per_cell, not value",
            "ns_per_cell": round(ms * 1e6 / n ** 3, 2),
            "config": {"workload": "configs[3] channel-gate, bounded sample %d^3 = %.4f of the metric's 256^3 cells"
                                   % (n, (n / 256.0) ** 3), "grid": [n, n, n], "tol": TOL},
            "cpu_baseline": {"value": round(ms, 1), "unit": "ms", "cores": _threads_used(),
                             "host_cores": os.cpu_count(), "kind": "oracle", "sample": sample},
            "e2e": {"value": round(ms, 1), "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def _apply_A_fp64(p, au, av, aw, c):
    """c G^T S G p in fp64 NumPy with homogeneous ghosts (acceptance check of the sweep; closed walls have alpha = 0)."""
    import numpy as np
    fu = np.zeros(au.shape); fv = np.zeros(av.shape); fw = np.zeros(aw.shape)
    fu[:, :, 1:-1] = au[:, :, 1:-1] * (p[:, :, 1:] - p[:, :, :-1])
    fu[:, :, 0] = au[:, :, 0] * p[:, :, 0]; fu[:, :, -1] = -au[:, :, -1] * p[:, :, -1]
    fv[:, 1:-1, :] = av[:, 1:-1, :] * (p[:, 1:, :] - p[:, :-1, :])
    fv[:, 0, :] = av[:, 0, :] * p[:, 0, :]; fv[:, -1, :] = -av[:, -1, :] * p[:, -1, :]
    fw[1:-1] = aw[1:-1] * (p[1:] - p[:-1])
    fw[0] = aw[0] * p[0]; fw[-1] = -aw[-1] * p[-1]
    return c * ((fu[:, :, :-1] - fu[:, :, 1:]) + (fv[:, :-1, :] - fv[:, 1:, :]) + (fw[:-1] - fw[1:]))


def run_sweep(args):
    """BASELINE.json configs[4]: MGPCG alone (nf_solve) on cubic all-Neumann grids with 200 random solid spheres
    (nf_set_solid alone, every fluid pocket kept), rhs N(0,1) with its mean removed on every pocket, tol 1e-6: iterations, ms, Mcell-iterations/s, and the fp64 true residual of the
    answer evaluated on the host (the oracle's operator, one pass; the oracle does not solve at these sizes)."""
    import numpy as np
    import torch
    from paper_2405_14903_b200 import api, workloads as wl
    api.load_library()
    torch.cuda.set_device(0)
    d = lambda a: torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    rows = []
    for n in [int(x) for x in args.sweep.split(",")]:
        phi = wl.config5_phi(n)
        g = api.Grid(n, n, n, 1.0 / n)
        g.set_solid(d(phi))           # nf_set_solid alone: the library finds the fluid pockets itself (R12)
        au, av, aw = [a.cpu().numpy() for a in g.get_weights()]
        labels, ncomp = wl.fluid_components(au, av, aw)
        active = labels > 0
        rhs = wl.config5_rhs_per_component(n, labels)
        ncomp_lib, nsing_lib = g.components()
        drhs = d(rhs)
        p = torch.empty(g.shape_p, dtype=torch.float32, device="cuda")
        for _ in range(3):
            rc = g.solve(drhs, p, tol=TOL, maxit=MAXIT)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 5
        e0.record()
        for _ in range(reps):
            rc = g.solve(drhs, p, tol=TOL, maxit=MAXIT)
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        info = g.last_solve_info()
        nact = int(active.sum())
        # per-kernel device time of one more solve (CUDA events around every launch) -> algorithmic GB/s per kernel
        g.profile_enable(True)
        g.solve(drhs, p, tol=TOL, maxit=MAXIT)
        prof = g.profile()
        g.profile_enable(False)
        per_kernel = {}
        sw = g.sweeps()
        bytes_of = dict(BYTES)
        bytes_of["vec_coarse"] = coarse_bytes_per_fine_cell(sw[2], sw[3])
        for name, (kms, cnt) in prof.items():
            if cnt and name in bytes_of:
                us = 1e3 * kms / cnt
                per_kernel[name] = {"us_per_launch": round(us, 2), "launches": cnt,
                                    "gbs": round(bytes_of[name] * n ** 3 / (us * 1e-6) / 1e9, 1)}
        res = rhs.astype(np.float64) - _apply_A_fp64(p.cpu().numpy().astype(np.float64), au, av, aw, float(n))
        res[~active] = 0.0
        rows.append({"n": n, "rc": int(rc), "iters": info["iters"], "ms": round(ms, 3), "active_cells": nact,
                     "fluid_components": int(ncomp), "components_found_by_library": [ncomp_lib, nsing_lib],
                     "levels": g.info()["levels"], "sweeps_fine_l1_deeper": [sw[0], sw[2], sw[3]],
                     "mcell_iters_per_s": round(nact * info["iters"] / (ms * 1e-3) / 1e6, 1),
                     "us_per_iter": round(1e3 * ms / max(info["iters"], 1), 1),
                     "recursive_relres": float(info["relres"]),
                     "true_relres_fp64": float(np.linalg.norm(res) / np.linalg.norm(rhs)),
                     "hbm_gbs_per_kernel": per_kernel})
        g.close()
        del p, drhs
        torch.cuda.empty_cache()
    print(json.dumps({"workload": "configs[4] pressure-solve sweep (200 random spheres, all-Neumann, rhs N(0,1))",
                      "tol": TOL, "dtype": "f32", "rows": rows}))


def run_geometry(args):
    """SURVEY.md 8f NEXT-2 at the headline grid size: a solid made of four polar-Bezier primitives (K = 4 key sections,
    N = 8 curves, M = 16 samples per curve: 128 polygon edges each; "union of four sub-geometries"),
    phi = union on the nodes, its reverse with dJ/dphi confined to the nodes next to the surface (what
    nf_weights_adjoint produces), and the solid velocity of one moving primitive with a band of 3 dx + its reverse.
    roofline: ALU-bound; one (node, edge) pair costs 19.25 SASS instructions in k_geom_sdf's scan loop (77 per 4 points,
    cuobjdump), so peak = 148 SMs x 128 lanes x SM clock / 19.25 pairs/s."""
    import numpy as np
    import torch
    from paper_2405_14903_b200 import api, workloads as wl
    api.load_library()
    torch.cuda.set_device(0)
    n, K, N, M = args.n, 4, 8, 16
    g = api.Grid(n, n, n, 1.0 / n)
    prims = [wl.geom_random_params(40 + i, K, N, 0.15 + 0.05 * i, 0.6 + 0.08 * i,
                                   (0.35 + 0.3 * (i % 2), 0.35 + 0.3 * (i // 2)), 0.17) for i in range(4)]
    phis = [torch.empty(g.shape_sdf, dtype=torch.float32, device="cuda") for _ in prims]
    acc = [torch.empty_like(phis[0]) for _ in range(3)]
    gacc = [torch.empty_like(phis[0]) for _ in range(8)]

    def forward():
        for p, f in zip(prims, phis):
            g.geom_sdf(p, K, N, M, f)
        g.geom_csg("union", phis[0], phis[1], acc[0])
        g.geom_csg("union", acc[0], phis[2], acc[1])
        g.geom_csg("union", acc[1], phis[3], acc[2])

    forward()
    gphi = torch.where(acc[2].abs() < 2.0 / n, torch.randn_like(acc[2]), torch.zeros_like(acc[2]))

    def backward():
        g.geom_csg_adjoint("union", acc[1], phis[3], gphi, gacc[0], gacc[1])
        g.geom_csg_adjoint("union", acc[0], phis[2], gacc[0], gacc[2], gacc[3])
        g.geom_csg_adjoint("union", phis[0], phis[1], gacc[2], gacc[4], gacc[5])
        return [g.geom_sdf_adjoint(p, K, N, M, gg) for p, gg in zip(prims, (gacc[4], gacc[5], gacc[3], gacc[1]))]

    pd = wl.geom_random_rates(3, K, N, 0.1)
    U = [torch.zeros(s, dtype=torch.float32, device="cuda") for s in (g.shape_u, g.shape_v, g.shape_w)]
    gU = [torch.randn_like(a) for a in U]
    legs = {"sdf_union_of_4": forward, "sdf_adjoint_4": backward,
            "velocity_1": lambda: g.geom_velocity(prims[0], pd, K, N, M, *U, band=3.0 / n),
            "velocity_adjoint_1": lambda: g.geom_velocity_adjoint(prims[0], K, N, M, *gU, band=3.0 / n)}
    clocks = ClockSampler(0)
    clocks.start()
    out = {}
    for name, fn in legs.items():
        for _ in range(max(args.warmup, 3)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        out[name] = round(e0.elapsed_time(e1) / args.steps, 4)
    ck = clocks.stop()
    # the dominant kernel alone
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        g.geom_sdf(prims[0], K, N, M, phis[0])
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    pairs = float((n + 1) ** 3) * N * M
    mhz = ck.get("sm_mhz") or 1900.0
    peak = 148 * 128 * mhz * 1e6 / 19.25
    traffic = None
    try:
        with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "r1_geom_traffic.json")) as f:
            traffic = float(json.load(f)["k_geom_sdf"]["traffic"])
    except Exception:
        pass
    print(json.dumps({"workload": "NEXT-2 parametric geometry, %d^3 grid, 4 primitives x (K=4, N=8, M=16)" % n,
                      "dtype": "f32", "ms": out, "clocks": ck,
                      "roofline": {"kernel": "k_geom_sdf", "bound": "alu", "achieved": round(pairs / (ms * 1e-3) / 1e9, 1),
                                   "peak": round(peak / 1e9, 1), "unit": "G(node,edge)/s",
                                   "frac": round(pairs / (ms * 1e-3) / peak, 3), "ms_per_launch": round(ms, 4),
                                   "frac_meaning": "issue efficiency: the peak is derived from THIS kernel's own "
                                                   "19.25 SASS instructions per (node, edge) pair, not from an "
                                                   "algorithmic flop count",
                                   "traffic": traffic}}))


def run_envs(args):
    """E concurrent small environments (paper_2405_14903_b200/envs.py: one handle, stream and host
    thread each) -- aggregate forward + adjoint projection steps per second at the paper's task sizes (PAPER.md:L151-160:
    40^3-48^3), a step = nf_set_solid + nf_project + nf_project_adjoint to 1e-6 on a sphere-in-channel grid."""
    import time
    import numpy as np
    import torch
    from paper_2405_14903_b200 import api, envs, workloads as wl
    api.load_library()
    torch.cuda.set_device(0)
    n = args.n
    i, j, k = wl.node_coords(n, n, n)
    phi = torch.from_numpy(wl.sdf_sphere(i, j, k, (n / 2 + 0.3, n / 2 - 0.2, n / 2 + 0.1), n / 5).astype(np.float32)).cuda()
    rows = []
    for E in [int(x) for x in args.envs.split(",")]:
        pool = envs.EnvPool(E, n, n, n, 1.0 / n)
        for g in pool.grids:
            g.set_domain_bc(0, 1, 1.0)
            g.set_domain_bc(1, 1, 0.0)
        rng = np.random.default_rng(1)
        U0 = [[torch.from_numpy((0.3 * rng.standard_normal(s)).astype(np.float32)).cuda() for s in wl.face_shapes(n, n, n)]
              for _ in range(E)]
        torch.cuda.synchronize()

        def work(reps):
            def fn(e, g):
                p = torch.empty(g.shape_p, dtype=torch.float32, device="cuda")
                its = 0
                for _ in range(reps):
                    V = [a.clone() for a in U0[e]]
                    g.set_solid(phi)
                    g.project(*V, p, tol=TOL, maxit=MAXIT)
                    its += g.last_solve_info()["iters"]
                    g.project_adjoint(*V, p_saved=p, uhat=U0[e], tol=TOL, maxit=MAXIT)
                    its += g.last_solve_info()["iters"]
                torch.cuda.current_stream().synchronize()
                return its
            return fn
        pool.run(work(max(args.warmup, 3)))
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        its = pool.run(work(args.steps))
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        rows.append({"mode": "threads (one handle + stream + host thread per environment)", "envs": E,
                     "env_steps_per_s": round(E * args.steps / dt, 1),
                     "ms_per_env_step": round(1e3 * dt / args.steps, 3),
                     "iters_per_solve": round(sum(its) / (2.0 * E * args.steps), 1)})
        pool.close()
        # the same work through the batched entry points: ONE host thread, one launch per solver pass for all E
        grids = [api.Grid(n, n, n, 1.0 / n) for _ in range(E)]
        for g in grids:
            g.set_domain_bc(0, 1, 1.0)
            g.set_domain_bc(1, 1, 0.0)
        ps = [torch.zeros(g.shape_p, dtype=torch.float32, device="cuda") for g in grids]
        ys = [torch.zeros(g.shape_p, dtype=torch.float32, device="cuda") for g in grids]

        def batched(reps, lo=0, hi=None):
            hi = E if hi is None else hi
            gg, its = grids[lo:hi], 0
            for _ in range(reps):
                V = [[a.clone() for a in U0[e]] for e in range(lo, hi)]
                for g in gg:
                    g.set_solid(phi)
                api.project_batch(gg, V, ps[lo:hi], tol=TOL, maxit=MAXIT)
                its += sum(g.last_solve_info()["iters"] for g in gg)
                api.project_adjoint_batch(gg, V, ys[lo:hi], p_saved=ps[lo:hi], uhat=U0[lo:hi], tol=TOL, maxit=MAXIT)
                its += sum(g.last_solve_info()["iters"] for g in gg)
            torch.cuda.current_stream().synchronize()
            return its
        batched(max(args.warmup, 3))
        l0 = sum(g.launch_count() for g in grids)
        t0 = time.perf_counter()
        its = batched(args.steps)
        dt = time.perf_counter() - t0
        rows.append({"mode": "batched (nf_project_batch / nf_project_adjoint_batch, one host thread)", "envs": E,
                     "env_steps_per_s": round(E * args.steps / dt, 1),
                     "ms_per_env_step": round(1e3 * dt / args.steps, 3),
                     "iters_per_solve": round(its / (2.0 * E * args.steps), 1),
                     "launches_per_env_step": round((sum(g.launch_count() for g in grids) - l0) / (E * args.steps), 1)})
        # groups of batched environments on their own streams / host threads: one group's nf_set_solid passes overlap
        # another group's solver passes
        for per in (2, 4, 8):
            if E < 2 * per:
                continue
            import threading
            T = E // per
            streams = [torch.cuda.Stream() for _ in range(T)]

            def grouped(reps):
                out = [0] * T

                def work(t):
                    with torch.cuda.stream(streams[t]):
                        out[t] = batched(reps, t * per, (t + 1) * per)
                th = [threading.Thread(target=work, args=(t,)) for t in range(T)]
                for x in th:
                    x.start()
                for x in th:
                    x.join()
                return sum(out)
            torch.cuda.synchronize()
            grouped(max(args.warmup, 3))
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            its = grouped(args.steps)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            rows.append({"mode": "batched groups of %d, one stream + host thread per group" % per, "envs": T * per,
                         "env_steps_per_s": round(T * per * args.steps / dt, 1),
                         "ms_per_env_step": round(1e3 * dt / args.steps, 3),
                         "iters_per_solve": round(its / (2.0 * T * per * args.steps), 1)})
        for g in grids:
            g.close()
    print(json.dumps({"workload": "NEXT-4 concurrent environments, %d^3 sphere-in-channel, forward + adjoint projection "
                                  "to %g (wall clock over all environments, host threads included)" % (n, TOL),
                      "dtype": "f32", "rows": rows}))


def run_config(args):
    """BASELINE.json configs[1] / configs[2] at their stated size and length through the C ABI (rollout.py sequences the
    calls): 64^3 x 10 full steps with two oscillating plates, gradient of the centre-block loss w.r.t. the plate
    amplitude; 128^3 x 50 steps of the chamber pump (static chamber, 16 Gaussian wall bumps modulated by sin(2 pi t/50),
    Dirichlet outlet), loss 1/2 sum u^2 on the outlet faces, gradient w.r.t. the 16 amplitudes, with the per-step state
    (U^n, Uhat, p: "checkpointed pressures") kept on the device.  Reports ms per step (forward + backward), the PCG
    iterations per step and the bytes of the tape."""
    import numpy as np
    import torch
    from paper_2405_14903_b200 import api, rollout as ro, workloads as wl
    api.load_library()
    torch.cuda.set_device(0)
    d = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).cuda()
    cfg = args.config
    if cfg == 2:
        n = args.n if args.n_forced else 64
        P = wl.config2_params(n)
        nsteps = P["steps"]
        geom = {}
        for st in range(1, nsteps + 1):
            v = wl.config2_solid(P, st, P["theta"])
            geom[st] = (d(v[0]), [d(a) for a in v[1]], d(v[2]), [d(a) for a in v[3]])
        solid = lambda st: geom[st]
        lo, hi = P["loss_lo"], P["loss_hi"]

        def loss(U):
            blk = U[0][lo:hi, lo:hi, lo:hi].double()
            G = [torch.zeros_like(a) for a in U]
            G[0][lo:hi, lo:hi, lo:hi] = (2.0 * blk).float()
            return (blk * blk).sum(), G
        name = "configs[1] two oscillating plates %d^3 x %d steps, dJ/d(amplitude)" % (n, nsteps)
    else:
        n = args.n if args.n_forced else 128
        P = wl.config3_params(n)
        nsteps = P["steps"]
        phi, us1 = wl.config3_solid(P, P["period"] / 4.0)              # modulation sin(pi/2) = 1: the unit wall field
        dphi_ = d(phi)
        unit = [d(a) for a in us1]
        basis = [[d(a) for a in wl.config3_us_basis(P, P["period"] / 4.0, k)] for k in range(16)]

        def solid(st):
            mod = float(np.sin(2 * np.pi * st / P["period"]))
            return dphi_, [mod * a for a in unit], None, {"basis": basis, "scale": mod}

        def loss(U):
            G = [torch.zeros_like(a) for a in U]
            out = U[0][:, :, -1].double()
            G[0][:, :, -1] = out.float()
            return 0.5 * (out * out).sum(), G
        name = "configs[2] chamber pump %d^3 x %d steps, dJ/d(16 bump amplitudes)" % (n, nsteps)
    g = api.Grid(n, n, n, P["dx"])
    g.set_dt_rho(P["dt_over_rho"])
    for f in range(6):
        g.set_domain_bc(f, P["bc_types"][f], P["bc_values"][f])
    U0 = [torch.zeros(sh, dtype=torch.float32, device="cuda") for sh in (g.shape_u, g.shape_v, g.shape_w)]
    run = lambda stats=None: ro.rollout(g, U0, solid, nsteps, P["dt"], loss, tol=TOL, maxit=MAXIT, stats=stats)
    for _ in range(max(1, min(args.warmup, 2))):
        run()
    torch.cuda.synchronize()
    reps = max(1, min(args.steps, 3))
    l0 = g.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.reset_peak_memory_stats()
    e0.record()
    for _ in range(reps):
        J, dJ, _ = run()
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / reps
    launches = (g.launch_count() - l0) // reps
    stats = {}
    run(stats)
    print(json.dumps({"workload": name, "dtype": "f32", "tol": TOL, "grid": [n, n, n], "steps": nsteps,
                      "ms_total_fwd_bwd": round(ms, 3), "ms_per_step_fwd_bwd": round(ms / nsteps, 3),
                      "iters_fwd_mean": round(float(np.mean(stats["iters_fwd"])), 1),
                      "iters_adj_mean": round(float(np.mean(stats["iters_adj"])), 1),
                      "iters_fwd_max": int(max(stats["iters_fwd"])), "iters_adj_max": int(max(stats["iters_adj"])),
                      "tape_bytes": ro.tape_bytes(g, nsteps),
                      "torch_peak_bytes": int(torch.cuda.max_memory_allocated()),
                      "gpu_launches_per_rollout": int(launches), "loss": J,
                      "dJ_dtheta": dJ if isinstance(dJ, list) else [dJ],
                      "paper_context": "RTX A6000, whole step at 64^3: 0.105 s forward / 0.117-0.301 s backward "
                                       "(PAPER.md Tables 2-3); memory 405 MB at 64^3 (Table 3)"}))


def run_karman(args):
    """the paper's 2-D validation case (appendix D: flow past a cylinder on a
    512 x 1024 grid with viscosity) as a timing workload -- nz = 1 grid of 1024 x 512 cells, inflow p = 1 / outflow p = 0,
    a cylinder of radius 40 cells, nu = 0.01; a step = nf_advect + nf_viscosity + nf_project (the solid is static)."""
    import numpy as np
    import torch
    from paper_2405_14903_b200 import api, workloads as wl
    api.load_library()
    torch.cuda.set_device(0)
    nx, ny = 1024, 512
    dx = 1.0 / ny
    g = api.Grid(nx, ny, 1, dx)
    g.set_domain_bc(0, 1, 1.0)
    g.set_domain_bc(1, 1, 0.0)
    i, j, k = wl.node_coords(nx, ny, 1)
    phi = (np.sqrt((i - 256.3) ** 2 + (j - 255.7) ** 2) - 40.0 + 0 * k).astype(np.float32)
    g.set_solid(torch.from_numpy(np.ascontiguousarray(phi)).cuda())
    rng = np.random.default_rng(0)
    U = [torch.from_numpy(((1.0 if c == 0 else 0.0) + 0.05 * rng.standard_normal(s)).astype(np.float32)).cuda()
         for c, s in enumerate(wl.face_shapes(nx, ny, 1))]
    p = torch.empty(g.shape_p, dtype=torch.float32, device="cuda")
    dt, nu = 0.5 * dx, 0.01
    its, pms = [], []

    def step():
        g.advect(*U, dt)
        g.viscosity(*U, nu, dt)
        g.project(*U, p, tol=TOL, maxit=MAXIT)
        info = g.last_solve_info()
        its.append(info["iters"])
        pms.append(info["ms"])
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    del its[:], pms[:]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    torch.cuda.synchronize()
    print(json.dumps({"workload": "NEXT-3 2-D mode: cylinder in a 1024 x 512 channel, advect + viscosity + projection to %g" % TOL,
                      "dtype": "f32", "ms_per_step": round(e0.elapsed_time(e1) / args.steps, 3),
                      "solve_ms": round(sum(pms) / len(pms), 3), "iters_per_solve": round(sum(its) / len(its), 1),
                      "levels": g.info()["levels"], "active_cells": g.info()["active_cells"]}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=256, help="grid size (the metric is quoted at 256)")
    ap.add_argument("--cpu-n", type=int, default=0,
                    help="grid size of the cpu_baseline sample (default 96: ~30-40 s of oracle time) / of --impl reference")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--warm-start", action="store_true",
                    help="nf_project starts from the previous step's pressure (default: x0 = 0, as BASELINE's metric)")
    ap.add_argument("--sweep", default="", help="comma-separated cubic sizes: run the configs[4] pressure-solve sweep "
                                                 "instead of the headline step, e.g. --sweep 64,128,256,384")
    ap.add_argument("--geometry", action="store_true",
                    help="time the NEXT-2 parametric-geometry kernels at --n instead of the headline step")
    ap.add_argument("--envs", default="", help="comma-separated environment counts: aggregate throughput of concurrent "
                                                "small grids of size --n (e.g. --envs 1,4,8 --n 48) instead of the headline step")
    ap.add_argument("--karman", action="store_true", help="time the 2-D cylinder-in-channel case (1024 x 512, nz = 1)")
    ap.add_argument("--config", type=int, default=0, choices=[0, 2, 3],
                    help="2: BASELINE configs[1] (64^3 x 10 steps fwd + backprop); 3: configs[2] (128^3 x 50 steps chamber pump)")
    args = ap.parse_args()
    args.n_forced = "--n" in sys.argv
    args.cpu_n_forced = args.cpu_n > 0
    if not args.cpu_n_forced:
        args.cpu_n = 96
    if args.config:
        run_config(args)
        return
    if args.karman:
        run_karman(args)
        return
    if args.envs:
        run_envs(args)
        return
    if args.sweep:
        run_sweep(args)
        return
    if args.geometry:
        run_geometry(args)
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
