#!/usr/bin/env python
"""bench.py -- decays/s of the whole hot path on the synthetic patient phantom (BASELINE.json cfg3).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--decays D] [--impl reference]

One step = one anm_run of D decays (default 1e9, the north-star target) on cfg3 (256x256x400 voxels of
2x2x4 mm, 27 organs, pairs of 0.511 MeV photons + 0.2498 MeV positron energy, 100 batches): source sampling,
Woodcock transport, tally, 100 batch folds with organ reduction, finalize -- every SURVEY.md §8(a) row.
`value` times K such runs with all inputs resident in HBM (CUDA events on the launching stream, max over ranks);
`e2e` times the same job through the C ABI from HOST buffers (phantom / activity / label upload, set-up, run,
dose + uncertainty + organ read-back to the host).  `roofline` is the ALU/issue roofline of the transport kernel
(DESIGN.md §6); `cpu_baseline` is the oracle timed on this box's host cores on a bounded sample.
With --impl reference the oracle itself is the timed arm (same metric / config, bounded sample per step).
Under torchrun (N > 1) the step is ONE logical run of N*D decays in N*100 batches: each rank simulates its own
whole-batch shard (history_offset = rank*D, no collective during transport) and the step ends with the merge of
the tallies (paper_2111_11687_b200.multi_gpu.run_sharded: in-place NCCL sum-all-reduce of the sum / sum-of-squares
volumes + organ rows, finalize on the merged volumes); per-GPU work is fixed, scaling = weak.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

WORKLOAD = "cfg3_patient 256x256x400 @2x2x4mm, 27 organs, pairs+positron KE, 100 batches"

# DESIGN.md §5.1 / §6: algorithmic thread-instructions per unit of the method = the SASS instructions the per-event device
# functions execute per lane, counted from the ncu source page of the transport kernel (profiles/r2_event_instr.md has the
# command, the per-region table and how each constant is put together); the event pool's scheduling (ring push / pick /
# pop), the slot loads / stores and the speculative half of a FLY event are NOT in them.  Multiplied by the units per
# decay a counted run of the same workload measures (anm_stats: n_steps, n_compton_tries, n_compton, ...).
INSTR_PHILOX = 46.2          # one Philox4x32-10 block (20 IMAD.WIDE + 20 LOP3 + counter set-up)
INSTR_U01 = 3.2              # one uniform (SHF + I2F + FFMA)
INSTR_SUBSTEP = 101.0        # half a block (23.1) + 2 uniforms (6.4) + fly_land (38.0) + half of fly_two (30.0) + texel load (3.5)
INSTR_COMPTON_TRY = 86.8     # block + 3 uniforms (9.6) + compton_try (31.0)
INSTR_COMPTON_ACCEPT = 51.2  # azimuth uniform (3.2) + rotate (35.0) + energy split, cutoff test, log, grid coordinate (13)
INSTR_RAYLEIGH_TRY = 291.0   # block + 2 uniforms + rayleigh_try (238: two bisections of the 256-point form-factor table)
INSTR_RAYLEIGH_ACCEPT = 44.0 # azimuth uniform + rotate + grid coordinate
INSTR_DEPOSIT = 9.7          # address of the decay's batch tally + fp32 RED (Compton, photoelectric, positron)
INSTR_SOURCE = 208.0         # 2 blocks (92.4) + 6 uniforms (19.2) + sample_source (86.0: alias bucket, voxel -> (ix, iy, iz), position,
                             # direction) + hull test (11.0)
LANES_PER_SM_PER_CLK = 128.0   # 4 SMSP x 32 lanes, one instruction per SMSP per clock
N_SM = 148


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self) -> dict:
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm = sorted(float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit())
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for i, n in enumerate(names) if any(len(r) > 3 + i and r[3 + i].lower().startswith("active") for r in self.rows)]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx[0] if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def run_reference(args, rank: int):
    """The oracle as the timed arm: cfg3, each step a bounded sample of the workload on the host cores."""
    if rank != 0:
        return
    import anm_inputs
    from oracle import anm_oracle
    cores = os.cpu_count() or 1
    cfg = anm_inputs.make_config(3)
    tables = anm_inputs.make_tables()
    n = cores * args.ref_decays_per_core
    o = anm_oracle.Oracle(cfg, tables, n_decays=n, n_batches=cores, seed=1042)
    for _ in range(args.warmup):
        o.run_parallel(cores)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.run_parallel(cores)
    dt = time.perf_counter() - t0
    val = n * args.steps / dt
    sample = "%d decays per step (%d per core) of cfg3, %d single-threaded processes, one batch each" % (n, args.ref_decays_per_core, cores)
    print(json.dumps({
        "impl": "reference", "metric": "decays/s (18F, patient phantom)", "value": val, "unit": "decays/s",
        "sec_per_1e9_decays": 1e9 / val, "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic", "config": {"workload": WORKLOAD, "decays_per_step": n, "sample": sample},
        "cpu_baseline": {"value": val, "unit": "decays/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": "decays/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--decays", type=float, default=1e9, help="decays per step per GPU")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-decays-per-core", type=int, default=400_000)
    ap.add_argument("--cpu-baseline-decays-per-core", type=int, default=400_000)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--config", type=int, default=3, choices=[3, 4],
                    help="BASELINE.json config to run: 3 = the bench workload (default); 4 = the 512x512x600 scale case, "
                         "for profiling only (use with --no-frontend --no-variants; its line is not a bench number; the "
                         "default run reports cfg4 under variants.cfg4_fullres)")
    ap.add_argument("--no-peaks", action="store_true", help="skip the roofline microbenchmarks (anm_measure_peaks)")
    ap.add_argument("--no-cfg4", action="store_true", help="skip the cfg4 scale case in variants")
    ap.add_argument("--no-frontend", action="store_true", help="skip the image front-end timing (anm_load_ct / anm_load_pet)")
    ap.add_argument("--no-variants", action="store_true", help="skip the electron-transport / history-by-history runs")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, rank)

    import numpy as np
    import torch
    import anm_inputs
    from paper_2111_11687_b200 import Simulation

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    dev = torch.device("cuda", local_rank)
    torch.cuda.set_device(dev)

    cfg = anm_inputs.make_config(args.config)
    tables = anm_inputs.make_tables()
    D = int(args.decays)
    B = cfg["n_batches"]
    V = int(np.prod(cfg["shape"]))
    phys = dict(photons_per_decay=2, rayleigh_on=1, photon_cutoff_MeV=0.010, positron_ke_MeV=cfg["positron_ke_mev"])
    opts = dict(n_batches=B, history_offset=rank * D, **phys)
    if world > 1:
        from paper_2111_11687_b200.multi_gpu import run_sharded

    def step(s):
        if world > 1:
            run_sharded(s, world * D, cfg["seed"], world * B, phys)      # this rank's shard + the NCCL merge
        else:
            s.run(D, cfg["seed"])

    # ---- device-resident arm ----------------------------------------------------------------------------
    stream = torch.cuda.Stream(device=dev)
    mat = torch.from_numpy(cfg["material"]).to(dev)
    rho = torch.from_numpy(cfg["density"]).to(dev)
    act = torch.from_numpy(cfg["activity"]).to(dev)
    lab = torch.from_numpy(cfg["labels"]).to(dev)
    sim = Simulation(local_rank)
    peaks_dev = None
    with torch.cuda.stream(stream):
        sim.set_stream(stream)
        if not args.no_peaks:
            # roofline microbenchmarks of THIS device: before the warm-up steps, so that the clock
            # the power-limited issue stream pulls down has recovered when the timed region starts
            peaks_dev = sim.measure_peaks(104_857_600, 629_145_600)
        sim.set_grid(cfg["shape"], cfg["spacing_mm"])
        sim.load_phantom(mat, rho)
        sim.load_activity(act)
        sim.load_organs(lab, cfg["n_organs"])
        sim.set_physics_tables(tables)
        # events per decay (properties of the method + majorant), from a short counted run
        sim.set_options(collect_stats=1, **opts)
        n_cnt = B * 100_000
        sim.run(n_cnt, cfg["seed"])
        cnt = sim.get_stats()
        per_decay = {k: cnt[k] / n_cnt for k in ("n_steps", "n_real", "n_pe", "n_compton", "n_rayleigh", "n_fly_trips",
                                                 "n_compton_tries", "n_rayleigh_tries")}
        sim.set_options(collect_stats=0, **opts)
        for _ in range(args.warmup):
            step(sim)
        if dist:
            dist.barrier()
        torch.cuda.synchronize(dev)
        clocks = ClockSampler(local_rank)
        clocks.start()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ms_t = ms_f = ms_fin = 0.0
        launches = 0
        e0.record(stream)
        for _ in range(args.steps):
            step(sim)
            st = sim.get_stats()
            ms_t += st["ms_transport"]; ms_f += st["ms_fold"]; ms_fin += st["ms_finalize"]
            launches += st["n_launches"]
        e1.record(stream)
        torch.cuda.synchronize(dev)
        if dist:
            dist.barrier()
        clk = clocks.stop()
    ms_total = e0.elapsed_time(e1)
    if dist:
        t = torch.tensor([ms_total], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    value = world * D * args.steps / (ms_total * 1e-3)

    # ---- roofline of the dominant kernel (transport), DESIGN.md §5.1 / §6 ------------------------------------------
    # Four resources, each with its algorithmic demand per decay and a MEASURED denominator:
    #   alu        thread-instructions of the method's arithmetic  vs  the issue rate of a dependency-free FFMA + LOP3
    #              stream (anm_measure_peaks), per clock, at the SM clock this run held
    #   l2_gather  one random 4-byte texel read per Woodcock sub-step  vs  random ld.global.nc over a 105 MB array
    #   red        one fp32 RED per deposit (Compton, photoelectric, positron)  vs  random RED.ADD over a 105 MB array
    #   hbm        algorithmic bytes (4 B texel, 8 B tally RMW, 16 B alias entry)  vs  MEASURED_PEAKS.json hbm_gbs
    # (cfg4 uses the 630 MB figures.)  The binding one is named by ncu (issue-slot utilisation vs L2 / DRAM throughput,
    # profiles/): the ALU / issue side on cfg3; `bound`, `achieved`, `peak`, `frac` repeat that entry.
    deposits = per_decay["n_compton"] + per_decay["n_pe"] + (1.0 if cfg["positron_ke_mev"] > 0 else 0.0)
    instr_per_decay = (per_decay["n_steps"] * INSTR_SUBSTEP + per_decay["n_compton_tries"] * INSTR_COMPTON_TRY +
                       per_decay["n_compton"] * INSTR_COMPTON_ACCEPT + per_decay["n_rayleigh_tries"] * INSTR_RAYLEIGH_TRY +
                       per_decay["n_rayleigh"] * INSTR_RAYLEIGH_ACCEPT + deposits * INSTR_DEPOSIT + INSTR_SOURCE)
    # One step = n_groups transport launches (anm_options.batches_per_launch: G batches per launch) + B folds + finalize.
    # With the launch pipeline ms_transport is the pipeline's wall time, folds included (conservative for `achieved`).
    G = int(st["batches_per_launch"])
    n_groups = (B + G - 1) // G
    launches_transport = n_groups * args.steps
    sec_per_launch = ms_t * 1e-3 / launches_transport
    decays_per_s_kernel = (D / n_groups) / sec_per_launch
    achieved = instr_per_decay * decays_per_s_kernel / 1e9                          # G thread-instr / s
    sm_max = clk.get("sm_max_mhz") or 1965.0
    sm_run = clk.get("sm_mhz") or sm_max
    nominal = N_SM * LANES_PER_SM_PER_CLK * sm_max * 1e6 / 1e9
    file_peaks = {}
    try:
        file_peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak = float(file_peaks.get("hbm_gbs", 6500.0))
    big = args.config == 4
    alg_bytes = 4.0 * per_decay["n_steps"] + 8.0 * deposits + 16.0
    if peaks_dev:
        slots_per_clk = peaks_dev["issue_gtis"] * 1e9 / (N_SM * LANES_PER_SM_PER_CLK * peaks_dev["issue_sm_mhz"] * 1e6)
        peak = slots_per_clk * N_SM * LANES_PER_SM_PER_CLK * sm_run * 1e6 / 1e9
        peak_source = ("anm_measure_peaks: %.1f Gthread-instr/s at %.0f MHz (power-limited) = %.3f of the issue slots per clock, "
                       "x 148 SM x 128 lanes x %.0f MHz held during the timed region" % (peaks_dev["issue_gtis"], peaks_dev["issue_sm_mhz"], slots_per_clk, sm_run))
        g_peak, r_peak = peaks_dev["gather_gps"][1 if big else 0], peaks_dev["red_gps"][1 if big else 0]
        m_peak = peaks_dev["mix_gps"][1 if big else 0]
    else:
        m_peak = None
        peak, peak_source = nominal, "nominal 148 SM x 4 SMSP x 32 lanes x %.0f MHz (clocks.max.sm); --no-peaks" % sm_max
        g_peak = r_peak = None
    g_ach = per_decay["n_steps"] * decays_per_s_kernel / 1e9
    r_ach = deposits * decays_per_s_kernel / 1e9
    h_ach = alg_bytes * decays_per_s_kernel / 1e9
    traffic, traffic_source = None, None   # dram__bytes_read.sum + dram__bytes_write.sum per launch, from the committed ncu capture
    instr_executed, instr_executed_source = None, None   # thread-instructions the kernel EXECUTES per decay, same capture
    tdir = os.path.join(ROOT, "profiles")
    for name in sorted(os.listdir(tdir) if os.path.isdir(tdir) else [], reverse=True):
        if name.endswith("_transport_traffic.csv"):
            import csv
            rows = list(csv.DictReader(open(os.path.join(tdir, name))))
            if rows and int(rows[-1]["decays_per_launch"]) == D // n_groups and args.config == 3:
                traffic = int(rows[-1]["dram_bytes_read"]) + int(rows[-1]["dram_bytes_write"])
                traffic_source = "profiles/%s (ncu --set full capture of this kernel and launch size; not measured in this run)" % name
                if rows[-1].get("warp_instr_executed") and rows[-1].get("lanes_per_warp_instr"):
                    # smsp__inst_executed.sum x smsp__thread_inst_executed_per_inst_executed.ratio / decays of the launch
                    instr_executed = float(rows[-1]["warp_instr_executed"]) * float(rows[-1]["lanes_per_warp_instr"]) / float(rows[-1]["decays_per_launch"])
                    instr_executed_source = "profiles/%s (same capture; goes stale with the next kernel edit until re-captured)" % name
            break
    roofline = {"bound": "alu", "kernel": "transport_pool_kernel", "achieved": achieved, "peak": peak, "unit": "Gthread-instr/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_source, "peak_source": peak_source,
                "alu": {"achieved": achieved, "peak": peak, "frac": achieved / peak, "unit": "Gthread-instr/s",
                        "numerator": "SASS-issued work: this build's instruction counts of the per-event device functions x the events a "
                                     "counted run measures (profiles/r2_event_instr.md) -- not a count derived from the method alone, so "
                                     "compare rounds on decays/s and on instr_per_decay_executed, not on this fraction",
                        "peak_nominal": nominal, "frac_nominal": achieved / nominal,
                        "peak_power_limited": peaks_dev["issue_gtis"] if peaks_dev else None},
                "l2_gather": {"achieved": g_ach, "peak": g_peak, "frac": g_ach / g_peak if g_peak else None, "unit": "G loads/s",
                              "array_bytes": peaks_dev["bytes"][1 if big else 0] if peaks_dev else None},
                "red": {"achieved": r_ach, "peak": r_peak, "frac": r_ach / r_peak if r_peak else None, "unit": "G atomics/s"},
                # both streams at once (loads 5 : REDs 2, UNIFORMLY random over two arrays of the volume's size).  A reference
                # point, not a ceiling: two 105 MB arrays no longer fit the L2 together, whereas the transport's accesses
                # are concentrated on the body (its hot part does fit), so the kernel can exceed it -- ratio > 1 measures
                # that locality.  The separate gather / red fractions share the L2 and the HBM and must not be added up.
                "mem_mix_uniform": {"achieved": g_ach + r_ach, "reference": m_peak, "ratio": (g_ach + r_ach) / m_peak if m_peak else None,
                                    "unit": "G accesses/s (texel loads + tally REDs)",
                                    "note": "uniform-random reference over 2 arrays, not a peak: the kernel's accesses have locality"},
                "hbm": {"achieved": h_ach, "peak": hbm_peak, "frac": h_ach / hbm_peak, "unit": "GB/s",
                        "peak_source": "MEASURED_PEAKS.json hbm_gbs" if file_peaks else "fallback 6500 GB/s"},
                "peaks_measured": peaks_dev,
                "instr_per_decay_algorithmic": instr_per_decay, "instr_per_decay_executed": instr_executed,
                "instr_per_decay_executed_source": instr_executed_source, "events_per_decay": per_decay,
                "avg_launch_ms": sec_per_launch * 1e3, "batches_per_launch": G, "transport_launches_per_step": n_groups,
                "decays_per_launch": D // n_groups, "share_of_step": ms_t / max(ms_t + ms_f + ms_fin, 1e-9),
                "texel_bytes_per_decay": 4.0 * per_decay["n_steps"], "tally_bytes_per_decay": 8.0 * deposits,
                "algorithmic_bytes_per_decay": alg_bytes}

    # ---- end to end through the C ABI from host buffers ----------------------------------------------------
    e2e = None
    if not args.no_e2e:
        hm, hr = torch.from_numpy(cfg["material"]).pin_memory(), torch.from_numpy(cfg["density"]).pin_memory()
        ha, hl = torch.from_numpy(cfg["activity"]).pin_memory(), torch.from_numpy(cfg["labels"]).pin_memory()
        out_d, out_u = torch.empty(V, dtype=torch.float32).pin_memory(), torch.empty(V, dtype=torch.float32).pin_memory()
        phases = {}

        def e2e_step():
            tp = time.perf_counter()

            def lap(name):
                nonlocal tp
                t = time.perf_counter()
                phases[name] = phases.get(name, 0.0) + (t - tp) * 1e3
                tp = t

            with Simulation(local_rank) as s2:
                s2.set_grid(cfg["shape"], cfg["spacing_mm"]); lap("create+set_grid")
                s2.load_phantom(hm, hr); lap("load_phantom (131 MB H2D + pack + hull)")
                s2.load_activity(ha); lap("load_activity (105 MB H2D + alias table)")
                s2.load_organs(hl, cfg["n_organs"]); lap("load_organs (26 MB H2D + masses)")
                s2.set_physics_tables(tables)
                s2.set_options(**opts); lap("tables+options")
                step(s2); lap("run")
                s2.get_dose(out_d); lap("get_dose (kernel + 105 MB D2H)")
                s2.get_uncertainty(out_u); lap("get_uncertainty (kernel + 105 MB D2H)")
                r = s2.get_organ_doses(), s2.get_stats()
            lap("organs+stats+destroy")
            return r

        e2e_step()                                   # untimed: first-touch of the pinned buffers, allocator warm-up
        phases.clear()
        if dist:
            dist.barrier()
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        for _ in range(args.steps):                  # every step: full set-up from host buffers, run, read-back
            organs, st2 = e2e_step()
        torch.cuda.synchronize(dev)
        dt = (time.perf_counter() - t0) / args.steps
        if dist:
            t = torch.tensor([dt], device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        assert float(out_d.sum()) > 0 and organs["mean_Gy_per_decay"].max() > 0
        e2e = {"value": world * D / dt, "unit": "decays/s", "h2d_bytes_per_step": V * (1 + 4 + 4 + 1),
               "d2h_bytes_per_step": V * 8 + 27 * 56, "seconds": dt, "ms_setup_device": st2["ms_setup"],
               "phases_ms": {k: v / args.steps for k, v in phases.items()},
               "what": "anm_set_grid + load_phantom/activity/organs (host) + tables + anm_run + get_dose + get_uncertainty + get_organ_doses (host)"}

    # ---- image front end: set-up, not part of decays/s; HBM roofline of its two kernels -------
    frontend = None
    if not args.no_frontend and world == 1 and args.config == 3:
        img = anm_inputs.make_ct_pet(cfg, ct_shape=(512, 512, 400))          # 1 x 1 x 4 mm CT over the cfg3 grid
        hu_d = torch.from_numpy(img["ct_hu"]).to(dev)
        pet_d = torch.from_numpy(img["pet_bqml"]).to(dev)
        with Simulation(local_rank) as s3:
            s3.set_grid(cfg["shape"], cfg["spacing_mm"])
            ms_ct, ms_pet = [], []
            for _ in range(5):
                s3.load_ct(hu_d, img["ct_shape"], img["ct_spacing_mm"], img["ct_offset_mm"])
                s3.load_pet(pet_d, img["pet_shape"], img["pet_spacing_mm"], img["pet_offset_mm"])
                st3 = s3.get_stats()
                ms_ct.append(st3["ms_load_ct"]); ms_pet.append(st3["ms_load_pet"])
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm = float(peaks.get("hbm_gbs", 6500.0))
        b_ct = hu_d.numel() * 2 + V * 4
        b_pet = pet_d.numel() * 4 + V * 4
        frontend = {"workload": "CT 512x512x400 int16 HU @1x1x4mm + PET 256x256x400 Bq/mL -> cfg3 grid",
                    "load_ct_ms": min(ms_ct[1:]), "load_ct_bytes": b_ct, "load_ct_gbs": b_ct / (min(ms_ct[1:]) * 1e-3) / 1e9,
                    "load_pet_ms": min(ms_pet[1:]), "load_pet_bytes": b_pet, "load_pet_gbs": b_pet / (min(ms_pet[1:]) * 1e-3) / 1e9,
                    "hbm_peak_gbs": hbm, "peak_source": "MEASURED_PEAKS.json hbm_gbs" if peaks else "fallback 6500 GB/s",
                    "load_ct_frac": b_ct / (min(ms_ct[1:]) * 1e-3) / 1e9 / hbm,
                    "load_pet_frac": b_pet / (min(ms_pet[1:]) * 1e-3) / 1e9 / hbm}
        del hu_d, pet_d

    # ---- the widened rows on the same workload: 1e8 decays each, device time of anm_run ----
    variants = None
    if not args.no_variants and world == 1:
        variants = {}
        nv = min(D, 100_000_000)
        with torch.cuda.stream(stream):
            sim.set_electron_tables(anm_inputs.make_electron_tables())
            for name, kw in (("default_same_size", {}), ("electron_transport", {"electron_transport": 1}), ("uncertainty_hbh", {"uncertainty": 1})):
                sim.set_options(collect_stats=0, **opts, **kw)
                sim.run(nv, cfg["seed"])                      # warm-up (first launch of this kernel variant)
                sim.run(nv, cfg["seed"])
                stv = sim.get_stats()
                ms = stv["ms_transport"] + stv["ms_fold"] + stv["ms_finalize"]
                variants[name] = {"decays": nv, "ms": ms, "value": nv / (ms * 1e-3), "unit": "decays/s"}
            sim.set_options(collect_stats=0, **opts)
        # BASELINE.json configs[4], the full-resolution scale case (tally 630 MB > L2: the HBM-atomic regime), 1e9 of its
        # decays, device time of anm_run; its own context (4.5 GB), released afterwards
        if not args.no_cfg4 and args.config == 3:
            del mat, rho, act, lab
            cfg4 = anm_inputs.make_config(4)
            with torch.cuda.stream(stream), Simulation(local_rank) as s4:
                s4.set_stream(stream)
                s4.load_config(cfg4, tables, n_batches=100, collect_stats=1)
                s4.run(10_000_000, cfg4["seed"])
                c4 = s4.get_stats()
                s4.set_options(n_batches=100, positron_ke_MeV=cfg4["positron_ke_mev"])
                n4 = min(D, 1_000_000_000)
                s4.run(n4, cfg4["seed"])
                s4.run(n4, cfg4["seed"])
                st4 = s4.get_stats()
                ms4 = st4["ms_transport"] + st4["ms_fold"] + st4["ms_finalize"]
                dps4 = n4 / (ms4 * 1e-3)
                steps4, dep4 = c4["n_steps"] / 1e7, (c4["n_compton"] + c4["n_pe"]) / 1e7 + 1.0
                v4 = {"workload": "cfg4_fullres 512x512x600 @0.98x0.98x3mm, 27 organs, pairs+positron KE, 100 batches",
                      "decays": n4, "ms": ms4, "value": dps4, "unit": "decays/s", "texel_bits": int(st4["texel_bits"]),
                      "batches_per_launch": int(st4["batches_per_launch"]),
                      "events_per_decay": {"n_steps": steps4, "deposits": dep4}}
                # the same phantom through the 32-bit texels: what a phantom that is NOT on the 2^-12 g/cm^3 density grid
                # gets -- every phantom loaded from a CT image (anm_load_ct stores densities on the 2^-20 grid), and cfg4
                # itself before its generator was put on the coarse grid (reading C18)
                s4.set_options(n_batches=100, positron_ke_MeV=cfg4["positron_ke_mev"], texel_bits=32)
                s4.run(n4, cfg4["seed"])
                s4.run(n4, cfg4["seed"])
                st32 = s4.get_stats()
                ms32 = st32["ms_transport"] + st32["ms_fold"] + st32["ms_finalize"]
                v4["texel_bits_32"] = {"decays": n4, "ms": ms32, "value": n4 / (ms32 * 1e-3), "unit": "decays/s",
                                       "texel_bits": int(st32["texel_bits"]),
                                       "note": "same phantom, 32-bit texels: the path of any phantom off the 2^-12 density grid (every CT-loaded one)"}
                s4.set_options(n_batches=100, positron_ke_MeV=cfg4["positron_ke_mev"])
                if D >= 1_000_000_000:      # the config's own size (BASELINE.json configs[4]: "Run 1e10 decays"), once
                    s4.run(10_000_000_000, cfg4["seed"])
                    st10 = s4.get_stats()
                    ms10 = st10["ms_transport"] + st10["ms_fold"] + st10["ms_finalize"]
                    v4["run_1e10"] = {"decays": 10_000_000_000, "ms": ms10, "value": 1e10 / (ms10 * 1e-3), "unit": "decays/s",
                                      "deposited_MeV": st10["deposited_MeV"], "rms_rel_sigma_gt10": st10["rms_rel_sigma_gt10"],
                                      "rms_rel_sigma_gt50": st10["rms_rel_sigma_gt50"]}
                if peaks_dev:      # the memory side binds here: random DRAM gathers + REDs over 630 MB volumes
                    t_model = steps4 / (peaks_dev["gather_gps"][1] * 1e9) + dep4 / (peaks_dev["red_gps"][1] * 1e9)
                    v4["roofline"] = {"bound": "hbm random access", "gather_frac": steps4 * dps4 / 1e9 / peaks_dev["gather_gps"][1],
                                      "red_frac": dep4 * dps4 / 1e9 / peaks_dev["red_gps"][1],
                                      "mem_mix_uniform_ratio": (steps4 + dep4) * dps4 / 1e9 / peaks_dev["mix_gps"][1],   # > 1: locality (see roofline.mem_mix_uniform)
                                      "decays_per_s_if_gathers_and_reds_were_serial_at_peak": 1.0 / t_model}
            variants["cfg4_fullres"] = v4
            del cfg4

    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return

    # ---- the oracle beside it, on this box's host cores (bounded sample) ------------------------------------
    cpu = None
    if not args.no_cpu_baseline and world == 1:
        from oracle import anm_oracle
        cores = os.cpu_count() or 1
        n = cores * args.cpu_baseline_decays_per_core
        o = anm_oracle.Oracle(cfg, tables, n_decays=n, n_batches=cores, seed=1042)
        r = o.run_parallel(cores)
        cpu = {"value": n / r["seconds"], "unit": "decays/s", "cores": r["cores"], "kind": "oracle",
               "sample": "%d decays of cfg3 (%d per core), one batch per single-threaded process, %.1f s wall" % (n, args.cpu_baseline_decays_per_core, r["seconds"]),
               "per_core": n / r["cpu_seconds"]}

    print(json.dumps({
        "metric": "decays/s (18F, patient phantom)", "value": value, "unit": "decays/s",
        "sec_per_1e9_decays": 1e9 / value, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": WORKLOAD if args.config == 3 else "cfg4_fullres 512x512x600 @0.98x0.98x3mm (profiling only, not the bench workload)",
                   "decays_per_step_per_gpu": D, "seed": cfg["seed"],
                   "l2": "working set (texels 105 MB + per-batch tallies (one 105 MB volume per batch in flight) + sum/sumsq 210 MB + alias 94 MB) exceeds the 126 MB L2; no flush needed",
                   "multi_gpu": "one logical run of N*D decays: whole-batch shards via history_offset, NCCL sum-all-reduce of the tallies + merged finalize at the end of every step" if world > 1 else "single GPU"},
        "clocks": clk, "e2e": e2e, "gpu_launches": int(launches),
        "phase_ms_per_step": {"transport": ms_t / args.steps, "fold": ms_f / args.steps, "finalize": ms_fin / args.steps},
        "roofline": roofline, "cpu_baseline": cpu, "frontend": frontend, "variants": variants,
        "paper_context": "ARCHER-NM on a Titan V: 1e9 decays in <0.5 min (>=3.3e7 decays/s), GATE 376 min (PAPER.md:L117); other hardware, other phantom, electron transport on",
    }))
    if dist:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
