#!/usr/bin/env python
"""bench.py -- throughput of the fp64 VL+CT MHD step (BASELINE.json metric) on B200.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c3|c5|c4|c1|c2|NxNxN] [--impl reference]

A "step" is one pass of the whole hot path: the CFL reduction (Eq. 11) followed by one full VL+CT
step (ghost fill, PCM+HLLD predictor, CT, half update, PLMC/PPMC+HLLD, CT, full update) on a
seeded synthetic grid.  `value` = cell updates per second with the state resident in HBM;
`e2e` = the same through the host-buffer C ABI (mhd_set_state + mhd_compute_dt + mhd_step +
mhd_get_state every step, pinned host memory).  N > 1 runs N independent replicas (DESIGN.md:
"replicas only", no collective); rank 0 prints ONE JSON line.
`--impl reference` times the CPU oracle (oracle/) on the host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
for _p in (ROOT, os.path.join(ROOT, "oracle")):
    if _p not in sys.path:
        sys.path.insert(0, _p)

import numpy as np  # noqa: E402

METRIC = "fp64 MHD cell updates/sec (VL+CT, HLLD, PLMC)"
UNIT = "cell updates/s"
CFL = 0.4

# Algorithmic work per cell update: fp64 FLOPs (dadd + dmul + 2 dfma,
# thread-level, predicated-on) executed per ACTIVE cell by each kernel as counted by ncu on the
# 256^3 PLMC workload (profiles/r1_ncu_kernels.md), and the HBM bytes each kernel must move per
# cell (compulsory reads + writes of its operand arrays, 8 B each).
KERNEL_MODEL = {
    #                          flop/cell  bytes/cell
    # U^n -> W^{n+1/2}, E_ref in one kernel.  1388 = the algorithmic count (PCM+HLLD 1169, CT 80, half
    # update 139, as counted on the three separate kernels); the kernel EXECUTES 1286 per cell (round 1: 1695) because
    # the halo columns of every 30 x 10 tile repeat their neighbours' Riemann solves.
    "k_predictor_stage":      (1388, (8 + 8 + 3) * 8),
    "k_flux_x":               (866, (8 + 7) * 8),               # W^{n+1/2} -> 7 fluxes
    "k_flux_march<1>":        (864, (8 + 7) * 8),
    "k_flux_march<2>+update": (924, (8 + 3 + 5 + 10 + 5) * 8),  # + U^n, x/y hydro fluxes -> U^{n+1} hydro
    "k_ct(corrector)":        (77, (9 + 3 + 3) * 8),            # mass/magnetic fluxes + E_ref -> edge E
    "k_update(B)+cfl":        (191, (3 + 3 + 5 + 3) * 8),       # B^n, edge E, U^{n+1} hydro -> B^{n+1}; CFL rate
}
# the same for PPMC (ncu capture of `--workload 256:ppmc`, profiles/r1_ncu_kernels.md): only the sweeps differ
KERNEL_MODEL_PPMC = dict(KERNEL_MODEL)
KERNEL_MODEL_PPMC.update({"k_flux_x": (1068, (8 + 7) * 8), "k_flux_march<1>": (1057, (8 + 7) * 8),
                          "k_flux_march<2>+update": (1121, (8 + 3 + 5 + 10 + 5) * 8),
                          "k_ct(corrector)": (76, (9 + 3 + 3) * 8), "k_update(B)+cfl": (190, (3 + 3 + 5 + 3) * 8)})
MODELS = {1: KERNEL_MODEL, 2: KERNEL_MODEL_PPMC}
# dram__bytes_read.sum + dram__bytes_write.sum per launch (GB) from the same ncu captures (256^3)
NCU_TRAFFIC_GB = {1: {"k_predictor_stage": 2.78, "k_flux_x": 2.07, "k_flux_march<1>": 2.13,
                      "k_flux_march<2>+update": 4.38, "k_ct(corrector)": 2.09, "k_update(B)+cfl": 1.93},
                  2: {"k_predictor_stage": 2.87, "k_flux_x": 2.11, "k_flux_march<1>": 2.20,
                      "k_flux_march<2>+update": 4.60, "k_ct(corrector)": 2.14, "k_update(B)+cfl": 1.98}}
STEP_FLOP_PER_CELL = sum(v[0] for v in KERNEL_MODEL.values())     # 4310 (PLMC; PPMC 4900), algorithmic
# what this build executes per active cell and step (ncu, profiles/r2_ncu_kernels.md): flop = dadd + dmul +
# 2 dfma summed over the step's kernels (halo columns of the stage kernel included); DRAM bytes read + written
EXECUTED_FLOP_PER_CELL = {1: 3598, 2: 4993}   # (the branch-free PPM limiter evaluates every candidate value)
NCU_STEP_DRAM_BYTES_PER_CELL = {1: 918, 2: 948}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=40)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="c3",
                    help="c1..c5 = BASELINE.json configs[0..4]; or NxNxN[:plmc|ppmc] turbulence cube")
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-sizes", action="store_true", help="skip the size sweep block (32^3 .. 640^3, PPMC 256^3 / 512^3)")
    ap.add_argument("--sizes-budget", type=float, default=420.0,
                    help="wall-clock seconds the size sweep may take; sizes that do not fit are reported as skipped")
    return ap.parse_args()


def make_problem(workload, small=False):
    """Seeded synthetic input (paper_2402_05240_b200/inputs.py) for a BASELINE.json config."""
    from paper_2402_05240_b200 import inputs
    w = workload.lower()
    if w == "c1":
        return inputs.linear_wave(32, 32, 32, "fast", recon=1), "c1: 32^3 linear fast wave, PLMC"
    if w == "c2":
        return inputs.riemann("brio_wu", 256, 16, axis=0, recon=1), "c2: 256x16x16 Brio-Wu, PLMC, outflow x"
    if w == "c3":
        return inputs.turbulence(256, recon=1), "c3: 256^3 Mach-1 beta-1 turbulence, PLMC (BASELINE.json configs[2])"
    if w == "c4":
        return inputs.blast(512, recon=2), "c4: 512^3 blast, PPMC (BASELINE.json configs[3])"
    if w == "c5":
        return inputs.turbulence(640, recon=1), "c5: 640^3 Mach-1 beta-1 turbulence, PLMC (BASELINE.json configs[4])"
    recon = 1
    if ":" in w:
        w, r = w.split(":")
        recon = {"plmc": 1, "ppmc": 2, "pcm": 0}[r]
    n = tuple(int(x) for x in w.split("x"))
    if len(n) == 1:
        n = n * 3
    return inputs.turbulence(n, recon=recon), "%dx%dx%d turbulence, recon=%d" % (n + (recon,))


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, reasons, pw = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) < 7:
                continue
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); pw.append(float(r[2]))
            except ValueError:
                continue
            for nm, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": float(max(smax)) if smax else None,
                "power_w_max": float(max(pw)) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(problem, n_steps, warmup=0, threads=None):
    """The oracle as it stands on the host cores: {compute_dt; step} x n_steps.
    threads=None: all cores, in this process.  threads=k: a child process with OMP_NUM_THREADS=k
    (the OpenMP runtime reads it once).  Returns (cells/s, seconds, cores)."""
    nc = problem.n[0] * problem.n[1] * problem.n[2]
    if threads is not None:
        code = ("import sys, time, json; sys.path.insert(0, %r); sys.path.insert(0, %r)\n"
                "import oracle as orc\nfrom paper_2402_05240_b200 import inputs\n"
                "p = inputs.turbulence(%d, recon=%d)\n"
                "o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc); o.set_state(p.state)\n"
                "t0 = time.perf_counter()\n"
                "for _ in range(%d): o.step(o.compute_dt(0.4))\n"
                "print(json.dumps([time.perf_counter() - t0, orc.num_threads()]))\n"
                % (ROOT, os.path.join(ROOT, "oracle"), problem.n[0], problem.recon, n_steps))
        env = dict(os.environ, OMP_NUM_THREADS=str(threads))
        out = subprocess.run([sys.executable, "-c", code], env=env, stdout=subprocess.PIPE, text=True, check=True)
        el, cores = json.loads(out.stdout.strip().splitlines()[-1])
        return nc * n_steps / el, el, cores
    import oracle as orc
    o = orc.Oracle(*problem.n, problem.gamma, problem.recon, problem.bc)
    o.set_state(problem.state)
    for _ in range(warmup):
        o.step(o.compute_dt(CFL))
    t0 = time.perf_counter()
    for _ in range(n_steps):
        dt = o.compute_dt(CFL)
        o.step(dt)
    el = time.perf_counter() - t0
    cores = orc.num_threads()
    o.close()
    return nc * n_steps / el, el, cores


def sample_problem(workload):
    """The oracle's workload: the configuration itself where the host can hold it and finish a step in
    seconds (c1, c2, c3 and 256^3 cubes IN FULL), else a bounded sample of the same recipe."""
    from paper_2402_05240_b200 import inputs
    w = workload.lower()
    if w in ("c1", "c2", "c3"):
        p, name = make_problem(w)
        return p, name + " (full size)", True
    if w == "c4":
        return inputs.blast(128, recon=2), "c4 recipe (blast, PPMC) at 128^3 (512^3 needs 43 GB and 100 s per step)", False
    if w == "c5":
        return inputs.turbulence(256, recon=1), "c5 recipe (Mach-1 beta-1 turbulence, PLMC) at 256^3 (640^3 needs 84 GB)", False
    recon = 2 if w.endswith(":ppmc") else 1
    n = int(w.split(":")[0].split("x")[0])
    if n <= 256:
        p, name = make_problem(w)
        return p, name + " (full size)", True
    return inputs.turbulence(256, recon=recon), "turbulence recipe, recon=%d, at 256^3" % recon, False


def run_reference(args):
    """The reference arm of this tier: the CPU oracle, as it stands, on the host cores, on the arm's own
    workload (c3 in full: 256^3; a step is ~3.5 s on 16 threads).  --steps is honoured up to a wall-clock
    budget of ~4 minutes; the line says how many steps were timed."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    p, sample, same = sample_problem(args.workload)
    _, wname = make_problem_name(args.workload)
    import oracle as orc
    o = orc.Oracle(*p.n, p.gamma, p.recon, p.bc)
    o.set_state(p.state)
    budget = 240.0
    t_w = time.perf_counter()
    done_w = 0
    for _ in range(args.warmup):
        o.step(o.compute_dt(CFL))
        done_w += 1
        if time.perf_counter() - t_w > 0.15 * budget:
            break
    t0 = time.perf_counter()
    done = 0
    for _ in range(args.steps):
        o.step(o.compute_dt(CFL))
        done += 1
        if time.perf_counter() - t0 > budget:
            break
    el = time.perf_counter() - t0
    cores = orc.num_threads()
    o.close()
    nc = p.n[0] * p.n[1] * p.n[2]
    val = nc * done / el
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
            "steps": done, "warmup": done_w, "ms_per_step": 1e3 * el / done,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wname, "sample": sample, "same_config": same,
                                            "steps_requested": args.steps},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def make_problem_name(workload):
    names = {"c1": "c1: 32^3 linear fast wave, PLMC", "c2": "c2: 256x16x16 Brio-Wu, PLMC, outflow x",
             "c3": "c3: 256^3 Mach-1 beta-1 turbulence, PLMC (BASELINE.json configs[2])",
             "c4": "c4: 512^3 blast, PPMC (BASELINE.json configs[3])",
             "c5": "c5: 640^3 Mach-1 beta-1 turbulence, PLMC (BASELINE.json configs[4])"}
    return None, names.get(workload.lower(), workload + " turbulence cube")


def job_value(ms_local, cells_per_rank, steps, world, device="cuda"):
    """Whole-job throughput of N independent replicas ("replicas only"): every
    rank advances its own grid; the job's time is the MAX over ranks of the device-timed region and
    the job's work the SUM of the cell updates.  Returns (cell updates/s, ms)."""
    ms = float(ms_local)
    if world > 1:
        import torch
        import torch.distributed as dist
        t = torch.tensor([ms], device=device, dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    return world * cells_per_rank * steps / (ms * 1e-3), ms


def load_measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as fh:
            d = json.load(fh)
        return float(d["hbm_gbs"]), "MEASURED_PEAKS.json"
    except (OSError, KeyError, ValueError):
        return 6650.0, "fallback (B200_PROFILING.md)"


SIZES = [("32^3 plmc", "c1"), ("256x16x16 plmc (c2)", "c2"), ("64^3 plmc", "64"), ("128^3 plmc", "128"),
         ("256^3 ppmc", "256:ppmc"), ("384^3 plmc", "384"), ("512^3 plmc", "512"), ("c4: 512^3 blast ppmc", "c4"),
         ("c5: 640^3 plmc", "c5")]


def size_sweep(mhd, torch, local, budget_s, fp64_tf, flop_cell):
    """north_star: cell updates/s from 32^3 to 640^3 (PLMC) and for PPMC at 256^3 / 512^3, each with its
    fraction of the fp64 roofline (counted flop / measured fp64 peak / step time) and the clocks seen."""
    out, t_start = [], time.perf_counter()
    for label, w in SIZES:
        if time.perf_counter() - t_start > budget_s:
            out.append({"size": label, "skipped": "size-sweep time budget (%.0f s) used up" % budget_s})
            continue
        t0 = time.perf_counter()
        p, _ = make_problem(w)
        t_gen = time.perf_counter() - t0
        nc = p.n[0] * p.n[1] * p.n[2]
        stream = torch.cuda.Stream()
        try:
            g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, stream=stream)
        except Exception as e:      # out of memory on a smaller part: reported, not fatal
            out.append({"size": label, "skipped": "init failed: %s" % str(e)[:80]})
            continue
        g.set_state(p.state)
        steps = 6 if nc >= 300 ** 3 else (12 if nc >= 2 ** 21 else 200)
        with torch.cuda.stream(stream):
            g.advance(4 if nc >= 2 ** 21 else 40, CFL)
            torch.cuda.synchronize()
            sampler = ClockSampler(local)
            sampler.start()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = []
            for _ in range(3):
                e0.record(stream)
                g.advance(steps, CFL)
                e1.record(stream)
                torch.cuda.synchronize()
                reps.append(e0.elapsed_time(e1) / steps)
            clocks = sampler.stop()
            ok = True
            try:
                g.compute_dt(CFL)
            except mhd.MhdError:
                ok = False
        g.close()
        del g
        torch.cuda.empty_cache()
        med = sorted(reps)[1]
        fc = flop_cell.get(p.recon)
        out.append({"size": label, "grid": list(p.n), "recon": p.recon, "steps": steps,
                    "ms_per_step_median": med, "ms_per_step_best": min(reps),
                    "cell_updates_per_s": nc / (med * 1e-3),
                    "frac_flop": (fc * nc / (fp64_tf * 1e12)) / (med * 1e-3) if fc else None,
                    "sm_mhz": clocks.get("sm_mhz"), "power_w_max": clocks.get("power_w_max"),
                    "reasons": clocks.get("reasons"), "state_ok": ok, "input_gen_s": round(t_gen, 1)})
        del p
    return out


def run_b200(args):
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the VL+CT step has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2402_05240_b200 import mhd
    from paper_2402_05240_b200.inputs import FIELDS

    p, wname = make_problem(args.workload)
    nc = p.n[0] * p.n[1] * p.n[2]
    stream = torch.cuda.Stream()
    g = mhd.Mhd(*p.n, p.gamma, p.recon, p.bc, stream=stream)
    g.set_state(p.state)

    def barrier():
        if world > 1:
            dist.barrier()

    with torch.cuda.stream(stream):
        g.advance(args.warmup, CFL)
        torch.cuda.synchronize()
        sampler = ClockSampler(local)
        if rank == 0:
            sampler.start()
        barrier()
        torch.cuda.synchronize()
        l0 = g.launch_count()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        g.advance(args.steps, CFL)
        e1.record(stream)
        torch.cuda.synchronize()
        barrier()
        ms = e0.elapsed_time(e1)
        launches = g.launch_count() - l0
        value, ms = job_value(ms, nc, args.steps, world)
        # ---- per-kernel live timing (CUDA events on the library stream) ----------------
        # Directly behind the timed region, the same K steps enqueued back to back in the same way with an
        # event after every launch (mhd_advance_profile): each kernel's duration averaged over the region,
        # in the steady state the headline number is measured in (same caches; a box that throttles under
        # the load does so progressively, hence next to the region that gives `value`).
        prof = {name: t_ms for name, t_ms in g.advance_profile(max(args.steps, 1), CFL)}
        # two more regions of the same length (median and best of 3); `value` is the first
        reps = [ms / args.steps]
        for _ in range(2):
            barrier()
            e0.record(stream)
            g.advance(args.steps, CFL)
            e1.record(stream)
            torch.cuda.synchronize()
            reps.append(job_value(e0.elapsed_time(e1), nc, args.steps, world)[1] / args.steps)
        clocks = sampler.stop() if rank == 0 else None   # sampled over the timed region, the profiled one and the repeats

        bad_state = False
        try:
            g.compute_dt(CFL)
        except mhd.MhdError:
            bad_state = True

        # ---- end to end through the host-buffer ABI ------------------------------------
        sh = mhd.field_shapes(*p.n)
        pin_in = {f: torch.from_numpy(np.ascontiguousarray(p.state[f])).pin_memory() for f in FIELDS}
        pin_out = {f: torch.empty(sh[f], dtype=torch.float64).pin_memory() for f in FIELDS}
        np_in = {f: pin_in[f].numpy() for f in FIELDS}
        np_out = {f: pin_out[f].numpy() for f in FIELDS}
        h2d = sum(int(np_in[f].nbytes) for f in FIELDS)
        d2h = sum(int(np_out[f].nbytes) for f in FIELDS) + 8

        def e2e_step():
            g.set_state(np_in)
            dt_ = g.compute_dt(CFL)
            g.step(dt_)
            g.get_state(np_out)

        e2e_step()
        barrier()
        torch.cuda.synchronize()
        e0.record(stream)
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            e2e_step()
        e1.record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        ms_e2e = max(e0.elapsed_time(e1), wall * 1e3)
        e2e_val, ms_e2e = job_value(ms_e2e, nc, args.e2e_steps, world)

    fp64_tf, copy_gbs = (None, None)
    if rank == 0:
        fp64_tf, copy_gbs = mhd.measure_peaks(1.0)
    g.close()

    if rank == 0:
        hbm_peak, hbm_src = load_measured_peaks()
        step_ms = sum(prof.values())
        model = MODELS.get(p.recon)   # FLOP counts were taken on the PLMC and PPMC builds
        top = max((k for k in prof if k in KERNEL_MODEL), key=lambda k: prof[k])
        flop_cell, byte_cell = (model or KERNEL_MODEL)[top]
        if model is None:
            flop_cell = None
        t_top = prof[top] * 1e-3
        traffic = NCU_TRAFFIC_GB[p.recon].get(top) if (tuple(p.n) == (256, 256, 256) and model) else None
        roof = {"kernel": top, "kernel_ms": prof[top], "share_of_step": prof[top] / step_ms,
                "traffic": traffic * 1e9 if traffic else None,
                "traffic_source": "profiles/r2_ncu_kernels.md (ncu --set full, 256^3)" if traffic else None}
        hbm_ach = byte_cell * nc / t_top / 1e9
        roof["algorithmic_bytes_per_launch"] = byte_cell * nc
        if flop_cell is not None and flop_cell * nc / (fp64_tf * 1e12) > byte_cell * nc / (hbm_peak * 1e9):
            ach = flop_cell * nc / t_top / 1e12
            roof.update({"bound": "alu", "achieved": ach, "peak": fp64_tf, "unit": "TFLOP/s",
                         "frac": ach / fp64_tf, "peak_source": "measured DFMA chain (mhd_measure_peaks, sustained)",
                         "hbm_achieved_gbs": hbm_ach})
        else:
            roof.update({"bound": "hbm", "achieved": hbm_ach, "peak": hbm_peak, "unit": "GB/s",
                         "frac": hbm_ach / hbm_peak, "peak_source": hbm_src})
            if flop_cell is not None:
                roof["fp64_achieved_tflops"] = flop_cell * nc / t_top / 1e12
        # whole-step roofline (north_star): counted FLOPs at the measured fp64 peak, counted bytes at the
        # measured HBM bandwidth, and the 128 B/cell floor beside them
        if model:
            step_flop = sum(v[0] for v in model.values())
            t_step = ms / args.steps * 1e-3
            t_flop = step_flop * nc / (fp64_tf * 1e12)
            ex_flop = EXECUTED_FLOP_PER_CELL.get(p.recon)
            dram = NCU_STEP_DRAM_BYTES_PER_CELL.get(p.recon)
            roof["step"] = {"flop_per_cell_algorithmic": step_flop, "flop_per_cell_executed": ex_flop,
                            "dram_bytes_per_cell_ncu": dram,
                            "frac_flop": t_flop / t_step,
                            "frac_flop_executed": (ex_flop * nc / (fp64_tf * 1e12)) / t_step if ex_flop else None,
                            "frac_counted_bytes": (dram * nc / (hbm_peak * 1e9)) / t_step if dram else None,
                            "frac_of_128B_floor": (128.0 * nc / (hbm_peak * 1e9)) / t_step,
                            "fp64_tflops_step_algorithmic": step_flop * nc / t_step / 1e12,
                            "basis": "algorithmic = dadd + dmul + 2 dfma per active cell of the plain formulation "
                                     "(round-1 ncu count, profiles/r1_ncu_kernels.md); executed = the same count on "
                                     "this build (profiles/r2_ncu_kernels.md)"}
        roof["kernels_ms"] = {k: round(v, 4) for k, v in prof.items()}
        roof["kernels_ms_source"] = ("mhd_advance_profile: CUDA events after every launch of %d back-to-back steps "
                                     "on the library stream, mean per kernel; sum = %.4f ms per step" % (args.steps, step_ms))
        roof["measured_here"] = {"fp64_tflops": fp64_tf, "copy_gbs": copy_gbs}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "ms_per_step_repeats": [round(x, 5) for x in reps], "ms_per_step_median": sorted(reps)[1],
                "ms_per_step_best": min(reps),
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": wname, "grid": list(p.n), "recon": p.recon, "cfl": CFL,
                           "parallelism": "replicas x%d" % world,
                           "l2": "inputs larger than L2 (state %.0f MB)" % (8 * 8 * nc / 1e6),
                           "step": "mhd_advance: CFL reduction + full VL+CT step, dt on device"},
                "clocks": clocks, "gpu_launches": int(launches),
                "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                        "steps": args.e2e_steps},
                "roofline": roof, "state_ok": not bad_state,
                "paper_context": {"a100_cell_updates_per_s": 2.59e8, "ratio": value / world / 2.59e8}}
        if world == 1 and not args.no_sizes:
            flop_cell = {r: sum(v[0] for v in m.values()) for r, m in MODELS.items()}
            line["sizes"] = size_sweep(mhd, torch, local, args.sizes_budget, fp64_tf, flop_cell)
        if world == 1 and not args.no_cpu_baseline:
            sp, sname, same = sample_problem(args.workload)
            big = sp.n[0] * sp.n[1] * sp.n[2] >= 2 ** 22
            v, el, cores = time_oracle(sp, 5 if big else 200, warmup=1 if big else 5)   # ~20 s of host work
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
                                    "sample": sname + ", %d steps, %.1f s" % (5 if big else 200, el),
                                    "same_config": same}
            if big:   # one thread, labelled: a smaller cube of the same recipe (a 256^3 step takes ~1 min on one core)
                from paper_2402_05240_b200 import inputs
                v1, el1, c1 = time_oracle(inputs.turbulence(128, recon=sp.recon), 2, threads=1)
                line["cpu_baseline"]["single_thread"] = {"value": v1, "cores": c1,
                                                         "sample": "same recipe at 128^3, 2 steps, %.1f s" % el1}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse_args()
    sys.exit(run_reference(a) if a.impl == "reference" else run_b200(a))
