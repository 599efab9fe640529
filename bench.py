#!/usr/bin/env python
"""bench.py -- throughput of the Vlasov full-step hot path on B200.

A "step" is one cycle of section 4.3 without the fluid solve, for all species:
currents (eq. 11) -> Maxwell half step -> one complete Vlasov step (x/2, y/2, vx, vy, vz, y/2, x/2, eq. 22)
with its moment reductions -> currents -> Maxwell half step; plus the ghost fill where a y side is FLUID.
metric = interior phase-space cell-updates/s (all species).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload gem128|gem64|band|nv16|nv24|nv32|nv48]
    python bench.py --impl reference ...     # the oracle, as it stands, on the host cores (rank 0 only)

Prints ONE JSON line (rank 0).  N > 1 = N independent replicas (the build is single-GPU by north_star,
DESIGN.md "Multi-GPU": replicas only, no collective on the data path); launched by torchrun.
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

import numpy as np

from paper_1406_5445_b200 import inputs

METRIC = "vlasov_phase_space_cell_updates_per_s"
UNIT = "cell-updates/s"

# Algorithmic HBM bytes per phase-space cell and launch of each f-sized kernel:
# a sweep reads and writes every cell once (8 + 8 B); the moments pass reads it once.
BYTES_PER_CELL = {"sweep_x": 16.0, "sweep_y": 16.0, "sweep_z": 16.0, "sweep_xy": 16.0, "sweep_yx": 16.0, "vsweep_x": 16.0, "vsweep_yz": 16.0,
                  "vsweep_xyz": 16.0, "moments": 8.0}


def make_workload(name):
    if name == "gem128":
        return inputs.gem_workload(nx=128, ny=64, nv=32, steps=20, name="gem_128x64x32^3_x2species")
    if name == "gem64":
        return inputs.gem_workload(nx=64, ny=32, nv=32, steps=50, name="gem_64x32x32^3_x2species")
    if name == "band":
        return inputs.band_workload()
    if name == "gem3d":
        return inputs.gem3d_workload()
    if name.startswith("nv"):
        nv = int(name[2:])
        return inputs.gem_workload(nx=64, ny=64, nv=nv, steps=10, name=f"gem_64x64x{nv}^3_x2species")
    raise SystemExit(f"unknown workload {name}")


def cpu_model():
    try:
        with open("/proc/cpuinfo") as fh:
            for ln in fh:
                if ln.lower().startswith("model name"):
                    return ln.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as fh:
            return float(json.load(fh)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


# ------------------------------------------------------------------------------------------------
# clocks sampled DURING the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap,power.draw")
    NAMES = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]

    def __init__(self, index):
        self.lines = []
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "100"],
                                      stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except OSError:
            self.p = None

    def _read(self):
        for ln in self.p.stdout:
            self.lines.append((time.time(), ln.strip()))

    def stop(self, t0, t1):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        sm, mx, pw, reasons = [], [], [], set()
        rows = [ln for (t, ln) in self.lines if t0 <= t <= t1 + 0.12] or [ln for (_, ln) in self.lines[-3:]]
        for ln in rows:
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[6]))
            except ValueError:
                continue
            for k, nm in enumerate(self.NAMES):
                if c[2 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm), "power_w_max": max(pw) if pw else None}


# ------------------------------------------------------------------------------------------------
# the oracle legs (cpu_baseline and --impl reference): only oracle/ is executed here
# ------------------------------------------------------------------------------------------------
def oracle_sample_workload(w, nx_s=16, ny_s=8):
    """A bounded sample of workload w: the same species, velocity grids, dt, dx, dy, profiles and noise on
    an nx_s x ny_s spatial cut around the sheet centre (y rows straddle y = 0)."""
    nx_s = min(nx_s, w.nx)
    ny_s = min(ny_s, w.ny)
    import copy
    ws = copy.deepcopy(w)
    ws.nx, ws.ny = nx_s, ny_s
    ws.lx, ws.ly = w.dx * nx_s, w.dy * ny_s
    ws.x0, ws.y0 = -ws.lx / 2, -ws.ly / 2
    ws.ly_domain = getattr(w, "ly_domain", w.ly)
    ws.name = f"{w.name}:cut{nx_s}x{ny_s}"
    return ws


class OracleRun:
    """State of an oracle run of a workload; the section-4.3 cycle itself is oracle.cycle (no CUDA)."""

    def __init__(self, ws):
        from oracle import oracle as orc
        self.orc, self.w = orc, ws
        orc.build()
        self.sp = []
        self.f = []
        for s, spec in enumerate(ws.species):
            self.f.append(inputs.gem_f(ws, s))
            spec.f_inf = inputs.gem_f_inf(ws, s)
            self.sp.append(orc.Species(spec.q, spec.m, spec.nv, spec.vmin, spec.vmax, spec.f_inf))
        self.E, self.B = inputs.gem_fields(ws)
        self.wall = 0 if ws.bc_y_lo == inputs.BC_PERIODIC else 1
        self.fluid = None
        self.mom = [orc.moments(f, sp, ws.nx, ws.ny, ws.nghost_y) for f, sp in zip(self.f, self.sp)]
        self.step_index = 0

    def cycle(self):
        orc, w = self.orc, self.w
        fluid = None
        if w.bc_y_lo == inputs.BC_FLUID:
            fluid = [(inputs.band_fluid_state(w, s, 0, self.step_index), inputs.band_fluid_state(w, s, 1, self.step_index))
                     for s in range(len(self.sp))]
        self.mom = orc.cycle(self.f, self.sp, self.mom, self.E, self.B, w.nx, w.ny, w.nghost_y, w.lx, w.ly, w.dt, w.nsub,
                             w.c, w.mu0, fields_yee=w.fields_yee, bc_lo=w.bc_y_lo, bc_hi=w.bc_y_hi, fluid=fluid)
        self.step_index += 1


def oracle_leg(w, steps, warmup, budget_s=25.0):
    """Time the oracle on a bounded sample.  Returns (cell-updates/s, ms/step, cores, sample text, steps done)."""
    ws = oracle_sample_workload(w)
    run = OracleRun(ws)
    cores = run.orc.num_threads()
    for _ in range(warmup):
        run.cycle()
    t0 = time.perf_counter()
    done = 0
    for _ in range(steps):
        run.cycle()
        done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    cells = ws.interior_cells
    sample = (f"{ws.nx}x{ws.ny} spatial cut of {w.name} (same species, {ws.species[0].nv[0]}^3 velocity cells each, dt, dx, dy, "
              f"profiles, noise), {done} full cycle(s) after {warmup} warm-up, {cells} interior cells/step")
    return cells * done / dt, 1e3 * dt / done, cores, sample, done


# ------------------------------------------------------------------------------------------------
# multi-GPU: replicas only -- the only cross-rank step is the timing reduction
# ------------------------------------------------------------------------------------------------
def max_over_ranks(ms, dist, device):
    """Device-timed milliseconds -> the maximum over all ranks (identity without a process group)."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(cells_per_replica, steps, ms, world):
    """Aggregate cell-updates/s of `world` independent replicas that all ran `steps` steps within `ms`."""
    return world * cells_per_replica * steps / (ms * 1e-3)


# ------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------
def upload_f(w, s, torch, device):
    """Seeded f of species s, generated row by row on the host and copied to the device."""
    sp = w.species[s]
    if getattr(w, "nz", 1) > 1:          # 3D3V: slab by slab
        f = torch.empty((w.nz, w.ny_g, w.nx) + tuple(sp.nv), dtype=torch.float64, device=device)
        for k in range(w.nz):
            f[k].copy_(torch.from_numpy(inputs.gem3d_f(w, s, k)))
        sp.f_inf = inputs.gem_f_inf(w, s)
        return f
    f = torch.empty((w.ny_g, w.nx) + tuple(sp.nv), dtype=torch.float64, device=device)
    for r in range(w.ny_g):
        f[r].copy_(torch.from_numpy(inputs.gem_f(w, s, rows=[r])[0]))
    sp.f_inf = inputs.gem_f_inf(w, s)
    return f


def gpu_arm(args):
    import torch
    from paper_1406_5445_b200 import binding
    binding.lib()                                  # fails loudly if the CUDA library is missing
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if world != args.gpus and world > 1:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=device)

    w = make_workload(args.workload)
    ns = len(w.species)
    fs = [upload_f(w, s, torch, device) for s in range(ns)]
    nz = getattr(w, "nz", 1)
    E0, B0 = inputs.gem3d_fields(w) if nz > 1 else inputs.gem_fields(w)
    stream = torch.cuda.current_stream()
    order = binding.ORDER_VXV if args.order == "vxv" else binding.ORDER_XVX
    ctx = binding.context_for(w, fs, order=order)
    Ed, Bd = torch.from_numpy(E0).to(device), torch.from_numpy(B0).to(device)
    fluid = None
    if w.bc_y_lo == inputs.BC_FLUID:
        # seeded 5-moment states, redrawn per step from the step index (config 4); resident before timing
        nstate = args.warmup + (args.reps + 2) * args.steps + 8
        fluid = [[[torch.from_numpy(inputs.band_fluid_state(w, s, side, k)).to(device) for side in (0, 1)]
                  for s in range(ns)] for k in range(nstate)]
    step_no = [0]
    live = None
    if fluid is not None and args.fluid == "live":
        # the fluid region of the coupled set-up as two live five-moment blocks (rest of the 128-row domain), fields of
        # the fluid blocks held at their initial values (the Maxwell solve of this bench covers the band)
        nyf = (round(w.ly_domain / w.dy) - w.ny) // 2
        live = {"nyf": nyf, "U": [], "E": [], "B": [], "blk": [], "q": [sp.q for sp in w.species], "m": [sp.m for sp in w.species],
                "b5": [[torch.empty((5, w.nghost_y, w.nx), dtype=torch.float64, device=device) for _ in (0, 1)] for _ in range(ns)],
                "mb": torch.empty((10, w.nghost_y, w.nx), dtype=torch.float64, device=device),
                "gh": [torch.zeros((3, ns, 5, 2, w.nx), dtype=torch.float64, device=device) for _ in (0, 1)]}
        for side in (0, 1):
            U0, Ef, Bf = inputs.band_fluid_block(w, nyf, side)
            live["U"].append(torch.from_numpy(U0).to(device))
            live["E"].append(torch.from_numpy(Ef).to(device)); live["B"].append(torch.from_numpy(Bf).to(device))
            live["blk"].append(binding.FluidBlock(w.nx, nyf, w.dx, w.dy, live["q"], live["m"],
                                                  binding.FLUID_BC_WALL if side == 0 else binding.FLUID_BC_COUPLED,
                                                  binding.FLUID_BC_COUPLED if side == 0 else binding.FLUID_BC_WALL))

    def live_before():
        """Ghost state of the band from the fluid rows next to it (section 4.2), and the mark of section 4.1."""
        g, nyf = w.nghost_y, live["nyf"]
        for side in (0, 1):
            rows = slice(2 + nyf - g, 2 + nyf) if side == 0 else slice(2, 2 + g)
            for s in range(ns):
                tmp = live["b5"][s][side]
                binding.vlasov_fluid_to_boundary(live["U"][side][s][:, rows].contiguous(), live["m"][s], tmp)
                lay = torch.flip(tmp, dims=[1]).contiguous() if side == 0 else tmp      # ghost layers count outward
                ctx.vlasov_set_boundary(s, side, inputs.BC_FLUID, lay)
        ctx.vlasov_fluid_boundary_mark()

    def live_after():
        """Ghost rows of the fluid blocks from the band's border rows at the Runge-Kutta stage times, then the fluid steps."""
        for side in (0, 1):
            pick = slice(0, 2) if side == 0 else slice(1, 3)
            for k, th in enumerate((0.0, 1.0, 0.5)):
                for s in range(ns):
                    ctx.vlasov_fluid_boundary(s, side, th, live["mb"])
                    binding.vlasov_fluid_from_moments(live["mb"][:, pick].contiguous(), live["m"][s], live["gh"][side][k, s])
            gl, gh = (None, live["gh"][0]) if side == 0 else (live["gh"][1], None)
            live["blk"][side].vlasov_fluid_step(w.dt, live["U"][side], live["E"][side], live["B"][side], gl, gh)

    def cycle():
        if live is not None:
            live_before()
            ctx.vlasov_cycle(w.dt, w.nsub, Ed, Bd)
            live_after()
        else:
            set_fluid()
            ctx.vlasov_cycle(w.dt, w.nsub, Ed, Bd)

    def set_fluid():
        if fluid is not None:
            st = fluid[step_no[0] % len(fluid)]
            for s in range(ns):
                for side in (0, 1):
                    ctx.vlasov_set_boundary(s, side, inputs.BC_FLUID, st[s][side])
        step_no[0] += 1

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    # ---- device-resident leg: `value` -------------------------------------------------------
    # Timed with the library's per-launch event pairs OFF.  REPS repetitions of the timed block (each EXACTLY
    # args.steps cycles between barrier + synchronize); the reported time is the median.
    for _ in range(args.warmup):
        cycle()
    ctx.vlasov_check()
    ctx.vlasov_timing_enable(False)
    sampler = ClockSampler(local) if rank == 0 else None
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rep_ms, launches = [], 0
    t_wall0 = time.time()
    for _ in range(max(1, args.reps)):
        barrier()
        l0 = ctx.launch_count()
        ev0.record(stream)
        for _ in range(args.steps):
            cycle()
        ev1.record(stream)
        barrier()
        launches = ctx.launch_count() - l0
        rep_ms.append(max_over_ranks(ev0.elapsed_time(ev1), dist, device))
    t_wall1 = time.time()
    ctx.vlasov_check()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    ms = float(np.median(rep_ms))
    cells = w.interior_cells * nz
    value = whole_job_value(cells, args.steps, ms, world)

    # ---- the same number of steps again with an event pair around every launch: the per-kernel table ----
    ctx.vlasov_timing_enable(True)
    barrier()
    ev0.record(stream)
    for _ in range(args.steps):
        cycle()
    ev1.record(stream)
    barrier()
    ms_instr = ev0.elapsed_time(ev1)
    per_kind = ctx.vlasov_timing_read()
    ctx.vlasov_timing_enable(False)

    # ---- end-to-end leg: HOST buffers through the C ABI (vlasov_cycle_host) -----------------
    ncell = w.ny_g * w.nx * nz
    Eh = torch.from_numpy(E0.copy()).pin_memory()
    Bh = torch.from_numpy(B0.copy()).pin_memory()
    Mh = torch.empty((ns, 10, nz * w.ny_g, w.nx), dtype=torch.float64).pin_memory()
    Eh.copy_(Ed.cpu()); Bh.copy_(Bd.cpu())
    e2e_steps = max(1, min(args.steps, 10))
    set_fluid()
    ctx.vlasov_cycle_host(w.dt, w.nsub, Eh, Bh, Mh)
    barrier()
    ev0.record(stream)
    for _ in range(e2e_steps):
        set_fluid()
        ctx.vlasov_cycle_host(w.dt, w.nsub, Eh, Bh, Mh)
    ev1.record(stream)
    barrier()
    ms_e = ev0.elapsed_time(ev1)
    ms_e = max_over_ranks(ms_e, dist, device)
    e2e = whole_job_value(cells, e2e_steps, ms_e, world)
    h2d = 6 * ncell * 8
    d2h = (6 + 10 * ns) * ncell * 8
    if not np.isfinite(Mh.numpy()).all():
        raise SystemExit("bench.py: non-finite moments")

    if rank != 0:
        ctx.close()
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (CUDA-event pairs around every launch, timed region) ----
    peak, peak_src = peaks()
    cells_all = sum(nz * w.ny_g * w.nx * s.ncell_v for s in w.species) / ns  # ghost-inclusive, per species launch
    cells_int = cells / ns                                                     # interior rows only
    kinds = {}
    tot_ms = sum(v[0] for v in per_kind.values())
    for k, (kms, cnt) in per_kind.items():
        if cnt == 0:
            continue
        ent = {"ms_per_step": kms / args.steps, "launches_per_step": cnt / args.steps, "share": kms / tot_ms}
        if k in BYTES_PER_CELL:
            # the fused spatial stages cover the interior rows (ghost rows are Dirichlet data, R16); the velocity sweeps and
            # the moments pass cover every row.  Ghost-fill launches have their own kinds (ghost_*) and are not mixed in.
            ncells = cells_int if k in ("sweep_xy", "sweep_yx") else cells_all
            ent["gbs"] = BYTES_PER_CELL[k] * ncells * cnt / (kms * 1e-3) / 1e9
            ent["frac_of_peak"] = ent["gbs"] / peak
            ent["cells_per_launch"] = ncells
        kinds[k] = ent
    ghost_ms = sum(v["ms_per_step"] for k, v in kinds.items() if k.startswith("ghost_"))
    dom = max((k for k in kinds if "gbs" in kinds[k]), key=lambda k: kinds[k]["share"], default=None)
    roofline = None
    if dom is not None:
        d = kinds[dom]
        roofline = {"kernel": dom, "bound": "hbm", "achieved": d["gbs"], "peak": peak, "unit": "GB/s",
                    "frac": d["gbs"] / peak, "traffic": None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": BYTES_PER_CELL[dom] * d["cells_per_launch"],
                    "avg_launch_ms": d["ms_per_step"] / d["launches_per_step"], "share_of_step": d["share"]}
        tr = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tr):
            with open(tr) as fh:
                tj = json.load(fh)
            if tj.get("workload") == w.name and dom in tj.get("dram_bytes_per_launch", {}):
                roofline["traffic"] = tj["dram_bytes_per_launch"][dom]
                roofline["traffic_source"] = tj.get("source")
            wi = tj.get("warp_instructions_per_launch", {}).get(dom) if tj.get("workload") == w.name else None
            if wi and clocks and clocks.get("sm_mhz"):
                # second roof of the same kernel: warp-instructions issued per second against 4 schedulers x SMs x
                # the SM clock sampled during the timed region (the vy+vz kernel is issue-bound)
                sms = torch.cuda.get_device_properties(0).multi_processor_count
                ipeak = 4.0 * sms * clocks["sm_mhz"] * 1e6
                iach = wi / (roofline["avg_launch_ms"] * 1e-3)
                roofline["issue"] = {"achieved": iach / 1e9, "peak": ipeak / 1e9, "unit": "G warp-instructions/s",
                                     "frac": iach / ipeak, "warp_instructions_per_launch": wi,
                                     "source": tj.get("warp_instructions_source")}
    # f-sized passes of one step and species (the ghost_* kinds are overhead of the FLUID border, not passes); the
    # one-direction sweeps count only when no fused stage ran.
    fused = any(k in kinds for k in ("sweep_xy", "sweep_yx"))

    def full_passes(k, v):
        n = v["launches_per_step"] / ns
        if k in ("sweep_x", "sweep_y"):
            return 0.0 if fused else n
        return n

    step_bytes = sum(BYTES_PER_CELL[k] * v["cells_per_launch"] * full_passes(k, v) * ns
                     for k, v in kinds.items() if k in BYTES_PER_CELL)
    pass_bytes = step_bytes / cells           # per interior cell-update

    # ---- the oracle timed beside it (reported baseline only) --------------------------------
    cpu = None
    if not args.no_cpu_baseline and nz == 1:        # (the oracle leg samples 2D cuts; the 3D workload is timed without it)
        v, _, cores, sample, _ = oracle_leg(make_workload(args.workload), steps=50, warmup=1, budget_s=args.cpu_budget)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "cpu_model": cpu_model(), "kind": "oracle", "sample": sample}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "timing": {"what": "median of the repetitions; each repetition times exactly `steps` cycles, per-launch event pairs off",
                   "repetitions": len(rep_ms), "ms_per_step_each": [m / args.steps for m in rep_ms],
                   "ms_per_step_with_per_launch_events": ms_instr / args.steps},
        "dtype": "f64", "data": "synthetic (seeded GEM Harris-sheet profiles + hash noise, DESIGN.md 'Input recipe')",
        "config": {"workload": w.name, "nx": w.nx, "ny": w.ny, "nz": nz, "nghost_y": w.nghost_y,
                   "nv": list(w.species[0].nv), "species": ns, "dt": w.dt, "maxwell_nsub": w.nsub,
                   "interior_cells_per_step": cells,
                   "fluid": (args.fluid if fluid is not None else None),
                   "order": "VXV (PAPER.md:420; moments fused into the last vy+vz pass)" if args.order == "vxv" else "XVX (eq. 22)", "parallelism": "replicas only" if world > 1 else "single GPU",
                   "l2": f"inputs larger than L2: {sum(f.numel() for f in fs) * 8 / 1e9:.2f} GB of f streamed by every pass (L2 126 MB)"},
        "clocks": clocks,
        "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
                "ms_per_step": ms_e / e2e_steps,
                "what": "vlasov_cycle_host: E,B from pinned host memory each step, E,B and all moments back; f resident (PAPER.md:86)"},
        "gpu_launches": launches,
        "roofline": roofline,
        "step_hbm": {"algorithmic_bytes_per_cell_update": pass_bytes,
                     "achieved_gbs": step_bytes * args.steps / (ms * 1e-3) / 1e9,
                     "note": "sum over the step's f-sized passes (cells each pass covers; ghost_* launches not credited) / step time"},
        "kernels": kinds,
        "cpu_baseline": cpu,
    }
    if fluid is not None:
        # what the FLUID border costs (ghost fill: edge moments + table + three remaps of the ghost
        # rows; x sweeps of the ghost rows), as a share of the per-launch-timed step
        out["ghost_fill_share_of_step"] = (ghost_ms + kinds.get("ghost_table", {}).get("ms_per_step", 0.0)) / (tot_ms / args.steps)
    out["step_hbm"]["frac_of_peak"] = out["step_hbm"]["achieved_gbs"] / peak
    # SURVEY.md 8(d) reporting rule: the same figure against the nominal 8 TB/s, and the "useful" fraction that
    # credits only the 48 B per cell-update of the 3-pass Strang floor (x/2 y/2, V, y/2 x/2 each once through HBM)
    out["step_hbm"]["frac_of_nominal_8tbs"] = out["step_hbm"]["achieved_gbs"] / 8000.0
    out["step_hbm"]["useful_frac_48B"] = 48.0 * value / max(world, 1) / 1e9 / peak
    print(json.dumps(out))
    ctx.close()
    if dist is not None:
        dist.destroy_process_group()


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = make_workload(args.workload)
    v, ms, cores, sample, done = oracle_leg(w, steps=args.steps, warmup=args.warmup, budget_s=args.ref_budget)
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": done,
           "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic (seeded GEM Harris-sheet profiles + hash noise)",
           "config": {"workload": w.name, "sample": sample},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "cpu_model": cpu_model(), "kind": "oracle", "sample": sample},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
           "gpu_launches": 0}
    print(json.dumps(out))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--reps", type=int, default=5, help="repetitions of the timed block of --steps cycles (median reported)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="gem128")
    ap.add_argument("--fluid", default="seeded", choices=["seeded", "live"],
                    help="band workload: ghost state from seeded fluid moments (BASELINE config 4) or from two live five-moment fluid blocks")
    ap.add_argument("--order", default="xvx", choices=["xvx", "vxv"], help="Strang order of the Vlasov step (R2); xvx is the benchmark")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=20.0, help="seconds of oracle time for the cpu_baseline leg")
    ap.add_argument("--ref-budget", type=float, default=150.0, help="seconds of oracle time for --impl reference")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        reference_arm(args)
    else:
        gpu_arm(args)


if __name__ == "__main__":
    main()
