#!/usr/bin/env python
"""bench.py -- ANI-2x energy+force MD throughput on B200 (BASELINE.json metric), one JSON line.

Workload (BASELINE.json configs[2], the configuration the metric is quoted on): 32,768 rigid-geometry waters
= 98,304 atoms in a periodic cube L = 99.4 A, seeded Maxwell-Boltzmann velocities at 300 K, velocity Verlet at
dt = 0.5 fs, Verlet skin 0.5 A with the displacement-triggered rebuild, one network of seeded Xavier weights,
fp32.  A "step" is one MD step = one pass of all five stages (neighbour rebuild when triggered, AEV, MLPs,
reverse pass + force scatter, integrator).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--mm-mode 0|1|2]

N > 1 (torchrun): the path does not shard (north_star: one GPU, no collectives) -> N independent replicas,
"scaling": "weak", value = sum of atom-steps over ranks / max time over ranks.
--impl reference: the fp64 CPU oracle (oracle/) as it stands on the host cores, on bounded samples.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "ANI-2x energy+force MD atom-steps/s (0.5 fs velocity Verlet, 98,304-atom water box)"
UNIT = "atom-steps/s"
DT_FS, SKIN, T_KELVIN = 0.5, 0.5, 300.0
N_WATERS = 32768
MM_NAMES = ["fp32_simt", "3xtf32_tcgen05", "tf32_tcgen05", "fp64_simt", "3xf16_tcgen05_fused"]
TRAJ_MAX = 1050   # longest stretch of one trajectory (steps): BASELINE.json's 1000-step run + the default warm-up
BOX_L = 99.4


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sus=d["bf16_tflops_sustained"],
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sus=1400.0, sm_max_mhz=1965.0, source="fallback")


class ClockSampler(threading.Thread):
    """nvidia-smi clocks/throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 7:
                    self.rows.append(f)
            except Exception:
                pass
            self.stop_flag.wait(0.2)

    def summary(self):
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]),
                "power_w_max": max(float(r[2]) for r in self.rows), "samples": len(self.rows), "reasons": reasons}


def oracle_model(n_nets=1):
    from oracle import nnp_oracle as orc
    from paper_2405_01491_b200 import inputs
    consts = inputs.ani2x_constants()
    params = inputs.make_weights(inputs.SEED0, n_nets, last_layer_scale=inputs.FORCE_SCALE_MD)
    return orc, orc.OracleModel(consts, inputs.WIDTHS, params, n_nets)


def time_oracle_md(n_waters, n_steps, seed, L=None):
    """Oracle MD on a water box of the workload's density.  orc.md evaluates the initial forces and then one
    force evaluation per step, so the timed work is n_steps + 1 step-equivalents (the integrator itself is
    negligible).  Returns (atom-steps, seconds, cores)."""
    from paper_2405_01491_b200 import inputs
    orc, om = oracle_model()
    sp, xyz, box = inputs.water_box(n_waters, L, seed=seed)
    v = inputs.maxwell_boltzmann(sp, T_KELVIN)
    t0 = time.perf_counter()
    orc.md(om, sp, xyz, v, inputs.MASS, box, DT_FS, inputs.ACCEL_CONV, n_steps, skin=SKIN,
           nbr_method=1 if n_waters >= 216 else 0)
    dt = time.perf_counter() - t0
    return len(sp) * (n_steps + 1), dt, orc.num_threads()


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    K, W = args.steps, args.warmup
    # calibrate on the smallest box, then pick the largest sample that keeps the run within ~3 minutes
    a, t, cores = time_oracle_md(64, 1, 1)
    rate = a / t                          # atom-steps/s
    budget = 150.0 / max(1, K + W + 1)
    n_waters = 64
    for cand in (216, 512, 1000, 4096, N_WATERS):
        if cand * 3 / rate <= budget:
            n_waters = cand
    atoms, secs, cores = time_oracle_md(n_waters, K + W, 2, BOX_L if n_waters == N_WATERS else None)
    secs_timed = secs * K / (K + W + 1)
    value = n_waters * 3 * K / secs_timed
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": K,
            "warmup": W, "ms_per_step": 1e3 * secs_timed / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "water_98304_md (configs[2]); each step = one oracle MD step of a %d-atom water box "
                                   "of the same density" % (n_waters * 3), "dt_fs": DT_FS, "skin_A": SKIN},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": "%d velocity-Verlet steps of a %d-atom water box (same density, same model)" %
                                       (K, n_waters * 3)},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def run_eval_config(args):
    """--config 1|2|4|5: the other BASELINE.json workloads.  A step = nnp_build_neighbors(skin 0) + nnp_energy_forces on
    inputs resident in HBM; same JSON line as the headline, roofline entry for the dominant stage."""
    import torch
    from paper_2405_01491_b200 import eval_timing, inputs, nnp
    import __graft_entry__
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:          # these lines are single-GPU measurements
        return 0
    torch.cuda.set_device(0)
    dev = torch.device("cuda", 0)
    __graft_entry__.build()
    nnp.lib()
    name, n_nets, sp, xyz, box, offs = eval_timing._workload(args.config)
    n = len(sp)
    n_mols = 1 if offs is None else len(offs) - 1
    consts = inputs.ani2x_constants()
    params = inputs.make_weights(inputs.SEED0 + args.config, n_nets, last_layer_scale=args.force_scale)
    p, keep = nnp.make_params(consts, inputs.WIDTHS, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=n_nets, mm_mode=args.mm_mode)
    stream = torch.cuda.Stream(device=dev)
    ctx = nnp.nnp_create(p, n, n_mols, 0, stream.cuda_stream)
    K, W = args.steps, args.warmup
    d_sp = torch.as_tensor(np.asarray(sp, dtype=np.int32), device=dev)
    d_x = torch.as_tensor(np.asarray(xyz, dtype=np.float32), device=dev).contiguous()
    d_mo = None if offs is None else torch.as_tensor(np.asarray(offs, dtype=np.int32), device=dev)
    d_E = torch.zeros(n_mols, dtype=torch.float64, device=dev)
    d_F = torch.zeros((n, 3), dtype=torch.float32, device=dev)
    flush = torch.empty(256 * 2**20, dtype=torch.uint8, device=dev)      # > the 126 MB L2
    torch.cuda.synchronize()
    nnp.nnp_set_system(ctx, n, d_sp, d_x, box, n_mols, d_mo)

    def step():
        nnp.nnp_build_neighbors(ctx, 0.0)
        nnp.nnp_energy_forces(ctx, d_E, d_F)

    with torch.cuda.stream(stream):
        for _ in range(W):
            step()
        nnp.nnp_sync(ctx)
        sampler = ClockSampler(0)
        sampler.start()
        l0 = nnp.nnp_launch_count(ctx)
        evs = []
        for _ in range(K):                      # L2 flushed between the timed iterations (outside the event pairs)
            flush.fill_(1)
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            step()
            b.record(stream)
            evs.append((a, b))
        nnp.nnp_sync(ctx)
        launches = nnp.nnp_launch_count(ctx) - l0
        sampler.stop_flag.set()
        ms = sum(a.elapsed_time(b) for a, b in evs)
        # counts of the method's own work, from the lists (skin 0: the rows are the in-cutoff neighbours)
        d_c = torch.zeros(n, dtype=torch.int32, device=dev)
        d_l = torch.zeros((n, 4), dtype=torch.int32, device=dev)
        nnp.nnp_get_neighbors(ctx, 0, d_c, d_l, 4)
        n_rad = int(d_c.sum().item())
        nnp.nnp_get_neighbors(ctx, 1, d_c, d_l, 4)
        ca = d_c.to(torch.int64)
        n_tri = int((ca * (ca - 1) // 2).sum().item())
        # per-stage pass (untimed)
        P = min(args.profile_steps, 20)
        nnp.nnp_profile(ctx, 1)
        for _ in range(P):
            flush.fill_(1)
            step()
        stage_ms, stage_n = nnp.nnp_profile_read(ctx)
        nnp.nnp_profile(ctx, 0)
    kact = nnp.nnp_aev_active_columns(ctx)
    sampler.join(timeout=2)
    # ---- end to end: host species / coordinates / offsets in, energies and forces out, every step (pinned buffers)
    h_sp = torch.as_tensor(np.asarray(sp, dtype=np.int32)).pin_memory()
    h_x = torch.as_tensor(np.asarray(xyz, dtype=np.float32)).contiguous().pin_memory()
    h_mo = None if offs is None else torch.as_tensor(np.asarray(offs, dtype=np.int32)).pin_memory()
    h_E = torch.zeros(n_mols, dtype=torch.float64).pin_memory()
    h_F = torch.zeros((n, 3), dtype=torch.float32).pin_memory()
    Ke = min(K, args.e2e_steps)
    for _ in range(3):
        nnp.nnp_energy_forces_host(ctx, n, h_sp, h_x, box, n_mols, h_mo, 0.0, h_E, h_F)
    torch.cuda.synchronize(dev)
    t0 = time.perf_counter()
    for _ in range(Ke):
        nnp.nnp_energy_forces_host(ctx, n, h_sp, h_x, box, n_mols, h_mo, 0.0, h_E, h_F)
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0
    nnp.nnp_destroy(ctx)

    pk, clocks = peaks(), sampler.summary()
    build_ms = stage_ms[1] / max(1, stage_n[1])
    per_stage = {nnp.STAGE_NAMES[k]: (stage_ms[k] / stage_n[k] if stage_n[k] else 0.0) for k in range(nnp.NNP_N_STAGES)}
    per_stage = {k: v for k, v in per_stage.items() if k not in ("kick_drift", "kick_ekin")}
    per_stage["neighbor_build"] = (ms / K) - sum(v for k, v in per_stage.items() if k != "neighbor_build")   # events cover E+F only
    del build_ms
    tot = sum(per_stage.values())
    mlp_ms = sum(v for k, v in per_stage.items() if k.startswith("mlp"))
    groups = {"mlp_all_layers": mlp_ms, **{k: v for k, v in per_stage.items() if not k.startswith("mlp")}}
    dom = max(groups, key=groups.get)
    kpad = (kact + 31) // 32 * 32
    fp32_peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
    if dom == "mlp_all_layers":
        counts = np.bincount(sp, minlength=7)
        Wd = inputs.WIDTHS
        macs = sum(int(counts[s]) * (kpad * int(Wd[s, 1]) + int(Wd[s, 1]) * int(Wd[s, 2]) + int(Wd[s, 2]) * int(Wd[s, 3]) + int(Wd[s, 3]))
                   for s in range(7))
        ach = 2.0 * 2.0 * macs * n_nets / (mlp_ms * 1e-3) / 1e12           # forward + input gradient
        peak = pk["bf16_sus"] if args.mm_mode == 4 else pk["bf16_sus"] * 0.5 if args.mm_mode in (1, 2) else fp32_peak   # fp16 operands: the bf16 rate; tf32: half of it
        roof = {"kernel": "mlp_all_layers (mm_mode 4: fused chain [+ layer 1 / dE/dG launches]; else 6 grouped GEMM launches per network batch)",
                "bound": "tensor" if args.mm_mode in (1, 2, 4) else "alu",
                "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
                "peak_source": "%s sustained bf16 cuBLAS%s; fp32-equivalent flops counted once (the split issues 3 MMAs per product)" % (pk["source"], "" if args.mm_mode == 4 else " x 0.5")}
    elif dom in ("aev_forward", "aev_backward_scatter"):
        flop = {"aev_forward": n_rad * 16 * 6 + n_tri * 150.0, "aev_backward_scatter": n_rad * 16 * 10 + n_tri * 330.0}[dom]
        ach = flop / (groups[dom] * 1e-3) / 1e12
        roof = {"kernel": dom, "bound": "alu", "achieved": ach, "peak": fp32_peak, "unit": "TFLOP/s", "frac": ach / fp32_peak,
                "traffic": None, "peak_source": "148 SM x 128 lanes x 2 x clocks.max.sm; work counted from the lists: %d radial terms, "
                "%d triplets" % (n_rad, n_tri)}
    else:
        byts = {"neighbor_build": (n_rad + int(ca.sum().item())) * 4.0 + n * 48.0, "energy_sum": n * 12.0}.get(dom, n * 64.0)
        ach = byts / (groups[dom] * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": pk["hbm"], "unit": "GB/s", "frac": ach / pk["hbm"],
                "traffic": None, "peak_source": pk["source"]}
    roof["traffic"] = traffic_from_profiles(dom, "config%d_mm%d" % (args.config, args.mm_mode))
    roof["stage_ms"] = {k: round(v, 4) for k, v in per_stage.items()}
    roof["stage_share"] = {k: round(v / tot, 4) for k, v in per_stage.items()} if tot else {}
    roof["stage_ms_source"] = "separate untimed pass of %d steps with CUDA events around every stage; neighbor_build = step - rest" % P
    line = {"metric": "ANI-2x energy+force atom-steps/s (one list build + one energy/force evaluation per step, %s)" % name,
            "value": n * K / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": K, "warmup": W, "ms_per_step": ms / K,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": name, "atoms": n, "structures": n_mols, "n_nets": n_nets, "aev_active_columns": kact,
                       "mm_mode": MM_NAMES[args.mm_mode],
                       "us_per_evaluation": 1e3 * ms / K, "force_scale": args.force_scale,
                       "radial_terms": n_rad, "triplets": n_tri,
                       "launch_path": "kernel_by_kernel (nnp_build_neighbors + nnp_energy_forces per step)",
                       "l2_policy": "L2 flushed (256 MB write) between timed iterations, outside the event pairs",
                       "parallelism": "single GPU"},
            "clocks": clocks,
            "e2e": {"value": n * Ke / e2e_s, "unit": UNIT, "steps": Ke,
                    "h2d_bytes_per_step": n * 16 + (4 * (n_mols + 1) if offs is not None else 0),
                    "d2h_bytes_per_step": n * 12 + 8 * n_mols + 12,
                    "api": "nnp_energy_forces_host (pinned host species, xyz[, offsets] up; energies, forces down; every step)"},
            "gpu_launches": launches, "roofline": roof}
    if not args.no_cpu_baseline:
        orc, om = oracle_model(1)
        om = orc.OracleModel(consts, inputs.WIDTHS, inputs.make_weights(inputs.SEED0 + args.config, 1, last_layer_scale=args.force_scale), 1)
        t0 = time.perf_counter()
        orc.energy_forces(om, sp, xyz, box, offs, nbr_method=1 if (box is not None and n >= 600) else 0)
        secs = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": n / secs, "unit": UNIT, "cores": orc.num_threads(), "kind": "oracle",
                                "sample": "one energy+force evaluation of the whole workload with ONE network (fp64 oracle, OpenMP; "
                                          "the workload's ensemble has %d)" % n_nets}
    print(json.dumps(line))
    return 0


# ---- the N > 1 path ("replicas only": independent trajectories, no data-path collective).  The three pieces of host
# logic it consists of are functions of their own so that tests/test_multi_rank.py can run them under gloo on CPU.
def replica_seed(base, rank):
    """Every rank simulates its own seeded system."""
    return base + 1000 * rank


def max_over_ranks(values, dist, device):
    """Timings are combined as the MAX over ranks (the job is as slow as its slowest replica)."""
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    if dist:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t.tolist()]


def whole_job_rate(world, atoms_per_rank, steps, ms_max):
    """Aggregate atom-steps/s of all replicas over the slowest replica's time (weak scaling)."""
    return world * atoms_per_rank * steps / (ms_max * 1e-3)


def run_ours(args):
    import torch
    from paper_2405_01491_b200 import inputs, nnp
    import __graft_entry__
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if rank == 0:
        __graft_entry__.build()
    if dist:
        dist.barrier()
    nnp.lib()          # fails loudly if the CUDA library is missing

    # ---- workload: replica `rank` gets its own seed (independent trajectories, "replicas only")
    sp, xyz, box = inputs.water_box(args.waters, BOX_L if args.waters == N_WATERS else None, seed=replica_seed(inputs.SEED0 + 3, rank))
    n = len(sp)
    vel = inputs.maxwell_boltzmann(sp, T_KELVIN, seed=inputs.SEED0 + 103 + 1000 * rank)
    consts = inputs.ani2x_constants()
    params = inputs.make_weights(inputs.SEED0, 1, last_layer_scale=args.force_scale)
    p, keep = nnp.make_params(consts, inputs.WIDTHS, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=1, mm_mode=args.mm_mode)
    stream = torch.cuda.Stream(device=dev)
    ctx = nnp.nnp_create(p, n, 1, local, stream.cuda_stream)

    d_sp = torch.as_tensor(sp, device=dev)
    d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
    d_v = torch.as_tensor(vel.astype(np.float32), device=dev)
    K, W = args.steps, args.warmup

    def barrier():
        if dist:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident run (value)
    o_ep = torch.zeros(1, dtype=torch.float64, device=dev)
    o_ek = torch.zeros(1, dtype=torch.float64, device=dev)
    o_nr = torch.zeros(1, dtype=torch.int32, device=dev)

    def restart():
        """(Re)loads the seeded start of the trajectory.  The random-weight model is not a bound liquid: the box heats up
        and collapses after ~1 ps (NNP_ECAPACITY near 2000 steps), so no trajectory is run past TRAJ_MAX steps -
        BASELINE.json's run length is 1000.  A run with --steps > TRAJ_MAX restarts inside the timed region (one upload-free
        nnp_set_system + nnp_md_init = one list build and one force evaluation per restart, < 0.2 % of the segment)."""
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box)
        nnp.nnp_md_init(ctx, d_v, DT_FS, SKIN)
        if args.langevin > 0:  # the paper's benchmarks run Langevin 300 K; not the default workload
            nnp.nnp_md_set_langevin(ctx, args.langevin, inputs.KB * T_KELVIN, inputs.SEED0 + 7 + rank)

    def read_state():
        nnp.nnp_get_state(ctx, None, None, o_ep, o_ek, o_nr)
        nnp.nnp_sync(ctx)
        return float(o_ep.item() + o_ek.item()), int(o_nr.item()), float(o_ek.item())

    st = {"since": 0, "rebuilds": 0, "restarts": 0, "e0": 0.0, "nr0": 0, "ek0": 0.0}

    def advance(n_steps):
        """n_steps of MD, restarting the trajectory whenever it has reached TRAJ_MAX steps (never with the defaults)."""
        left = n_steps
        while left > 0:
            if st["since"] >= TRAJ_MAX:
                st["rebuilds"] += read_state()[1] - st["nr0"]
                restart()
                st["restarts"] += 1
                st["e0"], st["nr0"], st["ek0"] = read_state()
                st["since"] = 0
            seg = min(left, TRAJ_MAX - st["since"])
            nnp.nnp_md_step(ctx, seg)
            left -= seg
            st["since"] += seg

    restart()
    advance(W)
    nnp.nnp_sync(ctx)
    st["e0"], st["nr0"], st["ek0"] = read_state()
    st["rebuilds"], st["restarts"] = 0, 0
    nnp.nnp_profile(ctx, 0)          # no instrumentation inside the timed region: every timed step is one CUDA-graph launch
    sampler = ClockSampler(local)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = nnp.nnp_launch_count(ctx)
    barrier()
    sampler.start()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        advance(K)
        ev1.record(stream)
    barrier()
    sampler.stop_flag.set()
    launches = nnp.nnp_launch_count(ctx) - l0   # kernels outside the conditional rebuild; + 8 per rebuild below
    kact = nnp.nnp_aev_active_columns(ctx)
    ms = ev0.elapsed_time(ev1)
    nnp.nnp_sync(ctx)
    e_end, nr_end, ek_end = read_state()
    e_start, ek_start = st["e0"], st["ek0"]          # energy drift and temperatures: over the last trajectory segment
    n_rebuilds, n_restarts = st["rebuilds"] + nr_end - st["nr0"], st["restarts"]
    sampler.join(timeout=2)

    # ---- per-stage timings: a SEPARATE, untimed pass (CUDA events around every stage need the kernel-by-kernel launch
    # path; the timed region above ran the graph path only).  Same trajectory, restarted so it stays on its healthy stretch.
    P = args.profile_steps
    restart()
    nnp.nnp_md_step(ctx, 20)
    nnp.nnp_sync(ctx)
    nnp.nnp_profile(ctx, 1)
    nnp.nnp_md_step(ctx, P)
    stage_ms, stage_n = nnp.nnp_profile_read(ctx)
    nnp.nnp_profile(ctx, 0)
    st["since"] = 20 + P

    # ---- end-to-end through the host entry point: every step uploads x,v and downloads x,v,E (pinned memory)
    Ke = min(K, args.e2e_steps, TRAJ_MAX // 2)
    if st["since"] + Ke + 3 > TRAJ_MAX + TRAJ_MAX // 4:   # keep the end-to-end leg on a healthy stretch of the trajectory as well
        restart()
        nnp.nnp_md_step(ctx, 20)
        nnp.nnp_sync(ctx)
    h_x = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    h_v = torch.empty((n, 3), dtype=torch.float32).pin_memory()
    h_e = torch.zeros(2, dtype=torch.float64).pin_memory()
    tmp_x, tmp_v = torch.zeros_like(d_x), torch.zeros_like(d_v)
    nnp.nnp_get_state(ctx, tmp_x, tmp_v, None, None, None)
    nnp.nnp_sync(ctx)
    h_x.copy_(tmp_x)
    h_v.copy_(tmp_v)
    for _ in range(3):
        nnp.nnp_md_step_host(ctx, h_x, h_v, 1, h_e[0:1], h_e[1:2])
    barrier()
    t0 = time.perf_counter()
    for _ in range(Ke):
        nnp.nnp_md_step_host(ctx, h_x, h_v, 1, h_e[0:1], h_e[1:2])
    torch.cuda.synchronize(dev)
    e2e_s = time.perf_counter() - t0

    # ---- max over ranks
    ms_max, e2e_ms_max = max_over_ranks([ms, e2e_s * 1e3], dist, dev)
    nnp.nnp_destroy(ctx)
    if rank != 0:
        if dist:
            dist.destroy_process_group()
        return 0

    pk = peaks()
    clocks = sampler.summary()
    value = whole_job_rate(world, n, K, ms_max)
    steps_per_s = K / (ms_max * 1e-3)
    per_stage = {nnp.STAGE_NAMES[k]: (stage_ms[k] / stage_n[k] if stage_n[k] else 0.0) for k in range(nnp.NNP_N_STAGES)}
    tot_stage = sum(per_stage.values())
    dom = max(per_stage, key=per_stage.get)
    kpad = (kact + 31) // 32 * 32
    roof = roofline_for(dom, per_stage[dom], n, sp, args.mm_mode, pk, clocks, kpad)
    roof["stage_ms_source"] = "separate untimed pass of %d kernel-by-kernel steps with CUDA events around every stage" % P
    roof["stage_ms"] = {k: round(v, 4) for k, v in per_stage.items()}
    roof["stage_share"] = {k: round(v / tot_stage, 4) for k, v in per_stage.items()} if tot_stage else {}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
        "ms_per_step": ms_max / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": "water_%d_md (BASELINE configs[2])" % n if args.waters == N_WATERS else "water_%d_md" % n,
                   "atoms": n, "box_A": float(box[0]), "dt_fs": DT_FS, "skin_A": SKIN, "n_nets": 1,
                   "integrator": "langevin_baoab gamma=%g/fs" % args.langevin if args.langevin > 0 else "velocity_verlet",
                   "mm_mode": MM_NAMES[args.mm_mode],
                   "force_scale": args.force_scale, "ns_per_day": steps_per_s * DT_FS * 1e-6 * 86400,
                   "rebuilds_in_timed_region": n_rebuilds, "trajectory_restarts_in_timed_region": n_restarts,
                   "temperature_K_end": 2 * ek_end / (3 * n * inputs.KB), "temperature_K_start": 2 * ek_start / (3 * n * inputs.KB),
                   "etot_drift_rel": (e_end - e_start) / abs(e_start) if e_start else None,
                   "aev_active_columns": kact,
                   "launch_path": "kernel_by_kernel" if os.environ.get("NNP_NO_GRAPH") == "1" else
                                  "cuda_graph (one graph launch per step, rebuild inside a conditional node)",
                   "l2_policy": "inputs larger than L2: per step the kernels stream G (%d MB), the activations (%d MB%s) and "
                                "the neighbour rows (%d MB); no flush needed"
                                % (n * kpad * 4 // 2**20, n * (448 if args.mm_mode == 4 else 608) * 4 // 2**20,
                                   ": only h1 and h2 leave the SM in mm_mode 4" if args.mm_mode == 4 else "", n * 224 * 4 // 2**20),
                   "parallelism": "replicas only" if world > 1 else "single GPU"},
        "clocks": clocks,
        "e2e": {"value": world * n * Ke / (e2e_ms_max * 1e-3), "unit": UNIT, "steps": Ke,
                "h2d_bytes_per_step": 2 * n * 12, "d2h_bytes_per_step": 2 * n * 12 + 40,  # x, v and one packed (epot, ekin, 3 flag words) record
                "api": "nnp_md_step_host (pinned host x,v up; x,v,epot,ekin down; every step)"},
        "gpu_launches": launches + 8 * n_rebuilds,
        "roofline": roof,
    }
    if world == 1 and not args.no_cpu_baseline:
        atoms, secs, cores = time_oracle_md(args.cpu_waters, args.cpu_steps, inputs.SEED0 + 3,
                                            BOX_L if args.cpu_waters == N_WATERS else None)
        line["cpu_baseline"] = {"value": atoms / secs, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": "%d velocity-Verlet steps (%d force evaluations) of %s (fp64 oracle, OpenMP)" %
                                          (args.cpu_steps, args.cpu_steps + 1,
                                           "the workload itself: the same seeded 98,304-atom water box" if args.cpu_waters == N_WATERS
                                           else "a %d-atom water box of the same density and model" % (args.cpu_waters * 3))}
    print(json.dumps(line))
    if dist:
        dist.destroy_process_group()
    return 0


TRAFFIC_FILE = os.path.join(ROOT, "profiles", "traffic_ncu.csv")


def kernel_source_hash():
    """sha256 over the CUDA sources: the stamp that ties an ncu capture to the kernels it was taken from (the GPU box has
    no .git, so the commit id itself cannot be checked there)."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2405_01491_b200", "csrc")
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")) and f != "no_alloc.cu":  # (nnp_neighbors_no_alloc: never called by bench.py)
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def traffic_from_profiles(stage, workload_key):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch [bytes] of the stage's kernel from the committed `ncu --set
    full` capture (profiles/traffic_ncu.csv: '# source=<hash>' header, rows workload,stage,read_bytes,write_bytes).
    None when there is no capture of this workload or the kernels have changed since it was taken."""
    if not os.path.exists(TRAFFIC_FILE):
        return None
    stamp, rows = None, {}
    for ln in open(TRAFFIC_FILE):
        ln = ln.strip()
        if ln.startswith("#"):
            if "source=" in ln:
                stamp = ln.split("source=")[1].split()[0]
            continue
        f = ln.split(",")
        if len(f) >= 4 and f[0] != "workload":
            rows[(f[0], f[1])] = float(f[2]) + float(f[3])
    if stamp != kernel_source_hash():
        return None
    return rows.get((workload_key, stage))


def roofline_for(stage, ms, n, sp, mm_mode, pk, clocks, kpad, workload_key=None):
    r = _roofline_for(stage, ms, n, sp, mm_mode, pk, clocks, kpad)
    if workload_key is None and n == 3 * N_WATERS:
        workload_key = "config3"
    r["traffic"] = traffic_from_profiles(stage, "%s_mm%d" % (workload_key, mm_mode)) if workload_key else None
    return r


def _roofline_for(stage, ms, n, sp, mm_mode, pk, clocks, kpad):
    """Roofline entry for the dominant stage (DESIGN.md 'Kernels and rooflines' gives the per-atom figures)."""
    from paper_2405_01491_b200 import inputs
    W = inputs.WIDTHS
    counts = np.bincount(sp, minlength=7)

    def macs(op):
        tot = 0
        for s in range(7):
            h1, h2, h3 = int(W[s, 1]), int(W[s, 2]), int(W[s, 3])
            tot += counts[s] * {"mlp_fwd_l1": kpad * h1, "mlp_fwd_l2": h1 * h2, "mlp_fwd_l3_out": h2 * h3 + h3,
                                "mlp_bwd_l3": h3 * h2, "mlp_bwd_l2": h2 * h1, "mlp_bwd_l1_dEdG": h1 * kpad}[op]
        return tot

    if stage == "mlp_fused_chain":
        ops = ["mlp_fwd_l1", "mlp_fwd_l2", "mlp_fwd_l3_out", "mlp_bwd_l3", "mlp_bwd_l2", "mlp_bwd_l1_dEdG"]
        flops = 2.0 * sum(macs(op) for op in ops)
        ach = flops / (ms * 1e-3) / 1e12 if ms else 0.0
        peak = pk["bf16_sus"]
        return {"kernel": "k_mlp_fused (%d GEMMs of the MLP chain in one launch, fp16 hi/lo split operands)" % len(ops), "bound": "tensor",
                "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak, "traffic": None,
                "peak_source": "%s sustained bf16 cuBLAS %.1f TF/s (fp16 operands run at the bf16 rate); algorithmic fp32 flops counted "
                               "once (the 3xF16 split issues 3 MMAs per product: a perfect kernel reads 1/3)" % (pk["source"], pk["bf16_sus"])}
    if stage.startswith("mlp"):
        flops = 2.0 * macs(stage)
        ach = flops / (ms * 1e-3) / 1e12 if ms else 0.0
        if mm_mode == 0:
            sm_mhz = clocks.get("sm_mhz") or pk["sm_max_mhz"]
            peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
            return {"kernel": stage, "bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                    "traffic": None, "peak_source": "148 SM x 128 FMA lanes x 2 x %.0f MHz (clocks.max.sm); median clock under load %s MHz"
                    % (pk["sm_max_mhz"], sm_mhz)}
        peak = pk["bf16_sus"] * 0.5
        return {"kernel": stage, "bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "traffic": None,
                "peak_source": "%s sustained bf16 cuBLAS %.1f TF/s x 0.5 (nominal tf32/bf16 ratio); algorithmic fp32 flops "
                               "counted once (3xTF32 issues 3 MMAs per product)" % (pk["source"], pk["bf16_sus"])}
    if stage in ("aev_forward", "aev_backward_scatter"):
        # algorithmic fp32 operations per atom for water at 1 g/cm3 (55.7 radial, 18.0 angular neighbours)
        per_atom = {"aev_forward": 55.7 * 16 * 6 + 153 * 150.0, "aev_backward_scatter": 55.7 * 16 * 10 + 153 * 330.0}[stage]
        ach = per_atom * n / (ms * 1e-3) / 1e12 if ms else 0.0
        peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
        return {"kernel": stage, "bound": "alu", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
                "traffic": None, "peak_source": "148 SM x 128 lanes x 2 x clocks.max.sm"}
    bytes_per_atom = {"kick_drift": 96.0, "kick_ekin": 52.0, "energy_sum": 12.0, "neighbor_build": 403.0 + 48.0}.get(stage, 64.0)
    ach = bytes_per_atom * n / (ms * 1e-3) / 1e9 if ms else 0.0
    return {"kernel": stage, "bound": "hbm", "achieved": ach, "peak": pk["hbm"], "unit": "GB/s", "frac": ach / pk["hbm"],
            "traffic": None, "peak_source": pk["source"]}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=50)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--mm-mode", type=int, default=int(os.environ.get("NNP_MM_MODE", "4")),
                    help="0 fp32 SIMT, 1 3xTF32 tcgen05 (six launches), 2 TF32, 3 fp64 SIMT, 4 3xF16 fused tcgen05 chain (default)")
    ap.add_argument("--waters", type=int, default=N_WATERS)
    ap.add_argument("--force-scale", type=float, default=None)
    ap.add_argument("--e2e-steps", type=int, default=200)
    ap.add_argument("--cpu-waters", type=int, default=N_WATERS, help="cpu_baseline: waters in the oracle's box (default: the workload)")
    ap.add_argument("--cpu-steps", type=int, default=2)
    ap.add_argument("--profile-steps", type=int, default=48, help="steps of the separate per-stage timing pass")
    ap.add_argument("--config", type=int, default=3, choices=[1, 2, 3, 4, 5],
                    help="BASELINE.json configuration (1-based): 3 = the headline MD workload; 1, 2, 4, 5 = one list build + one "
                         "energy/force evaluation per step")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--langevin", type=float, default=0.0, help="friction in 1/fs: BAOAB Langevin at 300 K instead of velocity Verlet")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    if args.force_scale is None:
        from paper_2405_01491_b200 import inputs
        args.force_scale = inputs.FORCE_SCALE_MD
    if args.impl == "reference":
        return run_reference(args)
    if args.config != 3:
        if args.steps == 1000 and args.warmup == 50:      # the MD defaults: an evaluation workload needs far fewer
            args.steps, args.warmup = 50, 5
        return run_eval_config(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
