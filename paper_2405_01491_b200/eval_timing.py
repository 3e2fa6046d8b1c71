"""Times one neighbour build + one energy/force evaluation on the BASELINE.json configurations that are not the
bench.py headline (configs 1, 2, 4, 5; config 3 = bench.py).  CUDA path only; prints one JSON line per configuration.

    python -m paper_2405_01491_b200.eval_timing [--reps 20] [--configs 1,2,4,5]

SURVEY.md 8(d): config 1 is launch-latency-bound (reported as microseconds per evaluation), configs 2 and 5 (8-network
ensembles) are MLP-dominated, config 4 exercises the ragged seven-species grouped GEMMs with the full 1008-column AEV.
Times are CUDA events on the library's stream around nnp_build_neighbors (skin 0) and nnp_energy_forces, median of
`reps` after 3 warm-up calls; the inputs stay resident in HBM.
"""
import argparse
import json

import numpy as np

from . import inputs, nnp


def _workload(cfg):
    """-> name, n_nets, species, xyz, box, mol_offsets"""
    if cfg == 1:
        sp, xyz, box = inputs.water_box(64, 12.42)
        return "water_192 (configs[0])", 1, sp, xyz, box, None
    if cfg == 2:
        sp, xyz, box = inputs.water_box(4096, 49.7, seed=inputs.SEED0 + 2)
        return "water_12288_ens8 (configs[1])", 8, sp, xyz, box, None
    if cfg == 4:
        sp, xyz, box = inputs.solvated_chain()
        return "solvated_chain_%d (configs[3])" % len(sp), 1, sp, xyz, box, None
    if cfg == 5:
        sp, xyz, offs = inputs.molecule_batch()
        return "molecules_8192_ens8 (configs[4])", 8, sp, xyz, None, offs
    raise ValueError("config %r: 1, 2, 4 or 5 (config 3 is bench.py)" % cfg)


def time_config(cfg, reps=20, mm_mode=1):
    import torch
    dev = torch.device("cuda:0")
    name, n_nets, sp, xyz, box, offs = _workload(cfg)
    n = len(sp)
    n_mols = 1 if offs is None else len(offs) - 1
    consts = inputs.ani2x_constants()
    params = inputs.make_weights(inputs.SEED0 + cfg, n_nets, last_layer_scale=2.0)
    p, keep = nnp.make_params(consts, inputs.WIDTHS, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=n_nets, mm_mode=mm_mode)
    stream = torch.cuda.Stream()
    ctx = nnp.nnp_create(p, n, n_mols, 0, stream.cuda_stream)
    try:
        d_sp = torch.as_tensor(np.asarray(sp, dtype=np.int32), device=dev)
        d_x = torch.as_tensor(np.asarray(xyz, dtype=np.float32), device=dev).contiguous()
        d_mo = None if offs is None else torch.as_tensor(np.asarray(offs, dtype=np.int32), device=dev)
        d_E = torch.zeros(n_mols, dtype=torch.float64, device=dev)
        d_F = torch.zeros((n, 3), dtype=torch.float32, device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box, n_mols, d_mo)
        t_build, t_eval = [], []
        with torch.cuda.stream(stream):
            for it in range(reps + 3):
                e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
                e0.record(stream)
                nnp.nnp_build_neighbors(ctx, 0.0)
                e1.record(stream)
                nnp.nnp_energy_forces(ctx, d_E, d_F)
                e2.record(stream)
                nnp.nnp_sync(ctx)
                if it >= 3:
                    t_build.append(e0.elapsed_time(e1))
                    t_eval.append(e1.elapsed_time(e2))
        ms_b, ms_e = float(np.median(t_build)), float(np.median(t_eval))
        return {"workload": name, "atoms": n, "structures": n_mols, "n_nets": n_nets,
                "aev_active_columns": nnp.nnp_aev_active_columns(ctx), "mm_mode": mm_mode,
                "neighbor_build_ms": round(ms_b, 4), "energy_forces_ms": round(ms_e, 4),
                "atom_evaluations_per_s": n / ((ms_b + ms_e) * 1e-3), "reps": reps}
    finally:
        nnp.nnp_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--configs", default="1,2,4,5")
    ap.add_argument("--mm-mode", type=int, default=1)
    a = ap.parse_args()
    for cfg in (int(c) for c in a.configs.split(",")):
        print(json.dumps(time_config(cfg, a.reps, a.mm_mode)), flush=True)


if __name__ == "__main__":
    main()
