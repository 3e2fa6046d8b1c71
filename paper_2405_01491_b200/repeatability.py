#!/usr/bin/env python
"""Repeatability stress: the same structure evaluated many times on one context must give the same energies and forces up
to the order of the fp32 atomics (forces are scattered with RED.ADD, energies summed with atomics in fp64 per structure).
A synchronisation bug in the tensor-core kernels (a consumer reading a tile or an operand chunk before it has arrived) shows
up here as an outlier - compute-sanitizer's racecheck is not available on the GPU pool this was developed on.

  python -m paper_2405_01491_b200.repeatability [--repeats 60] [--mm-mode 4]

Workloads: water (128 active AEV columns), a four-species system (384 columns: partial passes of the fused chain), the
seven-species solvated chain (1024 columns) and a molecule batch with an 8-network ensemble, each on the default stream and
on a side stream.  Prints one markdown row per workload; exits 1 if any repeat deviates by more than 1e-6 of sum |e_i| in
an atomic energy or 5e-4 in a force component.  Needs a GPU and the built library; nothing here touches the oracle."""
import argparse
import sys

import numpy as np


def run(name, sp, xyz, box, offs, n_nets, args, side):
    import torch
    from . import inputs, nnp
    dev = torch.device("cuda:0")
    consts = inputs.ani2x_constants()
    params = inputs.make_weights(inputs.SEED0 + 3, n_nets, last_layer_scale=20.0)
    n = len(sp)
    n_mols = 1 if offs is None else len(offs) - 1
    p, keep = nnp.make_params(consts, inputs.WIDTHS, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=n_nets, mm_mode=args.mm_mode)
    stream = torch.cuda.Stream(device=dev) if side else torch.cuda.current_stream()
    ctx = nnp.nnp_create(p, n, n_mols, 0, stream.cuda_stream)
    try:
        d_sp = torch.as_tensor(np.asarray(sp, dtype=np.int32), device=dev)
        d_x = torch.as_tensor(np.asarray(xyz, dtype=np.float32), device=dev).contiguous()
        d_o = None if offs is None else torch.as_tensor(np.asarray(offs, dtype=np.int32), device=dev)
        d_E = torch.zeros(n_mols, dtype=torch.float64, device=dev)
        d_F = torch.zeros((n, 3), dtype=torch.float32, device=dev)
        d_e = torch.zeros(n, dtype=torch.float32, device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box, n_mols, d_o)
        nnp.nnp_build_neighbors(ctx, 0.0)
        es, fs = [], []
        for _ in range(args.repeats):
            nnp.nnp_energy_forces(ctx, d_E, d_F)
            nnp.nnp_get_atomic_energies(ctx, d_e)
            nnp.nnp_sync(ctx)
            es.append(d_e.cpu().numpy().copy())
            fs.append(d_F.cpu().numpy().copy())
        es, fs = np.array(es), np.array(fs)
        scale = np.abs(np.median(es, axis=0)).sum()
        de = np.abs(es - np.median(es, axis=0)).max() / scale
        df = np.abs(fs - np.median(fs, axis=0)).max()
        ok = de <= 1e-6 and df <= 5e-4
        print("| %s | %s | %d | %d | %d | %.1e | %.1e | %s |" % (name, "side" if side else "default", n, nnp.nnp_aev_active_columns(ctx),
                                                                  args.repeats, de, df, "ok" if ok else "FAIL"), flush=True)
        return ok
    finally:
        nnp.nnp_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--repeats", type=int, default=60)
    ap.add_argument("--mm-mode", type=int, default=4)
    args = ap.parse_args()
    from . import inputs
    work = []
    sp, xyz, box = inputs.water_box(4096)
    work.append(("water 4096", sp, xyz, box, None, 1))
    sp, xyz, box = inputs.solvated_chain()
    work.append(("solvated chain, 7 species", sp, xyz, box, None, 1))
    work.append(("solvated chain, 4 species", np.minimum(sp, 3).astype(sp.dtype), xyz, box, None, 1))
    sp, xyz, offs = inputs.molecule_batch(1024)
    work.append(("1024 molecules, 8 networks", sp, xyz, None, offs, 8))
    print("| workload | stream | atoms | AEV columns | repeats | max |de_i| / sum |e_i| | max |dF| | |")
    print("|---|---|---:|---:|---:|---:|---:|---|")
    ok = True
    for w in work:
        for side in (0, 1):
            ok = run(*w, args, side) and ok
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
