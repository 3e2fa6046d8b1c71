#!/usr/bin/env python
"""Matmul-precision study in the manner of the paper's Fig. 3.

The paper runs NVE dynamics of a 216-molecule water box at dt = 0.1 fs, started from rest, with the network's matmuls in
bf16 ("default"), TF32 ("high"), fp32 ("highest") and fp64, and finds that only full fp32 conserves the total energy
(fluctuation < 0.1 %, no initial shift).  Here the same protocol runs on the library's five matmul modes:
    3  fp32 operands, fp64 products and sums (the fp64 leg)      0  fp32 SIMT      1  3xTF32 on tcgen05
    4  3xF16 fused tcgen05 chain (the default)                   2  plain TF32 on tcgen05
on a seeded 216-water box with seeded random-init weights (the paper's trained ANI-2x weights are not available, so the
comparison is qualitative: which modes conserve energy, not the paper's absolute numbers).

  python -m paper_2405_01491_b200.precision_study [--steps 3000] [--repeats 3] [--dt 0.1] [--scale 66] [--waters 216]

Prints one markdown table row per mode: maximum |E_tot(t) - E_tot(0)| (median and worst of the repeats), the linear drift over
the run, the median change of E_tot per sampling interval, the shift of the initial total energy against the fp64 leg
(Fig. 3's second criterion), all relative to the mean kinetic energy of the second half of the run (the quantity Fig. 3
plots against), and the final kinetic temperature.
The window is 0.3 ps by default on purpose.  The random-weight model is not a bound liquid: at 0.43 ps two hydrogens of the
seeded box pass within 0.035 A of each other, and the integration error of that unphysical geometry (a transient of 1e-5 ..
2e-4 <E_kin>, the same in every mode, fp64 included) then decides the maximum; repeats of one mode differ there by a factor
of ten because the order of the force reductions differs from run to run and the trajectories have diverged by then.
Before it the repeats of a mode agree to ~30 %.
Needs a GPU and the built library; nothing here touches the oracle.
"""
import argparse

import numpy as np


def run_mode(mm_mode, args):
    import torch
    from . import inputs, nnp
    dev = torch.device("cuda:0")
    consts = inputs.ani2x_constants()
    params = inputs.make_weights(inputs.SEED0, 1, last_layer_scale=args.scale)
    sp, xyz, box = inputs.water_box(args.waters, seed=inputs.SEED0 + 216)
    n = len(sp)
    p, keep = nnp.make_params(consts, inputs.WIDTHS, params, inputs.MASS, inputs.ACCEL_CONV, n_nets=1, mm_mode=mm_mode)
    stream = torch.cuda.Stream(device=dev)
    ctx = nnp.nnp_create(p, n, 1, 0, stream.cuda_stream)
    try:
        d_sp = torch.as_tensor(sp, device=dev)
        d_x = torch.as_tensor(xyz.astype(np.float32), device=dev)
        d_v = torch.zeros_like(d_x)                       # Fig. 3: started from rest
        o_ep = torch.zeros(1, dtype=torch.float64, device=dev)
        o_ek = torch.zeros(1, dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        nnp.nnp_set_system(ctx, n, d_sp, d_x, box)
        nnp.nnp_md_init(ctx, d_v, args.dt, 0.5)
        etot, ekin = [], []
        for k in range(args.steps // args.every + 1):
            nnp.nnp_get_state(ctx, None, None, o_ep, o_ek, None)
            nnp.nnp_sync(ctx)
            etot.append(float(o_ep.item()) + float(o_ek.item()))
            ekin.append(float(o_ek.item()))
            nnp.nnp_md_step(ctx, args.every)
        etot, ekin = np.array(etot), np.array(ekin)
        t = np.arange(len(etot)) * args.every * args.dt
        ke = ekin[len(ekin) // 2:].mean()
        drift = np.polyfit(t, etot, 1)[0] * t[-1]
        return dict(max_dev=np.abs(etot - etot[0]).max() / ke, drift=drift / ke, step_med=np.median(np.abs(np.diff(etot))) / ke,
                    T_end=2 * ekin[-1] / (3 * n * inputs.KB), ke=ke, e0=etot[0])
    finally:
        nnp.nnp_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=3000)
    ap.add_argument("--repeats", type=int, default=3)
    ap.add_argument("--every", type=int, default=20)
    ap.add_argument("--dt", type=float, default=0.1)
    ap.add_argument("--waters", type=int, default=216)
    ap.add_argument("--scale", type=float, default=None, help="last-layer weight scale (default inputs.FORCE_SCALE_WATER)")
    args = ap.parse_args()
    from . import inputs
    if args.scale is None:
        args.scale = inputs.FORCE_SCALE_WATER
    print("| matmul mode | max |dE_tot| / <E_kin>: median (worst) of %d runs | drift over run / <E_kin> | median |dE_tot| per %d steps / <E_kin> "
          "| E_tot(0) - E_tot(0)[fp64] / <E_kin> | T_end [K] |" % (args.repeats, args.every))
    print("|---|---:|---:|---:|---:|---:|")
    ref = None
    for mode, name in ((3, "fp64-accumulate SIMT"), (0, "fp32 SIMT"), (1, "3xTF32 tcgen05"), (4, "3xF16 fused tcgen05 (default)"),
                       (2, "TF32 tcgen05")):
        rs = [run_mode(mode, args) for _ in range(args.repeats)]
        med = lambda k: float(np.median([r[k] for r in rs]))  # noqa: E731
        if ref is None:
            ref = dict(e0=med("e0"), ke=med("ke"))
        print("| %s | %.2e (%.2e) | %+.2e | %.2e | %+.2e | %.0f |" % (name, med("max_dev"), max(r["max_dev"] for r in rs), med("drift"),
                                                                 med("step_med"), (med("e0") - ref["e0"]) / ref["ke"], med("T_end")), flush=True)


if __name__ == "__main__":
    main()
