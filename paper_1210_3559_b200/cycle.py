"""The paper's heating / cooling cycle through libscmd, as a usage example:

    python -m paper_1210_3559_b200.cycle [--shells 8] [--t-low 400] [--t-high 1400] [--rate 1.0] [--block 10000]

An n-shell Mackay icosahedron (8 shells = Ni2057) under the Langevin thermostat (gamma = 10 ps^-1,
dt = 1 fs) is heated from t_low to t_high and cooled back at `rate` K/ps; every `block` steps one line
"T_bath  T_kin  E_pot/atom" is printed (the caloric curve; the paper reads the melting and the
solidification temperature off its jump, ~400 K apart).  Everything runs in the CUDA kernels: one
cooperative launch per block of steps for N <= 2960 (the library's default; possible up to 6144).  The paper's cycle is 2 x 10^6 steps.
"""
from __future__ import annotations

import argparse
import time


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--shells", type=int, default=8)
    ap.add_argument("--t-low", type=float, default=400.0)
    ap.add_argument("--t-high", type=float, default=1400.0)
    ap.add_argument("--rate", type=float, default=1.0, help="K per ps")
    ap.add_argument("--block", type=int, default=10000, help="MD steps per output line (and per sc_step call)")
    ap.add_argument("--seed", type=int, default=2057)
    args = ap.parse_args()

    import torch
    from . import SuttonChen, langevin_thermostat
    from . import workloads as W

    w = W.mackay_cluster(args.shells, args.t_low, args.seed)
    n = w.n_atoms
    sc = SuttonChen(n)
    sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
    steps_per_leg = int(round((args.t_high - args.t_low) / args.rate * 1000.0))      # dt = 1 fs
    nblocks = max(1, steps_per_leg // args.block)
    print(f"# Ni{n} Mackay, Langevin gamma = 0.01 / fs, {args.rate} K/ps, {2 * nblocks * args.block} steps")
    print("# T_bath[K]  T_kin[K]  E_pot/atom[eV]")
    t0 = time.perf_counter()
    total = 0
    for leg, (ta, tb) in enumerate(((args.t_low, args.t_high), (args.t_high, args.t_low))):
        for b in range(nblocks):
            t_start = ta + (tb - ta) * b / nblocks
            t_end = ta + (tb - ta) * (b + 1) / nblocks
            sc.sc_step(1.0, args.block, langevin_thermostat(t_start, t_end, 0.01, args.seed))
            total += args.block
            _, t_kin = sc.sc_kinetic()
            print(f"{t_end:9.2f} {t_kin:9.2f} {sc.sc_energy() / n:12.6f}", flush=True)
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    print(f"# {total} steps in {dt:.1f} s = {total / dt:.0f} MD steps/s")
    sc.close()


if __name__ == "__main__":
    main()
