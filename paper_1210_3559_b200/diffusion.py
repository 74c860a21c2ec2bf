"""The paper's self-diffusion measurement (Eq. (12)) through libscmd, as a usage example:

    python -m paper_1210_3559_b200.diffusion [--shells 8] [--temperature 820] [--segments 10] [--segment-ps 100]

Procedure of PAPER.md:209: a window of the trajectory at the thermostat temperature is split into segments;
for each segment the cluster is "translated and rotated as a whole in order to minimize the root-mean-square
displacement of atoms from a reference structure" (the structure at the segment's start) and the
mean-square displacement of "all atoms located within 10 A of the cluster center of mass" gives
D = <dr^2> / (2 z dt), z = 3; the value reported is the average over the segments.  `sc_msd` does the fit
and the average on the device; this file only loops and converts units (1 A^2/fs = 0.1 cm^2/s).

Two states of the n-shell Mackay cluster at the same temperature are measured: the supercooled droplet
(melted at --melt-temperature, then cooled to the target in --quench-ps) and the solid icosahedron that was
never melted -- the paper's point is that D separates them ("drops abruptly" at solidification; molten
value ~2.3e-6 cm^2/s at 820 K).  Langevin thermostat, gamma = 10 ps^-1, dt = 1 fs.
"""
from __future__ import annotations

import argparse
import time

A2_PER_FS_IN_CM2_PER_S = 0.1


def diffusion_coefficient(msd_a2: float, dt_fs: float, z: int = 3) -> float:
    """Eq. (12): D = <dr^2> / (2 z dt), in cm^2/s from A^2 and fs."""
    return A2_PER_FS_IN_CM2_PER_S * msd_a2 / (2.0 * z * dt_fs)


def measure(sc, label: str, temperature: float, segments: int, seg_steps: int, r_centre: float, seed: int, block: int):
    from . import langevin_thermostat
    n = sc.n_atoms
    ds = []
    print(f"# {label}: {segments} segments of {seg_steps} steps at {temperature} K, atoms within {r_centre} A of the centre")
    print("# segment  n_sel  msd[A^2]   D[cm^2/s]   E_pot/atom[eV]  T_kin[K]")
    for s in range(segments):
        ref, _ = sc.sc_get_state(want_vel=False)
        done = 0
        while done < seg_steps:
            k = min(block, seg_steps - done)
            sc.sc_step(1.0, k, langevin_thermostat(temperature, temperature, 0.01, seed))
            done += k
        msd, n_sel, _ = sc.sc_msd(ref, r_centre, 2)
        d = diffusion_coefficient(msd, float(seg_steps))
        ds.append(d)
        _, t_kin = sc.sc_kinetic()
        print(f"{s:9d} {n_sel:6d} {msd:9.4f} {d:12.4e} {sc.sc_energy() / n:12.6f} {t_kin:9.2f}", flush=True)
    mean = sum(ds) / len(ds)
    print(f"# {label}: D = {mean:.3e} cm^2/s (mean of {len(ds)} segments, min {min(ds):.3e}, max {max(ds):.3e})")
    return mean


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--shells", type=int, default=8)
    ap.add_argument("--temperature", type=float, default=820.0)
    ap.add_argument("--melt-temperature", type=float, default=1400.0)
    ap.add_argument("--melt-ps", type=float, default=50.0)
    ap.add_argument("--quench-ps", type=float, default=50.0)
    ap.add_argument("--segments", type=int, default=10)
    ap.add_argument("--segment-ps", type=float, default=100.0)
    ap.add_argument("--r-centre", type=float, default=10.0)
    ap.add_argument("--block", type=int, default=20000, help="MD steps per sc_step call")
    ap.add_argument("--seed", type=int, default=2057)
    args = ap.parse_args()

    import torch
    from . import SuttonChen, langevin_thermostat
    from . import workloads as W

    seg_steps = int(round(args.segment_ps * 1000.0))
    t0 = time.perf_counter()
    total = 0
    out = {}
    for label in ("solid (icosahedron, never melted)", "supercooled droplet"):
        liquid = label.startswith("supercooled")
        w = W.mackay_cluster(args.shells, args.temperature, args.seed)
        sc = SuttonChen(w.n_atoms)
        sc.sc_set_state(torch.as_tensor(w.pos, device="cuda"), torch.as_tensor(w.vel, device="cuda"))
        if liquid:
            legs = ((args.melt_temperature, args.melt_temperature, args.melt_ps),
                    (args.melt_temperature, args.temperature, args.quench_ps))
        else:
            legs = ((args.temperature, args.temperature, 20.0),)
        for ta, tb, ps in legs:                                   # preparation, not measured
            steps = int(round(ps * 1000.0))
            nb = max(1, steps // args.block)
            for b in range(nb):
                sc.sc_step(1.0, steps // nb, langevin_thermostat(ta + (tb - ta) * b / nb, ta + (tb - ta) * (b + 1) / nb,
                                                                0.01, args.seed))
            total += steps
        out[label] = measure(sc, f"Ni{w.n_atoms} {label}", args.temperature, args.segments, seg_steps, args.r_centre,
                             args.seed, args.block)
        total += args.segments * seg_steps
        sc.close()
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    vals = list(out.values())
    print(f"# D(droplet) / D(solid) = {vals[1] / max(vals[0], 1e-300):.1f}")
    print(f"# {total} steps in {dt:.1f} s = {total / dt:.0f} MD steps/s")


if __name__ == "__main__":
    main()
