// sc_n3_loop.cuh -- n3_loop_kernel: all NVE steps of one sc_step call through the Newton's-third-law sweeps in ONE
// cooperative launch (velocity Verlet; the two sweeps of PAPER.md:127 with every unordered pair once).
//
// With the balanced plan (scmd.cu, plan_n3) a sweep is one CTA per SM, all resident, so the four kernels of a step --
// sweep 1, its finalize (rho_i, s'_i), sweep 2, its finalize (F_i, second half kick, next first half kick, drift) --
// can be four PHASES of one kernel separated by grid barriers: the same device functions as the stand-alone kernels
// (n3_sweep_piece / n3p_sweep_piece, n3_finalize_groups), the same sums in the same order, hence the same bits.  What
// goes away is the launch gap between dependent kernels (~3 us each, 12 us of a 29 us step at N = 2057 and of a 104 us
// step at N = 8000) and each kernel's ramp; what is paid is 4 barriers per step (~1 us each).
// Velocity rescaling (the cooling ramp of BASELINE.json config 3): the second finalize phase stops after the second
// half kick and leaves per-group sums of |v|^2; after the barrier that ends the step EVERY CTA adds them up in the same
// fixed order, forms lambda = sqrt(T_target / T) -- the expressions of reduce_ke_kernel -- and does the first half
// kick + drift of the next step for its share of the atoms with v <- lambda v first, as kick_drift_kernel does: one
// more phase and barrier per step (measured N = 8000: 114.8 us per step in seven launches -> see scmd.cu).
// The first half kick + drift of the call's first step is kick_drift_kernel, launched before this kernel; the kinetic
// energy of the last step is left as per-group partials (part_ke) for reduce_ke_kernel, the pair energy as per-CTA
// partials, U_emb as per-group partials: the host launches the scalar reductions after the loop, as on the other paths.
#pragma once
#include "sc_allpairs_n3.cuh"
#include "sc_integrate.cuh"

namespace scmd {

template <int IT, int NE, int ME, bool MIXED>
__global__ void __launch_bounds__(kN3Warps * 32, 1) n3_loop_kernel(const N3LoopArgs a) {
    __shared__ __align__(16) double buf[MIXED ? kN3pSmemDoubles<IT> : kN3Warps * IT * 3 * 32];
    double (&red)[kN3Warps][IT][3][32] = *reinterpret_cast<double (*)[kN3Warps][IT][3][32]>(buf);
    __shared__ double red_e[kN3Warps];
    __shared__ __align__(16) unsigned char slots[(kN3Warps / 2) * kN3SlotBytes];
    unsigned long long bar_target = a.barrier_base;
    auto grid_sync = [&]() { bar_target += gridDim.x; grid_barrier(a.barrier, bar_target); };
    constexpr int GB = 4;                                   // groups of 32 atoms a finalize phase handles at once
    static_assert(sizeof(double) * GB * kN3FinWarps * 3 * 32 <= sizeof(red), "finalize sums must fit into red");
    double(*fred)[kN3FinWarps][3][32] = reinterpret_cast<double(*)[kN3FinWarps][3][32]>(&red[0][0][0][0]);
    const int piece = blockIdx.x;
    const int ngroups = (a.f.n_atoms + kN3FinAtoms - 1) / kN3FinAtoms;
    N3FinalArgs f = a.f;
    __shared__ double s_lambda;
    for (long long k = 0; k < a.nsteps; ++k) {
        const bool last = k + 1 == a.nsteps;
        if (a.thermo == 1 && k > 0) {
            // k steps are done: scale to the ramp's temperature after step k, then first half kick + drift of step k + 1
            double v2 = 0.0;
            for (int j = threadIdx.x; j < ngroups; j += blockDim.x) v2 += f.part_ke[j];
            const double tot = block_sum(v2, red_e);
            if (threadIdx.x == 0) {
                const double target = a.T_start + (a.T_end - a.T_start) * double(k) / double(a.nsteps);
                const double ke = 0.5 * a.mass * tot / kAcc;
                const double temp = a.ndof > 0.0 ? 2.0 * ke / (kBoltzmann * a.ndof) : 0.0;
                s_lambda = temp > 0.0 ? sqrt(target / temp) : 1.0;
            }
            __syncthreads();
            const double lambda = s_lambda;
            for (int i = piece * blockDim.x + threadIdx.x; i < f.n_atoms; i += gridDim.x * blockDim.x) {
                double4 p = f.xs[i];
                double vx = f.vel[3 * size_t(i)] * lambda, vy = f.vel[3 * size_t(i) + 1] * lambda, vz = f.vel[3 * size_t(i) + 2] * lambda;
                vx = fma(f.hk, f.force[3 * size_t(i)], vx);
                vy = fma(f.hk, f.force[3 * size_t(i) + 1], vy);
                vz = fma(f.hk, f.force[3 * size_t(i) + 2], vz);
                p.x = fma(f.dt, vx, p.x); p.y = fma(f.dt, vy, p.y); p.z = fma(f.dt, vz, p.z);
                f.vel[3 * size_t(i)] = vx; f.vel[3 * size_t(i) + 1] = vy; f.vel[3 * size_t(i) + 2] = vz;
                f.xs[i] = p;
                if (f.xf) store_split_record(f.xf, i, p.x, p.y, p.z, float(p.w));
                if (f.xfr) f.xfr[i] = split_record(p);
            }
            grid_sync();
        }
        // sweep 1: density partials
        if constexpr (MIXED) n3p_sweep_piece<IT, NE, ME, false, false>(a.sf, piece, buf, red_e, slots);
        else n3_sweep_piece<IT, NE, ME, false, false>(a.s, piece, red, red_e, slots);
        grid_sync();
        f.fuse = 0;
        for (int g = piece; g < ngroups; g += GB * gridDim.x)
            n3_finalize_groups<false, GB>(f, g, gridDim.x, min(GB, (ngroups - g + int(gridDim.x) - 1) / int(gridDim.x)), fred);
        grid_sync();
        // sweep 2: force partials (+ pair energy)
        if (last || a.energy_every) {
            if constexpr (MIXED) n3p_sweep_piece<IT, NE, ME, true, true>(a.sf, piece, buf, red_e, slots);
            else n3_sweep_piece<IT, NE, ME, true, true>(a.s, piece, red, red_e, slots);
        } else {
            if constexpr (MIXED) n3p_sweep_piece<IT, NE, ME, true, false>(a.sf, piece, buf, red_e, slots);
            else n3_sweep_piece<IT, NE, ME, true, false>(a.s, piece, red, red_e, slots);
        }
        grid_sync();
        f.fuse = (last || a.thermo == 1) ? 1 : 2;
        for (int g = piece; g < ngroups; g += GB * gridDim.x)
            n3_finalize_groups<true, GB>(f, g, gridDim.x, min(GB, (ngroups - g + int(gridDim.x) - 1) / int(gridDim.x)), fred);
        if (!last) grid_sync();
    }
}

}  // namespace scmd
