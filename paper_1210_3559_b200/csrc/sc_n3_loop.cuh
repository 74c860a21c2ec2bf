// sc_n3_loop.cuh -- n3_loop_kernel: all NVE steps of one sc_step call through the Newton's-third-law sweeps in ONE
// cooperative launch (velocity Verlet; the two sweeps of PAPER.md:127 with every unordered pair once).
//
// With the balanced plan (scmd.cu, plan_n3) a sweep is one CTA per SM, all resident, so the four kernels of a step --
// sweep 1, its finalize (rho_i, s'_i), sweep 2, its finalize (F_i, second half kick, next first half kick, drift) --
// can be four PHASES of one kernel separated by grid barriers: the same device functions as the stand-alone kernels
// (n3_sweep_piece / n3p_sweep_piece, n3_finalize_groups), the same sums in the same order, hence the same bits.  What
// goes away is the launch gap between dependent kernels (~3 us each, 12 us of a 29 us step at N = 2057 and of a 104 us
// step at N = 8000) and each kernel's ramp; what is paid is 4 barriers per step (~1 us each).
// The first half kick + drift of the call's first step is kick_drift_kernel, launched before this kernel; the kinetic
// energy of the last step is left as per-group partials (part_ke) for reduce_ke_kernel, the pair energy as per-CTA
// partials, U_emb as per-group partials: the host launches the scalar reductions after the loop, as on the other paths.
#pragma once
#include "sc_allpairs_n3.cuh"

namespace scmd {

template <int IT, int NE, int ME, bool MIXED>
__global__ void __launch_bounds__(kN3Warps * 32, 1) n3_loop_kernel(const N3LoopArgs a) {
    __shared__ double red[kN3Warps][IT][3][32];
    __shared__ double red_e[kN3Warps];
    unsigned long long bar_target = a.barrier_base;
    auto grid_sync = [&]() { bar_target += gridDim.x; grid_barrier(a.barrier, bar_target); };
    constexpr int GB = 4;                                   // groups of 32 atoms a finalize phase handles at once
    static_assert(sizeof(double) * GB * kN3FinWarps * 3 * 32 <= sizeof(red), "finalize sums must fit into red");
    double(*fred)[kN3FinWarps][3][32] = reinterpret_cast<double(*)[kN3FinWarps][3][32]>(&red[0][0][0][0]);
    const int piece = blockIdx.x;
    const int ngroups = (a.f.n_atoms + kN3FinAtoms - 1) / kN3FinAtoms;
    N3FinalArgs f = a.f;
    for (long long k = 0; k < a.nsteps; ++k) {
        const bool last = k + 1 == a.nsteps;
        // sweep 1: density partials
        if constexpr (MIXED) n3p_sweep_piece<IT, NE, ME, false, false>(a.sf, piece, red, red_e);
        else n3_sweep_piece<IT, NE, ME, false, false>(a.s, piece, red, red_e);
        grid_sync();
        f.fuse = 0;
        for (int g = piece; g < ngroups; g += GB * gridDim.x)
            n3_finalize_groups<false, GB>(f, g, gridDim.x, min(GB, (ngroups - g + int(gridDim.x) - 1) / int(gridDim.x)), fred);
        grid_sync();
        // sweep 2: force partials (+ pair energy)
        if (last || a.energy_every) {
            if constexpr (MIXED) n3p_sweep_piece<IT, NE, ME, true, true>(a.sf, piece, red, red_e);
            else n3_sweep_piece<IT, NE, ME, true, true>(a.s, piece, red, red_e);
        } else {
            if constexpr (MIXED) n3p_sweep_piece<IT, NE, ME, true, false>(a.sf, piece, red, red_e);
            else n3_sweep_piece<IT, NE, ME, true, false>(a.s, piece, red, red_e);
        }
        grid_sync();
        f.fuse = last ? 1 : 2;
        for (int g = piece; g < ngroups; g += GB * gridDim.x)
            n3_finalize_groups<true, GB>(f, g, gridDim.x, min(GB, (ngroups - g + int(gridDim.x) - 1) / int(gridDim.x)), fred);
        if (!last) grid_sync();
    }
}

}  // namespace scmd
