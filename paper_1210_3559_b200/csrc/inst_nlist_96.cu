// inst_nlist_96.cu -- instantiations of nlist_kernel<TPA, 9, 6, FORCE, ENERGY, MIXED> (see sc_dispatch.h)
#include "sc_dispatch.h"

namespace scmd {
namespace {
template <int TPA>
cudaError_t launch(const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st) {
    const int atoms_per_block = kNlistBlock / TPA;
    const int grid = (a.n_atoms + atoms_per_block - 1) / atoms_per_block;
    auto go = [&](auto kernel) -> cudaError_t {
        kernel<<<grid, kNlistBlock, 0, st>>>(a);
        return cudaGetLastError();
    };
    if (!mixed) {
        if (!force) return go(nlist_kernel<TPA, 9, 6, false, false, false>);
        if (energy) return go(nlist_kernel<TPA, 9, 6, true, true, false>);
        return go(nlist_kernel<TPA, 9, 6, true, false, false>);
    }
    if (!force) return go(nlist_kernel<TPA, 9, 6, false, false, true>);
    if (energy) return go(nlist_kernel<TPA, 9, 6, true, true, true>);
    return go(nlist_kernel<TPA, 9, 6, true, false, true>);
}
}  // namespace

cudaError_t launch_nlist_96(int tpa, const NlistArgs &a, bool force, bool energy, bool mixed, cudaStream_t st) {
    switch (tpa) {
        case 1: return launch<1>(a, force, energy, mixed, st);
        case 2: return launch<2>(a, force, energy, mixed, st);
        case 4: return launch<4>(a, force, energy, mixed, st);
        case 8: return launch<8>(a, force, energy, mixed, st);
        case 16: return launch<16>(a, force, energy, mixed, st);
        case 32: return launch<32>(a, force, energy, mixed, st);
    }
    return cudaErrorInvalidConfiguration;
}
}  // namespace scmd
