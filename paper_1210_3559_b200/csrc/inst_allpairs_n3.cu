// inst_allpairs_n3.cu -- instantiations of allpairs_n3_kernel<IT, n, m, FORCE, ENERGY> (see sc_allpairs_n3.cuh)
#include "sc_allpairs_n3.cuh"

namespace scmd {
namespace {
template <int IT, int NE, int ME>
const void *pick(bool force, bool energy) {
    if (!force) return reinterpret_cast<const void *>(allpairs_n3_kernel<IT, NE, ME, false, false>);
    if (energy) return reinterpret_cast<const void *>(allpairs_n3_kernel<IT, NE, ME, true, true>);
    return reinterpret_cast<const void *>(allpairs_n3_kernel<IT, NE, ME, true, false>);
}
}  // namespace

namespace {
template <int IT, int NE, int ME>
const void *pickp(bool force, bool energy) {
    if (!force) return reinterpret_cast<const void *>(allpairs_n3p_kernel<IT, NE, ME, false, false>);
    if (energy) return reinterpret_cast<const void *>(allpairs_n3p_kernel<IT, NE, ME, true, true>);
    return reinterpret_cast<const void *>(allpairs_n3p_kernel<IT, NE, ME, true, false>);
}
}  // namespace

const void *allpairs_n3p_fn(int it, bool fast, bool force, bool energy) {
    if (it == 4) return fast ? pickp<4, 9, 6>(force, energy) : pickp<4, 0, 0>(force, energy);
    return nullptr;
}

const void *allpairs_n3_fn(int it, bool fast, bool force, bool energy) {
    if (it == 4) return fast ? pick<4, 9, 6>(force, energy) : pick<4, 0, 0>(force, energy);
    return nullptr;
}
}  // namespace scmd
