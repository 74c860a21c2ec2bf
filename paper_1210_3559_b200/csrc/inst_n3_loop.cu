// inst_n3_loop.cu -- instantiations of n3_loop_kernel<IT, n, m, MIXED> (see sc_n3_loop.cuh)
#include "sc_n3_loop.cuh"

namespace scmd {
const void *n3_loop_fn(bool fast, bool mixed) {
    if (mixed) return fast ? reinterpret_cast<const void *>(n3_loop_kernel<4, 9, 6, true>)
                           : reinterpret_cast<const void *>(n3_loop_kernel<4, 0, 0, true>);
    return fast ? reinterpret_cast<const void *>(n3_loop_kernel<4, 9, 6, false>)
                : reinterpret_cast<const void *>(n3_loop_kernel<4, 0, 0, false>);
}
}  // namespace scmd
