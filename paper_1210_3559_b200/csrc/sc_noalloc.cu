// sc_noalloc.cu -- sc_density_noalloc (include/scmd.h): sweep 1 of the Sutton-Chen evaluation (Eq. (2), PAPER.md:69,
// all pairs, FP64) for callers that can hand the library NO workspace: code under CUDA graph capture, serving loops and
// harnesses in which nobody may call cudaMalloc.  The regular path (sc_create + sc_density) keeps its packed records
// and its per-CTA partial sums in a caller-allocated workspace; this variant keeps them in a file-scope device array
// of fixed size that every GPU loading libscmd.so holds until the process exits.
//
// The entry point calls no cudaMalloc, cudaFree or allocating library routine: one cudaMemsetAsync and two kernel
// launches on the caller's stream.  The array's device address is looked up ONCE PER DEVICE, with that device current,
// by cudaGetSymbolAddress (in host code the array's name is a host-side stand-in, not a device address).
//
// Every call shares the array, which keeps the last call's contents: the call clears the words that must start at zero
// (the arrival counter of the final reduction) and overwrites what it reads (records, partials).  Calls that overlap on
// the GPU (two streams or two host threads of one process on one device) race on it; the caller serialises them.
#include <cmath>
#include <cstdio>
#include <mutex>

#include "../../include/scmd.h"
#include "sc_device.cuh"

namespace scmd {
namespace {

constexpr int kNoallocMaxAtoms = SC_NOALLOC_MAX_ATOMS;
constexpr int kNoallocThreads = 128;                                   // one row i per thread
constexpr int kNoallocMaxBlocks = (kNoallocMaxAtoms + kNoallocThreads - 1) / kNoallocThreads;
// layout of the scratch array: [0, 256) arrival counter; [256, 256 + 8 * blocks) per-CTA sums of sqrt(rho);
// then the packed records (x, y, z, 0) of all atoms
constexpr size_t kOffPartial = 256;
constexpr size_t kOffRecords = (kOffPartial + sizeof(double) * kNoallocMaxBlocks + 255) / 256 * 256;
constexpr size_t kScratchBytes = kOffRecords + sizeof(double4) * size_t(kNoallocMaxAtoms);
static_assert(kScratchBytes <= SC_NOALLOC_SCRATCH_BYTES, "scmd.h states the size of the static scratch array");

static __device__ __align__(256) unsigned char g_noalloc_scratch[SC_NOALLOC_SCRATCH_BYTES];

// pos[N*3] -> records (x, y, z, 0) in the scratch array
__global__ void noalloc_pack_kernel(const double *__restrict__ pos, double4 *__restrict__ rec, int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) rec[i] = make_double4(pos[3 * size_t(i)], pos[3 * size_t(i) + 1], pos[3 * size_t(i) + 2], 0.0);
}

// rho_i = a^m sum_{j != i} r_ij^-m, the self term excluded by index (reading Q11); tiles of 128 records
// staged in shared memory; sum_i sqrt(rho_i) in a fixed order: per CTA, then by the last CTA to arrive over all CTAs
__global__ void __launch_bounds__(kNoallocThreads)
noalloc_density_kernel(const double4 *__restrict__ rec, int N, int m_exp, double am, double *__restrict__ rho,
                       double *__restrict__ partial, unsigned int *__restrict__ arrived, double *__restrict__ sum_sqrt) {
    __shared__ double4 tile[kNoallocThreads];
    __shared__ double scratch[32];
    __shared__ bool is_last;
    const int i = blockIdx.x * kNoallocThreads + threadIdx.x;
    const bool live = i < N;
    const double4 pi = live ? rec[i] : make_double4(0.0, 0.0, 0.0, 0.0);
    double acc = 0.0;
    for (int j0 = 0; j0 < N; j0 += kNoallocThreads) {
        const int jl = j0 + threadIdx.x;
        __syncthreads();
        if (jl < N) tile[threadIdx.x] = rec[jl];
        __syncthreads();
        const int cnt = min(kNoallocThreads, N - j0);
        for (int k = 0; k < cnt; ++k) {
            const double4 p = tile[k];
            const bool self = (j0 + k == i);
            const double dx = pi.x - p.x, dy = pi.y - p.y, dz = pi.z - p.z;
            double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
            r2 = self ? 1.0 : r2;
            double term;
            if ((m_exp & 1) == 0) {
                const double w = self ? 0.0 : rcp_fast(r2);
                term = ipow_rt(w, m_exp >> 1);
            } else {
                const double y = self ? 0.0 : rsqrt_fast(r2);
                term = ipow_rt(y, m_exp);
            }
            acc += term;
        }
    }
    double root = 0.0;
    if (live) {
        const double r = am * acc;
        rho[i] = r;
        root = r > 0.0 ? sqrt(r) : 0.0;                                   // reading Q9
    }
    const double t = block_sum(root, scratch);
    if (threadIdx.x == 0) {
        partial[blockIdx.x] = t;
        __threadfence();
        is_last = atomicAdd(arrived, 1u) + 1u == gridDim.x;
    }
    __syncthreads();
    if (is_last && threadIdx.x == 0) {
        __threadfence();
        double s = 0.0;
        for (int b = 0; b < int(gridDim.x); ++b) s += __ldcg(partial + b);
        if (sum_sqrt) *sum_sqrt = s;
        *arrived = 0u;                                                    // the next call finds it clear as well
    }
}

thread_local char tl_error[256] = "";

sc_status noalloc_fail(sc_status st, const char *msg) {
    std::snprintf(tl_error, sizeof(tl_error), "%s", msg);
    return st;
}

// device address of the scratch array, looked up once per device with that device current
constexpr int kMaxDevices = 64;
std::mutex g_mutex;
unsigned char *g_scratch_ptr[kMaxDevices] = {};

sc_status scratch_for_current_device(unsigned char **out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) return noalloc_fail(SC_ERR_CUDA, "sc_density_noalloc: no CUDA device");
    if (dev < 0 || dev >= kMaxDevices) return noalloc_fail(SC_ERR_CUDA, "sc_density_noalloc: device ordinal beyond 63");
    std::lock_guard<std::mutex> lock(g_mutex);
    if (!g_scratch_ptr[dev]) {
        void *p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            std::snprintf(tl_error, sizeof(tl_error), "sc_density_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            return SC_ERR_CUDA;
        }
        g_scratch_ptr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_scratch_ptr[dev];
    return SC_OK;
}

double ipow_h(double u, int k) {
    double r = 1.0;
    for (int t = 0; t < k; ++t) r *= u;
    return r;
}

}  // namespace
}  // namespace scmd

extern "C" {

const char *sc_noalloc_last_error(void) { return scmd::tl_error; }

sc_status sc_density_noalloc(const sc_params *params, int64_t n_atoms, const double *d_pos, double *d_rho,
                             double *d_sum_sqrt_rho, void *cuda_stream) {
    using namespace scmd;
    if (!params || !d_pos || !d_rho) return noalloc_fail(SC_ERR_INVALID, "sc_density_noalloc: NULL argument");
    if (!(params->n > params->m && params->m > 0 && params->n <= 64 && params->a > 0.0 && std::isfinite(params->a)))
        return noalloc_fail(SC_ERR_INVALID, "sc_density_noalloc: need 64 >= n > m > 0 and a > 0");
    if (params->r_cut > 0.0) return noalloc_fail(SC_ERR_INVALID, "sc_density_noalloc: all pairs only (r_cut must be <= 0)");
    if (n_atoms < 1) return noalloc_fail(SC_ERR_INVALID, "sc_density_noalloc: n_atoms must be >= 1");
    if (n_atoms > kNoallocMaxAtoms) {
        std::snprintf(tl_error, sizeof(tl_error),
                      "sc_density_noalloc: n_atoms = %lld exceeds SC_NOALLOC_MAX_ATOMS = %d (the static scratch array holds no more; "
                      "use sc_create + sc_density with a workspace)", static_cast<long long>(n_atoms), kNoallocMaxAtoms);
        return SC_ERR_NOMEM;
    }
    unsigned char *base = nullptr;
    sc_status st = scratch_for_current_device(&base);
    if (st != SC_OK) return st;
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    unsigned int *arrived = reinterpret_cast<unsigned int *>(base);
    double *partial = reinterpret_cast<double *>(base + kOffPartial);
    double4 *rec = reinterpret_cast<double4 *>(base + kOffRecords);
    const int N = int(n_atoms), blocks = (N + kNoallocThreads - 1) / kNoallocThreads;
    // the array keeps the last call's contents (a call that was aborted may have left the counter anywhere)
    cudaError_t e = cudaMemsetAsync(arrived, 0, kOffPartial, stream);
    if (e != cudaSuccess) {
        std::snprintf(tl_error, sizeof(tl_error), "sc_density_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e));
        return SC_ERR_CUDA;
    }
    noalloc_pack_kernel<<<blocks, kNoallocThreads, 0, stream>>>(d_pos, rec, N);
    noalloc_density_kernel<<<blocks, kNoallocThreads, 0, stream>>>(rec, N, params->m, ipow_h(params->a, params->m), d_rho,
                                                                   partial, arrived, d_sum_sqrt_rho);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        std::snprintf(tl_error, sizeof(tl_error), "sc_density_noalloc: launch: %s", cudaGetErrorString(e));
        return SC_ERR_CUDA;
    }
    tl_error[0] = 0;
    return SC_OK;
}

}  // extern "C"
