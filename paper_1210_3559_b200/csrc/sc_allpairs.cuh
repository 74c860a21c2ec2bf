// sc_allpairs.cuh -- the two O(N^2) sweeps over all ordered pairs, FP64.
//
// Decomposition.  A CTA owns RPC = (32 / TPR) * IT complete rows i (so no cross-CTA reduction
// and no atomics: results are bit-reproducible).  Every consumer warp of the CTA holds the same
// rows in registers -- lane = g * TPR + q holds rows g*IT .. g*IT+IT-1 -- and the j range is
// split W * TPR ways (W consumer warps x TPR lanes): "j-lane" jl = w * TPR + q takes
// j = jl, jl + W*TPR, ... of every tile.  Lanes with equal q read the same shared-memory
// address (broadcast).  At the end the partial sums are reduced over q with warp shuffles and
// over the W warps through shared memory in a fixed order.
//
// The j stream.  Atoms live in HBM/L2 as one 32-byte record (x, y, z, s') per atom, where
// s'_j = eps (c m / 2) a^m rho_j^-1/2 is written by the first sweep's epilogue.  One extra
// "producer" warp streams the records through a ring of shared-memory tiles with 1-D bulk
// async copies (TMA; SASS UBLKCP) that complete on mbarriers; consumer warps hand a tile back
// through a second mbarrier.  All N records are re-read by every CTA from L2 (N <= 262144 is
// 8.4 MB), never from HBM after the first touch.
//
// Per ordered pair, (n, m) = (9, 6), FP64-pipe instructions (SASS-checked):
//   sweep 1: 3 (displacement) + 3 (r^2) + 3 (1/r^2) + 2 (cube, accumulate)            = 11
//   sweep 2: 3 + 3 + 5 (1/r) + 4 (powers) + 1 (s_i'+s_j') + 2 (bracket, x r^-8) + 3 (F) = 21
//            + 1 when the pair energy is accumulated                                     = 22
#pragma once
#include "sc_device.cuh"

namespace scmd {

constexpr int kTileAtoms = 512;     // records per shared-memory tile (16 KB)
constexpr int kStages = 4;          // ring depth
constexpr int kMaxConsumerWarps = 8;

struct PairConsts {
    double am;        // a^m                      rho_i = am * sum r^-m
    double An;        // eps * n * a^n
    double Bm;        // eps * (c m / 2) * a^m    s'_i = Bm * rho_i^-1/2
    double En;        // eps / 2 * a^n            U_pair = En * sum_i sum_j r^-n
    double eps_c;     // eps * c                  U_emb  = -eps_c * sum_i sqrt(rho_i)
    int n, m;
};

struct AllPairsArgs {
    double4 *xs;          // [N] (x, y, z, s')
    int n_atoms;
    double *rho;          // [N]    sweep 1 output
    double *force;        // [N*3]  sweep 2 output
    double *partial;      // [gridDim.x] per-CTA partial: sum sqrt(rho) (sweep 1) / sum r^-n (sweep 2)
    PairConsts c;
};

__host__ __device__ constexpr int allpairs_rows_per_cta(int IT, int TPR) { return (32 / TPR) * IT; }

constexpr int kBarrierBytes = 128;   // 2 * kStages mbarriers, padded
static_assert(2 * kStages * sizeof(uint64_t) <= kBarrierBytes, "barrier area too small");

inline size_t allpairs_smem_bytes(int IT, int TPR, int W) {
    size_t tiles = size_t(kStages) * kTileAtoms * sizeof(double4);
    size_t red = (size_t(W) * allpairs_rows_per_cta(IT, TPR) * 4 + allpairs_rows_per_cta(IT, TPR)) * sizeof(double);
    return kBarrierBytes + (tiles > red ? tiles : red);
}

// IT rows per thread, TPR lanes per row group, exponents NE/ME (0,0 = read from args at run time),
// FORCE: second sweep; ENERGY: also accumulate sum r^-n (second sweep only)
template <int IT, int TPR, int NE, int ME, bool FORCE, bool ENERGY>
__global__ void __launch_bounds__((kMaxConsumerWarps + 1) * 32, 1) allpairs64_kernel(const AllPairsArgs a) {
    constexpr int RPC = allpairs_rows_per_cta(IT, TPR);
    constexpr int NV = FORCE ? 4 : 1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    // layout: [0,128) mbarriers | [128, ...) tile ring, reused as reduction scratch after the sweep
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);
    double4 *tiles = reinterpret_cast<double4 *>(smem_raw + kBarrierBytes);
    double *red = reinterpret_cast<double *>(smem_raw + kBarrierBytes);
    uint64_t *empty = full + kStages;

    const int W = (blockDim.x >> 5) - 1;                  // consumer warps
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int N = a.n_atoms;
    const int ntiles = (N + kTileAtoms - 1) / kTileAtoms;

    if (threadIdx.x == 0) {
        for (int s = 0; s < kStages; ++s) { mbar_init(&full[s], 1); mbar_init(&empty[s], W); }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == W) {                                      // ---- producer warp ----
        if (lane == 0) {
            for (int t = 0; t < ntiles; ++t) {
                const int s = t % kStages, use = t / kStages;
                if (use > 0) mbar_wait(&empty[s], (use - 1) & 1);
                const int nj = min(kTileAtoms, N - t * kTileAtoms);
                const uint32_t bytes = uint32_t(nj) * sizeof(double4);
                mbar_arrive_expect_tx(&full[s], bytes);
                bulk_copy_g2s(tiles + size_t(s) * kTileAtoms, a.xs + size_t(t) * kTileAtoms, bytes, &full[s]);
            }
        }
        return;
    }

    // ---- consumer warps ----
    const int g = lane / TPR, q = lane % TPR;
    const int row0 = blockIdx.x * RPC;
    int irow[IT];
    double xi[IT], yi[IT], zi[IT], si[IT];
    double acc0[IT], acc1[IT], acc2[IT], acc3[IT];
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        irow[k] = row0 + g * IT + k;
        const double4 p = a.xs[min(irow[k], N - 1)];
        xi[k] = p.x; yi[k] = p.y; zi[k] = p.z; si[k] = p.w;
        acc0[k] = acc1[k] = acc2[k] = acc3[k] = 0.0;
    }
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An;
    const int jl = warp * TPR + q, jstride = W * TPR;

    auto pair = [&](const double4 &p, int k) {
        const double dx = xi[k] - p.x, dy = yi[k] - p.y, dz = zi[k] - p.z;
        const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
        if constexpr (!FORCE) {
            if constexpr (ME > 0 && ME % 2 == 0) {
                const double w = rcp_fast(r2);
                if constexpr (ME == 6) { acc0[k] = fma(w * w, w, acc0[k]); }
                else acc0[k] += ipow_c<ME / 2>(w);
            } else if constexpr (ME > 0) {
                acc0[k] += ipow_c<ME>(rsqrt_fast(r2));
            } else {
                acc0[k] += ipow_rt(rsqrt_fast(r2), m_exp);
            }
        } else {
            const double y = rsqrt_fast(r2);
            const double w = y * y;
            const double ss = si[k] + p.w;
            double coef, pn;
            if constexpr (NE == 9 && ME == 6) {
                const double w2 = w * w, w4 = w2 * w2, y3 = w * y;
                coef = w4 * fma(An, y3, -ss);              // r^-8 (An r^-3 - (s_i'+s_j'))
                if constexpr (ENERGY) acc3[k] = fma(w4, y, acc3[k]);
                pn = 0.0;
            } else {
                const double pm = (ME > 0) ? ipow_c<ME>(y) : ipow_rt(y, m_exp);
                pn = (NE > 0) ? ipow_c<NE>(y) : ipow_rt(y, n_exp);
                coef = w * fma(An, pn, -ss * pm);
                if constexpr (ENERGY) acc3[k] += pn;
            }
            acc0[k] = fma(coef, dx, acc0[k]);
            acc1[k] = fma(coef, dy, acc1[k]);
            acc2[k] = fma(coef, dz, acc2[k]);
        }
    };

    for (int t = 0; t < ntiles; ++t) {
        const int s = t % kStages, use = t / kStages;
        const int j0 = t * kTileAtoms;
        const int nj = min(kTileAtoms, N - j0);
        const double4 *tile = tiles + size_t(s) * kTileAtoms;
        mbar_wait(&full[s], use & 1);
        const bool diag = (j0 < row0 + RPC) && (j0 + nj > row0);      // CTA-uniform
        if (!diag) {
#pragma unroll 4
            for (int j = jl; j < nj; j += jstride) {
                const double4 p = tile[j];
#pragma unroll
                for (int k = 0; k < IT; ++k) pair(p, k);
            }
        } else {
            for (int j = jl; j < nj; j += jstride) {
                const double4 p = tile[j];
#pragma unroll
                for (int k = 0; k < IT; ++k)
                    if (j0 + j != irow[k]) pair(p, k);                 // self term excluded by index
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    // ---- reduce over the TPR lanes of a row group, then over the W warps (fixed order) ----
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        acc0[k] = group_sum<TPR>(acc0[k]);
        if constexpr (FORCE) {
            acc1[k] = group_sum<TPR>(acc1[k]);
            acc2[k] = group_sum<TPR>(acc2[k]);
            acc3[k] = group_sum<TPR>(acc3[k]);
        }
    }
    named_bar_sync(1, W * 32);                            // every consumer is done with the tiles
    if (q == 0) {
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            double *dst = red + (size_t(warp) * RPC + g * IT + k) * NV;
            dst[0] = acc0[k];
            if constexpr (FORCE) { dst[1] = acc1[k]; dst[2] = acc2[k]; dst[3] = acc3[k]; }
        }
    }
    named_bar_sync(1, W * 32);
    double *fin = red + size_t(W) * RPC * NV;             // per-row scalar for the CTA partial
    const int tid = threadIdx.x;
    for (int r = tid; r < RPC; r += W * 32) {
        double v[NV];
#pragma unroll
        for (int c = 0; c < NV; ++c) v[c] = 0.0;
        for (int w = 0; w < W; ++w)
#pragma unroll
            for (int c = 0; c < NV; ++c) v[c] += red[(size_t(w) * RPC + r) * NV + c];
        const int i = row0 + r;
        double contrib = 0.0;
        if (i < N) {
            if constexpr (!FORCE) {
                const double rho = a.c.am * v[0];
                if (a.rho) a.rho[i] = rho;
                const double root = rho > 0.0 ? sqrt(rho) : 0.0;       // reading Q9: rho = 0 -> 0
                a.xs[i].w = rho > 0.0 ? a.c.Bm / root : 0.0;
                contrib = root;
            } else {
                a.force[3 * size_t(i) + 0] = v[0];
                a.force[3 * size_t(i) + 1] = v[1];
                a.force[3 * size_t(i) + 2] = v[2];
                contrib = v[3];
            }
        }
        fin[r] = contrib;
    }
    named_bar_sync(1, W * 32);
    if (tid == 0 && a.partial) {
        double tot = 0.0;
        for (int r = 0; r < RPC; ++r) tot += fin[r];
        a.partial[blockIdx.x] = tot;
    }
}

}  // namespace scmd
