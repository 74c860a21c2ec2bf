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
#include <type_traits>

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
    int row_begin, row_end;   // rows i this launch computes: [row_begin, row_end) (all of them: 0, N); j always runs over all N
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
    const int row0 = a.row_begin + blockIdx.x * RPC;
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
        if (i < a.row_end) {
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

// ---------------------------------------------------------------------------------------------
// Mixed precision: binary32 pair arithmetic, binary64 accumulation (BASELINE.json "mixed FP32-pair /
// FP64-accumulate path").  Same decomposition and TMA ring as the FP64 sweeps.
//
// Coordinates are split, x = xh + xl with xh = fl32(x), xl = fl32(x - xh), so the displacement
// (xh_i - xh_j) + (xl_i - xl_j) keeps the accuracy of a binary64 subtraction to within binary32
// rounding OF THE DIFFERENCE (positions rounded to binary32 first lose the force tolerance at
// N = 65536: SURVEY 8c-M).  1/r and 1/r^2 come from the MUFU seed + one Newton step.
//
// Everything is computed with Blackwell's packed binary32 pair instructions (PTX add/mul/fma.f32x2,
// SASS FADD2 / FMUL2 / FFMA2): one instruction works on TWO j atoms for the same row i, which halves
// the issue slots per pair so that the FMA pipes, not the scheduler, bound the sweep.  Atoms are
// therefore stored two to a 64-byte record (FPair), j-side values NEGATED (-xh, -xl, -s') so that
// only additions are needed:   d = (xh_i + (-xh_j)) + (xl_i + (-xl_j)).
// Partial sums run in packed binary32 over kF32Chunk records (2 x 8 atoms) of a thread and are then
// added into binary64 accumulators: FP32->FP64 conversion is an XU-pipe instruction (16 lanes/SM) and
// would bound the sweep if issued per pair.
// FMA-pipe lane-operations per ordered pair, (9, 6): sweep 1: 9 + 3 + 2 + 2 = 16;
//   sweep 2: 9 + 3 + 4 (rsqrt) + 4 (powers) + 1 + 2 + 3 + 1 (energy) = 27.
// ---------------------------------------------------------------------------------------------
static_assert(sizeof(FPair) == 2 * sizeof(double4), "two atoms per 64-byte record: same tile geometry");

constexpr int kF32Chunk = 8;          // records (of 2 atoms) between flushes into binary64

typedef unsigned long long f2;        // two packed binary32 values in one 64-bit register pair
__device__ __forceinline__ f2 f2_make(float lo, float hi) {
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 f2_dup(float v) { return f2_make(v, v); }
__device__ __forceinline__ float f2_lo(f2 v) { return __uint_as_float(unsigned(v)); }
__device__ __forceinline__ float f2_hi(f2 v) { return __uint_as_float(unsigned(v >> 32)); }
__device__ __forceinline__ f2 f2_add(f2 a, f2 b) { f2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 f2_mul(f2 a, f2 b) { f2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f2 f2_fma(f2 a, f2 b, f2 c) { f2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ float mufu_rsq(float x) { float y; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float mufu_rcp(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
template <int K>
__device__ __forceinline__ f2 f2_ipow_c(f2 u) {
    if constexpr (K == 1) return u;
    else if constexpr (K % 2 == 0) { f2 h = f2_ipow_c<K / 2>(u); return f2_mul(h, h); }
    else return f2_mul(f2_ipow_c<K - 1>(u), u);
}
__device__ __forceinline__ f2 f2_ipow_rt(f2 u, int k) {   // k >= 1
    f2 r = f2_dup(1.0f), b = u;
    while (k) { if (k & 1) r = f2_mul(r, b); b = f2_mul(b, b); k >>= 1; }
    return r;
}

struct AllPairs32Args {
    FPair *xf;            // [(N + kTileAtoms) / 2 + 1] packed records (negated split coordinates, -s')
    double4 *xs;          // [N] binary64 records: sweep 1 stores s' here too
    int n_atoms;
    int row_begin, row_end;   // rows i this launch computes (see AllPairsArgs)
    double *rho;
    double *force;
    double *partial;
    PairConsts c;
};

template <int IT, int TPR, int NE, int ME, bool FORCE, bool ENERGY>
__global__ void __launch_bounds__((kMaxConsumerWarps + 1) * 32, 1) allpairs32_kernel(const AllPairs32Args a) {
    constexpr int RPC = allpairs_rows_per_cta(IT, TPR);
    constexpr int NV = FORCE ? 4 : 1;
    constexpr int kTileRecs = kTileAtoms / 2;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);
    FPair *tiles = reinterpret_cast<FPair *>(smem_raw + kBarrierBytes);
    double *red = reinterpret_cast<double *>(smem_raw + kBarrierBytes);
    uint64_t *empty = full + kStages;

    const int W = (blockDim.x >> 5) - 1;
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
                const uint32_t bytes = uint32_t((nj + 1) / 2) * sizeof(FPair);
                mbar_arrive_expect_tx(&full[s], bytes);
                bulk_copy_g2s(tiles + size_t(s) * kTileRecs, a.xf + size_t(t) * kTileRecs, bytes, &full[s]);
            }
        }
        return;
    }

    const int g = lane / TPR, q = lane % TPR;
    const int row0 = a.row_begin + blockIdx.x * RPC;
    int irow[IT];
    f2 xh[IT], yh[IT], zh[IT], xl[IT], yl[IT], zl[IT], nsi[IT];      // row values duplicated into both halves
    f2 f0[IT], f1[IT], f2_[IT], f3[IT];
    double acc0[IT], acc1[IT], acc2[IT], acc3[IT];
    const f2 zero2 = f2_dup(0.f);
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        irow[k] = row0 + g * IT + k;
        const int ii = min(irow[k], N - 1);
        const float *rec = reinterpret_cast<const float *>(a.xf + (ii >> 1)) + (ii & 1);
        xh[k] = f2_dup(-rec[0]); yh[k] = f2_dup(-rec[2]); zh[k] = f2_dup(-rec[4]); nsi[k] = f2_dup(rec[6]);
        xl[k] = f2_dup(-rec[8]); yl[k] = f2_dup(-rec[10]); zl[k] = f2_dup(-rec[12]);
        f0[k] = f1[k] = f2_[k] = f3[k] = zero2;
        acc0[k] = acc1[k] = acc2[k] = acc3[k] = 0.0;
    }
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const f2 An2 = f2_dup(float(a.c.An));
    const f2 one2 = f2_dup(1.0f), mone2 = f2_dup(-1.0f), mhalf2 = f2_dup(-0.5f);

    // one record (atoms 2r, 2r+1 of the tile) against row k.  MASKED: drop the half whose mask is set
    // (self term, or the slot beyond an odd tile tail) -- its r^2 is replaced by 1 and its terms by 0.
    auto pair2 = [&](const ulonglong2 &A, const ulonglong2 &B, const ulonglong2 &C, const ulonglong2 &D, int k,
                     auto masked, bool mlo, bool mhi) {
        // A = (nxh, nyh), B = (nzh, ns), C = (nxl, nyl), D = (nzl, -)
        const f2 dx = f2_add(f2_add(xh[k], A.x), f2_add(xl[k], C.x));
        const f2 dy = f2_add(f2_add(yh[k], A.y), f2_add(yl[k], C.y));
        const f2 dz = f2_add(f2_add(zh[k], B.x), f2_add(zl[k], D.x));
        f2 r2 = f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx)));
        if constexpr (decltype(masked)::value) r2 = f2_make(mlo ? 1.0f : f2_lo(r2), mhi ? 1.0f : f2_hi(r2));
        if constexpr (!FORCE) {
            f2 term = zero2;
            if constexpr (ME > 0 && ME % 2 == 0) {
                // nw = -(1/r^2): seed of -x, e = 1 + x * (-y0), nw = (-y0) + (-y0) e
                const f2 ny0 = f2_make(mufu_rcp(-f2_lo(r2)), mufu_rcp(-f2_hi(r2)));
                const f2 e = f2_fma(r2, ny0, one2);
                const f2 nw = f2_fma(ny0, e, ny0);
                const f2 w2 = f2_mul(nw, nw);
                if constexpr (ME == 6) {
                    if constexpr (decltype(masked)::value) term = f2_mul(w2, nw);
                    else { f0[k] = f2_fma(w2, nw, f0[k]); return; }              // accumulates -r^-6
                } else {
                    // (-w)^(ME/2): sign fixed so that the accumulated term is always -r^-ME
                    term = f2_ipow_c<ME / 2>(nw);
                    if constexpr ((ME / 2) % 2 == 0) term = f2_mul(term, mone2);
                }
            } else {
                const f2 y0 = f2_make(mufu_rsq(f2_lo(r2)), mufu_rsq(f2_hi(r2)));
                const f2 ep = f2_fma(f2_mul(r2, y0), y0, mone2);
                const f2 y = f2_fma(f2_mul(y0, ep), mhalf2, y0);
                term = (ME > 0) ? f2_ipow_c<(ME > 0 ? ME : 1)>(y) : f2_ipow_rt(y, m_exp);
                term = f2_mul(term, mone2);
            }
            if constexpr (decltype(masked)::value) term = f2_make(mlo ? 0.f : f2_lo(term), mhi ? 0.f : f2_hi(term));
            f0[k] = f2_add(f0[k], term);
        } else {
            const f2 y0 = f2_make(mufu_rsq(f2_lo(r2)), mufu_rsq(f2_hi(r2)));
            const f2 ep = f2_fma(f2_mul(r2, y0), y0, mone2);          // t y0 - 1
            const f2 y = f2_fma(f2_mul(y0, ep), mhalf2, y0);          // y0 - y0 e' / 2
            const f2 w = f2_mul(y, y);
            const f2 nss = f2_add(nsi[k], B.y);                       // -(s'_i + s'_j)
            f2 coef, et = zero2;
            if constexpr (NE == 9 && ME == 6) {
                const f2 w2 = f2_mul(w, w), w4 = f2_mul(w2, w2), y3 = f2_mul(w, y);
                coef = f2_mul(w4, f2_fma(An2, y3, nss));              // r^-8 (An r^-3 - (s_i'+s_j'))
                if constexpr (ENERGY) {
                    if constexpr (decltype(masked)::value) et = f2_mul(w4, y);
                    else f3[k] = f2_fma(w4, y, f3[k]);
                }
            } else {
                const f2 pm = (ME > 0) ? f2_ipow_c<(ME > 0 ? ME : 1)>(y) : f2_ipow_rt(y, m_exp);
                const f2 pn = (NE > 0) ? f2_ipow_c<(NE > 0 ? NE : 1)>(y) : f2_ipow_rt(y, n_exp);
                coef = f2_mul(w, f2_fma(An2, pn, f2_mul(nss, pm)));
                if constexpr (ENERGY) {
                    if constexpr (decltype(masked)::value || !(NE == 9 && ME == 6)) et = pn;
                }
            }
            if constexpr (decltype(masked)::value) {
                coef = f2_make(mlo ? 0.f : f2_lo(coef), mhi ? 0.f : f2_hi(coef));
                if constexpr (ENERGY) et = f2_make(mlo ? 0.f : f2_lo(et), mhi ? 0.f : f2_hi(et));
            }
            if constexpr (ENERGY && (decltype(masked)::value || !(NE == 9 && ME == 6))) f3[k] = f2_add(f3[k], et);
            f0[k] = f2_fma(coef, dx, f0[k]);
            f1[k] = f2_fma(coef, dy, f1[k]);
            f2_[k] = f2_fma(coef, dz, f2_[k]);
        }
    };
    auto flush = [&]() {
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            acc0[k] += double(f2_lo(f0[k]) + f2_hi(f0[k])); f0[k] = zero2;
            if constexpr (FORCE) {
                acc1[k] += double(f2_lo(f1[k]) + f2_hi(f1[k])); f1[k] = zero2;
                acc2[k] += double(f2_lo(f2_[k]) + f2_hi(f2_[k])); f2_[k] = zero2;
                if constexpr (ENERGY) { acc3[k] += double(f2_lo(f3[k]) + f2_hi(f3[k])); f3[k] = zero2; }
            }
        }
    };
    const std::integral_constant<bool, false> kPlain{};
    const std::integral_constant<bool, true> kMasked{};

    // the W warps take contiguous slices of a tile's records; the TPR lanes of a row group interleave
    const int slice = (kTileRecs + W - 1) / W;
    for (int t = 0; t < ntiles; ++t) {
        const int s = t % kStages, use = t / kStages;
        const int j0 = t * kTileAtoms;
        const int nj = min(kTileAtoms, N - j0);
        const int nfull = nj >> 1;                                   // records with both atoms real
        const ulonglong2 *tile = reinterpret_cast<const ulonglong2 *>(tiles + size_t(s) * kTileRecs);
        mbar_wait(&full[s], use & 1);
        const bool diag = (j0 < row0 + RPC) && (j0 + nj > row0);      // CTA-uniform
        const int sb = warp * slice, se = min(sb + slice, nfull);
        int r = sb + q;
        if (!diag) {
            for (; r + (kF32Chunk - 1) * TPR < se; r += kF32Chunk * TPR) {
#pragma unroll
                for (int u = 0; u < kF32Chunk; ++u) {
                    const ulonglong2 *p = tile + 4 * (r + u * TPR);
                    const ulonglong2 A = p[0], B = p[1], C = p[2], D = p[3];
#pragma unroll
                    for (int k = 0; k < IT; ++k) pair2(A, B, C, D, k, kPlain, false, false);
                }
                flush();
            }
            for (; r < se; r += TPR) {
                const ulonglong2 *p = tile + 4 * r;
                const ulonglong2 A = p[0], B = p[1], C = p[2], D = p[3];
#pragma unroll
                for (int k = 0; k < IT; ++k) pair2(A, B, C, D, k, kPlain, false, false);
            }
        } else {
            for (int u = 0; r < se; r += TPR, ++u) {
                const ulonglong2 *p = tile + 4 * r;
                const ulonglong2 A = p[0], B = p[1], C = p[2], D = p[3];
#pragma unroll
                for (int k = 0; k < IT; ++k)                           // self term excluded by index
                    pair2(A, B, C, D, k, kMasked, j0 + 2 * r == irow[k], j0 + 2 * r + 1 == irow[k]);
                if ((u & (kF32Chunk - 1)) == kF32Chunk - 1) flush();
            }
        }
        if ((nj & 1) && warp == 0 && q == 0) {                        // odd tail: the last record holds one atom
            const ulonglong2 *p = tile + 4 * nfull;
            const ulonglong2 A = p[0], B = p[1], C = p[2], D = p[3];
#pragma unroll
            for (int k = 0; k < IT; ++k) pair2(A, B, C, D, k, kMasked, j0 + 2 * nfull == irow[k], true);
        }
        flush();
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

#pragma unroll
    for (int k = 0; k < IT; ++k) {
        acc0[k] = group_sum<TPR>(acc0[k]);
        if constexpr (FORCE) {
            acc1[k] = group_sum<TPR>(acc1[k]);
            acc2[k] = group_sum<TPR>(acc2[k]);
            acc3[k] = group_sum<TPR>(acc3[k]);
        }
    }
    named_bar_sync(1, W * 32);
    if (q == 0) {
#pragma unroll
        for (int k = 0; k < IT; ++k) {
            double *dst = red + (size_t(warp) * RPC + g * IT + k) * NV;
            dst[0] = acc0[k];
            if constexpr (FORCE) { dst[1] = acc1[k]; dst[2] = acc2[k]; dst[3] = acc3[k]; }
        }
    }
    named_bar_sync(1, W * 32);
    double *fin = red + size_t(W) * RPC * NV;
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
        if (i < a.row_end) {
            if constexpr (!FORCE) {
                const double rho = a.c.am * -v[0];                     // the sweep accumulates -r^-m
                if (a.rho) a.rho[i] = rho;
                const double root = rho > 0.0 ? sqrt(rho) : 0.0;       // reading Q9
                const double sp = rho > 0.0 ? a.c.Bm / root : 0.0;
                a.xs[i].w = sp;
                reinterpret_cast<float *>(a.xf + (i >> 1))[6 + (i & 1)] = -float(sp);
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
