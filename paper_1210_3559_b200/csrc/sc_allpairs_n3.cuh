// sc_allpairs_n3.cuh -- the two all-pairs sweeps with Newton's third law: every UNORDERED pair is
// evaluated once and its term is added to both atoms, 13 / 25 FP64 instructions per unordered pair instead of
// 2 x 11 / 2 x 22 for the two ordered pairs (PAPER.md:127 has one particle per thread and full N^2).
//
// Decomposition.  A CTA (12 warps) owns a block of RB = 32 * IT rows i; lane t of EVERY warp holds rows
// row0 + k * 32 + t (k < IT) in registers.  The j range is cut into chunks of 32 atoms; the block takes the chunks
// from its own first chunk to the end (the upper triangle), warp w every 12th of them.  For a chunk, lane t loads
// atom j = 32 c + t and the warp ROTATES the chunk through its lanes: 32 steps, in each of which a lane evaluates
// its IT rows against the j record it currently holds and then passes the record -- together with the reaction
// sums accumulated on it so far -- to the next lane by warp shuffles.  After 32 steps every record is back in its
// home lane carrying the sum over the warp's 32 * IT rows, and is stored as this block's partial for j.  No atomics,
// no shared memory in the loop; rows i accumulate in registers as in the one-sided sweeps.
//
// Diagonal: in the chunks that overlap the block's own rows a pair counts iff j > i (by index); pairs with i or j
// beyond N are evaluated on dummy records 1e100 away, whose terms underflow to exact zeros.
//
// Sums.  part[b][j] (j >= first row of block b: triangular storage) holds block b's reaction sums, self[i] the
// row sums of i's own block, one per j segment; a finalize kernel adds self[0..][i] + part[0..block(i)][i] in that fixed order, so the
// result is bit-reproducible.  Storage: ~N^2 / (2 RB) records of 32 bytes (0.54 GB at N = 65536), which is what
// limits the variant to N <= 131072.
#pragma once
#include "sc_allpairs.cuh"
#include "sc_device.cuh"

namespace scmd {

constexpr int kN3Warps = 12;
constexpr double kN3Far = 1.0e100;

struct N3Args {
    const double4 *xs;      // [N] (x, y, z, s')
    int n_atoms, n_pad;     // n_pad = round_up(N, 32)
    double4 *part;          // triangular: block b at offset n3_part_offset(b), n_pad - b * RB records (FORCE) ...
    double *part_rho;       // ... or doubles (density sweep); the same memory
    double4 *self;          // [gridDim.y][n_pad] row sums per j segment (x, y, z) / (rho, -, -)
    double *partial;        // [gridDim.y * gridDim.x] per-CTA sum r^-n over ORDERED pairs (FORCE && ENERGY)
    int seg_chunks;         // chunks of 32 atoms per j segment: CTA (b, s) takes chunks cb(b) + s L .. + L of block b's
                            //   triangle, so that all CTAs carry about the same work (a triangle cut by rows only leaves
                            //   the SMs idle at the end: measured 6 % at N = 65536, 20 % at N = 32768)
    PairConsts c;
};

__host__ __device__ inline size_t n3_part_offset(int b, int n_pad, int rb) {
    return size_t(b) * size_t(n_pad) - size_t(rb) * (size_t(b) * size_t(b > 0 ? b - 1 : 0) / 2);
}
inline size_t n3_part_records(int n_atoms, int rb) {
    const int n_pad = (n_atoms + 31) / 32 * 32, nb = (n_atoms + rb - 1) / rb;
    return n3_part_offset(nb, n_pad, rb);
}

__device__ __forceinline__ double rot1(double v) { return __shfl_sync(0xffffffffu, v, (threadIdx.x + 1) & 31); }
__device__ __forceinline__ int rot1(int v) { return __shfl_sync(0xffffffffu, v, (threadIdx.x + 1) & 31); }

template <int IT, int NE, int ME, bool FORCE, bool ENERGY>
__global__ void __launch_bounds__(kN3Warps * 32, 1) allpairs_n3_kernel(const N3Args a) {
    constexpr int RB = 32 * IT;
    __shared__ double red[kN3Warps][IT][3][32];            // epilogue: per-warp row sums
    __shared__ double red_e[kN3Warps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = a.n_atoms;
    const int row0 = blockIdx.x * RB;
    if ((row0 >> 5) + int(blockIdx.y) * a.seg_chunks >= ((a.n_atoms + 31) >> 5)) {   // no such segment in this block's triangle
        if (FORCE && ENERGY && threadIdx.x == 0) a.partial[blockIdx.y * gridDim.x + blockIdx.x] = 0.0;
        return;
    }
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An;

    int irow[IT];
    double xi[IT], yi[IT], zi[IT], si[IT];
    double f0[IT], f1[IT], f2[IT];
    double esum = 0.0;
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        irow[k] = row0 + k * 32 + lane;
        if (irow[k] < N) {
            const double4 p = a.xs[irow[k]];
            xi[k] = p.x; yi[k] = p.y; zi[k] = p.z; si[k] = p.w;
        } else {                                           // dummy row: far from everything, also from the dummy j
            xi[k] = kN3Far * double(k + 2); yi[k] = -kN3Far * double(lane + 1); zi[k] = 0.0; si[k] = 0.0;
        }
        f0[k] = f1[k] = f2[k] = 0.0;
    }

    const int cb = row0 >> 5, nch = (N + 31) >> 5;
    const int c_begin = cb + int(blockIdx.y) * a.seg_chunks, c_end = min(nch, c_begin + a.seg_chunks);
    double4 *part = a.part + n3_part_offset(blockIdx.x, a.n_pad, RB);
    double *part_rho = a.part_rho + n3_part_offset(blockIdx.x, a.n_pad, RB);
    for (int c = c_begin + warp; c < c_end; c += kN3Warps) {
        int jidx = (c << 5) + lane;
        double xj, yj, zj, sj;
        if (jidx < N) {
            const double4 p = a.xs[jidx];
            xj = p.x; yj = p.y; zj = p.z; sj = p.w;
        } else {
            xj = -kN3Far * double(lane + 1); yj = kN3Far; zj = kN3Far; sj = 0.0;
        }
        const int jhome = jidx;
        double g0 = 0.0, g1 = 0.0, g2 = 0.0;               // reaction sums travelling with the record
        const bool diag = c < cb + IT;                     // warp-uniform
        auto step = [&](auto masked) {
            // the record of the NEXT step is fetched first (positions do not change): its shuffle latency hides
            // behind this step's arithmetic; only the reaction sums have to wait for it
            const double xn = rot1(xj), yn = rot1(yj), zn = rot1(zj);
            double sn = 0.0;
            if constexpr (FORCE) sn = rot1(sj);
            int jn = 0;
            if constexpr (decltype(masked)::value) jn = rot1(jidx);
#pragma unroll
            for (int k = 0; k < IT; ++k) {
                const double dx = xi[k] - xj, dy = yi[k] - yj, dz = zi[k] - zj;
                const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
                if constexpr (!FORCE) {
                    double term;
                    if constexpr (ME > 0 && ME % 2 == 0) {
                        double w = rcp_fast(r2);
                        if constexpr (decltype(masked)::value) w = jidx > irow[k] ? w : 0.0;
                        term = ipow_c<ME / 2>(w);
                    } else {
                        double y = rsqrt_fast(r2);
                        if constexpr (decltype(masked)::value) y = jidx > irow[k] ? y : 0.0;
                        term = (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
                    }
                    f0[k] += term;
                    g0 += term;
                } else {
                    double y = rsqrt_fast(r2);
                    if constexpr (decltype(masked)::value) y = jidx > irow[k] ? y : 0.0;
                    const double w = y * y;
                    const double ss = si[k] + sj;
                    double coef, pn;
                    if constexpr (NE == 9 && ME == 6) {
                        const double w2 = w * w, w4 = w2 * w2, y3 = w * y;
                        coef = w4 * fma(An, y3, -ss);
                        pn = w4 * y;
                    } else {
                        const double pm = (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
                        pn = (NE > 0) ? ipow_c<(NE > 0 ? NE : 1)>(y) : ipow_rt(y, n_exp);
                        coef = w * fma(An, pn, -ss * pm);
                    }
                    if constexpr (ENERGY) esum += pn;
                    f0[k] = fma(coef, dx, f0[k]); f1[k] = fma(coef, dy, f1[k]); f2[k] = fma(coef, dz, f2[k]);
                    g0 = fma(-coef, dx, g0); g1 = fma(-coef, dy, g1); g2 = fma(-coef, dz, g2);
                }
            }
            // pass the sums on with the record
            g0 = rot1(g0);
            if constexpr (FORCE) { g1 = rot1(g1); g2 = rot1(g2); sj = sn; }
            xj = xn; yj = yn; zj = zn;
            if constexpr (decltype(masked)::value) jidx = jn;
        };
        if (diag) {
            for (int s = 0; s < 32; ++s) step(std::integral_constant<bool, true>{});
        } else {
#pragma unroll 4
            for (int s = 0; s < 32; ++s) step(std::integral_constant<bool, false>{});
        }
        // the record is home again (32 rotations by one lane)
        if (jhome < N) {
            if constexpr (FORCE) part[jhome - row0] = make_double4(g0, g1, g2, 0.0);
            else part_rho[jhome - row0] = g0;
        }
    }

    // ---- rows i: sum over the warps of the CTA in a fixed order ----
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        red[warp][k][0][lane] = f0[k];
        if constexpr (FORCE) { red[warp][k][1][lane] = f1[k]; red[warp][k][2][lane] = f2[k]; }
    }
    if constexpr (FORCE && ENERGY) {
        esum = warp_sum(esum);
        if (lane == 0) red_e[warp] = esum;
    }
    __syncthreads();
    for (int r = threadIdx.x; r < RB; r += kN3Warps * 32) {
        const int k = r >> 5, l = r & 31, i = row0 + r;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        for (int w = 0; w < kN3Warps; ++w) {
            v0 += red[w][k][0][l];
            if constexpr (FORCE) { v1 += red[w][k][1][l]; v2 += red[w][k][2][l]; }
        }
        if (i < N) a.self[size_t(blockIdx.y) * a.n_pad + i] = make_double4(v0, v1, v2, 0.0);
    }
    if constexpr (FORCE && ENERGY) {
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < kN3Warps; ++w) tot += red_e[w];
            a.partial[blockIdx.y * gridDim.x + blockIdx.x] = 2.0 * tot;   // every unordered pair stands for two ordered ones
        }
    }
}

// ---- mixed precision: the same rotation in binary32 on split records (x = xh + xl, RecF), binary64 accumulation ----
// Rows accumulate in binary32 over one chunk (32 terms) and are then added into binary64 sums; the reaction sums
// travel in binary32 (128 terms) and are stored as binary64 partials.  No binary64 instruction in the rotation.
// Sweep 1 keeps TWO binary32 sums per accumulator, one for pairs closer than 20 A and one for the rest: a far term
// (r^-6 ~ 1e-11) added to a sum that already holds a nearest-neighbour term (4e-3) would be absorbed entirely, a
// one-sided loss that biased rho by ~1.5e-7 and the energy by 6-8e-8 of BASELINE.json's 1e-7 (measured before the
// split); the energy and force terms of sweep 2 fall off as r^-9, r^-10 and need no such care.
__device__ __forceinline__ float rot1(float v) { return __shfl_sync(0xffffffffu, v, (threadIdx.x + 1) & 31); }

struct N3FArgs {
    const RecF *xfr;        // [N] split binary32 records
    int n_atoms, n_pad;
    double4 *part;
    double *part_rho;
    double4 *self;
    double *partial;
    int seg_chunks;
    PairConsts c;
};

template <int IT, int NE, int ME, bool FORCE, bool ENERGY>
__global__ void __launch_bounds__(kN3Warps * 32, 1) allpairs_n3f_kernel(const N3FArgs a) {
    constexpr int RB = 32 * IT;
    __shared__ double red[kN3Warps][IT][3][32];
    __shared__ double red_e[kN3Warps];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int N = a.n_atoms;
    const int row0 = blockIdx.x * RB;
    if ((row0 >> 5) + int(blockIdx.y) * a.seg_chunks >= ((a.n_atoms + 31) >> 5)) {   // no such segment in this block's triangle
        if (FORCE && ENERGY && threadIdx.x == 0) a.partial[blockIdx.y * gridDim.x + blockIdx.x] = 0.0;
        return;
    }
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const float Anf = float(a.c.An);
    constexpr float kFarF = 1.0e15f;                       // r^2 ~ 1e30 stays finite, its reciprocal powers vanish

    int irow[IT];
    RecF pi[IT];
    double F0[IT], F1[IT], F2[IT];
    double esum = 0.0;
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        irow[k] = row0 + k * 32 + lane;
        if (irow[k] < N) pi[k] = a.xfr[irow[k]];
        else pi[k] = RecF{kFarF * float(k + 2), -kFarF * float(lane + 1), 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        F0[k] = F1[k] = F2[k] = 0.0;
    }
    const int cb = row0 >> 5, nch = (N + 31) >> 5;
    const int c_begin = cb + int(blockIdx.y) * a.seg_chunks, c_end = min(nch, c_begin + a.seg_chunks);
    double4 *part = a.part + n3_part_offset(blockIdx.x, a.n_pad, RB);
    double *part_rho = a.part_rho + n3_part_offset(blockIdx.x, a.n_pad, RB);
    for (int c = c_begin + warp; c < c_end; c += kN3Warps) {
        int jidx = (c << 5) + lane;
        RecF pj;
        if (jidx < N) pj = a.xfr[jidx];
        else pj = RecF{-kFarF * float(lane + 1), kFarF, kFarF, 0.f, 0.f, 0.f, 0.f, 0.f};
        const int jhome = jidx;
        float g0 = 0.f, g1 = 0.f, g2 = 0.f, e32 = 0.f, gfar = 0.f;
        float f0[IT], f1[IT], f2[IT], ffar[IT];
#pragma unroll
        for (int k = 0; k < IT; ++k) f0[k] = f1[k] = f2[k] = ffar[k] = 0.f;
        const bool diag = c < cb + IT;
        auto step = [&](auto masked) {
            RecF pn;
            pn.xh = rot1(pj.xh); pn.yh = rot1(pj.yh); pn.zh = rot1(pj.zh);
            pn.xl = rot1(pj.xl); pn.yl = rot1(pj.yl); pn.zl = rot1(pj.zl);
            pn.s = 0.f; pn.pad = 0.f;
            if constexpr (FORCE) pn.s = rot1(pj.s);
            int jn = 0;
            if constexpr (decltype(masked)::value) jn = rot1(jidx);
#pragma unroll
            for (int k = 0; k < IT; ++k) {
                const float dx = (pi[k].xh - pj.xh) + (pi[k].xl - pj.xl), dy = (pi[k].yh - pj.yh) + (pi[k].yl - pj.yl);
                const float dz = (pi[k].zh - pj.zh) + (pi[k].zl - pj.zl);
                const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
                if constexpr (!FORCE) {
                    float term;
                    if constexpr (ME > 0 && ME % 2 == 0) {
                        float w = rcp_fast_f(r2);
                        if constexpr (decltype(masked)::value) w = jidx > irow[k] ? w : 0.f;
                        term = ipow_cf<ME / 2>(w);
                    } else {
                        float y = rsqrt_fast_f(r2);
                        if constexpr (decltype(masked)::value) y = jidx > irow[k] ? y : 0.f;
                        term = (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
                    }
                    const bool far = r2 > 400.0f;                    // 20 A
                    const float tn = far ? 0.f : term, tf = far ? term : 0.f;
                    f0[k] += tn; ffar[k] += tf;
                    g0 += tn; gfar += tf;
                } else {
                    float y = rsqrt_fast_f(r2);
                    if constexpr (decltype(masked)::value) y = jidx > irow[k] ? y : 0.f;
                    const float w = y * y;
                    const float ss = pi[k].s + pj.s;
                    float coef, pnw;
                    if constexpr (NE == 9 && ME == 6) {
                        const float w2 = w * w, w4 = w2 * w2, y3 = w * y;
                        coef = w4 * fmaf(Anf, y3, -ss);
                        pnw = w4 * y;
                    } else {
                        const float pm = (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
                        pnw = (NE > 0) ? ipow_cf<(NE > 0 ? NE : 1)>(y) : ipow_rtf(y, n_exp);
                        coef = w * fmaf(Anf, pnw, -ss * pm);
                    }
                    if constexpr (ENERGY) e32 += pnw;
                    f0[k] = fmaf(coef, dx, f0[k]); f1[k] = fmaf(coef, dy, f1[k]); f2[k] = fmaf(coef, dz, f2[k]);
                    g0 = fmaf(-coef, dx, g0); g1 = fmaf(-coef, dy, g1); g2 = fmaf(-coef, dz, g2);
                }
            }
            g0 = rot1(g0);
            if constexpr (FORCE) { g1 = rot1(g1); g2 = rot1(g2); }
            else gfar = rot1(gfar);
            pj = pn;
            if constexpr (decltype(masked)::value) jidx = jn;
        };
        if (diag) {
            for (int s = 0; s < 32; ++s) step(std::integral_constant<bool, true>{});
        } else {
#pragma unroll 4
            for (int s = 0; s < 32; ++s) step(std::integral_constant<bool, false>{});
        }
        if (jhome < N) {
            if constexpr (FORCE) part[jhome - row0] = make_double4(double(g0), double(g1), double(g2), 0.0);
            else part_rho[jhome - row0] = double(g0) + double(gfar);
        }
#pragma unroll
        for (int k = 0; k < IT; ++k) {                     // one chunk of binary32 row sums into binary64
            F0[k] += double(f0[k]);
            if constexpr (!FORCE) F0[k] += double(ffar[k]);
            if constexpr (FORCE) { F1[k] += double(f1[k]); F2[k] += double(f2[k]); }
        }
        if constexpr (FORCE && ENERGY) esum += double(e32);
    }
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        red[warp][k][0][lane] = F0[k];
        if constexpr (FORCE) { red[warp][k][1][lane] = F1[k]; red[warp][k][2][lane] = F2[k]; }
    }
    if constexpr (FORCE && ENERGY) {
        esum = warp_sum(esum);
        if (lane == 0) red_e[warp] = esum;
    }
    __syncthreads();
    for (int r = threadIdx.x; r < RB; r += kN3Warps * 32) {
        const int k = r >> 5, l = r & 31, i = row0 + r;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        for (int w = 0; w < kN3Warps; ++w) {
            v0 += red[w][k][0][l];
            if constexpr (FORCE) { v1 += red[w][k][1][l]; v2 += red[w][k][2][l]; }
        }
        if (i < N) a.self[size_t(blockIdx.y) * a.n_pad + i] = make_double4(v0, v1, v2, 0.0);
    }
    if constexpr (FORCE && ENERGY) {
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < kN3Warps; ++w) tot += red_e[w];
            a.partial[blockIdx.y * gridDim.x + blockIdx.x] = 2.0 * tot;
        }
    }
}

// ---- finalize: self[i] + part[0 .. block(i)][i] in that order ----
struct N3FinalArgs {
    double4 *xs;
    RecF *xfr;                          // mixed: sweep 1 stores fl32(s') here as well (else NULL)
    FPair *xf;                          // mixed: ... and into the packed records of the one-sided sweeps
    const double4 *part;
    const double *part_rho;
    const double4 *self;
    double *rho, *force, *partial;      // partial: [gridDim.x] sum sqrt(rho) (density)
    int n_atoms, n_pad, rb, seg_chunks;
    PairConsts c;
};

#ifdef SCMD_MAIN_TU
template <bool FORCE>
__global__ void __launch_bounds__(256) n3_finalize_kernel(const N3FinalArgs a) {
    __shared__ double scratch[32];
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    double contrib = 0.0;
    if (i < a.n_atoms) {
        const int bi = i / a.rb;
        const int nseg = (((a.n_atoms + 31) >> 5) - ((bi * a.rb) >> 5) + a.seg_chunks - 1) / a.seg_chunks;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        for (int sg = 0; sg < nseg; ++sg) {                 // row sums of the segments of i's own block
            const double4 s = a.self[size_t(sg) * a.n_pad + i];
            v0 += s.x; v1 += s.y; v2 += s.z;
        }
        for (int b = 0; b <= bi; ++b) {
            const size_t at = n3_part_offset(b, a.n_pad, a.rb) + size_t(i - b * a.rb);
            if constexpr (FORCE) {
                const double4 p = a.part[at];
                v0 += p.x; v1 += p.y; v2 += p.z;
            } else {
                v0 += a.part_rho[at];
            }
        }
        if constexpr (FORCE) {
            a.force[3 * size_t(i)] = v0; a.force[3 * size_t(i) + 1] = v1; a.force[3 * size_t(i) + 2] = v2;
        } else {
            const double rho = a.c.am * v0;
            if (a.rho) a.rho[i] = rho;
            const double root = rho > 0.0 ? sqrt(rho) : 0.0;           // reading Q9
            const double sp = rho > 0.0 ? a.c.Bm / root : 0.0;
            a.xs[i].w = sp;
            if (a.xfr) a.xfr[i].s = float(sp);
            if (a.xf) reinterpret_cast<float *>(a.xf + (i >> 1))[6 + (i & 1)] = -float(sp);
            contrib = root;
        }
    }
    if constexpr (!FORCE) {
        const double t = block_sum(contrib, scratch);
        if (threadIdx.x == 0) a.partial[blockIdx.x] = t;
    }
}
#endif  // SCMD_MAIN_TU

// instantiated in inst_allpairs_n3.cu; nullptr if this shape is not compiled
const void *allpairs_n3_fn(int it, bool fast, bool force, bool energy);
const void *allpairs_n3f_fn(int it, bool fast, bool force, bool energy);      // mixed precision

}  // namespace scmd
