// sc_allpairs_n3.cuh -- the two all-pairs sweeps with Newton's third law: every UNORDERED pair is
// evaluated once and its term is added to both atoms, 13 / 25 FP64 instructions per unordered pair instead of
// 2 x 11 / 2 x 22 for the two ordered pairs (PAPER.md:127 has one particle per thread and full N^2).
//
// Decomposition.  A row block is RB = 32 * IT rows i; lane t of every warp that works on it holds rows
// row0 + k * 32 + t (k < IT) in registers.  (A CTA of 12 warps holds a PAIR of row blocks, six warps each: see
// n3_sweep_piece.)  The j range is cut into chunks of 32 atoms; a block takes the chunks from its own first chunk to the
// end (the upper triangle), its warps in turn.  For a chunk, lane t loads
// atom j = 32 c + t and the warp ROTATES the chunk through its lanes: 32 steps, in each of which a lane evaluates
// its IT rows against the j record it currently holds and then passes the record -- together with the reaction
// sums accumulated on it so far -- to the next lane by warp shuffles.  After 32 steps every record is back in its
// home lane carrying the sum over the warp's 32 * IT rows, and is stored as the block's partial for j (after the sums
// of the pair's second row block have been added).  No atomics; rows i accumulate in registers as in the one-sided
// sweeps.  (Since round 2 the records of the chunk sit in shared memory and only the sums travel: see the kernel.)
//
// Diagonal: in the chunks that overlap the block's own rows a pair counts iff j > i (by index); pairs with i or j
// beyond N are evaluated on dummy records 1e100 away, whose terms underflow to exact zeros.
//
// Sums.  part[b][j] (j >= first row of PAIR block b: triangular storage) holds the pair block's reaction sums, self[i]
// the row sums of i's own block, one per tile; a finalize kernel adds self[0..][i] + part[0..block(i)][i] in that fixed
// order, so the result is bit-reproducible.  Storage: ~N^2 / (4 RB) records of 32 bytes (0.27 GB at N = 65536, 4.3 GB at
// 262144, the top of the range: kN3MaxAtoms in scmd.cu).
#pragma once
#ifndef SCMD_N3P_UNROLL
#define SCMD_N3P_UNROLL 4      // rotation steps unrolled in the mixed sweeps: 2 x this
#endif
#include "sc_allpairs.cuh"
#include "sc_device.cuh"

namespace scmd {

constexpr int kN3Warps = 12;          // warps per SM the register allocation allows (168 registers): ONE CTA of 12 or TWO of 6
constexpr double kN3Far = 1.0e100;
constexpr float kN3FarTerm = 1.4901161193847656e-08f;   // 2^-26: r^-6 of a pair 20 A apart (mixed sweep 1: near / far sums)

// A tile: chunks [c_begin, c_end) of row block b's part of the triangle (chunks of 32 atoms, the packed mixed kernel: of
// 64), whose row sums go to self[slot].  The host cuts the triangle -- row block after row block, ~N^2 / 8192 chunks --
// into one PIECE per CTA of equal cost, a piece being a few consecutive tiles (a long row block is cut into several
// tiles, each with its own slot; a piece at the narrow end of the triangle holds several short row blocks).  Round 1 and
// early round 2 launched a (row block, j segment) grid with ONE segment length for all row blocks: at N = 8000 that is 140
// CTAs of 2 ... 6 rounds of the 12 warps each, and the sweep lasted as long as the 6-round ones.
struct N3Tile { int b, c_begin, c_end, slot; };

struct N3Args {
    const double4 *xs;      // [N] (x, y, z, s')
    int n_atoms, n_pad;     // n_pad = round_up(N, 32)
    double4 *part;          // triangular: block b at offset n3_part_offset(b), n_pad - b * RB records (FORCE) ...
    double *part_rho;       // ... or doubles (density sweep); the same memory
    double4 *self;          // [gridDim.y][n_pad] row sums per j segment (x, y, z) / (rho, -, -)
    double *partial;        // [gridDim.x] per-CTA sum r^-n over ORDERED pairs (FORCE && ENERGY)
    const N3Tile *tiles;    // the plan (scmd.cu, plan_n3): CTA p works through tiles[piece_start[p] .. piece_start[p + 1])
    const int *piece_start;
    PairConsts c;
};

__host__ __device__ inline size_t n3_part_offset(int b, int n_pad, int rb) {
    return size_t(b) * size_t(n_pad) - size_t(rb) * (size_t(b) * size_t(b > 0 ? b - 1 : 0) / 2);
}
inline size_t n3_part_records(int n_atoms, int rb) {
    const int n_pad = (n_atoms + 31) / 32 * 32, nb = (n_atoms + rb - 1) / rb;
    return n3_part_offset(nb, n_pad, rb);
}

__device__ __forceinline__ double rot1(double v) {   // as a 64-bit integer: two SHFL on the register pair, no repacking
    return __longlong_as_double(__shfl_sync(0xffffffffu, __double_as_longlong(v), (threadIdx.x + 1) & 31));
}
// The MUFU seeds of 1 / x and x^-1/2 come as a high word; the library form (sc_device.cuh) completes them with a ZERO low
// word, one move per seed (4 of the 116 instructions of a rotation step).  Any low word will do: it perturbs the seed by
// < 2^-20 relative, about the seed's own error, and the cubic refinement leaves (2 e0)^3 ~ 2^-57 of it.  Here the low
// word is that of `dead`, a value the caller no longer needs (the partial sum dx^2 + dy^2), so that the seed can take
// over its register pair and no move is issued.  Deterministic: the bits are a function of the inputs alone.
__device__ __forceinline__ double seed_with_low_of(double seed, double dead) {
    return __hiloint2double(__double2hiint(seed), __double2loint(dead));
}
__device__ __forceinline__ double rcp_fast_lo(double x, double dead) {
    const double y0 = seed_with_low_of(rcp_seed(x), dead);
    const double e = fma(-x, y0, 1.0);
    return fma(y0, fma(e, e, e), y0);
}
__device__ __forceinline__ double rsqrt_fast_lo(double x, double dead) {
    const double y0 = seed_with_low_of(rsqrt_seed(x), dead);
    const double tt = x * y0, e = fma(-tt, y0, 1.0);
    return fma(y0, e * fma(0.375, e, 0.5), y0);
}

// Row blocks come in PAIRS (late round 2): a tile is a run of chunks of a pair block of 2 RB rows.  Warps 0 .. NW/2 - 1 hold
// the first RB rows in registers (set A), warps NW/2 .. NW - 1 the second RB rows (set B); warp p of A and warp p of B
// rotate the SAME chunk, each against its own rows, B hands its reaction sums to A through shared memory (two named
// barriers of 64 threads per chunk) and A stores ONE partial record per (pair block, j): N^2 / 512 records instead of
// N^2 / 256 -- half the workspace (4.3 GB at N = 262144), half the DRAM writes of sweep 2 (215 MB at N = 65536) and half
// the reads of the finalize.  Set B has no pairs in the first IT chunks of the pair block (they are below its diagonal).
// The hand-over is a producer / consumer pair of named barriers per warp pair (PTX bar.arrive / bar.sync, 64 threads):
// FULL -- B arrives after writing a slot, A waits before reading it; EMPTY -- A arrives after reading, B waits before it
// writes the slot again.  Neither warp waits for the other in step: B may finish the next chunk's rotation before A has
// read this one, A waits only when B is behind.  ONE slot per pair: a barrier counts threads, not roles, so with two slots
// A could arrive twice at EMPTY before B waits once and complete it alone (tried: deadlock).  (One symmetric bar.sync per chunk cost the density sweep 1.5 %: the two warps stalled together.)
__device__ __forceinline__ void n3_full_arrive(int pair) {
    __threadfence_block();
    asm volatile("bar.arrive %0, 64;" ::"r"(2 * pair + 1) : "memory");
}
__device__ __forceinline__ void n3_full_wait(int pair) { asm volatile("bar.sync %0, 64;" ::"r"(2 * pair + 1) : "memory"); }
__device__ __forceinline__ void n3_empty_arrive(int pair) { asm volatile("bar.arrive %0, 64;" ::"r"(2 * pair + 2) : "memory"); }
__device__ __forceinline__ void n3_empty_wait(int pair) { asm volatile("bar.sync %0, 64;" ::"r"(2 * pair + 2) : "memory"); }
constexpr int kN3SlotBytes = 3 * 32 * 8;              // reaction sums of one warp's chunk on their way from set B to set A

// One CTA's piece of a sweep (the whole of allpairs_n3_kernel; a phase of n3_loop_kernel, sc_n3_loop.cuh).
// red: per-warp row sums of the epilogue, also the chunk records during the rotation; red_e: per-warp energy sums.
template <int IT, int NE, int ME, bool FORCE, bool ENERGY>
__device__ __forceinline__ void n3_sweep_piece(const N3Args &a, const int piece, double (&red)[kN3Warps][IT][3][32],
                                               double (&red_e)[kN3Warps], unsigned char *slots /* kN3Warps / 2 x kN3SlotBytes */) {
    constexpr int RB = 32 * IT;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int NW = blockDim.x >> 5;                          // 12, or 6 (two CTAs per SM: finer tiles for mid-size clusters)
    const int H = NW >> 1, set = warp >= H ? 1 : 0, wp = warp - set * H;   // row set (A: 0, B: 1), index of the warp pair
    double *slot = reinterpret_cast<double *>(slots + wp * kN3SlotBytes);
    int nx = 0;                                              // exchanges so far (the same count in both warps of the pair)
    const int N = a.n_atoms;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An;
    double esum = 0.0;
    const int t_end = a.piece_start[piece + 1];
    for (int t = a.piece_start[piece]; t < t_end; ++t) {
    const N3Tile tile = a.tiles[t];
    const int row0p = tile.b * 2 * RB;                       // first row of the pair block
    const int row0 = row0p + set * RB;                       // ... and of this warp's row set

    int irow[IT];
    double xi[IT], yi[IT], zi[IT], si[IT];
    double f0[IT], f1[IT], f2[IT];
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

    const int cb = row0 >> 5, cbB = (row0p >> 5) + IT;        // first chunk of this set's rows; of set B's rows
    const int c_begin = tile.c_begin, c_end = tile.c_end;
    double4 *part = a.part + n3_part_offset(tile.b, a.n_pad, 2 * RB);
    double *part_rho = a.part_rho + n3_part_offset(tile.b, a.n_pad, 2 * RB);
    // The 32 records of a chunk do not change while the warp rotates it: they sit in shared memory (1 KB per warp, in the
    // space the epilogue's reduction uses afterwards; (x, y) and (z, s') as two 16-byte arrays: conflict-free), and at
    // step s a lane READS the record of lane + s -- two LDS.128 instead of eight shuffles and the moves that go with
    // them.  Only the reaction sums travel from lane to lane.
    // Each record is stored twice, at lane and at lane + 32, so that the index lane + s + 1 never wraps: with the steps
    // unrolled the address is one register plus an immediate (3 integer instructions per step less).
    static_assert(IT >= 3, "2 KB of chunk records per warp must fit into the warp's part of red");
    double2 *jxy = reinterpret_cast<double2 *>(&red[0][0][0][0]) + warp * 128, *jzs = jxy + 64;
    for (int c = c_begin + wp; c < c_end; c += H) {
        const int jidx = (c << 5) + lane;
        const bool both = c >= cbB;                        // set B has pairs in this chunk (the same for the two warps)
        double g0 = 0.0, g1 = 0.0, g2 = 0.0;
        if (set == 0 || both) {
        double xj, yj, zj, sj;
        if (jidx < N) {
            const double4 p = a.xs[jidx];
            xj = p.x; yj = p.y; zj = p.z; sj = p.w;
        } else {
            xj = -kN3Far * double(lane + 1); yj = kN3Far; zj = kN3Far; sj = 0.0;
        }
        const bool diag = c < cb + IT;                     // warp-uniform
        // One rotation step: evaluate the IT rows against the record held (`in`), hand it on with the reaction sums
        // accumulated on it so far (`out`).  Two register sets alternate (A -> B, B -> A): no value is ever moved back
        // into a loop-carried register (10 moves per step when the step updated one set in place).
        struct JRec { double x, y, z, s, g0, g1, g2; };
        __syncwarp();                                      // the previous chunk's readers are done
        jxy[lane] = make_double2(xj, yj); jzs[lane] = make_double2(zj, sj);
        jxy[lane + 32] = make_double2(xj, yj); jzs[lane + 32] = make_double2(zj, sj);
        __syncwarp();
        const int jbase = c << 5;
        auto step = [&](auto masked, int s, const JRec &in, JRec &out) {
            const double xj = in.x, yj = in.y, zj = in.z, sj = in.s;
            const int jidx = jbase + ((lane + s) & 31);
            double g0 = in.g0, g1 = in.g1, g2 = in.g2;     // reaction sums travelling with the record
            {   // the record of the NEXT step is fetched first: its latency hides behind this step's arithmetic
                const int nx = lane + s + 1;               // <= 63: the second copy
                const double2 pxy = jxy[nx], pzs = jzs[nx];
                out.x = pxy.x; out.y = pxy.y; out.z = pzs.x; out.s = pzs.y;
            }
#pragma unroll
            for (int k = 0; k < IT; ++k) {
                const double dx = xi[k] - xj, dy = yi[k] - yj, dz = zi[k] - zj;
                const double r2xy = fma(dy, dy, dx * dx);
                const double r2 = fma(dz, dz, r2xy);
                if constexpr (!FORCE) {
                    double term;
                    if constexpr (ME > 0 && ME % 2 == 0) {
                        double w = rcp_fast_lo(r2, r2xy);
                        if constexpr (decltype(masked)::value) w = jidx > irow[k] ? w : 0.0;
                        term = ipow_c<ME / 2>(w);
                    } else {
                        double y = rsqrt_fast_lo(r2, r2xy);
                        if constexpr (decltype(masked)::value) y = jidx > irow[k] ? y : 0.0;
                        term = (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
                    }
                    f0[k] += term;
                    g0 += term;
                } else {
                    double y = rsqrt_fast_lo(r2, r2xy);
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
            out.g0 = rot1(g0);
            if constexpr (FORCE) { out.g1 = rot1(g1); out.g2 = rot1(g2); }
        };
        JRec A, B;
        A.x = xj; A.y = yj; A.z = zj; A.s = sj; A.g0 = A.g1 = A.g2 = 0.0;
        B = A;
        if (diag) {
            for (int s = 0; s < 32; s += 2) {
                step(std::integral_constant<bool, true>{}, s, A, B);
                step(std::integral_constant<bool, true>{}, s + 1, B, A);
            }
        } else {
#pragma unroll 4
            for (int s = 0; s < 32; s += 2) {
                step(std::integral_constant<bool, false>{}, s, A, B);
                step(std::integral_constant<bool, false>{}, s + 1, B, A);
            }
        }
        g0 = A.g0; g1 = A.g1; g2 = A.g2;                   // the record is home again (32 rotations by one lane)
        }
        if (both) {                                        // set B -> set A: reaction sums of the second RB rows
            if (set) {
                if (nx >= 1) n3_empty_wait(wp);            // A has read the slot's previous contents
                slot[lane] = g0;
                if constexpr (FORCE) { slot[32 + lane] = g1; slot[64 + lane] = g2; }
                n3_full_arrive(wp);
            } else {
                n3_full_wait(wp);
                g0 += slot[lane];
                if constexpr (FORCE) { g1 += slot[32 + lane]; g2 += slot[64 + lane]; }
                n3_empty_arrive(wp);
            }
            ++nx;
        }
        if (!set && jidx < N) {
            if constexpr (FORCE) part[jidx - row0p] = make_double4(g0, g1, g2, 0.0);
            else part_rho[jidx - row0p] = g0;
        }
    }

    // ---- rows i: sum over the warps of the CTA in a fixed order ----
    __syncthreads();                                       // every warp is done with its chunk records (same memory)
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        red[warp][k][0][lane] = f0[k];
        if constexpr (FORCE) { red[warp][k][1][lane] = f1[k]; red[warp][k][2][lane] = f2[k]; }
    }
    __syncthreads();
    for (int r = threadIdx.x; r < 2 * RB; r += NW * 32) {
        const int rs = r >= RB ? 1 : 0, k = (r - rs * RB) >> 5, l = r & 31, i = row0p + r;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        for (int w = rs * H; w < rs * H + H; ++w) {       // the warps that hold this row's set
            v0 += red[w][k][0][l];
            if constexpr (FORCE) { v1 += red[w][k][1][l]; v2 += red[w][k][2][l]; }
        }
        if (i < N) a.self[size_t(tile.slot) * a.n_pad + i] = make_double4(v0, v1, v2, 0.0);
    }
    __syncthreads();                                       // the next tile's chunk records go into the same memory
    }   // tiles of this CTA's piece
    if (set && nx >= 1) n3_empty_wait(wp);                 // absorb A's last arrival: the barriers are clean for the next sweep
    if constexpr (FORCE && ENERGY) {
        esum = warp_sum(esum);                             // over all tiles of the piece
        if (lane == 0) red_e[warp] = esum;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < NW; ++w) tot += red_e[w];
            a.partial[piece] = 2.0 * tot;        // every unordered pair stands for two ordered ones
        }
    }
}

template <int IT, int NE, int ME, bool FORCE, bool ENERGY>
__global__ void __launch_bounds__(kN3Warps * 32, 1) allpairs_n3_kernel(const N3Args a) {
    __shared__ double red[kN3Warps][IT][3][32];
    __shared__ double red_e[kN3Warps];
    __shared__ __align__(16) unsigned char slots[(kN3Warps / 2) * kN3SlotBytes];
    n3_sweep_piece<IT, NE, ME, FORCE, ENERGY>(a, blockIdx.x, red, red_e, slots);
}

// ---- mixed precision: the same rotation in binary32 on split records (x = xh + xl, RecF), binary64 accumulation ----
// Rows accumulate in binary32 over one chunk (32 terms) and are then added into binary64 sums; the reaction sums
// travel in binary32 (128 terms) and are stored as binary64 partials.  No binary64 instruction in the rotation.
// Sweep 1 keeps TWO binary32 sums per accumulator, one for pairs closer than 20 A and one for the rest: a far term
// (r^-6 ~ 1e-11) added to a sum that already holds a nearest-neighbour term (4e-3) would be absorbed entirely, a
// one-sided loss that biased rho by ~1.5e-7 and the energy by 6-8e-8 of BASELINE.json's 1e-7 (measured before the
// split).  The pair-energy sum of sweep 2 (r^-9) needs the same split, at 10 A: unsplit it lost 1e-7 of the energy of
// the N = 8000 liquid droplet (a lane's sum holds a nearest-neighbour term with probability ~1500 / N); the force
// terms have the same loss, far inside their 1e-5 tolerance.

struct N3FArgs {
    const RecF *xfr;        // [N] split binary32 records
    int n_atoms, n_pad;
    double4 *part;
    double *part_rho;
    double4 *self;
    double *partial;
    const N3Tile *tiles;    // chunks counted in units of 64 atoms here
    const int *piece_start;
    PairConsts c;
};

// Packed: a warp rotates a chunk of 64 atoms: lane t holds records j_a = 64 c + t and j_b = 64 c + 32 + t in the two
// halves of Blackwell's binary32 pair registers (PTX add / mul / fma.f32x2, SASS FADD2 / FMUL2 / FFMA2), j-side values
// NEGATED so that only additions are needed; the rows i are duplicated into both halves once per launch.  One
// rotation step is then 4 rows x 2 records = 8 pairs per lane for the instruction count of 4.
__device__ __forceinline__ f2 rot1_f2(f2 v) {      // the 64-bit shuffle: two SHFL on the register pair, no repacking moves
    return __shfl_sync(0xffffffffu, v, (threadIdx.x + 1) & 31);
}

// Shared memory of the mixed sweeps: per warp 3584 B of chunk records (below), in the same buffer the epilogue's row sums
// (kN3Warps x IT x 3 x 32 doubles) use afterwards
constexpr int kN3pWarpBytes = 3 * 64 * 16 + 64 * 8;
template <int IT>
constexpr int kN3pSmemDoubles =
    (kN3Warps * kN3pWarpBytes > kN3Warps * IT * 3 * 32 * 8 ? kN3Warps * kN3pWarpBytes : kN3Warps * IT * 3 * 32 * 8) / 8;
constexpr int kN3pUnroll = SCMD_N3P_UNROLL;

template <int IT, int NE, int ME, bool FORCE, bool ENERGY>
__device__ __forceinline__ void n3p_sweep_piece(const N3FArgs &a, const int piece, double *buf /* kN3pSmemDoubles<IT> */,
                                                double (&red_e)[kN3Warps], unsigned char *slots) {
    constexpr int RB = 32 * IT;
    constexpr bool kNeg = !FORCE && ME > 0 && ME % 2 == 0 && (ME / 2) % 2 == 1;   // sweep 1 sums -r^-m (see the term)
    double (&red)[kN3Warps][IT][3][32] = *reinterpret_cast<double (*)[kN3Warps][IT][3][32]>(buf);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int NW = blockDim.x >> 5;
    const int H = NW >> 1, set = warp >= H ? 1 : 0, wp = warp - set * H;   // as in n3_sweep_piece
    f2 *slot = reinterpret_cast<f2 *>(slots + wp * kN3SlotBytes);   // one slot per warp pair here (shared memory is full)
    int nx = 0;
    const int N = a.n_atoms;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const f2 An2 = f2_dup(float(a.c.An));
    const f2 zero2 = f2_dup(0.f), one2 = f2_dup(1.0f), mone2 = f2_dup(-1.0f), mhalf2 = f2_dup(-0.5f);
    constexpr float kFarF = 1.0e15f;
    double esum = 0.0;
    const int t_end = a.piece_start[piece + 1];
    for (int t = a.piece_start[piece]; t < t_end; ++t) {
    const N3Tile tile = a.tiles[t];
    const int row0p = tile.b * 2 * RB, row0 = row0p + set * RB;
    const int cb = row0 >> 6, cbB = (row0p >> 6) + IT / 2;
    const int c_begin = tile.c_begin, c_end = tile.c_end;   // chunks of 64 atoms

    int irow[IT];
    f2 xh[IT], yh[IT], zh[IT], xl[IT], yl[IT], zl[IT], si[IT];     // row values in both halves
    double F0[IT], F1[IT], F2[IT];
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        irow[k] = row0 + k * 32 + lane;
        RecF p;
        if (irow[k] < N) p = a.xfr[irow[k]];
        else p = RecF{kFarF * float(k + 2), -kFarF * float(lane + 1), 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        xh[k] = f2_dup(p.xh); yh[k] = f2_dup(p.yh); zh[k] = f2_dup(p.zh);
        xl[k] = f2_dup(p.xl); yl[k] = f2_dup(p.yl); zl[k] = f2_dup(p.zl); si[k] = f2_dup(-p.s);    // s' NEGATED on both sides: -(s'_i + s'_j) is one addition
        F0[k] = F1[k] = F2[k] = 0.0;
    }
    double4 *part = a.part + n3_part_offset(tile.b, a.n_pad, 2 * RB);
    double *part_rho = a.part_rho + n3_part_offset(tile.b, a.n_pad, 2 * RB);
    // chunk records of this warp, every record at lane AND lane + 32 so that the index lane + s + 1 never wraps (as in the
    // FP64 kernel): three arrays of 64 x 16 B -- (xh, yh), (zh, s'), (xl, yl) -- and one of 64 x 8 B (zl)
    ulonglong2 *jq = reinterpret_cast<ulonglong2 *>(reinterpret_cast<unsigned char *>(buf) + warp * kN3pWarpBytes);
    unsigned long long *jq3 = reinterpret_cast<unsigned long long *>(jq + 192);
    auto fetch = [&](int j) -> RecF {
        if (j < N) return a.xfr[j];
        return RecF{-kFarF * float((j & 63) + 1), kFarF, kFarF, 0.f, 0.f, 0.f, 0.f, 0.f};
    };
    for (int c = c_begin + wp; c < c_end; c += H) {
        const int ja = (c << 6) + lane, jb = ja + 32;
        const bool both = c >= cbB;
        f2 g0 = zero2, g1 = zero2, g2 = zero2, gfar = zero2;
        if (set == 0 || both) {
        const RecF pa = fetch(ja), pb = fetch(jb);
        // negated j records, (a, b) in the (low, high) halves
        f2 nxh = f2_make(-pa.xh, -pb.xh), nyh = f2_make(-pa.yh, -pb.yh), nzh = f2_make(-pa.zh, -pb.zh);
        f2 nxl = f2_make(-pa.xl, -pb.xl), nyl = f2_make(-pa.yl, -pb.yl), nzl = f2_make(-pa.zl, -pb.zl);
        const f2 sj = f2_make(-pa.s, -pb.s);
        f2 f0[IT], f1[IT], f2v[IT], ffar[IT];
#pragma unroll
        for (int k = 0; k < IT; ++k) f0[k] = f1[k] = f2v[k] = ffar[k] = zero2;
        const bool diag = c < cb + IT / 2;                 // the block's own rows span IT / 2 chunks of 64
        // One rotation step: the lane evaluates its IT rows against the two records it holds (`in`) and hands them, with
        // the sums accumulated on them, to the next lane (`out`).  Two register sets alternate (A -> B, B -> A), so no
        // value has to be moved back into a loop-carried register (44 moves per two steps when written in place).
        struct JRec { f2 xh, yh, zh, xl, yl, zl, s, g0, g1, g2, gf; };
        // the 2 x 32 records of the chunk sit in shared memory (see the FP64 kernel): at step s a lane reads the pair of
        // records of lane + s with four LDS.128 instead of fourteen shuffles; only the sums travel
        __syncwarp();
        jq[lane] = make_ulonglong2(nxh, nyh); jq[64 + lane] = make_ulonglong2(nzh, sj);
        jq[128 + lane] = make_ulonglong2(nxl, nyl); jq3[lane] = nzl;
        jq[32 + lane] = make_ulonglong2(nxh, nyh); jq[96 + lane] = make_ulonglong2(nzh, sj);
        jq[160 + lane] = make_ulonglong2(nxl, nyl); jq3[32 + lane] = nzl;
        __syncwarp();
        auto step = [&](auto masked, int s, const JRec &in, JRec &out) {
            const f2 nxh = in.xh, nyh = in.yh, nzh = in.zh, nxl = in.xl, nyl = in.yl, nzl = in.zl, sj = in.s;
            const int jidx_a = ja - lane + ((lane + s) & 31), jidx_b = jidx_a + 32;
            f2 g0 = in.g0, g1 = in.g1, g2 = in.g2, gfar = in.gf;
            {   // the records of the NEXT step first: their latency hides behind this step's arithmetic
                const int nx = lane + s + 1;               // <= 63: the second copy
                const ulonglong2 q0 = jq[nx], q1 = jq[64 + nx], q2 = jq[128 + nx];
                out.xh = q0.x; out.yh = q0.y; out.zh = q1.x; out.s = q1.y; out.xl = q2.x; out.yl = q2.y; out.zl = jq3[nx];
            }
            f2 estep = zero2;                              // sum r^-n over the 2 IT pairs of this step
#pragma unroll
            for (int k = 0; k < IT; ++k) {
                const f2 dx = f2_add(f2_add(xh[k], nxh), f2_add(xl[k], nxl));
                const f2 dy = f2_add(f2_add(yh[k], nyh), f2_add(yl[k], nyl));
                const f2 dz = f2_add(f2_add(zh[k], nzh), f2_add(zl[k], nzl));
                const f2 r2 = f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx)));
                bool ka = true, kb = true;                 // pair counts (diagonal chunks: iff j > i)
                if constexpr (decltype(masked)::value) { ka = jidx_a > irow[k]; kb = jidx_b > irow[k]; }
                if constexpr (!FORCE) {
                    f2 term;
                    if constexpr (ME > 0 && ME % 2 == 0) {
                        // seed of -x (the negation rides on the MUFU operand): e = 1 + x (-y0) in one rounding, w = -(1 / r^2),
                        // so no packed multiply by -1 is needed; for an odd ME / 2 the term and all sums of this sweep
                        // are then NEGATIVE (kNeg) and their sign is turned when they leave binary32
                        const f2 y0 = f2_make(mufu_rcp(-f2_lo(r2)), mufu_rcp(-f2_hi(r2)));
                        const f2 e = f2_fma(r2, y0, one2);
                        f2 w = f2_fma(y0, e, y0);
                        if constexpr (decltype(masked)::value) w = f2_make(ka ? f2_lo(w) : 0.f, kb ? f2_hi(w) : 0.f);
                        term = f2_ipow_c<ME / 2>(w);
                    } else {
                        const f2 y0 = f2_make(mufu_rsq(f2_lo(r2)), mufu_rsq(f2_hi(r2)));
                        const f2 ep = f2_fma(f2_mul(r2, y0), y0, mone2);
                        f2 y = f2_fma(f2_mul(y0, ep), mhalf2, y0);
                        if constexpr (decltype(masked)::value) y = f2_make(ka ? f2_lo(y) : 0.f, kb ? f2_hi(y) : 0.f);
                        term = (ME > 0) ? f2_ipow_c<(ME > 0 ? ME : 1)>(y) : f2_ipow_rt(y, m_exp);
                    }
                    // two sums per accumulator (see the header of this section), split WITHOUT selects: the part of a
                    // term below 2^-26 A^-m (r^-6 at 20 A) goes to the far sum, what exceeds it to the near sum:
                    // tf = min(term, T) is exact, tn = term - tf is 0 for a far term and one rounding for a near one
                    const f2 tf = kNeg ? f2_make(fmaxf(f2_lo(term), -kN3FarTerm), fmaxf(f2_hi(term), -kN3FarTerm))
                                       : f2_make(fminf(f2_lo(term), kN3FarTerm), fminf(f2_hi(term), kN3FarTerm));
                    const f2 tn = f2_fma(tf, mone2, term);
                    f0[k] = f2_add(f0[k], tn); ffar[k] = f2_add(ffar[k], tf);
                    g0 = f2_add(g0, tn); gfar = f2_add(gfar, tf);
                } else {
                    const f2 y0 = f2_make(mufu_rsq(f2_lo(r2)), mufu_rsq(f2_hi(r2)));
                    const f2 ep = f2_fma(f2_mul(r2, y0), y0, mone2);                     // t y0 - 1
                    f2 y = f2_fma(f2_mul(y0, ep), mhalf2, y0);                           // y0 - y0 e' / 2
                    if constexpr (decltype(masked)::value) y = f2_make(ka ? f2_lo(y) : 0.f, kb ? f2_hi(y) : 0.f);
                    const f2 w = f2_mul(y, y);
                    const f2 nss = f2_add(si[k], sj);                                    // -(s'_i + s'_j): both come negated
                    f2 coef, pnw;
                    if constexpr (NE == 9 && ME == 6) {
                        const f2 w2 = f2_mul(w, w), w4 = f2_mul(w2, w2), y3 = f2_mul(w, y);
                        coef = f2_mul(w4, f2_fma(An2, y3, nss));
                        pnw = f2_mul(w4, y);
                    } else {
                        const f2 pm = (ME > 0) ? f2_ipow_c<(ME > 0 ? ME : 1)>(y) : f2_ipow_rt(y, m_exp);
                        pnw = (NE > 0) ? f2_ipow_c<(NE > 0 ? NE : 1)>(y) : f2_ipow_rt(y, n_exp);
                        coef = f2_mul(w, f2_fma(An2, pnw, f2_mul(nss, pm)));
                    }
                    if constexpr (ENERGY) estep = f2_add(estep, pnw);
                    f0[k] = f2_fma(coef, dx, f0[k]); f1[k] = f2_fma(coef, dy, f1[k]); f2v[k] = f2_fma(coef, dz, f2v[k]);
                    // the reaction sums collect +coef d; their sign is turned when they are stored (one packed multiply per row
                    // and step less: binary32 pair instructions have no negated operands)
                    g0 = f2_fma(coef, dx, g0); g1 = f2_fma(coef, dy, g1); g2 = f2_fma(coef, dz, g2);
                }
            }
            // The pair energy leaves binary32 after EVERY step (2 IT terms): a sum that lived for a whole chunk lost
            // the far terms to the first nearest-neighbour term it met (1e-7 of the energy, measured in round 1, then
            // cured by two selected sums per pair: 24 instructions per step; this is 3)
            if constexpr (FORCE && ENERGY) esum += double(f2_lo(estep) + f2_hi(estep));
            // the sums travel with the record
            out.g0 = rot1_f2(g0);
            if constexpr (FORCE) { out.g1 = rot1_f2(g1); out.g2 = rot1_f2(g2); }
            else out.gf = rot1_f2(gfar);
        };
        JRec A, B;
        A.xh = nxh; A.yh = nyh; A.zh = nzh; A.xl = nxl; A.yl = nyl; A.zl = nzl; A.s = sj;
        A.g0 = A.g1 = A.g2 = A.gf = zero2;
        B = A;
        if (diag) {
            for (int s = 0; s < 32; s += 2) {
                step(std::integral_constant<bool, true>{}, s, A, B);
                step(std::integral_constant<bool, true>{}, s + 1, B, A);
            }
        } else {
#pragma unroll kN3pUnroll
            for (int s = 0; s < 32; s += 2) {
                step(std::integral_constant<bool, false>{}, s, A, B);
                step(std::integral_constant<bool, false>{}, s + 1, B, A);
            }
        }
        g0 = A.g0; g1 = A.g1; g2 = A.g2; gfar = A.gf;      // both records are home again
#pragma unroll
        for (int k = 0; k < IT; ++k) {                     // one chunk of binary32 row sums into binary64
            if constexpr (!FORCE && kNeg) F0[k] -= double(f2_lo(f0[k]) + f2_hi(f0[k]));
            else F0[k] += double(f2_lo(f0[k]) + f2_hi(f0[k]));
            if constexpr (FORCE) {
                F1[k] += double(f2_lo(f1[k]) + f2_hi(f1[k]));
                F2[k] += double(f2_lo(f2v[k]) + f2_hi(f2v[k]));
            } else {
                if constexpr (kNeg) F0[k] -= double(f2_lo(ffar[k]) + f2_hi(ffar[k]));
                else F0[k] += double(f2_lo(ffar[k]) + f2_hi(ffar[k]));
            }
        }
        }   // this set has pairs in the chunk
        f2 b0 = zero2, b1 = zero2, b2 = zero2;             // set B's sums (binary32, as they travelled)
        if (both) {
            if (set) {
                if (nx >= 1) n3_empty_wait(wp);
                slot[lane] = g0; slot[32 + lane] = FORCE ? g1 : gfar; if constexpr (FORCE) slot[64 + lane] = g2;
                n3_full_arrive(wp);
            } else {
                n3_full_wait(wp);
                b0 = slot[lane]; b1 = slot[32 + lane]; if constexpr (FORCE) b2 = slot[64 + lane];
                n3_empty_arrive(wp);
            }
            ++nx;
        }
        if (!set) {
            if constexpr (FORCE) {
                if (ja < N) part[ja - row0p] = make_double4(-(double(f2_lo(g0)) + double(f2_lo(b0))), -(double(f2_lo(g1)) + double(f2_lo(b1))),
                                                            -(double(f2_lo(g2)) + double(f2_lo(b2))), 0.0);
                if (jb < N) part[jb - row0p] = make_double4(-(double(f2_hi(g0)) + double(f2_hi(b0))), -(double(f2_hi(g1)) + double(f2_hi(b1))),
                                                            -(double(f2_hi(g2)) + double(f2_hi(b2))), 0.0);
            } else {
                const double sgn = kNeg ? -1.0 : 1.0;
                if (ja < N) part_rho[ja - row0p] = sgn * ((double(f2_lo(g0)) + double(f2_lo(gfar))) + (double(f2_lo(b0)) + double(f2_lo(b1))));
                if (jb < N) part_rho[jb - row0p] = sgn * ((double(f2_hi(g0)) + double(f2_hi(gfar))) + (double(f2_hi(b0)) + double(f2_hi(b1))));
            }
        }
    }
    __syncthreads();                                       // every warp is done with its chunk records (same memory)
#pragma unroll
    for (int k = 0; k < IT; ++k) {
        red[warp][k][0][lane] = F0[k];
        if constexpr (FORCE) { red[warp][k][1][lane] = F1[k]; red[warp][k][2][lane] = F2[k]; }
    }
    __syncthreads();
    for (int r = threadIdx.x; r < 2 * RB; r += NW * 32) {
        const int rs = r >= RB ? 1 : 0, k = (r - rs * RB) >> 5, l = r & 31, i = row0p + r;
        double v0 = 0.0, v1 = 0.0, v2 = 0.0;
        for (int w = rs * H; w < rs * H + H; ++w) {       // the warps that hold this row's set
            v0 += red[w][k][0][l];
            if constexpr (FORCE) { v1 += red[w][k][1][l]; v2 += red[w][k][2][l]; }
        }
        if (i < N) a.self[size_t(tile.slot) * a.n_pad + i] = make_double4(v0, v1, v2, 0.0);
    }
    __syncthreads();                                       // the next tile's chunk records go into the same memory
    }   // tiles of this CTA's piece
    if (set && nx >= 1) n3_empty_wait(wp);                 // absorb A's last arrival
    if constexpr (FORCE && ENERGY) {
        esum = warp_sum(esum);                             // over all tiles of the piece
        if (lane == 0) red_e[warp] = esum;
        __syncthreads();
        if (threadIdx.x == 0) {
            double tot = 0.0;
            for (int w = 0; w < NW; ++w) tot += red_e[w];
            a.partial[piece] = 2.0 * tot;
        }
    }
}

template <int IT, int NE, int ME, bool FORCE, bool ENERGY>
__global__ void __launch_bounds__(kN3Warps * 32, 1) allpairs_n3p_kernel(const N3FArgs a) {
    __shared__ __align__(16) double buf[kN3pSmemDoubles<IT>];
    __shared__ double red_e[kN3Warps];
    __shared__ __align__(16) unsigned char slots[(kN3Warps / 2) * kN3SlotBytes];
    n3p_sweep_piece<IT, NE, ME, FORCE, ENERGY>(a, blockIdx.x, buf, red_e, slots);
}

// ---- finalize: self[i] + part[0 .. block(i)][i] in that order ----
struct N3FinalArgs {
    double4 *xs;
    RecF *xfr;                          // mixed: sweep 1 stores fl32(s') here as well (else NULL)
    FPair *xf;                          // mixed: ... and into the packed records of the one-sided sweeps
    const double4 *part;
    const double *part_rho;
    const double4 *self;
    double *rho, *force, *partial;      // partial: [gridDim.x = ceil(N / 32)] sum sqrt(rho) (density)
    int n_atoms, n_pad, rb;
    const int *blk_slots;               // [row blocks] tiles (= self slots) of each row block in the plan
    PairConsts c;
    // NVE steps inside sc_step (FORCE only): the thread that has just formed F_i also does the velocity-Verlet updates
    // that follow, instead of two more launches.  fuse = 0: nothing; 1: second half kick of this step and the per-CTA
    // sum of |v|^2 (the call's last step); 2: second half kick, then the first half kick and the drift of the NEXT step
    int fuse;
    double *vel, *part_ke;              // [N*3]; [gridDim.x]
    double hk, dt;                      // dt/2 ACC/m; dt
};

constexpr int kN3FinAtoms = 32;         // atoms per CTA of the finalize kernel: one per lane
constexpr int kN3FinWarps = 8;          // its warps share the segments and the row blocks of those atoms

// A group of 32 consecutive atoms (one per lane: every load is a contiguous 256 B or 1 KB line run): warp w < 8 sums
// the tiles' row sums sg = w, w + 8, ... and the row blocks b = w, w + 8, ... <= block(i), then the 8 sums are added in
// warp order.  Always 8 summing warps, whatever the CTA (n3_finalize_kernel: 8 warps, one group per CTA; n3_loop_kernel:
// 12 warps, 4 of them idle in the first part), so that every path gives the same bits.
// (One thread per atom walking all blocks left 32 CTAs on 148 SMs at N = 8000: 21 us for the force variant.)
// Up to GB groups g0, g0 + gstride, ... at once: their loads are independent and issued together (the phase is a chain
// of L2 latencies: one group after the other cost the loop kernel 2 us per group), warp u then finishes group u.
template <bool FORCE, int GB>
__device__ __forceinline__ void n3_finalize_groups(const N3FinalArgs &a, const int g0, const int gstride, const int cnt,
                                                   double (*red)[kN3FinWarps][3][32]) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    double v[GB][3];
    int ii[GB], bi[GB], nseg[GB];
    int bmax = -1, smax = 0;
#pragma unroll
    for (int u = 0; u < GB; ++u) {
        v[u][0] = v[u][1] = v[u][2] = 0.0;
        ii[u] = (g0 + u * gstride) * kN3FinAtoms + lane;
        const bool live = u < cnt && ii[u] < a.n_atoms && w < kN3FinWarps;
        bi[u] = live ? ii[u] / a.rb : -1;
        nseg[u] = live ? a.blk_slots[bi[u]] : 0;
        bmax = max(bmax, bi[u]); smax = max(smax, nseg[u]);
    }
    for (int sg = w; sg < smax; sg += kN3FinWarps) {        // row sums of the tiles of i's own block
#pragma unroll
        for (int u = 0; u < GB; ++u)
            if (GB == 1 || sg < nseg[u]) {          // one group: the loop bound is its own
                const double4 s = a.self[size_t(sg) * a.n_pad + ii[u]];
                v[u][0] += s.x; v[u][1] += s.y; v[u][2] += s.z;
            }
    }
#pragma unroll 4
    for (int b = w; b <= bmax; b += kN3FinWarps) {
#pragma unroll
        for (int u = 0; u < GB; ++u)
            if (GB == 1 || b <= bi[u]) {
                const size_t at = n3_part_offset(b, a.n_pad, a.rb) + size_t(ii[u] - b * a.rb);
                if constexpr (FORCE) {
                    const double4 p = a.part[at];
                    v[u][0] += p.x; v[u][1] += p.y; v[u][2] += p.z;
                } else {
                    v[u][0] += a.part_rho[at];
                }
            }
    }
    if (w < kN3FinWarps) {
#pragma unroll
        for (int u = 0; u < GB; ++u) {
            red[u][w][0][lane] = v[u][0];
            if constexpr (FORCE) { red[u][w][1][lane] = v[u][1]; red[u][w][2][lane] = v[u][2]; }
        }
    }
    __syncthreads();
    if (w < cnt && w < GB) {                               // warp u finishes group u
    const int group = g0 + w * gstride;
    const int i = group * kN3FinAtoms + lane;
    double v0 = 0.0, v1 = 0.0, v2 = 0.0;
#pragma unroll
    for (int k = 0; k < kN3FinWarps; ++k) {
        v0 += red[w][k][0][lane];
        if constexpr (FORCE) { v1 += red[w][k][1][lane]; v2 += red[w][k][2][lane]; }
    }
    double contrib = 0.0;
    if (i < a.n_atoms) {
        if constexpr (FORCE) {
            a.force[3 * size_t(i)] = v0; a.force[3 * size_t(i) + 1] = v1; a.force[3 * size_t(i) + 2] = v2;
            if (a.fuse) {
                // the same fused multiply-adds, in the same order, as kick_ke_kernel and kick_drift_kernel
                double vx = fma(a.hk, v0, a.vel[3 * size_t(i)]), vy = fma(a.hk, v1, a.vel[3 * size_t(i) + 1]),
                       vz = fma(a.hk, v2, a.vel[3 * size_t(i) + 2]);
                if (a.fuse == 1) {
                    contrib = fma(vz, vz, fma(vy, vy, vx * vx));
                } else {
                    vx = fma(a.hk, v0, vx); vy = fma(a.hk, v1, vy); vz = fma(a.hk, v2, vz);
                    double4 p = a.xs[i];
                    p.x = fma(a.dt, vx, p.x); p.y = fma(a.dt, vy, p.y); p.z = fma(a.dt, vz, p.z);
                    a.xs[i] = p;
                    if (a.xf) store_split_record(a.xf, i, p.x, p.y, p.z, float(p.w));
                    if (a.xfr) a.xfr[i] = split_record(p);
                }
                a.vel[3 * size_t(i)] = vx; a.vel[3 * size_t(i) + 1] = vy; a.vel[3 * size_t(i) + 2] = vz;
            }
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
        const double t = warp_sum(contrib);
        if (lane == 0) a.partial[group] = t;
    } else {
        if (a.fuse == 1) {
            const double t = warp_sum(contrib);
            if (lane == 0) a.part_ke[group] = t;
        }
    }
    }   // finishing warp
    __syncthreads();                                       // red is free again
}

#ifdef SCMD_MAIN_TU
template <bool FORCE>
__global__ void __launch_bounds__(kN3FinWarps * 32) n3_finalize_kernel(const N3FinalArgs a) {
    __shared__ double red[1][kN3FinWarps][3][32];
    n3_finalize_groups<FORCE, 1>(a, blockIdx.x, 0, 1, red);
}
#endif  // SCMD_MAIN_TU

// ---- the whole sc_step loop in one cooperative launch (sc_n3_loop.cuh, instantiated in inst_n3_loop.cu) ----
struct N3LoopArgs {
    N3Args s;                           // FP64 sweeps ...
    N3FArgs sf;                         // ... or the mixed ones
    N3FinalArgs f;                      // finalize (fuse is set by the kernel)
    unsigned long long *barrier;        // grid barrier counter; the host tracks its value
    unsigned long long barrier_base;
    long long nsteps;
    int energy_every;                   // 1: the pair energy on every step (SC_OPT_ENERGY_EVERY_STEP), else on the last only
    int thermo;                         // 0: NVE; 1: velocity rescaling to the ramp T_start -> T_end
    double T_start, T_end, mass, ndof;
};
const void *n3_loop_fn(bool fast, bool mixed);

// instantiated in inst_allpairs_n3.cu; nullptr if this shape is not compiled
const void *allpairs_n3_fn(int it, bool fast, bool force, bool energy);
const void *allpairs_n3p_fn(int it, bool fast, bool force, bool energy);      // mixed precision, packed pairs

}  // namespace scmd
