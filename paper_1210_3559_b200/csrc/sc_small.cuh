// sc_small.cuh -- the whole velocity-Verlet loop of sc_step in ONE cooperative launch, for clusters
// small enough that a step is bound by launch latency rather than by the FP64 pipe (the paper's own
// production size, Ni2057 for 6.5e7 steps; BASELINE.json configs 1 and 2).
//
// The multi-launch path needs 6-7 dependent launches per step (~40-50 us at N <= 2000, of which the
// pair arithmetic is < 5 us).  Here the grid stays resident and the phases of a step are separated
// by grid-wide barriers instead of launch boundaries:
//
//   A  owners: v <- lambda v; v += hk F; x += dt v                     (rows of this CTA only)
//      ---- grid barrier 1: all positions of the step are in global memory ----
//   B  every CTA stages all N records into shared memory; sweep 1 for its own rows:
//      rho_i, s'_i = eps (c m / 2) a^m rho_i^-1/2 -> sprime[i]
//      ---- grid barrier 2: all s' are in global memory ----
//   C  stage the s' (8 bytes per atom); sweep 2 for its own rows: F_i and sum_j r^-n
//   D  owners: v += hk F [Langevin update]; |v|^2
//      rescale thermostat only: ---- grid barrier 3 ----, every CTA forms the same kinetic energy
//      from the per-CTA partials in a fixed order and scales its own velocities.
//
// Decomposition: a CTA owns `rows` consecutive atoms; JL (a power of two) threads share one row and
// stride the j range; a warp holds 32 / lq rows (lq threads of each), so its shared-memory loads are
// broadcast across rows; partial sums meet in a shuffle tree (and across the warps of a row through
// shared memory), always in the same order: results are bit-reproducible.  The row's first
// thread ("owner") keeps v and F of its atom in registers for the whole call.
#pragma once
#include "sc_allpairs.cuh"
#include "sc_device.cuh"
#include "sc_integrate.cuh"

namespace scmd {

constexpr int kSmallThreads = 512;
constexpr int kSmallMaxAtoms = 6144;         // N * 32 B of records must fit in shared memory

struct SmallStepArgs {
    double4 *xs;            // [N] (x, y, z, s'): the state at entry and at exit
    double4 *xs_b;          // [N] second buffer: step k works in (k odd ? xs_b : xs), so that a CTA already in
                            //     phase A of step k + 1 never overwrites records another CTA still stages
    double *vel, *force, *rho;
    FPair *xf;              // MIXED: the packed records of the multi-launch sweeps, refreshed at exit (may be NULL)
    RecF *xfr;              // MIXED: ... and the split records of the Newton's-third-law sweeps (may be NULL)
    double *part_emb, *part_pair, *part_ke;   // [gridDim.x]
    double *sprime;         // [N] s' of the current step, contiguous (phase C re-stages only these 8 bytes per atom)
    unsigned long long *barrier;      // grid barrier counter; grows by gridDim.x per barrier
    unsigned long long barrier_base;  // its value when this launch starts (the host keeps count)
    double *scal;
    int n_atoms, rows, jl;  // rows per CTA; threads per row (power of two)
    int lq;                 // threads of a row inside one warp (power of two, <= min(jl, 32)): a warp holds 32 / lq rows, so a
                            //   shared-memory load of 32 lanes touches lq records (broadcast across the rows);
                            //   round_up(rows, 32 / lq) * jl <= kSmallThreads
    long long nsteps;
    double hk, dt, mass, ndof;
    int thermo;             // sc_thermo_kind
    double T_start, T_end;
    double lg_c1, lg_pre;   // Langevin: c1 = exp(-gamma dt); c2_k = sqrt(lg_pre * T_k * ACC / mass), lg_pre = (1 - c1^2) kB
    uint32_t key0, key1;
    unsigned long long lg_step0;
    PairConsts c;
};

// Staged records in shared memory: blocks of 8 records, the 8 first halves (16 B: x, y / xh, yh, zh, s') followed by the
// 8 second halves (z, s' / xl, yl, zl).  The lq lanes of a row read lq CONSECUTIVE records: as whole 32-byte records
// that is a 16-byte access at a 32-byte stride -- 2 x the wavefronts, and at N = 1415 (16 lanes per row) ncu showed the
// shared-memory pipe saturated by 1.2 M bank conflicts per step; in this layout the same access is contiguous.
// A thread steps through records jl apart; jl is a multiple of 8, so its address advances by jl x 32 bytes.
__host__ __device__ inline int small_rec_off(int j) { return ((j >> 3) << 8) + ((j & 7) << 4); }
__host__ __device__ inline int small_rec_bytes(int n_atoms) { return ((n_atoms + 7) >> 3) << 8; }
inline size_t small_step_smem_bytes(int n_atoms) {
    return size_t(small_rec_bytes(n_atoms)) + (kSmallThreads / 32) * 8 * 4 * sizeof(double) + kSmallThreads * sizeof(double);
}

#ifdef SCMD_MAIN_TU
__device__ __forceinline__ double4 load_record_cg(const double4 *p) {    // L2 (coherent) load, bypasses L1
    double4 r;
    asm volatile("ld.global.cg.v4.f64 {%0, %1, %2, %3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}

// sum over the JL threads of a row; valid in the row's first thread.  The lq threads of a row inside a warp meet in
// a shuffle tree; when the row spans jl / lq warps, its first thread adds the per-warp values in order.
constexpr int kSmallMaxRowsPerWarp = 8;
template <int NV>
__device__ __forceinline__ void row_reduce(double (&v)[NV], int jl, int lq, int q, double *warp_red) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int off = lq >> 1; off > 0; off >>= 1)
#pragma unroll
        for (int c = 0; c < NV; ++c) v[c] += __shfl_xor_sync(0xffffffffu, v[c], off);
    if (jl > lq) {                                          // block-uniform
        const int rl = lane / lq;                           // row of this lane inside the warp
        __syncthreads();
        if (lane % lq == 0)
#pragma unroll
            for (int c = 0; c < NV; ++c) warp_red[(warp * kSmallMaxRowsPerWarp + rl) * 4 + c] = v[c];
        __syncthreads();
        if (q == 0) {                                       // first warp of the row's group, first lane of the row
            const int nw = jl / lq;
#pragma unroll
            for (int c = 0; c < NV; ++c) {
                double s = 0.0;
                for (int w = 0; w < nw; ++w) s += warp_red[((warp + w) * kSmallMaxRowsPerWarp + rl) * 4 + c];
                v[c] = s;
            }
        }
    }
}

// fixed-order sum of one value per row over the rows of the CTA; result valid in thread 0
__device__ __forceinline__ double rows_sum(double mine, bool owner, int r, int nrows, double *rowval) {
    __syncthreads();
    if (owner) rowval[r] = mine;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int k = 0; k < nrows; ++k) s += rowval[k];
    return s;
}

// fixed-order sum of part[0..n) by warp 0 (every CTA gets the same bits); valid in all lanes of warp 0
__device__ __forceinline__ double warp0_sum_partials(const double *part, int n) {
    const int lane = threadIdx.x & 31;
    double s = 0.0;
    for (int k = lane; k < n; k += 32) s += __ldcg(part + k);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    return s;
}

template <class Rec> __device__ __forceinline__ Rec small_load(const unsigned char *p);
template <> __device__ __forceinline__ double4 small_load<double4>(const unsigned char *p) {
    const double2 a = *reinterpret_cast<const double2 *>(p), b = *reinterpret_cast<const double2 *>(p + 128);
    return make_double4(a.x, a.y, b.x, b.y);
}
template <> __device__ __forceinline__ RecF small_load<RecF>(const unsigned char *p) {
    const float4 a = *reinterpret_cast<const float4 *>(p), b = *reinterpret_cast<const float4 *>(p + 128);
    return RecF{a.x, a.y, a.z, a.w, b.x, b.y, b.z, 0.f};
}
__device__ __forceinline__ void small_store(unsigned char *p, const double4 &r) {
    *reinterpret_cast<double2 *>(p) = make_double2(r.x, r.y);
    *reinterpret_cast<double2 *>(p + 128) = make_double2(r.z, r.w);
}
__device__ __forceinline__ void small_store(unsigned char *p, const RecF &r) {
    *reinterpret_cast<float4 *>(p) = make_float4(r.xh, r.yh, r.zh, r.s);
    *reinterpret_cast<float4 *>(p + 128) = make_float4(r.xl, r.yl, r.zl, 0.f);
}
// a thread's cursor in the staged records: [k] is the record k places further on (k a multiple of 8)
template <class Rec>
struct SmallCursor {
    const unsigned char *p;
    __device__ __forceinline__ Rec operator[](int k) const { return small_load<Rec>(p + k * 32); }
    __device__ __forceinline__ SmallCursor &operator+=(int k) { p += k * 32; return *this; }
};

// Lean FP64 terms (round 2; the list sweeps' form, sc_cutoff.cuh): the self term is excluded by ONE select -- the high
// word of the MUFU seed, whose low word is 0 anyway, is replaced by 0, so that every later product is an exact 0 (r^2 = 0
// of the self pair gives seed = inf, which the select discards before any arithmetic; 0 x 0 on the way, never 0 x inf) --
// instead of selects on r^2 and on the result around a branch, and the terms go into their sums by fused multiply-adds.
__device__ __forceinline__ double small_seed_or_zero(double seed, bool keep) {
    return __hiloint2double(keep ? __double2hiint(seed) : 0, 0);
}
template <int ME>
__device__ __forceinline__ void small_density_acc(const double4 &pi, const double4 &p, bool self, int m_exp, double &acc) {
    const double dx = pi.x - p.x, dy = pi.y - p.y, dz = pi.z - p.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    if constexpr (ME > 0 && ME % 2 == 0) {
        const double y0 = small_seed_or_zero(rcp_seed(r2), !self);
        const double e = fma(-r2, y0, 1.0);
        const double w = fma(y0, fma(e, e, e), y0);
        if constexpr (ME == 6) acc = fma(w * w, w, acc);
        else acc += ipow_c<ME / 2>(w);
    } else {
        const double y0 = small_seed_or_zero(rsqrt_seed(r2), !self);
        const double tt = r2 * y0, e = fma(-tt, y0, 1.0);
        const double y = fma(y0, e * fma(0.375, e, 0.5), y0);
        acc += (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
    }
}
template <int NE, int ME, bool ENERGY>
__device__ __forceinline__ void small_force_acc(const double4 &pi, const double4 &p, bool self, double An, int n_exp,
                                                int m_exp, double (&acc)[4]) {
    const double dx = pi.x - p.x, dy = pi.y - p.y, dz = pi.z - p.z;
    const double r2 = fma(dz, dz, fma(dy, dy, dx * dx));
    const double y0 = small_seed_or_zero(rsqrt_seed(r2), !self);
    const double tt = r2 * y0, e = fma(-tt, y0, 1.0);
    const double y = fma(y0, e * fma(0.375, e, 0.5), y0);
    const double w = y * y;
    const double ss = pi.w + p.w;
    double coef;
    if constexpr (NE == 9 && ME == 6) {
        const double w2 = w * w, w4 = w2 * w2, y3 = w * y;
        coef = w4 * fma(An, y3, -ss);
        if constexpr (ENERGY) acc[3] = fma(w4, y, acc[3]);
    } else {
        const double pm = (ME > 0) ? ipow_c<(ME > 0 ? ME : 1)>(y) : ipow_rt(y, m_exp);
        const double pn = (NE > 0) ? ipow_c<(NE > 0 ? NE : 1)>(y) : ipow_rt(y, n_exp);
        coef = w * fma(An, pn, -ss * pm);
        if constexpr (ENERGY) acc[3] += pn;
    }
    acc[0] = fma(coef, dx, acc[0]);
    acc[1] = fma(coef, dy, acc[1]);
    acc[2] = fma(coef, dz, acc[2]);
}
// Sweep 2 of one thread: records q, q + JL, ... of the staged array against row i, two chains of sums (a, b).  The four
// records of an iteration sit at pj, pj + JL, pj + 2 JL, pj + 3 JL: one pointer and three offsets kept in registers,
// the self test compares the distance i - j with the same offsets.
template <int NE, int ME, bool ENERGY>
__device__ __forceinline__ void small_sweep2(const unsigned char *sm, int N, int i, int q, int JL, double An, int n_exp, int m_exp,
                                             double (&acc)[4]) {
    const double4 pi = small_load<double4>(sm + small_rec_off(i));
    double b[4] = {0.0, 0.0, 0.0, 0.0};                            // second chain
    const int JL2 = 2 * JL, JL3 = 3 * JL;
    SmallCursor<double4> pj{sm + small_rec_off(q)};
    int d = i - q, left = N - q;                                    // self iff d == offset; records left from pj on
    for (; left > JL3; left -= 4 * JL, d -= 4 * JL, pj += 4 * JL) { // 4 independent pair terms in flight
        small_force_acc<NE, ME, ENERGY>(pi, pj[0], d == 0, An, n_exp, m_exp, acc);
        small_force_acc<NE, ME, ENERGY>(pi, pj[JL], d == JL, An, n_exp, m_exp, b);
        small_force_acc<NE, ME, ENERGY>(pi, pj[JL2], d == JL2, An, n_exp, m_exp, acc);
        small_force_acc<NE, ME, ENERGY>(pi, pj[JL3], d == JL3, An, n_exp, m_exp, b);
    }
    for (; left > 0; left -= JL, d -= JL, pj += JL) small_force_acc<NE, ME, ENERGY>(pi, pj[0], d == 0, An, n_exp, m_exp, acc);
#pragma unroll
    for (int c = 0; c < 4; ++c) acc[c] += b[c];
}

// ---- mixed precision (binary32 pair arithmetic on split coordinates, binary64 accumulation) ----
// staged record: x = xh + xl with xh = fl32(x), xl = fl32(x - xh), so that (xh_i - xh_j) + (xl_i - xl_j) keeps the
// accuracy of a binary64 subtraction to within binary32 rounding of the DIFFERENCE (as in allpairs32_kernel)
using SmallRecF = RecF;
// Lean binary32 terms: the self term by one select on the MUFU seed (a zero seed makes every later product an exact 0:
// the Newton step forms 0 x 0, never 0 x inf), sums by fused multiply-adds; ENERGY as in the FP64 form
template <int ME>
__device__ __forceinline__ void small_density_acc_f(const SmallRecF &pi, const SmallRecF &p, bool self, int m_exp, float &acc) {
    const float dx = (pi.xh - p.xh) + (pi.xl - p.xl), dy = (pi.yh - p.yh) + (pi.yl - p.yl), dz = (pi.zh - p.zh) + (pi.zl - p.zl);
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    if constexpr (ME > 0 && ME % 2 == 0) {
        float y0;
        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(r2));
        y0 = self ? 0.f : y0;
        const float w = fmaf(y0, fmaf(-r2, y0, 1.0f), y0);
        if constexpr (ME == 6) acc = fmaf(w * w, w, acc);
        else acc += ipow_cf<ME / 2>(w);
    } else {
        float y0;
        asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(r2));
        y0 = self ? 0.f : y0;
        const float e = fmaf(-(r2 * y0), y0, 1.0f);
        const float y = fmaf(y0 * e, 0.5f, y0);
        acc += (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
    }
}
template <int NE, int ME, bool ENERGY>
__device__ __forceinline__ void small_force_acc_f(const SmallRecF &pi, const SmallRecF &p, bool self, float Anf, int n_exp,
                                                  int m_exp, float (&acc)[4]) {
    const float dx = (pi.xh - p.xh) + (pi.xl - p.xl), dy = (pi.yh - p.yh) + (pi.yl - p.yl), dz = (pi.zh - p.zh) + (pi.zl - p.zl);
    const float r2 = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    float y0;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(r2));
    y0 = self ? 0.f : y0;
    const float e = fmaf(-(r2 * y0), y0, 1.0f);
    const float y = fmaf(y0 * e, 0.5f, y0);
    const float w = y * y;
    const float ss = pi.s + p.s;
    float coef;
    if constexpr (NE == 9 && ME == 6) {
        const float w2 = w * w, w4 = w2 * w2, y3 = w * y;
        coef = w4 * fmaf(Anf, y3, -ss);
        if constexpr (ENERGY) acc[3] = fmaf(w4, y, acc[3]);
    } else {
        const float pm = (ME > 0) ? ipow_cf<(ME > 0 ? ME : 1)>(y) : ipow_rtf(y, m_exp);
        const float pn = (NE > 0) ? ipow_cf<(NE > 0 ? NE : 1)>(y) : ipow_rtf(y, n_exp);
        coef = w * fmaf(Anf, pn, -ss * pm);
        if constexpr (ENERGY) acc[3] += pn;
    }
    acc[0] = fmaf(coef, dx, acc[0]);
    acc[1] = fmaf(coef, dy, acc[1]);
    acc[2] = fmaf(coef, dz, acc[2]);
}
// mixed sweep 2 of one thread: binary32 partial sums over <= 8 terms (two chains of four), then binary64
template <int NE, int ME, bool ENERGY>
__device__ __forceinline__ void small_sweep2_f(const unsigned char *sm, int N, int i, int q, int JL, float Anf, int n_exp,
                                               int m_exp, double (&acc)[4]) {
    const SmallRecF pi = small_load<SmallRecF>(sm + small_rec_off(i));
    SmallCursor<SmallRecF> pj{sm + small_rec_off(q)};
    int d = i - q, left = N - q;
    const int JL7 = 7 * JL;
    for (; left > JL7; left -= 8 * JL, d -= 8 * JL, pj += 8 * JL) {
        float fa[4] = {0.f, 0.f, 0.f, 0.f}, fb[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            small_force_acc_f<NE, ME, ENERGY>(pi, pj[(2 * u) * JL], d == (2 * u) * JL, Anf, n_exp, m_exp, fa);
            small_force_acc_f<NE, ME, ENERGY>(pi, pj[(2 * u + 1) * JL], d == (2 * u + 1) * JL, Anf, n_exp, m_exp, fb);
        }
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[c] += double(fa[c] + fb[c]);
    }
    if (left > 0) {                                                 // <= 7 records left
        float fa[4] = {0.f, 0.f, 0.f, 0.f};
        for (; left > 0; left -= JL, d -= JL, pj += JL) small_force_acc_f<NE, ME, ENERGY>(pi, pj[0], d == 0, Anf, n_exp, m_exp, fa);
#pragma unroll
        for (int c = 0; c < 4; ++c) acc[c] += double(fa[c]);
    }
}

template <int NE, int ME, bool MIXED>
__global__ void __launch_bounds__(kSmallThreads, 1) small_step_kernel(const SmallStepArgs a) {
    unsigned long long bar_target = a.barrier_base;
    auto grid_sync = [&]() { bar_target += gridDim.x; grid_barrier(a.barrier, bar_target); };
    extern __shared__ __align__(32) unsigned char smem_raw[];
    const int N = a.n_atoms;
    unsigned char *sm = smem_raw;                                       // staged records (small_rec_off); MIXED: split binary32
    double *warp_red = reinterpret_cast<double *>(smem_raw + small_rec_bytes(N));
    double *rowval = warp_red + (kSmallThreads / 32) * kSmallMaxRowsPerWarp * 4;
    __shared__ double s_lambda;

    // thread -> (row r of this CTA, q of the row's JL threads): a warp holds RPW = 32 / lq rows (lq consecutive q each);
    // a group of JL / lq consecutive warps covers the JL threads of its RPW rows
    const int t = threadIdx.x, JL = a.jl, LQ = a.lq;
    const int rpw = 32 / LQ, wpg = JL / LQ;
    const int r = ((t >> 5) / wpg) * rpw + (t & 31) / LQ;
    const int q = ((t >> 5) % wpg) * LQ + (t & 31) % LQ;
    const int row0 = blockIdx.x * a.rows;
    const int nrows = min(a.rows, N - row0);
    const int i = row0 + r;
    const bool rowlive = r < nrows;
    const bool owner = rowlive && q == 0;
    const int n_exp = (NE > 0) ? NE : a.c.n, m_exp = (ME > 0) ? ME : a.c.m;
    const double An = a.c.An;
    const float Anf = float(An);

    double vx = 0, vy = 0, vz = 0, fx = 0, fy = 0, fz = 0, my_rho = 0;
    if (owner) {
        vx = a.vel[3 * size_t(i)]; vy = a.vel[3 * size_t(i) + 1]; vz = a.vel[3 * size_t(i) + 2];
        fx = a.force[3 * size_t(i)]; fy = a.force[3 * size_t(i) + 1]; fz = a.force[3 * size_t(i) + 2];
    }
    double lambda = a.scal[kSlotLambda];                   // a scale left pending by an earlier call
    double e_emb = 0.0, e_pair = 0.0, ke_sum = 0.0;        // thread 0: this CTA's partials of the last step
    double ke_final = 0.0, temp_final = 0.0;

    double px = 0, py = 0, pz = 0, sp = 0;                 // owner: position and s' of its atom
    if (owner) {
        const double4 p = load_record_cg(a.xs + i);
        px = p.x; py = p.y; pz = p.z; sp = p.w;
    }
    // The two position buffers the steps alternate between hold the records ALREADY in the staged layout (and, MIXED,
    // already split): staging is one bulk async copy (TMA) per CTA instead of N / 512 load-convert-store rounds per
    // thread.  The copy runs in the async proxy and reads what other CTAs wrote through the generic proxy before the
    // grid barrier, hence the proxy fence.
    __shared__ uint64_t stage_bar;
    uint32_t stage_uses = 0;
    if (t == 0) { mbar_init(&stage_bar, 1); mbar_fence_init(); }
    __syncthreads();
    auto stage = [&](const double4 *cur) {
        __syncthreads();                                    // everyone is done with the previous contents
        if (t == 0) {
            asm volatile("fence.proxy.async.global;" ::: "memory");
            const uint32_t bytes = uint32_t(small_rec_bytes(N));
            mbar_arrive_expect_tx(&stage_bar, bytes);
            for (uint32_t off = 0; off < bytes; off += 32768u)
                bulk_copy_g2s(sm + off, reinterpret_cast<const unsigned char *>(cur) + off, min(32768u, bytes - off), &stage_bar);
        }
        mbar_wait(&stage_bar, stage_uses & 1u);
        ++stage_uses;
    };

    for (long long k = 1; k <= a.nsteps; ++k) {
        double4 *cur = (k & 1) ? a.xs_b : a.xs;
        // ---- A: first half kick + drift ----
        if (owner) {
            vx *= lambda; vy *= lambda; vz *= lambda;
            vx = fma(a.hk, fx, vx); vy = fma(a.hk, fy, vy); vz = fma(a.hk, fz, vz);
            px = fma(a.dt, vx, px); py = fma(a.dt, vy, py); pz = fma(a.dt, vz, pz);
            unsigned char *dst = reinterpret_cast<unsigned char *>(cur) + small_rec_off(i);
            if constexpr (MIXED) small_store(dst, split_record(make_double4(px, py, pz, sp)));
            else small_store(dst, make_double4(px, py, pz, sp));
        }
        lambda = 1.0;
        grid_sync();

        // ---- B: sweep 1 ----
        stage(cur);
        {
            double acc[1] = {0.0};
            if (rowlive && MIXED) {
                const SmallRecF pi = small_load<SmallRecF>(sm + small_rec_off(i));
                SmallCursor<SmallRecF> pj{sm + small_rec_off(q)};
                int d = i - q, left = N - q;
                const int JL7 = 7 * JL;
                for (; left > JL7; left -= 8 * JL, d -= 8 * JL, pj += 8 * JL) {   // binary32 partial sums over 8 terms, then binary64
                    float t0 = 0.f, t1 = 0.f;
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        small_density_acc_f<ME>(pi, pj[(2 * u) * JL], d == (2 * u) * JL, m_exp, t0);
                        small_density_acc_f<ME>(pi, pj[(2 * u + 1) * JL], d == (2 * u + 1) * JL, m_exp, t1);
                    }
                    acc[0] += double(t0 + t1);
                }
                if (left > 0) {
                    float t0 = 0.f;
                    for (; left > 0; left -= JL, d -= JL, pj += JL) small_density_acc_f<ME>(pi, pj[0], d == 0, m_exp, t0);
                    acc[0] += double(t0);
                }
            } else if (rowlive) {
                const double4 pi = small_load<double4>(sm + small_rec_off(i));
                double t0 = 0.0, t1 = 0.0, t2 = 0.0, t3 = 0.0;   // 4 independent chains; summed in a fixed order
                const int JL2 = 2 * JL, JL3 = 3 * JL;
                SmallCursor<double4> pj{sm + small_rec_off(q)};
                int d = i - q, left = N - q;                      // self term excluded by index: iff d == offset
                for (; left > JL3; left -= 4 * JL, d -= 4 * JL, pj += 4 * JL) {
                    small_density_acc<ME>(pi, pj[0], d == 0, m_exp, t0);
                    small_density_acc<ME>(pi, pj[JL], d == JL, m_exp, t1);
                    small_density_acc<ME>(pi, pj[JL2], d == JL2, m_exp, t2);
                    small_density_acc<ME>(pi, pj[JL3], d == JL3, m_exp, t3);
                }
                for (; left > 0; left -= JL, d -= JL, pj += JL) small_density_acc<ME>(pi, pj[0], d == 0, m_exp, t0);
                acc[0] = (t0 + t1) + (t2 + t3);
            }
            row_reduce<1>(acc, JL, LQ, q, warp_red);
            double root = 0.0;
            if (owner) {
                my_rho = a.c.am * acc[0];
                root = my_rho > 0.0 ? sqrt(my_rho) : 0.0;                    // reading Q9
                sp = my_rho > 0.0 ? a.c.Bm / root : 0.0;
                a.sprime[i] = sp;
            }
            if (k == a.nsteps) e_emb = rows_sum(root, owner, r, nrows, rowval);
        }
        grid_sync();

        // ---- C: sweep 2 (positions are still staged; fetch the s' of this step) ----
        for (int j = t; j < N; j += kSmallThreads) {
            if constexpr (MIXED) *reinterpret_cast<float *>(sm + small_rec_off(j) + 12) = float(__ldcg(a.sprime + j));
            else *reinterpret_cast<double *>(sm + small_rec_off(j) + 128 + 8) = __ldcg(a.sprime + j);
        }
        __syncthreads();
        {
            double acc[4] = {0.0, 0.0, 0.0, 0.0};
            if (rowlive && MIXED) {
                if (k == a.nsteps) small_sweep2_f<NE, ME, true>(sm, N, i, q, JL, Anf, n_exp, m_exp, acc);
                else small_sweep2_f<NE, ME, false>(sm, N, i, q, JL, Anf, n_exp, m_exp, acc);
            } else if (rowlive) {
                // the pair energy is formed on the call's last step only (block-uniform choice of the instantiation)
                if (k == a.nsteps) small_sweep2<NE, ME, true>(sm, N, i, q, JL, An, n_exp, m_exp, acc);
                else small_sweep2<NE, ME, false>(sm, N, i, q, JL, An, n_exp, m_exp, acc);
            }
            row_reduce<4>(acc, JL, LQ, q, warp_red);
            // ---- D: second half kick (+ Langevin), |v|^2 ----
            double v2 = 0.0;
            if (owner) {
                fx = acc[0]; fy = acc[1]; fz = acc[2];
                vx = fma(a.hk, fx, vx); vy = fma(a.hk, fy, vy); vz = fma(a.hk, fz, vz);
                if (a.thermo == 2) {
                    const double target = a.T_start + (a.T_end - a.T_start) * double(k) / double(a.nsteps);
                    const double c2 = sqrt(a.lg_pre * target * kAcc / a.mass);
                    const unsigned long long step = a.lg_step0 + (unsigned long long)(k - 1);
                    const uint4 wd = philox4x32_10(make_uint4(uint32_t(i), uint32_t(step), uint32_t(step >> 32), 0u), a.key0, a.key1);
                    const double ra = sqrt(-2.0 * log(unit_open(wd.x))), rb = sqrt(-2.0 * log(unit_open(wd.z)));
                    double sa, ca, sb, cb;
                    sincospi(2.0 * unit_open(wd.y), &sa, &ca);
                    sincospi(2.0 * unit_open(wd.w), &sb, &cb);
                    vx = fma(a.lg_c1, vx, c2 * (ra * ca));
                    vy = fma(a.lg_c1, vy, c2 * (ra * sa));
                    vz = fma(a.lg_c1, vz, c2 * (rb * cb));
                }
                v2 = fma(vz, vz, fma(vy, vy, vx * vx));
            }
            const bool last = (k == a.nsteps);
            if (last) e_pair = rows_sum(acc[3], owner, r, nrows, rowval);
            if (a.thermo == 1 || last) {
                ke_sum = rows_sum(v2, owner, r, nrows, rowval);
                if (t == 0) a.part_ke[blockIdx.x] = ke_sum;
                grid_sync();
                // every CTA forms the same total (same order, same bits)
                if (t < 32) {
                    const double tot = warp0_sum_partials(a.part_ke, int(gridDim.x));
                    if (t == 0) {
                        double ke = 0.5 * a.mass * tot / kAcc;
                        double temp = a.ndof > 0.0 ? 2.0 * ke / (kBoltzmann * a.ndof) : 0.0;
                        double lam = 1.0;
                        if (a.thermo == 1 && temp > 0.0) {
                            const double target = a.T_start + (a.T_end - a.T_start) * double(k) / double(a.nsteps);
                            lam = sqrt(target / temp);
                            ke *= lam * lam;
                            temp = a.ndof > 0.0 ? 2.0 * ke / (kBoltzmann * a.ndof) : 0.0;
                        }
                        s_lambda = lam; ke_final = ke; temp_final = temp;
                    }
                }
                __syncthreads();
                lambda = s_lambda;
            }
        }
    }

    // ---- epilogue: state back to global memory, scalars ----
    if (owner) {
        a.vel[3 * size_t(i)] = vx * lambda; a.vel[3 * size_t(i) + 1] = vy * lambda; a.vel[3 * size_t(i) + 2] = vz * lambda;
        a.force[3 * size_t(i)] = fx; a.force[3 * size_t(i) + 1] = fy; a.force[3 * size_t(i) + 2] = fz;
        a.rho[i] = my_rho;
        a.xs[i] = make_double4(px, py, pz, sp);             // after the last barrier: nobody stages any more (back to the plain layout)
        if (a.xf) store_split_record(a.xf, i, px, py, pz, float(sp));
        if (a.xfr) a.xfr[i] = split_record(make_double4(px, py, pz, sp));
    }
    // the staged layout spilled into the up to 7 padding records behind record N - 1 of xs: zero again, as sc_create left them
    if (blockIdx.x == 0 && t < 8 && N + t < ((N + 7) & ~7)) a.xs[N + t] = make_double4(0.0, 0.0, 0.0, 0.0);
    if (t == 0) { a.part_emb[blockIdx.x] = e_emb; a.part_pair[blockIdx.x] = e_pair; }
    grid_sync();
    if (blockIdx.x == 0 && t < 32) {
        const double emb = warp0_sum_partials(a.part_emb, int(gridDim.x));
        const double pair = warp0_sum_partials(a.part_pair, int(gridDim.x));
        if (t == 0) {
            a.scal[kSlotEEmb] = -a.c.eps_c * emb;
            a.scal[kSlotEPair] = a.c.En * pair;
            a.scal[kSlotKE] = ke_final;
            a.scal[kSlotTemp] = temp_final;
            a.scal[kSlotLambda] = 1.0;
        }
    }
}
#endif  // SCMD_MAIN_TU

}  // namespace scmd
