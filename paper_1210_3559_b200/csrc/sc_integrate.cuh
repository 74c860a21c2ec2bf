// sc_integrate.cuh -- O(N) kernels around the sweeps: state packing, velocity-Verlet kicks and
// drift (reading Q3), kinetic-energy / temperature reduction, rescale thermostat
// (reading Q6), fixed-order scalar reductions.  All streaming, 24..72 B per atom.
#pragma once
#include "sc_device.cuh"

namespace scmd {

constexpr double kAcc = 9.648533215665e-3;   // A fs^-2 per (eV A^-1 u^-1), CODATA-2018 e / u
constexpr double kBoltzmann = 8.617333262e-5;   // eV / K

// device scalar slots (double scal[kNumScalars])
enum ScalarSlot {
    kSlotEPair = 0,     // U_pair (eV)
    kSlotEEmb = 1,      // U_emb (eV)
    kSlotKE = 2,        // kinetic energy (eV)
    kSlotTemp = 3,      // temperature (K)
    kSlotLambda = 4,    // pending velocity scale of the rescale thermostat (1 = none)
    kSlotMaxDisp2 = 5,  // max squared displacement since the last list build (cutoff path)
    kNumScalars = 16
};

#ifdef SCMD_MAIN_TU   // the non-template kernels are compiled in scmd.cu only
// pos[N*3] -> xs[N] = (x, y, z, 0); xf (mixed all-pairs path, else NULL) gets the split record
__global__ void pack_positions_kernel(const double *__restrict__ pos, double4 *__restrict__ xs, FPair *__restrict__ xf, RecF *__restrict__ xfr,
                                      int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) {
        const double x = pos[3 * size_t(i)], y = pos[3 * size_t(i) + 1], z = pos[3 * size_t(i) + 2];
        xs[i] = make_double4(x, y, z, 0.0);
        if (xf) store_split_record(xf, i, x, y, z, 0.f);
        if (xfr) xfr[i] = split_record(make_double4(x, y, z, 0.0));     // mixed list sweeps
    }
}
__global__ void unpack_positions_kernel(const double4 *__restrict__ xs, double *__restrict__ pos, int N) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) {
        const double4 p = xs[i];
        pos[3 * size_t(i)] = p.x; pos[3 * size_t(i) + 1] = p.y; pos[3 * size_t(i) + 2] = p.z;
    }
}

// Row split over several GPUs (scmd.h: sc_step_rows): positions of atoms [first, last) out of the records into the
// caller's all-atoms array, and s' of EVERY record from the all-atoms densities the ranks exchanged (the same
// expression as the sweep-1 epilogues, so every rank forms the same bits).
__global__ void export_rows_kernel(const double4 *__restrict__ xs, double *__restrict__ pos_all, int first, int last) {
    const int i = first + blockIdx.x * blockDim.x + threadIdx.x;
    if (i < last) {
        const double4 p = xs[i];
        pos_all[3 * size_t(i)] = p.x; pos_all[3 * size_t(i) + 1] = p.y; pos_all[3 * size_t(i) + 2] = p.z;
    }
}
__global__ void import_density_kernel(const double *__restrict__ rho_all, double4 *__restrict__ xs, FPair *__restrict__ xf,
                                      RecF *__restrict__ xfr, double *__restrict__ rho, int N, double Bm) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) {
        const double r = rho_all[i];
        const double sp = r > 0.0 ? Bm / sqrt(r) : 0.0;                  // reading Q9
        xs[i].w = sp;
        rho[i] = r;
        if (xf) reinterpret_cast<float *>(xf + (i >> 1))[6 + (i & 1)] = -float(sp);
        if (xfr) xfr[i].s = float(sp);
    }
}

// first half kick + drift:  v <- lambda v (pending thermostat scale);  v += hk F;  x += dt v
// (hk = dt/2 * ACC / m).  ref (may be NULL): positions at the last list build; the largest squared
// displacement from it goes to scal[kSlotMaxDisp2] through an integer atomicMax (order-free).
__global__ void kick_drift_kernel(double4 *__restrict__ xs, double *__restrict__ vel, const double *__restrict__ force,
                                  double *__restrict__ scal, const double4 *__restrict__ ref, FPair *__restrict__ xf, RecF *__restrict__ xfr,
                                  int first, int N, double hk, double dt) {
    const int i = first + blockIdx.x * blockDim.x + threadIdx.x;       // atoms [first, N)
    double d2 = 0.0;
    if (i < N) {
        const double lambda = scal[kSlotLambda];
        double4 p = xs[i];
        double vx = vel[3 * size_t(i)] * lambda, vy = vel[3 * size_t(i) + 1] * lambda, vz = vel[3 * size_t(i) + 2] * lambda;
        vx = fma(hk, force[3 * size_t(i)], vx);
        vy = fma(hk, force[3 * size_t(i) + 1], vy);
        vz = fma(hk, force[3 * size_t(i) + 2], vz);
        p.x = fma(dt, vx, p.x); p.y = fma(dt, vy, p.y); p.z = fma(dt, vz, p.z);
        vel[3 * size_t(i)] = vx; vel[3 * size_t(i) + 1] = vy; vel[3 * size_t(i) + 2] = vz;
        xs[i] = p;
        if (xf) store_split_record(xf, i, p.x, p.y, p.z, float(p.w));
        if (xfr) xfr[i] = split_record(p);
        if (ref) {
            const double4 r = ref[i];
            const double ex = p.x - r.x, ey = p.y - r.y, ez = p.z - r.z;
            d2 = fma(ez, ez, fma(ey, ey, ex * ex));
        }
    }
    if (ref) {
        // non-negative doubles order like their bit patterns
        unsigned long long bits = __double_as_longlong(d2);
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            unsigned long long o = __shfl_xor_sync(0xffffffffu, bits, off);
            bits = o > bits ? o : bits;
        }
        if ((threadIdx.x & 31) == 0 && bits != 0ull)
            atomicMax(reinterpret_cast<unsigned long long *>(scal + kSlotMaxDisp2), bits);
    }
}

// second half kick + per-block sum of |v|^2 -> part[blockIdx.x]
__global__ void kick_ke_kernel(double *__restrict__ vel, const double *__restrict__ force, double *__restrict__ part,
                               int first, int N, double hk) {
    __shared__ double scratch[32];
    const int i = first + blockIdx.x * blockDim.x + threadIdx.x;       // atoms [first, N)
    double v2 = 0.0;
    if (i < N) {
        double vx = fma(hk, force[3 * size_t(i)], vel[3 * size_t(i)]);
        double vy = fma(hk, force[3 * size_t(i) + 1], vel[3 * size_t(i) + 1]);
        double vz = fma(hk, force[3 * size_t(i) + 2], vel[3 * size_t(i) + 2]);
        vel[3 * size_t(i)] = vx; vel[3 * size_t(i) + 1] = vy; vel[3 * size_t(i) + 2] = vz;
        v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    }
    const double t = block_sum(v2, scratch);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

// Langevin thermostat (reading Q18 of DESIGN.md): after the second half kick the exact
// Ornstein-Uhlenbeck update v <- c1 v + c2 xi, xi = three standard normals per (atom, step) from
// Philox4x32-10 keyed by the seed, counter = (caller's atom index, step lo, step hi, 0).
struct LangevinArgs {
    double c1, c2;                  // exp(-gamma dt), sqrt((1 - c1^2) kB T ACC / m)
    uint32_t key0, key1;            // seed lo, hi
    uint32_t step_lo, step_hi;      // generator step
    const int *perm;                // internal -> caller's atom index (cutoff path), else NULL
};

__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint32_t k0, uint32_t k1) {
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t h0 = __umulhi(0xD2511F53u, c.x), l0 = 0xD2511F53u * c.x;
        const uint32_t h1 = __umulhi(0xCD9E8D57u, c.z), l1 = 0xCD9E8D57u * c.z;
        c = make_uint4(h1 ^ c.y ^ k0, l1, h0 ^ c.w ^ k1, l0);
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return c;
}
__device__ __forceinline__ double unit_open(uint32_t w) { return (double(w) + 0.5) * 2.3283064365386963e-10; }  // 2^-32

// second half kick + Langevin update + per-block sum of |v|^2 -> part[blockIdx.x]
__global__ void kick_langevin_ke_kernel(double *__restrict__ vel, const double *__restrict__ force,
                                        double *__restrict__ part, int first, int N, double hk, const LangevinArgs lg) {
    __shared__ double scratch[32];
    const int i = first + blockIdx.x * blockDim.x + threadIdx.x;       // atoms [first, N)
    double v2 = 0.0;
    if (i < N) {
        double vx = fma(hk, force[3 * size_t(i)], vel[3 * size_t(i)]);
        double vy = fma(hk, force[3 * size_t(i) + 1], vel[3 * size_t(i) + 1]);
        double vz = fma(hk, force[3 * size_t(i) + 2], vel[3 * size_t(i) + 2]);
        const uint32_t atom = uint32_t(lg.perm ? lg.perm[i] : i);
        const uint4 w = philox4x32_10(make_uint4(atom, lg.step_lo, lg.step_hi, 0u), lg.key0, lg.key1);
        const double ra = sqrt(-2.0 * log(unit_open(w.x))), rb = sqrt(-2.0 * log(unit_open(w.z)));
        double sa, ca, sb, cb;
        sincospi(2.0 * unit_open(w.y), &sa, &ca);
        sincospi(2.0 * unit_open(w.w), &sb, &cb);
        vx = fma(lg.c1, vx, lg.c2 * (ra * ca));
        vy = fma(lg.c1, vy, lg.c2 * (ra * sa));
        vz = fma(lg.c1, vz, lg.c2 * (rb * cb));
        vel[3 * size_t(i)] = vx; vel[3 * size_t(i) + 1] = vy; vel[3 * size_t(i) + 2] = vz;
        v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    }
    const double t = block_sum(v2, scratch);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

// per-block sum of |v|^2 without a kick (sc_kinetic)
__global__ void sum_v2_kernel(const double *__restrict__ vel, double *__restrict__ part, int first, int N, double lambda_apply,
                              const double *__restrict__ scal) {
    __shared__ double scratch[32];
    const int i = first + blockIdx.x * blockDim.x + threadIdx.x;       // atoms [first, N)
    double v2 = 0.0;
    if (i < N) {
        const double l = lambda_apply != 0.0 ? scal[kSlotLambda] : 1.0;
        const double vx = vel[3 * size_t(i)] * l, vy = vel[3 * size_t(i) + 1] * l, vz = vel[3 * size_t(i) + 2] * l;
        v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    }
    const double t = block_sum(v2, scratch);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

// v <- lambda v, lambda <- 1  (flushes a pending thermostat scale)
__global__ void scale_velocities_kernel(double *__restrict__ vel, const double *__restrict__ scal, int n3) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n3) vel[i] *= scal[kSlotLambda];
}
__global__ void reset_lambda_kernel(double *__restrict__ scal) { scal[kSlotLambda] = 1.0; }

// one block: fixed-order sum of part[0..n) -> scal[slot] = scale * sum
__global__ void reduce_partials_kernel(const double *__restrict__ part, int n, double *__restrict__ scal, int slot,
                                       double scale) {
    __shared__ double scratch[32];
    double v = 0.0;
    for (int k = threadIdx.x; k < n; k += blockDim.x) v += part[k];
    const double t = block_sum(v, scratch);
    if (threadIdx.x == 0) scal[slot] = scale * t;
}

// the same with a count-proportional constant taken off the sum first (energy-shifted cutoff: every in-range ordered
// pair loses r_c^-n; the count is the one sweep 1 left for the same positions): scal[slot] = scale * (sum - shift * count)
__global__ void reduce_partials_shift_kernel(const double *__restrict__ part, int n, double *__restrict__ scal, int slot,
                                             double scale, const unsigned long long *__restrict__ count, double shift) {
    __shared__ double scratch[32];
    double v = 0.0;
    for (int k = threadIdx.x; k < n; k += blockDim.x) v += part[k];
    const double t = block_sum(v, scratch);
    if (threadIdx.x == 0) scal[slot] = scale * fma(-double(*count), shift, t);
}

// one block: KE and T from the per-block |v|^2 sums; optionally the rescale factor for T_target
//   KE = 1/2 m sum|v|^2 / ACC ;  T = 2 KE / (kB ndof) ;  lambda = sqrt(T_target / T)
// After a rescale the stored KE and T are those of the rescaled velocities.
__global__ void reduce_ke_kernel(const double *__restrict__ part, int n, double *__restrict__ scal, double mass,
                                 double ndof, int thermo, double t_target) {
    __shared__ double scratch[32];
    double v = 0.0;
    for (int k = threadIdx.x; k < n; k += blockDim.x) v += part[k];
    const double t = block_sum(v, scratch);
    if (threadIdx.x == 0) {
        double ke = 0.5 * mass * t / kAcc;
        double temp = ndof > 0.0 ? 2.0 * ke / (kBoltzmann * ndof) : 0.0;
        double lambda = 1.0;
        if (thermo == 1 && temp > 0.0) {
            lambda = sqrt(t_target / temp);
            ke *= lambda * lambda;
            temp = ndof > 0.0 ? 2.0 * ke / (kBoltzmann * ndof) : 0.0;
        }
        scal[kSlotKE] = ke;
        scal[kSlotTemp] = temp;
        scal[kSlotLambda] = lambda;
    }
}

#endif  // SCMD_MAIN_TU

}  // namespace scmd
