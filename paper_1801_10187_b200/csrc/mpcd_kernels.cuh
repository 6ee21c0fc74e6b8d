// mpcd_kernels.cuh -- the kernels of the MPCD solvent step (sm_100a).
//
// One templated per-particle pass covers every block of Fig. 1 and their fusions;
// compile-time flags select which blocks a launch contains:
//
//   kSRD      a5+a6  SRD collision, Alg. 1: gathers the sums {S, N} and the axis of the
//                    particle's cell, u = S / N, rotates in fp64
//   kATApply  a7     Andersen-thermostat update, eq. 4 PAPER.md:54 (regenerates dv from the tag)
//   kStream   a1     eq. 1 PAPER.md:35 + periodic wrap
//   kBin      a3+a4  shifted binning + fp64 cell accumulation
//   kEnergy   a4     also accumulate sum |v|^2 (kinetic energy, eq. 3)
//   kATDraw   a7     draw dv for the (new) step and accumulate its per-cell sum
//   kThermo   a6     with kSRD: scale the rotated relative velocity by the cell's xi (Maxwell-Boltzmann cell thermostat,
//                    Alg. 1 lines 8-10 PAPER.md:150-152); xi rides in the 4th word of the cell's axis sector
//   kATStored a7     inside mpcd_step: kATDraw leaves the drawn dv in vel.xyz instead of the velocity (the AT update
//                    v = u + dv - D/N_c does not depend on the old velocity, which has been summed by then), and the
//                    next kATApply takes it from there instead of regenerating it: one Gaussian draw per particle-step;
//                    the cell's accumulator then holds sum(v) - sum(dv) (all that eq. 4 needs: v' = (S - D) / N_c + dv),
//                    so there is one sum, one combining tree and one gathered sector per particle instead of two
//   kEmbedded a5     with kSRD: the cell mean is mass-weighted over the solvent sums and the embedded beads' sums
//                    (mpcd_embedded.cuh)
//   kFixed    a4     deterministic accumulation: the cell sums are 64-bit fixed-point integers (mpcd_device.cuh), both
//                    where they are accumulated (kBin) and where they are read (kSRD)
//   kCoherent        the cell arrays read by kSRD were written earlier in the SAME launch (mpcd_small.cuh): plain loads ordered
//                    by the grid barrier instead of the read-only (.nc) path, which promises data constant for the whole launch
//   kCarry           the caller keeps the thread's particle in registers from one pass to the next (mpcd_small.cuh: the same
//                    thread owns the same array slot in every phase between two sorts): no reload of what it has just stored
//   kSortOut  a8     sort by cell on the way out: instead of in place, the particle is written
//                    to slot cell_start[c] + (atomic cursor) of the duplicate arrays, c = its cell in the step
//                    being collided; the separate read-and-scatter pass of the sort disappears
//
// The steady-state step of mpcd_step is ONE particle launch, kSRD|kStream|kBin|kEnergy: the collision of
// step t fused with the streaming, binning and accumulation of step t+1, so each particle's 32 bytes
// (pos4 + vel4) are read once and written once per step.  The mean velocity is formed where it is used
// (u = S / N from the cell's sums), so the only per-cell work between two steps is cell_prepare: the axes
// of the next step and a zeroed accumulator set.
#pragma once
#include "mpcd_device.cuh"
#include "mpcd_embedded.cuh"

namespace mpcdk {

enum : unsigned { kSRD = 1u, kATApply = 2u, kStream = 4u, kBin = 8u, kEnergy = 16u, kATDraw = 32u, kSortOut = 64u, kThermo = 128u, kATStored = 256u, kEmbedded = 512u, kFixed = 1024u, kCoherent = 2048u, kCarry = 4096u };

template <typename T> struct PassArgs {
    typename Vec4<T>::type *pos;
    typename Vec4<T>::type *vel;
    uint32_t *tag;
    // cell arrays of the step being collided (read only)
    const double *sums;   // {Sx, Sy, Sz, N} per cell
    const double *dsum;   // {Dx, Dy, Dz, -} per cell: sum of the thermostat draws (AT)
    const double *axis;   // {nx, ny, nz, xi} per cell (SRD; xi = thermostat factor)
    const double *esum;   // {sum m v, sum m} of the embedded beads per cell (kEmbedded)
    double mass;          // solvent particle mass (kEmbedded)
    // accumulators of the step being binned
    double *acc;          // {Sx, Sy, Sz, N} per cell
    double *qacc;         // sum |v|^2 per cell (kEnergy)
    double *at_acc;       // {Dx, Dy, Dz, -} per cell (AT second reduction)
    // kSortOut: the duplicate particle arrays and the per-cell write cursor (exclusive scan of the counts)
    typename Vec4<T>::type *pos_out;
    typename Vec4<T>::type *vel_out;
    uint32_t *tag_out;
    int32_t *cursor;
    int64_t N, Nc;
    int32_t n[3];
    T dt, L[3], inv_a;
    T shift[3];           // grid shift of the step being binned
    double cos_a, sin_a, sigma;
    uint64_t seed, step_collide, step_bin;
};

// Probe: 1 = the SRD collision of the plain rule forms the cell's axis in registers instead of gathering it.
#ifndef MPCD_AXIS_REG
#define MPCD_AXIS_REG 0
#endif
constexpr bool kAxisReg = MPCD_AXIS_REG != 0;

#ifndef MPCD_PASS_THREADS
#define MPCD_PASS_THREADS 128
#endif
constexpr int kPassThreads = MPCD_PASS_THREADS;

// a3 (A6, A8): linear index of the collision cell of position p under grid shift s.
template <typename T, typename V4>
__device__ __forceinline__ int cell_of(const V4 &p, const T (&s)[3], T inv_a, const int32_t (&n)[3])
{
    const int ix = bin_axis<T>(p.x, s[0], inv_a, n[0]);
    const int iy = bin_axis<T>(p.y, s[1], inv_a, n[1]);
    const int iz = bin_axis<T>(p.z, s[2], inv_a, n[2]);
    return ix + n[0] * (iy + n[1] * iz);
}

// The cell index of the last binning is cached in the fourth component of the velocity vector, as in
// the paper ("cached into the fourth element of the particle velocity vector"): vel.w is
// loaded and stored with the 16-byte vector anyway, so the cache costs no HBM traffic, where a separate
// int32 array would cost 8 bytes per particle-step.  At the ABI vel.w stays unspecified padding (A9).
__device__ __forceinline__ float cell_to_w(int c, float) { return __int_as_float(c); }
__device__ __forceinline__ double cell_to_w(int c, double) { return __longlong_as_double((long long)c); }
__device__ __forceinline__ int w_to_cell(float w) { return __float_as_int(w); }
__device__ __forceinline__ int w_to_cell(double w) { return (int)__double_as_longlong(w); }

// Blocks of 128 threads per SM the register count is held to (measured best): 12 (<= 42 registers, 48
// warps) in the mixed model, 10 (<= 51 registers, 40 warps) in the fp64 model, whose 64-bit state needs the registers.
#ifndef MPCD_MINBLOCKS_F32
#define MPCD_MINBLOCKS_F32 12
#endif
#ifndef MPCD_MINBLOCKS_F64
#define MPCD_MINBLOCKS_F64 10
#endif
template <unsigned F> struct PassScratch {
    using type = typename std::conditional<(F & kBin) && (F & kATDraw) && !(F & kATStored), WarpScratchX, WarpScratch>::type;
    static constexpr int count = (F & (kBin | kATDraw)) ? kPassThreads / 32 : 1;     // one per warp when the pass accumulates
};

// The pass over one particle per thread (particle i = blockIdx.x * kPassThreads + threadIdx.x); `w` is the warp's scratch.
template <typename T, unsigned F>
__device__ __forceinline__ void pass_body(const PassArgs<T> &a, typename PassScratch<F>::type &w,
                                          typename Vec4<T>::type *carry_p = nullptr, typename Vec4<T>::type *carry_v = nullptr, bool have = false)
{
    using V4 = typename Vec4<T>::type;
    const int64_t i = (int64_t)blockIdx.x * kPassThreads + threadIdx.x;
    const bool valid = i < a.N;
    const int inactive = -1 - (int)(threadIdx.x & 31);
    V4 p = {}, v = {};
    uint32_t tag = 0;
    // Lanes past the end of the array (last block only) work on a copy of the last particle and simply do not store or
    // accumulate: no branch around the loads, the gather and the arithmetic, so the compiler schedules them as one block.
    const int64_t il = valid ? i : a.N - 1;
    if ((F & kCarry) && have) {
        v = *carry_v; p = *carry_p;
    } else {
        v = load4(a.vel + il);
        if (F & (kStream | kBin)) p = load4(a.pos + il);
    }
    if ((F & (kATDraw | kSortOut)) || ((F & kATApply) && !(F & kATStored))) tag = a.tag[il];
    int c = w_to_cell(v.w);                                      // cell of the last binning (the step being collided)
    int64_t o = i;                                               // where this particle is written
    if ((F & kSortOut) && valid) o = atomicAdd(a.cursor + c, 1); // issued early: its latency hides behind the gather
    if (F & kSRD) {
        {
            f64x4 s = (F & kCoherent) ? ld256(a.sums + 4 * (size_t)c) : ld256_nc(a.sums + 4 * (size_t)c);   // Alg. 1 lines 2-4: the cell's sums and axis, one sector each
            f64x4 n;
            if constexpr (kAxisReg && !(F & (kThermo | kFixed | kCoherent))) {   // probe: no second gathered sector (xi rides in the axis sector; the deterministic mode keeps every kernel on the stored bits)
                axis_in_registers<T>(a.seed, a.step_collide, (uint32_t)c, n.x, n.y, n.z);
                n.w = 1.0;
            } else {
                n = (F & kCoherent) ? ld256(a.axis + 4 * (size_t)c) : ld256_nc(a.axis + 4 * (size_t)c);
            }
            if (F & kFixed) { s.x = acc_value(s.x, true); s.y = acc_value(s.y, true); s.z = acc_value(s.z, true); s.w = acc_count(s.w, true); }
            double ux, uy, uz;
            if (F & kEmbedded) {
                embedded_mean(s, ld256_nc(a.esum + 4 * (size_t)c), a.mass, ux, uy, uz);
            } else {
                const double inv = __drcp_rn(s.w);               // N_c >= 1: this particle is a member
                ux = __dmul_rn(s.x, inv); uy = __dmul_rn(s.y, inv); uz = __dmul_rn(s.z, inv);
            }
            double ox, oy, oz;                                   // lines 5-12
            srd_rotate((double)v.x, (double)v.y, (double)v.z, ux, uy, uz, n.x, n.y, n.z, (F & kThermo) ? n.w : 1.0, a.cos_a, a.sin_a, ox, oy, oz);
            v.x = (T)ox; v.y = (T)oy; v.z = (T)oz;
        }
    }
    if (F & kATApply) {
        {                                                        // eq. 4: v = u + dv_i - D / N_c = (S - D) / N_c + dv_i
            const f64x4 s = ld256_nc(a.sums + 4 * (size_t)c);
            const double inv = __drcp_rn(s.w);
            if (F & kATStored) {                                 // inside mpcd_step the cell's one sum IS S - D (kMinus below), dv_i rides in vel.xyz
                v.x = (T)(s.x * inv + (double)v.x);
                v.y = (T)(s.y * inv + (double)v.y);
                v.z = (T)(s.z * inv + (double)v.z);
            } else {
                const f64x4 d = ld256_nc(a.dsum + 4 * (size_t)c);
                double g0, g1, g2;                               // dv_i of the step being collided
                draw_gauss3<T>(a.seed, a.step_collide, tag, g0, g1, g2);
                v.x = (T)((s.x - d.x) * inv + a.sigma * g0);
                v.y = (T)((s.y - d.y) * inv + a.sigma * g1);
                v.z = (T)((s.z - d.z) * inv + a.sigma * g2);
            }
        }
    }
    if (F & kStream) {
        p.x = stream_wrap<T>(p.x, v.x, a.dt, a.L[0]);
        p.y = stream_wrap<T>(p.y, v.y, a.dt, a.L[1]);
        p.z = stream_wrap<T>(p.z, v.z, a.dt, a.L[2]);
        if (valid) store4(((F & kSortOut) ? a.pos_out : a.pos) + o, p);
    }
    if (F & kBin) {
        c = cell_of<T>(p, a.shift, a.inv_a, a.n);
        v.w = cell_to_w(c, T(0));
    }
    V4 vs = v;                                                   // what goes back to the velocity array
    double ex = 0, ey = 0, ez = 0;                               // dv_i of the step being binned
    if (F & kATDraw) {
        {
            double g0, g1, g2;
            draw_gauss3<T>(a.seed, a.step_bin, tag, g0, g1, g2);
            ex = a.sigma * g0; ey = a.sigma * g1; ez = a.sigma * g2;
            if (F & kATStored) {                                 // the sum below must be the sum of what is stored
                vs.x = (T)ex; vs.y = (T)ey; vs.z = (T)ez;
                ex = (double)vs.x; ey = (double)vs.y; ez = (double)vs.z;
            }
        }
    }
    if ((F & (kSRD | kATApply | kBin)) && valid) store4(((F & kSortOut) ? a.vel_out : a.vel) + o, vs);
    if ((F & kSortOut) && valid) a.tag_out[o] = tag;
    if (F & kCarry) { *carry_p = p; *carry_v = vs; }
    if (!valid) c = inactive;                                    // takes no part in the sums
    if constexpr ((F & kBin) && (F & kATDraw) && (F & kATStored))   // ONE sum per cell: sum(v) - sum(dv) is all eq. 4 needs; the stored dv is what is subtracted
        warp_cell_accumulate<T, true, (F & kEnergy) != 0, false, false, true>(a.acc, a.qacc, w, c, v.x, v.y, v.z, nullptr, 0.0, 0.0, 0.0, vs.x, vs.y, vs.z);
    else if constexpr ((F & kBin) && (F & kATDraw))     // one match and one tree for both sums: same cell, same groups
        warp_cell_accumulate<T, true, (F & kEnergy) != 0, false, true>(a.acc, a.qacc, w, c, v.x, v.y, v.z, a.at_acc, ex, ey, ez);
    else if constexpr ((F & kBin) != 0) warp_cell_accumulate<T, true, (F & kEnergy) != 0, (F & kFixed) != 0>(a.acc, a.qacc, w, c, v.x, v.y, v.z);
    else if constexpr ((F & kATDraw) != 0) warp_cell_accumulate<double, false, false>(a.at_acc, nullptr, w, c, ex, ey, ez);
}

template <typename T, unsigned F>
__global__ void __launch_bounds__(kPassThreads, sizeof(T) == 4 ? MPCD_MINBLOCKS_F32 : MPCD_MINBLOCKS_F64) particle_pass(const PassArgs<T> a)
{
    __shared__ typename PassScratch<F>::type ws[PassScratch<F>::count];
    pass_body<T, F>(a, ws[PassScratch<F>::count > 1 ? (threadIdx.x >> 5) : 0]);
}

// Cell index of every particle (the cache in vel.w) as an int32 array, on demand (mpcd_get_state, mpcd_device_ptrs).
template <typename T>
__global__ void __launch_bounds__(256) cells_of_particles(const PassArgs<T> a, int32_t *cell)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.N) return;
    cell[i] = w_to_cell(load4(a.vel + i).w);
}

// ---------------------------------------------------------------------------------------
// a5, cell side: the random axis of every cell for one step (it depends on
// (seed, step, cell) only, so it can be drawn before that step's particles are binned) and / or a zeroed
// accumulator set.  Any pointer may be NULL.  One launch per step in mpcd_step: the axes of step t + 1
// together with the zeroing of the set of step t + 2.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) cell_prepare(double *axis, uint64_t seed, uint64_t step, double *zero_acc, double *zero_q, double *zero_at, double *zero_emb,
                                                    double *zero_embq, int64_t Nc)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= Nc) return;
    if (zero_acc) st256(zero_acc + 4 * c, 0.0, 0.0, 0.0, 0.0);
    if (zero_q) zero_q[c] = 0.0;
    if (zero_at) st256(zero_at + 4 * c, 0.0, 0.0, 0.0, 0.0);
    if (zero_emb) st256(zero_emb + 4 * c, 0.0, 0.0, 0.0, 0.0);
    if (zero_embq) { zero_embq[2 * c] = 0.0; zero_embq[2 * c + 1] = 0.0; }
    if (axis) {
        double nx, ny, nz;
        draw_axis(seed, step, (uint32_t)c, nx, ny, nz);
        st256(axis + 4 * c, nx, ny, nz, 0.0);
    }
}

// Maxwell-Boltzmann cell thermostat: once the sums of a step are complete, the scale factor
// xi = sqrt(E^ / E_k) of every cell, E_k = m (sum |v|^2 - |S|^2 / N_c) / 2 (eq. 3; A12), E^ drawn
// from the canonical distribution; xi = 1 for N_c < 2 and for E_k = 0.  Written into the 4th word of the cell's
// axis sector, which the collision gathers anyway.
__global__ void __launch_bounds__(256) cell_thermostat(const double *acc, const double *qacc, double *axis, int64_t Nc, double m, double kT,
                                                       uint64_t seed, uint64_t step, bool fixed, const double *esum, const double *eq)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= Nc) return;
    f64x4 s = ld256(acc + 4 * c);
    s.x = acc_value(s.x, fixed); s.y = acc_value(s.y, fixed); s.z = acc_value(s.z, fixed); s.w = acc_count(s.w, fixed);
    int n = (int)s.w;
    // kinetic energy, momentum and mass of the cell's particles: the solvent's, plus the embedded beads' (reading A28)
    double q2 = m * acc_value(qacc[c], fixed), Px = m * s.x, Py = m * s.y, Pz = m * s.z, M = m * s.w;
    if (esum) {
        const f64x4 e = ld256(esum + 4 * c);
        Px += e.x; Py += e.y; Pz += e.z; M += e.w;
        q2 += eq[2 * c];
        n += (int)eq[2 * c + 1];
    }
    double xi = 1.0;
    if (n >= 2) {
        // E_rel = KE - M_c u^2 / 2 (A12) cancels when the cell drifts much faster than it is warm: below 1e-9 of the cell's
        // kinetic energy the difference is rounding noise of the fp64 sums, and the cell is left alone like E_k = 0 (A26)
        const double erel = 0.5 * (q2 - (Px * Px + Py * Py + Pz * Pz) / M);
        const double ehat = draw_cell_energy(seed, step, (uint32_t)c, n, kT);
        if (erel > 1e-9 * 0.5 * q2) xi = sqrt(ehat / erel);
    }
    axis[4 * c + 3] = xi;
}

// Largest cell occupancy of a bin (mpcd_get_stats), from the counts in the accumulator set.
__global__ void __launch_bounds__(256) cell_max_occupancy(const double *acc, int64_t Nc, int *out, bool fixed)
{
    int nmax = 0;
    for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < Nc; c += (int64_t)gridDim.x * blockDim.x) {
        const int n = (int)acc_count(acc[4 * c + 3], fixed);
        nmax = n > nmax ? n : nmax;
    }
    nmax = __reduce_max_sync(0xffffffffu, nmax);
    if ((threadIdx.x & 31) == 0 && nmax > 0) atomicMax(out, nmax);
}

// a9. Net momentum, kinetic energy, pooled temperature by device-wide reduction.
// out = {sum Sx, sum Sy, sum Sz, sum Q, sum E_rel over N_c >= 2, sum 1.5 (N_c - 1)}
__global__ void __launch_bounds__(256) cell_thermo(const double *acc, const double *qacc, int64_t Nc, double m, double *out, bool fixed)
{
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < Nc; c += (int64_t)gridDim.x * blockDim.x) {
        double2 s0 = reinterpret_cast<const double2 *>(acc + 4 * c)[0];
        double2 s1 = reinterpret_cast<const double2 *>(acc + 4 * c)[1];
        s0.x = acc_value(s0.x, fixed); s0.y = acc_value(s0.y, fixed); s1.x = acc_value(s1.x, fixed); s1.y = acc_count(s1.y, fixed);
        const double q = acc_value(qacc[c], fixed), dn = s1.y;
        v[0] += s0.x; v[1] += s0.y; v[2] += s1.x; v[3] += q;
        if (dn >= 2.0) {
            v[4] += 0.5 * m * (q - (s0.x * s0.x + s0.y * s0.y + s1.x * s1.x) / dn);
            v[5] += 1.5 * (dn - 1.0);
        }
    }
    block_sum_to_global<6>(v, out);
}

// Unpack the cell arrays for mpcd_get_cells (SoA outputs on the device, copied by the host): u = S / N_c
// (PAPER.md:122), the cell temperature kT_c = 2 E_rel / (3 (N_c - 1)), E_rel = KE - M_c u^2 / 2
// (eq. 3; A11, A12).
__global__ void __launch_bounds__(256) cell_unpack(const double *acc, const double *qacc, const double *axis, int64_t Nc, double m, bool fixed,
                                                   int32_t *count, double *sumv3, double *ke, double *u3, double *axis3, double *kTc)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= Nc) return;
    const double dn = acc_count(acc[4 * c + 3], fixed);
    const double S[3] = {acc_value(acc[4 * c], fixed), acc_value(acc[4 * c + 1], fixed), acc_value(acc[4 * c + 2], fixed)};
    const double qc = acc_value(qacc[c], fixed);
    double u[3] = {0, 0, 0};
    if (dn > 0.0) { u[0] = S[0] / dn; u[1] = S[1] / dn; u[2] = S[2] / dn; }
    if (count) count[c] = (int32_t)dn;
    if (sumv3) { sumv3[3 * c] = S[0]; sumv3[3 * c + 1] = S[1]; sumv3[3 * c + 2] = S[2]; }
    if (ke) ke[c] = 0.5 * m * qc;
    if (u3) { u3[3 * c] = u[0]; u3[3 * c + 1] = u[1]; u3[3 * c + 2] = u[2]; }
    if (axis3) { axis3[3 * c] = axis[4 * c]; axis3[3 * c + 1] = axis[4 * c + 1]; axis3[3 * c + 2] = axis[4 * c + 2]; }
    if (kTc) {
        double kT = 0.0;
        if (dn >= 2.0) {
            const double erel = 0.5 * m * (qc - dn * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]));
            kT = 2.0 * erel / (3.0 * (dn - 1.0));
        }
        kTc[c] = kT;
    }
}

// ---------------------------------------------------------------------------------------
// a8. Sort by cell as a counting sort on the counts the binning already
// produced: exclusive scan of cnt -> cell_start, then scatter every particle to
// cell_start[c] + (atomic slot) in the duplicate buffers ("duplicate array").
// ---------------------------------------------------------------------------------------
constexpr int kScanThreads = 256, kScanItems = 16, kScanTile = kScanThreads * kScanItems;

// The scan runs over SORT KEYS (mpcd_device.cuh: the cell index, or the brick-major key); count of a key = count of its
// cell, 0 for a hole.  cell_start stays indexed by the cell; brick_start[b] (brick-major order only) = first slot of
// brick b, brick_start[number of bricks] = N.
__device__ __forceinline__ int key_count(const double *acc, int64_t key, const BrickGrid &g, bool fixed, int64_t &cell)
{
    cell = key < g.nkeys ? key_to_cell(key, g) : -1;
    return cell >= 0 ? (int)acc_count(acc[4 * cell + 3], fixed) : 0;
}

__global__ void __launch_bounds__(kScanThreads) scan_tile_sums(const double *acc, const BrickGrid g, int32_t *tile_sum, bool fixed)
{
    __shared__ int sm[kScanThreads / 32];
    const int64_t base = (int64_t)blockIdx.x * kScanTile;
    int s = 0;
    for (int k = 0; k < kScanItems; ++k) {
        int64_t c;
        s += key_count(acc, base + (int64_t)k * kScanThreads + threadIdx.x, g, fixed, c);
    }
    s = __reduce_add_sync(0xffffffffu, s);
    if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < kScanThreads / 32; ++w) t += sm[w];
        tile_sum[blockIdx.x] = t;
    }
}

// single block: exclusive scan of the tile sums in place
__global__ void __launch_bounds__(1024) scan_tile_offsets(int32_t *tile_sum, int ntiles)
{
    __shared__ int sm[1024];
    __shared__ int carry;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int base = 0; base < ntiles; base += 1024) {
        const int idx = base + threadIdx.x;
        const int x = idx < ntiles ? tile_sum[idx] : 0;
        sm[threadIdx.x] = x;
        __syncthreads();
        for (int o = 1; o < 1024; o <<= 1) {
            const int y = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
            __syncthreads();
            sm[threadIdx.x] += y;
            __syncthreads();
        }
        const int incl = sm[threadIdx.x];
        if (idx < ntiles) tile_sum[idx] = carry + incl - x;
        __syncthreads();
        if (threadIdx.x == 1023) carry += incl;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kScanThreads) scan_cells(const double *acc, const BrickGrid g, const int32_t *tile_off, int32_t *cell_start,
                                                           int32_t *brick_start, bool fixed)
{
    // thread t owns kScanItems consecutive keys of the tile
    __shared__ int sm[kScanThreads];
    const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    int x[kScanItems];
    int64_t cell[kScanItems];
    int s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { x[k] = key_count(acc, base + k, g, fixed, cell[k]); s += x[k]; }
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int o = 1; o < kScanThreads; o <<= 1) {
        const int y = threadIdx.x >= o ? sm[threadIdx.x - o] : 0;
        __syncthreads();
        sm[threadIdx.x] += y;
        __syncthreads();
    }
    int run = tile_off[blockIdx.x] + sm[threadIdx.x] - s;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) {
        if (cell[k] >= 0) cell_start[cell[k]] = run;
        if (g.on && base + k < g.nkeys && (base + k) % kBV == 0) brick_start[(base + k) / kBV] = run;
        run += x[k];
        if (g.on && base + k == g.nkeys - 1) brick_start[g.nkeys / kBV] = run;
    }
}

template <typename T>
__global__ void __launch_bounds__(256) sort_scatter(const PassArgs<T> a /* pos, vel, tag, shift: the current bin */, int32_t *cursor,
                                                    typename Vec4<T>::type *pos2, typename Vec4<T>::type *vel2, uint32_t *tag2)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.N) return;
    const auto p = load4(a.pos + i);
    const auto v = load4(a.vel + i);
    const uint32_t t = a.tag[i];
    const int c = w_to_cell(v.w);
    const int dst = atomicAdd(cursor + c, 1);
    store4(pos2 + dst, p);
    store4(vel2 + dst, v);
    tag2[dst] = t;
}

// ---------------------------------------------------------------------------------------
// Initial condition (A23).
// ---------------------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(256) init_particles(int64_t N, uint64_t seed, double Lx, double Ly, double Lz, double sigma,
                                                      const double *mean /* NULL in pass 1 */, double *vsum,
                                                      typename Vec4<T>::type *pos, typename Vec4<T>::type *vel, uint32_t *tag)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    double g[3] = {0, 0, 0};
    if (i < N) {
        double g0, g1, g2;
        gauss3_from_block(draw(seed, 0, (uint32_t)i, kDomInitVel), g0, g1, g2);
        g[0] = sigma * g0; g[1] = sigma * g1; g[2] = sigma * g2;
    }
    if (mean == nullptr) {
        block_sum_to_global<3>(g, vsum);
        return;
    }
    if (i >= N) return;
    const u32x4 b0 = draw(seed, 0, (uint32_t)i, kDomInitPos), b1 = draw(seed, 1, (uint32_t)i, kDomInitPos);
    const double U[3] = {u01_53(b0.x, b0.y), u01_53(b0.z, b0.w), u01_53(b1.x, b1.y)};
    const double L[3] = {Lx, Ly, Lz};
    T x[3];
#pragma unroll
    for (int d = 0; d < 3; ++d) { x[d] = (T)(U[d] * L[d]); if (x[d] >= (T)L[d]) x[d] = T(0); }
    typename Vec4<T>::type p, v;
    p.x = x[0]; p.y = x[1]; p.z = x[2]; p.w = T(0);
    v.x = (T)(g[0] - mean[0]); v.y = (T)(g[1] - mean[1]); v.z = (T)(g[2] - mean[2]); v.w = T(0);
    store4(pos + i, p);
    store4(vel + i, v);
    tag[i] = (uint32_t)i;
}

__global__ void iota_tags(int64_t N, uint32_t *tag)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < N) tag[i] = (uint32_t)i;
}

__global__ void philox_test_kernel(const uint32_t *ctr4, const uint32_t *key2, uint32_t *out4, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const u32x4 r = philox4x32_10(ctr4[4 * i], ctr4[4 * i + 1], ctr4[4 * i + 2], ctr4[4 * i + 3], key2[2 * i], key2[2 * i + 1]);
    out4[4 * i] = r.x; out4[4 * i + 1] = r.y; out4[4 * i + 2] = r.z; out4[4 * i + 3] = r.w;
}

}  // namespace mpcdk
