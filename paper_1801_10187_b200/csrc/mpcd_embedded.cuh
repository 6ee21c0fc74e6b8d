// mpcd_embedded.cuh -- embedded solute (BASELINE config 5): MD beads of
// linear harmonic chains that take part in the SRD collision.
//
// Beads are few (config 5: 50 000 against 5 000 000 solvent particles), so they are kept in double whatever the
// solvent's storage precision (reading A27) and handled by three small kernels of their own; the solvent's fused
// pass only learns to add the beads' momentum and mass to its cell mean (flag kEmbedded in mpcd_kernels.cuh).
//   pos[i] = {x, y, z, mass}        vel[i] = {vx, vy, vz, cell of the last binning (as bits)}
//   esum[c] = {sum m v (3), sum m} over the beads of cell c: one 32-byte sector, by step parity like the solvent sums
//   eq[c]   = {sum m |v|^2, number of beads} of cell c (only with the cell thermostat, reading A28: the cell's kinetic
//             energy and its number of particles count the beads)
#pragma once
#include "mpcd_device.cuh"

namespace mpcdk {

constexpr int kEmbThreads = 128;
constexpr int kMaxChainLen = 512;       // one block integrates one chain with its state in shared memory (80 B per bead)

__device__ __forceinline__ double4 ld_d4(const double4 *p)
{
    const f64x4 a = ld256(reinterpret_cast<const double *>(p));
    return double4{a.x, a.y, a.z, a.w};
}
__device__ __forceinline__ void st_d4(double4 *p, double4 v) { st256(reinterpret_cast<double *>(p), v.x, v.y, v.z, v.w); }

// Harmonic bond U = k (r - r0)^2 / 2 between beads at xa and xb (minimum image): g such that the force on b is g d and
// the force on a is -g d, d = xb - xa.
__device__ __forceinline__ void bond(const double *xa, const double *xb, const double (&L)[3], double k, double r0, double (&d)[3], double &g)
{
    double r2 = 0.0;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        d[a] = xb[a] - xa[a];
        d[a] -= L[a] * floor(d[a] / L[a] + 0.5);
        r2 += d[a] * d[a];
    }
    const double r = sqrt(r2);
    g = r > 0.0 ? -k * (r - r0) / r : 0.0;
}

struct MdArgs {
    double4 *pos, *vel;
    int32_t chain_len, nsub;
    double k, r0, dt, L[3];
};

struct EmbArgs {
    double4 *pos, *vel;
    int64_t nb;
    const double *sums, *esum, *axis;    // cell arrays of the step being collided
    double *eacc;                        // bead accumulators of the step being binned
    double *eqacc;                       // ... {sum m |v|^2, count} (thermostat only, else NULL)
    int32_t thermo;                      // the rotation scales the relative velocity by the cell's xi (4th word of the axis sector)
    int32_t n[3];
    double shift[3], inv_a, mass_solvent, cos_a, sin_a;
};

// Mass-weighted mean velocity of a cell holding solvent sums s = {S, N} and bead sums e = {P, M} (A10).
__device__ __forceinline__ void embedded_mean(const f64x4 &s, const f64x4 &e, double m, double &ux, double &uy, double &uz)
{
    const double inv = __drcp_rn(__fma_rn(m, s.w, e.w));     // contractions spelled out: every kernel forms the same bits
    ux = __dmul_rn(__fma_rn(m, s.x, e.x), inv); uy = __dmul_rn(__fma_rn(m, s.y, e.y), inv); uz = __dmul_rn(__fma_rn(m, s.z, e.z), inv);
}

// The bead kernel, one block per chain with the chain's state in shared memory ([x, v, f: 3 doubles each][mass] per
// bead = 80 B), any combination of:
//   kEmbRotate  SRD rotation of the beads (eq. 2, Alg. 1) about their cell's axis, relative to the mass-weighted mean
//   kEmbMd      velocity Verlet between two collisions, nsub steps of length dt
//   kEmbBinAcc  bin the beads under the step's grid shift (the solvent's expression, in double; A6) and add their
//               momentum and mass to their cells ("including the solute particles in ... cell property
//               calculation")
// Inside mpcd_step all three are ONE launch (config 5 is half launch-bound: 5 M solvent particles take 0.12 ms per
// step): collide with the complete sums of step t, MD over the next interval, bin under the shift of step t + 1.  The
// unfused ABI calls launch the single-flag instantiations.
enum : unsigned { kEmbRotate = 1u, kEmbMd = 2u, kEmbBinAcc = 4u };

template <unsigned G>
__global__ void __launch_bounds__(kEmbThreads) emb_step(const MdArgs a, const EmbArgs e)
{
    extern __shared__ double sm[];
    const int n = a.chain_len;
    double *sx = sm, *sv = sm + 3 * n, *sf = sm + 6 * n, *smass = sm + 9 * n;
    const int64_t base = (int64_t)blockIdx.x * n;
    const double L[3] = {a.L[0], a.L[1], a.L[2]};
    for (int j = threadIdx.x; j < n; j += kEmbThreads) {
        const double4 p = ld_d4(a.pos + base + j);
        double4 v = ld_d4(a.vel + base + j);
        if (G & kEmbRotate) {
            const size_t c = (size_t)__double_as_longlong(v.w);
            const f64x4 s = ld256(e.sums + 4 * c), b = ld256(e.esum + 4 * c), ax = ld256(e.axis + 4 * c);
            double ux, uy, uz;
            embedded_mean(s, b, e.mass_solvent, ux, uy, uz);
            srd_rotate(v.x, v.y, v.z, ux, uy, uz, ax.x, ax.y, ax.z, e.thermo ? ax.w : 1.0, e.cos_a, e.sin_a, v.x, v.y, v.z);
        }
        sx[3 * j] = p.x; sx[3 * j + 1] = p.y; sx[3 * j + 2] = p.z; smass[j] = p.w;
        sv[3 * j] = v.x; sv[3 * j + 1] = v.y; sv[3 * j + 2] = v.z;
    }
    __syncthreads();
    if (G & kEmbMd) {
        auto forces = [&]() {
            for (int j = threadIdx.x; j < n; j += kEmbThreads) {
                double d[3], g, fx = 0.0, fy = 0.0, fz = 0.0;
                if (j > 0) { bond(sx + 3 * (j - 1), sx + 3 * j, L, a.k, a.r0, d, g); fx = g * d[0]; fy = g * d[1]; fz = g * d[2]; }
                if (j + 1 < n) { bond(sx + 3 * j, sx + 3 * (j + 1), L, a.k, a.r0, d, g); fx -= g * d[0]; fy -= g * d[1]; fz -= g * d[2]; }
                sf[3 * j] = fx; sf[3 * j + 1] = fy; sf[3 * j + 2] = fz;
            }
        };
        forces();
        for (int s = 0; s < a.nsub; ++s) {
            __syncthreads();
            for (int j = threadIdx.x; j < n; j += kEmbThreads) {
                const double h = 0.5 * a.dt / smass[j];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    sv[3 * j + c] += h * sf[3 * j + c];
                    double x = sx[3 * j + c] + sv[3 * j + c] * a.dt;
                    if (x < 0.0) x += L[c];
                    if (x >= L[c]) x -= L[c];
                    sx[3 * j + c] = x;
                }
            }
            __syncthreads();
            forces();
            for (int j = threadIdx.x; j < n; j += kEmbThreads) {
                const double h = 0.5 * a.dt / smass[j];
#pragma unroll
                for (int c = 0; c < 3; ++c) sv[3 * j + c] += h * sf[3 * j + c];
            }
        }
    }
    for (int j = threadIdx.x; j < n; j += kEmbThreads) {
        double4 v = ld_d4(a.vel + base + j);             // keeps .w (the cached cell index) unless the beads are re-binned
        v.x = sv[3 * j]; v.y = sv[3 * j + 1]; v.z = sv[3 * j + 2];
        const double4 p = double4{sx[3 * j], sx[3 * j + 1], sx[3 * j + 2], smass[j]};
        if (G & kEmbBinAcc) {
            const int ix = bin_axis<double>(p.x, e.shift[0], e.inv_a, e.n[0]);
            const int iy = bin_axis<double>(p.y, e.shift[1], e.inv_a, e.n[1]);
            const int iz = bin_axis<double>(p.z, e.shift[2], e.inv_a, e.n[2]);
            const int c = ix + e.n[0] * (iy + e.n[1] * iz);
            v.w = __longlong_as_double((long long)c);
            double *q = e.eacc + 4 * (size_t)c;
            atomicAdd(q, p.w * v.x); atomicAdd(q + 1, p.w * v.y); atomicAdd(q + 2, p.w * v.z); atomicAdd(q + 3, p.w);
            if (e.eqacc) { atomicAdd(e.eqacc + 2 * (size_t)c, p.w * sq_norm(v.x, v.y, v.z)); atomicAdd(e.eqacc + 2 * (size_t)c + 1, 1.0); }
        }
        if (G & kEmbMd) st_d4(a.pos + base + j, p);
        st_d4(a.vel + base + j, v);
    }
}

}  // namespace mpcdk
