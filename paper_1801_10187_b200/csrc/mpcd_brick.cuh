// mpcd_brick.cuh -- the steady-state step kernel with spatial tiles: one CTA per BRICK of collision cells, the cell
// side of the step (gather of the cell means / axes, accumulation of the next step's sums) in shared memory.
//
// Why.  In the round-1 kernel (particle_pass, mpcd_kernels.cuh) a warp is 32 array-consecutive particles of an
// x-fastest cell sort.  After the random grid shift those 32 particles sit in ~17 distinct cells,
// so in-warp aggregation is capped at 2 : 1, every lane gathers two 32-byte cell sectors from L2 and every second lane
// issues five fp64 REDs: ~122 LSU data-pipe wavefronts per warp, of which only 16 are the particle stream, on a pipe
// that ncu shows at 82-83 %.  Here the sort (the order inside the sort is free, A20)
// orders particles BRICK-major: cells grouped in bricks of kBX x kBY x kBZ cells, bricks x-fastest, cells x-fastest
// inside the brick.  A CTA owns the array segment of one brick.  Between two sorts a particle drifts ~0.1 a per step
// (r.m.s. 0.5 a after 25 steps) and the grid shift moves every cell boundary by the same known vector, so nearly all
// cells its particles touch lie in a WINDOW of (kBX + kH) x (kBY + kH) x (kBZ + kH) cells whose origin follows the
// difference between the step's shift and the shift of the last sort.  Per CTA:
//   1. window build: for every window cell of the step being collided, u = S / N and the axis
//      (PAPER.md:134), from the same global sectors the round-1 kernel gathers, into shared memory (SoA doubles);
//   2. per particle: collide from shared memory (Alg. 1), stream (eq. 1), bin, and add
//      {v, |v|^2, 1} to the window accumulators of the step being binned;
//   3. flush: one fp64 RED per non-empty window cell and value.
// A particle whose cell lies outside the window (it drifted further than the halo) takes the round-1 route, per lane:
// global gather / direct global RED.  So the result never depends on the drift, only the speed does.
//
// Shared-memory accumulation.  sm_100a has native shared-memory atomics for 32-bit integers only: fp64, fp32 and
// 64-bit integer atomicAdd on shared memory compile to ATOMS.CAST.SPIN loops (measured: 108 cycles per warp of 32
// particles for 4 fp64 sums, against 29 for what follows).  The CTA-local partial sums are therefore 64-bit
// fixed-point integers held as two 32-bit limbs: add the low word with ATOMS.ADD, derive the carry from the returned
// old value, add high word + carry.  Integer addition is exact and associative, so the partial sum is the exact sum
// of the quantised values; the scale is 2^48 / unit for velocities and 2^44 / unit^2 for |v|^2, unit = the power of
// two >= sqrt(kT/m): an fp32 velocity is represented exactly down to 2^-24 unit, an fp64 one is rounded at 2^-49 unit
// (the resolution of a double near 8 unit is 2^-50 unit).  A velocity component >= 8 unit does not fit the headroom of
// kFlushLimit additions and takes the direct global route.  With opt.deterministic the quantisation is the library's
// global one (2^40, mpcd_device.cuh) and the flush is an integer RED, so trajectories stay bit-identical whichever
// kernel processed a particle.
#pragma once
#include "mpcd_kernels.cuh"

namespace mpcdk {

#ifndef MPCD_BRICK_THREADS
#define MPCD_BRICK_THREADS 128
#endif
#ifndef MPCD_BRICK_MINBLOCKS
#define MPCD_BRICK_MINBLOCKS 8
#endif
constexpr int kBrickThreads = MPCD_BRICK_THREADS;
constexpr int kFlushLimit = 2048;      // additions per window cell between two flushes that the fixed-point headroom allows

struct BrickArgs {
    const int32_t *brick_start;    // first array slot of every brick's segment, nbricks + 1 entries
    int32_t nb[3];
    int32_t og[3], oa[3];          // window origin minus the brick's first cell, per axis: step collided / step binned
    Div31 div_nx, div_nxy;
    double sv, inv_sv, sq, inv_sq; // fixed-point scales of the shared-memory partial sums (velocity, |v|^2) and their inverses
    double vmax;                   // |v_d| below this fits the headroom
};

// x += v on a 64-bit integer held as two 32-bit words in shared memory: native ATOMS.ADD on the low word, carry from
// the returned old value, native ATOMS.ADD of high word + carry.
__device__ __forceinline__ void smem_add64(unsigned *lo, unsigned *hi, long long v)
{
    const unsigned vl = (unsigned)(unsigned long long)v, vh = (unsigned)((unsigned long long)v >> 32);
    const unsigned old = atomicAdd(lo, vl);
    atomicAdd(hi, vh + ((unsigned)(old + vl) < old ? 1u : 0u));
}

__device__ __forceinline__ int pmod(int v, int n) { int r = v % n; return r < 0 ? r + n : r; }

template <typename T, unsigned F>
__global__ void __launch_bounds__(kBrickThreads, MPCD_BRICK_MINBLOCKS) brick_pass(const PassArgs<T> a, const BrickArgs g)
{
    using V4 = typename Vec4<T>::type;
    static_assert((F & kSRD) && (F & kStream) && (F & kBin), "the brick kernel is the fused steady-state SRD step");
    constexpr bool kE = (F & kEnergy) != 0, kFx = (F & kFixed) != 0, kTh = (F & kThermo) != 0, kEm = (F & kEmbedded) != 0, kSo = (F & kSortOut) != 0;
    constexpr int NV = kE ? 4 : 3;
    using Ops = AccOps<typename std::conditional<kFx, long long, double>::type>;
    __shared__ double sU[3][kW];                        // window of the step collided: mean velocity
    __shared__ double sA[kTh ? 4 : 3][kW];              // ... axis (and the thermostat's xi)
    __shared__ unsigned sLo[NV][kW], sHi[NV][kW], sCnt[kW];   // window of the step binned: fixed-point partial sums
    const int tid = threadIdx.x;
    const int b = blockIdx.x;
    const int lo = g.brick_start[b], hi = g.brick_start[b + 1];
    if (lo >= hi) return;                               // empty brick
    const int n0 = a.n[0], n1 = a.n[1], n2 = a.n[2];
    const int bx = b % g.nb[0], by = (b / g.nb[0]) % g.nb[1], bz = b / (g.nb[0] * g.nb[1]);
    const int gx0 = pmod(bx * kBX + g.og[0], n0), gy0 = pmod(by * kBY + g.og[1], n1), gz0 = pmod(bz * kBZ + g.og[2], n2);
    const int ax0 = pmod(bx * kBX + g.oa[0], n0), ay0 = pmod(by * kBY + g.oa[1], n1), az0 = pmod(bz * kBZ + g.oa[2], n2);

    // 1. window build
    for (int w = tid; w < kW; w += kBrickThreads) {
        const int lx = w % kWX, ly = (w / kWX) % kWY, lz = w / (kWX * kWY);
        int cx = gx0 + lx, cy = gy0 + ly, cz = gz0 + lz;
        while (cx >= n0) cx -= n0;
        while (cy >= n1) cy -= n1;
        while (cz >= n2) cz -= n2;
        const size_t c = (size_t)cx + (size_t)n0 * ((size_t)cy + (size_t)n1 * (size_t)cz);
        f64x4 s = ld256_nc(a.sums + 4 * c);
        const f64x4 n = ld256_nc(a.axis + 4 * c);
        if (kFx) { s.x = acc_value(s.x, true); s.y = acc_value(s.y, true); s.z = acc_value(s.z, true); s.w = acc_count(s.w, true); }
        double ux = 0.0, uy = 0.0, uz = 0.0;
        if (kEm) {
            const f64x4 e = ld256_nc(a.esum + 4 * c);
            if (a.mass * s.w + e.w > 0.0) embedded_mean(s, e, a.mass, ux, uy, uz);
        } else if (s.w > 0.0) {
            const double inv = __drcp_rn(s.w);
            ux = __dmul_rn(s.x, inv); uy = __dmul_rn(s.y, inv); uz = __dmul_rn(s.z, inv);
        }
        sU[0][w] = ux; sU[1][w] = uy; sU[2][w] = uz;
        sA[0][w] = n.x; sA[1][w] = n.y; sA[2][w] = n.z;
        if (kTh) sA[kTh ? 3 : 0][w] = n.w;
#pragma unroll
        for (int k = 0; k < NV; ++k) { sLo[k][w] = 0u; sHi[k][w] = 0u; }
        sCnt[w] = 0u;
    }
    __syncthreads();

    // 3. flush: the window's partial sums to the global accumulators (also used inside the loop when a brick holds more
    // particles than the fixed-point headroom allows)
    auto flush = [&]() {
        for (int idx = tid; idx < 4 * kW; idx += kBrickThreads) {      // 4 adjacent lanes = the 4 adjacent doubles {Sx, Sy, Sz, N} of one cell
            const int w = idx >> 2, k = idx & 3;
            const unsigned cnt = sCnt[w];
            if (cnt == 0u) continue;
            const int lx = w % kWX, ly = (w / kWX) % kWY, lz = w / (kWX * kWY);
            int cx = ax0 + lx, cy = ay0 + ly, cz = az0 + lz;
            while (cx >= n0) cx -= n0;
            while (cy >= n1) cy -= n1;
            while (cz >= n2) cz -= n2;
            const size_t c = (size_t)cx + (size_t)n0 * ((size_t)cy + (size_t)n1 * (size_t)cz);
            if (k < 3) {
                const long long x = (long long)(((unsigned long long)sHi[k][w] << 32) | sLo[k][w]);
                Ops::red(a.acc + 4 * c + k, kFx ? fixed_bits(x) : (double)x * g.inv_sv);
            } else {
                Ops::red(a.acc + 4 * c + 3, Ops::stage(Ops::count((int)cnt)));
                if (kE) {
                    const long long x = (long long)(((unsigned long long)sHi[NV - 1][w] << 32) | sLo[NV - 1][w]);
                    Ops::red(a.qacc + c, kFx ? fixed_bits(x) : (double)x * g.inv_sq);
                }
            }
        }
    };

    // 2. the particles of this brick's segment
    const uint32_t nxy = (uint32_t)n0 * (uint32_t)n1;
    int since = 0;
    for (int base = lo; base < hi; base += kBrickThreads) {
        if (since + kBrickThreads > kFlushLimit) {
            __syncthreads();
            flush();
            __syncthreads();
            for (int w = tid; w < kW; w += kBrickThreads) {
#pragma unroll
                for (int k = 0; k < NV; ++k) { sLo[k][w] = 0u; sHi[k][w] = 0u; }
                sCnt[w] = 0u;
            }
            __syncthreads();
            since = 0;
        }
        since += kBrickThreads;
        const int i = base + tid;
        const bool valid = i < hi;
        const int il = valid ? i : hi - 1;               // lanes past the end work on a copy of the last particle and store nothing
        V4 v = load4(a.vel + il);
        V4 p = load4(a.pos + il);
        uint32_t tag = 0;
        if (kSo) tag = a.tag[il];
        const int c = w_to_cell(v.w);                    // cell of the step being collided
        int64_t o = i;
        if (kSo && valid) o = atomicAdd(a.cursor + c, 1);
        {
            const uint32_t iz = div31((uint32_t)c, g.div_nxy), r = (uint32_t)c - iz * nxy;
            const uint32_t iy = div31(r, g.div_nx), ix = r - iy * (uint32_t)n0;
            int lx = (int)ix - gx0, ly = (int)iy - gy0, lz = (int)iz - gz0;
            if (lx < 0) lx += n0;
            if (ly < 0) ly += n1;
            if (lz < 0) lz += n2;
            double ux, uy, uz, nx, ny, nz, xi = 1.0;
            if (lx < kWX && ly < kWY && lz < kWZ) {
                const int w = lx + kWX * (ly + kWY * lz);
                ux = sU[0][w]; uy = sU[1][w]; uz = sU[2][w];
                nx = sA[0][w]; ny = sA[1][w]; nz = sA[2][w];
                if (kTh) xi = sA[kTh ? 3 : 0][w];
            } else {                                     // drifted out of the window: the round-1 gather
                f64x4 s = ld256_nc(a.sums + 4 * (size_t)c);
                const f64x4 n = ld256_nc(a.axis + 4 * (size_t)c);
                if (kFx) { s.x = acc_value(s.x, true); s.y = acc_value(s.y, true); s.z = acc_value(s.z, true); s.w = acc_count(s.w, true); }
                if (kEm) {
                    embedded_mean(s, ld256_nc(a.esum + 4 * (size_t)c), a.mass, ux, uy, uz);
                } else {
                    const double inv = __drcp_rn(s.w);
                    ux = __dmul_rn(s.x, inv); uy = __dmul_rn(s.y, inv); uz = __dmul_rn(s.z, inv);
                }
                nx = n.x; ny = n.y; nz = n.z;
                if (kTh) xi = n.w;
            }
            double ox, oy, oz;
            srd_rotate((double)v.x, (double)v.y, (double)v.z, ux, uy, uz, nx, ny, nz, xi, a.cos_a, a.sin_a, ox, oy, oz);
            v.x = (T)ox; v.y = (T)oy; v.z = (T)oz;
        }
        p.x = stream_wrap<T>(p.x, v.x, a.dt, a.L[0]);
        p.y = stream_wrap<T>(p.y, v.y, a.dt, a.L[1]);
        p.z = stream_wrap<T>(p.z, v.z, a.dt, a.L[2]);
        if (valid) store4((kSo ? a.pos_out : a.pos) + o, p);
        const int jx = bin_axis<T>(p.x, a.shift[0], a.inv_a, n0);
        const int jy = bin_axis<T>(p.y, a.shift[1], a.inv_a, n1);
        const int jz = bin_axis<T>(p.z, a.shift[2], a.inv_a, n2);
        const int cn = jx + n0 * (jy + n1 * jz);         // cell of the step being binned
        v.w = cell_to_w(cn, T(0));
        if (valid) {
            store4((kSo ? a.vel_out : a.vel) + o, v);
            if (kSo) a.tag_out[o] = tag;
            const double dx = (double)v.x, dy = (double)v.y, dz = (double)v.z;
            const double q = kE ? sq_norm(dx, dy, dz) : 0.0;
            int lx = jx - ax0, ly = jy - ay0, lz = jz - az0;
            if (lx < 0) lx += n0;
            if (ly < 0) ly += n1;
            if (lz < 0) lz += n2;
            const bool fits = kFx || (fabs(dx) < g.vmax && fabs(dy) < g.vmax && fabs(dz) < g.vmax);
            if (lx < kWX && ly < kWY && lz < kWZ && fits) {
                const int w = lx + kWX * (ly + kWY * lz);
                smem_add64(&sLo[0][w], &sHi[0][w], kFx ? to_fixed(dx) : __double2ll_rn(dx * g.sv));
                smem_add64(&sLo[1][w], &sHi[1][w], kFx ? to_fixed(dy) : __double2ll_rn(dy * g.sv));
                smem_add64(&sLo[2][w], &sHi[2][w], kFx ? to_fixed(dz) : __double2ll_rn(dz * g.sv));
                if (kE) smem_add64(&sLo[NV - 1][w], &sHi[NV - 1][w], kFx ? to_fixed(q) : __double2ll_rn(q * g.sq));
                atomicAdd(&sCnt[w], 1u);
            } else {                                     // outside the window (or too fast for the headroom): straight to the global sums
                double *s = a.acc + 4 * (size_t)cn;
                Ops::red(s, Ops::stage(Ops::from(dx)));
                Ops::red(s + 1, Ops::stage(Ops::from(dy)));
                Ops::red(s + 2, Ops::stage(Ops::from(dz)));
                Ops::red(s + 3, Ops::stage(Ops::count(1)));
                if (kE) Ops::red(a.qacc + cn, Ops::stage(Ops::from(q)));
            }
        }
    }
    __syncthreads();
    flush();
}

}  // namespace mpcdk
