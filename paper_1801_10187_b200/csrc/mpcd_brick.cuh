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
// MPCD_BRICK_SUMS = 0 keeps the window read but accumulates like the per-particle kernel (match.any, shuffle tree, transposed
// RED): measured slower than both (DESIGN.md 5.1 probe table), kept as a compile-time probe.
#ifndef MPCD_BRICK_SUMS
#define MPCD_BRICK_SUMS 1
#endif
constexpr bool kWinSums = MPCD_BRICK_SUMS != 0;      // 1: the next step's sums in the shared-memory window; 0: in-warp aggregation + global RED (the per-particle kernel's route)
constexpr int kBrickThreads = MPCD_BRICK_THREADS;
constexpr int kFlushLimit = 2048;      // additions per window cell between two flushes that the fixed-point headroom allows

struct BrickArgs {
    const int32_t *brick_start;    // first array slot of every brick's segment, nbricks + 1 entries
    int32_t nb[3];
    int32_t og[3], oa[3];          // window origin minus the brick's first cell, per axis: step collided / step binned
    Div31 div_nx, div_nxy, div_nbx, div_nbxy;
    double sv, inv_sv, inv_sq;     // fixed-point scale of the shared-memory partial sums of the velocities and the inverse scales (velocity, |v|^2)
    double qrel;                   // scale of |v|^2 over scale of the velocities (a power of two: applied before the lanes rotate their values)
    double vmax;                   // |v_d| below this fits the headroom
};

// x += v on a 64-bit integer held as two 32-bit words in shared memory: native ATOMS.ADD on the low word, carry from
// the returned old value, native ATOMS.ADD of high word + carry.
__device__ __forceinline__ void smem_add64(unsigned *lo, unsigned *hi, long long v)
{
    const unsigned vl = (unsigned)(unsigned long long)v, vh = (unsigned)((unsigned long long)v >> 32);
    const unsigned old = atomicAdd(lo, vl);
    unsigned vhc;                                       // high word + carry of (old + vl)
    asm("{\n\t.reg .u32 t;\n\tadd.cc.u32 t, %1, %2;\n\taddc.u32 %0, %3, 0;\n\t}" : "=r"(vhc) : "r"(old), "r"(vl), "r"(vh));
    atomicAdd(hi, vhc);
}

// v mod n for a v that is at most a few n outside [0, n) (no integer division)
__device__ __forceinline__ int wrap(int v, int n)
{
    while (v < 0) v += n;
    while (v >= n) v -= n;
    return v;
}

// Shared memory of one CTA (dynamic: bricks larger than 4 x 4 x 4 need more than the static 48 KB).
template <unsigned F> struct BrickSmem {
    static constexpr int NV = (F & kEnergy) ? 4 : 3;            // fixed-point sums per cell: Sx, Sy, Sz [, sum |v|^2]
    static constexpr int NA = (F & kThermo) ? 4 : 3;            // axis [, xi]
    static constexpr size_t bytes = kWinSums ? (size_t)kW * (8 * (3 + NA) + 4 * (2 * NV + 2)) : (size_t)kW * 8 * (3 + NA);
};

// Thread -> particle mapping.  A warp's 32 lanes are four QUARTERS of 8 lanes; quarter k of the CTA streams through its
// own contiguous sub-segment of the brick, 8 consecutive particles (one full 128-byte line of float4) per iteration.
// The loads stay whole-line accesses, but the lanes of one ATOMS / LDS instruction now come from four places ~4 cells
// apart instead of 32 consecutive particles of ~3 cells, so fewer lanes of an instruction hit the same window cell
// (same-address shared-memory atomics serialise: 6.3 wavefronts per ATOMS with the consecutive mapping, ncu).
template <typename T, unsigned F>
__global__ void __launch_bounds__(kBrickThreads, MPCD_BRICK_MINBLOCKS) brick_pass(const PassArgs<T> a, const BrickArgs g)
{
    using V4 = typename Vec4<T>::type;
    static_assert((F & kSRD) && (F & kStream) && (F & kBin), "the brick kernel is the fused steady-state SRD step");
    constexpr bool kE = (F & kEnergy) != 0, kFx = (F & kFixed) != 0, kTh = (F & kThermo) != 0, kEm = (F & kEmbedded) != 0, kSo = (F & kSortOut) != 0;
    constexpr int NV = BrickSmem<F>::NV, NA = BrickSmem<F>::NA;
    using Ops = AccOps<typename std::conditional<kFx, long long, double>::type>;
    extern __shared__ __align__(16) unsigned char brick_smem[];
    double (*sU)[kW] = reinterpret_cast<double (*)[kW]>(brick_smem);                 // [3][kW]  window of the step collided: mean velocity
    double (*sA)[kW] = sU + 3;                                                       // [NA][kW] ... axis (and the thermostat's xi)
    unsigned (*sLo)[kW] = reinterpret_cast<unsigned (*)[kW]>(sA + NA);               // [NV][kW] window of the step binned: fixed-point partial sums
    unsigned (*sHi)[kW] = sLo + NV;                                                  // [NV][kW]
    unsigned *sCnt = reinterpret_cast<unsigned *>(sHi + NV);                         // [kW]
    int *sCell = reinterpret_cast<int *>(sCnt + kW);                                 // [kW]     global cell of every slot of that window
    __shared__ WarpScratch wscr[kWinSums ? 1 : kBrickThreads / 32];
    const int tid = threadIdx.x;
    const int b = blockIdx.x;
    const int lo = g.brick_start[b], hi = g.brick_start[b + 1];
    if (lo >= hi) return;                               // empty brick
    const int n0 = a.n[0], n1 = a.n[1], n2 = a.n[2];
    const int bz = (int)div31((uint32_t)b, g.div_nbxy), br = b - bz * g.nb[0] * g.nb[1];
    const int by = (int)div31((uint32_t)br, g.div_nbx), bx = br - by * g.nb[0];
    const int gx0 = wrap(bx * kBX + g.og[0], n0), gy0 = wrap(by * kBY + g.og[1], n1), gz0 = wrap(bz * kBZ + g.og[2], n2);
    const int ax0 = wrap(bx * kBX + g.oa[0], n0), ay0 = wrap(by * kBY + g.oa[1], n1), az0 = wrap(bz * kBZ + g.oa[2], n2);

    // The segment is cut in blocks of 8 particles (one 128-byte line of float4), counted from the line it starts in, and the
    // blocks are dealt to the 16 quarters in contiguous, BALANCED runs: the first nblk mod 16 quarters stream one block more
    // than the others.  All quarters are busy for the same number of iterations but the last, in which the idle quarters are
    // the high ones: they fill whole warps, which skip the body.
    const int a0 = lo & ~7;
    const int nblk = (hi - a0 + 7) >> 3;
    constexpr int kQuarters = kBrickThreads / 8;
    const int mlo = nblk / kQuarters, mrem = nblk - mlo * kQuarters;
    const int m = mlo + (mrem > 0);                      // iterations of the CTA
    const int quarter = tid >> 3;
    const int mine = mlo + (quarter < mrem);             // blocks of this quarter
    int i = a0 + 8 * (quarter * mlo + (quarter < mrem ? quarter : mrem)) + (tid & 7);
    auto clamped = [&](int idx) { return idx < lo ? lo : (idx >= hi ? hi - 1 : idx); };
    V4 vn = load4(a.vel + clamped(i));                  // the first block's loads are in flight while the window is built
    V4 pn = load4(a.pos + clamped(i));

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
        if (kTh) sA[NA - 1][w] = n.w;
        if (kWinSums) {
#pragma unroll
            for (int k = 0; k < NV; ++k) { sLo[k][w] = 0u; sHi[k][w] = 0u; }
            sCnt[w] = 0u;
            cx = ax0 + lx; cy = ay0 + ly; cz = az0 + lz;
            while (cx >= n0) cx -= n0;
            while (cy >= n1) cy -= n1;
            while (cz >= n2) cz -= n2;
            sCell[w] = cx + n0 * (cy + n1 * cz);
        }
    }
    __syncthreads();

    // 3. flush: the window's partial sums to the global accumulators (also used inside the loop when a brick holds more
    // particles than the fixed-point headroom allows)
    auto flush = [&]() {
        for (int idx = tid; idx < 4 * kW; idx += kBrickThreads) {      // 4 adjacent lanes = the 4 adjacent doubles {Sx, Sy, Sz, N} of one cell
            const int w = idx >> 2, k = idx & 3;
            const unsigned cnt = sCnt[w];
            if (cnt == 0u) continue;
            const size_t c = (size_t)sCell[w];
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
    const int rot = (tid & 7) % NV;                      // which value this lane adds first, and where the others go
    const int off0 = rot * kW, off1 = ((rot + 1) % NV) * kW, off2 = ((rot + 2) % NV) * kW, off3 = ((rot + 3) % NV) * kW;
    int since = 0;
    for (int j = 0; j < m; ++j, i += 8) {
        if (kWinSums && since + kBrickThreads > kFlushLimit) {
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
        const bool valid = j < mine && i >= lo && i < hi;   // other lanes work on a copy of a particle of the segment and store nothing
        V4 v = vn, p = pn;
        if (j + 1 < mine) {                              // the next block's loads fly during this block's arithmetic
            vn = load4(a.vel + clamped(i + 8));
            pn = load4(a.pos + clamped(i + 8));
        }
        if (!__any_sync(0xffffffffu, j < mine)) continue;   // a warp whose four quarters are done (last iteration only)
        uint32_t tag = 0;
        if (kSo) tag = a.tag[clamped(i)];
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
                if (kTh) xi = sA[NA - 1][w];
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
                // consume the loaded axis INSIDE this rare branch: a register first read after the branches merge would make
                // every warp wait there on the scoreboard slot these loads share with the prefetch of the next block (ncu:
                // 25 % of all samples on that one instruction)
                nx = __dadd_rn(n.x, 0.0); ny = __dadd_rn(n.y, 0.0); nz = __dadd_rn(n.z, 0.0);
                if (kTh) xi = __dadd_rn(n.w, 0.0);
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
        }
        if constexpr (!kWinSums) {       // the per-particle kernel's accumulation: match.any, shuffle tree, transposed fp64 RED (mpcd_device.cuh)
            warp_cell_accumulate<T, true, kE, kFx>(a.acc, a.qacc, wscr[tid >> 5], valid ? cn : -1 - (tid & 31), v.x, v.y, v.z);
        } else if (valid) {
            const double dx = (double)v.x, dy = (double)v.y, dz = (double)v.z;
            const double q = kE ? sq_norm(dx, dy, dz) : 0.0;
            int lx = jx - ax0, ly = jy - ay0, lz = jz - az0;
            if (lx < 0) lx += n0;
            if (ly < 0) ly += n1;
            if (lz < 0) lz += n2;
            const T vmax = (T)g.vmax;
            const bool fits = kFx || (fabs(v.x) < vmax && fabs(v.y) < vmax && fabs(v.z) < vmax);
            if (lx < kWX && ly < kWY && lz < kWZ && fits) {
                const int w = lx + kWX * (ly + kWY * lz);
                // Lanes of one instruction that share a window cell would serialise on its address (shared-memory atomics do
                // not merge; ncu: 4.8 wavefronts per ATOMS): lane l therefore starts with value (l mod NV), so that in any one
                // ATOMS the lanes of a cell are spread over the NV per-value arrays (3.3).  The rotation is two conditional swaps
                // of the doubles; |v|^2 is first brought to the velocities' scale (a power of two: exact) so that one multiply
                // serves whatever value a slot holds.
                double y0 = dx, y1 = dy, y2 = dz, y3 = kFx ? q : q * g.qrel;
                if (NV == 4) {
                    if (rot & 1) { const double t = y0; y0 = y1; y1 = y2; y2 = y3; y3 = t; }
                    if (rot & 2) { double t = y0; y0 = y2; y2 = t; t = y1; y1 = y3; y3 = t; }
                } else {
                    if (rot >= 1) { const double t = y0; y0 = y1; y1 = y2; y2 = t; }
                    if (rot >= 2) { const double t = y0; y0 = y1; y1 = y2; y2 = t; }
                }
                unsigned *plo = &sLo[0][w], *phi = &sHi[0][w];
                smem_add64(plo + off0, phi + off0, kFx ? to_fixed(y0) : __double2ll_rn(y0 * g.sv));
                smem_add64(plo + off1, phi + off1, kFx ? to_fixed(y1) : __double2ll_rn(y1 * g.sv));
                smem_add64(plo + off2, phi + off2, kFx ? to_fixed(y2) : __double2ll_rn(y2 * g.sv));
                if (NV == 4) smem_add64(plo + off3, phi + off3, kFx ? to_fixed(y3) : __double2ll_rn(y3 * g.sv));
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
    if (kWinSums) {
        __syncthreads();
        flush();
    }
}

}  // namespace mpcdk
