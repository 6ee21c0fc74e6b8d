// mpcd_kernels.cuh -- the kernels of the MPCD solvent step (sm_100a).
//
// One templated per-particle pass covers every particle-side block of Fig. 1
// and their fusions; compile-time flags select which blocks a launch contains:
//
//   kSRD      a6  SRD collision, Alg. 1 PAPER.md:142-155 (gathers u, axis of the particle's cell)
//   kATApply  a7  Andersen-thermostat update, eq. 4 PAPER.md:54 (regenerates dv from the tag)
//   kStream   a1  eq. 1 PAPER.md:35 + periodic wrap
//   kBin      a3+a4  shifted binning + fp64 cell accumulation
//   kEnergy   a4  also accumulate sum |v|^2 (kinetic energy, eq. 3)
//   kATDraw   a7  draw dv for the (new) step and accumulate its per-cell sum
//
// The steady-state step of mpcd_step is ONE launch with kSRD|kStream|kBin: the collision of
// step t fused with the streaming, binning and accumulation of step t+1, so each particle's
// 36 bytes are read once and written once per step.
#pragma once
#include "mpcd_device.cuh"

namespace mpcdk {

enum : unsigned { kSRD = 1u, kATApply = 2u, kStream = 4u, kBin = 8u, kEnergy = 16u, kATDraw = 32u };

// Per-cell record the collision gathers: 64 bytes, 64-byte aligned (never straddles a line).
struct alignas(64) CellRec {
    double u[3];      // mean velocity
    double r[3];      // SRD: rotation axis.  AT: u - sum(dv)/N_c  (eq. 4 without dv_i)
    double kT;        // cell temperature, 0 if N_c < 2 (A11)
    long long count;  // N_c
};

template <typename T> struct PassArgs {
    typename Vec4<T>::type *pos;
    typename Vec4<T>::type *vel;
    uint32_t *tag;
    int32_t *cell;
    const CellRec *rec;   // results of the step being collided
    double *acc;          // accumulators of the step being binned: {Sx, Sy, Sz, N} per cell
    double *qacc;         // sum |v|^2 per cell (kEnergy)
    double *at_acc;       // {Dx, Dy, Dz, -} per cell (AT second reduction)
    int64_t N;
    int32_t n[3];
    T dt, L[3], shift[3], inv_a;
    double cos_a, sin_a, sigma;
    uint64_t seed, step_collide, step_bin;
};

constexpr int kPassThreads = 256;

template <typename T, unsigned F>
__global__ void __launch_bounds__(kPassThreads) particle_pass(const PassArgs<T> a)
{
    using V4 = typename Vec4<T>::type;
    __shared__ WarpScratch ws[(F & (kBin | kATDraw)) ? kPassThreads / 32 : 1];
    const int64_t i = (int64_t)blockIdx.x * kPassThreads + threadIdx.x;
    const bool valid = i < a.N;
    V4 p = {}, v = {};
    int c = 0;
    uint32_t tag = 0;
    if (valid) {
        if (F & (kStream | kBin)) p = load4(a.pos + i);
        if (F & (kSRD | kStream | kBin)) { if (!(F & kATApply)) v = load4(a.vel + i); }
        if (F & (kSRD | kATApply) || ((F & kATDraw) && !(F & kBin))) c = a.cell[i];
        if (F & (kATApply | kATDraw)) tag = a.tag[i];
    }
    if (F & kSRD) {
        if (valid) {
            // Alg. 1 lines 2-4: gather the cell's mean velocity and axis (3 x 16 B of one 64-B record)
            const double *r = reinterpret_cast<const double *>(a.rec + c);
            const f64x4 r0 = ld256_nc(r);                                    // one full sector
            const double2 r2 = __ldg(reinterpret_cast<const double2 *>(r + 4));
            const double ux = r0.x, uy = r0.y, uz = r0.z, nx = r0.w, ny = r2.x, nz = r2.y;
            const double wx = (double)v.x - ux, wy = (double)v.y - uy, wz = (double)v.z - uz;   // lines 5-6
            const double ndw = nx * wx + ny * wy + nz * wz;                                    // line 7
            const double omc = 1.0 - a.cos_a;
            const double rx = wx * a.cos_a + (ny * wz - nz * wy) * a.sin_a + nx * ndw * omc;
            const double ry = wy * a.cos_a + (nz * wx - nx * wz) * a.sin_a + ny * ndw * omc;
            const double rz = wz * a.cos_a + (nx * wy - ny * wx) * a.sin_a + nz * ndw * omc;
            v.x = (T)(ux + rx); v.y = (T)(uy + ry); v.z = (T)(uz + rz);                          // lines 11-12
            store4(a.vel + i, v);
        }
    }
    if (F & kATApply) {
        if (valid) {
            double g0, g1, g2;
            draw_gauss3(a.seed, a.step_collide, tag, g0, g1, g2);
            const double *r = reinterpret_cast<const double *>(a.rec + c);               // r[] = u - D/N_c
            const double2 r1 = __ldg(reinterpret_cast<const double2 *>(r + 2)), r2 = __ldg(reinterpret_cast<const double2 *>(r + 4));
            v.x = (T)(r1.y + a.sigma * g0); v.y = (T)(r2.x + a.sigma * g1); v.z = (T)(r2.y + a.sigma * g2);
            v.w = T(0);
            store4(a.vel + i, v);
        }
    }
    if (F & kStream) {
        if (valid) {
            p.x = stream_wrap<T>(p.x, v.x, a.dt, a.L[0]);
            p.y = stream_wrap<T>(p.y, v.y, a.dt, a.L[1]);
            p.z = stream_wrap<T>(p.z, v.z, a.dt, a.L[2]);
            store4(a.pos + i, p);
        }
    }
    if (F & kBin) {
        int c2 = -1 - (int)(threadIdx.x & 31);
        if (valid) {
            const int ix = bin_axis<T>(p.x, a.shift[0], a.inv_a, a.n[0]);
            const int iy = bin_axis<T>(p.y, a.shift[1], a.inv_a, a.n[1]);
            const int iz = bin_axis<T>(p.z, a.shift[2], a.inv_a, a.n[2]);
            c2 = ix + a.n[0] * (iy + a.n[1] * iz);                    // A8
            a.cell[i] = c2;
        }
        warp_cell_accumulate<true, (F & kEnergy) != 0>(a.acc, a.qacc, ws[threadIdx.x >> 5], c2, (double)v.x, (double)v.y, (double)v.z);
        c = c2;
    }
    if (F & kATDraw) {
        double g0 = 0, g1 = 0, g2 = 0;
        if (valid) draw_gauss3(a.seed, a.step_bin, tag, g0, g1, g2);
        warp_cell_accumulate<false, false>(a.at_acc, nullptr, ws[threadIdx.x >> 5], valid ? c : -1 - (int)(threadIdx.x & 31),
                                           a.sigma * g0, a.sigma * g1, a.sigma * g2);
    }
}

// ---------------------------------------------------------------------------------------
// a5. Per-cell finalize: u = S / N_c, E_rel = KE - M_c u^2 / 2 (A12), kT_c (A11), the
// random axis or, for AT, u - D / N_c; tracks the largest occupancy
// and zeroes the OTHER accumulator set so the next step can accumulate into it.
// ---------------------------------------------------------------------------------------
struct FinalizeArgs {
    const double *acc; const double *qacc; const double *at_acc;   // this step
    double *acc_next; double *qacc_next; double *at_acc_next;      // zeroed for the next step (may be NULL)
    CellRec *rec;
    int *max_occupancy;
    int64_t Nc;
    double m;
    uint64_t seed, step;
    int at_mode;      // 0: r = axis; 1: r = u - D/N_c
    int have_energy;
};

constexpr int kFinCells = 2;     // cells per thread: all loads are issued before any is used (memory-level parallelism)

__global__ void __launch_bounds__(256, 4) cell_finalize(const FinalizeArgs a)
{
    const int64_t c0 = (int64_t)blockIdx.x * (256 * kFinCells) + threadIdx.x;
    double2 s0[kFinCells], s1[kFinCells], d0[kFinCells], d1[kFinCells];
    double qq[kFinCells];
    int n[kFinCells];
#pragma unroll
    for (int k = 0; k < kFinCells; ++k) {
        const int64_t c = c0 + 256 * k;
        n[k] = 0;
        if (c < a.Nc) {
            s0[k] = reinterpret_cast<const double2 *>(a.acc + 4 * c)[0];
            s1[k] = reinterpret_cast<const double2 *>(a.acc + 4 * c)[1];
            qq[k] = a.have_energy ? a.qacc[c] : 0.0;
            if (a.at_mode) {
                d0[k] = reinterpret_cast<const double2 *>(a.at_acc + 4 * c)[0];
                d1[k] = reinterpret_cast<const double2 *>(a.at_acc + 4 * c)[1];
            }
        }
    }
    int nmax = 0;
#pragma unroll
    for (int k = 0; k < kFinCells; ++k) {
        const int64_t c = c0 + 256 * k;
        if (c >= a.Nc) continue;
        const double dn = s1[k].y;
        n[k] = (int)dn;
        double u[3] = {0, 0, 0}, kT = 0.0;
        if (n[k] > 0) { u[0] = s0[k].x / dn; u[1] = s0[k].y / dn; u[2] = s1[k].x / dn; }
        if (a.have_energy && n[k] >= 2) {
            const double erel = 0.5 * a.m * (qq[k] - dn * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]));
            kT = 2.0 * erel / (3.0 * (double)(n[k] - 1));
        }
        double r[3] = {0, 0, 0};
        if (a.at_mode) {
            if (n[k] > 0) { r[0] = u[0] - d0[k].x / dn; r[1] = u[1] - d0[k].y / dn; r[2] = u[2] - d1[k].x / dn; }
        } else {
            draw_axis(a.seed, a.step, (uint32_t)c, r[0], r[1], r[2]);
        }
        double2 *out = reinterpret_cast<double2 *>(a.rec + c);
        out[0] = double2{u[0], u[1]};
        out[1] = double2{u[2], r[0]};
        out[2] = double2{r[1], r[2]};
        out[3] = double2{kT, __longlong_as_double((long long)n[k])};
        if (a.acc_next) {
            reinterpret_cast<double2 *>(a.acc_next + 4 * c)[0] = double2{0.0, 0.0};
            reinterpret_cast<double2 *>(a.acc_next + 4 * c)[1] = double2{0.0, 0.0};
            if (a.qacc_next) a.qacc_next[c] = 0.0;
        }
        if (a.at_acc_next) {
            reinterpret_cast<double2 *>(a.at_acc_next + 4 * c)[0] = double2{0.0, 0.0};
            reinterpret_cast<double2 *>(a.at_acc_next + 4 * c)[1] = double2{0.0, 0.0};
        }
        nmax = n[k] > nmax ? n[k] : nmax;
    }
    const int wmax = __reduce_max_sync(0xffffffffu, nmax);
    if ((threadIdx.x & 31) == 0 && wmax > 0) atomicMax(a.max_occupancy, wmax);
}

// zero one accumulator set
__global__ void __launch_bounds__(256) cell_zero(double *acc, double *qacc, double *at_acc, int64_t Nc)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= Nc) return;
    if (acc) {
        reinterpret_cast<double2 *>(acc + 4 * c)[0] = double2{0.0, 0.0};
        reinterpret_cast<double2 *>(acc + 4 * c)[1] = double2{0.0, 0.0};
        qacc[c] = 0.0;
    }
    if (at_acc) {
        reinterpret_cast<double2 *>(at_acc + 4 * c)[0] = double2{0.0, 0.0};
        reinterpret_cast<double2 *>(at_acc + 4 * c)[1] = double2{0.0, 0.0};
    }
}

// a9. Net momentum, kinetic energy, pooled temperature by device-wide reduction.
// out = {sum Sx, sum Sy, sum Sz, sum Q, sum E_rel over N_c >= 2, sum 1.5 (N_c - 1)}
__global__ void __launch_bounds__(256) cell_thermo(const double *acc, const double *qacc, int64_t Nc, double m, double *out)
{
    double v[6] = {0, 0, 0, 0, 0, 0};
    for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < Nc; c += (int64_t)gridDim.x * blockDim.x) {
        const double2 s0 = reinterpret_cast<const double2 *>(acc + 4 * c)[0];
        const double2 s1 = reinterpret_cast<const double2 *>(acc + 4 * c)[1];
        const double q = qacc[c], dn = s1.y;
        v[0] += s0.x; v[1] += s0.y; v[2] += s1.x; v[3] += q;
        if (dn >= 2.0) {
            v[4] += 0.5 * m * (q - (s0.x * s0.x + s0.y * s0.y + s1.x * s1.x) / dn);
            v[5] += 1.5 * (dn - 1.0);
        }
    }
    block_sum_to_global<6>(v, out);
}

// Unpack the cell arrays for mpcd_get_cells (SoA outputs on the device, copied by the host).
__global__ void __launch_bounds__(256) cell_unpack(const double *acc, const double *qacc, const CellRec *rec, int64_t Nc, double m,
                                                   int32_t *count, double *sumv3, double *ke, double *u3, double *axis3, double *kTc)
{
    const int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= Nc) return;
    if (count) count[c] = (int32_t)acc[4 * c + 3];
    if (sumv3) { sumv3[3 * c] = acc[4 * c]; sumv3[3 * c + 1] = acc[4 * c + 1]; sumv3[3 * c + 2] = acc[4 * c + 2]; }
    if (ke) ke[c] = 0.5 * m * qacc[c];
    if (u3) { u3[3 * c] = rec[c].u[0]; u3[3 * c + 1] = rec[c].u[1]; u3[3 * c + 2] = rec[c].u[2]; }
    if (axis3) { axis3[3 * c] = rec[c].r[0]; axis3[3 * c + 1] = rec[c].r[1]; axis3[3 * c + 2] = rec[c].r[2]; }
    if (kTc) kTc[c] = rec[c].kT;
}

// ---------------------------------------------------------------------------------------
// a8. Sort by cell as a counting sort on the counts the binning already
// produced: exclusive scan of cnt -> cell_start, then scatter every particle to
// cell_start[c] + (atomic slot) in the duplicate buffers ("duplicate array").
// ---------------------------------------------------------------------------------------
constexpr int kScanThreads = 256, kScanItems = 16, kScanTile = kScanThreads * kScanItems;

__global__ void __launch_bounds__(kScanThreads) scan_tile_sums(const double *acc, int64_t Nc, int32_t *tile_sum)
{
    __shared__ int sm[kScanThreads / 32];
    const int64_t base = (int64_t)blockIdx.x * kScanTile;
    int s = 0;
    for (int k = 0; k < kScanItems; ++k) {
        const int64_t c = base + (int64_t)k * kScanThreads + threadIdx.x;
        if (c < Nc) s += (int)acc[4 * c + 3];
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

__global__ void __launch_bounds__(kScanThreads) scan_cells(const double *acc, int64_t Nc, const int32_t *tile_off, int32_t *cell_start)
{
    // thread t owns kScanItems consecutive cells of the tile
    __shared__ int sm[kScanThreads];
    const int64_t base = (int64_t)blockIdx.x * kScanTile + (int64_t)threadIdx.x * kScanItems;
    int x[kScanItems];
    int s = 0;
#pragma unroll
    for (int k = 0; k < kScanItems; ++k) { x[k] = (base + k < Nc) ? (int)acc[4 * (base + k) + 3] : 0; s += x[k]; }
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
    for (int k = 0; k < kScanItems; ++k) { if (base + k < Nc) cell_start[base + k] = run; run += x[k]; }
}

template <typename T>
__global__ void __launch_bounds__(256) sort_scatter(int64_t N, const typename Vec4<T>::type *pos, const typename Vec4<T>::type *vel,
                                                    const uint32_t *tag, const int32_t *cell, int32_t *cursor,
                                                    typename Vec4<T>::type *pos2, typename Vec4<T>::type *vel2, uint32_t *tag2, int32_t *cell2)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int c = cell[i];
    const auto p = load4(pos + i);
    const auto v = load4(vel + i);
    const uint32_t t = tag[i];
    const int dst = atomicAdd(cursor + c, 1);
    store4(pos2 + dst, p);
    store4(vel2 + dst, v);
    tag2[dst] = t;
    cell2[dst] = c;
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
