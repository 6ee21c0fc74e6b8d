// mpcd_device.cuh -- device-side building blocks of the MPCD solvent step for sm_100a.
//
// Citations are PAPER.md:<line> (the paper's text) and A<n> (readings in DESIGN.md).
// This file shares nothing with oracle/: the RNG, the uniform conversions and the
// domain constants are restated here.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda_runtime.h>

namespace mpcdk {

// ---------------------------------------------------------------------------------------
// Counter-based RNG: Philox4x32-10 keyed like the paper keys Saru, (cell index | tag,
// timestep, seed) (A24): key = seed, ctr = (index, t_lo, t_hi, domain).
// ---------------------------------------------------------------------------------------
enum : uint32_t { kDomShift = 1u, kDomAxis = 2u, kDomAT = 3u, kDomInitPos = 4u, kDomInitVel = 5u, kDomThermo = 6u };

struct u32x4 { uint32_t x, y, z, w; };

__host__ __device__ __forceinline__ u32x4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                          uint32_t k0, uint32_t k1)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        c1 = (uint32_t)p1; c3 = (uint32_t)p0; c0 = n0; c2 = n2;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    return u32x4{c0, c1, c2, c3};
}

__host__ __device__ __forceinline__ u32x4 draw(uint64_t seed, uint64_t step, uint32_t index, uint32_t domain)
{
    return philox4x32_10(index, (uint32_t)step, (uint32_t)(step >> 32), domain, (uint32_t)seed, (uint32_t)(seed >> 32));
}

// (b + 1/2) 2^-32 in (0,1), exact in binary64
__host__ __device__ __forceinline__ double u01_32(uint32_t b) { return ((double)b + 0.5) * 2.3283064365386962890625e-10; }
// 53-bit uniform in [0,1)
__host__ __device__ __forceinline__ double u01_53(uint32_t lo, uint32_t hi)
{
    return (double)((((uint64_t)hi << 32) | lo) >> 11) * 1.1102230246251565404236316680908203125e-16;
}

// Random unit axis by cylindrical projection (A13): U1 -> z, U2 -> azimuth.
__device__ __forceinline__ void draw_axis(uint64_t seed, uint64_t step, uint32_t cell, double &nx, double &ny, double &nz)
{
    const u32x4 b = draw(seed, step, cell, kDomAxis);
    const double z = 2.0 * u01_53(b.x, b.y) - 1.0;
    double s, c;
    sincospi(2.0 * u01_53(b.z, b.w), &s, &c);
    const double rho = sqrt((1.0 - z) * (1.0 + z));   // sqrt(1 - z^2) without cancellation near the poles
    nx = rho * c; ny = rho * s; nz = z;
}

// The same axis formed per PARTICLE in registers instead of being gathered from the per-cell array ("or
// recomputed per particle in a6"; probe MPCD_AXIS_REG): it depends on (seed, step, cell) only.  The fp64
// model evaluates draw_axis itself (the same bits as the stored axis).  The mixed model evaluates the transcendental part in
// fp32 (reading A13b): z, 1 - z and 1 + z exactly in double from the 53-bit uniform, rho = sqrtf of their product (relative
// error 1e-7, also at the poles), the azimuth from the top 32 of its 53 bits (angle error < 1.5e-9) split into 24 exact
// bits for sincospif + a first-order rotation; then the vector is renormalised in double (|n|^2 - 1 ~ 1e-20, so the
// rotation conserves the cell's energy as exactly as with the stored axis).  The direction differs from the fp64 axis
// by <= ~1.5e-7, i.e. velocities by <= 2 |v - u| 1.5e-7 < 1e-5 sigma.
template <typename T>
__device__ __forceinline__ void axis_in_registers(uint64_t seed, uint64_t step, uint32_t cell, double &nx, double &ny, double &nz)
{
    if (sizeof(T) == 8) { draw_axis(seed, step, cell, nx, ny, nz); return; }
    const u32x4 b = draw(seed, step, cell, kDomAxis);
    const double u = u01_53(b.x, b.y);
    const double z = 2.0 * u - 1.0;
    const float rho = sqrtf((float)((2.0 - 2.0 * u) * (2.0 * u)));                 // (1 - z)(1 + z), the factors exact
    const float hi = (float)(b.w >> 8) * 1.1920928955078125e-7f;                  // 2 U2 = b.w 2^-31 = hi + lo (units of pi): (b.w >> 8) 2^-23 + (b.w & 255) 2^-31
    const float lo = (float)(b.w & 255u) * 4.656612873077392578125e-10f;
    float sh, ch;
    sincospif(hi, &sh, &ch);
    const float d = 3.14159265358979323846f * lo;
    const double x = (double)(rho * fmaf(-d, sh, ch)), y = (double)(rho * fmaf(d, ch, sh));
    const double e = fma(x, x, fma(y, y, fma(z, z, -1.0)));                        // |n|^2 - 1, ~2e-7
    const double inv = fma(e, fma(e, 0.375, -0.5), 1.0);                           // (1 + e)^(-1/2) to O(e^3)
    nx = x * inv; ny = y * inv; nz = z * inv;
}

// Three Gaussians of unit variance by Box-Muller from one Philox block keyed by the particle
// tag (A17, A18); the fourth is discarded.
__device__ __forceinline__ void gauss3_from_block(const u32x4 b, double &g0, double &g1, double &g2)
{
    const double r01 = sqrt(-2.0 * log(u01_32(b.x)));
    const double r23 = sqrt(-2.0 * log(u01_32(b.z)));
    double s, c;
    sincospi(2.0 * u01_32(b.y), &s, &c);
    g0 = r01 * c; g1 = r01 * s;
    g2 = r23 * cospi(2.0 * u01_32(b.w));
}
// The same three Gaussians evaluated in fp32 for the mixed model (A17 allows it as long as the 1e-5 sigma velocity
// parity holds; no fast-math intrinsics): absolute error <= ~1e-6 against the fp64 evaluation, by construction:
//  - radius sqrt(-2 ln U): for U > 1/2 the exact small quantity is w = 1 - U = (2^32 - b - 1/2) 2^-32, so
//    ln U = log1pf(-w) keeps full RELATIVE accuracy where the radius is small; for U <= 1/2, ln U = log1pf(m - 1) - k ln 2
//    with the normalised mantissa m has absolute error ~1e-6 at most while the radius is > 1.17;
//  - angle 2 U1 (in units of pi) = hi + lo with hi the top 24 bits (exact in fp32) and lo < 2^-23 applied as a
//    first-order rotation of sincospif(hi), instead of rounding U1 itself to 24 bits.
__device__ __forceinline__ float bm_radius_f32(uint32_t b)
{
    // One log1pf for both regimes, no divergence: U = m 2^-k with k = clz(b), m in [1/2, 1).  For U > 1/2 (k = 0) the
    // argument m - 1 = -w is formed from the integer 2^32 - 1 - b and is exact; for U <= 1/2 the mantissa m carries a
    // relative rounding of 2^-24, harmless there (|ln U| > 0.69).
    const int k = __clz((int)b);                                            // 0 when the top bit is set; 32 for b = 0
    const float w = ((float)(0xffffffffu - b) + 0.5f) * 2.3283064365386962890625e-10f;
    const float m = ((float)(k < 32 ? b << k : 0u) + ldexpf(0.5f, k)) * 2.3283064365386962890625e-10f;
    const float x = k == 0 ? -w : m - 1.0f;
    const float lnu = fmaf(-(float)k, 0.693147182464599609375f, log1pf(x));
    return sqrtf(-2.0f * lnu);
}
__device__ __forceinline__ void bm_sincos_f32(uint32_t b, float &s, float &c)      // sin, cos of 2 pi (b + 1/2) 2^-32
{
    const float hi = (float)(b >> 8) * 1.1920928955078125e-7f;                     // (b >> 8) 2^-23: exact
    const float lo = ((float)(b & 255u) + 0.5f) * 4.656612873077392578125e-10f;    // ((b & 255) + 1/2) 2^-31: exact
    float sh, ch;
    sincospif(hi, &sh, &ch);
    const float d = 3.14159265358979323846f * lo;
    s = fmaf(d, ch, sh);
    c = fmaf(-d, sh, ch);
}
__device__ __forceinline__ void gauss3_from_block_f32(const u32x4 b, double &g0, double &g1, double &g2)
{
    const float r01 = bm_radius_f32(b.x), r23 = bm_radius_f32(b.z);
    float s1, c1, s3, c3;
    bm_sincos_f32(b.y, s1, c1);
    bm_sincos_f32(b.w, s3, c3);
    g0 = (double)(r01 * c1); g1 = (double)(r01 * s1); g2 = (double)(r23 * c3);
}
// T = the native precision of the model: the fp64 model evaluates the transform in double.
template <typename T>
__device__ __forceinline__ void draw_gauss3(uint64_t seed, uint64_t step, uint32_t tag, double &g0, double &g1, double &g2)
{
    const u32x4 b = draw(seed, step, tag, kDomAT);
    if (sizeof(T) == 4) gauss3_from_block_f32(b, g0, g1, g2);
    else gauss3_from_block(b, g0, g1, g2);
}

// Maxwell-Boltzmann cell thermostat (A26): the relative kinetic energy of a cell of n >= 2
// particles at kT, drawn from Gamma(shape 3 (n - 1) / 2, scale kT) by Marsaglia & Tsang's rejection method with a
// Box-Muller Gaussian; one Philox block per attempt, keyed (seed, step, cell, kDomThermo + 256 * attempt).
__device__ __forceinline__ double draw_cell_energy(uint64_t seed, uint64_t step, uint32_t cell, int n, double kT)
{
    const double k = 1.5 * (double)(n - 1);
    const double d = k - 1.0 / 3.0;
    const double c = 1.0 / sqrt(9.0 * d);
    for (uint32_t attempt = 0;; ++attempt) {
        const u32x4 b = draw(seed, step, cell, kDomThermo + 256u * attempt);
        const double x = sqrt(-2.0 * log(u01_32(b.x))) * cospi(2.0 * u01_32(b.y));
        const double t = 1.0 + c * x;
        const double v = t * t * t;
        if (v > 0.0 && log(u01_32(b.z)) < 0.5 * x * x + d - d * v + d * log(v)) return kT * d * v;
    }
}

// ---------------------------------------------------------------------------------------
// Native-precision arithmetic with explicit rounding: streaming and binning are DEFINED as
// separately rounded operations (A6, A7), so no FMA contraction may happen here.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ float  add_rn(float a, float b)   { return __fadd_rn(a, b); }
__device__ __forceinline__ double add_rn(double a, double b) { return __dadd_rn(a, b); }
__device__ __forceinline__ float  sub_rn(float a, float b)   { return __fsub_rn(a, b); }
__device__ __forceinline__ double sub_rn(double a, double b) { return __dsub_rn(a, b); }
__device__ __forceinline__ float  mul_rn(float a, float b)   { return __fmul_rn(a, b); }
__device__ __forceinline__ double mul_rn(double a, double b) { return __dmul_rn(a, b); }
__device__ __forceinline__ int floor_int(float q)  { return __float2int_rd(q); }
__device__ __forceinline__ int floor_int(double q) { return __double2int_rd(q); }

template <typename T> struct Vec4;
template <> struct Vec4<float>  { using type = float4; };
template <> struct Vec4<double> { using type = double4; };

// 16-byte vector accesses (north_star: "coalesced 16-byte HBM access"); double4 = two of them.
// The particle arrays are streamed once per pass (GBs), the cell arrays are revisited while the
// sweep is in their neighbourhood: particle data is therefore marked evict-first (.cs) so that
// it does not push the cell records / accumulators out of the 126 MB L2.
#ifndef MPCD_CS
#define MPCD_CS 1
#endif
#if MPCD_CS
__device__ __forceinline__ float4 load4(const float4 *p) { return __ldcs(p); }
__device__ __forceinline__ void store4(float4 *p, float4 v) { __stcs(p, v); }
__device__ __forceinline__ double4 load4(const double4 *p)
{
    const double2 a = __ldcs(reinterpret_cast<const double2 *>(p)), b = __ldcs(reinterpret_cast<const double2 *>(p) + 1);
    return double4{a.x, a.y, b.x, b.y};
}
__device__ __forceinline__ void store4(double4 *p, double4 v)
{
    __stcs(reinterpret_cast<double2 *>(p), double2{v.x, v.y});
    __stcs(reinterpret_cast<double2 *>(p) + 1, double2{v.z, v.w});
}
#else
__device__ __forceinline__ float4 load4(const float4 *p) { return *p; }
__device__ __forceinline__ void store4(float4 *p, float4 v) { *p = v; }
__device__ __forceinline__ double4 load4(const double4 *p)
{
    const double2 a = reinterpret_cast<const double2 *>(p)[0], b = reinterpret_cast<const double2 *>(p)[1];
    return double4{a.x, a.y, b.x, b.y};
}
__device__ __forceinline__ void store4(double4 *p, double4 v)
{
    reinterpret_cast<double2 *>(p)[0] = double2{v.x, v.y};
    reinterpret_cast<double2 *>(p)[1] = double2{v.z, v.w};
}
#endif

// 32-byte (one full sector) accesses for the per-cell records: sm_100 has 256-bit LDG/STG.
struct f64x4 { double x, y, z, w; };
__device__ __forceinline__ f64x4 ld256_nc(const double *p)     // read-only path
{
    f64x4 r;
    asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p));
    return r;
}
__device__ __forceinline__ f64x4 ld256(const double *p)
{
    f64x4 r;
    asm volatile("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(r.x), "=d"(r.y), "=d"(r.z), "=d"(r.w) : "l"(p) : "memory");
    return r;
}
__device__ __forceinline__ void st256(double *p, double a, double b, double c, double d)
{
    asm volatile("st.global.v4.f64 [%0], {%1,%2,%3,%4};" :: "l"(p), "d"(a), "d"(b), "d"(c), "d"(d) : "memory");
}

// eq. 1 PAPER.md:35 + periodic wrap (A7): x = fl(x + fl(v dt)); if x < 0: x += L; if x >= L: x -= L.
template <typename T> __device__ __forceinline__ T stream_wrap(T x, T v, T dt, T L)
{
    x = add_rn(x, mul_rn(v, dt));
    if (x < T(0)) x = add_rn(x, L);
    if (x >= L) x = sub_rn(x, L);
    return x;
}

// PAPER.md:110 + A6: i = floor(fl(fl(x + s) * inv_a)), integer periodic wrap.
template <typename T> __device__ __forceinline__ int bin_axis(T x, T s, T inv_a, int n)
{
    int i = floor_int(mul_rn(add_rn(x, s), inv_a));
    if (i < 0) i += n;
    if (i >= n) i -= n;
    return i;
}

// Alg. 1 lines 5-12: v' = u + xi R(alpha, n)(v - u), in double, with the contractions spelled out so
// that every kernel that collides a particle produces the same bits (opt.deterministic relies on it).
__device__ __forceinline__ void srd_rotate(double vx, double vy, double vz, double ux, double uy, double uz, double nx, double ny, double nz,
                                           double xi, double cos_a, double sin_a, double &ox, double &oy, double &oz)
{
    const double wx = vx - ux, wy = vy - uy, wz = vz - uz;                                      // lines 5-6
    const double ndw = __fma_rn(nz, wz, __fma_rn(ny, wy, __dmul_rn(nx, wx)));                   // line 7
    const double omc = 1.0 - cos_a;
    const double cx = __fma_rn(ny, wz, -__dmul_rn(nz, wy)), cy = __fma_rn(nz, wx, -__dmul_rn(nx, wz)), cz = __fma_rn(nx, wy, -__dmul_rn(ny, wx));
    const double rx = __fma_rn(__dmul_rn(nx, ndw), omc, __fma_rn(cx, sin_a, __dmul_rn(wx, cos_a)));
    const double ry = __fma_rn(__dmul_rn(ny, ndw), omc, __fma_rn(cy, sin_a, __dmul_rn(wy, cos_a)));
    const double rz = __fma_rn(__dmul_rn(nz, ndw), omc, __fma_rn(cz, sin_a, __dmul_rn(wz, cos_a)));
    ox = __fma_rn(rx, xi, ux); oy = __fma_rn(ry, xi, uy); oz = __fma_rn(rz, xi, uz);            // lines 8-12
}
__device__ __forceinline__ double sq_norm(double x, double y, double z) { return __fma_rn(z, z, __fma_rn(y, y, __dmul_rn(x, x))); }


// ---------------------------------------------------------------------------------------
// Warp-level machinery of the per-particle pass.
//
// What bounds the pass on a B200 is not HBM bandwidth alone but the SM's L1/LSU data pipe, one
// "wavefront" per cycle per SM (measured with micro-kernels under ncu): a coalesced
// 16-byte-per-lane access costs 4 wavefronts; a per-lane gather costs about 8 + bytes/2 per warp
// instruction whatever the number of distinct cells; a RED costs ~0.75 per leader record per
// instruction; a 32-bit SHFL costs 1.  So the accumulation is done "transposed": lanes that share a
// cell are found with match.any and combined, one leader per distinct cell is compacted into shared
// memory, and then 4 ADJACENT lanes issue the REDs on the 4 ADJACENT doubles of one cell's sector.
// ---------------------------------------------------------------------------------------
constexpr int kStagePitch = 36;    // doubles per staged component row: 4 rows land in disjoint banks for one half-warp
struct alignas(16) WarpScratch {   // per-warp shared memory of the accumulate phase
    double v[4][kStagePitch];      // [component][leader slot]
    int cell[32];                  // cell index of leader slot j
};
struct alignas(16) WarpScratchX : WarpScratch {   // ... with room for a second triple summed over the same groups (kExtra)
    double x[3][kStagePitch];
};

// ---------------------------------------------------------------------------------------
// Per-cell fp64 accumulation.  Layout in HBM: acc[c] = {Sx, Sy, Sz, N}
// (4 doubles = one 32-byte sector; the count N is kept as a double, exact below 2^53) and,
// when the kinetic energy is wanted, q[c] = sum |v|^2 in an array of its own.
// Lanes are first combined by cell inside the warp (match.any + a shuffle tree, ~2.3 particles
// per surviving leader on the benchmark fluid); the first round of the tree moves the particle
// values in their native precision (fp32 in the mixed model: half the shuffles) and upcasts at
// the receiver, as PAPER.md:124 asks ("all reductions are performed with double-precision
// values even if the particle velocities are stored in single precision").
// ---------------------------------------------------------------------------------------
#ifndef MPCD_TREE_ROUNDS
#define MPCD_TREE_ROUNDS 0
#endif
constexpr int kTreeRounds = MPCD_TREE_ROUNDS;   // rounds of the in-warp combining tree before the REDs; 0 = until one lane per cell is left

// Deterministic accumulation (the alternative PAPER.md:124-126 mentions): the cell sums are kept
// as 64-bit fixed-point integers with 40 fractional bits instead of doubles.  Integer addition is associative, so the
// sums -- and with them the whole trajectory -- no longer depend on the order in which warps and atomics happen to
// run.  An fp32 velocity is represented exactly whenever |v| >= 2^-17 (absolute rounding error <= 2^-41 otherwise, as
// for the fp64 value of |v|^2); the range is |sum| < 2^23.  The accumulator words hold the integers' bits.
constexpr double kFixScale = 1099511627776.0;            // 2^40
constexpr double kFixInv = 9.094947017729282379150390625e-13;   // 2^-40
__device__ __forceinline__ long long to_fixed(double x) { return __double2ll_rn(x * kFixScale); }
__device__ __forceinline__ double fixed_bits(long long x) { return __longlong_as_double(x); }
// value of an accumulator word: a double, or (fixed) the bits of a fixed-point integer / (count) of a plain integer
__device__ __forceinline__ double acc_value(double w, bool fixed) { return fixed ? (double)__double_as_longlong(w) * kFixInv : w; }
__device__ __forceinline__ double acc_count(double w, bool fixed) { return fixed ? (double)__double_as_longlong(w) : w; }

// The combining tree and the transposed REDs, on values of type A: double, or long long for the fixed-point sums.
template <typename A> struct AccOps;
template <> struct AccOps<double> {
    static __device__ __forceinline__ double from(double x) { return x; }
    static __device__ __forceinline__ double count(int n) { return (double)n; }
    static __device__ __forceinline__ double stage(double x) { return x; }
    static __device__ __forceinline__ void red(double *p, double staged) { atomicAdd(p, staged); }
};
template <> struct AccOps<long long> {
    static __device__ __forceinline__ long long from(double x) { return to_fixed(x); }
    static __device__ __forceinline__ long long count(int n) { return (long long)n; }
    static __device__ __forceinline__ double stage(long long x) { return fixed_bits(x); }
    static __device__ __forceinline__ void red(double *p, double staged)
    {
        atomicAdd(reinterpret_cast<unsigned long long *>(p), (unsigned long long)__double_as_longlong(staged));
    }
};

// kExtra: a second triple (ex, ey, ez), already double, is summed over the same groups into xacc[c] = {X, Y, Z, -} by the
// same match and the same tree (the AT rule's sum of the thermostat draws), instead of a second pass.
// kMinus: a second NATIVE triple (gx, gy, gz) is subtracted from the first before the summation (the difference of two
// native values is formed in double: exact), while the energy stays that of the first triple: inside mpcd_step the AT rule
// needs only sum(v) - sum(dv) of a cell (eq. 4: v' = (S - D) / N_c + dv), so ONE sum per cell carries both.
template <typename T, bool kCount, bool kEnergy, bool kFixed = false, bool kExtra = false, bool kMinus = false>
__device__ __forceinline__ void warp_cell_accumulate(double *__restrict__ acc, double *__restrict__ qacc,
                                                     typename std::conditional<kExtra, WarpScratchX, WarpScratch>::type &ws,
                                                     int c /* < 0 = inactive lane, unique per lane */, T fx, T fy, T fz,
                                                     double *__restrict__ xacc = nullptr, double ex = 0.0, double ey = 0.0, double ez = 0.0,
                                                     T gx = T(0), T gy = T(0), T gz = T(0))
{
    static_assert(!(kExtra && kFixed), "the second triple is summed in double");
    static_assert(!(kMinus && (kExtra || kFixed)), "the difference is summed in double, alone");
    using A = typename std::conditional<kFixed, long long, double>::type;
    using Ops = AccOps<A>;
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const double dx0 = (double)fx, dy0 = (double)fy, dz0 = (double)fz;
    A vx = Ops::from(kMinus ? dx0 - (double)gx : dx0), vy = Ops::from(kMinus ? dy0 - (double)gy : dy0), vz = Ops::from(kMinus ? dz0 - (double)gz : dz0);
    A q = kEnergy ? Ops::from(sq_norm(dx0, dy0, dz0)) : A(0);
    unsigned peers = __match_any_sync(full, c);
    const int size = __popc(peers);
    const int rank0 = __popc(peers & ((1u << lane) - 1u));
    int rank = rank0, rounds = 0;
    bool alive = true;                                     // not yet folded into a lower-ranked peer
    peers &= (0xfffffffeu << lane);                        // peers above this lane
    if (kTreeRounds == 1 || __any_sync(full, peers != 0u)) {   // round 1: raw particle values, native precision
        const int next = __ffs(peers);                     // 1-based lane of the next peer, 0 = none
        const int src = next ? next - 1 : lane;
        const T tx = __shfl_sync(full, fx, src), ty = __shfl_sync(full, fy, src), tz = __shfl_sync(full, fz, src);
        const T sx = kMinus ? __shfl_sync(full, gx, src) : T(0), sy = kMinus ? __shfl_sync(full, gy, src) : T(0), sz = kMinus ? __shfl_sync(full, gz, src) : T(0);
        alive = !(rank & 1);
        const double ux = kExtra ? __shfl_sync(full, ex, src) : 0.0, uy = kExtra ? __shfl_sync(full, ey, src) : 0.0,
                     uz = kExtra ? __shfl_sync(full, ez, src) : 0.0;
        if (next && alive) {
            const double dx = (double)tx, dy = (double)ty, dz = (double)tz;
            vx += Ops::from(kMinus ? dx - (double)sx : dx); vy += Ops::from(kMinus ? dy - (double)sy : dy); vz += Ops::from(kMinus ? dz - (double)sz : dz);
            if (kEnergy) q += Ops::from(sq_norm(dx, dy, dz));
            if (kExtra) { ex += ux; ey += uy; ez += uz; }
        }
        rounds = 1;
        if (kTreeRounds != 1) {
            peers &= __ballot_sync(full, alive);           // odd-ranked lanes have been absorbed
            rank >>= 1;
        }
    }
    if (kTreeRounds != 1) {
        while ((kTreeRounds == 0 || rounds < kTreeRounds) && __any_sync(full, alive && peers != 0u)) {   // log2(largest group) rounds at most
            const int next = __ffs(peers);
            const int src = next ? next - 1 : lane;
            const A tx = __shfl_sync(full, vx, src), ty = __shfl_sync(full, vy, src), tz = __shfl_sync(full, vz, src);
            const A tq = kEnergy ? __shfl_sync(full, q, src) : A(0);
            const double ux = kExtra ? __shfl_sync(full, ex, src) : 0.0, uy = kExtra ? __shfl_sync(full, ey, src) : 0.0,
                         uz = kExtra ? __shfl_sync(full, ez, src) : 0.0;
            if (next && alive && !(rank & 1)) { vx += tx; vy += ty; vz += tz; q += tq; if (kExtra) { ex += ux; ey += uy; ez += uz; } }
            alive = alive && !(rank & 1);
            peers &= __ballot_sync(full, alive);
            rank >>= 1;
            rounds += 1;
        }
    }
    // a surviving lane holds the sum over the original ranks [rank0, rank0 + 2^rounds) of its group
    const int span = 1 << rounds;
    const int mine = size - rank0 < span ? size - rank0 : span;
    const unsigned leaders = __ballot_sync(full, alive && c >= 0);
    const int nl = __popc(leaders);
    if (alive && c >= 0) {
        const int j = __popc(leaders & ((1u << lane) - 1u));
        ws.v[0][j] = Ops::stage(vx); ws.v[1][j] = Ops::stage(vy); ws.v[2][j] = Ops::stage(vz);
        if (kCount) ws.v[3][j] = Ops::stage(Ops::count(mine));
        if (kEnergy) Ops::red(qacc + c, Ops::stage(q));    // one 8-byte RED per leader, straight from its registers
        if constexpr (kExtra) { ws.x[0][j] = ex; ws.x[1][j] = ey; ws.x[2][j] = ez; }
        ws.cell[j] = c;
    }
    __syncwarp();
    const int comp = lane & 3;                             // 8 leaders per round, 4 lanes x 8 B = one 32-byte sector each
#pragma unroll
    for (int base = 0; base < 32; base += 8) {             // at most 32 leaders; fully unrolled, rounds past nl are predicated off
        if (base >= nl) break;
        const int j = base + (lane >> 2);
        if (j < nl && (kCount || comp < 3)) Ops::red(acc + 4 * (size_t)ws.cell[j] + comp, ws.v[comp][j]);
        if constexpr (kExtra) { if (j < nl && comp < 3) atomicAdd(xacc + 4 * (size_t)ws.cell[j] + comp, ws.x[comp][j]); }
    }
    __syncwarp();
}

// Block-wide sum of k doubles into out[0..k) with one atomic per block and value.
template <int K> __device__ __forceinline__ void block_sum_to_global(double (&v)[K], double *out)
{
    __shared__ double sm[32][K];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
#pragma unroll
    for (int k = 0; k < K; ++k)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_down_sync(0xffffffffu, v[k], o);
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < K; ++k) sm[warp][k] = v[k];
    __syncthreads();
    if (warp == 0) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            double x = lane < nw ? sm[lane][k] : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) x += __shfl_down_sync(0xffffffffu, x, o);
            if (lane == 0) atomicAdd(out + k, x);
        }
    }
    __syncthreads();
}

// ---------------------------------------------------------------------------------------
// Brick-major order of the sort and the tiles of the brick kernel (mpcd_brick.cuh).
// ---------------------------------------------------------------------------------------
#ifndef MPCD_BRICK_X
#define MPCD_BRICK_X 4
#endif
#ifndef MPCD_BRICK_Y
#define MPCD_BRICK_Y 4
#endif
#ifndef MPCD_BRICK_Z
#define MPCD_BRICK_Z 4
#endif
#ifndef MPCD_BRICK_HALO
#define MPCD_BRICK_HALO 2
#endif
constexpr int kBX = MPCD_BRICK_X, kBY = MPCD_BRICK_Y, kBZ = MPCD_BRICK_Z, kBV = kBX * kBY * kBZ;
constexpr int kH = MPCD_BRICK_HALO;
constexpr int kWX = kBX + kH, kWY = kBY + kH, kWZ = kBZ + kH, kW = kWX * kWY * kWZ;

// floor(n / d) for 0 <= n < 2^31 and a run-time invariant d >= 1: (n m) >> (31 + s), s = ceil(log2 d), m = ceil(2^(31+s) / d)
// (Granlund & Montgomery's round-up multiplier for 31-bit dividends: m < 2^32, the product fits 64 bits).
struct Div31 { uint32_t m, s; };
inline Div31 make_div31(uint32_t d)
{
    uint32_t s = 0;
    while (((uint64_t)1 << s) < d) ++s;
    const uint64_t two = (uint64_t)1 << (31 + s);
    return Div31{(uint32_t)((two + d - 1) / d), s};
}
__device__ __forceinline__ uint32_t div31(uint32_t n, const Div31 &dv) { return (uint32_t)(((uint64_t)n * dv.m) >> (31 + dv.s)); }

// The sort key.  Linear order (on == 0): key = cell index.  Brick-major order: key = brick * kBV + cell inside the brick,
// bricks x-fastest over nb = ceil(n / kB) per axis, cells x-fastest inside the brick; keys of cells outside the box
// (ragged last bricks) are holes with count 0.
struct BrickGrid {
    int32_t on;
    int32_t n[3], nb[3];
    int64_t nkeys;
};
__host__ __device__ __forceinline__ int64_t key_to_cell(int64_t k, const BrickGrid &g)       // -1 for a hole
{
    if (!g.on) return k;
    const int64_t b = k / kBV;
    const int l = (int)(k - b * kBV);
    const int lx = l % kBX, ly = (l / kBX) % kBY, lz = l / (kBX * kBY);
    const int bx = (int)(b % g.nb[0]), by = (int)((b / g.nb[0]) % g.nb[1]), bz = (int)(b / ((int64_t)g.nb[0] * g.nb[1]));
    const int ix = bx * kBX + lx, iy = by * kBY + ly, iz = bz * kBZ + lz;
    if (ix >= g.n[0] || iy >= g.n[1] || iz >= g.n[2]) return -1;
    return ix + (int64_t)g.n[0] * (iy + (int64_t)g.n[1] * iz);
}


}  // namespace mpcdk
