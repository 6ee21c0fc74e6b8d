// mpcd_static.cu -- mpcd_cell_sums_static: the shifted binning and fp64 cell reduction (a3 + a4, PAPER.md:110,
// :118-124) as ONE handle-free call that obtains no memory from anybody.
//
// Who this is for.  Everything else in this library works on a handle, and a handle gets its O(N) and O(N_cells)
// buffers from cudaMalloc or from the caller's allocator callback.  Some callers can do neither at the moment they need
// the cell sums: an analysis plug-in running inside a simulation whose device memory has been handed over, all of it,
// to another pool (PyTorch's caching allocator, an MPS client held to a fixed memory limit), where a cudaMalloc simply
// fails; and a caller inside a time-critical loop, where a cudaMalloc / cudaFree pair is not acceptable because both
// may synchronise the whole device.  For them the per-cell accumulators -- the one piece of memory the reduction needs
// beyond its inputs and outputs -- live in a fixed array inside this library.
//
// The price.  The array is MPCD_STATIC_MAX_CELLS * 40 bytes (1.25 MiB).  It is part of the library's device code, so a
// GPU holds that much from the moment this code is loaded onto it until the process exits, however rarely the entry
// point is called.  There is ONE array per GPU: all calls on that GPU share it, whatever their stream or host thread.
#include "../../include/mpcd.h"
#include "mpcd_device.cuh"

#include <cstdio>
#include <mutex>

using namespace mpcdk;

namespace {

constexpr int64_t kMaxCells = MPCD_STATIC_MAX_CELLS;
constexpr int kStaticThreads = 128;
constexpr int kMaxDevices = 64;

// The scratch: for a call with Nc cells, {Sx, Sy, Sz, N} per cell in the first 4 Nc doubles (one 32-byte sector per
// cell, what warp_cell_accumulate adds into), sum |v|^2 per cell in the Nc doubles after them.
//
// `g_cell_scratch` is a device symbol.  In HOST code that name is only a stand-in the runtime uses to look the symbol up;
// its host-side address is not device memory, and a kernel handed `g_cell_scratch` from host code would fault (or, on a
// system where the GPU can reach host memory, quietly add into the wrong place).  Host code therefore asks the runtime
// for the device address, once per device, and passes THAT to the kernels (scratch_for_current_device below).
static __device__ __align__(256) double g_cell_scratch[kMaxCells * 5];

std::mutex g_setup_lock;                       // guards g_scratch_ptr and g_sms
double *g_scratch_ptr[kMaxDevices] = {};       // device address of g_cell_scratch on device d, once looked up
int g_sms[kMaxDevices] = {};
thread_local char g_static_error[256] = "no error";

int fail(int code, const char *fmt, const char *detail = "")
{
    snprintf(g_static_error, sizeof(g_static_error), fmt, detail);
    return code;
}

// Set-up, done by the first call on each device with that device current: the device address of the scratch array
// (cudaGetSymbolAddress loads the module on the device if it is not loaded yet, which is why the first call should not
// be made while a stream is capturing) and the SM count for the grid of the unpack kernel.  No allocation.
int scratch_for_current_device(double **out, int *sms)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(MPCD_ECUDA, "cudaGetDevice: %s (no CUDA device: there is no CPU fallback)", cudaGetErrorString(e)); }
    if (dev < 0 || dev >= kMaxDevices) return fail(MPCD_ECUDA, "device ordinal out of range%s");
    std::lock_guard<std::mutex> guard(g_setup_lock);
    if (!g_scratch_ptr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress(reinterpret_cast<void **>(&p), g_cell_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return fail(MPCD_ECUDA, "cudaGetSymbolAddress(scratch): %s", cudaGetErrorString(e)); }
        int n = 0;
        e = cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess || n < 1) { cudaGetLastError(); return fail(MPCD_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e)); }
        g_sms[dev] = n;
        g_scratch_ptr[dev] = p;
    }
    *out = g_scratch_ptr[dev];
    *sms = g_sms[dev];
    return MPCD_OK;
}

template <typename T> struct StaticArgs {
    const typename Vec4<T>::type *pos;
    const typename Vec4<T>::type *vel;
    int64_t N;
    int32_t n[3];
    T inv_a;
    T shift[3];
    double *acc;      // {Sx, Sy, Sz, N} per cell, in the scratch
    double *qacc;     // sum |v|^2 per cell, in the scratch
};

// The variant of particle_pass<T, kBin | kEnergy> (mpcd_kernels.cuh) behind mpcd_shift_and_bin: the same binning
// (bin_axis: add the shift, multiply by 1/a, floor, wrap once, A6) and the same warp-level accumulation
// (match.any + shuffle tree + one fp64 RED per distinct cell and component), but the particle arrays
// are read-only (no cell cache is written into vel.w) and the accumulators are the static scratch.
template <typename T>
__global__ void __launch_bounds__(kStaticThreads) cell_sums_static_pass(const StaticArgs<T> a)
{
    __shared__ WarpScratch ws[kStaticThreads / 32];
    const int64_t i = (int64_t)blockIdx.x * kStaticThreads + threadIdx.x;
    const bool valid = i < a.N;
    const int64_t il = valid ? i : a.N - 1;            // lanes past the end work on a copy of the last particle and take no part
    const auto p = load4(a.pos + il);
    const auto v = load4(a.vel + il);
    const int ix = bin_axis<T>(p.x, a.shift[0], a.inv_a, a.n[0]);
    const int iy = bin_axis<T>(p.y, a.shift[1], a.inv_a, a.n[1]);
    const int iz = bin_axis<T>(p.z, a.shift[2], a.inv_a, a.n[2]);
    // A position outside [0, box) can land outside the grid even after the single wrap: such a particle is left out, so
    // that nothing is ever added outside the scratch array whatever the caller passes.
    const bool inside = ix >= 0 && ix < a.n[0] && iy >= 0 && iy < a.n[1] && iz >= 0 && iz < a.n[2];
    const int c = (valid && inside) ? ix + a.n[0] * (iy + a.n[1] * iz) : -1 - (int)(threadIdx.x & 31);
    warp_cell_accumulate<T, true, true>(a.acc, a.qacc, ws[threadIdx.x >> 5], c, v.x, v.y, v.z);
}

// Scratch -> the caller's outputs, in the layout of mpcd_get_cells: count, S, KE = m q / 2.
__global__ void __launch_bounds__(256) cell_sums_static_unpack(const double *acc, const double *qacc, int64_t Nc, double m,
                                                               int32_t *count, double *sumv3, double *ke)
{
    for (int64_t c = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; c < Nc; c += (int64_t)gridDim.x * blockDim.x) {
        const f64x4 s = ld256(acc + 4 * c);
        if (count) count[c] = (int32_t)s.w;
        if (sumv3) { sumv3[3 * c] = s.x; sumv3[3 * c + 1] = s.y; sumv3[3 * c + 2] = s.z; }
        if (ke) ke[c] = 0.5 * m * qacc[c];
    }
}

template <typename T>
int run(const void *pos4, const void *vel4, int64_t N, const int32_t n[3], double a, const double shift[3], double m, int64_t Nc,
        int32_t *count, double *sumv3, double *ke, cudaStream_t stream)
{
    double *scratch = nullptr;
    int sms = 0;
    int rc = scratch_for_current_device(&scratch, &sms);
    if (rc) return rc;
    double *acc = scratch, *qacc = scratch + 4 * Nc;
    // the array still holds the previous call's sums: everything this call adds into starts from zero
    cudaError_t e = cudaMemsetAsync(scratch, 0, (size_t)Nc * 5 * sizeof(double), stream);
    if (e != cudaSuccess) return fail(MPCD_ECUDA, "cudaMemsetAsync(scratch): %s", cudaGetErrorString(e));
    if (N > 0) {
        StaticArgs<T> s{};
        s.pos = static_cast<const typename Vec4<T>::type *>(pos4);
        s.vel = static_cast<const typename Vec4<T>::type *>(vel4);
        s.N = N;
        for (int d = 0; d < 3; ++d) { s.n[d] = n[d]; s.shift[d] = (T)shift[d]; }
        s.inv_a = (T)1 / (T)a;                         // as the handle forms it (mpcd.cu make_args)
        s.acc = acc; s.qacc = qacc;
        const unsigned grid = (unsigned)((N + kStaticThreads - 1) / kStaticThreads);
        cell_sums_static_pass<T><<<grid, kStaticThreads, 0, stream>>>(s);
        e = cudaGetLastError();
        if (e != cudaSuccess) return fail(MPCD_ECUDA, "cell_sums_static_pass launch: %s", cudaGetErrorString(e));
    }
    const int64_t want = (Nc + 255) / 256;
    const unsigned ugrid = (unsigned)(want < (int64_t)sms * 8 ? want : (int64_t)sms * 8);
    cell_sums_static_unpack<<<ugrid, 256, 0, stream>>>(acc, qacc, Nc, m, count, sumv3, ke);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(MPCD_ECUDA, "cell_sums_static_unpack launch: %s", cudaGetErrorString(e));
    return MPCD_OK;
}

}  // namespace

extern "C" int mpcd_cell_sums_static(const void *pos4, const void *vel4, int64_t N, int32_t precision, const int32_t n[3], double a,
                                     const double shift[3], double m, int32_t *count, double *sumv3, double *ke, void *stream)
{
    if (!n || !shift) return fail(MPCD_EINVAL, "cell_sums_static: n and shift are required%s");
    if (precision != MPCD_MIXED && precision != MPCD_FP64) return fail(MPCD_EINVAL, "cell_sums_static: precision must be MPCD_MIXED or MPCD_FP64%s");
    if (N < 0 || N >= ((int64_t)1 << 31)) return fail(MPCD_EINVAL, "cell_sums_static: N must be in [0, 2^31)%s");
    if (N > 0 && (!pos4 || !vel4)) return fail(MPCD_EINVAL, "cell_sums_static: pos4 and vel4 are required when N > 0%s");
    if (!(a > 0.0) || !(m > 0.0)) return fail(MPCD_EINVAL, "cell_sums_static: a and m must be positive%s");
    if (n[0] < 1 || n[1] < 1 || n[2] < 1) return fail(MPCD_EINVAL, "cell_sums_static: every n[d] must be >= 1%s");
    const int64_t n01 = (int64_t)n[0] * n[1];          // two factors < 2^31 fit; the third is multiplied in only once n01 is known to be small
    const int64_t Nc = n01 <= kMaxCells ? n01 * n[2] : n01;
    if (Nc > kMaxCells) {
        char what[128];
        snprintf(what, sizeof(what), "%d x %d x %d cells, the static scratch holds at most %lld", n[0], n[1], n[2], (long long)kMaxCells);
        return fail(MPCD_EINVAL, "cell_sums_static: %s (MPCD_STATIC_MAX_CELLS); use a handle and mpcd_shift_and_bin for larger grids", what);
    }
    for (int d = 0; d < 3; ++d)
        if (!(shift[d] > -a && shift[d] < a)) return fail(MPCD_EINVAL, "cell_sums_static: |shift[d]| must be below a (the binning wraps once)%s");
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    if (precision == MPCD_FP64) return run<double>(pos4, vel4, N, n, a, shift, m, Nc, count, sumv3, ke, s);
    return run<float>(pos4, vel4, N, n, a, shift, m, Nc, count, sumv3, ke, s);
}

extern "C" const char *mpcd_cell_sums_static_error(void) { return g_static_error; }
