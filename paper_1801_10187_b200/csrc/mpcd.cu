// mpcd.cu -- host side of the C ABI declared in include/mpcd.h: handle, memory, the step
// scheduler and the kernel launches.  All arithmetic of the method runs in the kernels of
// mpcd_kernels.cuh; the only method arithmetic on the host is the three-scalar grid-shift
// draw (a2) and cos/sin of the SRD angle (A15).
#include "../../include/mpcd.h"
#include "mpcd_brick.cuh"
#include "mpcd_small.cuh"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace mpcdk;

namespace {

thread_local char g_create_error[256] = "no error";

struct Buffer { void *ptr; size_t bytes; };

}  // namespace

struct mpcd {
    // parameters
    int64_t N = 0, Nc = 0;
    int32_t n[3] = {0, 0, 0};
    double box[3] = {0, 0, 0};
    double a = 1, m = 1, kT = 1, sigma = 1;
    uint64_t seed = 0;
    mpcd_options opt{};
    cudaStream_t stream = nullptr;
    // particle arrays, double-buffered for the sort
    void *pos[2] = {nullptr, nullptr}, *vel[2] = {nullptr, nullptr};
    uint32_t *tag[2] = {nullptr, nullptr};
    void *cells_stage = nullptr;   // mpcd_get_cells' staging buffer, from the allocator on first use
    int32_t *cell = nullptr;       // cell index per particle, filled on demand only (mpcd_get_state / mpcd_device_ptrs)
    int pcur = 0;
    // cell arrays, double-buffered by step parity: while the fused kernel reads the sums and axes of step t
    // (collision) it accumulates step t + 1 into the other set
    double *acc[2] = {nullptr, nullptr};      // {Sx, Sy, Sz, N} per cell
    double *qacc[2] = {nullptr, nullptr};     // sum |v|^2 per cell
    double *at_acc[2] = {nullptr, nullptr};   // {Dx, Dy, Dz, -} per cell (AT only, allocated on first use)
    double *axis[2] = {nullptr, nullptr};     // {nx, ny, nz, -} per cell
    // small systems (mpcd_small.cuh): a third accumulator set, allocated on first use; whether the cooperative kernel may be used
    double *acc_x = nullptr, *qacc_x = nullptr;
    bool small_ok = true;          // cleared for good once a property that cannot change rules the cooperative path out
    int small_capacity = -1;       // thread blocks of one resident wave of this handle's small_steps instantiation on this handle's device
    std::vector<const void *> smem_configured;   // brick kernels whose dynamic shared memory opt-in has been set on this handle's device
    // embedded solute (NEXT-1; mpcd_embedded.cuh): beads in double, their per-cell sums by step parity
    int64_t emb_n = 0;
    int32_t emb_chain_len = 0, emb_nsub = 0;
    double emb_k = 0, emb_r0 = 0;
    double4 *emb_pos = nullptr, *emb_vel = nullptr;
    double *emb_acc[2] = {nullptr, nullptr};
    double *emb_q[2] = {nullptr, nullptr};     // {sum m |v|^2, number of beads} per cell: only with the cell thermostat (A28)
    bool emb_zeroed[2] = {false, false};
    bool emb_binned = false;       // the beads are binned and summed for the current bin
    cudaStream_t emb_stream = nullptr;   // inside mpcd_step the bead kernel runs beside the solvent's step kernel (fork / join by events)
    cudaEvent_t emb_fork = nullptr, emb_join = nullptr;
    int32_t *cell_start = nullptr, *tile_sum = nullptr;
    // brick-major sort order and the brick-tiled step kernel (mpcd_brick.cuh)
    BrickGrid grid{};              // the sort keys: grid.on = 0 is the plain ascending-cell order
    int32_t nbricks = 0;
    int32_t *brick_start[2] = {nullptr, nullptr};   // segment starts of the current order / of the sort being prepared
    int bcur = 0;
    bool brick_valid = false;      // the particle arrays are in brick-major order of the bin whose shift is brick_shift
    double brick_shift[3] = {0, 0, 0};
    int *d_max_occ = nullptr;
    double *d_scalars = nullptr;   // 8 doubles of scratch for reductions
    int ccur = 0;                  // accumulator set of the current bin
    int num_sms = 148;
    bool debug_sync = false;       // MPCD_DEBUG_SYNC=1: synchronise after every launch (see LAUNCH_CHECK)
    bool zeroed[2] = {false, false}, at_zeroed[2] = {false, false};
    bool axis_valid[2] = {false, false}, xi_valid[2] = {false, false};   // xi: the thermostat factor in the axis sector's 4th word
    uint64_t axis_step[2] = {0, 0};
    int max_occ = 0;               // of the last bin whose counts were inspected
    // state machine
    uint64_t step = 0, bin_step = 0;
    bool bin_valid = false, sums_valid = false, energy_valid = false, counts_valid = false;
    double shift_used[3] = {0, 0, 0};
    // bookkeeping
    std::vector<Buffer> buffers;
    uint64_t launches = 0, sorts = 0, device_bytes = 0;
    // opt-in per-kernel timing (mpcd_set_profiling): CUDA events on the handle's stream
    bool profiling = false;
    struct Timed { cudaEvent_t a, b; int kind; };
    std::vector<Timed> timed;
    double prof_ms[MPCD_PROF_KINDS] = {0};
    uint64_t prof_n[MPCD_PROF_KINDS] = {0};
    char err[256] = "no error";
};

namespace {

int fail(mpcd_t *h, int code, const char *fmt, const char *detail = "")
{
    char *dst = h ? h->err : g_create_error;
    snprintf(dst, 256, fmt, detail);
    return code;
}

#define CUDA_TRY(h, expr)                                                        \
    do {                                                                         \
        cudaError_t e_ = (expr);                                                 \
        if (e_ != cudaSuccess) return fail((h), MPCD_ECUDA, #expr ": %s", cudaGetErrorString(e_)); \
    } while (0)

// After every kernel launch.  With MPCD_DEBUG_SYNC=1 in the environment the stream is synchronised here, so a
// faulting kernel is reported at its own launch site (source line, launch number) instead of at a later call.
#define LAUNCH_CHECK(h)                                                          \
    do {                                                                         \
        (h)->launches += 1;                                                      \
        cudaError_t e_ = cudaGetLastError();                                     \
        if (e_ == cudaSuccess && (h)->debug_sync) e_ = cudaStreamSynchronize((h)->stream); \
        if (e_ != cudaSuccess) {                                                 \
            char where_[96];                                                     \
            snprintf(where_, sizeof(where_), "%s (mpcd.cu:%d, launch %llu)", cudaGetErrorString(e_), __LINE__, (unsigned long long)(h)->launches); \
            return fail((h), MPCD_ECUDA, "kernel launch: %s", where_);          \
        }                                                                        \
    } while (0)

int dev_alloc(mpcd_t *h, void **out, size_t bytes)
{
    bytes = (bytes + 255) & ~(size_t)255;
    if (bytes == 0) bytes = 256;
    void *p = nullptr;
    if (h->opt.alloc_fn) {
        p = h->opt.alloc_fn(bytes, h->opt.alloc_user);
        if (!p) return fail(h, MPCD_ENOMEM, "allocator callback returned NULL%s");
    } else {
        cudaError_t e = cudaMalloc(&p, bytes);
        if (e != cudaSuccess) { cudaGetLastError(); return fail(h, MPCD_ENOMEM, "cudaMalloc: %s", cudaGetErrorString(e)); }
    }
    try {
        h->buffers.push_back(Buffer{p, bytes});
    } catch (...) {
        if (h->opt.free_fn) h->opt.free_fn(p, h->opt.alloc_user); else if (!h->opt.alloc_fn) cudaFree(p);
        return fail(h, MPCD_ENOMEM, "host bookkeeping allocation failed%s");
    }
    h->device_bytes += bytes;
    *out = p;
    return MPCD_OK;
}

template <typename P> int dev_alloc_t(mpcd_t *h, P **out, size_t count) { return dev_alloc(h, reinterpret_cast<void **>(out), count * sizeof(P)); }

inline size_t native_size(const mpcd_t *h) { return h->opt.precision == MPCD_FP64 ? sizeof(double) : sizeof(float); }
inline unsigned grid_for(int64_t n, int threads) { return (unsigned)((n + threads - 1) / threads); }

struct ProfScope {   // brackets the launches of one kind with a CUDA event pair when profiling is on
    mpcd_t *h; int kind; cudaEvent_t a = nullptr, b = nullptr;
    ProfScope(mpcd_t *h_, int kind_) : h(h_), kind(kind_)
    {
        if (!h->profiling) return;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { a = b = nullptr; return; }
        cudaEventRecord(a, h->stream);
    }
    ~ProfScope()
    {
        if (!a) return;
        cudaEventRecord(b, h->stream);
        try { h->timed.push_back(mpcd::Timed{a, b, kind}); } catch (...) { cudaEventDestroy(a); cudaEventDestroy(b); }
    }
};

void drain_profile(mpcd_t *h)
{
    for (const auto &t : h->timed) {
        float ms = 0.f;
        if (cudaEventSynchronize(t.b) == cudaSuccess && cudaEventElapsedTime(&ms, t.a, t.b) == cudaSuccess) {
            h->prof_ms[t.kind] += ms;
            h->prof_n[t.kind] += 1;
        }
        cudaEventDestroy(t.a);
        cudaEventDestroy(t.b);
    }
    h->timed.clear();
}

// a2: the step's grid shift, uniform on (-a/2, a/2)^3 from Philox(seed, (0, t, SHIFT)) (A4, A5)
void draw_shift(const mpcd_t *h, uint64_t step, double s[3])
{
    const u32x4 b = draw(h->seed, step, 0u, kDomShift);
    const uint32_t w[3] = {b.x, b.y, b.z};
    for (int d = 0; d < 3; ++d) s[d] = (u01_32(w[d]) - 0.5) * h->a;
}

inline bool thermostatted(const mpcd_t *h) { return h->opt.thermostat != 0; }
inline bool deterministic(const mpcd_t *h) { return h->opt.deterministic != 0; }
inline unsigned fixed_flag(const mpcd_t *h) { return h->opt.deterministic != 0 ? kFixed : 0u; }

// the shift as the binning applies it
inline void shift_for(const mpcd_t *h, uint64_t step, double out[3])
{
    draw_shift(h, step, out);
    if (h->opt.precision != MPCD_FP64) for (int d = 0; d < 3; ++d) out[d] = (double)(float)out[d];   // A5
}

// What one launch of the pass works on: `cset` = accumulator set of the step being collided (its sums, thermostat
// sums and, by step parity, its axes), `bset` = set of the step being binned.
struct PassPlan {
    int cset = 0, bset = 0;
    uint64_t step_collide = 0, step_bin = 0;
    double shift[3] = {0, 0, 0};      // grid shift of the step being binned
    double alpha = 0;
    bool sort_out = false;            // kSortOut: write the particles to the duplicate arrays in cell order
};

template <typename T> PassArgs<T> make_args(mpcd_t *h, const PassPlan &pl)
{
    PassArgs<T> a{};
    a.pos = static_cast<typename Vec4<T>::type *>(h->pos[h->pcur]);
    a.vel = static_cast<typename Vec4<T>::type *>(h->vel[h->pcur]);
    a.tag = h->tag[h->pcur];
    a.sums = h->acc[pl.cset];
    a.dsum = h->at_acc[pl.cset];
    a.axis = h->axis[pl.step_collide & 1];
    a.esum = h->emb_acc[pl.cset];
    a.mass = h->m;
    a.acc = h->acc[pl.bset];
    a.qacc = h->qacc[pl.bset];
    a.at_acc = h->at_acc[pl.bset];
    a.pos_out = static_cast<typename Vec4<T>::type *>(h->pos[h->pcur ^ 1]);
    a.vel_out = static_cast<typename Vec4<T>::type *>(h->vel[h->pcur ^ 1]);
    a.tag_out = h->tag[h->pcur ^ 1];
    a.cursor = h->cell_start;
    a.N = h->N;
    a.Nc = h->Nc;
    for (int d = 0; d < 3; ++d) {
        a.n[d] = h->n[d];
        a.L[d] = (T)h->box[d];
        a.shift[d] = (T)pl.shift[d];
    }
    a.dt = (T)h->opt.dt;
    a.inv_a = (T)1 / (T)h->a;
    a.cos_a = std::cos(pl.alpha);
    a.sin_a = std::sin(pl.alpha);
    a.sigma = h->sigma;
    a.seed = h->seed;
    a.step_collide = pl.step_collide;
    a.step_bin = pl.step_bin;
    return a;
}

template <typename T, unsigned F> void launch_pass_t(mpcd_t *h, const PassArgs<T> &a)
{
    particle_pass<T, F><<<grid_for(h->N, kPassThreads), kPassThreads, 0, h->stream>>>(a);
}

template <typename T> int launch_pass(mpcd_t *h, unsigned F, const PassPlan &pl)
{
    const PassArgs<T> a = make_args<T>(h, pl);
    switch (F) {
#define CASE(f) case (f): launch_pass_t<T, (f)>(h, a); break;
        CASE(kStream)
        CASE(kBin | kEnergy)
        CASE(kStream | kBin)
        CASE(kStream | kBin | kEnergy)
        CASE(kStream | kBin | kATDraw)
        CASE(kStream | kBin | kATDraw | kEnergy)
        CASE(kSRD)
        CASE(kSRD | kStream | kBin)
        CASE(kSRD | kStream | kBin | kEnergy)
        CASE(kATApply | kStream | kBin | kATDraw)
        CASE(kATApply | kStream | kBin | kATDraw | kEnergy)
        CASE(kSRD | kStream | kBin | kSortOut)
        CASE(kSRD | kStream | kBin | kEnergy | kSortOut)
        CASE(kATApply | kStream | kBin | kATDraw | kSortOut)
        CASE(kATApply | kStream | kBin | kATDraw | kEnergy | kSortOut)
        CASE(kSRD | kEmbedded)
        CASE(kSRD | kEmbedded | kStream | kBin)
        CASE(kSRD | kEmbedded | kStream | kBin | kEnergy)
        CASE(kSRD | kEmbedded | kStream | kBin | kSortOut)
        CASE(kSRD | kEmbedded | kStream | kBin | kEnergy | kSortOut)
        CASE(kSRD | kThermo | kEmbedded)
        CASE(kSRD | kThermo | kEmbedded | kStream | kBin | kEnergy)
        CASE(kSRD | kThermo | kEmbedded | kStream | kBin | kEnergy | kSortOut)
        CASE(kBin | kEnergy | kFixed)
        CASE(kStream | kBin | kFixed)
        CASE(kStream | kBin | kEnergy | kFixed)
        CASE(kSRD | kFixed)
        CASE(kSRD | kStream | kBin | kFixed)
        CASE(kSRD | kStream | kBin | kEnergy | kFixed)
        CASE(kSRD | kStream | kBin | kSortOut | kFixed)
        CASE(kSRD | kStream | kBin | kEnergy | kSortOut | kFixed)
        CASE(kSRD | kThermo | kFixed)
        CASE(kSRD | kThermo | kStream | kBin | kEnergy | kFixed)
        CASE(kSRD | kThermo | kStream | kBin | kEnergy | kSortOut | kFixed)
        CASE(kSRD | kThermo)
        CASE(kSRD | kThermo | kStream | kBin | kEnergy)
        CASE(kSRD | kThermo | kStream | kBin | kEnergy | kSortOut)
        CASE(kStream | kBin | kATDraw | kATStored)
        CASE(kStream | kBin | kATDraw | kEnergy | kATStored)
        CASE(kATApply | kStream | kBin | kATDraw | kATStored)
        CASE(kATApply | kStream | kBin | kATDraw | kEnergy | kATStored)
        CASE(kATApply | kStream | kBin | kATDraw | kATStored | kSortOut)
        CASE(kATApply | kStream | kBin | kATDraw | kEnergy | kATStored | kSortOut)
        CASE(kATApply | kATStored)
        CASE(kATDraw)
        CASE(kATApply)
#undef CASE
        default: return fail(h, MPCD_EINVAL, "internal: pass combination not instantiated%s");
    }
    LAUNCH_CHECK(h);
    return MPCD_OK;
}

// The brick kernel's view of one launch: the segment starts of the current order, where the two cell windows sit
// relative to a brick (the shift of the step collided / binned against the shift of the bin the arrays were sorted by,
// centred on the halo), and the fixed-point scales of the shared-memory partial sums (mpcd_brick.cuh).
BrickArgs brick_args(const mpcd_t *h, const PassPlan &pl)
{
    BrickArgs g{};
    g.brick_start = h->brick_start[h->bcur];
    double sc[3];
    shift_for(h, pl.step_collide, sc);
    for (int d = 0; d < 3; ++d) {
        g.nb[d] = h->grid.nb[d];
        g.og[d] = (int32_t)std::floor((sc[d] - h->brick_shift[d]) / h->a - 0.5 * kH + 0.5);
        g.oa[d] = (int32_t)std::floor((pl.shift[d] - h->brick_shift[d]) / h->a - 0.5 * kH + 0.5);
    }
    g.div_nx = make_div31((uint32_t)h->n[0]);
    g.div_nxy = make_div31((uint32_t)h->n[0] * (uint32_t)h->n[1]);
    g.div_nbx = make_div31((uint32_t)h->grid.nb[0]);
    g.div_nbxy = make_div31((uint32_t)h->grid.nb[0] * (uint32_t)h->grid.nb[1]);
    int e = 0;
    std::frexp(h->sigma, &e);                        // unit = 2^e >= sqrt(kT / m)
    if (deterministic(h)) {
        g.sv = kFixScale; g.inv_sv = g.inv_sq = kFixInv; g.qrel = 1.0; g.vmax = HUGE_VAL;
    } else {
        g.sv = std::ldexp(1.0, 48 - e); g.inv_sv = std::ldexp(1.0, e - 48);
        g.inv_sq = std::ldexp(1.0, 2 * e - 44); g.qrel = std::ldexp(1.0, -4 - e);
        g.vmax = std::ldexp(8.0, e);
    }
    return g;
}

template <typename T, unsigned F> int launch_brick_t(mpcd_t *h, const PassArgs<T> &a, const BrickArgs &g)
{
    // dynamic shared memory above 48 KB is opt-in per kernel AND per device: remembered on the handle (which lives on one
    // device and is used by one host thread at a time), not in a process-wide flag
    const void *kern = reinterpret_cast<const void *>(brick_pass<T, F>);
    bool configured = false;
    for (const void *k : h->smem_configured) configured = configured || k == kern;
    if (!configured) {
        CUDA_TRY(h, cudaFuncSetAttribute(brick_pass<T, F>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)BrickSmem<F>::bytes));
        try { h->smem_configured.push_back(kern); } catch (...) { /* not remembered: set again at the next launch */ }
    }
    brick_pass<T, F><<<(unsigned)h->nbricks, kBrickThreads, BrickSmem<F>::bytes, h->stream>>>(a, g);
    return MPCD_OK;
}

template <typename T> int launch_brick(mpcd_t *h, unsigned F, const PassPlan &pl)
{
    const PassArgs<T> a = make_args<T>(h, pl);
    const BrickArgs g = brick_args(h, pl);
    int rc = MPCD_OK;
    switch (F) {
#define CASE(f) case (f): rc = launch_brick_t<T, (f)>(h, a, g); break;
#define CASE_F32(f) case (f): if constexpr (sizeof(T) == 4) { rc = launch_brick_t<T, (f)>(h, a, g); break; } else return fail(h, MPCD_EINVAL, "internal: fixed-point sums need the mixed model%s");
        CASE(kSRD | kStream | kBin)
        CASE(kSRD | kStream | kBin | kEnergy)
        CASE(kSRD | kStream | kBin | kSortOut)
        CASE(kSRD | kStream | kBin | kEnergy | kSortOut)
        CASE(kSRD | kEmbedded | kStream | kBin)
        CASE(kSRD | kEmbedded | kStream | kBin | kEnergy)
        CASE(kSRD | kEmbedded | kStream | kBin | kSortOut)
        CASE(kSRD | kEmbedded | kStream | kBin | kEnergy | kSortOut)
        CASE(kSRD | kThermo | kStream | kBin | kEnergy)
        CASE(kSRD | kThermo | kStream | kBin | kEnergy | kSortOut)
        CASE(kSRD | kThermo | kEmbedded | kStream | kBin | kEnergy)
        CASE(kSRD | kThermo | kEmbedded | kStream | kBin | kEnergy | kSortOut)
        CASE_F32(kSRD | kStream | kBin | kFixed)
        CASE_F32(kSRD | kStream | kBin | kEnergy | kFixed)
        CASE_F32(kSRD | kStream | kBin | kSortOut | kFixed)
        CASE_F32(kSRD | kStream | kBin | kEnergy | kSortOut | kFixed)
        CASE_F32(kSRD | kThermo | kStream | kBin | kEnergy | kFixed)
        CASE_F32(kSRD | kThermo | kStream | kBin | kEnergy | kSortOut | kFixed)
#undef CASE
#undef CASE_F32
        default: return fail(h, MPCD_EINVAL, "internal: brick pass combination not instantiated%s");
    }
    if (rc) return rc;
    LAUNCH_CHECK(h);
    return MPCD_OK;
}

int pass(mpcd_t *h, unsigned F, const PassPlan &pl)
{
    const bool collide = (F & (kSRD | kATApply)) != 0, bin = (F & kBin) != 0;
    ProfScope prof(h, collide && bin ? ((F & kSortOut) ? MPCD_PROF_FUSED_SORT : MPCD_PROF_FUSED) : (collide ? MPCD_PROF_COLLIDE : (bin ? MPCD_PROF_BIN : MPCD_PROF_OTHER)));
    if (h->brick_valid && (F & kSRD) && (F & kStream) && (F & kBin))   // the arrays are in brick order: one CTA per brick
        return h->opt.precision == MPCD_FP64 ? launch_brick<double>(h, F, pl) : launch_brick<float>(h, F, pl);
    return h->opt.precision == MPCD_FP64 ? launch_pass<double>(h, F, pl) : launch_pass<float>(h, F, pl);
}

int ensure_at_buffers(mpcd_t *h)
{
    if (h->at_acc[0]) return MPCD_OK;
    for (int s = 0; s < 2; ++s) {
        int rc = dev_alloc_t(h, &h->at_acc[s], (size_t)h->Nc * 4);
        if (rc) return rc;
        h->at_zeroed[s] = false;
    }
    return MPCD_OK;
}

// Cell-side preparation, as ONE launch of cell_prepare doing whatever of this is still missing: accumulator set
// `zset` all-zero (its sums if `sums`, its thermostat sums if `at`; zset < 0 = none) and the axes of step
// `axis_step` in axis[axis_step & 1] (want_axes = false: none).
int prepare(mpcd_t *h, int zset, bool sums, bool at, bool want_axes, uint64_t axis_step)
{
    const bool zs = zset >= 0 && sums && !h->zeroed[zset];
    const bool za = zset >= 0 && at && h->at_acc[zset] && !h->at_zeroed[zset];
    const bool ze = zset >= 0 && sums && h->emb_acc[zset] && !h->emb_zeroed[zset];      // the beads' sums go with the solvent's
    const int b = (int)(axis_step & 1);
    const bool ax = want_axes && !(h->axis_valid[b] && h->axis_step[b] == axis_step);
    if (!zs && !za && !ze && !ax) return MPCD_OK;
    ProfScope prof(h, MPCD_PROF_CELLS);
    cell_prepare<<<grid_for(h->Nc, 256), 256, 0, h->stream>>>(ax ? h->axis[b] : nullptr, h->seed, axis_step, zs ? h->acc[zset] : nullptr,
                                                           zs ? h->qacc[zset] : nullptr, za ? h->at_acc[zset] : nullptr,
                                                           ze ? h->emb_acc[zset] : nullptr, ze ? h->emb_q[zset] : nullptr, h->Nc);
    LAUNCH_CHECK(h);
    if (zs) h->zeroed[zset] = true;
    if (za) h->at_zeroed[zset] = true;
    if (ze) h->emb_zeroed[zset] = true;
    if (ax) { h->axis_valid[b] = true; h->axis_step[b] = axis_step; h->xi_valid[b] = false; }
    return MPCD_OK;
}
inline int zero_set(mpcd_t *h, int s, bool sums, bool at) { return prepare(h, s, sums, at, false, 0); }
inline int ensure_axes(mpcd_t *h, uint64_t t) { return prepare(h, -1, false, false, true, t); }


// Maxwell-Boltzmann cell thermostat: xi of every cell from the complete sums (incl. energy) of step t in
// set t & 1, into the 4th word of that step's axis sectors.
int thermostat(mpcd_t *h, uint64_t t)
{
    const int b = (int)(t & 1);
    if (h->xi_valid[b] && h->axis_valid[b] && h->axis_step[b] == t) return MPCD_OK;
    int rc = ensure_axes(h, t);
    if (rc) return rc;
    ProfScope prof(h, MPCD_PROF_CELLS);
    cell_thermostat<<<grid_for(h->Nc, 256), 256, 0, h->stream>>>(h->acc[b], h->qacc[b], h->axis[b], h->Nc, h->m, h->kT, h->seed, t, deterministic(h),
                                                                 h->emb_acc[b], h->emb_q[b]);
    LAUNCH_CHECK(h);
    h->xi_valid[b] = true;
    return MPCD_OK;
}

// ---- embedded solute (NEXT-1) ----
inline bool embedded(const mpcd_t *h) { return h->emb_n > 0; }

EmbArgs emb_args(mpcd_t *h, int cset, int bset, uint64_t step_collide, const double shift[3], double alpha)
{
    EmbArgs e{};
    e.pos = h->emb_pos; e.vel = h->emb_vel; e.nb = h->emb_n;
    e.sums = h->acc[cset]; e.esum = h->emb_acc[cset]; e.axis = h->axis[step_collide & 1];
    e.eacc = h->emb_acc[bset];
    e.eqacc = h->emb_q[bset];
    e.thermo = h->opt.thermostat != 0;
    for (int d = 0; d < 3; ++d) { e.n[d] = h->n[d]; e.shift[d] = shift[d]; }
    e.inv_a = 1.0 / h->a;
    e.mass_solvent = h->m;
    e.cos_a = std::cos(alpha); e.sin_a = std::sin(alpha);
    return e;
}

MdArgs md_args(const mpcd_t *h)
{
    MdArgs a{};
    a.pos = h->emb_pos; a.vel = h->emb_vel; a.chain_len = h->emb_chain_len; a.nsub = h->emb_nsub;
    a.k = h->emb_k; a.r0 = h->emb_r0; a.dt = h->opt.dt / h->emb_nsub;
    for (int d = 0; d < 3; ++d) a.L[d] = h->box[d];
    return a;
}

// one launch of the bead kernel (one block per chain) on stream st
template <unsigned G> int emb_launch(mpcd_t *h, const EmbArgs &e, cudaStream_t st)
{
    ProfScope prof(h, MPCD_PROF_OTHER);              // (on the beads' own stream the pair of events on the handle's stream brackets nothing: the count is kept, the time is not)
    emb_step<G><<<(unsigned)(h->emb_n / h->emb_chain_len), kEmbThreads, (size_t)h->emb_chain_len * 10 * sizeof(double), st>>>(md_args(h), e);
    LAUNCH_CHECK(h);
    return MPCD_OK;
}

// the beads' "streaming": md_substeps velocity-Verlet steps over one collision interval
int emb_md(mpcd_t *h)
{
    const double zero[3] = {0, 0, 0};
    return emb_launch<kEmbMd>(h, emb_args(h, 0, 0, 0, zero, 0.0), h->stream);
}

// bin the beads under `shift` and add them to the (zeroed) bead sums of set `bset`
int emb_bin(mpcd_t *h, int bset, const double shift[3])
{
    int rc = emb_launch<kEmbBinAcc>(h, emb_args(h, bset, bset, 0, shift, 0.0), h->stream);
    h->emb_zeroed[bset] = false;
    return rc;
}

int emb_rotate(mpcd_t *h, int cset, uint64_t step_collide, double alpha)
{
    const double zero[3] = {0, 0, 0};
    return emb_launch<kEmbRotate>(h, emb_args(h, cset, cset, step_collide, zero, alpha), h->stream);
}

// inside mpcd_step: [collide(step_collide) with set cset] + MD + [bin under `shift` into set bset] as one launch
template <unsigned G> int emb_step_launch(mpcd_t *h, int cset, int bset, uint64_t step_collide, const double shift[3], double alpha, bool beside = false)
{
    // beside: on the beads' own stream, after everything enqueued so far on the handle's stream (fork); the caller joins
    cudaStream_t st = beside && h->emb_stream ? h->emb_stream : h->stream;
    if (st != h->stream) {
        CUDA_TRY(h, cudaEventRecord(h->emb_fork, h->stream));
        CUDA_TRY(h, cudaStreamWaitEvent(st, h->emb_fork, 0));
    }
    int rc = emb_launch<G>(h, emb_args(h, cset, bset, step_collide, shift, alpha), st);
    if (rc) return rc;
    if (st != h->stream) CUDA_TRY(h, cudaEventRecord(h->emb_join, st));
    if (G & kEmbBinAcc) h->emb_zeroed[bset] = false;
    return MPCD_OK;
}

// the handle's stream waits for the bead kernel launched beside it
int emb_join_stream(mpcd_t *h)
{
    if (h->emb_stream) CUDA_TRY(h, cudaStreamWaitEvent(h->stream, h->emb_join, 0));
    return MPCD_OK;
}

inline bool sort_due(const mpcd_t *h, uint64_t t) { return h->opt.sort_period > 0 && (t % (uint64_t)h->opt.sort_period) == 0; }

// Small systems: `n` consecutive fused steps (collide t .. t + n - 1, none of them a sort step) as ONE cooperative launch
// (mpcd_small.cuh).  Returns MPCD_OK with *done = false when the system is not eligible (too large for one resident wave,
// another rule, thermostat, beads, brick order, profiling): the caller then takes the ordinary per-step path.
// The instantiation of small_steps a handle uses (its precision, energy option and accumulation mode never change), or
// nullptr when there is none for these flags.
const void *small_kernel(const mpcd_t *h, unsigned F)
{
#define SMALL(T, f) reinterpret_cast<const void *>(small_steps<T, (f)>)
    if (h->opt.precision == MPCD_FP64) {
        switch (F) {
            case kSRD | kStream | kBin: return SMALL(double, kSRD | kStream | kBin);
            case kSRD | kStream | kBin | kEnergy: return SMALL(double, kSRD | kStream | kBin | kEnergy);
            default: return nullptr;
        }
    }
    switch (F) {
        case kSRD | kStream | kBin: return SMALL(float, kSRD | kStream | kBin);
        case kSRD | kStream | kBin | kEnergy: return SMALL(float, kSRD | kStream | kBin | kEnergy);
        case kSRD | kStream | kBin | kFixed: return SMALL(float, kSRD | kStream | kBin | kFixed);
        case kSRD | kStream | kBin | kEnergy | kFixed: return SMALL(float, kSRD | kStream | kBin | kEnergy | kFixed);
        default: return nullptr;
    }
#undef SMALL
}

// Whether the cooperative path can ever serve this handle, from what cannot change after mpcd_create.  Cheap, and evaluated
// before mpcd_step looks for a run of steps: a handle that fails it never pays for the search.
inline bool small_possible(mpcd_t *h)
{
    if (!h->small_ok) return false;
    if (h->opt.rule != MPCD_SRD || thermostatted(h) || h->grid.on
        || h->N > (int64_t)h->num_sms * 16 * kPassThreads                                 // cannot be one resident wave whatever the kernel
        || h->Nc > 4 * (int64_t)grid_for(h->N, kPassThreads) * kPassThreads)              // a dilute box: the cell side (an fp64 sincos per cell) would dominate the phase
        h->small_ok = false;
    return h->small_ok;
}

int small_run(mpcd_t *h, int set, uint64_t t, int32_t n, unsigned fe, bool *done)
{
    *done = false;
    if (!small_possible(h) || h->profiling || h->debug_sync || embedded(h)) return MPCD_OK;
    // one resident wave of THIS handle's kernel on THIS handle's device: asked once, before anything is allocated or zeroed;
    // N and the occupancy are fixed, so a handle that does not fit never comes back here
    const unsigned F = kSRD | kStream | kBin | fe | fixed_flag(h);
    const void *kern = small_kernel(h, F);
    if (!kern) { h->small_ok = false; return MPCD_OK; }
    if (h->small_capacity < 0) {
        int per_sm = 0;
        if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, kPassThreads, 0) != cudaSuccess) { cudaGetLastError(); per_sm = 0; }
        h->small_capacity = per_sm * h->num_sms;
    }
    const unsigned grid = grid_for(h->N, kPassThreads);
    if ((int64_t)grid > (int64_t)h->small_capacity) { h->small_ok = false; return MPCD_OK; }
    if (!h->acc_x) {
        int rc = dev_alloc_t(h, &h->acc_x, (size_t)h->Nc * 4);
        if (!rc) rc = dev_alloc_t(h, &h->qacc_x, (size_t)h->Nc);
        if (rc) return rc;
    }
    const int nxt = set ^ 1;
    int rc = zero_set(h, nxt, true, false);          // the set phase 0 accumulates into; the kernel zeroes the later ones itself
    if (rc) return rc;
    PassPlan pl;
    pl.cset = set; pl.bset = nxt;
    pl.step_collide = t; pl.step_bin = t + 1;
    pl.alpha = h->opt.alpha;
    SmallArgs sa{};
    sa.acc3[0] = h->acc[set]; sa.acc3[1] = h->acc[nxt]; sa.acc3[2] = h->acc_x;
    sa.qacc3[0] = h->qacc[set]; sa.qacc3[1] = h->qacc[nxt]; sa.qacc3[2] = h->qacc_x;
    sa.axis2[0] = h->axis[0]; sa.axis2[1] = h->axis[1];
    const int out = (int)((t + (uint64_t)n) & 1);
    sa.acc_out = h->acc[out]; sa.qacc_out = h->qacc[out];
    sa.t0 = t; sa.nphases = n; sa.a_cell = h->a;
    int32_t nsorts = 0, first_sort = n;              // sorts inside the launch (few cells only; else the caller ends the run before a sort step)
    for (int32_t k = 0; k < n; ++k)
        if (sort_due(h, t + (uint64_t)k)) { nsorts += 1; if (first_sort == n) first_sort = k; }
    if (nsorts > 0 && h->Nc > kSmallSortCells) return MPCD_OK;
    sa.sort_period = nsorts > 0 ? h->opt.sort_period : 0;
    sa.first_sort = first_sort;
    const PassArgs<double> a64 = make_args<double>(h, pl);
    const PassArgs<float> a32 = make_args<float>(h, pl);
    void *args[2] = {h->opt.precision == MPCD_FP64 ? (void *)&a64 : (void *)&a32, &sa};
    if (cudaLaunchCooperativeKernel(kern, dim3(grid), dim3(kPassThreads), args, 0, h->stream) != cudaSuccess) {
        cudaGetLastError();                          // no cooperative launch on this device / context: never try again
        h->small_ok = false;
        return MPCD_OK;
    }
    *done = true;
    LAUNCH_CHECK(h);
    // cell-array state after n phases: the sums of step t + n are complete in set (t + n) & 1, the axes of steps t + n and
    // t + n - 1 in their parities; every other set is dirty
    h->zeroed[0] = h->zeroed[1] = false;
    h->xi_valid[0] = h->xi_valid[1] = false;
    for (uint64_t u = t + (uint64_t)n - 1; u <= t + (uint64_t)n; ++u) { h->axis_valid[u & 1] = true; h->axis_step[u & 1] = u; }
    h->sorts += (uint64_t)nsorts;
    if (nsorts & 1) h->pcur ^= 1;                    // every sort inside the launch swapped the two sets of particle arrays
    return MPCD_OK;
}

// a8, first half: exclusive scan of the per-cell counts of accumulator set `s` in sort-key order -> cell_start (the
// write cursors) and, in brick-major order, the segment starts of the order being prepared (brick_start[bcur ^ 1])
int scan_counts(mpcd_t *h, int s)
{
    const int ntiles = (int)((h->grid.nkeys + kScanTile - 1) / kScanTile);
    ProfScope prof(h, MPCD_PROF_SORT);
    scan_tile_sums<<<ntiles, kScanThreads, 0, h->stream>>>(h->acc[s], h->grid, h->tile_sum, deterministic(h));
    LAUNCH_CHECK(h);
    scan_tile_offsets<<<1, 1024, 0, h->stream>>>(h->tile_sum, ntiles);
    LAUNCH_CHECK(h);
    scan_cells<<<ntiles, kScanThreads, 0, h->stream>>>(h->acc[s], h->grid, h->tile_sum, h->cell_start, h->brick_start[h->bcur ^ 1], deterministic(h));
    LAUNCH_CHECK(h);
    return MPCD_OK;
}

// The particle arrays have just been written out in sort-key order of the bin of step t.
void sorted_now(mpcd_t *h, uint64_t t)
{
    h->sorts += 1;
    h->bcur ^= 1;
    h->brick_valid = h->grid.on != 0;
    shift_for(h, t, h->brick_shift);
}

// a8 as a pass of its own: counting sort by cell on the counts of accumulator set `s` (the cell of every particle is
// cached in vel.w).  Inside mpcd_step the scatter is done by the next fused kernel instead (kSortOut).
int do_sort(mpcd_t *h, int s, uint64_t t)
{
    int rc = scan_counts(h, s);
    if (rc) return rc;
    ProfScope prof(h, MPCD_PROF_SORT);
    const int src = h->pcur, dst = src ^ 1;
    PassPlan pl;
    pl.cset = pl.bset = s;
    if (h->opt.precision == MPCD_FP64)
        sort_scatter<double><<<grid_for(h->N, 256), 256, 0, h->stream>>>(make_args<double>(h, pl), h->cell_start, (double4 *)h->pos[dst], (double4 *)h->vel[dst], h->tag[dst]);
    else
        sort_scatter<float><<<grid_for(h->N, 256), 256, 0, h->stream>>>(make_args<float>(h, pl), h->cell_start, (float4 *)h->pos[dst], (float4 *)h->vel[dst], h->tag[dst]);
    LAUNCH_CHECK(h);
    h->pcur = dst;
    sorted_now(h, t);
    return MPCD_OK;
}


// bin + accumulate (+ axes) for step t as a standalone block; energy always accumulated here
int bin_accumulate(mpcd_t *h, uint64_t t)
{
    PassPlan pl;
    shift_for(h, t, pl.shift);
    const int set = (int)(t & 1);
    pl.cset = pl.bset = set;
    pl.step_collide = pl.step_bin = t;
    pl.alpha = h->opt.alpha;
    int rc = zero_set(h, set, true, false);
    if (rc) return rc;
    h->zeroed[set] = false;
    h->xi_valid[set] = false;                         // the sums of this set are rewritten: its thermostat factors are stale
    rc = pass(h, kBin | kEnergy | fixed_flag(h), pl);
    if (rc) return rc;
    for (int d = 0; d < 3; ++d) h->shift_used[d] = pl.shift[d];
    h->ccur = set;
    h->bin_valid = true; h->bin_step = t;
    rc = ensure_axes(h, t);
    if (!rc && embedded(h)) { rc = emb_bin(h, set, pl.shift); h->emb_binned = rc == MPCD_OK; }
    if (!rc && thermostatted(h)) rc = thermostat(h, t);       // after the beads: they count in the cell's energy (A28)
    if (rc) return rc;
    h->sums_valid = true; h->energy_valid = true; h->counts_valid = true;
    return MPCD_OK;
}

// Cell index of every particle under the last bin's shift, computed on demand into h->cell (allocated on first use).
int fill_cells(mpcd_t *h)
{
    if (!h->bin_valid) return fail(h, MPCD_ESTATE, "no bin yet: cell indices are undefined%s");
    if (!h->cell) { int rc = dev_alloc_t(h, &h->cell, (size_t)h->N); if (rc) return rc; }
    PassPlan pl;
    pl.cset = pl.bset = h->ccur;
    if (h->opt.precision == MPCD_FP64)
        cells_of_particles<double><<<grid_for(h->N, 256), 256, 0, h->stream>>>(make_args<double>(h, pl), h->cell);
    else
        cells_of_particles<float><<<grid_for(h->N, 256), 256, 0, h->stream>>>(make_args<float>(h, pl), h->cell);
    LAUNCH_CHECK(h);
    return MPCD_OK;
}

int init_state(mpcd_t *h)
{
    CUDA_TRY(h, cudaMemsetAsync(h->d_scalars, 0, 8 * sizeof(double), h->stream));
    const unsigned g = grid_for(h->N, 256);
    if (h->opt.precision == MPCD_FP64)
        init_particles<double><<<g, 256, 0, h->stream>>>(h->N, h->seed, h->box[0], h->box[1], h->box[2], h->sigma, nullptr, h->d_scalars,
                                                       (double4 *)h->pos[0], (double4 *)h->vel[0], h->tag[0]);
    else
        init_particles<float><<<g, 256, 0, h->stream>>>(h->N, h->seed, h->box[0], h->box[1], h->box[2], h->sigma, nullptr, h->d_scalars,
                                                      (float4 *)h->pos[0], (float4 *)h->vel[0], h->tag[0]);
    LAUNCH_CHECK(h);
    double sum[3];
    CUDA_TRY(h, cudaMemcpyAsync(sum, h->d_scalars, 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    double mean[3] = {sum[0] / (double)h->N, sum[1] / (double)h->N, sum[2] / (double)h->N};
    CUDA_TRY(h, cudaMemcpyAsync(h->d_scalars + 4, mean, 3 * sizeof(double), cudaMemcpyHostToDevice, h->stream));
    if (h->opt.precision == MPCD_FP64)
        init_particles<double><<<g, 256, 0, h->stream>>>(h->N, h->seed, h->box[0], h->box[1], h->box[2], h->sigma, h->d_scalars + 4, nullptr,
                                                       (double4 *)h->pos[0], (double4 *)h->vel[0], h->tag[0]);
    else
        init_particles<float><<<g, 256, 0, h->stream>>>(h->N, h->seed, h->box[0], h->box[1], h->box[2], h->sigma, h->d_scalars + 4, nullptr,
                                                      (float4 *)h->pos[0], (float4 *)h->vel[0], h->tag[0]);
    LAUNCH_CHECK(h);
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return MPCD_OK;
}

void release(mpcd_t *h)
{
    if (h->emb_stream) { cudaStreamSynchronize(h->emb_stream); cudaStreamDestroy(h->emb_stream); h->emb_stream = nullptr; }
    if (h->emb_fork) { cudaEventDestroy(h->emb_fork); h->emb_fork = nullptr; }
    if (h->emb_join) { cudaEventDestroy(h->emb_join); h->emb_join = nullptr; }
    for (const Buffer &b : h->buffers) {
        if (h->opt.free_fn) h->opt.free_fn(b.ptr, h->opt.alloc_user);
        else if (!h->opt.alloc_fn) cudaFree(b.ptr);
    }
    h->buffers.clear();
}

}  // namespace

// =========================================================================================
// C ABI
// =========================================================================================
extern "C" {

int mpcd_default_options(mpcd_options *opt)
{
    if (!opt) return MPCD_EINVAL;
    std::memset(opt, 0, sizeof(*opt));
    opt->precision = MPCD_MIXED;
    opt->rule = MPCD_SRD;
    opt->dt = 0.1;
    opt->alpha = 130.0 * 3.14159265358979323846 / 180.0;
    opt->sort_period = 25;
    opt->cell_energy = 1;
    opt->init_state = 1;
    opt->brick = 0;
    return MPCD_OK;
}

int mpcd_create(mpcd_t **out, const double box[3], int64_t N, double a, double m, double kT, uint64_t seed)
{
    return mpcd_create_ex(out, box, N, a, m, kT, seed, nullptr);
}

int mpcd_create_ex(mpcd_t **out, const double box[3], int64_t N, double a, double m, double kT, uint64_t seed, const mpcd_options *opt)
{
    if (!out) return fail(nullptr, MPCD_EINVAL, "out is NULL%s");
    *out = nullptr;
    if (!box) return fail(nullptr, MPCD_EINVAL, "box is NULL%s");
    if (N < 1 || N >= ((int64_t)1 << 31)) return fail(nullptr, MPCD_EINVAL, "N must be in [1, 2^31)%s");
    if (!(a > 0) || !(m > 0) || !(kT > 0)) return fail(nullptr, MPCD_EINVAL, "a, m, kT must be positive%s");
    mpcd_options o;
    mpcd_default_options(&o);
    if (opt) o = *opt;
    if (o.precision != MPCD_MIXED && o.precision != MPCD_FP64) return fail(nullptr, MPCD_EINVAL, "bad precision%s");
    if (o.rule != MPCD_SRD && o.rule != MPCD_AT) return fail(nullptr, MPCD_EINVAL, "bad rule%s");
    if (o.thermostat != 0 && o.thermostat != 1) return fail(nullptr, MPCD_EINVAL, "thermostat must be 0 or 1%s");
    if (o.deterministic != 0 && (o.deterministic != 1 || o.precision != MPCD_MIXED || o.rule != MPCD_SRD))
        return fail(nullptr, MPCD_EINVAL, "deterministic accumulation is 0 or 1 and needs the mixed model and the SRD rule%s");
    if (o.brick != 0 && o.brick != 1) return fail(nullptr, MPCD_EINVAL, "brick must be 0 or 1%s");
    if (!(o.dt > 0) || o.sort_period < 0) return fail(nullptr, MPCD_EINVAL, "dt must be > 0 and sort_period >= 0%s");
    if ((o.alloc_fn == nullptr) != (o.free_fn == nullptr)) return fail(nullptr, MPCD_EINVAL, "alloc_fn and free_fn must be given together%s");
    int32_t n[3];
    double ncells = 1;
    for (int d = 0; d < 3; ++d) {
        const double q = box[d] / a;
        const double r = std::floor(q + 0.5);
        if (!(r >= 1) || std::fabs(q - r) > 1e-9 || r >= 2147483648.0) return fail(nullptr, MPCD_EINVAL, "box must be a positive integer multiple of a%s");
        n[d] = (int32_t)r;
        ncells *= r;
    }
    if (ncells >= 2147483648.0) return fail(nullptr, MPCD_EINVAL, "number of cells must be < 2^31%s");
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        return fail(nullptr, MPCD_ECUDA, "no CUDA device: this library has no CPU fallback%s");
    }
    mpcd_t *h = new (std::nothrow) mpcd();
    if (!h) return fail(nullptr, MPCD_ENOMEM, "host allocation failed%s");
    h->N = N; h->a = a; h->m = m; h->kT = kT; h->sigma = std::sqrt(kT / m); h->seed = seed; h->opt = o;
    h->stream = static_cast<cudaStream_t>(o.stream);
    for (int d = 0; d < 3; ++d) { h->n[d] = n[d]; h->box[d] = box[d]; }
    h->Nc = (int64_t)n[0] * n[1] * n[2];
    {   // the sort keys: brick-major when asked for and the key space (whole bricks) still fits int32, else the cell index
        BrickGrid &g = h->grid;
        double nkeys = (double)kBV;
        for (int d = 0; d < 3; ++d) g.n[d] = n[d];
        g.nb[0] = (n[0] + kBX - 1) / kBX; g.nb[1] = (n[1] + kBY - 1) / kBY; g.nb[2] = (n[2] + kBZ - 1) / kBZ;
        for (int d = 0; d < 3; ++d) nkeys *= (double)g.nb[d];
        g.on = (o.brick != 0 && nkeys < 2147483648.0) ? 1 : 0;
        g.nkeys = g.on ? (int64_t)g.nb[0] * g.nb[1] * g.nb[2] * kBV : h->Nc;
        h->nbricks = g.on ? g.nb[0] * g.nb[1] * g.nb[2] : 0;
    }
    if (const char *e = std::getenv("MPCD_DEBUG_SYNC")) h->debug_sync = std::atoi(e) != 0;
    if (const char *e = std::getenv("MPCD_NO_COOP")) h->small_ok = std::atoi(e) == 0;      // A/B timing of the small-system kernel
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0) h->num_sms = sms;
    }
    const size_t ns = native_size(h);
    int rc = MPCD_OK;
    for (int s = 0; s < 2 && !rc; ++s) {
        rc = dev_alloc(h, &h->pos[s], (size_t)N * 4 * ns);
        if (!rc) rc = dev_alloc(h, &h->vel[s], (size_t)N * 4 * ns);
        if (!rc) rc = dev_alloc_t(h, &h->tag[s], (size_t)N);
        if (!rc) rc = dev_alloc_t(h, &h->axis[s], (size_t)h->Nc * 4);
    }
    for (int s = 0; s < 2 && !rc; ++s) {
        rc = dev_alloc_t(h, &h->acc[s], (size_t)h->Nc * 4);
        if (!rc) rc = dev_alloc_t(h, &h->qacc[s], (size_t)h->Nc);
    }
    if (!rc) rc = dev_alloc_t(h, &h->cell_start, (size_t)h->Nc + 1);
    if (!rc) rc = dev_alloc_t(h, &h->tile_sum, (size_t)((h->grid.nkeys + kScanTile - 1) / kScanTile) + 1);
    for (int s = 0; s < 2 && !rc; ++s) rc = dev_alloc_t(h, &h->brick_start[s], (size_t)h->nbricks + 1);
    if (!rc) rc = dev_alloc_t(h, &h->d_max_occ, 64);
    if (!rc) rc = dev_alloc_t(h, &h->d_scalars, 32);
    if (!rc && o.rule == MPCD_AT) rc = ensure_at_buffers(h);
    if (!rc && o.init_state) rc = init_state(h);
    if (rc) {
        std::memcpy(g_create_error, h->err, sizeof(g_create_error));
        release(h);
        delete h;
        return rc;
    }
    *out = h;
    return MPCD_OK;
}

int mpcd_destroy(mpcd_t *h)
{
    if (!h) return MPCD_EINVAL;
    cudaStreamSynchronize(h->stream);
    drain_profile(h);
    release(h);
    delete h;
    return MPCD_OK;
}

int mpcd_stream(mpcd_t *h)
{
    if (!h) return MPCD_EINVAL;
    PassPlan pl;
    pl.cset = pl.bset = h->ccur;
    pl.step_collide = pl.step_bin = h->step;
    int rc = pass(h, kStream, pl);
    if (!rc && embedded(h)) rc = emb_md(h);          // the solute moves by MD over the same interval
    if (rc) return rc;
    h->bin_valid = false; h->sums_valid = false; h->energy_valid = false; h->counts_valid = false; h->emb_binned = false;
    h->xi_valid[0] = h->xi_valid[1] = false;
    return MPCD_OK;
}

int mpcd_shift_and_bin(mpcd_t *h)
{
    if (!h) return MPCD_EINVAL;
    return bin_accumulate(h, h->step);
}

int mpcd_collide_srd(mpcd_t *h, double alpha)
{
    if (!h) return MPCD_EINVAL;
    if (!(h->bin_valid && h->bin_step == h->step && h->sums_valid))
        return fail(h, MPCD_ESTATE, "collide_srd needs mpcd_shift_and_bin for the current step first%s");
    int rc = ensure_axes(h, h->step);
    if (!rc && thermostatted(h)) rc = h->energy_valid ? thermostat(h, h->step) : fail(h, MPCD_ESTATE, "thermostat needs the cell energies%s");
    if (rc) return rc;
    PassPlan pl;
    pl.cset = pl.bset = h->ccur;
    pl.step_collide = pl.step_bin = h->step;
    pl.alpha = alpha;
    if (embedded(h)) {
        if (!h->emb_binned) return fail(h, MPCD_ESTATE, "the embedded beads are not binned for this step: call mpcd_shift_and_bin%s");
        rc = emb_rotate(h, h->ccur, h->step, alpha);
        if (rc) return rc;
    }
    rc = pass(h, kSRD | (thermostatted(h) ? kThermo : 0u) | (embedded(h) ? kEmbedded : 0u) | fixed_flag(h), pl);
    if (rc) return rc;
    h->sums_valid = false; h->energy_valid = false; h->emb_binned = false;
    return MPCD_OK;
}

int mpcd_collide_at(mpcd_t *h)
{
    if (!h) return MPCD_EINVAL;
    if (!(h->bin_valid && h->bin_step == h->step && h->sums_valid))
        return fail(h, MPCD_ESTATE, "collide_at needs mpcd_shift_and_bin for the current step first%s");
    if (embedded(h)) return fail(h, MPCD_ESTATE, "embedded beads take part in the SRD rule only%s");
    int rc = ensure_at_buffers(h);
    if (rc) return rc;
    const int set = h->ccur;
    rc = zero_set(h, set, false, true);
    if (rc) return rc;
    h->at_zeroed[set] = false;
    PassPlan pl;
    pl.cset = pl.bset = set;
    pl.step_collide = pl.step_bin = h->step;
    pl.alpha = h->opt.alpha;
    rc = pass(h, kATDraw, pl);                       // second reduction
    if (!rc) rc = pass(h, kATApply, pl);
    if (rc) return rc;
    h->sums_valid = false; h->energy_valid = false;
    return MPCD_OK;
}

int mpcd_sort(mpcd_t *h)
{
    if (!h) return MPCD_EINVAL;
    if (!(h->bin_valid && h->counts_valid)) return fail(h, MPCD_ESTATE, "sort needs a valid bin (mpcd_shift_and_bin)%s");
    return do_sort(h, h->ccur, h->bin_step);
}

int mpcd_step(mpcd_t *h, int32_t nsteps)
{
    if (!h) return MPCD_EINVAL;
    if (nsteps < 0) return fail(h, MPCD_EINVAL, "nsteps must be >= 0%s");
    if (nsteps == 0) return MPCD_OK;
    const bool at = h->opt.rule == MPCD_AT;
    const bool emb = embedded(h);
    if (emb && at) return fail(h, MPCD_ESTATE, "embedded beads take part in the SRD rule only%s");
    const unsigned fb = (emb ? kEmbedded : 0u) | fixed_flag(h);    // flags of the SRD gather; kFixed also goes with every kBin
    const unsigned ft = (!at && thermostatted(h)) ? kThermo : 0u;
    const unsigned fe = (h->opt.cell_energy != 0 || ft) ? kEnergy : 0u;      // the thermostat needs the cell energies
    int rc = MPCD_OK;
    uint64_t t = h->step;
    int set = (int)(t & 1);                         // cell arrays of step k: set k & 1
    PassPlan pl;
    pl.alpha = h->opt.alpha;
    // first block: stream + bin + accumulate for step t
    // (AT: inside this call a cell's ONE accumulator holds sum(v) - sum(dv), kATStored; the second array is not touched)
    rc = prepare(h, set, true, false, !at, t);      // zeroed set of step t, axes of step t
    if (rc) return rc;
    shift_for(h, t, pl.shift);
    pl.cset = pl.bset = set;
    pl.step_collide = pl.step_bin = t;
    h->zeroed[set] = false;
    h->xi_valid[set] = false;
    rc = pass(h, kStream | kBin | fe | fixed_flag(h) | (at ? (kATDraw | kATStored) : 0u), pl);   // AT: vel.xyz carries dv between the launches of this call
    if (!rc && emb) rc = emb_step_launch<kEmbMd | kEmbBinAcc>(h, set, set, t, pl.shift, h->opt.alpha);
    if (rc) return rc;
    if (ft) { rc = thermostat(h, t); if (rc) return rc; }
    bool sort_pending = sort_due(h, t);            // sort by the cells of step t: done by the next fused kernel on its way out
    // steady state, two launches per step: cell_prepare (zeroed set and axes of step t + 1), then collide(t) fused with
    // stream + bin + accumulate (t + 1)
    for (int32_t j = 1; j < nsteps; ++j) {
        if (!at && nsteps - j >= 2 && (!sort_pending || h->Nc <= kSmallSortCells) && small_possible(h)) {   // small systems: a run of steps in one cooperative launch
            int32_t run = nsteps - j;                      // to the end of the call (few cells: the launch sorts itself) ...
            if (h->Nc > kSmallSortCells && h->opt.sort_period > 0) {   // ... or up to the next sort step, t + r with r >= 1
                const int64_t r = (int64_t)h->opt.sort_period - (int64_t)(t % (uint64_t)h->opt.sort_period);
                if (r < (int64_t)run) run = (int32_t)r;
            }
            bool done = false;
            if (run >= 2) { rc = small_run(h, set, t, run, fe, &done); if (rc) return rc; }
            if (done) {
                t += (uint64_t)run; set = (int)(t & 1); j += run - 1;
                shift_for(h, t, pl.shift);                 // the shift of the last bin (mpcd_get_shift)
                sort_pending = sort_due(h, t);
                continue;
            }
        }
        const int nxt = set ^ 1;
        rc = prepare(h, nxt, true, false, !at, t + 1);
        if (rc) return rc;
        if (sort_pending) { rc = scan_counts(h, set); if (rc) return rc; }
        shift_for(h, t + 1, pl.shift);
        if (emb) {            // beads, one launch: collide(t) with the complete sums of step t, MD over the next interval, bin(t + 1)
            rc = emb_step_launch<kEmbRotate | kEmbMd | kEmbBinAcc>(h, set, nxt, t, pl.shift, h->opt.alpha, true);   // beside the solvent's kernel
            if (rc) return rc;
        }
        pl.cset = set; pl.bset = nxt;
        pl.step_collide = t; pl.step_bin = t + 1;
        h->zeroed[nxt] = false;
        h->xi_valid[nxt] = false;
        rc = pass(h, (at ? (kATApply | kATDraw | kATStored) : (kSRD | ft | fb)) | kStream | kBin | fe | (sort_pending ? kSortOut : 0u), pl);
        if (rc) return rc;
        if (emb) { rc = emb_join_stream(h); if (rc) return rc; }
        if (sort_pending) { h->pcur ^= 1; sorted_now(h, t); }
        set = nxt; t += 1;
        if (ft) { rc = thermostat(h, t); if (rc) return rc; }
        sort_pending = sort_due(h, t);
    }
    if (sort_pending) { rc = do_sort(h, set, t); if (rc) return rc; }
    // last collision
    pl.cset = pl.bset = set;
    pl.step_collide = pl.step_bin = t;
    if (emb) { rc = emb_rotate(h, set, t, h->opt.alpha); if (rc) return rc; }
    rc = pass(h, at ? (kATApply | kATStored) : (kSRD | ft | fb), pl);
    if (rc) return rc;
    h->emb_binned = false;
    h->ccur = set;
    for (int d = 0; d < 3; ++d) h->shift_used[d] = pl.shift[d];
    h->bin_valid = true; h->bin_step = t; h->counts_valid = true;
    h->sums_valid = false; h->energy_valid = false;
    h->step = t + 1;
    return MPCD_OK;
}

int mpcd_get_state(mpcd_t *h, void *pos4, void *vel4, uint32_t *tag, int32_t *cell, uint64_t *step)
{
    if (!h) return MPCD_EINVAL;
    const size_t vb = (size_t)h->N * 4 * native_size(h);
    if (pos4) CUDA_TRY(h, cudaMemcpyAsync(pos4, h->pos[h->pcur], vb, cudaMemcpyDeviceToHost, h->stream));
    if (vel4) CUDA_TRY(h, cudaMemcpyAsync(vel4, h->vel[h->pcur], vb, cudaMemcpyDeviceToHost, h->stream));
    if (tag) CUDA_TRY(h, cudaMemcpyAsync(tag, h->tag[h->pcur], (size_t)h->N * 4, cudaMemcpyDeviceToHost, h->stream));
    if (cell && h->bin_valid) {                       // without a bin the cell indices are unspecified: the buffer is left untouched
        int rc = fill_cells(h);
        if (rc) return rc;
        CUDA_TRY(h, cudaMemcpyAsync(cell, h->cell, (size_t)h->N * 4, cudaMemcpyDeviceToHost, h->stream));
    }
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (step) *step = h->step;
    return MPCD_OK;
}

int mpcd_set_state(mpcd_t *h, const void *pos4, const void *vel4, const uint32_t *tag, uint64_t step)
{
    if (!h) return MPCD_EINVAL;
    if (!pos4 || !vel4) return fail(h, MPCD_EINVAL, "pos4 and vel4 are required%s");
    const size_t vb = (size_t)h->N * 4 * native_size(h);
    CUDA_TRY(h, cudaMemcpyAsync(h->pos[h->pcur], pos4, vb, cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(h->vel[h->pcur], vel4, vb, cudaMemcpyHostToDevice, h->stream));
    if (tag) {
        CUDA_TRY(h, cudaMemcpyAsync(h->tag[h->pcur], tag, (size_t)h->N * 4, cudaMemcpyHostToDevice, h->stream));
    } else {
        iota_tags<<<grid_for(h->N, 256), 256, 0, h->stream>>>(h->N, h->tag[h->pcur]);
        LAUNCH_CHECK(h);
    }
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    h->step = step;
    h->bin_valid = false; h->sums_valid = false; h->energy_valid = false; h->counts_valid = false; h->emb_binned = false;
    h->xi_valid[0] = h->xi_valid[1] = false;
    h->brick_valid = false;                           // the caller's order is arbitrary
    return MPCD_OK;
}

int mpcd_get_cells(mpcd_t *h, int32_t *count, double *sumv3, double *ke, double *u3, double *axis3, double *kTc)
{
    if (!h) return MPCD_EINVAL;
    if (!(h->sums_valid && h->energy_valid))
        return fail(h, MPCD_ESTATE, "cell sums are not valid: call mpcd_shift_and_bin first%s");
    if (axis3) { int rc0 = ensure_axes(h, h->bin_step); if (rc0) return rc0; }
    const size_t Nc = (size_t)h->Nc;
    // stage through one device buffer (SoA) obtained from the handle's allocator on first use and kept
    if (!h->cells_stage) {
        int rc0 = dev_alloc(h, &h->cells_stage, Nc * (4 + 8 * (3 + 1 + 3 + 3 + 1)));
        if (rc0) return rc0;
    }
    char *base = static_cast<char *>(h->cells_stage);
    double *d_sumv = reinterpret_cast<double *>(base);
    double *d_ke = d_sumv + 3 * Nc;
    double *d_u = d_ke + Nc;
    double *d_ax = d_u + 3 * Nc;
    double *d_kT = d_ax + 3 * Nc;
    int32_t *d_cnt = reinterpret_cast<int32_t *>(d_kT + Nc);
    cell_unpack<<<grid_for(h->Nc, 256), 256, 0, h->stream>>>(h->acc[h->ccur], h->qacc[h->ccur], h->axis[h->bin_step & 1], h->Nc, h->m, deterministic(h),
                                                          count ? d_cnt : nullptr, sumv3 ? d_sumv : nullptr, ke ? d_ke : nullptr, u3 ? d_u : nullptr,
                                                          axis3 ? d_ax : nullptr, kTc ? d_kT : nullptr);
    LAUNCH_CHECK(h);
    if (count) CUDA_TRY(h, cudaMemcpyAsync(count, d_cnt, Nc * 4, cudaMemcpyDeviceToHost, h->stream));
    if (sumv3) CUDA_TRY(h, cudaMemcpyAsync(sumv3, d_sumv, Nc * 24, cudaMemcpyDeviceToHost, h->stream));
    if (ke) CUDA_TRY(h, cudaMemcpyAsync(ke, d_ke, Nc * 8, cudaMemcpyDeviceToHost, h->stream));
    if (u3) CUDA_TRY(h, cudaMemcpyAsync(u3, d_u, Nc * 24, cudaMemcpyDeviceToHost, h->stream));
    if (axis3) CUDA_TRY(h, cudaMemcpyAsync(axis3, d_ax, Nc * 24, cudaMemcpyDeviceToHost, h->stream));
    if (kTc) CUDA_TRY(h, cudaMemcpyAsync(kTc, d_kT, Nc * 8, cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return MPCD_OK;
}

int mpcd_set_embedded(mpcd_t *h, int64_t nb, const double *pos3, const double *vel3, const double *mass, int32_t chain_len, double k, double r0,
                      int32_t md_substeps)
{
    if (!h) return MPCD_EINVAL;
    if (h->opt.rule != MPCD_SRD || deterministic(h))
        return fail(h, MPCD_EINVAL, "embedded beads need the SRD rule without deterministic accumulation%s");
    if (nb < 1 || !pos3 || !vel3 || !mass || chain_len < 1 || chain_len > kMaxChainLen || nb % chain_len != 0 || !(k >= 0) || !(r0 >= 0) || md_substeps < 1)
        return fail(h, MPCD_EINVAL, "set_embedded: nb >= 1 a multiple of chain_len in [1, 512], k, r0 >= 0, md_substeps >= 1%s");
    std::vector<double4> hp, hv;
    try { hp.resize((size_t)nb); hv.resize((size_t)nb); } catch (...) { return fail(h, MPCD_ENOMEM, "set_embedded: host staging allocation failed%s"); }
    for (int64_t i = 0; i < nb; ++i) {
        if (!(mass[i] > 0)) return fail(h, MPCD_EINVAL, "set_embedded: masses must be positive%s");
        for (int d = 0; d < 3; ++d)
            if (!(pos3[3 * i + d] >= 0.0 && pos3[3 * i + d] < h->box[d])) return fail(h, MPCD_EINVAL, "set_embedded: positions must lie in [0, box)%s");
        hp[i] = double4{pos3[3 * i], pos3[3 * i + 1], pos3[3 * i + 2], mass[i]};
        hv[i] = double4{vel3[3 * i], vel3[3 * i + 1], vel3[3 * i + 2], 0.0};
    }
    if (h->emb_n != nb) {
        if (h->emb_n != 0) return fail(h, MPCD_EINVAL, "set_embedded: the number of beads of a handle cannot change%s");
        int rc = dev_alloc_t(h, &h->emb_pos, (size_t)nb);
        if (!rc) rc = dev_alloc_t(h, &h->emb_vel, (size_t)nb);
        for (int s = 0; s < 2 && !rc; ++s) { rc = dev_alloc_t(h, &h->emb_acc[s], (size_t)h->Nc * 4); h->emb_zeroed[s] = false; }
        for (int s = 0; s < 2 && !rc && thermostatted(h); ++s) rc = dev_alloc_t(h, &h->emb_q[s], (size_t)h->Nc * 2);
        if (rc) return rc;
        if (cudaStreamCreateWithFlags(&h->emb_stream, cudaStreamNonBlocking) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->emb_fork, cudaEventDisableTiming) != cudaSuccess ||
            cudaEventCreateWithFlags(&h->emb_join, cudaEventDisableTiming) != cudaSuccess) {
            cudaGetLastError();                       // no side stream: the bead kernel simply runs in line
            if (h->emb_stream) cudaStreamDestroy(h->emb_stream);
            h->emb_stream = nullptr;
        }
    }
    CUDA_TRY(h, cudaMemcpyAsync(h->emb_pos, hp.data(), (size_t)nb * sizeof(double4), cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(h->emb_vel, hv.data(), (size_t)nb * sizeof(double4), cudaMemcpyHostToDevice, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    h->emb_n = nb; h->emb_chain_len = chain_len; h->emb_nsub = md_substeps; h->emb_k = k; h->emb_r0 = r0;
    h->bin_valid = false; h->sums_valid = false; h->energy_valid = false; h->counts_valid = false; h->emb_binned = false;
    h->xi_valid[0] = h->xi_valid[1] = false;
    return MPCD_OK;
}

int mpcd_get_embedded(mpcd_t *h, double *pos3, double *vel3, int32_t *cell)
{
    if (!h) return MPCD_EINVAL;
    if (!embedded(h)) return fail(h, MPCD_ESTATE, "no embedded beads%s");
    const size_t nb = (size_t)h->emb_n;
    std::vector<double4> hp, hv;
    try { hp.resize(nb); hv.resize(nb); } catch (...) { return fail(h, MPCD_ENOMEM, "get_embedded: host staging allocation failed%s"); }
    CUDA_TRY(h, cudaMemcpyAsync(hp.data(), h->emb_pos, nb * sizeof(double4), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaMemcpyAsync(hv.data(), h->emb_vel, nb * sizeof(double4), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    for (size_t i = 0; i < nb; ++i) {
        if (pos3) { pos3[3 * i] = hp[i].x; pos3[3 * i + 1] = hp[i].y; pos3[3 * i + 2] = hp[i].z; }
        if (vel3) { vel3[3 * i] = hv[i].x; vel3[3 * i + 1] = hv[i].y; vel3[3 * i + 2] = hv[i].z; }
        if (cell) { long long c; std::memcpy(&c, &hv[i].w, sizeof(c)); cell[i] = (int32_t)c; }
    }
    return MPCD_OK;
}

int mpcd_get_xi(mpcd_t *h, double *xi)
{
    if (!h || !xi) return MPCD_EINVAL;
    if (!thermostatted(h)) return fail(h, MPCD_ESTATE, "the thermostat is off (opt.thermostat)%s");
    if (!(h->bin_valid && h->sums_valid && h->energy_valid)) return fail(h, MPCD_ESTATE, "cell sums are not valid: call mpcd_shift_and_bin first%s");
    int rc = thermostat(h, h->bin_step);
    if (rc) return rc;
    CUDA_TRY(h, cudaMemcpy2DAsync(xi, sizeof(double), h->axis[h->bin_step & 1] + 3, 4 * sizeof(double), sizeof(double), (size_t)h->Nc,
                                  cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    return MPCD_OK;
}

int mpcd_get_shift(mpcd_t *h, double s[3])
{
    if (!h || !s) return MPCD_EINVAL;
    if (!h->bin_valid) return fail(h, MPCD_ESTATE, "no bin yet%s");
    for (int d = 0; d < 3; ++d) s[d] = h->shift_used[d];
    return MPCD_OK;
}

int mpcd_get_thermo(mpcd_t *h, double P[3], double *KE, double *kT)
{
    if (!h) return MPCD_EINVAL;
    if (!(h->sums_valid && h->energy_valid)) {
        int rc = bin_accumulate(h, h->bin_valid ? h->bin_step : h->step);
        if (rc) return rc;
    }
    CUDA_TRY(h, cudaMemsetAsync(h->d_scalars, 0, 8 * sizeof(double), h->stream));
    cell_thermo<<<h->num_sms * 4, 256, 0, h->stream>>>(h->acc[h->ccur], h->qacc[h->ccur], h->Nc, h->m, h->d_scalars, deterministic(h));
    LAUNCH_CHECK(h);
    double out[6];
    CUDA_TRY(h, cudaMemcpyAsync(out, h->d_scalars, sizeof(out), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    if (P) for (int d = 0; d < 3; ++d) P[d] = h->m * out[d];
    if (KE) *KE = 0.5 * h->m * out[3];
    if (kT) *kT = out[5] > 0 ? out[4] / out[5] : 0.0;
    return MPCD_OK;
}

int mpcd_get_stats(mpcd_t *h, mpcd_stats *out)
{
    if (!h || !out) return MPCD_EINVAL;
    std::memset(out, 0, sizeof(*out));
    out->N = h->N; out->Nc = h->Nc;
    for (int d = 0; d < 3; ++d) out->n[d] = h->n[d];
    if (h->bin_valid && h->counts_valid) {            // the counts of the last bin are still in its accumulator set
        CUDA_TRY(h, cudaMemsetAsync(h->d_max_occ, 0, sizeof(int), h->stream));
        cell_max_occupancy<<<h->num_sms * 8, 256, 0, h->stream>>>(h->acc[h->ccur], h->Nc, h->d_max_occ, deterministic(h));
        LAUNCH_CHECK(h);
        CUDA_TRY(h, cudaMemcpyAsync(&h->max_occ, h->d_max_occ, sizeof(int), cudaMemcpyDeviceToHost, h->stream));
        CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    }
    out->max_occupancy = h->max_occ;
    if (h->grid.on) { out->brick[0] = kBX; out->brick[1] = kBY; out->brick[2] = kBZ; out->brick[3] = kH; }
    out->step = h->step; out->kernel_launches = h->launches; out->sorts = h->sorts; out->device_bytes = h->device_bytes;
    return MPCD_OK;
}

int mpcd_device_ptrs(mpcd_t *h, void **pos4, void **vel4, uint32_t **tag, int32_t **cell)
{
    if (!h) return MPCD_EINVAL;
    if (pos4) *pos4 = h->pos[h->pcur];
    if (vel4) *vel4 = h->vel[h->pcur];
    if (tag) *tag = h->tag[h->pcur];
    if (cell) {
        int rc = fill_cells(h);
        if (rc) return rc;
        *cell = h->cell;
    }
    return MPCD_OK;
}

int mpcd_set_profiling(mpcd_t *h, int32_t on)
{
    if (!h) return MPCD_EINVAL;
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    drain_profile(h);
    h->profiling = on != 0;
    for (int k = 0; k < MPCD_PROF_KINDS; ++k) { h->prof_ms[k] = 0; h->prof_n[k] = 0; }
    return MPCD_OK;
}

int mpcd_get_profile(mpcd_t *h, double ms[MPCD_PROF_KINDS], uint64_t count[MPCD_PROF_KINDS])
{
    if (!h) return MPCD_EINVAL;
    CUDA_TRY(h, cudaStreamSynchronize(h->stream));
    drain_profile(h);
    for (int k = 0; k < MPCD_PROF_KINDS; ++k) {
        if (ms) ms[k] = h->prof_ms[k];
        if (count) count[k] = h->prof_n[k];
    }
    return MPCD_OK;
}

const char *mpcd_last_error(const mpcd_t *h) { return h ? h->err : g_create_error; }

int mpcd_abi_version(void) { return MPCD_ABI_VERSION; }

const char *mpcd_build_info(void)
{
    return "mpcd-b200 ABI 3, sm_100a, nvcc " __VERSION__
#ifdef __CUDACC_VER_MAJOR__
           " / CUDA"
#endif
        ;
}

int mpcd_test_philox(const uint32_t *ctr4, const uint32_t *key2, uint32_t *out4, int64_t n)
{
    if (!ctr4 || !key2 || !out4 || n < 0) return MPCD_EINVAL;
    if (n == 0) return MPCD_OK;
    uint32_t *d = nullptr;
    if (cudaMalloc(&d, (size_t)n * 10 * sizeof(uint32_t)) != cudaSuccess) { cudaGetLastError(); return MPCD_ECUDA; }
    uint32_t *dc = d, *dk = d + 4 * n, *dout = d + 6 * n;
    int rc = MPCD_OK;
    if (cudaMemcpy(dc, ctr4, (size_t)n * 16, cudaMemcpyHostToDevice) != cudaSuccess) rc = MPCD_ECUDA;
    if (!rc && cudaMemcpy(dk, key2, (size_t)n * 8, cudaMemcpyHostToDevice) != cudaSuccess) rc = MPCD_ECUDA;
    if (!rc) {
        philox_test_kernel<<<grid_for(n, 256), 256>>>(dc, dk, dout, n);
        if (cudaGetLastError() != cudaSuccess) rc = MPCD_ECUDA;
    }
    if (!rc && cudaMemcpy(out4, dout, (size_t)n * 16, cudaMemcpyDeviceToHost) != cudaSuccess) rc = MPCD_ECUDA;
    cudaFree(d);
    return rc;
}

}  // extern "C"
