// mpcd_small.cuh -- small systems (BASELINE config 1: 2560 particles, 512 cells): many steps in ONE cooperative launch.
//
// A system whose particle pass fits on the chip as one resident wave of thread blocks is bound by launches, not by
// bandwidth: mpcd_step issues cell_prepare + the fused step kernel per step, ~2 us of kernel each plus the host's launch
// cost (7.9 us per step measured on config 1 in round 1).  Here the grid stays resident and walks the steps itself:
//
//   phase k (collides step t = t0 + k):
//     every thread   the fused pass of its particle, exactly pass_body of mpcd_kernels.cuh: collide(t) with the complete sums
//                    of set k mod 3 and the axes of parity t & 1, stream, bin(t + 1) under the shift of step t + 1 -- drawn
//                    by the thread itself from Philox(seed, t + 1, SHIFT) as the host draws it (A4, A5) --
//                    accumulate into set (k + 1) mod 3;
//     grid-stride    the cell side of cell_prepare for the NEXT phase: axes of step t + 1 into the
//                    other parity, and a zeroed set (k + 2) mod 3.  Three accumulator sets instead of two make this legal
//                    inside the phase: nobody reads or adds to set (k + 2) mod 3 while phase k runs;
//     grid.sync()    the sums of step t + 1 are complete.
//
// The sort: with few cells (<= kSmallSortCells) a phase whose step must be sorted first lets block 0
// scan the counts of that step into the write cursors (one more grid barrier), then runs the pass with kSortOut -- the
// particles go to the duplicate arrays in cell order -- and swaps the two sets of arrays for the phases that follow.  With
// more cells a launch ends before a step that must be sorted, and mpcd_step runs that step through the ordinary kernels.
// Results are those of the ordinary path up to the order of the fp64 additions (bit for bit with opt.deterministic).
#pragma once
#include <cooperative_groups.h>
#include "mpcd_kernels.cuh"

namespace mpcdk {

constexpr int64_t kSmallSortCells = 8192;      // counts that one block scans in a few microseconds

struct SmallArgs {
    double *acc3[3], *qacc3[3];     // accumulator sets in the kernel's rotation: [0] holds the sums of step t0, [1] is zeroed
    double *axis2[2];               // axes by step parity; [t0 & 1] holds the axes of step t0
    double *acc_out, *qacc_out;     // where mpcd_step expects the sums of step t0 + nphases
    uint64_t t0;
    int32_t nphases;
    double a_cell;                  // cell edge (the shift is uniform on (-a/2, a/2))
    int32_t sort_period;            // > 0: steps with t % sort_period == 0 are sorted inside the launch (Nc <= kSmallSortCells)
    int32_t first_sort;             // ... the first such phase (>= nphases: none)
};

// Exclusive scan of the per-cell counts (4th word of the accumulator sectors) into the sort's write cursors, by ONE block.
__device__ __forceinline__ void small_scan_counts(const double *acc, int64_t Nc, int32_t *cursor, bool fixed)
{
    __shared__ int part[kPassThreads];
    const int per = (int)((Nc + kPassThreads - 1) / kPassThreads);
    const int64_t c0 = (int64_t)threadIdx.x * per;
    int sum = 0;
    for (int64_t c = c0; c < c0 + per && c < Nc; ++c) sum += (int)acc_count(ld256(acc + 4 * c).w, fixed);
    part[threadIdx.x] = sum;
    __syncthreads();
    for (int o = 1; o < kPassThreads; o <<= 1) {
        const int y = (int)threadIdx.x >= o ? part[threadIdx.x - o] : 0;
        __syncthreads();
        part[threadIdx.x] += y;
        __syncthreads();
    }
    int run = part[threadIdx.x] - sum;
    for (int64_t c = c0; c < c0 + per && c < Nc; ++c) {
        cursor[c] = run;
        run += (int)acc_count(ld256(acc + 4 * c).w, fixed);
    }
}

template <typename T, unsigned F>
__global__ void __launch_bounds__(kPassThreads, 4) small_steps(PassArgs<T> a, const SmallArgs s)
{
    static_assert((F & kSRD) && (F & kStream) && (F & kBin) && !(F & (kSortOut | kThermo | kEmbedded | kATApply | kATDraw)),
                  "the small-system kernel runs the plain fused SRD step");
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ typename PassScratch<F | kCoherent>::type ws[PassScratch<F | kCoherent>::count];
    const int64_t gtid = (int64_t)blockIdx.x * kPassThreads + threadIdx.x, gsize = (int64_t)gridDim.x * kPassThreads;
    int next_sort = s.sort_period > 0 ? s.first_sort : -1;
    typename Vec4<T>::type carry_p = {}, carry_v = {};
    bool have = false;
    for (int k = 0; k < s.nphases; ++k) {
        const uint64_t t = s.t0 + (uint64_t)k;
        const u32x4 b = draw(a.seed, t + 1, 0u, kDomShift);                   // a2: the grid shift of the step being binned
        a.shift[0] = (T)((u01_32(b.x) - 0.5) * s.a_cell);
        a.shift[1] = (T)((u01_32(b.y) - 0.5) * s.a_cell);
        a.shift[2] = (T)((u01_32(b.z) - 0.5) * s.a_cell);
        a.sums = s.acc3[k % 3];
        a.acc = s.acc3[(k + 1) % 3];
        a.qacc = s.qacc3[(k + 1) % 3];
        a.axis = s.axis2[t & 1];
        a.step_collide = t;
        a.step_bin = t + 1;
        const bool sort_now = k == next_sort;            // a8: sort by the cells of step t (t % sort_period == 0), on this pass's way out
        if (sort_now) {
            next_sort += s.sort_period;
            if (blockIdx.x == 0) small_scan_counts(a.sums, a.Nc, a.cursor, (F & kFixed) != 0);
            grid.sync();
            pass_body<T, F | kCoherent | kSortOut>(a, ws[threadIdx.x >> 5]);
            have = false;                                // the slot holds another particle from now on
        } else {
            pass_body<T, F | kCoherent | kCarry>(a, ws[threadIdx.x >> 5], &carry_p, &carry_v, have);
            have = true;                                 // this thread's particle stays in its registers for the next phase
        }
        double *ax = s.axis2[(t + 1) & 1], *z = s.acc3[(k + 2) % 3], *zq = s.qacc3[(k + 2) % 3];
        const bool more = k + 1 < s.nphases;
        for (int64_t c = gtid; c < a.Nc; c += gsize) {
            double nx, ny, nz;
            draw_axis(a.seed, t + 1, (uint32_t)c, nx, ny, nz);
            st256(ax + 4 * c, nx, ny, nz, 0.0);
            if (more) { st256(z + 4 * c, 0.0, 0.0, 0.0, 0.0); zq[c] = 0.0; }
        }
        grid.sync();
        if (sort_now) {                                  // the duplicate arrays hold the particles now
            auto *tp = a.pos; a.pos = a.pos_out; a.pos_out = tp;
            auto *tv = a.vel; a.vel = a.vel_out; a.vel_out = tv;
            uint32_t *tt = a.tag; a.tag = a.tag_out; a.tag_out = tt;
        }
    }
    const double *src = s.acc3[s.nphases % 3], *srcq = s.qacc3[s.nphases % 3];
    if (src != s.acc_out)
        for (int64_t c = gtid; c < a.Nc; c += gsize) {
            const f64x4 v = ld256(src + 4 * c);
            st256(s.acc_out + 4 * c, v.x, v.y, v.z, v.w);
            s.qacc_out[c] = srcq[c];
        }
}

}  // namespace mpcdk
