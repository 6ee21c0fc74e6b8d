/*
 * mpcd.h -- C ABI of the B200-native MPCD solvent step.
 *
 * The method is the multiparticle collision dynamics (MPCD) solvent of Howard,
 * Panagiotopoulos & Nikoubashman, arXiv 1801.10187.  Citations below are
 * "PAPER.md:<line>" (the text of the paper under /root/reference) plus the
 * section / equation / algorithm the line falls in; "A<n>" are the readings
 * listed in DESIGN.md where the paper is silent.
 *
 * One MPCD step (Fig. 1):
 *     stream (eq. 1) -> random grid shift + bin into cells (sect. 3.4)
 *       -> [sort by cell, every sort_period steps (sect. 3.8)]
 *       -> cell properties: count, sum v, kinetic energy in fp64 (sect. 3.5)
 *       -> collide: SRD (eq. 2, Alg. 1) or Andersen thermostat (eq. 4, sect. 3.7)
 *
 * Conventions
 *   - Every call returns int: 0 = MPCD_OK, negative = error.  Nothing throws,
 *     aborts or prints across the ABI.  mpcd_last_error() gives a description.
 *   - A handle is used from one host thread at a time.
 *   - All device work is enqueued on the handle's CUDA stream and is
 *     asynchronous, except mpcd_get_* / mpcd_set_state which synchronise that
 *     stream before returning.
 *   - "host" / "device" is stated for every pointer.  Particle vectors are
 *     N x 4 arrays of the NATIVE precision: float in MPCD_MIXED, double in
 *     MPCD_FP64 ("arrays of four-element floating-point vectors",
 *     PAPER.md:195 mixed-precision model).  The 4th components are padding (A9).
 *   - The box is [0, box[d]) per axis, periodic (A1); box[d] = n_d * a with
 *     integer n_d (A2).  Cell linear index c = ix + nx (iy + ny iz) (A8).
 *   - There is no CPU fallback: without a CUDA device every call that would
 *     compute returns MPCD_ECUDA.
 */
#ifndef MPCD_H_
#define MPCD_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MPCD_ABI_VERSION 3

/* status codes */
#define MPCD_OK      0
#define MPCD_EINVAL (-1)  /* bad argument (NULL handle, N < 1, box not a multiple of a, ...) */
#define MPCD_ENOMEM (-2)  /* the allocator (callback or cudaMalloc) failed */
#define MPCD_ECUDA  (-3)  /* a CUDA runtime call or kernel launch failed / no device */
#define MPCD_ESTATE (-4)  /* call not valid in the current state (e.g. collide without a bin) */

/* precision models */
#define MPCD_MIXED 0      /* fp32 particle data, fp64 cell sums and collision arithmetic */
#define MPCD_FP64  1      /* everything double */

/* collision rules */
#define MPCD_SRD 0        /* stochastic rotation dynamics, eq. 2 */
#define MPCD_AT  1        /* Andersen thermostat, eq. 4 */

typedef struct mpcd mpcd_t;   /* opaque */

/* Device-memory callbacks: PyTorch (or any caller) supplies every O(N) and
 * O(N_cells) buffer through these; `bytes` is a multiple of 256 and the returned
 * DEVICE pointer must be 256-byte aligned and stay valid until free_fn is called
 * with it.  alloc_fn returns NULL on failure.  When both are NULL the library
 * uses cudaMalloc / cudaFree. */
typedef void *(*mpcd_alloc_fn)(size_t bytes, void *user);
typedef void (*mpcd_free_fn)(void *device_ptr, void *user);

typedef struct mpcd_options {
    int32_t precision;     /* MPCD_MIXED (default) | MPCD_FP64 */
    int32_t rule;          /* MPCD_SRD (default) | MPCD_AT: the rule mpcd_step applies */
    double dt;             /* collision time, default 0.1 */
    double alpha;          /* SRD angle in radians (A15), default 130 deg */
    int32_t sort_period;   /* sort every k steps, t % k == 0 (A21); 0 = never; default 25 */
    int32_t cell_energy;   /* 1 (default): accumulate the per-cell kinetic energy every step (sect. 3.5);
                              0: momentum and count only (KE is then computed on demand by mpcd_get_cells / thermo) */
    int32_t init_state;    /* 1 (default): draw the initial condition on the device (A23); 0: leave the particle
                              arrays uninitialised, the caller must mpcd_set_state before stepping */
    int32_t thermostat;    /* 1: Maxwell-Boltzmann cell thermostat for the SRD rule (PAPER.md:45-50 eq. 3, :157): the relative
                              velocities of every cell with N_c >= 2 are scaled by xi = sqrt(E^/E_k), E^ ~ Gamma(3 (N_c - 1) / 2, kT);
                              default 0.  Ignored by the AT rule, which is isothermal by construction */
    int32_t deterministic; /* 1: deterministic accumulation (NEXT-3; PAPER.md:124-126 names the alternative): the cell sums are 64-bit
                              fixed-point integers (40 fractional bits), so the trajectory is bit-reproducible whatever the order of
                              warps, atomics and particles in memory; results stay within the mixed-model tolerance of the fp64
                              sums.  Mixed model + SRD rule only (MPCD_EINVAL otherwise; no embedded beads); default 0 */
    int32_t brick;         /* 1: the sort (sect. 3.8) orders the particles BRICK-major -- cells grouped in bricks of
                              brick[0] x brick[1] x brick[2] cells (mpcd_stats.brick; compile-time), bricks x-fastest over
                              ceil(n_d / brick[d]) per axis, cells x-fastest inside a brick -- and mpcd_step runs its steady-state kernel
                              with one thread block per brick and the cell side of the step in shared memory.  The
                              order inside the sort is free (A20): results are the same up to fp64 summation order, with one
                              qualification.  The block-local partial sums are fixed-point: with unit = the power of two >=
                              sqrt(kT/m) of mpcd_create, a velocity component is rounded to 2^-49 unit and |v|^2 to 2^-44 unit^2
                              before it is added (exact for fp32 state; for MPCD_FP64 about 16x coarser than a double at
                              |v| ~ unit: cell means move by <= 2^-50 unit, velocities after a collision by < 1e-13 unit, a
                              thermostat factor by ~1e-14 relative -- inside the 1e-12 tolerance, but not "summation order"
                              only).  A particle with any |v_d| >= 8 unit does not fit that format and takes the per-particle
                              route (direct fp64 atomics): correct, but slow if it is most of them, e.g. a state loaded with
                              mpcd_set_state at > 60x the kT given to mpcd_create or in a bulk drift above 8 unit.
                              0 (default): ascending cell index and the warp-level kernel (the faster of the two on the north-star workload,
                              DESIGN.md 5.1) */
    void *stream;          /* cudaStream_t the library enqueues on; NULL = the legacy default stream */
    mpcd_alloc_fn alloc_fn;
    mpcd_free_fn free_fn;
    void *alloc_user;
} mpcd_options;

/* Fills *opt with the defaults above.  opt: host. */
int mpcd_default_options(mpcd_options *opt);

/*
 * mpcd_create -- allocate a solvent of N particles of mass m in a periodic box
 * `box` (host, 3 doubles) of cubic collision cells of edge a, at
 * temperature kT, with RNG seed `seed` ("user-supplied seed").
 * Errors: MPCD_EINVAL if out == NULL, N < 1, N >= 2^31, a, m, kT <= 0, box[d]
 * not an integer multiple of a (|box/a - n_d| <= 1e-9) or n_x n_y n_z >= 2^31;
 * MPCD_ENOMEM / MPCD_ECUDA on allocation / device failure (then *out = NULL).
 * Initial state (A23): positions uniform in the box, velocities N(0, kT/m) with
 * the mean removed, tags 0..N-1, step counter 0.
 * The handle is owned by the caller until mpcd_destroy.
 */
int mpcd_create(mpcd_t **out, const double box[3], int64_t N, double a, double m, double kT, uint64_t seed);
int mpcd_create_ex(mpcd_t **out, const double box[3], int64_t N, double a, double m, double kT, uint64_t seed,
                   const mpcd_options *opt /* host, may be NULL */);
int mpcd_destroy(mpcd_t *h);

/* a1. Streaming, eq. 1: r <- r + v dt in native precision (two
 * roundings, no FMA, A7), wrapped into [0, L).  Invalidates the current bin. */
int mpcd_stream(mpcd_t *h);

/* a2-a5. For the current step counter t: draw the grid shift from
 * Philox(seed, t) (A4, A5), bin every particle with the shift
 * applied during binning only (A6), accumulate per cell the count,
 * sum of velocities and kinetic energy in fp64, and draw per cell
 * the random unit axis from Philox(seed, t, cell) by cylindrical projection
 * (A13).  The mean velocity u = S / N_c and the cell temperature
 * (eq. 3; A11) are functions of those sums: the collision forms u where
 * it uses it, mpcd_get_cells / mpcd_get_thermo report both.  With the thermostat
 * on, also the scale factor xi of every cell; with embedded beads,
 * their binning and mass-weighted sums.  Idempotent for a given (state, t).  Direct
 * accumulation has no capacity, so the overflow / rebuild path of PAPER.md:110 does
 * not exist. */
int mpcd_shift_and_bin(mpcd_t *h);

/* a6. SRD collision, eq. 2 / Algorithm 1, angle alpha in
 * radians about each cell's axis, fp64 arithmetic, native-precision store.
 * Needs a valid bin for the current step (else MPCD_ESTATE).  Does not advance
 * the step counter.  Invalidates the cell sums (velocities changed). */
int mpcd_collide_srd(mpcd_t *h, double alpha);

/* a7. Andersen-thermostat collision, eq. 4, sect. 3.7 PAPER.md:163:
 * per-particle Gaussians from Philox(seed, t, tag) by Box-Muller (A17, A18), a
 * second per-cell reduction, v <- u + dv - sum(dv)/N_c.  Same preconditions. */
int mpcd_collide_at(mpcd_t *h);

/* a8. Sort by cell, sect. 3.8: reorder pos, vel, tag and cell so
 * that the particles of a cell are contiguous, using the current bin (MPCD_ESTATE
 * if none).  Cells follow each other in ascending SORT KEY: the cell index with
 * opt.brick = 0; with opt.brick = 1, for cell (ix, iy, iz) and brick edges
 * B = mpcd_stats.brick[0..2], nb_d = ceil(n_d / B_d):
 *   key = (((iz/Bz) nb_y + iy/By) nb_x + ix/Bx) Bx By Bz + ((iz%Bz) By + iy%By) Bx + ix%Bx.
 * Order within a cell is unspecified (A20).  Tags travel with particles. */
int mpcd_sort(mpcd_t *h);

/* nsteps x { stream; shift_and_bin; sort if sort_period and t % sort_period == 0;
 * collide per opt.rule; t += 1 } (A3).  Internally the collision of
 * step t is fused with the streaming / binning / accumulation of step t + 1
 * (one pass over the particles per step), and on sort steps that pass also writes
 * the particles out in cell order; the result is the same as the unfused sequence
 * of calls up to fp64 summation order (exactly the same with opt.deterministic).
 * A system small enough to sit on the device as one resident wave of thread blocks
 * (plain SRD rule) runs its steps, sorts included, in one cooperative launch
 * (DESIGN.md 5.4); the results are the same.  All work is enqueued on the handle's
 * stream; the call does not synchronise. */
int mpcd_step(mpcd_t *h, int32_t nsteps);

/* Copies the particle state to caller-owned HOST buffers (any may be NULL):
 * pos4 / vel4 = N x 4 native precision, tag = N x u32, cell = N x i32 (last bin;
 * unspecified if none), step = the step counter.  Order is the current (possibly
 * sorted) order: compare by tag.  Synchronises the stream. */
int mpcd_get_state(mpcd_t *h, void *pos4, void *vel4, uint32_t *tag, int32_t *cell, uint64_t *step);

/* Overwrites the particle state from HOST buffers (pos4, vel4 required, N x 4
 * native precision; tag may be NULL = 0..N-1) and sets the step counter.
 * Positions must lie in [0, box).  Invalidates the bin.  Synchronises. */
int mpcd_set_state(mpcd_t *h, const void *pos4, const void *vel4, const uint32_t *tag, uint64_t step);

/* Per-cell results of the last mpcd_shift_and_bin to HOST buffers (any may be
 * NULL): count[Nc] i32, sumv3[Nc*3], ke[Nc], u3[Nc*3], axis3[Nc*3], kTc[Nc],
 * all double.  MPCD_ESTATE if the cell sums are not valid (no bin, or a
 * collision has changed the velocities since). */
int mpcd_get_cells(mpcd_t *h, int32_t *count, double *sumv3, double *ke, double *u3, double *axis3, double *kTc);

/* The shift used by the last bin, as applied (mixed mode: the fp32 value, A5).  s: host. */
int mpcd_get_shift(mpcd_t *h, double s[3]);

/* NEXT-1. Embedded solute (BASELINE config 5): nb beads of linear chains of chain_len beads each
 * (nb a multiple of chain_len, chain_len <= 512), bead i of mass mass[i], consecutive beads of a chain joined by the
 * harmonic bond U = k (r - r0)^2 / 2 (minimum image).  From then on the beads take part in the SRD collision -- the
 * cell mean becomes (m sum_solvent v + sum_beads m_b v_b) / (m N_c + sum_beads m_b) and the beads are rotated about
 * their cell's axis like the solvent -- and wherever the solvent streams over dt (mpcd_stream, mpcd_step) the beads
 * are advanced by md_substeps velocity-Verlet steps of dt / md_substeps.  Beads are kept in double whatever the
 * precision model (A27).  pos3, vel3: HOST, nb x 3 doubles, positions in [0, box); mass: HOST, nb doubles.  Needs the
 * SRD rule without deterministic accumulation (MPCD_EINVAL otherwise); the sort leaves the beads alone;
 * mpcd_get_cells / mpcd_get_thermo report the solvent only.  With opt.thermostat = 1 the beads are particles of their cell
 * for the thermostat too (A28): E_k of eq. 3 sums m_i |v_i - u|^2 / 2 over solvent and beads,
 * the drawn energy follows the cell's particle count incl. beads, and xi scales the beads' relative velocities as well.  Calling it again with the same nb replaces the state. */
int mpcd_set_embedded(mpcd_t *h, int64_t nb, const double *pos3, const double *vel3, const double *mass, int32_t chain_len, double k, double r0,
                      int32_t md_substeps);
/* Bead state to HOST buffers (any may be NULL): pos3, vel3 nb x 3 doubles, cell nb x i32 (last binning).  Synchronises. */
int mpcd_get_embedded(mpcd_t *h, double *pos3, double *vel3, int32_t *cell);

/* The thermostat's scale factor xi per cell for the current bin (opt.thermostat = 1; MPCD_ESTATE otherwise or when the
 * cell sums are not valid).  xi: host, Nc doubles.  Test accessor for the parity of PAPER.md:157. */
int mpcd_get_xi(mpcd_t *h, double *xi);

/* a9. Net momentum P (3), kinetic energy and pooled temperature (A11) of the
 * CURRENT velocities by device-wide reduction.  If no bin is valid
 * one is made for the current step.  Outputs: host, any may be NULL. */
int mpcd_get_thermo(mpcd_t *h, double P[3], double *KE, double *kT);

typedef struct mpcd_stats {
    int64_t N;              /* particles */
    int64_t Nc;             /* cells */
    int32_t n[3];           /* cells per axis */
    int32_t max_occupancy;  /* largest cell count seen in the last bin */
    uint64_t step;          /* step counter */
    uint64_t kernel_launches; /* kernels launched by this handle so far */
    uint64_t sorts;         /* sorts done so far */
    uint64_t device_bytes;  /* bytes obtained from the allocator */
    int32_t brick[4];       /* brick edges (cells) per axis and the window halo of the brick kernel; zeros with opt.brick = 0 */
} mpcd_stats;
int mpcd_get_stats(mpcd_t *h, mpcd_stats *out /* host */);

/* Opt-in per-kernel timing.  While on, every launch group is bracketed by a CUDA event
 * pair on the handle's stream (this costs a little, so leave it off for throughput runs).
 * mpcd_get_profile synchronises and returns, per kind, the summed device time in ms and the
 * number of launch groups since profiling was switched on.  ms, count: host, may be NULL. */
#define MPCD_PROF_FUSED    0   /* collide(t) + stream + bin + accumulate(t+1): the steady-state step kernel */
#define MPCD_PROF_BIN      1   /* [stream +] bin + accumulate without a collision */
#define MPCD_PROF_COLLIDE  2   /* collision only */
#define MPCD_PROF_CELLS    3   /* per-cell helper kernels outside the fused step (axes, zeroing) */
#define MPCD_PROF_SORT     4   /* scan of the cell counts; the scatter pass when the sort is not fused into a step kernel */
#define MPCD_PROF_OTHER    5
#define MPCD_PROF_FUSED_SORT 6 /* the fused step kernel on a sort step: it also writes the particles out in cell order */
#define MPCD_PROF_KINDS    7
int mpcd_set_profiling(mpcd_t *h, int32_t on);
int mpcd_get_profile(mpcd_t *h, double ms[MPCD_PROF_KINDS], uint64_t count[MPCD_PROF_KINDS]);

/* DEVICE pointers of the current particle arrays (for zero-copy inspection; they
 * change after a sort).  Any output may be NULL. */
int mpcd_device_ptrs(mpcd_t *h, void **pos4, void **vel4, uint32_t **tag, int32_t **cell);

/* Static description of the last error on this handle (or of the last failed
 * mpcd_create when h == NULL).  Never NULL. */
const char *mpcd_last_error(const mpcd_t *h);

/*
 * mpcd_cell_sums_static -- a3 + a4 without a handle and without any allocation: bins N particles into the shifted grid
 * (A6, A8) and accumulates per cell the count, the sum of velocities and the kinetic energy in fp64
 * (PAPER.md:118-124), exactly as mpcd_shift_and_bin does (same binning arithmetic, same warp-level reduction; the sums
 * agree with mpcd_get_cells up to fp64 summation order, the counts exactly).
 *
 * It exists for callers that cannot obtain device memory at the point where they need the cell sums: code running
 * beside an application that has given all device memory to another pool (a framework's caching allocator, an MPS
 * client with a fixed memory limit), so that cudaMalloc fails; and code in a time-critical loop that cannot afford
 * cudaMalloc / cudaFree because they may synchronise the device.  The call uses no cudaMalloc, no cudaFree, no
 * allocator callback and no allocating library routine.  The per-cell accumulators it needs sit in a fixed array of
 * MPCD_STATIC_MAX_CELLS * 40 bytes (1.25 MiB) inside the library, which each GPU holds from the time the library's
 * device code is loaded onto it until the process exits.
 *
 * Arguments.  pos4, vel4: DEVICE, N x 4 of the native precision (float for MPCD_MIXED, double for MPCD_FP64), read
 * only; the 4th components are ignored.  Positions must lie in [0, n[d] a) per axis (as for mpcd_set_state); a particle
 * that does not is left out of every sum (nothing is written out of bounds).  n: HOST, cells per axis; a: cell edge;
 * shift: HOST, the grid shift as applied, |shift[d]| < a (mixed model: pass the fp32 value, as mpcd_get_shift returns
 * it); m: particle mass.  Outputs, DEVICE, caller-owned, any may be NULL: count[Nc] int32, sumv3[Nc * 3] and ke[Nc]
 * double, Nc = n[0] n[1] n[2], cell index c = ix + n[0] (iy + n[1] iz), ke = m sum |v|^2 / 2.  N = 0 gives zeros.
 * stream: cudaStream_t of the CURRENT device (NULL = legacy default stream); the work is enqueued there and the call
 * does not synchronise.
 *
 * Errors: MPCD_EINVAL for Nc > MPCD_STATIC_MAX_CELLS (the message names the limit), N < 0 or >= 2^31, missing
 * pointers, bad precision, a, m <= 0, |shift| >= a; MPCD_ECUDA for a runtime failure or no device.  The text is
 * returned by mpcd_cell_sums_static_error() (per host thread; never NULL), not by mpcd_last_error.
 *
 * Sharing.  There is one scratch array per GPU and every call on that GPU uses it; it keeps the previous call's sums,
 * so each call first clears the part it will use (on `stream`).  Two calls whose device work can overlap -- different
 * streams, or different host threads -- race on it and give wrong sums: keep the calls of one GPU on one stream, or
 * order them with events.
 *
 * First call.  The first call on each device (with that device current) looks up the array's device address
 * (cudaGetSymbolAddress) and the SM count, under a lock, and keeps them; make that first call before any stream
 * capture begins.
 */
#define MPCD_STATIC_MAX_CELLS 32768
int mpcd_cell_sums_static(const void *pos4, const void *vel4, int64_t N, int32_t precision, const int32_t n[3], double a,
                          const double shift[3], double m, int32_t *count, double *sumv3, double *ke, void *stream);
const char *mpcd_cell_sums_static_error(void);

/* Library identification: ABI version; build string (arch, compiler). */
int mpcd_abi_version(void);
const char *mpcd_build_info(void);

/* Test hook: the library's own Philox4x32-10 block function evaluated ON THE
 * DEVICE for n (ctr, key) pairs; ctr4: host n x 4 u32, key2: host n x 2 u32,
 * out4: host n x 4 u32.  Used to pin the CUDA generator against the oracle and
 * cuRAND. */
int mpcd_test_philox(const uint32_t *ctr4, const uint32_t *key2, uint32_t *out4, int64_t n);

#ifdef __cplusplus
}
#endif
#endif /* MPCD_H_ */
