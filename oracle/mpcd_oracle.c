/*
 * mpcd_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU statement of the MPCD solvent step of
 * Howard, Panagiotopoulos & Nikoubashman (arXiv 1801.10187), written from
 * /root/reference/PAPER.md.  Citations are "PAPER.md:<line>" plus the section /
 * equation / algorithm.  Where the paper is silent the reading is the one in
 * SURVEY.md section 8(c) (A1..A25, G1..G4) and DESIGN.md "Readings".
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / reference
 * legs may load this library.  It shares no code, header, table or constant
 * generator with the CUDA path (paper_1801_10187_b200/csrc); neither includes
 * the other.
 *
 * Rules kept here so the file can be checked against the paper by eye:
 *   - one loop per step of the method, in the paper's order; no blocking,
 *     fusion, threading or reordering;
 *   - "native" precision (float in the mixed model, double in the fp64 model,
 *     PAPER.md:84, :195) for positions / velocities / streaming / binning;
 *     double for every cell sum and for the collision arithmetic
 *     (Alg. 1 line 5);
 *   - compiled with -O2 -ffp-contract=off (no FMA contraction, so
 *     fl(x + fl(v*dt)) is two roundings, reading A7), never -ffast-math.
 *
 * Pins (tests/test_oracle_*.py, all "-m 'not gpu'"): Philox block function vs
 * ATen's CPU engine and cuRAND's host path; uniform conversions by exactness;
 * binning vs exact-rational brute force; cell sums vs numpy bincount and exact
 * fsum; axis statistics; rotation vs scipy Rotation (handedness), RR^T = I;
 * per-cell momentum / energy conservation; one-step decorrelation closed forms;
 * Maxwell-Boltzmann KS test; viscosity 8.7 by transverse-mode
 * decay; AT conservation / Gaussianity / tag-keying; sort multiset + stability;
 * cell thermostat: drawn energies vs scipy's Gamma distribution, E_k' = E^ per cell,
 * one-collision thermalisation (test_oracle_thermostat.py); embedded solute: the
 * velocity-Verlet dimer against its closed form, forces vs numerical gradients, MD
 * momentum / bounded energy, mass-weighted collision invariants, equipartition
 * (test_oracle_embedded.py); initial condition oracle_init_*: A23 restated per particle from the
 * pinned Philox words, KS tests, zero net momentum; the rotation sense inside
 * oracle_collide_srd_beads against scipy's Rotation; oracle_collide_srd_xi bit-identical to
 * oracle_collide_srd at xi = 1 and doubling the relative velocity at xi = 2
 * (test_oracle_pins_r2.py); thermostat with beads (oracle_erel_about, oracle_embedded_energy,
 * oracle_collide_srd_beads_xi): E_k' = E^ per cell incl. the beads, cell momentum kept, agreement with the
 * pinned plain functions at xi = 1 / without beads, equipartition of hot beads under the thermostat
 * (test_oracle_embedded.py).
 * parity unpinned: none.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------- *
 * Counter-based RNG: Philox4x32-10 (the paper uses Saru keyed by (cell index,
 * timestep, seed); north_star replaces it by Philox4x32-10
 * with the same keying, reading A24).  Block function as published by Salmon
 * et al. (ref. [74] of the paper): 10 rounds of two 32x32->64
 * multiplies, key bumped by the Weyl constants between rounds.
 * ------------------------------------------------------------------------- */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Domain tags (4th counter word), reading A24. */
enum { DOM_SHIFT = 1, DOM_AXIS = 2, DOM_AT = 3, DOM_INITPOS = 4, DOM_INITVEL = 5, DOM_THERMO = 6 };

/* Philox(key = seed, ctr = (index, step_lo, step_hi, domain)), reading A24. */
static void draw_block(uint64_t seed, uint64_t step, uint32_t index, uint32_t domain, uint32_t out[4])
{
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t ctr[4] = { index, (uint32_t)step, (uint32_t)(step >> 32), domain };
    oracle_philox4x32_10(ctr, key, out);
}

/* 32-bit word -> U in (0,1): (b + 0.5) 2^-32, exact in binary64. */
double oracle_u01_32(uint32_t b) { return ((double)b + 0.5) * (1.0 / 4294967296.0); }

/* two words -> U in [0,1) with 53 bits: ((lo | hi<<32) >> 11) 2^-53. */
double oracle_u01_53(uint32_t lo, uint32_t hi)
{
    uint64_t w = ((uint64_t)lo | ((uint64_t)hi << 32)) >> 11;
    return (double)w * (1.0 / 9007199254740992.0);
}

/* ------------------------------------------------------------------------- *
 * a2. Random grid shift: one vector per step, each component uniform on
 * (-a/2, a/2) (PAPER.md:37 "random shift ... of +-a/2", :110; readings A4, A5).
 * Returned in double; the mixed model rounds it once to float (oracle_bin_f32).
 * ------------------------------------------------------------------------- */
void oracle_shift(uint64_t seed, uint64_t step, double a, double s[3])
{
    uint32_t b[4];
    draw_block(seed, step, 0u, DOM_SHIFT, b);
    for (int d = 0; d < 3; ++d) {
        double U = oracle_u01_32(b[d]);
        s[d] = (U - 0.5) * a;
    }
}

/* ------------------------------------------------------------------------- *
 * a5 (axis part). Random unit axis per cell by cylindrical projection from
 * two uniforms, keyed by (seed, step, global cell index)
 * (PAPER.md:138), stored in double.  Readings A13, A16.
 * ------------------------------------------------------------------------- */
void oracle_axis(uint64_t seed, uint64_t step, int64_t Nc, double *axis3)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t c = 0; c < Nc; ++c) {
        uint32_t b[4];
        draw_block(seed, step, (uint32_t)c, DOM_AXIS, b);
        double U1 = oracle_u01_53(b[0], b[1]);
        double U2 = oracle_u01_53(b[2], b[3]);
        double z = 2.0 * U1 - 1.0;
        double phi = two_pi * U2;
        double rho = sqrt((1.0 - z) * (1.0 + z));   /* = sqrt(1 - z^2) without the cancellation near the poles */
        axis3[3 * c + 0] = rho * cos(phi);
        axis3[3 * c + 1] = rho * sin(phi);
        axis3[3 * c + 2] = z;
    }
}

/* ------------------------------------------------------------------------- *
 * a7 (draw part). Andersen-thermostat random velocities: per particle three
 * Gaussians of variance kT/m by Box-Muller, RNG keyed by (timestep, particle
 * tag, seed).  Readings A17, A18.  Always double.
 * ------------------------------------------------------------------------- */
void oracle_at_draw(uint64_t seed, uint64_t step, int64_t N, const uint32_t *tag, double sigma, double *dv3)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t i = 0; i < N; ++i) {
        uint32_t b[4];
        draw_block(seed, step, tag[i], DOM_AT, b);
        double U0 = oracle_u01_32(b[0]), U1 = oracle_u01_32(b[1]);
        double U2 = oracle_u01_32(b[2]), U3 = oracle_u01_32(b[3]);
        double r01 = sqrt(-2.0 * log(U0));
        double r23 = sqrt(-2.0 * log(U2));
        double g0 = r01 * cos(two_pi * U1);
        double g1 = r01 * sin(two_pi * U1);
        double g2 = r23 * cos(two_pi * U3);   /* the fourth Gaussian is discarded */
        dv3[3 * i + 0] = sigma * g0;
        dv3[3 * i + 1] = sigma * g1;
        dv3[3 * i + 2] = sigma * g2;
    }
}

/* ------------------------------------------------------------------------- *
 * a8. Sort by cell: the permutation that puts particles in
 * cell order; stable (reading A20).  perm[k] = old index of the particle that
 * goes to slot k.
 * ------------------------------------------------------------------------- */
void oracle_sort_perm(int64_t N, const int32_t *cell, int64_t Nc, int64_t *perm)
{
    int64_t *start = (int64_t *)calloc((size_t)Nc + 1, sizeof(int64_t));
    for (int64_t i = 0; i < N; ++i) start[cell[i] + 1] += 1;
    for (int64_t c = 0; c < Nc; ++c) start[c + 1] += start[c];
    for (int64_t i = 0; i < N; ++i) { perm[start[cell[i]]] = i; start[cell[i]] += 1; }
    free(start);
}

/* ------------------------------------------------------------------------- *
 * NEXT-2. Maxwell-Boltzmann cell thermostat for SRD (eq. 3,
 * :157).  Per cell with N_c >= 2: a random kinetic energy E^ is drawn from the
 * Maxwell-Boltzmann (canonical) distribution of the relative kinetic energy of
 * N_c particles at kT, i.e. Gamma(shape k = 3 (N_c - 1) / 2, scale kT) (the
 * N_c - 1 relative velocities have 3 (N_c - 1) quadratic degrees of freedom),
 * by Marsaglia & Tsang's rejection method (ref. [75]):
 *     d = k - 1/3, c = 1 / sqrt(9 d);
 *     repeat: x ~ N(0,1), v = (1 + c x)^3, U ~ U(0,1);
 *             accept if v > 0 and ln U < x^2/2 + d - d v + d ln v;
 *     E^ = kT d v.
 * The Gaussian comes from the Box-Muller transformation of two uniforms
 * (PAPER.md:157).  xi = sqrt(E^ / E_k); xi = 1 for N_c < 2 (PAPER.md:157:
 * temperature undefined) and, reading A26, also when E_k = 0.
 * Reading A26 (paper silent): RNG keyed like the axis, Philox(seed, (cell,
 * t_lo, t_hi, DOM_THERMO + 256 * iteration)); words 0,1 -> the Gaussian
 * x = sqrt(-2 ln U0) cos(2 pi U1), word 2 -> U, all by (b + 1/2) 2^-32.
 * k >= 3/2 always, so the shape < 1 boost of the method is never needed.
 * ------------------------------------------------------------------------- */
void oracle_thermostat_xi(uint64_t seed, uint64_t step, int64_t Nc, double kT, const int32_t *count,
                          const double *erel, double *ehat, double *xi)
{
    const double two_pi = 6.283185307179586476925286766559;
    for (int64_t c = 0; c < Nc; ++c) {
        ehat[c] = 0.0;
        xi[c] = 1.0;
        if (count[c] < 2) continue;
        const double k = 1.5 * (double)(count[c] - 1);
        const double d = k - 1.0 / 3.0;
        const double cc = 1.0 / sqrt(9.0 * d);
        for (uint32_t it = 0;; ++it) {
            uint32_t b[4];
            draw_block(seed, step, (uint32_t)c, (uint32_t)DOM_THERMO + 256u * it, b);
            const double U0 = oracle_u01_32(b[0]), U1 = oracle_u01_32(b[1]), U = oracle_u01_32(b[2]);
            const double x = sqrt(-2.0 * log(U0)) * cos(two_pi * U1);
            const double t = 1.0 + cc * x;
            const double v = t * t * t;
            if (v > 0.0 && log(U) < 0.5 * x * x + d - d * v + d * log(v)) {
                ehat[c] = kT * d * v;
                break;
            }
        }
        if (erel[c] > 0.0) xi[c] = sqrt(ehat[c] / erel[c]);
    }
}

/* ------------------------------------------------------------------------- *
 * NEXT-1. Embedded solute (BASELINE config 5): MD beads that
 * take part in the collision.  Beads are kept in double whatever the solvent's
 * storage precision (reading A27: there are few of them), as nb x 3 arrays.
 *
 * Between collisions the beads follow "the standard MD equations of motion ...
 * using the velocity Verlet algorithm".  The only forces here are
 * harmonic bonds U = k (r - r0)^2 / 2 between consecutive beads of a linear chain
 * of chain_len beads (config 5; the paper's own polymer model, ref. [78], is not
 * specified in PAPER.md), with the minimum-image convention.
 * ------------------------------------------------------------------------- */
void oracle_md_forces(int64_t nb, int32_t chain_len, const double *pos3, double k, double r0, const double L[3], double *f3)
{
    for (int64_t i = 0; i < 3 * nb; ++i) f3[i] = 0.0;
    for (int64_t i = 0; i + 1 < nb; ++i) {
        if ((i + 1) % chain_len == 0) continue;                 /* i is the last bead of its chain */
        double d[3], r2 = 0.0;
        for (int a = 0; a < 3; ++a) {
            d[a] = pos3[3 * (i + 1) + a] - pos3[3 * i + a];
            d[a] -= L[a] * floor(d[a] / L[a] + 0.5);            /* minimum image */
            r2 += d[a] * d[a];
        }
        const double r = sqrt(r2);
        const double g = r > 0.0 ? -k * (r - r0) / r : 0.0;     /* force on bead i+1 = g d, on bead i = -g d */
        for (int a = 0; a < 3; ++a) { f3[3 * (i + 1) + a] += g * d[a]; f3[3 * i + a] -= g * d[a]; }
    }
}

/* nsub velocity-Verlet steps of length dt: v += f dt / 2m; x += v dt (wrapped into [0, L)); f = F(x); v += f dt / 2m. */
void oracle_md_verlet(int64_t nb, int32_t chain_len, double *pos3, double *vel3, const double *mass, double k, double r0,
                      const double L[3], double dt, int32_t nsub)
{
    double *f = (double *)malloc((size_t)nb * 3 * sizeof(double));
    oracle_md_forces(nb, chain_len, pos3, k, r0, L, f);
    for (int s = 0; s < nsub; ++s) {
        for (int64_t i = 0; i < nb; ++i)
            for (int a = 0; a < 3; ++a) {
                vel3[3 * i + a] += 0.5 * dt * f[3 * i + a] / mass[i];
                double x = pos3[3 * i + a] + vel3[3 * i + a] * dt;
                if (x < 0.0) x += L[a];
                if (x >= L[a]) x -= L[a];
                pos3[3 * i + a] = x;
            }
        oracle_md_forces(nb, chain_len, pos3, k, r0, L, f);
        for (int64_t i = 0; i < nb; ++i)
            for (int a = 0; a < 3; ++a) vel3[3 * i + a] += 0.5 * dt * f[3 * i + a] / mass[i];
    }
    free(f);
}

/* Mass-weighted cell mean with embedded particles ("the MD particles ... included in the collision step",
 * :159; reading A10): u = (m sum_solvent v + sum_beads m_b v_b) / (m N_solvent + sum_beads m_b). */
void oracle_embedded_means(int64_t Nc, double m, const int32_t *count, const double *sumv3, int64_t nb, const int32_t *cell_b,
                           const double *vel3_b, const double *mass_b, double *u3, double *Mc)
{
    double *P = (double *)calloc((size_t)Nc * 3, sizeof(double));
    for (int64_t c = 0; c < Nc; ++c) {
        Mc[c] = m * (double)count[c];
        for (int a = 0; a < 3; ++a) P[3 * c + a] = m * sumv3[3 * c + a];
    }
    for (int64_t i = 0; i < nb; ++i) {
        const int64_t c = cell_b[i];
        Mc[c] += mass_b[i];
        for (int a = 0; a < 3; ++a) P[3 * c + a] += mass_b[i] * vel3_b[3 * i + a];
    }
    for (int64_t c = 0; c < Nc; ++c)
        for (int a = 0; a < 3; ++a) u3[3 * c + a] = Mc[c] > 0.0 ? P[3 * c + a] / Mc[c] : 0.0;
    free(P);
}

/* SRD rotation of the beads about their cell's axis, relative to the (mass-weighted) cell mean: eq. (2), Alg. 1. */
void oracle_collide_srd_beads(int64_t nb, double *vel3, const int32_t *cell_b, const double *u3, const double *axis3,
                              double cos_a, double sin_a)
{
    for (int64_t i = 0; i < nb; ++i) {
        const int64_t c = cell_b[i];
        const double ux = u3[3 * c], uy = u3[3 * c + 1], uz = u3[3 * c + 2];
        const double nx = axis3[3 * c], ny = axis3[3 * c + 1], nz = axis3[3 * c + 2];
        const double wx = vel3[3 * i] - ux, wy = vel3[3 * i + 1] - uy, wz = vel3[3 * i + 2] - uz;
        const double ndw = nx * wx + ny * wy + nz * wz;
        const double cx = ny * wz - nz * wy, cy = nz * wx - nx * wz, cz = nx * wy - ny * wx;
        vel3[3 * i + 0] = ux + wx * cos_a + cx * sin_a + nx * ndw * (1.0 - cos_a);
        vel3[3 * i + 1] = uy + wy * cos_a + cy * sin_a + ny * ndw * (1.0 - cos_a);
        vel3[3 * i + 2] = uz + wz * cos_a + cz * sin_a + nz * ndw * (1.0 - cos_a);
    }
}

/* ... with the cell thermostat (PAPER.md:157 + :159 "including the solute particles in all stages of the algorithm";
 * reading A28): the beads' rotated relative velocities are scaled by the cell's xi like the solvent's (Alg. 1 lines 8-10). */
void oracle_collide_srd_beads_xi(int64_t nb, double *vel3, const int32_t *cell_b, const double *u3, const double *axis3,
                                 const double *xi, double cos_a, double sin_a)
{
    for (int64_t i = 0; i < nb; ++i) {
        const int64_t c = cell_b[i];
        const double ux = u3[3 * c], uy = u3[3 * c + 1], uz = u3[3 * c + 2];
        const double nx = axis3[3 * c], ny = axis3[3 * c + 1], nz = axis3[3 * c + 2];
        const double wx = vel3[3 * i] - ux, wy = vel3[3 * i + 1] - uy, wz = vel3[3 * i + 2] - uz;
        const double ndw = nx * wx + ny * wy + nz * wz;
        const double cx = ny * wz - nz * wy, cy = nz * wx - nx * wz, cz = nx * wy - ny * wx;
        double rx = wx * cos_a + cx * sin_a + nx * ndw * (1.0 - cos_a);
        double ry = wy * cos_a + cy * sin_a + ny * ndw * (1.0 - cos_a);
        double rz = wz * cos_a + cz * sin_a + nz * ndw * (1.0 - cos_a);
        rx = rx * xi[c]; ry = ry * xi[c]; rz = rz * xi[c];
        vel3[3 * i + 0] = ux + rx;
        vel3[3 * i + 1] = uy + ry;
        vel3[3 * i + 2] = uz + rz;
    }
}

/* The beads' share of a cell's relative kinetic energy and member count (eq. 3 PAPER.md:47 with the sum taken over ALL
 * particles of the cell, solvent and solute; reading A28): erel[c] += sum_beads m_b |v_b - u|^2 / 2 with the
 * mass-weighted mean u of oracle_embedded_means, ntot[c] = count[c] + beads in c.  erel comes in holding the solvent's share
 * about the SAME u (oracle_erel_about). */
void oracle_embedded_energy(int64_t Nc, const int32_t *count, int64_t nb, const int32_t *cell_b, const double *vel3_b, const double *mass_b,
                            const double *u3, double *erel, int32_t *ntot)
{
    for (int64_t c = 0; c < Nc; ++c) ntot[c] = count[c];
    for (int64_t i = 0; i < nb; ++i) {
        const int64_t c = cell_b[i];
        const double wx = vel3_b[3 * i] - u3[3 * c], wy = vel3_b[3 * i + 1] - u3[3 * c + 1], wz = vel3_b[3 * i + 2] - u3[3 * c + 2];
        erel[c] += 0.5 * mass_b[i] * (wx * wx + wy * wy + wz * wz);
        ntot[c] += 1;
    }
}

/* a4 (count part) + a9 helpers that do not depend on the storage precision. */

/* a9. Net momentum, kinetic energy and pooled temperature from the cell arrays
 * (PAPER.md:130); pooled estimator kT = sum E_rel / sum 1.5 (N_c - 1) over cells
 * with N_c >= 2 (reading A11). out = {Px, Py, Pz, KE, kT}. */
void oracle_thermo(int64_t Nc, double m, const int32_t *count, const double *sumv3, const double *ke,
                   const double *erel, double out[5])
{
    double P[3] = { 0, 0, 0 }, K = 0, E = 0, dof = 0;
    for (int64_t c = 0; c < Nc; ++c) {
        for (int d = 0; d < 3; ++d) P[d] += m * sumv3[3 * c + d];
        K += ke[c];
        if (count[c] >= 2) { E += erel[c]; dof += 1.5 * (double)(count[c] - 1); }
    }
    out[0] = P[0]; out[1] = P[1]; out[2] = P[2]; out[3] = K;
    out[4] = dof > 0 ? E / dof : 0.0;
}

/* ------------------------------------------------------------------------- *
 * Everything that touches particle storage exists once per storage precision.
 * ------------------------------------------------------------------------- */
#define REAL float
#define SUF(name) name##_f32
#include "mpcd_oracle_steps.inc"
#undef REAL
#undef SUF

#define REAL double
#define SUF(name) name##_f64
#include "mpcd_oracle_steps.inc"
#undef REAL
#undef SUF
