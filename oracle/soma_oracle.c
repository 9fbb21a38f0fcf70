/*
 * soma_oracle.c -- plain, slow, obviously-correct CPU oracle for the SCMF Monte-Carlo step of
 * SOMA (Schneider & Mueller, arXiv:1711.03828).
 *
 * THIS FILE IS TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no code
 * with the CUDA path under paper_1711_03828_b200/csrc/ (no common header, helper, table or
 * constant generator); neither side includes or imports the other.
 *
 * It follows the paper's algorithm step by step, in the paper's order:
 *   stage 1  densities n_i(c) (Eq. 4) and fields omega_i(c) (Eq. 12)
 *   stage 2  one Monte-Carlo sweep with omega frozen, iterating molecules in
 *            parallel and, inside a molecule, the independent sets sequentially -- Code 2,
 *            with the local-displacement Metropolis move of PAPER.md:206 and
 *            the energies of Eq. 2 and Eq. 15.
 * Where the paper is silent the readings R1..R14 of DESIGN.md ("Readings of the paper") apply;
 * each is named at the line that uses it.
 *
 * Arithmetic: the decision path is IEEE binary32 with every rounding written out (compile with
 * -ffp-contract=off; fused multiply-adds appear only as explicit fmaf()).  Self-checks that need
 * more precision live in tests/, in float64, and do not call back into this file for their
 * expected values.
 *
 * Pins (tests/test_oracle_*.py, all `-m "not gpu"`): Philox known-answer vectors + cuRAND host
 * generator; brute-force total-Hamiltonian differences; exact Metropolis ratio; Gaussian bond
 * statistics / <Re^2> / <Rg^2> of ideal chains; Boltzmann occupation of a two-level field;
 * histogram sum rules and brute-force counting; hand-computed field values and a finite
 * difference of Eq. 5.  Unpinned: exact trajectories (the paper prints none) -- the sweep as a
 * whole is pinned only through those statistical and incremental-vs-brute-force checks.
 * The Smart-MC proposal (sweep kind 2) follows the textbook Rossky-Doll-Friedman scheme because
 * the paper gives no formula (PAPER.md:206 names refs [28,29] only): its stationary distribution
 * is pinned, its exact formula is "parity unpinned" against the paper.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_MAX_TYPES 8

/* System description handed in by the caller (ctypes.Structure mirror in oracle/__init__.py). */
typedef struct {
    uint32_t        n_specs;       /* number of molecular architectures (all linear chains)     */
    const uint64_t *spec_n_chains; /* [n_specs] chains of each architecture, stored contiguously */
    const uint32_t *spec_n_beads;  /* [n_specs] beads per chain                                  */
    const uint8_t  *types;         /* concatenated per-architecture bead types                   */
    uint32_t        n_types;       /* n_t of PAPER.md:120                                        */
    uint32_t        N_ref;         /* reference N of PAPER.md:157                                */
    float           box[3];        /* L_x, L_y, L_z in units of R_e0                             */
    int32_t         grid[3];       /* cells per axis; Delta L_a = box[a]/grid[a]                 */
    float           chiN[ORACLE_MAX_TYPES * ORACLE_MAX_TYPES]; /* chi_ij N, symmetric, 0 diagonal */
    float           kappaN;        /* kappa N                                                    */
    float           A;             /* maximal step length a of PAPER.md:206                      */
    uint64_t        seed;
    int32_t         hamiltonian;   /* 0: K^0_inter (Eq. 7), 1: K^1_inter (Eq. 8)                 */
    float           smc_step;      /* Smart-MC step a_s in R_e0^2                                */
    int32_t         set_order;     /* 0: sets in the order even, odd (R11); 1: random order per   */
                                   /*    molecule and sweep (Code 2; R21)        */
    uint32_t        field_every;   /* omega refreshed after every field_every-th sweep (R22); 0, 1: every sweep */
    int32_t         scheme;        /* 0: independent sets (Code 2); 1: molecule-parallel, N random picks */
                                   /*    per molecule and sweep (Code 1; R24)           */
    const uint32_t *spec_n_bonds;  /* nullable; [n_specs] bonds of each architecture, 0 = linear chain   */
    const uint32_t *bonds;         /* concatenated (i, j) monomer pairs of the architectures with bonds  */
    const float    *ext_field;     /* nullable, [n_types][cells]: static external field added to omega   */
    const uint8_t  *forbidden;     /* nullable, [cells]: 1 = no particle may enter this cell             */
    /* A part of a larger system (molecules distributed over ranks).  nullable:         */
    const uint64_t *spec_first_bead; /* [n_specs] index in the whole system of the first bead of this part's */
                                   /* molecules of each architecture = their Philox counter words (R3)    */
    uint64_t        global_n_beads; /* beads of the whole system (rho_0 of Eq. 12); 0: this system is whole */
} oracle_system;

/* ------------------------------------------------------------------------------------------ */
/* a0  Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  PAPER.md:368 describes the           */
/* "hashed from the thread ID and the time step" generator family; north_star fixes Philox.     */
/* ------------------------------------------------------------------------------------------ */
void soma_oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        const uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        const uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n1 = lo1;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        const uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; /* key schedule between rounds (the bump after round 10 is unused) */
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* Reading R3: counter = (global bead index, sweep lo32, sweep hi32, tag), key = (seed lo32,
 * seed hi32), tag = (kind << 8) | sub; kind 0 = initial state, 1 = local move, 2 = Smart-MC. */
static void draw(const oracle_system *s, uint64_t bead, uint64_t sweep, uint32_t kind, uint32_t sub,
                 uint32_t out[4])
{
    const uint32_t ctr[4] = { (uint32_t)bead, (uint32_t)sweep, (uint32_t)(sweep >> 32),
                              (kind << 8) | sub };
    const uint32_t key[2] = { (uint32_t)s->seed, (uint32_t)(s->seed >> 32) };
    soma_oracle_philox4x32_10(ctr, key, out);
}

/* Reading R4: top 23 bits of a word become the mantissa of a float in [1,2), exactly. */
float soma_oracle_u23(uint32_t w)
{
    const uint32_t bits = 0x3F800000u | (w >> 9);
    float f;
    memcpy(&f, &bits, sizeof f);
    return f;
}

/* ------------------------------------------------------------------------------------------ */
/* bookkeeping of the chain-major bead array                                                    */
/* ------------------------------------------------------------------------------------------ */
uint64_t soma_oracle_n_beads(const oracle_system *s)
{
    uint64_t nb = 0;
    for (uint32_t a = 0; a < s->n_specs; ++a) nb += s->spec_n_chains[a] * s->spec_n_beads[a];
    return nb;
}

static int64_t n_cells(const oracle_system *s)
{
    return (int64_t)s->grid[0] * s->grid[1] * s->grid[2];
}

/* ------------------------------------------------------------------------------------------ */
/* Pi_c of Eq. 4: the cell that contains r.  Reading R7: coordinates are      */
/* stored unwrapped; per axis the position in units of the box length is the fp32 number         */
/* t = fl32(x * fl32(1/L)), and the cell is floor(t n) mod n = floor(t n) - n floor(t), both      */
/* floors taken of the exact values (t has 24 significant bits and n < 2^24, so the product is    */
/* exact in a double): half-open cells [i, i+1) DeltaL, periodic, no rounding after t.           */
/* Supported domain |t n| < 2^22.                                                                 */
/* ------------------------------------------------------------------------------------------ */
static int32_t axis_cell(float x, float L, int32_t n)
{
    const float inv_L = (float)(1.0 / (double)L);
    const float t = x * inv_L;
    const double k = floor((double)t * (double)n); /* exact product, exact floor */
    const double m = floor((double)t);
    return (int32_t)(k - (double)n * m);           /* in 0 .. n-1 */
}

int64_t soma_oracle_cell_index(const oracle_system *s, float x, float y, float z)
{
    const int32_t ix = axis_cell(x, s->box[0], s->grid[0]);
    const int32_t iy = axis_cell(y, s->box[1], s->grid[1]);
    const int32_t iz = axis_cell(z, s->box[2], s->grid[2]);
    return ((int64_t)ix * s->grid[1] + iy) * s->grid[2] + iz; /* R8: [ix][iy][iz], z fastest */
}

/* ------------------------------------------------------------------------------------------ */
/* a3  occupation numbers n_i(c) = rho_0 DeltaL^3 phi_i(c), Eq. 4           */
/* counts[type][cell], uint32                                                                   */
/* ------------------------------------------------------------------------------------------ */
void soma_oracle_histogram(const oracle_system *s, const float *x, const float *y, const float *z,
                           uint32_t *counts)
{
    const int64_t cells = n_cells(s);
    memset(counts, 0, sizeof(uint32_t) * (size_t)cells * s->n_types);
    uint64_t first = 0;
    const uint8_t *types = s->types;
    for (uint32_t a = 0; a < s->n_specs; ++a) {
        const uint32_t N = s->spec_n_beads[a];
        const int64_t n_mol = (int64_t)s->spec_n_chains[a];
#ifdef _OPENMP
#pragma omp parallel for schedule(static)
#endif
        for (int64_t m = 0; m < n_mol; ++m)
            for (uint32_t j = 0; j < N; ++j) {
                const uint64_t g = first + (uint64_t)m * N + j;
                uint32_t *slot = &counts[(int64_t)types[j] * cells + soma_oracle_cell_index(s, x[g], y[g], z[g])];
#ifdef _OPENMP
#pragma omp atomic
#endif
                *slot += 1u;
            }
        first += (uint64_t)n_mol * N;
        types += N;
    }
}

/* ------------------------------------------------------------------------------------------ */
/* a4  interaction fields, Eq. 12, both Hamiltonian options.                 */
/* phi_i(c) = n_i(c) / (rho_0 DeltaL^3) with rho_0 DeltaL^3 = beads / cells;*/
/* chi_0 = chiN / N_ref, kappa_0 = kappaN / N_ref.  Reading R9: each unordered    */
/* pair once in Eq. 7-8, so Eq. 12 holds as printed.  omega[type][cell], fp32.                   */
/* ------------------------------------------------------------------------------------------ */
/* External fields, reading R23.  "The second specifies a linear attraction for the */
/* particle of a specific type": a static, type-specific field ext_i(c) added to omega_i(c).  "The   */
/* first prevents any particle from entering a specific grid cell": omega_i(c) = +infinity for every */
/* type in such a cell, so Eq. 15 gives dE_nb = +inf for a move into it and the Metropolis rule       */
/* rejects it (a bead that starts inside may leave: dE_nb = -inf).  The mean occupancy rho_0 DeltaL^3 */
/* of PAPER.md:125, 241 then refers to the accessible volume: beads / (cells - forbidden cells).      */
void soma_oracle_fields(const oracle_system *s, const uint32_t *counts, float *omega)
{
    const int64_t cells = n_cells(s);
    const uint32_t nt = s->n_types;
    int64_t allowed = cells;
    if (s->forbidden)
        for (int64_t c = 0; c < cells; ++c) allowed -= s->forbidden[c] ? 1 : 0;
    const uint64_t beads_all = s->global_n_beads ? s->global_n_beads : soma_oracle_n_beads(s);
    const float inv_nbar = (float)((double)allowed / (double)beads_all);
    const float kappa0 = (float)((double)s->kappaN / (double)s->N_ref);
    float chi0[ORACLE_MAX_TYPES][ORACLE_MAX_TYPES], half_chi0[ORACLE_MAX_TYPES][ORACLE_MAX_TYPES];
    for (uint32_t i = 0; i < nt; ++i)
        for (uint32_t k = 0; k < nt; ++k) {
            chi0[i][k] = (float)((double)s->chiN[i * ORACLE_MAX_TYPES + k] / (double)s->N_ref);
            half_chi0[i][k] = (float)(0.5 * (double)s->chiN[i * ORACLE_MAX_TYPES + k] / (double)s->N_ref);
        }
    for (int64_t c = 0; c < cells; ++c) {
        float phi[ORACLE_MAX_TYPES];
        for (uint32_t i = 0; i < nt; ++i) phi[i] = (float)counts[(int64_t)i * cells + c] * inv_nbar;
        float sum = phi[0];
        for (uint32_t i = 1; i < nt; ++i) sum = sum + phi[i];
        const float P = kappa0 * (sum - 1.0f); /* kappa_0 (sum_k phi_k - 1) */
        for (uint32_t i = 0; i < nt; ++i) {
            float w = P;
            for (uint32_t k = 0; k < nt; ++k) {
                if (k == i) continue;
                if (s->hamiltonian == 0)
                    w = w - half_chi0[i][k] * (phi[i] - phi[k]); /* Eq. 12, K^0 line */
                else
                    w = w + chi0[i][k] * phi[k];                 /* Eq. 12, K^1 line */
            }
            if (s->ext_field) w = w + s->ext_field[(int64_t)i * cells + c];
            if (s->forbidden && s->forbidden[c]) w = INFINITY;
            omega[(int64_t)i * cells + c] = w;
        }
    }
}

/* ------------------------------------------------------------------------------------------ */
/* a1/a2  local random displacement + Metropolis                                 */
/* ------------------------------------------------------------------------------------------ */

/* Reading R5: trial displacement "uniformly chosen with a maximal step length, a, along each
 * Cartesian direction": d = A * ((2k+1) 2^-23 - 1), k = top 23 bits -- 2^23 equidistant values,
 * symmetric about 0, inside the open interval (-A, A); acceptance uniform u = k 2^-23 in [0,1). */
void soma_oracle_local_proposal(const oracle_system *s, uint64_t bead, uint64_t sweep, float d[3],
                                float *u)
{
    uint32_t w[4];
    draw(s, bead, sweep, 1u, 0u, w);
    const float c1 = (float)(2.0 * (double)s->A);
    const float c0 = (float)((double)s->A * (ldexp(1.0, -23) - 3.0));
    d[0] = fmaf(soma_oracle_u23(w[0]), c1, c0);
    d[1] = fmaf(soma_oracle_u23(w[1]), c1, c0);
    d[2] = fmaf(soma_oracle_u23(w[2]), c1, c0);
    *u = soma_oracle_u23(w[3]) - 1.0f;
}

/* Energy change of displacing one bead by d with everything else fixed.
 * Bonded (Eq. 2; k_0 = 3 (N_ref - 1) / R_e0^2 from b_0 = sqrt(3/k_0), PAPER.md:161,
 * with R_e0^2 = (N_ref - 1) b_0^2 -- reading R1):
 *     dE_b = k_0/2 sum_nb ( |b_nb + d|^2 - |b_nb|^2 ) = k_0/2 ( 2 d.s + m |d|^2 ),
 *     b_nb = r - r_nb,  s = sum_nb b_nb,  m = number of bonded neighbours
 * (the factored form avoids the cancellation of two nearly equal squares; reading R6 fixes the
 * fp32 operation order below).  Non-bonded (Eq. 15): dE_nb = omega_k(c') - omega_k(c),
 * with c' the cell of the stored trial position r' = fl32(r + d); exactly 0 when c' == c.
 * has_l / has_r say whether the chain neighbours at bead-1 / bead+1 exist. */
/* The same with the bond sum s = sum_nb (r - r_nb) and the number of bonded neighbours m handed in
 * (any molecular architecture). */
static void local_delta_e_core(const oracle_system *s, const float *x, const float *y, const float *z,
                               const float *omega, uint64_t bead, float sx, float sy, float sz, float mf,
                               uint32_t type, const float d[3], float *dE_b, float *dE_nb, float r_new[3]);

void soma_oracle_local_delta_e(const oracle_system *s, const float *x, const float *y, const float *z,
                               const float *omega, uint64_t bead, int has_l, int has_r, uint32_t type,
                               const float d[3], float *dE_b, float *dE_nb, float r_new[3])
{
    const float rx = x[bead], ry = y[bead], rz = z[bead];
    /* s = sum over existing neighbours of (r - r_nb); an absent neighbour contributes exactly 0 */
    const float blx = has_l ? rx - x[bead - 1] : 0.0f, brx = has_r ? rx - x[bead + 1] : 0.0f;
    const float bly = has_l ? ry - y[bead - 1] : 0.0f, bry = has_r ? ry - y[bead + 1] : 0.0f;
    const float blz = has_l ? rz - z[bead - 1] : 0.0f, brz = has_r ? rz - z[bead + 1] : 0.0f;
    const float mf = (float)((has_l ? 1 : 0) + (has_r ? 1 : 0));
    local_delta_e_core(s, x, y, z, omega, bead, blx + brx, bly + bry, blz + brz, mf, type, d, dE_b, dE_nb, r_new);
}

static void local_delta_e_core(const oracle_system *s, const float *x, const float *y, const float *z,
                               const float *omega, uint64_t bead, float sx, float sy, float sz, float mf,
                               uint32_t type, const float d[3], float *dE_b, float *dE_nb, float r_new[3])
{
    const float hk = (float)(1.5 * ((double)s->N_ref - 1.0)); /* k_0 / 2 with R_e0 = 1 */
    const float rx = x[bead], ry = y[bead], rz = z[bead];
    const float ds = fmaf(d[2], sz, fmaf(d[1], sy, d[0] * sx));
    const float dd = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
    *dE_b = hk * fmaf(2.0f, ds, mf * dd);

    r_new[0] = rx + d[0];
    r_new[1] = ry + d[1];
    r_new[2] = rz + d[2];
    const int64_t c_old = soma_oracle_cell_index(s, rx, ry, rz);
    const int64_t c_new = soma_oracle_cell_index(s, r_new[0], r_new[1], r_new[2]);
    if (c_new == c_old) {
        *dE_nb = 0.0f;
    } else {
        const int64_t cells = n_cells(s);
        *dE_nb = omega[(int64_t)type * cells + c_new] - omega[(int64_t)type * cells + c_old];
    }
}

/* Metropolis acceptance (reading R10: accept iff dE <= 0 or u < exp(-dE)). */
int soma_oracle_metropolis(float dE, float u)
{
    if (dE <= 0.0f) return 1;
    return u < expf(-dE) ? 1 : 0;
}

/* "MC scheme for particle ip" of Code 1/2, local-displacement variant. */
static int mc_local(const oracle_system *s, float *x, float *y, float *z, const float *omega,
                    uint64_t bead, uint64_t bead_rng, int has_l, int has_r, uint32_t type,
                    uint64_t sweep)
{
    float d[3], u, dE_b, dE_nb, r_new[3];
    soma_oracle_local_proposal(s, bead_rng, sweep, d, &u);
    soma_oracle_local_delta_e(s, x, y, z, omega, bead, has_l, has_r, type, d, &dE_b, &dE_nb, r_new);
    const float dE = dE_b + dE_nb;
    if (!soma_oracle_metropolis(dE, u)) return 0;
    x[bead] = r_new[0];
    y[bead] = r_new[1];
    z[bead] = r_new[2];
    return 1;
}

/* ------------------------------------------------------------------------------------------ */
/* a5  Smart Monte-Carlo move (refs [28,29]); reading R13 (Rossky-Doll-Friedman    */
/* with the bonded force only):                                                                  */
/*    F(r)  = -k_0 sum_nb (r - r_nb)                                                             */
/*    d     = a_s F(r) + sqrt(2 a_s) g,  g ~ N(0,1)^3                                            */
/*    F'    = F(r + d) with the neighbours fixed = F - k_0 m d                                   */
/*    accept iff u < exp( -dE - ( |d + a_s F'|^2 - |d - a_s F|^2 ) / (4 a_s) )                   */
/* with dE = dE_b + dE_nb as for the local move.  Gaussians: Box-Muller on Philox words of       */
/* call sub=0 (g_x,g_y from words 0,1; g_z from words 2,3); acceptance u from call sub=1 word 0. */
/* ------------------------------------------------------------------------------------------ */
void soma_oracle_smc_proposal(const oracle_system *s, uint64_t bead, uint64_t sweep, float g[3], float *u)
{
    uint32_t w[4], v[4];
    draw(s, bead, sweep, 2u, 0u, w);
    draw(s, bead, sweep, 2u, 1u, v);
    /* u1 = 2 - U23 in (0,1] (exact), u2 = U23 - 1 in [0,1) (exact) */
    const float u1a = 2.0f - soma_oracle_u23(w[0]), u2a = soma_oracle_u23(w[1]) - 1.0f;
    const float u1b = 2.0f - soma_oracle_u23(w[2]), u2b = soma_oracle_u23(w[3]) - 1.0f;
    const float ra = sqrtf(-2.0f * logf(u1a)), rb = sqrtf(-2.0f * logf(u1b));
    const float two_pi = 6.283185307179586f;
    g[0] = ra * cosf(two_pi * u2a);
    g[1] = ra * sinf(two_pi * u2a);
    g[2] = rb * cosf(two_pi * u2b);
    *u = soma_oracle_u23(v[0]) - 1.0f;
}

static void smc_delta_core(const oracle_system *s, const float *x, const float *y, const float *z,
                           const float *omega, uint64_t bead, float sx, float sy, float sz, float mf, uint32_t type,
                           const float g[3], float d[3], float *dE, float *log_ratio, float r_new[3]);

void soma_oracle_smc_delta(const oracle_system *s, const float *x, const float *y, const float *z,
                           const float *omega, uint64_t bead, int has_l, int has_r, uint32_t type,
                           const float g[3], float d[3], float *dE, float *log_ratio, float r_new[3])
{
    const float rx = x[bead], ry = y[bead], rz = z[bead];
    const float blx = has_l ? rx - x[bead - 1] : 0.0f, brx = has_r ? rx - x[bead + 1] : 0.0f;
    const float bly = has_l ? ry - y[bead - 1] : 0.0f, bry = has_r ? ry - y[bead + 1] : 0.0f;
    const float blz = has_l ? rz - z[bead - 1] : 0.0f, brz = has_r ? rz - z[bead + 1] : 0.0f;
    const float mf = (float)((has_l ? 1 : 0) + (has_r ? 1 : 0));
    smc_delta_core(s, x, y, z, omega, bead, blx + brx, bly + bry, blz + brz, mf, type, g, d, dE, log_ratio, r_new);
}

static void smc_delta_core(const oracle_system *s, const float *x, const float *y, const float *z,
                           const float *omega, uint64_t bead, float sx, float sy, float sz, float mf, uint32_t type,
                           const float g[3], float d[3], float *dE, float *log_ratio, float r_new[3])
{
    const float k0 = (float)(3.0 * ((double)s->N_ref - 1.0));
    const float a_s = s->smc_step;
    const float noise = sqrtf(2.0f * a_s);
    const float rx = x[bead], ry = y[bead], rz = z[bead];
    const float F[3] = { -k0 * sx, -k0 * sy, -k0 * sz };
    for (int a = 0; a < 3; ++a) d[a] = fmaf(a_s, F[a], noise * g[a]);
    const float ds = fmaf(d[2], sz, fmaf(d[1], sy, d[0] * sx));
    const float dd = fmaf(d[2], d[2], fmaf(d[1], d[1], d[0] * d[0]));
    const float dE_b = (0.5f * k0) * fmaf(2.0f, ds, mf * dd);
    r_new[0] = rx + d[0];
    r_new[1] = ry + d[1];
    r_new[2] = rz + d[2];
    const int64_t c_old = soma_oracle_cell_index(s, rx, ry, rz);
    const int64_t c_new = soma_oracle_cell_index(s, r_new[0], r_new[1], r_new[2]);
    float dE_nb = 0.0f;
    if (c_new != c_old) {
        const int64_t cells = n_cells(s);
        dE_nb = omega[(int64_t)type * cells + c_new] - omega[(int64_t)type * cells + c_old];
    }
    *dE = dE_b + dE_nb;
    /* proposal densities: forward T(r->r') ~ exp(-|d - a_s F|^2 / 4 a_s), reverse T(r'->r) ~
     * exp(-|-d - a_s F'|^2 / 4 a_s), F' = F - k_0 m d */
    float fwd = 0.0f, rev = 0.0f;
    for (int a = 0; a < 3; ++a) {
        const float Fp = F[a] - (k0 * mf) * d[a];
        const float ef = d[a] - a_s * F[a];
        const float er = d[a] + a_s * Fp;
        fwd = fmaf(ef, ef, fwd);
        rev = fmaf(er, er, rev);
    }
    *log_ratio = (rev - fwd) / (4.0f * a_s);
}

static int mc_smc(const oracle_system *s, float *x, float *y, float *z, const float *omega,
                  uint64_t bead, uint64_t bead_rng, int has_l, int has_r, uint32_t type, uint64_t sweep)
{
    float g[3], u, d[3], dE, log_ratio, r_new[3];
    soma_oracle_smc_proposal(s, bead_rng, sweep, g, &u);
    soma_oracle_smc_delta(s, x, y, z, omega, bead, has_l, has_r, type, g, d, &dE, &log_ratio, r_new);
    if (!soma_oracle_metropolis(dE + log_ratio, u)) return 0;
    x[bead] = r_new[0];
    y[bead] = r_new[1];
    z[bead] = r_new[2];
    return 1;
}

/* ------------------------------------------------------------------------------------------ */
/* General molecular architectures ("almost arbitrary architectures", 292,     */
/* 344-354).  An architecture with spec_n_bonds > 0 is given by its bond list; every bond is the  */
/* harmonic spring of Eq. 2 with the same k_0.  Reading R25:                                       */
/*  - neighbour lists in ascending monomer index; the bond sum s = sum_nb (r - r_nb) of Eq. 2 is   */
/*    accumulated in that order in fp32 (a linear chain given as bonds (j, j+1) then reproduces    */
/*    the chain code above bit for bit);                                                           */
/*  - independent sets ("a simple heuristics ... aiming for the minimal number of sets",            */
/*    PAPER.md:292): greedy first fit in monomer order -- monomer j joins the lowest-numbered set   */
/*    that holds none of its bonded neighbours; for a linear chain that is even / odd (Fig. 1);     */
/*  - the sets are worked through in the order 0, 1, ... (R11), their members in monomer order.     */
/* ------------------------------------------------------------------------------------------ */
static const uint32_t *spec_bonds(const oracle_system *s, uint32_t spec)
{
    const uint32_t *b = s->bonds;
    for (uint32_t a = 0; a < spec; ++a) b += 2u * s->spec_n_bonds[a];
    return b;
}

/* adjacency of one architecture: nbr_off[N+1], nbr[2 n_bonds] (ascending within a monomer) */
static void build_adjacency(uint32_t N, uint32_t n_bonds, const uint32_t *bonds, uint32_t *nbr_off, uint32_t *nbr)
{
    for (uint32_t j = 0; j <= N; ++j) nbr_off[j] = 0;
    for (uint32_t b = 0; b < n_bonds; ++b) { nbr_off[bonds[2 * b] + 1]++; nbr_off[bonds[2 * b + 1] + 1]++; }
    for (uint32_t j = 0; j < N; ++j) nbr_off[j + 1] += nbr_off[j];
    uint32_t *fill = (uint32_t *)calloc(N, sizeof(uint32_t));
    for (uint32_t b = 0; b < n_bonds; ++b) {
        const uint32_t i = bonds[2 * b], j = bonds[2 * b + 1];
        nbr[nbr_off[i] + fill[i]++] = j;
        nbr[nbr_off[j] + fill[j]++] = i;
    }
    free(fill);
    for (uint32_t j = 0; j < N; ++j)          /* insertion sort of each (short) list */
        for (uint32_t a = nbr_off[j] + 1; a < nbr_off[j + 1]; ++a) {
            const uint32_t v = nbr[a];
            uint32_t c = a;
            while (c > nbr_off[j] && nbr[c - 1] > v) { nbr[c] = nbr[c - 1]; --c; }
            nbr[c] = v;
        }
}

/* set_of[j] = independent set of monomer j of architecture `spec`; returns the number of sets */
uint32_t soma_oracle_sets(const oracle_system *s, uint32_t spec, uint32_t *set_of)
{
    const uint32_t N = s->spec_n_beads[spec];
    const uint32_t nb = s->spec_n_bonds ? s->spec_n_bonds[spec] : 0u;
    if (nb == 0) {                                   /* linear chain: even / odd (Fig. 1) */
        for (uint32_t j = 0; j < N; ++j) set_of[j] = j & 1u;
        return N > 1 ? 2u : 1u;
    }
    uint32_t *off = (uint32_t *)malloc(sizeof(uint32_t) * (N + 1)), *nbr = (uint32_t *)malloc(sizeof(uint32_t) * 2 * nb);
    build_adjacency(N, nb, spec_bonds(s, spec), off, nbr);
    uint32_t n_sets = 0;
    for (uint32_t j = 0; j < N; ++j) {
        uint32_t c = 0;
        for (;;) {                                   /* lowest set without a bonded neighbour (only j' < j are placed) */
            int clash = 0;
            for (uint32_t a = off[j]; a < off[j + 1]; ++a)
                if (nbr[a] < j && set_of[nbr[a]] == c) clash = 1;
            if (!clash) break;
            ++c;
        }
        set_of[j] = c;
        if (c + 1 > n_sets) n_sets = c + 1;
    }
    free(off); free(nbr);
    return n_sets;
}

/* one molecule of a general architecture, all sets in order */
static uint64_t sweep_general_molecule(const oracle_system *s, float *x, float *y, float *z, const float *omega,
                                       uint64_t first, uint32_t N, const uint8_t *types, const uint32_t *off,
                                       const uint32_t *nbr, const uint32_t *set_of, uint32_t n_sets,
                                       uint64_t sweep, int move_kind, uint8_t *decisions)
{
    uint64_t accepted = 0;
    for (uint32_t i_set = 0; i_set < n_sets; ++i_set)
        for (uint32_t ip = 0; ip < N; ++ip) {
            if (set_of[ip] != i_set) continue;
            const uint64_t bead = first + ip;
            float sx = 0.0f, sy = 0.0f, sz = 0.0f;
            const uint32_t m = off[ip + 1] - off[ip];
            for (uint32_t a = off[ip]; a < off[ip + 1]; ++a) {
                const uint64_t nb = first + nbr[a];
                const float bx = x[bead] - x[nb], by = y[bead] - y[nb], bz = z[bead] - z[nb];
                if (a == off[ip]) { sx = bx; sy = by; sz = bz; } else { sx = sx + bx; sy = sy + by; sz = sz + bz; }
            }
            float r_new[3], u, dE;
            if (move_kind == 2) {
                float g[3], d[3], lr;
                soma_oracle_smc_proposal(s, bead, sweep, g, &u);
                smc_delta_core(s, x, y, z, omega, bead, sx, sy, sz, (float)m, types[ip], g, d, &dE, &lr, r_new);
                dE = dE + lr;
            } else {
                float d[3], eb, enb;
                soma_oracle_local_proposal(s, bead, sweep, d, &u);
                local_delta_e_core(s, x, y, z, omega, bead, sx, sy, sz, (float)m, types[ip], d, &eb, &enb, r_new);
                dE = eb + enb;
            }
            const int acc = soma_oracle_metropolis(dE, u);
            if (acc) { x[bead] = r_new[0]; y[bead] = r_new[1]; z[bead] = r_new[2]; }
            accepted += (uint64_t)acc;
            if (decisions) decisions[bead] = (uint8_t)acc;
        }
    return accepted;
}

/* "Generate random permutation of the sets" (Code 2; "a pre-defined random order",
 * PAPER.md:294).  A linear chain has two sets, so the permutation is one fair bit per molecule and
 * sweep.  Reading R21: bit 31 of word 0 of Philox(counter = (global index of the molecule's first
 * bead, sweep lo32, sweep hi32, kind 3 << 8)); it names the set that goes first (0 even, 1 odd).
 * The bit does not depend on the configuration, so global balance holds. */
uint32_t soma_oracle_first_set(const oracle_system *s, uint64_t first_bead, uint64_t sweep)
{
    if (s->set_order == 0) return 0u;
    uint32_t w[4];
    draw(s, first_bead, sweep, 3u, 0u, w);
    return w[0] >> 31;
}

/* ------------------------------------------------------------------------------------------ */
/* Stage 2: one MC sweep, omega frozen.  Code 2: parallel loop over           */
/* molecules; inside a molecule the independent sets one after the other; for a linear chain the */
/* sets are the even and the odd monomers (Fig. 1).  Reading R11: the set order is */
/* even, then odd, every sweep, unless set_order = 1 (soma_oracle_first_set).                    */
/* decisions (nullable): one byte per bead, 1 = accepted.                                        */
/* move_kind: 1 = local displacement, 2 = Smart-MC.  Returns the number of accepted moves.       */
/* ------------------------------------------------------------------------------------------ */
uint64_t soma_oracle_sweep(const oracle_system *s, float *x, float *y, float *z, const float *omega,
                           uint64_t sweep, int move_kind, uint8_t *decisions)
{
    uint64_t accepted = 0;
    uint64_t spec_first_bead = 0;
    const uint8_t *types = s->types;
    for (uint32_t a = 0; a < s->n_specs; ++a) {
        const uint32_t N = s->spec_n_beads[a];
        const int64_t n_mol = (int64_t)s->spec_n_chains[a];
        if (s->spec_n_bonds && s->spec_n_bonds[a] > 0) {        /* general architecture (R25) */
            const uint32_t nb = s->spec_n_bonds[a];
            uint32_t *off = (uint32_t *)malloc(sizeof(uint32_t) * (N + 1));
            uint32_t *nbr = (uint32_t *)malloc(sizeof(uint32_t) * 2 * nb);
            uint32_t *set_of = (uint32_t *)malloc(sizeof(uint32_t) * N);
            build_adjacency(N, nb, spec_bonds(s, a), off, nbr);
            const uint32_t n_sets = soma_oracle_sets(s, a, set_of);
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : accepted)
#endif
            for (int64_t mol = 0; mol < n_mol; ++mol)
                accepted += sweep_general_molecule(s, x, y, z, omega, spec_first_bead + (uint64_t)mol * N, N, types,
                                                   off, nbr, set_of, n_sets, sweep, move_kind, decisions);
            free(off); free(nbr); free(set_of);
            spec_first_bead += (uint64_t)n_mol * N;
            types += N;
            continue;
        }
        /* a part of a larger system draws the numbers of its beads' indices in the whole system */
        const uint64_t rng_shift = s->spec_first_bead ? s->spec_first_bead[a] - spec_first_bead : 0;
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : accepted)
#endif
        for (int64_t mol = 0; mol < n_mol; ++mol) {
            const uint64_t first = spec_first_bead + (uint64_t)mol * N;
            const uint32_t first_set = soma_oracle_first_set(s, first + rng_shift, sweep);
            for (uint32_t k_set = 0; k_set < 2; ++k_set) {      /* the two sets, one after the other */
                const uint32_t i_set = k_set ^ first_set;       /* set_permutation[k_set]            */
                for (uint32_t ip = i_set; ip < N; ip += 2) {     /* members of the set                */
                    const uint64_t bead = first + ip;
                    const int has_l = ip > 0, has_r = ip + 1 < N;
                    const int acc = move_kind == 2
                        ? mc_smc(s, x, y, z, omega, bead, bead + rng_shift, has_l, has_r, types[ip], sweep)
                        : mc_local(s, x, y, z, omega, bead, bead + rng_shift, has_l, has_r, types[ip], sweep);
                    accepted += (uint64_t)acc;
                    if (decisions) decisions[bead] = (uint8_t)acc;
                }
            }
        }
        spec_first_bead += (uint64_t)n_mol * N;
        types += N;
    }
    return accepted;
}

/* ------------------------------------------------------------------------------------------ */
/* Stage 2, first scheme of the paper (Code 1): molecules in parallel; inside a  */
/* molecule "sequentially choosing a particle of this molecule at random for a MC move", N times, */
/* so that "on average, each particle of the molecules is attempted to be moved once during a MC  */
/* step".  Reading R24: attempt k = 0..N-1 of the molecule whose first bead has global index f    */
/* owns the Philox counter word f + k (unique per sweep); the particle is                          */
/* i = floor(w0 N / 2^32) with w0 = word 0 of the call of kind 4, and the move itself (local or    */
/* Smart-MC) takes its random numbers from the calls of kind 1 / 2 with that same counter word.    */
/* decisions[f + k] = outcome of attempt k.                                                        */
/* ------------------------------------------------------------------------------------------ */
uint32_t soma_oracle_pick(const oracle_system *s, uint64_t attempt_id, uint64_t sweep, uint32_t N)
{
    uint32_t w[4];
    draw(s, attempt_id, sweep, 4u, 0u, w);
    return (uint32_t)(((uint64_t)w[0] * (uint64_t)N) >> 32);
}

uint64_t soma_oracle_sweep_molecules(const oracle_system *s, float *x, float *y, float *z,
                                     const float *omega, uint64_t sweep, int move_kind, uint8_t *decisions)
{
    uint64_t accepted = 0;
    uint64_t spec_first_bead = 0;
    const uint8_t *types = s->types;
    for (uint32_t a = 0; a < s->n_specs; ++a) {
        const uint32_t N = s->spec_n_beads[a];
        const int64_t n_mol = (int64_t)s->spec_n_chains[a];
#ifdef _OPENMP
#pragma omp parallel for schedule(static) reduction(+ : accepted)
#endif
        for (int64_t mol = 0; mol < n_mol; ++mol) {
            const uint64_t first = spec_first_bead + (uint64_t)mol * N;
            for (uint32_t mono = 0; mono < N; ++mono) {          /* sequential iteration of particles */
                const uint64_t attempt = first + mono;
                const uint32_t ip = soma_oracle_pick(s, attempt, sweep, N);   /* select random particle */
                const uint64_t bead = first + ip;
                const int has_l = ip > 0, has_r = ip + 1 < N;
                const int acc = move_kind == 2
                    ? mc_smc(s, x, y, z, omega, bead, attempt, has_l, has_r, types[ip], sweep)
                    : mc_local(s, x, y, z, omega, bead, attempt, has_l, has_r, types[ip], sweep);
                accepted += (uint64_t)acc;
                if (decisions) decisions[attempt] = (uint8_t)acc;
            }
        }
        spec_first_bead += (uint64_t)n_mol * N;
        types += N;
    }
    return accepted;
}

/* One SCMF cycle as soma_step runs it: sweep with the current omega, then stage 1 for the new
 * configuration (fields refreshed "after each MC step"; reading R12). */
uint64_t soma_oracle_step(const oracle_system *s, float *x, float *y, float *z, uint32_t *counts,
                          float *omega, uint64_t sweep0, uint32_t n_sweeps, int move_kind,
                          uint8_t *decisions)
{
    uint64_t accepted = 0;
    for (uint32_t i = 0; i < n_sweeps; ++i) {
        accepted += s->scheme == 1
            ? soma_oracle_sweep_molecules(s, x, y, z, omega, sweep0 + i, move_kind, decisions)
            : soma_oracle_sweep(s, x, y, z, omega, sweep0 + i, move_kind, decisions);
        soma_oracle_histogram(s, x, y, z, counts);
        /* Reading R22: with field_every = k > 1 the fields are the "frequently updated" ones of
         * PAPER.md:200 refreshed only after sweeps number k, 2k, ... (counted from 1) */
        if (s->field_every <= 1 || (sweep0 + i + 1) % s->field_every == 0)
            soma_oracle_fields(s, counts, omega);
    }
    return accepted;
}

/* ------------------------------------------------------------------------------------------ */
/* Initial state of soma_init when no positions are handed in (BASELINE.json configs: "Gaussian  */
/* random walks, per-axis bond std R_e/sqrt(3 (N-1)), first bead uniform in the box").  Reading  */
/* R14: kind-0 Philox words of each bead; first bead L_a * w_a 2^-32; following beads add        */
/* sigma * Box-Muller Gaussians; the running sum is kept in double and rounded to fp32 once.     */
/* ------------------------------------------------------------------------------------------ */
void soma_oracle_init_positions(const oracle_system *s, float *x, float *y, float *z)
{
    const double two32 = 4294967296.0, two_pi = 6.283185307179586476925286766559;
    const double sigma = s->N_ref > 1 ? 1.0 / sqrt(3.0 * ((double)s->N_ref - 1.0)) : 0.0;
    uint64_t g = 0;
    for (uint32_t a = 0; a < s->n_specs; ++a) {
        const uint32_t N = s->spec_n_beads[a];
        for (uint64_t m = 0; m < s->spec_n_chains[a]; ++m) {
            double p[3] = { 0.0, 0.0, 0.0 };
            for (uint32_t j = 0; j < N; ++j, ++g) {
                uint32_t w[4];
                draw(s, g, 0u, 0u, 0u, w);
                if (j == 0) {
                    for (int c = 0; c < 3; ++c) p[c] = (double)s->box[c] * ((double)w[c] / two32);
                } else {
                    const double ra = sqrt(-2.0 * log(((double)w[0] + 1.0) / two32));
                    const double rb = sqrt(-2.0 * log(((double)w[2] + 1.0) / two32));
                    const double ta = two_pi * ((double)w[1] / two32);
                    const double tb = two_pi * ((double)w[3] / two32);
                    p[0] += sigma * (ra * cos(ta));
                    p[1] += sigma * (ra * sin(ta));
                    p[2] += sigma * (rb * cos(tb));
                }
                x[g] = (float)p[0];
                y[g] = (float)p[1];
                z[g] = (float)p[2];
            }
        }
    }
}

int soma_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void soma_oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n > 0 ? n : 1);
#else
    (void)n;
#endif
}
