// soma_kernels.cuh -- device code of the SCMF Monte-Carlo step for sm_100a (B200).
//
// Kernels (PAPER.md = arXiv:1711.03828 text; DESIGN.md has the data layout and rooflines):
//   fused_sweep_kernel    a1+a2(+a3): one warp owns 128 consecutive beads (= whole chains, N | 128),
//                         4 beads per lane in registers, even monomers then odd monomers
//                         (independent sets of Fig. 1 / Code 2), neighbours by
//                         warp shuffle, each position read and written once per sweep.
//   generic_move_kernel   a1 or a2 for any chain length: one thread per monomer of one parity.
//   arch_move_kernel      one independent set of a general architecture (bond lists): one thread per member
//   molecule_move_kernel  the paper's other scheme (Code 1): one thread per molecule, N random picks
//   histogram_kernel      a3  n_i(c), Eq. 4
//   field_kernel          a4  omega_i(c), Eq. 12
//   init_walk_kernel      Gaussian-walk start state (BASELINE.json configs)
//
// Compiled with -fmad=false: the only fused multiply-adds are the explicit fmaf() below, so every
// fp32 rounding on the decision path is the one written here.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace soma {

constexpr int kMaxTypes = 8;
constexpr int kTile = 128;          // beads per warp tile in the fused kernel (4 per lane)
constexpr int kAccSlots = 256;      // spread slots of the accepted-moves counter
constexpr int kFusedThreads = 640;  // threads per block of the fused kernel: one block of 20 warps per SM
constexpr int kFusedMinBlocks = 1;  // resident blocks per SM the fused kernel is compiled for (register cap: 96)
constexpr int kMolUnroll = 4;       // attempts of the staged molecule kernel unrolled together

struct GridP {
    float inv_L[3];   // fl32(1 / L_a)
    float nf[3];      // (float) n_a
    uint32_t n[3];
    uint32_t neg_n[3];  // -n_a (mod 2^32)
    uint32_t k_rec;     // f * ((K_x n_y + K_y) n_z + K_z) mod 2^32, K_a = (n_a - 1) 0x4B400000 (see cell_raw()); f = 1
                        // for planes, 2 for records per cell (see cell_at())
    uint32_t cells;
    uint32_t last;      // n_types * cells - 1: the last valid index of omega
};

struct MoveP {
    GridP g;
    float c0, c1;     // trial displacement d = fmaf(U23, c1, c0): c1 = 2A, c0 = A (2^-23 - 3)
    float hk;         // k_0 / 2 = 1.5 (N_ref - 1)        (Eq. 2)
    float k0;         // k_0
    float a_s;        // Smart-MC step
    float noise;      // sqrt(2 a_s)
    float four_as;    // 4 a_s
    uint32_t rk[10][2];           // Philox round keys: seed + r * (0x9E3779B9, 0xBB67AE85)
    uint32_t sweep_lo, sweep_hi;  // Philox counter words 1, 2
    uint32_t head[2][4];          // rounds 1-2 folded over the warp-uniform counter words, per sub-move (philox4x32_10_head)
};

struct FieldP {
    float inv_nbar;   // cells / beads = 1 / (rho_0 DeltaL^3)
    float kappa0;     // kappaN / N_ref
    float chi0[kMaxTypes][kMaxTypes];
    float half_chi0[kMaxTypes][kMaxTypes];
    int n_types;
    int hamiltonian;
    uint32_t cells;
};

// ------------------------------------------------------------------------------------------------
// a0  Philox4x32-10 (Salmon et al., SC'11): ten rounds of two 32x32->64 multiplies and two
// three-way xors; the key schedule adds the Weyl constants between rounds.  No state in memory
// (the paper keeps 16 B of PCG state per thread in device memory).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t a, uint32_t b, uint32_t c, uint32_t d,
                                              uint32_t ka, uint32_t kb, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long pa = (unsigned long long)a * 0xD2511F53ull;
        const unsigned long long pc = (unsigned long long)c * 0xCD9E8D57ull;
        const uint32_t na = (uint32_t)(pc >> 32) ^ b ^ ka;
        const uint32_t nc = (uint32_t)(pa >> 32) ^ d ^ kb;
        b = (uint32_t)pc;
        d = (uint32_t)pa;
        a = na;
        c = nc;
        ka += 0x9E3779B9u;
        kb += 0xBB67AE85u;
    }
    out[0] = a; out[1] = b; out[2] = c; out[3] = d;
}

// The same ten rounds with the key schedule precomputed on the host (MoveP::rk lives in the kernel's
// constant bank) for counter (gid, sweep_lo, sweep_hi, tag), where only word 0 differs between
// beads: in round 1 the product sweep_hi * M1 and in round 2 the product a1 * M0 are the same for
// every bead of the launch, so the host multiplies them once (soma_ctx::movep) and passes
//   h[0] = tag ^ rk[0][1]              c1 = hi(gid M0) ^ h[0],   d1 = lo(gid M0)
//   h[1] = lo(sweep_hi M1) ^ rk[1][0]  a2 = hi(c1 M1) ^ h[1],    b2 = lo(c1 M1)
//   h[2] = hi(a1 M0) ^ rk[1][1]        c2 = d1 ^ h[2]
//   h[3] = lo(a1 M0)                   d2 = h[3]
// with a1 = hi(sweep_hi M1) ^ sweep_lo ^ rk[0][0].  Rounds 3-10 are the generic ones.  The output is
// bit-identical to philox4x32_10; 18 instead of 20 wide multiplies per call.
// p1 = gid * M0, the one product of round 1 that differs between beads.  A lane of the fused kernel owns
// consecutive beads, whose products differ by M0: it multiplies once and adds (exact in 64 bits).
constexpr unsigned long long kPhiloxM0 = 0xD2511F53ull;
__device__ __forceinline__ void philox4x32_10_head_p(unsigned long long p1, const uint32_t (&h)[4],
                                                     const uint32_t (&rk)[10][2], uint32_t (&out)[4])
{
    const uint32_t c1 = (uint32_t)(p1 >> 32) ^ h[0];
    const unsigned long long p2 = (unsigned long long)c1 * 0xCD9E8D57ull;
    uint32_t a = (uint32_t)(p2 >> 32) ^ h[1], b = (uint32_t)p2, c = (uint32_t)p1 ^ h[2], d = h[3];
#pragma unroll
    for (int r = 2; r < 10; ++r) {
        const unsigned long long pa = (unsigned long long)a * 0xD2511F53ull;
        const unsigned long long pc = (unsigned long long)c * 0xCD9E8D57ull;
        const uint32_t na = (uint32_t)(pc >> 32) ^ b ^ rk[r][0];
        const uint32_t nc = (uint32_t)(pa >> 32) ^ d ^ rk[r][1];
        b = (uint32_t)pc;
        d = (uint32_t)pa;
        a = na;
        c = nc;
    }
    out[0] = a; out[1] = b; out[2] = c; out[3] = d;
}
__device__ __forceinline__ void philox4x32_10_head(uint32_t gid, const uint32_t (&h)[4],
                                                   const uint32_t (&rk)[10][2], uint32_t (&out)[4])
{
    philox4x32_10_head_p((unsigned long long)gid * kPhiloxM0, h, rk, out);
}

// "Generate random permutation of the sets" (Code 2): a linear chain has two sets, so
// the permutation is one bit per chain and sweep, bit 31 of word 0 of the Philox call with counter
// (global index of the chain's first bead, sweep, kind 3) -- DESIGN.md reading R21.  0: the even
// monomers move first, 1: the odd ones.
__device__ __forceinline__ uint32_t first_set_bit(uint32_t first_gid, uint32_t sweep_lo, uint32_t sweep_hi,
                                                  uint32_t key0, uint32_t key1)
{
    uint32_t w[4];
    philox4x32_10(first_gid, sweep_lo, sweep_hi, 0x300u, key0, key1, w);
    return w[0] >> 31;
}

// Programmatic dependent launch: a kernel launched with the programmatic-serialization attribute may
// become resident while its predecessor in the stream still runs.  pdl_trigger() lets the successor
// start launching; pdl_wait() returns once the predecessor grid has completed and its writes are
// visible.  Both are no-ops in a kernel launched the ordinary way.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// Positions cross the SM once per sweep: streaming (evict-first) loads and stores, so that they do not push
// the omega lines the gathers reuse out of L1.
__device__ __forceinline__ float4 ld_stream(const float* p)
{
    return __ldcs(reinterpret_cast<const float4*>(p));
}
__device__ __forceinline__ void st_stream(float* p, const float4& v)
{
    __stcs(reinterpret_cast<float4*>(p), v);
}

// top 23 bits -> float in [1, 2), exact
__device__ __forceinline__ float u23(uint32_t w) { return __uint_as_float(0x3F800000u | (w >> 9)); }

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ float sqrt_approx(float x)
{
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ------------------------------------------------------------------------------------------------
// Pi_c of Eq. 4: the cell that contains r, periodic (R7).  Per axis the
// position in units of the box length is the fp32 number t = x * (1/L); the cell is
//   floor(t n) mod n = floor(t n) - n floor(t),
// both floors of the exact values.  Both come out of one instruction each, as the low mantissa bits of
//   A = fl_down(t + 1.5 * 2^23)        bits(A) = 0x4B400000 + floor(t)
//   B = fl_down(t * n + 1.5 * 2^23)    bits(B) = 0x4B400000 + floor(t n)     (FFMA: exact product)
// exact for |t n| < 2^22 (the supported domain).  With K_a = (n_a - 1) 0x4B400000 the cell of axis a is
// bits(B) - n_a bits(A) + K_a in 32-bit wrap-around arithmetic; the three constants are folded into one,
//   cell = ((cx ny + cy) nz + cz) = (((Bx - nx Ax) ny + By - ny Ay) nz + Bz - nz Az) + k_tot,
// five IMADs.  FMUL, FADD.RM, FFMA.RM per axis; no FRND / F2I (XU pipe), no fold of the fraction, no
// per-axis clamp.  cell_raw() returns the sum without k_tot.  cell_at() returns the index of the bead's
// field value in omega; it adds k_tot and the type's offset in one go (tk = toff + k_rec; toff = type * cells
// for planes, = type for records: the table the host keeps per monomer), and its
// unsigned min keeps the index inside the array for every input (NaN, coordinates outside the domain).
// Two grid formats:
//   planes (kPack = false, any number of types)  omega[type][cell], counts uint32 [type][cell]; index = cell + tk
//   records (kPack = true, two types)            omega[cell] = {omega_A, omega_B}; the occupation numbers of a
//          cell are one 32-bit word, n_A in the low and n_B in the high 16 bits (the paper stores uint16,
//          PAPER.md:243): 12 instead of 16 bytes of grid data per cell, which pays once the grids outgrow L2.
//          index = 2 cell + type is one three-input add.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cell_raw(const GridP& g, float x, float y, float z)
{
    const float M = 12582912.0f;
    const float tx = x * g.inv_L[0], ty = y * g.inv_L[1], tz = z * g.inv_L[2];
    const uint32_t ax = __float_as_uint(__fadd_rd(tx, M)), bx = __float_as_uint(__fmaf_rd(tx, g.nf[0], M));
    const uint32_t ay = __float_as_uint(__fadd_rd(ty, M)), by = __float_as_uint(__fmaf_rd(ty, g.nf[1], M));
    const uint32_t az = __float_as_uint(__fadd_rd(tz, M)), bz = __float_as_uint(__fmaf_rd(tz, g.nf[2], M));
    uint32_t u = ax * g.neg_n[0] + bx;
    u = u * g.n[1] + by;
    u = ay * g.neg_n[1] + u;
    u = u * g.n[2] + bz;
    u = az * g.neg_n[2] + u;
    return u;
}

// tk = type + k_rec
template <bool kPack>
__device__ __forceinline__ uint32_t cell_at(const GridP& g, float x, float y, float z, uint32_t tk)
{
    const uint32_t u = cell_raw(g, x, y, z);
    return min(kPack ? u + u + tk : u + tk, g.last);
}

// ------------------------------------------------------------------------------------------------
// Pieces of one Monte-Carlo move of one bead ("MC scheme for particle ip", Code 2).
// They are separate functions so that the fused kernel can run them phase by phase over the four
// beads a lane owns (all random numbers, then all cell indices, then all field gathers in flight at
// once, then the decisions), while the generic kernel strings them together for one bead.
// ------------------------------------------------------------------------------------------------
struct Draw {            // what one move takes from Philox
    float a, b, c;       // local move: trial displacement d;  Smart-MC: the Gaussians g
    float u;             // acceptance uniform in [0, 1)
};

// -2 ln(u1) for the Box-Muller radius, u1 = 2 - U23(w) = 1 - delta in (0, 1], delta = k 2^-23 exact.
// lg2.approx has an absolute error of 2^-22, which is a relative one only while |ln u1| is not small; near
// u1 = 1 (delta < 1/16) the series -ln(1 - delta) = delta + delta^2/2 + ... + delta^5/5 takes over (truncation
// 1.6e-7 relative).  Relative error of the result <= 2.6e-6 (at the switch), of the radius half that: a Gaussian
// is off by < 5e-7.  13 instructions instead of the ~28 of logf with its special cases.
__device__ __forceinline__ float neg2ln_u1(uint32_t w)
{
    const float delta = u23(w) - 1.0f, u1 = 1.0f - delta;              // both exact
    float l2;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(l2) : "f"(u1));
    const float far = l2 * -1.3862943611198906f;                        // -2 ln 2 lg2(u1)
    float p = fmaf(delta, 0.4f, 0.5f);
    p = fmaf(delta, p, 0.6666666666666666f);
    p = fmaf(delta, p, 1.0f);
    p = fmaf(delta, p, 2.0f);
    return delta < 0.0625f ? delta * p : far;
}

// kMove 1: d uniform in (-A,A)^3, 2^23 equidistant values per axis.
// kMove 2: g ~ N(0,1)^3 by Box-Muller on the words of call sub=0, u from call sub=1.
template <int kMove>
__device__ __forceinline__ Draw draw_move_p(const MoveP& P, unsigned long long p1)   // p1 = gid * M0
{
    Draw r;
    if (kMove == 1) {
        uint32_t w[4];
        philox4x32_10_head_p(p1, P.head[0], P.rk, w);
        r.a = fmaf(u23(w[0]), P.c1, P.c0);
        r.b = fmaf(u23(w[1]), P.c1, P.c0);
        r.c = fmaf(u23(w[2]), P.c1, P.c0);
        r.u = u23(w[3]) - 1.0f;
    } else {
        uint32_t w[4], v[4];
        philox4x32_10_head_p(p1, P.head[0], P.rk, w);
        philox4x32_10_head_p(p1, P.head[1], P.rk, v);
        // Box-Muller with sin.approx / cos.approx (MUFU) for the angle, taken in [-pi, pi) where the
        // approximations are best (absolute error 2^-21.4): sin(t) = -sin(t - pi), cos(t) = -cos(t - pi), and
        // t - pi = 2 pi (U23 - 1.5) with an exact subtraction.  A Gaussian is then off by <= ~2e-6, a
        // displacement by sqrt(2 a_s) times that: inside the parity tolerance on positions (R17).
        // Radius: see neg2ln_u1().
        const float ra = sqrt_approx(neg2ln_u1(w[0]));                  // sqrt.approx: <= 2 ulp
        const float rb = sqrt_approx(neg2ln_u1(w[2]));
        const float two_pi = 6.283185307179586f;
        const float ta = two_pi * (u23(w[1]) - 1.5f), tb = two_pi * (u23(w[3]) - 1.5f);
        const float sa = -__sinf(ta), ca = -__cosf(ta), cb = -__cosf(tb);
        r.a = ra * ca; r.b = ra * sa; r.c = rb * cb;
        r.u = u23(v[0]) - 1.0f;
    }
    return r;
}

template <int kMove>
__device__ __forceinline__ Draw draw_move(const MoveP& P, uint32_t gid)
{
    return draw_move_p<kMove>(P, (unsigned long long)gid * kPhiloxM0);
}

// dE_nb = omega_k(c') - omega_k(c), Eq. 15; exactly 0 when the cell is kept.  The
// loads are predicated, not branched around, so several moves' gathers are in flight together.
__device__ __forceinline__ float field_delta(const float* __restrict__ omega, uint32_t i_old, uint32_t i_new)
{
    float w_new = 0.0f, w_old = 0.0f;
    if (i_new != i_old) {
        // ordinary loads: with programmatic dependent launch this kernel may be resident while the field
        // kernel still writes omega, which rules out the non-coherent path (ld.global.nc)
        asm("ld.global.f32 %0, [%1];" : "=f"(w_new) : "l"(omega + i_new));
        asm("ld.global.f32 %0, [%1];" : "=f"(w_old) : "l"(omega + i_old));
    }
    return w_new - w_old;
}

// s = sum over bonded neighbours of (r - r_nb); an absent neighbour is passed as the bead itself.
__device__ __forceinline__ void bond_sum(float x, float y, float z, float xl, float yl, float zl,
                                         float xr, float yr, float zr, float& sx, float& sy, float& sz)
{
    sx = (x - xl) + (x - xr);
    sy = (y - yl) + (y - yr);
    sz = (z - zl) + (z - zr);
}

// bonded: dE_b = k_0/2 (2 d.s + m |d|^2), Eq. 2
__device__ __forceinline__ float bonded_delta(float half_k0, float mf, float dx, float dy, float dz,
                                              float sx, float sy, float sz)
{
    const float ds = fmaf(dz, sz, fmaf(dy, sy, dx * sx));
    const float dd = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    return half_k0 * fmaf(2.0f, ds, mf * dd);
}

// Metropolis: accept iff dE <= 0 or u < exp(-dE).  u < 1 and ex2.approx(t) >= 1 for
// every t >= 0 (also t = +inf), so the single comparison already accepts every dE <= 0.
__device__ __forceinline__ bool metropolis(float dE, float u)
{
    return u < ex2_approx(dE * -1.4426950408889634f);
}

// Smart-MC proposal from the bonded force F = -k_0 s (refs [28,29]; R13):
//   d = a_s F + sqrt(2 a_s) g,   accept iff u < exp(-(dE_b + dE_nb + L)),
//   L = ln T(r->r') - ln T(r'->r) = (|d + a_s F'|^2 - |d - a_s F|^2) / (4 a_s),   F' = F - k_0 m d.
// With e_r - e_f = 2 a_s F - a_s k_0 m d and e_r + e_f = (2 - a_s k_0 m) d for e_f = d - a_s F, e_r = d + a_s F',
//   L = (2 - a_s k_0 m)/4 (2 F.d - k_0 m |d|^2) = -(1 - a_s k_0 m / 2) dE_b,      dE_b = k_0/2 (2 d.s + m |d|^2),
// so the exponent is dE_nb + (a_s k_0 m / 2) dE_b: one fused multiply-add instead of the two squared norms and
// their difference (which also loses digits to cancellation; the closed form is the more accurate of the two).
__device__ __forceinline__ void smc_proposal(const MoveP& P, float sx, float sy, float sz, const Draw& g,
                                             float& dx, float& dy, float& dz)
{
    const float Fx = -P.k0 * sx, Fy = -P.k0 * sy, Fz = -P.k0 * sz;
    dx = fmaf(P.a_s, Fx, P.noise * g.a);
    dy = fmaf(P.a_s, Fy, P.noise * g.b);
    dz = fmaf(P.a_s, Fz, P.noise * g.c);
}

// exponent of the Smart-MC acceptance: dE_nb + (a_s k_0 m / 2) dE_b;  half_as_k0 = a_s k_0 / 2
__device__ __forceinline__ float smc_exponent(float half_as_k0, float mf, float e_b, float e_nb)
{
    return fmaf(half_as_k0 * mf, e_b, e_nb);
}

// The occupation numbers follow an accepted move (+1 new cell, -1 old cell): integer arithmetic, so
// they stay identical to a fresh histogram (a3, Eq. 4).
// i_old, i_new: cell_at() of the old and the new position (same type).  kPack: the cell's word is index >> 1,
// the type's half index & 1; the sums are exact modulo 2^32 whatever the order of the updates, so the word
// always holds n_A + 65536 n_B (the field kernel checks that no half has outgrown its 16 bits).
//   tk: the bead's type + k_rec as handed to cell_at() (k_rec is even for records, so bit 0 is the type: the
//   increment does not depend on the cells and can be kept across tiles)
template <bool kPack>
__device__ __forceinline__ void count_follow(uint32_t* __restrict__ counts, bool acc, uint32_t i_old, uint32_t i_new,
                                             uint32_t tk)
{
    if (acc && i_new != i_old) {
        if (kPack) {
            const uint32_t one = 1u << ((tk & 1u) << 4);
            atomicAdd(counts + (i_new >> 1), one);
            atomicAdd(counts + (i_old >> 1), 0u - one);
        } else {
            atomicAdd(counts + i_new, 1u);
            atomicAdd(counts + i_old, 0xFFFFFFFFu);
        }
    }
}

// One whole move of one bead (generic kernels).  (x,y,z) is updated in place when accepted.
//   (sx,sy,sz)     s = sum over the bonded neighbours of (r - r_nb), Eq. 2
//   mf             number of bonded neighbours as float
//   toff           offset of the bead type in omega: type * cells (planes) or type (records)
//   gid            global bead index = Philox counter word 0
template <int kMove, bool kIncr, bool kPack>
__device__ __forceinline__ bool mc_move_s(const MoveP& P, const float* __restrict__ omega,
                                          uint32_t* __restrict__ counts, float& x, float& y, float& z,
                                          float sx, float sy, float sz, float mf, uint32_t toff, uint32_t gid)
{
    const Draw q = draw_move<kMove>(P, gid);
    float dx = q.a, dy = q.b, dz = q.c;
    if (kMove == 2) smc_proposal(P, sx, sy, sz, q, dx, dy, dz);
    const float x2 = x + dx, y2 = y + dy, z2 = z + dz;   // r' = fl32(r + d)
    const uint32_t i_old = cell_at<kPack>(P.g, x, y, z, toff + P.g.k_rec);
    const uint32_t i_new = cell_at<kPack>(P.g, x2, y2, z2, toff + P.g.k_rec);
    const float e_nb = field_delta(omega, i_old, i_new);
    const float e_b = bonded_delta(kMove == 1 ? P.hk : 0.5f * P.k0, mf, dx, dy, dz, sx, sy, sz);
    const float dE = kMove == 2 ? smc_exponent(P.four_as * 0.125f * P.k0, mf, e_b, e_nb) : e_b + e_nb;
    const bool acc = metropolis(dE, q.u);
    x = acc ? x2 : x;
    y = acc ? y2 : y;
    z = acc ? z2 : z;
    if (kIncr) count_follow<kPack>(counts, acc, i_old, i_new, toff + P.g.k_rec);
    return acc;
}

// The same for a monomer of a linear chain, from its two chain neighbours.
template <int kMove, bool kIncr, bool kPack>
__device__ __forceinline__ bool mc_move(const MoveP& P, const float* __restrict__ omega,
                                        uint32_t* __restrict__ counts, float& x, float& y, float& z,
                                        float xl, float yl, float zl, float xr, float yr, float zr,
                                        float mf, uint32_t toff, uint32_t gid)
{
    float sx, sy, sz;
    bond_sum(x, y, z, xl, yl, zl, xr, yr, zr, sx, sy, sz);
    return mc_move_s<kMove, kIncr, kPack>(P, omega, counts, x, y, z, sx, sy, sz, mf, toff, gid);
}

// ------------------------------------------------------------------------------------------------
// a1 + a2 (+ a3) fused, chain-resident.  Requires N in {4, 8, ..., 128} (N | 128) so that a 128-bead
// warp tile holds whole chains; the architecture's bead array starts 512-byte aligned.  Only full
// tiles are processed here; the host sends a ragged tail (< 128 beads, whole chains) to the generic
// kernel.  Block b owns the contiguous tile range [b T / B, (b+1) T / B); its warps take those tiles
// round-robin.  Per tile and lane (4 consecutive monomers in registers):
//   1. the tile's positions are requested (they are first needed after step 2, which hides the latency);
//   2. all four Philox draws (they depend on nothing loaded);
//   3. local move: all four trial positions, all eight cell indices, all eight omega gathers in
//      flight at once -- dE_nb (Eq. 15) does not depend on the neighbours, only dE_b does;
//   4. set 0 (even monomers) decides, then set 1 (odd monomers) with the moved even neighbours
//      (independent sets of Fig. 1 / Code 2); neighbours across lanes by shuffle;
//   5. count updates for the accepted moves, one 128-bit store per coordinate array.
// Smart-MC proposals depend on the neighbours, so there steps 3-4 run per set.
//   x,y,z       base of this architecture's beads (padded layout)
//   toff_tab    [N] offset of every monomer's type in omega (type * cells, or type for records per cell)
//   n_tiles     full tiles of this architecture (n_chains * N / 128)
//   gid0        global index of the architecture's first bead
//   orig        [n_chains] the caller's chain index of the chain in each slot (Philox counter, bitmap)
//   dec_words   decision bitmap (whole system), or unused
// kOrder: dynamic shared memory = four bytes per chain of the block's tile range (the host keeps the ranges
// short enough); the block draws the order bit of all its chains before it waits for its predecessor.
// ------------------------------------------------------------------------------------------------
// kAnyN: chain lengths that are a multiple of 4 up to 128 but do not divide 128 (12, 20, 24, 48, 100, ...): a tile
// holds floor(128 / N) whole chains, the lanes beyond them idle (they load harmlessly, decide nothing and
// store nothing); n_mask then carries N and log2N the chains per tile.
template <int kMove, bool kIncr, bool kRecord, bool kOrder, bool kPack, bool kAnyN = false>
__global__ void __launch_bounds__(kFusedThreads, kFusedMinBlocks)
fused_sweep_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                   const float* __restrict__ omega, uint32_t* __restrict__ counts,
                   const uint32_t* __restrict__ toff_tab, uint32_t n_mask, uint32_t n_tiles,
                   uint32_t gid0, const uint32_t* __restrict__ orig, uint32_t log2N,
                   uint32_t* __restrict__ dec_words, unsigned long long* __restrict__ acc_slots)
{
    constexpr uint32_t kFull = 0xFFFFFFFFu;
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t wib = threadIdx.x >> 5;
    constexpr uint32_t kWarps = kFusedThreads / 32;
    pdl_trigger();
    const uint32_t len = n_mask, cpt = log2N;                 // kAnyN: chain length, chains per tile
    const uint32_t cit_raw = kAnyN ? lane / (len >> 2) : 0u;  // kAnyN: this lane's chain in its tile
    const bool active = !kAnyN || cit_raw < cpt;
    const uint32_t cit = kAnyN ? min(cit_raw, cpt - 1u) : 0u;
    const uint32_t tile_beads = kAnyN ? cpt * len : kTile;
    const uint32_t j0 = kAnyN ? 4u * lane - cit_raw * len : (4u * lane) & n_mask;   // monomer index of slot 0
    const bool has_l0 = j0 != 0u;                             // slot 0 has a left neighbour
    const bool has_r3 = kAnyN ? j0 + 4u != len : ((j0 + 4u) & n_mask) != 0u;   // slot 3 has a right neighbour
    const uint4 toff = *reinterpret_cast<const uint4*>(toff_tab + j0);
    const uint4 tk = make_uint4(toff.x + P.g.k_rec, toff.y + P.g.k_rec, toff.z + P.g.k_rec, toff.w + P.g.k_rec);
    const float mf0 = has_l0 ? 2.0f : 1.0f, mf3 = has_r3 ? 2.0f : 1.0f;
    const float half_k0 = kMove == 1 ? P.hk : 0.5f * P.k0;
    uint32_t n_acc = 0;

    const uint32_t t_begin = (uint32_t)(((uint64_t)blockIdx.x * n_tiles) / gridDim.x);
    const uint32_t t_end = (uint32_t)(((uint64_t)(blockIdx.x + 1) * n_tiles) / gridDim.x);
    // The block's tiles are handed out dynamically: the first two rounds are fixed (tile = begin + warp,
    // + kWarps), after that a warp takes the next free tile from a shared-memory counter, one tile ahead
    // of the prefetch.  The schedulers do not serve their warps evenly; with a fixed share per warp the
    // favoured ones finished early and the SM ran its last tiles at low occupancy.
    __shared__ uint32_t s_next[2];
    const uint32_t zero = n_mask >> 8;                        // n_mask = N - 1 <= 127
    if (threadIdx.x == 0) s_next[0] = t_begin + 2u * kWarps;
    // kOrder: the chains of this block's tile range, regrouped (entry = index of the chain's first bead in this
    // architecture's arrays, bit 0 = odd set first)
    extern __shared__ __align__(16) uint32_t s_perm[];
    const uint32_t slot_begin = kAnyN ? t_begin * cpt : (t_begin * kTile) >> log2N;
    const uint32_t n_slots = kAnyN ? (t_end - t_begin) * cpt : ((t_end - t_begin) * kTile) >> log2N;
    const uint32_t cpt_shift = 7u - log2N, ci = kAnyN ? cit : (4u * lane) >> log2N;   // chains per tile = 128 / N; this lane's chain in its tile
    // list entry of the tile `t` for this lane; bead offset of a chain slot; chain slot of a bead offset
    auto entry_at = [&](uint32_t t) { return kAnyN ? (t - t_begin) * cpt + ci : ((t - t_begin) << cpt_shift) + ci; };
    auto beads_of = [&](uint32_t slot) { return kAnyN ? slot * len : slot << log2N; };
    if (kOrder) {
        // "Generate random permutation of the sets" (Code 2) for every chain this block will move:
        // needs nothing of the predecessor kernel (orig[] only changes in a re-sort), so it runs before the wait.
        // The lanes of a warp hold different chains, and a warp whose chains all start with the same set does
        // four evaluations per lane like the fixed order, a mixed one six (three phases); so the chains are
        // regrouped by their bit within groups of 64 consecutive chains -- tiles are made of 128 / N consecutive
        // entries of the list -- and (N = 32) at most one tile in sixteen is mixed, while a tile's chains stay
        // neighbours in the storage order.  A stable partition per group: a warp per group, two chains per lane.
        for (uint32_t lo0 = wib * 64u; lo0 < n_slots; lo0 += 4u * kWarps * 64u) {
            uint32_t first[8];                                // four groups' loads in flight
#pragma unroll
            for (uint32_t k = 0; k < 8u; ++k) {
                const uint32_t s = lo0 + (k >> 1) * kWarps * 64u + (k & 1u) * 32u + lane;
                first[k] = s < n_slots ? orig[slot_begin + s] : 0u;
            }
#pragma unroll
            for (uint32_t k = 0; k < 4u; ++k) {
                const uint32_t lo = lo0 + k * kWarps * 64u, sa = lo + lane, sb = sa + 32u;
                if (lo >= n_slots) break;
                const uint32_t ba = sa < n_slots ? first_set_bit(gid0 + beads_of(first[2 * k]), P.sweep_lo, P.sweep_hi, P.rk[0][0], P.rk[0][1]) : 0u;
                const uint32_t bb = sb < n_slots ? first_set_bit(gid0 + beads_of(first[2 * k + 1]), P.sweep_lo, P.sweep_hi, P.rk[0][0], P.rk[0][1]) : 0u;
                const uint32_t ones_a = __ballot_sync(kFull, ba != 0u), ones_b = __ballot_sync(kFull, bb != 0u);
                const uint32_t zeros_a = __ballot_sync(kFull, sa < n_slots) & ~ones_a, zeros_b = __ballot_sync(kFull, sb < n_slots) & ~ones_b;
                const uint32_t below = (1u << lane) - 1u;
                const uint32_t n_zero = __popc(zeros_a) + __popc(zeros_b);
                const uint32_t pos_a = ba ? n_zero + __popc(ones_a & below) : __popc(zeros_a & below);
                const uint32_t pos_b = bb ? n_zero + __popc(ones_a) + __popc(ones_b & below) : __popc(zeros_a) + __popc(zeros_b & below);
                if (sa < n_slots) s_perm[lo + pos_a] = beads_of(slot_begin + sa) | ba;   // 4 | N: the low bits are free
                if (sb < n_slots) s_perm[lo + pos_b] = beads_of(slot_begin + sb) | bb;
            }
        }
    }
    pdl_wait();                                               // omega of the preceding field kernel
    __syncthreads();
    uint32_t tile = t_begin + wib, tile_n = tile + kWarps;
    float4 X, Y, Z;
    uint32_t C = 0u;                                          // the caller's index of this lane's chain
    uint32_t E = 0u;                                          // kOrder: this lane's entry of the list
    if (tile < t_end) {
        if (kOrder) E = s_perm[entry_at(tile)];
        const uint32_t i0 = kOrder ? (E & ~1u) + j0 : tile * tile_beads + 4u * lane;
        C = orig[kAnyN ? (kOrder ? (E >> 2) / (len >> 2) : tile * cpt + cit) : i0 >> log2N];
    }
    while (tile < t_end) {
        const uint32_t i0 = kOrder ? (E & ~1u) + j0 : tile * tile_beads + 4u * lane;
        const uint32_t gid = gid0 + beads_of(C) + j0;
        // the tile after the next one.  The counter is addressed through `warp & zero` (zero: a kernel argument
        // bit that is never set): with a provably uniform address ptxas wraps the atomic of this single lane
        // into its warp-aggregation sequence (vote, popc, leader election: a dozen instructions per tile)
        uint32_t tile_nn = 0u;
        if (lane == 0) tile_nn = atomicAdd(s_next + (wib & zero), 1u);

        // 1. the chain index of the next tile of this warp (clamped to the last tile: a harmless re-read)
        uint32_t En = 0u;
        if (kOrder) En = s_perm[entry_at(min(tile_n, t_end - 1u))];
        const uint32_t i0n = kOrder ? (En & ~1u) + j0 : min(tile_n, t_end - 1u) * tile_beads + 4u * lane;
        // this tile's positions: asked for now, first needed after the four Philox draws below (~150
        // instructions of this warp and as many of each of its four neighbours on the scheduler), which covers
        // the latency without holding a second tile in registers
        X = ld_stream(x + i0);
        Y = ld_stream(y + i0);
        Z = ld_stream(z + i0);
        const uint32_t Cn = orig[kAnyN ? (kOrder ? (En >> 2) / (len >> 2) : min(tile_n, t_end - 1u) * cpt + cit) : i0n >> log2N];

        // 2. random numbers of the four moves
        // (round 1 of beads gid + 1 .. gid + 3 by addition: (gid + j) M0 = gid M0 + j M0, no carry out of 64 bits)
        const unsigned long long p1 = (unsigned long long)gid * kPhiloxM0;
        Draw q0 = draw_move_p<kMove>(P, p1), q1 = draw_move_p<kMove>(P, p1 + kPhiloxM0),
             q2 = draw_move_p<kMove>(P, p1 + 2ull * kPhiloxM0), q3 = draw_move_p<kMove>(P, p1 + 3ull * kPhiloxM0);
        if (kAnyN && !active)                                 // an idle lane compares with u = +inf, which accepts nothing
            q0.u = q1.u = q2.u = q3.u = __int_as_float(0x7F800000);

        bool a0, a1, a2, a3;
        if (kMove == 1) {
            // 3. trial positions r' = fl32(r + d), cells, field differences
            const float x0n = X.x + q0.a, y0n = Y.x + q0.b, z0n = Z.x + q0.c;
            const float x1n = X.y + q1.a, y1n = Y.y + q1.b, z1n = Z.y + q1.c;
            const float x2n = X.z + q2.a, y2n = Y.z + q2.b, z2n = Z.z + q2.c;
            const float x3n = X.w + q3.a, y3n = Y.w + q3.b, z3n = Z.w + q3.c;
            const uint32_t o0 = cell_at<kPack>(P.g, X.x, Y.x, Z.x, tk.x), n0 = cell_at<kPack>(P.g, x0n, y0n, z0n, tk.x);
            const uint32_t o1 = cell_at<kPack>(P.g, X.y, Y.y, Z.y, tk.y), n1 = cell_at<kPack>(P.g, x1n, y1n, z1n, tk.y);
            const uint32_t o2 = cell_at<kPack>(P.g, X.z, Y.z, Z.z, tk.z), n2 = cell_at<kPack>(P.g, x2n, y2n, z2n, tk.z);
            const uint32_t o3 = cell_at<kPack>(P.g, X.w, Y.w, Z.w, tk.w), n3 = cell_at<kPack>(P.g, x3n, y3n, z3n, tk.w);
            const float e0 = field_delta(omega, o0, n0), e1 = field_delta(omega, o1, n1),
                        e2 = field_delta(omega, o2, n2), e3 = field_delta(omega, o3, n3);

            if (!kOrder) {
                // 4a. set 0: even monomers (slots 0, 2) see the old odd monomers
                float xl = __shfl_up_sync(kFull, X.w, 1), yl = __shfl_up_sync(kFull, Y.w, 1), zl = __shfl_up_sync(kFull, Z.w, 1);
                xl = has_l0 ? xl : X.x; yl = has_l0 ? yl : Y.x; zl = has_l0 ? zl : Z.x;
                float sx, sy, sz;
                bond_sum(X.x, Y.x, Z.x, xl, yl, zl, X.y, Y.y, Z.y, sx, sy, sz);
                a0 = metropolis(bonded_delta(half_k0, mf0, q0.a, q0.b, q0.c, sx, sy, sz) + e0, q0.u);
                bond_sum(X.z, Y.z, Z.z, X.y, Y.y, Z.y, X.w, Y.w, Z.w, sx, sy, sz);
                a2 = metropolis(bonded_delta(half_k0, 2.0f, q2.a, q2.b, q2.c, sx, sy, sz) + e2, q2.u);
                X.x = a0 ? x0n : X.x; Y.x = a0 ? y0n : Y.x; Z.x = a0 ? z0n : Z.x;
                X.z = a2 ? x2n : X.z; Y.z = a2 ? y2n : Y.z; Z.z = a2 ? z2n : Z.z;

                // 4b. set 1: odd monomers (slots 1, 3) see the moved even monomers
                float xr = __shfl_down_sync(kFull, X.x, 1), yr = __shfl_down_sync(kFull, Y.x, 1), zr = __shfl_down_sync(kFull, Z.x, 1);
                xr = has_r3 ? xr : X.w; yr = has_r3 ? yr : Y.w; zr = has_r3 ? zr : Z.w;
                bond_sum(X.y, Y.y, Z.y, X.x, Y.x, Z.x, X.z, Y.z, Z.z, sx, sy, sz);
                a1 = metropolis(bonded_delta(half_k0, 2.0f, q1.a, q1.b, q1.c, sx, sy, sz) + e1, q1.u);
                bond_sum(X.w, Y.w, Z.w, X.z, Y.z, Z.z, xr, yr, zr, sx, sy, sz);
                a3 = metropolis(bonded_delta(half_k0, mf3, q3.a, q3.b, q3.c, sx, sy, sz) + e3, q3.u);
                X.y = a1 ? x1n : X.y; Y.y = a1 ? y1n : Y.y; Z.y = a1 ? z1n : Z.y;
                X.w = a3 ? x3n : X.w; Y.w = a3 ? y3n : Y.w; Z.w = a3 ? z3n : Z.w;
            } else {
                // 4'. random set order (SOMA_OPT_SET_ORDER = 1, "Generate random permutation of the sets", Code 2,
                // PAPER.md:302): the chain's bit says which set moves first, and the lanes of a warp hold
                // different chains.  Three phases: the odd monomers of the chains that start with their odd set,
                // the even monomers of every chain, the odd monomers of the chains that start with their even
                // set.  A chain takes part in the two phases that are its own order.  A phase no chain of the warp
                // takes part in is skipped: the block has grouped its chains by their bit, so all but one of its
                // tiles run two phases -- four evaluations per lane, as in the fixed order.
                const bool odd_first = (E & 1u) != 0u;
                const uint32_t vote = __ballot_sync(kFull, odd_first);
                a1 = a3 = false;
                auto even_set = [&]() {        // slots 0, 2 of every chain
                    float sx, sy, sz;
                    float xl = __shfl_up_sync(kFull, X.w, 1), yl = __shfl_up_sync(kFull, Y.w, 1), zl = __shfl_up_sync(kFull, Z.w, 1);
                    xl = has_l0 ? xl : X.x; yl = has_l0 ? yl : Y.x; zl = has_l0 ? zl : Z.x;
                    bond_sum(X.x, Y.x, Z.x, xl, yl, zl, X.y, Y.y, Z.y, sx, sy, sz);
                    a0 = metropolis(bonded_delta(half_k0, mf0, q0.a, q0.b, q0.c, sx, sy, sz) + e0, q0.u);
                    bond_sum(X.z, Y.z, Z.z, X.y, Y.y, Z.y, X.w, Y.w, Z.w, sx, sy, sz);
                    a2 = metropolis(bonded_delta(half_k0, 2.0f, q2.a, q2.b, q2.c, sx, sy, sz) + e2, q2.u);
                    X.x = a0 ? x0n : X.x; Y.x = a0 ? y0n : Y.x; Z.x = a0 ? z0n : Z.x;
                    X.z = a2 ? x2n : X.z; Y.z = a2 ? y2n : Y.z; Z.z = a2 ? z2n : Z.z;
                };
                auto odd_set = [&](float u1, float u3) {   // slots 1, 3; a chain whose turn it is not is given u = +inf
                    float sx, sy, sz;
                    float xr = __shfl_down_sync(kFull, X.x, 1), yr = __shfl_down_sync(kFull, Y.x, 1), zr = __shfl_down_sync(kFull, Z.x, 1);
                    xr = has_r3 ? xr : X.w; yr = has_r3 ? yr : Y.w; zr = has_r3 ? zr : Z.w;
                    bond_sum(X.y, Y.y, Z.y, X.x, Y.x, Z.x, X.z, Y.z, Z.z, sx, sy, sz);
                    const bool b1 = metropolis(bonded_delta(half_k0, 2.0f, q1.a, q1.b, q1.c, sx, sy, sz) + e1, u1);
                    bond_sum(X.w, Y.w, Z.w, X.z, Y.z, Z.z, xr, yr, zr, sx, sy, sz);
                    const bool b3 = metropolis(bonded_delta(half_k0, mf3, q3.a, q3.b, q3.c, sx, sy, sz) + e3, u3);
                    X.y = b1 ? x1n : X.y; Y.y = b1 ? y1n : Y.y; Z.y = b1 ? z1n : Z.y;
                    X.w = b3 ? x3n : X.w; Y.w = b3 ? y3n : Y.w; Z.w = b3 ? z3n : Z.w;
                    a1 = a1 || b1; a3 = a3 || b3;
                };
                if (vote == 0u) {              // every chain of the warp: even set, then odd set
                    even_set();
                    odd_set(q1.u, q3.u);
                } else if (vote == kFull) {    // every chain: odd set, then even set
                    odd_set(q1.u, q3.u);
                    even_set();
                } else {                       // mixed (one tile in 16)
                    const float inf = __int_as_float(0x7F800000);
                    odd_set(odd_first ? q1.u : inf, odd_first ? q3.u : inf);
                    even_set();
                    odd_set(odd_first ? inf : q1.u, odd_first ? inf : q3.u);
                }
            }

            // 5. occupation numbers follow the accepted moves
            if (kIncr) {
                count_follow<kPack>(counts, a0, o0, n0, tk.x);
                count_follow<kPack>(counts, a1, o1, n1, tk.y);
                count_follow<kPack>(counts, a2, o2, n2, tk.z);
                count_follow<kPack>(counts, a3, o3, n3, tk.w);
            }
        } else {
            // Smart-MC: the proposal needs the bonded force, i.e. the neighbours as they are now
            float xl = __shfl_up_sync(kFull, X.w, 1), yl = __shfl_up_sync(kFull, Y.w, 1), zl = __shfl_up_sync(kFull, Z.w, 1);
            xl = has_l0 ? xl : X.x; yl = has_l0 ? yl : Y.x; zl = has_l0 ? zl : Z.x;
            const float hak = P.four_as * 0.125f * P.k0;          // a_s k_0 / 2
            float sx0, sy0, sz0, sx2, sy2, sz2, dx0, dy0, dz0, dx2, dy2, dz2;
            bond_sum(X.x, Y.x, Z.x, xl, yl, zl, X.y, Y.y, Z.y, sx0, sy0, sz0);
            bond_sum(X.z, Y.z, Z.z, X.y, Y.y, Z.y, X.w, Y.w, Z.w, sx2, sy2, sz2);
            smc_proposal(P, sx0, sy0, sz0, q0, dx0, dy0, dz0);
            smc_proposal(P, sx2, sy2, sz2, q2, dx2, dy2, dz2);
            const float x0n = X.x + dx0, y0n = Y.x + dy0, z0n = Z.x + dz0;
            const float x2n = X.z + dx2, y2n = Y.z + dy2, z2n = Z.z + dz2;
            const uint32_t o0 = cell_at<kPack>(P.g, X.x, Y.x, Z.x, tk.x), n0 = cell_at<kPack>(P.g, x0n, y0n, z0n, tk.x);
            const uint32_t o2 = cell_at<kPack>(P.g, X.z, Y.z, Z.z, tk.z), n2 = cell_at<kPack>(P.g, x2n, y2n, z2n, tk.z);
            const float e0 = field_delta(omega, o0, n0), e2 = field_delta(omega, o2, n2);
            a0 = metropolis(smc_exponent(hak, mf0, bonded_delta(half_k0, mf0, dx0, dy0, dz0, sx0, sy0, sz0), e0), q0.u);
            a2 = metropolis(smc_exponent(hak, 2.0f, bonded_delta(half_k0, 2.0f, dx2, dy2, dz2, sx2, sy2, sz2), e2), q2.u);
            X.x = a0 ? x0n : X.x; Y.x = a0 ? y0n : Y.x; Z.x = a0 ? z0n : Z.x;
            X.z = a2 ? x2n : X.z; Y.z = a2 ? y2n : Y.z; Z.z = a2 ? z2n : Z.z;
            if (kIncr) { count_follow<kPack>(counts, a0, o0, n0, tk.x); count_follow<kPack>(counts, a2, o2, n2, tk.z); }

            float xr = __shfl_down_sync(kFull, X.x, 1), yr = __shfl_down_sync(kFull, Y.x, 1), zr = __shfl_down_sync(kFull, Z.x, 1);
            xr = has_r3 ? xr : X.w; yr = has_r3 ? yr : Y.w; zr = has_r3 ? zr : Z.w;
            float sx1, sy1, sz1, sx3, sy3, sz3, dx1, dy1, dz1, dx3, dy3, dz3;
            bond_sum(X.y, Y.y, Z.y, X.x, Y.x, Z.x, X.z, Y.z, Z.z, sx1, sy1, sz1);
            bond_sum(X.w, Y.w, Z.w, X.z, Y.z, Z.z, xr, yr, zr, sx3, sy3, sz3);
            smc_proposal(P, sx1, sy1, sz1, q1, dx1, dy1, dz1);
            smc_proposal(P, sx3, sy3, sz3, q3, dx3, dy3, dz3);
            const float x1n = X.y + dx1, y1n = Y.y + dy1, z1n = Z.y + dz1;
            const float x3n = X.w + dx3, y3n = Y.w + dy3, z3n = Z.w + dz3;
            const uint32_t o1 = cell_at<kPack>(P.g, X.y, Y.y, Z.y, tk.y), n1 = cell_at<kPack>(P.g, x1n, y1n, z1n, tk.y);
            const uint32_t o3 = cell_at<kPack>(P.g, X.w, Y.w, Z.w, tk.w), n3 = cell_at<kPack>(P.g, x3n, y3n, z3n, tk.w);
            const float e1 = field_delta(omega, o1, n1), e3 = field_delta(omega, o3, n3);
            a1 = metropolis(smc_exponent(hak, 2.0f, bonded_delta(half_k0, 2.0f, dx1, dy1, dz1, sx1, sy1, sz1), e1), q1.u);
            a3 = metropolis(smc_exponent(hak, mf3, bonded_delta(half_k0, mf3, dx3, dy3, dz3, sx3, sy3, sz3), e3), q3.u);
            X.y = a1 ? x1n : X.y; Y.y = a1 ? y1n : Y.y; Z.y = a1 ? z1n : Z.y;
            X.w = a3 ? x3n : X.w; Y.w = a3 ? y3n : Y.w; Z.w = a3 ? z3n : Z.w;
            if (kIncr) { count_follow<kPack>(counts, a1, o1, n1, tk.y); count_follow<kPack>(counts, a3, o3, n3, tk.w); }
        }

        if (active) {
            st_stream(x + i0, X);
            st_stream(y + i0, Y);
            st_stream(z + i0, Z);
        }

        const uint32_t nib = (a0 ? 1u : 0u) | (a1 ? 2u : 0u) | (a2 ? 4u : 0u) | (a3 ? 8u : 0u);
        n_acc += __popc(nib);
        if (kRecord) {
            // bit (b & 31) of word (b >> 5) for bead b; gid is a multiple of 4 only if gid0 is
            const unsigned long long bits = (unsigned long long)nib << (gid & 31u);
            if ((uint32_t)bits) atomicOr(dec_words + (gid >> 5), (uint32_t)bits);
            if ((uint32_t)(bits >> 32)) atomicOr(dec_words + (gid >> 5) + 1u, (uint32_t)(bits >> 32));
        }
        C = Cn;
        if (kOrder) E = En;
        tile = tile_n;
        tile_n = __shfl_sync(kFull, tile_nn, 0);
    }
    n_acc = __reduce_add_sync(kFull, n_acc);
    if (lane == 0 && n_acc)
        atomicAdd(acc_slots + ((blockIdx.x * kWarps + wib) % kAccSlots), (unsigned long long)n_acc);
}

// ------------------------------------------------------------------------------------------------
// a1 or a2 for any chain length: one thread per monomer of parity `parity` (set 0 / set 1).  The
// other parity is not written during this launch, so neighbours can be read from global memory.
//   half  = ceil(N / 2) threads per chain; n_items = n_chains * half; parity = 0, 1: first, second set
//   set_order  0: the first set is the even monomers; 1: the chain's first_set_bit decides
// ------------------------------------------------------------------------------------------------
template <int kMove, bool kIncr, bool kRecord, bool kPack>
__global__ void __launch_bounds__(256)
generic_move_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                    const float* __restrict__ omega, uint32_t* __restrict__ counts,
                    const uint32_t* __restrict__ toff_tab, uint32_t N, uint32_t half, uint32_t parity,
                    uint32_t set_order, uint64_t n_items, uint32_t gid0, const uint32_t* __restrict__ orig,
                    uint32_t* __restrict__ dec_words, unsigned long long* __restrict__ acc_slots)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool acc = false;
    uint64_t chain = 0;
    uint32_t j = N;
    if (t < n_items) {
        chain = t / half;
        uint32_t set = parity;       // launch 0 moves the first set of every chain, launch 1 the second
        if (set_order) set ^= first_set_bit(gid0 + orig[chain] * N, P.sweep_lo, P.sweep_hi, P.rk[0][0], P.rk[0][1]);
        j = 2u * (uint32_t)(t - chain * half) + set;
    }
    if (j < N) {                     // half = ceil(N / 2): the odd set of an odd-length chain has one member fewer
        const uint64_t i = chain * N + j;
        const bool has_l = j > 0u, has_r = j + 1u < N;
        float px = x[i], py = y[i], pz = z[i];
        const float xl = has_l ? x[i - 1] : px, yl = has_l ? y[i - 1] : py, zl = has_l ? z[i - 1] : pz;
        const float xr = has_r ? x[i + 1] : px, yr = has_r ? y[i + 1] : py, zr = has_r ? z[i + 1] : pz;
        const float mf = (float)((has_l ? 1 : 0) + (has_r ? 1 : 0));
        const uint32_t gid = gid0 + orig[chain] * N + j;   // the chain's identity, not its slot (soma_layout.cuh)
        acc = mc_move<kMove, kIncr, kPack>(P, omega, counts, px, py, pz, xl, yl, zl, xr, yr, zr, mf, toff_tab[j], gid);
        if (acc) { x[i] = px; y[i] = py; z[i] = pz; }
        if (kRecord && acc) atomicOr(dec_words + (gid >> 5), 1u << (gid & 31u));
    }
    const uint32_t n_acc = __popc(__ballot_sync(0xFFFFFFFFu, acc));
    if ((threadIdx.x & 31u) == 0 && n_acc)
        atomicAdd(acc_slots + ((t >> 5) % kAccSlots), (unsigned long long)n_acc);
}

// ------------------------------------------------------------------------------------------------
// Molecular architecture, stored once per molecule type as the array of 32-bit words of Fig. 2:
//   word 0                 N, the number of monomers
//   words 1 .. N           per monomer: upper 3 bytes = index (in this array) of its first bond word, 0 if it has
//                          no bond; lowest byte = its type
//   then the bond words    upper 27 bits = signed offset from the monomer to its bonded partner, next 4 bits =
//                          bond type (0: the harmonic spring of Eq. 2, the only one), lowest bit = 1 on the
//                          monomer's last bond.  A monomer's partners come in ascending order (R25).
// Behind it, what the set scheme needs (not part of Fig. 2):
//   members[N] (set by set) | set_off[n_sets + 1] | set_magic[n_sets] (floor(2^32 / set size) + 1)
// arch_bond_sum() walks the bond words of monomer j: s = sum over its partners of (r_j - r_partner) in list order
// (the first term assigned, the others added, so that a linear chain given as bonds reproduces the chain kernels
// bit for bit); returns the number of partners.  pos(k) gives the position of monomer k of the same molecule.
// ------------------------------------------------------------------------------------------------
template <typename PosOf>
__device__ __forceinline__ uint32_t arch_bond_sum(const uint32_t* __restrict__ arch, uint32_t j, float px, float py, float pz,
                                                  PosOf pos, float& sx, float& sy, float& sz)
{
    sx = sy = sz = 0.0f;
    uint32_t at = arch[1u + j] >> 8, n = 0u;
    if (at == 0u) return 0u;
    uint32_t w;
    do {
        w = arch[at++];
        const uint32_t k = j + (uint32_t)((int32_t)w >> 5);              // signed 27-bit offset
        float qx, qy, qz;
        pos(k, qx, qy, qz);
        const float bx = px - qx, by = py - qy, bz = pz - qz;
        if (n == 0u) { sx = bx; sy = by; sz = bz; } else { sx = sx + bx; sy = sy + by; sz = sz + bz; }
        ++n;
    } while (!(w & 1u));
    return n;
}

// ------------------------------------------------------------------------------------------------
// One independent set of a general molecular architecture (DESIGN.md
// R25): one thread per member of set `i_set` of every molecule; the host launches the sets one after the
// other.  arch: the architecture words above (global memory); members: the members of this set.
// ------------------------------------------------------------------------------------------------
template <int kMove, bool kIncr, bool kRecord, bool kPack>
__global__ void __launch_bounds__(256)
arch_move_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                 const float* __restrict__ omega, uint32_t* __restrict__ counts,
                 const uint32_t* __restrict__ toff_tab, const uint32_t* __restrict__ arch,
                 const uint32_t* __restrict__ members, uint32_t N,
                 uint32_t set_size, uint64_t n_items, uint32_t gid0, const uint32_t* __restrict__ orig,
                 uint32_t* __restrict__ dec_words, unsigned long long* __restrict__ acc_slots)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool acc = false;
    if (t < n_items) {
        const uint64_t mol = t / set_size;
        const uint32_t j = members[(uint32_t)(t - mol * set_size)];      // monomer of this set member
        const uint64_t base = mol * N, i = base + j;
        float px = x[i], py = y[i], pz = z[i];
        float sx, sy, sz;
        const uint32_t n_nb = arch_bond_sum(arch, j, px, py, pz,        // other sets: not written in this launch
            [&](uint32_t k, float& qx, float& qy, float& qz) { qx = x[base + k]; qy = y[base + k]; qz = z[base + k]; },
            sx, sy, sz);
        const uint32_t gid = gid0 + orig[mol] * N + j;
        acc = mc_move_s<kMove, kIncr, kPack>(P, omega, counts, px, py, pz, sx, sy, sz, (float)n_nb, toff_tab[j], gid);
        if (acc) { x[i] = px; y[i] = py; z[i] = pz; }
        if (kRecord && acc) atomicOr(dec_words + (gid >> 5), 1u << (gid & 31u));
    }
    const uint32_t n_acc = __popc(__ballot_sync(0xFFFFFFFFu, acc));
    if ((threadIdx.x & 31u) == 0 && n_acc)
        atomicAdd(acc_slots + ((t >> 5) % kAccSlots), (unsigned long long)n_acc);
}

// The same with the molecules staged in shared memory, all independent sets in one launch: a warp copies a
// group of consecutive molecules (group * N consecutive beads per coordinate array) with coalesced loads,
// works through the sets one after the other -- the members of a set of all molecules of the group spread over
// its lanes, neighbours read from shared memory, __syncwarp between sets -- and writes the group back: every
// position crosses HBM once per sweep, and the architecture (offsets, neighbour lists, set members: the
// compressed-architecture array of PAPER.md:344-354 in plain 32-bit words) sits in shared memory too.
//   arch        the architecture words above with members | set_off | set_magic behind them
//               (set_magic: item / set size by one multiply, exact below 2^16)
//   group       molecules per warp and pass (group * N <= 65535)
// Dynamic shared memory: arch words + toff[N], then warps * 3 * group * N floats.
template <int kMove, bool kIncr, bool kRecord, bool kPack>
__global__ void __launch_bounds__(256)
arch_staged_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                   const float* __restrict__ omega, uint32_t* __restrict__ counts,
                   const uint32_t* __restrict__ toff_tab, const uint32_t* __restrict__ arch, uint32_t n_arch_words,
                   uint32_t N, uint32_t n_bonds, uint32_t n_sets, uint32_t group, uint64_t n_mol, uint32_t gid0,
                   const uint32_t* __restrict__ orig, uint32_t* __restrict__ dec_words,
                   unsigned long long* __restrict__ acc_slots)
{
    extern __shared__ __align__(16) uint32_t s_words[];
    const uint32_t lane = threadIdx.x & 31u, wib = threadIdx.x >> 5, warps = blockDim.x >> 5;
    for (uint32_t k = threadIdx.x; k < n_arch_words; k += blockDim.x) s_words[k] = arch[k];
    for (uint32_t k = threadIdx.x; k < N; k += blockDim.x) s_words[n_arch_words + k] = toff_tab[k];
    __syncthreads();
    const uint32_t* members = s_words + 1u + N + 2u * n_bonds;
    const uint32_t* set_off = members + N;
    const uint32_t* set_magic = set_off + (n_sets + 1u);
    const uint32_t* toff = s_words + n_arch_words;
    const uint32_t head = (n_arch_words + N + 3u) & ~3u;
    float* sx = reinterpret_cast<float*>(s_words + head) + (size_t)wib * 3u * group * N;
    float* sy = sx + group * N;
    float* sz = sy + group * N;
    const uint64_t n_groups = (n_mol + group - 1u) / group;
    uint32_t n_acc = 0;
    for (uint64_t grp = (uint64_t)blockIdx.x * warps + wib; grp < n_groups; grp += (uint64_t)gridDim.x * warps) {
        const uint64_t m0 = grp * group, base = m0 * N;
        const uint32_t n_here = (uint32_t)min((uint64_t)group, n_mol - m0), n_floats = n_here * N;
        for (uint32_t e = lane; e < n_floats; e += 32u) {
            sx[e] = x[base + e];
            sy[e] = y[base + e];
            sz[e] = z[base + e];
        }
        __syncwarp();
        for (uint32_t i_set = 0; i_set < n_sets; ++i_set) {
            const uint32_t first = set_off[i_set], set_size = set_off[i_set + 1u] - first, magic = set_magic[i_set];
            const uint32_t items = n_here * set_size;
            for (uint32_t it = lane; it < items; it += 32u) {
                const uint32_t m = set_size == 1u ? it : __umulhi(it, magic);   // it / set_size (2^32 / 1 has no 32-bit magic)
                const uint32_t j = members[first + (it - m * set_size)];
                const uint32_t i = m * N + j;
                float px = sx[i], py = sy[i], pz = sz[i];
                float bsx, bsy, bsz;
                const uint32_t mol0 = m * N;
                const uint32_t n_nb = arch_bond_sum(s_words, j, px, py, pz,   // other sets: not written during this set
                    [&](uint32_t k, float& qx, float& qy, float& qz) { qx = sx[mol0 + k]; qy = sy[mol0 + k]; qz = sz[mol0 + k]; },
                    bsx, bsy, bsz);
                const uint32_t gid = gid0 + orig[m0 + m] * N + j;
                const bool acc = mc_move_s<kMove, kIncr, kPack>(P, omega, counts, px, py, pz, bsx, bsy, bsz, (float)n_nb,
                                                                toff[j], gid);
                if (acc) { sx[i] = px; sy[i] = py; sz[i] = pz; }
                if (kRecord && acc) atomicOr(dec_words + (gid >> 5), 1u << (gid & 31u));
                n_acc += acc ? 1u : 0u;
            }
            __syncwarp();
        }
        for (uint32_t e = lane; e < n_floats; e += 32u) {
            x[base + e] = sx[e];
            y[base + e] = sy[e];
            z[base + e] = sz[e];
        }
        __syncwarp();
    }
    n_acc = __reduce_add_sync(0xFFFFFFFFu, n_acc);
    if (lane == 0 && n_acc)
        atomicAdd(acc_slots + ((blockIdx.x * warps + wib) % kAccSlots), (unsigned long long)n_acc);
}

// ------------------------------------------------------------------------------------------------
// Molecule-parallel scheme (Code 1): one thread per molecule, which N times picks
// one of its particles at random and attempts to move it; attempts of one molecule are sequential
// (a particle picked twice, or a neighbour moved earlier, is seen in its new place), molecules are
// independent while omega is frozen.  Attempt k of the chain whose first bead has global index f owns
// the Philox counter word f + k: kind 4 picks the particle, i = floor(w0 N / 2^32); kind 1 / 2 gives
// the move's random numbers (R24).  The chain's 3 N floats are touched N times by the same
// thread, so they stay in L1; lanes of a warp work on 32 consecutive chains.
//   dec_words   bit of attempt f + k (not of a bead), or unused
// ------------------------------------------------------------------------------------------------
template <int kMove, bool kIncr, bool kRecord, bool kPack>
__global__ void __launch_bounds__(128)
molecule_move_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                     const float* __restrict__ omega, uint32_t* __restrict__ counts,
                     const uint32_t* __restrict__ toff_tab, uint32_t N, uint64_t n_chains, uint32_t gid0,
                     const uint32_t* __restrict__ orig, uint32_t* __restrict__ dec_words,
                     unsigned long long* __restrict__ acc_slots)
{
    const uint64_t chain = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t n_acc = 0;
    if (chain < n_chains) {
        const uint64_t base = chain * N;
        const uint32_t first = gid0 + orig[chain] * N;
        for (uint32_t k = 0; k < N; ++k) {                    // "sequential iteration of particles"
            const uint32_t attempt = first + k;
            uint32_t w[4];
            philox4x32_10(attempt, P.sweep_lo, P.sweep_hi, 0x400u, P.rk[0][0], P.rk[0][1], w);
            const uint32_t j = __umulhi(w[0], N);             // "select random particle to move"
            const uint64_t i = base + j;
            const bool has_l = j > 0u, has_r = j + 1u < N;
            float px = x[i], py = y[i], pz = z[i];
            const float xl = has_l ? x[i - 1] : px, yl = has_l ? y[i - 1] : py, zl = has_l ? z[i - 1] : pz;
            const float xr = has_r ? x[i + 1] : px, yr = has_r ? y[i + 1] : py, zr = has_r ? z[i + 1] : pz;
            const float mf = (float)((has_l ? 1 : 0) + (has_r ? 1 : 0));
            const bool acc = mc_move<kMove, kIncr, kPack>(P, omega, counts, px, py, pz, xl, yl, zl, xr, yr, zr, mf,
                                                   toff_tab[j], attempt);
            if (acc) { x[i] = px; y[i] = py; z[i] = pz; }
            if (kRecord && acc) atomicOr(dec_words + (attempt >> 5), 1u << (attempt & 31u));
            n_acc += acc ? 1u : 0u;
        }
    }
    n_acc = __reduce_add_sync(0xFFFFFFFFu, n_acc);
    if ((threadIdx.x & 31u) == 0 && n_acc)
        atomicAdd(acc_slots + ((chain >> 5) % kAccSlots), (unsigned long long)n_acc);
}

// The same scheme with the chains staged in shared memory: a warp copies 32 consecutive chains
// (32 N consecutive beads per coordinate array) with coalesced loads, every lane then runs the N
// attempts of its own chain out of shared memory, and the warp writes the 32 chains back coalesced --
// each position crosses HBM once per sweep, as in the fused kernel.  Dynamic shared memory:
// warps_per_block * 3 * 32 N floats.
template <int kMove, bool kIncr, bool kRecord, bool kPack>
__global__ void __launch_bounds__(128)
molecule_staged_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                       const float* __restrict__ omega, uint32_t* __restrict__ counts,
                       const uint32_t* __restrict__ toff_tab, uint32_t N, uint64_t n_chains, uint32_t gid0,
                       const uint32_t* __restrict__ orig, uint32_t* __restrict__ dec_words,
                       unsigned long long* __restrict__ acc_slots)
{
    extern __shared__ __align__(16) float stage_f[];
    const uint32_t lane = threadIdx.x & 31u, wib = threadIdx.x >> 5, warps = blockDim.x >> 5;
    float* sx = stage_f + (size_t)wib * 96u * N;              // this warp's 3 x 32 N floats
    float* sy = sx + 32u * N;
    float* sz = sy + 32u * N;
    const uint64_t n_groups = (n_chains + 31u) / 32u;
    uint32_t n_acc = 0;
    for (uint64_t grp = (uint64_t)blockIdx.x * warps + wib; grp < n_groups; grp += (uint64_t)gridDim.x * warps) {
        const uint64_t chain0 = grp * 32u, base = chain0 * N;
        const uint32_t n_here = (uint32_t)min((uint64_t)32u, n_chains - chain0), n_floats = n_here * N;
        for (uint32_t e = lane; e < n_floats; e += 32u) {
            sx[e] = x[base + e];
            sy[e] = y[base + e];
            sz[e] = z[base + e];
        }
        __syncwarp();
        if (lane < n_here) {
            const uint32_t mine = lane * N;
            const uint32_t first = gid0 + orig[chain0 + lane] * N;
            #pragma unroll kMolUnroll
            for (uint32_t k = 0; k < N; ++k) {                // "sequential iteration of particles"
                const uint32_t attempt = first + k;
                uint32_t w[4];
                philox4x32_10(attempt, P.sweep_lo, P.sweep_hi, 0x400u, P.rk[0][0], P.rk[0][1], w);
                const uint32_t j = __umulhi(w[0], N);         // "select random particle to move"
                const uint32_t i = mine + j;
                const bool has_l = j > 0u, has_r = j + 1u < N;
                float px = sx[i], py = sy[i], pz = sz[i];
                const float xl = has_l ? sx[i - 1] : px, yl = has_l ? sy[i - 1] : py, zl = has_l ? sz[i - 1] : pz;
                const float xr = has_r ? sx[i + 1] : px, yr = has_r ? sy[i + 1] : py, zr = has_r ? sz[i + 1] : pz;
                const float mf = (float)((has_l ? 1 : 0) + (has_r ? 1 : 0));
                const bool acc = mc_move<kMove, kIncr, kPack>(P, omega, counts, px, py, pz, xl, yl, zl, xr, yr, zr, mf,
                                                       toff_tab[j], attempt);
                if (acc) { sx[i] = px; sy[i] = py; sz[i] = pz; }
                if (kRecord && acc) atomicOr(dec_words + (attempt >> 5), 1u << (attempt & 31u));
                n_acc += acc ? 1u : 0u;
            }
        }
        __syncwarp();
        for (uint32_t e = lane; e < n_floats; e += 32u) {
            x[base + e] = sx[e];
            y[base + e] = sy[e];
            z[base + e] = sz[e];
        }
        __syncwarp();
    }
    n_acc = __reduce_add_sync(0xFFFFFFFFu, n_acc);
    if (lane == 0 && n_acc)
        atomicAdd(acc_slots + ((blockIdx.x * warps + wib) % kAccSlots), (unsigned long long)n_acc);
}

// ------------------------------------------------------------------------------------------------
// a3  occupation numbers from scratch (Eq. 4): one count per bead into the cell's record.
// ------------------------------------------------------------------------------------------------
template <bool kPack>
__global__ void __launch_bounds__(256)
histogram_kernel(const GridP g, const float* __restrict__ x, const float* __restrict__ y,
                 const float* __restrict__ z, const uint32_t* __restrict__ toff_tab, uint32_t N,
                 uint32_t n_beads, uint32_t* __restrict__ counts, uint32_t* __restrict__ n_outside)
{
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t bad = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_beads; i += stride) {   // 64-bit: n_beads may be 2^32 - 1
        const uint32_t j = (uint32_t)(i % N);
        const float xi = x[i], yi = y[i], zi = z[i];
        const uint32_t idx = cell_at<kPack>(g, xi, yi, zi, toff_tab[j] + g.k_rec);
        if (kPack) atomicAdd(counts + (idx >> 1), 1u << ((idx & 1u) << 4));
        else atomicAdd(counts + idx, 1u);
        // the supported coordinates of cell_raw(): |t n| < 2^22 per axis (a NaN fails the comparison too)
        const bool ok = fabsf(xi * g.inv_L[0] * g.nf[0]) < 4194304.0f && fabsf(yi * g.inv_L[1] * g.nf[1]) < 4194304.0f &&
                        fabsf(zi * g.inv_L[2] * g.nf[2]) < 4194304.0f;
        bad += ok ? 0u : 1u;
    }
    if (bad && n_outside) atomicAdd(n_outside, bad);
}

// ------------------------------------------------------------------------------------------------
// a4  omega_i(c) from n_i(c), Eq. 12: phi_i = n_i / (rho_0 DeltaL^3),
//     K^0: omega_i = kappa_0 (sum phi - 1) - sum_{k != i} chi_0ik/2 (phi_i - phi_k)
//     K^1: omega_i = kappa_0 (sum phi - 1) + sum_{k != i} chi_0ik phi_k
//     + ext_i(c) if an external field is set; +inf in forbidden cells, so that Eq. 15 makes every move
//     into such a cell cost +inf and the Metropolis rule rejects it (R23)
// ------------------------------------------------------------------------------------------------
// omega of one cell from its occupation numbers n[0 .. nt); ext is [type][cell] (the caller's layout)
template <int kTypes>
__device__ __forceinline__ void field_of_cell(const FieldP& F, const uint32_t (&n)[kMaxTypes], uint32_t c,
                                              const float* __restrict__ ext, const uint8_t* __restrict__ forbidden,
                                              float (&w_out)[kMaxTypes])
{
    const int nt = kTypes > 0 ? kTypes : F.n_types;
    float phi[kMaxTypes];
#pragma unroll
    for (int i = 0; i < kMaxTypes; ++i)
        if (i < nt) phi[i] = (float)n[i] * F.inv_nbar;
    float sum = phi[0];
#pragma unroll
    for (int i = 1; i < kMaxTypes; ++i)
        if (i < nt) sum = sum + phi[i];
    const float pressure = F.kappa0 * (sum - 1.0f);
#pragma unroll
    for (int i = 0; i < kMaxTypes; ++i) {
        if (i >= nt) continue;
        float w = pressure;
#pragma unroll
        for (int k = 0; k < kMaxTypes; ++k) {
            if (k >= nt || k == i) continue;
            if (F.hamiltonian == 0)
                w = w - F.half_chi0[i][k] * (phi[i] - phi[k]);
            else
                w = w + F.chi0[i][k] * phi[k];
        }
        // external fields: a static type-specific field; +inf where no particle may enter
        if (ext) w = w + ext[(size_t)i * F.cells + c];
        if (forbidden && forbidden[c]) w = __int_as_float(0x7F800000);
        w_out[i] = w;
    }
}

// Packed occupation numbers (kPack): has a 16-bit half overflowed?  The word of a cell is n_A + 65536 n_B
// modulo 2^32 exactly, so as long as both numbers are below 65536 the halves are the numbers and the sum of
// all halves is the number of beads counted; a number of 65536 or more lowers that sum (by 65535 per carry
// into the upper half, by 65536 per carry out of the word) and nothing can raise it.  The field kernel
// therefore adds up the halves it decodes anyway -- one atomic per block on *ticket_sum, block count in the
// bits from 40 up, sum below -- and the block that draws the last ticket compares the sum with the number
// of beads and sets the sticky flag *overflow (pinned host memory, written once if ever) if they differ.

// One thread per cell.  counts and omega as planes [type][cell], or (kPack, two types) as records per cell
// with packed counts.  kTypes = 0: any number of types (F.n_types).
//   exchange   NULL, or (a part of a system spread over several GPUs) the array the move
//              kernels of this rank counted into, summed over all ranks by the caller: the change of the whole
//              system's occupation numbers since the last call, in the format of counts.  It is added to counts
//              and cleared for the next sweep.  Sums of words are exact modulo 2^32, packed or not.
//   peers      NULL, or the exchange arrays of ALL ranks (this one included) in peer memory -- other GPUs over
//              NVLink / NVSwitch, or CUDA IPC mappings: the kernel does the reduction itself, word by word, instead
//              of a collective before it (n_peers pointers, each read at word offset peer_off).  Nobody may
//              still be writing them (the caller's barrier).  The arrays read are left as they are -- other
//              ranks read them too -- and `exchange` is then this rank's OTHER buffer, which every rank has
//              finished reading a sweep ago: it is cleared for the next sweep (double buffering, soma_b200.cu).
template <int kTypes, bool kPack>
__global__ void __launch_bounds__(256)
field_kernel(const FieldP F, uint32_t* __restrict__ counts, float* __restrict__ omega,
             const float* __restrict__ ext, const uint8_t* __restrict__ forbidden,
             unsigned long long* __restrict__ ticket_sum, uint32_t* __restrict__ overflow,
             unsigned long long n_counted, uint32_t* __restrict__ exchange,
             const uint32_t* const* __restrict__ peers, uint32_t n_peers, size_t peer_off)
{
    static_assert(!kPack || kTypes == 2, "packed occupation numbers: two types");
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    pdl_trigger();
    pdl_wait();                                               // counts of the preceding move kernel
    uint32_t total = 0;
    if (c < F.cells) {
        const int nt = kTypes > 0 ? kTypes : F.n_types;
        uint32_t n[kMaxTypes];
        float w[kMaxTypes];
        if (kPack) {
            uint32_t v = counts[c];
            if (peers) {
                for (uint32_t r = 0; r < n_peers; ++r) v += __ldcg(peers[r] + peer_off + c);
                counts[c] = v;
                exchange[c] = 0u;
            } else if (exchange) {
                v += exchange[c];
                counts[c] = v;
                exchange[c] = 0u;
            }
            n[0] = v & 0xFFFFu;
            n[1] = v >> 16;
            total = n[0] + n[1];
        } else {
#pragma unroll
            for (int i = 0; i < kMaxTypes; ++i) {
                if (i >= nt) continue;
                const size_t at = (size_t)i * F.cells + c;
                n[i] = counts[at];
                if (peers) {
                    for (uint32_t r = 0; r < n_peers; ++r) n[i] += __ldcg(peers[r] + peer_off + at);
                    counts[at] = n[i];
                    exchange[at] = 0u;
                } else if (exchange) {
                    n[i] += exchange[at];
                    counts[at] = n[i];
                    exchange[at] = 0u;
                }
            }
        }
        field_of_cell<kTypes>(F, n, c, ext, forbidden, w);
        if (kPack) {
            reinterpret_cast<float2*>(omega)[c] = make_float2(w[0], w[1]);
        } else {
#pragma unroll
            for (int i = 0; i < kMaxTypes; ++i)
                if (i < nt) omega[(size_t)i * F.cells + c] = w[i];
        }
    }
    if (kPack) {
        __shared__ uint32_t s_total;
        if (threadIdx.x == 0) s_total = 0u;
        __syncthreads();
        total = __reduce_add_sync(0xFFFFFFFFu, total);
        if ((threadIdx.x & 31u) == 0u && total) atomicAdd(&s_total, total);
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned long long mine = (1ull << 40) | (unsigned long long)s_total;
            const unsigned long long before = atomicAdd(ticket_sum, mine);
            if ((before >> 40) == (unsigned long long)(gridDim.x - 1u)) {      // the last block of this launch
                if (((before + mine) & ((1ull << 40) - 1ull)) != n_counted) *overflow = 1u;
                *ticket_sum = 0ull;                                            // for the next launch
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Grid arrays between the device format (planes, or records per cell with packed occupation numbers) and
// the caller's [type][cell] arrays of the C ABI.
// ------------------------------------------------------------------------------------------------
template <bool kPack>
__global__ void __launch_bounds__(256)
export_grid_kernel(const float* __restrict__ omega, const uint32_t* __restrict__ counts, uint32_t cells, uint32_t nt,
                   float* __restrict__ omega_out, uint32_t* __restrict__ counts_out)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (uint64_t)cells * nt) return;
    const uint32_t t = (uint32_t)(i / cells), c = (uint32_t)(i - (uint64_t)t * cells);
    if (omega_out) omega_out[i] = kPack ? omega[(size_t)c * nt + t] : omega[i];
    if (counts_out) {
        if (kPack) counts_out[i] = t ? counts[c] >> 16 : counts[c] & 0xFFFFu;
        else counts_out[i] = counts[i];
    }
}

// src: occupation numbers [type][cell] (e.g. summed over the ranks of a sharded system) -> internal layout
template <bool kPack>
__global__ void __launch_bounds__(256)
import_counts_kernel(const uint32_t* __restrict__ src, uint32_t cells, uint32_t nt, uint32_t* __restrict__ dst,
                     uint32_t* __restrict__ overflow)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= cells) return;
    if (kPack) {
        const uint32_t a = src[c], b = src[(size_t)cells + c];
        if ((a | b) >> 16) *overflow = 1u;
        dst[c] = a + (b << 16);
    } else {
        for (uint32_t t = 0; t < nt; ++t) dst[(size_t)t * cells + c] = src[(size_t)t * cells + c];
    }
}

// ------------------------------------------------------------------------------------------------
// Start state: one thread per chain walks its monomers.  Kind-0 Philox words of every bead; first
// bead uniform in the box, then Box-Muller Gaussian bonds of per-axis std sigma, running sum in
// double, one rounding to fp32.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
init_walk_kernel(float* __restrict__ x, float* __restrict__ y, float* __restrict__ z, uint64_t n_chains,
                 uint32_t N, uint32_t gid0, uint32_t key0, uint32_t key1, double Lx, double Ly, double Lz,
                 double sigma)
{
    const uint64_t chain = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (chain >= n_chains) return;
    const double inv32 = 1.0 / 4294967296.0, two_pi = 6.283185307179586476925286766559;
    double px = 0.0, py = 0.0, pz = 0.0;
    for (uint32_t j = 0; j < N; ++j) {
        const uint64_t i = chain * N + j;
        uint32_t w[4];
        philox4x32_10(gid0 + (uint32_t)i, 0u, 0u, 0u, key0, key1, w);
        if (j == 0) {
            px = Lx * ((double)w[0] * inv32);
            py = Ly * ((double)w[1] * inv32);
            pz = Lz * ((double)w[2] * inv32);
        } else {
            const double ra = sqrt(-2.0 * log(((double)w[0] + 1.0) * inv32));
            const double rb = sqrt(-2.0 * log(((double)w[2] + 1.0) * inv32));
            double sa, ca, sb, cb;
            sincos(two_pi * ((double)w[1] * inv32), &sa, &ca);
            sincos(two_pi * ((double)w[3] * inv32), &sb, &cb);
            px += sigma * (ra * ca);
            py += sigma * (ra * sa);
            pz += sigma * (rb * cb);
        }
        x[i] = (float)px; y[i] = (float)py; z[i] = (float)pz;
    }
}

// counts += exchange, exchange = 0: a sweep of a shard after which omega is not refreshed (SOMA_OPT_FIELD_INTERVAL)
__global__ void __launch_bounds__(256)
fold_exchange_kernel(uint32_t* __restrict__ counts, uint32_t* __restrict__ exchange, uint64_t n_words)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_words) return;
    counts[i] += exchange[i];
    exchange[i] = 0u;
}

}  // namespace soma
