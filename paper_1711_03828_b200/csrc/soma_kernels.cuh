// soma_kernels.cuh -- device code of the SCMF Monte-Carlo step for sm_100a (B200).
//
// Kernels (PAPER.md = arXiv:1711.03828 text; DESIGN.md has the data layout and rooflines):
//   fused_sweep_kernel    a1+a2(+a3): one warp owns 128 consecutive beads (= whole chains, N | 128),
//                         4 beads per lane in registers, even monomers then odd monomers
//                         (independent sets of Fig. 1 / Code 2), neighbours by
//                         warp shuffle, each position read and written once per sweep.
//   generic_move_kernel   a1 or a2 for any chain length: one thread per monomer of one parity.
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

#ifndef SOMA_FUSED_MIN_BLOCKS
#define SOMA_FUSED_MIN_BLOCKS 3      // resident 256-thread blocks per SM the fused kernel is compiled for
#endif

struct GridP {
    float inv_L[3];   // fl32(1 / L_a)
    float nf[3];      // (float) n_a
    uint32_t n[3];
    uint32_t nm1[3];  // n_a - 1
    uint32_t cells;
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

// Same generator with the key schedule precomputed on the host (MoveP::rk lives in the kernel's
// constant bank, so the round keys cost no instruction).
__device__ __forceinline__ void philox4x32_10_rk(uint32_t a, uint32_t b, uint32_t c, uint32_t d,
                                                 const uint32_t (&rk)[10][2], uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
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

// top 23 bits -> float in [1, 2), exact
__device__ __forceinline__ float u23(uint32_t w) { return __uint_as_float(0x3F800000u | (w >> 9)); }

__device__ __forceinline__ float ex2_approx(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// ------------------------------------------------------------------------------------------------
// Pi_c of Eq. 4: the cell that contains r, periodic.  Per axis: position in
// units of the box length t = x * (1/L), folded by its fractional part frac = t - floor(t), cell =
// floor(frac * n) (exact product) clamped to n-1.
// FRND and F2I run on the XU pipe (16 lanes/clk/SM, shared with MUFU) and saturated it in the first
// version of this kernel, so floor and float->int are done on the FMA/ALU pipes instead:
//   floor(t)       = fl_down(t + 1.5 * 2^23) - 1.5 * 2^23     exact for |t| < 2^22
//   floor(frac n)  = mantissa of fl_down(frac * n + 2^23)      exact for frac * n < 2^23
// FMUL, FADD.RM, FADD, FADD, FFMA.RM, IADD, VIMNMX.U32 per axis.  The unsigned min keeps the index
// in range for every input (also NaN and |t| >= 2^22, which is outside the supported domain:
// |x_a| < 2^22 L_a, R7).
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t axis_cell(float x, float inv_L, float nf, uint32_t n_minus_1)
{
    const float t = x * inv_L;
    const float fl = __fadd_rd(t, 12582912.0f) - 12582912.0f;
    const float frac = t - fl;
    const float s = __fmaf_rd(frac, nf, 8388608.0f);
    return min(__float_as_uint(s) - 0x4B000000u, n_minus_1);
}

__device__ __forceinline__ uint32_t cell_of(const GridP& g, float x, float y, float z)
{
    const uint32_t cx = axis_cell(x, g.inv_L[0], g.nf[0], g.nm1[0]);
    const uint32_t cy = axis_cell(y, g.inv_L[1], g.nf[1], g.nm1[1]);
    const uint32_t cz = axis_cell(z, g.inv_L[2], g.nf[2], g.nm1[2]);
    return (cx * g.n[1] + cy) * g.n[2] + cz;
}

// ------------------------------------------------------------------------------------------------
// One Monte-Carlo move of one bead ("MC scheme for particle ip", Code 2).
//   (x,y,z)        the bead, updated in place when the move is accepted
//   (xl..),(xr..)  chain neighbours; an absent neighbour is passed as the bead itself (bond 0)
//   mf             number of bonded neighbours as float
//   toff           type * cells, offset of this bead type's plane in omega / counts
//   gid            global bead index = Philox counter word 0
// kMove 1: local displacement uniform in (-A,A)^3 + Metropolis.
// kMove 2: Smart-MC, force-biased proposal from the bonded force + Metropolis-Hastings.
// kIncr: the occupation numbers follow the accepted move (+1 new cell, -1 old cell) -- integer
// arithmetic, so they stay identical to a fresh histogram (a3).  No branch on the hot path: the
// gathers and the count updates are predicated, so the two moves of a set interleave (ILP 2).
// ------------------------------------------------------------------------------------------------
template <int kMove, bool kIncr>
__device__ __forceinline__ bool mc_move(const MoveP& P, const float* __restrict__ omega,
                                        uint32_t* __restrict__ counts, float& x, float& y, float& z,
                                        float xl, float yl, float zl, float xr, float yr, float zr,
                                        float mf, uint32_t toff, uint32_t gid)
{
    // s = sum over neighbours of (r - r_nb)
    const float sx = (x - xl) + (x - xr);
    const float sy = (y - yl) + (y - yr);
    const float sz = (z - zl) + (z - zr);

    float dx, dy, dz, u, log_ratio = 0.0f;
    if (kMove == 1) {
        uint32_t w[4];
        philox4x32_10_rk(gid, P.sweep_lo, P.sweep_hi, 0x100u, P.rk, w);
        dx = fmaf(u23(w[0]), P.c1, P.c0);
        dy = fmaf(u23(w[1]), P.c1, P.c0);
        dz = fmaf(u23(w[2]), P.c1, P.c0);
        u = u23(w[3]) - 1.0f;
    } else {
        uint32_t w[4], v[4];
        philox4x32_10_rk(gid, P.sweep_lo, P.sweep_hi, 0x200u, P.rk, w);
        philox4x32_10_rk(gid, P.sweep_lo, P.sweep_hi, 0x201u, P.rk, v);
        const float ra = sqrtf(-2.0f * logf(2.0f - u23(w[0])));
        const float rb = sqrtf(-2.0f * logf(2.0f - u23(w[2])));
        const float two_pi = 6.283185307179586f;
        float sa, ca, sb, cb;
        sincosf(two_pi * (u23(w[1]) - 1.0f), &sa, &ca);
        sincosf(two_pi * (u23(w[3]) - 1.0f), &sb, &cb);
        const float gx = ra * ca, gy = ra * sa, gz = rb * cb;
        u = u23(v[0]) - 1.0f;
        const float Fx = -P.k0 * sx, Fy = -P.k0 * sy, Fz = -P.k0 * sz;   // bonded force
        dx = fmaf(P.a_s, Fx, P.noise * gx);
        dy = fmaf(P.a_s, Fy, P.noise * gy);
        dz = fmaf(P.a_s, Fz, P.noise * gz);
        // ln T(r->r') - ln T(r'->r) = ( |d + a_s F'|^2 - |d - a_s F|^2 ) / (4 a_s),  F' = F - k_0 m d
        const float km = P.k0 * mf;
        float fwd = 0.0f, rev = 0.0f;
        {
            const float ef = dx - P.a_s * Fx, er = dx + P.a_s * (Fx - km * dx);
            fwd = fmaf(ef, ef, fwd); rev = fmaf(er, er, rev);
        }
        {
            const float ef = dy - P.a_s * Fy, er = dy + P.a_s * (Fy - km * dy);
            fwd = fmaf(ef, ef, fwd); rev = fmaf(er, er, rev);
        }
        {
            const float ef = dz - P.a_s * Fz, er = dz + P.a_s * (Fz - km * dz);
            fwd = fmaf(ef, ef, fwd); rev = fmaf(er, er, rev);
        }
        log_ratio = (rev - fwd) / P.four_as;
    }

    const float x2 = x + dx, y2 = y + dy, z2 = z + dz;   // r' = fl32(r + d)

    // non-bonded: dE_nb = omega_k(c') - omega_k(c), Eq. 15; 0 when the cell is kept
    const uint32_t i_old = toff + cell_of(P.g, x, y, z);
    const uint32_t i_new = toff + cell_of(P.g, x2, y2, z2);
    const bool moved = i_new != i_old;
    float w_new = 0.0f, w_old = 0.0f;
    if (moved) {
        w_new = __ldg(omega + i_new);
        w_old = __ldg(omega + i_old);
    }
    const float e_nb = w_new - w_old;

    // bonded: dE_b = k_0/2 (2 d.s + m |d|^2), Eq. 2
    const float ds = fmaf(dz, sz, fmaf(dy, sy, dx * sx));
    const float dd = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
    const float e_b = (kMove == 1 ? P.hk : 0.5f * P.k0) * fmaf(2.0f, ds, mf * dd);

    float dE = e_b + e_nb;
    if (kMove == 2) dE = dE + log_ratio;

    // Metropolis: accept iff dE <= 0 or u < exp(-dE)
    const bool acc = (dE <= 0.0f) || (u < ex2_approx(dE * -1.4426950408889634f));
    x = acc ? x2 : x;
    y = acc ? y2 : y;
    z = acc ? z2 : z;
    if (kIncr && acc && moved) {
        atomicAdd(counts + i_new, 1u);
        atomicAdd(counts + i_old, 0xFFFFFFFFu);
    }
    return acc;
}

// ------------------------------------------------------------------------------------------------
// a1 + a2 fused, chain-resident.  Requires N in {4, 8, ..., 128} (N | 128) so that a 128-bead warp
// tile holds whole chains; the architecture's bead array starts 512-byte aligned.  Only full tiles
// are processed here; the host sends a ragged tail (< 128 beads, whole chains) to the generic kernel.
//   x,y,z       base of this architecture's beads (padded layout)
//   toff_tab    [N] type * cells of every monomer of the chain
//   n_tiles     full tiles of this architecture (n_chains * N / 128)
//   gid0        global index of the architecture's first bead
//   dec_bytes   decision bitmap of the architecture (byte view), or unused
// ------------------------------------------------------------------------------------------------
template <int kMove, bool kIncr, bool kRecord>
__global__ void __launch_bounds__(256, SOMA_FUSED_MIN_BLOCKS)
fused_sweep_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                   const float* __restrict__ omega, uint32_t* __restrict__ counts,
                   const uint32_t* __restrict__ toff_tab, uint32_t n_mask, uint32_t n_tiles,
                   uint32_t gid0, uint8_t* __restrict__ dec_bytes,
                   unsigned long long* __restrict__ acc_slots)
{
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const uint32_t n_warps = (gridDim.x * blockDim.x) >> 5;
    const uint32_t j0 = (4u * lane) & n_mask;                 // monomer index of slot 0
    const bool has_l0 = j0 != 0u;                             // slot 0 has a left neighbour
    const bool has_r3 = ((j0 + 4u) & n_mask) != 0u;           // slot 3 has a right neighbour
    const uint4 toff = *reinterpret_cast<const uint4*>(toff_tab + j0);
    const float mf0 = has_l0 ? 2.0f : 1.0f, mf3 = has_r3 ? 2.0f : 1.0f;
    uint32_t n_acc = 0;

    for (uint32_t tile = warp; tile < n_tiles; tile += n_warps) {
        const uint32_t i0 = tile * kTile + 4u * lane;
        float4 X = *reinterpret_cast<const float4*>(x + i0);
        float4 Y = *reinterpret_cast<const float4*>(y + i0);
        float4 Z = *reinterpret_cast<const float4*>(z + i0);
        const uint32_t gid = gid0 + i0;

        // ---- set 0: even monomers (slots 0, 2) see the old odd monomers --------------------
        float xl = __shfl_up_sync(0xFFFFFFFFu, X.w, 1), yl = __shfl_up_sync(0xFFFFFFFFu, Y.w, 1),
              zl = __shfl_up_sync(0xFFFFFFFFu, Z.w, 1);
        xl = has_l0 ? xl : X.x; yl = has_l0 ? yl : Y.x; zl = has_l0 ? zl : Z.x;
        const bool a0 = mc_move<kMove, kIncr>(P, omega, counts, X.x, Y.x, Z.x, xl, yl, zl, X.y, Y.y, Z.y, mf0, toff.x, gid);
        const bool a2 = mc_move<kMove, kIncr>(P, omega, counts, X.z, Y.z, Z.z, X.y, Y.y, Z.y, X.w, Y.w, Z.w, 2.0f, toff.z, gid + 2u);

        // ---- set 1: odd monomers (slots 1, 3) see the moved even monomers ------------------
        float xr = __shfl_down_sync(0xFFFFFFFFu, X.x, 1), yr = __shfl_down_sync(0xFFFFFFFFu, Y.x, 1),
              zr = __shfl_down_sync(0xFFFFFFFFu, Z.x, 1);
        xr = has_r3 ? xr : X.w; yr = has_r3 ? yr : Y.w; zr = has_r3 ? zr : Z.w;
        const bool a1 = mc_move<kMove, kIncr>(P, omega, counts, X.y, Y.y, Z.y, X.x, Y.x, Z.x, X.z, Y.z, Z.z, 2.0f, toff.y, gid + 1u);
        const bool a3 = mc_move<kMove, kIncr>(P, omega, counts, X.w, Y.w, Z.w, X.z, Y.z, Z.z, xr, yr, zr, mf3, toff.w, gid + 3u);

        *reinterpret_cast<float4*>(x + i0) = X;
        *reinterpret_cast<float4*>(y + i0) = Y;
        *reinterpret_cast<float4*>(z + i0) = Z;

        const uint32_t nib = (a0 ? 1u : 0u) | (a1 ? 2u : 0u) | (a2 ? 4u : 0u) | (a3 ? 8u : 0u);
        n_acc += __popc(nib);
        if (kRecord) {
            const uint32_t hi = __shfl_down_sync(0xFFFFFFFFu, nib, 1);
            if ((lane & 1u) == 0u) dec_bytes[i0 >> 3] = (uint8_t)(nib | (hi << 4));
        }
    }
    n_acc = __reduce_add_sync(0xFFFFFFFFu, n_acc);
    if (lane == 0 && n_acc) atomicAdd(acc_slots + (warp % kAccSlots), (unsigned long long)n_acc);
}

// ------------------------------------------------------------------------------------------------
// a1 or a2 for any chain length: one thread per monomer of parity `parity` (set 0 / set 1).  The
// other parity is not written during this launch, so neighbours can be read from global memory.
//   half  = monomers of this parity per chain; n_items = n_chains * half
// ------------------------------------------------------------------------------------------------
template <int kMove, bool kIncr, bool kRecord>
__global__ void __launch_bounds__(256)
generic_move_kernel(const MoveP P, float* __restrict__ x, float* __restrict__ y, float* __restrict__ z,
                    const float* __restrict__ omega, uint32_t* __restrict__ counts,
                    const uint32_t* __restrict__ toff_tab, uint32_t N, uint32_t half, uint32_t parity,
                    uint64_t n_items, uint32_t gid0, uint32_t* __restrict__ dec_words,
                    unsigned long long* __restrict__ acc_slots)
{
    const uint64_t t = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    bool acc = false;
    if (t < n_items) {
        const uint64_t chain = t / half;
        const uint32_t j = 2u * (uint32_t)(t - chain * half) + parity;
        const uint64_t i = chain * N + j;
        const bool has_l = j > 0u, has_r = j + 1u < N;
        float px = x[i], py = y[i], pz = z[i];
        const float xl = has_l ? x[i - 1] : px, yl = has_l ? y[i - 1] : py, zl = has_l ? z[i - 1] : pz;
        const float xr = has_r ? x[i + 1] : px, yr = has_r ? y[i + 1] : py, zr = has_r ? z[i + 1] : pz;
        const float mf = (float)((has_l ? 1 : 0) + (has_r ? 1 : 0));
        const uint32_t gid = gid0 + (uint32_t)i;
        acc = mc_move<kMove, kIncr>(P, omega, counts, px, py, pz, xl, yl, zl, xr, yr, zr, mf, toff_tab[j], gid);
        if (acc) { x[i] = px; y[i] = py; z[i] = pz; }
        if (kRecord && acc) atomicOr(dec_words + (gid >> 5), 1u << (gid & 31u));
    }
    const uint32_t n_acc = __popc(__ballot_sync(0xFFFFFFFFu, acc));
    if ((threadIdx.x & 31u) == 0 && n_acc)
        atomicAdd(acc_slots + ((t >> 5) % kAccSlots), (unsigned long long)n_acc);
}

// ------------------------------------------------------------------------------------------------
// a3  occupation numbers from scratch (Eq. 4): counts[type][cell] += 1 per bead.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
histogram_kernel(const GridP g, const float* __restrict__ x, const float* __restrict__ y,
                 const float* __restrict__ z, const uint32_t* __restrict__ toff_tab, uint32_t N,
                 uint32_t n_beads, uint32_t* __restrict__ counts)
{
    const uint32_t stride = gridDim.x * blockDim.x;
    for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < n_beads; i += stride) {
        const uint32_t j = i % N;
        atomicAdd(counts + toff_tab[j] + cell_of(g, x[i], y[i], z[i]), 1u);
    }
}

// ------------------------------------------------------------------------------------------------
// a4  omega_i(c) from n_i(c), Eq. 12: phi_i = n_i / (rho_0 DeltaL^3),
//     K^0: omega_i = kappa_0 (sum phi - 1) - sum_{k != i} chi_0ik/2 (phi_i - phi_k)
//     K^1: omega_i = kappa_0 (sum phi - 1) + sum_{k != i} chi_0ik phi_k
// ------------------------------------------------------------------------------------------------
template <int kTypes>
__global__ void __launch_bounds__(256)
field_kernel(const FieldP F, const uint32_t* __restrict__ counts, float* __restrict__ omega)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= F.cells) return;
    const int nt = kTypes > 0 ? kTypes : F.n_types;
    float phi[kMaxTypes];
#pragma unroll
    for (int i = 0; i < kMaxTypes; ++i)
        if (i < nt) phi[i] = (float)counts[(size_t)i * F.cells + c] * F.inv_nbar;
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
        omega[(size_t)i * F.cells + c] = w;
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

}  // namespace soma
