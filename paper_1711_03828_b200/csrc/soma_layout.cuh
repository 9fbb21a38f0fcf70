// soma_layout.cuh -- device code that keeps the chains in a spatially coherent order in HBM.
//
// Nothing here is part of the method's arithmetic (PAPER.md has no counterpart): it only decides
// WHERE a chain is stored.  A chain keeps its identity -- orig[slot] is the chain's index in the
// caller's order, and that index (not the slot) enters the Philox counter and the decision bitmap --
// so results do not depend on the layout.  Why a layout at all: with chains ordered along a Hilbert
// curve through their centres of mass, the tiles a block works on live in a small region of the grid,
// so the omega gathers and count updates of the move kernel hit in L1/L2 and touch fewer L2 slices
// (~3 % faster at C3; chains diffuse ~R_e per 1e5 sweeps, so the order ages slowly).
//
//   chain_key_kernel      Hilbert index of the centre of mass of every chain
//   (sort by key: cub::DeviceRadixSort in soma_b200.cu -- a library sort, off the hot path)
//   permute_chains_kernel gather one coordinate array into the new order
//   permute_ids_kernel    carry orig[] along
//   import/export kernels caller order <-> device order for soma_set_positions / soma_positions
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace soma {

// Hilbert index of a point of the 2^bits cube (Skilling's transposition: axes -> transposed index
// -> interleave).  bits <= 10.
__device__ __forceinline__ uint32_t hilbert3(uint32_t hx, uint32_t hy, uint32_t hz, uint32_t bits)
{
    uint32_t X[3] = {hx, hy, hz};
    const uint32_t M = 1u << (bits - 1u);
    for (uint32_t Q = M; Q > 1u; Q >>= 1) {          // inverse undo of the excess work
        const uint32_t Pm = Q - 1u;
#pragma unroll
        for (int i = 0; i < 3; ++i) {
            if (X[i] & Q) {
                X[0] ^= Pm;
            } else {
                const uint32_t t = (X[0] ^ X[i]) & Pm;
                X[0] ^= t;
                X[i] ^= t;
            }
        }
    }
    X[1] ^= X[0];                                    // Gray encode
    X[2] ^= X[1];
    uint32_t t = 0;
    for (uint32_t Q = M; Q > 1u; Q >>= 1)
        if (X[2] & Q) t ^= Q - 1u;
    X[0] ^= t; X[1] ^= t; X[2] ^= t;
    uint32_t code = 0;
    for (int b = (int)bits - 1; b >= 0; --b)
#pragma unroll
        for (int a = 0; a < 3; ++a) code = (code << 1) | ((X[a] >> b) & 1u);
    return code;
}

// fractional box coordinate in [0, 1) of a (mean) position -- layout heuristic, not Eq. 4
__device__ __forceinline__ float box_fraction(float x, float inv_L)
{
    const float t = x * inv_L;
    const float f = t - floorf(t);
    return f < 1.0f ? f : 0.0f;
}

// keys[c] = Hilbert index of the centre of mass of the chain in slot c, vals[c] = c
__global__ void __launch_bounds__(128)
chain_key_kernel(const float* __restrict__ x, const float* __restrict__ y, const float* __restrict__ z,
                 uint32_t n_chains, uint32_t N, float inv_Lx, float inv_Ly, float inv_Lz, uint32_t bits,
                 float side_x, float side_y, float side_z, uint32_t* __restrict__ keys, uint32_t* __restrict__ vals)
{
    const uint32_t c = blockIdx.x * blockDim.x + threadIdx.x;
    if (c >= n_chains) return;
    const size_t b = (size_t)c * N;
    float sx = 0.f, sy = 0.f, sz = 0.f;
    for (uint32_t j = 0; j < N; ++j) { sx += x[b + j]; sy += y[b + j]; sz += z[b + j]; }
    // side_a = units of the 2^bits cube the box spans along axis a: the same length per unit along x and y
    // (the longest axis fills the cube), a multiple of it along z, the direction in which the cells of omega
    // and counts are contiguous in memory (see resort()).
    const float inv_N = 1.0f / (float)N;
    const uint32_t top = (1u << bits) - 1u;
    const uint32_t hx = min((uint32_t)(box_fraction(sx * inv_N, inv_Lx) * side_x), top);
    const uint32_t hy = min((uint32_t)(box_fraction(sy * inv_N, inv_Ly) * side_y), top);
    const uint32_t hz = min((uint32_t)(box_fraction(sz * inv_N, inv_Lz) * side_z), top);
    keys[c] = hilbert3(hx, hy, hz, bits);
    vals[c] = c;
}

// dst[slot * N + j] = src[order[slot] * N + j]
__global__ void __launch_bounds__(256)
permute_chains_kernel(float* __restrict__ dst, const float* __restrict__ src,
                      const uint32_t* __restrict__ order, uint32_t N, uint64_t n_beads)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_beads) return;
    const uint32_t slot = (uint32_t)(i / N), j = (uint32_t)(i - (uint64_t)slot * N);
    dst[i] = src[(uint64_t)order[slot] * N + j];
}

__global__ void __launch_bounds__(256)
permute_ids_kernel(uint32_t* __restrict__ dst, const uint32_t* __restrict__ src,
                   const uint32_t* __restrict__ order, uint32_t n)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = src[order[i]];
}

__global__ void __launch_bounds__(256)
iota_kernel(uint32_t* __restrict__ dst, uint32_t n)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) dst[i] = i;
}

// Caller order (SoA x | y | z over all beads, bead = gid0 + chain * N + monomer) <-> device order
// (this architecture's padded segment, slot * N + monomer).
template <bool kToUser>
__global__ void __launch_bounds__(256)
reorder_kernel(float* __restrict__ user, uint64_t user_stride, float* __restrict__ x, float* __restrict__ y,
               float* __restrict__ z, const uint32_t* __restrict__ orig, uint32_t N, uint64_t n_beads,
               uint64_t gid0)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n_beads) return;
    const uint32_t slot = (uint32_t)(i / N), j = (uint32_t)(i - (uint64_t)slot * N);
    const uint64_t g = gid0 + (uint64_t)orig[slot] * N + j;
    if (kToUser) {
        user[g] = x[i];
        user[user_stride + g] = y[i];
        user[2 * user_stride + g] = z[i];
    } else {
        x[i] = user[g];
        y[i] = user[user_stride + g];
        z[i] = user[2 * user_stride + g];
    }
}

}  // namespace soma
