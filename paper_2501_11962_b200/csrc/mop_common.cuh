// mop_common.cuh -- shared declarations of the CUDA hot path (sm_100a).
//
// Data layout in HBM (per force bead n < nf, nf = max(N-1,1); S = padded slots per bead):
//   xq   [nf][S] float4  wrapped coordinates + charge, sorted by (column, z-bin), columns padded to 8
//   typ  [nf][S] int     type * n_types (row offset into the LJ table), sorted order
//   et   [nf][S] float4  eta^n (xyz) + type row offset (w, int bits), sorted order, pass-2 input
//   F4   [nf][S] float4  physical force F^n, sorted order (w unused)
//   H4   [nf][S] float4  H^n eta^n, sorted order (w unused)
//   perm [nf][S] int     sorted slot -> original atom (-1: padding);  slot_of [nf][Q] the inverse
// A cluster ("octet") = 8 consecutive slots: a compact group of ~8 atoms (thin x,y columns of side ~ (8/rho)^(1/3),
// sorted along z).  The same octets serve as i-clusters (one work unit each) and as j-clusters (four per warp step).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MOP_CL 8           // atoms per cluster (octet)
#define MOP_NG 4           // j-octets per warp step (lane = (j atom 0..7, group 0..3))
#define MOP_KE 138.935458f // Coulomb constant, kJ mol^-1 nm e^-2
#define MOP_MAX_TYPES 64
#define MOP_EXROWS 48      // max distinct j-octets holding exclusion partners of one i-octet (row 0: the octet itself)
#ifndef MOP_LBUF
#define MOP_LBUF 384       // per-warp staging capacity (candidate j-octets) in the list builder
#endif
#define MOP_NOSHIFT 21     // shift id (kx+1) | (ky+1) << 2 | (kz+1) << 4 of the zero shift

// -DMOP_CHECK: a checked build for tests/sanitizer_target.py (compute-sanitizer is closed on the GPU pool this was
// developed on): every index the list builder and the pair kernels derive from list data is tested against the size of
// the array it goes into; a violation prints the place and traps (the launch fails with cudaErrorAssert / launch failure).
#ifdef MOP_CHECK
#include <cstdio>
#define MOP_ASSERT(cond)                                                                   \
    do {                                                                                   \
        if (!(cond)) {                                                                     \
            printf("MOP_ASSERT failed: %s  (%s:%d)\n", #cond, __FILE__, __LINE__);         \
            __trap();                                                                      \
        }                                                                                  \
    } while (0)
#else
#define MOP_ASSERT(cond) ((void)0)
#endif

struct MopGrid {
    float box[3], inv_box[3]; // inv_box = 1.0f / box (FP32)
    float sc[3];              // (float)dims * inv_box (FP32 product): cell = min((int)(xw*sc), dims-1)
    int dims[3];              // nx, ny (columns), nz (thin z bins)
    int ncol, ncell;          // nx*ny, ncol*nz
    int S;                    // slots per bead (multiple of 32)
    int Q, nf;
    float colw[2];            // column widths box/dims
    int n0;                   // first bead of this launch of the S0 kernels (bead = n0 + blockIdx.y)
};

struct MopUnit {            // one work unit of the pair kernels: (bead, i-octet)
    int bead;
    int ci;                 // i-octet index within the bead (slot = ci*8 + k)
    unsigned start, count;  // range in the entry array; count is a multiple of MOP_NG (padded with pattern-0 entries)
    unsigned excl_base;     // first exclusion-mask row of this i-octet
    unsigned pad0, pad1, pad2;
};

// entry: x = j-octet index within the bead | shift id << 24  ((kx+1) | (ky+1) << 2 | (kz+1) << 4, MOP_NOSHIFT = none)
//        y = pattern (bits 0-3: row pair p = i atoms (2p, 2p+1) has a pair within r_list of this octet; 0: padding)
//            | (exclusion row + 1) << 8 (bits 8-15; 0: no exclusions in this octet pair)
//            | step information, the same in the four entries of a step: bits 16-19 union of their patterns,
//              bit 20 some entry is shifted, bit 21 some entry has an exclusion row or is padding
// The entries of a unit are ordered by pattern, so that the four octets of a warp step mostly share theirs.
typedef uint2 MopEntry;

struct MopCounters {
    unsigned n_units, n_entries, n_masks, overflow; // overflow: bit0 entries, bit1 units, bit2 masks, bit3 staging, bit4 excl rows
    unsigned n_units_bead0, nonfinite, work1, n_units_mid;  // nonfinite: an input coordinate was NaN/Inf or beyond 1e6 box lengths
                                                            // n_units_mid: units of the first bead group (split pass 2 of the host entry point)
    unsigned long long n_pairs;   // debug pair walker
    unsigned long long n_inrange; // in-range decisions counted by the production force kernel (counting variant)
    unsigned long long pair_hash; // ... and the sum (mod 2^64) of a 64-bit hash of (bead, i, j) over those decisions
};

// ---- G8: the FP32 expressions shared by every kernel that classifies (fixed order, never contracted) ----
__device__ __forceinline__ float mop_wrap1(float x, float L, float invL) {
    float t = __fmul_rn(x, invL);
    float f = floorf(t);
    float p = __fmul_rn(L, f);
    float xw = __fsub_rn(x, p);
    if (xw < 0.0f) xw = __fadd_rn(xw, L);
    if (xw >= L) xw = __fsub_rn(xw, L);
    return xw;
}

// clamped on both sides: a coordinate the wrap could not bring into [0, L) (|x| beyond ~1e7 L, NaN, Inf) still
// lands in a valid cell; k_bin raises the context's non-finite flag for it
__device__ __forceinline__ int mop_cell1(float xw, float sc, int n) {
    int v = (int)__fmul_rn(xw, sc);
    v = v > n - 1 ? n - 1 : v;
    return v < 0 ? 0 : v;
}

// padding slots sit far outside the box on a lattice of three box lengths: slot s -> (a, b, c) = its bit fields,
// x = -(3a + 2) Lx, y = -(3b + 2) Ly, z = -(3c + 2) Lz.  Two distinct dummies differ by >= 3 L in some component and a
// real atom (in [0, L)) is >= 2 L away from every dummy, so under any periodic shift (|k| <= 1) no pair that involves
// a dummy is within r_cut <= L/2: the pair predicate itself rejects them, with finite arithmetic; charge 0, type 0
__device__ __forceinline__ float4 mop_dummy_xq(int s, const float box[3]) {
    return make_float4(-(3.0f * (float)(s & 1023) + 2.0f) * box[0], -(3.0f * (float)((s >> 10) & 1023) + 2.0f) * box[1],
                       -(3.0f * (float)(s >> 20) + 2.0f) * box[2], 0.0f);
}

__device__ __forceinline__ void mop_red_add_f4(float4 *addr, float x, float y, float z) {
    asm volatile("red.relaxed.gpu.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(x), "f"(y), "f"(z),
                 "f"(0.0f)
                 : "memory");
}

__device__ __forceinline__ float mop_warp_sum(float v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
__device__ __forceinline__ double mop_warp_sum_d(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}
