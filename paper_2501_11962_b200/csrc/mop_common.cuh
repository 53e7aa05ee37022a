// mop_common.cuh -- shared declarations of the CUDA hot path (sm_100a).
//
// Data layout in HBM (per force bead n < nf, nf = max(N-1,1); S = padded slots per bead):
//   xq   [nf][S] float4  wrapped coordinates + charge, sorted by (column, z-bin), columns padded to 32
//   typ  [nf][S] int     type * n_types (row offset into the LJ table), sorted order
//   et   [nf][S] float4  eta^n (xyz) + type row offset (w, int bits), sorted order, pass-2 input
//   F4   [nf][S] float4  physical force F^n, sorted order (w unused)
//   H4   [nf][S] float4  H^n eta^n, sorted order (w unused)
//   perm [nf][S] int     sorted slot -> original atom (-1: padding);  slot_of [nf][Q] the inverse
// j-cluster = 32 consecutive slots (one warp lane each); i-cluster = 8 consecutive slots.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define MOP_CJ 32          // atoms per j-cluster (= warp lanes)
#define MOP_CI 8           // atoms per i-cluster (processed sequentially by one warp)
#define MOP_KE 138.935458f // Coulomb constant, kJ mol^-1 nm e^-2
#define MOP_MAX_TYPES 64
#define MOP_EXROWS 32      // max distinct j-clusters holding exclusion partners of one i-cluster
#define MOP_LBUF 448       // per-warp staging capacity (cluster-pair entries) in the list builder

struct MopGrid {
    float box[3], inv_box[3]; // inv_box = 1.0f / box (FP32)
    float sc[3];              // (float)dims * inv_box (FP32 product): cell = min((int)(xw*sc), dims-1)
    int dims[3];              // nx, ny (columns), nz (thin z bins)
    int ncol, ncell;          // nx*ny, ncol*nz
    int S;                    // slots per bead (multiple of 32)
    int Q, nf;
    float colw[2];            // column widths box/dims
};

struct MopUnit {            // one work unit of the pair kernels: (bead, i-cluster, periodic shift)
    int bead;
    int ci;                 // i-cluster index within the bead (slot = ci*8 + k)
    int shift;              // (kx+1) + 3*(ky+1) + 9*(kz+1); 13 = no shift
    unsigned start, count;  // range in the entry array
    unsigned excl_base;     // first exclusion-mask row of this i-cluster
    unsigned pad0, pad1;
};

// entry: x = j-cluster index within the bead; y = imask (bits 0-7: which i atoms can be in range)
//        | (exclusion row + 1) << 8 (0: no exclusions in this cluster pair)
typedef uint2 MopEntry;

struct MopCounters {
    unsigned n_units, n_entries, n_masks, overflow; // overflow: bit0 entries, bit1 units, bit2 masks, bit3 staging, bit4 excl rows
    unsigned n_units_bead0, work0, work1, pad;
    unsigned long long n_pairs; // debug pair walker
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

__device__ __forceinline__ int mop_cell1(float xw, float sc, int n) {
    int v = (int)__fmul_rn(xw, sc);
    return v > n - 1 ? n - 1 : v;
}

// padding slots sit far outside the box, every slot at its own place (no two dummies coincide)
__device__ __forceinline__ float4 mop_dummy_xq(int s) {
    return make_float4(-1000.0f - 4.0f * (float)(s & 1023), -1000.0f - 4.0f * (float)((s >> 10) & 1023),
                       -1000.0f - 4.0f * (float)(s >> 20), 0.0f);
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
