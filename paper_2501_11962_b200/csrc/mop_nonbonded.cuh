// mop_nonbonded.cuh -- declarations shared by the pair kernels (mop_nonbonded_packed.cuh: S2 pass 1 force / energy,
// S5 pass 2 fused force-scalar + Hessian-vector kernel) and the debug pair walker.
//
// Pair math (O2/O3 of DESIGN.md), u = LJ 12-6 + reaction field, d = r_i - r_j, x = 1/r^2, A = 6 C6 x^3,
// B = 12 C12 x^6, C = ke qi qj x^(3/2):
//   g = u'/r           = x (A - B) + ke qi qj 2 k_rf - C
//   h = (u''-u'/r)/r^2 = x (x (14 B - 8 A) + 3 C)
//   F_i -= g d ; (H s)_i += h (d.delta) d + g delta, delta = s_i - s_j   (and the opposite on j)
#pragma once
#include "mop_common.cuh"

enum { NB_FORCE = 0, NB_ENERGY = 1, NB_HVP = 2 };

struct NbArgs {
    int S, nt;
    float rc2;          // r_cut*r_cut (FP32 product, G8)
    float k2rf;         // 2 k_rf
    double krf_d, crf_d; // energy only: k_rf and c_rf = 1/r_c + k_rf r_c^2 in FP64 (applied once per step to FP32 partial sums)
    const float4 *xq;   // [nf][S]
    const int *typ;     // [nf][S] types (force pass)
    const float4 *et;   // [nf][S] eta + type bits (HVP pass)
    float4 *out;        // [nf][S] F4 or H4, accumulated with vector reductions
    const MopUnit *units;
    const MopEntry *entries;
    const unsigned long long *masks; // exclusion rows: byte jl = the i atoms (bits 0-7) j atom jl may interact with
    const MopCounters *ctr;
    unsigned cap_units;              // units beyond the allocation were never written (overflow): never read them
    unsigned cap_entries, cap_masks, n_slots;   // checked build only: sizes of entries, masks and of the [nf][S] arrays
    unsigned long long *n_inrange;   // counting variant only: in-range, non-excluded pair decisions of this launch
    unsigned long long *pair_hash;   // counting variant only: sum of mop_pair_hash over those decisions
    const int *perm;                 // counting variant only: [nf][S] sorted slot -> original atom
    int Q;                           // counting variant only
    unsigned *work;     // dynamic work counter (zeroed before the launch)
    int range;          // 0: units [0, n_units_bead0)   1: [n_units_bead0, n_units)   2: all   3: [0, n_units_mid)   4: [n_units_mid, n_units)
    const float2 *tab;  // [nt*nt] (6 C6, 12 C12)
    const float *tabs;  // [nt*nt] LJ energy shift C12 rc^-12 - C6 rc^-6 (0 when lj_shift = 0)
    double *energies;   // [0] U_lj, [1] U_coul
    float box[3];
};

// counting variant: order-independent fingerprint of the decided pair set.  key = (bead * Q + min(i,j)) * Q + max(i,j) in
// original atom indices, hashed by the SplitMix64 finaliser (Steele, Lea, Flood 2014; the published constants)
__device__ __forceinline__ unsigned long long mop_pair_hash(unsigned long long bead, unsigned long long Q, int i, int j) {
    const unsigned long long lo = (unsigned long long)min(i, j), hi = (unsigned long long)max(i, j);
    unsigned long long z = (bead * Q + lo) * Q + hi + 0x9E3779B97F4A7C15ULL;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}

__device__ __forceinline__ float mop_rsqrt(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// G8: the pair predicate.  d = (xw_i - xw_j) - k L (one rounding each; k L exact; d = xw_i - xw_j exactly for the zero
// shift), r2 = fma(dz,dz, fma(dy,dy, dx*dx)), in range iff r2 < rc*rc.  Swapping the roles of the two atoms (k -> -k)
// negates d bit for bit, so the result does not depend on which atom of a pair the list makes the i atom.
__device__ __forceinline__ float mop_r2(float dx, float dy, float dz) {
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

__device__ __forceinline__ void mop_unit_shift(int s, const float box[3], float &sx, float &sy, float &sz) {
    sx = (float)((s & 3) - 1) * box[0];
    sy = (float)(((s >> 2) & 3) - 1) * box[1];
    sz = (float)((s >> 4) - 1) * box[2];
}

// ---- debug: the set of in-range, non-excluded pairs of one bead, scalar restatement of the predicate over the list ----
struct PairDbgArgs {
    int S, bead;
    float rc2;
    const float4 *xq;
    const int *perm;
    const MopUnit *units;
    const MopEntry *entries;
    const unsigned long long *masks;
    MopCounters *ctr;
    unsigned cap_units;
    int *pairs;
    long long cap;
    float box[3];
};

__global__ void __launch_bounds__(128) k_debug_pairs(const PairDbgArgs a) {
    const int lane = threadIdx.x & 31, g = lane >> 3, jl = lane & 7;
    const unsigned nwarps = gridDim.x * (blockDim.x >> 5);
    const unsigned nu = min(a.ctr->n_units, a.cap_units);
    for (unsigned u = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); u < nu; u += nwarps) {
        const MopUnit un = a.units[u];
        if (un.bead != a.bead || un.count == 0) continue;
        const float4 *xq = a.xq + (size_t)un.bead * a.S;
        const int *perm = a.perm + (size_t)un.bead * a.S;
        for (unsigned e0 = un.start; e0 < un.start + un.count; e0 += MOP_NG) {
            const MopEntry cur = a.entries[e0 + g];
            const unsigned pat = cur.y & 15u;
            if (pat == 0) continue;
            const unsigned oc = cur.x & 0xffffffu, sid = cur.x >> 24, row1 = (cur.y >> 8) & 0xffu;
            float sx, sy, sz;
            mop_unit_shift((int)sid, a.box, sx, sy, sz);
            const float4 cp = xq[(size_t)oc * MOP_CL + jl];
            const int pj = perm[(size_t)oc * MOP_CL + jl];
            unsigned long long row = ~0ull;
            if (row1) row = a.masks[(size_t)un.excl_base + row1 - 1];
            for (int k = 0; k < MOP_CL; k++) {
                if (!((pat >> (k >> 1)) & 1u)) continue;
                const float4 pi = xq[un.ci * MOP_CL + k];
                const bool allowed = (row >> (8 * jl + k)) & 1ull;
                const float dx = __fsub_rn(__fsub_rn(pi.x, cp.x), sx), dy = __fsub_rn(__fsub_rn(pi.y, cp.y), sy),
                            dz = __fsub_rn(__fsub_rn(pi.z, cp.z), sz);
                const float r2 = mop_r2(dx, dy, dz);
                if ((r2 < a.rc2) && allowed) {
                    unsigned long long pos = atomicAdd(&a.ctr->n_pairs, 1ull);
                    if ((long long)pos < a.cap) {
                        a.pairs[2 * pos] = perm[un.ci * MOP_CL + k];
                        a.pairs[2 * pos + 1] = pj;
                    }
                }
            }
        }
    }
}
