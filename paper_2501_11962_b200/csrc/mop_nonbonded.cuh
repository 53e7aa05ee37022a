// mop_nonbonded.cuh -- S2 (pass 1: force, energy on bead 1) and S5 (pass 2: fused force-scalar + Hessian-vector
// pair kernel), SURVEY.md 8a.  FP32 ALU-bound; no tensor cores (not a dense contraction).
//
// One warp per work unit (bead, i-cluster, shift).  The 8 i atoms (pre-shifted by the unit's periodic image,
// charge pre-multiplied by k_e) are staged once per unit; lane l owns atom l of the current j-cluster (one
// coalesced float4 load per array per entry, issued one entry ahead; the entry words two ahead).  The warp walks
// the i atoms the list's imask allows, so
//   - the j-side result needs NO cross-lane reduction (each lane owns its j atom) and leaves the warp as one
//     16-byte vector reduction (red.global.add.v4.f32) per lane per entry,
//   - the i-side accumulators stay distributed over the lanes for the whole unit and are reduced by shuffles
//     once at the end.
// Pair math (O2/O3 of DESIGN.md), u = LJ 12-6 + reaction field, d = r_i - r_j, x = 1/r^2, A = 6 C6 x^3,
// B = 12 C12 x^6, C = ke qi qj x^(3/2):
//   g = u'/r           = x (A - B) + ke qi qj 2 k_rf - C
//   h = (u''-u'/r)/r^2 = x (x (14 B - 8 A) + 3 C)
//   F_i -= g d ; (H s)_i += h (d.delta) d + g delta, delta = s_i - s_j   (and the opposite on j)
// Out-of-range / excluded / padding slots are evaluated and discarded by ONE select on g (and h).
#pragma once
#include "mop_common.cuh"

enum { NB_FORCE = 0, NB_ENERGY = 1, NB_HVP = 2 };
// tuning variants (bit flags of the VAR template argument)
enum { NBV_ISMEM = 1,   // i atoms are read from shared memory per row (fewer registers) instead of registers
       NBV_ROWS2 = 2,   // rows are processed two at a time (more ILP, a few wasted rows)
       NBV_ZSKIP = 4 }; // a row with no lane in range is dropped after the distance test

struct NbArgs {
    int S, nt;
    float rc2;          // r_cut*r_cut (FP32 product, G8)
    float k2rf;         // 2 k_rf
    float krf, crf;     // energy only
    const float4 *xq;   // [nf][S]
    const int *typ;     // [nf][S] types (force pass)
    const float4 *et;   // [nf][S] eta + type bits (HVP pass)
    float4 *out;        // [nf][S] F4 or H4, accumulated with vector reductions
    const MopUnit *units;
    const MopEntry *entries;
    const unsigned *masks;
    const MopCounters *ctr;
    unsigned *work;     // dynamic work counter (zeroed before the launch)
    int range;          // 0: units [0, n_units_bead0)   1: [n_units_bead0, n_units)   2: all
    const float2 *tab;  // [nt*nt] (6 C6, 12 C12)
    const float2 *tabe; // [nt*nt] (C6, C12) as given (energy: no rounding bias from the prefactors)
    const float *tabs;  // [nt*nt] LJ energy shift C12 rc^-12 - C6 rc^-6 (0 when lj_shift = 0)
    double *energies;   // [0] U_lj, [1] U_coul
    float box[3];
};

__device__ __forceinline__ float mop_rsqrt(float x) {
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// G8: the pair predicate.  xs_i = xw_i - k L is formed once per unit (k L exact, one rounding); then
// d = xs_i - xw_j (one rounding per component), r2 = fma(dz,dz, fma(dy,dy, dx*dx)), in range iff r2 < rc*rc.
__device__ __forceinline__ float mop_r2(float dx, float dy, float dz) {
    return __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
}

__device__ __forceinline__ void mop_unit_shift(int s, const float box[3], float &sx, float &sy, float &sz) {
    sx = (float)(s % 3 - 1) * box[0];
    sy = (float)((s / 3) % 3 - 1) * box[1];
    sz = (float)(s / 9 - 1) * box[2];
}

__device__ __forceinline__ float2 mop_lds_f2(unsigned addr) { // shared-window byte address
    float2 v;
    asm("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(v.x), "=f"(v.y) : "r"(addr));
    return v;
}

template <int MODE, int VAR>
__device__ __forceinline__ void nb_unit(const NbArgs &a, const MopUnit &un, float4 *__restrict__ si,
                                        const unsigned tab, const float2 *__restrict__ tabe,
                                        const float *__restrict__ tabs, const int lane) {
    constexpr bool HVP = MODE == NB_HVP, ENERGY = MODE == NB_ENERGY;
    constexpr bool ISMEM = (VAR & NBV_ISMEM) != 0, ROWS2 = (VAR & NBV_ROWS2) != 0, ZSKIP = (VAR & NBV_ZSKIP) != 0;
    const size_t boff = (size_t)un.bead * a.S;
    const float4 *__restrict__ xq = a.xq + boff;
    const float4 *__restrict__ et = a.et + boff;
    const int *__restrict__ typ = a.typ + boff;
    float4 *__restrict__ out = a.out + boff;

    // ---- stage the i atoms: si[k] = (xs, ys, zs, ke q), si[8+k] = (s_x, s_y, s_z, byte offset of the LJ-table row)
    __syncwarp();
    if (lane < MOP_CI) {
        float sx, sy, sz;
        mop_unit_shift(un.shift, a.box, sx, sy, sz);
        float4 p = xq[un.ci * MOP_CI + lane];
        p.x = __fsub_rn(p.x, sx), p.y = __fsub_rn(p.y, sy), p.z = __fsub_rn(p.z, sz);
        p.w *= MOP_KE;
        float4 e = make_float4(0.f, 0.f, 0.f, 0.f);
        int ti;
        if (HVP) {
            e = et[un.ci * MOP_CI + lane];
            ti = __float_as_int(e.w);
        } else {
            ti = typ[un.ci * MOP_CI + lane];
        }
        e.w = __int_as_float((int)tab + ti * a.nt * 8);   // shared address of the i atom's LJ-table row
        si[lane] = p;
        si[MOP_CI + lane] = e;
    }
    __syncwarp();
    float4 ri[ISMEM ? 1 : MOP_CI], rs[ISMEM ? 1 : MOP_CI];
    if (!ISMEM) {
#pragma unroll
        for (int k = 0; k < MOP_CI; k++) ri[k] = si[k], rs[k] = si[MOP_CI + k];
    }
    float ax[MOP_CI], ay[MOP_CI], az[MOP_CI];
#pragma unroll
    for (int k = 0; k < MOP_CI; k++) ax[k] = ay[k] = az[k] = 0.f;
    double e_lj = 0.0, e_c = 0.0;

    const unsigned e0 = un.start, eend = un.start + un.count;
    MopEntry ent1 = a.entries[e0];                                         // entry e (then e+1)
    MopEntry ent2 = (e0 + 1 < eend) ? a.entries[e0 + 1] : make_uint2(0u, 0u); // entry e+1 (then e+2)
    float4 pj = xq[(size_t)ent1.x * MOP_CJ + lane];
    float4 ej = make_float4(0.f, 0.f, 0.f, 0.f);
    int tj = 0;
    if (HVP) ej = et[(size_t)ent1.x * MOP_CJ + lane];
    else tj = typ[(size_t)ent1.x * MOP_CJ + lane];

    for (unsigned e = e0; e < eend; e++) {
        const MopEntry cur = ent1;
        const float4 cp = pj;
        const float4 ce = ej;
        const int tj8 = (HVP ? __float_as_int(ej.w) : tj) * 8;
        ent1 = ent2;
        if (e + 2 < eend) ent2 = a.entries[e + 2];
        if (e + 1 < eend) { // the next entry's j atoms
            pj = xq[(size_t)ent1.x * MOP_CJ + lane];
            if (HVP) ej = et[(size_t)ent1.x * MOP_CJ + lane];
            else tj = typ[(size_t)ent1.x * MOP_CJ + lane];
        }
        const unsigned imask = cur.y & 0xffu;
        const unsigned row1 = cur.y >> 8;
        // lm: bit k set iff i atom k may interact with this lane's j atom (imask and exclusions)
        unsigned lm = imask;
        if (row1 != 0) {
            const uint4 *__restrict__ mrow =
                reinterpret_cast<const uint4 *>(a.masks + (size_t)(un.excl_base + row1 - 1) * MOP_CI);
            const uint4 m0 = mrow[0], m1 = mrow[1];
            const unsigned mm[8] = {m0.x, m0.y, m0.z, m0.w, m1.x, m1.y, m1.z, m1.w};
            unsigned al = 0;
#pragma unroll
            for (int k = 0; k < MOP_CI; k++) al |= ((mm[k] >> lane) & 1u) << k;
            lm &= al;
        }
        float jx = 0.f, jy = 0.f, jz = 0.f;
        float u_lj = 0.f, u_c = 0.f;

        auto row = [&](const int k) {
            const float4 pi = ISMEM ? si[k] : ri[k];
            const float4 ei = ISMEM ? si[MOP_CI + k] : rs[k];
            const float dx = __fsub_rn(pi.x, cp.x), dy = __fsub_rn(pi.y, cp.y), dz = __fsub_rn(pi.z, cp.z);
            const float r2 = mop_r2(dx, dy, dz);
            const bool inr = (r2 < a.rc2) && ((lm & (1u << k)) != 0u);
            if (ZSKIP) {
                if (!__any_sync(0xffffffffu, inr)) return;
            }
            float rinv = mop_rsqrt(r2);
            if (ENERGY) { // one Newton step: removes the approximation's bias from the energy sum
                const float er = __fmaf_rn(-__fmul_rn(r2, rinv), rinv, 1.0f);
                rinv = __fmaf_rn(0.5f * rinv, er, rinv);
            }
            const unsigned tofs = (unsigned)__float_as_int(ei.w) + (unsigned)tj8;
            const float2 cc = mop_lds_f2(tofs);
            const float x = rinv * rinv;
            const float x3 = x * x * x;
            const float A = cc.x * x3;
            const float B = cc.y * x3 * x3;
            const float qq = pi.w * cp.w;
            const float C = qq * (x * rinv);
            float g = fmaf(x, A - B, fmaf(qq, a.k2rf, -C));
            g = inr ? g : 0.f;
            if (!HVP) {
                ax[k] = fmaf(-g, dx, ax[k]), ay[k] = fmaf(-g, dy, ay[k]), az[k] = fmaf(-g, dz, az[k]);
                jx = fmaf(g, dx, jx), jy = fmaf(g, dy, jy), jz = fmaf(g, dz, jz);
                if (ENERGY) {
                    const int ti = (int)((tofs - tab) >> 3);
                    const float2 ce6 = tabe[ti];
                    const float r6i = x * x * x;
                    const float ulj = __fmaf_rn(ce6.y * r6i, r6i, -__fmaf_rn(ce6.x, r6i, tabs[ti]));
                    const float uc = qq * (rinv + a.krf * r2 - a.crf);
                    u_lj += inr ? ulj : 0.f;
                    u_c += inr ? uc : 0.f;
                }
            } else {
                float h = x * fmaf(x, fmaf(14.0f, B, -8.0f * A), 3.0f * C);
                h = inr ? h : 0.f;
                const float ddx = ei.x - ce.x, ddy = ei.y - ce.y, ddz = ei.z - ce.z;
                const float t = h * fmaf(dz, ddz, fmaf(dy, ddy, dx * ddx));
                ax[k] = fmaf(t, dx, fmaf(g, ddx, ax[k]));
                ay[k] = fmaf(t, dy, fmaf(g, ddy, ay[k]));
                az[k] = fmaf(t, dz, fmaf(g, ddz, az[k]));
                jx = fmaf(-t, dx, fmaf(-g, ddx, jx));
                jy = fmaf(-t, dy, fmaf(-g, ddy, jy));
                jz = fmaf(-t, dz, fmaf(-g, ddz, jz));
            }
        };

        if (ROWS2) {
#pragma unroll
            for (int k = 0; k < MOP_CI; k += 2)
                if (imask & (3u << k)) row(k), row(k + 1);
        } else {
#pragma unroll
            for (int k = 0; k < MOP_CI; k++)
                if (imask & (1u << k)) row(k);
        }
        mop_red_add_f4(out + (size_t)cur.x * MOP_CJ + lane, jx, jy, jz);
        if (ENERGY) e_lj += (double)u_lj, e_c += (double)u_c;
    }

    // i-side: reduce over the lanes, lane k writes atom k
    float ox = 0.f, oy = 0.f, oz = 0.f;
#pragma unroll
    for (int k = 0; k < MOP_CI; k++) {
        float vx = mop_warp_sum(ax[k]), vy = mop_warp_sum(ay[k]), vz = mop_warp_sum(az[k]);
        if (lane == k) ox = vx, oy = vy, oz = vz;
    }
    if (lane < MOP_CI) mop_red_add_f4(out + (size_t)un.ci * MOP_CI + lane, ox, oy, oz);
    if (ENERGY) {
        e_lj = mop_warp_sum_d(e_lj), e_c = mop_warp_sum_d(e_c);
        if (lane == 0) {
            atomicAdd(&a.energies[0], e_lj);
            atomicAdd(&a.energies[1], e_c);
        }
    }
}

// dynamic shared memory: [4 warps][16] float4 i-atom staging, then the LJ tables
__host__ __device__ inline size_t nb_smem_bytes(int nt) { return 4 * 16 * sizeof(float4) + (size_t)nt * nt * 20; }

template <int MODE, int VAR>
__global__ void __launch_bounds__(128) k_nonbonded(const NbArgs a) {
    extern __shared__ float4 s_dyn[];
    float4 *si = s_dyn + (threadIdx.x >> 5) * 16;
    float2 *tab = reinterpret_cast<float2 *>(s_dyn + 64);
    float2 *tabe = tab + a.nt * a.nt;
    float *tabs = reinterpret_cast<float *>(tabe + a.nt * a.nt);
    for (int t = threadIdx.x; t < a.nt * a.nt; t += blockDim.x) {
        tab[t] = a.tab[t];
        tabe[t] = a.tabe[t];
        tabs[t] = a.tabs[t];
    }
    __syncthreads();
    const int lane = threadIdx.x & 31;
    unsigned ubeg = 0, uend = a.ctr->n_units;
    if (a.range == 0) uend = a.ctr->n_units_bead0;
    else if (a.range == 1) ubeg = a.ctr->n_units_bead0;
    for (;;) {
        unsigned u = 0;
        if (lane == 0) u = atomicAdd(a.work, 1u);
        u = __shfl_sync(0xffffffffu, u, 0) + ubeg;
        if (u >= uend) break;
        const uint4 *up = reinterpret_cast<const uint4 *>(a.units + u);
        const uint4 u0 = up[0], u1 = up[1];
        MopUnit un;
        un.bead = (int)u0.x, un.ci = (int)u0.y, un.shift = (int)u0.z, un.start = u0.w;
        un.count = u1.x, un.excl_base = u1.y;
        if (un.count == 0) continue;
        nb_unit<MODE, VAR>(a, un, si, (unsigned)__cvta_generic_to_shared(tab), tabe, tabs, lane);
    }
}

// ---- debug: the set of in-range, non-excluded pairs of one bead, with the force kernel's predicate ----
struct PairDbgArgs {
    int S, bead;
    float rc2;
    const float4 *xq;
    const int *perm;
    const MopUnit *units;
    const MopEntry *entries;
    const unsigned *masks;
    MopCounters *ctr;
    int *pairs;
    long long cap;
    float box[3];
};

__global__ void __launch_bounds__(128) k_debug_pairs(const PairDbgArgs a) {
    const int lane = threadIdx.x & 31;
    const unsigned nwarps = gridDim.x * (blockDim.x >> 5);
    const unsigned nu = a.ctr->n_units;
    for (unsigned u = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); u < nu; u += nwarps) {
        const MopUnit un = a.units[u];
        if (un.bead != a.bead || un.count == 0) continue;
        const float4 *xq = a.xq + (size_t)un.bead * a.S;
        const int *perm = a.perm + (size_t)un.bead * a.S;
        float sx, sy, sz;
        mop_unit_shift(un.shift, a.box, sx, sy, sz);
        for (unsigned e = un.start; e < un.start + un.count; e++) {
            const MopEntry cur = a.entries[e];
            const float4 cp = xq[(size_t)cur.x * MOP_CJ + lane];
            const int pj = perm[(size_t)cur.x * MOP_CJ + lane];
            const unsigned row1 = cur.y >> 8;
            for (int k = 0; k < MOP_CI; k++) {
                if (!((cur.y >> k) & 1u)) continue;
                const float4 pi = xq[un.ci * MOP_CI + k];
                bool allowed = true;
                if (row1) allowed = (a.masks[(size_t)(un.excl_base + row1 - 1) * MOP_CI + k] >> lane) & 1u;
                const float dx = __fsub_rn(__fsub_rn(pi.x, sx), cp.x), dy = __fsub_rn(__fsub_rn(pi.y, sy), cp.y),
                            dz = __fsub_rn(__fsub_rn(pi.z, sz), cp.z);
                const float r2 = mop_r2(dx, dy, dz);
                if ((r2 < a.rc2) && allowed) {
                    unsigned long long pos = atomicAdd(&a.ctr->n_pairs, 1ull);
                    if ((long long)pos < a.cap) {
                        a.pairs[2 * pos] = perm[un.ci * MOP_CI + k];
                        a.pairs[2 * pos + 1] = pj;
                    }
                }
            }
        }
    }
}
