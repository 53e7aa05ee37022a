// mop_nonbonded.cuh -- S2 (pass 1: force, energy on bead 1) and S5 (pass 2: fused force-scalar + Hessian-vector
// pair kernel), SURVEY.md 8a.  FP32 ALU-bound; no tensor cores (not a dense contraction).
//
// One warp per work unit (bead, i-cluster, shift).  The 8 i atoms live in registers (warp-uniform values);
// lane l owns atom l of the current j-cluster (one coalesced float4 load per array per entry, prefetched one
// entry ahead).  The warp walks the i atoms sequentially, skipping those the list's imask rules out, so
//   - the j-side result needs NO cross-lane reduction (each lane owns its j atom) and leaves the warp as one
//     16-byte vector reduction (red.global.add.v4.f32) per entry,
//   - the i-side accumulators stay distributed over the lanes for the whole unit and are reduced by
//     shuffles once at the end.
// Pair math (O2/O3 of DESIGN.md), u = LJ 12-6 + reaction field, d = r_i - r_j:
//   g = u'/r        = (6 C6 r^-6 - 12 C12 r^-12) r^-2 + ke qi qj (2 k_rf - r^-3)
//   h = (u''-u'/r)/r^2 = (14*12 C12 r^-12 - 8*6 C6 r^-6) r^-4 + 3 ke qi qj r^-5
//   F_i -= g d ; (H s)_i += h (d.delta) d + g delta, delta = s_i - s_j   (and the opposite on j)
#pragma once
#include "mop_common.cuh"

struct NbArgs {
    int S, nt;
    float rc2;          // r_cut*r_cut (FP32 product, G8)
    float k2rf;         // 2 k_rf
    float krf, crf;     // energy only
    const float4 *xq;   // [nf][S]
    const int *typ;     // [nf][S] type row offsets (force pass)
    const float4 *et;   // [nf][S] eta + type row offset (HVP pass)
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

template <bool HVP, bool ENERGY, bool SHIFT>
__device__ __forceinline__ void nb_unit(const NbArgs &a, const MopUnit &un, const float2 *__restrict__ tab,
                                        const float2 *__restrict__ tabe, const float *__restrict__ tabs,
                                        const int lane) {
    const size_t boff = (size_t)un.bead * a.S;
    const float4 *__restrict__ xq = a.xq + boff;
    const float4 *__restrict__ et = a.et + boff;
    const int *__restrict__ typ = a.typ + boff;
    float sx = 0.f, sy = 0.f, sz = 0.f;
    if (SHIFT) {
        int s = un.shift;
        sx = (float)(s % 3 - 1) * a.box[0];
        sy = (float)((s / 3) % 3 - 1) * a.box[1];
        sz = (float)(s / 9 - 1) * a.box[2];
    }
    float xi[MOP_CI], yi[MOP_CI], zi[MOP_CI], qi[MOP_CI];
    float sxi[HVP ? MOP_CI : 1], syi[HVP ? MOP_CI : 1], szi[HVP ? MOP_CI : 1];
    int ri[MOP_CI];
    float ax[MOP_CI], ay[MOP_CI], az[MOP_CI];
#pragma unroll
    for (int k = 0; k < MOP_CI; k++) {
        float4 p = xq[un.ci * MOP_CI + k];
        xi[k] = p.x, yi[k] = p.y, zi[k] = p.z, qi[k] = MOP_KE * p.w;
        if (HVP) {
            float4 e = et[un.ci * MOP_CI + k];
            sxi[k] = e.x, syi[k] = e.y, szi[k] = e.z;
            ri[k] = __float_as_int(e.w) * a.nt;
        } else {
            ri[k] = typ[un.ci * MOP_CI + k] * a.nt;
        }
        ax[k] = ay[k] = az[k] = 0.f;
    }
    double e_lj = 0.0, e_c = 0.0;

    unsigned e = un.start;
    const unsigned eend = un.start + un.count;
    MopEntry ent = a.entries[e];
    float4 pj = xq[(size_t)ent.x * MOP_CJ + lane];
    float4 ej = make_float4(0.f, 0.f, 0.f, 0.f);
    int tj = 0;
    if (HVP) ej = et[(size_t)ent.x * MOP_CJ + lane];
    else tj = typ[(size_t)ent.x * MOP_CJ + lane];

    for (; e < eend; e++) {
        const MopEntry cur = ent;
        const float4 cp = pj;
        const float4 ce = ej;
        const int ctj = HVP ? __float_as_int(ej.w) : tj;
        if (e + 1 < eend) { // prefetch the next entry's j atoms
            ent = a.entries[e + 1];
            pj = xq[(size_t)ent.x * MOP_CJ + lane];
            if (HVP) ej = et[(size_t)ent.x * MOP_CJ + lane];
            else tj = typ[(size_t)ent.x * MOP_CJ + lane];
        }
        float jx = 0.f, jy = 0.f, jz = 0.f;
        float u_lj = 0.f, u_c = 0.f;
        const unsigned imask = cur.y & 0xffu;
        const unsigned row1 = cur.y >> 8;

        auto pair = [&](const int k, const bool allowed) {
            float dx = __fsub_rn(xi[k], cp.x), dy = __fsub_rn(yi[k], cp.y), dz = __fsub_rn(zi[k], cp.z);
            if (SHIFT) dx = __fsub_rn(dx, sx), dy = __fsub_rn(dy, sy), dz = __fsub_rn(dz, sz);
            const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            const bool inr = (r2 < a.rc2) && allowed;
            float rinv = rsqrtf(r2);
            if (ENERGY) { // one Newton step: removes the approximation's bias from the energy sum
                const float er = __fmaf_rn(-__fmul_rn(r2, rinv), rinv, 1.0f);
                rinv = __fmaf_rn(0.5f * rinv, er, rinv);
            }
            rinv = inr ? rinv : 0.f;
            const float qq = inr ? qi[k] * cp.w : 0.f;
            const float2 cc = tab[ri[k] + ctj];
            const float r2i = rinv * rinv;
            const float r6i = r2i * r2i * r2i;
            const float p6 = cc.x * r6i;
            const float p12 = cc.y * r6i * r6i;
            const float r3i = rinv * r2i;
            const float g = (p6 - p12) * r2i + qq * (a.k2rf - r3i);
            if (!HVP) {
                ax[k] = fmaf(-g, dx, ax[k]), ay[k] = fmaf(-g, dy, ay[k]), az[k] = fmaf(-g, dz, az[k]);
                jx = fmaf(g, dx, jx), jy = fmaf(g, dy, jy), jz = fmaf(g, dz, jz);
                if (ENERGY) {
                    const float sh = inr ? tabs[ri[k] + ctj] : 0.f;
                    const float2 ce6 = tabe[ri[k] + ctj];
                    u_lj += __fmaf_rn(ce6.y * r6i, r6i, -__fmaf_rn(ce6.x, r6i, sh));
                    u_c += qq * (rinv + a.krf * r2 - a.crf);
                }
            } else {
                const float h = r2i * ((14.0f * p12 - 8.0f * p6) * r2i + 3.0f * qq * r3i);
                const float ddx = sxi[k] - ce.x, ddy = syi[k] - ce.y, ddz = szi[k] - ce.z;
                const float t = h * (dx * ddx + dy * ddy + dz * ddz);
                const float ox = fmaf(t, dx, g * ddx), oy = fmaf(t, dy, g * ddy), oz = fmaf(t, dz, g * ddz);
                ax[k] += ox, ay[k] += oy, az[k] += oz;
                jx -= ox, jy -= oy, jz -= oz;
            }
        };

        if (row1 == 0) {
#pragma unroll
            for (int k = 0; k < MOP_CI; k++)
                if (imask & (1u << k)) pair(k, true);
        } else {
            const unsigned *__restrict__ mrow = a.masks + (size_t)(un.excl_base + row1 - 1) * MOP_CI;
#pragma unroll
            for (int k = 0; k < MOP_CI; k++)
                if (imask & (1u << k)) pair(k, (mrow[k] >> lane) & 1u);
        }
        mop_red_add_f4(a.out + boff + (size_t)cur.x * MOP_CJ + lane, jx, jy, jz);
        if (ENERGY) e_lj += (double)u_lj, e_c += (double)u_c;
    }

    // i-side: reduce over the lanes, lane k writes atom k
    float ox = 0.f, oy = 0.f, oz = 0.f;
#pragma unroll
    for (int k = 0; k < MOP_CI; k++) {
        float vx = mop_warp_sum(ax[k]), vy = mop_warp_sum(ay[k]), vz = mop_warp_sum(az[k]);
        if (lane == k) ox = vx, oy = vy, oz = vz;
    }
    if (lane < MOP_CI) mop_red_add_f4(a.out + boff + (size_t)un.ci * MOP_CI + lane, ox, oy, oz);
    if (ENERGY) {
        e_lj = mop_warp_sum_d(e_lj), e_c = mop_warp_sum_d(e_c);
        if (lane == 0) {
            atomicAdd(&a.energies[0], e_lj);
            atomicAdd(&a.energies[1], e_c);
        }
    }
}

template <bool HVP, bool ENERGY>
__global__ void __launch_bounds__(128) k_nonbonded(const NbArgs a) {
    extern __shared__ float4 s_dyn[];
    float2 *tab = reinterpret_cast<float2 *>(s_dyn);
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
        if (un.shift == 13) nb_unit<HVP, ENERGY, false>(a, un, tab, tabe, tabs, lane);
        else nb_unit<HVP, ENERGY, true>(a, un, tab, tabe, tabs, lane);
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
        const int s = un.shift;
        const float sx = (float)(s % 3 - 1) * a.box[0], sy = (float)((s / 3) % 3 - 1) * a.box[1],
                    sz = (float)(s / 9 - 1) * a.box[2];
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
                float dx = __fsub_rn(pi.x, cp.x), dy = __fsub_rn(pi.y, cp.y), dz = __fsub_rn(pi.z, cp.z);
                if (s != 13) dx = __fsub_rn(dx, sx), dy = __fsub_rn(dy, sy), dz = __fsub_rn(dz, sz);
                const float r2 = __fmaf_rn(dz, dz, __fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
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
