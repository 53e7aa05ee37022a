// mop_pairlist.cuh -- S1: octet-pair list with exact row-pair patterns.
//
// One warp per i-octet (8 consecutive sorted slots).  It lists every (j-octet, periodic shift) with j-octet index
// >= its own (half list) in which some atom pair comes within r_list, together with
//   - a 4-bit pattern: row pair p (i atoms 2p, 2p+1) has such a pair (evaluated atom by atom with the FP32 form of
//     the pair kernels' distance, against r_list^2 inflated by 1e-4: a superset of what the kernels accept),
//   - the index of an exclusion-mask row when the octet pair holds excluded pairs (or is the diagonal block, where
//     only j slot > i slot is allowed).
// The entries of a unit are written ordered by pattern, so that the four octets a warp of the pair kernels takes per
// step mostly share theirs, and padded to a multiple of four with pattern-0 entries.
// The list is only a superset; the pair kernels apply the exact FP32 predicate (G8) per atom pair.
#pragma once
#include "mop_common.cuh"
#include "mop_nonbonded.cuh"
#include "mop_f2.cuh"

struct PlArgs {
    MopGrid g;
    int bead0;
    float rl, rl2; // list radius, and its square inflated by 1e-4 (conservative against FP32 rounding)
    const int *perm, *slot_of;
    const float4 *xq, *blo, *bhi;
    const int *col_start, *cell_rel, *col_count;
    const int *excl_start, *excl_list; // may be NULL
    MopUnit *units;
    MopEntry *entries;
    unsigned long long *masks;
    MopCounters *ctr;
    unsigned long long *slots_active; // [0] sum over entries of popc(pattern) * 16; [1] sum over steps of popc(union pattern) * 64
    unsigned cap_units, cap_entries, cap_masks;
};

__device__ __forceinline__ float mop_gap(float lo_a, float hi_a, float lo_b, float hi_b) {
    // distance between intervals [lo_a,hi_a] and [lo_b,hi_b]
    return fmaxf(0.0f, fmaxf(lo_b - hi_a, lo_a - hi_b));
}

// bucket order of the 15 non-zero patterns: the contiguous runs (the usual patterns, the row pairs of an octet being
// ordered along z) as a chain in which neighbours differ by one row pair -- 1, 3, 7, 15, 14, 12, 8 -- so that a step of four
// entries that straddles two buckets evaluates at most one row pair too many; then the rest
__constant__ unsigned char c_pat_order[16] = {1, 3, 7, 15, 14, 12, 8, 6, 2, 4, 5, 9, 10, 11, 13, 0};

#define MOP_PL_WARPS 4     // warps (i-octets) per CTA of the list builder
#ifndef MOP_PL_MINB
#define MOP_PL_MINB 5      // resident CTAs per SM asked for (register cap 65536 / (128 * MINB))
#endif
__global__ void __launch_bounds__(32 * MOP_PL_WARPS, MOP_PL_MINB) k_pairlist(PlArgs a) {
    __shared__ int s_exJ[MOP_PL_WARPS][MOP_EXROWS];
    __shared__ unsigned s_exM[MOP_PL_WARPS][MOP_EXROWS][2];
    __shared__ int s_exN[MOP_PL_WARPS];
    __shared__ unsigned s_bcj[MOP_PL_WARPS][MOP_LBUF];
    __shared__ unsigned s_binfo[MOP_PL_WARPS][MOP_LBUF];
    __shared__ unsigned s_pcnt[MOP_PL_WARPS][32];
    __shared__ float4 s_j[MOP_PL_WARPS][32 * 9];

    const MopGrid &g = a.g;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = a.bead0 + blockIdx.y;
    const int ci = blockIdx.x * MOP_PL_WARPS + w;
    const int noc = g.S / MOP_CL;
    if (ci >= noc) return;
    const float4 blo = a.blo[(size_t)n * noc + ci], bhi = a.bhi[(size_t)n * noc + ci];
    if (__float_as_int(blo.w) == 0) return; // no real atom in this octet

    const int *perm = a.perm + (size_t)n * g.S;
    const int *slot_of = a.slot_of + (size_t)n * g.Q;
    const float4 *xq = a.xq + (size_t)n * g.S;
    const float4 *jlo = a.blo + (size_t)n * noc, *jhi = a.bhi + (size_t)n * noc;
    const int *col_start = a.col_start + (size_t)n * (g.ncol + 1);
    int *exJ = s_exJ[w];
    unsigned(*exM)[2] = s_exM[w];
    unsigned *bcj = s_bcj[w], *binfo = s_binfo[w], *pcnt = s_pcnt[w];
    float4 *sj = s_j[w];
    const int J0 = ci;

    if (lane < MOP_EXROWS) {
        // row 0: the octet itself, only j slot > i slot (byte k of the 64-bit row = allowed j slots of i atom k)
        unsigned lo = 0, hi = 0;
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 4; k++) {
                lo |= ((0xffu << (k + 1)) & 0xffu) << (8 * k);
                hi |= ((0xffu << (k + 5)) & 0xffu) << (8 * k);
            }
        }
        exM[lane][0] = lane == 0 ? lo : 0xffffffffu;
        exM[lane][1] = lane == 0 ? hi : 0xffffffffu;
    }
    for (int t = 32 + lane; t < MOP_EXROWS; t += 32) exM[t][0] = exM[t][1] = 0xffffffffu;
    pcnt[lane] = 0;
    if (lane == 0) {
        exJ[0] = J0;
        s_exN[w] = 1;
    }
    __syncwarp();

    // ---- exclusion rows: for each i atom, clear the bit of every excluded partner in its j-octet's row
    // (four lanes per i atom, so the dependent loads perm -> excl_start -> excl_list -> slot_of of the 8 atoms are
    // in flight together instead of one atom after the other)
    if (a.excl_start != nullptr) {
        const int k = lane >> 2, sub = lane & 3;
        const int orig = perm[ci * MOP_CL + k];
        int e0 = 0, e1 = 0;
        if (orig >= 0) e0 = a.excl_start[orig], e1 = a.excl_start[orig + 1];
        const int maxn = __reduce_max_sync(0xffffffffu, e1 - e0);
        for (int eb = 0; eb < maxn; eb += 4) {
            const int e = e0 + eb + sub;
            bool act = e < e1;
            int J = -1, bit = 0;
            if (act) {
                const int ps = slot_of[a.excl_list[e]];
                MOP_ASSERT(ps >= 0 && ps < g.S);
                J = ps >> 3;
                bit = ps & 7;
                if (J < J0) act = false; // never listed from this side
            }
            unsigned pend = __ballot_sync(0xffffffffu, act);
            while (pend) {
                const int leader = __ffs(pend) - 1;
                const int Jl = __shfl_sync(0xffffffffu, J, leader);
                const int nrow = s_exN[w];
                unsigned hit = __ballot_sync(0xffffffffu, lane < nrow && exJ[lane] == Jl);
                int row = hit ? __ffs(hit) - 1 : -1;
                if (!hit && nrow > 32) {
                    hit = __ballot_sync(0xffffffffu, lane + 32 < nrow && exJ[lane + 32] == Jl);
                    if (hit) row = 32 + __ffs(hit) - 1;
                }
                if (row < 0) {
                    if (nrow < MOP_EXROWS) {
                        row = nrow;
                        if (lane == 0) {
                            exJ[nrow] = Jl;
                            s_exN[w] = nrow + 1;
                        }
                    } else if (lane == 0) {
                        atomicOr(&a.ctr->overflow, 16u);
                    }
                }
                __syncwarp();
                const bool same = act && J == Jl;
                if (same && row >= 0) atomicAnd(&exM[row][k >> 2], ~(1u << (8 * (k & 3) + bit)));
                pend &= ~__ballot_sync(0xffffffffu, same);
                __syncwarp();
            }
        }
    }
    __syncwarp();
    const int exN = s_exN[w];

    // ---- phases 2 and 3 for the candidates staged so far: one work unit.  Called when the staging buffer is nearly
    // full (an i-octet with more candidates than it holds gets several units) and at the end.
    const int gq = lane >> 3, jl = lane & 7;
    f2 xi[4], yi[4], zi[4];
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float4 a0 = xq[ci * MOP_CL + 2 * p], a1 = xq[ci * MOP_CL + 2 * p + 1];
        xi[p] = f2_pack(a0.x, a1.x), yi[p] = f2_pack(a0.y, a1.y), zi[p] = f2_pack(a0.z, a1.z);
    }
    // The candidates of an i-octet are staged in shared memory; when the buffer is nearly full (rare: sparse columns
    // make long octets with many neighbours) one work unit is made from what is staged and phase 1 resumes where it
    // stopped, so an i-octet can have several units.
    unsigned mb = 0xffffffffu; // first exclusion-mask row of this i-octet (allocated by its first unit)
    int kz0 = -1, ob0 = 0, base0 = 0; // where phase 1 resumes
    for (;;) {
    int nbuf = 0;
    bool full = false;
        // ---- phase 1: candidate j-octets.  Each lane takes one neighbouring column (under its x,y periodic image)
        // and one z image; the column's z bins (S0's thin cells) give the slot range that can hold atoms within
        // r_list in z, hence a short run of octets.  The runs of the 32 lanes are enumerated flat (prefix sum +
        // binary search), so every lane tests one octet bounding box per iteration.
        const int nx = g.dims[0], ny = g.dims[1], nz = g.dims[2];
        const int cx = mop_cell1(blo.x, g.sc[0], nx), cy = mop_cell1(blo.y, g.sc[1], ny);
        const int mx = (int)floorf(a.rl / g.colw[0]) + 1, my = (int)floorf(a.rl / g.colw[1]) + 1;
        const int wy = 2 * my + 1, noff = (2 * mx + 1) * wy;
        const float marg = 1.0e-4f, mz = 1.0e-3f;
        const float zlo = blo.z - a.rl - mz, zhi = bhi.z + a.rl + mz;
        const int *cell_rel = a.cell_rel + (size_t)n * g.ncell;
        const int *col_count = a.col_count + (size_t)n * g.ncol;
        for (int kz = kz0; kz <= 1 && !full; kz++) {
            if (kz == -1 && !(zlo < 0.0f)) continue;
            if (kz == 1 && !(zhi > g.box[2])) continue;
            const float zoff = (float)kz * g.box[2];   // the column's atoms are seen at z + kz Lz
            for (int ob = kz == kz0 ? ob0 : 0; ob < noff && !full; ob += 32) {
                const int t = ob + lane;
                int first = 0, cnt = 0;
                unsigned sid = 0;
                if (t < noff) {
                    const int gx = cx + t / wy - mx, gy = cy + t % wy - my;
                    const int kx = gx < 0 ? -1 : (gx >= nx ? 1 : 0), ky = gy < 0 ? -1 : (gy >= ny ? 1 : 0);
                    const int colx = gx - kx * nx, coly = gy - ky * ny;
                    if (colx >= 0 && colx < nx && coly >= 0 && coly < ny) {
                        const float clo = (float)colx * g.colw[0] + (float)kx * g.box[0];
                        const float cylo = (float)coly * g.colw[1] + (float)ky * g.box[1];
                        const float dxg = mop_gap(blo.x, bhi.x, clo - marg * g.box[0], clo + g.colw[0] + marg * g.box[0]);
                        const float dyg = mop_gap(blo.y, bhi.y, cylo - marg * g.box[1], cylo + g.colw[1] + marg * g.box[1]);
                        const float dxy2 = dxg * dxg + dyg * dyg;
                        // the z window of THIS column: atoms within r_list of the i box lie within sqrt(r_list^2 - gap_xy^2)
                        // in z (a sphere, not a cylinder: a third fewer octets to test than with the full r_list)
                        const float reach = sqrtf(fmaxf(a.rl2 - dxy2, 0.0f)) + mz;
                        const float za = fmaxf(blo.z - reach - zoff, 0.0f), zb = fminf(bhi.z + reach - zoff, g.box[2]);
                        if (dxy2 < a.rl2 && za <= zb) {
                            const int b0 = max(mop_cell1(za, g.sc[2], nz) - 1, 0);
                            const int b1 = min(mop_cell1(zb, g.sc[2], nz) + 1, nz - 1);
                            const int col = colx * ny + coly;
                            const int s0 = col_start[col];
                            const int r0 = cell_rel[(size_t)col * nz + b0];
                            const int r1 = b1 + 1 < nz ? cell_rel[(size_t)col * nz + b1 + 1] : col_count[col];
                            if (r1 > r0) {
                                first = max((s0 + r0) >> 3, J0); // half list: never below the own octet
                                cnt = max(((s0 + r1 - 1) >> 3) - first + 1, 0);
                                sid = (unsigned)((kx + 1) | ((ky + 1) << 2) | ((kz + 1) << 4));
                            }
                        }
                    }
                }
                int incl = cnt;
    #pragma unroll
                for (int o = 1; o < 32; o <<= 1) {
                    const int v = __shfl_up_sync(0xffffffffu, incl, o);
                    if (lane >= o) incl += v;
                }
                const int total = __shfl_sync(0xffffffffu, incl, 31);
                for (int base = (kz == kz0 && ob == ob0) ? base0 : 0; base < total; base += 32) {
                    if (nbuf + 32 > MOP_LBUF) { // staging buffer nearly full: one unit from what is staged, then resume here
                        kz0 = kz, ob0 = ob, base0 = base;
                        full = true;
                        break;
                    }
                    const int f = base + lane;
                    int lo_s = 0, hi_s = 31;
    #pragma unroll
                    for (int it = 0; it < 5; it++) { // smallest lane s with incl[s] > f
                        const int mid = (lo_s + hi_s) >> 1;
                        const int v = __shfl_sync(0xffffffffu, incl, mid);
                        if (v > f) hi_s = mid;
                        else lo_s = mid + 1;
                    }
                    const int seg = min(lo_s, 31);
                    const int s_incl = __shfl_sync(0xffffffffu, incl, seg), s_cnt = __shfl_sync(0xffffffffu, cnt, seg);
                    const int s_first = __shfl_sync(0xffffffffu, first, seg);
                    const unsigned s_sid = __shfl_sync(0xffffffffu, sid, seg);
                    bool ok = f < total;
                    const int cj = s_first + (f - (s_incl - s_cnt));
                    if (ok) {
                        MOP_ASSERT(cj >= 0 && cj < noc);
                        float4 lo = jlo[cj], hi = jhi[cj];
                        ok = __float_as_int(lo.w) > 0;
                        float sx, sy, sz;
                        mop_unit_shift((int)s_sid, g.box, sx, sy, sz);
                        lo.x += sx, hi.x += sx, lo.y += sy, hi.y += sy, lo.z += sz, hi.z += sz;
                        const float ex = mop_gap(blo.x, bhi.x, lo.x, hi.x), ey = mop_gap(blo.y, bhi.y, lo.y, hi.y),
                                    ez = mop_gap(blo.z, bhi.z, lo.z, hi.z);
                        ok = ok && (ex * ex + ey * ey + ez * ez < a.rl2);
                    }
                    const unsigned bal = __ballot_sync(0xffffffffu, ok);
                    if (ok) {
                        MOP_ASSERT(nbuf + __popc(bal & ((1u << lane) - 1)) < MOP_LBUF);
                        bcj[nbuf + __popc(bal & ((1u << lane) - 1))] = (unsigned)cj | (s_sid << 24);
                    }
                    nbuf += __popc(bal);
                }
            }
        }
    __syncwarp();
    if (nbuf > 0) {
        do {
        __syncwarp();

        // ---- phase 2: one candidate per lane.  The 8 i atoms (packed two by two: the row pairs of the pair kernels)
        // against the 8 atoms of the lane's j-octet (xs_i = x_i - k L once per candidate, d = xs_i - x_j: the pair kernels'
        // d = (x_i - x_j) - k L up to a few ulp(L), far inside the 1e-4 inflation of r_list^2); pattern bit p = some pair of
        // row pair p within r_list.  Padding atoms are never within range (mop_dummy_xq).  Then the exclusion row of the
        // octet pair (at most one matches) and the position inside the bucket of (pattern, shifted or not): lanes with
        // equal keys are ranked with one match, the first of them draws the range from the bucket's counter.
        unsigned nslots = 0;
        const unsigned pcnt_addr = (unsigned)__cvta_generic_to_shared(pcnt);
        for (int b = 0; b < nbuf; b += 32) {
            const int idx = b + lane;
            const bool live = idx < nbuf;
            const unsigned cw = live ? bcj[idx] : ((unsigned)ci | ((unsigned)MOP_NOSHIFT << 24));
            const unsigned cj = cw & 0xffffffu, sid = cw >> 24;
            float sx, sy, sz;
            mop_unit_shift((int)sid, g.box, sx, sy, sz);
            const f2 hx = f2_bc(sx), hy = f2_bc(sy), hz = f2_bc(sz);
            f2 xs[4], ys[4], zs[4];
    #pragma unroll
            for (int p = 0; p < 4; p++) xs[p] = f2_sub(xi[p], hx), ys[p] = f2_sub(yi[p], hy), zs[p] = f2_sub(zi[p], hz);
            float best[4] = {3.0e38f, 3.0e38f, 3.0e38f, 3.0e38f}; // smallest r2 of each row pair
            // the 32 candidates' octets go through shared memory: coalesced loads (lane = (atom jl, candidate 4 t + gq)),
            // then every lane reads the 8 atoms of its own candidate (row stride 9 float4: conflict-free)
            __syncwarp();
    #pragma unroll
            for (int t = 0; t < 8; t++) {
                const unsigned cwt = __shfl_sync(0xffffffffu, cw, 4 * t + gq);
                sj[(4 * t + gq) * 9 + jl] = xq[(size_t)(cwt & 0xffffffu) * MOP_CL + jl];
            }
            __syncwarp();
    #pragma unroll
            for (int j = 0; j < MOP_CL; j++) {
                const float4 q = sj[lane * 9 + j];
                const f2 jx = f2_bc(q.x), jy = f2_bc(q.y), jz = f2_bc(q.z);
    #pragma unroll
                for (int p = 0; p < 4; p++) {
                    const f2 dx = f2_sub(xs[p], jx), dy = f2_sub(ys[p], jy), dz = f2_sub(zs[p], jz);
                    float r2a, r2b;
                    f2_unpack(f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx))), r2a, r2b);
                    best[p] = fminf(best[p], fminf(r2a, r2b));
                }
            }
            unsigned pat = 0;
    #pragma unroll
            for (int p = 0; p < 4; p++)
                if (best[p] < a.rl2) pat |= 1u << p;
            if (!live) pat = 0;
            unsigned row1 = 0;
            for (int t = 0; t < exN; t++)
                if ((unsigned)exJ[t] == cj) row1 = (unsigned)t + 1u;
            const unsigned key = pat == 0 ? 0u : (pat | (sid != MOP_NOSHIFT ? 16u : 0u));
            const unsigned same = __match_any_sync(0xffffffffu, key);
            const unsigned rank = __popc(same & ((1u << lane) - 1u));
            unsigned base = 0;
            if (rank == 0 && key != 0)
                asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(base) : "r"(pcnt_addr + key * 4u), "r"(__popc(same)) : "memory");
            base = __shfl_sync(0xffffffffu, base, __ffs(same) - 1);
            if (live) binfo[idx] = key == 0 ? 0u : (key | (row1 << 8) | ((base + rank) << 16));
            nslots += __popc(pat) * 16u;
        }
        __syncwarp();

        // ---- bucket starts: the 15 plain buckets in pattern order, then the 15 shifted ones in reverse pattern order (one
        // junction between plain and shifted entries, and between equal patterns: few steps take the general body for a
        // single shifted entry), total, padded total
        unsigned mycnt = 0, mykey = 0;
        if (lane < 30) {
            mykey = lane < 15 ? (unsigned)c_pat_order[lane] : ((unsigned)c_pat_order[29 - lane] | 16u);
            mycnt = pcnt[mykey];
        }
        unsigned incl = mycnt;
    #pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned v = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += v;
        }
        const unsigned total = __shfl_sync(0xffffffffu, incl, 31);
        if (total == 0) break;
        __syncwarp();
        if (lane < 30) pcnt[mykey] = incl - mycnt; // exclusive start of the bucket
        __syncwarp();
        const unsigned padded = (total + MOP_NG - 1) & ~(unsigned)(MOP_NG - 1);
        nslots = (unsigned)__reduce_add_sync(0xffffffffu, nslots);

        // ---- exclusion-mask rows of this i-octet, unit record, entries
        const bool first = mb == 0xffffffffu; // the mask rows are written with the i-octet's first unit
        unsigned st = 0, ui = 0;
        if (lane == 0) {
            atomicAdd(a.slots_active, (unsigned long long)nslots);
            if (first) mb = atomicAdd(&a.ctr->n_masks, (unsigned)exN);
            st = atomicAdd(&a.ctr->n_entries, padded);
            ui = atomicAdd(&a.ctr->n_units, 1u);
        }
        mb = __shfl_sync(0xffffffffu, mb, 0);
        st = __shfl_sync(0xffffffffu, st, 0);
        ui = __shfl_sync(0xffffffffu, ui, 0);
        const bool fits = mb + exN <= a.cap_masks && st + padded <= a.cap_entries && ui < a.cap_units;
        if (!fits) {
            if (lane == 0) {
                atomicOr(&a.ctr->overflow, (mb + exN > a.cap_masks ? 4u : 0u) | (st + padded > a.cap_entries ? 1u : 0u) |
                                               (ui >= a.cap_units ? 2u : 0u));
                if (ui < a.cap_units) {
                    MopUnit un = {n, ci, 0u, 0u, 0u, 0u, 0u, 0u};
                    a.units[ui] = un;
                }
            }
            break;
        }
        // mask rows leave transposed: byte jl of the 64-bit row = the i atoms (bits 0-7) j atom jl may interact with, so
        // that a lane of the pair kernels reads its 8 bits with one byte load (8x8 bit-matrix transpose, three swaps)
        for (int t = lane; first && t < exN; t += 32) {
            unsigned long long x = (unsigned long long)exM[t][0] | ((unsigned long long)exM[t][1] << 32), y;
            y = (x ^ (x >> 7)) & 0x00AA00AA00AA00AAull, x ^= y ^ (y << 7);
            y = (x ^ (x >> 14)) & 0x0000CCCC0000CCCCull, x ^= y ^ (y << 14);
            y = (x ^ (x >> 28)) & 0x00000000F0F0F0F0ull, x ^= y ^ (y << 28);
            MOP_ASSERT(mb + t < a.cap_masks);
            a.masks[(size_t)mb + t] = x;
        }
        // entries in their final order go through shared memory (the j staging buffer is free now), so that every step of
        // four can be given its union pattern and flags: y bits 16-19 union of the four patterns, bit 20 some entry of the
        // step is shifted, bit 21 some entry has an exclusion row or is padding.  The pair kernels branch on these.
        __syncwarp();
        uint2 *sorted = reinterpret_cast<uint2 *>(sj);
        for (int idx = lane; idx < nbuf; idx += 32) {
            const unsigned info = binfo[idx];
            if (info == 0) continue;
            MOP_ASSERT(pcnt[info & 31u] + (info >> 16) < (unsigned)(32 * 9 * 2));   // the j staging buffer, as uint2
            sorted[pcnt[info & 31u] + (info >> 16)] = make_uint2(bcj[idx], info & 0xff0fu);
        }
        if (lane < (int)(padded - total)) sorted[total + lane] = make_uint2((unsigned)ci | ((unsigned)MOP_NOSHIFT << 24), 0u);
        __syncwarp();
        unsigned nunion = 0;   // pair slots the pair kernels evaluate: 64 per row pair of every step's union pattern
        for (unsigned sidx = lane; sidx < padded / MOP_NG; sidx += 32) {
            uint2 e[MOP_NG];
            unsigned u = 0, fl = 0;
    #pragma unroll
            for (int q = 0; q < MOP_NG; q++) {
                e[q] = sorted[sidx * MOP_NG + q];
                u |= e[q].y & 15u;
                if ((e[q].x >> 24) != MOP_NOSHIFT) fl |= 1u << 20;
                if ((e[q].y >> 8) != 0u || (e[q].y & 15u) == 0u) fl |= 1u << 21;
            }
            fl |= u << 16;
            nunion += __popc(u) * 64u;
            MOP_ASSERT(st + (sidx + 1) * MOP_NG <= a.cap_entries && (st % MOP_NG) == 0);
            uint4 *dst = reinterpret_cast<uint4 *>(a.entries + st + sidx * MOP_NG); // st is a multiple of 4: 32 B aligned
            dst[0] = make_uint4(e[0].x, e[0].y | fl, e[1].x, e[1].y | fl);
            dst[1] = make_uint4(e[2].x, e[2].y | fl, e[3].x, e[3].y | fl);
        }
        nunion = (unsigned)__reduce_add_sync(0xffffffffu, nunion);
        if (lane == 0) {
            MopUnit un = {n, ci, st, padded, mb, 0u, 0u, 0u};
            a.units[ui] = un;
            atomicAdd(a.slots_active + 1, (unsigned long long)nunion);
        }
        } while (false);
    }
    if (!full) break;
    __syncwarp();
    pcnt[lane] = 0;
    __syncwarp();
    } // resume loop
}

__global__ void k_mark_bead0(MopCounters *ctr, unsigned cap_units) { ctr->n_units_bead0 = min(ctr->n_units, cap_units); }
__global__ void k_mark_mid(MopCounters *ctr, unsigned cap_units) { ctr->n_units_mid = min(ctr->n_units, cap_units); }
