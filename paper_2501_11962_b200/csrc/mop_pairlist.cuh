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
    unsigned long long *slots_active; // sum over entries of popc(pattern) * 16
    unsigned cap_units, cap_entries, cap_masks;
};

__device__ __forceinline__ float mop_gap(float lo_a, float hi_a, float lo_b, float hi_b) {
    // distance between intervals [lo_a,hi_a] and [lo_b,hi_b]
    return fmaxf(0.0f, fmaxf(lo_b - hi_a, lo_a - hi_b));
}

// bucket order of the 15 non-zero patterns: full first, then the contiguous runs (the usual partial patterns, the
// row pairs of an octet being ordered along z), then the rest
__constant__ unsigned char c_pat_order[16] = {15, 7, 3, 1, 14, 12, 8, 6, 2, 4, 5, 9, 10, 11, 13, 0};

__global__ void __launch_bounds__(128) k_pairlist(PlArgs a) {
    __shared__ int s_exJ[4][MOP_EXROWS];
    __shared__ unsigned s_exM[4][MOP_EXROWS][2];
    __shared__ int s_exN[4];
    __shared__ unsigned s_bcj[4][MOP_LBUF];
    __shared__ unsigned s_binfo[4][MOP_LBUF];
    __shared__ unsigned s_pcnt[4][16];

    const MopGrid &g = a.g;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = a.bead0 + blockIdx.y;
    const int ci = blockIdx.x * 4 + w;
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
    if (lane < 16) pcnt[lane] = 0;
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
    int nbuf = 0;
    for (int kz = -1; kz <= 1; kz++) {
        if (kz == -1 && !(zlo < 0.0f)) continue;
        if (kz == 1 && !(zhi > g.box[2])) continue;
        const float za = kz == 0 ? fmaxf(zlo, 0.0f) : (kz == -1 ? zlo + g.box[2] : 0.0f);
        const float zb = kz == 0 ? fminf(zhi, g.box[2]) : (kz == -1 ? g.box[2] : zhi - g.box[2]);
        const int b0 = max(mop_cell1(fmaxf(za, 0.0f), g.sc[2], nz) - 1, 0);
        const int b1 = min(mop_cell1(fminf(zb, g.box[2]), g.sc[2], nz) + 1, nz - 1);
        for (int ob = 0; ob < noff; ob += 32) {
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
                    if (dxg * dxg + dyg * dyg < a.rl2) {
                        const int col = colx * ny + coly;
                        const int s0 = col_start[col];
                        const int r0 = cell_rel[(size_t)col * nz + b0];
                        const int r1 = b1 + 1 < nz ? cell_rel[(size_t)col * nz + b1 + 1] : col_count[col];
                        if (r1 > r0) {
                            first = max((s0 + r0) >> 3, J0); // half list: never below the own octet
                            cnt = max(((s0 + r1 - 1) >> 3) - first + 1, 0);
                            sid = (unsigned)((kx + 1) + 3 * (ky + 1) + 9 * (kz + 1));
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
            for (int base = 0; base < total; base += 32) {
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
                    const int pos = nbuf + __popc(bal & ((1u << lane) - 1));
                    if (pos < MOP_LBUF) bcj[pos] = (unsigned)cj | (s_sid << 24);
                }
                nbuf += __popc(bal);
            }
        }
    }
    __syncwarp();
    if (nbuf > MOP_LBUF) {
        if (lane == 0) atomicOr(&a.ctr->overflow, 8u);
        nbuf = MOP_LBUF;
    }

    // ---- phase 2: four candidates per step, lane = (j atom jl, candidate g): the 8 i atoms (packed two by two, the
    // row pairs of the pair kernels) against the lane's j atom with the arithmetic of the pair kernels
    // (xs_i = x_i - k L, d = xs_i - x_j, r2 = fma(dz,dz,fma(dy,dy,dx dx)); x - 0 = x exactly, so the steps without a
    // shifted candidate skip the first subtraction); pattern bit p = some pair of row pair p within r_list.
    // Padding atoms are never within range (mop_dummy_xq).
    const int gq = lane >> 3, jl = lane & 7;
    f2 xi[4], yi[4], zi[4];
#pragma unroll
    for (int p = 0; p < 4; p++) {
        const float4 a0 = xq[ci * MOP_CL + 2 * p], a1 = xq[ci * MOP_CL + 2 * p + 1];
        xi[p] = f2_pack(a0.x, a1.x), yi[p] = f2_pack(a0.y, a1.y), zi[p] = f2_pack(a0.z, a1.z);
    }
    for (int b = 0; b < nbuf; b += MOP_NG) {
        const int idx = b + gq;
        const bool live = idx < nbuf;
        const unsigned cw = live ? bcj[idx] : ((unsigned)ci | ((unsigned)MOP_NOSHIFT << 24));
        const int cj = (int)(cw & 0xffffffu);
        const unsigned sid = cw >> 24;
        const float4 pj = xq[cj * MOP_CL + jl];
        const f2 jx = f2_bc(pj.x), jy = f2_bc(pj.y), jz = f2_bc(pj.z);
        unsigned pat = 0;
        if (__any_sync(0xffffffffu, sid != MOP_NOSHIFT)) {
            float sx, sy, sz;
            mop_unit_shift((int)sid, g.box, sx, sy, sz);
            const f2 hx = f2_bc(sx), hy = f2_bc(sy), hz = f2_bc(sz);
#pragma unroll
            for (int p = 0; p < 4; p++) {
                const f2 dx = f2_sub(f2_sub(xi[p], hx), jx), dy = f2_sub(f2_sub(yi[p], hy), jy),
                         dz = f2_sub(f2_sub(zi[p], hz), jz);
                float r2a, r2b;
                f2_unpack(f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx))), r2a, r2b);
                const unsigned bal = __ballot_sync(0xffffffffu, fminf(r2a, r2b) < a.rl2);
                if ((bal >> (8 * gq)) & 0xffu) pat |= 1u << p;
            }
        } else {
#pragma unroll
            for (int p = 0; p < 4; p++) {
                const f2 dx = f2_sub(xi[p], jx), dy = f2_sub(yi[p], jy), dz = f2_sub(zi[p], jz);
                float r2a, r2b;
                f2_unpack(f2_fma(dz, dz, f2_fma(dy, dy, f2_mul(dx, dx))), r2a, r2b);
                const unsigned bal = __ballot_sync(0xffffffffu, fminf(r2a, r2b) < a.rl2);
                if ((bal >> (8 * gq)) & 0xffu) pat |= 1u << p;
            }
        }
        if (live && jl == 0) binfo[idx] = pat;
    }
    __syncwarp();

    // ---- per candidate: exclusion row of its octet pair (at most one row matches) and position inside its pattern's
    // bucket (lanes with equal patterns are ranked with one match; the first of them draws the range from the counter)
    unsigned nslots = 0;
    const unsigned pcnt_addr = (unsigned)__cvta_generic_to_shared(pcnt);
    for (int b = 0; b < nbuf; b += 32) {
        const int idx = b + lane;
        unsigned pat = 0, cj = 0xffffffffu;
        if (idx < nbuf) pat = binfo[idx], cj = bcj[idx] & 0xffffffu;
        unsigned row1 = 0;
        for (int t = 0; t < exN; t++)
            if ((unsigned)exJ[t] == cj) row1 = (unsigned)t + 1u;
        const unsigned same = __match_any_sync(0xffffffffu, pat);
        const unsigned rank = __popc(same & ((1u << lane) - 1u));
        unsigned base = 0;
        if (rank == 0 && pat != 0)
            asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(base) : "r"(pcnt_addr + pat * 4u), "r"(__popc(same)) : "memory");
        base = __shfl_sync(0xffffffffu, base, __ffs(same) - 1);
        if (pat != 0) {
            binfo[idx] = pat | (row1 << 8) | ((base + rank) << 16);
            nslots += __popc(pat) * 16u;
        }
    }
    __syncwarp();

    // ---- bucket starts in pattern order, total, padded total
    unsigned mycnt = 0, mypat = 0;
    if (lane < 15) {
        mypat = c_pat_order[lane];
        mycnt = pcnt[mypat];
    }
    unsigned incl = mycnt;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        const unsigned v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += v;
    }
    const unsigned total = __shfl_sync(0xffffffffu, incl, 14);
    if (total == 0) return;
    __syncwarp();
    if (lane < 15) pcnt[mypat] = incl - mycnt; // exclusive start of the bucket
    __syncwarp();
    const unsigned padded = (total + MOP_NG - 1) & ~(unsigned)(MOP_NG - 1);
    nslots = (unsigned)__reduce_add_sync(0xffffffffu, nslots);

    // ---- exclusion-mask rows of this i-octet, unit record, entries
    unsigned mb = 0, st = 0, ui = 0;
    if (lane == 0) {
        atomicAdd(a.slots_active, (unsigned long long)nslots);
        mb = atomicAdd(&a.ctr->n_masks, (unsigned)exN);
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
        return;
    }
    for (int t = lane; t < exN; t += 32)
        a.masks[(size_t)mb + t] = (unsigned long long)exM[t][0] | ((unsigned long long)exM[t][1] << 32);
    for (int idx = lane; idx < nbuf; idx += 32) {
        const unsigned info = binfo[idx];
        if (info == 0) continue;
        const unsigned pos = st + pcnt[info & 15u] + (info >> 16);
        a.entries[pos] = make_uint2(bcj[idx], info & 0xffffu);
    }
    if (lane < (int)(padded - total))
        a.entries[st + total + lane] = make_uint2((unsigned)ci | ((unsigned)MOP_NOSHIFT << 24), 0u);
    if (lane == 0) {
        MopUnit un = {n, ci, st, padded, mb, 0u, 0u, 0u};
        a.units[ui] = un;
    }
}

__global__ void k_mark_bead0(MopCounters *ctr, unsigned cap_units) { ctr->n_units_bead0 = min(ctr->n_units, cap_units); }
