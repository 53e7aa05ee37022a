// mop_pairlist.cuh -- S1: cluster-pair list.
//
// One warp per i-cluster (8 consecutive sorted slots).  For every periodic shift it lists the j-clusters
// (32 slots, index >= the i-cluster's own j-cluster: half list) whose bounding box comes within r_list of the
// i-cluster's box, with an 8-bit mask of the i atoms that come within r_list of the j box, and the index of
// an exclusion-mask row when the cluster pair holds excluded pairs (or is the diagonal block, where only
// lane > own lane is allowed).  Output: work units (bead, i-cluster, shift) -> contiguous entry ranges.
// The list is only a superset; the pair kernels apply the exact FP32 predicate (G8) per atom pair.
#pragma once
#include "mop_common.cuh"

struct PlArgs {
    MopGrid g;
    int bead0;
    float rl, rl2; // list radius, and its square inflated by 1e-4 (conservative against FP32 rounding)
    const int *perm, *slot_of;
    const float4 *xq, *jlo, *jhi, *ilo, *ihi;
    const int *col_start, *cell_rel, *col_count;
    const int *excl_start, *excl_list; // may be NULL
    MopUnit *units;
    MopEntry *entries;
    unsigned *masks;
    MopCounters *ctr;
    unsigned long long *slots_active; // sum over entries of popc(imask)
    unsigned cap_units, cap_entries, cap_masks;
};

__device__ __forceinline__ float mop_gap(float lo_a, float hi_a, float lo_b, float hi_b) {
    // distance between intervals [lo_a,hi_a] and [lo_b,hi_b]
    return fmaxf(0.0f, fmaxf(lo_b - hi_a, lo_a - hi_b));
}

__global__ void __launch_bounds__(128) k_pairlist(PlArgs a) {
    __shared__ float4 s_ia[4][MOP_CI];
    __shared__ int s_exJ[4][MOP_EXROWS];
    __shared__ unsigned s_exM[4][MOP_EXROWS][MOP_CI];
    __shared__ int s_exN[4];
    __shared__ int s_bcj[4][MOP_LBUF];
    __shared__ unsigned s_binfo[4][MOP_LBUF];

    const MopGrid &g = a.g;
    const int w = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int n = a.bead0 + blockIdx.y;
    const int ci = blockIdx.x * 4 + w;
    const int nci = g.S / MOP_CI, ncj = g.S / MOP_CJ;
    if (ci >= nci) return;
    const float4 blo = a.ilo[(size_t)n * nci + ci], bhi = a.ihi[(size_t)n * nci + ci];
    if (__float_as_int(blo.w) == 0) return; // no real atom in this i-cluster

    const int *perm = a.perm + (size_t)n * g.S;
    const int *slot_of = a.slot_of + (size_t)n * g.Q;
    const float4 *xq = a.xq + (size_t)n * g.S;
    const float4 *jlo = a.jlo + (size_t)n * ncj, *jhi = a.jhi + (size_t)n * ncj;
    const int *col_start = a.col_start + (size_t)n * (g.ncol + 1);
    float4 *ia = s_ia[w];
    int *exJ = s_exJ[w];
    unsigned(*exM)[MOP_CI] = s_exM[w];
    int *bcj = s_bcj[w];
    unsigned *binfo = s_binfo[w];
    const int J0 = ci >> 2;

    if (lane < MOP_CI) {
        int s = ci * MOP_CI + lane;
        float4 p = xq[s];
        p.w = perm[s] >= 0 ? 1.0f : 0.0f;
        ia[lane] = p;
        int li = (ci & 3) * MOP_CI + lane; // own lane inside the diagonal j-cluster: only lanes > li are allowed
        exM[0][lane] = li == 31 ? 0u : (0xffffffffu << (li + 1));
    }
    if (lane == 0) {
        exJ[0] = J0;
        s_exN[w] = 1;
    }
    __syncwarp();

    // ---- exclusion rows: for each i atom, clear the bit of every excluded partner in its j-cluster's row
    // (four lanes per i atom, so the dependent loads perm -> excl_start -> excl_list -> slot_of of the 8 atoms are
    // in flight together instead of one atom after the other)
    if (a.excl_start != nullptr) {
        const int k = lane >> 2, sub = lane & 3;
        const int orig = perm[ci * MOP_CI + k];
        int e0 = 0, e1 = 0;
        if (orig >= 0) e0 = a.excl_start[orig], e1 = a.excl_start[orig + 1];
        const int maxn = __reduce_max_sync(0xffffffffu, e1 - e0);
        for (int eb = 0; eb < maxn; eb += 4) {
            const int e = e0 + eb + sub;
            bool act = e < e1;
            int J = -1, bit = 0;
            if (act) {
                const int ps = slot_of[a.excl_list[e]];
                J = ps >> 5;
                bit = ps & 31;
                if (J < J0) act = false; // never listed from this side
            }
            unsigned pend = __ballot_sync(0xffffffffu, act);
            while (pend) {
                const int leader = __ffs(pend) - 1;
                const int Jl = __shfl_sync(0xffffffffu, J, leader);
                const int nrow = s_exN[w];
                const unsigned hit = __ballot_sync(0xffffffffu, lane < nrow && exJ[lane] == Jl);
                int row;
                if (hit) {
                    row = __ffs(hit) - 1;
                } else if (nrow < MOP_EXROWS) {
                    row = nrow;
                    if (lane == 0) {
                        exJ[nrow] = Jl;
                        s_exN[w] = nrow + 1;
                    }
                    if (lane < MOP_CI) exM[nrow][lane] = 0xffffffffu;
                } else {
                    row = -1;
                    if (lane == 0) atomicOr(&a.ctr->overflow, 16u);
                }
                __syncwarp();
                const bool same = act && J == Jl;
                if (same && row >= 0) atomicAnd(&exM[row][k], ~(1u << bit));
                pend &= ~__ballot_sync(0xffffffffu, same);
                __syncwarp();
            }
        }
    }
    __syncwarp();
    const int exN = s_exN[w];

    // ---- phase 1: candidate j-clusters.  Each lane takes one neighbouring column (under its x,y periodic image)
    // and one z image; the column's z bins (S0's thin cells) give the slot range that can hold atoms within
    // r_list in z, hence a short run of j-clusters.  The runs of the 32 lanes are enumerated flat (prefix sum +
    // binary search), so every lane tests one cluster bounding box per iteration.
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
                            first = max((s0 + r0) >> 5, J0); // half list: never below the own j-cluster
                            cnt = max(((s0 + r1 - 1) >> 5) - first + 1, 0);
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
                    if (pos < MOP_LBUF) {
                        bcj[pos] = cj;
                        binfo[pos] = s_sid;
                    }
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
    // ---- phase 2: per candidate, which i atoms come within r_list of the j box (imask), and the exclusion row
    unsigned shift_seen = 0;
    unsigned nslots = 0;
    for (int b = 0; b < nbuf; b += 32) {
        const int idx = b + lane;
        unsigned info = 0xffffffffu; // dead
        if (idx < nbuf) {
            const int cj = bcj[idx];
            const unsigned sid = binfo[idx];
            float4 lo = jlo[cj], hi = jhi[cj];
            float sx, sy, sz;
            mop_unit_shift((int)sid, g.box, sx, sy, sz);
            lo.x += sx, hi.x += sx, lo.y += sy, hi.y += sy, lo.z += sz, hi.z += sz;
            unsigned imask = 0;
#pragma unroll
            for (int k = 0; k < MOP_CI; k++) {
                const float4 p = ia[k];
                const float px = mop_gap(p.x, p.x, lo.x, hi.x), py = mop_gap(p.y, p.y, lo.y, hi.y),
                            pz = mop_gap(p.z, p.z, lo.z, hi.z);
                if (p.w != 0.0f && px * px + py * py + pz * pz < a.rl2) imask |= 1u << k;
            }
            if (imask != 0) {
                unsigned row1 = 0;
                for (int t = 0; t < exN; t++)
                    if (exJ[t] == cj) row1 = (unsigned)t + 1;
                info = imask | (row1 << 8) | (sid << 16);
                nslots += __popc(imask);
            }
            binfo[idx] = info;
        }
        // the shifts that occur among the live candidates of this batch
        unsigned live = __ballot_sync(0xffffffffu, info != 0xffffffffu);
        while (live) {
            const int l = __ffs(live) - 1;
            const unsigned sidl = __shfl_sync(0xffffffffu, info, l) >> 16;
            shift_seen |= 1u << sidl;
            live &= ~__ballot_sync(0xffffffffu, info != 0xffffffffu && (info >> 16) == sidl);
        }
    }
    __syncwarp();
    if (shift_seen == 0) return;
    nslots = (unsigned)__reduce_add_sync(0xffffffffu, nslots);
    if (lane == 0) atomicAdd(a.slots_active, (unsigned long long)nslots);

    // ---- exclusion-mask rows of this i-cluster
    unsigned mb = 0;
    if (lane == 0) mb = atomicAdd(&a.ctr->n_masks, (unsigned)exN);
    mb = __shfl_sync(0xffffffffu, mb, 0);
    if (mb + exN > a.cap_masks) {
        if (lane == 0) atomicOr(&a.ctr->overflow, 4u);
        return;
    }
    for (int t = lane; t < exN * MOP_CI; t += 32) a.masks[(size_t)mb * MOP_CI + t] = exM[t / MOP_CI][t % MOP_CI];

    // ---- one unit per shift that occurred; its entries are copied out contiguously
    while (shift_seen) {
        unsigned sid = (unsigned)__ffs(shift_seen) - 1;
        shift_seen &= shift_seen - 1;
        unsigned cnt = 0;
        for (int b = 0; b < nbuf; b += 32) {
            int idx = b + lane;
            bool m = idx < nbuf && binfo[idx] != 0xffffffffu && (binfo[idx] >> 16) == sid;
            cnt += __popc(__ballot_sync(0xffffffffu, m));
        }
        if (cnt == 0) continue;
        unsigned st = 0, ui = 0;
        if (lane == 0) {
            st = atomicAdd(&a.ctr->n_entries, cnt);
            ui = atomicAdd(&a.ctr->n_units, 1u);
        }
        st = __shfl_sync(0xffffffffu, st, 0);
        ui = __shfl_sync(0xffffffffu, ui, 0);
        if (st + cnt > a.cap_entries || ui >= a.cap_units) {
            if (lane == 0) atomicOr(&a.ctr->overflow, st + cnt > a.cap_entries ? 1u : 2u);
            if (ui < a.cap_units && lane == 0) {
                MopUnit un = {n, ci, (int)sid, 0u, 0u, mb, 0u, 0u};
                a.units[ui] = un;
            }
            continue;
        }
        unsigned wr = 0;
        for (int b = 0; b < nbuf; b += 32) {
            int idx = b + lane;
            bool m = idx < nbuf && binfo[idx] != 0xffffffffu && (binfo[idx] >> 16) == sid;
            unsigned bal = __ballot_sync(0xffffffffu, m);
            if (m) {
                unsigned pos = st + wr + __popc(bal & ((1u << lane) - 1));
                a.entries[pos] = make_uint2((unsigned)bcj[idx], binfo[idx] & 0xffffu);
            }
            wr += __popc(bal);
        }
        if (lane == 0) {
            MopUnit un = {n, ci, (int)sid, st, cnt, mb, 0u, 0u};
            a.units[ui] = un;
        }
    }
}

__global__ void k_mark_bead0(MopCounters *ctr) { ctr->n_units_bead0 = min(ctr->n_units, 0xffffffffu); }
