// mop_grid.cuh -- S0: bead-batched cell-list build.
// wrap -> cell id -> histogram -> column scan (columns padded to 32 slots) -> STABLE scatter
// (within a cell ascending original index, reading G13) -> sorted float4 (x,y,z,q) + type + permutation.
// A launch processes the beads g.n0, g.n0 + 1, ... (bead = g.n0 + blockIdx.y; all nf force beads, or one group of them
// in the pipelined host entry point).  HBM-bound.
#pragma once
#include "mop_common.cuh"

// cell id of every atom + per-cell histogram.  A coordinate that is not finite, or so large that the FP32 wrap cannot
// bring it into [0, L), raises the sticky non-finite flag (reported as MOP_ERR_NONFINITE at the next synchronising call)
__global__ void __launch_bounds__(256) k_bin(const float *__restrict__ R, MopGrid g, int *__restrict__ cell,
                                             int *__restrict__ cell_count, unsigned *__restrict__ nonfinite) {
    int n = g.n0 + blockIdx.y;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Q) return;
    const float *r = R + ((size_t)n * g.Q + i) * 3;
    int c[3];
    bool ok = true;
#pragma unroll
    for (int d = 0; d < 3; d++) {
        const float xw = mop_wrap1(r[d], g.box[d], g.inv_box[d]);
        // false for NaN/Inf; beyond 1e6 box lengths the FP32 wrap has no resolution left (ulp(x) > L / 16)
        ok = ok && (xw >= 0.0f) && (xw < g.box[d]) && (fabsf(r[d]) <= 1.0e6f * g.box[d]);
        c[d] = mop_cell1(xw, g.sc[d], g.dims[d]);
    }
    if (!ok) *nonfinite = 1u;
    int id = (c[0] * g.dims[1] + c[1]) * g.dims[2] + c[2];
    MOP_ASSERT(id >= 0 && id < g.ncell);
    cell[(size_t)n * g.Q + i] = id;
    atomicAdd(&cell_count[(size_t)n * g.ncell + id], 1);
}

// one warp per column: exclusive scan of the cell counts inside the column + the column total
__global__ void __launch_bounds__(128) k_colscan(MopGrid g, const int *__restrict__ cell_count,
                                                 int *__restrict__ cell_rel, int *__restrict__ col_count) {
    int n = g.n0 + blockIdx.y;
    int col = blockIdx.x * 4 + (threadIdx.x >> 5);
    int lane = threadIdx.x & 31;
    if (col >= g.ncol) return;
    size_t base = (size_t)n * g.ncell + (size_t)col * g.dims[2];
    int run = 0;
    for (int z0 = 0; z0 < g.dims[2]; z0 += 32) {
        int z = z0 + lane;
        int c = z < g.dims[2] ? cell_count[base + z] : 0;
        int inc = c;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (z < g.dims[2]) cell_rel[base + z] = run + inc - c;
        run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) col_count[(size_t)n * g.ncol + col] = run;
}

// one CTA per bead: exclusive scan of the column counts rounded up to the cluster size -> col_start[n][0..ncol]
__global__ void __launch_bounds__(1024) k_colstart(MopGrid g, const int *__restrict__ col_count,
                                                   int *__restrict__ col_start) {
    __shared__ int wsum[32];
    __shared__ int carry;
    int n = g.n0 + blockIdx.x;
    int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    if (threadIdx.x == 0) carry = 0;
    __syncthreads();
    for (int c0 = 0; c0 < g.ncol; c0 += 1024) {
        int col = c0 + threadIdx.x;
        int v = col < g.ncol ? ((col_count[(size_t)n * g.ncol + col] + MOP_CL - 1) & ~(MOP_CL - 1)) : 0;
        int inc = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, inc, o);
            if (lane >= o) inc += t;
        }
        if (lane == 31) wsum[w] = inc;
        __syncthreads();
        if (w == 0) {
            int s = wsum[lane];
            int si = s;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int t = __shfl_up_sync(0xffffffffu, si, o);
                if (lane >= o) si += t;
            }
            wsum[lane] = si - s;
        }
        __syncthreads();
        int excl = carry + wsum[w] + inc - v;
        if (col < g.ncol) col_start[(size_t)n * (g.ncol + 1) + col] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) carry = excl + v;
        __syncthreads();
    }
    if (threadIdx.x == 0) col_start[(size_t)n * (g.ncol + 1) + g.ncol] = carry;
}

// every slot starts as padding
__global__ void __launch_bounds__(256) k_fill_pad(MopGrid g, int *__restrict__ perm, float4 *__restrict__ xq,
                                                  int *__restrict__ typ) {
    int n = g.n0 + blockIdx.y;
    int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= g.S) return;
    size_t o = (size_t)n * g.S + s;
    perm[o] = -1;
    xq[o] = mop_dummy_xq(s, g.box);
    typ[o] = 0;
}

// unstable placement inside the cell's slot range (arrival order)
__global__ void __launch_bounds__(256) k_place(MopGrid g, const int *__restrict__ cell,
                                               const int *__restrict__ cell_rel, const int *__restrict__ col_start,
                                               int *__restrict__ cell_fill, int *__restrict__ tmp) {
    int n = g.n0 + blockIdx.y;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Q) return;
    int c = cell[(size_t)n * g.Q + i];
    int col = c / g.dims[2];
    int base = col_start[(size_t)n * (g.ncol + 1) + col] + cell_rel[(size_t)n * g.ncell + c];
    int pos = atomicAdd(&cell_fill[(size_t)n * g.ncell + c], 1);
    tmp[(size_t)n * g.S + base + pos] = i;
}

// stable rank = number of atoms of the same cell with a smaller original index; writes the sorted arrays
__global__ void __launch_bounds__(256) k_rank(const float *__restrict__ R, MopGrid g, const int *__restrict__ cell,
                                              const int *__restrict__ cell_rel, const int *__restrict__ col_start,
                                              const int *__restrict__ cell_count, const int *__restrict__ tmp,
                                              const float *__restrict__ charge, const int *__restrict__ type_row,
                                              int *__restrict__ perm, int *__restrict__ slot_of,
                                              float4 *__restrict__ xq, int *__restrict__ typ) {
    int n = g.n0 + blockIdx.y;
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Q) return;
    int c = cell[(size_t)n * g.Q + i];
    int col = c / g.dims[2];
    int base = col_start[(size_t)n * (g.ncol + 1) + col] + cell_rel[(size_t)n * g.ncell + c];
    int cnt = cell_count[(size_t)n * g.ncell + c];
    const int *t = tmp + (size_t)n * g.S + base;
    int rank = 0;
    for (int k = 0; k < cnt; k++) rank += (t[k] < i);
    int s = base + rank;
    MOP_ASSERT(base >= 0 && base + cnt <= g.S && rank < cnt);
    const float *r = R + ((size_t)n * g.Q + i) * 3;
    size_t o = (size_t)n * g.S + s;
    perm[o] = i;
    slot_of[(size_t)n * g.Q + i] = s;
    xq[o] = make_float4(mop_wrap1(r[0], g.box[0], g.inv_box[0]), mop_wrap1(r[1], g.box[1], g.inv_box[1]),
                        mop_wrap1(r[2], g.box[2], g.inv_box[2]), charge[i]);
    typ[o] = type_row[i];
}

// bounding box over the real atoms of every octet (8 slots); lo.w = number of real atoms (int bits)
__global__ void __launch_bounds__(128) k_bbox(MopGrid g, const int *__restrict__ perm, const float4 *__restrict__ xq,
                                              float4 *__restrict__ blo, float4 *__restrict__ bhi) {
    const int n = g.n0 + blockIdx.y;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;   // S is a multiple of 32: whole warps in range
    if (s >= g.S) return;
    const size_t o = (size_t)n * g.S + s;
    const bool real = perm[o] >= 0;
    const float4 p = xq[o];
    float lo[3], hi[3];
    const float BIG = 1.0e30f;
    lo[0] = real ? p.x : BIG, lo[1] = real ? p.y : BIG, lo[2] = real ? p.z : BIG;
    hi[0] = real ? p.x : -BIG, hi[1] = real ? p.y : -BIG, hi[2] = real ? p.z : -BIG;
    int cnt = real ? 1 : 0;
#pragma unroll
    for (int off = 1; off < MOP_CL; off <<= 1) {
#pragma unroll
        for (int d = 0; d < 3; d++) {
            lo[d] = fminf(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], off));
            hi[d] = fmaxf(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], off));
        }
        cnt += __shfl_xor_sync(0xffffffffu, cnt, off);
    }
    if ((s & (MOP_CL - 1)) == 0) {
        const size_t oc = (size_t)n * (g.S / MOP_CL) + s / MOP_CL;
        blo[oc] = make_float4(lo[0], lo[1], lo[2], __int_as_float(cnt));
        bhi[oc] = make_float4(hi[0], hi[1], hi[2], 0.0f);
    }
}

// ---- reuse of a buffered list (r_buf > 0): refresh the sorted coordinates in place -------------------------------
// Every atom keeps the slot and the periodic image it had when the list was built:
//   xq[slot] = wrap(R_ref) + (R - R_ref)      (never re-wrapped: the list's unit shifts stay valid)
// and the flag is raised when some atom has moved farther than r_buf / 2 from R_ref (the list then misses pairs and
// the caller rebuilds).  One thread per (bead, atom).
__global__ void __launch_bounds__(256) k_refresh(const float *__restrict__ R, const float *__restrict__ Rref, MopGrid g,
                                                 float half_buf2, const int *__restrict__ slot_of,
                                                 float4 *__restrict__ xq, int *__restrict__ flag) {
    const int n = g.n0 + blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.Q) return;
    const float *r = R + ((size_t)n * g.Q + i) * 3, *f = Rref + ((size_t)n * g.Q + i) * 3;
    const float dx = r[0] - f[0], dy = r[1] - f[1], dz = r[2] - f[2];
    if (!(dx * dx + dy * dy + dz * dz <= half_buf2)) *flag = 1;   // also catches NaN
    float4 *p = xq + (size_t)n * g.S + slot_of[(size_t)n * g.Q + i];
    p->x = mop_wrap1(f[0], g.box[0], g.inv_box[0]) + dx;
    p->y = mop_wrap1(f[1], g.box[1], g.inv_box[1]) + dy;
    p->z = mop_wrap1(f[2], g.box[2], g.inv_box[2]) + dz;
}
