// mop_bonded.cuh -- S3 (harmonic bond/angle forces, energies on bead 1) and S6 (their Hessian-vector products),
// SURVEY.md 8a.  One thread per term per bead; coordinates are the caller's (never wrapped) with a minimum image
// on the difference; results are scattered into the sorted-order force / H.eta arrays with float atomics.
//   bond   u = k_b/2 (r-b0)^2 : g = u'/r = k_b (1 - b0/r), h = (u''-u'/r)/r^2 = k_b b0 / r^3, pair form as in pass 2
//   angle  u = k_t/2 (theta-theta0)^2, theta = acos(a^.b^), a = r_i-r_j, b = r_k-r_j:
//          dtheta/da = -(b^ - c a^)/(|a| sin), dtheta/db = -(a^ - c b^)/(|b| sin);
//          H.s by forward-mode differentiation of the gradient along (da, db) = (s_i-s_j, s_k-s_j).
#pragma once
#include "mop_common.cuh"

struct BondedArgs {
    int Q, S, n_bonds, n_angles;
    const float *R;          // [N][Q][3] caller coordinates
    const int *slot_of;      // [nf][Q]
    const int *bond_ij;      // [n_bonds][2]
    const float2 *bond_par;  // (b0, kb)
    const int *angle_ijk;    // [n_angles][3]
    const float2 *angle_par; // (theta0, kt)
    const float4 *et;        // [nf][S] direction (HVP)
    float4 *out;             // [nf][S] F4 or H4
    double *energies;        // [2] U_bond, [3] U_angle (bead 0 only)
    float box[3], inv_box[3];
};

__device__ __forceinline__ void mop_mi(const float *a, const float *b, const BondedArgs &A, float d[3]) {
#pragma unroll
    for (int q = 0; q < 3; q++) {
        float t = a[q] - b[q];
        d[q] = t - A.box[q] * rintf(t * A.inv_box[q]);
    }
}

__device__ __forceinline__ void mop_atomic_add3(float4 *p, float x, float y, float z) {
    float *f = reinterpret_cast<float *>(p);
    atomicAdd(f, x);
    atomicAdd(f + 1, y);
    atomicAdd(f + 2, z);
}

template <bool HVP>
__global__ void __launch_bounds__(128) k_bonded(const BondedArgs A) {
    const int n = blockIdx.y;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    const float *R = A.R + (size_t)n * A.Q * 3;
    const int *slot_of = A.slot_of + (size_t)n * A.Q;
    const float4 *et = A.et + (size_t)n * A.S;
    float4 *out = A.out + (size_t)n * A.S;
    double ub = 0.0, ua = 0.0;
    if (t < A.n_bonds) {
        const int i = A.bond_ij[2 * t], j = A.bond_ij[2 * t + 1];
        const float2 par = A.bond_par[t];
        float d[3];
        mop_mi(R + 3 * (size_t)i, R + 3 * (size_t)j, A, d);
        const float r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
        const float r = sqrtf(r2);
        const float g = par.y * (1.0f - par.x / r);
        const int si = slot_of[i], sj = slot_of[j];
        if (!HVP) {
            mop_atomic_add3(out + si, -g * d[0], -g * d[1], -g * d[2]);
            mop_atomic_add3(out + sj, g * d[0], g * d[1], g * d[2]);
            if (n == 0) ub = 0.5 * (double)par.y * (double)(r - par.x) * (double)(r - par.x);
        } else {
            const float h = par.y * par.x / (r2 * r);
            const float4 ei = et[si], ej = et[sj];
            const float e0 = ei.x - ej.x, e1 = ei.y - ej.y, e2 = ei.z - ej.z;
            const float hd = h * (d[0] * e0 + d[1] * e1 + d[2] * e2);
            const float o0 = hd * d[0] + g * e0, o1 = hd * d[1] + g * e1, o2 = hd * d[2] + g * e2;
            mop_atomic_add3(out + si, o0, o1, o2);
            mop_atomic_add3(out + sj, -o0, -o1, -o2);
        }
    } else if (t < A.n_bonds + A.n_angles) {
        const int ta = t - A.n_bonds;
        const int i = A.angle_ijk[3 * ta], j = A.angle_ijk[3 * ta + 1], k = A.angle_ijk[3 * ta + 2];
        const float2 par = A.angle_par[ta];
        float a[3], b[3];
        mop_mi(R + 3 * (size_t)i, R + 3 * (size_t)j, A, a);
        mop_mi(R + 3 * (size_t)k, R + 3 * (size_t)j, A, b);
        const float la = sqrtf(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
        const float lb = sqrtf(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
        const float ila = 1.0f / la, ilb = 1.0f / lb;
        float ah[3], bh[3];
#pragma unroll
        for (int q = 0; q < 3; q++) ah[q] = a[q] * ila, bh[q] = b[q] * ilb;
        float c = ah[0] * bh[0] + ah[1] * bh[1] + ah[2] * bh[2];
        c = fminf(1.0f, fmaxf(-1.0f, c));
        const float th = acosf(c);
        const float sg = sqrtf(fmaxf(1.0f - c * c, 1.0e-12f));
        const float pref = par.y * (th - par.x);
        const float ias = 1.0f / (la * sg), ibs = 1.0f / (lb * sg);
        float p[3], qv[3], ga[3], gb[3];
#pragma unroll
        for (int q = 0; q < 3; q++) {
            p[q] = bh[q] - c * ah[q];
            qv[q] = ah[q] - c * bh[q];
            ga[q] = -p[q] * ias;
            gb[q] = -qv[q] * ibs;
        }
        const int si = slot_of[i], sj = slot_of[j], sk = slot_of[k];
        if (!HVP) {
            float fi[3], fk[3];
#pragma unroll
            for (int q = 0; q < 3; q++) fi[q] = -pref * ga[q], fk[q] = -pref * gb[q];
            mop_atomic_add3(out + si, fi[0], fi[1], fi[2]);
            mop_atomic_add3(out + sk, fk[0], fk[1], fk[2]);
            mop_atomic_add3(out + sj, -(fi[0] + fk[0]), -(fi[1] + fk[1]), -(fi[2] + fk[2]));
            if (n == 0) ua = 0.5 * (double)par.y * (double)(th - par.x) * (double)(th - par.x);
        } else {
            const float4 ei = et[si], ej = et[sj], ek = et[sk];
            const float da[3] = {ei.x - ej.x, ei.y - ej.y, ei.z - ej.z};
            const float db[3] = {ek.x - ej.x, ek.y - ej.y, ek.z - ej.z};
            float dth = 0.f, dla = 0.f, dlb = 0.f;
#pragma unroll
            for (int q = 0; q < 3; q++) {
                dth += ga[q] * da[q] + gb[q] * db[q];
                dla += ah[q] * da[q];
                dlb += bh[q] * db[q];
            }
            float dah[3], dbh[3];
            float dc = 0.f;
#pragma unroll
            for (int q = 0; q < 3; q++) {
                dah[q] = (da[q] - ah[q] * dla) * ila;
                dbh[q] = (db[q] - bh[q] * dlb) * ilb;
                dc += dah[q] * bh[q] + ah[q] * dbh[q];
            }
            const float dsg = -c * dc / sg;
            const float wa = (dla * sg + la * dsg) * ias * ias; // d(|a| sin)/(|a| sin)^2
            const float wb = (dlb * sg + lb * dsg) * ibs * ibs;
            float hi[3], hk[3];
#pragma unroll
            for (int q = 0; q < 3; q++) {
                const float dp = dbh[q] - dc * ah[q] - c * dah[q];
                const float dq = dah[q] - dc * bh[q] - c * dbh[q];
                const float dga = -dp * ias + p[q] * wa;
                const float dgb = -dq * ibs + qv[q] * wb;
                hi[q] = par.y * dth * ga[q] + pref * dga;
                hk[q] = par.y * dth * gb[q] + pref * dgb;
            }
            mop_atomic_add3(out + si, hi[0], hi[1], hi[2]);
            mop_atomic_add3(out + sk, hk[0], hk[1], hk[2]);
            mop_atomic_add3(out + sj, -(hi[0] + hk[0]), -(hi[1] + hk[1]), -(hi[2] + hk[2]));
        }
    }
    if (!HVP && n == 0) { // energies of bead 1: warp reduce, one double atomic per warp
        ub = mop_warp_sum_d(ub);
        ua = mop_warp_sum_d(ua);
        if ((threadIdx.x & 31) == 0) {
            if (ub != 0.0) atomicAdd(&A.energies[2], ub);
            if (ua != 0.0) atomicAdd(&A.energies[3], ua);
        }
    }
}
