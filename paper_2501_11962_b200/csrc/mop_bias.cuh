// mop_bias.cuh -- the metadynamics-of-paths bias.
//   CV   S_e2e = s(R^N) - s(R^1)  (eq. 8);  s(R) = distance between the centres of mass of two atom groups
//   V(S) = sum_k w exp(-(S - S_k)^2 / (2 sigma^2)),  dV/dR^N = V'(S) ds/dR^N,  dV/dR^1 = -V'(S) ds/dR^1
// Touches beads 1 and N only.  Three tiny launches per evaluation (COM reductions in FP64, CV + hills, force).
#pragma once
#include "mop_common.cuh"

#define MOP_MAX_HILLS 65536

struct BiasArgs {
    int Q, N, na, nb;
    const int *ga, *gb;     // atom indices of the two groups
    const float *mass;
    float box[3];
    double sigma, w;
    double *hills;          // [MOP_MAX_HILLS] centres S_k
    int *n_hills;
    double *com;            // [2 beads][2 groups][4]: sum m x, sum m y, sum m z, sum m
    double *state;          // [0] S [1] s(R^1) [2] s(R^N) [3] V [4] dV/dS [5..7] unit vector bead 1 [8..10] bead N
};

// block (group g = blockIdx.x, end bead e = blockIdx.y): mass-weighted coordinate sums in FP64
__global__ void __launch_bounds__(256) k_bias_com(BiasArgs a, const float *__restrict__ R) {
    const int g = blockIdx.x, e = blockIdx.y;
    const int *idx = g ? a.gb : a.ga;
    const int n = g ? a.nb : a.na;
    const float *X = R + (size_t)(e ? a.N - 1 : 0) * a.Q * 3;
    double s[4] = {0.0, 0.0, 0.0, 0.0};
    for (int k = threadIdx.x; k < n; k += blockDim.x) {
        const int i = idx[k];
        const double m = (double)a.mass[i];
        s[0] += m * (double)X[3 * (size_t)i], s[1] += m * (double)X[3 * (size_t)i + 1], s[2] += m * (double)X[3 * (size_t)i + 2];
        s[3] += m;
    }
    __shared__ double sh[8][4];
#pragma unroll
    for (int q = 0; q < 4; q++) s[q] = mop_warp_sum_d(s[q]);
    if ((threadIdx.x & 31) == 0)
        for (int q = 0; q < 4; q++) sh[threadIdx.x >> 5][q] = s[q];
    __syncthreads();
    if (threadIdx.x < 4) {
        double t = 0.0;
        for (int w = 0; w < (int)(blockDim.x >> 5); w++) t += sh[w][threadIdx.x];
        a.com[(e * 2 + g) * 4 + threadIdx.x] = t;
    }
}

// one warp: the two COM distances (minimum image), S, optional hill deposition at S, then V and dV/dS over the hills
__global__ void __launch_bounds__(32) k_bias_cv(BiasArgs a, int deposit) {
    const int lane = threadIdx.x;
    double sv[2], u[2][3];
    for (int e = 0; e < 2; e++) {
        double r2 = 0.0;
        for (int q = 0; q < 3; q++) {
            const double L = (double)a.box[q];
            double d = a.com[(e * 2 + 0) * 4 + q] / a.com[(e * 2 + 0) * 4 + 3] - a.com[(e * 2 + 1) * 4 + q] / a.com[(e * 2 + 1) * 4 + 3];
            d -= L * floor(d / L + 0.5);
            u[e][q] = d;
            r2 += d * d;
        }
        sv[e] = sqrt(r2);
        for (int q = 0; q < 3; q++) u[e][q] = sv[e] > 0.0 ? u[e][q] / sv[e] : 0.0;
    }
    const double S = sv[1] - sv[0];
    int nh = *a.n_hills;
    if (deposit && nh < MOP_MAX_HILLS) {
        if (lane == 0) a.hills[nh] = S, *a.n_hills = nh + 1;
        nh += 1;
    }
    __syncwarp();
    double V = 0.0, dV = 0.0;
    for (int k = lane; k < nh; k += 32) {
        const double t = (S - a.hills[k]) / a.sigma, ex = a.w * exp(-0.5 * t * t);
        V += ex;
        dV += -ex * t / a.sigma;
    }
    V = mop_warp_sum_d(V), dV = mop_warp_sum_d(dV);
    if (lane == 0) {
        a.state[0] = S, a.state[1] = sv[0], a.state[2] = sv[1], a.state[3] = V, a.state[4] = dV;
        for (int q = 0; q < 3; q++) a.state[5 + q] = u[0][q], a.state[8 + q] = u[1][q];
    }
}

// grad[bead][i] += (+/-) V'(S) (m_i / M_group) u   for the group atoms of beads 1 (sign -) and N (sign +)
__global__ void __launch_bounds__(256) k_bias_apply(BiasArgs a, float *__restrict__ grad) {
    const int e = blockIdx.y;
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= a.na + a.nb) return;
    const int g = t >= a.na;
    const int i = g ? a.gb[t - a.na] : a.ga[t];
    const double f = (e ? 1.0 : -1.0) * (g ? -1.0 : 1.0) * a.state[4] * (double)a.mass[i] / a.com[(e * 2 + g) * 4 + 3];
    float *gp = grad + ((size_t)(e ? a.N - 1 : 0) * a.Q + i) * 3;
    for (int q = 0; q < 3; q++) atomicAdd(gp + q, (float)(f * a.state[5 + 3 * e + q]));
}
