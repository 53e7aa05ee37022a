// mop_path.cuh -- S4 (displacements eta^n and spring energy: the paper's PMD kernels 1 and 7),
// S7 (gradient assembly: PMD kernels 4-6, eqs (5),(6),(7)) and S8 (velocity Verlet on
// eq. (4)).  Elementwise, HBM-bound.
#pragma once
#include "mop_common.cuh"

// eta^n_i = (R^{n+1}_i - R^n_i) - a_i F^n_i,  a_i = dt/(m_i nu)  (L^n = a F^n, reading G1)
// E_spring += K_i/2 |eta^n_i|^2, K_i = m_i nu/(2 dt), accumulated in FP64.  One thread per sorted slot.
// R_next: bead-block mode only -- the bead after the block (the right neighbour's first bead, [Q][3]) for the block's
// last bead n_local - 1; otherwise bead n + 1 is read from R itself
__global__ void __launch_bounds__(256) k_eta(int Q, int S, int n_local, const float *__restrict__ R,
                                             const float *__restrict__ R_next,
                                             const int *__restrict__ perm, const int *__restrict__ typ,
                                             const float4 *__restrict__ F4, const float *__restrict__ a_i,
                                             const float *__restrict__ K_i, float4 *__restrict__ et,
                                             double *__restrict__ e_spring) {
    const int n = blockIdx.y;
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    double e = 0.0;
    if (s < S) {
        const size_t o = (size_t)n * S + s;
        const int i = perm[o];
        float4 out = make_float4(0.f, 0.f, 0.f, __int_as_float(typ[o]));
        if (i >= 0) {
            const float *r0 = R + ((size_t)n * Q + i) * 3;
            const float *r1 = n + 1 < n_local ? r0 + (size_t)Q * 3 : R_next + (size_t)i * 3;
            const float4 f = F4[o];
            const float a = a_i[i];
            out.x = __fmaf_rn(-a, f.x, r1[0] - r0[0]);
            out.y = __fmaf_rn(-a, f.y, r1[1] - r0[1]);
            out.z = __fmaf_rn(-a, f.z, r1[2] - r0[2]);
            e = 0.5 * (double)K_i[i] *
                ((double)out.x * (double)out.x + (double)out.y * (double)out.y + (double)out.z * (double)out.z);
        }
        et[o] = out;
    }
    __shared__ double sh[8];
    e = mop_warp_sum_d(e);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x < 32) {
        double v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
        v = mop_warp_sum_d(v);
        if (threadIdx.x == 0 && v != 0.0) atomicAdd(e_spring, v);
    }
}

// dV_eff/dR^n_i (= -F_eff of eqs 5,6,7 with the bracket at its eps->0 limit -1/2 H eta):
//   n = 1     : -F^1 - K eta^1 + 1/2 H^1 eta^1          (N = 1: -F^1)
//   1 < n < N : K eta^{n-1} - K eta^n + 1/2 H^n eta^n
//   n = N     : K eta^{N-1}
// over the N_local beads of the context: has_u1 = its first bead is bead 1 of the path, nh = beads that have eta and
// H.eta (all but the path's last bead), keta_left = K eta of the bead before the block ([Q][3], original order; the left
// neighbour's halo in bead-block mode) or NULL
// (n_first: first bead of this launch; the host entry point assembles and copies out the beads in two groups)
__global__ void __launch_bounds__(256) k_assemble(int Q, int S, int n_first, int N_local, int nh, int has_u1,
                                                  const int *__restrict__ slot_of,
                                                  const float4 *__restrict__ F4, const float4 *__restrict__ et,
                                                  const float4 *__restrict__ H4, const float *__restrict__ K_i,
                                                  const float *__restrict__ keta_left, float *__restrict__ grad) {
    const int n = n_first + blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Q) return;
    float gx = 0.f, gy = 0.f, gz = 0.f;
    const float K = K_i[i];
    if (n == 0 && has_u1) {
        const float4 f = F4[slot_of[i]];
        gx -= f.x, gy -= f.y, gz -= f.z;
    }
    if (n > 0) {
        const float4 e = et[(size_t)(n - 1) * S + slot_of[(size_t)(n - 1) * Q + i]];
        gx = fmaf(K, e.x, gx), gy = fmaf(K, e.y, gy), gz = fmaf(K, e.z, gz);
    } else if (keta_left) {
        gx += keta_left[3 * (size_t)i], gy += keta_left[3 * (size_t)i + 1], gz += keta_left[3 * (size_t)i + 2];
    }
    if (n < nh) {
        const size_t o = (size_t)n * S + slot_of[(size_t)n * Q + i];
        const float4 e = et[o], h = H4[o];
        gx += fmaf(-K, e.x, 0.5f * h.x), gy += fmaf(-K, e.y, 0.5f * h.y), gz += fmaf(-K, e.z, 0.5f * h.z);
    }
    float *g = grad + ((size_t)n * Q + i) * 3;
    g[0] = gx, g[1] = gy, g[2] = gz;
}

// bead-block mode: K eta of local bead n in original atom order, the halo the right neighbour's assembly needs
__global__ void __launch_bounds__(256) k_keta_out(int Q, int S, int n, const int *__restrict__ slot_of,
                                                  const float4 *__restrict__ et, const float *__restrict__ K_i,
                                                  float *__restrict__ out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Q) return;
    const float4 e = et[(size_t)n * S + slot_of[(size_t)n * Q + i]];
    const float K = K_i[i];
    out[3 * (size_t)i] = K * e.x, out[3 * (size_t)i + 1] = K * e.y, out[3 * (size_t)i + 2] = K * e.z;
}

// sorted float4 array -> original-order [nf][Q][3]
__global__ void __launch_bounds__(256) k_gather3(int Q, int S, const int *__restrict__ slot_of,
                                                 const float4 *__restrict__ src, float *__restrict__ dst,
                                                 float scale) {
    const int n = blockIdx.y;
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= Q) return;
    const float4 v = src[(size_t)n * S + slot_of[(size_t)n * Q + i]];
    float *d = dst + ((size_t)n * Q + i) * 3;
    d[0] = scale * v.x, d[1] = scale * v.y, d[2] = scale * v.z;
}

// user direction s [Q][3] -> et of bead slot 0 (mop_force_hvp)
__global__ void __launch_bounds__(256) k_set_dir(int S, const int *__restrict__ perm, const int *__restrict__ typ,
                                                 const float *__restrict__ sdir, float4 *__restrict__ et) {
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= S) return;
    const int i = perm[s];
    float4 out = make_float4(0.f, 0.f, 0.f, __int_as_float(typ[s]));
    if (i >= 0) out.x = sdir[3 * (size_t)i], out.y = sdir[3 * (size_t)i + 1], out.z = sdir[3 * (size_t)i + 2];
    et[s] = out;
}

// velocity Verlet: mode 0  v += (dt/2)(-G)/m ; R += dt v      mode 1  v += (dt/2)(-G)/m (+ kinetic energy)
__global__ void __launch_bounds__(256) k_verlet(size_t total, int Q, float dt, int mode, const float *__restrict__ inv_m,
                                                const float *__restrict__ m, const float *__restrict__ G,
                                                float *__restrict__ R, float *__restrict__ V,
                                                double *__restrict__ e_kin) {
    const size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    double ek = 0.0;
    if (o < total) {
        const int i = (int)((o / 3) % (size_t)Q);
        float v = V[o];
        v = fmaf(-0.5f * dt * inv_m[i], G[o], v);
        V[o] = v;
        if (mode == 0) R[o] = fmaf(dt, v, R[o]);
        else if (e_kin) ek = 0.5 * (double)m[i] * (double)v * (double)v;
    }
    if (mode == 1 && e_kin) {
        __shared__ double sh[8];
        ek = mop_warp_sum_d(ek);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = ek;
        __syncthreads();
        if (threadIdx.x < 32) {
            double v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
            v = mop_warp_sum_d(v);
            if (threadIdx.x == 0) atomicAdd(e_kin, v);
        }
    }
}

// ---- the paper's finite-difference form of the Hessian term (NEXT-1) ----
// paper kernel 2: displaced coordinates R^n +- eps eta^n (original atom order, eta in original order)
__global__ void __launch_bounds__(256) k_displace(size_t total, float eps, const float *__restrict__ R,
                                                  const float *__restrict__ eta, float *__restrict__ Rd) {
    const size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (o < total) Rd[o] = __fmaf_rn(eps, eta[o], R[o]);
}

// paper kernels 3-6 in gradient form, original atom order:
//   dV_eff/dR^n = [n = 1: -F^1] + K eta^{n-1} - K eta^n - [F(R^n + eps eta^n) - F(R^n - eps eta^n)] / (4 eps)
// (eqs (5),(6),(7) with K a_i = 1/2; the bracket replaces -1/2 H^n eta^n)
__global__ void __launch_bounds__(256) k_assemble_fd(int Q, int N, float inv4eps, const float *__restrict__ F,
                                                     const float *__restrict__ eta, const float *__restrict__ Fp,
                                                     const float *__restrict__ Fm, const float *__restrict__ K_i,
                                                     float *__restrict__ grad) {
    const int n = blockIdx.y;
    const size_t t = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= (size_t)Q * 3) return;
    const float K = K_i[t / 3];
    const size_t o = (size_t)n * Q * 3 + t;
    float g = 0.f;
    if (n == 0) g -= F[t];
    if (n > 0) g = fmaf(K, eta[o - (size_t)Q * 3], g);
    if (n < N - 1) g += fmaf(-K, eta[o], -inv4eps * (Fp[o] - Fm[o]));
    grad[o] = g;
}

// ---- Langevin thermostat of the NVT runs (NEXT-2; reading G19 of DESIGN.md) ----
// Counter-based noise: 64 bits from (seed, step, index of the coordinate in [N][Q][3]) by two SplitMix64
// finalisers, two 32-bit uniforms, Box-Muller.  The integer part is bit-identical to the oracle's generator
// (written independently there); the transcendental part is FP32 here and FP64 there.
__device__ __forceinline__ unsigned long long mop_mix64(unsigned long long z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ULL;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBULL;
    return z ^ (z >> 31);
}
__device__ __forceinline__ unsigned long long mop_noise_bits(unsigned long long seed, unsigned long long step,
                                                             unsigned long long idx) {
    return mop_mix64(mop_mix64(seed + 0x9E3779B97F4A7C15ULL * (step + 1ULL)) ^ (idx * 0xD1342543DE82EF95ULL + 1ULL));
}
__device__ __forceinline__ float mop_noise_normal(unsigned long long seed, unsigned long long step, unsigned long long idx) {
    const unsigned long long b = mop_noise_bits(seed, step, idx);
    const double u1 = ((double)(unsigned)(b >> 32) + 0.5) * (1.0 / 4294967296.0);   // exact in FP64, in (0,1)
    const float u2 = (float)(((double)(unsigned)b + 0.5) * (1.0 / 4294967296.0));
    return sqrtf(-2.0f * (float)log(u1)) * cospif(2.0f * u2);
}

// exact Ornstein-Uhlenbeck velocity update over dt: v <- c v + sqrt((1 - c^2) kT / m) xi  (+ kinetic energy)
// idx0: index of V[0] in the whole path's [N][Q][3] array (0 unless V is a bead block of a longer path: the generator is
// keyed by the coordinate's place in the WHOLE path, so a sharded run draws the numbers the unsharded one does)
__global__ void __launch_bounds__(256) k_ou(size_t total, int Q, float c, float amp, unsigned long long seed,
                                            unsigned long long step, unsigned long long idx0, const float *__restrict__ inv_m,
                                            const float *__restrict__ m, float *__restrict__ V,
                                            double *__restrict__ e_kin) {
    const size_t o = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    double ek = 0.0;
    if (o < total) {
        const int i = (int)((o / 3) % (size_t)Q);
        const float v = fmaf(c, V[o], amp * sqrtf(inv_m[i]) * mop_noise_normal(seed, step, idx0 + o));
        V[o] = v;
        if (e_kin) ek = 0.5 * (double)m[i] * (double)v * (double)v;
    }
    if (e_kin) {
        __shared__ double sh[8];
        ek = mop_warp_sum_d(ek);
        if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = ek;
        __syncthreads();
        if (threadIdx.x < 32) {
            double v = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
            v = mop_warp_sum_d(v);
            if (threadIdx.x == 0) atomicAdd(e_kin, v);
        }
    }
}

// debug: the generator's raw bits for idx = 0..n-1 (bit-exact comparison with the oracle)
__global__ void k_noise_bits(int n, unsigned long long seed, unsigned long long step, unsigned long long *out) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = mop_noise_bits(seed, step, (unsigned long long)i);
}
