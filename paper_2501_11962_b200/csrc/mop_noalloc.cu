// mop_noalloc.cu -- mop_eta_spring_noalloc (include/mop.h): the paper's PMD kernels 1 and 7 (
// stage S4 of the hot path) as ONE stateless call that never allocates.
//
// Who this is for.  Some programs that want eta^n and the spring energy are not in a position to let a library call
// cudaMalloc on their behalf: an MD engine or plug-in host that hands out every byte of device memory from its own
// pool at start-up and treats any later driver allocation as an error; a process whose other framework has already
// reserved (nearly) all of HBM, so that a late cudaMalloc fails or stalls; a latency-critical stepping loop, where
// cudaMalloc / cudaFree are off limits because they synchronise the whole device.  mop_create and the context-based
// calls allocate, so such callers cannot use them.  This entry point takes caller-owned inputs and outputs only and
// keeps the one piece of working memory it needs -- one FP64 partial sum per thread block plus a ticket counter -- in
// a fixed array that is part of the library image (g_scratch below).  It calls no cudaMalloc, cudaMallocHost, cudaFree
// or any library routine that allocates.
//
// What that costs.  The array has a fixed size (MOP_NOALLOC_SCRATCH_BYTES, about 1 MiB), and every GPU on which this
// process uses the library holds it until the process exits.  Its size bounds the problem: at most
// MOP_NOALLOC_MAX_ATOM_BEADS = 33,554,432 (atom, bead) pairs per call, larger calls are refused.  There is ONE array
// per device, shared by every call from every thread and stream: two calls that are in flight on the same GPU at the
// same time race on it (wrong energy, or a lost ticket).  Put such calls on one stream, or order them with events.
//
// First call on a device.  In host code the name `g_scratch` is only a handle for the device array, not its address;
// the first call on each device looks the address up (cudaGetSymbolAddress, with that device current) and caches it.
// Make that first call outside any stream capture.
#include "../../include/mop.h"

#include <cstdio>
#include <mutex>

#define NA_THREADS 256
#define NA_MAX_BLOCKS (MOP_NOALLOC_MAX_ATOM_BEADS / NA_THREADS)   // 131,072 partial sums
#define NA_HEADER_BYTES 256                                        // ticket counter, alone in its 256-byte line
#define NA_MAX_DEVICES 64

static_assert(MOP_NOALLOC_MAX_ATOM_BEADS % NA_THREADS == 0, "whole thread blocks");
static_assert(MOP_NOALLOC_SCRATCH_BYTES == NA_HEADER_BYTES + NA_MAX_BLOCKS * 8, "mop.h states the size of the array");

// The working memory: [0, 4) ticket counter (must be 0 when a call starts), [256, 256 + 8 * blocks) FP64 partials.
// Device code may name it directly; host code must go through scratch_of().
static __device__ __align__(256) unsigned char g_scratch[MOP_NOALLOC_SCRATCH_BYTES];

// eta^n_i = (R^{n+1}_i - R^n_i) - a_i F^n_i with a_i = dt/(m_i nu) (L^n = a F^n: reading G1 of DESIGN.md), and
// E_spring = sum_{n,i} K_i/2 |eta^n_i|^2 with K_i = m_i nu/(2 dt), in FP64.  Same arithmetic, operation
// for operation, as k_eta + mop_set_topology of the context path, but in the caller's atom order, with a_i and K_i
// formed on the fly from the masses, and with a two-level sum in a fixed order (block partials in the scratch array,
// added up by whichever block finishes last) instead of atomics on one double: E_spring is bit-reproducible.
__global__ void __launch_bounds__(NA_THREADS) k_eta_spring_noalloc(int Q, int total, double dt, double nu,
                                                                   const float *__restrict__ R,
                                                                   const float *__restrict__ F,
                                                                   const float *__restrict__ mass,
                                                                   float *__restrict__ eta, unsigned char *scratch,
                                                                   double *__restrict__ e_out) {
    unsigned *ticket = reinterpret_cast<unsigned *>(scratch);
    double *partial = reinterpret_cast<double *>(scratch + NA_HEADER_BYTES);
    const int t = blockIdx.x * NA_THREADS + threadIdx.x;   // (bead n, atom i) = (t / Q, t % Q)
    double e = 0.0;
    if (t < total) {
        const int i = t % Q;
        const double m = (double)mass[i];
        const float a = (float)(dt / (m * nu));
        const float K = (float)(m * nu / (2.0 * dt));
        const size_t o = (size_t)t * 3;
        const float *r0 = R + o, *r1 = r0 + (size_t)Q * 3, *f = F + o;
        const float ex = __fmaf_rn(-a, f[0], r1[0] - r0[0]);
        const float ey = __fmaf_rn(-a, f[1], r1[1] - r0[1]);
        const float ez = __fmaf_rn(-a, f[2], r1[2] - r0[2]);
        eta[o] = ex, eta[o + 1] = ey, eta[o + 2] = ez;
        e = 0.5 * (double)K * ((double)ex * (double)ex + (double)ey * (double)ey + (double)ez * (double)ez);
    }
    // block sum in a fixed order: shuffle tree per warp, then the 8 warp sums one after the other
    __shared__ double sh[NA_THREADS / 32];
    __shared__ bool is_last;
    for (int d = 16; d > 0; d >>= 1) e += __shfl_down_sync(0xffffffffu, e, d);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = e;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int w = 0; w < NA_THREADS / 32; w++) v += sh[w];
        partial[blockIdx.x] = v;
        __threadfence();                                   // the partial is visible before the ticket is taken
        is_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!is_last) return;
    // the last block to finish adds up all partials: thread k takes k, k + 256, ... in order, then the same tree
    __threadfence();
    double s = 0.0;
    for (unsigned k = threadIdx.x; k < gridDim.x; k += NA_THREADS) s += __ldcg(partial + k);
    for (int d = 16; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    __syncthreads();                                       // sh is reused
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double v = 0.0;
        for (int w = 0; w < NA_THREADS / 32; w++) v += sh[w];
        *e_out = v;
        *ticket = 0u;                                      // leave the counter clean as well (the host clears it anyway)
    }
}

// Device address of g_scratch on `device`, looked up once per device with that device current.
static cudaError_t scratch_of(int device, unsigned char **out) {
    static std::mutex mu;
    static unsigned char *addr[NA_MAX_DEVICES] = {nullptr};
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        unsigned char *p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void **)&p, g_scratch);   // current device = `device` (set by the caller)
        if (e != cudaSuccess) return e;
        addr[device] = p;
    }
    *out = addr[device];
    return cudaSuccess;
}

static mop_status na_fail(char *err, size_t err_len, mop_status code, const char *msg, const char *detail = nullptr) {
    if (err && err_len) snprintf(err, err_len, "mop_eta_spring_noalloc: %s%s%s", msg, detail ? ": " : "", detail ? detail : "");
    return code;
}

extern "C" mop_status mop_eta_spring_noalloc(int device, void *stream, int n_atoms, int n_beads, double dt_path, double nu,
                                             const float *R_dev, const float *F_dev, const float *mass_dev,
                                             float *eta_dev, double *e_spring_dev, char *err, size_t err_len) {
    if (err && err_len) err[0] = 0;
    if (n_atoms < 1 || n_beads < 2) return na_fail(err, err_len, MOP_ERR_INVALID_ARG, "need n_atoms >= 1 and n_beads >= 2");
    if (!(dt_path > 0.0) || !(nu > 0.0)) return na_fail(err, err_len, MOP_ERR_INVALID_ARG, "dt_path and nu must be > 0");
    if (!R_dev || !F_dev || !mass_dev || !eta_dev || !e_spring_dev)
        return na_fail(err, err_len, MOP_ERR_INVALID_ARG, "NULL device pointer");
    if (device < 0 || device >= NA_MAX_DEVICES) return na_fail(err, err_len, MOP_ERR_INVALID_ARG, "device ordinal out of range");
    const long long total = (long long)n_atoms * (long long)(n_beads - 1);
    if (total > (long long)MOP_NOALLOC_MAX_ATOM_BEADS) {
        char b[320];
        snprintf(b, sizeof b, "n_atoms * (n_beads - 1) = %lld exceeds MOP_NOALLOC_MAX_ATOM_BEADS = %d (the fixed scratch array "
                 "holds one partial sum per 256 of them); split the path into shorter bead ranges", total,
                 (int)MOP_NOALLOC_MAX_ATOM_BEADS);
        return na_fail(err, err_len, MOP_ERR_INVALID_ARG, b);
    }
    int prev = -1;
    cudaError_t e = cudaGetDevice(&prev);
    if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
    if (e != cudaSuccess) return na_fail(err, err_len, MOP_ERR_CUDA, "cannot select the device (no CPU fallback)", cudaGetErrorString(e));
    unsigned char *scratch = nullptr;
    mop_status rc = MOP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    if ((e = scratch_of(device, &scratch)) != cudaSuccess) {
        rc = na_fail(err, err_len, MOP_ERR_CUDA, "cudaGetSymbolAddress", cudaGetErrorString(e));
    } else if ((e = cudaMemsetAsync(scratch, 0, NA_HEADER_BYTES, st)) != cudaSuccess) {
        // the array keeps whatever the last call left (or an aborted one): the ticket counter must start at zero; the
        // partials need no clearing, every slot that is read has been written by this launch
        rc = na_fail(err, err_len, MOP_ERR_CUDA, "cudaMemsetAsync", cudaGetErrorString(e));
    } else {
        const unsigned blocks = (unsigned)((total + NA_THREADS - 1) / NA_THREADS);
        k_eta_spring_noalloc<<<blocks, NA_THREADS, 0, st>>>(n_atoms, (int)total, dt_path, nu, R_dev, F_dev, mass_dev, eta_dev,
                                                            scratch, e_spring_dev);
        if ((e = cudaGetLastError()) != cudaSuccess) rc = na_fail(err, err_len, MOP_ERR_CUDA, "kernel launch", cudaGetErrorString(e));
    }
    if (prev >= 0 && prev != device) cudaSetDevice(prev);
    return rc;
}
