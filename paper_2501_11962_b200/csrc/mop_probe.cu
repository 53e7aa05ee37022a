// mop_probe.cu -- FP32-pipe probe (measurement aid for bench.py; its own small library, libmop_probe.so, not part of
// the product library).  TFLOP/s of dependent-free FMA streams of three operand shapes, FMA = 2 flop.
#include <cuda_runtime.h>

#include "mop_probe.cuh"

extern "C" int mop_probe_fp32(int device, double out[4]) {
    if (!out) return 1;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev || cudaSetDevice(device) != cudaSuccess) {
        cudaGetLastError();
        return 5;
    }
    int sms = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    const int grid = sms * 4, block = 256;
    float *buf = nullptr;
    if (cudaMalloc((void **)&buf, (size_t)grid * block * sizeof(float)) != cudaSuccess) return 4;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0), cudaEventCreate(&e1);
    void (*ks[3])(float *, float) = {k_probe_fp32<0>, k_probe_fp32<1>, k_probe_fp32<2>};
    const double fma_per_thread[3] = {8.0 * MOP_PROBE_ITER, 8.0 * MOP_PROBE_ITER, 16.0 * MOP_PROBE_ITER};
    for (int m = 0; m < 3; m++) {
        float best = 1e30f;
        for (int rep = 0; rep < 4; rep++) {
            cudaEventRecord(e0);
            ks[m]<<<grid, block>>>(buf, 1.0001f);
            cudaEventRecord(e1);
            cudaEventSynchronize(e1);
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (rep > 0 && ms < best) best = ms;
        }
        out[m] = 2.0 * fma_per_thread[m] * (double)grid * block / (best * 1e-3) / 1e12;
    }
    out[3] = (double)sms;
    cudaEventDestroy(e0), cudaEventDestroy(e1);
    cudaFree(buf);
    return cudaGetLastError() == cudaSuccess ? 0 : 5;
}
