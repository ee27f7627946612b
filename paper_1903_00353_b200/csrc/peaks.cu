// peaks.cu -- measurement support (BASELINE.json north_star: "the slower of the grid plus
// feature bytes at HBM peak and the candidate cell x feature distance evaluations at FP32 peak"): the FP32
// leg of the roofline needs a measured FP32 peak, and MEASURED_PEAKS.json (driver-written) holds none.
// sdf_measure_fp32_peak runs a register-resident FMA loop on every SM and reports the rate.
#include "common.cuh"

#define PK_BT 512
#define PK_CHAINS 16          // independent FMA chains per thread: hides the 4-cycle FMA latency at any occupancy
#define PK_ITERS 4096

__global__ void __launch_bounds__(PK_BT) fp32_fma_peak_kernel(float *__restrict__ sink, float a, float b) {
    float x[PK_CHAINS];
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) x[c] = (float)(threadIdx.x + c) * 1e-3f;
#pragma unroll 8
    for (int it = 0; it < PK_ITERS; it++) {
#pragma unroll
        for (int c = 0; c < PK_CHAINS; c++) x[c] = __fmaf_rn(x[c], a, b);
    }
    float s = 0.0f;
#pragma unroll
    for (int c = 0; c < PK_CHAINS; c++) s += x[c];
    if (s == 123.456f) sink[blockIdx.x * PK_BT + threadIdx.x] = s;      // never true: keeps the loop alive
}

extern "C" int sdf_measure_fp32_peak(double *tflops_out, int *sm_count_out, void *stream) {
    if (!tflops_out) return SDF_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    if (sm_count_out) *sm_count_out = sms;
    const int blocks = sms * 4 * 8;           // 4 resident blocks per SM (2048 threads), 8 waves
    float *sink = nullptr;
    CK(cudaMallocAsync((void **)&sink, sizeof(float) * (size_t)blocks * PK_BT, st));
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    double best = 0.0;
    for (int rep = 0; rep < 6; rep++) {       // first repetitions warm the clocks up; the best one counts
        CK(cudaEventRecord(e0, st));
        KL; fp32_fma_peak_kernel<<<blocks, PK_BT, 0, st>>>(sink, 0.999f, 1e-3f);
        CK(cudaEventRecord(e1, st));
        CK(cudaEventSynchronize(e1));
        float ms = 0.0f;
        CK(cudaEventElapsedTime(&ms, e0, e1));
        const double flop = 2.0 * (double)blocks * PK_BT * PK_CHAINS * PK_ITERS;
        const double tf = flop / ((double)ms * 1e-3) / 1e12;
        if (tf > best) best = tf;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    CK(cudaFreeAsync(sink, st));
    CK(cudaGetLastError());
    *tflops_out = best;
    return SDF_OK;
}
