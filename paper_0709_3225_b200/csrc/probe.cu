// md_probe_fp32_peak: the FP32 FMA rate of the current device, measured, so that bench.py can put a live number
// beside the "alu" roofline peak it derives from unit counts and clocks (SMs x 128 lanes x 2 flop x clocks.max.sm;
// SURVEY 8(d)).  Not part of the MD path: a calibration helper.
//
// Every thread runs PR_CHAINS independent chains of dependent FFMAs (a <- a * x + y) out of registers; with 2048
// resident threads per SM the FMA pipe never waits on a dependency, and nothing but FFMA and the loop branch is issued.
// The result is written only under a condition that never holds, which keeps the compiler from removing the chains
// without a single store in the timed kernel.
#include "common.cuh"

#define PR_T 256
#define PR_CHAINS 8
#define PR_UNROLL 16

static __device__ float g_probe_sink[PR_CHAINS];

__global__ void __launch_bounds__(PR_T)
k_probe_ffma(int iters, float x, float y)
{
    float a[PR_CHAINS];
#pragma unroll
    for (int k = 0; k < PR_CHAINS; k++) a[k] = (float)(threadIdx.x + k) * 1e-3f;
    for (int it = 0; it < iters; it++) {
#pragma unroll
        for (int u = 0; u < PR_UNROLL; u++) {
#pragma unroll
            for (int k = 0; k < PR_CHAINS; k++) a[k] = fmaf(a[k], x, y);
        }
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < PR_CHAINS; k++) s += a[k];
    if (s == 123456.789f) g_probe_sink[threadIdx.x % PR_CHAINS] = s;      // never true for the x, y passed below
}

extern "C" int md_probe_fp32_peak(double *tflops, double *ms, void *cuda_stream)
{
    if (!tflops) return MD_EINVAL;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int blocks = sms * (2048 / PR_T);
    const int iters = 4096;
    cudaEvent_t e0, e1;
    CK(cudaEventCreate(&e0));
    CK(cudaEventCreate(&e1));
    float best = 1e30f;
    int rc = MD_OK;
    for (int rep = 0; rep < 4 && rc == MD_OK; rep++) {                // the first launch warms up; best of the other three
        cudaEventRecord(e0, st);
        k_probe_ffma<<<blocks, PR_T, 0, st>>>(iters, 0.999f, 1e-3f);
        cudaEventRecord(e1, st);
        cudaError_t e = cudaGetLastError();
        if (e == cudaSuccess) e = cudaEventSynchronize(e1);
        float t = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&t, e0, e1);
        if (e != cudaSuccess) { ljmd_note_cuda_error(e, "md_probe_fp32_peak", __FILE__, __LINE__); rc = MD_ECUDA; }
        if (rep > 0 && t < best) best = t;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    if (rc) return rc;
    const double flop = 2.0 * (double)blocks * PR_T * PR_CHAINS * PR_UNROLL * (double)iters;
    *tflops = flop / ((double)best * 1e-3) / 1e12;
    if (ms) *ms = best;
    return MD_OK;
}
