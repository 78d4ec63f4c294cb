// pt_probe.cu -- measured ALU peaks of the device, reported by bench.py beside the derived roofline.  NOT part of libpt.so:
// built into its own library (libpt_probe.so, `build.build_probe()`), which only bench.py loads.
// kind 0 = dependent-free FFMA stream, kind 1 = MUFU.COS stream.
#include <cuda_runtime.h>
#include <stdint.h>

namespace pt {

constexpr int kProbeIters = 4096;
constexpr int kProbeIlp = 16;

__global__ void __launch_bounds__(512, 1) probe_ffma(float a, float b, float* out) {
    float v[kProbeIlp];
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) v[k] = (float)(threadIdx.x + k);
#pragma unroll 1
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int k = 0; k < kProbeIlp; ++k) v[k] = fmaf(v[k], a, b);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
}

__global__ void __launch_bounds__(512, 1) probe_mufu(float a, float* out) {
    float v[kProbeIlp];
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) v[k] = (float)(threadIdx.x + k) * a;
#pragma unroll 1
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int k = 0; k < kProbeIlp; ++k) v[k] = __cosf(v[k]);
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
}

}  // namespace pt

// Writes operations per second (fp32 lane-operations of the probed kind) to *ops_per_s [host].  Synchronous.
// Returns 0, or -1 for a bad argument, or -3 when a CUDA call failed.
extern "C" __attribute__((visibility("default"))) int32_t pt_bench_peak_probe(int32_t kind, double* ops_per_s) {
    using namespace pt;
    if (!ops_per_s || kind < 0 || kind > 1) return -1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    float* out = nullptr;
    if (cudaMalloc(&out, 4) != cudaSuccess) return -3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 4, thr = 512;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        if (kind == 0) probe_ffma<<<grid, thr>>>(1.0001f, 0.5f, out);
        else probe_mufu<<<grid, thr>>>(0.37f, out);
        cudaEventRecord(e1);
        if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); return -3; }
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (rep > 0 && ms < best_ms) best_ms = ms;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(out);
    const double ops = (double)grid * thr * (double)kProbeIters * kProbeIlp;
    *ops_per_s = ops / (best_ms * 1e-3);
    return 0;
}
