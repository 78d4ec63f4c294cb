// pt_probe.cu -- measured ALU peaks of the device (pt_peak_probe), reported by bench.py beside the derived
// roofline: kind 0 = dependent-free FFMA stream, kind 1 = MUFU.COS stream, kind 2 = the instruction mix of one
// sample-evaluation of the fitness loop (7 FP32-pipe + 1 MUFU), kind 3 = FFMA whose three sources are distinct
// registers (register-file port check).
#include "pt_internal.h"

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

__global__ void __launch_bounds__(512, 1) probe_ffma3(float a, float* out) {
    // v[k] = v[k] * w[k] + u[k]: three distinct source registers per FFMA
    float v[kProbeIlp], w[kProbeIlp], u[kProbeIlp];
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) {
        v[k] = (float)(threadIdx.x + k);
        w[k] = a + (float)k * 1e-3f;
        u[k] = a * (float)(k + 1);
    }
#pragma unroll 1
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int k = 0; k < kProbeIlp; ++k) v[k] = fmaf(v[k], w[k], u[k]);
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

__global__ void __launch_bounds__(512, 1) probe_mix(float a, float b, float* out) {
    // per "sample-evaluation": FADD, FFMA, FFMA, (FMUL + MUFU.COS), FFMA, FFMA, FFMA
    float acc[kProbeIlp], t[kProbeIlp];
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) { acc[k] = 0.f; t[k] = (float)(threadIdx.x + k) * a; }
    const float d0 = a, d1 = b, d2 = a * b, a0 = 1.0f + a, a1 = b * 0.5f;
#pragma unroll 1
    for (int it = 0; it < kProbeIters; ++it) {
#pragma unroll
        for (int k = 0; k < kProbeIlp; ++k) {
            const float wd = t[k] + d0;
            const float h = fmaf(t[k], d2, d1);
            const float y = fmaf(t[k], h, wd);
            const float c = __cosf(y);
            const float A = fmaf(t[k], a1, a0);
            const float r = fmaf(-A, c, t[k]);
            acc[k] = fmaf(r, r, acc[k]);
        }
#pragma unroll
        for (int k = 0; k < kProbeIlp; ++k) t[k] += a;   // keep the inputs moving (1 extra FADD per evaluation)
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) s += acc[k];
    if (s == 123.456f) out[0] = s;
}

int peak_probe(int kind, double* ops_per_s) {
    int dev = 0, sms = 0;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return -3;
    if (check_cuda(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute")) return -3;
    float* out = nullptr;
    if (check_cuda(cudaMalloc(&out, 4), "cudaMalloc")) return -3;
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    const int grid = sms * 4, thr = 512;
    float best_ms = 1e30f;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0);
        switch (kind) {
            case 0: probe_ffma<<<grid, thr>>>(1.0001f, 0.5f, out); break;
            case 1: probe_mufu<<<grid, thr>>>(0.37f, out); break;
            case 2: probe_mix<<<grid, thr>>>(0.37f, 0.11f, out); break;
            default: probe_ffma3<<<grid, thr>>>(1.0001f, out); break;
        }
        cudaEventRecord(e1);
        if (check_cuda(cudaEventSynchronize(e1), "probe kernel")) { cudaFree(out); return -3; }
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

}  // namespace pt
