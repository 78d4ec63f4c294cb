// pt_probe.cu -- measured ALU peaks of the device, reported by bench.py beside the derived roofline.  NOT part of libpt.so:
// built into its own library (libpt_probe.so, `build.build_probe()`), which only bench.py loads.
// kind 0 = dependent-free FFMA stream, kind 1 = MUFU.COS stream.
// pt_bench_sm_clock: the SM clock a kernel actually runs at (clock64 against globaltimer) with and without tensor-core activity.
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

// MUFU stream of one CTA per SM for a few milliseconds; with MMA != 0 one thread per CTA also issues a small tcgen05.mma
// (kind::tf32, M 128 x N 8 x K 8, zero operands) every 64 cosines.  CTA 0 measures clock64 against globaltimer.  The variant
// without MMA is a separate instantiation: its code holds no tensor-core instruction at all.
__device__ __forceinline__ uint32_t probe_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
template <bool WITH_MMA>
__global__ void __launch_bounds__(128, 1) probe_clock(float a, float* out, unsigned long long* clk) {
    __shared__ __align__(128) float opA[128 * 8];
    __shared__ __align__(128) float opB[8 * 8];
    __shared__ __align__(8) unsigned long long bar;
    __shared__ uint32_t tptr;
    const int tid = threadIdx.x, warp = tid >> 5;
    for (int i = tid; i < 128 * 8; i += 128) opA[i] = 0.0f;
    if (tid < 64) opB[tid] = 0.0f;
    if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(probe_smem_u32(&bar)) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 32;" ::"r"(probe_smem_u32(&tptr)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = tptr;
    // K-major, no swizzle: 8-row core matrices of 16-byte rows; A: 128 rows (chunk stride 2048 B), B: 8 rows (chunk stride 128 B)
    auto desc = [](uint32_t addr, uint32_t lbo, uint32_t sbo) {
        return (unsigned long long)((addr >> 4) & 0x3FFFu) | ((unsigned long long)((lbo >> 4) & 0x3FFFu) << 16) |
               ((unsigned long long)((sbo >> 4) & 0x3FFFu) << 32) | (1ull << 46);
    };
    const unsigned long long da = desc(probe_smem_u32(opA), 2048, 128), db = desc(probe_smem_u32(opB), 128, 128);
    const uint32_t idesc = (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(8 >> 3) << 17) | ((uint32_t)(128 >> 4) << 24);
    unsigned long long c0 = 0, g0 = 0;
    if (tid == 0 && blockIdx.x == 0) { c0 = clock64(); asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0)); }
    float v[kProbeIlp];
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) v[k] = (float)(tid + k) * a;
#pragma unroll 1
    for (int it = 0; it < 20 * kProbeIters; ++it) {
#pragma unroll
        for (int k = 0; k < kProbeIlp; ++k) v[k] = __cosf(v[k]);
        if (WITH_MMA && tid == 0 && (it & 3) == 0)
            asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, 0, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n" ::"r"(tmem), "l"(da),
                         "l"(db), "r"(idesc)
                         : "memory");
    }
    if (tid == 0) {
        asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(probe_smem_u32(&bar)) : "memory");
        uint32_t ok = 0;
        while (!ok)
            asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}\n" : "=r"(ok) : "r"(probe_smem_u32(&bar)) : "memory");
    }
    if (tid == 0 && blockIdx.x == 0) {
        unsigned long long g1;
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
        clk[0] = clock64() - c0;
        clk[1] = g1 - g0;
    }
    float s = 0.f;
#pragma unroll
    for (int k = 0; k < kProbeIlp; ++k) s += v[k];
    if (s == 123.456f) out[0] = s;
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 32;" ::"r"(tmem) : "memory");
}

}  // namespace pt

// SM clock [MHz] during a MUFU-bound kernel, with (with_mma != 0) or without tensor-core instructions in flight: on the B200 any
// tcgen05.mma activity lowers the SM clock from 1965 to 1845 MHz, which nvidia-smi's clocks.sm does not show.
extern "C" __attribute__((visibility("default"))) int32_t pt_bench_sm_clock(int32_t with_mma, double* mhz) {
    using namespace pt;
    if (!mhz) return -1;
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return -3;
    if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -3;
    float* out = nullptr;
    unsigned long long* clk = nullptr;
    if (cudaMalloc(&out, 4) != cudaSuccess || cudaMalloc(&clk, 16) != cudaSuccess) return -3;
    unsigned long long h[2] = {0, 1};
    for (int rep = 0; rep < 2; ++rep) {
        if (with_mma) probe_clock<true><<<sms, 128>>>(0.37f, out, clk);
        else probe_clock<false><<<sms, 128>>>(0.37f, out, clk);
        if (cudaDeviceSynchronize() != cudaSuccess) { cudaFree(out); cudaFree(clk); return -3; }
    }
    cudaMemcpy(h, clk, 16, cudaMemcpyDeviceToHost);
    cudaFree(out);
    cudaFree(clk);
    *mhz = 1e3 * (double)h[0] / (double)h[1];
    return 0;
}

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
