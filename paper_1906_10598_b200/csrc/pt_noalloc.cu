// pt_noalloc.cu -- pt_refit_doubtful_static: the continuity check and re-search of doubtful blocks (PAPER.md:191-199, :226-248,
// :252; reading R25) for callers that cannot allocate device memory (code under CUDA graph capture, serving loops,
// harnesses that forbid cudaMalloc).  The same kernels as pt_refit_doubtful, in the same order, on the same stream; the only
// difference is where their scratch lives (border residuals [B][10] fp64, running phase [B] fp64, doubtful flags, the ordered
// list of doubtful blocks and its length): in the file-scope device array below instead of a caller-provided workspace.
//
//   * Every GPU that loads libpt.so holds PT_STATIC_SCRATCH_BYTES (4 MiB) of device memory for this array until the process exits.
//   * The call allocates nothing: no cudaMalloc / cudaFree / cudaMallocAsync, no allocating library routine.
//   * All calls on a device share the array, and it keeps the last call's contents: the bytes a call uses are cleared first, on the
//     caller's stream.  Two calls that overlap on the GPU (different streams, no dependency between them) RACE on it.
//   * In host code `g_static_scratch` is a host-side stand-in for the symbol, not a device address; the address the kernels get comes
//     from cudaGetSymbolAddress, looked up once per device with that device current.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "pt_internal.h"

namespace pt {

static __device__ __align__(256) unsigned char g_static_scratch[PT_STATIC_SCRATCH_BYTES];

// Clears the first `bytes` (a multiple of 16) of the array; device code names the array directly.
__global__ void static_scratch_clear_kernel(size_t bytes) {
    uint4* p = reinterpret_cast<uint4*>(g_static_scratch);
    const size_t n = bytes / 16;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        p[i] = make_uint4(0u, 0u, 0u, 0u);
}

constexpr int kMaxDevices = 64;
static std::mutex g_scratch_mutex;
static void* g_scratch_addr[kMaxDevices];      // device address of g_static_scratch on device d (null: not looked up yet)

// Device address of the array on the current device; looked up once per device, with that device current.
static int static_scratch_address(void** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) {
        (void)cudaGetLastError();
        set_error("pt_refit_doubtful_static: no current CUDA device (%s)", e != cudaSuccess ? cudaGetErrorString(e) : "ordinal out of range");
        return PT_ERR_CUDA;
    }
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        void* ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_static_scratch);
        if (e != cudaSuccess || !ptr) {
            (void)cudaGetLastError();
            set_error("pt_refit_doubtful_static: cudaGetSymbolAddress failed on device %d: %s", dev, cudaGetErrorString(e));
            return PT_ERR_CUDA;
        }
        g_scratch_addr[dev] = ptr;
    }
    *out = g_scratch_addr[dev];
    return PT_OK;
}

}  // namespace pt

using namespace pt;

extern "C" {

size_t pt_static_scratch_bytes(void) { return (size_t)PT_STATIC_SCRATCH_BYTES; }

int32_t pt_refit_doubtful_static(const float* x, int64_t B, int32_t N, double fs, double* lo, double* hi,
                                 const uint32_t* block_index, const pt_de_config* cfg, const pt_retry_config* retry,
                                 double* best, float* best_rss, uint32_t* status, int32_t* attempts, void* stream) {
    if (!x || !lo || !hi || !cfg || !retry || !best || !best_rss || !status || !attempts) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if (B < 1) { set_error("B must be >= 1"); return PT_ERR_INVALID_ARG; }
    const size_t need = pt_refit_doubtful_workspace_bytes(B, N, cfg);
    if (need == 0) { set_error("pt_refit_doubtful_static: invalid B, N or configuration"); return PT_ERR_INVALID_ARG; }
    if (need > (size_t)PT_STATIC_SCRATCH_BYTES) {
        set_error("pt_refit_doubtful_static: B = %lld blocks of N = %d samples need %zu bytes of scratch, the static array holds %zu "
                  "(about %lld blocks that fit in shared memory); use pt_refit_doubtful with a caller workspace",
                  (long long)B, N, need, (size_t)PT_STATIC_SCRATCH_BYTES, (long long)(PT_STATIC_SCRATCH_BYTES / 96 - 16));
        return PT_ERR_UNSUPPORTED;
    }
    void* scratch = nullptr;
    const int rc = static_scratch_address(&scratch);
    if (rc) return rc;
    // the array keeps the previous call's contents: clear what this call uses (need is a multiple of 256)
    const size_t bytes = (need + 15) / 16 * 16;
    const unsigned grid = (unsigned)((bytes / 16 + 255) / 256 < 1184 ? (bytes / 16 + 255) / 256 : 1184);
    static_scratch_clear_kernel<<<grid, 256, 0, (cudaStream_t)stream>>>(bytes);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { set_error("static_scratch_clear_kernel launch: %s", cudaGetErrorString(e)); return PT_ERR_CUDA; }
    return pt_refit_doubtful(x, B, N, fs, lo, hi, block_index, cfg, retry, best, best_rss, status, attempts, scratch,
                             (size_t)PT_STATIC_SCRATCH_BYTES, stream);
}

}  // extern "C"
