// pt_api.cu -- the C ABI of libpt.so (include/pt.h): argument checks, launch planning, kernel launches.
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <cmath>
#include <algorithm>
#include <mutex>
#include <vector>

#include "../../include/pt.h"
#include "pt_de_kernel.cuh"
#include "pt_tc_kernel.cuh"
#include "pt_run_kernel.cuh"
#include "pt_internal.h"

namespace pt {

static thread_local char g_err[512] = "no error";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

int check_cuda(cudaError_t e, const char* what) {
    if (e == cudaSuccess) return 0;
    set_error("%s: %s", what, cudaGetErrorString(e));
    return 1;
}

// ---------------------------------------------------------------------------------------------------
// Launch plan of the block kernel.
// ---------------------------------------------------------------------------------------------------
struct Plan {
    int C, threads, Wg, Ws, ctas_per_sm, grid, smem, Npad, NPpad, resident, sms;
    int TS, S;              // streamed path: samples per tile, ring stages (0, 0 when resident)
    size_t ws_bytes;        // device workspace the launch needs (streamed path only)
    int K, NpadS;           // cluster path: CTAs per block, padded samples of the largest slice (K = 1: Npad)
    int tc;                 // 1: the tensor-core kernel (pt_tc_kernel.cuh) fits these blocks
    int tc_slots;           //    data blocks one of its CTAs fits at the same time (2 when shared memory allows)
    int run;                // 1: the run-local kernel (pt_run_kernel.cuh) fits these blocks
};

// Per-device facts and per-device launch attributes, keyed by the CUDA device ordinal and guarded by one mutex: a process may
// drive several devices, from several host threads.
constexpr int kMaxDevices = 64;
static std::mutex g_dev_mutex;
struct DeviceFacts { int known, sms, smem_optin; };
static DeviceFacts g_dev[kMaxDevices];

// *_host entry points: a stream-ordered memory pool and a stream per device, kept between calls so that a repeated call pays
// neither cudaMalloc / cudaFree (0.5 ms each, with occasional outliers of 10-100 ms) nor stream creation.
struct HostCache { int ready; cudaMemPool_t pool; cudaStream_t stream; };
static HostCache g_host_cache[kMaxDevices];

static int host_cache_get(cudaMemPool_t* pool, cudaStream_t* stream) {
    int dev = 0;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return 1;
    if (dev < 0 || dev >= kMaxDevices) { set_error("device ordinal %d beyond the compiled limit %d", dev, kMaxDevices); return 1; }
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    HostCache& c = g_host_cache[dev];
    if (!c.ready) {
        cudaMemPoolProps props;
        memset(&props, 0, sizeof(props));
        props.allocType = cudaMemAllocationTypePinned;
        props.handleTypes = cudaMemHandleTypeNone;
        props.location.type = cudaMemLocationTypeDevice;
        props.location.id = dev;
        if (check_cuda(cudaMemPoolCreate(&c.pool, &props), "cudaMemPoolCreate")) return 1;
        unsigned long long keep = ~0ull;        // freed blocks stay in the pool until pt_host_cache_release()
        if (check_cuda(cudaMemPoolSetAttribute(c.pool, cudaMemPoolAttrReleaseThreshold, &keep), "cudaMemPoolSetAttribute")) return 1;
        if (check_cuda(cudaStreamCreateWithFlags(&c.stream, cudaStreamNonBlocking), "cudaStreamCreate")) return 1;
        c.ready = 1;
    }
    *pool = c.pool;
    *stream = c.stream;
    return 0;
}

static int device_info(int* sms, int* smem_optin, int* dev_out = nullptr) {
    int dev = 0;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return 1;
    if (dev < 0 || dev >= kMaxDevices) { set_error("device ordinal %d beyond the compiled limit %d", dev, kMaxDevices); return 1; }
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    DeviceFacts& f = g_dev[dev];
    if (!f.known) {
        if (check_cuda(cudaDeviceGetAttribute(&f.sms, cudaDevAttrMultiProcessorCount, dev), "cudaDeviceGetAttribute")) return 1;
        if (check_cuda(cudaDeviceGetAttribute(&f.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev), "cudaDeviceGetAttribute")) return 1;
        f.known = 1;
    }
    *sms = f.sms;
    *smem_optin = f.smem_optin;
    if (dev_out) *dev_out = dev;
    return 0;
}

static bool have_device() {
    int n = 0;
    if (cudaGetDeviceCount(&n) != cudaSuccess || n == 0) { (void)cudaGetLastError(); return false; }
    return true;
}
static int device_smem_optin() {
    int sms = 148, smem_optin = 232448;
    if (!have_device() || device_info(&sms, &smem_optin)) return 232448;
    return smem_optin;
}

// Warp grid (Wg candidate-group columns x Ws sample slices) with the smallest per-warp load.
static void choose_warp_grid(int warps, int groups, int nch, int* Wg, int* Ws) {
    long long best = -1;
    for (int wg = 1; wg <= warps; ++wg) {
        if (warps % wg) continue;
        const int ws = warps / wg;
        const long long load = (long long)((groups + wg - 1) / wg) * ((nch + ws - 1) / ws);
        // prefer fewer slices on ties (fewer partial sums to combine)
        if (best < 0 || load < best || (load == best && ws < *Ws)) { best = load; *Wg = wg; *Ws = ws; }
    }
}

// Which evaluation kernel fits a block: pt_run_kernel (thread = candidate, phase by run-local Horner with immediate indices: the
// default), pt_block_kernel (lanes own samples, phase relative to a reference array) or pt_tc_kernel (phase on the tensor cores).
// Automatic choice = whichever measured fastest on the B200 (profiles/r2_kernel_choice.md): pt_run_kernel
// everywhere.  PT_KERNEL=run / tc / classic in the environment forces one of them where it applies (tests, A/B measurements).
static int kernel_override() {
    const char* e = getenv("PT_KERNEL");
    if (!e || !*e) return 0;
    if (!strcmp(e, "tc")) return 1;
    if (!strcmp(e, "classic")) return 2;
    if (!strcmp(e, "run")) return 3;
    return 0;
}
static bool want_tc(int N, int NP, int D, int objective) {
    (void)N; (void)D; (void)objective;
    if (NP > kTcMaxNP) return false;
    return kernel_override() == 1;
}
static bool want_run() {
    const int o = kernel_override();
    return o == 0 || o == 3;
}

// Plan of pt_run_kernel: one CTA of 1024 threads per SM, or 2 x 512 / 4 x 256 / 8 x 128 (short blocks) when shared memory and the number of blocks allow (the
// DE step of one CTA then overlaps with the evaluation of the others); with few blocks a cluster of K CTAs per block; blocks
// larger than shared memory are streamed through a ring of 3 tiles.
// Sample slices of pt_run_kernel's evaluation: NP x S work items over `threads` threads, `len` samples per tile.  Picks the S that
// maximises (thread utilisation in whole rounds) x (useful share of a run: a run of L samples pays about 32 sample-evaluations of
// re-expansion), smallest S on ties; at most two rounds of items.
static int choose_slices(int NP, int threads, int len) {
    int best = 1;
    double best_score = -1.0;
    const int cap = 2 * (threads > NP ? threads : NP);
    for (int S = 1; S <= 64 && (long long)NP * S <= cap; ++S) {
        const int per = len / S;
        if (S > 1 && per < 64) break;
        const long long items = (long long)NP * S, rounds = (items + threads - 1) / threads;
        const double util = (double)items / (double)(rounds * threads);
        const double L = per < kRun ? (double)per : (double)kRun;
        const double score = util * L / (L + 32.0);
        if (score > best_score + 1e-9) { best_score = score; best = S; }
    }
    return best;
}

// Short blocks (measured on the config-4 sweep, profiles/r2_kernel_choice.md): with NP x N <= kRunCps8Max sample-evaluations per
// generation a block runs on a CTA of 128 threads, eight per SM; with NP x N <= kRunPartialMax the remainder of a launch list stays
// one partly filled round instead of being cut into exactly full grids of fewer, larger CTAs per SM (whose DE steps are exposed).
constexpr long long kRunCps8Max = 1 << 18;
constexpr long long kRunPartialMax = 1 << 19;
constexpr int kRunMaxCps = 8;
static int make_plan_run(long long B, int N, int NP, int D, int sms, int smem_optin, int force_K, Plan* pl, int max_cps = kRunMaxCps) {
    pl->sms = sms;
    pl->tc = 0; pl->tc_slots = 1; pl->run = 1;
    pl->C = 1; pl->NPpad = NP; pl->Wg = 1; pl->Ws = 1;
    pl->Npad = (N + 3) & ~3;
    pl->K = 1; pl->NpadS = pl->Npad; pl->TS = 0; pl->S = 0; pl->ws_bytes = 0; pl->resident = 1;
    const int per_sm_total = smem_optin + 1024;   // 228 KB per SM, 1 KB reserved per resident CTA
    const int quads = pl->Npad / 4;
    {
        // few blocks, many SMs: K = the largest power of two <= min(8, SMs / B) that leaves every CTA at least two runs of samples
        int K = 1;
        while (K * 2 <= 8 && (long long)B * (K * 2) <= sms && N / (K * 2) >= 2 * kRun) K *= 2;
        if (force_K > 0) { K = force_K; while (K > 1 && quads / K < 1) --K; }
        if (K > 1) {
            // (splitting the cluster further into 2 x 512 or 4 x 256-thread CTAs per SM, so that the replicated DE step of one block
            // overlaps with the evaluation of another, was measured on config 1 and lost: 26.8 / 27.7 ms against 21.3 ms)
            const int NresMax = ((quads + K - 1) / K + 1) * 4;
            const int slices = choose_slices(NP, kRunMaxThreads, N / K);
            const RunSmemLayout L(NresMax, NP, D, slices, 0, 0, K);
            if (L.total <= smem_optin) {
                pl->threads = kRunMaxThreads; pl->ctas_per_sm = 1; pl->smem = L.total; pl->K = K; pl->NpadS = NresMax; pl->Ws = slices;
                const long long want = (long long)(sms / K) * K;
                pl->grid = (int)((long long)B * K < want ? (long long)B * K : want);
                return 0;
            }
        }
    }
    for (int cps = max_cps; cps >= 1; cps >>= 1) {
        if (cps > 1 && B <= (long long)sms * (cps / 2)) continue;   // not enough blocks to want that many CTAs
        const int threads = kRunMaxThreads / cps;
        const int slices = choose_slices(NP, threads, N);
        // eight CTAs of 128 threads: blocks so short that a generation is a few thousand cycles (slices of whole runs, and seven
        // other CTAs evaluating while one is in its DE step)
        if (cps == 8 && (long long)NP * N > kRunCps8Max) continue;
        const RunSmemLayout L(pl->Npad, NP, D, slices);
        if (L.total > smem_optin) continue;
        if ((long long)(L.total + 1024) * cps > per_sm_total) continue;
        pl->threads = threads; pl->ctas_per_sm = cps; pl->smem = L.total; pl->Ws = slices;
        const long long want = (long long)sms * cps;
        pl->grid = (int)(B < want ? B : want);
        return 0;
    }
    // streamed
    pl->resident = 0;
    for (int TS = 16384; TS >= 1024; TS >>= 1) {
        const int slices = choose_slices(NP, kRunMaxThreads, TS);
        const RunSmemLayout L(pl->Npad, NP, D, slices, TS, 3);
        if (L.total > smem_optin) continue;
        pl->threads = kRunMaxThreads; pl->ctas_per_sm = 1; pl->smem = L.total; pl->TS = TS; pl->S = 3; pl->Ws = slices;
        pl->grid = (int)(B < sms ? B : sms);
        pl->ws_bytes = (size_t)pl->grid * pl->Npad * sizeof(float);      // aligned fp32 copies of unaligned / quantised rows
        return 0;
    }
    return 1;
}

// sms / smem_optin are passed in so that the plan can also be computed without a device (defaults of B200).
// force_K > 0 overrides the cluster-size choice (tests, tuning); 0 = automatic
static int make_plan(long long B, int N, int NP, int D, int sms, int smem_optin, int force_K, Plan* pl, int objective = 0) {
    if (want_run() && make_plan_run(B, N, NP, D, sms, smem_optin, force_K, pl) == 0) return 0;
    pl->sms = sms;
    pl->tc = 0; pl->tc_slots = 1; pl->run = 0;
    pl->C = (NP % 8 == 0) ? 8 : 4;
    pl->NPpad = (NP + pl->C - 1) / pl->C * pl->C;
    pl->Npad = (N + kChunk - 1) / kChunk * kChunk;
    const int groups = pl->NPpad / pl->C, nch = pl->Npad / kChunk;
    const int per_sm_total = smem_optin + 1024;   // 228 KB per SM, 1 KB reserved per resident CTA
    int chosen = 0;
    pl->K = 1; pl->NpadS = pl->Npad;
    // Few blocks, many SMs: a thread-block cluster of K CTAs (K SMs) per block, each owning 1/K of the samples.
    // K = the largest power of two <= min(8, SMs / B) that leaves every CTA at least two chunks of samples.
    {
        int K = 1;
        while (K * 2 <= 8 && (long long)B * (K * 2) <= sms && nch / (K * 2) >= 2) K *= 2;
        if (force_K > 0) { K = force_K; while (K > 1 && nch / K < 1) --K; }
        if (K > 1) {
            const int threads = 512, warps = threads / 32;
            const int nchS = (nch + K - 1) / K;
            int Wg = 1, Ws = warps;
            choose_warp_grid(warps, groups, nchS, &Wg, &Ws);
            const SmemLayout L(nchS * kChunk, NP, pl->NPpad, D, Ws, 0, 0, K);
            if (L.total <= smem_optin) {
                pl->threads = threads; pl->Wg = Wg; pl->Ws = Ws; pl->ctas_per_sm = 1; pl->smem = L.total;
                pl->K = K; pl->NpadS = nchS * kChunk;
                pl->resident = 1; pl->TS = 0; pl->S = 0; pl->ws_bytes = 0;
                const long long want = (long long)(sms / K) * K;
                pl->grid = (int)((long long)B * K < want ? (long long)B * K : want);
                return 0;
            }
        }
    }
    if (want_tc(N, NP, D, objective)) {
        // one CTA of 640 threads per SM; shared memory holds the samples only, so the block must be resident
        for (int slots = 2; slots >= 1; --slots) {
            const TcSmemLayout L(N, NP, D, slots);
            if (L.total > smem_optin) continue;
            pl->tc = 1; pl->tc_slots = slots; pl->C = 1; pl->NPpad = kTcMaxNP; pl->threads = kTcThreads; pl->Wg = 4; pl->Ws = 4;
            pl->ctas_per_sm = 1; pl->smem = L.total; pl->resident = 1; pl->TS = 0; pl->S = 0; pl->ws_bytes = 0;
            pl->grid = (int)(B < sms ? B : sms);
            return 0;
        }
    }
    for (int cps = 4; cps >= 1; cps >>= 1) {
        if (cps > 1 && B <= (long long)sms * (cps / 2)) continue;   // not enough blocks to want that many CTAs
        const int threads = 512 / cps, warps = threads / 32;
        int Wg = 1, Ws = warps;
        choose_warp_grid(warps, groups, nch, &Wg, &Ws);
        const SmemLayout L(pl->Npad, NP, pl->NPpad, D, Ws);
        if (L.total > smem_optin) continue;
        if ((long long)(L.total + 1024) * cps > per_sm_total) continue;
        pl->threads = threads; pl->Wg = Wg; pl->Ws = Ws; pl->ctas_per_sm = cps; pl->smem = L.total;
        chosen = 1;
        break;
    }
    pl->resident = chosen;
    pl->TS = 0; pl->S = 0; pl->ws_bytes = 0;
    if (!chosen) {
        // streamed: one CTA of 512 threads per SM, ring of 3 stages, the largest tile that fits
        const int threads = 512, warps = threads / 32, S = 3;
        for (int TS = 8192; TS >= 1024 && !chosen; TS >>= 1) {
            int Wg = 1, Ws = warps;
            choose_warp_grid(warps, groups, TS / kChunk, &Wg, &Ws);
            const SmemLayout L(pl->Npad, NP, pl->NPpad, D, Ws, TS, S);
            if (L.total > smem_optin) continue;
            pl->threads = threads; pl->Wg = Wg; pl->Ws = Ws; pl->ctas_per_sm = 1; pl->smem = L.total;
            pl->TS = TS; pl->S = S;
            chosen = 1;
        }
        if (!chosen) return 1;
    }
    const long long want = (long long)sms * pl->ctas_per_sm;
    pl->grid = (int)(B < want ? B : want);
    if (pl->S > 0) pl->ws_bytes = (size_t)pl->grid * pl->Npad * sizeof(float) * 2;   // reference-phase rows + aligned copies
    return 0;
}

// PT_CLUSTER=<K> in the environment forces the cluster size (1 = never cluster); unset/0 = automatic.
static int force_cluster() {
    const char* e = getenv("PT_CLUSTER");
    if (!e || !*e) return 0;
    const int k = atoi(e);
    return (k >= 1 && k <= 8) ? k : 0;
}

// plan with the current device's limits, or B200's when no device is present (the query entry points)
static int plan_for(long long B, int N, int NP, int D, Plan* pl, bool need_device, int force_K = 0, int objective = 0) {
    int sms = 148, smem_optin = 232448;
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) == cudaSuccess && dev_count > 0) {
        if (device_info(&sms, &smem_optin)) return PT_ERR_CUDA;
    } else {
        (void)cudaGetLastError();
        if (need_device) { set_error("no CUDA device"); return PT_ERR_CUDA; }
    }
    if (make_plan(B, N, NP, D, sms, smem_optin, force_K > 0 ? force_K : force_cluster(), pl, objective)) {
        set_error("N = %d with NP = %d: population tables alone exceed shared memory", N, NP);
        return PT_ERR_UNSUPPORTED;
    }
    return PT_OK;
}

static void cluster_launch_config(const Plan& pl, int grid, cudaStream_t st, cudaLaunchConfig_t* cfg, cudaLaunchAttribute* attr) {
    memset(cfg, 0, sizeof(*cfg));
    cfg->gridDim = dim3((unsigned)grid);
    cfg->blockDim = dim3((unsigned)pl.threads);
    cfg->dynamicSmemBytes = (size_t)pl.smem;
    cfg->stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)pl.K; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
    cfg->attrs = attr; cfg->numAttrs = 1;
}

template <int C, int D, int MODE, bool STREAM, int OBJ>
static int configure_smem(const Plan& pl) {
    // cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device attribute of the kernel: remember the largest value set on
    // each device (one table per template instantiation)
    static int configured_smem[kMaxDevices];
    int dev = 0;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return PT_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) { set_error("device ordinal %d beyond the compiled limit %d", dev, kMaxDevices); return PT_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (pl.smem > configured_smem[dev]) {
        if (check_cuda(cudaFuncSetAttribute(pt_block_kernel<C, D, MODE, STREAM, OBJ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                            pl.smem),
                       "cudaFuncSetAttribute"))
            return PT_ERR_CUDA;
        configured_smem[dev] = pl.smem;
    }
    return PT_OK;
}

// clusters of pl.K CTAs that can be resident at once (0 if the query fails)
template <int C, int D, int MODE, bool STREAM, int OBJ>
static int max_resident_clusters(const Plan& pl) {
    if (configure_smem<C, D, MODE, STREAM, OBJ>(pl)) return 0;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    cluster_launch_config(pl, pl.K, nullptr, &cfg, attr);
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, pt_block_kernel<C, D, MODE, STREAM, OBJ>, &cfg) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return n;
}

template <int C, int D, int MODE, bool STREAM, int OBJ>
static int launch_block_kernel(const BlockParams& p, const Plan& pl, cudaStream_t st) {
    if (configure_smem<C, D, MODE, STREAM, OBJ>(pl)) return PT_ERR_CUDA;
    if (pl.K > 1) {
        // one thread-block cluster of K CTAs per data block
        int grid = pl.grid;
        const int max_clusters = max_resident_clusters<C, D, MODE, STREAM, OBJ>(pl);
        if (max_clusters > 0 && grid > max_clusters * pl.K) grid = max_clusters * pl.K;   // persistent: resident clusters only
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute attr[1];
        cluster_launch_config(pl, grid, st, &cfg, attr);
        if (check_cuda(cudaLaunchKernelEx(&cfg, pt_block_kernel<C, D, MODE, STREAM, OBJ>, p), "pt_block_kernel cluster launch"))
            return PT_ERR_CUDA;
        return PT_OK;
    }
    pt_block_kernel<C, D, MODE, STREAM, OBJ><<<pl.grid, pl.threads, pl.smem, st>>>(p);
    if (check_cuda(cudaGetLastError(), "pt_block_kernel launch")) return PT_ERR_CUDA;
    return PT_OK;
}

template <int MODE, bool STREAM, int OBJ>
static int dispatch3(const BlockParams& p, const Plan& pl, int D, cudaStream_t st) {
    if (pl.C == 8)
        return D == 5 ? launch_block_kernel<8, 5, MODE, STREAM, OBJ>(p, pl, st) : launch_block_kernel<8, 6, MODE, STREAM, OBJ>(p, pl, st);
    return D == 5 ? launch_block_kernel<4, 5, MODE, STREAM, OBJ>(p, pl, st) : launch_block_kernel<4, 6, MODE, STREAM, OBJ>(p, pl, st);
}

template <int MODE, bool STREAM>
static int dispatch2(const BlockParams& p, const Plan& pl, int D, int objective, cudaStream_t st) {
    return objective == kObjCor ? dispatch3<MODE, STREAM, kObjCor>(p, pl, D, st) : dispatch3<MODE, STREAM, kObjChi2>(p, pl, D, st);
}

template <int D, int MODE, int OBJ>
static int launch_tc_kernel(const BlockParams& p, const Plan& pl, cudaStream_t st) {
    static int configured_smem[kMaxDevices];
    int dev = 0;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return PT_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) { set_error("device ordinal %d beyond the compiled limit %d", dev, kMaxDevices); return PT_ERR_CUDA; }
    {
        std::lock_guard<std::mutex> lock(g_dev_mutex);
        if (pl.smem > configured_smem[dev]) {
            if (check_cuda(cudaFuncSetAttribute(pt_tc_kernel<D, MODE, OBJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem), "cudaFuncSetAttribute"))
                return PT_ERR_CUDA;
            configured_smem[dev] = pl.smem;
        }
    }
    pt_tc_kernel<D, MODE, OBJ><<<pl.grid, pl.threads, pl.smem, st>>>(p);
    if (check_cuda(cudaGetLastError(), "pt_tc_kernel launch")) return PT_ERR_CUDA;
    return PT_OK;
}

template <int MODE>
static int dispatch_tc(const BlockParams& p, const Plan& pl, int D, int objective, cudaStream_t st) {
    if (objective == kObjCor) return D == 5 ? launch_tc_kernel<5, MODE, kObjCor>(p, pl, st) : launch_tc_kernel<6, MODE, kObjCor>(p, pl, st);
    return D == 5 ? launch_tc_kernel<5, MODE, kObjChi2>(p, pl, st) : launch_tc_kernel<6, MODE, kObjChi2>(p, pl, st);
}

// ---- pt_run_kernel ----
template <int D, int MODE, bool STREAM, int OBJ>
static int run_configure_smem(const Plan& pl) {
    static int configured_smem[kMaxDevices];
    int dev = 0;
    if (check_cuda(cudaGetDevice(&dev), "cudaGetDevice")) return PT_ERR_CUDA;
    if (dev < 0 || dev >= kMaxDevices) { set_error("device ordinal %d beyond the compiled limit %d", dev, kMaxDevices); return PT_ERR_CUDA; }
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    if (pl.smem > configured_smem[dev]) {
        if (check_cuda(cudaFuncSetAttribute(pt_run_kernel<D, MODE, STREAM, OBJ>, cudaFuncAttributeMaxDynamicSharedMemorySize, pl.smem), "cudaFuncSetAttribute"))
            return PT_ERR_CUDA;
        configured_smem[dev] = pl.smem;
    }
    return PT_OK;
}

template <int D, int MODE, bool STREAM, int OBJ>
static int run_max_resident_clusters(const Plan& pl) {
    if (run_configure_smem<D, MODE, STREAM, OBJ>(pl)) return 0;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    cluster_launch_config(pl, pl.K, nullptr, &cfg, attr);
    int n = 0;
    if (cudaOccupancyMaxActiveClusters(&n, pt_run_kernel<D, MODE, STREAM, OBJ>, &cfg) != cudaSuccess) {
        (void)cudaGetLastError();
        return 0;
    }
    return n;
}

template <int D, int MODE, bool STREAM, int OBJ>
static int launch_run_kernel(const BlockParams& p, const Plan& pl, cudaStream_t st) {
    if (run_configure_smem<D, MODE, STREAM, OBJ>(pl)) return PT_ERR_CUDA;
    if (pl.K > 1) {
        int grid = pl.grid;
        const int max_clusters = run_max_resident_clusters<D, MODE, STREAM, OBJ>(pl);
        if (max_clusters > 0 && grid > max_clusters * pl.K) grid = max_clusters * pl.K;   // persistent: resident clusters only
        cudaLaunchConfig_t cfg;
        cudaLaunchAttribute attr[1];
        cluster_launch_config(pl, grid, st, &cfg, attr);
        if (check_cuda(cudaLaunchKernelEx(&cfg, pt_run_kernel<D, MODE, STREAM, OBJ>, p), "pt_run_kernel cluster launch")) return PT_ERR_CUDA;
        return PT_OK;
    }
    pt_run_kernel<D, MODE, STREAM, OBJ><<<pl.grid, pl.threads, pl.smem, st>>>(p);
    if (check_cuda(cudaGetLastError(), "pt_run_kernel launch")) return PT_ERR_CUDA;
    return PT_OK;
}

template <int MODE, bool STREAM>
static int dispatch_run2(const BlockParams& p, const Plan& pl, int D, int objective, cudaStream_t st) {
    if (objective == kObjCor) return D == 5 ? launch_run_kernel<5, MODE, STREAM, kObjCor>(p, pl, st) : launch_run_kernel<6, MODE, STREAM, kObjCor>(p, pl, st);
    return D == 5 ? launch_run_kernel<5, MODE, STREAM, kObjChi2>(p, pl, st) : launch_run_kernel<6, MODE, STREAM, kObjChi2>(p, pl, st);
}

template <int MODE>
static int dispatch_run(const BlockParams& p, const Plan& pl, int D, int objective, cudaStream_t st) {
    return pl.S > 0 ? dispatch_run2<MODE, true>(p, pl, D, objective, st) : dispatch_run2<MODE, false>(p, pl, D, objective, st);
}

template <int MODE>
static int dispatch(const BlockParams& p, const Plan& pl, int D, int objective, cudaStream_t st) {
    if (pl.run) return dispatch_run<MODE>(p, pl, D, objective, st);
    if (pl.tc) return dispatch_tc<MODE>(p, pl, D, objective, st);
    return pl.S > 0 ? dispatch2<MODE, true>(p, pl, D, objective, st) : dispatch2<MODE, false>(p, pl, D, objective, st);
}

// the shared-memory footprint, register count and launch bounds do not depend on the objective
static int fit_max_resident_clusters(const Plan& pl, int D) {
    if (pl.run) return D == 5 ? run_max_resident_clusters<5, kModeFit, false, kObjChi2>(pl) : run_max_resident_clusters<6, kModeFit, false, kObjChi2>(pl);
    if (pl.C == 8) return D == 5 ? max_resident_clusters<8, 5, kModeFit, false, kObjChi2>(pl) : max_resident_clusters<8, 6, kModeFit, false, kObjChi2>(pl);
    return D == 5 ? max_resident_clusters<4, 5, kModeFit, false, kObjChi2>(pl) : max_resident_clusters<4, 6, kModeFit, false, kObjChi2>(pl);
}

// Tail wave.  B blocks on a persistent grid of `sms` single-CTA blocks take ceil(B / sms) waves; when the last wave
// is at most half full its `rem` blocks are fitted by a second launch in which a cluster of K = floor(sms / rem)
// CTAs shares each block, so the tail costs 1/K of a wave.  K is lowered until `rem` clusters are resident at once.
// Returns the number of tail blocks (0: single launch) and their plan.
static long long plan_tail(long long B, int N, int NP, int D, const Plan& pl, Plan* tail) {
    const long long slots = (long long)pl.sms * pl.ctas_per_sm;
    if (force_cluster() != 0 || pl.K != 1 || pl.S != 0 || (pl.ctas_per_sm != 1 && !pl.run) || B <= slots) return 0;
    const long long rem = B % slots;
    if (rem == 0 || rem * 2 > pl.sms) return 0;
    int sms = 0, smem_optin = 0;
    if (device_info(&sms, &smem_optin)) return 0;
    for (int K = (int)(sms / rem) < 8 ? (int)(sms / rem) : 8; K >= 2; --K) {
        Plan t;
        if (make_plan(rem, N, NP, D, sms, smem_optin, K, &t) || t.K != K) continue;
        if (fit_max_resident_clusters(t, D) >= rem) { *tail = t; return rem; }
    }
    return 0;
}

// Launch list of pt_run_kernel.  All blocks take the same time, so a persistent grid is balanced only when every CTA fits the same
// number of blocks and every SM holds the same number of CTAs -- and which CTAs share an SM is the block scheduler's business
// (measured on the B200: consecutive CTAs, not CTA i and i + SMs), so a partly filled last round can leave half of the SMs idle.
// The blocks are therefore cut into segments, one launch each, in which the grid is exactly full: whole rounds of SMs x c CTAs,
// then the remainder with fewer (larger) CTAs per SM, and the last < SMs / 2 blocks on clusters of K = SMs / rem CTAs per block.
struct Segment { long long first, count; Plan pl; };
static int run_launch_list(long long B, int N, int NP, int D, int sms, int smem_optin, std::vector<Segment>* out) {
    long long done = 0;
    int max_cps = kRunMaxCps;
    while (done < B) {
        const long long left = B - done;
        Segment sg;
        sg.first = done;
        if (left * 2 <= sms) {
            // the last few blocks: clusters, as many CTAs per block as are resident at once
            bool ok = false;
            int Kmax = (int)(sms / left) < 8 ? (int)(sms / left) : 8;
            if (Kmax > N / (2 * kRun)) Kmax = N / (2 * kRun);           // every CTA keeps at least two runs of samples
            for (int K = Kmax; K >= 2 && !ok; --K) {
                if (make_plan_run(left, N, NP, D, sms, smem_optin, K, &sg.pl) || sg.pl.K != K) continue;
                ok = !have_device() || fit_max_resident_clusters(sg.pl, D) >= left;      // no device: the plan of a B200, residency assumed
            }
            if (!ok && make_plan_run(left, N, NP, D, sms, smem_optin, 1, &sg.pl, 1)) return 1;
            sg.count = left;
        } else {
            if (make_plan_run(left, N, NP, D, sms, smem_optin, 1, &sg.pl, max_cps)) return 1;
            const long long slots = (long long)sms * sg.pl.ctas_per_sm;
            if (left >= slots) {
                sg.count = left / slots * slots;
            } else if (sg.pl.ctas_per_sm > 1 && (long long)NP * N <= kRunPartialMax) {
                // blocks so short that a generation is bound by the latency of its DE step as much as by the XU pipe: fewer, larger
                // CTAs per SM would expose it (measured: N 1024 NP 128, 4 + 2 + 1 CTAs per SM in three launches 68.8 %, one partly
                // filled round of 8 per SM 76.6 %), so the remainder stays one partly filled round
                sg.count = left;
            } else if (sg.pl.ctas_per_sm > 1) {
                // fewer blocks than CTA slots: the largest c' <= left / SMs CTAs per SM, exactly full
                int c = sg.pl.ctas_per_sm;
                while (c > 1 && (long long)sms * c > left) c >>= 1;
                if (make_plan_run((long long)sms * c, N, NP, D, sms, smem_optin, 1, &sg.pl, c)) return 1;
                sg.count = left < (long long)sms * sg.pl.ctas_per_sm ? left : (long long)sms * sg.pl.ctas_per_sm;
            } else {
                sg.count = left;
            }
            max_cps = sg.pl.ctas_per_sm;
            sg.pl.grid = (int)(sg.count < (long long)sms * sg.pl.ctas_per_sm ? sg.count : (long long)sms * sg.pl.ctas_per_sm);
        }
        out->push_back(sg);
        done += sg.count;
    }
    return 0;
}

// streamed path: hand the workspace rows to the kernel
static int attach_workspace(BlockParams* p, const Plan& pl, void* workspace, size_t workspace_bytes) {
    p->TS = pl.TS; p->S = pl.S;
    p->K = pl.K; p->NpadS = pl.NpadS; p->tc_slots = pl.tc_slots;
    if (pl.run) { p->Npad = pl.Npad; p->NPpad = pl.NPpad; }
    if (pl.S == 0) return PT_OK;
    if (!workspace || workspace_bytes < pl.ws_bytes) {
        set_error("streamed path (N = %d does not fit in shared memory) needs %zu bytes of workspace, got %zu", p->N, pl.ws_bytes,
                  workspace ? workspace_bytes : (size_t)0);
        return PT_ERR_UNSUPPORTED;
    }
    if (reinterpret_cast<uintptr_t>(workspace) % 16) { set_error("workspace must be 16-byte aligned"); return PT_ERR_INVALID_ARG; }
    p->ws_wref = reinterpret_cast<float*>(workspace);
    p->ws_x = pl.run ? p->ws_wref : p->ws_wref + (size_t)pl.grid * pl.Npad;      // pt_run_kernel has no reference-phase rows
    return PT_OK;
}

static uint32_t cr32_of(double CR) {
    const double v = floor(CR * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

static int check_common(long long B, int N, double fs, int NP, int D) {
    if (B < 1) { set_error("B must be >= 1"); return PT_ERR_INVALID_ARG; }
    if (N < 8 || (N & 1)) { set_error("N must be even and >= 8 (got %d)", N); return PT_ERR_INVALID_ARG; }
    if (N > PT_MAX_N) { set_error("N = %d exceeds PT_MAX_N = %d (sample indices are carried exactly in fp32)", N, PT_MAX_N); return PT_ERR_UNSUPPORTED; }
    if (!(fs > 0.0)) { set_error("fs must be > 0"); return PT_ERR_INVALID_ARG; }
    if (D != 5 && D != 6) { set_error("D must be 5 or 6 (got %d)", D); return PT_ERR_INVALID_ARG; }
    if (NP < 4) { set_error("NP must be >= 4 (got %d)", NP); return PT_ERR_INVALID_ARG; }
    if (NP > PT_MAX_NP) { set_error("NP = %d exceeds PT_MAX_NP = %d", NP, PT_MAX_NP); return PT_ERR_UNSUPPORTED; }
    return PT_OK;
}

static int check_quant(const pt_quant* q, int64_t row_bytes, int N, Quant* out) {
    if (!q) { set_error("quant is null"); return PT_ERR_INVALID_ARG; }
    if (q->bits != 1 && q->bits != 2 && q->bits != 4 && q->bits != 8 && q->bits != 16) {
        set_error("quant.bits must be 1, 2, 4, 8 or 16 (got %d)", q->bits);
        return PT_ERR_INVALID_ARG;
    }
    if (!std::isfinite(q->scale) || !std::isfinite(q->offset)) { set_error("quant.scale and quant.offset must be finite"); return PT_ERR_INVALID_ARG; }
    if (row_bytes * 8 < (int64_t)N * q->bits) { set_error("row_bytes = %lld holds fewer than N = %d samples of %d bits", (long long)row_bytes, N, q->bits); return PT_ERR_INVALID_ARG; }
    out->bits = q->bits; out->is_signed = q->is_signed ? 1 : 0; out->scale = q->scale; out->offset = q->offset;
    return PT_OK;
}

static int check_cfg(const pt_de_config* cfg) {
    if (!cfg) { set_error("cfg is null"); return PT_ERR_INVALID_ARG; }
    if (cfg->generations < 0) { set_error("generations must be >= 0"); return PT_ERR_INVALID_ARG; }
    if (!(cfg->F >= 0.0 && cfg->F <= 2.0)) { set_error("F must be in [0, 2]"); return PT_ERR_INVALID_ARG; }
    if (!(cfg->CR >= 0.0 && cfg->CR <= 1.0)) { set_error("CR must be in [0, 1]"); return PT_ERR_INVALID_ARG; }
    if (!std::isfinite(cfg->t0)) { set_error("t0 must be finite"); return PT_ERR_INVALID_ARG; }
    if (cfg->strategy < 0 || cfg->strategy > 6) { set_error("strategy must be 1..6 (0 = DE/rand/1), got %d", cfg->strategy); return PT_ERR_INVALID_ARG; }
    if (cfg->objective != PT_OBJECTIVE_CHI2 && cfg->objective != PT_OBJECTIVE_COR) { set_error("objective must be 0 (chi^2) or 1 (correlation), got %d", cfg->objective); return PT_ERR_INVALID_ARG; }
    return PT_OK;
}

// ---------------------------------------------------------------------------------------------------
// small parity / debug kernels: same device functions as the DE kernel
// ---------------------------------------------------------------------------------------------------
template <int D>
__global__ void de_draws_kernel(const uint32_t* __restrict__ q, long long Q, uint32_t NP, uint32_t CR32, uint32_t k0,
                                uint32_t k1, int32_t* __restrict__ out) {
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= Q) return;
    const Draws d = de_draws<D>(q[3 * k + 2], q[3 * k + 1], q[3 * k + 0], NP, CR32, k0, k1);
    out[5 * k + 0] = d.r1; out[5 * k + 1] = d.r2; out[5 * k + 2] = d.r3; out[5 * k + 3] = d.jrand;
    out[5 * k + 4] = (int32_t)d.mask;
}

template <int D>
__global__ void init_population_kernel(const double* __restrict__ lo, const double* __restrict__ hi,
                                       const uint32_t* __restrict__ block_index, long long B, int NP, uint32_t k0,
                                       uint32_t k1, double* __restrict__ pop0) {
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k >= B * NP) return;
    const long long b = k / NP;
    const int i = (int)(k % NP);
    double l[D], h[D], th[D];
#pragma unroll
    for (int j = 0; j < D; ++j) { l[j] = lo[b * D + j]; h[j] = hi[b * D + j]; }
    init_member<D>((uint32_t)i, block_index ? block_index[b] : (uint32_t)b, k0, k1, l, h, th);
#pragma unroll
    for (int j = 0; j < D; ++j) pop0[k * D + j] = th[j];
}

__global__ void unpack_samples_kernel(const unsigned char* __restrict__ xq, long long row_bytes, long long B, int N, Quant q,
                                      float* __restrict__ x) {
    const long long total = B * (long long)N;
    for (long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x; k < total; k += (long long)gridDim.x * blockDim.x) {
        const long long b = k / N;
        x[k] = unpack_sample(xq + b * row_bytes, k - b * N, q);
    }
}

}  // namespace pt

using namespace pt;

extern "C" {

const char* pt_last_error_string(void) { return g_err; }
const char* pt_version(void) { return "pt 0.1 (sm_100a)"; }

size_t pt_fitness_workspace_bytes(int64_t B, int32_t N, int32_t NP, int32_t D) {
    Plan pl;
    if (check_common(B, N, 1.0, NP, D) || plan_for(B, N, NP, D, &pl, false)) return 0;
    return pl.ws_bytes;
}

int32_t pt_objective(const float* x, int64_t B, int32_t N, double fs, double t0, const float* pop, int32_t NP, int32_t D,
                     int32_t objective, float* fitness, void* workspace, size_t workspace_bytes, void* stream) {
    if (!x || !pop || !fitness) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    int rc = check_common(B, N, fs, NP, D);
    if (rc) return rc;
    if (!std::isfinite(t0)) { set_error("t0 must be finite"); return PT_ERR_INVALID_ARG; }
    if (objective != PT_OBJECTIVE_CHI2 && objective != PT_OBJECTIVE_COR) { set_error("objective must be 0 (chi^2) or 1 (correlation), got %d", objective); return PT_ERR_INVALID_ARG; }
    Plan pl;
    rc = plan_for(B, N, NP, D, &pl, true, 0, objective);
    if (rc) return rc;
    BlockParams p;
    memset(&p, 0, sizeof(p));
    p.x = x; p.pop_in = pop; p.fitness_out = fitness;
    p.B = B; p.N = N; p.Npad = pl.Npad; p.NP = NP; p.NPpad = pl.NPpad; p.G = 0;
    p.fs = fs; p.t0 = t0; p.Wg = pl.Wg; p.Ws = pl.Ws; p.strategy = kRand1;
    p.dt = 1.0 / fs; p.dtf = (float)p.dt; p.t0f = (float)t0;
    p.use_bulk = ((N % 4) == 0 && (reinterpret_cast<uintptr_t>(x) % 16) == 0) ? 1 : 0;
    rc = attach_workspace(&p, pl, workspace, workspace_bytes);
    if (rc) return rc;
    return dispatch<kModeFitness>(p, pl, D, objective, (cudaStream_t)stream);
}

int32_t pt_fitness(const float* x, int64_t B, int32_t N, double fs, double t0, const float* pop, int32_t NP, int32_t D,
                   float* fitness, void* workspace, size_t workspace_bytes, void* stream) {
    return pt_objective(x, B, N, fs, t0, pop, NP, D, PT_OBJECTIVE_CHI2, fitness, workspace, workspace_bytes, stream);
}

size_t pt_fit_blocks_workspace_bytes(int64_t B, int32_t N, const pt_de_config* cfg) {
    Plan pl;
    if (!cfg || check_common(B, N, 1.0, cfg->NP, cfg->D) || plan_for(B, N, cfg->NP, cfg->D, &pl, false, 0, cfg->objective)) return 0;
    return pl.ws_bytes;
}

int32_t pt_fit_blocks_plan(int64_t B, int32_t N, const pt_de_config* cfg, int32_t out[8]) {
    if (!cfg || !out) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    int rc = check_common(B, N, 1.0, cfg->NP, cfg->D);
    if (rc) return rc;
    Plan pl;
    rc = plan_for(B, N, cfg->NP, cfg->D, &pl, false, 0, cfg->objective);
    if (rc) return rc;
    out[7] = 0;
    if (pl.run) {
        // the plan of the FIRST launch of the launch list (run_launch_list), and the cluster size of the last one
        std::vector<Segment> segs;
        if (force_cluster() == 0 && pl.K == 1 && pl.S == 0 && run_launch_list(B, N, cfg->NP, cfg->D, pl.sms, device_smem_optin(), &segs) == 0 &&
            !segs.empty()) {
            pl = segs.front().pl;
            if (segs.size() > 1 && segs.back().pl.K > 1) out[7] = segs.back().pl.K;
        }
    } else if (have_device()) {
        Plan tl;
        if (plan_tail(B, N, cfg->NP, cfg->D, pl, &tl) > 0) out[7] = tl.K;
    }
    out[0] = pl.grid; out[1] = pl.threads; out[2] = pl.smem; out[3] = pl.resident; out[4] = pl.C; out[5] = pl.ctas_per_sm;
    out[6] = pl.K;
    return PT_OK;
}

int32_t pt_fit_blocks_launches(int64_t B, int32_t N, const pt_de_config* cfg, int32_t* out, int32_t max_launches) {
    if (!cfg || (!out && max_launches > 0)) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    int rc = check_common(B, N, 1.0, cfg->NP, cfg->D);
    if (rc) return rc;
    Plan pl;
    rc = plan_for(B, N, cfg->NP, cfg->D, &pl, false, 0, cfg->objective);
    if (rc) return rc;
    std::vector<Segment> segs;
    if (pl.run && force_cluster() == 0 && pl.K == 1 && pl.S == 0) {
        if (run_launch_list(B, N, cfg->NP, cfg->D, pl.sms, device_smem_optin(), &segs)) { set_error("no launch plan"); return PT_ERR_UNSUPPORTED; }
    } else {
        Plan tl;
        const long long rem = have_device() ? plan_tail(B, N, cfg->NP, cfg->D, pl, &tl) : 0;
        segs.push_back(Segment{0, B - rem, pl});
        if (rem > 0) segs.push_back(Segment{B - rem, rem, tl});
    }
    for (size_t k = 0; k < segs.size() && (int32_t)k < max_launches; ++k) {
        out[5 * k + 0] = (int32_t)segs[k].first; out[5 * k + 1] = (int32_t)segs[k].count; out[5 * k + 2] = segs[k].pl.grid;
        out[5 * k + 3] = segs[k].pl.threads; out[5 * k + 4] = segs[k].pl.K;
    }
    return (int32_t)segs.size();
}

static int32_t fit_blocks_impl(const float* x, const unsigned char* xq, const pt_quant* quant, int64_t row_bytes, int64_t B,
                               int32_t N, double fs, const double* lo, const double* hi, const uint32_t* block_index,
                               const pt_de_config* cfg, double* best, float* best_rss, uint32_t* status, float* final_pop,
                               float* final_fit, void* workspace, size_t workspace_bytes, void* stream,
                               const uint32_t* sel = nullptr, const int* count = nullptr) {
    // sel != null: work item j is data block sel[j] of the caller's arrays; count (device scalar) = how many items there are,
    // at most B (pt_refit_doubtful: the number of doubtful blocks is known on the device only, so the launch geometry is that
    // of B single-CTA blocks and CTAs without an item exit at once)
    if ((!x && !xq) || !lo || !hi || !best || !best_rss || !status) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_common(B, N, fs, cfg->NP, cfg->D);
    if (rc) return rc;
    BlockParams p;
    memset(&p, 0, sizeof(p));
    if (xq) {
        rc = check_quant(quant, row_bytes, N, &p.q);
        if (rc) return rc;
    }
    Plan pl;
    rc = plan_for(B, N, cfg->NP, cfg->D, &pl, true, count ? 1 : 0, cfg->objective);
    if (rc) return rc;
    p.x = x; p.xq = xq; p.row_bytes = row_bytes;
    p.lo = lo; p.hi = hi; p.block_index = block_index; p.sel = sel; p.count = count;
    p.best = best; p.best_rss = best_rss; p.status = status; p.final_pop = final_pop; p.final_fit = final_fit;
    p.B = B; p.N = N; p.Npad = pl.Npad; p.NP = cfg->NP; p.NPpad = pl.NPpad; p.G = cfg->generations;
    p.fs = fs; p.t0 = cfg->t0; p.F = cfg->F;
    p.dt = 1.0 / fs; p.dtf = (float)p.dt; p.t0f = (float)cfg->t0;
    p.CR32 = cr32_of(cfg->CR);
    p.key0 = (uint32_t)(cfg->seed & 0xFFFFFFFFull); p.key1 = (uint32_t)(cfg->seed >> 32);
    p.Wg = pl.Wg; p.Ws = pl.Ws;
    p.strategy = cfg->strategy == 0 ? kRand1 : cfg->strategy;
    p.use_bulk = (!xq && (N % 4) == 0 && (reinterpret_cast<uintptr_t>(x) % 16) == 0) ? 1 : 0;
    rc = attach_workspace(&p, pl, workspace, workspace_bytes);
    if (rc) return rc;
    if (pl.run && !count && force_cluster() == 0 && pl.K == 1 && pl.S == 0) {
        // segments of exactly full grids (run_launch_list); every launch reads its own geometry from its plan
        std::vector<Segment> segs;
        if (run_launch_list(B, N, cfg->NP, cfg->D, pl.sms, device_smem_optin(), &segs)) { set_error("no launch plan"); return PT_ERR_UNSUPPORTED; }
        for (const Segment& sg : segs) {
            BlockParams q = p;
            q.blk0 = sg.first; q.B = sg.first + sg.count;
            q.Npad = sg.pl.Npad; q.NPpad = sg.pl.NPpad; q.Wg = sg.pl.Wg; q.Ws = sg.pl.Ws;
            rc = attach_workspace(&q, sg.pl, nullptr, 0);
            if (rc) return rc;
            rc = dispatch<kModeFit>(q, sg.pl, cfg->D, cfg->objective, (cudaStream_t)stream);
            if (rc) return rc;
        }
        return PT_OK;
    }
    Plan tl;
    const long long rem = count ? 0 : plan_tail(B, N, cfg->NP, cfg->D, pl, &tl);
    if (rem == 0) return dispatch<kModeFit>(p, pl, cfg->D, cfg->objective, (cudaStream_t)stream);
    // full waves on single CTAs, then the last partial wave on clusters
    p.B = B - rem;
    rc = dispatch<kModeFit>(p, pl, cfg->D, cfg->objective, (cudaStream_t)stream);
    if (rc) return rc;
    BlockParams q = p;
    q.blk0 = B - rem; q.B = B;
    q.Wg = tl.Wg; q.Ws = tl.Ws; q.Npad = tl.Npad; q.NPpad = tl.NPpad;   // the tail plan is always pt_block_kernel's
    rc = attach_workspace(&q, tl, nullptr, 0);
    if (rc) return rc;
    return dispatch<kModeFit>(q, tl, cfg->D, cfg->objective, (cudaStream_t)stream);
}

int32_t pt_fit_blocks(const float* x, int64_t B, int32_t N, double fs, const double* lo, const double* hi,
                      const uint32_t* block_index, const pt_de_config* cfg, double* best, float* best_rss,
                      uint32_t* status, float* final_pop, float* final_fit, void* workspace, size_t workspace_bytes,
                      void* stream) {
    if (!x) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    return fit_blocks_impl(x, nullptr, nullptr, 0, B, N, fs, lo, hi, block_index, cfg, best, best_rss, status, final_pop,
                           final_fit, workspace, workspace_bytes, stream);
}

int32_t pt_fit_blocks_q(const void* xq, const pt_quant* quant, int64_t row_bytes, int64_t B, int32_t N, double fs,
                        const double* lo, const double* hi, const uint32_t* block_index, const pt_de_config* cfg,
                        double* best, float* best_rss, uint32_t* status, float* final_pop, float* final_fit,
                        void* workspace, size_t workspace_bytes, void* stream) {
    if (!xq) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    return fit_blocks_impl(nullptr, static_cast<const unsigned char*>(xq), quant, row_bytes, B, N, fs, lo, hi, block_index,
                           cfg, best, best_rss, status, final_pop, final_fit, workspace, workspace_bytes, stream);
}

int32_t pt_unpack_samples(const void* xq, const pt_quant* quant, int64_t row_bytes, int64_t B, int32_t N, float* x,
                          void* stream) {
    if (!xq || !x) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if (B < 1 || N < 1) { set_error("B and N must be >= 1"); return PT_ERR_INVALID_ARG; }
    Quant q;
    int rc = check_quant(quant, row_bytes, N, &q);
    if (rc) return rc;
    const long long total = B * (long long)N;
    const int thr = 256;
    const unsigned grid = (unsigned)std::min<long long>((total + thr - 1) / thr, 148LL * 16);
    unpack_samples_kernel<<<grid, thr, 0, (cudaStream_t)stream>>>(static_cast<const unsigned char*>(xq), row_bytes, B, N, q, x);
    if (check_cuda(cudaGetLastError(), "unpack_samples_kernel launch")) return PT_ERR_CUDA;
    return PT_OK;
}

int32_t pt_acquire(const float* x, int64_t B, int32_t N, double fs, int32_t D, const pt_acq_config* acq, double* est,
                   double* lo, double* hi, void* stream) {
    if (!x || !acq || !est || !lo || !hi) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if (B < 1 || N < 8 || !(fs > 0.0) || (D != 5 && D != 6)) { set_error("invalid B, N, fs or D"); return PT_ERR_INVALID_ARG; }
    const int M = acq->M;
    if (M < 8 || (M & (M - 1))) { set_error("acq.M must be a power of two >= 8 (got %d)", M); return PT_ERR_INVALID_ARG; }
    if (M > 8192) { set_error("acq.M = %d exceeds the compiled limit 8192", M); return PT_ERR_UNSUPPORTED; }
    if (acq->spacing < 1 || (long long)M + 2LL * acq->spacing > N) { set_error("pieces do not fit: M + 2 spacing must be <= N"); return PT_ERR_INVALID_ARG; }
    const double v[6] = {acq->f_rel, acq->f_bins, acq->fdot_bins, acq->a_rel, acq->a1_rel, acq->fddot_hw};
    for (int k = 0; k < 6; ++k)
        if (!(v[k] >= 0.0) || !std::isfinite(v[k])) { set_error("acq half-widths must be finite and >= 0"); return PT_ERR_INVALID_ARG; }
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) { (void)cudaGetLastError(); set_error("no CUDA device"); return PT_ERR_CUDA; }
    if (acquire_launch(x, B, N, fs, D, acq, est, lo, hi, (cudaStream_t)stream)) return PT_ERR_CUDA;
    return PT_OK;
}

static void refit_layout(int64_t B, size_t fit_ws, size_t* o_pb, size_t* o_tp, size_t* o_flags, size_t* o_list, size_t* o_cnt,
                         size_t* o_fit, size_t* total) {
    size_t off = 0;
    auto take = [&off](size_t bytes) { size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
    *o_pb = take((size_t)B * 10 * 8); *o_tp = take((size_t)B * 8); *o_flags = take((size_t)B * 4); *o_list = take((size_t)B * 4);
    *o_cnt = take(sizeof(int));
    *o_fit = take(fit_ws);
    *total = off;
}

// workspace of the re-fit launches: the plan of B single-CTA blocks (see fit_blocks_impl, count != null)
static size_t refit_fit_workspace_bytes(int64_t B, int32_t N, const pt_de_config* cfg) {
    Plan pl;
    if (!cfg || check_common(B, N, 1.0, cfg->NP, cfg->D) || plan_for(B, N, cfg->NP, cfg->D, &pl, false, 1, cfg->objective)) return 0;
    return pl.ws_bytes;
}

size_t pt_refit_doubtful_workspace_bytes(int64_t B, int32_t N, const pt_de_config* cfg) {
    if (!cfg || B < 1) return 0;
    size_t a, b, c, d, e, f, total;
    refit_layout(B, refit_fit_workspace_bytes(B, N, cfg), &a, &b, &c, &d, &e, &f, &total);
    return total;
}

int32_t pt_refit_doubtful(const float* x, int64_t B, int32_t N, double fs, double* lo, double* hi, const uint32_t* block_index,
                          const pt_de_config* cfg, const pt_retry_config* retry, double* best, float* best_rss,
                          uint32_t* status, int32_t* attempts, void* workspace, size_t workspace_bytes, void* stream) {
    if (!x || !lo || !hi || !best || !best_rss || !status || !attempts || !retry) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_common(B, N, fs, cfg->NP, cfg->D);
    if (rc) return rc;
    if (!(retry->phi_tol > 0.0) || !(retry->F_tol > 0.0) || retry->max_attempts < 0 || retry->max_attempts > 16 ||
        !(retry->grow >= 1.0) || !(retry->f_floor >= 0.0) || !(retry->fdot_floor >= 0.0) || !(retry->a_rel >= 0.0) ||
        !std::isfinite(retry->phi_tol + retry->F_tol + retry->grow + retry->f_floor + retry->fdot_floor + retry->a_rel)) {
        set_error("invalid retry configuration");
        return PT_ERR_INVALID_ARG;
    }
    const size_t fit_ws = refit_fit_workspace_bytes(B, N, cfg);
    size_t o_pb, o_tp, o_flags, o_list, o_cnt, o_fit, total;
    refit_layout(B, fit_ws, &o_pb, &o_tp, &o_flags, &o_list, &o_cnt, &o_fit, &total);
    if (!workspace || workspace_bytes < total) { set_error("pt_refit_doubtful needs %zu bytes of workspace, got %zu", total, workspace ? workspace_bytes : (size_t)0); return PT_ERR_UNSUPPORTED; }
    if (reinterpret_cast<uintptr_t>(workspace) % 16) { set_error("workspace must be 16-byte aligned"); return PT_ERR_INVALID_ARG; }
    int dev_count = 0;
    if (cudaGetDeviceCount(&dev_count) != cudaSuccess || dev_count == 0) { (void)cudaGetLastError(); set_error("no CUDA device"); return PT_ERR_CUDA; }
    unsigned char* ws = static_cast<unsigned char*>(workspace);
    double* per_block = reinterpret_cast<double*>(ws + o_pb);
    double* total_phase = reinterpret_cast<double*>(ws + o_tp);
    uint32_t* flags = reinterpret_cast<uint32_t*>(ws + o_flags);
    uint32_t* list = reinterpret_cast<uint32_t*>(ws + o_list);
    int* count = reinterpret_cast<int*>(ws + o_cnt);
    cudaStream_t st = (cudaStream_t)stream;
    const int D = cfg->D;
    const double T = (double)N / fs;
    if (check_cuda(cudaMemsetAsync(attempts, 0, (size_t)B * sizeof(int32_t), st), "cudaMemsetAsync")) return PT_ERR_CUDA;
    // Eq. 8 residuals of the current solution -> flags of the doubtful blocks -> their ordered list and its length, all on the device
    auto flag_blocks = [&]() -> int {
        if (doppler_launch(best, B, D, T, 0.0, nullptr, 0, per_block, total_phase, nullptr, st)) return PT_ERR_CUDA;
        if (check_cuda(cudaGetLastError(), "doppler kernels launch")) return PT_ERR_CUDA;
        if (retry_flag_launch(per_block, B, retry->phi_tol, retry->F_tol, flags, st)) return PT_ERR_CUDA;
        if (retry_compact_launch(flags, B, list, count, st)) return PT_ERR_CUDA;
        return PT_OK;
    };
    // Every attempt is enqueued unconditionally: with no doubtful block left its kernels find *count == 0 and do nothing
    // (a few launch latencies), which is what lets the call stay asynchronous.
    double g = 1.0;
    for (int a = 1; a <= retry->max_attempts; ++a, g *= retry->grow) {
        rc = flag_blocks();
        if (rc) return rc;
        if (retry_box_launch(flags, best, lo, hi, B, D, T, g, retry, st)) return PT_ERR_CUDA;
        pt_de_config c = *cfg;
        c.seed = cfg->seed + (uint64_t)a * 0x9E3779B97F4A7C15ull;
        rc = fit_blocks_impl(x, nullptr, nullptr, 0, B, N, fs, lo, hi, block_index, &c, best, best_rss, status, nullptr, nullptr,
                             fit_ws ? ws + o_fit : nullptr, fit_ws, st, list, count);
        if (rc) return rc;
        if (retry_count_launch(list, count, B, attempts, st)) return PT_ERR_CUDA;
    }
    rc = flag_blocks();
    if (rc) return rc;
    if (retry->max_attempts > 0)
        if (retry_abandon_launch(flags, B, status, st)) return PT_ERR_CUDA;
    return PT_OK;
}

int32_t pt_doppler_products(const double* best, int64_t B, int32_t D, double T, double los_scale,
                            const int32_t* blocks_per_interval, int32_t n_intervals, double* per_block,
                            double* total_phase, double* const* interval_out, void* stream) {
    if (!best || !per_block || !total_phase) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if (B < 1 || (D != 5 && D != 6) || !(T > 0.0) || n_intervals < 0) { set_error("invalid B, D, T or n_intervals"); return PT_ERR_INVALID_ARG; }
    if (n_intervals > 0 && (!blocks_per_interval || !interval_out)) { set_error("null interval arguments"); return PT_ERR_INVALID_ARG; }
    for (int k = 0; k < n_intervals; ++k) {
        if (blocks_per_interval[k] < 1) { set_error("blocks_per_interval[%d] must be >= 1", k); return PT_ERR_INVALID_ARG; }
        if (B / blocks_per_interval[k] > 0 && !interval_out[k]) { set_error("interval_out[%d] is null", k); return PT_ERR_INVALID_ARG; }
    }
    doppler_launch(best, B, D, T, los_scale, blocks_per_interval, n_intervals, per_block, total_phase, interval_out,
                   (cudaStream_t)stream);
    if (check_cuda(cudaGetLastError(), "doppler kernels launch")) return PT_ERR_CUDA;
    return PT_OK;
}

int32_t pt_de_draws(const uint32_t* query, int64_t Q, int32_t NP, int32_t D, double CR, uint64_t seed, int32_t* out,
                    void* stream) {
    if (!query || !out) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if (Q < 1 || NP < 4 || (D != 5 && D != 6) || !(CR >= 0.0 && CR <= 1.0)) { set_error("invalid Q, NP, D or CR"); return PT_ERR_INVALID_ARG; }
    const int thr = 128;
    const unsigned grid = (unsigned)((Q + thr - 1) / thr);
    const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    if (D == 5) de_draws_kernel<5><<<grid, thr, 0, (cudaStream_t)stream>>>(query, Q, (uint32_t)NP, cr32_of(CR), k0, k1, out);
    else de_draws_kernel<6><<<grid, thr, 0, (cudaStream_t)stream>>>(query, Q, (uint32_t)NP, cr32_of(CR), k0, k1, out);
    if (check_cuda(cudaGetLastError(), "de_draws_kernel launch")) return PT_ERR_CUDA;
    return PT_OK;
}

int32_t pt_init_population(const double* lo, const double* hi, const uint32_t* block_index, int64_t B, int32_t NP,
                           int32_t D, uint64_t seed, double* pop0, void* stream) {
    if (!lo || !hi || !pop0) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if (B < 1 || NP < 1 || (D != 5 && D != 6)) { set_error("invalid B, NP or D"); return PT_ERR_INVALID_ARG; }
    const int thr = 128;
    const unsigned grid = (unsigned)((B * NP + thr - 1) / thr);
    const uint32_t k0 = (uint32_t)(seed & 0xFFFFFFFFull), k1 = (uint32_t)(seed >> 32);
    if (D == 5) init_population_kernel<5><<<grid, thr, 0, (cudaStream_t)stream>>>(lo, hi, block_index, B, NP, k0, k1, pop0);
    else init_population_kernel<6><<<grid, thr, 0, (cudaStream_t)stream>>>(lo, hi, block_index, B, NP, k0, k1, pop0);
    if (check_cuda(cudaGetLastError(), "init_population_kernel launch")) return PT_ERR_CUDA;
    return PT_OK;
}

static int32_t track_host_impl(const float* x, const void* xq, const pt_quant* quant, int64_t row_bytes, int64_t B, int32_t N,
                               double fs, const double* lo, const double* hi, const pt_de_config* cfg, double los_scale,
                               const int32_t* blocks_per_interval, int32_t n_intervals, double* best, float* best_rss,
                               uint32_t* status, double* per_block, double* total_phase, double* const* interval_out,
                               const pt_acq_config* acq = nullptr, const pt_retry_config* retry = nullptr,
                               double* lo_out = nullptr, double* hi_out = nullptr, int32_t* attempts = nullptr) {
    // acq != null: the ranges come from pt_acquire (lo, hi are not read); retry != null: pt_refit_doubtful after the fit
    if ((!x && !xq) || (!acq && (!lo || !hi))) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    if ((acq || retry) && xq) { set_error("acquisition and re-search take fp32 samples"); return PT_ERR_UNSUPPORTED; }
    if (xq) {
        Quant qq;
        const int rq = check_quant(quant, row_bytes, N, &qq);
        if (rq) return rq;
    }
    int rc = check_cfg(cfg);
    if (rc) return rc;
    rc = check_common(B, N, fs, cfg->NP, cfg->D);
    if (rc) return rc;
    if (n_intervals < 0 || (n_intervals > 0 && (!blocks_per_interval || !interval_out))) { set_error("invalid interval arguments"); return PT_ERR_INVALID_ARG; }
    for (long long k = 0; !acq && k < B * cfg->D; ++k)
        if (!(lo[k] <= hi[k])) { set_error("lo > hi at element %lld", k); return PT_ERR_INVALID_ARG; }
    const int D = cfg->D;
    const size_t nx = xq ? (size_t)B * (size_t)row_bytes : (size_t)B * N * sizeof(float), nbox = (size_t)B * D * sizeof(double);
    // one device arena for everything
    size_t off = 0;
    auto take = [&off](size_t bytes) { size_t o = off; off += (bytes + 255) / 256 * 256; return o; };
    const size_t o_x = take(nx), o_lo = take(nbox), o_hi = take(nbox), o_best = take(nbox);
    const size_t o_rss = take((size_t)B * 4), o_st = take((size_t)B * 4), o_pb = take((size_t)B * 10 * 8), o_tp = take((size_t)B * 8);
    const size_t ws_bytes = pt_fit_blocks_workspace_bytes(B, N, cfg);
    const size_t o_ws = take(ws_bytes);
    const size_t o_est = take(acq ? (size_t)B * 8 * 8 : 0), o_att = take(retry ? (size_t)B * 4 : 0);
    const size_t rws_bytes = retry ? pt_refit_doubtful_workspace_bytes(B, N, cfg) : 0;
    const size_t o_rws = take(rws_bytes);
    std::vector<size_t> o_iv(n_intervals);
    std::vector<long long> cnt(n_intervals);
    for (int k = 0; k < n_intervals; ++k) {
        if (blocks_per_interval[k] < 1) { set_error("blocks_per_interval[%d] must be >= 1", k); return PT_ERR_INVALID_ARG; }
        cnt[k] = B / blocks_per_interval[k];
        o_iv[k] = take((size_t)(cnt[k] > 0 ? cnt[k] : 1) * 16);
    }
    cudaMemPool_t pool;
    cudaStream_t st = nullptr;
    if (host_cache_get(&pool, &st)) return PT_ERR_CUDA;
    unsigned char* arena = nullptr;
    if (check_cuda(cudaMallocFromPoolAsync(reinterpret_cast<void**>(&arena), off, pool, st), "cudaMallocFromPoolAsync")) return PT_ERR_CUDA;
    int ret = PT_OK;
    std::vector<double*> d_iv(n_intervals > 0 ? n_intervals : 1, nullptr);
    for (int k = 0; k < n_intervals; ++k) d_iv[k] = reinterpret_cast<double*>(arena + o_iv[k]);
    do {
        if (check_cuda(cudaMemcpyAsync(arena + o_x, xq ? xq : static_cast<const void*>(x), nx, cudaMemcpyHostToDevice, st), "H2D x")) { ret = PT_ERR_CUDA; break; }
        if (acq) {
            ret = pt_acquire(reinterpret_cast<float*>(arena + o_x), B, N, fs, D, acq, reinterpret_cast<double*>(arena + o_est),
                             reinterpret_cast<double*>(arena + o_lo), reinterpret_cast<double*>(arena + o_hi), st);
            if (ret) break;
        } else {
            if (check_cuda(cudaMemcpyAsync(arena + o_lo, lo, nbox, cudaMemcpyHostToDevice, st), "H2D lo")) { ret = PT_ERR_CUDA; break; }
            if (check_cuda(cudaMemcpyAsync(arena + o_hi, hi, nbox, cudaMemcpyHostToDevice, st), "H2D hi")) { ret = PT_ERR_CUDA; break; }
        }
        ret = fit_blocks_impl(xq ? nullptr : reinterpret_cast<float*>(arena + o_x), xq ? arena + o_x : nullptr, quant, row_bytes, B,
                              N, fs, reinterpret_cast<double*>(arena + o_lo), reinterpret_cast<double*>(arena + o_hi), nullptr,
                              cfg, reinterpret_cast<double*>(arena + o_best), reinterpret_cast<float*>(arena + o_rss),
                              reinterpret_cast<uint32_t*>(arena + o_st), nullptr, nullptr, ws_bytes ? arena + o_ws : nullptr,
                              ws_bytes, st);
        if (ret) break;
        if (retry) {
            ret = pt_refit_doubtful(reinterpret_cast<float*>(arena + o_x), B, N, fs, reinterpret_cast<double*>(arena + o_lo),
                                    reinterpret_cast<double*>(arena + o_hi), nullptr, cfg, retry,
                                    reinterpret_cast<double*>(arena + o_best), reinterpret_cast<float*>(arena + o_rss),
                                    reinterpret_cast<uint32_t*>(arena + o_st), reinterpret_cast<int32_t*>(arena + o_att),
                                    arena + o_rws, rws_bytes, st);
            if (ret) break;
        }
        ret = pt_doppler_products(reinterpret_cast<double*>(arena + o_best), B, D, (double)N / fs, los_scale,
                                  blocks_per_interval, n_intervals, reinterpret_cast<double*>(arena + o_pb),
                                  reinterpret_cast<double*>(arena + o_tp), d_iv.data(), st);
        if (ret) break;
        cudaError_t e = cudaSuccess;
        if (best) e = cudaMemcpyAsync(best, arena + o_best, nbox, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && best_rss) e = cudaMemcpyAsync(best_rss, arena + o_rss, (size_t)B * 4, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && status) e = cudaMemcpyAsync(status, arena + o_st, (size_t)B * 4, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && per_block) e = cudaMemcpyAsync(per_block, arena + o_pb, (size_t)B * 80, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && total_phase) e = cudaMemcpyAsync(total_phase, arena + o_tp, (size_t)B * 8, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && lo_out) e = cudaMemcpyAsync(lo_out, arena + o_lo, nbox, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && hi_out) e = cudaMemcpyAsync(hi_out, arena + o_hi, nbox, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess && attempts && retry) e = cudaMemcpyAsync(attempts, arena + o_att, (size_t)B * 4, cudaMemcpyDeviceToHost, st);
        for (int k = 0; k < n_intervals && e == cudaSuccess; ++k)
            if (cnt[k] > 0 && interval_out[k])
                e = cudaMemcpyAsync(interval_out[k], arena + o_iv[k], (size_t)cnt[k] * 16, cudaMemcpyDeviceToHost, st);
        if (check_cuda(e, "D2H results")) { ret = PT_ERR_CUDA; break; }
        if (check_cuda(cudaStreamSynchronize(st), "pt_track_host")) { ret = PT_ERR_CUDA; break; }
    } while (0);
    if (ret != PT_OK) cudaStreamSynchronize(st);
    cudaFreeAsync(arena, st);            // back to the pool (kept for the next call); ordered after everything above
    return ret;
}

int32_t pt_host_cache_release(void) {
    std::lock_guard<std::mutex> lock(g_dev_mutex);
    int rc = PT_OK;
    int cur = 0;
    if (cudaGetDevice(&cur) != cudaSuccess) { (void)cudaGetLastError(); return PT_OK; }      // no device: nothing was ever cached
    for (int dev = 0; dev < kMaxDevices; ++dev) {
        HostCache& c = g_host_cache[dev];
        if (!c.ready) continue;
        cudaSetDevice(dev);
        if (cudaStreamSynchronize(c.stream) != cudaSuccess) rc = PT_ERR_CUDA;
        cudaStreamDestroy(c.stream);
        cudaMemPoolDestroy(c.pool);
        c.ready = 0;
    }
    cudaSetDevice(cur);
    return rc;
}

int32_t pt_track_host(const float* x, int64_t B, int32_t N, double fs, const double* lo, const double* hi,
                      const pt_de_config* cfg, double los_scale, const int32_t* blocks_per_interval, int32_t n_intervals,
                      double* best, float* best_rss, uint32_t* status, double* per_block, double* total_phase,
                      double* const* interval_out) {
    if (!x) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    return track_host_impl(x, nullptr, nullptr, 0, B, N, fs, lo, hi, cfg, los_scale, blocks_per_interval, n_intervals, best,
                           best_rss, status, per_block, total_phase, interval_out);
}

int32_t pt_track_auto_host(const float* x, int64_t B, int32_t N, double fs, const pt_de_config* cfg, const pt_acq_config* acq,
                           const pt_retry_config* retry, double los_scale, const int32_t* blocks_per_interval,
                           int32_t n_intervals, double* lo, double* hi, double* best, float* best_rss, uint32_t* status,
                           int32_t* attempts, double* per_block, double* total_phase, double* const* interval_out) {
    if (!x || !acq) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    return track_host_impl(x, nullptr, nullptr, 0, B, N, fs, nullptr, nullptr, cfg, los_scale, blocks_per_interval, n_intervals,
                           best, best_rss, status, per_block, total_phase, interval_out, acq, retry, lo, hi, attempts);
}

int32_t pt_track_host_q(const void* xq, const pt_quant* quant, int64_t row_bytes, int64_t B, int32_t N, double fs,
                        const double* lo, const double* hi, const pt_de_config* cfg, double los_scale,
                        const int32_t* blocks_per_interval, int32_t n_intervals, double* best, float* best_rss,
                        uint32_t* status, double* per_block, double* total_phase, double* const* interval_out) {
    if (!xq) { set_error("null pointer argument"); return PT_ERR_INVALID_ARG; }
    return track_host_impl(nullptr, xq, quant, row_bytes, B, N, fs, lo, hi, cfg, los_scale, blocks_per_interval, n_intervals,
                           best, best_rss, status, per_block, total_phase, interval_out);
}

}  // extern "C"
