// pt_retry.cu -- continuity check and run-time ranges of the re-search of doubtful blocks (section 3.1.1,
// :226-248 section 3.1.3 Eq. 8, :252 section 3.1.4; reading R25).  Small fp64 kernels, one thread per block;
// pt_refit_doubtful in pt_api.cu strings them together with the DE kernel, all on the caller's stream (no host round trip).
#include <cmath>

#include "pt_internal.h"

namespace pt {

// Border j (between blocks j and j+1) is bad if the phase or frequency residual of Eq. 8 exceeds its threshold;
// a block is doubtful if every border it has is bad.  per_block is pt_doppler_products' [B][10] output:
// column 8 = wrapped phase residual to block b+1 [rad], column 9 = frequency residual [rad/s].
__global__ void retry_flag_kernel(const double* __restrict__ per_block, long long B, double phi_tol, double F_tol_rad,
                                  uint32_t* __restrict__ flags) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B) return;
    auto bad = [&](long long j) {
        return fabs(per_block[j * 10 + 8]) > phi_tol || fabs(per_block[j * 10 + 9]) > F_tol_rad;
    };
    int borders = 0, bad_borders = 0;
    if (b > 0) { ++borders; bad_borders += bad(b - 1) ? 1 : 0; }
    if (b < B - 1) { ++borders; bad_borders += bad(b) ? 1 : 0; }
    flags[b] = (borders > 0 && bad_borders == borders) ? 1u : 0u;
}

// New ranges of every doubtful block from the nearest trusted block n (left on equal distance), k = b - n:
//   F(t) = f + fdot t + fddot t^2/2,  F'(t) = fdot + fddot t  of block n,
//   f    in mid[F((k-1/2)T), F((k+1/2)T)] -+ g max(half their distance, f_floor)
//   fdot in mid[F'((k-1/2)T), F'((k+1/2)T)] -+ g max(half their distance, fdot_floor)
//   a0   in a0^n (1 -+ g a_rel)
//   phi0 in [-pi, pi]; a1 and fddot keep their ranges
// With no trusted block at all, the block's own box is widened by `grow` about its centre.
__global__ void retry_box_kernel(const uint32_t* __restrict__ flags, const double* __restrict__ best, double* __restrict__ lo,
                                 double* __restrict__ hi, long long B, int D, double T, double g, double grow, double f_floor,
                                 double fdot_floor, double a_rel) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B || !flags[b]) return;
    long long nl = b - 1, nr = b + 1;
    while (nl >= 0 && flags[nl]) --nl;
    while (nr < B && flags[nr]) ++nr;
    double* l = lo + b * D;
    double* h = hi + b * D;
    if (nl < 0 && nr >= B) {
        for (int j = 0; j < D; ++j) {
            const double c = 0.5 * (l[j] + h[j]), w = 0.5 * (h[j] - l[j]) * grow;
            l[j] = c - w; h[j] = c + w;
        }
        return;
    }
    const long long n = (nl >= 0 && (nr >= B || b - nl <= nr - b)) ? nl : nr;
    const double k = (double)(b - n);
    const double* th = best + n * D;
    const double a0 = th[0], f = th[3], fdot = th[4], fddot = (D == 6) ? th[5] : 0.0;
    const double t1 = (k - 0.5) * T, t2 = (k + 0.5) * T;
    const double e1 = f + fdot * t1 + fddot * t1 * t1 / 2.0, e2 = f + fdot * t2 + fddot * t2 * t2 / 2.0;
    const double d1 = fdot + fddot * t1, d2 = fdot + fddot * t2;
    double hw = g * fmax(fabs(e2 - e1) / 2.0, f_floor);
    l[3] = (e1 + e2) / 2.0 - hw; h[3] = (e1 + e2) / 2.0 + hw;
    hw = g * fmax(fabs(d2 - d1) / 2.0, fdot_floor);
    l[4] = (d1 + d2) / 2.0 - hw; h[4] = (d1 + d2) / 2.0 + hw;
    double al = a0 * (1.0 - g * a_rel), ah = a0 * (1.0 + g * a_rel);
    if (al > ah) { const double tmp = al; al = ah; ah = tmp; }
    l[0] = al; h[0] = ah;
    l[2] = -kPi; h[2] = kPi;
}

// Ordered compaction of the doubtful blocks: list[0 .. *count) = ascending indices b with flags[b] != 0.  One CTA walks the
// flags in chunks of its size with a block-wide exclusive scan (B is a few 10^4: a few dozen trips), so the list is in the same
// order a host loop would produce and no host round trip is needed.
__global__ void __launch_bounds__(1024) retry_compact_kernel(const uint32_t* __restrict__ flags, long long B, uint32_t* __restrict__ list,
                                                             int* __restrict__ count) {
    __shared__ int warp_tot[32];
    __shared__ int base;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) base = 0;
    __syncthreads();
    for (long long b0 = 0; b0 < B; b0 += blockDim.x) {
        const long long b = b0 + tid;
        const int f = (b < B && flags[b]) ? 1 : 0;
        int incl = f;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const int v = __shfl_up_sync(0xffffffffu, incl, off);
            if (lane >= off) incl += v;
        }
        if (lane == 31) warp_tot[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int t = warp_tot[lane];
#pragma unroll
            for (int off = 1; off < 32; off <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, t, off);
                if (lane >= off) t += v;
            }
            warp_tot[lane] = t;      // inclusive totals of the warps
        }
        __syncthreads();
        const int before = base + (warp > 0 ? warp_tot[warp - 1] : 0) + incl - f;
        if (f) list[before] = (uint32_t)b;
        __syncthreads();
        if (tid == 0) base += warp_tot[31];
        __syncthreads();
    }
    if (tid == 0) *count = base;
}

__global__ void retry_count_kernel(const uint32_t* __restrict__ sel, const int* __restrict__ n, long long B, int32_t* __restrict__ attempts) {
    const long long k = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (k < B && k < *n) attempts[sel[k]] += 1;
}

__global__ void retry_abandon_kernel(const uint32_t* __restrict__ flags, long long B, uint32_t* __restrict__ status) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b < B && flags[b]) status[b] |= 4u;
}

static unsigned grid_for(long long n) { return (unsigned)((n + 127) / 128); }

int retry_flag_launch(const double* per_block, long long B, double phi_tol, double F_tol_hz, uint32_t* flags, cudaStream_t st) {
    retry_flag_kernel<<<grid_for(B), 128, 0, st>>>(per_block, B, phi_tol, 2.0 * kPi * F_tol_hz, flags);
    return check_cuda(cudaGetLastError(), "retry_flag_kernel launch");
}

int retry_box_launch(const uint32_t* flags, const double* best, double* lo, double* hi, long long B, int D, double T, double g,
                     const pt_retry_config* rc, cudaStream_t st) {
    retry_box_kernel<<<grid_for(B), 128, 0, st>>>(flags, best, lo, hi, B, D, T, g, rc->grow, rc->f_floor, rc->fdot_floor,
                                                   rc->a_rel);
    return check_cuda(cudaGetLastError(), "retry_box_kernel launch");
}

int retry_compact_launch(const uint32_t* flags, long long B, uint32_t* list, int* count, cudaStream_t st) {
    retry_compact_kernel<<<1, 1024, 0, st>>>(flags, B, list, count);
    return check_cuda(cudaGetLastError(), "retry_compact_kernel launch");
}

int retry_count_launch(const uint32_t* sel, const int* n, long long B, int32_t* attempts, cudaStream_t st) {
    retry_count_kernel<<<grid_for(B), 128, 0, st>>>(sel, n, B, attempts);
    return check_cuda(cudaGetLastError(), "retry_count_kernel launch");
}

int retry_abandon_launch(const uint32_t* flags, long long B, uint32_t* status, cudaStream_t st) {
    retry_abandon_kernel<<<grid_for(B), 128, 0, st>>>(flags, B, status);
    return check_cuda(cudaGetLastError(), "retry_abandon_kernel launch");
}

}  // namespace pt
