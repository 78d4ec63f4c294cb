// pt_doppler.cu -- Doppler products from the fitted parameters, fp64.
//   phi(t) = phi0 + 2 pi (f t + fdot t^2/2 + fddot t^3/6), F(t) = dphi/dt [rad/s]      PAPER.md:228-234 (Eq. 7)
//   border phases / frequencies at t = -T/2, +T/2 and their continuity residuals          PAPER.md:237-246 (Eq. 8)
//   dphi_block = phi(T/2) - phi(-T/2); total-count phase; Phi_total, F_int over m blocks   PAPER.md:343-351 (Eq. 16-17)
//   a_los = los_scale * fdot                                                              PAPER.md:376-378 (Eq. 19)
// The total phase reaches 5e7 rad and is wanted to mrad, hence fp64 everywhere.
#include "pt_internal.h"

namespace pt {

__device__ __forceinline__ double phase_at(const double* th, int D, double t) {
    const double fddot = (D >= 6) ? th[5] : 0.0;
    return th[2] + kTwoPi * (th[3] * t + th[4] * t * t / 2.0 + fddot * t * t * t / 6.0);
}
__device__ __forceinline__ double freq_at(const double* th, int D, double t) {
    const double fddot = (D >= 6) ? th[5] : 0.0;
    return kTwoPi * (th[3] + th[4] * t + fddot * t * t / 2.0);
}
__device__ __forceinline__ double mod_2pi(double v) {
    double r = fmod(v, kTwoPi);
    if (r < 0.0) r += kTwoPi;
    if (r >= kTwoPi) r -= kTwoPi;
    return r;
}
__device__ __forceinline__ double wrap_pi(double v) {   // to (-pi, pi]
    double r = fmod(v, kTwoPi);
    if (r <= -kPi) r += kTwoPi;
    if (r > kPi) r -= kTwoPi;
    return r;
}

// one thread per block: the ten per-block columns
__global__ void doppler_per_block_kernel(const double* __restrict__ best, long long B, int D, double T, double los_scale,
                                         double* __restrict__ per_block) {
    const long long b = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (b >= B) return;
    double th[6] = {0, 0, 0, 0, 0, 0};
    for (int j = 0; j < D; ++j) th[j] = best[b * D + j];
    const double pl = phase_at(th, D, -0.5 * T), pr = phase_at(th, D, 0.5 * T);
    double* o = per_block + b * 10;
    o[0] = th[3];
    o[1] = th[4];
    o[2] = los_scale * th[4];
    o[3] = mod_2pi(pl);
    o[4] = mod_2pi(pr);
    o[5] = freq_at(th, D, -0.5 * T);
    const double fr = freq_at(th, D, 0.5 * T);
    o[6] = fr;
    o[7] = pr - pl;
    if (b + 1 < B) {
        double nx[6] = {0, 0, 0, 0, 0, 0};
        for (int j = 0; j < D; ++j) nx[j] = best[(b + 1) * D + j];
        o[8] = wrap_pi(phase_at(nx, D, -0.5 * T) - pr);
        o[9] = freq_at(nx, D, -0.5 * T) - fr;
    } else {
        o[8] = nan("");
        o[9] = nan("");
    }
}

// inclusive running sum of dphi_block (column 7) over all B blocks: one CTA, each thread owns a contiguous
// run of blocks, CTA-wide scan of the run totals, then the runs are replayed with their offsets.
__global__ void __launch_bounds__(1024, 1) doppler_scan_kernel(const double* __restrict__ per_block, long long B,
                                                               double* __restrict__ total_phase) {
    __shared__ double warp_tot[32];
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const long long per = (B + nthr - 1) / nthr;
    const long long lo = min(B, (long long)tid * per), hi = min(B, lo + per);
    double s = 0.0;
    for (long long b = lo; b < hi; ++b) s += per_block[b * 10 + 7];
    double incl = s;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        const double o = __shfl_up_sync(0xffffffffu, incl, off);
        if (lane >= off) incl += o;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        double w = (lane < (nthr >> 5)) ? warp_tot[lane] : 0.0;
#pragma unroll
        for (int off = 1; off < 32; off <<= 1) {
            const double o = __shfl_up_sync(0xffffffffu, w, off);
            if (lane >= off) w += o;
        }
        warp_tot[lane] = w;
    }
    __syncthreads();
    double run = (incl - s) + (warp > 0 ? warp_tot[warp - 1] : 0.0);
    for (long long b = lo; b < hi; ++b) {
        run += per_block[b * 10 + 7];
        total_phase[b] = run;
    }
}

// Phi_total and F_int of each run of m blocks (Eq. 16-17): one thread per interval, sequential sum.
__global__ void doppler_interval_kernel(const double* __restrict__ per_block, long long count, int m, double T,
                                        double* __restrict__ out) {
    const long long j = blockIdx.x * (long long)blockDim.x + threadIdx.x;
    if (j >= count) return;
    double s = 0.0;
    for (int q = 0; q < m; ++q) s += per_block[(j * m + q) * 10 + 7];
    out[2 * j + 0] = s;
    out[2 * j + 1] = s / ((double)m * T);
}

int doppler_launch(const double* best, long long B, int D, double T, double los_scale, const int32_t* m, int n_intervals,
                   double* per_block, double* total_phase, double* const* interval_out, cudaStream_t st) {
    const int thr = 256;
    doppler_per_block_kernel<<<(unsigned)((B + thr - 1) / thr), thr, 0, st>>>(best, B, D, T, los_scale, per_block);
    doppler_scan_kernel<<<1, 1024, 0, st>>>(per_block, B, total_phase);
    for (int k = 0; k < n_intervals; ++k) {
        const long long count = B / m[k];
        if (count > 0)
            doppler_interval_kernel<<<(unsigned)((count + thr - 1) / thr), thr, 0, st>>>(per_block, count, m[k], T,
                                                                                         interval_out[k]);
    }
    return 0;
}

}  // namespace pt
