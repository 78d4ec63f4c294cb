// pt_acquire.cu -- initial range determination (section 3.1.1 items 1-6; reading R24):
// per data block, three Hann-windowed FFTs of M-sample pieces around the block centre give the centre frequency and
// amplitude (peak of |X|^2, log-parabolic refinement) and, by central difference, the frequency rate; the boxes the DE
// fit searches follow the paper's percentages.  One CTA per data block, all blocks in parallel (the step is independent
// per block); the FFT is an in-place radix-2 decimation-in-time transform in shared memory, fp32 butterflies with
// sincospif twiddles, the refinement and the boxes in fp64.
#include <cmath>

#include "../../include/pt.h"
#include "pt_device.cuh"
#include "pt_internal.h"

namespace pt {

struct AcqParams {
    const float* x;      // [B][N]
    double* est;         // [B][8]
    double* lo;          // [B][D]
    double* hi;          // [B][D]
    long long B;
    int N, D, M, logM, S;
    double fs, f_rel, f_bins, fdot_bins, a_rel, a1_rel, fddot_hw;
};

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
    return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x));
}

__global__ void __launch_bounds__(256) acquire_kernel(const AcqParams p) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float2* buf = reinterpret_cast<float2*>(smem_raw);
    __shared__ float s_val[8];
    __shared__ int s_idx[8];
    __shared__ double s_f[3], s_a[3];
    __shared__ int s_k[3];
    const int tid = threadIdx.x, nthr = blockDim.x, lane = tid & 31, warp = tid >> 5;
    const int M = p.M;
    for (long long b = blockIdx.x; b < p.B; b += gridDim.x) {
        const float* xb = p.x + b * (long long)p.N;
        for (int piece = 0; piece < 3; ++piece) {
            const int i0 = p.N / 2 + (piece - 1) * p.S - M / 2;
            // periodic Hann window, bit-reversed store
            for (int m = tid; m < M; m += nthr) {
                const float w = 0.5f - 0.5f * cospif(2.0f * (float)m / (float)M);
                const int r = (int)(__brev((unsigned)m) >> (32 - p.logM));
                buf[r] = make_float2(__ldg(xb + i0 + m) * w, 0.0f);
            }
            __syncthreads();
            for (int s = 1; s <= p.logM; ++s) {
                const int half = 1 << (s - 1);
                for (int j = tid; j < M / 2; j += nthr) {
                    const int pos = j & (half - 1);
                    const int a0 = ((j >> (s - 1)) << s) + pos, a1 = a0 + half;
                    float sn, cs;
                    sincospif(-(float)pos / (float)half, &sn, &cs);
                    const float2 u = buf[a0], v = cmul(buf[a1], make_float2(cs, sn));
                    buf[a0] = make_float2(u.x + v.x, u.y + v.y);
                    buf[a1] = make_float2(u.x - v.x, u.y - v.y);
                }
                __syncthreads();
            }
            // peak of |X_k|^2 over 1 <= k <= M/2 - 1, lowest k on ties
            float bv = -1.0f;
            int bk = 0x7fffffff;
            for (int k = 1 + tid; k <= M / 2 - 1; k += nthr) {
                const float2 X = buf[k];
                const float P = fmaf(X.x, X.x, X.y * X.y);
                if (P > bv || (P == bv && k < bk)) { bv = P; bk = k; }
            }
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) {
                const float ov = __shfl_xor_sync(0xffffffffu, bv, off);
                const int ok = __shfl_xor_sync(0xffffffffu, bk, off);
                if (ov > bv || (ov == bv && ok < bk)) { bv = ov; bk = ok; }
            }
            if (lane == 0) { s_val[warp] = bv; s_idx[warp] = bk; }
            __syncthreads();
            if (tid == 0) {
                for (int w = 1; w < nthr / 32; ++w)
                    if (s_val[w] > bv || (s_val[w] == bv && s_idx[w] < bk)) { bv = s_val[w]; bk = s_idx[w]; }
                const float2 Xm = buf[bk - 1], X0 = buf[bk], Xp = buf[bk + 1];
                const double Pm = (double)Xm.x * Xm.x + (double)Xm.y * Xm.y;
                const double P0 = (double)X0.x * X0.x + (double)X0.y * X0.y;
                const double Pp = (double)Xp.x * Xp.x + (double)Xp.y * Xp.y;
                const double lm = log(Pm), l0 = log(P0), lp = log(Pp);
                const double den = lm - 2.0 * l0 + lp;
                const double delta = den != 0.0 ? 0.5 * (lm - lp) / den : 0.0;
                const double sinc = delta != 0.0 ? sinpi(delta) / (kPi * delta) : 1.0;
                const double lobe = sinc / (1.0 - delta * delta);
                s_f[piece] = ((double)bk + delta) * p.fs / (double)M;
                s_a[piece] = 4.0 * sqrt(P0) / (double)M / lobe;
                s_k[piece] = bk;
            }
            __syncthreads();
        }
        if (tid == 0) {
            const double T = (double)p.N / p.fs, dts = (double)p.S / p.fs;
            const double a = s_a[1], fc = s_f[1];
            const double fdot = (s_f[2] - s_f[0]) / (2.0 * dts);
            double* e = p.est + b * 8;
            e[0] = a; e[1] = s_f[0]; e[2] = fc; e[3] = s_f[2]; e[4] = fdot;
            e[5] = (double)s_k[0]; e[6] = (double)s_k[1]; e[7] = (double)s_k[2];
            const double f_hw = fmax(p.f_rel * fabs(fc), p.f_bins * p.fs / (double)M);
            const double fdot_hw = p.fdot_bins * (p.fs / (double)M) / dts;
            double* lo = p.lo + b * p.D;
            double* hi = p.hi + b * p.D;
            lo[0] = a * (1.0 - p.a_rel); hi[0] = a * (1.0 + p.a_rel);
            lo[1] = -p.a1_rel * a / T; hi[1] = p.a1_rel * a / T;
            lo[2] = -kPi; hi[2] = kPi;
            lo[3] = fc - f_hw; hi[3] = fc + f_hw;
            lo[4] = fdot - fdot_hw; hi[4] = fdot + fdot_hw;
            if (p.D == 6) { lo[5] = -p.fddot_hw; hi[5] = p.fddot_hw; }
        }
        __syncthreads();
    }
}

int acquire_launch(const float* x, long long B, int N, double fs, int D, const pt_acq_config* a, double* est, double* lo,
                   double* hi, cudaStream_t st) {
    AcqParams p;
    p.x = x; p.est = est; p.lo = lo; p.hi = hi; p.B = B; p.N = N; p.D = D; p.M = a->M; p.S = a->spacing;
    p.logM = 0;
    while ((1 << p.logM) < a->M) ++p.logM;
    p.fs = fs; p.f_rel = a->f_rel; p.f_bins = a->f_bins; p.fdot_bins = a->fdot_bins; p.a_rel = a->a_rel; p.a1_rel = a->a1_rel;
    p.fddot_hw = a->fddot_hw;
    const size_t smem = (size_t)a->M * sizeof(float2);
    if (smem > 48 * 1024) {
        if (check_cuda(cudaFuncSetAttribute(acquire_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem),
                       "cudaFuncSetAttribute(acquire_kernel)"))
            return 1;
    }
    const unsigned grid = (unsigned)(B < 148LL * 8 ? B : 148LL * 8);
    acquire_kernel<<<grid, 256, smem, st>>>(p);
    return check_cuda(cudaGetLastError(), "acquire_kernel launch");
}

}  // namespace pt
