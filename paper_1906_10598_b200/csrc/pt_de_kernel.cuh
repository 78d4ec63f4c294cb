// pt_de_kernel.cuh -- the persistent one-CTA-per-data-block kernel: stages a block's samples into shared
// memory once (bulk async copy), then runs the whole Differential Evolution fit on-chip; the same kernel in
// FITNESS mode evaluates a caller-given population (pt_fitness).
//
// Hot loop = the chi^2 objective (Eq. 4) of the model (Eq. 2):
//     RSS_i = sum_n [ x_n - (a0 + a1 t_n) cos(phi_i(t_n)) ]^2 .
// Arithmetic per sample and candidate ("sample-evaluation"), D = 5:
//     FADD  wd = W_n + d0            W_n: fp64 reference phase of the block, reduced mod 2 pi, stored fp32
//     FFMA  h  = t d2 + d1           d*: candidate's offset from the reference, phase-polynomial coefficients
//     FFMA  y  = t h + wd
//     FMUL  + MUFU.COS  c = cos(y)   (cos.approx = multiply by 1/2pi, then the hardware cosine in turns)
//     FFMA  A  = t a1 + a0
//     FFMA  r  = x - A c
//     FFMA  acc += r r
// i.e. 7 FP32-pipe instructions + 1 MUFU per sample-evaluation (one more FFMA for D = 6).  Lanes own samples,
// every thread carries C candidates in registers (register blocking), so the shared-memory loads and the
// t_n computation are amortised over C.
#pragma once
#include "pt_device.cuh"

namespace pt {

constexpr int kChunk = 128;        // samples per warp step: 32 lanes x 4 consecutive samples (one LDS.128 each)
constexpr int kCandStride = 8;     // floats per candidate in the evaluation table (a0,a1,d0,d1,d2,d3,-,-)

enum Mode { kModeFit = 0, kModeFitness = 1 };

struct BlockParams {
    const float* x;               // [B][N]
    const double* lo;             // [B][D]  (fit)
    const double* hi;             // [B][D]  (fit)
    const uint32_t* block_index;  // [B] or null (fit)
    const float* pop_in;          // [B][NP][D] (fitness)
    float* fitness_out;           // [B][NP]    (fitness)
    double* best;                 // [B][D]
    float* best_rss;              // [B]
    uint32_t* status;             // [B]
    float* final_pop;             // [B][NP][D] or null
    float* final_fit;             // [B][NP] or null
    long long B;
    int N, Npad, NP, NPpad, G;
    double fs, t0, F;
    uint32_t CR32, key0, key1;
    int Wg, Ws;                   // warp grid of the evaluation phase, Wg * Ws = warps per CTA
    int use_bulk;                 // rows of x are 16-byte aligned and N % 4 == 0
};

// Shared-memory carve-up, identical on host and device.
struct SmemLayout {
    int off_bar, off_xs, off_ws, off_popA, off_popT, off_box, off_fit, off_cand, off_part, total;
    __host__ __device__ static int align_up(int v, int a) { return (v + a - 1) / a * a; }
    __host__ __device__ SmemLayout(int Npad, int NP, int NPpad, int D, int Ws) {
        int o = 0;
        off_bar = o; o += 16;
        off_xs = o; o += Npad * 4;
        off_ws = o; o += Npad * 4;
        o = align_up(o, 16);
        off_popA = o; o += NP * D * 8;
        off_popT = o; o += NP * D * 8;
        off_box = o; o += 3 * 8 * 8;          // base[8], lo[8], hi[8]
        off_fit = o; o += NPpad * 4;
        o = align_up(o, 16);
        off_cand = o; o += NPpad * kCandStride * 4;
        off_part = o; o += Ws * NPpad * 4;
        total = align_up(o, 16);
    }
};

// ---------------------------------------------------------------------------------------------------
// Evaluation of one group of C candidates over chunks [kb, ke) of the resident block.
// ---------------------------------------------------------------------------------------------------
template <int C, int D, bool MASKED>
__device__ __forceinline__ void eval_chunk(const float4 xv, const float4 wv, const float nf, const float dtf,
                                           const float (&tb)[4], const int n_left, const float (&a0)[C],
                                           const float (&a1)[C], const float (&d0)[C], const float (&d1)[C],
                                           const float (&d2)[C], const float (&d3)[C], float (&acc)[C]) {
    const float xs4[4] = {xv.x, xv.y, xv.z, xv.w};
    const float ws4[4] = {wv.x, wv.y, wv.z, wv.w};
    float t[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) t[j] = fmaf(nf, dtf, tb[j]);
#pragma unroll
    for (int c = 0; c < C; ++c) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            float h;
            if (D == 6) h = fmaf(t[j], fmaf(t[j], d3[c], d2[c]), d1[c]);
            else h = fmaf(t[j], d2[c], d1[c]);
            const float y = fmaf(t[j], h, ws4[j] + d0[c]);
            const float cs = __cosf(y);
            const float A = fmaf(t[j], a1[c], a0[c]);
            float r = fmaf(-A, cs, xs4[j]);
            if (MASKED) r = (j < n_left) ? r : 0.0f;
            acc[c] = fmaf(r, r, acc[c]);
        }
    }
}

template <int C>
__device__ __forceinline__ void reduce_and_store(float (&acc)[C], const int lane, float* out) {
    // butterfly with halving: after log2(C) exchange steps every lane holds one candidate's partial sum
    int cidx = 0;
    int off = 16;
#pragma unroll
    for (int half = C / 2; half >= 1; half >>= 1, off >>= 1) {
        const bool upper = (lane & off) != 0;
#pragma unroll
        for (int c = 0; c < half; ++c) {
            const float send = upper ? acc[c] : acc[c + half];
            const float keep = upper ? acc[c + half] : acc[c];
            acc[c] = keep + __shfl_xor_sync(0xffffffffu, send, off);
        }
        cidx += upper ? half : 0;
    }
    float v = acc[0];
    for (; off >= 1; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    if ((lane & (32 / C - 1)) == 0) out[cidx] = v;
}

template <int C, int D>
__device__ __forceinline__ void eval_population(const BlockParams& p, const float* __restrict__ xs,
                                                const float* __restrict__ wref, const float* __restrict__ cand,
                                                float* __restrict__ part, const int warp, const int lane) {
    const int wg = warp % p.Wg, wsl = warp / p.Wg;
    const int nch = p.Npad / kChunk;
    const int kb = (int)(((long long)wsl * nch) / p.Ws), ke = (int)(((long long)(wsl + 1) * nch) / p.Ws);
    const bool tail = (p.N % kChunk) != 0;             // the last chunk of the block is partial
    const int ke_full = (tail && ke == nch) ? ke - 1 : ke;
    const double dt = 1.0 / p.fs;
    const float dtf = (float)dt;
    float tb[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) tb[j] = (float)(p.t0 + j * dt);
    float* out_row = part + wsl * p.NPpad;
    const int groups = p.NPpad / C;
    for (int g = wg; g < groups; g += p.Wg) {
        float a0[C], a1[C], d0[C], d1[C], d2[C], d3[C], acc[C];
        const float4* cg = reinterpret_cast<const float4*>(cand + (size_t)g * C * kCandStride);
#pragma unroll
        for (int c = 0; c < C; ++c) {
            const float4 u = cg[2 * c], v = cg[2 * c + 1];
            a0[c] = u.x; a1[c] = u.y; d0[c] = u.z; d1[c] = u.w; d2[c] = v.x; d3[c] = v.y;
            acc[c] = 0.0f;
        }
        const float4* xp = reinterpret_cast<const float4*>(xs) + kb * 32 + lane;
        const float4* wp = reinterpret_cast<const float4*>(wref) + kb * 32 + lane;
        float nf = (float)(kb * kChunk + lane * 4);
#pragma unroll 1
        for (int k = kb; k < ke_full; ++k) {
            eval_chunk<C, D, false>(*xp, *wp, nf, dtf, tb, 4, a0, a1, d0, d1, d2, d3, acc);
            xp += 32; wp += 32; nf += (float)kChunk;
        }
        if (ke_full < ke) {
            const int n_left = p.N - ((nch - 1) * kChunk + lane * 4);     // valid samples of this lane (may be <= 0)
            eval_chunk<C, D, true>(*xp, *wp, nf, dtf, tb, n_left, a0, a1, d0, d1, d2, d3, acc);
        }
        reduce_and_store<C>(acc, lane, out_row + g * C);
    }
}

// Evaluation-table entry of one member: absolute amplitudes, phase-polynomial offsets from the block's fp64
// reference (radians): d0 = phi0 - phi0_b, d1 = 2 pi (f - f_b), d2 = pi (fdot - fdot_b), d3 = (pi/3)(fddot - fddot_b).
template <int D>
__device__ __forceinline__ void write_cand(float* ce, const double* th, const double* base) {
    float4 u, v;
    u.x = (float)th[0];
    u.y = (float)th[1];
    u.z = (float)(th[2] - base[2]);
    u.w = (float)(kTwoPi * (th[3] - base[3]));
    v.x = (float)(kPi * (th[4] - base[4]));
    v.y = (D == 6) ? (float)((kPi / 3.0) * (th[5] - base[5])) : 0.0f;
    v.z = 0.0f; v.w = 0.0f;
    reinterpret_cast<float4*>(ce)[0] = u;
    reinterpret_cast<float4*>(ce)[1] = v;
}

template <int C, int D, int MODE>
__global__ void __launch_bounds__(512, 1) pt_block_kernel(const BlockParams p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const SmemLayout L(p.Npad, p.NP, p.NPpad, D, p.Ws);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.off_bar);
    float* xs = reinterpret_cast<float*>(smem + L.off_xs);
    float* wref = reinterpret_cast<float*>(smem + L.off_ws);
    double* popA = reinterpret_cast<double*>(smem + L.off_popA);
    double* popT = reinterpret_cast<double*>(smem + L.off_popT);
    double* base = reinterpret_cast<double*>(smem + L.off_box);
    double* lo_s = base + 8;
    double* hi_s = base + 16;
    float* fit = reinterpret_cast<float*>(smem + L.off_fit);
    float* cand = reinterpret_cast<float*>(smem + L.off_cand);
    float* part = reinterpret_cast<float*>(smem + L.off_part);

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31;
    uint32_t parity = 0;

    if (tid == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    // padded evaluation-table rows evaluate a zero model; their sums are never read
    for (int i = p.NP * kCandStride + tid; i < p.NPpad * kCandStride; i += nthr) cand[i] = 0.0f;
    __syncthreads();

    for (long long blk = blockIdx.x; blk < p.B; blk += gridDim.x) {
        const float* xg = p.x + blk * (long long)p.N;
        // ---- a0: stage the block's samples (PAPER.md:121 data block) into shared memory, once ----
        if (p.use_bulk) {
            if (tid == 0) {
                fence_proxy_async();   // earlier generic-proxy reads of xs are ordered before the async writes
                const uint32_t bytes = (uint32_t)p.N * 4u;
                mbar_arrive_expect_tx(bar, bytes);
                for (uint32_t o = 0; o < bytes; o += 32768u) {
                    const uint32_t len = min(32768u, bytes - o);
                    bulk_g2s(reinterpret_cast<unsigned char*>(xs) + o, reinterpret_cast<const unsigned char*>(xg) + o,
                             len, bar);
                }
            }
        } else {
            for (int n = tid; n < p.N; n += nthr) xs[n] = __ldg(xg + n);
        }
        for (int n = p.N + tid; n < p.Npad; n += nthr) xs[n] = 0.0f;

        // ---- box, reference point ----
        if (MODE == kModeFit) {
            if (tid < D) {
                const double l = p.lo[blk * D + tid], h = p.hi[blk * D + tid];
                lo_s[tid] = l; hi_s[tid] = h;
                base[tid] = 0.5 * (l + h);
            }
        } else {
            if (tid < D) {   // mid-range of the given population
                const float* pp = p.pop_in + blk * (long long)p.NP * D + tid;
                float mn = pp[0], mx = pp[0];
                for (int i = 1; i < p.NP; ++i) { const float v = pp[(size_t)i * D]; mn = fminf(mn, v); mx = fmaxf(mx, v); }
                base[tid] = 0.5 * ((double)mn + (double)mx);
            }
        }
        __syncthreads();

        // ---- reference phase W_n = [phi_b(t_n)] mod 2 pi in fp64, stored fp32 in [-pi, pi) ----
        {
            const double b0 = base[2] * (1.0 / kTwoPi), b1 = base[3], b2 = 0.5 * base[4];
            const double b3 = (D == 6) ? base[5] * (1.0 / 6.0) : 0.0;
            const double dt = 1.0 / p.fs;
            for (int n = tid; n < p.Npad; n += nthr) {
                const double t = p.t0 + (double)n * dt;
                double u = b0 + t * (b1 + t * (b2 + t * b3));     // turns
                u -= rint(u);
                wref[n] = (float)(kTwoPi * u);
            }
        }

        // ---- a1: generation 0 ----
        const uint32_t bidx = (MODE == kModeFit) ? (p.block_index ? p.block_index[blk] : (uint32_t)blk) : 0u;
        for (int i = tid; i < p.NP; i += nthr) {
            double th[D];
            if (MODE == kModeFit) {
                init_member<D>((uint32_t)i, bidx, p.key0, p.key1, lo_s, hi_s, th);
#pragma unroll
                for (int j = 0; j < D; ++j) popA[i * D + j] = th[j];
            } else {
                const float* pp = p.pop_in + (blk * (long long)p.NP + i) * D;
#pragma unroll
                for (int j = 0; j < D; ++j) th[j] = (double)pp[j];
            }
            write_cand<D>(cand + (size_t)i * kCandStride, th, base);
        }
        if (p.use_bulk) mbar_wait(bar, parity);
        parity ^= 1u;
        __syncthreads();

        eval_population<C, D>(p, xs, wref, cand, part, warp, lane);
        __syncthreads();
        for (int i = tid; i < p.NP; i += nthr) {
            float s = 0.0f;
            for (int w = 0; w < p.Ws; ++w) s += part[w * p.NPpad + i];
            fit[i] = s;
            if (MODE == kModeFitness) p.fitness_out[blk * (long long)p.NP + i] = s;
        }
        __syncthreads();

        if (MODE == kModeFit) {
            // ---- a2..a7: generations ----
            for (int g = 1; g <= p.G; ++g) {
                for (int i = tid; i < p.NP; i += nthr) {
                    const Draws dr = de_draws<D>((uint32_t)i, (uint32_t)g, bidx, (uint32_t)p.NP, p.CR32, p.key0, p.key1);
                    double th[D];
#pragma unroll
                    for (int j = 0; j < D; ++j) {
                        const double parent = popA[i * D + j];
                        const double mut = mutate_coord(popA[dr.r1 * D + j], popA[dr.r2 * D + j], popA[dr.r3 * D + j],
                                                        p.F, lo_s[j], hi_s[j]);
                        th[j] = ((dr.mask >> j) & 1u) ? mut : parent;
                        popT[i * D + j] = th[j];
                    }
                    write_cand<D>(cand + (size_t)i * kCandStride, th, base);
                }
                __syncthreads();
                eval_population<C, D>(p, xs, wref, cand, part, warp, lane);
                __syncthreads();
                // ---- a6: greedy selection, accept on <= ----
                for (int i = tid; i < p.NP; i += nthr) {
                    float s = 0.0f;
                    for (int w = 0; w < p.Ws; ++w) s += part[w * p.NPpad + i];
                    if (s <= fit[i]) {
                        fit[i] = s;
#pragma unroll
                        for (int j = 0; j < D; ++j) popA[i * D + j] = popT[i * D + j];
                    }
                }
                __syncthreads();
            }

            // ---- a8: best member (lowest index on ties), status, optional final population ----
            if (warp == 0) {
                float bv = INFINITY, mx = -INFINITY;
                int bi = 0x7fffffff;
                for (int i = lane; i < p.NP; i += 32) {
                    const float v = fit[i];
                    if (v < bv || (v == bv && i < bi)) { bv = v; bi = i; }
                    mx = fmaxf(mx, v);
                }
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) {
                    const float ov = __shfl_xor_sync(0xffffffffu, bv, off);
                    const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
                    const float om = __shfl_xor_sync(0xffffffffu, mx, off);
                    if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
                    mx = fmaxf(mx, om);
                }
                if (lane == 0) {
                    uint32_t st = 0;
#pragma unroll
                    for (int j = 0; j < D; ++j) {
                        const double v = popA[bi * D + j];
                        p.best[blk * D + j] = v;
                        const double w = hi_s[j] - lo_s[j];
                        if (w > 0.0 && (v - lo_s[j] <= 1e-6 * w || hi_s[j] - v <= 1e-6 * w)) st |= 1u;
                    }
                    if (mx - bv > 1e-6f * bv) st |= 2u;
                    p.best_rss[blk] = bv;
                    p.status[blk] = st;
                }
            }
            if (p.final_pop) {
                float* fp = p.final_pop + blk * (long long)p.NP * D;
                for (int i = tid; i < p.NP * D; i += nthr) fp[i] = (float)popA[i];
            }
            if (p.final_fit) {
                float* ff = p.final_fit + blk * (long long)p.NP;
                for (int i = tid; i < p.NP; i += nthr) ff[i] = fit[i];
            }
        }
        __syncthreads();   // xs / popA are reused by the next block of this CTA
    }
}

}  // namespace pt
