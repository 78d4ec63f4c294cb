// pt_run_kernel.cuh -- the run-local variant of the persistent one-CTA-per-data-block DE kernel (rows a0-a8 of SURVEY 8(a)).
// Same method, same DE step (Philox draws, fp64 mutation / crossover / bounds, greedy selection) and same outputs as
// pt_block_kernel; what differs is the layout and the arithmetic of the evaluation loop (row a5, Eq. 2-4):
//
//   * transposed layout: a THREAD owns one candidate and walks a contiguous slice of the block's samples (thread = candidate x
//     slice); the sample values are warp-uniform shared-memory broadcasts (one LDS.128 per four sample-evaluations of a warp),
//     there is no shuffle reduction and no reference-phase array (shared memory holds 4 bytes per sample);
//   * the samples are walked in RUNS of kRun = 256.  Per run the phase polynomial of Eq. 3, P(t) = phi0/2pi + f t + fdot t^2/2 +
//     fddot t^3/6 [turns], is re-expanded at the run centre t_c in fp64: E0 = 2 pi frac(P(t_c)), E1 = 2 pi dt P1(t_c),
//     E2 = 2 pi dt^2 P2(t_c)/2, E3 = 2 pi dt^3 P3/6 (Pk = k-th derivative), so that phase(j) = E0 + j (E1 + j (E2 + j E3)) for the
//     sample j steps from the centre.  The large part of the phase (6e3 ... 3e5 rad) is removed exactly and fp32 never sees more
//     than pi + 128 |E1|.  Inside the run the index j is a COMPILE-TIME constant of the fully unrolled instruction stream, so
//     the Horner scheme needs no index arithmetic at all; per PAIR of consecutive samples (j, j + 1), with packed coefficient pairs
//     whose second lane holds the polynomial shifted by one sample:
//         FFMA2 h = E2 j + E1,  FFMA2 y = h j + E0          phase of samples (j, j + 1); j is a 32-bit immediate (FFMA2 R, R, -128, R)
//         2 x (FMUL + MUFU.COS)                              cos.approx
//         FFMA2 A = G j + Ac                                 negated amplitude -(a0 + a1 t)
//         FFMA2 r = A c + x,  FFMA2 acc += r r
//     i.e. 6 FP32-pipe lane operations + 1 MUFU per sample-evaluation for D = 5 (pt_block_kernel: 7) and the same for D = 6 whenever
//     the cubic term cannot matter inside a run (|E3| 128^3 below 1e-7 rad over the whole box: the run then carries the exact value,
//     first and second derivative of the cubic at its centre); 7 otherwise.  4.75 issue slots per sample-evaluation (5.3);
//   * 64 registers per thread: 32 warps per SM (one CTA of 1024 threads, or 2 x 512 / 4 x 256 / 8 x 128 for shorter blocks, whose DE steps
//     then overlap with the other CTAs' evaluation), against 16 warps of 128 registers in pt_block_kernel.
// Every phase is rounded on its own: there is no recurrence.  (A forward-difference recurrence y += d, d += dd was measured first
// and dropped: with dd below half an ulp of d the second difference is lost and the phase drifts by E2 j^2, 1e-5 rad at j = 64.
// The run length trades the per-run re-expansion (about 60 instructions, a serial fp64 chain) against the size of the fp32 phases:
// measured on config 2, 64 / 128 / 256 samples per run give 80.5 / 86.5 / 89.2 % of the XU roofline and a largest objective error of
// 1.5e-7 / 4e-7 / 1.7e-6 relative; 256 is also the tile of pt_tc_kernel.)
// Summation: fp32 FMA over a run (128 terms per accumulator), error-free two-sum of the run's value into a (hi, lo) pair, fp64 from
// there on (partials, objective values, selection), as in pt_tc_kernel (R18, R20).
// Measured numbers and the comparison with the other two evaluation kernels: DESIGN.md section 5.13, profiles/r2_*.
#pragma once
#include "pt_de_kernel.cuh"

namespace pt {

#ifndef PT_RUN_SAMPLES
#define PT_RUN_SAMPLES 256
#endif
#ifndef PT_RUN_INLINE
#define PT_RUN_INLINE __noinline__
#endif
constexpr int kRun = PT_RUN_SAMPLES;      // samples per run
constexpr int kRunMaxThreads = 1024;
enum RunAmp { kRunAmpLinear = 0, kRunAmpConst = 1, kRunAmpCor = 2 };

// Shared-memory carve-up of pt_run_kernel, identical on host and device.
struct RunSmemLayout {
    int off_bar, off_xs, off_popA, off_popT, off_box, off_fit, off_part, off_xpart, total;
    __host__ __device__ static int align_up(int v, int a) { return (v + a - 1) / a * a; }
    // Nres: samples this CTA keeps resident (its slice when K > 1); TS/S: tile samples and ring stages of the streamed path
    // slices: sample slices of the evaluation (work items = NP x slices)
    __host__ __device__ RunSmemLayout(int Nres, int NP, int D, int slices, int TS = 0, int S = 0, int K = 1) {
        int o = 0;
        off_bar = o; o += kBarBytes;               // [0] staging barrier, [1..S] full, [1+S..2S] empty
        off_xs = o; o += (S > 0) ? S * TS * 4 : align_up(Nres, 4) * 4;
        o = align_up(o, 16);
        off_popA = o; o += NP * D * 8;
        off_popT = o; o += NP * D * 8;
        off_box = o; o += 3 * 8 * 8;               // flags[8], lo[8], hi[8]
        off_fit = o; o += NP * 8;                  // objective values of the members, fp64
        off_part = o; o += NP * slices * 8;        // [slice][candidate] partial sums, fp64
        off_xpart = o; o += (K > 1) ? 2 * K * NP * 8 : 0;           // [2][K][NP]: the cluster peers' sums, double-buffered
        total = align_up(o, 16);
    }
};

__device__ __forceinline__ void st_cluster_f64(uint32_t addr, double v) {
    asm volatile("st.shared::cluster.f64 [%0], %1;" ::"r"(addr), "d"(v) : "memory");
}
__device__ __forceinline__ f32x2 run_bc2(float v) { return pack2(v, v); }

// One run of one candidate, two consecutive samples at a time.  The run's polynomial phase(j) = E0 + j (E1 + j (E2 + j E3)) is
// evaluated by Horner's rule at EVEN j with packed coefficient pairs: lane 0 holds the coefficients themselves (sample j), lane 1
// the same polynomial shifted by one sample (sample j + 1), so that one FFMA2 chain yields the phases of samples (j, j + 1) and j
// enters as a broadcast scalar -- in a full run a 32-bit immediate of the unrolled instruction stream (SASS: FFMA2 R, R, -128, R).
//   chi^2 (Eq. 4): r = A' cos(y) + x with the negated amplitude A'(j) = Ac + j G, acc += r^2;   correlation (Eq. 5-6): acc += x cos(y).
struct RunCoef { f32x2 E0, E1, E2, E3, Ac, G; };

template <int AMP, bool CUB>
__device__ __forceinline__ void run_pair(const RunCoef& c, const float jf, const float x0, const float x1, f32x2& acc) {
    const f32x2 j2 = pack2(jf, jf);
    f32x2 y;
    if (CUB) y = fma2(fma2(fma2(c.E3, j2, c.E2), j2, c.E1), j2, c.E0);
    else y = fma2(fma2(c.E2, j2, c.E1), j2, c.E0);
    float y0, y1;
    unpack2(y, y0, y1);
    const f32x2 cc = pack2(__cosf(y0), __cosf(y1));
    if (AMP == kRunAmpCor) {
        acc = fma2(cc, pack2(x0, x1), acc);
    } else {
        const f32x2 A = (AMP == kRunAmpLinear) ? fma2(c.G, j2, c.Ac) : c.Ac;
        const f32x2 r = fma2(A, cc, pack2(x0, x1));
        acc = fma2(r, r, acc);
    }
}

// a full run of kRun samples centred at j = 0: fully unrolled, every j is a compile-time constant
template <int AMP, bool CUB>
__device__ __forceinline__ void run_full(const float* __restrict__ xr, const RunCoef& c, f32x2& acc) {
#pragma unroll
    for (int k = 0; k < kRun; k += 4) {
        const float4 q = *reinterpret_cast<const float4*>(xr + k);
        run_pair<AMP, CUB>(c, (float)(k - kRun / 2), q.x, q.y, acc);
        run_pair<AMP, CUB>(c, (float)(k + 2 - kRun / 2), q.z, q.w, acc);
    }
}
// a shorter run (the last one of a slice): `len` (even) samples, the first one at j = jf0 (an integer, carried exactly in fp32)
template <int AMP, bool CUB>
__device__ __forceinline__ void run_part(const float* __restrict__ xr, const int len, const float jf0, const RunCoef& c, f32x2& acc) {
    float jf = jf0;
    int k = 0;
    for (; k + 16 <= len; k += 16, jf += 16.0f) {
#pragma unroll
        for (int u = 0; u < 16; u += 4) {
            const float4 q = *reinterpret_cast<const float4*>(xr + k + u);
            run_pair<AMP, CUB>(c, jf + (float)u, q.x, q.y, acc);
            run_pair<AMP, CUB>(c, jf + (float)(u + 2), q.z, q.w, acc);
        }
    }
#pragma unroll 1
    for (; k < len; k += 2, jf += 2.0f) {
        const float2 q = *reinterpret_cast<const float2*>(xr + k);
        run_pair<AMP, CUB>(c, jf, q.x, q.y, acc);
    }
}

// double -> float by integer operations on the bits (round to nearest, ties away; |v| < 2^-126 gives 0): the conversion
// instruction F2F.F32.F64 executes on the XU pipe, the pipe the cosines saturate (measured: 4 conversions per run = 3.5 % of the
// XU cycles of this kernel).
__device__ __forceinline__ float run_d2f(const double v) {
    const unsigned long long b = (unsigned long long)__double_as_longlong(v) + 0x10000000ull;      // + half an fp32 ulp
    const uint32_t hi = (uint32_t)(b >> 32), lo = (uint32_t)b;
    const uint32_t mag = hi & 0x7FFFFFFFu;
    const uint32_t fb = __funnelshift_l(lo, mag - 0x38000000u, 3) | (hi & 0x80000000u);          // re-biased exponent, 23 mantissa bits
    return __uint_as_float(mag >= 0x38100000u ? fb : 0u);
}

// One evaluation pass over a tile of samples that sits in shared memory: xs[0 .. len_t) are samples n_t0 .. n_t0 + len_t of the
// data block (the whole block, a cluster CTA's slice of it, or one tile of the streamed ring).  Work item = (candidate, slice):
// the tile is cut into S = p.Ws contiguous ranges on 4-sample boundaries (the planner picks S so that NP x S items fill the
// threads of the CTA in whole rounds); item i is candidate i % NP over slice i / NP, and thread t takes items t, t + threads, ...
// The item's sum goes to part[i] (added when `accumulate`).
// Not inlined: the loop's register allocation then does not depend on the code around it.
template <int D, int AMP, bool CUB>
__device__ PT_RUN_INLINE void run_eval_tile(const BlockParams& p, const float* __restrict__ xs, const int n_t0, const int len_t,
                                          const double* __restrict__ pop, double* __restrict__ part, const bool accumulate, const int tid,
                                          const int nthr) {
    const int NP = p.NP;
    const int S = p.Ws;
    const int quads = (len_t + 3) >> 2;
    const f32x2 neg1 = run_bc2(-1.0f);
    for (int item = tid; item < NP * S; item += nthr) {
        const int cand = item % NP, slice = item / NP;
        const int nb = (int)(((long long)slice * quads) / S) * 4;
        const int ne = min(len_t, (int)(((long long)(slice + 1) * quads) / S) * 4);
        const double* th = pop + cand * D;
        // phase polynomial in turns (Eq. 3): P = c0 + t (f + t (fdot/2 + t fddot/6)); only c0, f, fdot, fddot stay
        // in registers, the halves and thirds are formed where they are used (the fp64 pipe is 2 % busy, registers are scarce)
        const double c0 = th[2] * (1.0 / kTwoPi), f1 = th[3], f2 = th[4], f3 = (D == 6) ? th[5] : 0.0;
        const float na0 = -(float)th[0], na1 = (AMP == kRunAmpLinear) ? -(float)th[1] : 0.0f;
        f32x2 hi = run_bc2(0.0f), lo = run_bc2(0.0f);
        // block-relative index of the run's first sample, in both precisions (exact: < 2^24; a conversion would run on the XU pipe)
        double nd = (double)(n_t0 + nb);
        float nf = (float)(n_t0 + nb);
        // D = 5: the full runs of a slice follow each other at a fixed step, so their re-expansions are carried instead of recomputed.
        // frac(P(t_c)) lives in 64-bit fixed point (turns x 2^64: the integer addition wraps exactly where the phase does, so there is
        // no range reduction) and advances by its first and second differences; E1 advances in fp64 by its constant step; E2 is a
        // constant of the candidate.  Per run: four integer additions, one DADD and one double -> float instead of a serial chain of
        // a dozen fp64 operations and three conversions.  Quantisation 2^-64 turns per addition; E0 is read off with 2^-23 turns.
        unsigned long long Pfix = 0, d1fix = 0, d2fix = 0;
        double e1s = 0.0, de1s = 0.0;
        float E2s = 0.0f;
        if (D == 5 && ne - nb >= kRun) {
            const double dt = p.dt, step = (double)kRun * dt;
            const double tc = fma(nd + (double)(kRun / 2), dt, p.t0);               // centre of the slice's first run
            auto fix = [](const double v) -> unsigned long long { return __double2ull_rn((v - floor(v)) * 18446744073709551616.0); };
            const double slope = fma(f2, tc, f1);                                   // P'(t_c) [turns / s]
            Pfix = fix(fma(tc, fma(tc, 0.5 * f2, f1), c0));
            d1fix = fix(fma(step, slope, 0.5 * f2 * step * step));                  // P(t_c + step) - P(t_c)
            d2fix = fix(f2 * step * step);
            e1s = (kTwoPi * dt) * slope;
            de1s = (kTwoPi * dt) * f2 * step;
            E2s = run_d2f((kTwoPi * dt * dt) * (0.5 * f2));
        }
        for (int n0 = nb; n0 < ne; n0 += kRun, nd += (double)kRun, nf += (float)kRun) {
            f32x2 acc = run_bc2(0.0f);
            // The polynomial is re-expanded at sample h of the run (its centre; a short last run of a slice: ITS centre, so that a
            // block of a few samples is evaluated next to the expansion point).
            auto coefficients = [&](const float hf, const double hd) -> RunCoef {
                const double dt = p.dt;
                const double tcen = fma(nd + hd, dt, p.t0);
                const double w1 = kTwoPi * dt;
                double P, e1, e2;
                if (D == 6) {
                    const double h3 = 0.5 * f3;
                    P = fma(tcen, fma(tcen, fma(tcen, f3 * (1.0 / 6.0), 0.5 * f2), f1), c0);
                    e1 = w1 * fma(tcen, fma(tcen, h3, f2), f1);                 // 2 pi dt P'(t_c)
                    e2 = (w1 * dt) * fma(tcen, h3, 0.5 * f2);                   // 2 pi dt^2 P''(t_c) / 2
                } else {
                    P = fma(tcen, fma(tcen, 0.5 * f2, f1), c0);
                    e1 = w1 * fma(tcen, f2, f1);
                    e2 = (w1 * dt) * (0.5 * f2);
                }
                P -= __dadd_rn(__dadd_rn(P, 6755399441055744.0), -6755399441055744.0);      // P - rint(P), |P| < 2^51
                const float E0 = run_d2f(kTwoPi * P), E1 = run_d2f(e1), E2 = run_d2f(e2);
                RunCoef c;
                // lane 1 = the polynomial in (j + 1): E0 + E1 + E2 + E3, E1 + 2 E2 + 3 E3, E2 + 3 E3, E3
                if (CUB) {
                    const float E3 = run_d2f((w1 * dt) * dt * (f3 * (1.0 / 6.0)));
                    c.E0 = pack2(E0, (E0 + E1) + (E2 + E3));
                    c.E1 = pack2(E1, fmaf(3.0f, E3, fmaf(2.0f, E2, E1)));
                    c.E2 = pack2(E2, fmaf(3.0f, E3, E2));
                    c.E3 = run_bc2(E3);
                } else {
                    c.E0 = pack2(E0, (E0 + E1) + E2);
                    c.E1 = pack2(E1, fmaf(2.0f, E2, E1));
                    c.E2 = run_bc2(E2);
                    c.E3 = run_bc2(0.0f);
                }
                if (AMP == kRunAmpLinear) {
                    const float dtf = p.dtf, g1 = na1 * dtf;
                    const float Ac = fmaf(na1, fmaf(nf + hf, dtf, p.t0f), na0);      // -(a0 + a1 t_c), t_c in fp32: |t| ulp 3e-8 relative
                    c.Ac = pack2(Ac, Ac + g1);
                    c.G = run_bc2(g1);
                } else {
                    c.Ac = run_bc2(na0);
                    c.G = run_bc2(0.0f);
                }
                return c;
            };
            if (n0 + kRun <= ne) {
                RunCoef c;
                if (D == 5) {
                    // coefficients of a full run from the carried state (see below): no fp64 chain, no range reduction
                    const int sfrac = (int)((uint32_t)(Pfix >> 32) + 256u);                         // frac(P) in [-1/2, 1/2) turns x 2^32, + half a step
                    const float kf = __int_as_float(0x4B400000 + (sfrac >> 9)) - 12582912.0f;       // ... x 2^23, rounded, exact in fp32
                    const float E0 = kf * (float)(kTwoPi / 8388608.0), E1 = run_d2f(e1s);
                    Pfix += d1fix; d1fix += d2fix; e1s += de1s;
                    c.E0 = pack2(E0, (E0 + E1) + E2s);
                    c.E1 = pack2(E1, fmaf(2.0f, E2s, E1));
                    c.E2 = run_bc2(E2s);
                    c.E3 = run_bc2(0.0f);
                    if (AMP == kRunAmpLinear) {
                        const float dtf = p.dtf, g1 = na1 * dtf;
                        const float Ac = fmaf(na1, fmaf(nf + (float)(kRun / 2), dtf, p.t0f), na0);
                        c.Ac = pack2(Ac, Ac + g1);
                        c.G = run_bc2(g1);
                    } else {
                        c.Ac = run_bc2(na0);
                        c.G = run_bc2(0.0f);
                    }
                } else {
                    c = coefficients((float)(kRun / 2), (double)(kRun / 2));
                }
                run_full<AMP, CUB>(xs + n0, c, acc);
            } else {
                const int len = ne - n0, h = len >> 1;
                const RunCoef c = coefficients((float)h, (double)h);
                run_part<AMP, CUB>(xs + n0, len, -(float)h, c, acc);
            }
            // (hi, lo) += acc without losing the rounding error of the addition (Knuth's two-sum, packed)
            const f32x2 sum = add2(hi, acc);
            const f32x2 bp = fma2(hi, neg1, sum);                              // sum - hi
            const f32x2 e1 = fma2(fma2(bp, neg1, sum), neg1, hi);              // hi - (sum - bp)
            const f32x2 e2 = fma2(bp, neg1, acc);                              // acc - bp
            lo = add2(lo, add2(e1, e2));
            hi = sum;
        }
        float h0, h1, l0, l1;
        unpack2(hi, h0, h1);
        unpack2(lo, l0, l1);
        const double v = ((double)h0 + (double)h1) + ((double)l0 + (double)l1);
        part[item] = accumulate ? part[item] + v : v;
    }
}

// Streamed path (blocks larger than shared memory): the block's samples move through a ring of S stages of TS samples by 1-D bulk
// async copies with a full/empty mbarrier pair per stage; thread 0 is the producer and refills the stage that tile c - 2 used.
// Only the samples are streamed (4 bytes per sample and pass, from L2): there is no reference-phase array.
struct RunStream {
    uint64_t* full; uint64_t* empty;
    float* stages;
    const float* xsrc;       // the block's samples in global memory (16-byte aligned row of at least align4(N) floats)
    uint32_t cons, prod, to_issue;
    int j_issue;
};

__device__ __forceinline__ void run_stream_issue_one(const BlockParams& p, RunStream& st) {
    const int s = (int)(st.prod % (uint32_t)p.S);
    const uint32_t k = st.prod / (uint32_t)p.S;
    if (k >= 1) mbar_wait_suspended(&st.empty[s], (k - 1) & 1u);        // every warp has released the previous fill
    const int n0 = st.j_issue * p.TS;
    const int N4 = p.use_bulk ? p.N : (p.N + 3) & ~3;         // N % 4 == 0 on the direct path, else the zero-padded workspace copy
    const uint32_t xb = (uint32_t)min(p.TS, N4 - n0) * 4u;
    mbar_arrive_expect_tx(&st.full[s], xb);
    bulk_g2s(st.stages + (size_t)s * p.TS, st.xsrc + n0, xb, &st.full[s]);
    ++st.prod; --st.to_issue;
    st.j_issue = (st.j_issue + 1 == (p.N + p.TS - 1) / p.TS) ? 0 : st.j_issue + 1;
}

template <int D, int MODE, bool STREAM, int OBJ>
__global__ void __launch_bounds__(kRunMaxThreads, 1) pt_run_kernel(const __grid_constant__ BlockParams p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31;
    const RunSmemLayout L(p.NpadS, p.NP, D, p.Ws, p.TS, p.S, p.K);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.off_bar);
    float* xs = reinterpret_cast<float*>(smem + L.off_xs);
    double* popA = reinterpret_cast<double*>(smem + L.off_popA);
    double* popT = reinterpret_cast<double*>(smem + L.off_popT);
    double* flags = reinterpret_cast<double*>(smem + L.off_box);      // [5] cubic loop, [6] bad box, [7] a1 fixed at zero
    double* lo_s = flags + 8;
    double* hi_s = flags + 16;
    double* fit = reinterpret_cast<double*>(smem + L.off_fit);
    double* part = reinterpret_cast<double*>(smem + L.off_part);
    double* xpart = reinterpret_cast<double*>(smem + L.off_xpart);
    uint32_t parity = 0;
    const double dt = 1.0 / p.fs;

    // ---- cluster geometry: CTA `rank` of K owns samples [n_lo, n_hi) of every block its cluster fits (4-sample boundaries) ----
    const int K = STREAM ? 1 : p.K;
    const int rank = (K > 1) ? (int)cluster_ctarank() : 0;
    const long long first_blk = (K > 1) ? (long long)cluster_id_x() : (long long)blockIdx.x;
    const long long blk_stride = (long long)gridDim.x / K;
    const int quads_blk = (p.N + 3) >> 2;
    const int n_lo = (int)(((long long)rank * quads_blk) / K) * 4;
    const int n_hi = min(p.N, (int)(((long long)(rank + 1) * quads_blk) / K) * 4);
    const int Nown = n_hi - n_lo;
    uint32_t xchg = 0;             // exchanges of partial sums done so far (selects the xpart buffer)
    const int S_sl = p.Ws;         // slices of the evaluation (run_eval_tile)

    RunStream st;
    if (STREAM) {
        st.full = bar + 1; st.empty = bar + 1 + p.S;
        st.stages = xs;
        st.cons = 0; st.prod = 0; st.to_issue = 0; st.j_issue = 0;
    }
    if (tid == 0) {
        mbar_init(bar, 1);
        if (STREAM)
            for (int k = 0; k < p.S; ++k) { mbar_init(&st.full[k], 1); mbar_init(&st.empty[k], (uint32_t)(nthr >> 5)); }
        fence_mbar_init();
    }
    __syncthreads();
    if (K > 1) cluster_sync_all();     // every CTA of the cluster is running before any peer store is issued
    // Objective value of member i: the slices' partial sums in fixed order; with a cluster, the K CTAs' sums are exchanged through
    // distributed shared memory and added in rank order, so every CTA of the cluster holds the same fp64 value.
    auto combine_begin = [&]() {
        if (K > 1) {
            double* buf = xpart + (size_t)(xchg & 1u) * K * p.NP;
            for (int i = tid; i < p.NP; i += nthr) {
                double s = 0.0;
                for (int w = 0; w < S_sl; ++w) s += part[w * p.NP + i];
                const double* slot = buf + (size_t)rank * p.NP + i;
                for (int r = 0; r < K; ++r) st_cluster_f64(mapa_shared(slot, (uint32_t)r), s);
            }
            cluster_sync_all();
        }
    };
    auto combined = [&](int i, const double* pop) -> double {
        double s = 0.0;
        if (K > 1) {
            const double* buf = xpart + (size_t)(xchg & 1u) * K * p.NP;
            for (int r = 0; r < K; ++r) s += buf[(size_t)r * p.NP + i];
        } else {
            for (int w = 0; w < S_sl; ++w) s += part[w * p.NP + i];
        }
        // Eq. 5-6: s = sum x cos(phi); the value minimised is -cor = (-a0) s, with a0 rounded to fp32 as the evaluation sees it
        if (OBJ == kObjCor) s *= (double)(-(float)pop[i * D]);
        return s;
    };
    // argmin of fit[0..NP) with the lowest index on ties, and the maximum (a NaN is read as +inf); every lane gets them
    auto warp_argmin = [&](double& bv, int& bi, double& mx) {
        const double inf = __longlong_as_double(0x7ff0000000000000LL);
        bv = inf; mx = -inf; bi = 0x7fffffff;
        for (int i = lane; i < p.NP; i += 32) {
            double v = fit[i];
            if (!(v == v)) v = inf;
            if (v < bv || (v == bv && i < bi)) { bv = v; bi = i; }
            mx = fmax(mx, v);
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const double ov = __shfl_xor_sync(0xffffffffu, bv, off);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, off);
            const double om = __shfl_xor_sync(0xffffffffu, mx, off);
            if (ov < bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
            mx = fmax(mx, om);
        }
    };
    auto reported = [&](double v) -> double {       // F_cor - 1/pi of cor = -v for the correlation objective
        if (OBJ == kObjCor) return 1.0 / (atan(-v) + 0.5 * kPi) - 1.0 / kPi;
        return v;
    };

    const long long item_end = p.count ? min(p.B, p.blk0 + (long long)*p.count) : p.B;
    for (long long item = p.blk0 + first_blk; item < item_end; item += blk_stride) {
        const long long blk = p.sel ? (long long)p.sel[item] : item;
        const bool quantised = p.q.bits != 0;
        const float* xg = quantised ? nullptr : p.x + blk * (long long)p.N + n_lo;      // this CTA's samples of the block
        const unsigned char* xqrow = quantised ? p.xq + blk * p.row_bytes : nullptr;
        // ---- a0: stage the block's samples (PAPER.md:121 data block) into shared memory, once (streamed path: tiles are staged
        //      every pass; an unaligned or quantised row is first written to the workspace as fp32) ----
        const float* xrow = xg;
        if (STREAM) {
            if (quantised || !p.use_bulk) {
                float* xw = p.ws_x + (size_t)blockIdx.x * p.Npad;
                const int N4 = (p.N + 3) & ~3;
                if (quantised) for (int n = tid; n < N4; n += nthr) xw[n] = (n < p.N) ? unpack_sample(xqrow, n, p.q) : 0.0f;
                else for (int n = tid; n < N4; n += nthr) xw[n] = (n < p.N) ? __ldg(xg + n) : 0.0f;
                xrow = xw;
            }
        } else if (quantised) {
            for (int n = tid; n < Nown; n += nthr) xs[n] = unpack_sample(xqrow, (long long)n_lo + n, p.q);
        } else if (p.use_bulk) {
            if (tid == 0) {
                fence_proxy_async();   // earlier generic-proxy reads of xs are ordered before the async writes
                const uint32_t bytes = (uint32_t)Nown * 4u;
                mbar_arrive_expect_tx(bar, bytes);
                for (uint32_t o = 0; o < bytes; o += 32768u)
                    bulk_g2s(reinterpret_cast<unsigned char*>(xs) + o, reinterpret_cast<const unsigned char*>(xg) + o, min(32768u, bytes - o), bar);
            }
        } else {
            for (int n = tid; n < Nown; n += nthr) xs[n] = __ldg(xg + n);
        }

        // ---- box and per-block switches ----
        if (MODE == kModeFit) {
            if (tid < D) {
                const double l = p.lo[blk * D + tid], h = p.hi[blk * D + tid];
                lo_s[tid] = l; hi_s[tid] = h;
                if (tid == 1) flags[7] = (l == 0.0 && h == 0.0) ? 1.0 : 0.0;     // amplitude slope fixed at zero
                // the cubic term inside a run of kRun samples: |E3| (kRun/2)^3 over the whole box
                if (tid == 5) flags[5] = ((kTwoPi / 6.0) * fmax(fabs(l), fabs(h)) * dt * dt * dt * (double)(kRun / 2) * (kRun / 2) * (kRun / 2) > 1.0e-7) ? 1.0 : 0.0;
            }
            if (tid == 32) {   // lo <= hi is the caller's contract (pt.h); an asynchronous call reports a violation in status bit 4
                bool bad = false;
                for (int j = 0; j < D; ++j) bad = bad || !(p.lo[blk * D + j] <= p.hi[blk * D + j]);
                flags[6] = bad ? 1.0 : 0.0;
            }
        } else {
            // a1 == 0 for every given member (warp 0); the largest |fddot| (warp 1, D = 6): the lanes stride over the members
            if (warp < 2 && (warp == 0 || D == 6)) {
                const int col = warp == 0 ? 1 : 5;
                const float* pp = p.pop_in + blk * (long long)p.NP * D + col;
                float amax = 0.0f;
                for (int i = lane; i < p.NP; i += 32) amax = fmaxf(amax, fabsf(__ldg(pp + (size_t)i * D)));
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, off));
                if (lane == 0) {
                    if (warp == 0) flags[7] = (amax == 0.0f) ? 1.0 : 0.0;
                    else flags[5] = ((kTwoPi / 6.0) * (double)amax * dt * dt * dt * (double)(kRun / 2) * (kRun / 2) * (kRun / 2) > 1.0e-7) ? 1.0 : 0.0;
                }
            }
            if (tid == 64 % nthr) flags[6] = 0.0;
        }
        if (D == 5 && tid == 65 % nthr) flags[5] = 0.0;
        __syncthreads();

        const bool a1z = (OBJ == kObjChi2) && flags[7] != 0.0;
        const bool cub = (D == 6) && flags[5] != 0.0;
        // one evaluation pass of the population `pop` over the samples this CTA holds (or streams)
        auto eval_tile = [&](const float* tile, int n_t0, int len_t, const double* pop, bool accumulate) {
            if (D == 6 && cub) {
                if (OBJ == kObjCor) run_eval_tile<D, kRunAmpCor, true>(p, tile, n_t0, len_t, pop, part, accumulate, tid, nthr);
                else if (a1z) run_eval_tile<D, kRunAmpConst, true>(p, tile, n_t0, len_t, pop, part, accumulate, tid, nthr);
                else run_eval_tile<D, kRunAmpLinear, true>(p, tile, n_t0, len_t, pop, part, accumulate, tid, nthr);
            } else {
                if (OBJ == kObjCor) run_eval_tile<D, kRunAmpCor, false>(p, tile, n_t0, len_t, pop, part, accumulate, tid, nthr);
                else if (a1z) run_eval_tile<D, kRunAmpConst, false>(p, tile, n_t0, len_t, pop, part, accumulate, tid, nthr);
                else run_eval_tile<D, kRunAmpLinear, false>(p, tile, n_t0, len_t, pop, part, accumulate, tid, nthr);
            }
        };
        auto evaluate = [&](const double* pop) {
            if (STREAM) {
                const int nT = (p.N + p.TS - 1) / p.TS;
                for (int jt = 0; jt < nT; ++jt) {
                    if (tid == 0 && st.to_issue > 0) run_stream_issue_one(p, st);
                    const int s = (int)(st.cons % (uint32_t)p.S);
                    mbar_wait_suspended(&st.full[s], (st.cons / (uint32_t)p.S) & 1u);
                    eval_tile(st.stages + (size_t)s * p.TS, jt * p.TS, min(p.TS, p.N - jt * p.TS), pop, jt > 0);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&st.empty[s]);
                    ++st.cons;
                }
            } else {
                eval_tile(xs, n_lo, Nown, pop, false);
            }
        };

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
                for (int j = 0; j < D; ++j) popA[i * D + j] = (double)pp[j];
            }
        }
        if (STREAM) {
            fence_proxy_async_global();      // a workspace row written above is read by the bulk copies below
            __syncthreads();
            if (tid == 0) {
                st.xsrc = xrow;
                st.to_issue = ((MODE == kModeFit) ? (uint32_t)p.G + 1u : 1u) * (uint32_t)((p.N + p.TS - 1) / p.TS);
                st.j_issue = 0;
                for (int k = 0; k < p.S - 2 && st.to_issue > 0; ++k) run_stream_issue_one(p, st);
            }
        } else {
            if (p.use_bulk && !quantised) mbar_wait(bar, parity);
            parity ^= 1u;
            __syncthreads();
        }
        evaluate(popA);
        __syncthreads();
        combine_begin();
        for (int i = tid; i < p.NP; i += nthr) {
            const double s = combined(i, popA);
            fit[i] = s;
            if (MODE == kModeFitness && rank == 0) p.fitness_out[blk * (long long)p.NP + i] = (float)reported(s);
        }
        ++xchg;
        __syncthreads();

        if (MODE == kModeFit) {
            // ---- a2..a7: generations ----
            for (int g = 1; g <= p.G; ++g) {
                // best member of the population the trials are built from (strategies 2 and 3); every warp finds it
                int ibest = 0;
                if (p.strategy == kLocalToBest1 || p.strategy == kBest1Jitter) {
                    double bv, mx;
                    warp_argmin(bv, ibest, mx);
                }
                for (int i = tid; i < p.NP; i += nthr) {
                    const Draws dr = de_draws<D>((uint32_t)i, (uint32_t)g, bidx, (uint32_t)p.NP, p.CR32, p.key0, p.key1);
                    double th[D];
                    if (p.strategy == kRand1) {
#pragma unroll
                        for (int j = 0; j < D; ++j) {
                            const double parent = popA[i * D + j];
                            const double mut = mutate_coord(popA[dr.r1 * D + j], popA[dr.r2 * D + j], popA[dr.r3 * D + j], p.F, lo_s[j], hi_s[j]);
                            th[j] = ((dr.mask >> j) & 1u) ? mut : parent;
                        }
                    } else {
                        const AuxDraws ax = aux_draws<D>(p.strategy, (uint32_t)i, (uint32_t)g, bidx, p.key0, p.key1);
#pragma unroll
                        for (int j = 0; j < D; ++j) {
                            const double parent = popA[i * D + j];
                            const double v = mutant_coord(p.strategy, parent, popA[dr.r1 * D + j], popA[dr.r2 * D + j], popA[dr.r3 * D + j],
                                                          popA[ibest * D + j], p.F, ax.jit[j], ax.u);
                            th[j] = ((dr.mask >> j) & 1u) ? bound_coord(v, lo_s[j], hi_s[j]) : parent;
                        }
                    }
#pragma unroll
                    for (int j = 0; j < D; ++j) popT[i * D + j] = th[j];
                }
                __syncthreads();
                evaluate(popT);
                __syncthreads();
                combine_begin();
                // ---- a6: greedy selection, accept on <= ----
                for (int i = tid; i < p.NP; i += nthr) {
                    const double s = combined(i, popT);
                    if (s <= fit[i]) {
                        fit[i] = s;
#pragma unroll
                        for (int j = 0; j < D; ++j) popA[i * D + j] = popT[i * D + j];
                    }
                }
                ++xchg;
                __syncthreads();
            }

            // ---- a8: best member (lowest index on ties), status, optional final population (cluster: CTA 0 writes) ----
            if (warp == 0 && rank == 0) {
                double bv, mx;
                int bi;
                warp_argmin(bv, bi, mx);
                if (lane == 0) {
                    uint32_t stw = 0;
#pragma unroll
                    for (int j = 0; j < D; ++j) {
                        const double v = popA[bi * D + j];
                        p.best[blk * D + j] = v;
                        const double w = hi_s[j] - lo_s[j];
                        if (w > 0.0 && (v - lo_s[j] <= 1e-6 * w || hi_s[j] - v <= 1e-6 * w)) stw |= 1u;
                    }
                    const double braw = fit[bi];                       // as evaluated (NaN stays NaN in the output)
                    if (OBJ == kObjCor) {
                        const double fb = reported(bv), fw = reported(mx);
                        if (fw - fb > 1e-3 * fb) stw |= 2u;
                        p.best_rss[blk] = (float)reported(braw);
                    } else {
                        if (mx - bv > 1e-3 * bv) stw |= 2u;
                        p.best_rss[blk] = (float)braw;
                    }
                    if (!(fabs(braw) <= 3.0e38)) stw |= 8u;            // objective of the best member is not finite
                    if (flags[6] != 0.0) stw |= 16u;                   // the caller's box has lo > hi (or NaN) in some coordinate
                    p.status[blk] = stw;
                }
            }
            if (p.final_pop && rank == 0) {
                float* fp = p.final_pop + blk * (long long)p.NP * D;
                for (int i = tid; i < p.NP * D; i += nthr) fp[i] = (float)popA[i];
            }
            if (p.final_fit && rank == 0) {
                float* ff = p.final_fit + blk * (long long)p.NP;
                for (int i = tid; i < p.NP; i += nthr) ff[i] = (float)reported(fit[i]);
            }
        }
        __syncthreads();   // xs / popA are reused by the next block of this CTA
    }
    // no CTA of a cluster exits while a peer may still store into its shared memory
    if (K > 1) cluster_sync_all();
}

}  // namespace pt
