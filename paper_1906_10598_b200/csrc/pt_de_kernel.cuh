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
//     FFMA  A' = t (-a1) + (-a0)
//     FFMA  r  = A' c + x
//     FFMA  acc += r r
// i.e. 7 FP32-pipe operations + 1 MUFU per sample-evaluation (one more FFMA for D = 6).  Lanes own samples and
// every thread carries C candidates in registers (register blocking), so the shared-memory loads and the t_n
// computation are amortised over C.  The six FADD/FFMA are issued as Blackwell packed-pair instructions
// (PTX add/fma.rn.f32x2 -> SASS FADD2/FFMA2) over PAIRS OF CANDIDATES with the sample value as the broadcast
// scalar operand: 5.4 issue slots per sample-evaluation instead of 8.4, which is what lets the XU (MUFU) pipe,
// the roofline of this loop, stay fed (measured: 10.9 -> 13.2 sample-evaluations/clk/SM).
#pragma once
#include "pt_device.cuh"

namespace pt {

constexpr int kChunk = 128;        // samples per warp step: 32 lanes x 4 consecutive samples (one LDS.128 each)
constexpr int kCandStride = 8;     // floats per candidate in the evaluation table
constexpr int kPairStride = 16;    // floats per candidate PAIR: (-a0,-a1,d0,d1,d2,d3,-,-) interleaved lo/hi
constexpr int kBarBytes = 128;     // mbarrier area at the start of shared memory
constexpr int kMaxStages = 7;

enum Mode { kModeFit = 0, kModeFitness = 1 };
// Objective: chi^2 of Eq. 4 or the correlation objective of Eq. 5-6,
//     F_cor = 1 / (arctan(cor) + pi/2),  cor = sum_n x_n a0 cos(phi(t_n))       (constant amplitude a0, a1 unused).
// F_cor is strictly decreasing in cor, so the kernel minimises -cor (fp32) and maps to F_cor only on output.
enum Objective { kObjChi2 = 0, kObjCor = 1 };
// Third evaluation kind, chosen per block at run time under kObjChi2: the amplitude slope is fixed at zero (the caller's a1
// box is [0, 0]; "c5 ... can be ignored when amplitude change is small with data length below 10 seconds"),
// so A(t) = a0 and the amplitude FFMA2 drops out: 6 instead of 7 FP32 operations per sample-evaluation.
constexpr int kEvalChi2Const = 2;

struct BlockParams {
    const float* x;               // [B][N] fp32 samples, or null when the samples are quantised:
    const unsigned char* xq;      // [B][row_bytes] packed samples (Quant q says how), unpacked while staging
    long long row_bytes;
    Quant q;
    const double* lo;             // [B][D]  (fit)
    const double* hi;             // [B][D]  (fit)
    const uint32_t* block_index;  // [B] or null (fit)
    const uint32_t* sel;          // [B] or null: when given, work item j of [blk0, B) is data block sel[j] (re-search of a subset)
    const int* count;             // device scalar or null: when given, only work items [blk0, blk0 + *count) exist (the length of
                                  // sel, known on the device only: pt_refit_doubtful never synchronises)
    const float* pop_in;          // [B][NP][D] (fitness)
    float* fitness_out;           // [B][NP]    (fitness)
    double* best;                 // [B][D]
    float* best_rss;              // [B]
    uint32_t* status;             // [B]
    float* final_pop;             // [B][NP][D] or null
    float* final_fit;             // [B][NP] or null
    long long B;                  // blocks [blk0, B) are fitted by this launch
    long long blk0;
    int N, Npad, NP, NPpad, G;
    double fs, t0, F;
    double dt;                    // 1 / fs (set on the host: pt_run_kernel reads it once per run instead of dividing)
    float dtf, t0f;               // dt and t0 rounded to fp32 (amplitude time base of pt_run_kernel)
    uint32_t CR32, key0, key1;
    int strategy;                 // Strategy (pt_device.cuh), 1..6
    int Wg, Ws;                   // warp grid of the evaluation phase, Wg * Ws = warps per CTA
    int use_bulk;                 // rows of x are 16-byte aligned and N % 4 == 0
    // streamed path (blocks larger than shared memory): tiles of TS samples move through a ring of S stages
    float* ws_wref;               // [grid][Npad] device workspace: reference phase of the block a CTA is fitting
    float* ws_x;                  // [grid][Npad] device workspace: 16-byte aligned copy of the block (only if !use_bulk)
    int TS, S;                    // samples per tile (multiple of kChunk), ring stages; S == 0: resident path
    // cluster path (few blocks, many SMs): K CTAs of one thread-block cluster fit ONE block together.  CTA r owns the
    // chunks [r nch / K, (r+1) nch / K) of the block (its own slice of the samples in shared memory), evaluates every
    // candidate over that slice, and the K partial sums of every candidate are exchanged through distributed shared
    // memory; the DE step itself is replicated (counter-based RNG, fp64: bit-identical in every CTA).
    int K;                        // CTAs per cluster = per block; 1: no cluster
    int tc_slots;                 // pt_tc_kernel: data blocks a CTA fits at the same time (1 or 2)
    int NpadS;                    // padded samples of the largest slice (= Npad when K == 1)
};

// The samples one CTA evaluates: the whole block (K == 1) or its slice of it.
struct Slice {
    int N, Npad;                  // valid / padded samples of the slice
    double t0;                    // time of the slice's first sample relative to the block centre
};

// Shared-memory carve-up, identical on host and device.
struct SmemLayout {
    int off_bar, off_xs, off_ws, off_popA, off_popT, off_box, off_fit, off_cand, off_part, off_xpart, total;
    __host__ __device__ static int align_up(int v, int a) { return (v + a - 1) / a * a; }
    // TS/S: tile samples and stages of the streamed path; S == 0: the whole block (xs, wref) is resident
    // Npad: padded samples this CTA keeps resident (its slice when K > 1); K: CTAs per cluster
    __host__ __device__ SmemLayout(int Npad, int NP, int NPpad, int D, int Ws, int TS = 0, int S = 0, int K = 1) {
        int o = 0;
        off_bar = o; o += kBarBytes;          // [0] staging barrier, [1..S] full, [1+S..2S] empty
        if (S > 0) {
            off_xs = o; o += S * TS * 8;      // stage s: x tile [TS] then reference-phase tile [TS]
            off_ws = off_xs;
        } else {
            off_xs = o; o += Npad * 4;
            off_ws = o; o += Npad * 4;
        }
        o = align_up(o, 16);
        off_popA = o; o += NP * D * 8;
        off_popT = o; o += NP * D * 8;
        off_box = o; o += 3 * 8 * 8;          // base[8], lo[8], hi[8]
        off_fit = o; o += NPpad * 4;
        o = align_up(o, 16);
        off_cand = o; o += NPpad * kCandStride * 4;
        off_part = o; o += Ws * NPpad * 4;
        off_xpart = o; o += (K > 1) ? 2 * K * NPpad * 4 : 0;     // [2][K][NPpad]: peers' partial sums, double-buffered
        total = align_up(o, 16);
    }
};

// ---------------------------------------------------------------------------------------------------
// Packed fp32 pairs (sm_100 FADD2 / FFMA2).
// ---------------------------------------------------------------------------------------------------
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) {
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}

// ---------------------------------------------------------------------------------------------------
// Evaluation of one group of C = 2 P candidates over one chunk: 4 consecutive samples of this lane.
// ---------------------------------------------------------------------------------------------------
template <int P, int D, bool MASKED, int OBJ>
__device__ __forceinline__ void eval_chunk(const float4 xv, const float4 wv, const float nf, const float dtf,
                                           const float (&tb)[4], const int n_left, const f32x2 (&na0)[P],
                                           const f32x2 (&na1)[P], const f32x2 (&d0)[P], const f32x2 (&d1)[P],
                                           const f32x2 (&d2)[P], const f32x2 (&d3)[P], f32x2 (&acc)[P]) {
    const float xs4[4] = {xv.x, xv.y, xv.z, xv.w};
    const float ws4[4] = {wv.x, wv.y, wv.z, wv.w};
    float t[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) t[j] = fmaf(nf, dtf, tb[j]);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        // the sample's scalars as broadcast operands (SASS: Rn.F32, no extra registers)
        const f32x2 t2 = pack2(t[j], t[j]), w2 = pack2(ws4[j], ws4[j]);
        const float xm = (MASKED && j >= n_left) ? 0.0f : xs4[j];
        const f32x2 x2 = pack2(xm, xm);
#pragma unroll
        for (int q = 0; q < P; ++q) {
            f32x2 h;
            if (D == 6) h = fma2(fma2(d3[q], t2, d2[q]), t2, d1[q]);
            else h = fma2(d2[q], t2, d1[q]);
            const f32x2 y = fma2(h, t2, add2(d0[q], w2));
            float y0, y1;
            unpack2(y, y0, y1);
            const f32x2 cs = pack2(__cosf(y0), __cosf(y1));
            if (OBJ == kObjCor) {
                acc[q] = fma2(cs, x2, acc[q]);                     // Eq. 5-6: sum x cos(phi); a padded sample has x = 0
            } else {
                f32x2 A;
                if (OBJ == kEvalChi2Const) A = na0[q];             // constant amplitude (a1 = 0)
                else A = fma2(na1[q], t2, na0[q]);
                if (MASKED && j >= n_left) A = pack2(0.0f, 0.0f);  // padded sample: residual 0 - 0 * c
                const f32x2 r = fma2(A, cs, x2);
                acc[q] = fma2(r, r, acc[q]);
            }
        }
    }
}

template <int C>
__device__ __forceinline__ void reduce_and_store(float (&acc)[C], const int lane, float* out, const bool accumulate = false) {
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
    if ((lane & (32 / C - 1)) == 0) out[cidx] = accumulate ? out[cidx] + v : v;
}

// Not inlined on purpose: the loop's register allocation (which decides the operand-bank conflicts of the FFMA2 stream, the
// binding resource of this loop) then does not depend on the code around it in the kernel.  Measured on config 2: 2101 ms
// inlined vs 2071 ms as a call, with identical instruction mixes.
template <int C, int D, int OBJ>
__device__ __noinline__ void eval_population(const BlockParams& p, const Slice& sl, const float* __restrict__ xs,
                                                const float* __restrict__ wref, const float* __restrict__ cand,
                                                float* __restrict__ part, const int warp, const int lane) {
    constexpr int P = C / 2;
    const int wg = warp % p.Wg, wsl = warp / p.Wg;
    const int nch = sl.Npad / kChunk;
    const int kb = (int)(((long long)wsl * nch) / p.Ws), ke = (int)(((long long)(wsl + 1) * nch) / p.Ws);
    const bool tail = (sl.N % kChunk) != 0;            // the last chunk of the slice is partial
    const int ke_full = (tail && ke == nch) ? ke - 1 : ke;
    const double dt = 1.0 / p.fs;
    const float dtf = (float)dt;
    float tb[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) tb[j] = (float)(sl.t0 + j * dt);
    float* out_row = part + wsl * p.NPpad;
    const int groups = p.NPpad / C;
    for (int g = wg; g < groups; g += p.Wg) {
        f32x2 na0[P], na1[P], d0[P], d1[P], d2[P], d3[P], acc[P];
        const ulonglong2* cg = reinterpret_cast<const ulonglong2*>(cand + (size_t)g * P * kPairStride);
#pragma unroll
        for (int q = 0; q < P; ++q) {
            const ulonglong2 u = cg[4 * q], v = cg[4 * q + 1], w = cg[4 * q + 2];
            na0[q] = u.x; na1[q] = u.y; d0[q] = v.x; d1[q] = v.y; d2[q] = w.x; d3[q] = w.y;
            acc[q] = pack2(0.0f, 0.0f);
        }
        const float4* xp = reinterpret_cast<const float4*>(xs) + kb * 32 + lane;
        const float4* wp = reinterpret_cast<const float4*>(wref) + kb * 32 + lane;
        float nf = (float)(kb * kChunk + lane * 4);
#pragma unroll 4   // four chunks per trip: fewer drain/fill bubbles of the MUFU results (+2 % on config 2)
        for (int k = kb; k < ke_full; ++k) {
            eval_chunk<P, D, false, OBJ>(*xp, *wp, nf, dtf, tb, 4, na0, na1, d0, d1, d2, d3, acc);
            xp += 32; wp += 32; nf += (float)kChunk;
        }
        if (ke_full < ke) {
            const int n_left = sl.N - ((nch - 1) * kChunk + lane * 4);    // valid samples of this lane (may be <= 0)
            eval_chunk<P, D, true, OBJ>(*xp, *wp, nf, dtf, tb, n_left, na0, na1, d0, d1, d2, d3, acc);
        }
        float accs[C];
#pragma unroll
        for (int q = 0; q < P; ++q) unpack2(acc[q], accs[2 * q], accs[2 * q + 1]);
        reduce_and_store<C>(accs, lane, out_row + g * C);
    }
}

// ---------------------------------------------------------------------------------------------------
// Streamed evaluation (blocks larger than shared memory, BASELINE config 4: 64 K and 256 K samples).
// The block's samples and its fp32 reference phase (computed once per block into the device workspace) move
// through a ring of S shared-memory stages, TS samples per tile, by 1-D bulk async copies (UBLKCP) with a
// full/empty mbarrier pair per stage.  Thread 0 is the producer: at tile c it refills the stage that tile
// c - 2 used, so it only ever waits for warps that are two tiles behind.  The tile sequence simply repeats for
// every generation (the data do not depend on the generation), so copies keep flowing through the DE step.
// Per tile every warp evaluates its candidate groups over its slice of the tile with the same eval_chunk as
// the resident path and adds its partial sums to part[slice][candidate].
// ---------------------------------------------------------------------------------------------------
struct Stream {
    uint64_t* full;          // [S]
    uint64_t* empty;         // [S]
    float* stages;           // S x (x tile [TS], wref tile [TS])
    const float* xsrc;       // block's samples in global memory (16-byte aligned rows)
    const float* wsrc;       // block's reference phase in the workspace
    uint32_t cons;           // tiles consumed since kernel start (all threads)
    uint32_t prod;           // tiles issued since kernel start (thread 0)
    uint32_t to_issue;       // tiles of the current block not yet issued (thread 0)
    int j_issue;             // tile index within the pass of the next tile to issue (thread 0)
};

__device__ __forceinline__ void stream_issue_one(const BlockParams& p, Stream& st) {
    const int s = (int)(st.prod % (uint32_t)p.S);
    const uint32_t k = st.prod / (uint32_t)p.S;
    if (k >= 1) mbar_wait(&st.empty[s], (k - 1) & 1u);        // every warp has released the previous fill
    const int n0 = st.j_issue * p.TS;
    // sizes are multiples of 16 bytes: N % 4 == 0 on the direct path, else the source is the zero-padded workspace copy
    const uint32_t wb = (uint32_t)min(p.TS, p.Npad - n0) * 4u;
    const uint32_t xb = p.use_bulk ? (uint32_t)min(p.TS, p.N - n0) * 4u : wb;
    float* dx = st.stages + (size_t)s * 2 * p.TS;
    mbar_arrive_expect_tx(&st.full[s], xb + wb);
    bulk_g2s(dx, st.xsrc + n0, xb, &st.full[s]);
    bulk_g2s(dx + p.TS, st.wsrc + n0, wb, &st.full[s]);
    ++st.prod; --st.to_issue;
    st.j_issue = (st.j_issue + 1 == (p.Npad + p.TS - 1) / p.TS) ? 0 : st.j_issue + 1;
}

// called by thread 0 after the block's workspace rows are written and fenced: tiles of `passes` evaluation passes
__device__ __forceinline__ void stream_begin_block(const BlockParams& p, Stream& st, const float* xsrc, const float* wsrc,
                                                   uint32_t passes) {
    st.xsrc = xsrc; st.wsrc = wsrc;
    st.to_issue = passes * (uint32_t)((p.Npad + p.TS - 1) / p.TS);
    st.j_issue = 0;
    for (int k = 0; k < p.S - 2 && st.to_issue > 0; ++k) stream_issue_one(p, st);
}

template <int C, int D, int OBJ>
__device__ __forceinline__ void eval_population_streamed(const BlockParams& p, Stream& st, const float* __restrict__ cand,
                                                         float* __restrict__ part, const int tid, const int warp,
                                                         const int lane) {
    constexpr int P = C / 2;
    const int wg = warp % p.Wg, wsl = warp / p.Wg;
    const int nT = (p.Npad + p.TS - 1) / p.TS;
    const int nch = p.Npad / kChunk;
    const bool tail = (p.N % kChunk) != 0;
    const double dt = 1.0 / p.fs;
    const float dtf = (float)dt;
    float tb[4];
#pragma unroll
    for (int j = 0; j < 4; ++j) tb[j] = (float)(p.t0 + j * dt);
    float* out_row = part + wsl * p.NPpad;
    const int groups = p.NPpad / C;
    for (int jt = 0; jt < nT; ++jt) {
        if (tid == 0 && st.to_issue > 0) stream_issue_one(p, st);
        const int s = (int)(st.cons % (uint32_t)p.S);
        mbar_wait(&st.full[s], (st.cons / (uint32_t)p.S) & 1u);
        const float* xs = st.stages + (size_t)s * 2 * p.TS;
        const float* wref = xs + p.TS;
        const int c0 = jt * (p.TS / kChunk);                          // first chunk of this tile in the block
        const int nct = min(p.TS / kChunk, nch - c0);                 // chunks in this tile
        const int kb = (int)(((long long)wsl * nct) / p.Ws), ke = (int)(((long long)(wsl + 1) * nct) / p.Ws);
        const int ke_full = (tail && c0 + ke == nch) ? ke - 1 : ke;
        for (int g = wg; g < groups; g += p.Wg) {
            f32x2 na0[P], na1[P], d0[P], d1[P], d2[P], d3[P], acc[P];
            const ulonglong2* cg = reinterpret_cast<const ulonglong2*>(cand + (size_t)g * P * kPairStride);
#pragma unroll
            for (int q = 0; q < P; ++q) {
                const ulonglong2 u = cg[4 * q], v = cg[4 * q + 1], w = cg[4 * q + 2];
                na0[q] = u.x; na1[q] = u.y; d0[q] = v.x; d1[q] = v.y; d2[q] = w.x; d3[q] = w.y;
                acc[q] = pack2(0.0f, 0.0f);
            }
            const float4* xp = reinterpret_cast<const float4*>(xs) + kb * 32 + lane;
            const float4* wp = reinterpret_cast<const float4*>(wref) + kb * 32 + lane;
            float nf = (float)((c0 + kb) * kChunk + lane * 4);
#pragma unroll 2   // measured: 1 -> 2 gives +2 points at D = 6, NP = 400 (paper-shaped blocks), neutral at D = 5; 4 is worse
            for (int k = kb; k < ke_full; ++k) {
                eval_chunk<P, D, false, OBJ>(*xp, *wp, nf, dtf, tb, 4, na0, na1, d0, d1, d2, d3, acc);
                xp += 32; wp += 32; nf += (float)kChunk;
            }
            if (ke_full < ke) {
                const int n_left = p.N - ((nch - 1) * kChunk + lane * 4);
                eval_chunk<P, D, true, OBJ>(*xp, *wp, nf, dtf, tb, n_left, na0, na1, d0, d1, d2, d3, acc);
            }
            float accs[C];
#pragma unroll
            for (int q = 0; q < P; ++q) unpack2(acc[q], accs[2 * q], accs[2 * q + 1]);
            reduce_and_store<C>(accs, lane, out_row + g * C, jt > 0);
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&st.empty[s]);
        ++st.cons;
    }
}

// Evaluation-table entry of member i: NEGATED amplitudes (so that the residual is one FMA, r = A' c + x) and the
// phase-polynomial offsets from the block's fp64 reference, in radians: d0 = phi0 - phi0_b, d1 = 2 pi (f - f_b),
// d2 = pi (fdot - fdot_b), d3 = (pi/3)(fddot - fddot_b).  Members 2q and 2q+1 share a row, interleaved lo/hi,
// so that the evaluation loop loads candidate PAIRS straight into 64-bit registers.
template <int D>
__device__ __forceinline__ void write_cand(float* cand, const int i, const double* th, const double* base) {
    float* ce = cand + (size_t)(i >> 1) * kPairStride + (i & 1);
    ce[0] = -(float)th[0];
    ce[2] = -(float)th[1];
    ce[4] = (float)(th[2] - base[2]);
    ce[6] = (float)(kTwoPi * (th[3] - base[3]));
    ce[8] = (float)(kPi * (th[4] - base[4]));
    ce[10] = (D == 6) ? (float)((kPi / 3.0) * (th[5] - base[5])) : 0.0f;
}

template <int C, int D, int MODE, bool STREAM, int OBJ>
__global__ void __launch_bounds__(512, 1) pt_block_kernel(const BlockParams p) {
    extern __shared__ __align__(16) unsigned char smem[];
    const SmemLayout L(p.NpadS, p.NP, p.NPpad, D, p.Ws, p.TS, p.S, p.K);
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
    float* xpart = reinterpret_cast<float*>(smem + L.off_xpart);

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31;
    uint32_t parity = 0;

    // ---- cluster geometry: CTA `rank` of K owns the chunks [c_lo, c_hi) of every block its cluster fits ----
    const int K = STREAM ? 1 : p.K;
    const int rank = (K > 1) ? (int)cluster_ctarank() : 0;
    const long long first_blk = (K > 1) ? (long long)cluster_id_x() : (long long)blockIdx.x;
    const long long blk_stride = (long long)gridDim.x / K;
    Slice sl;
    int n_lo = 0;
    {
        const int nch_blk = p.Npad / kChunk;
        const int c_lo = (int)(((long long)rank * nch_blk) / K), c_hi = (int)(((long long)(rank + 1) * nch_blk) / K);
        n_lo = c_lo * kChunk;
        sl.Npad = (c_hi - c_lo) * kChunk;
        sl.N = max(0, min(p.N, c_hi * kChunk) - n_lo);
        sl.t0 = p.t0 + (double)n_lo * (1.0 / p.fs);
    }
    uint32_t xchg = 0;             // exchanges of partial sums done so far (selects the xpart buffer)

    Stream st;
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
    // padded evaluation-table rows evaluate a zero model; their sums are never read
    for (int i = tid; i < p.NPpad * kCandStride; i += nthr) cand[i] = 0.0f;
    __syncthreads();
    if (K > 1) cluster_sync_all();     // every CTA of the cluster is running before any peer store is issued

    // Sum of the Ws slice partials of member i; with a cluster, the K CTAs' sums are exchanged through distributed
    // shared memory and added in rank order, so every CTA of the cluster holds the same fp32 value.
    auto combine_begin = [&]() {
        if (K > 1) {
            float* buf = xpart + (size_t)(xchg & 1u) * K * p.NPpad;
            for (int i = tid; i < p.NP; i += nthr) {
                float s = 0.0f;
                for (int w = 0; w < p.Ws; ++w) s += part[w * p.NPpad + i];
                const float* slot = buf + (size_t)rank * p.NPpad + i;
                for (int r = 0; r < K; ++r) st_cluster_f32(mapa_shared(slot, (uint32_t)r), s);
            }
            cluster_sync_all();
        }
    };
    auto combined = [&](int i) -> float {
        float s = 0.0f;
        if (K > 1) {
            const float* buf = xpart + (size_t)(xchg & 1u) * K * p.NPpad;
            for (int r = 0; r < K; ++r) s += buf[(size_t)r * p.NPpad + i];
        } else {
            for (int w = 0; w < p.Ws; ++w) s += part[w * p.NPpad + i];
        }
        // Eq. 5-6: s = sum x cos(phi); the value minimised is -cor = (-a0) s   (first entry of member i's table row)
        if (OBJ == kObjCor) s *= cand[(size_t)(i >> 1) * kPairStride + (i & 1)];
        return s;
    };
    // argmin of fit[0..NP) with the lowest index on ties, and the maximum; every lane of the calling warp gets them
    auto warp_argmin = [&](float& bv, int& bi, float& mx) {
        // a NaN objective (a non-finite sample makes every member's sum NaN) compares false with everything: it is read
        // as +inf, so that the index stays inside the population (all NaN -> member 0) and the block is flagged by status bit 3
        bv = INFINITY; mx = -INFINITY; bi = 0x7fffffff;
        for (int i = lane; i < p.NP; i += 32) {
            float v = fit[i];
            if (!(v == v)) v = INFINITY;
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
    };
    // value reported for a minimised fp32 value v: the RSS itself, or F_cor - 1/pi of cor = -v (PAPER.md:161 displays
    // the correlation objective with the constant 0.31830988618 subtracted), computed in fp64
    auto reported = [&](float v) -> double {
        if (OBJ == kObjCor) return 1.0 / (atan(-(double)v) + 0.5 * kPi) - 1.0 / kPi;
        return (double)v;
    };

    const long long item_end = p.count ? min(p.B, p.blk0 + (long long)*p.count) : p.B;
    for (long long item = p.blk0 + first_blk; item < item_end; item += blk_stride) {
        const long long blk = p.sel ? (long long)p.sel[item] : item;
        const bool quantised = p.q.bits != 0;
        const float* xg = quantised ? nullptr : p.x + blk * (long long)p.N + n_lo;      // this CTA's slice of the block
        const unsigned char* xqrow = quantised ? p.xq + blk * p.row_bytes : nullptr;
        // ---- a0: stage the block's samples (PAPER.md:121 data block) into shared memory, once ----
        //      (streamed path: tiles are staged every pass; an unaligned or quantised row is first written to the
        //       workspace as fp32).  Quantised samples (Table 3) are unpacked here, once per block.
        float* wrow = STREAM ? p.ws_wref + (size_t)blockIdx.x * p.Npad : nullptr;
        const float* xrow = xg;
        if (STREAM) {
            if (quantised || !p.use_bulk) {
                float* xw = p.ws_x + (size_t)blockIdx.x * p.Npad;
                if (quantised) for (int n = tid; n < p.Npad; n += nthr) xw[n] = (n < p.N) ? unpack_sample(xqrow, n, p.q) : 0.0f;
                else for (int n = tid; n < p.Npad; n += nthr) xw[n] = (n < p.N) ? __ldg(xg + n) : 0.0f;
                xrow = xw;
            }
        } else if (quantised) {
            for (int n = tid; n < sl.N; n += nthr) xs[n] = unpack_sample(xqrow, (long long)n_lo + n, p.q);
        } else if (p.use_bulk) {
            if (tid == 0) {
                fence_proxy_async();   // earlier generic-proxy reads of xs are ordered before the async writes
                const uint32_t bytes = (uint32_t)sl.N * 4u;
                mbar_arrive_expect_tx(bar, bytes);
                for (uint32_t o = 0; o < bytes; o += 32768u) {
                    const uint32_t len = min(32768u, bytes - o);
                    bulk_g2s(reinterpret_cast<unsigned char*>(xs) + o, reinterpret_cast<const unsigned char*>(xg) + o,
                             len, bar);
                }
            }
        } else {
            for (int n = tid; n < sl.N; n += nthr) xs[n] = __ldg(xg + n);
        }
        if (!STREAM)
            for (int n = sl.N + tid; n < sl.Npad; n += nthr) xs[n] = 0.0f;

        // ---- box, reference point ----
        if (MODE == kModeFit) {
            if (tid < D) {
                const double l = p.lo[blk * D + tid], h = p.hi[blk * D + tid];
                lo_s[tid] = l; hi_s[tid] = h;
                base[tid] = 0.5 * (l + h);
                if (tid == 1) base[7] = (l == 0.0 && h == 0.0) ? 1.0 : 0.0;     // amplitude slope fixed at zero
            }
            if (tid == 32) {   // lo <= hi is the caller's contract (pt.h); an asynchronous call reports a violation in status bit 4
                bool bad = false;
                for (int j = 0; j < D; ++j) bad = bad || !(p.lo[blk * D + j] <= p.hi[blk * D + j]);
                base[6] = bad ? 1.0 : 0.0;
            }
        } else {
            if (tid < D) {   // mid-range of the given population
                const float* pp = p.pop_in + blk * (long long)p.NP * D + tid;
                float mn = pp[0], mx = pp[0];
                for (int i = 1; i < p.NP; ++i) { const float v = pp[(size_t)i * D]; mn = fminf(mn, v); mx = fmaxf(mx, v); }
                base[tid] = 0.5 * ((double)mn + (double)mx);
                if (tid == 1) base[7] = (mn == 0.0f && mx == 0.0f) ? 1.0 : 0.0;
            }
            if (tid == 32) base[6] = 0.0;
        }
        __syncthreads();

        // ---- reference phase W_n = [phi_b(t_n)] mod 2 pi in fp64, stored fp32 in [-pi, pi) ----
        {
            const double b0 = base[2] * (1.0 / kTwoPi), b1 = base[3], b2 = 0.5 * base[4];
            const double b3 = (D == 6) ? base[5] * (1.0 / 6.0) : 0.0;
            const double dt = 1.0 / p.fs;
            const int nw = STREAM ? p.Npad : sl.Npad;
            for (int n = tid; n < nw; n += nthr) {
                const double t = sl.t0 + (double)n * dt;
                double u = b0 + t * (b1 + t * (b2 + t * b3));     // turns
                u -= rint(u);
                if (STREAM) wrow[n] = (float)(kTwoPi * u);
                else wref[n] = (float)(kTwoPi * u);
            }
        }

        // one evaluation pass of the table `cand`; the constant-amplitude loop when this block's a1 is fixed at zero
        const bool a1z = (OBJ == kObjChi2) && base[7] != 0.0;
        auto evaluate = [&]() {
            if (STREAM) {
                if (a1z) eval_population_streamed<C, D, (OBJ == kObjChi2 ? kEvalChi2Const : OBJ)>(p, st, cand, part, tid, warp, lane);
                else eval_population_streamed<C, D, OBJ>(p, st, cand, part, tid, warp, lane);
            } else {
                if (a1z) eval_population<C, D, (OBJ == kObjChi2 ? kEvalChi2Const : OBJ)>(p, sl, xs, wref, cand, part, warp, lane);
                else eval_population<C, D, OBJ>(p, sl, xs, wref, cand, part, warp, lane);
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
                for (int j = 0; j < D; ++j) th[j] = (double)pp[j];
            }
            write_cand<D>(cand, i, th, base);
        }
        if (STREAM) {
            fence_proxy_async_global();      // workspace rows written above are read by the bulk copies below
            __syncthreads();
            if (tid == 0) stream_begin_block(p, st, xrow, wrow, (MODE == kModeFit) ? (uint32_t)p.G + 1u : 1u);
            evaluate();
        } else {
            if (p.use_bulk) mbar_wait(bar, parity);
            parity ^= 1u;
            __syncthreads();
            evaluate();
        }
        __syncthreads();
        combine_begin();
        for (int i = tid; i < p.NP; i += nthr) {
            const float s = combined(i);
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
                    float bv, mx;
                    warp_argmin(bv, ibest, mx);
                }
                for (int i = tid; i < p.NP; i += nthr) {
                    const Draws dr = de_draws<D>((uint32_t)i, (uint32_t)g, bidx, (uint32_t)p.NP, p.CR32, p.key0, p.key1);
                    double th[D];
                    if (p.strategy == kRand1) {
#pragma unroll
                        for (int j = 0; j < D; ++j) {
                            const double parent = popA[i * D + j];
                            const double mut = mutate_coord(popA[dr.r1 * D + j], popA[dr.r2 * D + j], popA[dr.r3 * D + j],
                                                            p.F, lo_s[j], hi_s[j]);
                            th[j] = ((dr.mask >> j) & 1u) ? mut : parent;
                        }
                    } else {
                        const AuxDraws ax = aux_draws<D>(p.strategy, (uint32_t)i, (uint32_t)g, bidx, p.key0, p.key1);
#pragma unroll
                        for (int j = 0; j < D; ++j) {
                            const double parent = popA[i * D + j];
                            const double v = mutant_coord(p.strategy, parent, popA[dr.r1 * D + j], popA[dr.r2 * D + j],
                                                          popA[dr.r3 * D + j], popA[ibest * D + j], p.F, ax.jit[j], ax.u);
                            th[j] = ((dr.mask >> j) & 1u) ? bound_coord(v, lo_s[j], hi_s[j]) : parent;
                        }
                    }
#pragma unroll
                    for (int j = 0; j < D; ++j) popT[i * D + j] = th[j];
                    write_cand<D>(cand, i, th, base);
                }
                __syncthreads();
                evaluate();
                __syncthreads();
                combine_begin();
                // ---- a6: greedy selection, accept on <= ----
                for (int i = tid; i < p.NP; i += nthr) {
                    const float s = combined(i);
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
                float bv, mx;
                int bi;
                warp_argmin(bv, bi, mx);
                if (lane == 0) {
                    uint32_t st = 0;
#pragma unroll
                    for (int j = 0; j < D; ++j) {
                        const double v = popA[bi * D + j];
                        p.best[blk * D + j] = v;
                        const double w = hi_s[j] - lo_s[j];
                        if (w > 0.0 && (v - lo_s[j] <= 1e-6 * w || hi_s[j] - v <= 1e-6 * w)) st |= 1u;
                    }
                    const float braw = fit[bi];                        // as evaluated (NaN stays NaN in the output)
                    if (OBJ == kObjCor) {
                        const double fb = reported(bv), fw = reported(mx);
                        if (fw - fb > 1e-3 * fb) st |= 2u;
                        p.best_rss[blk] = (float)reported(braw);
                    } else {
                        if (mx - bv > 1e-3f * bv) st |= 2u;
                        p.best_rss[blk] = braw;
                    }
                    if (!(fabsf(braw) <= 3.0e38f)) st |= 8u;           // objective of the best member is not finite
                    if (base[6] != 0.0) st |= 16u;                     // the caller's box has lo > hi (or NaN) in some coordinate
                    p.status[blk] = st;
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
