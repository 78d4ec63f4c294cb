// pt_tc_kernel.cuh -- the tensor-core variant of the persistent one-CTA-per-data-block DE kernel (rows a0-a8 of SURVEY 8(a)).
//
// Same method, same DE step (Philox draws, fp64 mutation / crossover / bounds, selection on the fp32 objective) and same
// outputs as pt_block_kernel; what differs is who computes the phase of Eq. 3.  Here the phase of all 128
// candidates over a tile of 256 samples is ONE tcgen05.mma (kind::tf32, K = 16, fp32 accumulators in tensor memory):
//     phase[c][j] = sum_k A[c][k] B[j][k],   A = tile-local Taylor coefficients of candidate c in tf32-exact pieces,
//                                            B = the fixed basis (1, j, j^2, j^3), j = sample index - tile centre.
// Warp roles (640 threads, one CTA per SM):
//   warps 16-19  "producers": thread = candidate (of up to two data blocks in flight).  DE step; per tile the candidate's phase polynomial is re-expanded at the
//                tile centre in fp64 (value reduced mod 1 turn, so that fp32 never sees more than |E1| 128 rad), split into
//                tf32-exact pieces by integer bit operations and stored as a row of the A operand (ring of 4 operands);
//                lane 0 of warp 16 issues the MMAs (ring of 2 accumulators = all 512 TMEM columns) and commits to mbarriers;
//   warps 0-15   "consumers": TMEM lane = candidate (32 (warp % 4) + lane), warp / 4 = which 64 of the tile's 256 columns.
//                tcgen05.ld brings 16 phases at a time; per sample-evaluation: FMUL + MUFU.COS (cos.approx), 1/2 FADD2
//                (amplitude a0 + a1 t by a running sum), 1/2 FFMA2 (residual), 1/2 FFMA2 (square-accumulate): 4 FP32 lane
//                operations instead of pt_block_kernel's 7 (8 for D = 6), no shuffle reduction (a thread owns its candidate),
//                the sample value is a warp-uniform shared-memory broadcast.  D = 6 costs the same as D = 5: the cubic term
//                is three more slots of K.
// No reference-phase array: shared memory holds the samples only (4 bytes per sample), so blocks up to ~45 000 samples stay
// resident.  Measured numbers, the profile and the comparison with pt_block_kernel: DESIGN.md section 5.12, profiles/r2_*.
#pragma once
#include "pt_de_kernel.cuh"
#include "pt_tc_device.cuh"

namespace pt {

constexpr int kTcConsumerWarps = 16, kTcProducerWarps = 4;
constexpr int kTcThreads = (kTcConsumerWarps + kTcProducerWarps) * 32;     // 640
constexpr int kTcMaxNP = 128;                                              // one MMA M-tile of candidates
enum TcAmp { kTcAmpLinear = 0, kTcAmpConst = 1, kTcAmpCor = 2 };

// Shared-memory carve-up of the tensor-core kernel, identical on host and device.  A CTA fits `nslots` (1 or 2) data blocks
// at the same time ("slots"): while the producers run the DE step of one, the consumers evaluate the other, so the serial part
// of a generation (selection, trial vectors, first coefficient rows, pipeline fill) is hidden.
struct TcSmemLayout {
    int off_bar, off_tptr, off_opB, off_opA, off_slot, slot_stride;
    int s_popA, s_popT, s_box, s_fit, s_amp, s_part, s_xs;       // offsets inside a slot
    int total;
    __host__ __device__ static int align_up(int v, int a) { return (v + a - 1) / a * a; }
    __host__ __device__ TcSmemLayout(int N, int NP, int D, int nslots) {
        const int Npad = align_up(N, tc::kTile);
        int o = 0;
        off_bar = o; o += 16 * 8;              // [0] staging, a_full[4], a_empty[4], t_full[2], t_empty[2]
        off_tptr = o; o += 16;
        o = align_up(o, 128);
        off_opB = o; o += tc::kBBytes;
        off_opA = o; o += tc::kAStages * tc::kABytes;
        off_slot = o;
        int q = 0;
        s_popA = q; q += NP * D * 8;
        s_popT = q; q += NP * D * 8;
        s_box = q; q += 3 * 8 * 8;
        s_fit = q; q += kTcMaxNP * 8;          // objective values of the members, fp64 (see tc_consumer_pass)
        s_amp = q; q += kTcMaxNP * 2 * 4;      // (-a0, -a1) of every member: what the consumers need of a candidate
        s_part = q; q += 4 * kTcMaxNP * 8;     // [column group][candidate] partial sums, fp64
        q = align_up(q, 16);
        s_xs = q; q += Npad * 4;
        slot_stride = align_up(q, 128);
        total = off_slot + nslots * slot_stride;
    }
};

__device__ __forceinline__ f32x2 bc2(float v) { return pack2(v, v); }

// 16 consecutive samples of one candidate: u = phases [rad] from TMEM, xt = the samples (warp-uniform broadcast loads).
//   chi^2 (Eq. 4): r = A' cos(u) + x with the NEGATED amplitude A'(i) running in A2, acc += r^2; a padded sample has x = 0 and
//   is given A' = 0 (MASKED).   correlation (Eq. 5-6): acc += x cos(u).
template <int AMP, bool MASKED>
__device__ __forceinline__ void tc_consume16(const uint32_t (&u)[16], const float* __restrict__ xt, f32x2& A2, const f32x2 step, f32x2& acc,
                                             const int nvalid) {
    float xv[16];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        const float4 q = *reinterpret_cast<const float4*>(xt + 4 * k);
        xv[4 * k] = q.x; xv[4 * k + 1] = q.y; xv[4 * k + 2] = q.z; xv[4 * k + 3] = q.w;
    }
#pragma unroll
    for (int i = 0; i < 16; i += 2) {
        const f32x2 cc = pack2(__cosf(__uint_as_float(u[i])), __cosf(__uint_as_float(u[i + 1])));
        const f32x2 x2 = pack2(xv[i], xv[i + 1]);
        if (AMP == kTcAmpCor) {
            acc = fma2(cc, x2, acc);
        } else {
            f32x2 Ap = A2;
            if (AMP == kTcAmpLinear) A2 = add2(A2, step);
            if (MASKED) {
                float A0, A1;
                unpack2(Ap, A0, A1);
                if (i >= nvalid) A0 = 0.0f;
                if (i + 1 >= nvalid) A1 = 0.0f;
                Ap = pack2(A0, A1);
            }
            const f32x2 r = fma2(Ap, cc, x2);
            acc = fma2(r, r, acc);
        }
    }
}

struct TcConsumer {          // per-warp pipeline state of a consumer
    uint64_t* t_full; uint64_t* t_empty;
    uint32_t tbase;          // TMEM address of this warp's lane quarter and first column (buffer 0)
    uint32_t it;             // tiles consumed since kernel start (selects the accumulator and its mbarrier phase)
    int lane;
};

// Chunk K of a tile for a warp that owns 64 columns (four x16 loads through two 16-register buffers).  On entry chunk K is in
// flight into `cur`; the next chunk (or chunk 0 of the next tile) is started into `nxt` before chunk K is evaluated.
// INTERIOR: all 64 columns of the warp are samples of the block (every tile but the first and last of a block): no bounds
// checks, and the amplitude runs on from chunk to chunk.
template <int AMP, int K, bool INTERIOR>
__device__ __forceinline__ void tc_tile_chunk(uint32_t (&cur)[16], uint32_t (&nxt)[16], TcConsumer& st, const float* __restrict__ xw,
                                              const int n_first, const int N, const float g0w, const float g1, f32x2& A2, const f32x2 step,
                                              f32x2& acc, const bool has_next) {
    constexpr int nchunk = 4;
    tc::wait_ld();
    if (K == nchunk - 1) {
        // every load of this tile has landed: hand the accumulator back to the MMA issuer, then start on the next tile
        tc::fence_before_sync();
        __syncwarp();
        if (st.lane == 0) mbar_arrive(&st.t_empty[st.it % tc::kTmemBufs]);
        ++st.it;
        if (has_next) {
            if (st.lane == 0) tc::mbar_wait_sleep(&st.t_full[st.it % tc::kTmemBufs], (st.it / tc::kTmemBufs) & 1u);
            __syncwarp();
            tc::fence_after_sync();
            tc::tmem_ld16(st.tbase + (st.it % tc::kTmemBufs) * tc::kTile, nxt);
        }
    } else {
        tc::tmem_ld16(st.tbase + (st.it % tc::kTmemBufs) * tc::kTile + (K + 1) * 16, nxt);
    }
    if (INTERIOR) {
        tc_consume16<AMP, false>(cur, xw + K * 16, A2, step, acc, 16);
    } else {
        // sample index of the chunk's first column (a multiple of 16; negative or >= N: the chunk is padding and is skipped)
        const int n0 = n_first + K * 16;
        if (n0 >= 0 && n0 < N) {
            f32x2 Ac = (AMP == kTcAmpLinear) ? pack2(fmaf(g1, (float)(K * 16), g0w), fmaf(g1, (float)(K * 16 + 1), g0w)) : bc2(g0w);
            if (n0 + 16 <= N) tc_consume16<AMP, false>(cur, xw + K * 16, Ac, step, acc, 16);
            else tc_consume16<AMP, true>(cur, xw + K * 16, Ac, step, acc, N - n0);
        }
    }
    if constexpr (K + 1 < nchunk) tc_tile_chunk<AMP, K + 1, INTERIOR>(nxt, cur, st, xw, n_first, N, g0w, g1, A2, step, acc, has_next);
}

// One evaluation pass of a consumer warp over the block: sum over its 64 columns of every tile for its lane's candidate.
// Summation: fp32 FMA accumulation over the thread's 64 columns of a tile (two packed accumulators of 32 terms), then an
// error-free two-sum of the tile's value into a (hi, lo) pair -- 7 packed operations per tile and thread -- and fp64 from there
// on (partials, the members' objective values, the selection).  A plain fp32 accumulator over a thread's N/4 terms would carry
// ~1e-4 of absolute rounding at N = 10 000, two orders above what a 1e-3 Hz step of f moves the chi^2 of a faded block by
// (R20).
template <int AMP>
__device__ __forceinline__ double tc_consumer_pass(TcConsumer& st, const float* __restrict__ xs, const int N, const int nT, const int c0,
                                                   const int off, const float na0, const float na1, const float dtf, const float Ldtf,
                                                   const float tw0) {
    f32x2 hi = pack2(0.0f, 0.0f), lo = pack2(0.0f, 0.0f);
    const f32x2 neg1 = bc2(-1.0f);
    uint32_t ua[16], ub[16];
    const float g1 = na1 * dtf;
    const f32x2 step = bc2(2.0f * g1);
    float tauf = 0.0f;
    if (st.lane == 0) tc::mbar_wait_sleep(&st.t_full[st.it % tc::kTmemBufs], (st.it / tc::kTmemBufs) & 1u);
    __syncwarp();
    tc::fence_after_sync();
    tc::tmem_ld16(st.tbase + (st.it % tc::kTmemBufs) * tc::kTile, ua);
    for (int tau = 0; tau < nT; ++tau) {
        // negated amplitude A'(t) = -a0 - a1 t at the warp's first column of this tile (tw0 = its time in tile 0)
        const float g0w = (AMP == kTcAmpLinear) ? fmaf(na1, fmaf(tauf, Ldtf, tw0), na0) : na0;
        tauf += 1.0f;
        const int col = tau * tc::kTile + c0;          // position of the warp's first column in the padded sample array
        const int n_first = col - off;                 // its sample index
        f32x2 A2 = (AMP == kTcAmpLinear) ? pack2(g0w, g0w + g1) : bc2(g0w);
        f32x2 acc = pack2(0.0f, 0.0f);
        if (n_first >= 0 && n_first + 64 <= N) tc_tile_chunk<AMP, 0, true>(ua, ub, st, xs + col, n_first, N, g0w, g1, A2, step, acc, tau + 1 < nT);
        else tc_tile_chunk<AMP, 0, false>(ua, ub, st, xs + col, n_first, N, g0w, g1, A2, step, acc, tau + 1 < nT);
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
    return ((double)h0 + (double)h1) + ((double)l0 + (double)l1);
}

// argmin of fit[0..NP) with the lowest index on ties, and the maximum (a NaN is read as +inf); every lane gets them
__device__ __forceinline__ void tc_warp_argmin(const double* fit, const int NP, const int lane, double& bv, int& bi, double& mx) {
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    bv = inf; mx = -inf; bi = 0x7fffffff;
    for (int i = lane; i < NP; i += 32) {
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
}

// amp(slot): producers -> consumers, the amplitude table of the slot's candidates of this generation is written;
// part(slot): consumers -> producers, the slot's partial sums of this generation are written; kBarProd: producers only.
__device__ __forceinline__ int bar_amp(int slot) { return slot ? 4 : 1; }
__device__ __forceinline__ int bar_part(int slot) { return slot ? 5 : 2; }
constexpr int kBarProd = 3;
__device__ __forceinline__ void named_sync(int id, int count) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory"); }
__device__ __forceinline__ void named_arrive(int id, int count) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(count) : "memory"); }

struct TcProducer {          // per-thread pipeline state of a producer
    uint64_t* a_full; uint64_t* a_empty; uint64_t* t_full; uint64_t* t_empty;
    unsigned char* opA;
    uint32_t tmem, idesc;
    uint64_t db0, db1;       // descriptors of the two K halves of the basis operand
    uint32_t pit;            // tiles produced since kernel start
};

// All tiles of one evaluation pass for member `row` with parameters th (absolute, fp64): per tile the phase polynomial
//     P(t) = phi0/2pi + f t + fdot t^2/2 + fddot t^3/6   [turns]                       PAPER.md:132-137 (Eq. 3)
// is re-expanded at the tile centre t_c: E0 = 2 pi frac(P(t_c)), E1 = 2 pi dt P1(t_c), E2 = 2 pi dt^2 P2(t_c)/2,
// E3 = 2 pi dt^3 P3/6 (Pk = k-th derivative), so that phase(j) = E0 + E1 j + E2 j^2 + E3 j^3 for the sample j steps from
// the centre.  All in fp64 without a single conversion instruction (round-to-integer by the magic constant, pieces by bit
// operations): conversions would run on the XU pipe.
template <int D>
__device__ __forceinline__ void tc_produce_pass(TcProducer& pr, const BlockParams& p, const double* th, const bool active, const int row,
                                                const int nT, const int off, const int warp, const int lane) {
    const double dt = 1.0 / p.fs;
    const double c0 = th[2] * (1.0 / kTwoPi), c1 = th[3], c2 = 0.5 * th[4], c3 = (D == 6) ? th[5] * (1.0 / 6.0) : 0.0;
    const double k1 = kTwoPi * dt * c1, k2 = kTwoPi * dt * 2.0 * c2, k3 = kTwoPi * dt * 3.0 * c3;
    const double m2 = kTwoPi * dt * dt * c2, m3 = kTwoPi * dt * dt * 3.0 * c3;
    float E3h, E3m;
    tc::split2(kTwoPi * c3 * dt * dt * dt, E3h, E3m);
    const double Ldt = (double)tc::kTile * dt, tc0 = p.t0 + (double)(tc::kTile / 2 - off) * dt;
    double taud = 0.0;
    for (int tau = 0; tau < nT; ++tau, ++pr.pit) {
        const int s = (int)(pr.pit % tc::kAStages);
        if (pr.pit >= (uint32_t)tc::kAStages) {
            if (lane == 0) tc::mbar_wait_sleep(&pr.a_empty[s], ((pr.pit / tc::kAStages) - 1) & 1u);
            __syncwarp();
        }
        if (active) {
            const double tcen = fma(taud, Ldt, tc0);
            double P = fma(tcen, fma(tcen, fma(tcen, c3, c2), c1), c0);
            P -= __dadd_rn(__dadd_rn(P, 6755399441055744.0), -6755399441055744.0);      // P - rint(P), |P| < 2^51
            float e[16];
            tc::coef_row(kTwoPi * P, fma(tcen, fma(tcen, k3, k2), k1), fma(tcen, m3, m2), E3h, E3m, e);
            tc::write_row(pr.opA + s * tc::kABytes, row, e, tc::kAChunk);
        }
        taud += 1.0;
        fence_proxy_async();             // the rows are read by the tensor core through the async proxy
        __syncwarp();
        if (lane == 0) mbar_arrive(&pr.a_full[s]);
        if (warp == kTcConsumerWarps) {
            // ===== MMA issue: one thread on behalf of the CTA =====
            if (lane == 0) {
                const int b = (int)(pr.pit % tc::kTmemBufs);
                tc::mbar_wait_sleep(&pr.a_full[s], (pr.pit / tc::kAStages) & 1u);
                if (pr.pit >= (uint32_t)tc::kTmemBufs) tc::mbar_wait_sleep(&pr.t_empty[b], ((pr.pit / tc::kTmemBufs) - 1) & 1u);
                tc::fence_after_sync();
                const uint32_t abase = smem_u32(pr.opA + s * tc::kABytes);
                tc::mma_tf32(pr.tmem + b * tc::kTile, tc::make_desc(abase, tc::kAChunk, 128), pr.db0, pr.idesc, 0);
                tc::mma_tf32(pr.tmem + b * tc::kTile, tc::make_desc(abase + 2 * tc::kAChunk, tc::kAChunk, 128), pr.db1, pr.idesc, 1);
                tc::commit(&pr.a_empty[s]);      // the operand may be overwritten once both MMAs have read it
                tc::commit(&pr.t_full[b]);       // the accumulator is complete
            }
            __syncwarp();
        }
    }
}

template <int D, int MODE, int OBJ>
__global__ void __launch_bounds__(kTcThreads, 1) pt_tc_kernel(const BlockParams p) {
    extern __shared__ __align__(16) unsigned char smem[];   // operands need 16-byte alignment (no swizzle)
    const int nslots = p.tc_slots;
    const TcSmemLayout L(p.N, p.NP, D, nslots);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.off_bar);
    uint64_t* a_full = bar + 1;
    uint64_t* a_empty = a_full + tc::kAStages;
    uint64_t* t_full = a_empty + tc::kAStages;
    uint64_t* t_empty = t_full + tc::kTmemBufs;
    uint32_t* tptr = reinterpret_cast<uint32_t*>(smem + L.off_tptr);
    unsigned char* opB = smem + L.off_opB;
    unsigned char* opA = smem + L.off_opA;
    // per-slot arrays
    auto slot = [&](int s) -> unsigned char* { return smem + L.off_slot + s * L.slot_stride; };
    auto popA_of = [&](int s) { return reinterpret_cast<double*>(slot(s) + L.s_popA); };
    auto popT_of = [&](int s) { return reinterpret_cast<double*>(slot(s) + L.s_popT); };
    auto box_of = [&](int s) { return reinterpret_cast<double*>(slot(s) + L.s_box); };     // [6] bad box, [7] a1 fixed, +8 lo, +16 hi
    auto fit_of = [&](int s) { return reinterpret_cast<double*>(slot(s) + L.s_fit); };
    auto amp_of = [&](int s) { return reinterpret_cast<float*>(slot(s) + L.s_amp); };
    auto part_of = [&](int s) { return reinterpret_cast<double*>(slot(s) + L.s_part); };
    auto xs_of = [&](int s) { return reinterpret_cast<float*>(slot(s) + L.s_xs); };

    const int tid = threadIdx.x, nthr = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31;
    const int Npad = TcSmemLayout::align_up(p.N, tc::kTile), nT = Npad / tc::kTile;
    // The N samples sit in the middle of the nT tiles (offset a multiple of the 16-column chunk): sample n is column off + n.
    // A short block is then evaluated next to its tile's centre, where the re-expanded polynomial has the smallest terms.
    const int off = ((Npad - p.N) / 2) & ~15;
    const double dt = 1.0 / p.fs;
    uint32_t parity = 0;

    if (tid == 0) {
        mbar_init(bar, 1);
        for (int k = 0; k < tc::kAStages; ++k) { mbar_init(&a_full[k], kTcProducerWarps); mbar_init(&a_empty[k], 1); }
        for (int k = 0; k < tc::kTmemBufs; ++k) { mbar_init(&t_full[k], 1); mbar_init(&t_empty[k], kTcConsumerWarps); }
        fence_mbar_init();
    }
    if (warp == kTcConsumerWarps) tc::tmem_alloc(tptr, tc::kTmemCols);
    if (tid < tc::kTile) {           // the basis operand: the same for every tile, block and generation
        float e[16];
        tc::basis_row(tid - tc::kTile / 2, e);
        tc::write_row(opB, tid, e, tc::kBChunk);
    }
    // rows of candidates beyond NP stay zero (phase 0): their lanes compute sums nobody reads
    for (int i = tid; i < tc::kAStages * tc::kABytes / 16; i += nthr) reinterpret_cast<float4*>(opA)[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    fence_proxy_async();
    tc::fence_before_sync();
    __syncthreads();
    tc::fence_after_sync();
    const uint32_t tmem = *tptr;

    TcConsumer cs;
    cs.t_full = t_full; cs.t_empty = t_empty; cs.it = 0; cs.lane = lane;
    cs.tbase = tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 64);
    TcProducer pr;
    pr.a_full = a_full; pr.a_empty = a_empty; pr.t_full = t_full; pr.t_empty = t_empty; pr.opA = opA; pr.tmem = tmem;
    pr.idesc = tc::make_idesc_tf32(tc::kRowsA, tc::kTile);
    pr.db0 = tc::make_desc(smem_u32(opB), tc::kBChunk, 128);
    pr.db1 = tc::make_desc(smem_u32(opB) + 2 * tc::kBChunk, tc::kBChunk, 128);
    pr.pit = 0;

    auto reported = [&](double v) -> double {       // F_cor - 1/pi of cor = -v for the correlation objective
        if (OBJ == kObjCor) return 1.0 / (atan(-v) + 0.5 * kPi) - 1.0 / kPi;
        return v;
    };
    const int passes = (MODE == kModeFit) ? p.G + 1 : 1;
    const long long item_end = p.count ? min(p.B, p.blk0 + (long long)*p.count) : p.B;
    // This CTA's work items are blk0 + blockIdx.x + k gridDim.x; it takes them `nslots` at a time.
    for (long long item0 = p.blk0 + blockIdx.x; item0 < item_end; item0 += (long long)nslots * gridDim.x) {
        const int na = (nslots == 2 && item0 + gridDim.x < item_end) ? 2 : 1;      // slots in use this round
        long long blk_of[2];
        for (int s = 0; s < na; ++s) {
            const long long item = item0 + (long long)s * gridDim.x;
            blk_of[s] = p.sel ? (long long)p.sel[item] : item;
        }
        // ---- a0: stage the blocks' samples into shared memory, once (PAPER.md:121 data block) ----
        const bool bulk = p.q.bits == 0 && p.use_bulk;
        if (bulk && tid == 0) {
            fence_proxy_async();           // earlier generic-proxy reads of xs are ordered before the async writes
            const uint32_t bytes = (uint32_t)p.N * 4u;
            mbar_arrive_expect_tx(bar, bytes * (uint32_t)na);
            for (int s = 0; s < na; ++s) {
                const float* xg = p.x + blk_of[s] * (long long)p.N;
                for (uint32_t o = 0; o < bytes; o += 32768u)
                    bulk_g2s(reinterpret_cast<unsigned char*>(xs_of(s) + off) + o, reinterpret_cast<const unsigned char*>(xg) + o,
                             min(32768u, bytes - o), bar);
            }
        }
        for (int s = 0; s < na; ++s) {
            const long long blk = blk_of[s];
            float* xs = xs_of(s);
            double* box = box_of(s);
            if (p.q.bits != 0) {
                const unsigned char* xqrow = p.xq + blk * p.row_bytes;
                for (int n = tid; n < p.N; n += nthr) xs[off + n] = unpack_sample(xqrow, n, p.q);
            } else if (!p.use_bulk) {
                const float* xg = p.x + blk * (long long)p.N;
                for (int n = tid; n < p.N; n += nthr) xs[off + n] = __ldg(xg + n);
            }
            for (int n = tid; n < off; n += nthr) xs[n] = 0.0f;
            for (int n = off + p.N + tid; n < Npad; n += nthr) xs[n] = 0.0f;
            if (MODE == kModeFit) {
                if (tid < D) {
                    const double l = p.lo[blk * D + tid], h = p.hi[blk * D + tid];
                    box[8 + tid] = l; box[16 + tid] = h;
                    if (tid == 1) box[7] = (l == 0.0 && h == 0.0) ? 1.0 : 0.0;      // amplitude slope fixed at zero
                }
                if (tid == 32) {      // lo <= hi is the caller's contract; a violation is reported in status bit 4
                    bool bad = false;
                    for (int j = 0; j < D; ++j) bad = bad || !(p.lo[blk * D + j] <= p.hi[blk * D + j]);
                    box[6] = bad ? 1.0 : 0.0;
                }
            } else if (tid == 0) {
                const float* pp = p.pop_in + blk * (long long)p.NP * D + 1;
                bool z = true;
                for (int i = 0; i < p.NP; ++i) z = z && (pp[(size_t)i * D] == 0.0f);
                box[7] = z ? 1.0 : 0.0;
                box[6] = 0.0;
            }
        }
        if (bulk) { mbar_wait(bar, parity); parity ^= 1u; }
        __syncthreads();

        if (warp < kTcConsumerWarps) {
            // ================= consumers: pass-major, slot-minor -- the order in which the producers emit the tiles =================
            const int cand = (warp & 3) * 32 + lane, cg = warp >> 2, c0 = cg * 64;
            const float dtf = (float)dt, Ldtf = (float)((double)tc::kTile * dt), tw0 = (float)(p.t0 + (double)(c0 - off) * dt);
            for (int g = 0; g < passes; ++g) {
                for (int s = 0; s < na; ++s) {
                    const float* xs = xs_of(s);
                    const float* amp = amp_of(s);
                    const bool a1z = (OBJ == kObjChi2) && box_of(s)[7] != 0.0;
                    named_sync(bar_amp(s), kTcThreads);
                    const float na0 = amp[2 * cand], na1 = amp[2 * cand + 1];
                    double sum;
                    if (OBJ == kObjCor) sum = tc_consumer_pass<kTcAmpCor>(cs, xs, p.N, nT, c0, off, na0, na1, dtf, Ldtf, tw0);
                    else if (a1z) sum = tc_consumer_pass<kTcAmpConst>(cs, xs, p.N, nT, c0, off, na0, na1, dtf, Ldtf, tw0);
                    else sum = tc_consumer_pass<kTcAmpLinear>(cs, xs, p.N, nT, c0, off, na0, na1, dtf, Ldtf, tw0);
                    part_of(s)[cg * kTcMaxNP + cand] = sum;
                    named_arrive(bar_part(s), kTcThreads);
                }
            }
        } else {
            // ================= producers: thread i = member i of both slots =================
            const int i = tid - kTcConsumerWarps * 32;
            const bool active = i < p.NP;
            // sum of the four column groups' partials of member i, in fixed order; Eq. 5-6: the value minimised is -cor = (-a0) S
            auto combined = [&](int s) -> double {
                const double* part = part_of(s);
                double v = ((part[i] + part[kTcMaxNP + i]) + part[2 * kTcMaxNP + i]) + part[3 * kTcMaxNP + i];
                if (OBJ == kObjCor) v *= (double)amp_of(s)[2 * i];
                return v;
            };
            // hand the candidate to the consumers (amplitude table), then emit the coefficient rows of all its tiles
            auto evaluate = [&](int s, const double* th) {
                float* amp = amp_of(s);
                amp[2 * i] = -(float)th[0];
                amp[2 * i + 1] = -(float)th[1];
                named_arrive(bar_amp(s), kTcThreads);
                tc_produce_pass<D>(pr, p, th, active, i, nT, off, warp, lane);
            };
            auto bidx_of = [&](int s) -> uint32_t { return p.block_index ? p.block_index[blk_of[s]] : (uint32_t)blk_of[s]; };
            // ---- a1: generation 0 of every slot ----
            for (int s = 0; s < na; ++s) {
                double th[D];
#pragma unroll
                for (int j = 0; j < D; ++j) th[j] = 0.0;
                if (active) {
                    if (MODE == kModeFit) {
                        init_member<D>((uint32_t)i, bidx_of(s), p.key0, p.key1, box_of(s) + 8, box_of(s) + 16, th);
#pragma unroll
                        for (int j = 0; j < D; ++j) popA_of(s)[i * D + j] = th[j];
                    } else {
                        const float* pp = p.pop_in + (blk_of[s] * (long long)p.NP + i) * D;
#pragma unroll
                        for (int j = 0; j < D; ++j) th[j] = (double)pp[j];
                    }
                }
                evaluate(s, th);
            }
            // ---- a2..a7: generations.  For slot s: selection of generation g - 1, then the trials of generation g; meanwhile
            //      the consumers are still busy with the other slot's tiles (emitted just before) ----
            for (int g = 1; g <= passes; ++g) {
                for (int s = 0; s < na; ++s) {
                    double* popA = popA_of(s);
                    double* popT = popT_of(s);
                    double* fit = fit_of(s);
                    const double* lo_s = box_of(s) + 8;
                    const double* hi_s = box_of(s) + 16;
                    named_sync(bar_part(s), kTcThreads);               // the slot's sums of generation g - 1 are complete
                    if (active) {
                        const double v = combined(s);
                        if (g == 1) {
                            fit[i] = v;
                            if (MODE == kModeFitness) p.fitness_out[blk_of[s] * (long long)p.NP + i] = (float)reported(v);
                        } else if (v <= fit[i]) {                      // a6: greedy selection, accept on <=
                            fit[i] = v;
#pragma unroll
                            for (int j = 0; j < D; ++j) popA[i * D + j] = popT[i * D + j];
                        }
                    }
                    named_sync(kBarProd, kTcProducerWarps * 32);       // population and objective values visible to every producer
                    if (g == passes) continue;                          // last selection done: results are written below
                    const uint32_t bidx = bidx_of(s);
                    int ibest = 0;
                    if (p.strategy == kLocalToBest1 || p.strategy == kBest1Jitter) {
                        double bv, mx;
                        tc_warp_argmin(fit, p.NP, lane, bv, ibest, mx);
                    }
                    double th[D];
#pragma unroll
                    for (int j = 0; j < D; ++j) th[j] = 0.0;
                    if (active) {
                        const Draws dr = de_draws<D>((uint32_t)i, (uint32_t)g, bidx, (uint32_t)p.NP, p.CR32, p.key0, p.key1);
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
                    // every producer has read the parents before anybody's next selection can overwrite them: the next write to
                    // popA of this slot happens after the next bar_part(s), which all producers pass only after this point
                    evaluate(s, th);
                }
            }
            // ---- a8: best member (lowest index on ties), status, optional final population ----
            if (MODE == kModeFit) {
                for (int s = 0; s < na; ++s) {
                    const long long blk = blk_of[s];
                    const double* popA = popA_of(s);
                    const double* fit = fit_of(s);
                    const double* box = box_of(s);
                    if (warp == kTcConsumerWarps) {
                        double bv, mx;
                        int bi;
                        tc_warp_argmin(fit, p.NP, lane, bv, bi, mx);
                        if (lane == 0) {
                            uint32_t st = 0;
#pragma unroll
                            for (int j = 0; j < D; ++j) {
                                const double v = popA[bi * D + j];
                                p.best[blk * D + j] = v;
                                const double w = box[16 + j] - box[8 + j];
                                if (w > 0.0 && (v - box[8 + j] <= 1e-6 * w || box[16 + j] - v <= 1e-6 * w)) st |= 1u;
                            }
                            const double braw = fit[bi];
                            if (OBJ == kObjCor) {
                                const double fb = reported(bv), fw = reported(mx);
                                if (fw - fb > 1e-3 * fb) st |= 2u;
                                p.best_rss[blk] = (float)reported(braw);
                            } else {
                                if (mx - bv > 1e-3 * bv) st |= 2u;
                                p.best_rss[blk] = (float)braw;
                            }
                            if (!(fabs(braw) <= 3.0e38)) st |= 8u;         // objective of the best member is not finite
                            if (box[6] != 0.0) st |= 16u;                  // the caller's box has lo > hi (or NaN) in some coordinate
                            p.status[blk] = st;
                        }
                    }
                    if (p.final_pop) {
                        float* fp = p.final_pop + blk * (long long)p.NP * D;
                        for (int k = i; k < p.NP * D; k += kTcProducerWarps * 32) fp[k] = (float)popA[k];
                    }
                    if (p.final_fit && active) p.final_fit[blk * (long long)p.NP + i] = (float)reported(fit[i]);
                }
            }
        }
        __syncthreads();   // samples, populations and boxes are reused by the next blocks of this CTA
    }
    tc::fence_before_sync();
    __syncthreads();
    if (warp == kTcConsumerWarps) tc::tmem_dealloc(tmem, tc::kTmemCols);
}

}  // namespace pt
