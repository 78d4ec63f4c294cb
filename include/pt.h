/*
 * pt.h -- C ABI of libpt.so: B200-native (sm_100a) phase tracking by Differential Evolution,
 *         the data-parallel hot path of arxiv 1906.10598 ("The GPU-based Phase Tracking method for
 *         Planetary Radio Science applications").  Citations are PAPER.md line numbers.
 *
 * Parameterisation.  theta = (a0, a1, phi0, f, fdot[, fddot]), D = 5 or 6, and the signal model is
 *     s(t) = (a0 + a1 t) cos(phi0 + 2 pi (f t + fdot t^2/2 + fddot t^3/6)),   t in [-T/2, T/2)
 * which is PAPER.md:128-137 (Eq. 2-3) with c0 = phi0, c1 = 2 pi f, c2 = pi fdot, c3 = (pi/3) fddot,
 * c4 = a0, c5 = a1.  Sample n of a block sits at t_n = t0 + n/fs; t0 = -N/(2 fs) puts sample N/2 at
 * the block centre.
 *
 * Conventions (all entry points).
 *   - Return value: PT_OK (0) or a negative pt_status.  Nothing throws, nothing aborts, nothing prints.
 *     pt_last_error_string() describes the last failure of the calling thread.
 *   - Unless a parameter is marked [host], every array pointer is a DEVICE pointer owned by the caller
 *     (the Python binding allocates them with torch).  Layouts are dense row-major.  Inputs are never
 *     modified.  The device entry points keep no device memory between calls; scratch is passed in by the caller
 *     and sized by the *_workspace_bytes query.  (The *_host entry points keep a stream-ordered memory pool and a
 *     stream per device between calls, so that a repeated call pays no cudaMalloc; pt_host_cache_release() frees them.)
 *   - Device entry points are asynchronous on the given stream and never synchronise the device or the stream.
 *     The *_host entry points are synchronous and own their temporary device memory.
 *   - One process may drive several devices from several host threads: per-device state inside the library is keyed by
 *     the CUDA device current at the call and guarded by a mutex.
 *   - The stream argument is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - There is no CPU fallback: without a CUDA device every compute call returns PT_ERR_CUDA.
 */
#ifndef PT_H_
#define PT_H_

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define PT_API __attribute__((visibility("default")))
#else
#define PT_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    PT_OK = 0,
    PT_ERR_INVALID_ARG = -1, /* null pointer, N odd or < 8, D not 5/6, NP < 4, fs <= 0, F or CR out of range; lo > hi in
                                HOST boxes (*_host entries; device boxes: status bit4 of the block)            */
    PT_ERR_UNSUPPORTED = -2, /* NP or N beyond the compiled limits, workspace too small                               */
    PT_ERR_CUDA = -3         /* a CUDA call failed; see pt_last_error_string()                                        */
} pt_status;

#define PT_MAX_NP 1024      /* population limit of the DE kernel                                  */
#define PT_MAX_N 16777216   /* samples per block: the evaluation loop carries the sample index exactly in fp32 (2^24) */
#define PT_PER_BLOCK_COLS 10 /* columns of pt_doppler_products' per_block output                  */

/*
 * Mutation strategies.  PAPER.md:205: "There are six kind of mutation operations strategies in the DE algorithm
 * [Price et al., 2006].  Among these strategies the third is the best choice for objective function Eq. 4 and the
 * sixth for Eq. 5"; Table 4 sets "strategy 3 6".  The paper does not define them; they are taken as
 * the six strategies of Price, Storn & Lampinen (2006), all with binomial crossover (reading R21).
 * x_r1, x_r2, x_r3: distinct random members != i; x_best: best member of the previous generation; rand: uniform [0,1).
 */
typedef enum {
    PT_STRATEGY_RAND1 = 1,             /* v = x_r1 + F (x_r2 - x_r3)                                              */
    PT_STRATEGY_LOCAL_TO_BEST1 = 2,    /* v = x_i + F (x_best - x_i) + F (x_r2 - x_r3)                            */
    PT_STRATEGY_BEST1_JITTER = 3,      /* v_j = x_best,j + (x_r2,j - x_r3,j) (F + 0.0001 rand_j)                  */
    PT_STRATEGY_RAND1_VEC_DITHER = 4,  /* v = x_r1 + (F + (1 - F) rand_i) (x_r2 - x_r3), one rand per vector      */
    PT_STRATEGY_RAND1_GEN_DITHER = 5,  /* same, one rand per generation                                           */
    PT_STRATEGY_EITHER_OR = 6          /* rand_i < 0.5: as 1; else v = x_r1 + 0.5 (F + 1) (x_r2 + x_r3 - 2 x_r1)  */
} pt_strategy;

/*
 * Objectives.  PT_OBJECTIVE_CHI2: Eq. 4, the residual sum of squares of the model of Eq. 2.
 * PT_OBJECTIVE_COR: Eq. 5, F_cor = 1 / (arctan(cor) + pi/2) with the constant-amplitude model of Eq. 6,
 * s(t) = a0 cos(phi(t)) (a1 is not used), and cor = sum_n x_n s(t_n), the un-normalised correlation sum (the only
 * reading under which F_cor "shall converge to 1/pi"; reading R22).  With a free amplitude
 * this objective diverges: give a0 a zero-width box.  F_cor is strictly decreasing in cor; the
 * kernel maximises the fp32 correlation sum and reports F_cor - 1/pi (fp64 arithmetic, rounded to fp32), the
 * quantity the paper displays ("subtracted a constant of 0.31830988618"): it tends to 0 from above.
 */
typedef enum { PT_OBJECTIVE_CHI2 = 0, PT_OBJECTIVE_COR = 1 } pt_objective_kind;

/* DE control record: the paper's Table 4 plus the population size it never states. */
typedef struct {
    int32_t D;           /* 5: (a0,a1,phi0,f,fdot)   6: (+fddot)                     PAPER.md:213 Dim_XC */
    int32_t NP;          /* population size, 4 <= NP <= PT_MAX_NP                                         */
    int32_t generations; /* itermax; the fixed-count stop rule  */
    double F;            /* mutation scaling factor F_XC, in [0, 2]         */
    double CR;           /* crossover factor CR_XC, in [0, 1]         */
    uint64_t seed;       /* Philox4x32-10 key (low word, high word)                                       */
    double t0;           /* time of sample 0 relative to the block centre [s]; -N/(2 fs) by default       */
    int32_t strategy;    /* pt_strategy, Table 4 "strategy" (0 is read as PT_STRATEGY_RAND1) */
    int32_t objective;   /* pt_objective_kind: chi^2 (Eq. 4) or correlation (Eq. 5-6)  */
} pt_de_config;

/*
 * pt_fitness -- the chi^2 objective with sigma_i = 1 (Eq. 4):
 *     fitness[b][i] = sum_n ( x[b][n] - s(pop[b][i], t_n) )^2 .
 * x        [B][N]      fp32 baseband samples (PAPER.md:121 data block; N even, N >= 8)
 * pop      [B][NP][D]  fp32 ABSOLUTE parameter values (no per-block offset), so that a reference
 *                      implementation can be fed exactly the same numbers
 * fitness  [B][NP]     fp32 out
 * Runs the same per-sample code as the DE kernel: fp32 FMA + one hardware cosine per sample and candidate,
 * phase taken relative to a per-block fp64 reference trajectory.  Blocks larger than shared memory are
 * streamed; then workspace (>= pt_fitness_workspace_bytes) is required, else it may be NULL.
 */
PT_API size_t pt_fitness_workspace_bytes(int64_t B, int32_t N, int32_t NP, int32_t D);
PT_API int32_t pt_fitness(const float* x, int64_t B, int32_t N, double fs, double t0, const float* pop, int32_t NP,
                   int32_t D, float* fitness, void* workspace, size_t workspace_bytes, void* stream);

/*
 * pt_objective -- like pt_fitness for either objective: objective = PT_OBJECTIVE_CHI2 writes Eq. 4,
 * PT_OBJECTIVE_COR writes F_cor - 1/pi of Eq. 5-6 (see pt_objective_kind).  Same arguments otherwise.
 */
PT_API int32_t pt_objective(const float* x, int64_t B, int32_t N, double fs, double t0, const float* pop, int32_t NP,
                     int32_t D, int32_t objective, float* fitness, void* workspace, size_t workspace_bytes,
                     void* stream);

/*
 * pt_fit_blocks -- Differential Evolution fit of every block (PAPER.md:39-43 Fig. 1, :203-224 Table 4):
 * NP members drawn uniformly in the box [lo, hi], then `generations` synchronous
 * generations of mutation by cfg->strategy (default DE/rand/1: v = x_r1 + F (x_r2 - x_r3)), binomial crossover
 * with factor CR, reflect-then-clamp bound handling, evaluation of cfg->objective (default chi^2, Eq. 4) and
 * greedy selection (accept on <=).
 * Random numbers are Philox4x32-10 with counter (slot, candidate, generation, block_index) and key = seed,
 * so every draw is independent of any floating-point decision.
 * x            [B][N]     fp32 samples
 * lo, hi       [B][D]     fp64 parameter box per block (XCmin / XCmax); lo == hi is legal
 * block_index  [B]        u32 Philox counter word of each block, or NULL for 0..B-1
 * best         [B][D]     fp64 out: member with the smallest RSS (lowest index on ties)
 * best_rss     [B]        fp32 out: its RSS (the "RSS" column of the paper's output record);
 *                                   F_cor - 1/pi for PT_OBJECTIVE_COR
 * status       [B]        u32 out: bit0 (1) = best lies within 1e-6 (hi-lo) of a box face;
 *                                  bit1 (2) = population not collapsed (max RSS - min RSS > 1e-3 min RSS; for the
 *                                         correlation objective the same rule on F_cor - 1/pi);
 *                                  bit2 (4) = abandoned by pt_refit_doubtful;
 *                                  bit3 (8) = the best member's objective is not finite (a NaN or Inf sample in the
 *                                         block): the block's outputs are meaningless, the other blocks are unaffected;
 *                                  bit4 (16) = the block's box has lo > hi (or a NaN) in some coordinate.  The device
 *                                         entry points are asynchronous and cannot return PT_ERR_INVALID_ARG for the
 *                                         contents of device arrays; pt_track_host checks its host boxes and does.
 * final_pop    [B][NP][D] fp32 out, optional (NULL): final population rounded to fp32
 * final_fit    [B][NP]    fp32 out, optional (NULL)
 * workspace               >= pt_fit_blocks_workspace_bytes(B, N, cfg) bytes of device scratch (may be NULL if 0)
 */
PT_API size_t pt_fit_blocks_workspace_bytes(int64_t B, int32_t N, const pt_de_config* cfg /*[host]*/);
PT_API int32_t pt_fit_blocks(const float* x, int64_t B, int32_t N, double fs, const double* lo, const double* hi,
                      const uint32_t* block_index, const pt_de_config* cfg /*[host]*/, double* best,
                      float* best_rss, uint32_t* status, float* final_pop, float* final_fit, void* workspace,
                      size_t workspace_bytes, void* stream);

/*
 * Quantised samples.  PAPER.md:104-117 (Table 3): the receiver records 8- or 16-bit samples in its narrow-band modes and
 * 1-, 2-, 4- or 8-bit samples in its wide-band modes; "s_i is the quantized signal value".  The paper gives
 * no packing or level table; this library takes (reading R23): sample n of a block is the bits-wide field n of
 * the block's row, fields packed from the least significant bit of each byte upwards, 16-bit samples little-endian; the
 * field is an unsigned integer (is_signed = 0) or two's complement (is_signed != 0); the sample value is
 *     s = scale * (code + offset),   evaluated in fp64 and rounded once to fp32.
 * (offset-binary 2-bit data with levels -1.5, -0.5, 0.5, 1.5 times a step: is_signed = 0, offset = -1.5, scale = step.)
 */
typedef struct {
    int32_t bits;      /* 1, 2, 4, 8 or 16 */
    int32_t is_signed; /* 0: unsigned field, else two's complement */
    double scale;
    double offset;
} pt_quant;

/*
 * pt_fit_blocks_q -- pt_fit_blocks on quantised samples: every block's row is unpacked to fp32 while it is staged into
 * shared memory (or, for blocks larger than shared memory, into the workspace row), once per block; everything after
 * that is pt_fit_blocks, and the results are bit-identical to pt_fit_blocks on the unpacked samples.
 * xq         [B][row_bytes]  device, packed samples; row_bytes * 8 >= N * bits
 * quant      [host]
 * Workspace: pt_fit_blocks_workspace_bytes(B, N, cfg).
 */
PT_API int32_t pt_fit_blocks_q(const void* xq, const pt_quant* quant /*[host]*/, int64_t row_bytes, int64_t B, int32_t N,
                        double fs, const double* lo, const double* hi, const uint32_t* block_index,
                        const pt_de_config* cfg /*[host]*/, double* best, float* best_rss, uint32_t* status,
                        float* final_pop, float* final_fit, void* workspace, size_t workspace_bytes, void* stream);

/* pt_unpack_samples -- the same unpacking as a stand-alone call (parity / inspection): xq[B][row_bytes] -> x[B][N] fp32,
 * both device pointers. */
PT_API int32_t pt_unpack_samples(const void* xq, const pt_quant* quant /*[host]*/, int64_t row_bytes, int64_t B, int32_t N,
                          float* x, void* stream);

/*
 * pt_acquire -- initial range determination (section 3.1.1 items 1-6): per block, the centre frequency
 * and amplitude from the FFT of "a small piece of data extracted from block center", the frequency rate by "central
 * difference method through three equally spaced frequency values near block center", and the parameter boxes
 *     phi0 in [-pi, pi] (item 1: a full turn), f in f_c -+ max(f_rel |f_c|, f_bins fs/M) (item 2: +-10 %),
 *     fdot in fdot_est -+ fdot_bins (fs/M)/(spacing/fs) (the paper gives no range for c2), fddot in -+ fddot_hw
 *     (item 4: c3 in [-50, 50], i.e. 150/pi), a0 in a_est (1 -+ a_rel) (item 5: +-10 %), a1 in -+ a1_rel a_est/T (item 6).
 * What the paper leaves open (reading R24): piece k = -1, 0, 1 is samples [N/2 + k spacing - M/2, N/2 + k spacing
 * + M/2) of the block, weighted by the periodic Hann window; its frequency is the largest |X_k|^2 over 1 <= k <= M/2 - 1
 * (lowest k on ties) refined by a parabola through the logarithms of the three powers around it; its amplitude is
 * 4 |X_k| / M divided by the Hann main-lobe factor sinc(delta)/(1 - delta^2).
 * x    [B][N]  fp32 samples (device)
 * acq  [host]  M: power of two, 8 <= M <= 8192, M + 2 spacing <= N, spacing >= 1
 * est  [B][8]  fp64 out: a_est, f(-1), f(0), f(+1), fdot_est, peak bins of the three pieces
 * lo, hi [B][D] fp64 out: the boxes, ready for pt_fit_blocks
 * All blocks are independent: one CTA per block, no sequential dependence between blocks.
 */
typedef struct {
    int32_t M;        /* piece length (power of two)                                              */
    int32_t spacing;  /* samples between piece centres                                            */
    double f_rel;     /* 0.1 in the paper                                          */
    double f_bins;    /* alternative half-width in FFT bins (the larger of the two is taken)      */
    double fdot_bins; /* half-width of fdot in frequency bins per spacing                         */
    double a_rel;     /* 0.1 in the paper                                          */
    double a1_rel;    /* 0.2 in the paper                                          */
    double fddot_hw;  /* 150/pi in the paper's units; used when D = 6              */
} pt_acq_config;

PT_API int32_t pt_acquire(const float* x, int64_t B, int32_t N, double fs, int32_t D, const pt_acq_config* acq /*[host]*/,
                   double* est, double* lo, double* hi, void* stream);

/*
 * pt_refit_doubtful -- continuity check and re-search of doubtful blocks (section 3.1.3, Eq. 8: a solution
 * is judged by "the continuity of instantaneous phase and frequency at the bound of two adjacent data block ... within
 * the threshold of noise"; :191-197 run-time ranges extrapolated from a solved block; :252 "the software will
 * automatically adjust parameters range and try to search again.  The data block will be abandoned after three attempts").
 * The paper walks the blocks one by one; here all blocks are fitted first (pt_fit_blocks) and then, per attempt a = 1 ..
 * max_attempts (reading R25):
 *   border j (blocks j, j+1) is bad if |wrapped phase residual| > phi_tol or |frequency residual| > F_tol;
 *   a block is doubtful if every border it has is bad;
 *   a doubtful block b takes ranges from the nearest trusted block n (left on equal distance), k = b - n, with
 *   F(t) = f + fdot t + fddot t^2/2 of block n:  f in mid[F((k-1/2)T), F((k+1/2)T)] -+ g max(half distance, f_floor),
 *   fdot likewise from F'(t) with fdot_floor, a0 in a0^n (1 -+ g a_rel), phi0 in [-pi, pi], a1 and fddot unchanged,
 *   g = grow^(a-1); with no trusted block its own box is widened by grow;
 *   the doubtful blocks (only they) are fitted again with key seed + a * 0x9E3779B97F4A7C15 and replace their solution.
 * Blocks still doubtful after the last attempt get status bit 2 (value 4, "abandoned").
 * lo, hi, best, best_rss, status [B]... are those of the preceding pt_fit_blocks call and are updated in place;
 * attempts [B] int32 device out: re-searches each block took (set to 0 first).
 * workspace: >= pt_refit_doubtful_workspace_bytes(B, N, cfg) device bytes, 16-byte aligned.
 * Asynchronous like every device entry point: the list of doubtful blocks and its length stay on the device (ordered
 * compaction kernel), every attempt is enqueued unconditionally and its kernels do nothing once no block is doubtful.  The
 * re-fit launch therefore has the geometry of B single-CTA blocks; CTAs without a doubtful block exit at once.
 */
typedef struct {
    double phi_tol;       /* rad                                                              */
    double F_tol;         /* Hz                                                               */
    int32_t max_attempts; /* 3 in the paper                                    */
    double grow;          /* enlargement of the ranges per attempt                            */
    double f_floor;       /* Hz: smallest half-width of the extrapolated f range (times g)    */
    double fdot_floor;    /* Hz/s                                                             */
    double a_rel;         /* 0.1 in the paper                                  */
} pt_retry_config;

PT_API size_t pt_refit_doubtful_workspace_bytes(int64_t B, int32_t N, const pt_de_config* cfg /*[host]*/);
PT_API int32_t pt_refit_doubtful(const float* x, int64_t B, int32_t N, double fs, double* lo, double* hi,
                          const uint32_t* block_index, const pt_de_config* cfg /*[host]*/,
                          const pt_retry_config* retry /*[host]*/, double* best, float* best_rss, uint32_t* status,
                          int32_t* attempts, void* workspace, size_t workspace_bytes, void* stream);

/*
 * pt_refit_doubtful_static -- pt_refit_doubtful for callers that cannot allocate device memory (code under CUDA graph capture,
 * serving loops, harnesses that forbid cudaMalloc): same arguments without the workspace, same kernels in the same order on the
 * same stream, identical results.  The scratch of the continuity check (Eq. 8 border residuals [B][10] fp64,
 * running phase, doubtful flags, the ordered list of doubtful blocks and its length) lives in a file-scope device array of
 * PT_STATIC_SCRATCH_BYTES (csrc/pt_noalloc.cu) that every GPU which loads the library holds until the process exits.
 * The call itself allocates nothing (no cudaMalloc / cudaFree, no allocating library routine).
 * Limit: pt_refit_doubtful_workspace_bytes(B, N, cfg) <= PT_STATIC_SCRATCH_BYTES, i.e. about 43 000 blocks that fit in shared
 * memory (96 bytes per block; blocks streamed from global memory need rows of their own and are refused); beyond it the call
 * returns PT_ERR_UNSUPPORTED with a message and launches nothing.
 * All calls on a device share the array and it keeps the last call's contents: the bytes a call uses are cleared first, on the
 * caller's stream.  Calls that overlap on the GPU (different streams with no dependency between them) race on it.
 * pt_static_scratch_bytes() returns the compiled size.
 */
#define PT_STATIC_SCRATCH_BYTES (4 * 1024 * 1024)
PT_API size_t pt_static_scratch_bytes(void);
PT_API int32_t pt_refit_doubtful_static(const float* x, int64_t B, int32_t N, double fs, double* lo, double* hi,
                                 const uint32_t* block_index, const pt_de_config* cfg /*[host]*/,
                                 const pt_retry_config* retry /*[host]*/, double* best, float* best_rss, uint32_t* status,
                                 int32_t* attempts, void* stream);

/*
 * pt_doppler_products -- observables from the fitted parameters, fp64 throughout.  T = N/fs.
 *     phi(t) = phi0 + 2 pi (f t + fdot t^2/2 + fddot t^3/6),  F(t) = dphi/dt  [rad/s]    PAPER.md:228-234 (Eq. 7)
 *     border values at t = -T/2, +T/2, phases reduced to [0, 2 pi)                      PAPER.md:237-246 (Eq. 8)
 *     dphi_block = phi(T/2) - phi(-T/2)                                                 PAPER.md:349 (Eq. 17 summand)
 *     Phi_total = sum of m consecutive dphi_block,  F_int = Phi_total / (m T)           PAPER.md:343-351 (Eq. 16-17)
 *     a_los = los_scale * fdot, los_scale = c/f0 (1-way) or c/(2 M2 f0) (3-way); 0 skips  PAPER.md:376-378 (Eq. 19)
 * best         [B][D]   fp64 fitted parameters (as written by pt_fit_blocks)
 * per_block    [B][10]  fp64 out: f, fdot, a_los, phi(-T/2) mod 2pi, phi(+T/2) mod 2pi, F(-T/2), F(+T/2),
 *                        dphi_block, border_dphi (to block b+1, wrapped to (-pi, pi]), border_dF;
 *                        the two border columns of the last block are NaN
 * total_phase  [B]      fp64 out: inclusive running sum of dphi_block (total-count phase)
 * blocks_per_interval [n_intervals] [host] int32: m_k = Tc_k / T
 * interval_out [n_intervals] [host] array of DEVICE pointers; interval_out[k] is [floor(B/m_k)][2] fp64 out:
 *                        (Phi_total, F_int) of each run of m_k blocks
 */
PT_API int32_t pt_doppler_products(const double* best, int64_t B, int32_t D, double T, double los_scale,
                            const int32_t* blocks_per_interval /*[host]*/, int32_t n_intervals,
                            double* per_block, double* total_phase, double* const* interval_out /*[host]*/,
                            void* stream);

/*
 * pt_track_host -- the whole hot path on HOST buffers: copy x, lo, hi to the device, pt_fit_blocks,
 * pt_doppler_products, copy the results back; synchronous.  Every pointer is a [host] pointer
 * (pinned memory makes the copies asynchronous-capable, pageable memory works).  Outputs that are NULL are skipped.
 * interval_out[k] is a [host] pointer to [floor(B/m_k)][2] fp64.
 */
PT_API int32_t pt_track_host(const float* x, int64_t B, int32_t N, double fs, const double* lo, const double* hi,
                      const pt_de_config* cfg, double los_scale, const int32_t* blocks_per_interval,
                      int32_t n_intervals, double* best, float* best_rss, uint32_t* status, double* per_block,
                      double* total_phase, double* const* interval_out);

/* pt_host_cache_release -- destroys the per-device memory pools and streams the *_host entry points keep between calls
 * (synchronises those streams).  The next *_host call creates them again.  Returns PT_OK or PT_ERR_CUDA. */
PT_API int32_t pt_host_cache_release(void);

/* pt_track_host_q -- pt_track_host on quantised HOST samples xq[B][row_bytes] (see pt_quant): the host-to-device copy
 * moves the packed bytes (bits/32 of the fp32 volume). */
PT_API int32_t pt_track_host_q(const void* xq, const pt_quant* quant, int64_t row_bytes, int64_t B, int32_t N, double fs,
                        const double* lo, const double* hi, const pt_de_config* cfg, double los_scale,
                        const int32_t* blocks_per_interval, int32_t n_intervals, double* best, float* best_rss,
                        uint32_t* status, double* per_block, double* total_phase, double* const* interval_out);

/*
 * pt_track_auto_host -- the paper's whole process flow (section 3.1.4) on HOST buffers, with no
 * caller-supplied ranges: copy x to the device, pt_acquire (initial ranges), pt_fit_blocks, pt_refit_doubtful when
 * `retry` is not NULL (continuity check and re-search), pt_doppler_products, copy the results back; synchronous.
 * Every pointer is a [host] pointer; outputs that are NULL are skipped.  lo, hi [B][D] out: the ranges finally used;
 * attempts [B] int32 out (only with retry).  Results are identical to calling the four device entry points in turn.
 */
PT_API int32_t pt_track_auto_host(const float* x, int64_t B, int32_t N, double fs, const pt_de_config* cfg,
                           const pt_acq_config* acq, const pt_retry_config* retry, double los_scale,
                           const int32_t* blocks_per_interval, int32_t n_intervals, double* lo, double* hi, double* best,
                           float* best_rss, uint32_t* status, int32_t* attempts, double* per_block, double* total_phase,
                           double* const* interval_out);

/*
 * pt_de_draws -- debug/parity entry: the integer random draws the DE kernel uses, for Q queries.
 * query  [Q][3]  u32 device: (block_index, generation >= 1, candidate)
 * out    [Q][5]  i32 device: r1, r2, r3, jrand, crossover mask (bit j set = coordinate j takes the mutant)
 * Runs the same device functions as pt_fit_blocks (Philox4x32-10, index map, CR threshold).
 */
PT_API int32_t pt_de_draws(const uint32_t* query, int64_t Q, int32_t NP, int32_t D, double CR, uint64_t seed,
                    int32_t* out, void* stream);

/*
 * pt_init_population -- debug/parity entry: the generation-0 population of the DE kernel,
 * pop0[B][NP][D] fp64 device = lo + (hi - lo) u, u = (Philox word >> 8) 2^-24.
 */
PT_API int32_t pt_init_population(const double* lo, const double* hi, const uint32_t* block_index, int64_t B, int32_t NP,
                           int32_t D, uint64_t seed, double* pop0, void* stream);

/* Launch geometry the library would use for pt_fit_blocks (for reporting): out[0] = grid, out[1] = threads per CTA,
 * out[2] = dynamic shared memory bytes, out[3] = 1 if the block's samples stay resident in shared memory, 0 if streamed,
 * out[4] = candidates per thread (register blocking), out[5] = CTAs per SM, out[6] = CTAs per data block (size of the
 * thread-block cluster that fits one block together when there are fewer blocks than SMs; 1 = no cluster), out[7] = cluster
 * size of the second launch that fits the last partial wave of blocks (0 = single launch; needs a device to be known).
 * The environment variable PT_CLUSTER = 1..8 overrides the automatic cluster size and disables the tail launch (tests and tuning). */
PT_API int32_t pt_fit_blocks_plan(int64_t B, int32_t N, const pt_de_config* cfg /*[host]*/, int32_t out[8] /*[host]*/);

/* The DE-kernel launches pt_fit_blocks issues for B blocks (for reporting; without a device: the list for a B200, with the
 * tail clusters assumed resident).  Blocks all take the same time, so the
 * library cuts them into segments whose grids are exactly full: whole rounds of SMs x c CTAs, the remainder with fewer, larger CTAs
 * per SM, the last few blocks on clusters.  (Short blocks, NP N <= 2^19 sample-evaluations per generation, keep their remainder as one
 * partly filled round; with NP N <= 2^18 a block runs on a CTA of 128 threads, eight per SM.)  Launch k is described by out[5 k .. 5 k + 4] = first block, number of blocks, grid,
 * threads per CTA, CTAs per data block (cluster size).  Returns the number of launches (at most `max_launches` are written), or a
 * negative pt_status.
 * Evaluation kernels (row a5: Eq. 2-4): pt_run_kernel (thread = candidate, run-local Horner; the automatic choice),
 * pt_block_kernel (lanes own samples, reference-phase array), pt_tc_kernel (phase on the tensor cores; NP <= 128).  The environment
 * variable PT_KERNEL = run | classic | tc forces one of them where it applies (tests and A/B measurements); results agree within
 * the tolerances of the objective (fp32 rounding differs), random streams and trial vectors are identical. */
PT_API int32_t pt_fit_blocks_launches(int64_t B, int32_t N, const pt_de_config* cfg /*[host]*/, int32_t* out /*[host]*/, int32_t max_launches);

PT_API const char* pt_last_error_string(void);
PT_API const char* pt_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PT_H_ */
