/*
 * pt_oracle.c -- plain fp64 CPU oracle of the phase-tracking hot path of arxiv 1906.10598.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may build, load or call it.  It shares no
 * code, header, table or constant generator with the CUDA path under paper_1906_10598_b200/.
 *
 * What it computes (citations are PAPER.md line numbers; "SURVEY 8(c)" is /root/repo/SURVEY.md):
 *   - the signal model  s(t) = (c4 + c5 t) cos(c0 + c1 t + c2 t^2 + c3 t^3)          PAPER.md:128-137 (Eq. 2-3)
 *     in the Hz-based parameterisation theta = (a0, a1, phi0, f, fdot[, fddot]):
 *     s(t) = (a0 + a1 t) cos(phi0 + 2 pi (f t + fdot t^2/2 + fddot t^3/6))           SURVEY 8, mapping c0=phi0,
 *     c1 = 2 pi f, c2 = pi fdot, c3 = (pi/3) fddot, c4 = a0, c5 = a1
 *   - the chi^2 objective with sigma_i = 1,  F = sum_i [s_i - s(c, t_i)]^2           PAPER.md:143-146 (Eq. 4)
 *   - Differential Evolution (random initial population in the parameter box, mutation with a
 *     weighting factor, crossover, selection, fixed iteration count)
 *     as DE/rand/1/bin, step by step as SURVEY 8(c) items 1-6 state it; the other five mutation
 *     strategies of Table 4's "strategy" item as DESIGN.md reading R21 takes them
 *   - the correlation objective F_cor = 1 / (arctan(cor(s_i, s(c_k, t_i))) + pi/2) with the
 *     constant-amplitude model s(t) = A cos(phi(t))                                  PAPER.md:148-155 (Eq. 5-6)
 *   - the Doppler products: phase / frequency at block borders, continuity residuals,
 *     total-count phase, integration Doppler, line-of-sight acceleration             PAPER.md:228-246 (Eq. 7-8),
 *                                                                                    :343-352 (Eq. 16-17), :376-379 (Eq. 19)
 *
 * Everything is fp64, evaluated literally (no Horner, no blocking, no reordering); random
 * numbers and index logic are exact integer arithmetic (Philox4x32-10).
 *
 * Pins (tests/test_oracle_*.py): Philox known answers; exhaustive index-draw checks; closed-form
 * fitness values; brute-force grid; Levenberg-Marquardt agreement; Appendix A of the paper;
 * for the mutation strategies the invariants of their definitions on every trial vector and the
 * Levenberg-Marquardt optimum (the paper prints no values: it does not define them, reading R21);
 * for Eq. 5 the limit the paper prints (0.31830988618), closed forms on whole cycles and the
 * least-squares phase; for the sample unpacking hand-decoded bytes and numpy's integer views.
 * Parity unpinned, by design: fdot / fddot / a1 where the data cannot observe them.
 *
 * OpenMP is used only to spread independent blocks (or independent candidates of one
 * generation) over the host cores; it changes no arithmetic and no summation order.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC -o libpt_oracle.so pt_oracle.c -lm
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define PTO_PI 3.14159265358979323846264338327950288

typedef struct {
    int32_t D;           /* 5 or 6                                  PAPER.md:213 (Dim_XC) */
    int32_t NP;          /* population size (never stated by the paper)       */
    int32_t generations; /* itermax, fixed-count stop   */
    double F;            /* mutation scaling factor F_XC         */
    double CR;           /* crossover factor CR_XC         */
    uint64_t seed;       /* Philox key                                                   */
    double t0;           /* time of sample 0 relative to the block centre */
    int32_t strategy;    /* 1..6, Table 4 "strategy"   */
    int32_t objective;   /* 0: chi^2 (Eq. 4)   1: correlation (Eq. 5-6) */
} pto_de_config;

int pto_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), SURVEY 8(c) item 3.
 * One round: (hi0,lo0) = M0*c0, (hi1,lo1) = M1*c2; c' = (hi1^c1^k0, lo1, hi0^c3^k1, lo0).
 * The key is bumped by (W0, W1) between rounds; ten rounds in all.
 * ------------------------------------------------------------------------------------------- */
void pto_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* counter = (slot, i, g, b); key = (seed low word, seed high word).  SURVEY 8(c) item 3. */
static void draw_words(uint64_t seed, uint32_t slot, uint32_t i, uint32_t g, uint32_t b, uint32_t w[4]) {
    uint32_t ctr[4] = {slot, i, g, b};
    uint32_t key[2] = {(uint32_t)(seed & 0xFFFFFFFFu), (uint32_t)(seed >> 32)};
    pto_philox4x32_10(ctr, key, w);
}

static uint32_t mulhi32(uint32_t w, uint32_t n) { return (uint32_t)(((uint64_t)w * (uint64_t)n) >> 32); }

/* CR32 = min(2^32 - 1, floor(CR * 2^32)), computed once in fp64 and used as an integer. */
uint32_t pto_cr32(double CR) {
    double v = floor(CR * 4294967296.0);
    if (v >= 4294967295.0) return 0xFFFFFFFFu;
    if (v <= 0.0) return 0u;
    return (uint32_t)v;
}

/* Index logic of one candidate from the four words of slot 0:
 * a = mulhi(wa, NP-1), b' = mulhi(wb, NP-2), c = mulhi(wc, NP-3), jrand = mulhi(wj, D);
 * r1 = a skipping i; r2 = b' skipping {i, r1} in ascending order; r3 = c skipping {i, r1, r2} in
 * ascending order.  Uniform over ordered triples of distinct indices different from i.
 * out = {r1, r2, r3, jrand}. */
void pto_indices_from_words(const uint32_t w[4], uint32_t i, int32_t NP, int32_t D, int32_t out[4]) {
    uint32_t r1 = mulhi32(w[0], (uint32_t)(NP - 1));
    uint32_t r2 = mulhi32(w[1], (uint32_t)(NP - 2));
    uint32_t r3 = mulhi32(w[2], (uint32_t)(NP - 3));
    uint32_t jrand = mulhi32(w[3], (uint32_t)D);
    if (r1 >= i) r1 += 1;
    {
        uint32_t e0 = i < r1 ? i : r1, e1 = i < r1 ? r1 : i;
        if (r2 >= e0) r2 += 1;
        if (r2 >= e1) r2 += 1;
    }
    {
        uint32_t e[3] = {i, r1, r2};
        for (int a = 0; a < 3; ++a)
            for (int c = a + 1; c < 3; ++c)
                if (e[c] < e[a]) { uint32_t tmp = e[a]; e[a] = e[c]; e[c] = tmp; }
        for (int a = 0; a < 3; ++a)
            if (r3 >= e[a]) r3 += 1;
    }
    out[0] = (int32_t)r1; out[1] = (int32_t)r2; out[2] = (int32_t)r3; out[3] = (int32_t)jrand;
}

/* The integer draws of generation g >= 1 for candidate i of block b:
 * slot 0 -> indices, slot 1 -> crossover words of coordinates 0..3, slot 2 -> coordinates 4..7.
 * out = {r1, r2, r3, jrand, mask}, mask bit j set iff coordinate j takes the mutant, i.e.
 * word_j < CR32 or j == jrand. */
void pto_de_draws(uint64_t seed, uint32_t b, uint32_t g, uint32_t i, int32_t NP, int32_t D, uint32_t CR32,
                  int32_t out[5]) {
    uint32_t w[4], x1[4], x2[4];
    int32_t idx[4];
    draw_words(seed, 0u, i, g, b, w);
    pto_indices_from_words(w, i, NP, D, idx);
    draw_words(seed, 1u, i, g, b, x1);
    draw_words(seed, 2u, i, g, b, x2);
    uint32_t mask = 0;
    for (int j = 0; j < D; ++j) {
        uint32_t word = j < 4 ? x1[j] : x2[j - 4];
        if (word < CR32 || j == idx[3]) mask |= (1u << j);
    }
    out[0] = idx[0]; out[1] = idx[1]; out[2] = idx[2]; out[3] = idx[3]; out[4] = (int32_t)mask;
}

/* The D uniform numbers u_j in [0,1) of the initial population (g = 0): u_j = (w_j >> 8) * 2^-24. */
void pto_init_uniforms(uint64_t seed, uint32_t b, uint32_t i, int32_t D, double* u) {
    uint32_t wa[4], wb[4];
    draw_words(seed, 0u, i, 0u, b, wa);
    draw_words(seed, 1u, i, 0u, b, wb);
    for (int j = 0; j < D; ++j) {
        uint32_t word = j < 4 ? wa[j] : wb[j - 4];
        u[j] = (double)(word >> 8) * (1.0 / 16777216.0);
    }
}

/* ---------------------------------------------------------------------------------------------
 * Model and objective.  PAPER.md:128-130 (Eq. 2), :143-146 (Eq. 4, sigma_i = 1).
 * ------------------------------------------------------------------------------------------- */
double pto_phase(const double* th, int32_t D, double t) {
    double fddot = (D >= 6) ? th[5] : 0.0;
    return th[2] + 2.0 * PTO_PI * (th[3] * t + th[4] * t * t / 2.0 + fddot * t * t * t / 6.0);
}

double pto_model(const double* th, int32_t D, double t) {
    return (th[0] + th[1] * t) * cos(pto_phase(th, D, t));
}

/* RSS of one parameter vector over one block; t_n = t0 + n/fs. */
double pto_rss(const float* x, int32_t N, double fs, double t0, const double* th, int32_t D) {
    double sum = 0.0;
    for (int32_t n = 0; n < N; ++n) {
        double t = t0 + (double)n / fs;
        double r = (double)x[n] - pto_model(th, D, t);
        sum += r * r;
    }
    return sum;
}

/* Fitness of given populations: pop[B][NP][D] are fp32 values promoted to fp64 (so that the
 * GPU is fed exactly the same numbers), fitness[B][NP] in fp64. */
void pto_fitness(const float* x, int64_t B, int32_t N, double fs, double t0, const float* pop, int32_t NP,
                 int32_t D, double* fitness) {
    int64_t total = B * (int64_t)NP;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < total; ++k) {
        int64_t b = k / NP;
        double th[6] = {0, 0, 0, 0, 0, 0};
        for (int j = 0; j < D; ++j) th[j] = (double)pop[k * D + j];
        fitness[k] = pto_rss(x + b * (int64_t)N, N, fs, t0, th, D);
    }
}

/* ---------------------------------------------------------------------------------------------
 * Correlation objective.  PAPER.md:148-155 (Eq. 5-6):
 *     F_cor(c_k) = 1 / ( arctan[ cor(s_i, s(c_k, t_i)) ] + pi/2 ),   s(t) = A cos(c0 + c1 t + c2 t^2 + c3 t^3).
 * Reading R22: cor is the plain (un-normalised) correlation sum  cor = sum_i s_i s(c_k, t_i);
 * only then does F_cor "converge to 1/pi ~ 0.318" -- a normalised coefficient <= 1 would stop
 * at 1/(pi/4 + pi/2) = 0.424.  A = th[0] (a0, "the average amplitude of signal"); th[1] (a1) is not used.
 * ------------------------------------------------------------------------------------------- */
double pto_cor(const float* x, int32_t N, double fs, double t0, const double* th, int32_t D) {
    double sum = 0.0;
    for (int32_t n = 0; n < N; ++n) {
        double t = t0 + (double)n / fs;
        double s = th[0] * cos(pto_phase(th, D, t));     /* Eq. 6 */
        sum += (double)x[n] * s;
    }
    return sum;
}

double pto_fcor_of_cor(double cor) { return 1.0 / (atan(cor) + PTO_PI / 2.0); }   /* Eq. 5 */

double pto_fcor(const float* x, int32_t N, double fs, double t0, const double* th, int32_t D) {
    return pto_fcor_of_cor(pto_cor(x, N, fs, t0, th, D));
}

/* objective 0: Eq. 4, objective 1: Eq. 5 */
double pto_objective(const float* x, int32_t N, double fs, double t0, const double* th, int32_t D, int32_t objective) {
    return objective == 1 ? pto_fcor(x, N, fs, t0, th, D) : pto_rss(x, N, fs, t0, th, D);
}

/* Objective of given populations, like pto_fitness. */
void pto_fitness_obj(const float* x, int64_t B, int32_t N, double fs, double t0, const float* pop, int32_t NP,
                     int32_t D, int32_t objective, double* fitness) {
    int64_t total = B * (int64_t)NP;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < total; ++k) {
        int64_t b = k / NP;
        double th[6] = {0, 0, 0, 0, 0, 0};
        for (int j = 0; j < D; ++j) th[j] = (double)pop[k * D + j];
        fitness[k] = pto_objective(x + b * (int64_t)N, N, fs, t0, th, D, objective);
    }
}

/* ---------------------------------------------------------------------------------------------
 * Mutation strategies.  PAPER.md:205: "There are six kind of mutation operations strategies in the DE
 * algorithm [Price et al., 2006]. Among these strategies the third is the best choice for objective
 * function Eq. 4 and the sixth for Eq. 5"; Table 4 "strategy  3 6".  The paper never
 * defines them.  Reading R21: the six strategies of Price, Storn & Lampinen (2006), whose
 * control-parameter names Table 4 mirrors, all with binomial crossover:
 *   1  DE/rand/1                        v = x_r1 + F (x_r2 - x_r3)
 *   2  DE/local-to-best/1               v = x_i + F (x_best - x_i) + F (x_r2 - x_r3)
 *   3  DE/best/1 with jitter            v_j = x_best,j + (x_r2,j - x_r3,j) (F + 0.0001 rand_j)
 *   4  DE/rand/1, per-vector dither     v = x_r1 + (F + (1 - F) rand_i) (x_r2 - x_r3)
 *   5  DE/rand/1, per-generation dither v = x_r1 + (F + (1 - F) rand_g) (x_r2 - x_r3)
 *   6  DE/rand/1 either-or              v = x_r1 + F (x_r2 - x_r3)               if rand_i < 0.5
 *                                       v = x_r1 + K (x_r2 + x_r3 - 2 x_r1), K = 0.5 (F + 1)   otherwise
 * x_best = the member with the smallest objective in the population the trials are built from (lowest index
 * on ties).  Uniform numbers are (word >> 8) 2^-24 of Philox counters (slot, i, g, b): jitter rand_j = slot 3
 * words 0..3 (j = 0..3) and slot 4 words 0..3 (j = 4..7); rand_i = slot 3 word 0; rand_g = slot 3 word 0 of
 * candidate index 0xFFFFFFFF.  Indices r1, r2, r3, jrand and the crossover mask are those of SURVEY 8(c) item 3
 * for every strategy.
 * ------------------------------------------------------------------------------------------- */
static double unit_uniform(uint32_t word) { return (double)(word >> 8) * (1.0 / 16777216.0); }

/* the D + 2 auxiliary uniforms of candidate i in generation g: u[0..D-1] jitter, u[8] per-vector, u[9] per-generation */
void pto_aux_uniforms(uint64_t seed, uint32_t b, uint32_t g, uint32_t i, double u[10]) {
    uint32_t w3[4], w4[4], wg[4];
    draw_words(seed, 3u, i, g, b, w3);
    draw_words(seed, 4u, i, g, b, w4);
    draw_words(seed, 3u, 0xFFFFFFFFu, g, b, wg);
    for (int j = 0; j < 4; ++j) { u[j] = unit_uniform(w3[j]); u[4 + j] = unit_uniform(w4[j]); }
    u[8] = unit_uniform(w3[0]);
    u[9] = unit_uniform(wg[0]);
}

/* Trial vector of candidate i in generation g >= 1 of block b, built from the population P[NP][D] of generation
 * g-1 whose best member is ibest: mutation by cfg->strategy, binomial crossover, reflect-then-clamp bounds. */
void pto_de_trial(const pto_de_config* cfg, uint32_t b, uint32_t g, uint32_t i, const double* P, int32_t ibest,
                  const double* lo, const double* hi, double* trial) {
    const int32_t D = cfg->D, NP = cfg->NP;
    const double F = cfg->F;
    int32_t d[5];
    double u[10];
    pto_de_draws(cfg->seed, b, g, i, NP, D, pto_cr32(cfg->CR), d);
    pto_aux_uniforms(cfg->seed, b, g, i, u);
    const double* xi = P + (int64_t)i * D;
    const double* x1 = P + (int64_t)d[0] * D;
    const double* x2 = P + (int64_t)d[1] * D;
    const double* x3 = P + (int64_t)d[2] * D;
    const double* xb = P + (int64_t)ibest * D;
    for (int j = 0; j < D; ++j) {
        double v;
        if (!((d[4] >> j) & 1)) { trial[j] = xi[j]; continue; }       /* crossover keeps the parent */
        switch (cfg->strategy) {
            case 2: v = (xi[j] + F * (xb[j] - xi[j])) + F * (x2[j] - x3[j]); break;
            case 3: v = xb[j] + (x2[j] - x3[j]) * (F + 0.0001 * u[j]); break;
            case 4: v = x1[j] + (F + (1.0 - F) * u[8]) * (x2[j] - x3[j]); break;
            case 5: v = x1[j] + (F + (1.0 - F) * u[9]) * (x2[j] - x3[j]); break;
            case 6:
                if (u[8] < 0.5) v = x1[j] + F * (x2[j] - x3[j]);
                else v = x1[j] + (0.5 * (F + 1.0)) * ((x2[j] + x3[j]) - 2.0 * x1[j]);
                break;
            default: v = x1[j] + F * (x2[j] - x3[j]); break;         /* 1: rand/1 */
        }
        /* bound handling: reflect once, then clamp */
        if (v < lo[j]) v = 2.0 * lo[j] - v;
        else if (v > hi[j]) v = 2.0 * hi[j] - v;
        if (v < lo[j]) v = lo[j];
        if (v > hi[j]) v = hi[j];
        trial[j] = v;
    }
}

static int32_t argmin_lowest(const double* fit, int32_t NP) {
    int32_t ib = 0;
    for (int32_t i = 1; i < NP; ++i) if (fit[i] < fit[ib]) ib = i;
    return ib;
}

/* ---------------------------------------------------------------------------------------------
 * DE on one block.  SURVEY 8(c) items 3-6; strategy and objective as cfg says.
 * Workspace: pop, trial [NP][D], fit, tfit [NP].  par != 0: spread the NP evaluations of one
 * generation over the host cores (independent; the arithmetic of each is unchanged).
 * ------------------------------------------------------------------------------------------- */
static void evaluate_all(const float* x, int32_t N, double fs, double t0, const double* P, int32_t NP, int32_t D,
                         int32_t objective, double* out, int par) {
    if (par) {
#pragma omp parallel for schedule(static)
        for (int32_t i = 0; i < NP; ++i) out[i] = pto_objective(x, N, fs, t0, P + (int64_t)i * D, D, objective);
    } else {
        for (int32_t i = 0; i < NP; ++i) out[i] = pto_objective(x, N, fs, t0, P + (int64_t)i * D, D, objective);
    }
}

static void fit_one_block(const float* x, uint32_t b, int32_t N, double fs, const double* lo, const double* hi,
                          const pto_de_config* cfg, double* best, double* best_rss, uint32_t* status,
                          double* final_pop, double* final_fit, double* trace, int par) {
    const int32_t D = cfg->D, NP = cfg->NP, G = cfg->generations;
    double* pop = (double*)malloc(sizeof(double) * (size_t)NP * D);
    double* trial = (double*)malloc(sizeof(double) * (size_t)NP * D);
    double* fit = (double*)malloc(sizeof(double) * (size_t)NP);
    double* tfit = (double*)malloc(sizeof(double) * (size_t)NP);

    /* g = 0: uniform in the box, then the fitness of every member */
    for (int32_t i = 0; i < NP; ++i) {
        double u[8];
        pto_init_uniforms(cfg->seed, b, (uint32_t)i, D, u);
        for (int j = 0; j < D; ++j) pop[(int64_t)i * D + j] = lo[j] + (hi[j] - lo[j]) * u[j];
    }
    evaluate_all(x, N, fs, cfg->t0, pop, NP, D, cfg->objective, fit, par);
    if (trace) {
        double m = fit[0];
        for (int32_t i = 1; i < NP; ++i) if (fit[i] < m) m = fit[i];
        trace[0] = m;
    }

    for (int32_t g = 1; g <= G; ++g) {
        /* all trials of generation g are built from the population of generation g-1 (and its best member) */
        const int32_t ibest = argmin_lowest(fit, NP);
        for (int32_t i = 0; i < NP; ++i)
            pto_de_trial(cfg, b, (uint32_t)g, (uint32_t)i, pop, ibest, lo, hi, trial + (int64_t)i * D);
        evaluate_all(x, N, fs, cfg->t0, trial, NP, D, cfg->objective, tfit, par);
        /* selection: replace if F_obj(u) <= F_obj(x_i) */
        for (int32_t i = 0; i < NP; ++i) {
            if (tfit[i] <= fit[i]) {
                fit[i] = tfit[i];
                memcpy(pop + (int64_t)i * D, trial + (int64_t)i * D, sizeof(double) * D);
            }
        }
        if (trace) {
            double m = fit[0];
            for (int32_t i = 1; i < NP; ++i) if (fit[i] < m) m = fit[i];
            trace[g] = m;
        }
    }

    /* result: argmin, lowest index on ties; status bits */
    int32_t ib = 0;
    double fmin = fit[0], fmax = fit[0];
    for (int32_t i = 1; i < NP; ++i) {
        if (fit[i] < fmin) { fmin = fit[i]; ib = i; }
        if (fit[i] > fmax) fmax = fit[i];
    }
    uint32_t st = 0;
    for (int j = 0; j < D; ++j) {
        double v = pop[(int64_t)ib * D + j];
        best[j] = v;
        double w = hi[j] - lo[j];
        if (w > 0.0 && (v - lo[j] <= 1e-6 * w || hi[j] - v <= 1e-6 * w)) st |= 1u;
    }
    /* DESIGN.md reading R7: 1e-3, not SURVEY's 1e-6; for Eq. 5 the spread is taken on F_cor - 1/pi, the quantity
       the paper displays, which is what tends to zero there */
    if (cfg->objective == 1) {
        if (fmax - fmin > 1e-3 * (fmin - 1.0 / PTO_PI)) st |= 2u;
    } else if (fmax - fmin > 1e-3 * fmin) st |= 2u;
    *best_rss = fmin;
    *status = st;
    if (final_pop) memcpy(final_pop, pop, sizeof(double) * (size_t)NP * D);
    if (final_fit) memcpy(final_fit, fit, sizeof(double) * (size_t)NP);
    free(pop); free(trial); free(fit); free(tfit);
}

/* DE fit of blocks.  x[B][N] fp32; lo, hi [B][D]; outputs best[B][D], best_rss[B], status[B];
 * optional final_pop[B][NP][D], final_fit[B][NP], trace[B][G+1] (best RSS after each generation).
 * block_index[B] (may be NULL = 0..B-1) is the Philox counter word of each block, so a subset of
 * a larger run can be fitted with the draws of the full run. */
int32_t pto_fit_blocks(const float* x, int64_t B, int32_t N, double fs, const double* lo, const double* hi,
                       const pto_de_config* cfg, const uint32_t* block_index, double* best, double* best_rss,
                       uint32_t* status, double* final_pop, double* final_fit, double* trace) {
    if (!x || !lo || !hi || !cfg || !best || !best_rss || !status) return -1;
    if (cfg->NP < 4 || (cfg->D != 5 && cfg->D != 6) || cfg->generations < 0 || N < 1 || fs <= 0.0) return -1;
    if (cfg->strategy < 1 || cfg->strategy > 6 || cfg->objective < 0 || cfg->objective > 1) return -1;
    const int32_t D = cfg->D, NP = cfg->NP, G = cfg->generations;
    int nthreads = pto_num_threads();
    if (B >= nthreads) {
#pragma omp parallel for schedule(dynamic, 1)
        for (int64_t b = 0; b < B; ++b) {
            uint32_t bi = block_index ? block_index[b] : (uint32_t)b;
            fit_one_block(x + b * (int64_t)N, bi, N, fs, lo + b * D, hi + b * D, cfg, best + b * D, best_rss + b,
                          status + b, final_pop ? final_pop + b * (int64_t)NP * D : NULL,
                          final_fit ? final_fit + b * (int64_t)NP : NULL, trace ? trace + b * (int64_t)(G + 1) : NULL,
                          0);
        }
    } else {
        for (int64_t b = 0; b < B; ++b) {
            uint32_t bi = block_index ? block_index[b] : (uint32_t)b;
            fit_one_block(x + b * (int64_t)N, bi, N, fs, lo + b * D, hi + b * D, cfg, best + b * D, best_rss + b,
                          status + b, final_pop ? final_pop + b * (int64_t)NP * D : NULL,
                          final_fit ? final_fit + b * (int64_t)NP : NULL, trace ? trace + b * (int64_t)(G + 1) : NULL,
                          1);
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Quantised samples.  PAPER.md:104-117 (Table 3): the receiver records 8- or 16-bit (narrow band) and 1-, 2-, 4-
 * or 8-bit (wide band) samples; "s_i is the quantized signal value".  The paper gives no packing or
 * level table.  Reading R23: sample n of a block is the bits-wide field n of the block's row, fields
 * packed from the least significant bit of each byte upwards, 16-bit samples little-endian; the field is read as
 * an unsigned integer (is_signed = 0) or as two's complement (is_signed = 1); the sample value is
 *     s_i = scale * (code + offset)
 * evaluated in fp64 and rounded once to fp32 (the input type of every other function here).
 * xq[B][row_bytes] -> x[B][N].  Returns -1 on invalid arguments.
 * ------------------------------------------------------------------------------------------- */
int32_t pto_unpack_samples(const uint8_t* xq, int64_t row_bytes, int64_t B, int32_t N, int32_t bits, int32_t is_signed,
                           double scale, double offset, float* x) {
    if (!xq || !x || B < 1 || N < 1) return -1;
    if (bits != 1 && bits != 2 && bits != 4 && bits != 8 && bits != 16) return -1;
    if (row_bytes * 8 < (int64_t)N * bits) return -1;
    for (int64_t b = 0; b < B; ++b) {
        const uint8_t* row = xq + b * row_bytes;
        for (int32_t n = 0; n < N; ++n) {
            uint32_t field;
            if (bits == 16) {
                field = (uint32_t)row[2 * (int64_t)n] | ((uint32_t)row[2 * (int64_t)n + 1] << 8);
            } else {
                int64_t bit = (int64_t)n * bits;
                field = ((uint32_t)row[bit / 8] >> (bit % 8)) & ((1u << bits) - 1u);
            }
            int32_t code = (int32_t)field;
            if (is_signed && (field >> (bits - 1)) & 1u) code = (int32_t)field - (int32_t)(1u << bits);
            x[b * (int64_t)N + n] = (float)(scale * ((double)code + offset));
        }
    }
    return 0;
}

/* ---------------------------------------------------------------------------------------------
 * Doppler products.  SURVEY 8(c) item 7.
 *   phi(t) = phi0 + 2 pi (f t + fdot t^2/2 + fddot t^3/6)                  PAPER.md:230 (Eq. 7)
 *   F(t)   = dphi/dt = 2 pi (f + fdot t + fddot t^2/2)   [rad/s]           PAPER.md:232-234 (Eq. 7)
 *   border values at t = +-T/2, phases mod 2 pi in [0, 2 pi)                PAPER.md:239-245 (Eq. 8), Appendix A
 *   dphi_b = phi_b(T/2) - phi_b(-T/2)                                      PAPER.md:349 (Eq. 17 summand)
 *   Phi_total = sum of m consecutive dphi_b, F_int = Phi_total / (m T)     PAPER.md:343-351 (Eq. 16-17)
 *   a_los = los_scale * fdot, los_scale = c/f0 (1-way) or c/(2 M2 f0)      PAPER.md:376-378 (Eq. 19)
 * per_block[B][10] = f, fdot, a_los, phi(-T/2) mod 2pi, phi(+T/2) mod 2pi, F(-T/2), F(+T/2),
 *                    dphi_block, border_dphi (to block b+1, wrapped to (-pi, pi]), border_dF;
 *                    the two border entries of the last block are NaN (it has no right neighbour).
 * total_phase[B] = inclusive running sum of dphi_block.
 * interval_out[k][j][2] = (Phi_total, F_int) of the j-th run of blocks_per_interval[k] blocks.
 * ------------------------------------------------------------------------------------------- */
static double mod_2pi(double v) {
    double r = fmod(v, 2.0 * PTO_PI);
    if (r < 0.0) r += 2.0 * PTO_PI;
    if (r >= 2.0 * PTO_PI) r -= 2.0 * PTO_PI;
    return r;
}

static double wrap_pi(double v) { /* to (-pi, pi] */
    double r = fmod(v, 2.0 * PTO_PI);
    if (r <= -PTO_PI) r += 2.0 * PTO_PI;
    if (r > PTO_PI) r -= 2.0 * PTO_PI;
    return r;
}

static double freq_rad(const double* th, int32_t D, double t) {
    double fddot = (D >= 6) ? th[5] : 0.0;
    return 2.0 * PTO_PI * (th[3] + th[4] * t + fddot * t * t / 2.0);
}

int32_t pto_doppler_products(const double* best, int64_t B, int32_t D, double T, double los_scale,
                             const int32_t* blocks_per_interval, int32_t n_intervals, double* per_block,
                             double* total_phase, double** interval_out) {
    if (!best || !per_block || !total_phase || B < 1 || (D != 5 && D != 6) || T <= 0.0) return -1;
    double run = 0.0;
    for (int64_t b = 0; b < B; ++b) {
        const double* th = best + b * D;
        double* o = per_block + b * 10;
        double pl = pto_phase(th, D, -T / 2.0), pr = pto_phase(th, D, T / 2.0);
        o[0] = th[3];
        o[1] = th[4];
        o[2] = los_scale * th[4];
        o[3] = mod_2pi(pl);
        o[4] = mod_2pi(pr);
        o[5] = freq_rad(th, D, -T / 2.0);
        o[6] = freq_rad(th, D, T / 2.0);
        o[7] = pr - pl;
        if (b + 1 < B) {
            const double* nx = best + (b + 1) * D;
            o[8] = wrap_pi(pto_phase(nx, D, -T / 2.0) - pr);
            o[9] = freq_rad(nx, D, -T / 2.0) - o[6];
        } else {
            o[8] = NAN;
            o[9] = NAN;
        }
        run += o[7];
        total_phase[b] = run;
    }
    for (int32_t k = 0; k < n_intervals; ++k) {
        int32_t m = blocks_per_interval[k];
        if (m < 1) return -1;
        int64_t cnt = B / m;
        for (int64_t j = 0; j < cnt; ++j) {
            double s = 0.0;
            for (int32_t q = 0; q < m; ++q) s += per_block[(j * m + q) * 10 + 7];
            interval_out[k][2 * j + 0] = s;
            interval_out[k][2 * j + 1] = s / ((double)m * T);
        }
    }
    return 0;
}
