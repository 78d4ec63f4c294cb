// pt_device.cuh -- device helpers of libpt.so (sm_100a): Philox4x32-10, the DE index map, fp64 helpers that
// round exactly as written (no FMA contraction), mbarrier / bulk-copy wrappers.
// Citations: PAPER.md line numbers; "SURVEY 8(c)" = /root/repo/SURVEY.md section 8(c).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace pt {

constexpr double kPi = 3.14159265358979323846264338327950288;
constexpr double kTwoPi = 6.28318530717958647692528676655900577;

// ---------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon et al., SC'11).  Counter-based: every draw of the DE kernel is a pure function of
// (slot, candidate, generation, block index, seed), independent of any floating-point decision.
// ---------------------------------------------------------------------------------------------------
struct U4 {
    uint32_t x, y, z, w;
};

__device__ __forceinline__ U4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                            uint32_t k1) {
    constexpr uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(M0, c0), lo0 = M0 * c0;
        const uint32_t hi1 = __umulhi(M1, c2), lo1 = M1 * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0;
        const uint32_t n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += W0; k1 += W1;
    }
    return U4{c0, c1, c2, c3};
}

// counter = (slot, candidate i, generation g, block index b); key = (seed low, seed high).
__device__ __forceinline__ U4 draw_words(uint32_t slot, uint32_t i, uint32_t g, uint32_t b, uint32_t k0, uint32_t k1) {
    return philox4x32_10(slot, i, g, b, k0, k1);
}

struct Draws {
    int r1, r2, r3, jrand;
    uint32_t mask;  // bit j set: coordinate j takes the mutant
};

// DE/rand/1/bin integer draws of candidate i in generation g >= 1: three distinct
// indices != i by the skip construction (uniform over ordered triples), jrand, and the crossover mask
// word_j < CR32 || j == jrand with CR32 = min(2^32-1, floor(CR 2^32)).
template <int D>
__device__ __forceinline__ Draws de_draws(uint32_t i, uint32_t g, uint32_t b, uint32_t NP, uint32_t CR32, uint32_t k0,
                                          uint32_t k1) {
    const U4 w = draw_words(0u, i, g, b, k0, k1);
    uint32_t r1 = __umulhi(w.x, NP - 1u);
    uint32_t r2 = __umulhi(w.y, NP - 2u);
    uint32_t r3 = __umulhi(w.z, NP - 3u);
    const uint32_t jrand = __umulhi(w.w, (uint32_t)D);
    r1 += (r1 >= i);
    {
        const uint32_t e0 = min(i, r1), e1 = max(i, r1);
        r2 += (r2 >= e0);
        r2 += (r2 >= e1);
    }
    {
        // ascending order of {i, r1, r2}
        const uint32_t lo = min(min(i, r1), r2), hi = max(max(i, r1), r2);
        const uint32_t mid = i + r1 + r2 - lo - hi;
        r3 += (r3 >= lo);
        r3 += (r3 >= mid);
        r3 += (r3 >= hi);
    }
    const U4 x1 = draw_words(1u, i, g, b, k0, k1);
    const U4 x2 = draw_words(2u, i, g, b, k0, k1);
    const uint32_t cw[8] = {x1.x, x1.y, x1.z, x1.w, x2.x, x2.y, x2.z, x2.w};
    uint32_t mask = 0;
#pragma unroll
    for (int j = 0; j < D; ++j) mask |= ((cw[j] < CR32) || ((uint32_t)j == jrand)) ? (1u << j) : 0u;
    Draws d;
    d.r1 = (int)r1; d.r2 = (int)r2; d.r3 = (int)r3; d.jrand = (int)jrand; d.mask = mask;
    return d;
}

// Generation-0 uniforms: u_j = (word_j >> 8) 2^-24 from slots 0 and 1; x = lo + (hi - lo) u, each fp64
// operation rounded on its own (no contraction) so that the population is bit-identical to a plain fp64
// evaluation of the same expression.
template <int D>
__device__ __forceinline__ void init_member(uint32_t i, uint32_t b, uint32_t k0, uint32_t k1, const double* lo,
                                            const double* hi, double* out) {
    const U4 a = draw_words(0u, i, 0u, b, k0, k1);
    const U4 c = draw_words(1u, i, 0u, b, k0, k1);
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, c.x, c.y, c.z, c.w};
#pragma unroll
    for (int j = 0; j < D; ++j) {
        const double u = (double)(w[j] >> 8) * (1.0 / 16777216.0);
        out[j] = __dadd_rn(lo[j], __dmul_rn(__dsub_rn(hi[j], lo[j]), u));
    }
}

// Bound handling of one coordinate: reflect once at the violated face, then clamp.
__device__ __forceinline__ double bound_coord(double u, double lo, double hi) {
    if (u < lo) u = __dsub_rn(__dmul_rn(2.0, lo), u);
    else if (u > hi) u = __dsub_rn(__dmul_rn(2.0, hi), u);
    if (u < lo) u = lo;
    if (u > hi) u = hi;
    return u;
}

// Mutation + bound handling of one coordinate, DE/rand/1: v = x1 + F (x2 - x3).
__device__ __forceinline__ double mutate_coord(double x1, double x2, double x3, double F, double lo, double hi) {
    return bound_coord(__dadd_rn(x1, __dmul_rn(F, __dsub_rn(x2, x3))), lo, hi);
}

// The other mutation strategies of Table 4's "strategy" item (reading R21: the six
// strategies of Price, Storn & Lampinen 2006).  Uniform numbers are (word >> 8) 2^-24 of Philox counters
// (slot, i, g, b): slot 3 words 0..3 and slot 4 words 0..3 = per-coordinate jitter; slot 3 word 0 = per-vector
// number; slot 3 word 0 of candidate 0xFFFFFFFF = per-generation number.
enum Strategy {
    kRand1 = 1,          // v = x1 + F (x2 - x3)
    kLocalToBest1 = 2,   // v = xi + F (xb - xi) + F (x2 - x3)
    kBest1Jitter = 3,    // v_j = xb_j + (x2_j - x3_j) (F + 0.0001 rand_j)
    kRand1VecDither = 4, // v = x1 + (F + (1 - F) rand_i) (x2 - x3)
    kRand1GenDither = 5, // v = x1 + (F + (1 - F) rand_g) (x2 - x3)
    kEitherOr = 6        // v = x1 + F (x2 - x3) if rand_i < 0.5 else x1 + 0.5 (F + 1) (x2 + x3 - 2 x1)
};

__device__ __forceinline__ double unit_uniform(uint32_t w) { return (double)(w >> 8) * (1.0 / 16777216.0); }

struct AuxDraws {
    double jit[8];     // per-coordinate jitter numbers (strategy 3)
    double u;          // per-vector (strategies 4, 6) or per-generation (strategy 5) number
};

template <int D>
__device__ __forceinline__ AuxDraws aux_draws(int strategy, uint32_t i, uint32_t g, uint32_t b, uint32_t k0, uint32_t k1) {
    AuxDraws a;
#pragma unroll
    for (int j = 0; j < 8; ++j) a.jit[j] = 0.0;
    a.u = 0.0;
    if (strategy == kBest1Jitter) {
        const U4 w3 = draw_words(3u, i, g, b, k0, k1);
        a.jit[0] = unit_uniform(w3.x); a.jit[1] = unit_uniform(w3.y); a.jit[2] = unit_uniform(w3.z); a.jit[3] = unit_uniform(w3.w);
        if (D > 4) {
            const U4 w4 = draw_words(4u, i, g, b, k0, k1);
            a.jit[4] = unit_uniform(w4.x); a.jit[5] = unit_uniform(w4.y); a.jit[6] = unit_uniform(w4.z); a.jit[7] = unit_uniform(w4.w);
        }
    } else if (strategy == kRand1VecDither || strategy == kEitherOr) {
        a.u = unit_uniform(draw_words(3u, i, g, b, k0, k1).x);
    } else if (strategy == kRand1GenDither) {
        a.u = unit_uniform(draw_words(3u, 0xFFFFFFFFu, g, b, k0, k1).x);
    }
    return a;
}

// mutant value of one coordinate before bound handling; every fp64 operation rounds on its own, in this order
__device__ __forceinline__ double mutant_coord(int strategy, double xi, double x1, double x2, double x3, double xb,
                                               double F, double jit, double u) {
    switch (strategy) {
        case kLocalToBest1:
            return __dadd_rn(__dadd_rn(xi, __dmul_rn(F, __dsub_rn(xb, xi))), __dmul_rn(F, __dsub_rn(x2, x3)));
        case kBest1Jitter:
            return __dadd_rn(xb, __dmul_rn(__dsub_rn(x2, x3), __dadd_rn(F, __dmul_rn(0.0001, jit))));
        case kRand1VecDither:
        case kRand1GenDither:
            return __dadd_rn(x1, __dmul_rn(__dadd_rn(F, __dmul_rn(__dsub_rn(1.0, F), u)), __dsub_rn(x2, x3)));
        case kEitherOr:
            if (u < 0.5) return __dadd_rn(x1, __dmul_rn(F, __dsub_rn(x2, x3)));
            return __dadd_rn(x1, __dmul_rn(__dmul_rn(0.5, __dadd_rn(F, 1.0)), __dsub_rn(__dadd_rn(x2, x3), __dmul_rn(2.0, x1))));
        default:
            return __dadd_rn(x1, __dmul_rn(F, __dsub_rn(x2, x3)));
    }
}

// ---------------------------------------------------------------------------------------------------
// Quantised samples (Table 3: 1/2/4/8/16-bit recording modes; reading R23).
// Sample n of a row is its bits-wide field n, packed from the least significant bit of each byte upwards (16-bit:
// little-endian); read as unsigned or two's complement; value = scale (code + offset) in fp64, rounded once to fp32.
// ---------------------------------------------------------------------------------------------------
struct Quant {
    int bits;          // 0: the samples are fp32 already
    int is_signed;
    double scale, offset;
};

__device__ __forceinline__ float unpack_sample(const unsigned char* __restrict__ row, long long n, const Quant& q) {
    uint32_t field;
    if (q.bits == 16) {
        field = (uint32_t)__ldg(row + 2 * n) | ((uint32_t)__ldg(row + 2 * n + 1) << 8);
    } else {
        const long long bit = n * q.bits;
        field = ((uint32_t)__ldg(row + (bit >> 3)) >> (int)(bit & 7)) & ((1u << q.bits) - 1u);
    }
    int code = (int)field;
    if (q.is_signed && ((field >> (q.bits - 1)) & 1u)) code = (int)field - (int)(1u << q.bits);
    return __double2float_rn(__dmul_rn(q.scale, __dadd_rn((double)code, q.offset)));
}

// ---------------------------------------------------------------------------------------------------
// mbarrier + 1-D bulk async copy (TMA engine, SASS UBLKCP) -- global -> shared staging of a data block.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// generic-proxy writes to GLOBAL memory made visible to later bulk async copies that read them
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
    }
}
// try_wait with a suspend-time hint: the thread sleeps in hardware until the phase completes (or the hint expires) instead of
// spinning on the issue slots of the warps that compute
__device__ __forceinline__ void mbar_wait_suspended(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity), "r"(1000000u) : "memory");
    } while (!ok);
}
// bytes must be a multiple of 16, src and dst 16-byte aligned
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Thread-block clusters: rank / size of this CTA's cluster, peer shared-memory stores (DSMEM), cluster barrier.
// A launch without the cluster attribute is a cluster of one CTA: the special registers read 0 / 1.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_id_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
// address of the same shared-memory location in CTA `rank` of this cluster (shared::cluster window)
__device__ __forceinline__ uint32_t mapa_shared(const void* p, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_u32(p)), "r"(rank));
    return r;
}
__device__ __forceinline__ void st_cluster_f32(uint32_t addr, float v) {
    asm volatile("st.shared::cluster.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
// all threads of all CTAs of the cluster; release/acquire orders the peer stores before the reads after it
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

}  // namespace pt
