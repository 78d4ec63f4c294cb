// pt_tc_device.cuh -- tcgen05 / TMEM helpers of the tensor-core evaluation path (pt_tc_kernel.cuh), sm_100a only.
//
// The phase of candidate c at sample n of a 256-sample tile is a small dense contraction,
//     phase[c][j] = E0_c + E1_c j + E2_c j^2 + E3_c j^3 = sum_k A[c][k] B[j][k],      j = n - (tile centre),
// (Eq. 3, re-expanded about the tile centre) with A = the candidate's coefficients split into tf32-exact
// pieces and B = the fixed basis (1, j, j^2, j^3, also in tf32-exact pieces).  It runs on the 5th-generation tensor cores
// (tcgen05.mma kind::tf32, fp32 accumulators in TMEM), which takes the four phase operations per sample-evaluation off the
// FP32 pipe.  Every operand entry has at most 11 significant bits, so every product is exact and the only rounding is the
// fp32 accumulation of 11 terms inside the tensor core.
#pragma once
#include "pt_device.cuh"

namespace pt {
namespace tc {

constexpr int kTile = 256;                 // samples per MMA tile (UMMA N = 256, the largest)
constexpr int kRowsA = 128;                // candidates per MMA (UMMA M = 128 = the TMEM lanes)
constexpr int kK = 16;                     // tf32 entries per operand row: two K = 8 instructions
constexpr int kABytes = kRowsA * kK * 4;   // 8 KB: one coefficient operand
constexpr int kBBytes = kTile * kK * 4;    // 16 KB: the basis operand
constexpr int kAChunk = kRowsA * 16;       // bytes between consecutive 16-byte K chunks of A (chunk-major [kc][row])
constexpr int kBChunk = kTile * 16;        // the same for B
constexpr int kAStages = 4;                // ring of coefficient operands
constexpr int kTmemBufs = 2;               // ring of 256-column accumulators: all 512 TMEM columns
constexpr int kTmemCols = 512;

__device__ __forceinline__ void tmem_alloc(uint32_t* dst_smem, uint32_t cols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "r"(cols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t addr, uint32_t cols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(addr), "r"(cols) : "memory");
}
__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// arrives on the mbarrier once every tcgen05 operation this thread issued before has completed
__device__ __forceinline__ void commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// try_wait with a suspend-time hint: the thread sleeps in hardware until the phase completes (or the hint expires)
__device__ __forceinline__ void mbar_wait_sleep(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    do {
        asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\nselp.u32 %0, 1, 0, p;\n}\n"
                     : "=r"(ok) : "r"(smem_u32(bar)), "r"(parity), "r"(1000000u) : "memory");
    } while (!ok);
}

// Shared-memory matrix descriptor, K-major, no swizzle: a core matrix is 8 rows x 16 bytes (rows 16 bytes apart);
// SBO = bytes between 8-row groups, LBO = bytes between the two 16-byte K chunks one instruction reads; version 1 (sm_100).
__device__ __forceinline__ uint64_t make_desc(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
    uint64_t d = 0;
    d |= (uint64_t)((saddr >> 4) & 0x3FFFu);
    d |= (uint64_t)((lbo >> 4) & 0x3FFFu) << 16;
    d |= (uint64_t)((sbo >> 4) & 0x3FFFu) << 32;
    d |= (uint64_t)1 << 46;
    return d;
}
// Instruction descriptor of kind::tf32: D fp32 (bits 4-5 = 1), A and B tf32 (bits 7-9, 10-12 = 2), both K-major, N >> 3 at
// bit 17, M >> 4 at bit 24.
__host__ __device__ constexpr uint32_t make_idesc_tf32(int M, int N) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(N >> 3) << 17) | ((uint32_t)(M >> 4) << 24);
}
// D[tmem] (+)= A[smem] . B[smem]^T, issued by ONE thread on behalf of the CTA
__device__ __forceinline__ void mma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile("{\n.reg .pred p;\nsetp.ne.b32 p, %4, 0;\ntcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n}\n"
                 ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate) : "memory");
}
// 16 consecutive columns of this thread's TMEM lane (lane = 32 (warp % 4) + lane id)
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
                   "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                 : "r"(taddr) : "memory");
}

// One tf32-exact piece of a double by integer operations on its bits only -- no F2F conversion: conversions execute on the
// XU pipe, the pipe the cosines saturate (measured: 16 % of the XU cycles went to conversions in the first prototype).
// h = v truncated toward zero to 11 significant bits, as fp32 bits; hd = the same value as a double.  |v| < 2^-126 gives 0.
__device__ __forceinline__ void tf32_piece(double v, float& h, double& hd) {
    const uint32_t hi = (uint32_t)__double2hiint(v);
    const uint32_t mag = hi & 0x7FFFFFFFu;
    const bool ok = mag >= 0x38100000u;                                    // biased exponent >= 897  <=>  |v| >= 2^-126
    const uint32_t fb = (((mag - 0x38000000u) << 3) & 0x7FFFE000u) | (hi & 0x80000000u);
    h = __uint_as_float(ok ? fb : 0u);
    hd = __hiloint2double(ok ? (int)(hi & 0xFFFFFC00u) : 0, 0);
}
// v = h + m + l to 33 bits / v = h + m to 22 bits, every piece tf32-exact
__device__ __forceinline__ void split3(double v, float& h, float& m, float& l) {
    double hd, md, ld;
    tf32_piece(v, h, hd);
    const double r1 = v - hd;
    tf32_piece(r1, m, md);
    tf32_piece(r1 - md, l, ld);
}
__device__ __forceinline__ void split2(double v, float& h, float& m) {
    double hd, md;
    tf32_piece(v, h, hd);
    tf32_piece(v - hd, m, md);
}

// Row `row` of an operand (16 fp32 entries), chunk-major layout [kc][row] of 16-byte vectors: conflict-free 128-bit stores
__device__ __forceinline__ void write_row(unsigned char* op, int row, const float (&e)[16], int chunk_stride) {
#pragma unroll
    for (int kc = 0; kc < 4; ++kc)
        *reinterpret_cast<float4*>(op + kc * chunk_stride + row * 16) = make_float4(e[4 * kc], e[4 * kc + 1], e[4 * kc + 2], e[4 * kc + 3]);
}

// Basis row of sample j in [-128, 128): slots 0-2 -> 1, 3-5 -> j, 6 and 8 -> (j^2)_h, 7 -> (j^2)_l, 9 and 11 -> (j^3)_h,
// 10 -> (j^3)_l, 12-15 -> 0.  j^2 <= 2^14 and |j^3| <= 2^21 split exactly into an 11-bit head and a tail of <= 10 bits.
__device__ __forceinline__ void basis_row(int j, float (&e)[16]) {
    const float jf = (float)j;
    const float j2 = jf * jf, j3 = j2 * jf;
    const float j2h = __uint_as_float(__float_as_uint(j2) & 0xFFFFE000u), j2l = j2 - j2h;
    const float j3h = __uint_as_float(__float_as_uint(j3) & 0xFFFFE000u), j3l = j3 - j3h;
    e[0] = e[1] = e[2] = 1.0f;
    e[3] = e[4] = e[5] = jf;
    e[6] = j2h; e[7] = j2l; e[8] = j2h;
    e[9] = j3h; e[10] = j3l; e[11] = j3h;
    e[12] = e[13] = e[14] = e[15] = 0.0f;
}
// Coefficient row of phase(j) = E0 + E1 j + E2 j^2 + E3 j^3 [rad]: E0, E1 to 33 bits (|E1 j| reaches 400 rad at Nyquist),
// E2, E3 to 22 bits; slots pair with basis_row (E2_h with both pieces of j^2, E2_m with its head; the same for E3).
__device__ __forceinline__ void coef_row(double E0, double E1, double E2, const float E3h, const float E3m, float (&e)[16]) {
    split3(E0, e[0], e[1], e[2]);
    split3(E1, e[3], e[4], e[5]);
    float h, m;
    split2(E2, h, m);
    e[6] = h; e[7] = h; e[8] = m;
    e[9] = E3h; e[10] = E3h; e[11] = E3m;
    e[12] = e[13] = e[14] = e[15] = 0.0f;
}

}  // namespace tc
}  // namespace pt
