// tc_common.cuh — tile geometry, PTX wrappers (mbarrier, cp.async.bulk, tcgen05.*) and shared-memory descriptors used by
// libgpmap's tensor-core kernels (scoring_tc.cu, scoring_seq20.cu).  Private to the library; not used by oracle/.
#pragma once
#include "device_common.cuh"

namespace tc {

constexpr int MT = 4;                 // genotype tiles per supertile
constexpr int TM = 128, TN = 128;     // weight tile: 128 structures; genotype tile: 128 rows
constexpr int HN = 64;                // the epilogue folds 64 columns at a time
constexpr int ROWB = 128;             // bytes per operand row = one 128-byte swizzle span = up to 128 int8 features
constexpr int TILE_BYTES = TM * ROWB; // 16 KB, A tile and B stage alike
constexpr int NSTAGE = 6;
constexpr int SUPER = MT * TM;        // 512 genotypes
constexpr int NISS = 2;                // MMA issuer warps of scoring_kernel (each owns MT / NISS accumulators)
constexpr int EPI_WARPS = 4 * MT;     // warp group m = warps 1+NISS+4m .. drains accumulator m
constexpr int THREADS = 32 * (1 + NISS + EPI_WARPS);  // warp 0 TMA producer, warps 1..NISS MMA issuers, then feature build + epilogue
constexpr int MAX_FB = 22;            // 2 + 22 + 100 pairs = 124 <= 128 columns
constexpr int KEY_SHIFT = 17;         // key = E * 2^17 + column (D < 2^17, |E| < 2^13)
constexpr int E_NONE = 16383;         // INT32_MAX >> KEY_SHIFT: "no energy yet"
constexpr int E_PAD = 8191;           // energy of the pad structures D..n_tiles*128-1 (bias columns 127*64 + 63): above
                                      // every real energy (|E| <= 8190 is checked in gp_check_hp), so a pad never wins

struct Cols {        // column c of the folded contraction: A byte = val * h_i * h_j  (bit 31 of the row word is always 1)
    uint8_t i[ROWB], j[ROWB], val[ROWB];
};

// ---- PTX wrappers ------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// TMA engine, 1-D bulk copy global -> shared, completion counted in bytes on an mbarrier
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[smem] . B[smem]^T, int8 x int8 -> int32
__device__ __forceinline__ void mma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc),
        "r"(accumulate) : "memory");
}
template <bool ACC>
__device__ __forceinline__ void mma_i8_c(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc) {
    if (ACC)
        asm volatile("{\n\t.reg .pred p;\n\tsetp.eq.u32 p, 1, 1;\n\t"
                     "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc) : "memory");
    else
        asm volatile("{\n\t.reg .pred p;\n\tsetp.eq.u32 p, 1, 0;\n\t"
                     "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc) : "memory");
}
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0;
}
// 128 accumulator columns as 64 registers: .pack::16b keeps the low 16 bits of each 32-bit column and packs two
// adjacent columns per register (column 2i in the low half of v[i], column 2i+1 in the high half).  Energies are
// |E| <= 8191, so the low 16 bits are the exact int16 value.
__device__ __forceinline__ void tmem_ld64_pack16(uint32_t taddr, uint32_t (&v)[64]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x64.pack::16b.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63}, [%64];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]), "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]), "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31]), "=r"(v[32]), "=r"(v[33]), "=r"(v[34]), "=r"(v[35]), "=r"(v[36]), "=r"(v[37]), "=r"(v[38]), "=r"(v[39]), "=r"(v[40]), "=r"(v[41]), "=r"(v[42]), "=r"(v[43]), "=r"(v[44]), "=r"(v[45]), "=r"(v[46]), "=r"(v[47]), "=r"(v[48]), "=r"(v[49]), "=r"(v[50]), "=r"(v[51]), "=r"(v[52]), "=r"(v[53]), "=r"(v[54]), "=r"(v[55]), "=r"(v[56]), "=r"(v[57]), "=r"(v[58]), "=r"(v[59]), "=r"(v[60]), "=r"(v[61]), "=r"(v[62]), "=r"(v[63])
        : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// shared-memory matrix descriptor: K-major, 128-byte swizzle, 8-row groups 1024 B apart (rows are 128 B)
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ULL << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ULL << 46) | (2ULL << 61);
}
// instruction descriptor: D = s32, A = B = s8, both K-major, N = n, M = 128
__host__ __device__ constexpr uint32_t idesc_for(int n) {
    return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(TM >> 4) << 24);
}

// byte offset of (row r, byte c) inside a 128-byte-swizzled tile with 128-byte rows
__host__ __device__ __forceinline__ uint32_t swz(uint32_t r, uint32_t c) {
    return r * ROWB + ((((c >> 4) ^ (r & 7u)) << 4) | (c & 15u));
}
// the same for rows of RB = 64 bytes (64-byte swizzle: 16-byte chunk index ^ bits 1-2 of the row) or 128 bytes
template <int RB>
__host__ __device__ __forceinline__ uint32_t swz_rb(uint32_t r, uint32_t c) {
    return RB == 128 ? swz(r, c) : r * 64u + ((((c >> 4) ^ ((r >> 1) & 3u)) << 4) | (c & 15u));
}
// K-major shared-memory descriptor for rows of RB bytes: 8-row groups RB*8 bytes apart, 128- or 64-byte swizzle
template <int RB>
__device__ __forceinline__ uint64_t smem_desc_rb(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ULL << 16) | ((uint64_t)((RB * 8) >> 4) << 32) | (1ULL << 46) |
           ((RB == 128 ? 2ULL : 4ULL) << 61);
}

}  // namespace tc
