// scoring_seq20.cu — explicit / seeded sequences over ANY alphabet (the 20-letter MJ-style model, a8) on the tensor
// cores: the paper's sampling runs at their Table-3 sizes (MJ 6x6 and MJ 3x3x3).
//
// E(seq, S) = sum over the contacts (i,j) of S of M[s_i][s_j] (Eq. 1, :67-69).  Per sequence the P monomer pairs that can
// ever touch get a non-negative cost c_p = emax - M[s_i][s_j], split into two int8 limbs c_p = lo_p + 64 hi_p
// (lo < 64, hi <= 127).  The structure side is a 0/-1 incidence matrix X[S][p] (-1 where p is a contact of S): it does
// not depend on the energies, is built once per lattice and cached in the handle.  Two tcgen05.mma kind::i8 chains per
// (128 sequences x 128 structures) share every incidence block:  acc_lo = lo . X^T,  acc_hi = hi . X^T,  and the epilogue
// recombines  v = acc_lo + 64 acc_hi = -(cost of S) = E - NBP emax  on packed int16 pairs before the same filtered
// min / second-min / argmin fold as scoring_tc.cu (ties -> null, R6, R7).  Pad structures get v = +127 from a constant
// column, above every real v <= 0.  Exact integer arithmetic throughout.
//
// Bound (profiles/r2_seq20_ncu.md): with one 128-sequence tile per CTA every incidence block feeds only two MMAs (lo, hi),
// 2 KB of shared-memory ingest per 66-clock MMA = 31 B/clk/SM, and an SM takes 20-25 B/clk from L2 whatever the
// mechanism (one cp.async.bulk per tile, per block, or a warp of 16-byte cp.async), ring depth or number of SMs running:
// the kernel is bound by that feed at about 55 % tensor-pipe activity.
#include <vector>

#include "tc_common.cuh"

namespace tc {

constexpr int QRB = 64;                          // bytes per operand row of a column block (64-byte swizzle): two K steps
constexpr int QBLK = TM * QRB;                   // 8 KB: one column block of 128 rows
constexpr int Q_KB_MAX = 6;                      // column blocks per limb set: 2 + P <= 384 columns
constexpr int Q_STAGES_MAX = 6;                  // structure tiles (kb x 16 KB of incidence blocks each) in flight
constexpr int Q_PARTS = 4;                       // column parts of a structure tile, one epilogue warp each per lane quarter
constexpr int Q_THREADS = 32 * (2 + 4 * Q_PARTS); // warp 0 TMA producer, warp 1 MMA issuer, 16 builder / epilogue warps
constexpr int Q_ROWS = TM;                       // sequences per item
constexpr int V_PAD = 127;                       // value of the pad structures
constexpr int V_NONE = 32767;

enum { QSRC_SEQS = 0, QSRC_SEEDED = 1 };

struct QArgs {
    const int8_t* img;        // [n_tiles][kb][QBLK] incidence blocks
    const uint16_t* class_of;
    const uint8_t* seqs;      // count x N letters (QSRC_SEQS)
    const uint8_t* pair_ij;   // P x 2 monomers of every pair column
    uint16_t* pheno;
    int16_t* gap;             // nullable
    uint64_t count, first, seed;
    uint32_t n_items, n_tiles;
    int N, P, kb, ksteps, alphabet, threshold, src, stages;
    int16_t cost[400];        // emax - M[a][b]
};

struct __align__(16) QBarriers {
    uint64_t b_full[Q_STAGES_MAX], b_empty[Q_STAGES_MAX];
    uint64_t acc_full[2], acc_empty[2];
    uint64_t a_full, a_empty;
    uint32_t tmem_base;
};

// 32 accumulator columns as 16 registers of two int16
__device__ __forceinline__ void tmem_ld16_pack16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.pack::16b.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr) : "memory");
}

// the filtered fold of scoring_tc.cu on 64-bit keys: v spans 16 bits here, so v * 2^17 + column needs more than 32
template <int NG>   // NG groups of 8 columns (4 registers each)
__device__ __forceinline__ void fold_packed64(const uint32_t* w, uint32_t col0, long long& k1, long long& k2, uint32_t& E2) {
    uint32_t g[NG];
#pragma unroll
    for (int s = 0; s < NG; s++)
        g[s] = __vimin3_s16x2(w[4 * s], w[4 * s + 1], __vmins2(w[4 * s + 2], w[4 * s + 3]));
    uint32_t all = g[0];
#pragma unroll
    for (int s = 1; s < NG; s++) all = __vmins2(all, g[s]);
    if (__vmins2(all, E2) != E2) {
#pragma unroll
        for (int s = 0; s < NG; s++) {
            if (__vmins2(g[s], E2) != E2) {
#pragma unroll
                for (int j = 0; j < 4; j++) {
                    const uint32_t x = w[4 * s + j];
                    const long long lo = (long long)(int16_t)(x & 0xFFFFu), hi = (long long)((int32_t)x >> 16);
                    const long long c = (long long)(col0 + 8 * s + 2 * j);
                    const long long key0 = lo * (1 << KEY_SHIFT) + c, key1 = hi * (1 << KEY_SHIFT) + c + 1;
                    k2 = min(k2, max(k1, key0));
                    k1 = min(k1, key0);
                    k2 = min(k2, max(k1, key1));
                    k1 = min(k1, key1);
                }
                const long long e2 = k2 >> KEY_SHIFT;
                E2 = (uint32_t)((e2 > V_NONE ? V_NONE : (int32_t)e2) & 0xFFFF) * 0x10001u;
            }
        }
    }
}

// Incidence image: one block = one 128-structure tile; thread = structure; the column blocks are built one by one.
__global__ void __launch_bounds__(TN) build_pair_image_kernel(const uint16_t* __restrict__ pairidx, int8_t* __restrict__ img,
                                                              uint32_t D, int NBP, int kb) {
    __shared__ __align__(16) int8_t tile[QBLK];
    const uint32_t r = threadIdx.x, n = blockIdx.x, d = n * TN + r;
    for (int b = 0; b < kb; b++) {
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < QBLK / 16; i += TN) reinterpret_cast<uint4*>(tile)[i] = make_uint4(0, 0, 0, 0);
        __syncthreads();
        const int c0 = b * QRB;
        if (d < D) {
            const uint16_t* px = pairidx + (size_t)d * NBP;
            for (int k = 0; k < NBP; k++) {
                const int c = 2 + px[k] - c0;
                if (c >= 0 && c < QRB) tile[swz_rb<QRB>(r, c)] = -1;
            }
        } else if (b == 0) {
            tile[swz_rb<QRB>(r, 0)] = V_PAD;   // pad structure: the constant column gives it v = +127
        }
        __syncthreads();
        uint4* dst = reinterpret_cast<uint4*>(img + ((uint64_t)n * kb + b) * QBLK);
        for (uint32_t i = threadIdx.x; i < QBLK / 16; i += TN) dst[i] = reinterpret_cast<const uint4*>(tile)[i];
    }
}

template <int SRC>
__global__ void __launch_bounds__(Q_THREADS, 1) seq20_kernel(const QArgs a) {
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;                                           // [lo | hi][kb][8 KB]
    uint8_t* sB = sA + 2 * a.kb * QBLK;                           // a.stages x kb x 8 KB
    QBarriers* bar = reinterpret_cast<QBarriers*>(sB + a.stages * a.kb * QBLK);
    const uint32_t Q_STAGES = (uint32_t)a.stages;
    uint8_t* let = reinterpret_cast<uint8_t*>(bar + 1);           // [N][128] letters of the item's sequences
    uint8_t* pij = let + a.N * Q_ROWS;                            // [P][2]
    int16_t* cost = reinterpret_cast<int16_t*>(pij + ((2 * a.P + 15) & ~15));
    long long* merge = reinterpret_cast<long long*>(cost + 400);  // [Q_PARTS][128][2] partial (k1, k2) per item
    constexpr uint32_t IDESC = idesc_for(TN);

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (int i = threadIdx.x; i < 2 * a.P; i += Q_THREADS) pij[i] = a.pair_ij[i];
    for (int i = threadIdx.x; i < a.alphabet * a.alphabet; i += Q_THREADS) cost[i] = a.cost[i];
    if (threadIdx.x == 0) {
        for (uint32_t s = 0; s < Q_STAGES; s++) { mbar_init(&bar->b_full[s], 1); mbar_init(&bar->b_empty[s], 1); }
        for (int b = 0; b < 2; b++) { mbar_init(&bar->acc_full[b], 1); mbar_init(&bar->acc_empty[b], 4 * Q_PARTS); }
        mbar_init(&bar->a_full, Q_ROWS * Q_PARTS);
        mbar_init(&bar->a_empty, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == 1) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&bar->tmem_base)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = bar->tmem_base;

    if (warp == 0) {
        // ===== producer: one bulk copy per structure tile (its kb incidence blocks are contiguous), once per item =====
        const uint32_t stage_bytes = (uint32_t)a.kb * QBLK;
        uint32_t it = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x)
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                const uint32_t s = it % Q_STAGES, ph = (it / Q_STAGES) & 1;
                mbar_wait(&bar->b_empty[s], ph ^ 1);
                if (elect_one()) {
                    mbar_expect_tx(&bar->b_full[s], stage_bytes);
                    bulk_g2s(sB + s * stage_bytes, a.img + (uint64_t)n * stage_bytes, stage_bytes, &bar->b_full[s]);
                }
                __syncwarp();
            }
    } else if (warp == 1) {
        // ===== MMA issuer: two chains (lo, hi limbs) per structure tile share every incidence block; accumulator pairs
        // double-buffered =====
        const uint64_t a_lo0 = smem_desc_rb<QRB>(smem_u32(sA)), a_hi0 = smem_desc_rb<QRB>(smem_u32(sA + a.kb * QBLK));
        const uint64_t b_desc0 = smem_desc_rb<QRB>(smem_u32(sB));
        uint32_t tile_no = 0, item_no = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x, item_no++) {
            mbar_wait(&bar->a_full, item_no & 1);
            tc_fence_after();
            for (uint32_t n = 0; n < a.n_tiles; n++, tile_no++) {
                const uint32_t buf = tile_no & 1;
                mbar_wait(&bar->acc_empty[buf], ((tile_no >> 1) & 1) ^ 1);
                tc_fence_after();
                const uint32_t d_lo = tmem + (2 * buf) * TN, d_hi = d_lo + TN;
                const uint32_t s = tile_no % Q_STAGES, ph = (tile_no / Q_STAGES) & 1;
                mbar_wait(&bar->b_full[s], ph);
                tc_fence_after();
                if (elect_one()) {
                    const uint64_t bd0 = b_desc0 + (uint64_t)s * (uint64_t)((a.kb * QBLK) >> 4);
                    for (int b = 0; b < a.kb; b++) {
                        const uint64_t blk = (uint64_t)((b * QBLK) >> 4);
                        const int nks = a.ksteps - 2 * b < 2 ? a.ksteps - 2 * b : 2;   // a 64-byte block holds two K steps
                        for (int ks = 0; ks < nks; ks++) {
                            const uint32_t acc = (b | ks) != 0;
                            mma_i8(d_lo, a_lo0 + blk + 2 * ks, bd0 + blk + 2 * ks, IDESC, acc);
                            mma_i8(d_hi, a_hi0 + blk + 2 * ks, bd0 + blk + 2 * ks, IDESC, acc);
                        }
                    }
                    tc_commit(&bar->b_empty[s]);
                    tc_commit(&bar->acc_full[buf]);
                }
                __syncwarp();
            }
            if (elect_one()) tc_commit(&bar->a_empty);
            __syncwarp();
        }
    } else {
        // ===== limb rows + epilogue: 16 warps.  Warp = (TMEM lane quarter, column part): the four warps of a quarter share
        // the 32 sequences of that quarter and split the 128 columns of every structure tile (one warp per SM
        // sub-partition cannot hide its own latencies: profiles/r2_seq20_ncu.md); their (k1, k2) are merged per item. =====
        const uint32_t quarter = warp & 3, part = (warp - 2) >> 2;
        const uint32_t r = quarter * 32 + lane;
        const uint32_t t_lane = tmem + ((quarter * 32u) << 16) + part * 32u;
        uint8_t* my_let = let + r;
        uint32_t tile_no = 0, item_no = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x, item_no++) {
            const uint64_t q = (uint64_t)item * Q_ROWS + r;
            for (int i = 0; i < a.N; i++) {   // the row's four threads each need all letters: every one writes the same bytes
                uint32_t l = 0;
                if (q < a.count) l = SRC == QSRC_SEQS ? a.seqs[q * a.N + i] : gp_letter(a.seed, a.first + q, i, (uint32_t)a.alphabet);
                my_let[i * Q_ROWS] = (uint8_t)min(l, (uint32_t)a.alphabet - 1u);  // a letter outside the alphabet counts as the last one
            }
            mbar_wait(&bar->a_empty, (item_no & 1) ^ 1);
            for (int b = part; b < 2 * a.kb; b += Q_PARTS)
#pragma unroll
                for (int c16 = 0; c16 < QRB / 16; c16++)
                    *reinterpret_cast<uint4*>(sA + b * QBLK + r * QRB + c16 * 16) = make_uint4(0, 0, 0, 0);
            asm volatile("bar.sync %0, 128;" ::"r"(quarter + 1) : "memory");   // the row is zeroed before its bytes are set
            if (part == 0) sA[swz_rb<QRB>(r, 0)] = 1;                        // constant column (lo limb set only)
            uint8_t* sHi = sA + a.kb * QBLK;
            for (int p = part; p < a.P; p += Q_PARTS) {
                const uint32_t c = (uint32_t)cost[my_let[pij[2 * p] * Q_ROWS] * a.alphabet + my_let[pij[2 * p + 1] * Q_ROWS]];
                const uint32_t col = 2u + p, off = (col >> 6) * QBLK + swz_rb<QRB>(r, col & 63u);
                sA[off] = (uint8_t)(c & 63u);
                sHi[off] = (uint8_t)(c >> 6);
            }
            fence_proxy_async();
            mbar_arrive(&bar->a_full);

            long long k1 = LLONG_MAX, k2 = LLONG_MAX;
            uint32_t E2 = (uint32_t)V_NONE * 0x10001u;
#pragma unroll 1
            for (uint32_t n = 0; n < a.n_tiles; n++, tile_no++) {
                const uint32_t buf = tile_no & 1;
                mbar_wait(&bar->acc_full[buf], (tile_no >> 1) & 1);
                tc_fence_after();
                uint32_t wl[16], wh[16];
                tmem_ld16_pack16(t_lane + (2 * buf) * TN, wl);
                tmem_ld16_pack16(t_lane + (2 * buf + 1) * TN, wh);
                tmem_ld_wait();
                tc_fence_before();       // this warp's share of both accumulators is in registers
                __syncwarp();
                if (lane == 0) mbar_arrive(&bar->acc_empty[buf]);
#pragma unroll
                for (int i = 0; i < 16; i++) wl[i] = __vadd2(wl[i], (wh[i] << 6) & 0xFFC0FFC0u);  // v = -(lo + 64 hi), per int16
                fold_packed64<4>(wl, n * TN + part * 32u, k1, k2, E2);
            }
            // merge the four column parts of every sequence: the two smallest of eight distinct keys
            merge[(part * Q_ROWS + r) * 2] = k1;
            merge[(part * Q_ROWS + r) * 2 + 1] = k2;
            asm volatile("bar.sync %0, 128;" ::"r"(quarter + 1) : "memory");
            if (part == 0) {
#pragma unroll
                for (int o = 1; o < Q_PARTS; o++) {
                    const long long x1 = merge[(o * Q_ROWS + r) * 2], x2 = merge[(o * Q_ROWS + r) * 2 + 1];
                    k2 = min(min(k2, x2), max(k1, x1));
                    k1 = min(k1, x1);
                }
                if (q < a.count) {
                    const long long e1 = k1 >> KEY_SHIFT, e2 = k2 >> KEY_SHIFT;
                    const uint32_t col = (uint32_t)(k1 & ((1LL << KEY_SHIFT) - 1));
                    const bool single = e2 >= V_PAD;   // D = 1: the runner-up is a pad structure
                    const bool folds = single || (e2 - e1 >= a.threshold);
                    a.pheno[q] = folds ? a.class_of[col] : (uint16_t)GP_NULL_PHENO;
                    if (a.gap) a.gap[q] = (int16_t)(single ? GP_GAP_NONE : (e1 - e2 < -32768 ? -32768 : e1 - e2));
                }
            }
            asm volatile("bar.sync %0, 128;" ::"r"(quarter + 1) : "memory");   // merge[] is free again
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
}

}  // namespace tc

// Any-alphabet sequences on the tensor cores.  GP_UNSUPPORTED_LATTICE = not eligible (too many pair columns, energies
// whose spread does not fit the limbs / int16 values): the caller falls back to the CUDA-core kernel.
gp_status gp_launch_seq20_tc(const gp_structures_s* s, const gp_energies* en, int seeded, const uint8_t* d_seqs, uint64_t seed,
                             uint64_t first, uint64_t count, uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st) {
    using namespace tc;
    const int A = en->alphabet, ncol = 2 + s->P;
    if (ncol > Q_KB_MAX * QRB || s->N > 64 || s->D >= (1u << KEY_SHIFT) || A < 2 || A > 20) return GP_UNSUPPORTED_LATTICE;
    int32_t emax = INT32_MIN, emin = INT32_MAX;
    for (int i = 0; i < A * A; i++) { emax = en->e[i] > emax ? en->e[i] : emax; emin = en->e[i] < emin ? en->e[i] : emin; }
    if ((long long)emax - emin > 8191 || ((long long)emax - emin) * s->NBP > 32000) return GP_UNSUPPORTED_LATTICE;
    QArgs a;
    for (int i = 0; i < A * A; i++) a.cost[i] = (int16_t)(emax - en->e[i]);
    const int kb = (ncol + QRB - 1) / QRB;
    const uint32_t n_tiles = (s->D + TN - 1) / TN;
    {   // incidence image: depends on the lattice only; built once, other streams wait on its event
        std::lock_guard<std::mutex> lk(s->mu);
        if (!s->d_pair_img) {
            int8_t* img = nullptr;
            GP_CUDA(cudaMalloc(&img, (size_t)n_tiles * kb * QBLK));  // first use on this handle only
            build_pair_image_kernel<<<n_tiles, TN, 0, st>>>(s->d_pairidx, img, s->D, s->NBP, kb);
            cudaError_t e = cudaGetLastError();
            cudaEvent_t ev = nullptr;
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventRecord(ev, st);
            if (e != cudaSuccess) { cudaFree(img); gp_set_cuda_error(e, "pair image"); return GP_CUDA_ERROR; }
            gp_count_launches(1);
            s->d_pair_img = img;
            s->pair_img_ready = ev;
        } else {
            GP_CUDA(cudaStreamWaitEvent(st, (cudaEvent_t)s->pair_img_ready, 0));
        }
    }
    a.img = s->d_pair_img; a.class_of = s->d_class_of; a.seqs = d_seqs; a.pair_ij = s->d_pair_ij; a.pheno = d_pheno; a.gap = d_gap;
    a.count = count; a.first = first; a.seed = seed;
    a.n_items = (uint32_t)((count + Q_ROWS - 1) / Q_ROWS); a.n_tiles = n_tiles;
    a.N = s->N; a.P = s->P; a.kb = kb; a.ksteps = (ncol + 31) / 32; a.alphabet = A; a.threshold = en->threshold;
    a.src = seeded ? QSRC_SEEDED : QSRC_SEQS;
    int dev = 0, sms = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t aux = sizeof(QBarriers) + (size_t)s->N * Q_ROWS + ((2 * (size_t)s->P + 15) & ~(size_t)15) + 800 +
                       (size_t)Q_PARTS * Q_ROWS * 16 + 1024 + 64;
    // a stage holds the kb incidence blocks of one structure tile, fetched by ONE bulk copy (16 KB copies were measured
    // to deliver a block per 940 clocks and SM, whatever the ring depth: profiles/r2_seq20_ncu.md)
    int stages = (int)(((227 * 1024 - aux) / QBLK - 2 * kb) / kb);
    if (stages > Q_STAGES_MAX) stages = Q_STAGES_MAX;
    if (stages < 2) return GP_UNSUPPORTED_LATTICE;
    a.stages = stages;
    const size_t smem = (size_t)(2 * kb + stages * kb) * QBLK + aux;
    void (*k)(const QArgs) = seeded ? seq20_kernel<QSRC_SEEDED> : seq20_kernel<QSRC_SEQS>;
    GP_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const unsigned grid = a.n_items < (uint32_t)sms ? a.n_items : (uint32_t)sms;
    const uint64_t tk1 = gp_time_begin(GP_KERNEL_SCORING, st);
    k<<<grid, Q_THREADS, smem, st>>>(a);
    gp_time_end(GP_KERNEL_SCORING, tk1, st);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}
