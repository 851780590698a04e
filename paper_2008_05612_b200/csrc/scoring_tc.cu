// scoring_tc.cu — a1-a4 of the hot path on the 5th-generation tensor cores (sm_100a):
//   a1 feature rows built in shared memory from the genotype index bits (genotypes are implicit)
//   a2 E(g,S) = sum_contacts e(h_i,h_j) (Eq. 1, :67-69) as an int8 contraction  E = x(g) . W[S]  (tcgen05.mma kind::i8,
//      accumulators in TMEM, weight tiles fetched by the TMA engine with cp.async.bulk)
//   a3 min / second-min / argmin with strict uniqueness (:81, :552-575) fused on the TMEM read-out
//   a4 one uint16 phenotype (and optional int16 gap) per genotype; the energy matrix never reaches HBM.
//
// Prefix folding.  With e(0,0)=a, lin=b-a, quad=c-2b+a:
//   E(g,S) - a*NBP = lin * sum_k c_k(S) h_k + quad * sum_{contacts} h_i h_j.
// A launch batch shares the genotype bits >= FB ("prefix"); only the low FB bits vary.  For one prefix every term with a
// fixed monomer folds into the weights: a constant bias(S), and w_i(S) = lin*c_i(S) + quad*#(H partners of i in the
// prefix).  The contraction then has K' = 2 + FB + pairs(FB) <= 128 columns instead of N + P (325 for 6x6), and the
// per-prefix weight image W' [D x 128 B] is rebuilt by a small kernel (build_image_kernel) before each batch.
//
// Tiling.  A CTA processes a "supertile" of MT*128 = 512 consecutive genotypes: four 128-row A tiles stay in shared
// memory while every 128-structure weight tile streams through a 6-stage ring once and is used by four MMAs
// (M=128, N=128, K=32 x k_steps), one per A tile, into four TMEM accumulators (4 x 128 columns = all 512).  Sixteen
// epilogue warps drain them: warp group m (four warps, one per TMEM lane quarter; thread = genotype row) owns
// accumulator m, so every SM sub-partition has four warps whose TMEM loads and min/max work overlap, and the drain loop
// is one small rolled body that stays in the instruction cache (the first version unrolled 16 copies of it, 100 KB of
// SASS, and spent its time in instruction-fetch stalls: profiles/r1_scoring_v1_ncu.md).
#include <vector>

#include "device_common.cuh"

#include "tc_common.cuh"

namespace tc {

struct Args {
    const int8_t* img;        // [n_batches][n_tiles][TILE_BYTES]
    const uint16_t* class_of;
    uint16_t* pheno;          // indexed by g - out_base
    int16_t* gap;             // nullable
    uint64_t g_first;         // first genotype of this launch (multiple of SUPER)
    uint64_t g_end;           // one past the last genotype to store
    uint64_t out_base;        // genotype that maps to pheno[0]
    uint32_t n_items;         // supertiles in this launch
    uint32_t n_tiles;         // ceil(D / TN)
    uint32_t D;
    int fb;                   // folded (varying) low bits
    int k_steps;              // 32-byte K steps actually used (1..4)
    int threshold;
    int4* hrec;               // map mode (gp_enumerate_map): per genotype (k1, k2) over all columns and the snapshot of
                              // (k1, k2) after the first n_snap weight tiles; indexed like pheno; pheno/gap unused
    uint32_t n_snap;
};

// ---- a1: feature rows -----------------------------------------------------------------------------------------------
// Row r of A tile m holds genotype g0 + m*128 + r: byte c = val[c] * h_{i[c]} * h_{j[c]} on its low `fb` bits.
// `pk` = the column table in shared memory, one word per column: the mask (1 << i) | (1 << j); the feature is 1 iff the
// row word has all mask bits set (3 ALU operations per byte instead of 10; the build is ALU-bound: clock64 timeline in
// profiles/r1_scoring_v4_ncu.md).  Column 0 (the x64 bias column) is the only one whose value is not 1.
template <int RB>
__device__ __forceinline__ void build_a_row(uint8_t* a_tile, uint32_t r, uint32_t glow, const uint32_t* pk) {
    const uint32_t w = glow | 0x80000000u;  // bit 31: the constant-1 "monomer" used by the bias columns
    const uint32_t sw = RB == 128 ? (r & 7u) : ((r >> 1) & 3u);
#pragma unroll 1
    for (uint32_t c16 = 0; c16 < RB / 16; c16++) {
        uint32_t q[4];
#pragma unroll
        for (int wd = 0; wd < 4; wd++) {
            const uint4 t4 = *reinterpret_cast<const uint4*>(pk + c16 * 16 + wd * 4);
            const uint32_t t[4] = {t4.x, t4.y, t4.z, t4.w};
            uint32_t x = 0;
#pragma unroll
            for (int b = 0; b < 4; b++) x |= ((w & t[b]) == t[b] ? 1u : 0u) << (8 * b);
            q[wd] = x;
        }
        if (c16 == 0) q[0] = (q[0] & ~0xFFu) | 64u;
        *reinterpret_cast<uint4*>(a_tile + r * RB + ((c16 ^ sw) << 4)) = make_uint4(q[0], q[1], q[2], q[3]);
    }
}

// ---- a3: exact min / second-min / argmin on packed keys -------------------------------------------------------------
// key = E * 2^17 + column.  (k1, k2) = the two smallest keys seen.  Keys are distinct, so k2 >> 17 is the second-smallest
// energy counted with multiplicity (R6), and a tie at the minimum shows as equal energies in k1 and k2.
// Filter: eight columns are rescanned only if their minimum is strictly below the current second-smallest energy;
// an energy equal to it cannot change (k1, k2) because columns arrive in increasing order.

// Packed int16 pairs (two columns per register, tcgen05.ld .pack::16b): per-halfword signed min (VIMNMX.S16X2-class
// DPX instructions).  One test on the minimum of 64 columns (22 ALU ops); only when some energy is strictly below the
// running second-smallest are the eight 8-column groups tested and the hit ones rescanned.  "some halfword of x is
// below e2" <=> min(x, E2) != E2 with E2 = (e2, e2).
__device__ __forceinline__ uint32_t pmin3(uint32_t a, uint32_t b, uint32_t c) { return __vimin3_s16x2(a, b, c); }
__device__ __forceinline__ uint32_t pmin(uint32_t a, uint32_t b) { return __vmins2(a, b); }
__device__ __forceinline__ uint32_t pack2(int32_t e) { return ((uint32_t)e & 0xFFFFu) * 0x10001u; }

__device__ __forceinline__ void fold_half_packed(const uint32_t* w, uint32_t col0, int32_t& k1, int32_t& k2, uint32_t& E2) {
    uint32_t g[8];
#pragma unroll
    for (int s = 0; s < 8; s++) g[s] = pmin3(w[4 * s], w[4 * s + 1], pmin(w[4 * s + 2], w[4 * s + 3]));
    const uint32_t all = pmin3(pmin3(g[0], g[1], g[2]), pmin3(g[3], g[4], g[5]), pmin(g[6], g[7]));
    if (pmin(all, E2) != E2) {
#pragma unroll
        for (int s = 0; s < 8; s++) {
            if (pmin(g[s], E2) != E2) {
#pragma unroll
                for (int j = 0; j < 4; j++) {
                    const uint32_t x = w[4 * s + j];
                    const int32_t lo = (int32_t)(int16_t)(x & 0xFFFFu), hi = (int32_t)x >> 16;
                    const int32_t c = (int32_t)(col0 + 8 * s + 2 * j);
                    const int32_t key0 = lo * (1 << KEY_SHIFT) + c, key1 = hi * (1 << KEY_SHIFT) + c + 1;
                    k2 = min(k2, max(k1, key0));
                    k1 = min(k1, key0);
                    k2 = min(k2, max(k1, key1));
                    k1 = min(k1, key1);
                }
                E2 = pack2(k2 >> KEY_SHIFT);
            }
        }
    }
}

struct __align__(16) Barriers {
    uint64_t b_full[NSTAGE], b_empty[NSTAGE];
    uint64_t acc_full[MT], acc_empty[MT];
    uint64_t a_full, a_empty;
    uint32_t tmem_base;
};

// KS = 32-byte K steps per MMA chain (1..4).  One N=128 MMA chain per accumulator; the epilogue reads the whole
// accumulator as packed int16 pairs, releases it at once and folds with two-lane SIMD min.
// RB = bytes per operand row: 64 when the contraction has at most 64 columns (half the weight-tile and feature-row traffic)
template <int KS, int RB>
__global__ void __launch_bounds__(THREADS, 1) scoring_kernel(const Args a, const Cols cols_in) {
    constexpr int TB = TM * RB;                           // bytes of an A tile / a weight tile
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;                                   // MT tiles
    uint8_t* sB = smem + MT * TB;                         // NSTAGE tiles
    Barriers* bar = reinterpret_cast<Barriers*>(sB + NSTAGE * TB);
    uint32_t* pk = reinterpret_cast<uint32_t*>(bar + 1);  // packed column table, ROWB words
    constexpr uint32_t IDESC = idesc_for(TN);

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    // the service warps have the highest warp ids: the sub-partition arbiter favours high ids, and their few instructions
    // per tile are the critical path
    constexpr uint32_t W_ISS = EPI_WARPS, W_PROD = EPI_WARPS + NISS;

    for (uint32_t c = threadIdx.x; c < ROWB; c += THREADS)
        pk[c] = cols_in.val[c] ? ((1u << cols_in.i[c]) | (1u << cols_in.j[c])) : 0xFFFFFFFFu;  // unused column: never all set
    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; s++) { mbar_init(&bar->b_full[s], 1); mbar_init(&bar->b_empty[s], NISS); }
        for (int m = 0; m < MT; m++) { mbar_init(&bar->acc_full[m], 1); mbar_init(&bar->acc_empty[m], 4); }
        mbar_init(&bar->a_full, 32 * EPI_WARPS);
        mbar_init(&bar->a_empty, NISS);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == W_ISS) {  // TMEM: all 512 columns (one CTA per SM)
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&bar->tmem_base)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = bar->tmem_base;

    if (warp == W_PROD) {
        // ===== producer: stream every weight tile of the item's batch image through the ring.  The whole warp runs the
        // loop (uniform control flow); one elected lane issues the copies. =====
        uint32_t it = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x) {
            const uint64_t g0 = a.g_first + (uint64_t)item * SUPER;
            const uint64_t batch = (g0 >> a.fb) - (a.g_first >> a.fb);
            const int8_t* img = a.img + batch * (uint64_t)a.n_tiles * TB;
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                const uint32_t s = it % NSTAGE, ph = (it / NSTAGE) & 1;
                mbar_wait(&bar->b_empty[s], ph ^ 1);
                if (elect_one()) {
                    mbar_expect_tx(&bar->b_full[s], TB);
                    bulk_g2s(sB + s * TB, img + (uint64_t)n * TB, TB, &bar->b_full[s]);
                }
                __syncwarp();
            }
        }
    } else if (warp >= W_ISS) {
        // ===== MMA issuers: NISS warps, issuer h owns accumulators h*MT/NISS ..; warp-uniform loop, one elected lane issues.
        // One issuer's own instruction latencies (wait, fence, elect, two MMAs, commit: 170 clocks per chain and 290 per
        // tile, clock64 trace in profiles/r2_scoring_ncu.md) were longer than the 528 clocks of tensor work per tile. =====
        constexpr int MPI = MT / NISS;                  // accumulators per issuer
        const uint32_t m0 = (warp - W_ISS) * MPI;
        const uint64_t a_desc0 = smem_desc_rb<RB>(smem_u32(sA));
        const uint64_t b_desc0 = smem_desc_rb<RB>(smem_u32(sB));
        uint32_t it = 0, item_no = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x, item_no++) {
            mbar_wait(&bar->a_full, item_no & 1);
            tc_fence_after();
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                const uint32_t s = it % NSTAGE, ph = (it / NSTAGE) & 1;
                mbar_wait(&bar->b_full[s], ph);
                tc_fence_after();
                const uint64_t bd = b_desc0 + (uint64_t)(s * (TB >> 4));
#pragma unroll
                for (int j = 0; j < MPI; j++) {
                    const uint32_t m = m0 + j;
                    mbar_wait(&bar->acc_empty[m], (it & 1) ^ 1);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t d = tmem + m * TN;
                        const uint64_t ad = a_desc0 + (uint64_t)((m * TB) >> 4);
                        mma_i8_c<false>(d, ad, bd, IDESC);
#pragma unroll
                        for (int k = 1; k < KS; k++) mma_i8_c<true>(d, ad + 2 * k, bd + 2 * k, IDESC);
                        tc_commit(&bar->acc_full[m]);
                    }
                    __syncwarp();
                }
                if (elect_one()) tc_commit(&bar->b_empty[s]);
                __syncwarp();
            }
            if (elect_one()) tc_commit(&bar->a_empty);
            __syncwarp();
        }
    } else {
        // ===== feature build + epilogue: 16 warps; warp group m owns A tile m and accumulator m; thread = genotype row =====
        const uint32_t m = warp >> 2;                   // accumulator / A tile of this warp group
        const uint32_t quarter = warp & 3;              // TMEM lanes 32*quarter .. +31 are the ones this warp may read
        const uint32_t r = quarter * 32 + lane;         // row within the 128-row tile
        const uint32_t t_acc = tmem + ((quarter * 32u) << 16) + m * TN;
        const uint32_t lowmask = a.fb >= 32 ? 0xFFFFFFFFu : ((1u << a.fb) - 1u);
        uint32_t it = 0, item_no = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x, item_no++) {
            const uint64_t g = a.g_first + (uint64_t)item * SUPER + m * TM + r;
            mbar_wait(&bar->a_empty, (item_no & 1) ^ 1);
            build_a_row<RB>(sA + m * TB, r, (uint32_t)g & lowmask, pk);
            fence_proxy_async();
            mbar_arrive(&bar->a_full);

            int32_t k1 = INT32_MAX, k2 = INT32_MAX, s1 = INT32_MAX, s2 = INT32_MAX;
            uint32_t E2 = pack2(E_NONE);
#pragma unroll 1
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                if (n == a.n_snap) { s1 = k1; s2 = k2; }
                mbar_wait(&bar->acc_full[m], it & 1);
                tc_fence_after();
                uint32_t w[2 * 32];
                tmem_ld64_pack16(t_acc, w);
                tmem_ld_wait();
                tc_fence_before();  // the accumulator is in registers: hand it back to the MMA warp
                __syncwarp();
                if (lane == 0) mbar_arrive(&bar->acc_empty[m]);
                fold_half_packed(&w[0], n * TN, k1, k2, E2);
                fold_half_packed(&w[32], n * TN + HN, k1, k2, E2);
            }
            if (a.n_snap >= a.n_tiles) { s1 = k1; s2 = k2; }
            if (a.hrec) {
                if (g < a.g_end) a.hrec[g] = make_int4(k1, k2, s1, s2);
            } else if (g < a.g_end && g >= a.out_base) {
                const int32_t e1 = k1 >> KEY_SHIFT, e2v = k2 >> KEY_SHIFT;
                const uint32_t col = (uint32_t)k1 & ((1u << KEY_SHIFT) - 1u);
                const bool single = (e2v >= E_PAD);  // D = 1: the runner-up is a pad structure
                const bool folds = single || (e2v - e1 >= a.threshold);
                a.pheno[g - a.out_base] = folds ? a.class_of[col] : (uint16_t)GP_NULL_PHENO;
                if (a.gap) a.gap[g - a.out_base] = (int16_t)(single ? GP_GAP_NONE : max(e1 - e2v, -32768));
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == W_ISS) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
}

typedef void (*scoring_fn)(const Args, const Cols);
template <int RB>
scoring_fn scoring_for(int ks) {
    switch (ks) {
        case 1: return scoring_kernel<1, RB>;
        case 2: return scoring_kernel<2, RB>;
        case 3: return scoring_kernel<3, RB>;
        default: return scoring_kernel<4, RB>;
    }
}

// ---- per-prefix weight image ----------------------------------------------------------------------------------------
struct Slots {  // column of pair (li, lj) of LOCAL bits li < lj in the folded contraction (0 = not a column), and
    uint8_t pair[MAX_FB * MAX_FB];  // the local bit of every monomer (-1 = the monomer is fixed within an image)
    int8_t loc[64];
};

struct ImgArgs {
    const uint8_t* contacts;   // D * NBP * 2
    const uint16_t* class_of;  // D; 0xFFFF marks a pad column inside the list
    int8_t* img;               // [n_images][n_tiles][TILE_BYTES]
    const uint32_t* units;     // nullable (prefix path): fixed-bit value of image y is gfix_first + y.  Map path: the
                               // unit table; see image_mid()
    uint64_t gfix_first;
    uint64_t unit_first;
    int paired, mid;           // map path: images 2j, 2j+1 = (m, rev m) of unit unit_first + j, else image j = m
    int gfix_shift;            // genotype with the fixed bits of image y in place = value << gfix_shift
    uint32_t D, n_tiles;
    int NBP, lin, quad;
};

// Map path: middle-bit value of image y of a launch group
__device__ __forceinline__ uint32_t image_mid(const uint32_t* units, uint64_t unit_first, int paired, int mid, uint32_t y) {
    const uint32_t m = units[unit_first + (paired ? (y >> 1) : y)];
    return (paired && (y & 1u)) ? (mid ? (__brev(m) >> (32 - mid)) : 0u) : m;
}

// One block = one 128-structure tile of IMG_PER_BLOCK consecutive images; thread = structure = one weight row.
// Only the first 2 + fb columns of a row depend on the image (the fixed monomers' letters G); the pair columns do not:
//   bias          = lin * sum over fixed monomers j of h_j * deg(j)  +  quad * #(contacts between two fixed H monomers)
//   column 2 + l  = lin * deg(l)  +  quad * popc(G & F_l),   F_l = the fixed monomers in contact with free monomer l
// (deg = contacts of the monomer in this structure).  The block prepares, once, the image-independent part of the tile
// in shared memory (already in the swizzled layout the MMA reads) and per thread deg, F_l, the degree bit-planes of the
// fixed monomers and the list of fixed-fixed contacts; per image a thread then evaluates 2 + fb bytes with popc,
// overwrites them in its row and its warp copies its 32 rows out, coalesced.  No barrier after the setup.
constexpr int IMG_PER_BLOCK = 32;

template <int RB>
__global__ void build_image_kernel(const ImgArgs a, const Slots slots_in, uint32_t n_images, int fb);

template <int RB>
size_t build_image_smem(int fb) {
    return (size_t)TM * RB + TN * 64 + (size_t)fb * TN * 8 + (((size_t)fb * TN + 15) & ~(size_t)15) + 32 * TN * 2 + sizeof(Slots) + 16;
}

template <int RB>
__global__ void __launch_bounds__(TN) build_image_kernel(const ImgArgs a, const Slots slots_in, uint32_t n_images, int fb) {
    constexpr int TB = TM * RB;
    extern __shared__ __align__(16) unsigned char img_smem[];
    int8_t* tile = reinterpret_cast<int8_t*>(img_smem);
    uint8_t* s_con = img_smem + TB;                          // contacts of the tile's structures: NBP <= 32 pairs each
    uint64_t* maskF = reinterpret_cast<uint64_t*>(s_con + TN * 64);    // [fb][TN]
    uint8_t* degL = reinterpret_cast<uint8_t*>(maskF + (size_t)fb * TN);   // [fb][TN]
    uint16_t* ffl = reinterpret_cast<uint16_t*>(degL + (((size_t)fb * TN + 15) & ~(size_t)15));  // [32][TN]: i | j << 8
    Slots* slots = reinterpret_cast<Slots*>(ffl + 32 * TN);
    const uint32_t r = threadIdx.x, n = blockIdx.x, lane = r & 31u;
    const uint32_t d = n * TN + r;
    const int row = a.NBP * 2;
    {
        const uint32_t first = n * TN, cnt = (a.D - first < (uint32_t)TN ? a.D - first : (uint32_t)TN) * row;
        const uint8_t* src = a.contacts + (size_t)first * row;
        for (uint32_t i = threadIdx.x; i < cnt; i += TN) s_con[i] = src[i];
        for (uint32_t i = threadIdx.x; i < sizeof(Slots); i += TN)
            reinterpret_cast<uint8_t*>(slots)[i] = reinterpret_cast<const uint8_t*>(&slots_in)[i];
        for (uint32_t i = threadIdx.x; i < TB / 16; i += TN) reinterpret_cast<uint4*>(tile)[i] = make_uint4(0, 0, 0, 0);
        for (int l = 0; l < fb; l++) { maskF[l * TN + r] = 0; degL[l * TN + r] = 0; }
    }
    __syncthreads();
    const bool real = d < a.D && a.class_of[d] != GP_NULL_PHENO;
    uint64_t dm0 = 0, dm1 = 0, dm2 = 0;     // bit-planes of deg(j) over the fixed monomers j (bit j - gfix_shift)
    int nff = 0;
    if (real) {
        const uint8_t* c = s_con + r * row;
        for (int k = 0; k < a.NBP; k++) {
            const int i = c[2 * k], j = c[2 * k + 1];  // i < j
            const int li = slots->loc[i], lj = slots->loc[j];
            const uint64_t bi = 1ULL << ((i - a.gfix_shift) & 63), bj = 1ULL << ((j - a.gfix_shift) & 63);
            if (li >= 0) degL[li * TN + r]++;
            else { const uint64_t c0 = dm0 & bi; dm0 ^= bi; const uint64_t c1 = dm1 & c0; dm1 ^= c0; dm2 ^= c1; }
            if (lj >= 0) degL[lj * TN + r]++;
            else { const uint64_t c0 = dm0 & bj; dm0 ^= bj; const uint64_t c1 = dm1 & c0; dm1 ^= c0; dm2 ^= c1; }
            if (li >= 0 && lj >= 0) tile[swz_rb<RB>(r, slots->pair[li * MAX_FB + lj])] = (int8_t)a.quad;
            else if (li >= 0) maskF[li * TN + r] |= bj;
            else if (lj >= 0) maskF[lj * TN + r] |= bi;
            else ffl[(nff++) * TN + r] = (uint16_t)(((i - a.gfix_shift) & 63) | (((j - a.gfix_shift) & 63) << 8));
        }
    } else {                                         // pad structure: energy E_PAD for every genotype
        tile[swz_rb<RB>(r, 0)] = 127;
        tile[swz_rb<RB>(r, 1)] = 63;
    }
    const int ncol = 2 + fb, nw = (ncol + 3) >> 2;   // image-dependent columns / the 32-bit words that hold them
    // the last of those words may also hold pair columns: keep its image-independent bytes
    const uint32_t last_base = *reinterpret_cast<const uint32_t*>(tile + swz_rb<RB>(r, 4 * (nw - 1)));
    const uint32_t* trow = reinterpret_cast<const uint32_t*>(tile);
    for (uint32_t y = blockIdx.y * IMG_PER_BLOCK; y < n_images && y < (blockIdx.y + 1) * IMG_PER_BLOCK; y++) {
        const uint64_t G = a.units ? (uint64_t)image_mid(a.units, a.unit_first, a.paired, a.mid, y) : a.gfix_first + y;
        if (real) {
            int bias = a.lin * (__popcll(G & dm0) + 2 * __popcll(G & dm1) + 4 * __popcll(G & dm2));
            for (int k = 0; k < nff; k++) {
                const uint32_t e = ffl[k * TN + r];
                bias += a.quad * (int)((G >> (e & 255u)) & (G >> (e >> 8)) & 1ULL);
            }
#pragma unroll
            for (int w = 0; w < (2 + MAX_FB + 3) / 4; w++) {
                if (w >= nw) break;
                uint32_t x = w == nw - 1 ? last_base : 0u;
#pragma unroll
                for (int b = 0; b < 4; b++) {
                    const int col = 4 * w + b;
                    if (col >= ncol) break;
                    int v;
                    if (col == 0) v = bias >> 6;          // x 64
                    else if (col == 1) v = bias & 63;     // x 1
                    else v = a.lin * (int)degL[(col - 2) * TN + r] + a.quad * __popcll(G & maskF[(col - 2) * TN + r]);
                    x = (x & ~(0xFFu << (8 * b))) | (((uint32_t)v & 0xFFu) << (8 * b));
                }
                *reinterpret_cast<uint32_t*>(tile + swz_rb<RB>(r, 4 * w)) = x;
            }
        }
        __syncwarp();
        // rows 32 * warp .. + 31 are contiguous in the tile and in the image
        uint4* dst = reinterpret_cast<uint4*>(a.img + ((uint64_t)y * a.n_tiles + n) * TB) + (r & ~31u) * (RB / 16);
        const uint4* srcw = reinterpret_cast<const uint4*>(trow) + (r & ~31u) * (RB / 16);
#pragma unroll
        for (uint32_t i = 0; i < RB / 16; i++) dst[i * 32 + lane] = srcw[i * 32 + lane];
        __syncwarp();
    }
}

// Columns of the folded contraction for a set of free monomers mon[0..fb-1] (increasing): 2 bias columns, fb monomer
// columns, one column per pair of free monomers that can touch (j - i odd and >= 3).  Returns the column count.
static int make_columns(const int* mon, int fb, int N, Cols& cols, Slots& slots) {
    memset(&slots, 0, sizeof(slots));
    for (int i = 0; i < 64; i++) slots.loc[i] = -1;
    for (int l = 0; l < fb; l++) slots.loc[mon[l]] = (int8_t)l;
    for (int c = 0; c < ROWB; c++) { cols.i[c] = 31; cols.j[c] = 31; cols.val[c] = 0; }
    cols.val[0] = 64;
    cols.val[1] = 1;
    int nc = 2;
    for (int l = 0; l < fb; l++, nc++) { cols.i[nc] = cols.j[nc] = (uint8_t)l; cols.val[nc] = 1; }
    for (int li = 0; li < fb; li++)
        for (int lj = li + 1; lj < fb; lj++) {
            const int dist = mon[lj] - mon[li];
            if (dist < 3 || (dist & 1) == 0) continue;
            if (nc < ROWB) {
                cols.i[nc] = (uint8_t)li; cols.j[nc] = (uint8_t)lj; cols.val[nc] = 1;
                slots.pair[li * MAX_FB + lj] = (uint8_t)nc;
            }
            nc++;
        }
    (void)N;
    return nc;
}

// ---- map mode: merge the two half-lists of a genotype and its reversal -------------------------
struct CombArgs {
    const int4* hrec;           // [n_images][2^fb]
    const uint32_t* units;      // unit table of the map
    const uint16_t* class_sym;
    uint16_t* pheno;
    int16_t* gap;               // nullable
    uint64_t unit_first;
    uint64_t compact_base;      // compact layout: output index of this group's image 0, local genotype 0
    uint32_t n_images;
    int paired, mid;            // the image holding the reversed genotypes of image y is y ^ 1 (paired) or y itself
    int fb, k, N, threshold, compact;
};

__global__ void __launch_bounds__(256) combine_kernel(const CombArgs a) {
    const uint64_t total = (uint64_t)a.n_images << a.fb;
    const uint32_t tmask = (1u << a.fb) - 1u, kmask = (1u << a.k) - 1u;
    for (uint64_t idx = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t y = (uint32_t)(idx >> a.fb), t = (uint32_t)idx & tmask;
        const uint32_t yp = a.paired ? (y ^ 1u) : y;
        const uint32_t tr = __brev(t) >> (32 - a.fb);
        const int4 A = a.hrec[idx];
        const int4 B = a.hrec[((uint64_t)yp << a.fb) + tr];
        // own list: all class representatives; reversed genotype's list: the same structures read backwards, i.e. the
        // other member of every two-member class (self-reverse classes are in the own list only)
        const int32_t a1 = A.x >> KEY_SHIFT, a2 = A.y >> KEY_SHIFT, b1 = B.z >> KEY_SHIFT, b2 = B.w >> KEY_SHIFT;
        const bool own = a1 <= b1;
        const int32_t m1 = own ? a1 : b1;
        const int32_t m2 = own ? min(a2, b1) : min(b2, a1);
        const uint32_t col = (uint32_t)(own ? A.x : B.z) & ((1u << KEY_SHIFT) - 1u);
        const bool single = (m2 >= E_PAD);
        const bool folds = single || (m2 - m1 >= a.threshold);
        const uint64_t g = a.compact ? a.compact_base + idx
                                     : ((uint64_t)(t >> a.k) << (a.N - a.k)) |
                                           ((uint64_t)image_mid(a.units, a.unit_first, a.paired, a.mid, y) << a.k) | (t & kmask);
        a.pheno[g] = folds ? a.class_sym[col] : (uint16_t)GP_NULL_PHENO;
        if (a.gap) a.gap[g] = (int16_t)(single ? GP_GAP_NONE : max(m1 - m2, -32768));
    }
}

// =====================================================================================================================
// Explicit sequences on the tensor cores (the paper's sampling runs, Table 3).
// Random sequences share no prefix, so the contraction keeps all K = 2 + N + P columns (two constant columns that give
// pad structures the energy E_PAD, N monomer columns with weight lin*c_i(S), P pair columns with weight quad):
// 327 columns for 6x6 = three 128-byte column blocks, eleven K steps per chain.  The weight image is built once per
// (lattice, energies) and cached in the handle.  Chains are long (11 x 64 clk), so two genotype tiles with
// double-buffered accumulators (2 x 2 x 128 TMEM columns) keep the tensor pipe busy.
constexpr int SQ_KB = 3;                       // 128-byte column blocks per operand row
constexpr int SQ_MT = 2;                       // sequence tiles per CTA
constexpr int SQ_ROWS = SQ_MT * TM;            // 256 sequences per item
constexpr int SQ_STAGES = 2;
constexpr int SQ_TILE = SQ_KB * TILE_BYTES;    // 48 KB: one operand tile, all column blocks
constexpr int SQ_EPI_WARPS = 4 * SQ_MT;
constexpr int SQ_THREADS = 32 * (2 + SQ_EPI_WARPS);
constexpr int SQ_MAXCOL = SQ_KB * ROWB;        // 384

struct SqCols {  // column c of the full contraction: feature = val * h_i * h_j; i = j for monomers; bit 63 is always 1
    uint8_t i[SQ_MAXCOL], j[SQ_MAXCOL];
};

struct SqImgArgs {
    const uint8_t* contacts;   // D * NBP * 2
    const uint16_t* pairidx;   // D * NBP: pair-feature index of each contact
    int8_t* img;               // [n_tiles][SQ_KB][TILE_BYTES]
    uint32_t D;
    int N, NBP, lin, quad;
};

// One block = one 128-structure tile; thread = structure; the three column blocks are built one after the other.
__global__ void __launch_bounds__(TN) build_full_image_kernel(const SqImgArgs a) {
    __shared__ __align__(16) int8_t tile[TILE_BYTES];
    const uint32_t r = threadIdx.x, n = blockIdx.x;
    const uint32_t d = n * TN + r;
    for (int kb = 0; kb < SQ_KB; kb++) {
        __syncthreads();
        for (uint32_t i = threadIdx.x; i < TILE_BYTES / 16; i += TN) reinterpret_cast<uint4*>(tile)[i] = make_uint4(0, 0, 0, 0);
        __syncthreads();
        const int c0 = kb * ROWB;
        if (d < a.D) {
            const uint8_t* c = a.contacts + (size_t)d * a.NBP * 2;
            const uint16_t* px = a.pairidx + (size_t)d * a.NBP;
            for (int k = 0; k < a.NBP; k++) {
                const int ci = 2 + c[2 * k] - c0, cj = 2 + c[2 * k + 1] - c0, cp = 2 + a.N + px[k] - c0;
                if (ci >= 0 && ci < ROWB) tile[swz(r, ci)] += (int8_t)a.lin;
                if (cj >= 0 && cj < ROWB) tile[swz(r, cj)] += (int8_t)a.lin;
                if (cp >= 0 && cp < ROWB) tile[swz(r, cp)] = (int8_t)a.quad;
            }
        } else if (kb == 0) {  // pad structure: energy E_PAD for every sequence
            tile[swz(r, 0)] = 127;
            tile[swz(r, 1)] = 63;
        }
        __syncthreads();
        uint4* dst = reinterpret_cast<uint4*>(a.img + ((uint64_t)n * SQ_KB + kb) * TILE_BYTES);
        for (uint32_t i = threadIdx.x; i < TILE_BYTES / 16; i += TN) dst[i] = reinterpret_cast<const uint4*>(tile)[i];
    }
}

struct SqArgs {
    const int8_t* img;        // [n_tiles][SQ_KB][TILE_BYTES]
    const uint16_t* class_of;
    const uint8_t* seqs;      // count x N letters (0 / 1); NULL: letters drawn from the seeded stream (seed, first)
    uint64_t seed, first;
    uint16_t* pheno;
    int16_t* gap;             // nullable
    uint64_t count;
    uint32_t n_items, n_tiles;
    int N, ksteps, threshold;
};

struct __align__(8) SqBarriers {
    uint64_t b_full[SQ_STAGES], b_empty[SQ_STAGES];
    uint64_t acc_full[SQ_MT][2], acc_empty[SQ_MT][2];
    uint64_t a_full, a_empty;
    uint32_t tmem_base;
};

__global__ void __launch_bounds__(SQ_THREADS, 1) sequence_kernel(const SqArgs a, const SqCols cols_in) {
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
    uint8_t* sA = smem;                                    // SQ_MT tiles x SQ_KB blocks
    uint8_t* sB = smem + SQ_MT * SQ_TILE;                  // SQ_STAGES tiles x SQ_KB blocks
    SqBarriers* bar = reinterpret_cast<SqBarriers*>(sB + SQ_STAGES * SQ_TILE);
    SqCols* cols = reinterpret_cast<SqCols*>(bar + 1);
    constexpr uint32_t IDESC = idesc_for(TN);

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    for (uint32_t i = threadIdx.x; i < sizeof(SqCols); i += SQ_THREADS)
        reinterpret_cast<uint8_t*>(cols)[i] = reinterpret_cast<const uint8_t*>(&cols_in)[i];
    if (threadIdx.x == 0) {
        for (int s = 0; s < SQ_STAGES; s++) { mbar_init(&bar->b_full[s], 1); mbar_init(&bar->b_empty[s], 1); }
        for (int m = 0; m < SQ_MT; m++)
            for (int h = 0; h < 2; h++) { mbar_init(&bar->acc_full[m][h], 1); mbar_init(&bar->acc_empty[m][h], 4); }
        mbar_init(&bar->a_full, 32 * SQ_EPI_WARPS);
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
        // ===== producer: whole 48 KB weight tiles =====
        uint32_t it = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x) {
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                const uint32_t s = it % SQ_STAGES, ph = (it / SQ_STAGES) & 1;
                mbar_wait(&bar->b_empty[s], ph ^ 1);
                if (elect_one()) {
                    mbar_expect_tx(&bar->b_full[s], SQ_TILE);
                    bulk_g2s(sB + s * SQ_TILE, a.img + (uint64_t)n * SQ_TILE, SQ_TILE, &bar->b_full[s]);
                }
                __syncwarp();
            }
        }
    } else if (warp == 1) {
        // ===== MMA issuer: chains of a.ksteps K steps over the column blocks, accumulators double-buffered =====
        const uint64_t a_desc0 = smem_desc(smem_u32(sA));
        const uint64_t b_desc0 = smem_desc(smem_u32(sB));
        uint32_t it = 0, item_no = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x, item_no++) {
            mbar_wait(&bar->a_full, item_no & 1);
            tc_fence_after();
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                const uint32_t s = it % SQ_STAGES, ph = (it / SQ_STAGES) & 1;
                const uint32_t buf = it & 1;
                mbar_wait(&bar->b_full[s], ph);
                tc_fence_after();
                const uint64_t bd = b_desc0 + (uint64_t)(s * (SQ_TILE >> 4));
#pragma unroll
                for (int m = 0; m < SQ_MT; m++) {
                    mbar_wait(&bar->acc_empty[m][buf], ((it >> 1) & 1) ^ 1);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t d = tmem + (m * 2 + buf) * TN;
                        const uint64_t ad = a_desc0 + (uint64_t)((m * SQ_TILE) >> 4);
                        for (int ks = 0; ks < a.ksteps; ks++) {
                            const uint64_t off = (uint64_t)(((ks >> 2) * TILE_BYTES + (ks & 3) * 32) >> 4);
                            mma_i8(d, ad + off, bd + off, IDESC, ks > 0);
                        }
                        tc_commit(&bar->acc_full[m][buf]);
                    }
                    __syncwarp();
                }
                if (elect_one()) tc_commit(&bar->b_empty[s]);
                __syncwarp();
            }
            if (elect_one()) tc_commit(&bar->a_empty);
            __syncwarp();
        }
    } else {
        // ===== feature rows + epilogue: warp group m owns sequence tile m; thread = sequence =====
        const uint32_t m = (warp - 2) >> 2;
        const uint32_t quarter = warp & 3;
        const uint32_t r = quarter * 32 + lane;
        const uint32_t t_lane = tmem + ((quarter * 32u) << 16) + m * 2 * TN;
        uint32_t it = 0, item_no = 0;
        for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x, item_no++) {
            const uint64_t q = (uint64_t)item * SQ_ROWS + m * TM + r;
            unsigned long long h = 1ULL << 63;  // bit 63: the constant-1 feature; bit 62 stays 0 for unused columns
            if (q < a.count) {
                if (a.seqs)
                    for (int i = 0; i < a.N; i++) h |= (unsigned long long)(a.seqs[q * a.N + i] != 0) << i;  // a letter outside {0, 1} is the last letter, H (R19)
                else
                    for (int i = 0; i < a.N; i++) h |= (unsigned long long)gp_letter(a.seed, a.first + q, i, 2u) << i;
            }
            mbar_wait(&bar->a_empty, (item_no & 1) ^ 1);
#pragma unroll 1
            for (uint32_t c16 = 0; c16 < SQ_MAXCOL / 16; c16++) {
                uint32_t w4[4];
#pragma unroll
                for (int wd = 0; wd < 4; wd++) {
                    uint32_t x = 0;
#pragma unroll
                    for (int b = 0; b < 4; b++) {
                        const uint32_t c = c16 * 16 + wd * 4 + b;
                        const uint32_t bit = (uint32_t)((h >> cols->i[c]) & (h >> cols->j[c]) & 1ULL);
                        x |= (bit * (c == 0 ? 64u : 1u)) << (8 * b);
                    }
                    w4[wd] = x;
                }
                uint8_t* blk = sA + (m * SQ_KB + (c16 >> 3)) * TILE_BYTES;
                *reinterpret_cast<uint4*>(blk + r * ROWB + (((c16 & 7) ^ (r & 7u)) << 4)) = make_uint4(w4[0], w4[1], w4[2], w4[3]);
            }
            fence_proxy_async();
            mbar_arrive(&bar->a_full);

            int32_t k1 = INT32_MAX, k2 = INT32_MAX;
            uint32_t E2 = pack2(E_NONE);
#pragma unroll 1
            for (uint32_t n = 0; n < a.n_tiles; n++, it++) {
                const uint32_t buf = it & 1;
                mbar_wait(&bar->acc_full[m][buf], (it >> 1) & 1);
                tc_fence_after();
                uint32_t w[2 * 32];
                tmem_ld64_pack16(t_lane + buf * TN, w);
                tmem_ld_wait();
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&bar->acc_empty[m][buf]);
                fold_half_packed(&w[0], n * TN, k1, k2, E2);
                fold_half_packed(&w[32], n * TN + HN, k1, k2, E2);
            }
            if (q < a.count) {
                const int32_t e1 = k1 >> KEY_SHIFT, e2v = k2 >> KEY_SHIFT;
                const uint32_t col = (uint32_t)k1 & ((1u << KEY_SHIFT) - 1u);
                const bool single = (e2v >= E_PAD);
                const bool folds = single || (e2v - e1 >= a.threshold);
                a.pheno[q] = folds ? a.class_of[col] : (uint16_t)GP_NULL_PHENO;
                if (a.gap) a.gap[q] = (int16_t)(single ? GP_GAP_NONE : max(e1 - e2v, -32768));
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
}


// ---- MMA-only probe: the measured int8 tensor peak this kernel family can be held against -----------------------------
// One CTA per SM issues the scoring kernel's own instruction stream — chains of KS tcgen05.mma kind::i8 M128 x N128 x
// K32 into four TMEM accumulators, operands in the same swizzled shared-memory layout — with no TMA traffic, no TMEM
// read-out and no epilogue: one commit per 64 MMAs, at most two commit groups in flight.
template <int KS, int RB>
__global__ void __launch_bounds__(128, 1) mma_probe_kernel(uint32_t groups, unsigned long long* cycles) {
    constexpr int TB = TM * RB;
    extern __shared__ unsigned char smem_dyn[];
    unsigned char* smem = reinterpret_cast<unsigned char*>(((uintptr_t)smem_dyn + 1023) & ~(uintptr_t)1023);
    __shared__ __align__(8) uint64_t done[2];
    __shared__ uint32_t tmem_base;
    for (uint32_t i = threadIdx.x; i < 2 * TB / 4; i += blockDim.x)  // pseudo-random operand bytes (zeros would flatter the clocks)
        reinterpret_cast<uint32_t*>(smem)[i] = (uint32_t)gp_mix64(i + 977u * blockIdx.x);
    if (threadIdx.x == 0) {
        mbar_init(&done[0], 1);
        mbar_init(&done[1], 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    const uint32_t warp = threadIdx.x >> 5;
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(smem_u32(&tmem_base)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = tmem_base;
    if (warp == 0) {
        constexpr uint32_t IDESC = idesc_for(TN);
        const uint64_t ad = smem_desc_rb<RB>(smem_u32(smem)), bd = smem_desc_rb<RB>(smem_u32(smem + TB));
        const long long t0 = clock64();
        for (uint32_t g = 0; g < groups; g++) {
            if (g >= 2) mbar_wait(&done[g & 1], ((g >> 1) - 1) & 1);
            if (elect_one()) {
#pragma unroll 4
                for (int c = 0; c < 64 / KS; c++) {
                    const uint32_t d = tmem + (c & 3) * TN;
                    mma_i8_c<false>(d, ad, bd, IDESC);
#pragma unroll
                    for (int k = 1; k < KS; k++) mma_i8_c<true>(d, ad + 2 * k, bd + 2 * k, IDESC);
                }
                tc_commit(&done[g & 1]);
            }
            __syncwarp();
        }
        for (uint32_t g = groups > 2 ? groups - 2 : 0; g < groups; g++) mbar_wait(&done[g & 1], (g >> 1) & 1);
        const long long t1 = clock64();
        if (threadIdx.x == 0) cycles[blockIdx.x] = (unsigned long long)(t1 - t0);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) {
        tc_fence_after();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tmem) : "memory");
    }
}

}  // namespace tc

// ---- tuning (include/gpmap.h: gp_tuning) ------------------------------------------------------------------------------
extern "C" gp_status gp_tuning_get(const gp_structures_t* s, gp_tuning* out) {
    if (!s || !out) return GP_INVALID_ARG;
    *out = s->tuning;
    return GP_OK;
}

extern "C" gp_status gp_tuning_set(gp_structures_t* s, const gp_tuning* t) {
    if (!s || !t) return GP_INVALID_ARG;
    if (t->fold_bits < 9 || t->fold_bits > tc::MAX_FB || t->sym_bits < 5 || 2 * t->sym_bits > tc::MAX_FB) return GP_INVALID_ARG;
    if ((t->narrow_rows | 1) != 1 || t->seq_tensor < 0 || t->seq_tensor > 2) return GP_INVALID_ARG;
    const bool rebuild = t->sym_bits != s->tuning.sym_bits;
    const gp_tuning old = s->tuning;
    s->tuning = *t;
    if (rebuild) {
        gp_status st = gp_build_map_units(s);
        if (st != GP_OK) { s->tuning = old; gp_build_map_units(s); return st; }
    }
    return GP_OK;
}

namespace {

// Geometry of one scoring launch family: contraction columns, K steps, operand rows, kernel and its shared memory
struct Plan {
    tc::Cols cols;
    tc::Slots slots;
    int nc = 0, k_steps = 0;
    bool narrow = false;
    uint32_t n_tiles = 0;
    size_t tile_bytes = 0, img_bytes = 0, smem = 0;
    tc::scoring_fn kernel = nullptr;
    int sms = 0, threads = 0;
};

gp_status make_plan(const gp_structures_s* s, const int* mon, int fb, uint32_t n_columns, Plan& p) {
    using namespace tc;
    p.nc = make_columns(mon, fb, s->N, p.cols, p.slots);
    if (p.nc > ROWB || s->NBP > 32) return GP_UNSUPPORTED_LATTICE;  // build_image_kernel stages 32 contacts per structure
    p.k_steps = (p.nc + 31) / 32;
    p.n_tiles = (n_columns + TN - 1) / TN;
    p.narrow = p.nc <= 64 && s->tuning.narrow_rows;  // at most 64 columns: 64-byte operand rows
    p.tile_bytes = (size_t)TM * (p.narrow ? 64 : 128);
    p.img_bytes = (size_t)p.n_tiles * p.tile_bytes;
    p.smem = (size_t)(MT + NSTAGE) * p.tile_bytes + sizeof(Barriers) + ROWB * sizeof(uint32_t) + 1024 + 64;
    p.threads = THREADS;
    p.kernel = p.narrow ? scoring_for<64>(p.k_steps) : scoring_for<128>(p.k_steps);
    int dev = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&p.sms, cudaDevAttrMultiProcessorCount, dev));
    GP_CUDA(cudaFuncSetAttribute(p.kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem));
    return GP_OK;
}

}  // namespace

// Weight images of launch group g + 1 are built on a side stream while the scoring kernel of group g runs on the caller's
// stream (two image buffers); events tie the side stream in, so that to the caller everything is ordered on `st`.
struct ImagePipeline {
    cudaStream_t side = nullptr, post = nullptr;   // post (map path): the combine of group g runs beside the scoring of g + 1
    cudaStream_t alt = nullptr;   // map path: odd scoring launches go here, so the blocks of launch g + 1 take over the SMs
                                  // one by one as the blocks of launch g retire (no idle tail at the end of a launch)
    cudaEvent_t built[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr}, posted[2] = {nullptr, nullptr}, start = nullptr;
    gp_status open(cudaStream_t st, bool with_post = false) {   // call after the buffers were allocated on st
        GP_CUDA(cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking));
        GP_CUDA(cudaEventCreateWithFlags(&start, cudaEventDisableTiming));
        for (int b = 0; b < 2; b++) {
            GP_CUDA(cudaEventCreateWithFlags(&built[b], cudaEventDisableTiming));
            GP_CUDA(cudaEventCreateWithFlags(&freed[b], cudaEventDisableTiming));
        }
        GP_CUDA(cudaEventRecord(start, st));
        GP_CUDA(cudaStreamWaitEvent(side, start, 0));
        if (with_post) {
            GP_CUDA(cudaStreamCreateWithFlags(&post, cudaStreamNonBlocking));
            GP_CUDA(cudaStreamCreateWithFlags(&alt, cudaStreamNonBlocking));
            for (int b = 0; b < 2; b++) GP_CUDA(cudaEventCreateWithFlags(&posted[b], cudaEventDisableTiming));
            GP_CUDA(cudaStreamWaitEvent(post, start, 0));
            GP_CUDA(cudaStreamWaitEvent(alt, start, 0));
        }
        return GP_OK;
    }
    cudaStream_t scoring_stream(uint64_t g, cudaStream_t st) { return alt && (g & 1) ? alt : st; }
    // record buffer g & 1 may be overwritten by scoring launch g once the combine of group g - 2 has read it
    void before_scoring(uint64_t g, cudaStream_t st) { if (post && g >= 2) cudaStreamWaitEvent(st, posted[g & 1], 0); }
    // the stream the combine of group g goes to (after after_scoring(g)): it waits for that scoring launch
    cudaStream_t post_stream(uint64_t g, cudaStream_t st) {
        if (!post) return st;
        cudaStreamWaitEvent(post, freed[g & 1], 0);
        return post;
    }
    void after_post(uint64_t g) { if (post) cudaEventRecord(posted[g & 1], post); }
    // the caller's stream continues only after every combine (n_groups launched)
    void join_post(uint64_t n_groups, cudaStream_t st) {
        if (!post) return;
        for (uint64_t g = n_groups >= 2 ? n_groups - 2 : 0; g < n_groups; g++) cudaStreamWaitEvent(st, posted[g & 1], 0);
    }
    // side stream may overwrite buffer b once the scoring launch that read it (two groups ago) is done
    void before_build(uint64_t g) { if (g >= 2) cudaStreamWaitEvent(side, freed[g & 1], 0); }
    void after_build(uint64_t g, cudaStream_t st) { cudaEventRecord(built[g & 1], side); cudaStreamWaitEvent(st, built[g & 1], 0); }
    void after_scoring(uint64_t g, cudaStream_t st) { cudaEventRecord(freed[g & 1], st); }
    ~ImagePipeline() {   // destroying a stream / event with work pending is deferred by the runtime
        for (int b = 0; b < 2; b++) { if (built[b]) cudaEventDestroy(built[b]); if (freed[b]) cudaEventDestroy(freed[b]); }
        for (int b = 0; b < 2; b++) if (posted[b]) cudaEventDestroy(posted[b]);
        if (start) cudaEventDestroy(start);
        if (side) cudaStreamDestroy(side);
        if (post) cudaStreamDestroy(post);
        if (alt) cudaStreamDestroy(alt);
    }
};

// Images per launch: the largest count under `cap` whose supertiles fill whole rounds of the persistent grid best
// (a launch of 59.3 rounds costs 60); `step` keeps pairs of images together on the map path.
static size_t tc_group_size(size_t cap, size_t step, uint64_t items_per_image, int sms) {
    if (cap < step) return step;
    size_t best = cap - cap % step;
    double best_eff = 0.0;
    for (size_t g = cap - cap % step; g >= step && g * 4 >= cap * 3; g -= step) {
        const uint64_t items = g * items_per_image, rounds = (items + sms - 1) / sms;
        const double eff = (double)items / (double)(rounds * sms);
        if (eff > best_eff + 1e-9) { best_eff = eff; best = g; }
    }
    return best;
}

gp_status gp_launch_scoring_tc(const gp_structures_s* s, const gp_hp_params& hp, uint64_t g_begin, uint64_t g_count,
                               uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st) {
    using namespace tc;
    const int N = s->N;
    const int fb = N < s->tuning.fold_bits ? N : s->tuning.fold_bits;
    if (s->D >= (1u << KEY_SHIFT)) return GP_UNSUPPORTED_LATTICE;
    Plan p;
    int mon[MAX_FB];
    for (int i = 0; i < fb; i++) mon[i] = i;
    gp_status stt = make_plan(s, mon, fb, s->D, p);
    if (stt != GP_OK) return stt == GP_UNSUPPORTED_LATTICE ? GP_INVALID_ARG : stt;

    // batches of 2^fb genotypes share a weight image; a launch covers up to `group` batches
    const uint64_t g_end = g_begin + g_count;
    uint64_t group = (640ULL << 20) / p.img_bytes;  // two buffers of <= 640 MB of images: one is built while the other is scored
    if (group < 1) group = 1;
    if (group > 256) group = 256;
    group = tc_group_size((size_t)group, 1, ((1ULL << fb) + SUPER - 1) / SUPER, p.sms);
    const uint64_t n_batches_all = ((g_end - 1) >> fb) - (g_begin >> fb) + 1;
    if (group > n_batches_all) group = n_batches_all;
    gp_pool_mem work;  // per-call working memory from the stream-ordered pool: calls on other streams have their own
    GP_CUDA(work.alloc(2 * p.img_bytes * (size_t)group, st));
    int8_t* d_img0 = work.as<int8_t>();
    ImagePipeline pipe;
    {
        gp_status ps = pipe.open(st);
        if (ps != GP_OK) return ps;
    }
    if (p.narrow) GP_CUDA(cudaFuncSetAttribute(build_image_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)build_image_smem<64>(fb)));
    else GP_CUDA(cudaFuncSetAttribute(build_image_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)build_image_smem<128>(fb)));
    uint64_t g = g_begin & ~(uint64_t)(SUPER - 1);  // g_begin is a multiple of gp_tile() = SUPER already
    gp_status result = GP_OK;
    for (uint64_t grp = 0; g < g_end; grp++) {
        int8_t* d_img = d_img0 + (grp & 1) * p.img_bytes * (size_t)group;
        const uint64_t b0 = g >> fb;
        uint64_t stop = (b0 + group) << fb;
        if (stop > g_end) stop = g_end;
        const uint32_t n_batches = (uint32_t)(((stop - 1) >> fb) - b0 + 1);
        ImgArgs ia;
        ia.contacts = s->d_contacts; ia.class_of = s->d_class_of; ia.img = d_img; ia.units = nullptr;
        ia.gfix_first = b0; ia.unit_first = 0; ia.paired = 0; ia.mid = 0; ia.gfix_shift = fb; ia.D = s->D; ia.n_tiles = p.n_tiles;
        ia.NBP = s->NBP; ia.lin = hp.lin; ia.quad = hp.quad;
        pipe.before_build(grp);
        const uint64_t tk1 = gp_time_begin(GP_KERNEL_IMAGE, pipe.side);
        if (p.narrow) build_image_kernel<64><<<dim3(p.n_tiles, (n_batches + IMG_PER_BLOCK - 1) / IMG_PER_BLOCK), TN, build_image_smem<64>(fb), pipe.side>>>(ia, p.slots, n_batches, fb);
        else build_image_kernel<128><<<dim3(p.n_tiles, (n_batches + IMG_PER_BLOCK - 1) / IMG_PER_BLOCK), TN, build_image_smem<128>(fb), pipe.side>>>(ia, p.slots, n_batches, fb);
        gp_time_end(GP_KERNEL_IMAGE, tk1, pipe.side);
        pipe.after_build(grp, st);
        Args a;
        a.img = d_img; a.class_of = s->d_class_of; a.pheno = d_pheno; a.gap = d_gap;
        a.g_first = g; a.g_end = stop; a.out_base = g_begin;
        a.n_items = (uint32_t)((stop - g + SUPER - 1) / SUPER);
        a.n_tiles = p.n_tiles; a.D = s->D; a.fb = fb; a.k_steps = p.k_steps; a.threshold = hp.threshold;
        a.hrec = nullptr; a.n_snap = p.n_tiles;
        const unsigned grid = a.n_items < (uint32_t)p.sms ? a.n_items : (uint32_t)p.sms;
        const uint64_t tk2 = gp_time_begin(GP_KERNEL_SCORING, st);
        p.kernel<<<grid, p.threads, p.smem, st>>>(a, p.cols);
        gp_time_end(GP_KERNEL_SCORING, tk2, st);
        pipe.after_scoring(grp, st);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { gp_set_cuda_error(e, "scoring launch"); result = GP_CUDA_ERROR; break; }
        gp_count_launches(2);
        g = stop;
    }
    if (result != GP_OK) return result;  // `work` drains the device before it gives the buffers back
    GP_CUDA(work.release());
    return GP_OK;
}

// ---- whole map through the reversal identity E(g, rev S) = E(rev g, S) ---------------
// Every genotype is scored on ONE representative per class (C columns instead of D); the energies of the other class
// members are those of the reversed genotype on the same representatives.  An image holds the 2^(2k) genotypes that
// share their middle N - 2k bits m, so the reversed genotypes of image m are exactly image rev(m), read in bit-reversed
// local order.  A unit = {m, rev m}; the table lists m <= rev m, pairs first (include/gpmap.h).
static int map_k_for(const gp_structures_s* s) {
    using namespace tc;
    const int N = s->N;
    const int k = s->tuning.sym_bits < N / 2 ? s->tuning.sym_bits : N / 2;
    const int fb = 2 * k, mid = N - fb;
    if (fb < 9 || mid > 26 || s->D_sym >= (1u << KEY_SHIFT)) return 0;
    Cols cols;
    Slots slots;
    int mon[MAX_FB];
    for (int l = 0; l < k; l++) { mon[l] = l; mon[k + l] = N - k + l; }
    return make_columns(mon, fb, N, cols, slots) <= ROWB ? k : 0;
}

gp_status gp_build_map_units(gp_structures_s* s) {
    if (s->d_units) { cudaFree(s->d_units); s->d_units = nullptr; }
    s->units.clear();
    s->map_k = map_k_for(s);
    if (!s->map_k) { s->n_units = 1; s->n_pair_units = 0; return GP_OK; }  // one unit = the whole map (prefix path)
    const int mid = s->N - 2 * s->map_k;
    const uint32_t n_mid = 1u << mid;
    std::vector<uint32_t> pal;
    for (uint32_t m = 0; m < n_mid; m++) {
        uint32_t r = 0;
        for (int b = 0; b < mid; b++) r |= ((m >> b) & 1u) << (mid - 1 - b);
        if (r > m) s->units.push_back(m);
        else if (r == m) pal.push_back(m);
    }
    s->n_pair_units = s->units.size();
    s->units.insert(s->units.end(), pal.begin(), pal.end());
    s->n_units = s->units.size();
    if (s->device >= 0) {
        GP_CUDA(cudaMalloc(&s->d_units, s->units.size() * sizeof(uint32_t)));
        GP_CUDA(cudaMemcpy(s->d_units, s->units.data(), s->units.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
    }
    return GP_OK;
}

extern "C" uint64_t gp_map_units(const gp_structures_t* s) { return s ? s->n_units : 0; }

extern "C" gp_status gp_map_unit(const gp_structures_t* s, uint64_t unit, uint64_t* m, int* k) {
    if (!s) return GP_INVALID_ARG;
    if (unit >= s->n_units) return GP_RANGE;
    if (m) *m = s->map_k ? s->units[unit] : 0;
    if (k) *k = s->map_k;  // 0: the single unit is the whole map
    return GP_OK;
}

static gp_status gp_launch_map_range(const gp_structures_s* s, const gp_hp_params& hp, uint64_t u_first, uint64_t u_count,
                                     uint16_t* d_pheno, int16_t* d_gap, int compact, cudaStream_t st) {
    using namespace tc;
    const int N = s->N, k = s->map_k, fb = 2 * k, mid = N - fb;
    Plan p;
    int mon[MAX_FB];
    for (int l = 0; l < k; l++) { mon[l] = l; mon[k + l] = N - k + l; }
    gp_status stt = make_plan(s, mon, fb, s->D_sym, p);
    if (stt != GP_OK) return stt;
    const size_t rec_bytes = sizeof(int4) << fb;
    size_t group = (1280ULL << 20) / (2 * p.img_bytes + 2 * rec_bytes);  // <= 1.25 GB: two image buffers + two record buffers
    if (group > 512) group = 512;
    group = tc_group_size(group, 2, ((1ULL << fb) + SUPER - 1) / SUPER, p.sms);
    if (group < 2) group = 2;
    {   // never more than the range needs
        const uint64_t pairs = u_first < s->n_pair_units ? (u_first + u_count < s->n_pair_units ? u_count : s->n_pair_units - u_first) : 0;
        const uint64_t most = 2 * pairs > u_count - pairs ? 2 * pairs : u_count - pairs;
        if (group > most) group = (size_t)((most + 1) & ~1ULL);
    }
    gp_pool_mem work;
    GP_CUDA(work.alloc((2 * p.img_bytes + 2 * rec_bytes) * group, st));
    char* d_work = work.as<char>();
    int4* d_rec0 = (int4*)(d_work + 2 * p.img_bytes * group);
    ImagePipeline pipe;
    {
        gp_status ps = pipe.open(st, u_count >= 1024);   // small ranges: a few launches, not worth two more streams
        if (ps != GP_OK) return ps;
    }
    if (p.narrow) GP_CUDA(cudaFuncSetAttribute(build_image_kernel<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)build_image_smem<64>(fb)));
    else GP_CUDA(cudaFuncSetAttribute(build_image_kernel<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)build_image_smem<128>(fb)));
    gp_status result = GP_OK;
    uint64_t u = u_first, images_done = 0, n_groups = 0;
    const uint64_t u_end = u_first + u_count;
    for (uint64_t grp = 0; u < u_end; grp++) {
        int8_t* d_img = (int8_t*)d_work + (grp & 1) * p.img_bytes * group;
        const int paired = u < s->n_pair_units;
        uint64_t stop = paired ? u + group / 2 : u + group;
        const uint64_t limit = paired && s->n_pair_units < u_end ? s->n_pair_units : u_end;
        if (stop > limit) stop = limit;
        const uint32_t n_img = (uint32_t)(stop - u) * (paired ? 2u : 1u);
        ImgArgs ia;
        ia.contacts = s->d_contacts_sym; ia.class_of = s->d_class_sym; ia.img = d_img; ia.units = s->d_units;
        ia.gfix_first = 0; ia.unit_first = u; ia.paired = paired; ia.mid = mid; ia.gfix_shift = k; ia.D = s->D_sym;
        ia.n_tiles = p.n_tiles; ia.NBP = s->NBP; ia.lin = hp.lin; ia.quad = hp.quad;
        pipe.before_build(grp);
        const uint64_t tk3 = gp_time_begin(GP_KERNEL_IMAGE, pipe.side);
        if (p.narrow) build_image_kernel<64><<<dim3(p.n_tiles, (n_img + IMG_PER_BLOCK - 1) / IMG_PER_BLOCK), TN, build_image_smem<64>(fb), pipe.side>>>(ia, p.slots, n_img, fb);
        else build_image_kernel<128><<<dim3(p.n_tiles, (n_img + IMG_PER_BLOCK - 1) / IMG_PER_BLOCK), TN, build_image_smem<128>(fb), pipe.side>>>(ia, p.slots, n_img, fb);
        gp_time_end(GP_KERNEL_IMAGE, tk3, pipe.side);
        cudaStream_t sg = pipe.scoring_stream(grp, st);
        pipe.after_build(grp, sg);
        Args a;
        a.img = d_img; a.class_of = s->d_class_sym; a.pheno = nullptr; a.gap = nullptr;
        a.g_first = 0; a.g_end = (uint64_t)n_img << fb; a.out_base = 0;
        a.n_items = (uint32_t)((a.g_end + SUPER - 1) / SUPER);
        a.n_tiles = p.n_tiles; a.D = s->D_sym; a.fb = fb; a.k_steps = p.k_steps; a.threshold = hp.threshold;
        int4* d_rec = d_rec0 + (grp & 1) * (group << fb);
        a.hrec = d_rec; a.n_snap = s->n_snap;
        const unsigned grid = a.n_items < (uint32_t)p.sms ? a.n_items : (uint32_t)p.sms;
        pipe.before_scoring(grp, sg);
        const uint64_t tk4 = gp_time_begin(GP_KERNEL_SCORING, sg);
        p.kernel<<<grid, p.threads, p.smem, sg>>>(a, p.cols);
        gp_time_end(GP_KERNEL_SCORING, tk4, sg);
        pipe.after_scoring(grp, sg);
        CombArgs ca;
        ca.hrec = d_rec; ca.units = s->d_units; ca.class_sym = s->d_class_sym;
        ca.pheno = d_pheno; ca.gap = d_gap; ca.unit_first = u; ca.n_images = n_img; ca.paired = paired; ca.mid = mid;
        ca.fb = fb; ca.k = k; ca.N = N; ca.threshold = hp.threshold; ca.compact = compact; ca.compact_base = images_done << fb;
        images_done += n_img;
        const uint64_t work = ((uint64_t)n_img << fb) / 256;
        combine_kernel<<<(unsigned)(work < (uint64_t)p.sms * 8 ? (work ? work : 1) : (uint64_t)p.sms * 8), 256, 0, pipe.post_stream(grp, st)>>>(ca);
        pipe.after_post(grp);
        n_groups = grp + 1;
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { gp_set_cuda_error(e, "map launch"); result = GP_CUDA_ERROR; break; }
        gp_count_launches(3);
        u = stop;
    }
    pipe.join_post(n_groups, st);
    if (result != GP_OK) return result;  // `work` drains the device before it gives the buffers back
    GP_CUDA(work.release());
    return GP_OK;
}

extern "C" uint64_t gp_map_range_genotypes(const gp_structures_t* s, uint64_t unit_first, uint64_t unit_count) {
    if (!s || unit_first > s->n_units || unit_count > s->n_units - unit_first) return 0;
    if (!s->map_k) return unit_count ? 1ULL << s->N : 0;
    const uint64_t end = unit_first + unit_count;
    const uint64_t pairs = unit_first < s->n_pair_units ? (end < s->n_pair_units ? end : s->n_pair_units) - unit_first : 0;
    return (2 * pairs + (unit_count - pairs)) << (2 * s->map_k);
}

extern "C" gp_status gp_enumerate_map_range(const gp_structures_t* s, const gp_energies* en, uint64_t unit_first,
                                            uint64_t unit_count, uint16_t* d_pheno, int16_t* d_gap, int layout,
                                            void* stream) {
    gp_hp_params hp;
    gp_status stt = gp_check_hp(s, en, &hp);
    if (stt != GP_OK) return stt;
    if (!d_pheno || (layout != GP_MAP_FULL_STORE && layout != GP_MAP_COMPACT)) return GP_INVALID_ARG;
    if (unit_first > s->n_units || unit_count > s->n_units - unit_first) return GP_RANGE;
    if (s->device < 0) { gp_set_cuda_error(cudaErrorNoDevice, "handle has no device tables"); return GP_CUDA_ERROR; }
    if (s->N >= 64) return GP_UNSUPPORTED_LATTICE;
    if (unit_count == 0) return GP_OK;
    if (!s->map_k)  // chains too short for the scheme: the single unit is the whole map on the prefix path
        return gp_launch_scoring_tc(s, hp, 0, 1ULL << s->N, d_pheno, d_gap, (cudaStream_t)stream);
    return gp_launch_map_range(s, hp, unit_first, unit_count, d_pheno, d_gap, layout == GP_MAP_COMPACT, (cudaStream_t)stream);
}

extern "C" gp_status gp_enumerate_map(const gp_structures_t* s, const gp_energies* en, uint16_t* d_pheno, int16_t* d_gap,
                                      void* stream) {
    if (!s) return GP_INVALID_ARG;
    return gp_enumerate_map_range(s, en, 0, s->n_units, d_pheno, d_gap, GP_MAP_FULL_STORE, stream);
}

// Explicit HP sequences on the tensor cores (sequence_kernel).  GP_UNSUPPORTED_LATTICE = this lattice needs more than
// 384 columns: the caller falls back to the CUDA-core kernel.
gp_status gp_launch_sequences_tc(const gp_structures_s* s, const gp_hp_params& hp, const uint8_t* d_seqs, uint64_t seed,
                                 uint64_t first, uint64_t count, uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st) {
    using namespace tc;
    const int ncol = 2 + s->N + s->P;
    if (ncol > SQ_MAXCOL || s->N > 62 || s->D >= (1u << KEY_SHIFT)) return GP_UNSUPPORTED_LATTICE;
    const uint32_t n_tiles = (s->D + TN - 1) / TN;
    // weight image of (lin, quad): cached in the handle, immutable once built; other streams wait on its event
    const int8_t* d_img = nullptr;
    gp_pool_mem private_img;      // cache full: a per-call image from the stream-ordered pool
    {
        std::lock_guard<std::mutex> lk(s->mu);
        for (const gp_weight_image& w : s->wimgs)
            if (w.lin == hp.lin && w.quad == hp.quad) {
                GP_CUDA(cudaStreamWaitEvent(st, (cudaEvent_t)w.ready, 0));
                d_img = w.d_img;
            }
        if (!d_img) {
            gp_weight_image w;
            w.lin = hp.lin; w.quad = hp.quad;
            const bool cache = s->wimgs.size() < 8;
            if (cache) GP_CUDA(cudaMalloc(&w.d_img, (size_t)n_tiles * SQ_TILE));  // first use of these energies only
            else { GP_CUDA(private_img.alloc((size_t)n_tiles * SQ_TILE, st)); w.d_img = private_img.as<int8_t>(); }
            SqImgArgs ia;
            ia.contacts = s->d_contacts; ia.pairidx = s->d_pairidx; ia.img = w.d_img; ia.D = s->D;
            ia.N = s->N; ia.NBP = s->NBP; ia.lin = hp.lin; ia.quad = hp.quad;
            build_full_image_kernel<<<n_tiles, TN, 0, st>>>(ia);
            cudaError_t e = cudaGetLastError();
            cudaEvent_t ev = nullptr;
            if (e == cudaSuccess && cache) {
                e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming);
                if (e == cudaSuccess) e = cudaEventRecord(ev, st);
            }
            if (e != cudaSuccess) {   // an image that never reached the cache is not kept
                gp_set_cuda_error(e, "gp_enumerate_seqs: weight image build");
                if (ev) cudaEventDestroy(ev);
                if (cache) { cudaStreamSynchronize(st); cudaFree(w.d_img); }
                return GP_CUDA_ERROR;
            }
            gp_count_launches(1);
            if (cache) {
                w.ready = ev;
                s->wimgs.push_back(w);
            }
            d_img = w.d_img;
        }
    }
    SqCols cols;
    for (int c = 0; c < SQ_MAXCOL; c++) cols.i[c] = cols.j[c] = 62;  // bit 62 of the letter word is always 0
    cols.i[0] = cols.j[0] = cols.i[1] = cols.j[1] = 63;             // constant 1 (x64 and x1)
    for (int i = 0; i < s->N; i++) cols.i[2 + i] = cols.j[2 + i] = (uint8_t)i;
    for (int i = 0; i < s->N; i++)
        for (int j = 0; j < s->N; j++) {
            const int p = s->pair_index[(size_t)i * s->N + j];
            if (p >= 0 && i < j) { cols.i[2 + s->N + p] = (uint8_t)i; cols.j[2 + s->N + p] = (uint8_t)j; }
        }
    int dev = 0, sms = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t smem = (size_t)(SQ_MT + SQ_STAGES) * SQ_TILE + sizeof(SqBarriers) + sizeof(SqCols) + 1024 + 64;
    GP_CUDA(cudaFuncSetAttribute(sequence_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    SqArgs a;
    a.img = d_img; a.class_of = s->d_class_of; a.seqs = d_seqs; a.seed = seed; a.first = first; a.pheno = d_pheno; a.gap = d_gap; a.count = count;
    a.n_items = (uint32_t)((count + SQ_ROWS - 1) / SQ_ROWS); a.n_tiles = n_tiles;
    a.N = s->N; a.ksteps = (ncol + 31) / 32; a.threshold = hp.threshold;
    const unsigned grid = a.n_items < (uint32_t)sms ? a.n_items : (uint32_t)sms;
    const uint64_t tk5 = gp_time_begin(GP_KERNEL_SCORING, st);
    sequence_kernel<<<grid, SQ_THREADS, smem, st>>>(a, cols);
    gp_time_end(GP_KERNEL_SCORING, tk5, st);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    GP_CUDA(private_img.release());
    return GP_OK;
}

extern "C" uint64_t gp_tile(void) { return tc::SUPER; }

extern "C" gp_status gp_enumerate(const gp_structures_t* s, const gp_energies* en, uint64_t g_begin, uint64_t g_count,
                                  uint16_t* d_pheno, int16_t* d_gap, void* stream) {
    gp_hp_params hp;
    gp_status stt = gp_check_hp(s, en, &hp);
    if (stt != GP_OK) return stt;
    if (!d_pheno && g_count) return GP_INVALID_ARG;
    const uint64_t total = s->N >= 64 ? ~0ULL : (1ULL << s->N);
    if (g_begin > total || g_count > total - g_begin || (g_begin % tc::SUPER) != 0) return GP_RANGE;
    if (s->device < 0) { gp_set_cuda_error(cudaErrorNoDevice, "handle has no device tables"); return GP_CUDA_ERROR; }
    if (g_count == 0) return GP_OK;
    return gp_launch_scoring_tc(s, hp, g_begin, g_count, d_pheno, d_gap, (cudaStream_t)stream);
}

// Measured int8 MMA-only peak (include/gpmap.h).  Synchronous.
extern "C" gp_status gp_probe_i8_peak(int k_steps, double seconds, double* ops_per_s, double* clk_per_mma, double* sm_mhz) {
    using namespace tc;
    if (k_steps < 1 || k_steps > 4 || !(seconds > 0) || seconds > 30 || !ops_per_s) return GP_INVALID_ARG;
    int dev = 0, sms = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    typedef void (*probe_fn)(uint32_t, unsigned long long*);
    const probe_fn fn = k_steps == 1 ? mma_probe_kernel<1, 64> : k_steps == 2 ? mma_probe_kernel<2, 64>
                      : k_steps == 3 ? mma_probe_kernel<3, 128> : mma_probe_kernel<4, 128>;
    const size_t smem = 2 * (size_t)TM * (k_steps <= 2 ? 64 : 128) + 1024;
    GP_CUDA(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    unsigned long long* d_cycles = nullptr;
    GP_CUDA(cudaMalloc(&d_cycles, sms * sizeof(unsigned long long)));
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    {
        cudaError_t e = cudaEventCreate(&e0);
        if (e == cudaSuccess) e = cudaEventCreate(&e1);
        if (e != cudaSuccess) {
            gp_set_cuda_error(e, "gp_probe_i8_peak: cudaEventCreate");
            if (e0) cudaEventDestroy(e0);
            cudaFree(d_cycles);
            return GP_CUDA_ERROR;
        }
    }
    const uint32_t mma_per_group = (64 / k_steps) * k_steps;
    uint32_t groups = 2000;  // ~4 ms; then scaled to the requested duration
    float ms = 0;
    gp_status st = GP_OK;
    for (int round = 0; round < 2 && st == GP_OK; round++) {
        cudaEventRecord(e0, 0);
        fn<<<sms, 128, smem, 0>>>(groups, d_cycles);
        cudaEventRecord(e1, 0);
        cudaError_t e = cudaEventSynchronize(e1);
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
        if (e != cudaSuccess) { gp_set_cuda_error(e, "gp_probe_i8_peak"); st = GP_CUDA_ERROR; break; }
        gp_count_launches(1);
        if (round == 0) {
            double want = groups * (seconds * 1e3 / (ms > 0.01f ? ms : 0.01f));
            groups = (uint32_t)(want < 4 ? 4 : want > 4e8 ? 4e8 : want);
        }
    }
    if (st == GP_OK) {
        std::vector<unsigned long long> cyc(sms);
        cudaMemcpy(cyc.data(), d_cycles, sms * sizeof(unsigned long long), cudaMemcpyDeviceToHost);
        double mean = 0;
        for (int i = 0; i < sms; i++) mean += (double)cyc[i] / sms;
        const double mmas = (double)groups * mma_per_group;
        *ops_per_s = mmas * sms * (2.0 * TM * TN * 32) / (ms * 1e-3);
        if (clk_per_mma) *clk_per_mma = mean / mmas;
        if (sm_mhz) *sm_mhz = mean / (ms * 1e-3) / 1e6;
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    cudaFree(d_cycles);
    return st;
}
