// reductions.cu — a5 designability, a6 one-point-mutation neighbourhood (:138-147, Eq. 2) and
// a7 neutral-network components (:19) over the uint16 phenotype store.  HBM-streaming kernels.
#include "device_common.cuh"

namespace {

constexpr uint32_t NULLP = GP_NULL_PHENO;

// ---------------------------------------------------------------------------------------------------------------
// a5. Histogram.  Each block keeps a private u32 histogram of all classes in shared memory (up to 56 K bins = 224 KB);
// nulls — the majority of entries (:216: 95 % for 3x3x3) — never touch it: they are counted with a warp ballot.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) hist_kernel(const uint16_t* __restrict__ pheno, uint64_t count, uint32_t C,
                                                    unsigned long long* __restrict__ hist, int use_smem) {
    extern __shared__ uint32_t sh[];
    if (use_smem)
        for (uint32_t i = threadIdx.x; i < C; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    unsigned long long nulls = 0;
    const uint64_t nvec = count / 8;
    const uint4* v = reinterpret_cast<const uint4*>(pheno);
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += 4 * stride) {
        uint4 xs[4];  // four independent 16-byte loads in flight per thread
#pragma unroll
        for (int u = 0; u < 4; u++) xs[u] = (i + u * stride < nvec) ? __ldg(v + i + u * stride) : make_uint4(~0u, ~0u, ~0u, ~0u);
#pragma unroll
        for (int u = 0; u < 4; u++) {
            if (i + u * stride >= nvec) break;
            const uint32_t w[4] = {xs[u].x, xs[u].y, xs[u].z, xs[u].w};
            // nulls: per half min(~id, 1) is 0 exactly for 0xFFFF; four words summed, halves added at the end
            const uint32_t nn = __vminu2(~w[0], 0x00010001u) + __vminu2(~w[1], 0x00010001u) + __vminu2(~w[2], 0x00010001u) +
                                __vminu2(~w[3], 0x00010001u);
            nulls += 8u - (nn & 0xFFFFu) - (nn >> 16);
            // one compare per id: the null id 0xFFFF is >= C like every id the caller's n_classes does not cover
#pragma unroll
            for (int j = 0; j < 4; j++) {
                const uint32_t p0 = w[j] & 0xFFFFu, p1 = w[j] >> 16;
                if (use_smem) {
                    if (p0 < C) atomicAdd(&sh[p0], 1u);
                    if (p1 < C) atomicAdd(&sh[p1], 1u);
                } else {
                    if (p0 < C) atomicAdd(&hist[p0], 1ULL);
                    if (p1 < C) atomicAdd(&hist[p1], 1ULL);
                }
            }
        }
    }
    // ragged tail (count not a multiple of 8)
    for (uint64_t i = nvec * 8 + (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count;
         i += (uint64_t)gridDim.x * blockDim.x) {
        uint32_t p = pheno[i];
        if (p == NULLP) nulls++;
        else if (p < C) {
            if (use_smem) atomicAdd(&sh[p], 1u);
            else atomicAdd(&hist[p], 1ULL);
        }
    }
    for (int o = 16; o > 0; o >>= 1) nulls += __shfl_down_sync(0xFFFFFFFFu, nulls, o);
    if ((threadIdx.x & 31) == 0 && nulls) atomicAdd(&hist[C], nulls);
    __syncthreads();
    if (use_smem)
        for (uint32_t i = threadIdx.x; i < C; i += blockDim.x)
            if (sh[i]) atomicAdd(&hist[i], (unsigned long long)sh[i]);
}

// ---------------------------------------------------------------------------------------------------------------
// a6. Neighbour pass, bit-tiled.  The n_bits flips are handled in passes; each pass reads the
// store ONCE.  A block stages a tile of 2^tb phenotypes in shared memory: 2^h segments (all values of the h "spread"
// genotype bits hi_pos..hi_pos+h-1) of 2^c consecutive ids each (c = tb - h; 128-byte segments when the tile allows,
// never under 16 bytes, so loads stay vectorised / coalesced).  Pass 0 has h = 0 and flips the tb low bits; every later
// pass flips its own h spread bits, all on chip.  n_bits = 36, tb = 16: 16 + 10 + 10 bits = 3 passes instead of 20
// partner sweeps.  A thread owns 8 consecutive ids (one 16-byte shared-memory vector); flips of local bits 0-2 stay
// inside the vector, higher local bits are one LDS.128 of the partner vector.
// ---------------------------------------------------------------------------------------------------------------
struct RobArgs {
    const uint16_t* pheno;
    int n_bits;
    uint32_t C;
    unsigned long long *R, *Dl, *O;
    uint32_t* bitmap;  // nullable; bit (min*C + max)
    int tb, c, h, hi_pos, f0;  // tile bits, contiguous low bits, spread bits, their position, first local bit to flip
};

// record the connected pair (p, q) in the C x C bitmap (tiny-store and cross-shard kernels; the tile kernel has its own
// filtered path)
__device__ __forceinline__ void note_pair(const RobArgs& a, uint32_t p, uint32_t q) {
    if (q < p) { const uint32_t t = p; p = q; q = t; }
    if (q >= a.C) return;
    const uint64_t bit = (uint64_t)p * a.C + q;
    uint32_t* w = a.bitmap + (bit >> 5);
    const uint32_t m = 1u << (bit & 31);
    if (!(*(volatile uint32_t*)w & m)) atomicOr(w, m);
}

__device__ __forceinline__ void unpack8(const uint4& x, uint32_t (&q)[8]) {
    q[0] = x.x & 0xFFFF; q[1] = x.x >> 16; q[2] = x.y & 0xFFFF; q[3] = x.y >> 16;
    q[4] = x.z & 0xFFFF; q[5] = x.z >> 16; q[6] = x.w & 0xFFFF; q[7] = x.w >> 16;
}

constexpr uint32_t ROB_FLUSH_TILES = 64;  // the class-count cache is written back every so many tiles (u32 counters)

// ---------------------------------------------------------------------------------------------------------------
// a6, the tile kernel.  The per-flip work is cut to what the counts need:
//   * "differs" per genotype pair = XOR + one unsigned 16x2 min with 1 (VIMNMX.U16x2): 2 ALU ops per two genotypes,
//     summed in packed halves (rne); neutral = flips - differs - (null neighbours) for a non-null genotype;
//   * null neighbours come from a per-tile bitmask (one byte per 8-genotype vector, built while staging): the partner
//     vector's byte is spread to eight nibbles by a 256-entry table and added to a nibble-packed counter;
//   * "some genotype of this vector has a neighbour of another class" = (differs byte) & (partner non-null byte) &
//     (own non-null byte) != 0: one test per vector-flip; only then are the events walked for the pair bitmap;
//   * class counts: (n, r, d) per run of equal class into the shared-memory cache; other = flips*n - r - d when the
//     cache is written back; n also yields the designability histogram when the caller wants it (pass 0).
// ---------------------------------------------------------------------------------------------------------------
constexpr int ROB2_TB_MAX = 16;     // 2^16 phenotypes = 128 KB of shared memory, one block of 1024 threads per SM
constexpr int R2THREADS = 1024;
struct Rob2Slot { uint32_t key, n, r, d; };

struct Rob2Args {
    const uint16_t* pheno;
    int n_bits;
    uint32_t C;
    unsigned long long *R, *Dl, *O, *hist;  // hist nullable: hist[p] += genotypes of class p, hist[C] += nulls
    uint32_t* bitmap;                        // nullable
    int tb, c, h, hi_pos, f0;
};

constexpr uint32_t ROB2_SLOTS = 4096;   // class-count cache of the second kernel: 64 KB, two probes (slot, slot ^ 1)

__device__ __forceinline__ void rob2_add(const Rob2Args& a, Rob2Slot* cache, uint32_t n_flip, uint32_t p, uint32_t n,
                                         uint32_t r, uint32_t d) {
    if (p >= a.C) return;
    Rob2Slot* s = cache + ((p * 2654435761u) >> 20);
    uint32_t k = s->key;
    if (k != p) {
        if (k == NULLP) k = atomicCAS(&s->key, NULLP, p), k = (k == NULLP) ? p : k;
        if (k != p) {                       // second probe
            s = cache + (((p * 2654435761u) >> 20) ^ 1u);
            k = s->key;
            if (k == NULLP) k = atomicCAS(&s->key, NULLP, p), k = (k == NULLP) ? p : k;
        }
    }
    if (k == p) {
        atomicAdd(&s->n, n);
        if (r) atomicAdd(&s->r, r);
        if (d) atomicAdd(&s->d, d);
    } else {                                // both slots hold other classes: straight to global memory
        if (r) atomicAdd(&a.R[p], (unsigned long long)r);
        if (d) atomicAdd(&a.Dl[p], (unsigned long long)d);
        const uint32_t o = n * n_flip - r - d;
        if (o) atomicAdd(&a.O[p], (unsigned long long)o);
        if (a.hist) atomicAdd(&a.hist[p], (unsigned long long)n);
    }
}

__device__ __forceinline__ void rob2_flush(const Rob2Args& a, Rob2Slot* cache, uint32_t n_flip) {
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < ROB2_SLOTS; i += blockDim.x) {
        const Rob2Slot s = cache[i];
        if (s.key != NULLP) {
            if (s.r) atomicAdd(&a.R[s.key], (unsigned long long)s.r);
            if (s.d) atomicAdd(&a.Dl[s.key], (unsigned long long)s.d);
            const unsigned long long o = (unsigned long long)s.n * n_flip - s.r - s.d;
            if (o) atomicAdd(&a.O[s.key], o);
            if (a.hist && s.n) atomicAdd(&a.hist[s.key], (unsigned long long)s.n);
        }
        cache[i] = Rob2Slot{NULLP, 0, 0, 0};
    }
    __syncthreads();
}

constexpr uint32_t ROB2_PF_SLOTS = 4096;  // per-block filter of recently recorded class pairs (16 KB)

// Pair events are not walked where they are found (a quarter of the lanes would work while the rest wait): a lane
// that has some pushes ONE record (vector, flipped bit, event byte) into its warp's shared-memory ring, and whenever 32
// records are pending the whole warp drains them, one record per lane.
constexpr uint32_t ROB2_RING = 64;   // records per warp

__device__ __forceinline__ void rob2_events(const RobArgs& pa, const uint16_t* seg, uint32_t* pf, uint32_t& last_key, uint32_t rec) {
    const uint32_t v = rec & 0x1FFFu, flipmask = 1u << ((rec >> 13) & 15u);
    uint32_t ob = rec >> 17;
    while (ob) {
        const uint32_t l = (v << 3) + (__ffs(ob) - 1);
        ob &= ob - 1;
        const uint32_t p = seg[l], qq = seg[l ^ flipmask];
        const uint32_t key = (min(p, qq) << 16) | max(p, qq);
        if (key != last_key) {
            last_key = key;
            uint32_t* slot = pf + ((key * 2654435761u) >> 20);
            if (*(volatile uint32_t*)slot != key) {   // not seen by this block lately (racy update is harmless: the bitmap is the truth)
                *(volatile uint32_t*)slot = key;
                const uint32_t q = key & 0xFFFFu;
                if (q < pa.C) {                       // fire-and-forget RED.OR: no read of the bitmap, nothing to wait for
                    const uint64_t bit = (uint64_t)(key >> 16) * pa.C + q;
                    atomicOr(pa.bitmap + (bit >> 5), 1u << (bit & 31));
                }
            }
        }
    }
}

// One flip of one 8-genotype vector: q = the neighbours' class words, Bp = their non-null byte, keep = which of the 8
// genotypes are the end of their edge that records pair events (the end whose flipped bit is 0).  Called by all 32
// lanes of the warp together (the ballot).
template <bool PAIRS>
__device__ __forceinline__ void rob2_flip(const RobArgs& pa, const uint16_t* seg, uint32_t* pf, uint32_t& last_key,
                                          uint32_t* ring, uint32_t& head, uint32_t& tail,
                                          const uint32_t (&m)[4], uint32_t q0, uint32_t q1, uint32_t q2, uint32_t q3,
                                          uint32_t Bm, uint32_t Bp, uint32_t keep, uint32_t v, uint32_t k,
                                          const uint32_t* lut, uint32_t (&rne)[4], uint32_t& nn) {
    const uint32_t e0 = __vminu2(q0 ^ m[0], 0x00010001u), e1 = __vminu2(q1 ^ m[1], 0x00010001u);
    const uint32_t e2 = __vminu2(q2 ^ m[2], 0x00010001u), e3 = __vminu2(q3 ^ m[3], 0x00010001u);
    rne[0] += e0; rne[1] += e1; rne[2] += e2; rne[3] += e3;
    nn += lut[Bp];
    if (PAIRS) {
        const uint32_t tt = e0 + (e1 << 2) + (e2 << 4) + (e3 << 6);
        const uint32_t ob = (tt | (tt >> 15)) & Bp & Bm & keep;     // differs, both ends non-null, recording end
        const uint32_t has = __ballot_sync(0xFFFFFFFFu, ob != 0);
        if (has) {
            const uint32_t lane = threadIdx.x & 31u;
            if (ob) ring[(tail + __popc(has & ((1u << lane) - 1u))) & (ROB2_RING - 1)] = v | (k << 13) | (ob << 17);
            tail += __popc(has);
            if (tail - head >= 32) {
                __syncwarp();
                rob2_events(pa, seg, pf, last_key, ring[(head + lane) & (ROB2_RING - 1)]);
                head += 32;
                __syncwarp();
            }
        }
    }
}

template <bool PAIRS>
__global__ void __launch_bounds__(R2THREADS, 1) robustness2_kernel(Rob2Args a) {
    extern __shared__ __align__(16) uint16_t seg[];
    const uint32_t n_vec = 1u << (a.tb - 3);                       // 16-byte vectors per tile
    uint8_t* nnb = reinterpret_cast<uint8_t*>(seg + ((size_t)1 << a.tb));  // per vector: bit i = genotype i is NOT null
    uint32_t* lut = reinterpret_cast<uint32_t*>(nnb + ((n_vec + 15u) & ~15u));  // byte -> eight nibbles
    Rob2Slot* cache = reinterpret_cast<Rob2Slot*>(lut + 256);
    uint32_t* pf = reinterpret_cast<uint32_t*>(cache + ROB2_SLOTS);
    uint32_t* ring = pf + ROB2_PF_SLOTS + (threadIdx.x >> 5) * ROB2_RING;  // this warp's event ring (PAIRS only)
    uint32_t head = 0, tail = 0;
    for (uint32_t i = threadIdx.x; i < 256; i += blockDim.x) {
        uint32_t x = 0;
        for (int b = 0; b < 8; b++) x |= ((i >> b) & 1u) << (4 * b);
        lut[i] = x;
    }
    for (uint32_t i = threadIdx.x; i < ROB2_SLOTS; i += blockDim.x) cache[i] = Rob2Slot{NULLP, 0, 0, 0};
    if (PAIRS)
        for (uint32_t i = threadIdx.x; i < ROB2_PF_SLOTS; i += blockDim.x) pf[i] = 0xFFFFFFFFu;
    uint32_t tiles_done = 0, last_key = 0xFFFFFFFFu;
    unsigned long long nulls = 0;
    const uint64_t n_tiles = 1ULL << (a.n_bits - a.tb);
    const uint32_t cmask = (1u << a.c) - 1u;
    const int lo_outer = a.hi_pos - a.c;                           // outer-index bits that sit below the spread bits
    const uint32_t n_flip = (uint32_t)(a.tb - a.f0);
    const int k_lo = a.f0 < 3 ? 3 : a.f0;                          // first flip that needs a partner vector
    const int k_mid = k_lo + 8 < a.tb ? k_lo + 8 : a.tb;           // nibble counters hold 8 flips each
    const uint4* sv = reinterpret_cast<const uint4*>(seg);
    const RobArgs pa = {a.pheno, a.n_bits, a.C, a.R, a.Dl, a.O, a.bitmap, a.tb, a.c, a.h, a.hi_pos, a.f0};
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const uint64_t base = ((t & ((1ULL << lo_outer) - 1ULL)) << a.c) | ((t >> lo_outer) << (a.hi_pos + a.h));
        __syncthreads();
        for (uint32_t v = threadIdx.x; v < n_vec; v += R2THREADS) {
            const uint32_t l = v << 3;
            const uint64_t g = base | (l & cmask) | ((uint64_t)(l >> a.c) << a.hi_pos);
            const uint4 x = __ldg(reinterpret_cast<const uint4*>(a.pheno + g));
            reinterpret_cast<uint4*>(seg)[v] = x;
            // non-null bits: per half min(~x, 1)
            const uint32_t n0 = __vminu2(~x.x, 0x00010001u), n1 = __vminu2(~x.y, 0x00010001u);
            const uint32_t n2 = __vminu2(~x.z, 0x00010001u), n3 = __vminu2(~x.w, 0x00010001u);
            const uint32_t tt = n0 + (n1 << 2) + (n2 << 4) + (n3 << 6);
            const uint32_t nb = (tt | (tt >> 15)) & 0xFFu;
            nnb[v] = (uint8_t)nb;
            nulls += 8 - __popc(nb);
        }
        __syncthreads();
        for (uint32_t v0 = 0; v0 < n_vec; v0 += R2THREADS) {       // uniform trip count: the warp stays converged
            const uint32_t v = v0 + threadIdx.x;
            const bool live = v < n_vec;
            const uint32_t Bm = live ? nnb[v] : 0u;
            if (__all_sync(0xFFFFFFFFu, Bm == 0)) continue;         // the warp's 256 genotypes are all null: nothing to count
            const uint4 mv = live ? sv[v] : make_uint4(~0u, ~0u, ~0u, ~0u);
            const uint32_t m[4] = {mv.x, mv.y, mv.z, mv.w};
            uint32_t rne[4] = {0, 0, 0, 0};                        // per half: flips whose neighbour differs (class or null)
            uint32_t nnL = 0, nnA = 0, nnB = 0;                    // per nibble: non-null neighbours (in-register flips / first 8 / rest)
            if (a.f0 == 0) {                                       // flips of local bits 0-2 stay inside the vector
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, __funnelshift_l(m[0], m[0], 16),
                                 __funnelshift_l(m[1], m[1], 16), __funnelshift_l(m[2], m[2], 16), __funnelshift_l(m[3], m[3], 16),
                                 Bm, ((Bm & 0x55u) << 1) | ((Bm >> 1) & 0x55u), 0x55u, v, 0u, lut, rne, nnL);
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, m[1], m[0], m[3], m[2], Bm,
                                 ((Bm & 0x33u) << 2) | ((Bm >> 2) & 0x33u), 0x33u, v, 1u, lut, rne, nnL);
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, m[2], m[3], m[0], m[1], Bm,
                                 ((Bm & 0x0Fu) << 4) | (Bm >> 4), 0x0Fu, v, 2u, lut, rne, nnL);
            }
#pragma unroll 4
            for (int k = k_lo; k < k_mid; k++) {
                const uint32_t pv = (v ^ (1u << (k - 3))) & (n_vec - 1);
                const uint4 x = sv[pv];
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, x.x, x.y, x.z, x.w, Bm, nnb[pv],
                                 pv > v ? 0xFFu : 0u, v, (uint32_t)k, lut, rne, nnA);
            }
#pragma unroll 4
            for (int k = k_mid; k < a.tb; k++) {
                const uint32_t pv = (v ^ (1u << (k - 3))) & (n_vec - 1);
                const uint4 x = sv[pv];
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, x.x, x.y, x.z, x.w, Bm, nnb[pv],
                                 pv > v ? 0xFFu : 0u, v, (uint32_t)k, lut, rne, nnB);
            }
            // per genotype: differs = rne half, non-null neighbours = nibbles of nnL + nnA + nnB;
            // neutral = flips - differs; to null = flips - non-null neighbours.  Runs of equal class are merged.
            uint32_t run = 0, r_acc = 0, d_acc = 0;
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const uint32_t p = (m[j >> 1] >> (16 * (j & 1))) & 0xFFFFu;
                if (p == NULLP) continue;
                run++;
                r_acc += n_flip - ((rne[j >> 1] >> (16 * (j & 1))) & 0xFFFFu);
                d_acc += n_flip - ((nnL >> (4 * j)) & 15u) - ((nnA >> (4 * j)) & 15u) - ((nnB >> (4 * j)) & 15u);
                const uint32_t nxt = j < 7 ? (m[(j + 1) >> 1] >> (16 * ((j + 1) & 1))) & 0xFFFFu : NULLP;
                if (nxt == p) continue;
                rob2_add(a, cache, n_flip, p, run, r_acc, d_acc);
                run = 0; r_acc = 0; d_acc = 0;
            }
        }
        if (PAIRS && tail != head) {                                // events left in the ring: the tile is about to be replaced
            __syncwarp();
            const uint32_t lane = threadIdx.x & 31u;
            if (lane < tail - head) rob2_events(pa, seg, pf, last_key, ring[(head + lane) & (ROB2_RING - 1)]);
            head = tail;
            __syncwarp();
        }
        if (++tiles_done % ROB_FLUSH_TILES == 0) rob2_flush(a, cache, n_flip);
    }
    rob2_flush(a, cache, n_flip);
    if (a.hist) {
        for (int o = 16; o > 0; o >>= 1) nulls += __shfl_down_sync(0xFFFFFFFFu, nulls, o);
        if ((threadIdx.x & 31) == 0 && nulls) atomicAdd(&a.hist[a.C], nulls);
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a6, the tile kernel with a DIRECT class table (used whenever 4 C bytes fit beside a 2^15 tile: every box of the paper).
// The flips are those of robustness2_kernel; what changes is where the per-genotype counts go.  One 32-bit word per
// class holds three fields, neutral (10 bits) | to-null (11 bits) | other (11 bits), and every non-null genotype does
// ONE shared-memory atomic add of its (r, d, o) word (at most 15 flips per pass, so each term is at most 15).  The add
// returns the old word, from which the carries out of the three fields are known exactly ((old & w) | ((old | w) &
// ~(old + w))): a carry out of a field is booked in the 64-bit global counters (+2^bits for the field that wrapped,
// -1 for the field above it that received the carry), so the fields may wrap as often as they like and the table is
// written back once, when the block has done all its tiles.  No hashing, no probing, no runs, no periodic flush.
// The genotype count per class (designability) is (r + d + o) / flips; the launcher reads it from per-call totals.
// ---------------------------------------------------------------------------------------------------------------
constexpr int ROB3_TB_MAX = 15;
constexpr uint32_t ROB3_C_MAX = 34304;   // 4 C bytes + 64 KB tile + bitmask + table + pair filter + rings <= 227 KB

__device__ __noinline__ void rob3_carry(const Rob2Args& a, uint32_t p, uint32_t c) {
    if (c & 0x200u) { atomicAdd(&a.R[p], 1024ULL); atomicAdd(&a.Dl[p], ~0ULL); }
    if (c & 0x100000u) { atomicAdd(&a.Dl[p], 2048ULL); atomicAdd(&a.O[p], ~0ULL); }
    if (c & 0x80000000u) atomicAdd(&a.O[p], 2048ULL);
}

template <bool PAIRS>
__global__ void __launch_bounds__(R2THREADS, 1) robustness3_kernel(Rob2Args a) {
    extern __shared__ __align__(16) uint16_t seg[];
    const uint32_t n_vec = 1u << (a.tb - 3);                       // 16-byte vectors per tile
    uint8_t* nnb = reinterpret_cast<uint8_t*>(seg + ((size_t)1 << a.tb));  // per vector: bit i = genotype i is NOT null
    uint32_t* lut = reinterpret_cast<uint32_t*>(nnb + ((n_vec + 15u) & ~15u));  // byte -> eight nibbles
    uint32_t* tab = lut + 256;                                     // per class: r | d << 10 | o << 21
    uint32_t* pf = tab + ((a.C + 3u) & ~3u);
    uint32_t* ring = pf + ROB2_PF_SLOTS + (threadIdx.x >> 5) * ROB2_RING;  // this warp's event ring (PAIRS only)
    uint32_t head = 0, tail = 0;
    for (uint32_t i = threadIdx.x; i < 256; i += blockDim.x) {
        uint32_t x = 0;
        for (int b = 0; b < 8; b++) x |= ((i >> b) & 1u) << (4 * b);
        lut[i] = x;
    }
    for (uint32_t i = threadIdx.x; i < a.C; i += blockDim.x) tab[i] = 0;
    if (PAIRS)
        for (uint32_t i = threadIdx.x; i < ROB2_PF_SLOTS; i += blockDim.x) pf[i] = 0xFFFFFFFFu;
    uint32_t last_key = 0xFFFFFFFFu;
    unsigned long long nulls = 0;
    const uint64_t n_tiles = 1ULL << (a.n_bits - a.tb);
    const uint32_t cmask = (1u << a.c) - 1u;
    const int lo_outer = a.hi_pos - a.c;                           // outer-index bits that sit below the spread bits
    const uint32_t n_flip = (uint32_t)(a.tb - a.f0);
    const int k_lo = a.f0 < 3 ? 3 : a.f0;                          // first flip that needs a partner vector
    // word of one genotype = (nf - rn) | (nf - nn) << 10 | (rn - nf + nn) << 21, rn = differing, nn = non-null neighbours
    const uint32_t w0 = n_flip * (1u + (1u << 10) - (1u << 21)), w_rn = (1u << 21) - 1u, w_nn = (1u << 21) - (1u << 10);
    const uint4* sv = reinterpret_cast<const uint4*>(seg);
    const RobArgs pa = {a.pheno, a.n_bits, a.C, a.R, a.Dl, a.O, a.bitmap, a.tb, a.c, a.h, a.hi_pos, a.f0};
    for (uint64_t t = blockIdx.x; t < n_tiles; t += gridDim.x) {
        const uint64_t base = ((t & ((1ULL << lo_outer) - 1ULL)) << a.c) | ((t >> lo_outer) << (a.hi_pos + a.h));
        __syncthreads();
        for (uint32_t v = threadIdx.x; v < n_vec; v += R2THREADS) {
            const uint32_t l = v << 3;
            const uint64_t g = base | (l & cmask) | ((uint64_t)(l >> a.c) << a.hi_pos);
            const uint4 x = __ldg(reinterpret_cast<const uint4*>(a.pheno + g));
            reinterpret_cast<uint4*>(seg)[v] = x;
            const uint32_t n0 = __vminu2(~x.x, 0x00010001u), n1 = __vminu2(~x.y, 0x00010001u);
            const uint32_t n2 = __vminu2(~x.z, 0x00010001u), n3 = __vminu2(~x.w, 0x00010001u);
            const uint32_t tt = n0 + (n1 << 2) + (n2 << 4) + (n3 << 6);
            const uint32_t nb = (tt | (tt >> 15)) & 0xFFu;
            nnb[v] = (uint8_t)nb;
            nulls += 8 - __popc(nb);
        }
        __syncthreads();
        if (t + gridDim.x < n_tiles) {                              // the next tile of this block: pull it into L2 meanwhile
            const uint64_t tn = t + gridDim.x;
            const uint64_t bn = ((tn & ((1ULL << lo_outer) - 1ULL)) << a.c) | ((tn >> lo_outer) << (a.hi_pos + a.h));
            const uint32_t step = a.c >= 6 ? 64u : (1u << a.c);     // genotypes per prefetch: a 128-byte line or one segment
            for (uint32_t l = threadIdx.x * step; l < (1u << a.tb); l += R2THREADS * step) {
                const uint64_t g = bn | (l & cmask) | ((uint64_t)(l >> a.c) << a.hi_pos);
                asm volatile("prefetch.global.L2 [%0];" ::"l"(a.pheno + g));
            }
        }
        for (uint32_t v0 = 0; v0 < n_vec; v0 += R2THREADS) {       // uniform trip count: the warp stays converged
            const uint32_t v = v0 + threadIdx.x;
            const bool live = v < n_vec;
            const uint32_t Bm = live ? nnb[v] : 0u;
            if (__all_sync(0xFFFFFFFFu, Bm == 0)) continue;         // the warp's 256 genotypes are all null: nothing to count
            const uint4 mv = live ? sv[v] : make_uint4(~0u, ~0u, ~0u, ~0u);
            const uint32_t m[4] = {mv.x, mv.y, mv.z, mv.w};
            uint32_t rne[4] = {0, 0, 0, 0};                        // per half: flips whose neighbour differs (class or null)
            uint32_t nn = 0;                                       // per nibble: non-null neighbours (at most 15 flips)
            if (a.f0 == 0) {                                       // flips of local bits 0-2 stay inside the vector
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, __funnelshift_l(m[0], m[0], 16),
                                 __funnelshift_l(m[1], m[1], 16), __funnelshift_l(m[2], m[2], 16), __funnelshift_l(m[3], m[3], 16),
                                 Bm, ((Bm & 0x55u) << 1) | ((Bm >> 1) & 0x55u), 0x55u, v, 0u, lut, rne, nn);
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, m[1], m[0], m[3], m[2], Bm,
                                 ((Bm & 0x33u) << 2) | ((Bm >> 2) & 0x33u), 0x33u, v, 1u, lut, rne, nn);
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, m[2], m[3], m[0], m[1], Bm,
                                 ((Bm & 0x0Fu) << 4) | (Bm >> 4), 0x0Fu, v, 2u, lut, rne, nn);
            }
#pragma unroll 4
            for (int k = k_lo; k < a.tb; k++) {
                const uint32_t pv = (v ^ (1u << (k - 3))) & (n_vec - 1);
                const uint4 x = sv[pv];
                rob2_flip<PAIRS>(pa, seg, pf, last_key, ring, head, tail, m, x.x, x.y, x.z, x.w, Bm, nnb[pv],
                                 pv > v ? 0xFFu : 0u, v, (uint32_t)k, lut, rne, nn);
            }
            uint32_t old[8], w[8];
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const uint32_t p = (m[j >> 1] >> (16 * (j & 1))) & 0xFFFFu;
                w[j] = w0 + ((rne[j >> 1] >> (16 * (j & 1))) & 0xFFFFu) * w_rn + ((nn >> (4 * j)) & 15u) * w_nn;
                old[j] = 0;
                if (p < a.C) old[j] = atomicAdd(&tab[p], w[j]); else w[j] = 0;
            }
#pragma unroll
            for (int j = 0; j < 8; j++) {
                const uint32_t c = ((old[j] & w[j]) | ((old[j] | w[j]) & ~(old[j] + w[j]))) & 0x80100200u;
                if (c) rob3_carry(a, (m[j >> 1] >> (16 * (j & 1))) & 0xFFFFu, c);
            }
        }
        if (PAIRS && tail != head) {                                // events left in the ring: the tile is about to be replaced
            __syncwarp();
            const uint32_t lane = threadIdx.x & 31u;
            if (lane < tail - head) rob2_events(pa, seg, pf, last_key, ring[(head + lane) & (ROB2_RING - 1)]);
            head = tail;
            __syncwarp();
        }
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < a.C; i += blockDim.x) {
        const uint32_t w = tab[i];
        if (w & 1023u) atomicAdd(&a.R[i], (unsigned long long)(w & 1023u));
        if ((w >> 10) & 2047u) atomicAdd(&a.Dl[i], (unsigned long long)((w >> 10) & 2047u));
        if (w >> 21) atomicAdd(&a.O[i], (unsigned long long)(w >> 21));
    }
    if (a.hist) {                                                   // only the null count: the classes come from the totals
        for (int o = 16; o > 0; o >>= 1) nulls += __shfl_down_sync(0xFFFFFFFFu, nulls, o);
        if ((threadIdx.x & 31) == 0 && nulls) atomicAdd(&a.hist[a.C], nulls);
    }
}

// After a pass whose (R, D, O) went to per-call totals: add them to the caller's arrays; every genotype of class p gave
// exactly `flips` to r + d + o, so the class's genotype count is the sum / flips.
__global__ void rob3_finish_kernel(const unsigned long long* tot, uint32_t C, uint32_t flips, unsigned long long* R,
                                   unsigned long long* Dl, unsigned long long* O, unsigned long long* hist) {
    const uint32_t p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= C) return;
    const unsigned long long r = tot[p], d = tot[C + p], o = tot[2 * (size_t)C + p];
    R[p] += r; Dl[p] += d; O[p] += o;
    hist[p] += (r + d + o) / flips;
}

// n_bits < 3 (fewer than 8 genotypes): one thread per genotype, straight from global memory.
__global__ void robustness_tiny_kernel(RobArgs a) {
    const uint32_t g = threadIdx.x;
    if (g >= (1u << a.n_bits)) return;
    const uint32_t p = a.pheno[g];
    if (p == NULLP || p >= a.C) return;
    unsigned long long r = 0, d = 0, o = 0;
    for (int k = 0; k < a.n_bits; k++) {
        const uint32_t q = a.pheno[g ^ (1u << k)];
        if (q == p) r++;
        else if (q == NULLP) d++;
        else { o++; if (a.bitmap) note_pair(a, p, q); }
    }
    if (r) atomicAdd(&a.R[p], r);
    if (d) atomicAdd(&a.Dl[p], d);
    if (o) atomicAdd(&a.O[p], o);
}

// phi row (Figs. 9-12): for a target class q, row[p] = number of (genotype, flip) pairs that lead from
// class p into q; row[C] = the same from null genotypes.  Adjacency is symmetric, so the kernel walks the genotypes OF
// class q (one streaming read, 16-byte vectors) and histograms their neighbours' classes.
__global__ void __launch_bounds__(256) phi_row_kernel(const uint16_t* __restrict__ pheno, int n_bits, uint32_t C, uint32_t q,
                                                      unsigned long long* __restrict__ row) {
    const uint64_t n = 1ULL << n_bits;
    const uint64_t n_vec = n >> 3;
    const uint32_t qq = q * 0x10001u;
    for (uint64_t v = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; v < (n_vec ? n_vec : 1);
         v += (uint64_t)gridDim.x * blockDim.x) {
        uint32_t mine[8];
        if (n_vec) {
            const uint4 x = __ldg(reinterpret_cast<const uint4*>(pheno) + v);
            if (!__vcmpeq2(x.x, qq) && !__vcmpeq2(x.y, qq) && !__vcmpeq2(x.z, qq) && !__vcmpeq2(x.w, qq)) continue;
            unpack8(x, mine);
        } else {
            for (int j = 0; j < 8; j++) mine[j] = (uint64_t)j < n ? pheno[j] : NULLP;
        }
        for (int j = 0; j < 8; j++) {
            if (mine[j] != q) continue;
            const uint64_t g = v * 8 + j;
            for (int k = 0; k < n_bits; k++) {
                const uint32_t p = pheno[g ^ (1ULL << k)];
                if (p == NULLP || p < C) atomicAdd(&row[p == NULLP ? C : p], 1ULL);
            }
        }
    }
}

// Flips of a bit that selects the shard (multi-GPU): entry i of `mine` and entry i of `partner` are
// neighbours.  Counts go to the classes of `mine` only (the partner's owner runs the mirror call).
__global__ void __launch_bounds__(256) robustness_cross_kernel(RobArgs a, const uint16_t* __restrict__ partner, uint64_t count) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t p = a.pheno[i];
        if (p == NULLP || p >= a.C) continue;
        const uint32_t q = partner[i];
        if (q == p) atomicAdd(&a.R[p], 1ULL);
        else if (q == NULLP) atomicAdd(&a.Dl[p], 1ULL);
        else {
            atomicAdd(&a.O[p], 1ULL);
            if (a.bitmap && q < a.C) note_pair(a, p, q);
        }
    }
}

// The same with a per-block class table in shared memory: one packed u32 per class, fields neutral (bits 0-10) |
// to-null (11-21) | other (22-31), one shared-memory atomic per non-null entry.  A field is emptied through its HALF
// mark: the one thread whose add takes a field from HALF - 1 to HALF subtracts HALF from the field and books HALF in
// the global counter.  Until that subtraction lands at most blockDim - 1 further adds can reach the field, so with
// XT = 512 threads it stays below 2 * HALF (other: 512 + 511 = 1023) and never carries into its neighbour; what is left
// in the table at the end is flushed class by class.  Global atomics per block: one per HALF entries of a class and
// field, plus at most three per class seen — instead of one per non-null entry, all ranks hammering the few designable
// classes (3 x 2^33 entries per rank for 6x6 on 8 GPUs).
constexpr int XT = 512;
constexpr uint32_t X_RBITS = 11, X_DBITS = 11, X_OBITS = 10;
__device__ __forceinline__ void xtab_add(uint32_t* tab, const RobArgs& a, uint32_t p, uint32_t shift, uint32_t bits,
                                         unsigned long long* global) {
    const uint32_t half = 1u << (bits - 1), mask = (1u << bits) - 1u;
    const uint32_t old = atomicAdd(&tab[p], 1u << shift);
    if (((old >> shift) & mask) + 1u == half) {
        atomicSub(&tab[p], half << shift);
        atomicAdd(&global[p], (unsigned long long)half);
    }
}
__global__ void __launch_bounds__(XT, 1) robustness_cross_table_kernel(RobArgs a, const uint16_t* __restrict__ partner,
                                                                       uint64_t count) {
    extern __shared__ uint32_t xtab[];
    for (uint32_t c = threadIdx.x; c < a.C; c += XT) xtab[c] = 0;
    __syncthreads();
    auto one = [&](uint32_t p, uint32_t q) {
        if (p == NULLP || p >= a.C) return;
        if (q == p) xtab_add(xtab, a, p, 0, X_RBITS, a.R);
        else if (q == NULLP) xtab_add(xtab, a, p, X_RBITS, X_DBITS, a.Dl);
        else {
            xtab_add(xtab, a, p, X_RBITS + X_DBITS, X_OBITS, a.O);
            if (a.bitmap && q < a.C) note_pair(a, p, q);
        }
    };
    // 16-byte vectors where both shards allow it (they are 2^k-entry device arrays in practice), scalars for the rest
    const bool vec = (((uintptr_t)a.pheno | (uintptr_t)partner) & 15) == 0;
    const uint64_t n_vec = vec ? count >> 3 : 0;
    for (uint64_t v = (uint64_t)blockIdx.x * XT + threadIdx.x; v < n_vec; v += (uint64_t)gridDim.x * XT) {
        const uint4 x = __ldg(reinterpret_cast<const uint4*>(a.pheno) + v);
        if (x.x == 0xFFFFFFFFu && x.y == 0xFFFFFFFFu && x.z == 0xFFFFFFFFu && x.w == 0xFFFFFFFFu) continue;  // eight nulls
        const uint4 y = __ldg(reinterpret_cast<const uint4*>(partner) + v);
        uint32_t mine[8], theirs[8];
        unpack8(x, mine);
        unpack8(y, theirs);
#pragma unroll
        for (int j = 0; j < 8; j++) one(mine[j], theirs[j]);
    }
    for (uint64_t i = n_vec * 8 + (uint64_t)blockIdx.x * XT + threadIdx.x; i < count; i += (uint64_t)gridDim.x * XT)
        one(a.pheno[i], partner[i]);
    __syncthreads();
    for (uint32_t c = threadIdx.x; c < a.C; c += XT) {
        const uint32_t w = xtab[c];
        if (!w) continue;
        const uint32_t r = w & ((1u << X_RBITS) - 1u), d = (w >> X_RBITS) & ((1u << X_DBITS) - 1u), o = w >> (X_RBITS + X_DBITS);
        if (r) atomicAdd(&a.R[c], (unsigned long long)r);
        if (d) atomicAdd(&a.Dl[c], (unsigned long long)d);
        if (o) atomicAdd(&a.O[c], (unsigned long long)o);
    }
}

__global__ void bitmap_or_kernel(uint32_t* __restrict__ dst, const uint32_t* __restrict__ src, uint64_t n_words) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t v = src[i];
        if (v) dst[i] |= v;
    }
}

__global__ void popcount_kernel(const uint32_t* __restrict__ words, uint64_t n_words, unsigned long long* out) {
    unsigned long long c = 0;
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (uint64_t)gridDim.x * blockDim.x)
        c += __popc(words[i]);
    for (int o = 16; o > 0; o >>= 1) c += __shfl_down_sync(0xFFFFFFFFu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(out, c);
}

// ---------------------------------------------------------------------------------------------------------------
// f4. Threshold sweep: designability at several energy thresholds from ONE
// read of the (phenotype, gap) stores of a threshold-1 enumeration.  A genotype folds at threshold t iff it has a
// unique ground state and second_min - min = -gap >= t.  bins[j][c] counts the genotypes of class c that fold at
// exactly j of the (ascending) thresholds; suffix sums over j give the histogram per threshold.
// ---------------------------------------------------------------------------------------------------------------
constexpr int SWEEP_MAX = 16;
struct SweepThr { int32_t t[SWEEP_MAX]; int n; };

__global__ void __launch_bounds__(512) sweep_kernel(const uint16_t* __restrict__ pheno, const int16_t* __restrict__ gap,
                                                    uint64_t count, uint32_t C, SweepThr thr,
                                                    unsigned long long* __restrict__ bins, int use_smem) {
    extern __shared__ uint32_t sh[];
    const uint32_t n_bins = (uint32_t)(thr.n + 1) * C;
    if (use_smem)
        for (uint32_t i = threadIdx.x; i < n_bins; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t p = pheno[i];
        if (p >= C) continue;  // null (or an id outside n_classes)
        const int32_t gp = gap[i];
        const int32_t margin = gp == GP_GAP_NONE ? INT32_MAX : -gp;
        int j = 0;
        for (int k = 0; k < thr.n; k++) j += (margin >= thr.t[k]);
        if (use_smem) atomicAdd(&sh[(uint32_t)j * C + p], 1u);
        else atomicAdd(&bins[(uint64_t)j * C + p], 1ULL);
    }
    __syncthreads();
    if (use_smem)
        for (uint32_t i = threadIdx.x; i < n_bins; i += blockDim.x)
            if (sh[i]) atomicAdd(&bins[i], (unsigned long long)sh[i]);
}

// block t: hist[slot[t]][c] = sum_{j > t} bins[j][c]; folding and null counts
__global__ void __launch_bounds__(256) sweep_finish_kernel(const unsigned long long* __restrict__ bins, uint64_t count,
                                                           uint32_t C, int n, const int* __restrict__ slot_of,
                                                           unsigned long long* __restrict__ folding,
                                                           unsigned long long* __restrict__ hist) {
    __shared__ unsigned long long part[256];
    const int t = blockIdx.x, out = slot_of[t];
    unsigned long long sum = 0;
    for (uint32_t c = threadIdx.x; c < C; c += blockDim.x) {
        unsigned long long v = 0;
        for (int j = t + 1; j <= n; j++) v += bins[(uint64_t)j * C + c];
        hist[(uint64_t)out * (C + 1) + c] = v;
        sum += v;
    }
    part[threadIdx.x] = sum;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) part[threadIdx.x] += part[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        folding[out] = part[0];
        hist[(uint64_t)out * (C + 1) + C] = count - part[0];
    }
}

// ---------------------------------------------------------------------------------------------------------------
// a7. Components: lock-free union-find over the hypercube edges that join equal non-null phenotypes.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t uf_find(uint32_t* parent, uint32_t x) {
    uint32_t p = parent[x];
    while (p != x) {
        uint32_t gp = parent[p];
        if (gp != p) parent[x] = gp;  // path halving (benign race: only ever points further up the same tree)
        x = p;
        p = parent[x];
    }
    return x;
}

__global__ void uf_init_kernel(uint32_t* parent, uint64_t n) {
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (uint64_t)gridDim.x * blockDim.x)
        parent[i] = (uint32_t)i;
}

__global__ void uf_link_kernel(const uint16_t* __restrict__ pheno, uint32_t* parent, int n_bits) {
    const uint64_t n = 1ULL << n_bits;
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n; g += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t p = pheno[g];
        if (p == NULLP) continue;
        for (int k = 0; k < n_bits; k++) {
            const uint64_t h = g ^ (1ULL << k);
            if (h < g || pheno[h] != p) continue;  // each edge once, from its lower end
            uint32_t x = uf_find(parent, (uint32_t)g), y = uf_find(parent, (uint32_t)h);
            while (x != y) {                       // hook the larger root under the smaller
                if (x < y) { uint32_t t = x; x = y; y = t; }
                uint32_t old = atomicCAS(&parent[x], x, y);
                if (old == x) break;
                x = uf_find(parent, old);
                y = uf_find(parent, y);
            }
        }
    }
}

__global__ void uf_count_kernel(const uint16_t* __restrict__ pheno, const uint32_t* __restrict__ parent, uint64_t n,
                                uint32_t C, uint32_t* ncomp) {
    for (uint64_t g = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; g < n; g += (uint64_t)gridDim.x * blockDim.x) {
        const uint32_t p = pheno[g];
        if (p != NULLP && p < C && parent[g] == (uint32_t)g) atomicAdd(&ncomp[p], 1u);
    }
}

int sm_count() {
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return sms;
}

}  // namespace

extern "C" gp_status gp_designability(const uint16_t* d_pheno, uint64_t count, uint32_t n_classes, uint64_t* d_hist,
                                      void* stream) {
    if (!d_hist || (!d_pheno && count) || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (((uintptr_t)d_pheno & 15) != 0) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    GP_CUDA(cudaMemsetAsync(d_hist, 0, ((size_t)n_classes + 1) * sizeof(uint64_t), st));
    if (count == 0) return GP_OK;
    const size_t smem = (size_t)n_classes * 4;
    const int use_smem = smem <= 224 * 1024;
    if (use_smem) GP_CUDA(cudaFuncSetAttribute(hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const uint64_t want = (count / 8 + 1023) / 1024;
    const int per_sm = use_smem ? (int)((224 * 1024) / (smem + 1024) > 2 ? 2 : 1) : 2;
    unsigned grid = (unsigned)(want < (uint64_t)sm_count() * per_sm ? (want ? want : 1) : (uint64_t)sm_count() * per_sm);
    const uint64_t tk1 = gp_time_begin(GP_KERNEL_HIST, st);
    hist_kernel<<<grid, 1024, use_smem ? smem : 0, st>>>(d_pheno, count, n_classes,
                                                         reinterpret_cast<unsigned long long*>(d_hist), use_smem);
    gp_time_end(GP_KERNEL_HIST, tk1, st);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}

extern "C" uint64_t gp_pair_bitmap_words(uint32_t n_classes) { return ((uint64_t)n_classes * n_classes + 31) / 32; }

static gp_status robustness_passes(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_neutral,
                                   uint64_t* d_deleterious, uint64_t* d_other, uint64_t* d_hist, uint32_t* d_pair_bitmap,
                                   int tile_bits, cudaStream_t st) {
    if (!d_pheno || !d_neutral || !d_deleterious || !d_other) return GP_INVALID_ARG;
    if (n_bits < 1 || n_bits > 40 || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (tile_bits != 0 && (tile_bits < 4 || tile_bits > ROB2_TB_MAX)) return GP_INVALID_ARG;
    if (((uintptr_t)d_pheno & 15) != 0) return GP_INVALID_ARG;
    RobArgs a;
    a.pheno = d_pheno; a.n_bits = n_bits; a.C = n_classes;
    a.R = reinterpret_cast<unsigned long long*>(d_neutral);
    a.Dl = reinterpret_cast<unsigned long long*>(d_deleterious);
    a.O = reinterpret_cast<unsigned long long*>(d_other);
    a.bitmap = d_pair_bitmap;
    if (n_bits < 3) {
        const uint64_t tk2 = gp_time_begin(GP_KERNEL_ROBUSTNESS, st);
        robustness_tiny_kernel<<<1, 32, 0, st>>>(a);
        gp_time_end(GP_KERNEL_ROBUSTNESS, tk2, st);
        GP_CUDA(cudaGetLastError());
        gp_count_launches(1);
        if (d_hist) {
            hist_kernel<<<1, 1024, 0, st>>>(d_pheno, 1ULL << n_bits, n_classes, reinterpret_cast<unsigned long long*>(d_hist), 0);
            GP_CUDA(cudaGetLastError());
            gp_count_launches(1);
        }
        return GP_OK;
    }
    // the direct-table kernel whenever the class table fits beside a 2^15 tile; tile_bits = 16 asks for the hashed one
    const bool direct = n_classes <= ROB3_C_MAX && tile_bits <= ROB3_TB_MAX;
    int tb = tile_bits ? tile_bits : (direct ? ROB3_TB_MAX : ROB2_TB_MAX);
    if (tb > n_bits) tb = n_bits;
    const uint64_t n_tiles = 1ULL << (n_bits - tb);
    const uint64_t cap = (uint64_t)sm_count();
    const unsigned grid = (unsigned)(n_tiles < cap ? n_tiles : cap);
    const size_t smem_tile = ((size_t)2 << tb) + ((((size_t)1 << (tb - 3)) + 15) & ~(size_t)15) + 1024 +
                             ROB2_PF_SLOTS * sizeof(uint32_t) + (R2THREADS / 32) * ROB2_RING * sizeof(uint32_t);
    const size_t smem = smem_tile + (direct ? (size_t)((n_classes + 3u) & ~3u) * 4 : ROB2_SLOTS * sizeof(Rob2Slot));
    if (direct) {
        if (d_pair_bitmap) GP_CUDA(cudaFuncSetAttribute(robustness3_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        else GP_CUDA(cudaFuncSetAttribute(robustness3_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    } else {
        if (d_pair_bitmap) GP_CUDA(cudaFuncSetAttribute(robustness2_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        else GP_CUDA(cudaFuncSetAttribute(robustness2_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    }
    a.tb = tb;
    // pass 0: the tb low bits; every later pass flips its own spread bits: segments of 2^c consecutive ids (128 bytes
    // with the hashed kernel's 2^16 tiles, 32 or 64 bytes with the direct kernel's 2^15, never under 16), all 2^h values
    // of the spread bits on chip; the remaining bits are split evenly over the fewest passes
    const int seg_bits = direct ? 4 : 6;
    const int hmax = tb - seg_bits > 1 ? tb - seg_bits : (tb - 3 > 1 ? tb - 3 : 1);
    int passes_left = (n_bits - tb + hmax - 1) / hmax;
    gp_pool_mem tot_mem;                                // direct kernel, pass 0 with the histogram: per-call totals
    int done = 0;
    bool first = true;
    while (done < n_bits) {
        if (done == 0) { a.c = tb; a.h = 0; a.hi_pos = tb; a.f0 = 0; done = tb; }
        else {
            const int h = (n_bits - done + passes_left - 1) / passes_left;
            passes_left--;
            a.h = h; a.c = tb - h; a.hi_pos = done; a.f0 = a.c; done += h;
        }
        const uint64_t tk3 = gp_time_begin(GP_KERNEL_ROBUSTNESS, st);
        {
            Rob2Args b;
            b.pheno = a.pheno; b.n_bits = n_bits; b.C = n_classes; b.R = a.R; b.Dl = a.Dl; b.O = a.O;
            b.hist = first ? reinterpret_cast<unsigned long long*>(d_hist) : nullptr;
            b.bitmap = a.bitmap; b.tb = a.tb; b.c = a.c; b.h = a.h; b.hi_pos = a.hi_pos; b.f0 = a.f0;
            if (direct) {
                if (b.hist) {
                    GP_CUDA(tot_mem.alloc(3 * (size_t)n_classes * sizeof(unsigned long long), st));
                    unsigned long long* tot = tot_mem.as<unsigned long long>();
                    GP_CUDA(cudaMemsetAsync(tot, 0, 3 * (size_t)n_classes * sizeof(unsigned long long), st));
                    b.R = tot; b.Dl = tot + n_classes; b.O = tot + 2 * (size_t)n_classes;
                }
                if (d_pair_bitmap) robustness3_kernel<true><<<grid, R2THREADS, smem, st>>>(b);
                else robustness3_kernel<false><<<grid, R2THREADS, smem, st>>>(b);
                if (b.hist) {
                    rob3_finish_kernel<<<(n_classes + 255) / 256, 256, 0, st>>>(tot_mem.as<unsigned long long>(), n_classes, (uint32_t)(b.tb - b.f0), a.R, a.Dl, a.O, b.hist);
                    gp_count_launches(1);
                }
            } else {
                if (d_pair_bitmap) robustness2_kernel<true><<<grid, R2THREADS, smem, st>>>(b);
                else robustness2_kernel<false><<<grid, R2THREADS, smem, st>>>(b);
            }
        }
        gp_time_end(GP_KERNEL_ROBUSTNESS, tk3, st);
        GP_CUDA(cudaGetLastError());
        gp_count_launches(1);
        GP_CUDA(tot_mem.release());
        first = false;
    }
    return GP_OK;
}

extern "C" gp_status gp_robustness_partial(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_neutral,
                                           uint64_t* d_deleterious, uint64_t* d_other, uint32_t* d_pair_bitmap,
                                           int tile_bits, void* stream) {
    return robustness_passes(d_pheno, n_bits, n_classes, d_neutral, d_deleterious, d_other, nullptr, d_pair_bitmap, tile_bits,
                             (cudaStream_t)stream);
}

extern "C" gp_status gp_robustness_cross(const uint16_t* d_mine, const uint16_t* d_partner, uint64_t count,
                                         uint32_t n_classes, uint64_t* d_neutral, uint64_t* d_deleterious,
                                         uint64_t* d_other, uint32_t* d_pair_bitmap, void* stream) {
    if (!d_mine || !d_partner || !d_neutral || !d_deleterious || !d_other) return GP_INVALID_ARG;
    if (n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (count == 0) return GP_OK;
    cudaStream_t st = (cudaStream_t)stream;
    RobArgs a;
    a.pheno = d_mine; a.n_bits = 0; a.C = n_classes;
    a.R = reinterpret_cast<unsigned long long*>(d_neutral);
    a.Dl = reinterpret_cast<unsigned long long*>(d_deleterious);
    a.O = reinterpret_cast<unsigned long long*>(d_other);
    a.bitmap = d_pair_bitmap;
    // the class table in shared memory whenever it fits one block per SM and the shard is long enough to repay zeroing
    // and flushing it; otherwise one global atomic per non-null entry
    const size_t table = (size_t)n_classes * sizeof(uint32_t);
    const bool use_table = table <= 220 * 1024 && count >= 16 * (uint64_t)n_classes;
    if (use_table) GP_CUDA(cudaFuncSetAttribute(robustness_cross_table_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)table));
    const uint64_t tk4 = gp_time_begin(GP_KERNEL_ROBUSTNESS, st);
    if (use_table) {
        const uint64_t want = (count / 8 + XT - 1) / XT, cap = (uint64_t)sm_count();
        robustness_cross_table_kernel<<<(unsigned)(want < cap ? (want ? want : 1) : cap), XT, table, st>>>(a, d_partner, count);
    } else {
        const uint64_t want = (count + 255) / 256, cap = (uint64_t)sm_count() * 8;
        robustness_cross_kernel<<<(unsigned)(want < cap ? want : cap), 256, 0, st>>>(a, d_partner, count);
    }
    gp_time_end(GP_KERNEL_ROBUSTNESS, tk4, st);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}

extern "C" gp_status gp_pair_bitmap_or(uint32_t* d_dst, const uint32_t* d_src, uint32_t n_classes, void* stream) {
    if (!d_dst || !d_src || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    const uint64_t n_words = gp_pair_bitmap_words(n_classes);
    bitmap_or_kernel<<<(unsigned)((n_words + 255) / 256 < 4096 ? (n_words + 255) / 256 : 4096), 256, 0, (cudaStream_t)stream>>>(
        d_dst, d_src, n_words);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}

extern "C" gp_status gp_pair_bitmap_count(const uint32_t* d_bitmap, uint32_t n_classes, uint64_t* d_count, void* stream) {
    if (!d_bitmap || !d_count || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t n_words = gp_pair_bitmap_words(n_classes);
    GP_CUDA(cudaMemsetAsync(d_count, 0, sizeof(uint64_t), st));
    popcount_kernel<<<(unsigned)((n_words + 255) / 256 < 4096 ? (n_words + 255) / 256 : 4096), 256, 0, st>>>(
        d_bitmap, n_words, reinterpret_cast<unsigned long long*>(d_count));
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}

extern "C" gp_status gp_reduce_store(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_hist,
                                     uint64_t* d_neutral, uint64_t* d_deleterious, uint64_t* d_other, uint64_t* d_pair_count,
                                     void* stream) {
    if (!d_pheno || !d_neutral || !d_deleterious || !d_other) return GP_INVALID_ARG;
    if (n_bits < 1 || n_bits > 40 || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t cb = (size_t)n_classes * sizeof(uint64_t);
    GP_CUDA(cudaMemsetAsync(d_neutral, 0, cb, st));
    GP_CUDA(cudaMemsetAsync(d_deleterious, 0, cb, st));
    GP_CUDA(cudaMemsetAsync(d_other, 0, cb, st));
    if (d_hist) GP_CUDA(cudaMemsetAsync(d_hist, 0, cb + sizeof(uint64_t), st));
    gp_pool_mem bitmap_mem;
    if (d_pair_count) {
        const uint64_t n_words = gp_pair_bitmap_words(n_classes);
        GP_CUDA(bitmap_mem.alloc(n_words * 4, st));
        GP_CUDA(cudaMemsetAsync(bitmap_mem.p, 0, n_words * 4, st));
    }
    uint32_t* bitmap = bitmap_mem.as<uint32_t>();
    gp_status stt = robustness_passes(d_pheno, n_bits, n_classes, d_neutral, d_deleterious, d_other, d_hist, bitmap, 0, st);
    if (stt == GP_OK && d_pair_count) stt = gp_pair_bitmap_count(bitmap, n_classes, d_pair_count, stream);
    if (stt != GP_OK) return stt;
    GP_CUDA(bitmap_mem.release());
    return GP_OK;
}

extern "C" gp_status gp_robustness(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_neutral,
                                   uint64_t* d_deleterious, uint64_t* d_other, uint64_t* d_pair_count, void* stream) {
    return gp_reduce_store(d_pheno, n_bits, n_classes, nullptr, d_neutral, d_deleterious, d_other, d_pair_count, stream);
}

extern "C" gp_status gp_threshold_sweep(const uint16_t* d_pheno, const int16_t* d_gap, uint64_t count, uint32_t n_classes,
                                        const int32_t* thresholds, int n_thresholds, uint64_t* d_folding,
                                        uint64_t* d_hist, void* stream) {
    if ((!d_pheno || !d_gap) && count) return GP_INVALID_ARG;
    if (!thresholds || !d_folding || !d_hist || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (n_thresholds < 1 || n_thresholds > SWEEP_MAX) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    // ascending thresholds; slot[r] = position of the r-th smallest in the caller's order
    SweepThr thr;
    int slot[SWEEP_MAX];
    thr.n = n_thresholds;
    for (int i = 0; i < n_thresholds; i++) {
        if (thresholds[i] < 1) return GP_INVALID_ARG;
        int r = i;
        while (r > 0 && thr.t[r - 1] > thresholds[i]) { thr.t[r] = thr.t[r - 1]; slot[r] = slot[r - 1]; r--; }
        thr.t[r] = thresholds[i]; slot[r] = i;
    }
    const size_t n_bins = (size_t)(n_thresholds + 1) * n_classes;
    gp_pool_mem work_mem;  // bins | slot table
    GP_CUDA(work_mem.alloc(n_bins * 8 + SWEEP_MAX * sizeof(int), st));
    char* work = work_mem.as<char>();
    unsigned long long* bins = reinterpret_cast<unsigned long long*>(work);
    int* d_slot = reinterpret_cast<int*>(work + n_bins * 8);
    GP_CUDA(cudaMemsetAsync(bins, 0, n_bins * 8, st));
    GP_CUDA(cudaMemcpyAsync(d_slot, slot, n_thresholds * sizeof(int), cudaMemcpyHostToDevice, st));  // pageable: staged before return
    const size_t smem = n_bins * 4;
    const int use_smem = smem <= 200 * 1024;
    if (use_smem) GP_CUDA(cudaFuncSetAttribute(sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (count) {
        const uint64_t want = (count + 511) / 512, cap = (uint64_t)sm_count() * (use_smem && smem > 100 * 1024 ? 1 : 2);
        sweep_kernel<<<(unsigned)(want < cap ? want : cap), 512, use_smem ? smem : 0, st>>>(
            d_pheno, d_gap, count, n_classes, thr, bins, use_smem);
        GP_CUDA(cudaGetLastError());
    }
    sweep_finish_kernel<<<n_thresholds, 256, 0, st>>>(bins, count, n_classes, n_thresholds, d_slot,
                                                      reinterpret_cast<unsigned long long*>(d_folding),
                                                      reinterpret_cast<unsigned long long*>(d_hist));
    GP_CUDA(cudaGetLastError());
    gp_count_launches(count ? 2 : 1);
    GP_CUDA(work_mem.release());
    return GP_OK;
}

extern "C" gp_status gp_phi_row(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint32_t q, uint64_t* d_row,
                                void* stream) {
    if (!d_pheno || !d_row || n_classes == 0 || n_classes >= NULLP || q >= n_classes) return GP_INVALID_ARG;
    if (n_bits < 1 || n_bits > 40 || ((uintptr_t)d_pheno & 15) != 0) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    GP_CUDA(cudaMemsetAsync(d_row, 0, ((size_t)n_classes + 1) * sizeof(uint64_t), st));
    const uint64_t n_vec = (1ULL << n_bits) >> 3;
    const uint64_t want = (n_vec + 255) / 256, cap = (uint64_t)sm_count() * 8;
    phi_row_kernel<<<(unsigned)(want < cap ? (want ? want : 1) : cap), 256, 0, st>>>(
        d_pheno, n_bits, n_classes, q, reinterpret_cast<unsigned long long*>(d_row));
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}

extern "C" gp_status gp_nn_components(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint32_t* d_ncomp,
                                      void* stream) {
    if (!d_pheno || !d_ncomp || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (n_bits < 1 || n_bits > 30) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t n = 1ULL << n_bits;
    gp_pool_mem parent_mem;
    GP_CUDA(parent_mem.alloc(n * sizeof(uint32_t), st));
    uint32_t* parent = parent_mem.as<uint32_t>();
    GP_CUDA(cudaMemsetAsync(d_ncomp, 0, (size_t)n_classes * sizeof(uint32_t), st));
    const unsigned grid = (unsigned)((n + 255) / 256 < (uint64_t)sm_count() * 16 ? (n + 255) / 256 : (uint64_t)sm_count() * 16);
    uf_init_kernel<<<grid, 256, 0, st>>>(parent, n);
    uf_link_kernel<<<grid, 256, 0, st>>>(d_pheno, parent, n_bits);
    uf_count_kernel<<<grid, 256, 0, st>>>(d_pheno, parent, n, n_classes, d_ncomp);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(3);
    GP_CUDA(parent_mem.release());
    GP_CUDA(cudaStreamSynchronize(st));
    return GP_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// gp_threshold_sweep_static (gpmap.h): the threshold sweep for callers that may not allocate device memory at run
// time — a process that gave its whole memory budget away at start-up, one whose pool is capped or disabled, a loop
// that cannot afford an allocator call.  The counter table that gp_threshold_sweep takes from the stream-ordered pool
// lives here in a file-scope device array of GP_SWEEP_STATIC_MAX_BINS counters (4 MiB, resident on every GPU that
// loads this code until the process ends).
//
// In HOST code `g_sweep_static_bins` is only a handle for the symbol, not a device address: handing it to a kernel
// would fault, or on a system where the GPU can reach host memory quietly count into the wrong place.  The address a
// kernel may use comes from cudaGetSymbolAddress, asked once per device with that device current and kept in
// g_sweep_static_ptr.  sweep_kernel is the same kernel the allocating path launches; only the table it is handed
// differs.  The slot table of the finish step travels as a kernel parameter, so there is no host-to-device copy either.
// ---------------------------------------------------------------------------------------------------------------
static __device__ __align__(256) unsigned long long g_sweep_static_bins[GP_SWEEP_STATIC_MAX_BINS];

namespace {

constexpr int SWEEP_STATIC_DEVICES = 64;  // device ordinals with a remembered address; higher ones are looked up per call
std::mutex g_sweep_static_mu;
unsigned long long* g_sweep_static_ptr[SWEEP_STATIC_DEVICES] = {};

struct SweepSlots { int s[SWEEP_MAX]; };

// sweep_finish_kernel with the slot table passed by value.  block t: hist[slots.s[t]][c] = sum_{j > t} bins[j][c]
__global__ void __launch_bounds__(256) sweep_finish_slots_kernel(const unsigned long long* __restrict__ bins, uint64_t count,
                                                                 uint32_t C, int n, SweepSlots slots,
                                                                 unsigned long long* __restrict__ folding,
                                                                 unsigned long long* __restrict__ hist) {
    __shared__ unsigned long long part[256];
    const int t = blockIdx.x, out = slots.s[t];
    unsigned long long sum = 0;
    for (uint32_t c = threadIdx.x; c < C; c += blockDim.x) {
        unsigned long long v = 0;
        for (int j = t + 1; j <= n; j++) v += bins[(uint64_t)j * C + c];
        hist[(uint64_t)out * (C + 1) + c] = v;
        sum += v;
    }
    part[threadIdx.x] = sum;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) part[threadIdx.x] += part[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        folding[out] = part[0];
        hist[(uint64_t)out * (C + 1) + C] = count - part[0];
    }
}

// Device address of g_sweep_static_bins on the CURRENT device.  The first call per device does the lookup (this is the
// set-up the header asks callers to keep outside stream capture); afterwards it is a table read.
gp_status sweep_static_table(unsigned long long** out) {
    int dev = -1;
    GP_CUDA(cudaGetDevice(&dev));
    const bool remembered = dev >= 0 && dev < SWEEP_STATIC_DEVICES;
    std::lock_guard<std::mutex> lk(g_sweep_static_mu);
    if (remembered && g_sweep_static_ptr[dev]) { *out = g_sweep_static_ptr[dev]; return GP_OK; }
    unsigned long long* p = nullptr;
    GP_CUDA(cudaGetSymbolAddress((void**)&p, g_sweep_static_bins));
    if (!p) { gp_set_cuda_error(cudaErrorInvalidSymbol, "gp_threshold_sweep_static: no device address for the scratch array"); return GP_CUDA_ERROR; }
    if (remembered) g_sweep_static_ptr[dev] = p;
    *out = p;
    return GP_OK;
}

}  // namespace

extern "C" gp_status gp_threshold_sweep_static(const uint16_t* d_pheno, const int16_t* d_gap, uint64_t count,
                                               uint32_t n_classes, const int32_t* thresholds, int n_thresholds,
                                               uint64_t* d_folding, uint64_t* d_hist, void* stream) {
    if ((!d_pheno || !d_gap) && count) return GP_INVALID_ARG;
    if (!thresholds || !d_folding || !d_hist || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (n_thresholds < 1 || n_thresholds > SWEEP_MAX) return GP_INVALID_ARG;
    const size_t n_bins = (size_t)(n_thresholds + 1) * n_classes;
    if (n_bins > GP_SWEEP_STATIC_MAX_BINS) return GP_TOO_LARGE;  // refused before anything is touched or launched
    cudaStream_t st = (cudaStream_t)stream;
    // ascending thresholds; slots.s[r] = position of the r-th smallest in the caller's order
    SweepThr thr;
    SweepSlots slots;
    thr.n = n_thresholds;
    for (int i = 0; i < SWEEP_MAX; i++) { thr.t[i] = 0; slots.s[i] = 0; }
    for (int i = 0; i < n_thresholds; i++) {
        if (thresholds[i] < 1) return GP_INVALID_ARG;
        int r = i;
        while (r > 0 && thr.t[r - 1] > thresholds[i]) { thr.t[r] = thr.t[r - 1]; slots.s[r] = slots.s[r - 1]; r--; }
        thr.t[r] = thresholds[i]; slots.s[r] = i;
    }
    unsigned long long* bins = nullptr;
    gp_status stt = sweep_static_table(&bins);
    if (stt != GP_OK) return stt;
    // the array keeps whatever the previous call counted: everything this call reads must start at zero
    GP_CUDA(cudaMemsetAsync(bins, 0, n_bins * sizeof(unsigned long long), st));
    const size_t smem = n_bins * 4;
    const int use_smem = smem <= 200 * 1024;
    if (use_smem) GP_CUDA(cudaFuncSetAttribute(sweep_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (count) {
        const uint64_t want = (count + 511) / 512, cap = (uint64_t)sm_count() * (use_smem && smem > 100 * 1024 ? 1 : 2);
        sweep_kernel<<<(unsigned)(want < cap ? want : cap), 512, use_smem ? smem : 0, st>>>(
            d_pheno, d_gap, count, n_classes, thr, bins, use_smem);
        GP_CUDA(cudaGetLastError());
    }
    sweep_finish_slots_kernel<<<n_thresholds, 256, 0, st>>>(bins, count, n_classes, n_thresholds, slots,
                                                            reinterpret_cast<unsigned long long*>(d_folding),
                                                            reinterpret_cast<unsigned long long*>(d_hist));
    GP_CUDA(cudaGetLastError());
    gp_count_launches(count ? 2 : 1);
    return GP_OK;
}
