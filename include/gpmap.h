/* gpmap.h — C ABI of libgpmap: exhaustive HP-model genotype-phenotype map on one B200 (sm_100a).
 *
 * What is computed follows arXiv 2008.05612 (citations are PAPER.md:LINE; readings R1.. are DESIGN.md section 2):
 *   fold library  = all compact self-avoiding walks of a box, one per symmetry class          (:65, :654-694)
 *   energy        = H = sum_{i<j} E[s_i][s_j] Delta(r_i - r_j), Delta = lattice but not chain neighbours (:67-69, Eq. 1)
 *   phenotype     = the unique minimum-energy fold, else "does not fold" (null)               (:81, :552-575)
 *   designability = number of genotypes per phenotype                                         (:138)
 *   robustness    = one-point-mutation neighbourhood counts, Eq. 2                            (:138-147)
 *   neutral nets  = connected same-phenotype genotype sets                                    (:19)
 *
 * Conventions
 *   - Every call returns a gp_status; nothing throws or exits across the ABI (the paper's gpuAssert exits, :470-485).
 *   - Pointers named d_* are DEVICE pointers, allocated and freed by the caller.  Pointers without the prefix are HOST
 *     pointers.  The library owns only the opaque gp_structures_t handle (its device tables included) and a private
 *     scratch it frees in gp_structures_free.
 *   - `stream` is a cudaStream_t passed as void* (NULL = default stream).  Compute calls are asynchronous on it and
 *     never synchronise the device or the stream unless their comment says so (gp_nn_components, gp_enumerate_host);
 *     a non-zero status reports argument or launch errors only.  Device output arrays are fully overwritten unless a
 *     call says it accumulates.  Working memory of a call comes from the device's stream-ordered pool
 *     (cudaMallocAsync on `stream`) and goes back to it on the same stream, so calls on one handle may run
 *     concurrently on different streams and threads; only gp_tuning_set and gp_structures_free must not overlap a
 *     call on the same handle.  A call may run part of its work (building weight images ahead of the scoring kernel)
 *     on an internal stream of its own; events tie it into `stream`, so the caller sees everything ordered on `stream`.
 *   - Genotype g: bit i of g is the letter of monomer i, 1 = H (R3).  Null phenotype = GP_NULL_PHENO (R7).
 *   - Phenotype ids are reversal-reduced class ids 0..C-1 in the canonical order of DESIGN.md section 3 (R1, R8).
 */
#ifndef GPMAP_H
#define GPMAP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define GP_NULL_PHENO 0xFFFFu
#define GP_GAP_NONE (-32768) /* gap reported when there is no second structure (D = 1), R6 */

typedef enum {
    GP_OK = 0,
    GP_INVALID_ARG = 1,         /* null pointer, bad alphabet, asymmetric or out-of-range energies, threshold < 1 */
    GP_UNSUPPORTED_LATTICE = 2, /* box with fewer than 2 or more than 64 sites, or more classes than a u16 holds */
    GP_OUT_OF_MEMORY = 3,
    GP_CUDA_ERROR = 4,          /* gp_last_cuda_error() has the CUDA text */
    GP_RANGE = 5,               /* genotype range outside [0, 2^N) or not aligned to gp_tile() */
    GP_TOO_LARGE = 6            /* problem exceeds the fixed scratch array of an entry point that never allocates */
} gp_status;

typedef struct gp_structures_s gp_structures_t; /* opaque */

/* Contact energies (PAPER.md:77-79 Table 1, integer units :132, :519-525).  e is a HOST array, alphabet*alphabet,
 * row-major, symmetric.  alphabet = 2: e = {E_PP, E_HP, E_HP, E_HH} (HP x10: 0,-10,-10,-23).  alphabet = 20: 0.01 units.
 * A sequence folds iff second_min - min >= threshold (threshold >= 1; 1 = strict uniqueness, R5). */
typedef struct {
    int32_t alphabet;
    const int32_t* e;
    int32_t threshold;
} gp_energies;

/* a0. Host setup: enumerate the Hamiltonian walks of the nx x ny x nz box (nz = 1 for 2D), keep one per
 * point-group class (D directed structures), pair each with its chain reversal (C classes), build contact tables and
 * upload them to the current CUDA device.  With no CUDA device the handle is host-only: the queries below work and
 * compute calls return GP_CUDA_ERROR.  *out is set to NULL on error. */
gp_status gp_structures(int nx, int ny, int nz, gp_structures_t** out);
void gp_structures_free(gp_structures_t* s);
int gp_structures_length(const gp_structures_t* s);            /* N, chain length                       */
uint32_t gp_structures_directed(const gp_structures_t* s);     /* D, scored structures                  */
uint32_t gp_structures_classes(const gp_structures_t* s);      /* C, phenotype ids are 0..C-1           */
uint32_t gp_structures_self_reverse(const gp_structures_t* s); /* classes equal to their own reversal   */
uint64_t gp_structures_walks(const gp_structures_t* s);        /* directed Hamiltonian walks = D * |G|  */
int gp_structures_contacts_per_fold(const gp_structures_t* s); /* NBP = #edges - (N-1)                  */
int gp_structures_features(const gp_structures_t* s);          /* K = N + P: columns of the contraction */
/* Directed structure d: sites[N] (site = x + nx*(y + ny*z)), contacts[2*NBP] monomer pairs i<j, class id.  HOST out
 * arrays, each nullable.  GP_RANGE if d >= D. */
gp_status gp_structures_get(const gp_structures_t* s, uint32_t d, uint8_t* sites, uint8_t* contacts, uint16_t* class_id);

/* Tuning of one handle.  Every setting gives the same results (the parity tests sweep them); they trade tensor work
 * against weight-image traffic and let tests force code paths that small inputs do not reach.
 * gp_structures starts a handle at the defaults below. */
typedef struct {
    int32_t fold_bits;   /* gp_enumerate: low genotype bits kept as contraction columns, 9..22 (default 15)          */
    int32_t sym_bits;    /* gp_enumerate_map*: k, monomers free at each chain end inside one image, 5..11 (default 7) */
    int32_t narrow_rows; /* 1 (default): 64-byte operand rows when the folded contraction has at most 64 columns     */
    int32_t seq_tensor;  /* gp_enumerate_seqs / _seeded: 1 (default) tensor cores where they pay, 2 wherever eligible, 0 never */
} gp_tuning;
gp_status gp_tuning_get(const gp_structures_t* s, gp_tuning* out);
/* GP_INVALID_ARG if a field is out of range (nothing is changed then).  Rebuilds the handle's unit table of
 * gp_enumerate_map_range when sym_bits changes (synchronous host work + one blocking upload). */
gp_status gp_tuning_set(gp_structures_t* s, const gp_tuning* t);

/* Genotype-range granularity of gp_enumerate (g_begin must be a multiple of it). */
uint64_t gp_tile(void);

/* a1-a4. Score genotypes g_begin .. g_begin+g_count-1 (alphabet 2, implicit) on all D directed structures
 * (Eq. 1, :67-69; :530-545), take min / second min / argmin (:552-567) and write d_pheno[g - g_begin] = class of the
 * argmin if second_min - min >= threshold else GP_NULL_PHENO (:81, :573), and, if d_gap is not NULL,
 * d_gap[g - g_begin] = min - second_min (:575; GP_GAP_NONE when D = 1).  The energy matrix never reaches HBM.
 * Runs the tcgen05 int8 contraction.  Errors: GP_INVALID_ARG (energies outside the int8 weight bound, asymmetric),
 * GP_RANGE. */
gp_status gp_enumerate(const gp_structures_t* s, const gp_energies* en, uint64_t g_begin, uint64_t g_count,
                       uint16_t* d_pheno, int16_t* d_gap, void* stream);

/* a1-a4 for the WHOLE map (g = 0 .. 2^N-1, d_pheno and the nullable d_gap hold 2^N entries), same results as
 * gp_enumerate(s, en, 0, 2^N, ...), at half the work: by the reversal identity E(g, rev S) = E(rev g, S) (:391) each
 * genotype is scored on one representative structure per class, and a genotype's list is merged with its reversed
 * genotype's list before the uniqueness test.  executed evaluations = 2^N * C, effective = 2^N * D. */
gp_status gp_enumerate_map(const gp_structures_t* s, const gp_energies* en, uint16_t* d_pheno, int16_t* d_gap,
                           void* stream);

/* The same map in resumable / shardable pieces (the paper's own 110-day job survived by appending results run by run,
 * PAPER.md:206-208, :754, :806).  The map is cut into gp_map_units(s) UNITS.  A unit is the pair of "images" {m, rev m}
 * (one image when m is a palindrome): image m = the 2^(2k) genotypes whose middle N-2k bits equal m, i.e.
 *   g = (hi << (N-k)) | (m << k) | lo,   0 <= hi, lo < 2^k,   k = gp_tuning.sym_bits (clamped to N/2),
 * and rev m = m with its N-2k bits reversed, so that a unit is closed under chain reversal.  Units 0 .. are ordered:
 * first the non-palindromic m < rev m in increasing m, then the palindromic m in increasing m; gp_map_unit reports m
 * and k of a unit so a caller can tell which genotypes a range of units covers.
 * gp_enumerate_map_range scores units unit_first .. unit_first+unit_count-1 and writes the phenotype (and the gap if
 * d_gap is not NULL) of exactly the genotypes of those units, in one of two layouts:
 *   GP_MAP_FULL_STORE: d_pheno / d_gap are the FULL stores of 2^N entries indexed by g; all other entries are left
 *     untouched.  Any partition of 0..gp_map_units-1 into ranges, in any order, on any streams, fills the same store
 *     as gp_enumerate_map.
 *   GP_MAP_COMPACT: d_pheno / d_gap hold gp_map_range_genotypes(s, unit_first, unit_count) entries: the images of the
 *     range one after the other (per unit: image m, then image rev m if the unit is a pair), each as its 2^(2k)
 *     genotypes in the order of the local index (hi << k) | lo.  This is the piece a resumable run appends to its
 *     output, or a rank that holds no full store keeps.
 * Lattices too small for the scheme (N < 10) have one unit that covers the map (k reported as 0; both layouts are
 * then the plain store).  Errors: GP_RANGE if the unit range leaves [0, gp_map_units). */
enum { GP_MAP_FULL_STORE = 0, GP_MAP_COMPACT = 1 };
uint64_t gp_map_units(const gp_structures_t* s);
gp_status gp_map_unit(const gp_structures_t* s, uint64_t unit, uint64_t* m, int* k);
uint64_t gp_map_range_genotypes(const gp_structures_t* s, uint64_t unit_first, uint64_t unit_count);
gp_status gp_enumerate_map_range(const gp_structures_t* s, const gp_energies* en, uint64_t unit_first,
                                 uint64_t unit_count, uint16_t* d_pheno, int16_t* d_gap, int layout, void* stream);

/* Same contract as gp_enumerate, computed by the plain CUDA-core kernel that walks the contact table like the paper's
 * listing (:530-570).  Kept as the in-library cross-check and timing strawman; no alignment requirement. */
gp_status gp_enumerate_simple(const gp_structures_t* s, const gp_energies* en, uint64_t g_begin, uint64_t g_count,
                              uint16_t* d_pheno, int16_t* d_gap, void* stream);

/* a8 / f3. Explicit sequences (the paper's SeqRnd path, :510-516, :762-775; its sampling runs :195-204 Table 3):
 * d_seqs[count][N] letters < alphabet (2..20; a letter outside the alphabet is read as the last letter), e symmetric
 * alphabet x alphabet.  Three kernels, chosen per call, all exact:
 *   - two-letter sequences whose energies fit the int8 weights (same bound as gp_enumerate): tensor cores, the full
 *     2 + N + P feature columns against the per-energy weight image (sequence_kernel);
 *   - any alphabet with (emax - emin) <= 8191 and NBP * (emax - emin) <= 32000 (the seeded 20-letter matrix on every
 *     BASELINE lattice): tensor cores, the P pair energies of a sequence as two int8 limbs against the 0/-1 contact
 *     incidence matrix of the lattice (seq20_kernel), limbs recombined on the TMEM read-out;
 *     by default only on lattices with at least 4096 directed structures (the per-sequence limb rows need a long
 *     structure list to pay; gp_tuning.seq_tensor = 2 takes it wherever eligible);
 *   - everything else, batches under 128 sequences, and gp_tuning.seq_tensor = 0: the CUDA-core kernel.
 * The first call on a handle that needs an image allocates it (cudaMalloc). */
gp_status gp_enumerate_seqs(const gp_structures_t* s, const gp_energies* en, const uint8_t* d_seqs, uint64_t count,
                            uint16_t* d_pheno, int16_t* d_gap, void* stream);
/* a8 / f3. Sequences first..first+count-1 of the counter-based generator of DESIGN.md section 4 over en->alphabet letters
 * (2..20), drawn on chip ("generation of random numbers on the GPU"): alphabet 20 with the seeded matrix is
 * BASELINE config 5, alphabet 2 the random H/P sampling runs (:195-204 Table 3 HP rows) with no sequence upload.  Same
 * kernel choice and same results as gp_enumerate_seqs on gp_seeded_letters(seed, first, count, N, alphabet). */
gp_status gp_enumerate_seeded(const gp_structures_t* s, const gp_energies* en, uint64_t seed, uint64_t first,
                              uint64_t count, uint16_t* d_pheno, int16_t* d_gap, void* stream);
/* Host helpers for the same generator: the seeded 20x20 matrix and sequences. */
gp_status gp_seeded_matrix(uint64_t seed, int32_t* m400);
gp_status gp_seeded_sequences(uint64_t seed, uint64_t first, uint64_t count, int n, uint8_t* seqs);                /* 20 letters */
gp_status gp_seeded_letters(uint64_t seed, uint64_t first, uint64_t count, int n, int alphabet, uint8_t* seqs);   /* 2..20 */

/* a5. Designability (:138): d_hist[c] = #{g : d_pheno[g] = c} for c < n_classes, d_hist[n_classes] = #null. */
gp_status gp_designability(const uint16_t* d_pheno, uint64_t count, uint32_t n_classes, uint64_t* d_hist, void* stream);

/* a6. One-point-mutation neighbourhood (:138-147, Eq. 2) over the FULL store of 2^n_bits entries.  For every non-null
 * g of class p and each of the n_bits flips, q = d_pheno[g ^ (1 << k)]: d_neutral[p] += (q == p),
 * d_deleterious[p] += (q null), d_other[p] += (q another class).  If d_pair_count is not NULL it receives the number
 * of unordered pairs of distinct non-null classes joined by at least one mutation (R11).  rho_p = neutral[p] /
 * (n_bits * hist[p]) etc. are host divisions (R9). */
gp_status gp_robustness(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_neutral,
                        uint64_t* d_deleterious, uint64_t* d_other, uint64_t* d_pair_count, void* stream);

/* a5 + a6 in one sweep: the first pass of the neighbour kernel stages every phenotype on chip anyway, so it also counts
 * them: d_hist (nullable; uint64[n_classes+1]) receives what gp_designability would write, the other outputs what
 * gp_robustness writes, at one read of the store less.  Full store of 2^n_bits entries. */
gp_status gp_reduce_store(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_hist, uint64_t* d_neutral,
                          uint64_t* d_deleterious, uint64_t* d_other, uint64_t* d_pair_count, void* stream);

/* a6 in pieces, for stores sharded over several GPUs on the top genotype bits and for resumable runs.
 * All three ADD into d_neutral / d_deleterious / d_other (uint64[n_classes], zeroed by the caller) and OR into
 * d_pair_bitmap (nullable; gp_pair_bitmap_words(n_classes) uint32 words, zeroed by the caller; bit p*n_classes+q,
 * p < q, is set when classes p and q are joined by a mutation):
 *   gp_robustness_partial: the flips of the n_bits LOCAL bits of a sub-cube store of 2^n_bits entries (a shard, or
 *     the whole map).  tile_bits = 0 takes the default on-chip tile; 4..16 forces a tile of 2^tile_bits entries (any
 *     value gives the same counts; small tiles exercise the multi-pass path on small stores).
 *   gp_robustness_cross: the flip of ONE bit outside the sub-cube: entry i of d_mine and entry i of d_partner (the
 *     shard whose index differs in that bit; may be peer memory) are neighbours; counts go to the classes found in
 *     d_mine only (the partner's owner makes the mirror call).
 * Per-class counts of shards add; bitmaps OR (gp_pair_bitmap_or: d_dst |= d_src); gp_pair_bitmap_count writes the
 * number of set bits (R11) to d_count[0].  gp_robustness = zero + gp_robustness_partial + gp_pair_bitmap_count. */
uint64_t gp_pair_bitmap_words(uint32_t n_classes);
gp_status gp_robustness_partial(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_neutral,
                                uint64_t* d_deleterious, uint64_t* d_other, uint32_t* d_pair_bitmap, int tile_bits,
                                void* stream);
gp_status gp_robustness_cross(const uint16_t* d_mine, const uint16_t* d_partner, uint64_t count, uint32_t n_classes,
                              uint64_t* d_neutral, uint64_t* d_deleterious, uint64_t* d_other, uint32_t* d_pair_bitmap,
                              void* stream);
gp_status gp_pair_bitmap_or(uint32_t* d_dst, const uint32_t* d_src, uint32_t n_classes, void* stream);
gp_status gp_pair_bitmap_count(const uint32_t* d_bitmap, uint32_t n_classes, uint64_t* d_count, void* stream);

/* phi row of target class q (:138-147 Eq. 2 numerators, Figs. 9-12): d_row[p] = number of
 * (genotype, flip) pairs that lead from a genotype of class p to a genotype of class q, p < n_classes (p = q: the
 * neutral count of q); d_row[n_classes] = the same from null genotypes.  phi_pq = d_row[p] / (n_bits * hist[p]).  Full
 * store of 2^n_bits entries. */
gp_status gp_phi_row(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint32_t q, uint64_t* d_row, void* stream);

/* f4. Energy-threshold sweep (PAPER.md:81 "within this threshold ... does not fold", :278, :466; R5) from the stores of
 * ONE threshold-1 enumeration: d_pheno / d_gap as written by gp_enumerate* with threshold = 1 over `count` genotypes.
 * For each thresholds[t] >= 1 (HOST array, n_thresholds <= 16, any order): a genotype folds iff it has a unique ground
 * state and second_min - min = -gap >= thresholds[t].  d_folding[t] = number of folding genotypes, d_hist[t][c]
 * (row length n_classes+1) = designability of class c, last entry = non-folding; the same values gp_enumerate with that
 * threshold followed by gp_designability gives, from one read of the two stores. */
gp_status gp_threshold_sweep(const uint16_t* d_pheno, const int16_t* d_gap, uint64_t count, uint32_t n_classes,
                             const int32_t* thresholds, int n_thresholds, uint64_t* d_folding, uint64_t* d_hist,
                             void* stream);

/* f4 without any allocation: gp_threshold_sweep for callers that must not, or cannot, allocate device memory while
 * they run.  Who that is: a service that hands its whole device-memory budget out at start-up and treats any later
 * cudaMalloc / cudaMallocAsync as a fault; code running under a memory pool that has been capped or switched off;
 * a latency-critical loop where an allocator call (which may take a driver lock or synchronise) is not acceptable.
 * gp_threshold_sweep needs a per-call table of (n_thresholds + 1) * n_classes 64-bit counters and takes it from the
 * stream-ordered pool; this entry point keeps that table in a fixed array that is part of the library image instead.
 *   Same arguments, same results and same asynchrony as gp_threshold_sweep.  The caller still owns every input and
 *   output (d_pheno, d_gap, d_folding, d_hist are device arrays, thresholds a host array).
 *   Limit: (n_thresholds + 1) * n_classes <= GP_SWEEP_STATIC_MAX_BINS (2^19 counters = 4 MiB; enough for 16
 *   thresholds on the 6x6 map's 28 728 classes, or 9 on the 3x3x3 map's 51 704).  Anything larger is refused with
 *   GP_TOO_LARGE and nothing is launched.  The 4 MiB are held on every GPU on which this process loads the library's
 *   device code, from that load until the process exits, whether or not this call is ever made.
 *   Set-up: the first call on each device (with that device current) looks up the device address of the array and
 *   keeps it; make that first call outside any stream capture.  Later calls on that device do no set-up.
 *   It calls no cudaMalloc, cudaMallocAsync, cudaFree or other allocating routine; the table is cleared on `stream`
 *   at the start of every call, so what an earlier call left behind never shows.
 *   All calls in a process share the one array of a device: two calls whose GPU work can overlap (different streams,
 *   or different host threads on different streams) race on it and give wrong counts.  Keep them on one stream, or
 *   order them with events. */
#define GP_SWEEP_STATIC_MAX_BINS (1u << 19)
gp_status gp_threshold_sweep_static(const uint16_t* d_pheno, const int16_t* d_gap, uint64_t count, uint32_t n_classes,
                                    const int32_t* thresholds, int n_thresholds, uint64_t* d_folding, uint64_t* d_hist,
                                    void* stream);

/* a7. Neutral-network components (:19, R12): d_ncomp[p] = number of connected components of {g : pheno = p} under
 * single-bit flips.  Needs 4 bytes of private scratch per genotype; n_bits <= 30.  Synchronises the stream. */
gp_status gp_nn_components(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint32_t* d_ncomp, void* stream);

/* Whole hot path from HOST buffers (the end-to-end call): enumerate [g_begin, g_begin+g_count) (a1-a4), copy the
 * phenotypes to pheno (host, g_count, nullable) and the histogram (a5) to hist (host, n_classes+1).  If rdo is not
 * NULL the range must be an aligned sub-cube (g_count a power of two dividing g_begin, else GP_RANGE); the neighbour
 * pass (a6) then runs over its log2(g_count) mutable bits and rdo (host, 3*n_classes) receives neutral | deleterious |
 * other, pair_count (host, 1, nullable) the number of connected class pairs.  The energy matrix (16 bytes) is the only
 * host input: genotypes are implicit.  Synchronous; its device buffers live in the handle between calls. */
gp_status gp_enumerate_host(const gp_structures_t* s, const gp_energies* en, uint64_t g_begin, uint64_t g_count,
                            uint16_t* pheno, uint64_t* hist, uint64_t* rdo, uint64_t* pair_count);

/* Number of CUDA kernels this library has launched in this process so far (all calls, all streams). */
uint64_t gp_launch_count(void);

/* Per-kernel device timing for bench.py's roofline line.  While enabled, every launch of the kernels below is
 * bracketed by a CUDA event pair on its own stream.  gp_kernel_time waits for those launches, returns the summed device
 * time in milliseconds and the number of launches since the last query, and forgets them.  Off by default.  The sum is
 * over launches, not wall time: the scoring launches of gp_enumerate_map_range alternate between two streams and overlap,
 * and the image builder runs beside the scoring kernel, so their sums can exceed the elapsed time of the call. */
enum { GP_KERNEL_SCORING = 0, GP_KERNEL_IMAGE = 1, GP_KERNEL_HIST = 2, GP_KERNEL_ROBUSTNESS = 3, GP_KERNEL_COUNT = 4 };
void gp_kernel_timing(int enable);
gp_status gp_kernel_time(int which, double* ms_total, uint64_t* launches);

/* The int8 tensor-core peak the scoring kernel is held against ("the build must
 * measure an MMA-only kind::i8 peak itself"), measured on the current device: one CTA per SM issues the scoring
 * kernel's own MMA stream (chains of k_steps tcgen05.mma kind::i8 M128 x N128 x K32 into four TMEM accumulators,
 * operands in shared memory, 64-byte rows for k_steps <= 2 else 128-byte rows) for about `seconds` with no TMA traffic,
 * no TMEM read-out and no epilogue.  *ops_per_s = int8 multiply-adds x 2 per second over all SMs; *clk_per_mma (nullable) =
 * SM clocks per MMA (64 nominal); *sm_mhz (nullable) = the SM clock it ran at (clock64 / event time).  Synchronous, on
 * the default stream. */
gp_status gp_probe_i8_peak(int k_steps, double seconds, double* ops_per_s, double* clk_per_mma, double* sm_mhz);

const char* gp_strerror(gp_status st);
const char* gp_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* GPMAP_H */
