// scoring_simple.cu — CUDA-core scorer for any alphabet: gp_enumerate_simple (implicit HP genotypes, the in-library
// cross-check of the tensor-core path), gp_enumerate_seqs (the paper's SeqRnd path) and
// gp_enumerate_seeded (20-letter variant, a8).
//
// One thread per sequence, like the paper's kernel (:193, :487-578), but the per-contact matrix look-up of the
// listing (:537-545) is hoisted: each thread first gathers the energies of all P monomer pairs that can ever touch
// (pe[p] = e[s_i][s_j], staged in shared memory, 20x20 matrix in shared memory too), then a structure is an NBP-term
// sum of pe[] entries addressed by the structure's pair indices, which all threads of a block read as broadcasts.
// min / second-min / argmin use the strict '<' updates of :552-567 with true-minimum initialisation (R6).
#include "device_common.cuh"

namespace {

enum { SRC_BITS = 0, SRC_SEQS = 1, SRC_SEEDED = 2 };
constexpr int CHUNK = 256;  // structures staged per shared-memory refill

struct SimpleArgs {
    const uint16_t* pairidx;  // D * NBP
    const uint8_t* pair_ij;   // P * 2
    const uint16_t* class_of;
    const uint8_t* seqs;
    uint16_t* pheno;
    int16_t* gap;
    uint64_t first, count, seed;
    uint32_t D;
    int N, NBP, P, alphabet, threshold, emax;
};

// Two sequences per thread: the pair energies are stored as non-negative 16-bit costs (emax - e) packed two to a word,
// so one shared-memory load and one integer add serve both sequences, with no carry between the halves
// (NBP * (emax - emin) < 2^16 is checked by the launcher).  The minimum energy is the maximum cost.
template <int SRC>
__global__ void __launch_bounds__(128) score_simple_kernel(SimpleArgs a, const int16_t* __restrict__ e_dev) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int BD = blockDim.x, tid = threadIdx.x;
    uint32_t* pe = reinterpret_cast<uint32_t*>(smem_raw);                 // [P][BD] packed costs of the thread's two sequences
    uint16_t* sidx = reinterpret_cast<uint16_t*>(pe + (size_t)a.P * BD);  // [CHUNK][NBP] pair index * BD
    int16_t* em = reinterpret_cast<int16_t*>(sidx + (size_t)CHUNK * a.NBP);  // [alphabet^2]
    uint8_t* let = reinterpret_cast<uint8_t*>(em + 400);                  // [N][2 BD]
    uint8_t* pij = let + (size_t)a.N * 2 * BD;                            // [P][2]

    for (int i = tid; i < a.alphabet * a.alphabet; i += BD) em[i] = e_dev[i];
    for (int i = tid; i < 2 * a.P; i += BD) pij[i] = a.pair_ij[i];

    const uint64_t n_tiles = (a.count + 2 * BD - 1) / (2 * BD);
    for (uint64_t tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const uint64_t q[2] = {tile * 2 * BD + tid, tile * 2 * BD + BD + tid};  // sequence numbers within the call
        const bool live[2] = {q[0] < a.count, q[1] < a.count};
        __syncthreads();
#pragma unroll
        for (int h = 0; h < 2; h++)
            for (int k = 0; k < a.N; k++) {
                uint32_t l = 0;
                if (live[h]) {
                    if (SRC == SRC_BITS) l = (uint32_t)(((a.first + q[h]) >> k) & 1ULL);
                    else if (SRC == SRC_SEQS) l = min((uint32_t)a.seqs[q[h] * a.N + k], (uint32_t)a.alphabet - 1u);  // outside the alphabet = the last letter
                    else l = gp_letter(a.seed, a.first + q[h], k, (uint32_t)a.alphabet);
                }
                let[(k * 2 + h) * BD + tid] = (uint8_t)l;
            }
        for (int p = 0; p < a.P; p++) {
            const int i = pij[2 * p], j = pij[2 * p + 1];
            const uint32_t c0 = (uint32_t)(a.emax - em[let[(i * 2) * BD + tid] * a.alphabet + let[(j * 2) * BD + tid]]);
            const uint32_t c1 = (uint32_t)(a.emax - em[let[(i * 2 + 1) * BD + tid] * a.alphabet + let[(j * 2 + 1) * BD + tid]]);
            pe[p * BD + tid] = c0 | (c1 << 16);
        }
        int32_t M1[2] = {-1, -1}, M2[2] = {-1, -1};  // largest and second-largest cost (with multiplicity)
        uint32_t arg[2] = {0, 0};
        for (uint32_t d0 = 0; d0 < a.D; d0 += CHUNK) {
            const uint32_t nd = min((uint32_t)CHUNK, a.D - d0);
            __syncthreads();
            for (uint32_t i = tid; i < nd * a.NBP; i += BD) sidx[i] = (uint16_t)(a.pairidx[(size_t)d0 * a.NBP + i] * BD);
            __syncthreads();
            const uint32_t* mine = pe + tid;
            for (uint32_t c = 0; c < nd; c++) {
                const uint16_t* ix = sidx + c * a.NBP;
                uint32_t S = 0;
                for (int k = 0; k < a.NBP; k++) S += mine[ix[k]];
#pragma unroll
                for (int h = 0; h < 2; h++) {
                    const int32_t cost = (int32_t)(h ? (S >> 16) : (S & 0xFFFFu));
                    if (cost > M1[h]) { M2[h] = M1[h]; M1[h] = cost; arg[h] = d0 + c; }
                    else if (cost > M2[h]) { M2[h] = cost; }
                }
            }
        }
#pragma unroll
        for (int h = 0; h < 2; h++)
            if (live[h]) {
                const bool folds = (M2[h] < 0) || (M1[h] - M2[h] >= a.threshold);
                a.pheno[q[h]] = folds ? a.class_of[arg[h]] : (uint16_t)GP_NULL_PHENO;
                if (a.gap) a.gap[q[h]] = (int16_t)((M2[h] < 0) ? GP_GAP_NONE : max(M2[h] - M1[h], -32768));
            }
    }
}

gp_status launch_simple(const gp_structures_s* s, const gp_energies* en, int src, const uint8_t* d_seqs, uint64_t seed,
                        uint64_t first, uint64_t count, uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st) {
    if (!s || !en || !en->e || !d_pheno) return GP_INVALID_ARG;
    if (en->alphabet < 2 || en->alphabet > 20 || en->threshold < 1) return GP_INVALID_ARG;
    if (src == SRC_SEQS && !d_seqs) return GP_INVALID_ARG;
    if (s->device < 0) { gp_set_cuda_error(cudaErrorNoDevice, "handle has no device tables"); return GP_CUDA_ERROR; }
    const int A = en->alphabet;
    int16_t h_e[400];
    int32_t emax = INT32_MIN, emin = INT32_MAX;
    for (int i = 0; i < A; i++)
        for (int j = 0; j < A; j++) {
            int32_t v = en->e[i * A + j];
            if (v != en->e[j * A + i]) return GP_INVALID_ARG;
            if ((long long)v * s->NBP > 32767 || (long long)v * s->NBP < -32767) return GP_INVALID_ARG;
            h_e[i * A + j] = (int16_t)v;
            emax = v > emax ? v : emax;
            emin = v < emin ? v : emin;
        }
    if ((long long)(emax - emin) * s->NBP > 65535 || (size_t)s->P * 128 > 65535) return GP_INVALID_ARG;  // packed 16-bit costs / offsets
    if (count == 0) return GP_OK;
    gp_pool_mem e_mem;
    GP_CUDA(e_mem.alloc(sizeof(h_e), st));
    int16_t* d_e = e_mem.as<int16_t>();
    GP_CUDA(cudaMemcpyAsync(d_e, h_e, sizeof(int16_t) * A * A, cudaMemcpyHostToDevice, st));  // pageable: staged before return

    SimpleArgs a;
    a.pairidx = s->d_pairidx; a.pair_ij = s->d_pair_ij; a.class_of = s->d_class_of; a.seqs = d_seqs;
    a.pheno = d_pheno; a.gap = d_gap; a.first = first; a.count = count; a.seed = seed;
    a.D = s->D; a.N = s->N; a.NBP = s->NBP; a.P = s->P; a.alphabet = A; a.threshold = en->threshold; a.emax = emax;
    const int BD = 128;
    size_t smem = (size_t)s->P * BD * 4 + (size_t)CHUNK * s->NBP * 2 + 800 + (size_t)s->N * 2 * BD + (size_t)s->P * 2 + 16;
    int dev = 0, sms = 0;
    GP_CUDA(cudaGetDevice(&dev));
    GP_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    uint64_t tiles = (count + 2 * BD - 1) / (2 * BD);
    int per_sm = (int)(200 * 1024 / smem);
    if (per_sm < 1) per_sm = 1;
    if (per_sm > 8) per_sm = 8;
    unsigned grid = (unsigned)(tiles < (uint64_t)sms * per_sm ? tiles : (uint64_t)sms * per_sm);
    void (*k)(SimpleArgs, const int16_t*) = src == SRC_BITS ? score_simple_kernel<SRC_BITS>
                                             : src == SRC_SEQS ? score_simple_kernel<SRC_SEQS>
                                                               : score_simple_kernel<SRC_SEEDED>;
    GP_CUDA(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    k<<<grid, BD, smem, st>>>(a, d_e);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    GP_CUDA(e_mem.release());
    return GP_OK;
}

}  // namespace

extern "C" gp_status gp_enumerate_simple(const gp_structures_t* s, const gp_energies* en, uint64_t g_begin,
                                         uint64_t g_count, uint16_t* d_pheno, int16_t* d_gap, void* stream) {
    if (!s || !en || en->alphabet != 2) return GP_INVALID_ARG;
    const uint64_t total = s->N >= 64 ? ~0ULL : (1ULL << s->N);
    if (g_begin > total || g_count > total - g_begin) return GP_RANGE;
    return launch_simple(s, en, SRC_BITS, nullptr, 0, g_begin, g_count, d_pheno, d_gap, (cudaStream_t)stream);
}

// any-alphabet sequences: tensor cores (scoring_seq20.cu) when the handle's tuning allows, the batch is worth a launch and
// the energies are eligible; the CUDA-core kernel otherwise.  Arguments are validated here for both.
static gp_status seqs_any_alphabet(const gp_structures_t* s, const gp_energies* en, int seeded, const uint8_t* d_seqs,
                                   uint64_t seed, uint64_t first, uint64_t count, uint16_t* d_pheno, int16_t* d_gap,
                                   cudaStream_t st) {
    // auto (1): the limb kernel pays a per-sequence row build that only a long structure list amortises (4x4, D = 69: the
    // CUDA-core kernel is 3x faster; 6x6 / 3x3x3: the tensor cores are 20x faster)
    const bool want_tc = s && (s->tuning.seq_tensor == 2 || (s->tuning.seq_tensor == 1 && s->D >= 4096));
    if (want_tc && en && en->e && d_pheno && count >= 128 && s->device >= 0 && en->alphabet >= 2 &&
        en->alphabet <= 20 && en->threshold >= 1 && (seeded || d_seqs != nullptr)) {
        bool symmetric = true;
        for (int i = 0; i < en->alphabet && symmetric; i++)
            for (int j = 0; j < i; j++)
                if (en->e[i * en->alphabet + j] != en->e[j * en->alphabet + i]) { symmetric = false; break; }
        if (symmetric) {
            gp_status stt = gp_launch_seq20_tc(s, en, seeded, d_seqs, seed, first, count, d_pheno, d_gap, st);
            if (stt != GP_UNSUPPORTED_LATTICE) return stt;
        }
    }
    return launch_simple(s, en, seeded ? SRC_SEEDED : SRC_SEQS, d_seqs, seed, first, count, d_pheno, d_gap, st);
}

extern "C" gp_status gp_enumerate_seqs(const gp_structures_t* s, const gp_energies* en, const uint8_t* d_seqs,
                                       uint64_t count, uint16_t* d_pheno, int16_t* d_gap, void* stream) {
    // two-letter sequences whose energies fit the int8 weights go to the tensor cores (sequence_kernel)
    gp_hp_params hp;
    if (s && s->tuning.seq_tensor && en && en->alphabet == 2 && d_seqs && d_pheno && count >= 256 && s->device >= 0 &&
        gp_check_hp(s, en, &hp) == GP_OK) {
        gp_status st = gp_launch_sequences_tc(s, hp, d_seqs, 0, 0, count, d_pheno, d_gap, (cudaStream_t)stream);
        if (st != GP_UNSUPPORTED_LATTICE) return st;
    }
    return seqs_any_alphabet(s, en, 0, d_seqs, 0, 0, count, d_pheno, d_gap, (cudaStream_t)stream);
}

extern "C" gp_status gp_enumerate_seeded(const gp_structures_t* s, const gp_energies* en, uint64_t seed, uint64_t first,
                                         uint64_t count, uint16_t* d_pheno, int16_t* d_gap, void* stream) {
    // seeded H/P sequences whose energies fit the int8 weights: sequence_kernel draws its feature rows from the counter
    gp_hp_params hp;
    if (s && s->tuning.seq_tensor && en && en->alphabet == 2 && d_pheno && count >= 256 && s->device >= 0 &&
        gp_check_hp(s, en, &hp) == GP_OK) {
        gp_status st = gp_launch_sequences_tc(s, hp, nullptr, seed, first, count, d_pheno, d_gap, (cudaStream_t)stream);
        if (st != GP_UNSUPPORTED_LATTICE) return st;
    }
    return seqs_any_alphabet(s, en, 1, nullptr, seed, first, count, d_pheno, d_gap, (cudaStream_t)stream);
}
