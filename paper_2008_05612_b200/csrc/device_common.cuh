// device_common.cuh — error plumbing and small helpers shared by libgpmap's .cu files (private; not used by oracle/).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "gpmap_internal.h"

void gp_set_cuda_error(cudaError_t e, const char* where);
void gp_count_launches(unsigned n);  // feeds gp_launch_count(): every kernel launch of the library is counted
// Optional per-kernel device timing (gp_kernel_timing / gp_kernel_time): CUDA events around one launch on its stream.
// gp_time_begin returns a token naming ITS event pair (0 = timing off); gp_time_end records the end on that pair, so
// calls that run concurrently on one handle from several threads cannot close each other's pairs.
uint64_t gp_time_begin(int which, cudaStream_t st);
void gp_time_end(int which, uint64_t token, cudaStream_t st);

#define GP_CUDA(call)                                 \
    do {                                              \
        cudaError_t e_ = (call);                      \
        if (e_ != cudaSuccess) {                      \
            gp_set_cuda_error(e_, #call);             \
            return e_ == cudaErrorMemoryAllocation ? GP_OUT_OF_MEMORY : GP_CUDA_ERROR; \
        }                                             \
    } while (0)

// Per-call working memory from the device's stream-ordered pool that finds its way back on EVERY exit path of a call
// (GP_CUDA returns early).  release() is the normal end: freed in stream order on the call's stream.  A destructor that
// still holds the block is an error path: other streams of the call (image builder, combine) may have work pending on
// it, so the device is drained before the block goes back.
struct gp_pool_mem {
    void* p = nullptr;
    cudaStream_t st = nullptr;
    gp_pool_mem() = default;
    gp_pool_mem(const gp_pool_mem&) = delete;
    gp_pool_mem& operator=(const gp_pool_mem&) = delete;
    cudaError_t alloc(size_t bytes, cudaStream_t s) { st = s; return cudaMallocAsync(&p, bytes, s); }
    template <class T> T* as() const { return static_cast<T*>(p); }
    cudaError_t release() {
        cudaError_t e = p ? cudaFreeAsync(p, st) : cudaSuccess;
        p = nullptr;
        return e;
    }
    ~gp_pool_mem() {
        if (!p) return;
        cudaDeviceSynchronize();
        cudaFreeAsync(p, st);
    }
};

// Validated alphabet-2 energies in the form the kernels use:
//   E(g,S) = a*NBP + lin * sum_k c_k(S) h_k + quad * #HH-contacts,  lin = b - a, quad = c - 2b + a
struct gp_hp_params {
    int32_t a, lin, quad, threshold;
};
gp_status gp_check_hp(const gp_structures_s* s, const gp_energies* en, gp_hp_params* out);

// 64-bit counter-based generator of DESIGN.md section 4 (splitmix finaliser)
__host__ __device__ inline uint64_t gp_mix64(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
__host__ __device__ inline uint64_t gp_draw(uint64_t seed, uint64_t ctr) {
    return gp_mix64(seed + (ctr + 1) * 0x9E3779B97F4A7C15ULL);
}
// letter k of sequence seq over `alphabet` letters: floor(alphabet * hi32(draw) / 2^32); alphabet 2 = the top bit, 1 = H
__host__ __device__ inline uint32_t gp_letter(uint64_t seed, uint64_t seq, int k, uint32_t alphabet) {
    uint64_t u = gp_draw(seed, seq * 64 + (uint64_t)k);
    return (uint32_t)(((u >> 32) * alphabet) >> 32);
}
__host__ __device__ inline uint32_t gp_letter20(uint64_t seed, uint64_t seq, int k) { return gp_letter(seed, seq, k, 20u); }

// scoring_tc.cu
gp_status gp_launch_scoring_tc(const gp_structures_s* s, const gp_hp_params& hp, uint64_t g_begin, uint64_t g_count,
                               uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st);
// d_seqs = NULL: the two-letter sequences first .. first+count-1 of the seeded stream, drawn on chip
gp_status gp_launch_sequences_tc(const gp_structures_s* s, const gp_hp_params& hp, const uint8_t* d_seqs, uint64_t seed,
                                 uint64_t first, uint64_t count, uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st);
// scoring_seq20.cu
gp_status gp_launch_seq20_tc(const gp_structures_s* s, const gp_energies* en, int seeded, const uint8_t* d_seqs, uint64_t seed,
                             uint64_t first, uint64_t count, uint16_t* d_pheno, int16_t* d_gap, cudaStream_t st);
