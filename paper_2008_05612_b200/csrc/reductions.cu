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
    for (uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (uint64_t)gridDim.x * blockDim.x) {
        uint4 x = __ldg(v + i);
        uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
        for (int j = 0; j < 4; j++) {
#pragma unroll
            for (int h = 0; h < 2; h++) {
                uint32_t p = h ? (w[j] >> 16) : (w[j] & 0xFFFFu);
                if (p == NULLP) nulls++;
                else if (p < C) {
                    if (use_smem) atomicAdd(&sh[p], 1u);
                    else atomicAdd(&hist[p], 1ULL);
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
// a6. Neighbour pass.  A block owns 2^TB consecutive genotypes staged in shared memory: flips of the low TB bits are
// served on chip; each higher bit k is one coalesced, vectorised read of the partner segment base ^ 2^k.  Counts are
// packed per genotype and flushed per class with 64-bit reductions; distinct-class pairs go to a C x C bitmap.
// ---------------------------------------------------------------------------------------------------------------
constexpr int TB = 13;              // 2^13 genotypes = 16 KB per staged segment
constexpr int RTHREADS = 1024;      // 8 genotypes per thread

struct RobArgs {
    const uint16_t* pheno;
    int n_bits;
    uint32_t C;
    unsigned long long *R, *Dl, *O;
    uint32_t* bitmap;  // nullable; bit (min*C + max)
};

__device__ __forceinline__ void note_pair(const RobArgs& a, uint32_t p, uint32_t q) {
    uint32_t lo = min(p, q), hi = max(p, q);
    uint64_t bit = (uint64_t)lo * a.C + hi;
    uint32_t* w = a.bitmap + (bit >> 5);
    uint32_t m = 1u << (bit & 31);
    if (!(__ldg(w) & m) && !(*(volatile uint32_t*)w & m)) atomicOr(w, m);
}

__global__ void __launch_bounds__(RTHREADS) robustness_kernel(RobArgs a) {
    __shared__ __align__(16) uint16_t seg[1 << TB];
    const int tb = min(TB, a.n_bits);
    const uint64_t seg_len = 1ULL << tb;
    const uint64_t n_seg = 1ULL << (a.n_bits - tb);
    const int per_thread = (int)((seg_len + RTHREADS - 1) / RTHREADS);  // 8 when tb = 13
    for (uint64_t s = blockIdx.x; s < n_seg; s += gridDim.x) {
        const uint64_t base = s << tb;
        __syncthreads();
        if (seg_len >= 8 * RTHREADS) {
            const uint4* src = reinterpret_cast<const uint4*>(a.pheno + base);
            reinterpret_cast<uint4*>(seg)[threadIdx.x] = __ldg(src + threadIdx.x);
        } else {
            for (uint32_t i = threadIdx.x; i < seg_len; i += RTHREADS) seg[i] = a.pheno[base + i];
        }
        __syncthreads();
        // this thread's genotypes: local ids l0 .. l0+per_thread-1 (contiguous, so high-bit partners are one vector)
        const uint32_t l0 = threadIdx.x * per_thread;
        if (l0 >= seg_len) continue;
        uint32_t mine[8], r[8], dl[8], o[8];
#pragma unroll
        for (int j = 0; j < 8; j++) { mine[j] = (j < per_thread) ? seg[l0 + j] : NULLP; r[j] = dl[j] = o[j] = 0; }
        bool any = false;
#pragma unroll
        for (int j = 0; j < 8; j++) any |= (mine[j] != NULLP);
        // low bits: on chip
        for (int k = 0; k < tb; k++) {
#pragma unroll
            for (int j = 0; j < 8; j++) {
                if (j < per_thread && mine[j] != NULLP) {
                    uint32_t q = seg[(l0 + j) ^ (1u << k)];
                    if (q == mine[j]) r[j]++;
                    else if (q == NULLP) dl[j]++;
                    else { o[j]++; if (a.bitmap) note_pair(a, mine[j], q); }
                }
            }
        }
        // high bits: partner segment, one 16-byte load per thread per bit (skipped when all 8 are null)
        for (int k = tb; k < a.n_bits; k++) {
            if (!any) break;
            const uint16_t* part = a.pheno + (base ^ (1ULL << k)) + l0;
            uint32_t q8[8];
            if (per_thread == 8) {
                uint4 x = __ldg(reinterpret_cast<const uint4*>(part));
                q8[0] = x.x & 0xFFFF; q8[1] = x.x >> 16; q8[2] = x.y & 0xFFFF; q8[3] = x.y >> 16;
                q8[4] = x.z & 0xFFFF; q8[5] = x.z >> 16; q8[6] = x.w & 0xFFFF; q8[7] = x.w >> 16;
            } else {
#pragma unroll
                for (int j = 0; j < 8; j++) q8[j] = (j < per_thread) ? part[j] : NULLP;
            }
#pragma unroll
            for (int j = 0; j < 8; j++) {
                if (j < per_thread && mine[j] != NULLP) {
                    uint32_t q = q8[j];
                    if (q == mine[j]) r[j]++;
                    else if (q == NULLP) dl[j]++;
                    else { o[j]++; if (a.bitmap) note_pair(a, mine[j], q); }
                }
            }
        }
        // flush, merging runs of equal class among this thread's 8 genotypes
#pragma unroll
        for (int j = 0; j < 8; j++) {
            if (mine[j] == NULLP) continue;
            if (j < 7 && mine[j + 1] == mine[j]) { r[j + 1] += r[j]; dl[j + 1] += dl[j]; o[j + 1] += o[j]; continue; }
            if (r[j]) atomicAdd(&a.R[mine[j]], (unsigned long long)r[j]);
            if (dl[j]) atomicAdd(&a.Dl[mine[j]], (unsigned long long)dl[j]);
            if (o[j]) atomicAdd(&a.O[mine[j]], (unsigned long long)o[j]);
        }
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
    gp_time_begin(GP_KERNEL_HIST, st);
    hist_kernel<<<grid, 1024, use_smem ? smem : 0, st>>>(d_pheno, count, n_classes,
                                                         reinterpret_cast<unsigned long long*>(d_hist), use_smem);
    gp_time_end(GP_KERNEL_HIST, st);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    return GP_OK;
}

extern "C" gp_status gp_robustness(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint64_t* d_neutral,
                                   uint64_t* d_deleterious, uint64_t* d_other, uint64_t* d_pair_count, void* stream) {
    if (!d_pheno || !d_neutral || !d_deleterious || !d_other) return GP_INVALID_ARG;
    if (n_bits < 1 || n_bits > 40 || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (((uintptr_t)d_pheno & 15) != 0) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t cb = (size_t)n_classes * sizeof(uint64_t);
    GP_CUDA(cudaMemsetAsync(d_neutral, 0, cb, st));
    GP_CUDA(cudaMemsetAsync(d_deleterious, 0, cb, st));
    GP_CUDA(cudaMemsetAsync(d_other, 0, cb, st));
    RobArgs a;
    a.pheno = d_pheno; a.n_bits = n_bits; a.C = n_classes;
    a.R = reinterpret_cast<unsigned long long*>(d_neutral);
    a.Dl = reinterpret_cast<unsigned long long*>(d_deleterious);
    a.O = reinterpret_cast<unsigned long long*>(d_other);
    a.bitmap = nullptr;
    uint64_t n_words = 0;
    if (d_pair_count) {
        n_words = ((uint64_t)n_classes * n_classes + 31) / 32;
        GP_CUDA(cudaMallocAsync(&a.bitmap, n_words * 4, st));
        GP_CUDA(cudaMemsetAsync(a.bitmap, 0, n_words * 4, st));
        GP_CUDA(cudaMemsetAsync(d_pair_count, 0, sizeof(uint64_t), st));
    }
    const uint64_t n_seg = 1ULL << (n_bits > TB ? n_bits - TB : 0);
    const uint64_t cap = (uint64_t)sm_count() * 2;
    gp_time_begin(GP_KERNEL_ROBUSTNESS, st);
    robustness_kernel<<<(unsigned)(n_seg < cap ? n_seg : cap), RTHREADS, 0, st>>>(a);
    gp_time_end(GP_KERNEL_ROBUSTNESS, st);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(1);
    if (d_pair_count) {
        popcount_kernel<<<(unsigned)((n_words + 255) / 256 < 4096 ? (n_words + 255) / 256 : 4096), 256, 0, st>>>(
            a.bitmap, n_words, reinterpret_cast<unsigned long long*>(d_pair_count));
        GP_CUDA(cudaGetLastError());
        gp_count_launches(1);
        GP_CUDA(cudaFreeAsync(a.bitmap, st));
    }
    return GP_OK;
}

extern "C" gp_status gp_nn_components(const uint16_t* d_pheno, int n_bits, uint32_t n_classes, uint32_t* d_ncomp,
                                      void* stream) {
    if (!d_pheno || !d_ncomp || n_classes == 0 || n_classes >= NULLP) return GP_INVALID_ARG;
    if (n_bits < 1 || n_bits > 30) return GP_INVALID_ARG;
    cudaStream_t st = (cudaStream_t)stream;
    const uint64_t n = 1ULL << n_bits;
    uint32_t* parent = nullptr;
    GP_CUDA(cudaMallocAsync(&parent, n * sizeof(uint32_t), st));
    GP_CUDA(cudaMemsetAsync(d_ncomp, 0, (size_t)n_classes * sizeof(uint32_t), st));
    const unsigned grid = (unsigned)((n + 255) / 256 < (uint64_t)sm_count() * 16 ? (n + 255) / 256 : (uint64_t)sm_count() * 16);
    uf_init_kernel<<<grid, 256, 0, st>>>(parent, n);
    uf_link_kernel<<<grid, 256, 0, st>>>(d_pheno, parent, n_bits);
    uf_count_kernel<<<grid, 256, 0, st>>>(d_pheno, parent, n, n_classes, d_ncomp);
    GP_CUDA(cudaGetLastError());
    gp_count_launches(3);
    GP_CUDA(cudaFreeAsync(parent, st));
    GP_CUDA(cudaStreamSynchronize(st));
    return GP_OK;
}
