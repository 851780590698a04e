// api.cu — C-ABI entry points of libgpmap (include/gpmap.h): argument checks, handle lifetime, dispatch to the kernels.
#include <cstdio>
#include <cstring>
#include <atomic>
#include <mutex>
#include <vector>
#include <new>

#include "device_common.cuh"

static thread_local char g_cuda_error[512] = "";

void gp_set_cuda_error(cudaError_t e, const char* where) {
    snprintf(g_cuda_error, sizeof(g_cuda_error), "%s: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e), where);
}

extern "C" const char* gp_last_cuda_error(void) { return g_cuda_error; }

static std::atomic<uint64_t> g_launches{0};
void gp_count_launches(unsigned n) { g_launches.fetch_add(n, std::memory_order_relaxed); }
extern "C" uint64_t gp_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

// ---- optional per-kernel timing: one CUDA event pair per launch, on the launching stream ----
namespace {
struct EvPair { cudaEvent_t a, b; uint64_t serial; bool ended; };
std::mutex g_time_mu;
bool g_time_on = false;
uint64_t g_time_serial = 0;
std::vector<EvPair> g_time_ev[GP_KERNEL_COUNT];
}  // namespace

uint64_t gp_time_begin(int which, cudaStream_t st) {
    if (!g_time_on) return 0;
    std::lock_guard<std::mutex> lk(g_time_mu);
    EvPair p;
    if (cudaEventCreate(&p.a) != cudaSuccess) return 0;
    if (cudaEventCreate(&p.b) != cudaSuccess) { cudaEventDestroy(p.a); return 0; }
    cudaEventRecord(p.a, st);
    p.serial = ++g_time_serial;
    p.ended = false;
    g_time_ev[which].push_back(p);
    return p.serial;
}
void gp_time_end(int which, uint64_t token, cudaStream_t st) {
    if (!token) return;
    std::lock_guard<std::mutex> lk(g_time_mu);
    std::vector<EvPair>& v = g_time_ev[which];
    for (size_t i = v.size(); i-- > 0;)   // the pair is near the back; it is gone if gp_kernel_time ran in between
        if (v[i].serial == token) { cudaEventRecord(v[i].b, st); v[i].ended = true; return; }
}
extern "C" void gp_kernel_timing(int enable) {
    std::lock_guard<std::mutex> lk(g_time_mu);
    g_time_on = enable != 0;
}
extern "C" gp_status gp_kernel_time(int which, double* ms_total, uint64_t* launches) {
    if (which < 0 || which >= GP_KERNEL_COUNT || !ms_total || !launches) return GP_INVALID_ARG;
    std::lock_guard<std::mutex> lk(g_time_mu);
    double tot = 0;
    uint64_t n = 0;
    gp_status st = GP_OK;
    for (EvPair& p : g_time_ev[which]) {
        if (p.ended) {   // a pair whose launch is still between begin and end on another thread is dropped, not waited for
            float ms = 0;
            cudaError_t e = cudaEventSynchronize(p.b);
            if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, p.a, p.b);
            if (e == cudaSuccess) { tot += ms; n++; }
            else { gp_set_cuda_error(e, "gp_kernel_time"); st = GP_CUDA_ERROR; }
        }
        cudaEventDestroy(p.a);
        cudaEventDestroy(p.b);
    }
    g_time_ev[which].clear();
    *ms_total = tot;
    *launches = n;
    return st;
}

extern "C" const char* gp_strerror(gp_status st) {
    switch (st) {
        case GP_OK: return "ok";
        case GP_INVALID_ARG: return "invalid argument";
        case GP_UNSUPPORTED_LATTICE: return "unsupported lattice";
        case GP_OUT_OF_MEMORY: return "out of memory";
        case GP_CUDA_ERROR: return "CUDA error (see gp_last_cuda_error)";
        case GP_RANGE: return "genotype range or index out of range / misaligned";
        case GP_TOO_LARGE: return "problem larger than the fixed scratch array of this no-allocation entry point";
    }
    return "unknown status";
}

gp_status gp_upload_tables(gp_structures_s* s) {
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        s->device = -1;  // host-only handle
        return GP_OK;
    }
    GP_CUDA(cudaGetDevice(&s->device));
    {   // the reductions take their scratch (pair bitmap, union-find parents) from the stream-ordered pool: keep freed
        // blocks in the pool instead of handing them back to the driver at every synchronisation
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, s->device) == cudaSuccess) {
            uint64_t keep = ~0ULL;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
        cudaGetLastError();
    }
    GP_CUDA(cudaMalloc(&s->d_contacts, s->contacts.size()));
    GP_CUDA(cudaMemcpy(s->d_contacts, s->contacts.data(), s->contacts.size(), cudaMemcpyHostToDevice));
    GP_CUDA(cudaMalloc(&s->d_class_of, s->class_of.size() * sizeof(uint16_t)));
    GP_CUDA(cudaMemcpy(s->d_class_of, s->class_of.data(), s->class_of.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
    std::vector<uint16_t> pidx(s->contacts.size() / 2);
    for (size_t k = 0; k < pidx.size(); k++)
        pidx[k] = (uint16_t)s->pair_index[(size_t)s->contacts[2 * k] * s->N + s->contacts[2 * k + 1]];
    GP_CUDA(cudaMalloc(&s->d_pairidx, pidx.size() * sizeof(uint16_t)));
    GP_CUDA(cudaMemcpy(s->d_pairidx, pidx.data(), pidx.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
    std::vector<uint8_t> ij((size_t)s->P * 2);
    for (int i = 0; i < s->N; i++)
        for (int j = 0; j < s->N; j++) {
            int p = s->pair_index[(size_t)i * s->N + j];
            if (p >= 0) { ij[2 * p] = (uint8_t)i; ij[2 * p + 1] = (uint8_t)j; }
        }
    GP_CUDA(cudaMalloc(&s->d_pair_ij, ij.size()));
    GP_CUDA(cudaMemcpy(s->d_pair_ij, ij.data(), ij.size(), cudaMemcpyHostToDevice));
    // one representative (smallest directed index) per class; classes with two members first
    {
        std::vector<uint32_t> members(s->C, 0), rep(s->C, 0xFFFFFFFFu);
        for (uint32_t d = 0; d < s->D; d++) {
            members[s->class_of[d]]++;
            if (rep[s->class_of[d]] == 0xFFFFFFFFu) rep[s->class_of[d]] = d;
        }
        std::vector<uint32_t> order;
        for (uint32_t c = 0; c < s->C; c++) if (members[c] == 2) order.push_back(rep[c]);
        const uint32_t n_nsr = (uint32_t)order.size();
        s->n_snap = (n_nsr + 127) / 128;
        order.resize((size_t)s->n_snap * 128, 0xFFFFFFFFu);
        for (uint32_t c = 0; c < s->C; c++) if (members[c] == 1) order.push_back(rep[c]);
        s->D_sym = (uint32_t)order.size();
        const size_t row = (size_t)s->NBP * 2;
        std::vector<uint8_t> csym(order.size() * row, 0);
        std::vector<uint16_t> ksym(order.size(), (uint16_t)GP_NULL_PHENO);
        for (size_t k = 0; k < order.size(); k++)
            if (order[k] != 0xFFFFFFFFu) {
                memcpy(&csym[k * row], &s->contacts[order[k] * row], row);
                ksym[k] = s->class_of[order[k]];
            }
        GP_CUDA(cudaMalloc(&s->d_contacts_sym, csym.size() ? csym.size() : 1));
        GP_CUDA(cudaMemcpy(s->d_contacts_sym, csym.data(), csym.size(), cudaMemcpyHostToDevice));
        GP_CUDA(cudaMalloc(&s->d_class_sym, ksym.size() * sizeof(uint16_t)));
        GP_CUDA(cudaMemcpy(s->d_class_sym, ksym.data(), ksym.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
    }
    return gp_build_map_units(s);
}

void gp_release_device(gp_structures_s* s) {
    if (s->device < 0) return;
    cudaFree(s->d_contacts);
    cudaFree(s->d_class_of);
    cudaFree(s->d_pairidx);
    cudaFree(s->d_pair_ij);
    cudaFree(s->d_contacts_sym);
    cudaFree(s->d_class_sym);
    s->d_contacts_sym = nullptr; s->d_class_sym = nullptr;
    for (gp_weight_image& w : s->wimgs) {
        cudaFree(w.d_img);
        if (w.ready) cudaEventDestroy((cudaEvent_t)w.ready);
    }
    s->wimgs.clear();
    cudaFree(s->d_pair_img);
    s->d_pair_img = nullptr;
    if (s->pair_img_ready) cudaEventDestroy((cudaEvent_t)s->pair_img_ready);
    s->pair_img_ready = nullptr;
    cudaFree(s->d_units);
    s->d_units = nullptr;
    cudaFree(s->d_host_store);
    s->d_host_store = nullptr; s->host_store_bytes = 0;
    s->d_contacts = nullptr; s->d_class_of = nullptr; s->d_pairidx = nullptr; s->d_pair_ij = nullptr;
}

extern "C" gp_status gp_structures(int nx, int ny, int nz, gp_structures_t** out) {
    if (!out) return GP_INVALID_ARG;
    *out = nullptr;
    gp_structures_s* s = new (std::nothrow) gp_structures_s();
    if (!s) return GP_OUT_OF_MEMORY;
    gp_status st;
    try {
        st = gp_build_host_tables(nx, ny, nz, s);
    } catch (const std::bad_alloc&) {
        st = GP_OUT_OF_MEMORY;
    }
    if (st == GP_OK) st = gp_upload_tables(s);
    if (st == GP_OK && s->device < 0) st = gp_build_map_units(s);  // host-only handle: the unit queries still work
    if (st != GP_OK) {
        gp_release_device(s);
        delete s;
        return st;
    }
    *out = s;
    return GP_OK;
}

extern "C" void gp_structures_free(gp_structures_t* s) {
    if (!s) return;
    gp_release_device(s);
    delete s;
}

extern "C" int gp_structures_length(const gp_structures_t* s) { return s ? s->N : 0; }
extern "C" uint32_t gp_structures_directed(const gp_structures_t* s) { return s ? s->D : 0; }
extern "C" uint32_t gp_structures_classes(const gp_structures_t* s) { return s ? s->C : 0; }
extern "C" uint32_t gp_structures_self_reverse(const gp_structures_t* s) { return s ? s->n_self_reverse : 0; }
extern "C" uint64_t gp_structures_walks(const gp_structures_t* s) { return s ? (uint64_t)s->D * (uint64_t)s->group : 0; }
extern "C" int gp_structures_contacts_per_fold(const gp_structures_t* s) { return s ? s->NBP : 0; }
extern "C" int gp_structures_features(const gp_structures_t* s) { return s ? s->K : 0; }

extern "C" gp_status gp_structures_get(const gp_structures_t* s, uint32_t d, uint8_t* sites, uint8_t* contacts,
                                       uint16_t* class_id) {
    if (!s) return GP_INVALID_ARG;
    if (d >= s->D) return GP_RANGE;
    if (sites) memcpy(sites, &s->walks[(size_t)d * s->N], s->N);
    if (contacts) memcpy(contacts, &s->contacts[(size_t)d * s->NBP * 2], (size_t)s->NBP * 2);
    if (class_id) *class_id = s->class_of[d];
    return GP_OK;
}

// alphabet-2 energies -> (a, lin, quad); bounds so that every weight fits int8 and every energy fits the packed key
gp_status gp_check_hp(const gp_structures_s* s, const gp_energies* en, gp_hp_params* out) {
    if (!s || !en || !en->e || en->alphabet != 2 || en->threshold < 1) return GP_INVALID_ARG;
    const int32_t a = en->e[0], b = en->e[1], b2 = en->e[2], c = en->e[3];
    if (b != b2) return GP_INVALID_ARG;
    if (a < -10000 || a > 10000 || b < -10000 || b > 10000 || c < -10000 || c > 10000) return GP_INVALID_ARG;
    int32_t lin = b - a, quad = c - 2 * b + a;
    // a monomer has at most 5 contacts on a cubic lattice (6 neighbours minus one chain bond), 3 in 2D
    int cmax = (s->nz > 1 && s->ny > 1 && s->nx > 1) ? 5 : 3;
    // int8 weights (scoring_tc.cu build_image_kernel): a pair column holds quad; a monomer column accumulates, over the
    // monomer's <= cmax contacts, lin (free partner), lin + quad (fixed H partner) or lin (fixed P partner)
    const int32_t alin = lin < 0 ? -lin : lin, alq = lin + quad < 0 ? -(lin + quad) : lin + quad;
    if (cmax * (alin > alq ? alin : alq) > 127 || quad > 127 || quad < -127) return GP_INVALID_ARG;
    long long bound = (long long)s->NBP * (2LL * (lin < 0 ? -lin : lin) + (quad < 0 ? -quad : quad));
    if (bound > 8190) return GP_INVALID_ARG;  // pad structures score 8191 (scoring_tc.cu E_PAD)
    out->a = a; out->lin = lin; out->quad = quad; out->threshold = en->threshold;
    return GP_OK;
}

extern "C" gp_status gp_seeded_matrix(uint64_t seed, int32_t* m400) {
    if (!m400) return GP_INVALID_ARG;
    for (int a = 0; a < 20; a++)
        for (int b = a; b < 20; b++) {
            uint64_t u = gp_draw(seed, (1ULL << 62) + (uint64_t)(20 * a + b));
            int32_t v = -750 + (int32_t)(((u >> 32) * 701) >> 32);
            m400[20 * a + b] = m400[20 * b + a] = v;
        }
    return GP_OK;
}

extern "C" gp_status gp_seeded_sequences(uint64_t seed, uint64_t first, uint64_t count, int n, uint8_t* seqs) {
    if (!seqs || n < 1 || n > 64) return GP_INVALID_ARG;
    for (uint64_t q = 0; q < count; q++)
        for (int k = 0; k < n; k++) seqs[q * n + k] = (uint8_t)gp_letter20(seed, first + q, k);
    return GP_OK;
}

extern "C" gp_status gp_seeded_letters(uint64_t seed, uint64_t first, uint64_t count, int n, int alphabet, uint8_t* seqs) {
    if (!seqs || n < 1 || n > 64 || alphabet < 2 || alphabet > 20) return GP_INVALID_ARG;
    for (uint64_t q = 0; q < count; q++)
        for (int k = 0; k < n; k++) seqs[q * n + k] = (uint8_t)gp_letter(seed, first + q, k, (uint32_t)alphabet);
    return GP_OK;
}

// End-to-end call from host buffers: device store allocated here, results copied back.
extern "C" gp_status gp_enumerate_host(const gp_structures_t* s, const gp_energies* en, uint64_t g_begin,
                                       uint64_t g_count, uint16_t* pheno, uint64_t* hist, uint64_t* rdo,
                                       uint64_t* pair_count) {
    if (!s || !hist) return GP_INVALID_ARG;
    if (s->device < 0) { gp_set_cuda_error(cudaErrorNoDevice, "handle has no device tables"); return GP_CUDA_ERROR; }
    const uint32_t C = s->C;
    int n_bits = 0;
    if (rdo) {  // the neighbour pass needs an aligned sub-cube of the genotype space
        while ((1ULL << n_bits) < g_count) n_bits++;
        if (g_count == 0 || (1ULL << n_bits) != g_count || (g_begin & (g_count - 1)) != 0) return GP_RANGE;
    } else if (pair_count) {
        return GP_INVALID_ARG;
    }
    // one device buffer, kept in the handle between calls: outputs (hist[C+1] | R[C] | D[C] | O[C] | pair_count), then the store
    const size_t n_out = (size_t)C + 1 + 3 * (size_t)C + 1;
    const size_t out_bytes = (n_out * sizeof(uint64_t) + 255) & ~(size_t)255;
    const size_t need = out_bytes + (g_count ? g_count : 1) * sizeof(uint16_t);
    const gp_structures_s* hs = s;
    std::lock_guard<std::mutex> lk(hs->mu);  // synchronous call: one at a time per handle shares the kept device buffers
    if (hs->host_store_bytes < need) {
        if (hs->d_host_store) GP_CUDA(cudaFree(hs->d_host_store));
        hs->d_host_store = nullptr; hs->host_store_bytes = 0;
        GP_CUDA(cudaMalloc(&hs->d_host_store, need));
        hs->host_store_bytes = need;
    }
    uint64_t* d_out = reinterpret_cast<uint64_t*>(hs->d_host_store);
    uint16_t* d_pheno = reinterpret_cast<uint16_t*>(reinterpret_cast<char*>(hs->d_host_store) + out_bytes);
    uint64_t* d_hist = d_out;
    uint64_t* d_rdo = d_out + C + 1;
    uint64_t* d_pc = d_rdo + 3 * (size_t)C;
    gp_status st = gp_enumerate(s, en, g_begin, g_count, d_pheno, nullptr, nullptr);
    if (st == GP_OK) {  // with the neighbour pass, its first sweep of the store also counts the classes (gp_reduce_store)
        if (rdo) st = gp_reduce_store(d_pheno, n_bits, C, d_hist, d_rdo, d_rdo + C, d_rdo + 2 * (size_t)C, pair_count ? d_pc : nullptr, nullptr);
        else st = gp_designability(d_pheno, g_count, C, d_hist, nullptr);
    }
    if (st == GP_OK) {
        cudaError_t e = cudaSuccess;
        if (pheno && g_count) e = cudaMemcpy(pheno, d_pheno, g_count * sizeof(uint16_t), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess) e = cudaMemcpy(hist, d_hist, ((size_t)C + 1) * sizeof(uint64_t), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess && rdo) e = cudaMemcpy(rdo, d_rdo, 3 * (size_t)C * sizeof(uint64_t), cudaMemcpyDeviceToHost);
        if (e == cudaSuccess && pair_count) e = cudaMemcpy(pair_count, d_pc, sizeof(uint64_t), cudaMemcpyDeviceToHost);
        if (e != cudaSuccess) { gp_set_cuda_error(e, "gp_enumerate_host copy-back"); st = GP_CUDA_ERROR; }
    }
    return st;
}
