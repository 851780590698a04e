// gp_oracle.cpp — CPU ORACLE for the HP/MJ-style lattice genotype-phenotype map.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may build, load or call it.
// It shares no code, header, table or helper with paper_2008_05612_b200/ (the CUDA
// path), and neither side imports the other.
//
// It is a plain, slow, single-threaded restatement of what the paper computes
// (arXiv 2008.05612; citations are PAPER.md:LINE):
//   * fold library = all compact self-avoiding walks of the lattice       (:65)
//   * H = sum_{i<j} E[s_i][s_j] * Delta(r_i - r_j), Delta = 1 iff lattice
//     neighbours but not chain neighbours                                (:67-69, Eq. 1)
//   * HP energies E_HH=-2.3, E_HP=-1, E_PP=0, used as integers x10         (:77-79, :519-525)
//   * ground state = unique minimum-energy fold, else "does not fold";
//     optional threshold on the gap to the second-lowest fold            (:81, :552-575)
//   * designability N_q                                                  (:138)
//   * one-point-mutation neighbourhood, phi_pq, robustness, phi_del      (:138-147, Eq. 2)
//   * neutral networks = connected sets of same-phenotype genotypes      (:19)
// No blocking, fusion or reordering: nested loops in the paper's order (listing
// lines 71-94).  Readings of ambiguous passages follow
// DESIGN.md "Readings" (R1..): all directed symmetry classes are scored, a tie
// between any two directed threadings is "does not fold", ids are reversal-reduced.
//
// Parity pins: see tests/test_oracle_*.py.  Every function below is pinned there
// (brute force on tiny lattices, paper-printed counts, closed forms, invariants).
//
// Build: g++ -O2 -std=c++17 -shared -fPIC gp_oracle.cpp -o liboracle.so

#include <algorithm>
#include <climits>
#include <cstdint>
#include <cstring>
#include <map>
#include <set>
#include <utility>
#include <vector>

namespace {

typedef std::vector<uint8_t> Walk;  // site index of monomer 0..N-1

struct Lattice {
    int dims[3];
    int N;
    std::vector<std::vector<int> > nbr;      // nearest-neighbour sites of each site
    std::vector<std::vector<uint8_t> > sym;  // point group of the box: site -> image site

    int site(int x, int y, int z) const { return x + dims[0] * (y + dims[1] * z); }

    Lattice(int nx, int ny, int nz) {
        dims[0] = nx; dims[1] = ny; dims[2] = nz;
        N = nx * ny * nz;
        nbr.resize(N);
        for (int z = 0; z < nz; z++)
            for (int y = 0; y < ny; y++)
                for (int x = 0; x < nx; x++) {
                    int s = site(x, y, z);
                    if (x > 0) nbr[s].push_back(site(x - 1, y, z));
                    if (x + 1 < nx) nbr[s].push_back(site(x + 1, y, z));
                    if (y > 0) nbr[s].push_back(site(x, y - 1, z));
                    if (y + 1 < ny) nbr[s].push_back(site(x, y + 1, z));
                    if (z > 0) nbr[s].push_back(site(x, y, z - 1));
                    if (z + 1 < nz) nbr[s].push_back(site(x, y, z + 1));
                    std::sort(nbr[s].begin(), nbr[s].end());
                }
        // Symmetries of the box = signed axis permutations that keep its extents:
        // 8 for a square, 48 for a cube, 4 for a non-square rectangle.
        int perm[3] = {0, 1, 2};
        std::set<std::vector<uint8_t> > seen;
        do {
            bool keeps = true;
            for (int a = 0; a < 3; a++)
                if (dims[perm[a]] != dims[a]) keeps = false;
            if (!keeps) continue;
            for (int flip = 0; flip < 8; flip++) {
                std::vector<uint8_t> map(N);
                for (int z = 0; z < nz; z++)
                    for (int y = 0; y < ny; y++)
                        for (int x = 0; x < nx; x++) {
                            int c[3] = {x, y, z};
                            int img[3];
                            for (int a = 0; a < 3; a++) {
                                int v = c[perm[a]];
                                if (flip & (1 << a)) v = dims[a] - 1 - v;
                                img[a] = v;
                            }
                            map[site(x, y, z)] = (uint8_t)site(img[0], img[1], img[2]);
                        }
                if (seen.insert(map).second) sym.push_back(map);
            }
        } while (std::next_permutation(perm, perm + 3));
    }
};

struct Structures {
    Lattice lat;
    int N, NBP;
    uint64_t n_walks;            // directed Hamiltonian walks of the box (before symmetry)
    uint32_t D, C, n_self_reverse;
    std::vector<Walk> walks;     // D directed-canonical walks, sorted lexicographically
    std::vector<uint8_t> contacts;  // D * NBP * 2 monomer indices (i<j)
    std::vector<uint32_t> class_of; // D -> class id 0..C-1

    Structures(int nx, int ny, int nz) : lat(nx, ny, nz), N(lat.N), NBP(0), n_walks(0), D(0), C(0), n_self_reverse(0) {}
};

// lexicographically smallest image of w under the point group
Walk canonical_directed(const Lattice& lat, const Walk& w) {
    Walk best = w;
    Walk img(w.size());
    for (size_t g = 0; g < lat.sym.size(); g++) {
        for (size_t i = 0; i < w.size(); i++) img[i] = lat.sym[g][w[i]];
        if (img < best) best = img;
    }
    return best;
}

void dfs(const Lattice& lat, Walk& w, std::vector<char>& used, uint64_t& n_walks, std::vector<Walk>& keep) {
    if ((int)w.size() == lat.N) {
        n_walks++;
        if (canonical_directed(lat, w) == w) keep.push_back(w);
        return;
    }
    int last = w.back();
    for (size_t k = 0; k < lat.nbr[last].size(); k++) {
        int s = lat.nbr[last][k];
        if (used[s]) continue;
        used[s] = 1;
        w.push_back((uint8_t)s);
        dfs(lat, w, used, n_walks, keep);
        w.pop_back();
        used[s] = 0;
    }
}

bool adjacent(const Lattice& lat, int a, int b) {
    for (size_t k = 0; k < lat.nbr[a].size(); k++)
        if (lat.nbr[a][k] == b) return true;
    return false;
}

Structures* build_structures(int nx, int ny, int nz) {
    Structures* S = new Structures(nx, ny, nz);
    const Lattice& lat = S->lat;
    // 1. all compact self-avoiding walks, from every start site
    for (int s = 0; s < lat.N; s++) {
        Walk w(1, (uint8_t)s);
        std::vector<char> used(lat.N, 0);
        used[s] = 1;
        dfs(lat, w, used, S->n_walks, S->walks);
    }
    // 2. directed classes: canonical walks sorted lexicographically
    std::sort(S->walks.begin(), S->walks.end());
    S->D = (uint32_t)S->walks.size();
    // 3. classes under point group + chain reversal
    std::map<Walk, uint32_t> index_of;
    for (uint32_t d = 0; d < S->D; d++) index_of[S->walks[d]] = d;
    std::vector<uint32_t> rep(S->D);
    std::set<uint32_t> reps;
    for (uint32_t d = 0; d < S->D; d++) {
        Walk r(S->walks[d].rbegin(), S->walks[d].rend());
        uint32_t dr = index_of.at(canonical_directed(lat, r));
        if (dr == d) S->n_self_reverse++;
        rep[d] = std::min(d, dr);
        reps.insert(rep[d]);
    }
    std::map<uint32_t, uint32_t> class_id;  // representative directed index -> class id (sorted order)
    for (std::set<uint32_t>::iterator it = reps.begin(); it != reps.end(); ++it) {
        uint32_t id = (uint32_t)class_id.size();
        class_id[*it] = id;
    }
    S->C = (uint32_t)class_id.size();
    S->class_of.resize(S->D);
    for (uint32_t d = 0; d < S->D; d++) S->class_of[d] = class_id.at(rep[d]);
    // 4. contacts: i<j, sites adjacent, not chain neighbours (Delta of Eq. 1)
    for (uint32_t d = 0; d < S->D; d++) {
        int n = 0;
        for (int i = 0; i < S->N; i++)
            for (int j = i + 2; j < S->N; j++)
                if (adjacent(lat, S->walks[d][i], S->walks[d][j])) {
                    S->contacts.push_back((uint8_t)i);
                    S->contacts.push_back((uint8_t)j);
                    n++;
                }
        if (d == 0) S->NBP = n;
        if (n != S->NBP) { delete S; return NULL; }  // every compact walk has the same count
    }
    return S;
}

// Eq. 1 for one sequence on one directed structure (listing lines 76-80)
int32_t energy_of(const Structures* S, uint32_t d, const uint8_t* letters, int alphabet, const int32_t* e) {
    int32_t E = 0;
    const uint8_t* c = &S->contacts[(size_t)d * S->NBP * 2];
    for (int k = 0; k < S->NBP; k++) {
        int loc1 = c[2 * k], loc2 = c[2 * k + 1];
        E += e[letters[loc1] * alphabet + letters[loc2]];
    }
    return E;
}

const uint16_t NULL_PHENO = 0xFFFF;

// ground state of one sequence: two smallest energies with multiplicity, strict '<' updates
// (PAPER.md:552-567), true-minimum initialisation (reading R6).
void ground_state(const Structures* S, const uint8_t* letters, int alphabet, const int32_t* e, int32_t threshold,
                  uint16_t* pheno, int32_t* gap) {
    int64_t m1 = INT64_MAX, m2 = INT64_MAX;
    uint32_t arg = 0;
    for (uint32_t d = 0; d < S->D; d++) {
        int64_t E = energy_of(S, d, letters, alphabet, e);
        if (E < m1) { m2 = m1; m1 = E; arg = d; }
        else if (E < m2) { m2 = E; }
    }
    bool folds = (m2 == INT64_MAX) || (m2 - m1 >= threshold);
    *pheno = folds ? (uint16_t)S->class_of[arg] : NULL_PHENO;
    if (gap) {
        int64_t g = (m2 == INT64_MAX) ? (int64_t)INT16_MIN : m1 - m2;  // m1 - m2 <= 0
        if (g < INT16_MIN) g = INT16_MIN;
        *gap = (int32_t)g;
    }
}

uint64_t mix64(uint64_t z) {  // 64-bit splitmix finaliser
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
uint64_t draw(uint64_t seed, uint64_t ctr) { return mix64(seed + (ctr + 1) * 0x9E3779B97F4A7C15ULL); }

}  // namespace

extern "C" {

void* oracle_structures_create(int nx, int ny, int nz) {
    if (nx < 1 || ny < 1 || nz < 1 || nx * ny * nz > 64 || nx * ny * nz < 2) return NULL;
    return build_structures(nx, ny, nz);
}
void oracle_structures_free(void* h) { delete (Structures*)h; }
int oracle_length(void* h) { return ((Structures*)h)->N; }
int oracle_contacts_per_fold(void* h) { return ((Structures*)h)->NBP; }
uint32_t oracle_directed(void* h) { return ((Structures*)h)->D; }
uint32_t oracle_classes(void* h) { return ((Structures*)h)->C; }
uint32_t oracle_self_reverse(void* h) { return ((Structures*)h)->n_self_reverse; }
uint64_t oracle_walk_count(void* h) { return ((Structures*)h)->n_walks; }
int oracle_group_order(void* h) { return (int)((Structures*)h)->lat.sym.size(); }

// sites[N], contacts[2*NBP], class id of directed structure d
void oracle_structure_get(void* h, uint32_t d, uint8_t* sites, uint8_t* contacts, uint32_t* class_id) {
    Structures* S = (Structures*)h;
    if (sites) memcpy(sites, S->walks[d].data(), S->N);
    if (contacts) memcpy(contacts, &S->contacts[(size_t)d * S->NBP * 2], (size_t)S->NBP * 2);
    if (class_id) *class_id = S->class_of[d];
}

int32_t oracle_energy(void* h, uint32_t d, const uint8_t* letters, int alphabet, const int32_t* e) {
    return energy_of((Structures*)h, d, letters, alphabet, e);
}

// implicit binary genotypes g_begin .. g_begin+count-1; bit i of g = letter of monomer i
// (1 = H: e[1*2+1] = E_HH).  DESIGN.md reading R3.
void oracle_enumerate(void* h, const int32_t* e /*4*/, int32_t threshold, uint64_t g_begin, uint64_t count,
                      uint16_t* pheno, int32_t* gap /*nullable*/) {
    Structures* S = (Structures*)h;
    uint8_t letters[64];
    for (uint64_t n = 0; n < count; n++) {
        uint64_t g = g_begin + n;
        for (int i = 0; i < S->N; i++) letters[i] = (uint8_t)((g >> i) & 1);
        ground_state(S, letters, 2, e, threshold, &pheno[n], gap ? &gap[n] : NULL);
    }
}

// explicit sequences seqs[count][N] over `alphabet` letters (the paper's SeqRnd path).  The paper
// only ever generates letters inside the alphabet (:762-775) and says nothing about others; reading R19: a
// byte >= alphabet is read as the LAST letter, alphabet - 1, so the look-up e[l1 * alphabet + l2] stays inside e[].
void oracle_enumerate_seqs(void* h, int alphabet, const int32_t* e, int32_t threshold, const uint8_t* seqs,
                           uint64_t count, uint16_t* pheno, int32_t* gap /*nullable*/) {
    Structures* S = (Structures*)h;
    uint8_t letters[64];
    for (uint64_t n = 0; n < count; n++) {
        for (int i = 0; i < S->N; i++) {
            uint8_t l = seqs[n * S->N + i];
            letters[i] = l < alphabet ? l : (uint8_t)(alphabet - 1);
        }
        ground_state(S, letters, alphabet, e, threshold, &pheno[n], gap ? &gap[n] : NULL);
    }
}

uint64_t oracle_draw(uint64_t seed, uint64_t ctr) { return draw(seed, ctr); }

// counter-based generator of DESIGN.md "Input recipe": letter k of sequence s is drawn at counter 64 s + k (a stride of
// 64 >= the longest chain, so that the sequences of chains longer than 16 share no draws: DESIGN.md section 4)
void oracle_seeded_sequences(uint64_t seed, uint64_t first, uint64_t count, int N, uint8_t* seqs) {
    for (uint64_t n = 0; n < count; n++)
        for (int k = 0; k < N; k++) {
            uint64_t u = draw(seed, (first + n) * 64 + (uint64_t)k);
            seqs[n * N + k] = (uint8_t)(((u >> 32) * 20) >> 32);
        }
}
// the same stream cut into `alphabet` letters (letter = floor(alphabet * hi32(draw) / 2^32); alphabet
// 20 is oracle_seeded_sequences, alphabet 2 — the paper's random H/P sampling runs, PAPER.md:195-204, :762-775 — takes
// the top bit of the draw, 1 = H)
void oracle_seeded_letters(uint64_t seed, uint64_t first, uint64_t count, int N, int alphabet, uint8_t* seqs) {
    for (uint64_t n = 0; n < count; n++)
        for (int k = 0; k < N; k++) {
            uint64_t u = draw(seed, (first + n) * 64 + (uint64_t)k);
            seqs[n * N + k] = (uint8_t)(((u >> 32) * (uint64_t)alphabet) >> 32);
        }
}
// symmetric 20x20 matrix, entries -750..-50 (units of 0.01)
void oracle_seeded_matrix(uint64_t seed, int32_t* M /*400*/) {
    for (int a = 0; a < 20; a++)
        for (int b = a; b < 20; b++) {
            uint64_t u = draw(seed, (1ULL << 62) + (uint64_t)(a * 20 + b));
            int32_t v = -750 + (int32_t)(((u >> 32) * 701) >> 32);
            M[a * 20 + b] = v;
            M[b * 20 + a] = v;
        }
}

// designability: hist[c] for c < C, hist[C] = null count
void oracle_designability(const uint16_t* pheno, uint64_t count, uint32_t C, uint64_t* hist) {
    for (uint32_t c = 0; c <= C; c++) hist[c] = 0;
    for (uint64_t n = 0; n < count; n++) hist[pheno[n] == NULL_PHENO ? C : pheno[n]]++;
}

// one-point-mutation neighbourhood: per class p, over its genotypes and
// their n_bits single flips: R = neutral, Dl = to null, O = to another non-null class.
// pair_count = unordered pairs of distinct non-null classes joined by >= 1 mutation.
void oracle_robustness(const uint16_t* pheno, int n_bits, uint32_t C, uint64_t* R, uint64_t* Dl, uint64_t* O,
                       uint64_t* pair_count /*nullable*/) {
    for (uint32_t c = 0; c < C; c++) R[c] = Dl[c] = O[c] = 0;
    std::set<std::pair<uint32_t, uint32_t> > pairs;
    uint64_t total = 1ULL << n_bits;
    for (uint64_t g = 0; g < total; g++) {
        uint32_t p = pheno[g];
        if (p == NULL_PHENO) continue;
        for (int k = 0; k < n_bits; k++) {
            uint32_t q = pheno[g ^ (1ULL << k)];
            if (q == p) R[p]++;
            else if (q == NULL_PHENO) Dl[p]++;
            else { O[p]++; pairs.insert(std::make_pair(std::min(p, q), std::max(p, q))); }
        }
    }
    if (pair_count) *pair_count = pairs.size();
}

// ordered transition counts T[p*C+q] (p,q non-null) for small C — used only by invariant tests
void oracle_transitions(const uint16_t* pheno, int n_bits, uint32_t C, uint64_t* T) {
    for (uint64_t i = 0; i < (uint64_t)C * C; i++) T[i] = 0;
    uint64_t total = 1ULL << n_bits;
    for (uint64_t g = 0; g < total; g++) {
        uint32_t p = pheno[g];
        if (p == NULL_PHENO) continue;
        for (int k = 0; k < n_bits; k++) {
            uint32_t q = pheno[g ^ (1ULL << k)];
            if (q != NULL_PHENO) T[(uint64_t)p * C + q]++;
        }
    }
}

// neutral-network components: connected components of each class's genotype set
// under single-bit-flip adjacency; breadth-first flood fill.
void oracle_nn_components(const uint16_t* pheno, int n_bits, uint32_t C, uint32_t* ncomp) {
    for (uint32_t c = 0; c < C; c++) ncomp[c] = 0;
    uint64_t total = 1ULL << n_bits;
    std::vector<char> seen(total, 0);
    std::vector<uint64_t> queue;
    for (uint64_t g0 = 0; g0 < total; g0++) {
        uint32_t p = pheno[g0];
        if (p == NULL_PHENO || seen[g0]) continue;
        ncomp[p]++;
        queue.clear();
        queue.push_back(g0);
        seen[g0] = 1;
        for (size_t head = 0; head < queue.size(); head++) {
            uint64_t g = queue[head];
            for (int k = 0; k < n_bits; k++) {
                uint64_t nb = g ^ (1ULL << k);
                if (!seen[nb] && pheno[nb] == p) { seen[nb] = 1; queue.push_back(nb); }
            }
        }
    }
}

}  // extern "C"
