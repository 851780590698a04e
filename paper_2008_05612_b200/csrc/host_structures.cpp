// host_structures.cpp — a0 `gp_structures`: the fold library ("all compact self-avoiding walks"; the paper
// reads it from files, :654-694).  Host-side setup of libgpmap; written independently of oracle/ (different search:
// orbit-minimal start sites, dead-end pruning, early-exit canonical test, binary search for the reversed walk).
//
// Canonical order: site = x + nx*(y + ny*z); a directed structure is the lexicographically
// smallest image of a walk under the box's point group; directed structures are sorted lexicographically; a class is
// {d, reverse(d)}, numbered by its smaller member.
#include <algorithm>
#include <cstring>

#include "gpmap_internal.h"

namespace {

struct Box {
    int ext[3];
    int n;
    std::vector<std::vector<uint8_t> > nbr;  // neighbours of each site
    std::vector<std::vector<uint8_t> > sym;  // point group as site permutations (identity first)
};

void make_box(int nx, int ny, int nz, Box& b) {
    b.ext[0] = nx; b.ext[1] = ny; b.ext[2] = nz;
    b.n = nx * ny * nz;
    b.nbr.assign(b.n, std::vector<uint8_t>());
    const int step[3] = {1, nx, nx * ny};
    for (int s = 0; s < b.n; s++) {
        int c[3] = {s % nx, (s / nx) % ny, s / (nx * ny)};
        for (int a = 0; a < 3; a++) {
            if (c[a] > 0) b.nbr[s].push_back((uint8_t)(s - step[a]));
            if (c[a] + 1 < b.ext[a]) b.nbr[s].push_back((uint8_t)(s + step[a]));
        }
    }
    // signed axis permutations that keep the extents; duplicates (flat axes) removed
    static const int perms[6][3] = {{0, 1, 2}, {0, 2, 1}, {1, 0, 2}, {1, 2, 0}, {2, 0, 1}, {2, 1, 0}};
    for (int p = 0; p < 6; p++) {
        const int* pm = perms[p];
        if (b.ext[pm[0]] != nx || b.ext[pm[1]] != ny || b.ext[pm[2]] != nz) continue;
        for (int f = 0; f < 8; f++) {
            std::vector<uint8_t> m(b.n);
            for (int s = 0; s < b.n; s++) {
                int c[3] = {s % nx, (s / nx) % ny, s / (nx * ny)};
                int t[3];
                for (int a = 0; a < 3; a++) {
                    t[a] = c[pm[a]];
                    if ((f >> a) & 1) t[a] = b.ext[a] - 1 - t[a];
                }
                m[s] = (uint8_t)(t[0] + nx * (t[1] + ny * t[2]));
            }
            if (std::find(b.sym.begin(), b.sym.end(), m) == b.sym.end()) b.sym.push_back(m);
        }
    }
}

// true iff no symmetry image of w is lexicographically smaller than w
bool is_canonical(const Box& b, const uint8_t* w) {
    for (size_t g = 1; g < b.sym.size(); g++) {
        const uint8_t* m = b.sym[g].data();
        for (int i = 0; i < b.n; i++) {
            int a = m[w[i]];
            if (a < w[i]) return false;
            if (a > w[i]) break;
        }
    }
    return true;
}

void canonical_image(const Box& b, const uint8_t* w, uint8_t* out) {
    std::vector<uint8_t> img(b.n);
    memcpy(out, w, b.n);
    for (size_t g = 1; g < b.sym.size(); g++) {
        const uint8_t* m = b.sym[g].data();
        for (int i = 0; i < b.n; i++) img[i] = m[w[i]];
        if (memcmp(img.data(), out, b.n) < 0) memcpy(out, img.data(), b.n);
    }
}

struct Search {
    const Box& b;
    std::vector<uint8_t> w;
    std::vector<char> used;
    std::vector<int> freedeg;  // unvisited neighbours of each site
    std::vector<uint8_t>& keep;
    int len;
    Search(const Box& box, std::vector<uint8_t>& out) : b(box), w(box.n), used(box.n, 0), freedeg(box.n), keep(out), len(0) {
        for (int s = 0; s < b.n; s++) freedeg[s] = (int)b.nbr[s].size();
    }
    void visit(int s) {
        used[s] = 1;
        w[len++] = (uint8_t)s;
        for (uint8_t u : b.nbr[s]) freedeg[u]--;
    }
    void leave(int s) {
        for (uint8_t u : b.nbr[s]) freedeg[u]++;
        used[s] = 0;
        len--;
    }
    void extend() {
        if (len == b.n) {
            if (is_canonical(b, w.data())) keep.insert(keep.end(), w.begin(), w.end());
            return;
        }
        int head = w[len - 1];
        for (uint8_t s : b.nbr[head]) {
            if (used[s]) continue;
            visit(s);
            // dead-end pruning: an unvisited neighbour of the old head that has no way in any more
            bool dead = false;
            if (len < b.n) {
                for (uint8_t u : b.nbr[head]) {
                    if (used[u]) continue;
                    bool touches_head = false;
                    for (uint8_t v : b.nbr[u]) touches_head |= (v == s);
                    if (freedeg[u] == 0 && !touches_head) { dead = true; break; }
                }
            }
            if (!dead) extend();
            leave(s);
        }
    }
};

}  // namespace

gp_status gp_build_host_tables(int nx, int ny, int nz, gp_structures_s* S) {
    if (nx < 1 || ny < 1 || nz < 1) return GP_UNSUPPORTED_LATTICE;
    long long n = (long long)nx * ny * nz;
    if (n < 2 || n > 64) return GP_UNSUPPORTED_LATTICE;
    Box b;
    make_box(nx, ny, nz, b);
    S->nx = nx; S->ny = ny; S->nz = nz;
    S->N = b.n;
    S->group = (int)b.sym.size();

    // 1. walks from orbit-minimal start sites only (a canonical walk starts on the smallest site of its orbit)
    std::vector<uint8_t> found;
    for (int s0 = 0; s0 < b.n; s0++) {
        bool minimal = true;
        for (size_t g = 1; g < b.sym.size(); g++) minimal &= (b.sym[g][s0] >= s0);
        if (!minimal) continue;
        Search q(b, found);
        q.visit(s0);
        q.extend();
    }
    size_t D = found.size() / b.n;
    if (D == 0) return GP_UNSUPPORTED_LATTICE;  // box has no Hamiltonian walk
    // 2. sort lexicographically -> directed index
    std::vector<uint32_t> order(D);
    for (size_t d = 0; d < D; d++) order[d] = (uint32_t)d;
    const int N = b.n;
    const uint8_t* base = found.data();
    std::sort(order.begin(), order.end(),
              [&](uint32_t x, uint32_t y) { return memcmp(base + (size_t)x * N, base + (size_t)y * N, N) < 0; });
    S->walks.resize(D * N);
    for (size_t d = 0; d < D; d++) memcpy(&S->walks[d * N], base + (size_t)order[d] * N, N);
    S->D = (uint32_t)D;

    // 3. reversal partner by binary search; classes numbered by smaller member
    std::vector<uint32_t> partner(D);
    std::vector<uint8_t> rev(N), can(N);
    S->n_self_reverse = 0;
    for (size_t d = 0; d < D; d++) {
        const uint8_t* w = &S->walks[d * N];
        for (int i = 0; i < N; i++) rev[i] = w[N - 1 - i];
        canonical_image(b, rev.data(), can.data());
        size_t lo = 0, hi = D;
        while (lo < hi) {
            size_t mid = (lo + hi) / 2;
            if (memcmp(&S->walks[mid * N], can.data(), N) < 0) lo = mid + 1; else hi = mid;
        }
        if (lo >= D || memcmp(&S->walks[lo * N], can.data(), N) != 0) return GP_UNSUPPORTED_LATTICE;  // cannot happen
        partner[d] = (uint32_t)lo;
        if (lo == d) S->n_self_reverse++;
    }
    uint32_t C = (uint32_t)((D + S->n_self_reverse) / 2);
    if (C >= GP_NULL_PHENO) return GP_UNSUPPORTED_LATTICE;
    S->class_of.assign(D, 0);
    uint32_t next = 0;
    for (size_t d = 0; d < D; d++) {
        if (partner[d] < d) S->class_of[d] = S->class_of[partner[d]];
        else S->class_of[d] = (uint16_t)next++;
    }
    S->C = next;

    // 4. contacts: monomer pairs on adjacent sites that are not chain neighbours (Delta of Eq. 1, :69)
    std::vector<int8_t> pos(N);
    S->NBP = -1;
    for (size_t d = 0; d < D; d++) {
        const uint8_t* w = &S->walks[d * N];
        for (int i = 0; i < N; i++) pos[w[i]] = (int8_t)i;
        int cnt = 0;
        for (int i = 0; i < N; i++)
            for (uint8_t u : b.nbr[w[i]]) {
                int j = pos[u];
                if (j > i + 1) { S->contacts.push_back((uint8_t)i); S->contacts.push_back((uint8_t)j); cnt++; }
            }
        if (S->NBP < 0) S->NBP = cnt;
        if (cnt != S->NBP) return GP_UNSUPPORTED_LATTICE;  // every compact walk has #edges-(N-1) contacts
        // sort this structure's contact list by (i, j)
        uint8_t* c = &S->contacts[d * (size_t)S->NBP * 2];
        std::vector<std::pair<uint8_t, uint8_t> > v(cnt);
        for (int k = 0; k < cnt; k++) v[k] = std::make_pair(c[2 * k], c[2 * k + 1]);
        std::sort(v.begin(), v.end());
        for (int k = 0; k < cnt; k++) { c[2 * k] = v[k].first; c[2 * k + 1] = v[k].second; }
    }

    // 5. feature columns of the contraction: N monomer letters, then the pairs that can ever touch
    //    (bipartite lattice: j - i odd and >= 3)
    S->pair_index.assign((size_t)N * N, -1);
    int P = 0;
    for (int i = 0; i < N; i++)
        for (int j = i + 3; j < N; j += 2) S->pair_index[(size_t)i * N + j] = (int16_t)P++;
    S->P = P;
    S->K = N + P;
    for (size_t k = 0; k < S->contacts.size(); k += 2)
        if (S->pair_index[(size_t)S->contacts[k] * N + S->contacts[k + 1]] < 0) return GP_UNSUPPORTED_LATTICE;
    return GP_OK;
}
