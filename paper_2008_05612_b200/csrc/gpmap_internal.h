// gpmap_internal.h — private to libgpmap (host setup + CUDA kernels).  Not part of the ABI, not used by oracle/.
#pragma once
#include <stdint.h>

#include <mutex>
#include <vector>

#include "gpmap.h"

// Cached device image of the weight matrix W for one (b-a, c-2b+a) pair, in the tile layout the tcgen05 kernel
// bulk-copies into shared memory (see scoring_tc.cu).
// Entries are immutable once built: a call that needs another (lin, quad) adds an entry; `ready` is recorded on the
// building stream and waited on by every other stream that uses the image.
struct gp_weight_image {
    int32_t lin = 0, quad = 0;  // (b-a), (c-2b+a): weight of a monomer feature per contact, of a pair feature
    int8_t* d_img = nullptr;    // [n_tiles][k_blocks][TILE_N rows][128 B], 128B-swizzled
    void* ready = nullptr;      // cudaEvent_t
};

struct gp_structures_s {
    int nx = 0, ny = 0, nz = 0;
    int N = 0, NBP = 0, group = 0;
    uint32_t D = 0, C = 0, n_self_reverse = 0;
    int P = 0, K = 0;                    // pair features, total features N + P
    std::vector<uint8_t> walks;          // D * N site indices
    std::vector<uint8_t> contacts;       // D * NBP * 2 monomer indices, i < j
    std::vector<uint16_t> class_of;      // D
    std::vector<int16_t> pair_index;     // N * N -> index into the P pair features, -1 if (i,j) can never touch
    // device side (null when no CUDA device)
    int device = -1;
    uint8_t* d_contacts = nullptr;
    uint16_t* d_class_of = nullptr;
    uint16_t* d_pairidx = nullptr;       // D * NBP: pair-feature index of each contact
    uint8_t* d_pair_ij = nullptr;        // P * 2: monomers (i, j) of each pair feature
    // reversal-reduced structure list for gp_enumerate_map (one representative per class; scoring_tc.cu): first the
    // classes that differ from their reversal, padded to a multiple of 128 columns, then the self-reverse classes
    uint8_t* d_contacts_sym = nullptr;   // D_sym * NBP * 2 (pad entries zero)
    uint16_t* d_class_sym = nullptr;     // D_sym: class id of the column, 0xFFFF = pad column
    uint32_t D_sym = 0, n_snap = 0;      // columns incl. interior pads; weight tiles holding non-self-reverse classes
    // units of gp_enumerate_map_range for the current tuning.sym_bits: middle-bit values m <= rev m, the
    // non-palindromic ones first; rebuilt by gp_tuning_set only
    uint32_t* d_units = nullptr;
    std::vector<uint32_t> units;
    uint64_t n_units = 0, n_pair_units = 0;  // all units; units that hold two images
    int map_k = 0;                            // k the table was built for (0: the lattice is too small, one unit)
    gp_tuning tuning = {15, 7, 1, 1};
    // mutable state behind `mu`: the cache of full-contraction weight images (sequence_kernel) and the device buffers
    // of the synchronous gp_enumerate_host.  Compute calls take everything else from the stream-ordered pool.
    mutable std::mutex mu;
    mutable std::vector<gp_weight_image> wimgs;
    mutable int8_t* d_pair_img = nullptr;    // 0/-1 contact-incidence image of seq20_kernel (lattice only), built once
    mutable void* pair_img_ready = nullptr;  // cudaEvent_t
    mutable void* d_host_store = nullptr;
    mutable size_t host_store_bytes = 0;
};

// host_structures.cpp
gp_status gp_build_host_tables(int nx, int ny, int nz, gp_structures_s* s);
// device.cu
gp_status gp_upload_tables(gp_structures_s* s);
void gp_release_device(gp_structures_s* s);
// scoring_tc.cu: (re)build the unit table of the map path for s->tuning.sym_bits and upload it
gp_status gp_build_map_units(gp_structures_s* s);
