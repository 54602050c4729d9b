// Internal declarations shared by the host setup and the CUDA translation units of libpff.
// Not part of the public boundary (include/pff.h is).
#pragma once
#include <cstdint>
#include <string>
#include <vector>

#include "pff.h"

namespace pff {

// One CTA chunk = a contiguous range of (renumbered) elements + the nodes they touch.
// Local node index: [0, n_int) are the chunk's interior nodes (global ids node_start + i, touched by
// no other chunk); [n_int, n_int + n_halo) are interface nodes, global ids halo_ids[halo_off + j].
struct ChunkMeta {
    int32_t elem_start, n_elem;
    int32_t node_start, n_int;
    int32_t halo_off, n_halo;
    int32_t ell_off, ell_w;  // ELL gather table: ell[ell_off + k * nloc + i], k < ell_w
};

struct HostMesh {
    int64_t N = 0, Ne = 0, C = 0, N_int = 0, N_sh = 0;
    int32_t chunk_elems = 0, max_nloc = 0, max_ell_w = 0;
    double hmin = 0.0;
    std::vector<int32_t> node_new_of_old, elem_new_of_old, node_old_of_new;
    std::vector<int32_t> conn4;    // [Ne][4] global internal node ids, 4th lane = 0
    std::vector<uint16_t> lconn4;  // [Ne][4] chunk-local node ids, 4th lane = 0
    std::vector<double> g12;       // [Ne][4] = (dx phi1, dy phi1, dx phi2, dy phi2); grad phi3 = -(1+2)
    std::vector<double> area;      // [Ne]
    std::vector<double> mass;      // [N] lumped mass, internal order
    std::vector<ChunkMeta> meta;
    std::vector<int32_t> halo_ids;  // global internal ids (all >= N_int)
    std::vector<uint16_t> ell;      // (local elem << 2 | corner), 0xFFFF = empty
    std::vector<int32_t> sh_rowptr, sh_slots;  // per interface node: halo slots (ascending chunk)
    std::vector<double> xy_user;    // copy of the input coordinates (traction lengths)
};

// Builds everything above. Returns PFF_OK or an error with `err` filled.
pff_status build_host_mesh(int64_t n_nodes, const double* xy, int64_t n_elems, const int32_t* tri,
                           double rho, int order, int chunk_elems, size_t real_bytes, size_t smem_limit,
                           HostMesh& hm, std::string& err);

void set_error(const std::string& s);

}  // namespace pff
