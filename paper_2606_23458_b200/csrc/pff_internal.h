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
    int32_t ell_off, ell_w;  // ELL gather table: ell[ell_off + k * nloc + i], k < ell_w (ell_off multiple of 8)
};

// Shared-memory stage of one chunk (byte offsets, all 16-byte aligned).  Every contiguous array of the chunk
// is streamed into the stage by TMA; nodal arrays hold [shift | interior | pad | halo] (node_len entries each).
// Per-element results live in "slots" addressed as corner * EC + local element, with one zero slot at 3 * EC
// that the padding entries of the gather table point to.
//   kind 0: explicit step   10 nodal arrays + flags; fp64: the force pairs of corners 1, 2 overwrite the element's own
//                           staged geometry and corner 3 follows contiguously (pair index); fp32: separate pair slots
//   kind 1: damage iteration  x r p q 1/D lb + mask; scalar slots [3 EC + 1]
//   kind 2: damage setup      x; scalar slots q, D, b each [3 EC + 1]
struct StageLayout {
    uint32_t lconn, geo, slots, area, H, node[10], flags, ell, bar, total;
    uint32_t slot_stride;  // kind 2: bytes between the q, D, b slot arrays
};
inline StageLayout make_stage_layout(int kind, int EC, int node_len, int flag_len, int ell_len, size_t rb)
{
    StageLayout L{};
    auto up16 = [](size_t v) { return uint32_t((v + 15) / 16 * 16); };
    uint32_t o = 0;
    L.lconn = o; o += up16(size_t(8) * EC);
    L.geo = o; o += up16(size_t(4) * rb * EC);
    if (kind == 0) {
        if (rb == 8) { L.slots = L.geo; o += up16(size_t(16) * (EC + 1)); }      // [ga | gb | third | zero] as double2
        else { L.slots = o; o += up16(size_t(8) * (3 * EC + 1)); }                // float2 [3 EC + 1]
    } else if (kind == 1) {
        L.slots = o; o += up16(rb * (size_t(3) * EC + 1));
    } else {
        L.slots = o; L.slot_stride = up16(rb * (size_t(3) * EC + 1)); o += 3 * L.slot_stride;
    }
    L.area = o; o += up16(rb * EC);
    L.H = o; o += up16(rb * EC);
    const int nn = kind == 0 ? 10 : (kind == 1 ? 6 : 1);
    for (int k = 0; k < nn; ++k) { L.node[k] = o; o += up16(rb * node_len); }
    L.flags = o; o += up16(kind == 2 ? 0 : flag_len);
    L.ell = o; o += up16(size_t(2) * ell_len);
    L.bar = o; o += 16;
    L.total = o;
    return L;
}
inline size_t chunk_smem_bytes(int kind, int EC, int node_len, int flag_len, int ell_len, size_t rb)
{
    return make_stage_layout(kind, EC, node_len, flag_len, ell_len, rb).total;
}

struct HostMesh {
    int64_t N = 0, Ne = 0, C = 0, N_int = 0, N_sh = 0;
    int32_t chunk_elems = 0, max_nloc = 0, max_ell_w = 0;
    int32_t node_len = 0;   // entries per staged nodal array: max over chunks of round_up(shift + n_int, A) + n_halo
    int32_t flag_len = 0;   // entries of the staged uint8 flag / mask array
    int32_t ell_len = 0;    // max over chunks of ell_w * nloc, rounded up to 8
    int32_t max_nhalo = 0;
    double hmin = 0.0;
    std::vector<int32_t> node_new_of_old, elem_new_of_old, node_old_of_new;
    std::vector<int32_t> conn4;    // [Ne][4] global internal node ids, 4th lane = 0
    std::vector<uint16_t> lconn4;  // [Ne][4] shared-memory node slots (shift + i interior, hb + j halo), 4th lane = 0
    std::vector<double> g12;       // [Ne][4] = (dx phi1, dy phi1, dx phi2, dy phi2); grad phi3 = -(1+2)
    std::vector<double> area;      // [Ne]
    std::vector<double> mass;      // [N] lumped mass, internal order
    std::vector<ChunkMeta> meta;
    std::vector<int32_t> halo_ids;  // global internal ids (all >= N_int)
    std::vector<uint16_t> ell;      // slot index corner * EC + local element; padding entries = 3 * EC (zero slot)
    std::vector<int32_t> sh_rowptr;  // per interface node: its range of partial slots (ascending chunk order)
    std::vector<int32_t> halo_dst;   // per (chunk, halo node) entry: the partial slot it writes
    std::vector<double> xy_user;    // copy of the input coordinates (traction lengths)
};

// Builds everything above. chunk_elems = 0 picks the default and shrinks it until three CTAs fit one SM;
// an explicit chunk_elems is only shrunk when a single CTA would not fit.  Returns PFF_OK or an error with `err` filled.
pff_status build_host_mesh(int64_t n_nodes, const double* xy, int64_t n_elems, const int32_t* tri,
                           double rho, int order, int chunk_elems, size_t real_bytes, HostMesh& hm, std::string& err);

constexpr size_t kSmemPerSM = 227 * 1024;   // usable shared memory of one sm_100a SM / one CTA
constexpr size_t kSmemCtaReserve = 1024;    // driver-reserved bytes per resident CTA
constexpr size_t kSmemStatic = 2304;        // static shared memory of the chunk kernels (reduction scratch)

void set_error(const std::string& s);

}  // namespace pff
