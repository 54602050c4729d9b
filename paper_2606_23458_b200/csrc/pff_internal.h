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
//   kind 1: damage iteration  x r p q 1/D lb + mask; scalar slots [3 EC + 1]  (one-rendezvous kernel: r p s w 1/D + halo partials)
//   kind 2: damage setup      x; scalar slots q, D, b each [3 EC + 1]
//   kind 5: kind 0 + the hold region of the fused damage setup (pff_step.cu MODE_STEPSU)
//   kind 3: quasi-static CG iteration (explicit-step kernel, MODE_EQ): 13 nodal arrays u_x u_y d p_x p_y r_x r_y q_x q_y
//                           1/D_x 1/D_y du_x du_y, no history array; force-pair slots as kind 0
constexpr int kIfaceWidth = 4;  // fixed partial slots per interface node (one per touching chunk)
struct StageLayout {
    // offsets relative to the base of a stage (stage s starts at s * stage_bytes)
    uint32_t lconn, geo, area, H, node[13], flags, ell;
    uint32_t hids, hflag, hdst;  // per halo node: global id, the 32-bit word holding its flag byte, its partial slot
    uint32_t hnext;              // global ids of the NEXT chunk's halo nodes (arrive with this stage, feed its gathers)
    uint32_t stage_bytes, n_stages;
    // absolute offsets of what the stages share
    uint32_t slot_base;    // the per-element result slots (one copy; only one stage computes at a time)
    uint32_t slot_stride;  // kind 2: bytes between the q, D, b slot arrays
    uint32_t meta;         // persistent kernels: ring of ChunkMeta of the chunks this CTA owns
    uint32_t hid0;         // persistent kernels: halo ids of the CTA's FIRST chunk (re-gathered every CG iteration)
    uint32_t hold;         // kind 5: (q, D) pairs of element corners 1 and 2 (fp32: 1, 2, 3) of the fused damage setup (one copy)
    uint32_t bar;          // one mbarrier per stage
    uint32_t total;
};
constexpr int kMetaCap = 32;  // chunk metas a persistent CTA keeps in shared memory per epoch
inline StageLayout make_stage_layout(int kind, int EC, int node_len, int flag_len, int ell_len, int max_nhalo, size_t rb,
                                     int n_stages = 1)
{
    StageLayout L{};
    auto up16 = [](size_t v) { return uint32_t((v + 15) / 16 * 16); };
    uint32_t o = 0;
    L.lconn = o; o += up16(size_t(8) * EC);
    L.geo = o; o += up16(size_t(4) * rb * EC);
    L.area = o; o += up16(kind == 1 ? 0 : rb * EC);  // kind 1 stages the 4 element-operator coefficients as "geometry"
    L.H = o; o += up16(kind == 1 || kind == 3 ? 0 : rb * EC);
    const bool fused = kind == 5;  // kind 5 = kind 0 + the hold region (explicit step with the damage setup fused in, fp64)
    if (fused) kind = 0;
    const int nn = kind == 0 ? 10 : (kind == 1 ? 6 : (kind == 3 ? 13 : 1));
    for (int k = 0; k < nn; ++k) {
        // kind 1, array 5: the lower bounds of the projected solver, or (one-rendezvous CG kernel) the kIfaceWidth partial
        // slots of every halo node
        const int len = (kind == 1 && k == 5) ? (node_len > kIfaceWidth * max_nhalo ? node_len : kIfaceWidth * max_nhalo) : node_len;
        L.node[k] = o; o += up16(rb * len);
    }
    L.flags = o; o += up16(flag_len);
    L.ell = o; o += up16(size_t(2) * ell_len);
    L.hids = o; o += up16(size_t(4) * max_nhalo);
    L.hflag = o; o += up16(size_t(4) * max_nhalo);
    L.hdst = o; o += up16(size_t(4) * (max_nhalo + 4));
    L.hnext = o; o += up16(n_stages > 1 ? size_t(4) * (max_nhalo + 4) : 0);
    L.stage_bytes = (o + 127) / 128 * 128;
    L.n_stages = uint32_t(n_stages);
    o = L.stage_bytes * uint32_t(n_stages);
    if (kind == 0 || kind == 3) {  // force-pair slots corner * EC + e (+ one zero pair).  fp64: corners 1, 2 overwrite the element's
        // own staged geometry (pair index into the stage's geometry) and only corner 3 + the zero pair live here
        L.slot_base = o; o += up16(rb == 8 ? size_t(16) * (EC + 1) : size_t(8) * (3 * EC + 1));
    }
    if (kind == 1) { L.slot_base = o; o += up16(rb * (size_t(3) * EC + 1)); }
    if (kind == 2) { L.slot_base = o; L.slot_stride = up16(rb * (size_t(3) * EC + 1)); o += 3 * L.slot_stride; }
    L.hold = o; o += up16(fused ? size_t(2) * rb * (rb == 8 ? 2 : 3) * EC : 0);  // fp32: all three corners (nothing to reuse there)
    L.meta = o; o += n_stages > 1 ? uint32_t(32 * kMetaCap) : 0;
    L.hid0 = o; o += up16(n_stages > 1 ? size_t(4) * max_nhalo : 0);
    L.bar = o; o += 16 * uint32_t(n_stages);
    L.total = o;
    return L;
}
// stages of each chunk kernel: all three (step, CG, damage setup) are persistent and double-buffered
inline int chunk_kernel_stages(int) { return 2; }
inline size_t chunk_smem_bytes(int kind, int EC, int node_len, int flag_len, int ell_len, int max_nhalo, size_t rb)
{
    return make_stage_layout(kind, EC, node_len, flag_len, ell_len, max_nhalo, rb, chunk_kernel_stages(kind)).total;
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
    std::vector<int32_t> sh_rowptr;  // per interface node: its range in the OVERFLOW partial slots (all zero on regular meshes)
    int32_t n_ovf = 0;               // overflow partial slots
    std::vector<int32_t> halo_dst;   // per (chunk, halo node) entry: the partial slot it writes
    std::vector<double> xy_user;    // copy of the input coordinates (traction lengths)
};

// Builds everything above. chunk_elems = 0 picks the default: the largest size for which three CTAs fit one SM, then the
// best-balanced size at or below it for the persistent CG kernel's grid (mesh_setup.cpp);
// an explicit chunk_elems is only shrunk when a single CTA would not fit.  Returns PFF_OK or an error with `err` filled.
pff_status build_host_mesh(int64_t n_nodes, const double* xy, int64_t n_elems, const int32_t* tri,
                           double rho, int order, int chunk_elems, size_t real_bytes, HostMesh& hm, std::string& err,
                           int cg_ctas = 0);  // CTAs of the persistent CG kernel on the target GPU (0: a B200's 444)

// Host-side bounds proof of every staged (widened) copy of every chunk; false + `err` on violation (mesh_setup.cpp).
bool verify_stage_extents(const HostMesh& hm, int64_t ell_total, int64_t n_entries, size_t real_bytes, std::string& err);

constexpr size_t kSmemPerSM = 227 * 1024;   // usable shared memory of one sm_100a SM / one CTA
constexpr size_t kSmemCtaReserve = 1024;    // driver-reserved bytes per resident CTA
constexpr size_t kSmemStatic = 1280;        // static shared memory of the damage chunk kernels (reduction scratch 8 x 16 doubles,
                                            // control block; checked against ptxas: 1,208 B)

void set_error(const std::string& s);

}  // namespace pff
