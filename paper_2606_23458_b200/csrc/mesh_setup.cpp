// Host-side mesh setup (Eq. 9): orientation, P1 geometry, lumped mass,
// h_min, element ordering along a Morton curve, CTA chunks with interior-first / interface-last node
// numbering, chunk-local connectivity and the shared-memory gather tables.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <numeric>
#include <thread>

#include "pff_internal.h"

namespace pff {

static inline uint32_t spread16(uint32_t v)
{
    v &= 0xFFFFu;
    v = (v | (v << 8)) & 0x00FF00FFu;
    v = (v | (v << 4)) & 0x0F0F0F0Fu;
    v = (v | (v << 2)) & 0x33333333u;
    v = (v | (v << 1)) & 0x55555555u;
    return v;
}

// Recursive coordinate bisection of the (Morton-ordered) elements into chunks of exactly EC elements (the last one
// ragged): every cut is a median cut across the longer side of the bounding box of the centroids, placed at a
// multiple of EC, so the chunks are compact near-square patches whatever EC is (a Morton range of a length that is
// not a power of two is ragged and has ~1.7x more interface nodes).  Leaves keep Morton order inside.
static void bisect_into_chunks(const std::vector<int32_t>& morton_order, const std::vector<float>& cx,
                               const std::vector<float>& cy, int EC, std::vector<int32_t>& elem_old_of_new)
{
    const int64_t Ne = (int64_t)morton_order.size();
    std::vector<int32_t> pos(Ne);  // positions in Morton order, permuted in place
    std::iota(pos.begin(), pos.end(), 0);
    struct Range { int64_t lo, hi; };
    std::vector<Range> stack{{0, Ne}};
    while (!stack.empty()) {
        const Range r = stack.back();
        stack.pop_back();
        const int64_t n = r.hi - r.lo, chunks = (n + EC - 1) / EC;
        if (chunks <= 1) { std::sort(pos.begin() + r.lo, pos.begin() + r.hi); continue; }
        float x0 = 3.4e38f, x1 = -3.4e38f, y0 = 3.4e38f, y1 = -3.4e38f;
        for (int64_t i = r.lo; i < r.hi; ++i) {
            const int32_t e = pos[i];
            x0 = std::min(x0, cx[e]); x1 = std::max(x1, cx[e]); y0 = std::min(y0, cy[e]); y1 = std::max(y1, cy[e]);
        }
        const std::vector<float>& key = (x1 - x0 >= y1 - y0) ? cx : cy;
        const int64_t mid = r.lo + (chunks / 2) * EC;
        std::nth_element(pos.begin() + r.lo, pos.begin() + mid, pos.begin() + r.hi,
                         [&](int32_t a, int32_t b) { return key[a] < key[b] || (key[a] == key[b] && a < b); });
        stack.push_back({mid, r.hi});
        stack.push_back({r.lo, mid});
    }
    for (int64_t i = 0; i < Ne; ++i) elem_old_of_new[i] = morton_order[pos[i]];
}

// Bank balance of the gather table.  Column w of the table is read by a warp as 32 consecutive local nodes, each fetching
// the result slot of its w-th incident element: slots idx and idx' collide when idx = idx' (mod n_banks) (n_banks slots
// of one real span the 128-byte bank row), and a column costs as many shared-memory wavefronts as its fullest class.  The
// order of a node's incident elements is free (it only fixes the order of its sum), so per group of 32 nodes the entries
// are dealt to the columns greedily, each to the free column where its class is rarest, followed by two sweeps of
// pairwise swaps that lower the wavefront count; padding entries (the zero slot, read as a broadcast) fill the rest.
// On the 10^6-node square this takes the slot reads from 4.1 to 2.6 wavefronts per column (the floor is 1.8).
static void balance_gather_columns(uint16_t* T, int nloc, int W, uint16_t pad, int n_banks)
{
    if (W < 2 || W > 32) return;
    std::vector<int> cc(size_t(W) * n_banks);
    std::vector<uint16_t> out;
    int mx[32];
    auto colmax = [&](int c) { int mx = 0; for (int b = 0; b < n_banks; ++b) mx = std::max(mx, cc[size_t(c) * n_banks + b]); return mx; };
    for (int g0 = 0; g0 < nloc; g0 += 32) {
        const int gn = std::min(32, nloc - g0);
        std::fill(cc.begin(), cc.end(), 0);
        out.assign(size_t(W) * gn, pad);
        for (int i = 0; i < gn; ++i) {
            unsigned used = 0;
            for (int w = 0; w < W; ++w) {
                const uint16_t idx = T[size_t(w) * nloc + g0 + i];
                if (idx == pad) continue;
                const int cl = idx % n_banks;
                int best = -1;
                for (int c = 0; c < W; ++c)
                    if (!((used >> c) & 1u) && (best < 0 || cc[size_t(c) * n_banks + cl] < cc[size_t(best) * n_banks + cl])) best = c;
                used |= 1u << best;
                ++cc[size_t(best) * n_banks + cl];
                out[size_t(best) * gn + i] = idx;
            }
        }
        for (int c = 0; c < W; ++c) mx[c] = colmax(c);
        for (int sweep = 0; sweep < 2; ++sweep) {
            bool any = false;
            for (int i = 0; i < gn; ++i)
                for (int a = 0; a < W; ++a)
                    for (int b = a + 1; b < W; ++b) {
                        const uint16_t xa = out[size_t(a) * gn + i], xb = out[size_t(b) * gn + i];
                        const int ca = xa == pad ? -1 : xa % n_banks, cb = xb == pad ? -1 : xb % n_banks;
                        if (ca == cb) continue;
                        int* A = &cc[size_t(a) * n_banks];
                        int* B = &cc[size_t(b) * n_banks];
                        // the swap moves class ca from column a to b and class cb from b to a
                        const bool grows = (cb >= 0 && A[cb] + 1 > mx[a]) || (ca >= 0 && B[ca] + 1 > mx[b]);
                        const bool may_drop = (ca >= 0 && A[ca] == mx[a]) || (cb >= 0 && B[cb] == mx[b]);
                        int sq = 0;  // change of the sum of squared class counts: the tie-break
                        if (ca >= 0) sq += 2 * (B[ca] - A[ca]) + 2;
                        if (cb >= 0) sq += 2 * (A[cb] - B[cb]) + 2;
                        if (!may_drop && (grows || sq >= 0)) continue;
                        if (ca >= 0) { --A[ca]; ++B[ca]; }
                        if (cb >= 0) { --B[cb]; ++A[cb]; }
                        const int na = colmax(a), nb = colmax(b), m0 = mx[a] + mx[b], m1 = na + nb;
                        if (m1 < m0 || (m1 == m0 && sq < 0)) {
                            std::swap(out[size_t(a) * gn + i], out[size_t(b) * gn + i]);
                            mx[a] = na; mx[b] = nb; any = true;
                        } else {
                            if (ca >= 0) { ++A[ca]; --B[ca]; }
                            if (cb >= 0) { ++B[cb]; --A[cb]; }
                        }
                    }
            if (!any) break;
        }
        for (int w = 0; w < W; ++w)
            for (int i = 0; i < gn; ++i) T[size_t(w) * nloc + g0 + i] = out[size_t(w) * gn + i];
    }
}

pff_status build_host_mesh(int64_t N, const double* xy, int64_t Ne, const int32_t* tri_in, double rho,
                           int order, int chunk_elems, size_t real_bytes, HostMesh& hm, std::string& err, int cg_ctas)
{
    if (N < 3 || Ne < 1) { err = "mesh needs at least 3 nodes and 1 element"; return PFF_EINVAL; }
    if (N >= (int64_t(1) << 30) || Ne >= (int64_t(1) << 30)) { err = "mesh too large (>= 2^30)"; return PFF_EMESH; }
    hm.N = N; hm.Ne = Ne;
    hm.xy_user.assign(xy, xy + 2 * N);

    // ---- orientation, areas, Eq. 9 gradients (fp64), h_min, in user order
    std::vector<int32_t> tri(3 * Ne);
    std::vector<double> g12u(4 * Ne), areau(Ne);
    double xmin = std::numeric_limits<double>::infinity(), xmax = -xmin, ymin = xmin, ymax = -xmin;
    for (int64_t i = 0; i < N; ++i) {
        double x = xy[2 * i], y = xy[2 * i + 1];
        if (!std::isfinite(x) || !std::isfinite(y)) { err = "non-finite node coordinate"; return PFF_EMESH; }
        xmin = std::min(xmin, x); xmax = std::max(xmax, x);
        ymin = std::min(ymin, y); ymax = std::max(ymax, y);
    }
    double hmin = std::numeric_limits<double>::infinity();
    for (int64_t e = 0; e < Ne; ++e) {
        int32_t n1 = tri_in[3 * e], n2 = tri_in[3 * e + 1], n3 = tri_in[3 * e + 2];
        if (n1 < 0 || n2 < 0 || n3 < 0 || n1 >= N || n2 >= N || n3 >= N) {
            err = "element " + std::to_string(e) + ": node index out of range"; return PFF_EMESH;
        }
        double x1 = xy[2 * n1], y1 = xy[2 * n1 + 1], x2 = xy[2 * n2], y2 = xy[2 * n2 + 1];
        double x3 = xy[2 * n3], y3 = xy[2 * n3 + 1];
        double twoA = (x2 - x1) * (y3 - y1) - (x3 - x1) * (y2 - y1);
        if (twoA < 0.0) { std::swap(n2, n3); std::swap(x2, x3); std::swap(y2, y3); twoA = -twoA; }
        double l12 = std::hypot(x2 - x1, y2 - y1), l23 = std::hypot(x3 - x2, y3 - y2), l31 = std::hypot(x1 - x3, y1 - y3);
        double lmax = std::max(l12, std::max(l23, l31));
        if (!(0.5 * twoA > 1e-14 * lmax * lmax)) {
            err = "element " + std::to_string(e) + ": zero or near-zero area"; return PFF_EMESH;
        }
        tri[3 * e] = n1; tri[3 * e + 1] = n2; tri[3 * e + 2] = n3;
        areau[e] = 0.5 * twoA;
        g12u[4 * e + 0] = (y2 - y3) / twoA; g12u[4 * e + 1] = (x3 - x2) / twoA;
        g12u[4 * e + 2] = (y3 - y1) / twoA; g12u[4 * e + 3] = (x1 - x3) / twoA;
        hmin = std::min(hmin, 4.0 * areau[e] / (l12 + l23 + l31));
    }
    hm.hmin = hmin;

    // ---- element order: Morton key of the centroid (or user order)
    std::vector<int32_t> elem_old_of_new(Ne);
    std::vector<float> ccx, ccy;  // centroids in Morton order (bisection only)
    if (order == PFF_ORDER_MORTON || order == PFF_ORDER_BISECTION) {
        std::vector<uint64_t> keyed(Ne);
        double sx = (xmax > xmin) ? 65535.0 / (xmax - xmin) : 0.0, sy = (ymax > ymin) ? 65535.0 / (ymax - ymin) : 0.0;
        for (int64_t e = 0; e < Ne; ++e) {
            const int32_t* t = &tri[3 * e];
            double cx = (xy[2 * t[0]] + xy[2 * t[1]] + xy[2 * t[2]]) / 3.0;
            double cy = (xy[2 * t[0] + 1] + xy[2 * t[1] + 1] + xy[2 * t[2] + 1]) / 3.0;
            uint32_t qx = (uint32_t)std::min(65535.0, std::max(0.0, (cx - xmin) * sx));
            uint32_t qy = (uint32_t)std::min(65535.0, std::max(0.0, (cy - ymin) * sy));
            uint32_t key = spread16(qx) | (spread16(qy) << 1);
            keyed[e] = (uint64_t(key) << 32) | uint64_t(uint32_t(e));
        }
        std::sort(keyed.begin(), keyed.end());
        for (int64_t e = 0; e < Ne; ++e) elem_old_of_new[e] = int32_t(keyed[e] & 0xFFFFFFFFu);
        if (order == PFF_ORDER_BISECTION) {
            ccx.resize(Ne); ccy.resize(Ne);
            for (int64_t e = 0; e < Ne; ++e) {
                // key = midpoint of the LONGEST edge: two triangles that share it (the two halves of a quad) get the
                // same key and stay on the same side of a cut, which keeps the cut lines straight
                const int32_t* t = &tri[3 * elem_old_of_new[e]];
                double best = -1.0, mx = 0.0, my = 0.0;
                for (int k = 0; k < 3; ++k) {
                    const int32_t p = t[k], q = t[(k + 1) % 3];
                    const double dx = xy[2 * p] - xy[2 * q], dy = xy[2 * p + 1] - xy[2 * q + 1], l2 = dx * dx + dy * dy;
                    if (l2 > best) { best = l2; mx = 0.5 * (xy[2 * p] + xy[2 * q]); my = 0.5 * (xy[2 * p + 1] + xy[2 * q + 1]); }
                }
                ccx[e] = float(mx - xmin);
                ccy[e] = float(my - ymin);
            }
        }
    } else {
        std::iota(elem_old_of_new.begin(), elem_old_of_new.end(), 0);
    }
    const std::vector<int32_t> morton_order = elem_old_of_new;  // bisection re-partitions this order per chunk size

    // ---- chunks; shrink the chunk until the shared-memory footprints of the chunk kernels fit.  Default chunk: the
    // largest size for which THREE double-buffered CTAs of the CG kernel (12 of 13 launches-worth of work per step)
    // and TWO of the step / setup kernels fit one SM (measured best, profiles/r1c); explicit chunk: one CTA of each.
    const int A = int(16 / real_bytes);  // reals per 16-byte TMA granule
    const bool user_chunk = chunk_elems > 0;
    int EC = user_chunk ? chunk_elems : (real_bytes == 8 ? 512 : 1024);
    EC = std::max(32, std::min(8192, (EC / 32) * 32));
    const size_t limit_cg = (user_chunk ? kSmemPerSM : kSmemPerSM / 3) - kSmemCtaReserve;
    const size_t limit_other = (user_chunk ? kSmemPerSM : kSmemPerSM / 2) - kSmemCtaReserve;
    std::vector<int32_t> cmin(N), cmax(N);
    bool balanced = false;  // the balance-aware choice below has been made
    for (;;) {
        if (order == PFF_ORDER_BISECTION) bisect_into_chunks(morton_order, ccx, ccy, EC, elem_old_of_new);
        std::fill(cmin.begin(), cmin.end(), std::numeric_limits<int32_t>::max());
        std::fill(cmax.begin(), cmax.end(), -1);
        for (int64_t en = 0; en < Ne; ++en) {
            int32_t c = int32_t(en / EC);
            const int32_t* t = &tri[3 * elem_old_of_new[en]];
            for (int k = 0; k < 3; ++k) { cmin[t[k]] = std::min(cmin[t[k]], c); cmax[t[k]] = std::max(cmax[t[k]], c); }
        }
        // per-chunk local node count and valence (bounds for the staged array lengths) via first-touch stamps
        int64_t C = (Ne + EC - 1) / EC;
        std::vector<int32_t> stamp(N, -1), valence(N, 0);
        int32_t max_nloc = 0, max_ell = 0, max_nh = 0;
        for (int64_t c = 0; c < C; ++c) {
            int32_t nloc = 0, w = 0, nh = 0;
            for (int64_t en = c * EC; en < std::min<int64_t>(Ne, (c + 1) * EC); ++en) {
                const int32_t* t = &tri[3 * elem_old_of_new[en]];
                for (int k = 0; k < 3; ++k) {
                    if (stamp[t[k]] != c) { stamp[t[k]] = int32_t(c); valence[t[k]] = 0; ++nloc; nh += cmin[t[k]] != cmax[t[k]]; }
                    w = std::max(w, ++valence[t[k]]);
                }
            }
            max_nloc = std::max(max_nloc, nloc);
            max_nh = std::max(max_nh, nh);
            max_ell = std::max(max_ell, w * nloc);
        }
        const int node_len_b = (max_nloc + 2 * A + A - 1) / A * A, flag_len_b = (max_nloc + 32 + 15) / 16 * 16;
        const int ell_len_b = (max_ell + 7) / 8 * 8;
        // dynamic + static shared memory per kernel (the step kernel has no static part)
        const size_t smem_step = chunk_smem_bytes(0, EC, node_len_b, flag_len_b, ell_len_b, max_nh, real_bytes);
        const size_t smem_cg = chunk_smem_bytes(1, EC, node_len_b, flag_len_b, ell_len_b, max_nh, real_bytes) + kSmemStatic;
        const size_t smem_su = chunk_smem_bytes(2, EC, node_len_b, flag_len_b, ell_len_b, max_nh, real_bytes) + kSmemStatic;
        const bool fits = smem_cg <= limit_cg && std::max(smem_step, smem_su) <= limit_other && max_nloc < 16384;
        if (fits || EC <= 32) {
            if (std::max(smem_cg, std::max(smem_step, smem_su)) > kSmemPerSM - kSmemCtaReserve) {
                err = "chunk does not fit shared memory"; return PFF_EMESH;
            }
            if (!user_chunk && !balanced && EC > 128) {
                // EC is the largest chunk that fits.  The persistent CG kernel (most of a staggered step) gives CTA b the
                // chunks b, b + G, ...: its chunk phase lasts ceil(C / G) chunks, so a chunk count just above a multiple of
                // G leaves most CTAs idle for a whole chunk (fp32 at 10^6 nodes: 3125 chunks of 640 on 444 CTAs = 8 rounds
                // where 7.04 would do).  Pick, among the sizes that fit, the one with the smallest modelled phase length:
                // rounds x (chunk + a fixed per-chunk cost), weighted by the growth of the interface (~ 1 / sqrt(chunk)).
                balanced = true;
                const int64_t G = cg_ctas > 0 ? cg_ctas : 444;
                auto cost = [&](int ec) {
                    const int64_t rounds = ((Ne + ec - 1) / ec + G - 1) / G;
                    return double(rounds) * double(ec + 60) * (1.0 + 0.3 * (std::sqrt(double(EC) / double(ec)) - 1.0));
                };
                int best = EC;
                for (int ec = EC - 32; ec >= 128; ec -= 32)
                    if (cost(ec) < 0.97 * cost(best)) best = ec;  // only a clear gain justifies more interface nodes
                if (best != EC) { EC = best; continue; }
            }
            hm.max_nloc = max_nloc; hm.C = C;
            break;
        }
        {   // footprints are nearly linear in EC: jump close to the fitting size, then step down by 32
            const double ratio = std::min(double(limit_cg) / double(smem_cg), double(limit_other) / double(std::max(smem_step, smem_su)));
            const int jump = int(EC * std::min(ratio, 1.0)) / 32 * 32 + 32;
            EC = std::max(32, std::min(EC - 32, jump));
        }
    }
    hm.chunk_elems = EC;
    hm.elem_new_of_old.resize(Ne);
    for (int64_t e = 0; e < Ne; ++e) hm.elem_new_of_old[elem_old_of_new[e]] = int32_t(e);
    const int64_t C = hm.C;
    for (int64_t i = 0; i < N; ++i)
        if (cmax[i] < 0) { err = "node " + std::to_string(i) + " belongs to no element (orphan)"; return PFF_EMESH; }

    // ---- node numbering: chunk by chunk the interior nodes in first-touch order, then interface nodes
    hm.node_new_of_old.assign(N, -1);
    hm.meta.resize(C);
    int32_t next = 0;
    for (int64_t c = 0; c < C; ++c) {
        ChunkMeta& m = hm.meta[c];
        m.elem_start = int32_t(c * EC);
        m.n_elem = int32_t(std::min<int64_t>(Ne, (c + 1) * EC) - c * EC);
        m.node_start = next;
        for (int64_t en = m.elem_start; en < m.elem_start + m.n_elem; ++en) {
            const int32_t* t = &tri[3 * elem_old_of_new[en]];
            for (int k = 0; k < 3; ++k)
                if (cmin[t[k]] == cmax[t[k]] && hm.node_new_of_old[t[k]] < 0) hm.node_new_of_old[t[k]] = next++;
        }
        m.n_int = next - m.node_start;
    }
    hm.N_int = next;
    for (int64_t en = 0; en < Ne; ++en) {
        const int32_t* t = &tri[3 * elem_old_of_new[en]];
        for (int k = 0; k < 3; ++k)
            if (hm.node_new_of_old[t[k]] < 0) hm.node_new_of_old[t[k]] = next++;
    }
    hm.N_sh = N - hm.N_int;
    hm.node_old_of_new.resize(N);
    for (int64_t i = 0; i < N; ++i) hm.node_old_of_new[hm.node_new_of_old[i]] = int32_t(i);

    // ---- per-chunk tables
    hm.conn4.assign(4 * Ne, 0);
    hm.lconn4.assign(4 * Ne, 0);
    hm.g12.resize(4 * Ne);
    hm.area.resize(Ne);
    hm.mass.assign(N, 0.0);
    std::vector<int32_t> sh_stamp(hm.N_sh, -1), sh_local(hm.N_sh, 0), sh_count(hm.N_sh + 1, 0);
    std::vector<int32_t> val;  // valence per local node
    std::vector<int32_t> lloc(size_t(3) * EC);  // chunk-local node index of each element corner
    hm.halo_ids.clear();
    hm.ell.clear();
    for (int64_t c = 0; c < C; ++c) {
        ChunkMeta& m = hm.meta[c];
        m.halo_off = int32_t(hm.halo_ids.size());
        int32_t nh = 0;
        for (int64_t en = m.elem_start; en < m.elem_start + m.n_elem; ++en) {
            int64_t eo = elem_old_of_new[en];
            for (int k = 0; k < 3; ++k) {
                int32_t g = hm.node_new_of_old[tri[3 * eo + k]];
                int32_t l;  // chunk-local node index: interior first, then halo in first-touch order
                if (g < hm.N_int) l = g - m.node_start;
                else {
                    int32_t s = g - int32_t(hm.N_int);
                    if (sh_stamp[s] != c) { sh_stamp[s] = int32_t(c); sh_local[s] = nh++; hm.halo_ids.push_back(g); ++sh_count[s + 1]; }
                    l = m.n_int + sh_local[s];
                }
                hm.conn4[4 * en + k] = g;
                lloc[3 * (en - m.elem_start) + k] = l;
            }
            for (int k = 0; k < 4; ++k) hm.g12[4 * en + k] = g12u[4 * eo + k];
            hm.area[en] = areau[eo];
        }
        m.n_halo = nh;
        const int32_t nloc = m.n_int + nh;
        // shared-memory slot of a local node: staged arrays hold [shift | interior | pad to 16 B | halo]
        const int32_t shift = m.node_start % A, hb = (shift + m.n_int + A - 1) / A * A;
        for (int64_t en = m.elem_start; en < m.elem_start + m.n_elem; ++en)
            for (int k = 0; k < 3; ++k) {
                const int32_t l = lloc[3 * (en - m.elem_start) + k];
                hm.lconn4[4 * en + k] = uint16_t(l < m.n_int ? shift + l : hb + (l - m.n_int));
            }
        hm.node_len = std::max(hm.node_len, (hb + nh + A - 1) / A * A);
        hm.flag_len = std::max(hm.flag_len, (m.node_start % 16 + m.n_int + 15) / 16 * 16);
        hm.max_nhalo = std::max(hm.max_nhalo, nh);
        val.assign(nloc, 0);
        for (int64_t en = m.elem_start; en < m.elem_start + m.n_elem; ++en)
            for (int k = 0; k < 3; ++k) ++val[lloc[3 * (en - m.elem_start) + k]];
        int32_t w = 0;
        for (int32_t i = 0; i < nloc; ++i) w = std::max(w, val[i]);
        m.ell_w = w;
        hm.ell.resize((hm.ell.size() + 7) / 8 * 8, uint16_t(3 * EC));  // 16-byte aligned table start
        m.ell_off = int32_t(hm.ell.size());
        hm.ell_len = std::max(hm.ell_len, (w * nloc + 7) / 8 * 8);
        if (hm.ell.size() + size_t(w) * nloc > size_t(std::numeric_limits<int32_t>::max())) {
            err = "gather table too large"; return PFF_EMESH;
        }
        hm.ell.resize(hm.ell.size() + size_t(w) * nloc, uint16_t(3 * EC));  // padding -> zero slot
        std::fill(val.begin(), val.end(), 0);
        for (int64_t en = m.elem_start; en < m.elem_start + m.n_elem; ++en)
            for (int k = 0; k < 3; ++k) {
                int32_t l = lloc[3 * (en - m.elem_start) + k];
                hm.ell[size_t(m.ell_off) + size_t(val[l]++) * nloc + l] = uint16_t(k * EC + (en - m.elem_start));
            }
        hm.max_ell_w = std::max(hm.max_ell_w, w);
    }
    hm.ell.resize((hm.ell.size() + 7) / 8 * 8 + 8, uint16_t(3 * EC));  // the widened TMA copy stays in bounds
    {   // bank balance of every chunk's table (chunks are independent: spread over the host cores; the result does not
        // depend on the thread count)
        const unsigned nt = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
        std::vector<std::thread> pool;
        for (unsigned t = 0; t < nt; ++t)
            pool.emplace_back([&, t]() {
                for (int64_t c = t; c < C; c += nt) {
                    const ChunkMeta& m = hm.meta[c];
                    balance_gather_columns(hm.ell.data() + m.ell_off, m.n_int + m.n_halo, m.ell_w, uint16_t(3 * EC), int(128 / real_bytes));
                }
            });
        for (auto& th : pool) th.join();
    }
    // interface-node CSR over halo slots, ascending chunk (chunks were visited in order)
    // Partial slots: kIfaceWidth fixed slots per interface node (slot kIfaceWidth * s + k for the k-th touching chunk,
    // ascending chunk order; never-written slots stay zero), the rare further ones in an overflow CSR behind them.
    hm.sh_rowptr.assign(hm.N_sh + 1, 0);
    for (int64_t s = 0; s < hm.N_sh; ++s)
        hm.sh_rowptr[s + 1] = hm.sh_rowptr[s] + std::max(0, sh_count[s + 1] - kIfaceWidth);
    hm.n_ovf = hm.sh_rowptr[hm.N_sh];
    hm.halo_dst.resize(hm.halo_ids.size());
    std::vector<int32_t> fill(hm.N_sh, 0);
    for (size_t slot = 0; slot < hm.halo_ids.size(); ++slot) {
        int32_t s = hm.halo_ids[slot] - int32_t(hm.N_int);
        const int32_t k = fill[s]++;
        hm.halo_dst[slot] = k < kIfaceWidth ? kIfaceWidth * s + k : int32_t(kIfaceWidth * hm.N_sh) + hm.sh_rowptr[s] + (k - kIfaceWidth);
    }
    // lumped mass m_i = rho sum A_e / 3 (L169), summed in internal element order
    for (int64_t en = 0; en < Ne; ++en)
        for (int k = 0; k < 3; ++k) hm.mass[hm.conn4[4 * en + k]] += rho * hm.area[en] / 3.0;
    return PFF_OK;
}

// Bounds proof of the widened bulk copies (stage_issue_desc, pff_tma.cuh), chunk by chunk: the device copies the
// 16-byte-granule cover [a0, a1) of every contiguous range it stages, a0 = start rounded down, a1 = end rounded up but
// never beyond the last full granule of the array.  Here the same arithmetic is restated on the host and checked
// against (i) the array length (source side) and (ii) the capacity of the stage region the range lands in
// (destination side: the lengths make_stage_layout is given).  Also checks that the (bank-balanced) gather table of every
// chunk is exactly the node-element incidence.  Any violation fails mesh creation.
bool verify_stage_extents(const HostMesh& hm, int64_t ell_total, int64_t n_entries, size_t rb, std::string& err)
{
    struct Range { int64_t start, count, total; int esize; int64_t cap_bytes; const char* what; };
    auto up16 = [](int64_t v) { return (v + 15) / 16 * 16; };
    const int EC = hm.chunk_elems;
    for (int64_t c = 0; c < hm.C; ++c) {
        const ChunkMeta& m = hm.meta[c];
        const int64_t nloc = m.n_int + m.n_halo;
        const int64_t next_off = c + 1 < hm.C ? hm.meta[c + 1].halo_off : 0, next_n = c + 1 < hm.C ? hm.meta[c + 1].n_halo : 0;
        const Range rs[] = {
            {m.elem_start, m.n_elem, hm.Ne, 8, up16(8 * (int64_t)EC), "local connectivity"},
            {m.elem_start, m.n_elem, hm.Ne, 16, 16 * (int64_t)EC, "geometry / coefficient pair"},
            {m.elem_start, m.n_elem, hm.Ne, (int)rb, up16((int64_t)rb * EC), "area / history"},
            {m.node_start, m.n_int, hm.N, (int)rb, up16((int64_t)rb * hm.node_len), "nodal array"},
            {m.node_start, m.n_int, hm.N, 1, up16(hm.flag_len), "flag bytes"},
            {m.ell_off, (int64_t)m.ell_w * nloc, ell_total, 2, up16(2 * (int64_t)hm.ell_len), "gather table"},
            {m.halo_off, m.n_halo, n_entries, 4, up16(4 * ((int64_t)hm.max_nhalo + 4)), "halo partial slots"},
            {next_off, next_n, n_entries, 4, up16(4 * ((int64_t)hm.max_nhalo + 4)), "next chunk's halo ids"},
        };
        for (const Range& r : rs) {
            if (r.count <= 0) continue;
            const int64_t A1 = 16 / r.esize - 1;
            const int64_t a0 = r.start & ~A1, end = r.start + r.count;
            const int64_t a1 = std::max(a0, std::min((end + A1) & ~A1, r.total & ~A1));
            const bool src_ok = a0 >= 0 && a1 <= r.total && end <= r.total;
            // destination: the bulk part [a0, a1) and the plain-load tail [a1, end) both land at (index - a0) * esize
            const bool dst_ok = (std::max(a1, end) - a0) * r.esize <= r.cap_bytes;
            if (!src_ok || !dst_ok) {
                err = std::string("internal: staged range of the ") + r.what + " of chunk " + std::to_string(c) +
                      (src_ok ? " overruns its shared-memory region" : " leaves its array");
                return false;
            }
        }
        // halo nodes sit behind the interior block of every staged nodal array
        const int64_t A = 16 / (int64_t)rb, hb = ((m.node_start % A) + m.n_int + A - 1) / A * A;
        if (hb + m.n_halo > hm.node_len || m.n_halo > hm.max_nhalo) {
            err = "internal: halo slots of chunk " + std::to_string(c) + " overrun the staged nodal arrays";
            return false;
        }
        // gather table (after the bank balance): the row of a local node lists exactly the result slots corner * EC + e of
        // the element corners that reference it, each once; everything else is the zero slot
        {
            const uint16_t* T = hm.ell.data() + m.ell_off;
            const int64_t shift = m.node_start % A;
            std::vector<uint8_t> seen(size_t(3) * EC, 0);
            for (int64_t l = 0; l < nloc; ++l) {
                const uint16_t slot = uint16_t(l < m.n_int ? shift + l : hb + (l - m.n_int));
                for (int w = 0; w < m.ell_w; ++w) {
                    const int idx = T[size_t(w) * nloc + l];
                    if (idx == 3 * EC) continue;
                    const int k = idx / EC, e = idx % EC;
                    if (k > 2 || e >= m.n_elem || seen[idx] || hm.lconn4[4 * (m.elem_start + e) + k] != slot) {
                        err = "internal: gather table of chunk " + std::to_string(c) + " is not the incidence of its nodes";
                        return false;
                    }
                    seen[idx] = 1;
                }
            }
            for (int64_t e = 0; e < m.n_elem; ++e)
                for (int k = 0; k < 3; ++k)
                    if (!seen[size_t(k) * EC + e]) {
                        err = "internal: gather table of chunk " + std::to_string(c) + " misses an element corner";
                        return false;
                    }
        }
    }
    return true;
}

}  // namespace pff
