// Geometric-multigrid-preconditioned CG for the AT2 damage solve ("preconditioned
// conjugate gradients ... AMG typically reducing the CG iteration count by a factor of 5 to 20 on fine meshes").
//
// The caller supplies a hierarchy of coarser meshes of the same domain (each an ordinary pff_mesh); the library builds,
// on the host, the P1 interpolation P_l from level l + 1 to level l by point location (every node of level l in a
// triangle of level l + 1, barycentric weights), its transpose as a gather table, and the parent element of every
// element of level l.  Coarse operators are RE-DISCRETISED: the same matrix-free operator (Gc / l0 + 2 H) M + Gc l0 K
// (L173, L185) on the coarse mesh with the history field averaged over each coarse element's children (area weights; the
// operator is linear in H).  One V(1,1) cycle with damped-Jacobi smoothing is the preconditioner:
//     x = w D^-1 b;  r = b - A x;  x += P V_{l+1}(P^T r);  x += w D^-1 (b - A x)          (coarsest: k Jacobi sweeps)
// symmetric and positive definite for w lambda_max(D^-1 A) < 2 (P1 mass + stiffness: lambda_max <= 2, w = 2/3), so the
// outer iteration is plain PCG and converges to the same unique solution as the Jacobi-PCG of pff_damage_solve.
// Every operator application is the chunk kernel of pff_damage.cu (plain mode); everything else is the small vector
// kernels below.  All reductions have a fixed order (block partials summed by the last block in index order).
#include <algorithm>
#include <atomic>
#include <cmath>
#include <functional>
#include <thread>
#include <string>
#include <vector>

#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

#define MG_CUDA(call)                                         \
    do {                                                      \
        pff_status st__ = pff::cuda_check((call), #call);     \
        if (st__ != PFF_OK) return st__;                      \
    } while (0)

struct MgTransfer {  // level l (fine) <-> level l + 1 (coarse); device arrays, internal numbering of both meshes
    int32_t* p_idx = nullptr;  // [3 N_l] coarse nodes of the triangle that holds fine node i
    void* p_w = nullptr;       // [3 N_l] barycentric weights
    int32_t *r_ptr = nullptr, *r_idx = nullptr;  // P^T as CSR over coarse nodes (entries ascending in the fine index)
    void* r_w = nullptr;
    int32_t *c_ptr = nullptr, *c_idx = nullptr;  // children (fine elements) of every coarse element
    void* c_w = nullptr;                         // area of the child / area of all children
};

struct MgLevel {
    pff_mesh* m = nullptr;
    pff_state st{};  // level >= 1: d = 0, H = restricted history; level 0: the caller's state
    void *b = nullptr, *x = nullptr, *t = nullptr, *dinv = nullptr, *zero = nullptr, *H = nullptr;
    MgTransfer tr;  // to the next coarser level (unused on the coarsest)
};

struct MgData {
    std::vector<MgLevel> lv;
    void *r = nullptr, *p = nullptr, *q = nullptr, *lb = nullptr;  // outer PCG vectors (finest level; z is level 0's x)
    void* dfull = nullptr;  // AT1: 1/D of every non-fixed node (level 0's dinv then holds the inactive set's)
    double *part = nullptr, *sc = nullptr, *h_sc = nullptr;
    unsigned int* ticket = nullptr;
    int n_part = 0;
    double omega = 2.0 / 3.0;
    int coarse_sweeps = 4;
    int last_cycles = 0;
    // one outer iteration (V-cycle, both inner products, direction and update: ~50 small launches) captured once and
    // replayed; key = everything the captured kernel arguments depend on
    // (two entries: the forward solve iterates on state->d, the adjoint solve on lambda)
    struct Graph {
        cudaGraphExec_t exec = nullptr;
        const void *x = nullptr, *b = nullptr;
        double omega = 0.0;
        int sweeps = 0, launches = 0;
        unsigned long long used = 0;
    } graphs[2];
    unsigned long long graph_clock = 0;
    cudaStream_t cap_stream = nullptr;
    bool graph_refused = false;
};

struct MgAdjoint {  // pff_damage_adjoint through the multigrid solver: right-hand side g, caller-given free set, result lambda
    const void* g;
    const uint8_t* free_mask;
    void* lambda;
};

enum { SC_PQ = 0, SC_RZ = 1, SC_RR = 2, SC_RZN = 3, SC_BB = 4, SC_R0 = 5, SC_CHG = 6, SC_N = 8 };

// ---- host: point location of the nodes / element centroids of a fine mesh in the triangles of a coarse mesh --------------
struct Locator {
    const HostMesh& c;
    double x0, y0, inv;
    int nb;
    std::vector<int32_t> ptr, items;
    const double* xy(int32_t node) const { return &c.xy_user[2 * size_t(c.node_old_of_new[node])]; }
    explicit Locator(const HostMesh& cm) : c(cm)
    {
        double x1 = -1e300, y1 = -1e300;
        x0 = y0 = 1e300;
        for (int64_t i = 0; i < c.N; ++i) {
            x0 = std::min(x0, c.xy_user[2 * i]); x1 = std::max(x1, c.xy_user[2 * i]);
            y0 = std::min(y0, c.xy_user[2 * i + 1]); y1 = std::max(y1, c.xy_user[2 * i + 1]);
        }
        nb = std::max(1, (int)std::sqrt(double(c.Ne) / 2.0));
        const double ext = std::max(std::max(x1 - x0, y1 - y0), 1e-300);
        inv = nb / ext;
        std::vector<int32_t> cnt(size_t(nb) * nb + 1, 0);
        auto range = [&](int64_t e, int& i0, int& i1, int& j0, int& j1) {
            double ax = 1e300, bx = -1e300, ay = 1e300, by = -1e300;
            for (int k = 0; k < 3; ++k) {
                const double* p = xy(c.conn4[4 * e + k]);
                ax = std::min(ax, p[0]); bx = std::max(bx, p[0]); ay = std::min(ay, p[1]); by = std::max(by, p[1]);
            }
            i0 = cell(ax - x0); i1 = cell(bx - x0); j0 = cell(ay - y0); j1 = cell(by - y0);
        };
        for (int pass = 0; pass < 2; ++pass) {
            for (int64_t e = 0; e < c.Ne; ++e) {
                int i0, i1, j0, j1;
                range(e, i0, i1, j0, j1);
                for (int j = j0; j <= j1; ++j)
                    for (int i = i0; i <= i1; ++i) {
                        if (pass == 0) ++cnt[size_t(j) * nb + i + 1];
                        else items[ptr[size_t(j) * nb + i] + cnt[size_t(j) * nb + i]++] = int32_t(e);
                    }
            }
            if (pass == 0) {
                ptr.assign(cnt.size(), 0);
                for (size_t k = 1; k < cnt.size(); ++k) ptr[k] = ptr[k - 1] + cnt[k];
                items.resize(ptr.back());
                std::fill(cnt.begin(), cnt.end(), 0);
            }
        }
    }
    int cell(double d) const { return std::min(nb - 1, std::max(0, (int)(d * inv))); }
    // triangle holding (px, py): the candidate with the largest smallest barycentric coordinate; w = its coordinates
    int32_t locate(double px, double py, double w[3]) const
    {
        const int ci = cell(px - x0), cj = cell(py - y0);
        int32_t best = -1;
        double best_min = -1e300;
        for (int32_t k = ptr[size_t(cj) * nb + ci]; k < ptr[size_t(cj) * nb + ci + 1]; ++k) {
            const int32_t e = items[k];
            const double *a = xy(c.conn4[4 * e]), *b = xy(c.conn4[4 * e + 1]), *d = xy(c.conn4[4 * e + 2]);
            const double det = (b[0] - a[0]) * (d[1] - a[1]) - (d[0] - a[0]) * (b[1] - a[1]);
            const double l1 = ((px - a[0]) * (d[1] - a[1]) - (d[0] - a[0]) * (py - a[1])) / det;
            const double l2 = ((b[0] - a[0]) * (py - a[1]) - (px - a[0]) * (b[1] - a[1])) / det;
            const double l0 = 1.0 - l1 - l2, mn = std::min(l0, std::min(l1, l2));
            if (mn > best_min) { best_min = mn; best = e; w[0] = l0; w[1] = l1; w[2] = l2; }
        }
        if (best < 0 || best_min < -1e-6) return -1;
        for (int k = 0; k < 3; ++k) w[k] = std::fabs(w[k]) < 1e-12 ? 0.0 : std::max(w[k], 0.0);  // on an edge / at a node
        const double s = w[0] + w[1] + w[2];
        for (int k = 0; k < 3; ++k) w[k] /= s;
        return best;
    }
};

// ---- device: vector kernels ---------------------------------------------------------------------------------------------
// Block partial -> part[slot * n_part + block]; the LAST block to finish sums each slot's partials in index order into
// sc[slots[k]] (deterministic), so one launch yields the scalars.
template <int NS>
__device__ __forceinline__ void reduce_to_scalars(const double (&v)[NS], const int (&slots)[NS], double* part, int n_part,
                                                  double* sc, unsigned int* ticket)
{
    __shared__ double s_red[32];
#pragma unroll
    for (int k = 0; k < NS; ++k) {
        const double t = block_sum(v[k], s_red);
        if (threadIdx.x == 0) part[(size_t)k * n_part + blockIdx.x] = t;
    }
    if (last_block(ticket)) {
#pragma unroll
        for (int k = 0; k < NS; ++k) {
            double a = 0.0;
            for (int i = threadIdx.x; i < (int)gridDim.x; i += blockDim.x) a += __ldcg(part + (size_t)k * n_part + i);
            const double t = block_sum(a, s_red);
            if (threadIdx.x == 0) sc[slots[k]] = t;
        }
    }
}

// dinv = 1 / D on free nodes, 0 on damage-Dirichlet nodes (flags bit 2; flags may be null: no constraint on coarse levels)
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_dinv_kernel(int N, const R* D, const uint8_t* flags, R* dinv)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N) dinv[i] = (flags && (flags[i] & 4)) ? R(0) : R(1) / D[i];
}

// adjoint solve: nodes outside the caller's free set are fixed as well
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_mask_kernel(int N, const uint8_t* free_mask, R* dinv)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N && !free_mask[i]) dinv[i] = R(0);
}

// H_c[E] = sum over the children e of E of w_e H[e]
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_restrict_H_kernel(int NeC, const int32_t* ptr, const int32_t* idx, const R* w, const R* H, R* Hc)
{
    const int E = blockIdx.x * kTPB + threadIdx.x;
    if (E >= NeC) return;
    R s = R(0);
    for (int k = ptr[E]; k < ptr[E + 1]; ++k) s = rfma(w[k], H[idx[k]], s);
    Hc[E] = s;
}

// The operator's chunk kernel leaves A x of an interface node as per-chunk partials (pff_damage.cu); the vector kernel
// that consumes A x sums them itself, in slot order, instead of a separate interface kernel per application.
template <typename R>
struct IfaceSum {
    const R* part;
    const int32_t* rowptr;
    int N_int, N_sh, n_ovf;
    __device__ __forceinline__ R operator()(const R* t, int i) const
    {
        return i < N_int ? t[i] : iface_sum<R>(part, i - N_int, N_sh, n_ovf, rowptr);
    }
};

// x = w D^-1 b  (first smoothing step from a zero guess)
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_smooth0_kernel(int N, R omega, const R* dinv, const R* b, R* x)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N) x[i] = omega * dinv[i] * b[i];
}

// x += w D^-1 (b - t), t = A x
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_smooth_kernel(int N, R omega, const R* dinv, const R* b, const R* t, IfaceSum<R> ifs, R* x)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N) x[i] = rfma(omega * dinv[i], b[i] - ifs(t, i), x[i]);
}

// x += w D^-1 (b - t) and sc[RZN] = b . x: the last smoothing step of level 0 inside the solve, where b is the residual r
// and x becomes z
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_smooth_dot_kernel(int N, R omega, const R* dinv, const R* b, const R* t, IfaceSum<R> ifs, R* x,
                                                             double* part, int n_part, double* sc, unsigned int* ticket)
{
    double v[1] = {0.0};
    for (int i = blockIdx.x * kTPB + threadIdx.x; i < N; i += gridDim.x * kTPB) {
        const R bi = b[i], xi = rfma(omega * dinv[i], bi - ifs(t, i), x[i]);
        x[i] = xi;
        v[0] += double(bi) * double(xi);
    }
    const int slots[1] = {SC_RZN};
    reduce_to_scalars<1>(v, slots, part, n_part, sc, ticket);
}

// t <- b - t on the free nodes, 0 elsewhere (the residual the restriction gathers)
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_residual_kernel(int N, const R* dinv, const R* b, IfaceSum<R> ifs, R* t)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N) t[i] = dinv[i] != R(0) ? b[i] - ifs(t, i) : R(0);
}

// b_c[I] = sum_j P[j, I] res[j]
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_restrict_kernel(int NC, const int32_t* ptr, const int32_t* idx, const R* w, const R* res, R* bc)
{
    const int I = blockIdx.x * kTPB + threadIdx.x;
    if (I >= NC) return;
    R s = R(0);
    for (int k = ptr[I]; k < ptr[I + 1]; ++k) s = rfma(w[k], res[idx[k]], s);
    bc[I] = s;
}

// x[i] += (P x_c)[i] on the free fine nodes
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_prolong_kernel(int N, const int32_t* pidx, const R* pw, const R* dinv, const R* xc, R* x)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N || dinv[i] == R(0)) return;
    const R c = rfma(pw[3 * i + 2], xc[pidx[3 * i + 2]], rfma(pw[3 * i + 1], xc[pidx[3 * i + 1]], pw[3 * i] * xc[pidx[3 * i]]));
    x[i] += c;
}

// r = mask (b - t), lb = x (the lower bound d_n of the clamp);  sc[RR] = r.r, sc[BB] = b.b
// (the kernels with a reduction walk the vector with a grid stride: at most kRedBlocks block partials)
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_residual0_kernel(int N, int mask_b, int write_lb, const R* dinv, const R* b, const R* t, const R* x,
                                                            R* r, R* lb, double* part, int n_part, double* sc, unsigned int* ticket)
{
    double v[2] = {0.0, 0.0};
    for (int i = blockIdx.x * kTPB + threadIdx.x; i < N; i += gridDim.x * kTPB) {
        const bool fr = dinv[i] != R(0);
        const R ri = fr ? b[i] - t[i] : R(0);
        r[i] = ri;
        if (write_lb) lb[i] = x[i];
        v[0] += double(ri) * double(ri);
        v[1] += (fr || !mask_b) ? double(b[i]) * double(b[i]) : 0.0;  // ||b|| over all nodes, as the oracle's stopping rule
                                                                        // (R10); adjoint: over the free set (g_F is the rhs)
    }
    const int slots[2] = {SC_RR, SC_BB};
    reduce_to_scalars<2>(v, slots, part, n_part, sc, ticket);
}

// sc[slot] = a . b
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_dot_kernel(int N, const R* a, const R* b, int slot, double* part, int n_part, double* sc,
                                                      unsigned int* ticket)
{
    double v[1] = {0.0};
    for (int i = blockIdx.x * kTPB + threadIdx.x; i < N; i += gridDim.x * kTPB) v[0] += double(a[i]) * double(b[i]);
    const int slots[1] = {slot};
    reduce_to_scalars<1>(v, slots, part, n_part, sc, ticket);
}

// sc[PQ] = p . q, with q of the interface nodes completed (summed and stored) on the way
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_pq_kernel(int N, const R* p, R* q, IfaceSum<R> ifs, double* part, int n_part, double* sc,
                                                     unsigned int* ticket)
{
    double v[1] = {0.0};
    for (int i = blockIdx.x * kTPB + threadIdx.x; i < N; i += gridDim.x * kTPB) {
        R qi = q[i];
        if (i >= ifs.N_int) { qi = ifs(q, i); q[i] = qi; }
        v[0] += double(p[i]) * double(qi);
    }
    const int slots[1] = {SC_PQ};
    reduce_to_scalars<1>(v, slots, part, n_part, sc, ticket);
}

// alpha = (r.z)_new / p.q;  x += alpha p;  r -= alpha q on the free nodes;  sc[RR] = r.r; afterwards (r.z)_old <- (r.z)_new
// (no block of this launch reads (r.z)_old; the direction kernel that does has finished)
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_update_kernel(int N, const R* dinv, const R* p, const R* q, R* x, R* r, double* part, int n_part,
                                                         double* sc, unsigned int* ticket)
{
    const double rzn = sc[SC_RZN];
    const R alpha = R(rzn / sc[SC_PQ]);
    double v[1] = {0.0};
    for (int i = blockIdx.x * kTPB + threadIdx.x; i < N; i += gridDim.x * kTPB) {
        x[i] = rfma(alpha, p[i], x[i]);
        const R ri = dinv[i] != R(0) ? rfma(-alpha, q[i], r[i]) : R(0);
        r[i] = ri;
        v[0] += double(ri) * double(ri);
    }
    const int slots[1] = {SC_RR};
    reduce_to_scalars<1>(v, slots, part, n_part, sc, ticket);
    if (blockIdx.x == 0 && threadIdx.x == 0) sc[SC_RZ] = rzn;
}

// p = z + beta p, beta = (r.z)_new / (r.z)_old.  The first iteration runs the same kernel with p = 0 and (r.z)_old = 1.
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_direction_kernel(int N, const R* z, R* p, const double* sc)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N) return;
    const R beta = R(sc[SC_RZN] / sc[SC_RZ]);
    p[i] = rfma(beta, p[i], z[i]);
}

__global__ void mg_init_rz_kernel(double* sc) { sc[SC_RZ] = 1.0; }
// pff_run_steps: counters of this solve into the device-resident tally (as the CG kernels do for the Jacobi solver)
__global__ void mg_tally_kernel(RunTally* t, int iters, int noconv) { t->iters += iters; t->solves += 1; t->noconv += noconv; }

// ---- AT1 (L181): primal-dual active set around the multigrid-preconditioned linear solve ---------------------------------
// One outer step: with r = b - A x (t = A x, all nodes), a non-fixed node is ACTIVE when r / D + (x - lb) < 0 (the multiplier
// estimate -r outweighs the distance to the bound, scaled by the diagonal): it is put on its bound and masked (dinv = 0)
// for the linear solve that follows; the others form the inactive set (dinv = 1 / D).  first = 1 also stores lb = x.
// sc[CHG] = nodes that changed sets, sc[R0] = |r|^2 over the non-fixed nodes, sc[BB] = |b|^2.
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_pdas_sets_kernel(int N, int first, const R* dfull, const R* b, const R* t, R* x, R* lb, R* dinv,
                                                            double* part, int n_part, double* sc, unsigned int* ticket)
{
    double v[3] = {0.0, 0.0, 0.0};
    for (int i = blockIdx.x * kTPB + threadIdx.x; i < N; i += gridDim.x * kTPB) {
        const R xi = x[i], ri = b[i] - t[i], di = dfull[i];
        if (first) lb[i] = xi;
        const R lo = first ? xi : lb[i];
        const bool fixed = di == R(0);
        const bool was_inactive = first ? !fixed : dinv[i] != R(0);
        const bool act = !fixed && (ri * di + (xi - lo) < R(0));
        if (act) x[i] = lo;
        dinv[i] = (!fixed && !act) ? di : R(0);
        v[0] += (!fixed && was_inactive == act) ? 1.0 : 0.0;
        v[1] += fixed ? 0.0 : double(ri) * double(ri);
        v[2] += double(b[i]) * double(b[i]);
    }
    const int slots[3] = {SC_CHG, SC_R0, SC_BB};
    reduce_to_scalars<3>(v, slots, part, n_part, sc, ticket);
}

// d <- min(1, max(d_n, d)) (L179)
template <typename R>
__global__ void __launch_bounds__(kTPB) mg_clamp_kernel(int N, const R* lb, R* x)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N) x[i] = rmin(R(1), rmax(lb[i], x[i]));
}

// ---- host: hierarchy set-up ---------------------------------------------------------------------------------------------
template <typename T>
static pff_status to_device(T** dst, const std::vector<T>& src, cudaStream_t s)
{
    MG_CUDA(cudaMalloc((void**)dst, std::max<size_t>(src.size(), 1) * sizeof(T)));
    if (!src.empty()) MG_CUDA(cudaMemcpyAsync(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice, s));
    return PFF_OK;
}

template <typename R>
static pff_status upload_reals(void** dst, const std::vector<double>& src, cudaStream_t s)
{
    std::vector<R> v(src.begin(), src.end());
    R* p = nullptr;
    pff_status st = to_device(&p, v, s);
    if (st == PFF_OK) st = cuda_check(cudaStreamSynchronize(s), "multigrid: upload");  // v goes out of scope
    *dst = p;
    return st;
}

template <typename R>
static pff_status build_transfer(const pff_mesh* mf, const pff_mesh* mc, MgTransfer& tr, int level)
{
    const HostMesh &f = mf->hm, &c = mc->hm;
    const Locator loc(c);
    cudaStream_t s = mf->stream;
    // interpolation: every fine node in a coarse triangle
    std::vector<int32_t> p_idx(size_t(3) * f.N);
    std::vector<double> p_w(size_t(3) * f.N);
    std::vector<int32_t> r_cnt(c.N + 1, 0);
    // (point location is independent per node / element: spread over the host cores; the tables do not depend on the
    // thread count)
    const unsigned nt = std::max(1u, std::min(16u, std::thread::hardware_concurrency()));
    auto parallel_for = [&](int64_t n, const std::function<void(int64_t)>& body) {
        std::vector<std::thread> pool;
        for (unsigned t = 0; t < nt; ++t)
            pool.emplace_back([&, t]() { for (int64_t i = t; i < n; i += nt) body(i); });
        for (auto& th : pool) th.join();
    };
    std::atomic<int> outside{0};
    parallel_for(f.N, [&](int64_t i) {
        const double* p = &f.xy_user[2 * size_t(f.node_old_of_new[i])];
        double w[3];
        const int32_t e = loc.locate(p[0], p[1], w);
        if (e < 0) { outside = 1; return; }
        for (int k = 0; k < 3; ++k) { p_idx[3 * i + k] = c.conn4[4 * size_t(e) + k]; p_w[3 * i + k] = w[k]; }
    });
    if (outside) {
        set_error("pff_mg_attach: a node of level " + std::to_string(level) + " lies in no triangle of level " +
                  std::to_string(level + 1) + " (the meshes must cover the same domain)");
        return PFF_EMESH;
    }
    for (int64_t i = 0; i < f.N; ++i)
        for (int k = 0; k < 3; ++k)
            if (p_w[3 * i + k] != 0.0) ++r_cnt[p_idx[3 * i + k] + 1];
    // its transpose, rows = coarse nodes, entries ascending in the fine index (fixed summation order)
    std::vector<int32_t> r_ptr(c.N + 1, 0);
    for (int64_t I = 0; I < c.N; ++I) r_ptr[I + 1] = r_ptr[I] + r_cnt[I + 1];
    std::vector<int32_t> r_idx(r_ptr[c.N]), fill(c.N, 0);
    std::vector<double> r_w(r_ptr[c.N]);
    for (int64_t i = 0; i < f.N; ++i)
        for (int k = 0; k < 3; ++k)
            if (p_w[3 * i + k] != 0.0) {
                const int32_t I = p_idx[3 * i + k], at = r_ptr[I] + fill[I]++;
                r_idx[at] = int32_t(i); r_w[at] = p_w[3 * i + k];
            }
    // parent element of every fine element (centroid), child weights = area fractions
    std::vector<int32_t> parent(f.Ne), c_ptr(c.Ne + 1, 0);
    std::vector<double> asum(c.Ne, 0.0);
    parallel_for(f.Ne, [&](int64_t e) {
        double cx = 0.0, cy = 0.0;
        for (int k = 0; k < 3; ++k) {
            const double* p = &f.xy_user[2 * size_t(f.node_old_of_new[f.conn4[4 * e + k]])];
            cx += p[0] / 3.0; cy += p[1] / 3.0;
        }
        double w[3];
        const int32_t E = loc.locate(cx, cy, w);
        if (E < 0) outside = 1;
        parent[e] = E;
    });
    if (outside) { set_error("pff_mg_attach: an element of level " + std::to_string(level) + " lies in no triangle of the next level"); return PFF_EMESH; }
    for (int64_t e = 0; e < f.Ne; ++e) { ++c_ptr[parent[e] + 1]; asum[parent[e]] += f.area[e]; }
    for (int64_t E = 0; E < c.Ne; ++E) c_ptr[E + 1] += c_ptr[E];
    std::vector<int32_t> c_idx(f.Ne), cfill(c.Ne, 0);
    std::vector<double> c_w(f.Ne);
    for (int64_t e = 0; e < f.Ne; ++e) {
        const int32_t E = parent[e], at = c_ptr[E] + cfill[E]++;
        c_idx[at] = int32_t(e); c_w[at] = f.area[e] / asum[E];
    }
    pff_status st;
    if ((st = to_device(&tr.p_idx, p_idx, s)) != PFF_OK) return st;
    if ((st = to_device(&tr.r_ptr, r_ptr, s)) != PFF_OK) return st;
    if ((st = to_device(&tr.r_idx, r_idx, s)) != PFF_OK) return st;
    if ((st = to_device(&tr.c_ptr, c_ptr, s)) != PFF_OK) return st;
    if ((st = to_device(&tr.c_idx, c_idx, s)) != PFF_OK) return st;
    if ((st = upload_reals<R>(&tr.p_w, p_w, s)) != PFF_OK) return st;
    if ((st = upload_reals<R>(&tr.r_w, r_w, s)) != PFF_OK) return st;
    if ((st = upload_reals<R>(&tr.c_w, c_w, s)) != PFF_OK) return st;
    return cuda_check(cudaStreamSynchronize(s), "multigrid: transfer upload");
}

void mg_free(pff_mesh* m)
{
    MgData* g = static_cast<MgData*>(m->mg);
    if (!g) return;
    for (MgLevel& L : g->lv) {
        void* ps[] = {L.b, L.x, L.t, L.dinv, L.zero, L.H, L.tr.p_idx, L.tr.p_w, L.tr.r_ptr, L.tr.r_idx, L.tr.r_w, L.tr.c_ptr, L.tr.c_idx, L.tr.c_w};
        for (void* p : ps) if (p) cudaFree(p);
    }
    void* ps[] = {g->r, g->p, g->q, g->lb, g->dfull, g->part, g->sc, g->ticket};
    for (void* p : ps) if (p) cudaFree(p);
    if (g->h_sc) cudaFreeHost(g->h_sc);
    for (auto& gr : g->graphs) if (gr.exec) cudaGraphExecDestroy(gr.exec);
    if (g->cap_stream) cudaStreamDestroy(g->cap_stream);
    delete g;
    m->mg = nullptr;
}

template <typename R>
static pff_status mg_attach_t(pff_mesh* m, int n_coarse, pff_mesh* const* coarse)
{
    mg_free(m);
    MgData* g = new MgData;
    m->mg = g;
    g->lv.resize(size_t(n_coarse) + 1);
    g->lv[0].m = m;
    for (int l = 1; l <= n_coarse; ++l) g->lv[l].m = coarse[l - 1];
    cudaStream_t s = m->stream;
    int64_t max_blocks = 1;
    for (size_t l = 0; l < g->lv.size(); ++l) {
        MgLevel& L = g->lv[l];
        const size_t nb = size_t(L.m->hm.N) * sizeof(R);
        max_blocks = std::max<int64_t>(max_blocks, (L.m->hm.N + kTPB - 1) / kTPB);
        for (void** p : {&L.b, &L.x, &L.t, &L.dinv}) MG_CUDA(cudaMalloc(p, nb));
        if (l > 0) {  // the coarse levels' own state: d = 0, H = restricted history, everything else a zero vector
            MG_CUDA(cudaMalloc(&L.zero, nb));
            MG_CUDA(cudaMemsetAsync(L.zero, 0, nb, s));
            MG_CUDA(cudaMalloc(&L.H, size_t(L.m->hm.Ne) * sizeof(R)));
            L.st = pff_state{L.zero, L.zero, L.zero, L.zero, L.zero, L.zero, L.zero, L.H, L.zero, L.zero};
        }
        if (l + 1 < g->lv.size()) {
            pff_status st = build_transfer<R>(L.m, g->lv[l + 1].m, L.tr, (int)l);
            if (st != PFF_OK) return st;
        }
    }
    const size_t nb0 = size_t(m->hm.N) * sizeof(R);
    for (void** p : {&g->r, &g->p, &g->q, &g->lb, &g->dfull}) MG_CUDA(cudaMalloc(p, nb0));
    g->n_part = (int)max_blocks;
    MG_CUDA(cudaMalloc((void**)&g->part, sizeof(double) * 4 * g->n_part));
    MG_CUDA(cudaMalloc((void**)&g->sc, sizeof(double) * SC_N));
    MG_CUDA(cudaMalloc((void**)&g->ticket, sizeof(unsigned int)));
    MG_CUDA(cudaMemsetAsync(g->ticket, 0, sizeof(unsigned int), s));
    MG_CUDA(cudaMallocHost((void**)&g->h_sc, sizeof(double) * SC_N));
    return cuda_check(cudaStreamSynchronize(s), "pff_mg_attach");
}

pff_status mg_attach(pff_mesh* m, int n_coarse, pff_mesh* const* coarse)
{
    for (int l = 0; l < n_coarse; ++l) {
        const pff_mesh* c = coarse[l];
        if (!c || c == m || c->opt.precision != m->opt.precision || c->device != m->device || c->stream != m->stream ||
            c->opt.scatter != PFF_SCATTER_GATHER) {
            set_error("pff_mg_attach: every coarse mesh must be a distinct gather mesh of the same precision, device and stream");
            return PFF_EINVAL;
        }
    }
    pff_status st = m->opt.precision == PFF_F32 ? mg_attach_t<float>(m, n_coarse, coarse) : mg_attach_t<double>(m, n_coarse, coarse);
    if (st != PFF_OK) mg_free(m);
    return st;
}

// ---- host: V-cycle and the outer PCG --------------------------------------------------------------------------------------
static inline unsigned nblk(int64_t n) { return (unsigned)std::max<int64_t>(1, (n + kTPB - 1) / kTPB); }

// Operators of this solve on every level: restricted history, coefficient form (first operator application refreshes it),
// Jacobi diagonal.  Level 0 uses the caller's state.
template <typename R>
static pff_status mg_setup_operators(MgData* g, const pff_state* s0)
{
    pff_mesh* m0 = g->lv[0].m;
    cudaStream_t s = m0->stream;
    g->lv[0].st = *s0;
    for (size_t l = 0; l < g->lv.size(); ++l) {
        MgLevel& L = g->lv[l];
        const int N = (int)L.m->hm.N;
        if (l > 0) {
            const MgLevel& F = g->lv[l - 1];
            mg_restrict_H_kernel<R><<<nblk(L.m->hm.Ne), kTPB, 0, s>>>((int)L.m->hm.Ne, F.tr.c_ptr, F.tr.c_idx, (const R*)F.tr.c_w,
                                                                      (const R*)F.st.H, (R*)L.H);
            ++m0->n_launches;
        }
        // b (unused on the coarse levels: scratch x), D -> t
        pff_status st = damage_rhs_diag(L.m, &L.st, l == 0 ? L.b : L.x, L.t);
        if (st != PFF_OK) return st;
        mg_dinv_kernel<R><<<nblk(N), kTPB, 0, s>>>(N, (const R*)L.t, l == 0 ? L.m->d_flags : nullptr, (R*)L.dinv);
        ++m0->n_launches;
        // coefficient form of the operator (one refresh per solve; every apply below reuses it)
        if ((st = damage_refresh_coef(L.m, &L.st)) != PFF_OK) return st;
    }
    return cuda_check(cudaGetLastError(), "multigrid: operator set-up");
}

// x_l = V(b_l) on level l (b_l, x_l, t_l are the level's vectors)
template <typename R>
static IfaceSum<R> iface_of(const pff_mesh* m)
{
    return IfaceSum<R>{(const R*)m->d_halo_part, m->d_sh_rowptr, (int)m->hm.N_int, (int)m->hm.N_sh, m->hm.n_ovf};
}

constexpr int kRedBlocks = 592;  // 4 per SM of a B200
static inline unsigned nred(int64_t n) { return (unsigned)std::min<int64_t>(kRedBlocks, std::max<int64_t>(1, (n + kTPB - 1) / kTPB)); }

template <typename R>
static pff_status mg_vcycle(MgData* g, size_t l, bool dot_rz = false)
{
    MgLevel& L = g->lv[l];
    pff_mesh* m0 = g->lv[0].m;
    cudaStream_t s = m0->stream;
    const int N = (int)L.m->hm.N;
    const R om = R(g->omega);
    pff_status st;
    mg_smooth0_kernel<R><<<nblk(N), kTPB, 0, s>>>(N, om, (const R*)L.dinv, (const R*)L.b, (R*)L.x);
    ++m0->n_launches;
    if (l + 1 == g->lv.size()) {  // coarsest level: a fixed number of damped-Jacobi sweeps (a fixed symmetric operator)
        for (int k = 1; k < g->coarse_sweeps; ++k) {
            if ((st = damage_matvec(L.m, &L.st, L.x, L.t, false, true)) != PFF_OK) return st;
            mg_smooth_kernel<R><<<nblk(N), kTPB, 0, s>>>(N, om, (const R*)L.dinv, (const R*)L.b, (const R*)L.t, iface_of<R>(L.m), (R*)L.x);
            ++m0->n_launches;
        }
        return PFF_OK;
    }
    MgLevel& Cl = g->lv[l + 1];
    const int NC = (int)Cl.m->hm.N;
    if ((st = damage_matvec(L.m, &L.st, L.x, L.t, false, true)) != PFF_OK) return st;
    mg_residual_kernel<R><<<nblk(N), kTPB, 0, s>>>(N, (const R*)L.dinv, (const R*)L.b, iface_of<R>(L.m), (R*)L.t);
    mg_restrict_kernel<R><<<nblk(NC), kTPB, 0, s>>>(NC, L.tr.r_ptr, L.tr.r_idx, (const R*)L.tr.r_w, (const R*)L.t, (R*)Cl.b);
    m0->n_launches += 2;
    if ((st = mg_vcycle<R>(g, l + 1)) != PFF_OK) return st;
    mg_prolong_kernel<R><<<nblk(N), kTPB, 0, s>>>(N, L.tr.p_idx, (const R*)L.tr.p_w, (const R*)L.dinv, (const R*)Cl.x, (R*)L.x);
    ++m0->n_launches;
    if ((st = damage_matvec(L.m, &L.st, L.x, L.t, false, true)) != PFF_OK) return st;
    if (dot_rz)
        mg_smooth_dot_kernel<R><<<nred(N), kTPB, 0, s>>>(N, om, (const R*)L.dinv, (const R*)L.b, (const R*)L.t, iface_of<R>(L.m), (R*)L.x,
                                                         g->part, g->n_part, g->sc, g->ticket);
    else
        mg_smooth_kernel<R><<<nblk(N), kTPB, 0, s>>>(N, om, (const R*)L.dinv, (const R*)L.b, (const R*)L.t, iface_of<R>(L.m), (R*)L.x);
    ++m0->n_launches;
    return PFF_OK;
}

// z = V(r) with the operator of state->H (test hook: the preconditioner alone)
template <typename R>
static pff_status mg_apply_t(pff_mesh* m, const pff_state* s0, const void* r, void* z)
{
    MgData* g = static_cast<MgData*>(m->mg);
    pff_status st = mg_setup_operators<R>(g, s0);
    if (st != PFF_OK) return st;
    const size_t nb = size_t(m->hm.N) * sizeof(R);
    MG_CUDA(cudaMemcpyAsync(g->lv[0].b, r, nb, cudaMemcpyDeviceToDevice, m->stream));
    if ((st = mg_vcycle<R>(g, 0)) != PFF_OK) return st;
    MG_CUDA(cudaMemcpyAsync(z, g->lv[0].x, nb, cudaMemcpyDeviceToDevice, m->stream));
    return cuda_check(cudaStreamSynchronize(m->stream), "pff_mg_apply");
}

template <typename R>
static pff_status mg_solve_t(pff_mesh* m, const pff_state* s0, double rel_tol, int max_iter, int* iters, double* relres,
                             const MgAdjoint* adj = nullptr)
{
    MgData* g = static_cast<MgData*>(m->mg);
    MgLevel& F = g->lv[0];
    cudaStream_t s = m->stream;
    const int N = (int)m->hm.N;
    const unsigned nb = nblk(N);
    R* x = adj ? (R*)adj->lambda : (R*)s0->d;
    pff_status st = mg_setup_operators<R>(g, s0);  // F.b = b(H)
    if (st != PFF_OK) return st;
    void* const b_own = F.b;
    if (adj) {  // A_FF lambda_F = g_F from lambda = 0 (the caller zeroed it): rhs g, free set = the caller's minus the fixed nodes
        if (adj->free_mask) { mg_mask_kernel<R><<<nb, kTPB, 0, s>>>(N, adj->free_mask, (R*)F.dinv); ++m->n_launches; }
        F.b = const_cast<void*>(adj->g);
    }
    struct Restore { MgLevel& F; void* b; ~Restore() { F.b = b; } } restore{F, b_own};
    auto read_scalars = [&]() -> pff_status {
        MG_CUDA(cudaMemcpyAsync(g->h_sc, g->sc, sizeof(double) * SC_N, cudaMemcpyDeviceToHost, s));
        return cuda_check(cudaStreamSynchronize(s), "pff_damage_solve_mg: sync");
    };
    const bool pdas = !adj && m->mat.model == PFF_AT1;  // bound-constrained problem: active-set outer loop (below)
    double nrm = 0.0, lim = 0.0, rr = 0.0;
    if (!pdas) {
        // r0 = mask (b - A d_n), lb = d_n; stopping rule of pff_damage_solve (R10)
        if ((st = damage_matvec(m, s0, x, F.t, false)) != PFF_OK) return st;
        mg_residual0_kernel<R><<<nred(N), kTPB, 0, s>>>(N, adj ? 1 : 0, 1, (const R*)F.dinv, (const R*)F.b, (const R*)F.t, x, (R*)g->r, (R*)g->lb,
                                                        g->part, g->n_part, g->sc, g->ticket);
        ++m->n_launches;
        if ((st = read_scalars()) != PFF_OK) return st;
        nrm = std::sqrt(std::max(g->h_sc[SC_BB], g->h_sc[SC_RR]));
        lim = rel_tol * nrm;
        rr = g->h_sc[SC_RR];
    } else {
        MG_CUDA(cudaMemcpyAsync(g->dfull, F.dinv, size_t(N) * sizeof(R), cudaMemcpyDeviceToDevice, s));
    }
    int it = 0;
    void* b_keep = F.b;  // the V-cycle's right-hand side on level 0 is the residual: swap the buffer in, b stays in b_keep
    pff_status result = PFF_OK;
    MG_CUDA(cudaMemsetAsync(g->p, 0, size_t(N) * sizeof(R), s));
    mg_init_rz_kernel<<<1, 1, 0, s>>>(g->sc);
    // one outer iteration on the levels' (common) stream
    auto iteration = [&]() -> pff_status {
        cudaStream_t cs = m->stream;
        F.b = g->r;
        pff_status e = mg_vcycle<R>(g, 0, g->lv.size() > 1);  // z = V(r) -> F.x, (r.z) with the last smoothing step
        F.b = b_keep;
        if (e != PFF_OK) return e;
        if (g->lv.size() == 1) {
            mg_dot_kernel<R><<<nred(N), kTPB, 0, cs>>>(N, (const R*)g->r, (const R*)F.x, SC_RZN, g->part, g->n_part, g->sc, g->ticket);
            ++m->n_launches;
        }
        mg_direction_kernel<R><<<nb, kTPB, 0, cs>>>(N, (const R*)F.x, (R*)g->p, g->sc);
        if ((e = damage_matvec(m, s0, g->p, g->q, false, true)) != PFF_OK) return e;  // q = A p (interface sums in the next kernel)
        mg_pq_kernel<R><<<nred(N), kTPB, 0, cs>>>(N, (const R*)g->p, (R*)g->q, iface_of<R>(m), g->part, g->n_part, g->sc, g->ticket);
        mg_update_kernel<R><<<nred(N), kTPB, 0, cs>>>(N, (const R*)F.dinv, (const R*)g->p, (const R*)g->q, x, (R*)g->r, g->part, g->n_part,
                                                      g->sc, g->ticket);
        m->n_launches += 3;
        return cuda_check(cudaGetLastError(), "pff_damage_solve_mg: iteration");
    };
    // captured once per (x, omega, sweeps): recorded on a stream of the library's own (the caller's may be the legacy
    // default stream, which cannot capture); every level launches on the recording stream while it is recorded
    const bool want_graph = m->graph_mode != 0 && !g->graph_refused && !m->prof_on;
    MgData::Graph* gr = nullptr;
    if (want_graph) {
        for (auto& c : g->graphs)
            if (c.exec && c.x == (const void*)x && c.b == (const void*)b_keep && c.omega == g->omega && c.sweeps == g->coarse_sweeps) gr = &c;
        if (!gr) {  // record into the least recently used entry
            gr = g->graphs[0].used <= g->graphs[1].used ? &g->graphs[0] : &g->graphs[1];
            if (gr->exec) { cudaGraphExecDestroy(gr->exec); gr->exec = nullptr; }
            cudaError_t ce = g->cap_stream ? cudaSuccess : cudaStreamCreateWithFlags(&g->cap_stream, cudaStreamNonBlocking);
            cudaGraph_t graph = nullptr;
            pff_status cst = PFF_OK;
            if (ce == cudaSuccess) ce = cudaStreamBeginCapture(g->cap_stream, cudaStreamCaptureModeThreadLocal);
            if (ce == cudaSuccess) {
                std::vector<int64_t> before;
                for (MgLevel& L : g->lv) { before.push_back(L.m->n_launches); L.m->stream = g->cap_stream; }
                cst = iteration();
                gr->launches = 0;
                for (size_t l = 0; l < g->lv.size(); ++l) {
                    MgLevel& L = g->lv[l];
                    L.m->stream = s;
                    gr->launches += int(L.m->n_launches - before[l]);
                    L.m->n_launches = before[l];  // recorded, not launched
                }
                ce = cudaStreamEndCapture(g->cap_stream, &graph);
            }
            if (ce == cudaSuccess && cst == PFF_OK && graph) ce = cudaGraphInstantiate(&gr->exec, graph, 0);
            if (graph) cudaGraphDestroy(graph);
            if (ce != cudaSuccess || cst != PFF_OK || !gr->exec) { cudaGetLastError(); gr->exec = nullptr; gr = nullptr; g->graph_refused = true; }
            else { gr->x = x; gr->b = b_keep; gr->omega = g->omega; gr->sweeps = g->coarse_sweeps; }
        }
        if (gr) gr->used = ++g->graph_clock;
    }
    // PCG on the masked system from the current x, r (p = 0, (r.z)_old = 1 set by the caller) until |r| <= target
    auto pcg = [&](double target) -> pff_status {
        while (std::sqrt(rr) > target) {
            if (it >= max_iter) { set_error("pff_damage_solve_mg: max_iter reached"); result = PFF_ENOCONV; return PFF_OK; }
            if (gr) {
                MG_CUDA(cudaGraphLaunch(gr->exec, s));
                m->n_launches += gr->launches;
            } else {
                pff_status e = iteration();
                if (e != PFF_OK) return e;
            }
            ++it;
            pff_status e = read_scalars();
            if (e != PFF_OK) return e;
            rr = g->h_sc[SC_RR];
            if (!(g->h_sc[SC_PQ] > 0.0) || !std::isfinite(rr)) {
                set_error("pff_damage_solve_mg: breakdown (p.Ap <= 0)"); result = PFF_ENOCONV; return PFF_OK;
            }
        }
        return PFF_OK;
    };
    int outer = 0;
    if (!pdas) {
        if ((st = pcg(lim)) != PFF_OK) return st;
    } else {
        // AT1 (L181): min 1/2 d'Ad - b'd, d >= d_n by a primal-dual active set method: the active nodes sit on their bound,
        // the inactive ones solve their linear system (PCG with the cycle masked to them, the loop above), the sets are
        // re-derived from the multiplier estimate, until they stop changing and the inactive residual meets the tolerance.
        // While the sets still move the linear solves are very inexact (residual x 0.3 per outer step: their only job is to
        // move the sets; measured at 10^6 nodes: 48 cycles in all against 116 with x 0.01 and 165 with x 0.001).
        for (;; ++outer) {
            if ((st = damage_matvec(m, s0, x, F.t, false)) != PFF_OK) return st;
            mg_pdas_sets_kernel<R><<<nred(N), kTPB, 0, s>>>(N, outer == 0, (const R*)g->dfull, (const R*)F.b, (const R*)F.t, x, (R*)g->lb,
                                                           (R*)F.dinv, g->part, g->n_part, g->sc, g->ticket);
            ++m->n_launches;
            if ((st = read_scalars()) != PFF_OK) return st;
            const double changed = g->h_sc[SC_CHG];
            if (outer == 0) { nrm = std::max(std::sqrt(std::max(g->h_sc[SC_BB], g->h_sc[SC_R0])), 1e-300); lim = rel_tol * nrm; }
            // residual of the inactive set after the projection
            if ((st = damage_matvec(m, s0, x, F.t, false)) != PFF_OK) return st;
            mg_residual0_kernel<R><<<nred(N), kTPB, 0, s>>>(N, 0, 0, (const R*)F.dinv, (const R*)F.b, (const R*)F.t, x, (R*)g->r, (R*)g->lb,
                                                            g->part, g->n_part, g->sc, g->ticket);
            MG_CUDA(cudaMemsetAsync(g->p, 0, size_t(N) * sizeof(R), s));
            mg_init_rz_kernel<<<1, 1, 0, s>>>(g->sc);
            m->n_launches += 2;
            if ((st = read_scalars()) != PFF_OK) return st;
            rr = g->h_sc[SC_RR];
            if (outer > 0 && changed == 0.0 && std::sqrt(rr) <= lim) break;  // KKT: sets stable, inactive residual converged
            if (outer >= 100 || it >= max_iter || result != PFF_OK) {
                if (result == PFF_OK) set_error("pff_damage_solve_mg: the active set did not settle (max_iter / 100 outer steps)");
                result = PFF_ENOCONV; break;
            }
            if ((st = pcg(changed == 0.0 ? lim : std::max(lim, 0.3 * std::sqrt(rr)))) != PFF_OK) return st;
        }
        m->last_restarts = outer; m->last_truncs = 0;
    }
    if (!adj) {
        mg_clamp_kernel<R><<<nb, kTPB, 0, s>>>(N, (const R*)g->lb, x);
        ++m->n_launches;
    }
    if ((st = cuda_check(cudaStreamSynchronize(s), "pff_damage_solve_mg: sync")) != PFF_OK) return st;
    g->last_cycles = it;
    if (!adj && m->defer && m->d_tally) {  // inside pff_run_steps: tallied on the device, reported once at the end of the run
        mg_tally_kernel<<<1, 1, 0, s>>>(m->d_tally, it, result == PFF_ENOCONV ? 1 : 0);
        ++m->n_launches;
        return PFF_OK;
    }
    if (iters) *iters = it;
    if (relres) *relres = nrm > 0.0 ? std::sqrt(rr) / nrm : 0.0;
    return result;
}

static pff_status mg_check(pff_mesh* m, const char* who)
{
    if (!m->mg) { set_error(std::string(who) + ": no hierarchy attached (pff_mg_attach)"); return PFF_EINVAL; }
    return PFF_OK;
}

pff_status mg_apply(pff_mesh* m, const pff_state* s, const void* r, void* z)
{
    pff_status st = mg_check(m, "pff_mg_apply");
    if (st != PFF_OK) return st;
    return m->opt.precision == PFF_F32 ? mg_apply_t<float>(m, s, r, z) : mg_apply_t<double>(m, s, r, z);
}

pff_status mg_solve(pff_mesh* m, pff_state* s, double rel_tol, int max_iter, int* iters, double* relres)
{
    pff_status st = mg_check(m, "pff_damage_solve_mg");
    if (st != PFF_OK) return st;
    return m->opt.precision == PFF_F32 ? mg_solve_t<float>(m, s, rel_tol, max_iter, iters, relres)
                                       : mg_solve_t<double>(m, s, rel_tol, max_iter, iters, relres);
}

// pff_damage_adjoint with the multigrid solver (a linear solve on a given free set: AT1 and AT2 alike)
pff_status mg_adjoint(pff_mesh* m, const pff_state* s, const void* gvec, const uint8_t* free_mask, void* lambda, double rel_tol,
                      int max_iter, int* iters, double* relres)
{
    if (!m->mg) { set_error("pff_damage_adjoint: no hierarchy attached"); return PFF_EINVAL; }
    const MgAdjoint adj{gvec, free_mask, lambda};
    return m->opt.precision == PFF_F32 ? mg_solve_t<float>(m, s, rel_tol, max_iter, iters, relres, &adj)
                                       : mg_solve_t<double>(m, s, rel_tol, max_iter, iters, relres, &adj);
}

pff_status mg_set_params(pff_mesh* m, double omega, int coarse_sweeps)
{
    if (!m->mg) { set_error("pff_mg_set_params: no hierarchy attached"); return PFF_EINVAL; }
    if (!(omega > 0.0) || !(omega < 1.0) || coarse_sweeps < 1) { set_error("pff_mg_set_params: need 0 < omega < 1, coarse_sweeps >= 1"); return PFF_EINVAL; }
    MgData* g = static_cast<MgData*>(m->mg);
    g->omega = omega; g->coarse_sweeps = coarse_sweeps;
    return PFF_OK;
}

}  // namespace pff
