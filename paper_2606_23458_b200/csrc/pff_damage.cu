// Damage sub-problem (Eq. 6-8): matrix-free operator with consistent mass,
// Jacobi-preconditioned CG (AT2, then clamp, L179) and projected CG with an active set (AT1, L181).
//
// Kernels per CG iteration (all early-exit when the device-resident control block says done):
//   dmg_matvec_chunk   one CTA per chunk: forms the new search direction p = z + beta p for the nodes it
//                      touches (z = D^-1 r on the free set), stages it in shared memory, element pass
//                      q^e = (c_e M^e + kappa K^e) p^e into slots, ordered node gather, q and the p.q partial.
//   dmg_matvec_shared  interface nodes; the last CTA reduces the partials in a fixed order and sets
//                      alpha = rho / p.q (and the AT1 step bound) in the control block.
//   dmg_vector         x += alpha p, r -= alpha q, next free set, r.z and ||r|| partials; the last CTA
//                      decides continue / restart / converged and sets beta, rho.
// alpha, beta, rho, norms never leave the device; the host polls the control block every few iterations.
#include <algorithm>
#include <cstring>

#include "pff_device.cuh"
#include "pff_mesh.h"

struct DamageCtrl {
    double rho, pq, alpha, beta, amax, nb, tol, relres;
    int iters, max_iter, done, status, sel, first, truncated, restarts;
};

namespace pff {

constexpr int kPartStride = 4;  // partial-sum channels per block

template <typename R>
struct DmgArgs {
    const ChunkMeta* meta;
    const ushort4* lconn;
    const void *ga, *gb;
    const R* area;
    const int32_t* halo_ids;
    const uint16_t* ell;
    const uint8_t* flags;
    R* halo_part;  // [3][n_slots]
    int64_t n_slots;
    int EC, max_nloc, N, N_int, N_sh, C, nbs;
    const int32_t *sh_rowptr, *sh_slots;
    const R* H;
    R* x;  // = state.d
    R *lb, *r, *p, *q, *dinv;
    uint8_t* mask;  // [2][N]
    const R* p_in;  // plain mat-vec / hooks
    R *q_out, *b_out, *D_out;
    double* part;
    int64_t part_n;  // blocks per channel
    DamageCtrl* ctrl;
    unsigned int* ticket;
    MatC<R> mat;
};

__device__ __forceinline__ bool last_block(unsigned int* ticket)
{
    __shared__ bool s_last;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned t = atomicAdd(ticket, 1u);
        s_last = (t == gridDim.x - 1);
        if (s_last) *ticket = 0u;
    }
    __syncthreads();
    if (s_last) __threadfence();
    return s_last;
}

// fixed-order sum / min of n block partials by one CTA
__device__ __forceinline__ double reduce_partials_sum(const double* part, int64_t n, double* s_red)
{
    double v = 0.0;
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) v += __ldcg(part + i);
    return block_sum(v, s_red);
}
__device__ __forceinline__ double reduce_partials_min(const double* part, int64_t n, double* s_red)
{
    double v = INFINITY;
    for (int64_t i = threadIdx.x; i < n; i += blockDim.x) v = fmin(v, __ldcg(part + i));
    return block_min(v, s_red);
}

enum { DM_CG = 0, DM_PLAIN = 1 };

// new search direction of node gid (identical expression in the chunk and the interface kernel)
template <typename R>
__device__ __forceinline__ R new_direction(const DmgArgs<R>& a, int gid, int sel, double beta)
{
    if (!a.mask[(int64_t)sel * a.N + gid]) return R(0);
    const R z = a.r[gid] * a.dinv[gid];
    return beta == 0.0 ? z : rfma(R(beta), a.p[gid], z);
}

template <typename R, int MODE, bool PROJ>
__global__ void __launch_bounds__(kTPB) dmg_matvec_chunk(const DmgArgs<R> a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_red[32];
    R* s_p = reinterpret_cast<R*>(smem_raw);
    R* s_q = s_p + a.max_nloc;  // [3][EC]
    int sel = 0;
    double beta = 0.0;
    if (MODE == DM_CG) {
        if (a.ctrl->done) return;
        sel = a.ctrl->sel; beta = a.ctrl->beta;
    }
    const ChunkMeta cm = a.meta[blockIdx.x];
    const int nloc = cm.n_int + cm.n_halo, tid = threadIdx.x;
    double amax = INFINITY;

    for (int i = tid; i < nloc; i += kTPB) {
        const int gid = i < cm.n_int ? cm.node_start + i : a.halo_ids[cm.halo_off + i - cm.n_int];
        R pn;
        if (MODE == DM_CG) {
            pn = new_direction<R>(a, gid, sel, beta);
            if (i < cm.n_int) {
                a.p[gid] = pn;
                if (PROJ && pn < R(0)) amax = fmin(amax, (double(a.lb[gid]) - double(a.x[gid])) / double(pn));
            }
        } else {
            pn = a.p_in[gid];
        }
        s_p[i] = pn;
    }
    __syncthreads();

    for (int e = tid; e < cm.n_elem; e += kTPB) {
        const int ge = cm.elem_start + e;
        const ushort4 c = __ldg(a.lconn + ge);
        R b1, c1, b2, c2;
        Geo<R>::load(a.ga, a.gb, ge, b1, c1, b2, c2);
        const R A = __ldg(a.area + ge);
        const R ce = a.mat.c0 + R(2) * a.H[ge];  // reaction coefficient (Eq. 6 / Eq. 8)
        const R p1 = s_p[c.x], p2 = s_p[c.y], p3 = s_p[c.z];
        const R m12 = ce * A * R(1.0 / 12.0), sum = p1 + p2 + p3;  // consistent mass A(1+delta_ij)/12 (L185)
        const R gx = b1 * (p1 - p3) + b2 * (p2 - p3), gy = c1 * (p1 - p3) + c2 * (p2 - p3);
        const R kA = a.mat.kappa * A;
        const R k1 = kA * (b1 * gx + c1 * gy), k2 = kA * (b2 * gx + c2 * gy);
        s_q[e] = m12 * (p1 + sum) + k1;
        s_q[a.EC + e] = m12 * (p2 + sum) + k2;
        s_q[2 * a.EC + e] = m12 * (p3 + sum) - (k1 + k2);
    }
    __syncthreads();

    const uint16_t* ell = a.ell + cm.ell_off;
    double pq = 0.0;
    for (int i = tid; i < nloc; i += kTPB) {
        R qs = R(0);
        for (int k = 0; k < cm.ell_w; ++k) {
            const unsigned ent = ell[k * nloc + i];
            if (ent != 0xFFFFu) qs += s_q[(ent & 3) * a.EC + (ent >> 2)];
        }
        if (i < cm.n_int) {
            const int gid = cm.node_start + i;
            if (MODE == DM_CG) { a.q[gid] = qs; pq += double(s_p[i]) * double(qs); }
            else a.q_out[gid] = qs;
        } else {
            a.halo_part[cm.halo_off + i - cm.n_int] = qs;
        }
    }
    if (MODE == DM_CG) {
        const double t = block_sum(pq, s_red);
        const double tm = PROJ ? block_min(amax, s_red) : INFINITY;
        if (tid == 0) { a.part[blockIdx.x] = t; a.part[a.part_n + blockIdx.x] = tm; }
    }
}

template <typename R, int MODE, bool PROJ>
__global__ void __launch_bounds__(kTPB) dmg_matvec_shared(const DmgArgs<R> a)
{
    __shared__ double s_red[32];
    int sel = 0;
    double beta = 0.0;
    if (MODE == DM_CG) {
        if (a.ctrl->done) return;
        sel = a.ctrl->sel; beta = a.ctrl->beta;
    }
    const int s = blockIdx.x * kTPB + threadIdx.x;
    double pq = 0.0, amax = INFINITY;
    if (s < a.N_sh) {
        const int gid = a.N_int + s;
        R qs = R(0);
        for (int k = a.sh_rowptr[s]; k < a.sh_rowptr[s + 1]; ++k) qs += a.halo_part[a.sh_slots[k]];
        if (MODE == DM_CG) {
            const R pn = new_direction<R>(a, gid, sel, beta);
            a.p[gid] = pn; a.q[gid] = qs;
            pq = double(pn) * double(qs);
            if (PROJ && pn < R(0)) amax = (double(a.lb[gid]) - double(a.x[gid])) / double(pn);
        } else {
            a.q_out[gid] = qs;
        }
    }
    if (MODE != DM_CG) return;
    const double t = block_sum(pq, s_red);
    const double tm = PROJ ? block_min(amax, s_red) : INFINITY;
    if (threadIdx.x == 0) { a.part[a.C + blockIdx.x] = t; a.part[a.part_n + a.C + blockIdx.x] = tm; }
    if (last_block(a.ticket)) {
        const int64_t nb = a.C + gridDim.x;
        const double pqs = reduce_partials_sum(a.part, nb, s_red);
        const double am = PROJ ? reduce_partials_min(a.part + a.part_n, nb, s_red) : INFINITY;
        if (threadIdx.x == 0) {
            DamageCtrl* c = a.ctrl;
            double alpha = c->rho / pqs;
            c->pq = pqs; c->amax = am;
            c->truncated = (PROJ && alpha >= am) ? 1 : 0;
            if (c->truncated) alpha = am;
            c->alpha = alpha;
            c->iters += 1;
        }
    }
}

// x += alpha p, r -= alpha q; candidate free set; partial sums.  One thread per node.
template <typename R, bool PROJ>
__global__ void __launch_bounds__(kTPB) dmg_vector(const DmgArgs<R> a)
{
    __shared__ double s_red[32];
    DamageCtrl* c = a.ctrl;
    if (c->done) return;
    const int first = c->first, sel = c->sel, trunc = c->truncated;
    const double alpha = first ? 0.0 : c->alpha;
    const int i = blockIdx.x * kTPB + threadIdx.x;
    double rn_old = 0.0, rz_old = 0.0, rn_new = 0.0, rz_new = 0.0;
    if (i < a.N) {
        const bool fixed = (a.flags[i] & 4) != 0;
        const bool m_old = !first && a.mask[(int64_t)sel * a.N + i];
        R x = a.x[i], r = a.r[i];
        const R lb = a.lb[i];
        if (!first) {
            const R p = a.p[i], q = a.q[i];
            if (m_old) {
                R xn = rfma(R(alpha), p, x);
                if (PROJ) {
                    // snap the node(s) that define the truncated step, and never leave the feasible set
                    if (trunc && p < R(0) && (double(lb) - double(x)) / double(p) <= alpha * (1.0 + 1e-12)) xn = lb;
                    if (xn < lb) xn = lb;
                }
                x = xn;
                a.x[i] = x;
            }
            r = rfma(R(-alpha), q, r);  // residual kept current on ALL nodes
            a.r[i] = r;
        }
        const bool m_new = !fixed && (!PROJ || x > lb || r > R(0));
        a.mask[(int64_t)(1 - sel) * a.N + i] = m_new ? 1 : 0;
        const double rr = double(r) * double(r), rz = rr * double(a.dinv[i]);
        if (m_old) { rn_old = rr; rz_old = rz; }
        if (m_new) { rn_new = rr; rz_new = rz; }
    }
    const double t0 = block_sum(rn_old, s_red), t1 = block_sum(rz_old, s_red);
    const double t2 = block_sum(rn_new, s_red), t3 = block_sum(rz_new, s_red);
    if (threadIdx.x == 0) {
        a.part[blockIdx.x] = t0; a.part[a.part_n + blockIdx.x] = t1;
        a.part[2 * a.part_n + blockIdx.x] = t2; a.part[3 * a.part_n + blockIdx.x] = t3;
    }
    if (last_block(a.ticket)) {
        const double rno = reduce_partials_sum(a.part, gridDim.x, s_red);
        const double rzo = reduce_partials_sum(a.part + a.part_n, gridDim.x, s_red);
        const double rnn = reduce_partials_sum(a.part + 2 * a.part_n, gridDim.x, s_red);
        const double rzn = reduce_partials_sum(a.part + 3 * a.part_n, gridDim.x, s_red);
        if (threadIdx.x == 0) {
            const double lim = c->tol * c->nb;
            bool restart = first || trunc || sqrt(rno) <= lim;
            if (restart) {
                c->relres = sqrt(rnn) / c->nb;
                if (sqrt(rnn) <= lim) { c->done = 1; c->status = PFF_OK; }
                else { c->sel = 1 - sel; c->rho = rzn; c->beta = 0.0; c->restarts += 1; }
            } else {
                c->relres = sqrt(rno) / c->nb;
                c->beta = rzo / c->rho;
                c->rho = rzo;
            }
            if (!c->done && c->iters >= c->max_iter) { c->done = 1; c->status = PFF_ENOCONV; }
            c->first = 0; c->truncated = 0;
        }
    }
}

// setup: r0 = b - A x0, D^-1, lb = d_n, norms (one chunk pass + interface pass).  HOOK: only b / D out.
template <typename R, bool HOOK>
__global__ void __launch_bounds__(kTPB) dmg_setup_chunk(const DmgArgs<R> a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_red[32];
    R* s_p = reinterpret_cast<R*>(smem_raw);
    R* s_q = s_p + a.max_nloc;  // [7][EC]: q1 q2 q3 D1 D2 D3 b
    const ChunkMeta cm = a.meta[blockIdx.x];
    const int nloc = cm.n_int + cm.n_halo, tid = threadIdx.x;
    for (int i = tid; i < nloc; i += kTPB) {
        const int gid = i < cm.n_int ? cm.node_start + i : a.halo_ids[cm.halo_off + i - cm.n_int];
        s_p[i] = a.x[gid];
    }
    __syncthreads();
    for (int e = tid; e < cm.n_elem; e += kTPB) {
        const int ge = cm.elem_start + e;
        const ushort4 c = __ldg(a.lconn + ge);
        R b1, c1, b2, c2;
        Geo<R>::load(a.ga, a.gb, ge, b1, c1, b2, c2);
        const R A = __ldg(a.area + ge);
        const R He = a.H[ge];
        const R ce = a.mat.c0 + R(2) * He, se = R(2) * He - a.mat.s0;
        const R p1 = s_p[c.x], p2 = s_p[c.y], p3 = s_p[c.z];
        const R m12 = ce * A * R(1.0 / 12.0), sum = p1 + p2 + p3;
        const R gx = b1 * (p1 - p3) + b2 * (p2 - p3), gy = c1 * (p1 - p3) + c2 * (p2 - p3);
        const R kA = a.mat.kappa * A;
        const R k1 = kA * (b1 * gx + c1 * gy), k2 = kA * (b2 * gx + c2 * gy);
        s_q[e] = m12 * (p1 + sum) + k1;
        s_q[a.EC + e] = m12 * (p2 + sum) + k2;
        s_q[2 * a.EC + e] = m12 * (p3 + sum) - (k1 + k2);
        const R b3 = -(b1 + b2), c3 = -(c1 + c2);
        s_q[3 * a.EC + e] = R(2) * m12 + kA * (b1 * b1 + c1 * c1);  // A_ii = c A/6 + kappa A |grad phi_i|^2
        s_q[4 * a.EC + e] = R(2) * m12 + kA * (b2 * b2 + c2 * c2);
        s_q[5 * a.EC + e] = R(2) * m12 + kA * (b3 * b3 + c3 * c3);
        s_q[6 * a.EC + e] = se * A * R(1.0 / 3.0);  // int s phi_i
    }
    __syncthreads();
    const uint16_t* ell = a.ell + cm.ell_off;
    double nb2 = 0.0, nr2 = 0.0;
    for (int i = tid; i < nloc; i += kTPB) {
        R qs = R(0), Ds = R(0), bs = R(0);
        for (int k = 0; k < cm.ell_w; ++k) {
            const unsigned ent = ell[k * nloc + i];
            if (ent != 0xFFFFu) {
                const int e = ent >> 2, cn = ent & 3;
                qs += s_q[cn * a.EC + e]; Ds += s_q[(3 + cn) * a.EC + e]; bs += s_q[6 * a.EC + e];
            }
        }
        if (i < cm.n_int) {
            const int gid = cm.node_start + i;
            if (HOOK) {
                if (a.b_out) a.b_out[gid] = bs;
                if (a.D_out) a.D_out[gid] = Ds;
            } else {
                const R r = bs - qs;
                a.r[gid] = r; a.dinv[gid] = R(1) / Ds; a.lb[gid] = s_p[i];
                nb2 += double(bs) * double(bs);
                if (!(a.flags[gid] & 4)) nr2 += double(r) * double(r);
            }
        } else {
            const int64_t slot = cm.halo_off + i - cm.n_int;
            a.halo_part[slot] = qs; a.halo_part[a.n_slots + slot] = Ds; a.halo_part[2 * a.n_slots + slot] = bs;
        }
    }
    if (!HOOK) {
        const double t0 = block_sum(nb2, s_red), t1 = block_sum(nr2, s_red);
        if (tid == 0) { a.part[blockIdx.x] = t0; a.part[a.part_n + blockIdx.x] = t1; }
    }
}

template <typename R, bool HOOK>
__global__ void __launch_bounds__(kTPB) dmg_setup_shared(const DmgArgs<R> a)
{
    __shared__ double s_red[32];
    const int s = blockIdx.x * kTPB + threadIdx.x;
    double nb2 = 0.0, nr2 = 0.0;
    if (s < a.N_sh) {
        const int gid = a.N_int + s;
        R qs = R(0), Ds = R(0), bs = R(0);
        for (int k = a.sh_rowptr[s]; k < a.sh_rowptr[s + 1]; ++k) {
            const int slot = a.sh_slots[k];
            qs += a.halo_part[slot]; Ds += a.halo_part[a.n_slots + slot]; bs += a.halo_part[2 * a.n_slots + slot];
        }
        if (HOOK) {
            if (a.b_out) a.b_out[gid] = bs;
            if (a.D_out) a.D_out[gid] = Ds;
        } else {
            const R r = bs - qs;
            a.r[gid] = r; a.dinv[gid] = R(1) / Ds; a.lb[gid] = a.x[gid];
            nb2 = double(bs) * double(bs);
            if (!(a.flags[gid] & 4)) nr2 = double(r) * double(r);
        }
    }
    if (HOOK) return;
    const double t0 = block_sum(nb2, s_red), t1 = block_sum(nr2, s_red);
    if (threadIdx.x == 0) { a.part[a.C + blockIdx.x] = t0; a.part[a.part_n + a.C + blockIdx.x] = t1; }
    if (last_block(a.ticket)) {
        const int64_t nb = a.C + gridDim.x;
        const double sb = reduce_partials_sum(a.part, nb, s_red);
        const double sr = reduce_partials_sum(a.part + a.part_n, nb, s_red);
        if (threadIdx.x == 0) a.ctrl->nb = fmax(fmax(sqrt(sb), sqrt(sr)), 1e-300);
    }
}

// d <- min(1, max(d_n, x)) on the non-Dirichlet nodes (L179)
template <typename R>
__global__ void __launch_bounds__(kTPB) dmg_finalize(int N, R* x, const R* lb, const uint8_t* flags)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N || (flags[i] & 4)) return;
    R v = x[i];
    const R l = lb[i];
    if (v < l) v = l;
    if (v > R(1)) v = R(1);
    x[i] = v;
}

template <typename R>
static DmgArgs<R> make_args(pff_mesh* m, const pff_state* s)
{
    const HostMesh& hm = m->hm;
    DmgArgs<R> a{};
    a.meta = m->d_meta; a.lconn = (const ushort4*)m->d_lconn; a.ga = m->d_ga; a.gb = m->d_gb;
    a.area = (const R*)m->d_area; a.halo_ids = m->d_halo_ids; a.ell = m->d_ell; a.flags = m->d_flags;
    a.halo_part = (R*)m->d_halo_part; a.n_slots = m->n_slots;
    a.EC = hm.chunk_elems; a.max_nloc = hm.max_nloc; a.N = (int)hm.N; a.N_int = (int)hm.N_int; a.N_sh = (int)hm.N_sh;
    a.C = (int)hm.C; a.nbs = (int)std::max<int64_t>(1, (hm.N_sh + kTPB - 1) / kTPB);
    a.sh_rowptr = m->d_sh_rowptr; a.sh_slots = m->d_sh_slots;
    a.H = (const R*)s->H; a.x = (R*)s->d;
    a.lb = (R*)m->d_lb; a.r = (R*)m->d_r; a.p = (R*)m->d_p; a.q = (R*)m->d_q; a.dinv = (R*)m->d_dinv;
    a.mask = m->d_mask; a.part = m->d_part; a.part_n = m->n_part_blocks;
    a.ctrl = m->d_ctrl; a.ticket = m->d_ticket;
    a.mat = make_matc<R>(m->mat);
    return a;
}

static pff_status ensure_workspace(pff_mesh* m)
{
    if (m->d_ctrl) return PFF_OK;
    const HostMesh& hm = m->hm;
    const int64_t nbs = std::max<int64_t>(1, (hm.N_sh + kTPB - 1) / kTPB), nbv = (hm.N + kTPB - 1) / kTPB;
    m->n_part_blocks = std::max<int64_t>(hm.C + nbs, nbv);
    pff_status st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_part, sizeof(double) * kPartStride * m->n_part_blocks), "damage: partials")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_ctrl, sizeof(DamageCtrl)), "damage: ctrl")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_ticket, sizeof(unsigned int)), "damage: ticket")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMemset(m->d_ticket, 0, sizeof(unsigned int)), "damage: ticket")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMallocHost((void**)&m->h_ctrl, 2 * sizeof(DamageCtrl)), "damage: pinned ctrl")) != PFF_OK) return st;
    return PFF_OK;
}

// Opt a kernel instantiation in to `bytes` of dynamic shared memory (kept as a per-instantiation high-water
// mark: the limit is 227 KB minus the kernel's static shared memory, so only what is needed is requested).
template <typename K>
static pff_status set_smem(K kern, int bytes, int& granted)
{
    if (bytes <= granted) return PFF_OK;
    pff_status st = cuda_check(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes), "cudaFuncSetAttribute(damage kernel)");
    if (st == PFF_OK) granted = bytes;
    return st;
}

template <typename R, bool PROJ>
static pff_status damage_solve_t(pff_mesh* m, pff_state* s, double rel_tol, int max_iter, int* iters, double* relres)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    const HostMesh& hm = m->hm;
    DmgArgs<R> a = make_args<R>(m, s);
    cudaStream_t cs = m->stream;
    const int smem_mv = int((size_t(hm.max_nloc) + size_t(3) * hm.chunk_elems) * sizeof(R));
    const int smem_su = int((size_t(hm.max_nloc) + size_t(7) * hm.chunk_elems) * sizeof(R));
    static int g_mv = 48 * 1024, g_su = 48 * 1024;
    if ((st = set_smem(dmg_matvec_chunk<R, DM_CG, PROJ>, smem_mv, g_mv)) != PFF_OK) return st;
    if ((st = set_smem(dmg_setup_chunk<R, false>, smem_su, g_su)) != PFF_OK) return st;
    DamageCtrl* h = m->h_ctrl;  // [0]: upload image, [1]: download image
    std::memset(&h[0], 0, sizeof(DamageCtrl));
    h[0].tol = rel_tol; h[0].max_iter = max_iter; h[0].first = 1; h[0].status = PFF_ENOCONV;
    if ((st = cuda_check(cudaMemcpyAsync(m->d_ctrl, &h[0], sizeof(DamageCtrl), cudaMemcpyHostToDevice, cs), "damage: ctrl upload")) != PFF_OK) return st;
    const unsigned nbv = (unsigned)((hm.N + kTPB - 1) / kTPB);
    PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_setup_chunk<R, false><<<(unsigned)hm.C, kTPB, smem_su, cs>>>(a)));
    PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_setup_shared<R, false><<<(unsigned)a.nbs, kTPB, 0, cs>>>(a)));
    PFF_LAUNCH(m, PFF_K_CG_VECTOR, (dmg_vector<R, PROJ><<<nbv, kTPB, 0, cs>>>(a)));
    int launched = 0, batch = 2;
    for (;;) {
        for (int k = 0; k < batch; ++k) {
            PFF_LAUNCH(m, PFF_K_MATVEC_CHUNK, (dmg_matvec_chunk<R, DM_CG, PROJ><<<(unsigned)hm.C, kTPB, smem_mv, cs>>>(a)));
            PFF_LAUNCH(m, PFF_K_MATVEC_SHARED, (dmg_matvec_shared<R, DM_CG, PROJ><<<(unsigned)a.nbs, kTPB, 0, cs>>>(a)));
            PFF_LAUNCH(m, PFF_K_CG_VECTOR, (dmg_vector<R, PROJ><<<nbv, kTPB, 0, cs>>>(a)));
        }
        launched += batch;
        if ((st = cuda_check(cudaMemcpyAsync(&h[1], m->d_ctrl, sizeof(DamageCtrl), cudaMemcpyDeviceToHost, cs), "damage: ctrl download")) != PFF_OK) return st;
        if ((st = cuda_check(cudaStreamSynchronize(cs), "damage: sync")) != PFF_OK) return st;
        if (h[1].done || launched >= max_iter + 1) break;
        batch = std::min(8, batch * 2);
    }
    PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_finalize<R><<<nbv, kTPB, 0, cs>>>((int)hm.N, a.x, a.lb, a.flags)));
    if ((st = cuda_check(cudaGetLastError(), "damage solve launch")) != PFF_OK) return st;
    if ((st = cuda_check(cudaStreamSynchronize(cs), "damage: final sync")) != PFF_OK) return st;
    if (iters) *iters = h[1].iters;
    if (relres) *relres = h[1].relres;
    if (!h[1].done || h[1].status == PFF_ENOCONV) {
        set_error("pff_damage_solve: max_iter reached, relres = " + std::to_string(h[1].relres));
        return PFF_ENOCONV;
    }
    return PFF_OK;
}

pff_status damage_solve(pff_mesh* m, pff_state* s, double rel_tol, int max_iter, int* iters, double* relres)
{
    const bool proj = m->mat.model == PFF_AT1;
    if (m->opt.precision == PFF_F32)
        return proj ? damage_solve_t<float, true>(m, s, rel_tol, max_iter, iters, relres)
                    : damage_solve_t<float, false>(m, s, rel_tol, max_iter, iters, relres);
    return proj ? damage_solve_t<double, true>(m, s, rel_tol, max_iter, iters, relres)
                : damage_solve_t<double, false>(m, s, rel_tol, max_iter, iters, relres);
}

template <typename R>
static pff_status damage_matvec_t(pff_mesh* m, const pff_state* s, const void* p, void* q)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    DmgArgs<R> a = make_args<R>(m, s);
    a.p_in = (const R*)p; a.q_out = (R*)q;
    const int smem_mv = int((size_t(m->hm.max_nloc) + size_t(3) * m->hm.chunk_elems) * sizeof(R));
    static int g_mv = 48 * 1024;
    if ((st = set_smem(dmg_matvec_chunk<R, DM_PLAIN, false>, smem_mv, g_mv)) != PFF_OK) return st;
    if (m->only_kernel != 3) {
        PFF_LAUNCH(m, PFF_K_MATVEC_CHUNK, (dmg_matvec_chunk<R, DM_PLAIN, false><<<(unsigned)m->hm.C, kTPB, smem_mv, m->stream>>>(a)));
    }
    if (m->only_kernel != 2) {
        PFF_LAUNCH(m, PFF_K_MATVEC_SHARED, (dmg_matvec_shared<R, DM_PLAIN, false><<<(unsigned)a.nbs, kTPB, 0, m->stream>>>(a)));
    }
    return cuda_check(cudaGetLastError(), "damage matvec launch");
}

pff_status damage_matvec(pff_mesh* m, const pff_state* s, const void* p, void* q)
{
    return m->opt.precision == PFF_F32 ? damage_matvec_t<float>(m, s, p, q) : damage_matvec_t<double>(m, s, p, q);
}

template <typename R>
static pff_status damage_rhs_diag_t(pff_mesh* m, const pff_state* s, void* b, void* D)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    DmgArgs<R> a = make_args<R>(m, s);
    a.b_out = (R*)b; a.D_out = (R*)D;
    const int smem_su = int((size_t(m->hm.max_nloc) + size_t(7) * m->hm.chunk_elems) * sizeof(R));
    static int g_su = 48 * 1024;
    if ((st = set_smem(dmg_setup_chunk<R, true>, smem_su, g_su)) != PFF_OK) return st;
    PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_setup_chunk<R, true><<<(unsigned)m->hm.C, kTPB, smem_su, m->stream>>>(a)));
    PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_setup_shared<R, true><<<(unsigned)a.nbs, kTPB, 0, m->stream>>>(a)));
    return cuda_check(cudaGetLastError(), "damage rhs/diag launch");
}

pff_status damage_rhs_diag(pff_mesh* m, const pff_state* s, void* b, void* D)
{
    return m->opt.precision == PFF_F32 ? damage_rhs_diag_t<float>(m, s, b, D) : damage_rhs_diag_t<double>(m, s, b, D);
}

}  // namespace pff
