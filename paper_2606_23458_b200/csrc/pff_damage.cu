// Damage sub-problem (Eq. 6-8): matrix-free operator with consistent mass,
// Jacobi-preconditioned CG (AT2, then clamp, L179) and projected CG with an active set (AT1, L181).
//
// pff_damage_solve = ONE cooperative launch of dmg_setup_chunk + ONE cooperative launch of dmg_iter_chunk<DM_CG>
// (DESIGN.md "Damage solve"):
//   dmg_setup_chunk   persistent, TMA-fed: rhs b, Jacobi diagonal, r0 = b - A d_n, lb = d_n, free-set mask, the
//                     element operator in coefficient form (4 reals per element) and the block partials of the norms.
//                     After a grid barrier the same kernel handles the interface nodes; the last CTA to finish sets
//                     ||b||, ||r0|| (and the zero-iteration flag) in the control block.
//   dmg_iter_chunk    persistent + cooperative: runs EVERY CG iteration.  Per iteration: chunk phase (double-buffered
//                     TMA stages, cp.async halo gathers one chunk ahead; node prologue applies the PREVIOUS step
//                     x += alpha p, r -= alpha q, re-derives the free set on a restart and forms p = z + beta p;
//                     element pass q^e = (c_e M^e + kappa K^e) p^e; ordered node gather; partial sums of p.q, r.z,
//                     r.r and of the four sums that PREDICT r.z and r.r after the coming step, so beta is known
//                     without another pass over the vectors), grid barrier, interface phase, grid barrier, then
//                     every CTA reduces the block partials in the same fixed order and advances its own copy of
//                     alpha, beta and the restart / truncation / convergence flags.  After the last iteration the
//                     same kernel applies the pending step and the clamp d <- min(1, max(d_n, d)) (L179).
// alpha, beta and the norms never leave the device; the control block is initialised by the setup kernel (tolerance and
// iteration cap travel as kernel arguments: nothing is uploaded) and the host reads it back once per solve.
// Convergence is declared on the TRUE residual norm, or (AT2) on the predicted one when its rounding error bound
// is far below the tolerance.
#include <algorithm>
#include <cstring>

#include "pff_device.cuh"
#include "pff_mesh.h"

#include "pff_tma.cuh"


namespace pff {

constexpr int kMaxSharedBlocks = 1184;  // interface kernel grid cap (8 CTAs per SM, grid-stride)

template <typename R>
struct DmgArgs {
    const ChunkMeta* meta;
    const ushort4* lconn;
    const void *ga, *gb;
    void *ca, *cb;  // element-operator coefficients of the current solve (written by the setup pass)
    const R* area;
    const int32_t* halo_ids;
    const uint16_t* ell;
    const uint8_t* flags;
    R* halo_part;  // [3][n_slots]
    int64_t n_slots, n_entries, ell_total;
    int EC, N, Ne, N_int, N_sh, C, n_ovf;
    const int32_t *sh_rowptr, *halo_dst;
    StageLayout lay;
    StagePlan plan;
    const R* H;
    R* x;  // = state.d
    R *lb, *r, *p, *q, *dinv;
    uint8_t* mask;  // [N]: bit0 = in the free set, bit1 = damage-Dirichlet
    const R* p_in;  // plain mat-vec / hooks
    // adjoint solve (pff_damage_adjoint): right-hand side g instead of b(H), optional caller-given free set, and no
    // clamp of the result
    const R* rhs;
    const uint8_t* free_in;
    int no_clamp;
    int zero_dinv_fixed;  // setup pass: store 1/D = 0 on nodes outside the free set (the one-rendezvous CG masks with it)
    R *q_out, *b_out, *D_out;
    double* part;    // [kCh][part_n] chunk-kernel block partials
    int64_t part_n;
    long long* trace;        // phase timestamps (PFF_TRACE builds), CG iteration trace_iter only
    int trace_iter;
    DamageCtrl* ctrl;
    RunTally* tally;         // may be null: device-resident counters of a pff_run_steps call
    double tol;              // stopping tolerance and iteration cap of this solve (the setup kernel writes them into ctrl)
    int max_iter;
    unsigned int* ticket;    // [0] last-block ticket, [1] grid barrier of the CG kernel (zeroed by the setup kernel before it),
                             // [2] grid barrier of the setup kernel (only grows), [3] its value at the start of the launch
    MatC<R> mat;
};

enum { DM_CG = 0, DM_PLAIN = 1 };



struct IterScalars {
    double alpha, beta;
    int first, restart, trunc;
};

// The per-node prologue of one CG iteration, identical for interior, halo and interface nodes:
// applies the previous step, re-derives the free set on a restart and returns the new direction.
// x, r, mk are updated in place (mk: bit0 free, bit1 fixed).
template <typename R, bool PROJ>
__device__ __forceinline__ R cg_node_prologue(const IterScalars& sc, R& x, R& r, R p, R q, R dinv, R lb, uint8_t& mk)
{
    bool free = (mk & 1) != 0;
    const bool fixed = (mk & 2) != 0;
    if (!sc.first) {
        if (free) {
            R xn = rfma(R(sc.alpha), p, x);
            if (PROJ) {
                // snap the node(s) that define a truncated step, and never leave the feasible set
                if (sc.trunc && p < R(0) && (double(lb) - double(x)) / double(p) <= sc.alpha * (1.0 + 1e-12)) xn = lb;
                if (xn < lb) xn = lb;
            }
            x = xn;
        }
        r = rfma(R(-sc.alpha), q, r);  // residual kept current on ALL nodes
    }
    if (sc.restart) {
        free = !fixed && (!PROJ || x > lb || r > R(0));
        mk = uint8_t((free ? 1 : 0) | (fixed ? 2 : 0));
    }
    if (!free) return R(0);
    const R z = r * dinv;
    return sc.restart ? z : rfma(R(sc.beta), p, z);
}

// (elem_damage_apply and elem_coefficients live in pff_device.cuh: the explicit-step kernel's fused setup uses them too)
template <typename R>
__device__ __forceinline__ void elem_damage_apply_coef(R m, R w12, R w13, R w23, R p1, R p2, R p3, R& q1, R& q2, R& q3)
{
    const R sum = p1 + p2 + p3, d12 = p1 - p2, d13 = p1 - p3, d23 = p2 - p3;
    q1 = m * (p1 + sum) + (w12 * d12 + w13 * d13);
    q2 = m * (p2 + sum) + (w23 * d23 - w12 * d12);
    q3 = m * (p3 + sum) - (w13 * d13 + w23 * d23);
}

// Scalar step of the recurrence, run by one thread after the fixed-order reduction of all partials.
// t[]: p.q, r.z, r.r (free set, residual BEFORE the coming step), z.q, q.Dinv.q, r.q, q.q, step bound.
template <bool PROJ>
__device__ __forceinline__ void cg_scalar_step(DamageCtrl* c, const double t[kCh])
{
    const double pq = t[0], rz = t[1], rr = t[2], lim = c->tol * c->nb;
    const int was_restart = c->restart;
    c->iters += 1;
    c->first = 0;
    c->relres = sqrt(rr) / c->nb;
    // true residual norm: AT2 every iteration; AT1 on the freshly derived free set (then KKT holds)
    if ((was_restart || !PROJ) && sqrt(rr) <= lim) { c->done = 1; c->status = PFF_OK; c->pending = 0; return; }
    if (was_restart && c->iters > 1) c->restarts += 1;  // the first free set is not a RE-start
    double alpha = pq > 0.0 ? rz / pq : 0.0;
    const int trunc = (PROJ && alpha >= t[kCh - 1]) ? 1 : 0;
    if (trunc) { alpha = t[kCh - 1]; c->truncs += 1; }
    // r.z and r.r after the step, from the sums gathered in this pass (no extra pass over the vectors)
    const double rz_pred = fmax(rz - 2.0 * alpha * t[3] + alpha * alpha * t[4], 0.0);
    const double rr_pred = rr - 2.0 * alpha * t[5] + alpha * alpha * t[6];
    c->alpha = alpha; c->trunc = trunc; c->amax = t[kCh - 1]; c->rz = rz;
    c->beta = rz > 0.0 ? rz_pred / rz : 0.0;
    c->pending = 1;
    if (PROJ) {
        c->restart = (trunc || sqrt(fmax(rr_pred, 0.0)) <= lim) ? 1 : 0;
    } else {
        c->restart = 0;
        // predicted norm trusted only when its rounding-error bound is itself far below the tolerance
        const double err = 64.0 * 2.220446049250313e-16 * (rr + 2.0 * alpha * fabs(t[5]) + alpha * alpha * t[6]);
        if (rr_pred + err <= lim * lim) {
            c->done = 1; c->status = PFF_OK; c->relres = sqrt(fmax(rr_pred, 0.0)) / c->nb;
            return;
        }
    }
    if (c->iters >= c->max_iter) { c->done = 1; c->status = PFF_ENOCONV; }
}

// Indexed gather of one halo node's CG vectors into the halo slots of a stage, as asynchronous copies (LDGSTS):
// no register or scoreboard is held while the data is in flight.  The flag byte travels inside its 32-bit word.
template <typename R, int MODE, bool PROJ>
__device__ __forceinline__ void halo_gather_async(const DmgArgs<R>& a, const StageLayout& L, unsigned char* stg, int slot,
                                                  int j, int gid)
{
    constexpr int B = sizeof(R);
    reinterpret_cast<int*>(stg + L.hids)[j] = gid;
    if (MODE == DM_CG) {
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[0]) + slot, a.x + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[1]) + slot, a.r + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[2]) + slot, a.p + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[3]) + slot, a.q + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[4]) + slot, a.dinv + gid);
        if (PROJ) cp_async<B>(reinterpret_cast<R*>(stg + L.node[5]) + slot, a.lb + gid);
        cp_async<4>(reinterpret_cast<int*>(stg + L.hflag) + j, a.mask + (gid & ~3));
    } else {
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[2]) + slot, a.p_in + gid);
    }
}

// prologue of one halo node from the gathered values in its stage slot; leaves the new direction in s_p[slot]
template <typename R, int MODE, bool PROJ>
__device__ __forceinline__ void halo_prologue(const IterScalars& sc, const StageLayout& L, unsigned char* stg, int slot, int j)
{
    if (MODE != DM_CG) return;
    R* s_p = reinterpret_cast<R*>(stg + L.node[2]);
    R x = reinterpret_cast<const R*>(stg + L.node[0])[slot], r = reinterpret_cast<const R*>(stg + L.node[1])[slot];
    const R p = s_p[slot], q = reinterpret_cast<const R*>(stg + L.node[3])[slot];
    const R dinv = reinterpret_cast<const R*>(stg + L.node[4])[slot];
    const R lb = PROJ ? reinterpret_cast<const R*>(stg + L.node[5])[slot] : R(0);
    const int gid = reinterpret_cast<const int*>(stg + L.hids)[j];
    uint8_t mk = uint8_t(reinterpret_cast<const unsigned*>(stg + L.hflag)[j] >> (8 * (gid & 3)));
    s_p[slot] = cg_node_prologue<R, PROJ>(sc, x, r, p, q, dinv, lb, mk);
}

// PERSISTENT, double-buffered CG iteration kernel: gridDim.x CTAs, CTA b owns chunks b, b + G, b + 2G, ...
// While chunk k is computed, the bulk copies of chunk k + 1 are in flight into the other stage and its halo
// gathers sit in registers, so no load latency is exposed between chunks.  Shared memory (StageLayout kind 1,
// two stages): per stage lconn | geometry | area | H | x r p q 1/D lb [node_len] | mask | gather table;
// shared by both stages: scalar slots [3 EC + 1], the chunk-meta ring, two mbarriers.
template <typename R, int MODE, bool PROJ>
__global__ void __launch_bounds__(kTPB, 3) dmg_iter_chunk(const DmgArgs<R> a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ double s_w[kCh * kRedWarps], s_out[kCh];
    constexpr int A = 16 / sizeof(R);
    __shared__ DamageCtrl s_ctrl;  // every CTA keeps its own, identical copy of the recurrence scalars
    IterScalars sc{0.0, 0.0, 1, 1, 0};
    if (MODE == DM_CG && threadIdx.x == 0) s_ctrl = *a.ctrl;  // tol, max_iter, nb (setup kernels), first = restart = 1
    const StageLayout& L = a.lay;
    R* s_slot = reinterpret_cast<R*>(smem + L.slot_base);
    ChunkMeta* s_meta = reinterpret_cast<ChunkMeta*>(smem + L.meta);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.bar);
    const int tid = threadIdx.x, G = gridDim.x, EC = a.EC;
    const int n_my = (a.C - (int)blockIdx.x + G - 1) / G;  // chunks this CTA owns
    // The LAST warp is the producer: it issues the bulk copies (one lane per array) and ALL halo gathers of the next
    // chunk and takes no part in the node prologue and the element pass (the other kWorkers threads synchronise on a
    // named barrier between those two phases); it rejoins for the node gather.
    constexpr int kWorkers = kTPB - 32;
    const int lane = tid & 31;
    const bool issuer = tid >= kWorkers;
    const bool have_desc = issuer && lane < a.plan.n;
    StageDesc my_desc{};
    if (have_desc) my_desc = a.plan.d[lane];
    int* s_hid0 = reinterpret_cast<int*>(smem + L.hid0);

    if (tid == 0) { mbar_init(bar, 1 + kTPB); mbar_init(bar + 2, 1 + kTPB); s_slot[3 * EC] = R(0); }
    double acc[kCh];
    const bool single_epoch = n_my <= kMetaCap;
    bool pre_issued = false;  // the next CG iteration's first chunk is already streaming in
    bool gathers_issued = false;  // ... and its halo gathers have been issued as well
    // halo gathers of the first chunk of an epoch into its stage + every thread's arrival on the stage barrier.  The ids of
    // the CTA's very first chunk are kept in shared memory (s_hid0) and reused by every later CG iteration.
    auto issue_first_gathers = [&](unsigned char* stg, uint64_t* sbar, const ChunkMeta& cm, bool from_global) {
        if (issuer) {
            const int hb0 = ((cm.node_start & (A - 1)) + cm.n_int + A - 1) & ~(A - 1);
            const bool first_chunk = cm.elem_start == s_meta[0].elem_start && single_epoch;
            for (int j = lane; j < cm.n_halo; j += 32) {
                int gid;
                if (from_global) { gid = __ldg(a.halo_ids + cm.halo_off + j); if (first_chunk) s_hid0[j] = gid; }
                else gid = s_hid0[j];
                halo_gather_async<R, MODE, PROJ>(a, L, stg, hb0 + j, j, gid);
            }
        }
        cp_async_mbar_arrive(sbar);
    };
    unsigned int gb_target = 0;  // grid-barrier epoch target (thread 0)
    int cg_it = 0;  // CG iterations done (phase trace)
    int it = 0;  // stage uses so far (global over epochs and CG iterations): stage = it & 1, mbarrier parity = (it >> 1) & 1
    if (MODE == DM_CG) {
        __syncthreads();  // s_ctrl loaded
        if (s_ctrl.done) goto finalize;  // converged before the first iteration (setup pass)
    }
  for (;;) {  // CG iterations (DM_CG); one pass otherwise
    const bool tr_on = MODE == DM_CG && cg_it == a.trace_iter;
    int tr_k = 0;
    PFF_TR(a.trace, tr_on, 0);
#pragma unroll
    for (int c = 0; c < kCh; ++c) acc[c] = 0.0;
    acc[kCh - 1] = INFINITY;
    for (int e0 = 0; e0 < n_my; e0 += kMetaCap) {
        const int n_ep = min(kMetaCap, n_my - e0);
        if (!pre_issued) {
            __syncthreads();  // previous epoch fully consumed (also publishes the mbarrier init)
            if (tid < n_ep) s_meta[tid] = a.meta[blockIdx.x + (e0 + tid) * G];
            __syncthreads();
        }
        // epoch prologue: chunk 0 of the epoch.  First CG iteration / several epochs: loaded with exposed latency.
        // Later CG iterations of a single-epoch CTA: the bulk copies were issued right after the chunk phase of
        // the previous iteration and the halo ids are still in a register: only the gathers are issued here.
        {
            const ChunkMeta cm = s_meta[0];
            unsigned char* stg = smem + (it & 1) * L.stage_bytes;
            if (issuer && !pre_issued) {
                const ChunkRange cr{cm.elem_start, cm.n_elem, a.Ne, cm.node_start, cm.n_int, a.N, cm.ell_off,
                                    cm.ell_w * (cm.n_int + cm.n_halo), (int)a.ell_total, cm.halo_off, cm.n_halo, (int)a.n_entries,
                                    n_ep > 1 ? s_meta[1].halo_off : 0, n_ep > 1 ? s_meta[1].n_halo : 0};
                fence_proxy_async();
                stage_issue_desc(my_desc, have_desc, stg, bar + 2 * (it & 1), lane, cr);
            }
            if (!gathers_issued) issue_first_gathers(stg, bar + 2 * (it & 1), cm, !pre_issued || e0 > 0);
            gathers_issued = false;
            pre_issued = false;
        }
        for (int k = 0; k < n_ep; ++k, ++it) {
            const int st = it & 1;
            unsigned char* stg = smem + st * L.stage_bytes;
            const ushort4* s_lconn = reinterpret_cast<const ushort4*>(stg + L.lconn);
            const unsigned char* s_geo = stg + L.geo;
            R* s_x = reinterpret_cast<R*>(stg + L.node[0]);
            R* s_r = reinterpret_cast<R*>(stg + L.node[1]);
            R* s_p = reinterpret_cast<R*>(stg + L.node[2]);
            R* s_q = reinterpret_cast<R*>(stg + L.node[3]);
            const R* s_dinv = reinterpret_cast<const R*>(stg + L.node[4]);
            const R* s_lb = reinterpret_cast<const R*>(stg + L.node[5]);
            uint8_t* s_mask = stg + L.flags;
            const uint16_t* s_ell = reinterpret_cast<const uint16_t*>(stg + L.ell);
            const ChunkMeta cm = s_meta[k];
            const int nloc = cm.n_int + cm.n_halo;
            const int shift = cm.node_start & (A - 1), hb = (shift + cm.n_int + A - 1) & ~(A - 1), fshift = cm.node_start & 15;
            const int* s_hdst = reinterpret_cast<const int*>(stg + L.hdst) + (cm.halo_off & 3);

            // bulk copies AND every thread's halo gathers of this chunk (all issued one iteration ago)
            mbar_wait(bar + 2 * st, (it >> 1) & 1);
            PFF_TR(a.trace, tr_on && tr_k < 24, 1 + 4 * tr_k);
            // ---- prefetch chunk k + 1 into the other stage: bulk copies (with the halo ids of chunk k + 2) and
            // asynchronous halo gathers; the ids it needs arrived with THIS stage.  No register is held in flight.
            if (k + 1 < n_ep) {
                const ChunkMeta cn = s_meta[k + 1];
                unsigned char* stn = smem + (st ^ 1) * L.stage_bytes;
                if (issuer) {
                    const ChunkRange cr{cn.elem_start, cn.n_elem, a.Ne, cn.node_start, cn.n_int, a.N, cn.ell_off,
                                        cn.ell_w * (cn.n_int + cn.n_halo), (int)a.ell_total, cn.halo_off, cn.n_halo, (int)a.n_entries,
                                        k + 2 < n_ep ? s_meta[k + 2].halo_off : 0, k + 2 < n_ep ? s_meta[k + 2].n_halo : 0};
                    fence_proxy_async();
                    stage_issue_desc(my_desc, have_desc, stn, bar + 2 * (st ^ 1), lane, cr);
                }
                if (issuer) {
                    const int hbn = ((cn.node_start & (A - 1)) + cn.n_int + A - 1) & ~(A - 1);
                    const int* ids = reinterpret_cast<const int*>(stg + L.hnext) + (cn.halo_off & 3);
                    for (int j = lane; j < cn.n_halo; j += 32) halo_gather_async<R, MODE, PROJ>(a, L, stn, hbn + j, j, ids[j]);
                }
                cp_async_mbar_arrive(bar + 2 * (st ^ 1));
            }
            // ---- interior nodes: apply the previous step, form the new direction (owner writes)
            // (workers only, one local node each: interior nodes, then the halo nodes whose gathered values become the
            // new direction in their stage slots)
            if (MODE == DM_CG && !issuer) {
                for (int i = tid; i < nloc; i += kWorkers) {
                    if (i >= cm.n_int) { halo_prologue<R, MODE, PROJ>(sc, L, stg, hb + i - cm.n_int, i - cm.n_int); continue; }
                    const int s = shift + i, gid = cm.node_start + i;
                    R x = R(0), r = s_r[s], p = R(0), q = R(0), lb = R(0);
                    const R dinv = s_dinv[s];
                    uint8_t mk = s_mask[fshift + i];
                    const uint8_t mk0 = mk;
                    if (!sc.first) { x = s_x[s]; p = s_p[s]; q = s_q[s]; }
                    if (PROJ) { if (sc.first) x = s_x[s]; lb = s_lb[s]; }
                    const R pn = cg_node_prologue<R, PROJ>(sc, x, r, p, q, dinv, lb, mk);
                    if (!sc.first) { if (mk0 & 1) a.x[gid] = x; a.r[gid] = r; }
                    if (mk != mk0) a.mask[gid] = mk;
                    a.p[gid] = pn;
                    s_p[s] = pn; s_r[s] = r; s_mask[fshift + i] = mk;
                    if (mk & 1) {
                        const double rd = double(r), zd = rd * double(dinv);
                        acc[1] += rd * zd; acc[2] += rd * rd;
                        if (PROJ && pn < R(0)) acc[kCh - 1] = fmin(acc[kCh - 1], (double(lb) - double(x)) / double(pn));
                    }
                }
            }
            if (!issuer) asm volatile("bar.sync 1, %0;" ::"n"(kWorkers) : "memory");  // workers only
            PFF_TR(a.trace, tr_on && tr_k < 24, 2 + 4 * tr_k);

            // ---- element pass (workers)
            for (int e = tid; e < (issuer ? 0 : cm.n_elem); e += kWorkers) {
                const ushort4 c = s_lconn[e];
                R cm_, w12, w13, w23, q1, q2, q3;
                Geo<R>::load_smem(s_geo, e, EC, cm_, w12, w13, w23);  // the staged "geometry" is the coefficient stream
                elem_damage_apply_coef<R>(cm_, w12, w13, w23, s_p[c.x], s_p[c.y], s_p[c.z], q1, q2, q3);
                s_slot[e] = q1; s_slot[EC + e] = q2; s_slot[2 * EC + e] = q3;
            }
            __syncthreads();
            PFF_TR(a.trace, tr_on && tr_k < 24, 3 + 4 * tr_k);

            // ---- ordered node gather, q, partial sums
            for (int i = tid; i < nloc; i += kTPB) {
                R qs = R(0);
                const uint16_t* row = s_ell + i;
#pragma unroll 4
                for (int w = 0; w < cm.ell_w; ++w) qs += s_slot[row[w * nloc]];
                if (i < cm.n_int) {
                    const int gid = cm.node_start + i, s = shift + i;
                    if (MODE == DM_CG) {
                        a.q[gid] = qs;
                        const double qd = double(qs);
                        acc[0] += double(s_p[s]) * qd;
                        if (s_mask[fshift + i] & 1) {
                            const double rd = double(s_r[s]), dv = double(s_dinv[s]);
                            acc[3] += rd * dv * qd; acc[4] += dv * qd * qd; acc[5] += rd * qd; acc[6] += qd * qd;
                        }
                    } else {
                        a.q_out[gid] = qs;
                    }
                } else {
                    a.halo_part[s_hdst[i - cm.n_int]] = qs;
                }
            }
            __syncthreads();  // stage st and the slots are free again
            PFF_TR(a.trace, tr_on && tr_k < 24, 4 + 4 * tr_k);
            ++tr_k;
        }
    }
    if (MODE != DM_CG) break;
    PFF_TR(a.trace, tr_on, 100);
    fence_proxy_async_global();
    // ---- interface nodes (owned by no chunk): ordered sum of the chunk partials, same prologue; grid-wide phase
    grid_barrier(a.ticket + 1, gb_target, (unsigned)G);
    PFF_TR(a.trace, tr_on, 101);
    // every interior value is final: start streaming the first chunk of the next CG iteration
    if (single_epoch) {
        if (issuer) {
            const ChunkMeta cm = s_meta[0];
            const ChunkRange cr{cm.elem_start, cm.n_elem, a.Ne, cm.node_start, cm.n_int, a.N, cm.ell_off,
                                cm.ell_w * (cm.n_int + cm.n_halo), (int)a.ell_total, cm.halo_off, cm.n_halo, (int)a.n_entries,
                                n_my > 1 ? s_meta[1].halo_off : 0, n_my > 1 ? s_meta[1].n_halo : 0};
            fence_proxy_async();
            stage_issue_desc(my_desc, have_desc, smem + (it & 1) * L.stage_bytes, bar + 2 * (it & 1), lane, cr);
        }
        pre_issued = true;
    }
    {
        // Equal slice per CTA, TWO nodes per thread and trip: every load of both nodes is issued before anything is
        // computed or stored, so a trip costs one memory round trip (the slice is ~1.3 nodes per thread at 10^6 nodes).
        struct IfNode { R qs, x, r, p, q, lb, dinv; uint8_t mk; };
        auto if_load = [&](int sn, IfNode& v) {
            const int gid = a.N_int + sn;
            v.qs = iface_sum<R>(a.halo_part, sn, a.N_sh, a.n_ovf, a.sh_rowptr);
            v.r = a.r[gid]; v.dinv = a.dinv[gid]; v.mk = a.mask[gid];
            v.x = R(0); v.p = R(0); v.q = R(0); v.lb = R(0);
            if (!sc.first) { v.x = a.x[gid]; v.p = a.p[gid]; v.q = a.q[gid]; }
            if (PROJ) { if (sc.first) v.x = a.x[gid]; v.lb = a.lb[gid]; }
        };
        auto if_finish = [&](int sn, IfNode& v) {
            const int gid = a.N_int + sn;
            const uint8_t mk0 = v.mk;
            const R pn = cg_node_prologue<R, PROJ>(sc, v.x, v.r, v.p, v.q, v.dinv, v.lb, v.mk);
            if (!sc.first) { if (mk0 & 1) a.x[gid] = v.x; a.r[gid] = v.r; }
            if (v.mk != mk0) a.mask[gid] = v.mk;
            a.p[gid] = pn; a.q[gid] = v.qs;
            const double qd = double(v.qs);
            acc[0] += double(pn) * qd;
            if (v.mk & 1) {
                const double rd = double(v.r), dv = double(v.dinv);
                acc[1] += rd * rd * dv; acc[2] += rd * rd;
                acc[3] += rd * dv * qd; acc[4] += dv * qd * qd; acc[5] += rd * qd; acc[6] += qd * qd;
                if (PROJ && pn < R(0)) acc[kCh - 1] = fmin(acc[kCh - 1], (double(v.lb) - double(v.x)) / double(pn));
            }
        };
        const int if_per = (a.N_sh + G - 1) / G, if_end = min(a.N_sh, ((int)blockIdx.x + 1) * if_per);
        for (int s0 = blockIdx.x * if_per + tid; s0 < if_end; s0 += 2 * kTPB) {
            const int s1 = s0 + kTPB;
            const bool two = s1 < if_end;
            IfNode n0, n1;
            if_load(s0, n0);
            if (two) if_load(s1, n1);
            if_finish(s0, n0);
            if (two) if_finish(s1, n1);
        }
    }
    PFF_TR(a.trace, tr_on, 102);
    __syncthreads();  // reconverge before the shuffle tree (measured: 10 us per iteration faster than without)
    block_reduce_ch(acc, s_w, s_out);
    if (tid < kCh) a.part[(int64_t)tid * a.part_n + blockIdx.x] = s_out[tid];
    PFF_TR(a.trace, tr_on, 103);
    fence_proxy_async_global();
    grid_barrier(a.ticket + 1, gb_target, (unsigned)G);
    PFF_TR(a.trace, tr_on, 104);
    // ---- every value of this iteration is final: the halo gathers of the next iteration's first chunk go out now and
    // fly while the scalars are reduced (they are harmless if the solve turns out to be finished)
    if (pre_issued) {
        issue_first_gathers(smem + (it & 1) * L.stage_bytes, bar + 2 * (it & 1), s_meta[0], false);
        gathers_issued = true;
    }
    // ---- every CTA reduces all block partials in the same fixed order and advances its copy of the scalars
    {
        const int w = tid >> 5;
        constexpr int kChUsed = PROJ ? kCh : kCh - 1;  // the step-bound channel (a minimum) exists only for the projected solver
        if (w < kChUsed) {
            const double ident = (w == kCh - 1) ? INFINITY : 0.0;
            double v = ident;
            constexpr int kB = 14;  // partials per lane and batch, all loads of a batch in flight at once (G <= 448: one batch)
            for (int base = 0; base < G; base += 32 * kB) {
                double u[kB];
#pragma unroll
                for (int j = 0; j < kB; ++j) {
                    const int i = base + 32 * j + lane;
                    u[j] = i < G ? __ldcg(a.part + (int64_t)w * a.part_n + i) : ident;
                }
#pragma unroll
                for (int j = 0; j < kB; ++j) v = (w == kCh - 1) ? fmin(v, u[j]) : v + u[j];
            }
            for (int o = 16; o > 0; o >>= 1) {
                const double u = __shfl_xor_sync(0xffffffffu, v, o);
                v = (w == kCh - 1) ? fmin(v, u) : v + u;
            }
            if (lane == 0) s_out[w] = v;
        }
        __syncthreads();
        if (tid == 0) {
            double t[kCh];
            for (int c = 0; c < kCh; ++c) t[c] = c < kChUsed ? s_out[c] : INFINITY;
            cg_scalar_step<PROJ>(&s_ctrl, t);
        }
        __syncthreads();
        sc.alpha = s_ctrl.alpha; sc.beta = s_ctrl.beta; sc.first = s_ctrl.first; sc.restart = s_ctrl.restart;
        sc.trunc = s_ctrl.trunc;
        PFF_TR(a.trace, tr_on, 105);
        ++cg_it;
        if (s_ctrl.done) {
            if (pre_issued) {  // drain the stage that was streamed ahead before leaving
                if (!gathers_issued) cp_async_mbar_arrive(bar + 2 * (it & 1));
                mbar_wait(bar + 2 * (it & 1), (it >> 1) & 1);
            }
            break;
        }
    }
  }
    if (MODE != DM_CG) return;
finalize:
    // ---- converged (or out of iterations): apply the pending last step, then d <- min(1, max(d_n, x)) (L179)
    {
        const bool pending = s_ctrl.pending != 0;
        for (int i = blockIdx.x * kTPB + tid; i < a.N; i += G * kTPB) {
            const uint8_t mk = a.mask[i];
            if (mk & 2) continue;
            R v = a.x[i];
            const R l = a.lb[i];
            if (pending && (mk & 1)) {
                const R p = a.p[i];
                R xn = rfma(R(sc.alpha), p, v);
                if (PROJ && sc.trunc && p < R(0) && (double(l) - double(v)) / double(p) <= sc.alpha * (1.0 + 1e-12)) xn = l;
                v = xn;
            }
            if (!a.no_clamp) {
                if (v < l) v = l;
                if (v > R(1)) v = R(1);
            }
            a.x[i] = v;
        }
        if (blockIdx.x == 0 && tid == 0) {
            *a.ctrl = s_ctrl;
            if (a.tally) {  // single writer, stream-ordered between solves
                a.tally->iters += s_ctrl.iters; a.tally->solves += 1;
                a.tally->noconv += (!s_ctrl.done || s_ctrl.status == PFF_ENOCONV) ? 1 : 0;
                a.tally->restarts += s_ctrl.restarts; a.tally->truncs += s_ctrl.truncs;
            }
        }
    }
}

}  // namespace pff
#include "pff_damage_cg2.cuh"
namespace pff {

// interface nodes of a plain operator apply (test hook pff_damage_matvec): ordered sum of the chunk partials
template <typename R>
__global__ void __launch_bounds__(kTPB) dmg_plain_shared(const DmgArgs<R> a)
{
    for (int s = blockIdx.x * kTPB + threadIdx.x; s < a.N_sh; s += gridDim.x * kTPB)
        a.q_out[a.N_int + s] = iface_sum<R>(a.halo_part, s, a.N_sh, a.n_ovf, a.sh_rowptr);
}

// operator coefficients from the geometry and the current history field (hook path: the solve gets them from the setup pass)
template <typename R>
__global__ void __launch_bounds__(kTPB) dmg_coef_kernel(const DmgArgs<R> a)
{
    const int e = blockIdx.x * kTPB + threadIdx.x;
    if (e >= a.Ne) return;
    R b1, c1, b2, c2, m, w12, w13, w23;
    Geo<R>::load(a.ga, a.gb, e, b1, c1, b2, c2);
    elem_coefficients<R>(a.mat, b1, c1, b2, c2, a.area[e], a.H[e], m, w12, w13, w23);
    Geo<R>::store_global(a.ca, a.cb, e, m, w12, w13, w23);
}

// setup: r0 = b - A x0, D^-1, lb = d_n, mask, operator coefficients, norms (chunk pass + interface pass).  HOOK: only
// b / D out.  PERSISTENT and double-buffered like the step and CG kernels (same pipeline: TMA burst + cp.async halo
// gathers of chunk k + 1 while chunk k is computed).  Stage = StageLayout kind 2: lconn | geometry | area | H |
// x [node_len] | gather table | halo ids / partial slots; shared by both stages: slots q, D, b (each [3 EC + 1]).
template <typename R, bool HOOK>
__global__ void __launch_bounds__(kTPB, 2) dmg_setup_chunk(const DmgArgs<R> a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ double s_w[kCh * kRedWarps], s_out[kCh];
    constexpr int A = 16 / sizeof(R), B = sizeof(R);
    const StageLayout& L = a.lay;
    R* s_sq = reinterpret_cast<R*>(smem + L.slot_base);
    R* s_sD = reinterpret_cast<R*>(smem + L.slot_base + L.slot_stride);
    R* s_sb = reinterpret_cast<R*>(smem + L.slot_base + 2 * L.slot_stride);
    ChunkMeta* s_meta = reinterpret_cast<ChunkMeta*>(smem + L.meta);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.bar);
    const int tid = threadIdx.x, lane = tid & 31, G = gridDim.x, EC = a.EC;
    const int n_my = (a.C - (int)blockIdx.x + G - 1) / G;
    constexpr int kWorkers = kTPB - 32;  // the last warp is the producer (bulk copies + halo gathers), as in the CG kernel
    const bool adj = !HOOK && a.rhs != nullptr;
    const bool issuer = tid >= kWorkers;
    const bool have_desc = issuer && lane < a.plan.n;
    StageDesc my_desc{};
    if (have_desc) my_desc = a.plan.d[lane];

    if (tid == 0) {
        mbar_init(bar, 1 + kTPB); mbar_init(bar + 2, 1 + kTPB);
        s_sq[3 * EC] = R(0); s_sD[3 * EC] = R(0); s_sb[3 * EC] = R(0);
        // the CG kernel that follows in stream order counts its grid barriers from zero (the previous one has finished)
        if (blockIdx.x == 0) a.ticket[1] = 0u;
    }
    unsigned int su_epoch = 0;  // thread 0: value of the setup barrier counter before this launch
    if (tid == 0 && a.N_sh > 0) su_epoch = *reinterpret_cast<volatile unsigned int*>(a.ticket + 3);
    double acc[kCh];
#pragma unroll
    for (int c = 0; c < kCh; ++c) acc[c] = 0.0;
    int it = 0;
    for (int e0 = 0; e0 < n_my; e0 += kMetaCap) {
        const int n_ep = min(kMetaCap, n_my - e0);
        __syncthreads();
        if (tid < n_ep) s_meta[tid] = a.meta[blockIdx.x + (e0 + tid) * G];
        __syncthreads();
        {   // epoch prologue: first chunk with exposed latency
            const ChunkMeta cm = s_meta[0];
            unsigned char* stg = smem + (it & 1) * L.stage_bytes;
            if (issuer) {
                const ChunkRange cr{cm.elem_start, cm.n_elem, a.Ne, cm.node_start, cm.n_int, a.N, cm.ell_off,
                                    cm.ell_w * (cm.n_int + cm.n_halo), (int)a.ell_total, cm.halo_off, cm.n_halo, (int)a.n_entries,
                                    n_ep > 1 ? s_meta[1].halo_off : 0, n_ep > 1 ? s_meta[1].n_halo : 0};
                fence_proxy_async();
                stage_issue_desc(my_desc, have_desc, stg, bar + 2 * (it & 1), lane, cr);
            }
            if (issuer) {
                const int hb0 = ((cm.node_start & (A - 1)) + cm.n_int + A - 1) & ~(A - 1);
                for (int j = lane; j < cm.n_halo; j += 32)
                    cp_async<B>(reinterpret_cast<R*>(stg + L.node[0]) + hb0 + j, a.x + __ldg(a.halo_ids + cm.halo_off + j));
            }
            cp_async_mbar_arrive(bar + 2 * (it & 1));
        }
        for (int k = 0; k < n_ep; ++k, ++it) {
            const int st = it & 1;
            unsigned char* stg = smem + st * L.stage_bytes;
            const ushort4* s_lconn = reinterpret_cast<const ushort4*>(stg + L.lconn);
            const unsigned char* s_geo = stg + L.geo;
            const R* s_area = reinterpret_cast<const R*>(stg + L.area);
            const R* s_H = reinterpret_cast<const R*>(stg + L.H);
            R* s_x = reinterpret_cast<R*>(stg + L.node[0]);
            const uint16_t* s_ell = reinterpret_cast<const uint16_t*>(stg + L.ell);
            const ChunkMeta cm = s_meta[k];
            const int nloc = cm.n_int + cm.n_halo;
            const int shift = cm.node_start & (A - 1), fshift = cm.node_start & 15;
            const int* s_hdst = reinterpret_cast<const int*>(stg + L.hdst) + (cm.halo_off & 3);
            const uint8_t* s_flags = stg + L.flags;

            mbar_wait(bar + 2 * st, (it >> 1) & 1);
            if (k + 1 < n_ep) {  // prefetch chunk k + 1 (its halo ids arrived with this stage)
                const ChunkMeta cn = s_meta[k + 1];
                unsigned char* stn = smem + (st ^ 1) * L.stage_bytes;
                if (issuer) {
                    const ChunkRange cr{cn.elem_start, cn.n_elem, a.Ne, cn.node_start, cn.n_int, a.N, cn.ell_off,
                                        cn.ell_w * (cn.n_int + cn.n_halo), (int)a.ell_total, cn.halo_off, cn.n_halo, (int)a.n_entries,
                                        k + 2 < n_ep ? s_meta[k + 2].halo_off : 0, k + 2 < n_ep ? s_meta[k + 2].n_halo : 0};
                    fence_proxy_async();
                    stage_issue_desc(my_desc, have_desc, stn, bar + 2 * (st ^ 1), lane, cr);
                }
                if (issuer) {
                    const int hbn = ((cn.node_start & (A - 1)) + cn.n_int + A - 1) & ~(A - 1);
                    const int* ids = reinterpret_cast<const int*>(stg + L.hnext) + (cn.halo_off & 3);
                    for (int j = lane; j < cn.n_halo; j += 32) cp_async<B>(reinterpret_cast<R*>(stn + L.node[0]) + hbn + j, a.x + ids[j]);
                }
                cp_async_mbar_arrive(bar + 2 * (st ^ 1));
            }

            for (int e = tid; e < (issuer ? 0 : cm.n_elem); e += kWorkers) {  // element pass: workers only
                const ushort4 c = s_lconn[e];
                R b1, c1, b2, c2, q1, q2, q3;
                Geo<R>::load_smem(s_geo, e, EC, b1, c1, b2, c2);
                const R Ar = s_area[e], He = s_H[e];
                elem_damage_apply<R>(a.mat, b1, c1, b2, c2, Ar, He, s_x[c.x], s_x[c.y], s_x[c.z], q1, q2, q3);
                {   // the operator of this solve in coefficient form, streamed by every CG iteration
                    R m, w12, w13, w23;
                    elem_coefficients<R>(a.mat, b1, c1, b2, c2, Ar, He, m, w12, w13, w23);
                    Geo<R>::store_global(a.ca, a.cb, cm.elem_start + e, m, w12, w13, w23);
                }
                s_sq[e] = q1; s_sq[EC + e] = q2; s_sq[2 * EC + e] = q3;
                const R ce = a.mat.c0 + R(2) * He, se = R(2) * He - a.mat.s0;
                const R m12 = ce * Ar * R(1.0 / 12.0), kA = a.mat.kappa * Ar;
                const R b3 = -(b1 + b2), c3 = -(c1 + c2);
                s_sD[e] = R(2) * m12 + kA * (b1 * b1 + c1 * c1);  // A_ii = c A/6 + kappa A |grad phi_i|^2
                s_sD[EC + e] = R(2) * m12 + kA * (b2 * b2 + c2 * c2);
                s_sD[2 * EC + e] = R(2) * m12 + kA * (b3 * b3 + c3 * c3);
                const R be = se * Ar * R(1.0 / 3.0);  // int s phi_i
                s_sb[e] = be; s_sb[EC + e] = be; s_sb[2 * EC + e] = be;
            }
            __syncthreads();
            for (int i = tid; i < nloc; i += kTPB) {
                R qs = R(0), Ds = R(0), bs = R(0);
                const uint16_t* row = s_ell + i;
                for (int w = 0; w < cm.ell_w; ++w) {
                    const int idx = row[w * nloc];
                    qs += s_sq[idx]; Ds += s_sD[idx]; bs += s_sb[idx];
                }
                if (i < cm.n_int) {
                    const int gid = cm.node_start + i;
                    if (HOOK) {
                        if (a.b_out) a.b_out[gid] = bs;
                        if (a.D_out) a.D_out[gid] = Ds;
                    } else {
                        bool fixed = (s_flags[fshift + i] & 4) != 0;
                        R rhs = bs;
                        if (adj) {  // adjoint: nodes outside the caller's free set are held at lambda = 0 like Dirichlet nodes
                            fixed = fixed || (a.free_in && !a.free_in[gid]);
                            rhs = fixed ? R(0) : a.rhs[gid];
                        }
                        const R r = rhs - qs;
                        a.r[gid] = r; a.dinv[gid] = (a.zero_dinv_fixed && fixed) ? R(0) : R(1) / Ds; a.lb[gid] = s_x[shift + i];
                        a.mask[gid] = fixed ? 2 : 1;
                        acc[0] += double(rhs) * double(rhs);
                        if (!fixed) acc[1] += double(r) * double(r);
                        if (!fixed && (adj || a.mat.model != PFF_AT1 || r > R(0))) acc[2] += double(r) * double(r);  // solver's first free set
                    }
                } else {
                    const int slot = s_hdst[i - cm.n_int];
                    a.halo_part[slot] = qs; a.halo_part[a.n_slots + slot] = Ds; a.halo_part[2 * a.n_slots + slot] = bs;
                }
            }
            __syncthreads();  // stage st and the slots are free again
        }
    }
    // ---- interface nodes after a grid-wide barrier: ordered sums of the three partial planes, same outputs
    if (a.N_sh > 0) {
        unsigned int target = su_epoch;
        grid_barrier(a.ticket + 2, target, (unsigned)G);
        if (blockIdx.x == 0 && tid == 0) a.ticket[3] = target;  // all CTAs have read the epoch and arrived: next launch's epoch
        // equal slice per CTA, two nodes per thread and trip with all loads issued first (one memory round trip per trip)
        struct IfNode { R qs, Ds, bs, x, rhs; bool fixed; };
        auto if_load = [&](int sn, IfNode& v) {
            const int gid = a.N_int + sn;
            v.qs = iface_sum<R>(a.halo_part, sn, a.N_sh, a.n_ovf, a.sh_rowptr);
            v.Ds = iface_sum<R>(a.halo_part + a.n_slots, sn, a.N_sh, a.n_ovf, a.sh_rowptr);
            v.bs = iface_sum<R>(a.halo_part + 2 * a.n_slots, sn, a.N_sh, a.n_ovf, a.sh_rowptr);
            if (HOOK) return;
            v.fixed = (a.flags[gid] & 4) != 0;
            v.x = a.x[gid];
            v.rhs = v.bs;
            if (adj) {  // adjoint: nodes outside the caller's free set are held at lambda = 0 like Dirichlet nodes
                v.fixed = v.fixed || (a.free_in && !a.free_in[gid]);
                v.rhs = a.rhs[gid];
            }
        };
        auto if_finish = [&](int sn, const IfNode& v) {
            const int gid = a.N_int + sn;
            if (HOOK) {
                if (a.b_out) a.b_out[gid] = v.bs;
                if (a.D_out) a.D_out[gid] = v.Ds;
                return;
            }
            const R rhs = (adj && v.fixed) ? R(0) : v.rhs;
            const R r = rhs - v.qs;
            a.r[gid] = r; a.dinv[gid] = (a.zero_dinv_fixed && v.fixed) ? R(0) : R(1) / v.Ds; a.lb[gid] = v.x;
            a.mask[gid] = v.fixed ? 2 : 1;
            acc[0] += double(rhs) * double(rhs);
            if (!v.fixed) acc[1] += double(r) * double(r);
            if (!v.fixed && (adj || a.mat.model != PFF_AT1 || r > R(0))) acc[2] += double(r) * double(r);
        };
        const int per = (a.N_sh + G - 1) / G, end = min(a.N_sh, ((int)blockIdx.x + 1) * per);
        for (int s0 = blockIdx.x * per + tid; s0 < end; s0 += 2 * kTPB) {
            const int s1 = s0 + kTPB;
            const bool two = s1 < end;
            IfNode n0, n1;
            if_load(s0, n0);
            if (two) if_load(s1, n1);
            if_finish(s0, n0);
            if (two) if_finish(s1, n1);
        }
    }
    if (HOOK) return;
    // ---- norms: one block reduction per CTA; the last CTA to arrive sums the block partials in a fixed order
    __syncthreads();
    block_reduce_ch(acc, s_w, s_out);
    if (tid < kCh) a.part[(int64_t)tid * a.part_n + blockIdx.x] = s_out[tid];
    if (last_block(a.ticket)) {
        const int w = tid >> 5;
        if (w < 3) {
            double v = 0.0;
            for (int i = lane; i < G; i += 32) v += __ldcg(a.part + (int64_t)w * a.part_n + i);
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) s_out[w] = v;
        }
        __syncthreads();
        if (tid == 0) {  // the control block of this solve, written in full (nothing is uploaded by the host)
            DamageCtrl c{};
            c.tol = a.tol; c.max_iter = a.max_iter; c.first = 1; c.restart = 1; c.status = PFF_ENOCONV;
            c.nb = fmax(fmax(sqrt(s_out[0]), sqrt(s_out[1])), 1e-300);
            // d_n already solves the system to the tolerance (no history growth since the last solve; AT1: KKT holds with
            // the free set the solver would start from): no CG iteration is needed, the cooperative kernel only clamps
            if (sqrt(s_out[2]) <= c.tol * c.nb) { c.done = 1; c.status = PFF_OK; c.relres = sqrt(s_out[2]) / c.nb; }
            *a.ctrl = c;
        }
    }
}

template <typename R>
static DmgArgs<R> make_args(pff_mesh* m, const pff_state* s)
{
    const HostMesh& hm = m->hm;
    DmgArgs<R> a{};
    a.meta = m->d_meta; a.lconn = (const ushort4*)m->d_lconn; a.ga = m->d_ga; a.gb = m->d_gb; a.ca = m->d_ca; a.cb = m->d_cb;
    a.area = (const R*)m->d_area; a.halo_ids = m->d_halo_ids; a.ell = m->d_ell; a.flags = m->d_flags;
    a.halo_part = (R*)m->d_halo_part; a.n_slots = m->n_slots; a.n_entries = m->n_entries; a.ell_total = m->ell_total; a.n_ovf = hm.n_ovf;
    a.EC = hm.chunk_elems;
    a.N = (int)hm.N; a.Ne = (int)hm.Ne; a.N_int = (int)hm.N_int; a.N_sh = (int)hm.N_sh; a.C = (int)hm.C;
    a.sh_rowptr = m->d_sh_rowptr; a.halo_dst = m->d_halo_dst;
    a.H = (const R*)s->H; a.x = (R*)s->d;
    a.lb = (R*)m->d_lb; a.r = (R*)m->d_r; a.p = (R*)m->d_p; a.q = (R*)m->d_q; a.dinv = (R*)m->d_dinv;
    a.mask = m->d_mask; a.part = m->d_part; a.part_n = m->n_part_blocks;
    a.ctrl = m->d_ctrl; a.ticket = m->d_ticket; a.trace = m->d_trace; a.trace_iter = m->trace_iter;
    a.mat = make_matc<R>(m->mat);
    return a;
}

// TMA plan of a damage chunk kernel: which = 0 CG iteration (lb only for the projected variant), 1 plain
// mat-vec (trial vector only), 2 setup (x only).  Kinds: 0 elements, 1 interior nodes, 2 gather table.
template <typename R>
static void set_plan(pff_mesh* m, DmgArgs<R>& a, int which, bool proj)
{
    const StageLayout& L = which == 2 ? m->lay_su : m->lay_mv;
    a.lay = L;
    StagePlan& P = a.plan;
    P.n = 0;
    const uint16_t lr = sizeof(R) == 8 ? 3 : 2;
    auto add = [&](const void* src, uint32_t off, uint16_t l, uint16_t kind) { P.d[P.n++] = StageDesc{src, off, l, kind}; };
    add(m->d_lconn, L.lconn, 3, 0);
    const void *g0 = which == 2 ? m->d_ga : m->d_ca, *g1 = which == 2 ? m->d_gb : m->d_cb;  // geometry / coefficients
    if (sizeof(R) == 8) { add(g0, L.geo, 4, 0); add(g1, L.geo + 16u * (uint32_t)m->hm.chunk_elems, 4, 0); }
    else add(g0, L.geo, 4, 0);
    if (which == 2) { add(m->d_area, L.area, lr, 0); add(a.H, L.H, lr, 0); }
    add(m->d_ell, L.ell, 1, 2);
    add(m->d_halo_dst, L.hdst, 2, 3);   // partial slots of the chunk's halo nodes
    add(m->d_halo_ids, L.hnext, 2, 4);  // ids of the next chunk's halo nodes
    if (which == 0) {
        add(a.x, L.node[0], lr, 1); add(a.r, L.node[1], lr, 1); add(a.p, L.node[2], lr, 1); add(a.q, L.node[3], lr, 1);
        add(a.dinv, L.node[4], lr, 1);
        if (proj) add(a.lb, L.node[5], lr, 1);
        add(a.mask, L.flags, 0, 1);
    } else if (which == 1) {
        add(a.p_in, L.node[2], lr, 1);
    } else {
        add(a.x, L.node[0], lr, 1);
        add(m->d_flags, L.flags, 0, 1);
    }
}

static unsigned shared_grid(const HostMesh& hm)
{
    return (unsigned)std::min<int64_t>(kMaxSharedBlocks, std::max<int64_t>(1, (hm.N_sh + kTPB - 1) / kTPB));
}

static pff_status ensure_workspace(pff_mesh* m)
{
    if (m->d_ctrl) return PFF_OK;
    const HostMesh& hm = m->hm;
    m->n_part_blocks = hm.C;
    pff_status st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_part, sizeof(double) * kCh * m->n_part_blocks), "damage: partials")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_ctrl, sizeof(DamageCtrl)), "damage: ctrl")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_ticket, 4 * sizeof(unsigned int)), "damage: ticket")) != PFF_OK) return st;  // [0] last-block ticket, [1] CG grid barrier, [2] setup grid barrier
    if ((st = cuda_check(cudaMemset(m->d_ticket, 0, 4 * sizeof(unsigned int)), "damage: ticket")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMallocHost((void**)&m->h_ctrl, sizeof(DamageCtrl)), "damage: pinned ctrl")) != PFF_OK) return st;
    return PFF_OK;
}

// One cooperative launch of a setup-kernel instantiation (chunk phase, grid barrier, interface phase, norms).  Its grid
// barrier counter only grows; the epoch lives on the device and is advanced by the kernel itself (graph-replayable).
template <typename R>
static pff_status launch_setup(pff_mesh* m, DmgArgs<R>& asu, const void* kern, unsigned g, int smem)
{
    void* kargs[] = {(void*)&asu};
    prof_mark(m, PFF_K_DAMAGE_SETUP);
    cudaError_t e = launch_cooperative(kern, g, kTPB, kargs, (size_t)smem, m->stream);
    prof_mark(m, PFF_K_DAMAGE_SETUP);
    if (e != cudaSuccess) return cuda_check(e, "damage: setup launch");
    ++m->n_launches;
    return PFF_OK;
}

// Which CG kernel an unconstrained / projected forward solve of this mesh runs (see damage_solve_t): true = the
// one-rendezvous kernel.  Shared with the fused setup of the explicit-step kernel, which must store 1/D the same way.
template <typename R>
static pff_status solve_uses_cg2(pff_mesh* m, bool proj, bool* cg2, int* grid_cg2_out = nullptr)
{
    int grid_cg2 = 0;
    pff_status st = persistent_config(m, (const void*)dmg_cg2_chunk<R>, (int)m->lay_mv.total, &grid_cg2);
    if (st != PFF_OK) return st;
    const bool eligible = !proj && m->hm.n_ovf == 0;
    *cg2 = eligible && (m->cg_variant == 2 || (m->cg_variant == 0 && m->hm.C <= (int64_t)16 * grid_cg2));
    if (grid_cg2_out) *grid_cg2_out = grid_cg2;
    return PFF_OK;
}

struct AdjointIn {
    const void* g;
    const uint8_t* free_mask;
    void* lambda;
};

template <typename R, bool PROJ>
static pff_status damage_solve_t(pff_mesh* m, const pff_state* s, double rel_tol, int max_iter, int* iters, double* relres,
                                 const AdjointIn* adj = nullptr)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    const HostMesh& hm = m->hm;
    DmgArgs<R> a = make_args<R>(m, s);
    if (adj) { a.x = (R*)adj->lambda; a.rhs = (const R*)adj->g; a.free_in = adj->free_mask; a.no_clamp = 1; }
    DmgArgs<R> asu = a;
    set_plan<R>(m, a, 0, PROJ);
    set_plan<R>(m, asu, 2, PROJ);
    const int smem_mv = (int)m->lay_mv.total, smem_su = (int)m->lay_su.total;
    cudaStream_t cs = m->stream;
    int grid_mv = 0, grid_su = 0;
    // Unconstrained solves (AT2, adjoint) on meshes without overflow partial slots run the one-rendezvous kernel
    // (pff_damage_cg2.cuh) as long as a CTA of the persistent grid owns at most 16 chunks (~1.4e6 nodes in fp64): its pass is
    // 33 % (10^4 nodes) to 7 % (10^6 nodes) shorter because the grid-wide tail is a large part of a pass there, which pays
    // for its one extra (cheaper) pass per solve: -25 % per solve up to 10^5 nodes, a tie at 10^6 nodes and 12 passes, -5 % at
    // 85 passes (profiles/r2_cg_kernels.md).  On larger meshes the tail is amortised and the extra pass is a loss (4e6
    // nodes, 12 passes: +6 %).  The projected solver (AT1) and irregular decompositions keep the two-rendezvous kernel.
    bool cg2 = false;
    if ((st = solve_uses_cg2<R>(m, PROJ, &cg2)) != PFF_OK) return st;
    m->last_cg_kernel = cg2 ? 2 : 1;
    const void* cg_kernel = cg2 ? (const void*)dmg_cg2_chunk<R> : (const void*)dmg_iter_chunk<R, DM_CG, PROJ>;
    Cg2Args<R> c2{};
    if (cg2) {
        const size_t ld = ((size_t)hm.N + 15) & ~size_t(15);
        if (!m->d_cg2) {
            if ((st = cuda_check(cudaMalloc(&m->d_cg2, 6 * ld * m->rb), "damage: second vector set")) != PFF_OK) return st;
        }
        R* base = (R*)m->d_cg2;
        c2.x[0] = a.x; c2.x[1] = base; c2.r[0] = a.r; c2.r[1] = base + ld; c2.p[0] = a.p; c2.p[1] = base + 2 * ld;
        c2.s[0] = a.q; c2.s[1] = base + 3 * ld; c2.w[0] = base + 4 * ld; c2.w[1] = base + 5 * ld;
        c2.hpart[0] = a.halo_part; c2.hpart[1] = a.halo_part + m->n_slots;
        c2.x_out = a.x;
        asu.zero_dinv_fixed = 1;
    }
    if ((st = persistent_config(m, cg_kernel, smem_mv, &grid_mv)) != PFF_OK) return st;
    if ((st = persistent_config(m, (const void*)dmg_setup_chunk<R, false>, smem_su, &grid_su)) != PFF_OK) return st;
    const unsigned gmv = (unsigned)std::min<int64_t>(grid_mv, hm.C), gsu = (unsigned)std::min<int64_t>(grid_su, hm.C);
    asu.tol = rel_tol; asu.max_iter = max_iter;
    a.tally = m->defer ? m->d_tally : nullptr;
    if (cg2) {  // bulk-copy plans of the two vector sets (StageLayout kind 1 re-read: r, p, s, w, 1/D, halo partial slots)
        for (int par = 0; par < 2; ++par) {
            StagePlan& P = par == 0 ? a.plan : c2.plan1;
            const StageLayout& L = m->lay_mv;
            P.n = 0;
            const uint16_t lr = sizeof(R) == 8 ? 3 : 2;
            auto add = [&](const void* src, uint32_t off, uint16_t l, uint16_t kind) { P.d[P.n++] = StageDesc{src, off, l, kind}; };
            add(m->d_lconn, L.lconn, 3, 0);
            if (sizeof(R) == 8) { add(m->d_ca, L.geo, 4, 0); add(m->d_cb, L.geo + 16u * (uint32_t)hm.chunk_elems, 4, 0); }
            else add(m->d_ca, L.geo, 4, 0);
            add(m->d_ell, L.ell, 1, 2);
            add(m->d_halo_dst, L.hdst, 2, 3);
            add(m->d_halo_ids, L.hnext, 2, 4);
            add(c2.r[par], L.node[0], lr, 1); add(c2.p[par], L.node[1], lr, 1); add(c2.s[par], L.node[2], lr, 1);
            add(c2.w[par], L.node[3], lr, 1); add(a.dinv, L.node[4], lr, 1);
        }
        c2.d = a;
    }
    // the explicit-step kernel of pff_run_steps may have done this solve's setup pass already (pff_step.cu MODE_STEPSU)
    const bool fused = m->su_ready && !adj && m->su_tol == rel_tol && m->su_max_iter == max_iter && m->su_zero_dinv == asu.zero_dinv_fixed;
    m->su_ready = false;
    if (!fused && (st = launch_setup(m, asu, (const void*)dmg_setup_chunk<R, false>, gsu, smem_su)) != PFF_OK) return st;
    // ONE cooperative launch runs every CG iteration (grid-wide barriers between the chunk phase, the interface
    // phase and the scalar recurrence), applies the last step and the clamp, and writes the control block back
    {
        void* kargs[] = {cg2 ? (void*)&c2 : (void*)&a};
        prof_mark(m, PFF_K_MATVEC_CHUNK);
        cudaError_t e = launch_cooperative(cg_kernel, gmv, kTPB, kargs, (size_t)smem_mv, cs);
        prof_mark(m, PFF_K_MATVEC_CHUNK);
        ++m->n_launches;
        if ((st = cuda_check(e, "damage: cooperative launch")) != PFF_OK) return st;
    }
    if (m->defer) return PFF_OK;  // pff_run_steps: the kernel has tallied its counters on the device; nothing is read back here
    DamageCtrl* h = m->h_ctrl;  // pinned download image; the stream is synchronised before it is read or reused
    if ((st = cuda_check(cudaMemcpyAsync(h, m->d_ctrl, sizeof(DamageCtrl), cudaMemcpyDeviceToHost, cs), "damage: ctrl download")) != PFF_OK) return st;
    if ((st = cuda_check(cudaStreamSynchronize(cs), "damage: sync")) != PFF_OK) return st;
    m->last_restarts = h->restarts; m->last_truncs = h->truncs;
    if (iters) *iters = h->iters;
    if (relres) *relres = h->relres;
    if (!h->done || h->status == PFF_ENOCONV) {
        set_error("pff_damage_solve: max_iter reached, relres = " + std::to_string(h->relres));
        return PFF_ENOCONV;
    }
    return PFF_OK;
}

// Buffers and options of the setup pass of the NEXT forward solve of this mesh (tolerance and cap in m->su_tol /
// m->su_max_iter), for the explicit-step kernel that performs it (pff_step.cu MODE_STEPSU).
pff_status damage_fused_setup(pff_mesh* m, FusedSetup* fs)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    bool cg2 = false;
    st = m->opt.precision == PFF_F32 ? solve_uses_cg2<float>(m, m->mat.model == PFF_AT1, &cg2)
                                     : solve_uses_cg2<double>(m, m->mat.model == PFF_AT1, &cg2);
    if (st != PFF_OK) return st;
    if (!m->d_su_part) {
        const size_t nb = size_t(3) * std::max<int64_t>(m->n_slots, 1) * m->rb;
        if ((st = cuda_check(cudaMalloc(&m->d_su_part, nb), "fused setup: partial planes")) != PFF_OK) return st;
        if ((st = cuda_check(cudaMemsetAsync(m->d_su_part, 0, nb, m->stream), "fused setup: partial planes")) != PFF_OK) return st;  // unused slots stay zero
    }
    fs->ca = m->d_ca; fs->cb = m->d_cb; fs->r = m->d_r; fs->dinv = m->d_dinv; fs->lb = m->d_lb; fs->mask = m->d_mask;
    fs->part3 = m->d_su_part; fs->part = m->d_part; fs->part_n = m->n_part_blocks; fs->ticket = m->d_ticket; fs->ctrl = m->d_ctrl;
    fs->tol = m->su_tol; fs->max_iter = m->su_max_iter; fs->zero_dinv_fixed = cg2 ? 1 : 0;
    m->su_zero_dinv = fs->zero_dinv_fixed;
    m->su_ready = true;
    return PFF_OK;
}

// gather meshes with the Jacobi solver whose fused stage still leaves two CTAs per SM; off with pff_set_fused_setup(mesh, 0)
bool fused_setup_ok(const pff_mesh* m)
{
    return m->fuse_setup != 0 && m->opt.scatter == PFF_SCATTER_GATHER && !(m->damage_solver == 1 && m->mg) &&
           2 * (m->lay_stepsu.total + kSmemCtaReserve) <= kSmemPerSM;
}

pff_status damage_solve(pff_mesh* m, pff_state* s, double rel_tol, int max_iter, int* iters, double* relres)
{
    // the multigrid-preconditioned solver where the caller selected it (pff_set_damage_solver) and it applies
    if (m->damage_solver == 1 && m->mg) return mg_solve(m, s, rel_tol, max_iter, iters, relres);
    const bool proj = m->mat.model == PFF_AT1;
    if (m->opt.precision == PFF_F32)
        return proj ? damage_solve_t<float, true>(m, s, rel_tol, max_iter, iters, relres)
                    : damage_solve_t<float, false>(m, s, rel_tol, max_iter, iters, relres);
    return proj ? damage_solve_t<double, true>(m, s, rel_tol, max_iter, iters, relres)
                : damage_solve_t<double, false>(m, s, rel_tol, max_iter, iters, relres);
}

// Adjoint of the converged damage system (section 4.2, Eq. 23): A_FF lambda_F = g_F with the operator of state->H,
// by the same setup + cooperative CG kernels as the forward solve (unprojected, from lambda = 0, no clamp).
pff_status damage_adjoint(pff_mesh* m, const pff_state* s, const void* g, const uint8_t* free_mask, void* lambda, double rel_tol,
                          int max_iter, int* iters, double* relres)
{
    pff_status st = cuda_check(cudaMemsetAsync(lambda, 0, (size_t)m->hm.N * m->rb, m->stream), "adjoint: zero lambda");
    if (st != PFF_OK) return st;
    // a linear solve on a given free set: the multigrid solver takes it for both models where the caller selected it
    if (m->damage_solver == 1 && m->mg) return mg_adjoint(m, s, g, free_mask, lambda, rel_tol, max_iter, iters, relres);
    const AdjointIn in{g, free_mask, lambda};
    if (m->opt.precision == PFF_F32) return damage_solve_t<float, false>(m, s, rel_tol, max_iter, iters, relres, &in);
    return damage_solve_t<double, false>(m, s, rel_tol, max_iter, iters, relres, &in);
}

template <typename R>
static pff_status damage_matvec_t(pff_mesh* m, const pff_state* s, const void* p, void* q, bool refresh_coef, bool skip_interface)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    DmgArgs<R> a = make_args<R>(m, s);
    a.p_in = (const R*)p; a.q_out = (R*)q;
    set_plan<R>(m, a, 1, false);
    const int smem_mv = (int)m->lay_mv.total;
    int grid_mv = 0;
    if ((st = persistent_config(m, (const void*)dmg_iter_chunk<R, DM_PLAIN, false>, smem_mv, &grid_mv)) != PFF_OK) return st;
    grid_mv = (int)std::min<int64_t>(grid_mv, m->hm.C);
    if (refresh_coef && m->only_kernel < 0) {  // the operator of state->H in coefficient form (timing hook, multigrid cycles: reuse the previous one)
        PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_coef_kernel<R><<<(unsigned)((m->hm.Ne + kTPB - 1) / kTPB), kTPB, 0, m->stream>>>(a)));
    }
    if (m->only_kernel != 3) {
        PFF_LAUNCH(m, PFF_K_MATVEC_CHUNK, (dmg_iter_chunk<R, DM_PLAIN, false><<<(unsigned)grid_mv, kTPB, smem_mv, m->stream>>>(a)));
    }
    if (m->only_kernel != 2 && !skip_interface) {  // (multigrid: the consumer of q sums the interface partials itself)
        PFF_LAUNCH(m, PFF_K_MATVEC_SHARED, (dmg_plain_shared<R><<<shared_grid(m->hm), kTPB, 0, m->stream>>>(a)));
    }
    return cuda_check(cudaGetLastError(), "damage matvec launch");
}

// operator coefficients of state->H alone (multigrid set-up: the cycles then apply the operator with refresh_coef = false)
template <typename R>
static pff_status damage_refresh_coef_t(pff_mesh* m, const pff_state* s)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    DmgArgs<R> a = make_args<R>(m, s);
    PFF_LAUNCH(m, PFF_K_DAMAGE_SETUP, (dmg_coef_kernel<R><<<(unsigned)((m->hm.Ne + kTPB - 1) / kTPB), kTPB, 0, m->stream>>>(a)));
    return cuda_check(cudaGetLastError(), "damage coefficients launch");
}

pff_status damage_refresh_coef(pff_mesh* m, const pff_state* s)
{
    return m->opt.precision == PFF_F32 ? damage_refresh_coef_t<float>(m, s) : damage_refresh_coef_t<double>(m, s);
}

pff_status damage_matvec(pff_mesh* m, const pff_state* s, const void* p, void* q, bool refresh_coef, bool skip_interface)
{
    return m->opt.precision == PFF_F32 ? damage_matvec_t<float>(m, s, p, q, refresh_coef, skip_interface)
                                       : damage_matvec_t<double>(m, s, p, q, refresh_coef, skip_interface);
}

template <typename R>
static pff_status damage_rhs_diag_t(pff_mesh* m, const pff_state* s, void* b, void* D)
{
    pff_status st = ensure_workspace(m);
    if (st != PFF_OK) return st;
    DmgArgs<R> a = make_args<R>(m, s);
    a.b_out = (R*)b; a.D_out = (R*)D;
    set_plan<R>(m, a, 2, false);
    const int smem_su = (int)m->lay_su.total;
    int grid_su = 0;
    if ((st = persistent_config(m, (const void*)dmg_setup_chunk<R, true>, smem_su, &grid_su)) != PFF_OK) return st;
    return launch_setup(m, a, (const void*)dmg_setup_chunk<R, true>, (unsigned)std::min<int64_t>(grid_su, m->hm.C), smem_su);
}

pff_status damage_rhs_diag(pff_mesh* m, const pff_state* s, void* b, void* D)
{
    return m->opt.precision == PFF_F32 ? damage_rhs_diag_t<float>(m, s, b, D) : damage_rhs_diag_t<double>(m, s, b, D);
}

}  // namespace pff
