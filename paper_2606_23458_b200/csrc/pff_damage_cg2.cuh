// One-rendezvous CG kernel of the damage solve (included by pff_damage.cu; AT2 and the adjoint solve: no bounds).
//
// dmg_iter_chunk needs TWO grid-wide rendezvous per iteration: one before the interface nodes can be summed (their new
// direction enters the dot products p.q, q.q ...), one before alpha and beta are known.  The Chronopoulos-Gear form of CG
// applies the operator to z = D^-1 r instead of p and keeps s = A p by recurrence:
//     p_i = z_i + beta_i p_{i-1},  s_i = w_i + beta_i s_{i-1},  x_{i+1} = x_i + alpha_i p_i,  r_{i+1} = r_i - alpha_i s_i,
//     z_{i+1} = D^-1 r_{i+1},  w_{i+1} = A z_{i+1},  gamma = (r_{i+1}, z_{i+1}),  delta = (w_{i+1}, z_{i+1}),
//     beta_{i+1} = gamma_{i+1} / gamma_i,  alpha_{i+1} = gamma_{i+1} / (delta_{i+1} - beta_{i+1} gamma_{i+1} / alpha_i).
// Both inner products are LINEAR in the freshly applied operator: gamma is nodal on known values, delta = sum over elements
// of z^e . (A^e z^e) needs no assembled w.  So the interface sums can wait: w at an interface node is only needed by the
// NEXT pass's node prologue, where every chunk that touches the node sums the (by then complete) partial slots itself.
// One pass = chunk phase, ONE grid barrier, redundant sum of 3 x G block partials: no interface phase, no second barrier.
// Same iterates as standard CG in exact arithmetic (tests converge both to 1e-12..1e-13); the price is one vector more
// (s) read and written per node and one more pass per solve (the first pass only applies the operator to z_0; it writes
// no vector and does not swap the sets).
//
// Hazards: a chunk writes the new x, r, p, s of the nodes it owns (its interior nodes; interface nodes belong to the chunk
// holding their partial slot 0) while other chunks still read the old values of the same interface nodes; and it writes
// new partials while others still read the old ones.  Every vector and the partial plane therefore exist twice: a pass
// reads set `par` and writes set `par ^ 1`.  Summation orders are fixed (gather table, slot order, block order): the solve
// is bit-reproducible.
#pragma once

namespace pff {

template <typename R>
struct Cg2Args {
    DmgArgs<R> d;          // mesh tables, coefficients, 1/D (0 on nodes outside the free set), control block, partials
    R *x[2], *r[2], *p[2], *s[2], *w[2];
    R* hpart[2];           // interface partial slots of w, one plane per set
    StagePlan plan1;       // bulk-copy plan of set 1 (d.plan: set 0)
    R* x_out;              // where the result goes (state->d / lambda)
};

// stage arrays (StageLayout kind 1 re-read): node[0] r, [1] p -> z, [2] s -> new p, [3] w, [4] 1/D, [5] halo partial slots
template <typename R>
__device__ __forceinline__ void cg2_halo_gather(const Cg2Args<R>& c, int par, const StageLayout& L, unsigned char* stg, int slot,
                                                int j, int gid)
{
    constexpr int B = sizeof(R);
    reinterpret_cast<int*>(stg + L.hids)[j] = gid;
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[0]) + slot, c.r[par] + gid);
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[1]) + slot, c.p[par] + gid);
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[2]) + slot, c.s[par] + gid);
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[4]) + slot, c.d.dinv + gid);
    const R* src = c.hpart[par] + (size_t)kIfaceWidth * (gid - c.d.N_int);
    R* dst = reinterpret_cast<R*>(stg + L.node[5]) + kIfaceWidth * j;
    if (B == 8) { cp_async<16>(dst, src); cp_async<16>(dst + 2, src + 2); }
    else cp_async<16>(dst, src);
}

__device__ __forceinline__ void cg2_scalar_step(DamageCtrl* c, double gamma, double delta, double rr)
{
    const double lim = c->tol * c->nb;
    c->iters += 1;  // operator applications
    c->relres = sqrt(rr) / c->nb;
    c->pending = 0;
    if (sqrt(rr) <= lim) { c->done = 1; c->status = PFF_OK; return; }
    if (c->first) {
        c->first = 0; c->beta = 0.0;
        c->alpha = delta > 0.0 ? gamma / delta : 0.0;
    } else {
        const double beta = c->rz > 0.0 ? gamma / c->rz : 0.0;
        const double den = delta - beta * gamma / c->alpha;
        c->beta = beta;
        c->alpha = den > 0.0 ? gamma / den : 0.0;
    }
    c->rz = gamma;
    if (!(c->alpha > 0.0) || c->iters >= c->max_iter) { c->done = 1; c->status = PFF_ENOCONV; }
}

template <typename R>
__global__ void __launch_bounds__(kTPB, 3) dmg_cg2_chunk(const Cg2Args<R> c)
{
    extern __shared__ __align__(128) unsigned char smem[];
    constexpr int kC2 = 3;  // channels: gamma, delta, r.r
    __shared__ double s_w[kC2 * 32], s_out[kC2];
    __shared__ DamageCtrl s_ctrl;
    constexpr int A = 16 / sizeof(R);
    const DmgArgs<R>& a = c.d;
    const StageLayout& L = a.lay;
    R* s_slot = reinterpret_cast<R*>(smem + L.slot_base);
    ChunkMeta* s_meta = reinterpret_cast<ChunkMeta*>(smem + L.meta);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.bar);
    int* s_hid0 = reinterpret_cast<int*>(smem + L.hid0);
    const int tid = threadIdx.x, lane = tid & 31, G = gridDim.x, EC = a.EC;
    const int n_my = (a.C - (int)blockIdx.x + G - 1) / G;
    constexpr int kWorkers = kTPB - 32;  // the last warp is the producer (bulk copies + halo gathers), as in dmg_iter_chunk
    const bool issuer = tid >= kWorkers;
    StageDesc my_desc[2] = {};
    const bool have_desc = issuer && lane < a.plan.n;
    if (have_desc) { my_desc[0] = a.plan.d[lane]; my_desc[1] = c.plan1.d[lane]; }
    if (tid == 0) { mbar_init(bar, 1 + kTPB); mbar_init(bar + 2, 1 + kTPB); s_slot[3 * EC] = R(0); s_ctrl = *a.ctrl; }
    const bool single_epoch = n_my <= kMetaCap;
    bool pre_issued = false;  // the next pass's first chunk (bulk copies + halo gathers) is already on its way
    unsigned int gb_target = 0;
    int it = 0;   // stage uses so far: stage = it & 1, mbarrier parity = (it >> 1) & 1
    int par = 0;  // the set the coming pass reads; it writes par ^ 1
    int pass = 0;
    double alpha = 0.0, beta = 0.0;
    bool first = true, second = false;  // the pass that only applies the operator to z_0; the one after it
    __syncthreads();
    if (s_ctrl.done) goto finalize;  // the warm start already satisfies the stopping test (setup pass)

    for (;;) {
        const bool tr_on = pass == a.trace_iter;
        int tr_k = 0;
        PFF_TR(a.trace, tr_on, 0);
        double acc_g = 0.0, acc_d = 0.0, acc_r = 0.0;
        const R al = R(alpha), be = R(beta);
        const int wr = first ? 0 : 1;  // 0: write into the set that is read (first pass), 1: into the other one
        auto chunk_range = [&](const ChunkMeta& cm, const ChunkMeta* nx) {
            return ChunkRange{cm.elem_start, cm.n_elem, a.Ne, cm.node_start, cm.n_int, a.N, cm.ell_off,
                              cm.ell_w * (cm.n_int + cm.n_halo), (int)a.ell_total, cm.halo_off, cm.n_halo, (int)a.n_entries,
                              nx ? nx->halo_off : 0, nx ? nx->n_halo : 0};
        };
        for (int e0 = 0; e0 < n_my; e0 += kMetaCap) {
            const int n_ep = min(kMetaCap, n_my - e0);
            if (!pre_issued) {
                __syncthreads();  // previous epoch fully consumed (also publishes the mbarrier init)
                if (tid < n_ep) s_meta[tid] = a.meta[blockIdx.x + (e0 + tid) * G];
                __syncthreads();
                const ChunkMeta cm = s_meta[0];
                unsigned char* stg = smem + (it & 1) * L.stage_bytes;
                if (issuer) {
                    fence_proxy_async();
                    stage_issue_desc(my_desc[par], have_desc, stg, bar + 2 * (it & 1), lane, chunk_range(cm, n_ep > 1 ? &s_meta[1] : nullptr));
                    const int hb0 = ((cm.node_start & (A - 1)) + cm.n_int + A - 1) & ~(A - 1);
                    for (int j = lane; j < cm.n_halo; j += 32) {
                        const int gid = __ldg(a.halo_ids + cm.halo_off + j);
                        if (e0 == 0 && single_epoch) s_hid0[j] = gid;
                        cg2_halo_gather<R>(c, par, L, stg, hb0 + j, j, gid);
                    }
                }
                cp_async_mbar_arrive(bar + 2 * (it & 1));
            }
            pre_issued = false;
            for (int k = 0; k < n_ep; ++k, ++it) {
                const int st = it & 1;
                unsigned char* stg = smem + st * L.stage_bytes;
                const ushort4* s_lconn = reinterpret_cast<const ushort4*>(stg + L.lconn);
                const unsigned char* s_geo = stg + L.geo;
                R* s_r = reinterpret_cast<R*>(stg + L.node[0]);
                R* s_z = reinterpret_cast<R*>(stg + L.node[1]);   // p on arrival, z = D^-1 r_new after the prologue
                R* s_pn = reinterpret_cast<R*>(stg + L.node[2]);  // s on arrival, the new p after the prologue
                const R* s_wv = reinterpret_cast<const R*>(stg + L.node[3]);
                const R* s_dinv = reinterpret_cast<const R*>(stg + L.node[4]);
                const R* s_hp = reinterpret_cast<const R*>(stg + L.node[5]);
                const int* s_hids = reinterpret_cast<const int*>(stg + L.hids);
                const uint16_t* s_ell = reinterpret_cast<const uint16_t*>(stg + L.ell);
                const ChunkMeta cm = s_meta[k];
                const int nloc = cm.n_int + cm.n_halo;
                const int shift = cm.node_start & (A - 1), hb = (shift + cm.n_int + A - 1) & ~(A - 1);
                const int* s_hdst = reinterpret_cast<const int*>(stg + L.hdst) + (cm.halo_off & 3);

                mbar_wait(bar + 2 * st, (it >> 1) & 1);
                PFF_TR(a.trace, tr_on && tr_k < 24, 1 + 4 * tr_k);
                if (k + 1 < n_ep) {  // prefetch chunk k + 1 into the other stage (its halo ids arrived with this stage)
                    const ChunkMeta cn = s_meta[k + 1];
                    unsigned char* stn = smem + (st ^ 1) * L.stage_bytes;
                    if (issuer) {
                        fence_proxy_async();
                        stage_issue_desc(my_desc[par], have_desc, stn, bar + 2 * (st ^ 1), lane, chunk_range(cn, k + 2 < n_ep ? &s_meta[k + 2] : nullptr));
                        const int hbn = ((cn.node_start & (A - 1)) + cn.n_int + A - 1) & ~(A - 1);
                        const int* ids = reinterpret_cast<const int*>(stg + L.hnext) + (cn.halo_off & 3);
                        for (int j = lane; j < cn.n_halo; j += 32) cg2_halo_gather<R>(c, par, L, stn, hbn + j, j, ids[j]);
                    }
                    cp_async_mbar_arrive(bar + 2 * (st ^ 1));
                }
                // x of the node this thread finishes in the gather phase: requested now, consumed two phases later, so its
                // latency hides behind the prologue and the element pass (x is read and written once per pass and nothing
                // else needs it: it is not worth a shared-memory array)
                R x_pre = R(0);
                if (!first && tid < nloc) {
                    const bool interior = tid < cm.n_int;
                    const int j = tid - cm.n_int;
                    if (interior || (s_hdst[j] & (kIfaceWidth - 1)) == 0) x_pre = c.x[par][interior ? cm.node_start + tid : s_hids[j]];
                }
                // ---- node prologue (workers): s, r, p of this pass for every local node; owned nodes are written to the other set
                // (letting the producer warp take the few nodes beyond the worker count costs more than the second trip: 41.1
                // against 38.9 us per pass)
                if (!issuer) {
                    for (int i = tid; i < nloc; i += kWorkers) {
                        const bool interior = i < cm.n_int;
                        const int j = i - cm.n_int, sl = interior ? shift + i : hb + j;
                        const R dinv = s_dinv[sl], r0 = s_r[sl];
                        R rn = r0, pn = R(0), sn = R(0);
                        if (!first) {
                            const R w = interior ? s_wv[sl] : ((s_hp[4 * j] + s_hp[4 * j + 1]) + s_hp[4 * j + 2]) + s_hp[4 * j + 3];
                            // the pass after the first finds no p and s yet (the first pass wrote none): p_0 = z_0, s_0 = w_0
                            sn = second ? w : rfma(be, s_pn[sl], w);
                            rn = rfma(-al, sn, r0);
                            pn = second ? dinv * r0 : rfma(be, s_z[sl], dinv * r0);
                        }
                        const R zn = dinv * rn;
                        const bool owned = interior || (s_hdst[j] & (kIfaceWidth - 1)) == 0;
                        if (owned) {
                            if (!first) {  // the first pass changes nothing but w: no vector is written
                                const int gid = interior ? cm.node_start + i : s_hids[j];
                                c.r[par ^ 1][gid] = rn; c.p[par ^ 1][gid] = pn; c.s[par ^ 1][gid] = sn;
                            }
                            if (dinv != R(0)) { acc_g += double(rn) * double(zn); acc_r += double(rn) * double(rn); }
                        }
                        s_z[sl] = zn; s_pn[sl] = pn;
                    }
                }
                if (!issuer) asm volatile("bar.sync 1, %0;" ::"n"(kWorkers) : "memory");
                PFF_TR(a.trace, tr_on && tr_k < 24, 2 + 4 * tr_k);
                // ---- element pass (workers): q^e = A^e z^e into the slots, delta += z^e . q^e
                for (int e = tid; e < (issuer ? 0 : cm.n_elem); e += kWorkers) {
                    const ushort4 cn = s_lconn[e];
                    R m_, w12, w13, w23, q1, q2, q3;
                    Geo<R>::load_smem(s_geo, e, EC, m_, w12, w13, w23);
                    const R z1 = s_z[cn.x], z2 = s_z[cn.y], z3 = s_z[cn.z];
                    elem_damage_apply_coef<R>(m_, w12, w13, w23, z1, z2, z3, q1, q2, q3);
                    s_slot[e] = q1; s_slot[EC + e] = q2; s_slot[2 * EC + e] = q3;
                    acc_d += double(z1) * double(q1) + double(z2) * double(q2) + double(z3) * double(q3);
                }
                __syncthreads();
                PFF_TR(a.trace, tr_on && tr_k < 24, 3 + 4 * tr_k);
                // ---- ordered node gather: w = A z (interior: stored; halo: this chunk's partial), x += alpha p for owned nodes
                for (int i = tid; i < nloc; i += kTPB) {
                    const bool interior = i < cm.n_int;
                    const int j = i - cm.n_int, sl = interior ? shift + i : hb + j;
                    const int hslot = interior ? 0 : s_hdst[j];
                    const bool owned = interior || (hslot & (kIfaceWidth - 1)) == 0;
                    const int gid = interior ? cm.node_start + i : s_hids[j];
                    R xv = x_pre;
                    if (owned && i >= kTPB) xv = c.x[par][gid];  // only chunks with more local nodes than threads
                    R qs = R(0);
                    const uint16_t* row = s_ell + i;
#pragma unroll 4
                    for (int w = 0; w < cm.ell_w; ++w) qs += s_slot[row[w * nloc]];
                    // the first pass leaves its w and partials in the set it read (nobody reads either during that pass) and
                    // the sets are not swapped after it
                    if (interior) c.w[par ^ wr][gid] = qs;
                    else c.hpart[par ^ wr][hslot] = qs;
                    if (owned && !first) c.x[par ^ 1][gid] = rfma(al, s_pn[sl], xv);
                }
                __syncthreads();  // stage st and the slots are free again
                PFF_TR(a.trace, tr_on && tr_k < 24, 4 + 4 * tr_k);
                ++tr_k;
            }
        }
        PFF_TR(a.trace, tr_on, 100);
        // ---- the only grid-wide rendezvous of the pass: block partials, barrier, every CTA sums them in the same order
        {
            double v[kC2] = {acc_g, acc_d, acc_r};
#pragma unroll
            for (int ch = 0; ch < kC2; ++ch)
                for (int o = 16; o > 0; o >>= 1) v[ch] += __shfl_xor_sync(0xffffffffu, v[ch], o);
            __syncthreads();
            if (lane == 0) { for (int ch = 0; ch < kC2; ++ch) s_w[ch * 32 + (tid >> 5)] = v[ch]; }
            __syncthreads();
            if (tid < kC2 * 32) {
                const int ch = tid >> 5;
                double t = lane < kTPB / 32 ? s_w[ch * 32 + lane] : 0.0;
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0) a.part[(int64_t)ch * a.part_n + blockIdx.x] = t;
            }
        }
        PFF_TR(a.trace, tr_on, 103);
        fence_proxy_async_global();
        grid_barrier(a.ticket + 1, gb_target, (unsigned)G);
        PFF_TR(a.trace, tr_on, 104);
        par ^= wr;
        // every value of set `par` is final: the first chunk of the next pass starts streaming under the scalar reduction
        if (single_epoch) {
            const ChunkMeta cm = s_meta[0];
            unsigned char* stg = smem + (it & 1) * L.stage_bytes;
            if (issuer) {
                fence_proxy_async();
                stage_issue_desc(my_desc[par], have_desc, stg, bar + 2 * (it & 1), lane, chunk_range(cm, n_my > 1 ? &s_meta[1] : nullptr));
                const int hb0 = ((cm.node_start & (A - 1)) + cm.n_int + A - 1) & ~(A - 1);
                for (int j = lane; j < cm.n_halo; j += 32) cg2_halo_gather<R>(c, par, L, stg, hb0 + j, j, s_hid0[j]);
            }
            cp_async_mbar_arrive(bar + 2 * (it & 1));
            pre_issued = true;
        }
        {
            const int w = tid >> 5;
            if (w < kC2) {
                double u[14], t = 0.0;
                for (int base = 0; base < G; base += 32 * 14) {
#pragma unroll
                    for (int q = 0; q < 14; ++q) {
                        const int i = base + 32 * q + lane;
                        u[q] = i < G ? __ldcg(a.part + (int64_t)w * a.part_n + i) : 0.0;
                    }
#pragma unroll
                    for (int q = 0; q < 14; ++q) t += u[q];
                }
                for (int o = 16; o > 0; o >>= 1) t += __shfl_xor_sync(0xffffffffu, t, o);
                if (lane == 0) s_out[w] = t;
            }
            __syncthreads();
            if (tid == 0) cg2_scalar_step(&s_ctrl, s_out[0], s_out[1], s_out[2]);
            __syncthreads();
            second = first;
            alpha = s_ctrl.alpha; beta = s_ctrl.beta; first = s_ctrl.first != 0;
            PFF_TR(a.trace, tr_on, 105);
            ++pass;
            if (s_ctrl.done) {
                if (pre_issued) mbar_wait(bar + 2 * (it & 1), (it >> 1) & 1);  // drain the stage that was streamed ahead
                break;
            }
        }
    }
finalize:
    // ---- the latest iterate sits in set `par`: d <- min(1, max(d_n, x)) (L179) unless the caller wants it raw (adjoint)
    for (int i = blockIdx.x * kTPB + tid; i < a.N; i += G * kTPB) {
        R v = c.x[par][i];
        if (!a.no_clamp && !(a.mask[i] & 2)) {
            const R l = a.lb[i];
            if (v < l) v = l;
            if (v > R(1)) v = R(1);
        }
        c.x_out[i] = v;
    }
    if (blockIdx.x == 0 && tid == 0) {
        *a.ctrl = s_ctrl;
        if (a.tally) {
            a.tally->iters += s_ctrl.iters; a.tally->solves += 1;
            a.tally->noconv += (!s_ctrl.done || s_ctrl.status == PFF_ENOCONV) ? 1 : 0;
        }
    }
}

}  // namespace pff
