// Explicit step kernels (Eq. 16-18; element math L42, L71-93, L124):
//
//   step_chunk_kernel   PERSISTENT CTAs, each owning every G-th chunk of elements; two shared-memory stages: the
//                       contiguous arrays of chunk k + 1 stream in by TMA (cp.async.bulk) and its halo nodes by
//                       cp.async while chunk k is computed.  Phase 1 forms the predictor u_{n+1} (Eq. 16) of all
//                       nodes the chunk touches in place in the stage; phase 2 is the fused element pass
//                       (strain -> split -> degradation -> stress -> force -> history) writing element forces
//                       to shared-memory slots; phase 3 gathers each node's incident slots in a fixed order
//                       (chunk-local ELL table) and, for interior nodes, completes Eq. 17-18 in the same
//                       kernel -- f_int never reaches HBM.  Interface nodes get one partial sum per chunk.
//                       After a grid-wide barrier (cooperative launch) the same kernel finishes the interface
//                       nodes: ordered sum of the per-chunk partials, then the same Eq. 16-18.
//   elem_atomic_kernel / node_atomic_kernel   PFF_SCATTER_ATOMIC variant: thread per element, global
//                       floating-point atomics (the paper's "atomic indexed accumulation", L43, L124).
//   dirichlet_kernel    writes u_bar, v_bar into the Dirichlet dofs before the step (Eq. 5, R8).
#include <algorithm>

#include "pff_device.cuh"
#include "pff_mesh.h"
#include "pff_tma.cuh"

namespace pff {

// MODE_TANGENT: matrix-free stiffness action q = f_int(u + p) - f_int(u) (Eq. 13), both forces in ONE element pass
// MODE_EQ: one WHOLE iteration of the quasi-static mechanics CG (pff_equilibrium.cu) in one pass: the node prologue applies
// the previous step (du += alpha p, r -= alpha q) and forms p = D^-1 r + beta p, the element pass is MODE_TANGENT's, the
// gather leaves q = K p and the sums that give alpha and PREDICT beta; the last CTA advances the scalars.
// MODE_STEPSU: the explicit step with the SETUP PASS of the damage solve that follows it fused in (pff_run_steps): the
// step kernel already has everything that pass reads in shared memory -- connectivity, geometry, area, the new history
// value, d -- so the element pass also forms the damage operator's coefficients (streamed to HBM for the CG iterations),
// its action on d_n, its diagonal and the right-hand side, and the one gather walk sums them next to the forces: the
// setup kernel's 120 MB of re-reads, its pipeline fill and its grid-wide tail disappear.  Same arithmetic in the same
// order as dmg_setup_chunk (pff_damage.cu): bit-identical r0, 1/D, coefficients, norms.
enum { MODE_STEP = 0, MODE_INIT = 1, MODE_FORCE = 2, MODE_TANGENT = 3, MODE_EQ = 4, MODE_STEPSU = 5 };

template <typename R>
struct StepArgs {
    const ChunkMeta* meta;
    const ushort4* lconn;
    const int4* conn;
    const void *ga, *gb;
    const R* area;
    const int32_t* halo_ids;
    const uint16_t* ell;
    const uint8_t* flags;
    const R* minv;
    R* halo_part;  // [2][n_slots]
    int64_t n_slots;
    int EC, N, Ne, N_int, N_sh, n_ovf, C;
    int64_t ell_total, n_entries;
    const int32_t *sh_rowptr, *halo_dst;
    unsigned int* gbar;    // [0] grid-barrier arrival counter (only grows), [1] its value when this launch started: kept on
                           // the device and advanced by the kernel itself, so a launch can be replayed from a CUDA graph
    StageLayout lay;
    StagePlan plan;
    R *ux, *uy, *vx, *vy, *ax, *ay;
    const R* d;
    R* H;
    const R *fex, *fey;
    R *fx_out, *fy_out, *psi_out;
    const R *px, *py;  // MODE_TANGENT: trial direction
    // MODE_EQ: CG vectors of the quasi-static solve (du, r, p, q in/out; 1/D in), its control block, block partials, ticket
    R *ex, *ey, *rx, *ry, *cpx, *cpy;
    const R *dix, *diy;
    DamageCtrl* eq_ctrl;
    double* eq_part;   // [kCh][gridDim.x]
    unsigned int* eq_ticket;
    R *fwx, *fwy;
    FusedSetup su;  // MODE_STEPSU: outputs of the fused damage setup (pff_mesh.h)
    R dt, hdt, hdt2, S;
    MatC<R> mat;
    long long* trace;  // phase timestamps (PFF_TRACE builds)
};

// Eq. 16 with the Dirichlet overwrite: flagged dofs hold u_bar already (dirichlet_kernel).
template <typename R, int MODE>
__device__ __forceinline__ void predict(const StepArgs<R>& a, int gid, R& upx, R& upy)
{
    const R ux = a.ux[gid], uy = a.uy[gid];
    if (MODE != MODE_STEP) { upx = ux; upy = uy; return; }
    const uint8_t fl = a.flags[gid];
    const R px = rfma(a.hdt2, a.ax[gid], rfma(a.dt, a.vx[gid], ux));
    const R py = rfma(a.hdt2, a.ay[gid], rfma(a.dt, a.vy[gid], uy));
    upx = (fl & 1) ? ux : px;
    upy = (fl & 2) ? uy : py;
}

// Eq. 17-18 for one node given its assembled internal force.
template <typename R, int MODE>
__device__ __forceinline__ void finish_node(const StepArgs<R>& a, int gid, R upx, R upy, R fx, R fy)
{
    if (MODE == MODE_FORCE || MODE == MODE_TANGENT) { a.fx_out[gid] = fx; a.fy_out[gid] = fy; return; }
    const uint8_t fl = a.flags[gid];
    const R minv = a.minv[gid];
    R axn = (a.S * a.fex[gid] - fx) * minv;
    R ayn = (a.S * a.fey[gid] - fy) * minv;
    if (fl & 1) axn = R(0);
    if (fl & 2) ayn = R(0);
    if (MODE == MODE_STEP) {
        const R vxo = a.vx[gid], vyo = a.vy[gid], axo = a.ax[gid], ayo = a.ay[gid];
        a.ux[gid] = upx; a.uy[gid] = upy;
        a.vx[gid] = (fl & 1) ? vxo : rfma(a.hdt, axo + axn, vxo);
        a.vy[gid] = (fl & 2) ? vyo : rfma(a.hdt, ayo + ayn, vyo);
    }
    a.ax[gid] = axn; a.ay[gid] = ayn;
}

// Fused element pass for one element: returns the 3 nodal forces, updates / emits history.
template <typename R, int SPLIT>
__device__ __forceinline__ void element_forces(const MatC<R>& mat, R b1, R c1, R b2, R c2, R A, R u1x, R u1y, R u2x,
                                               R u2y, R u3x, R u3y, R dsum, R& psi_p, R f[6])
{
    // strain (L69): grad phi3 = -(grad phi1 + grad phi2)  =>  eps from differences to node 3
    const R ax = u1x - u3x, bx = u2x - u3x, ay = u1y - u3y, by = u2y - u3y;
    const R exx = b1 * ax + b2 * bx;
    const R eyy = c1 * ay + c2 * by;
    const R exy = R(0.5) * (c1 * ax + c2 * bx + b1 * ay + b2 * by);
    const R de = dsum * R(1.0 / 3.0);  // centroid damage (R3)
    const R g = (R(1) - de) * (R(1) - de) + mat.eta;
    R psi_m, sxx, syy, sxy;
    elem_response<R, SPLIT>(mat, exx, eyy, exy, g, psi_p, psi_m, sxx, syy, sxy);
    // f_i = A sigma . grad phi_i (L124)
    f[0] = A * (sxx * b1 + sxy * c1); f[1] = A * (sxy * b1 + syy * c1);
    f[2] = A * (sxx * b2 + sxy * c2); f[3] = A * (sxy * b2 + syy * c2);
    f[4] = -(f[0] + f[2]); f[5] = -(f[1] + f[3]);
}

// Indexed gather of one halo node's kinematic state into the halo slots of a stage, as asynchronous copies
// (LDGSTS): nothing is held in registers while the data is in flight.  The flag byte travels in its 32-bit word.
template <typename R, int MODE>
__device__ __forceinline__ void step_halo_gather(const StepArgs<R>& a, const StageLayout& L, unsigned char* stg, int slot, int j,
                                                 int gid)
{
    constexpr int B = sizeof(R);
    reinterpret_cast<int*>(stg + L.hids)[j] = gid;
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[0]) + slot, a.ux + gid);
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[1]) + slot, a.uy + gid);
    cp_async<B>(reinterpret_cast<R*>(stg + L.node[2]) + slot, a.d + gid);
    if (MODE == MODE_STEP) {
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[3]) + slot, a.vx + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[4]) + slot, a.vy + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[5]) + slot, a.ax + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[6]) + slot, a.ay + gid);
        cp_async<4>(reinterpret_cast<int*>(stg + L.hflag) + j, a.flags + (gid & ~3));
    }
    if (MODE == MODE_TANGENT) {  // the trial direction travels in the velocity slots
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[3]) + slot, a.px + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[4]) + slot, a.py + gid);
    }
    if (MODE == MODE_EQ) {  // old p, r, old q, 1/D: the prologue of a halo node is recomputed by every chunk that touches it
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[3]) + slot, a.cpx + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[4]) + slot, a.cpy + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[5]) + slot, a.rx + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[6]) + slot, a.ry + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[7]) + slot, a.fx_out + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[8]) + slot, a.fy_out + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[9]) + slot, a.dix + gid);
        cp_async<B>(reinterpret_cast<R*>(stg + L.node[10]) + slot, a.diy + gid);
    }
}

// Scalar step of the quasi-static CG, run by one thread of the last CTA of a MODE_EQ launch after the fixed-order sums
// t[] = p.q, r.z, r.r (residual BEFORE the coming step), z.q, q.Dinv.q, r.q, q.q.  Same predicted-beta recurrence as the
// damage CG (pff_damage.cu): r.z and r.r after the step follow from the sums of this pass, so the next pass can form
// p = z + beta p in its prologue.  Stops on ||r|| <= tol ||r0||, on the iteration cap, or on a breakdown p.Kp <= 0 (the
// shifted difference of a non-isotropic split need not be positive definite): then no step is applied along p.
__device__ __forceinline__ void eq_scalar_step(DamageCtrl* c, const double* t)
{
    const double pq = t[0], rz = t[1], rr = t[2];
    if (c->first) { c->nb = sqrt(rr); c->first = 0; }
    c->pending = 0;
    c->relres = c->nb > 0.0 ? sqrt(rr) / c->nb : 0.0;
    const double lim = c->tol * c->nb;
    if (sqrt(rr) <= lim) { c->done = 1; c->status = PFF_OK; return; }
    if (c->iters >= c->max_iter) { c->done = 1; c->status = PFF_ENOCONV; return; }
    if (!(pq > 0.0) || !isfinite(pq)) { c->done = 1; c->status = PFF_ENOCONV; c->restart = 1; return; }  // restart = breakdown flag
    c->iters += 1;
    const double alpha = rz / pq;
    const double rz_pred = fmax(rz - 2.0 * alpha * t[3] + alpha * alpha * t[4], 0.0);
    const double rr_pred = rr - 2.0 * alpha * t[5] + alpha * alpha * t[6];
    c->alpha = alpha; c->rz = rz;
    c->beta = rz > 0.0 ? rz_pred / rz : 0.0;
    c->pending = 1;  // du += alpha p is applied by the next pass (or by the finish kernel)
    const double err = 64.0 * 2.220446049250313e-16 * (rr + 2.0 * alpha * fabs(t[5]) + alpha * alpha * t[6]);
    if (rr_pred + err <= lim * lim) { c->done = 1; c->status = PFF_OK; c->relres = sqrt(fmax(rr_pred, 0.0)) / c->nb; }
}

// PERSISTENT, double-buffered explicit-step kernel: gridDim.x CTAs, CTA b owns chunks b, b + G, b + 2G, ...
// While chunk k is computed, the bulk copies (TMA) of chunk k + 1 stream into the other stage and its halo
// gathers (cp.async) land in that stage's halo slots; one mbarrier per stage counts the TMA arrival and every
// thread's cp.async arrival.  Per chunk: predictor (Eq. 16) -> fused element pass (strain, split, degradation,
// stress, force, history) -> ordered gather + Eq. 17-18.  Stage = StageLayout kind 0 (pff_internal.h).
template <typename R, int SPLIT, int MODE>
__global__ void __launch_bounds__(kStepTPB, 2) step_chunk_kernel(const StepArgs<R> a)
{
    extern __shared__ __align__(128) unsigned char smem[];
    typedef typename Geo<R>::Pair Pair;
    constexpr int A = 16 / sizeof(R);
    const StageLayout& L = a.lay;
    unsigned char* s_shared_slots = smem + L.slot_base;
    ChunkMeta* s_meta = reinterpret_cast<ChunkMeta*>(smem + L.meta);
    uint64_t* bar = reinterpret_cast<uint64_t*>(smem + L.bar);
    const int tid = threadIdx.x, lane = tid & 31, G = gridDim.x, EC = a.EC;
    const int n_my = (a.C - (int)blockIdx.x + G - 1) / G;  // chunks this CTA owns
    // the LAST warp issues the bulk copies (one lane per array); the halo gathers are issued from the top thread down
    // the LAST warp is the producer (bulk copies + all halo gathers of the next chunk); the other kWorkers threads run the
    // predictor and the element pass and synchronise between them on a named barrier; the producer rejoins for the gather
    constexpr int kWorkers = kStepTPB - 32;
    const bool issuer = tid >= kWorkers;
    const bool have_desc = issuer && lane < a.plan.n;
    StageDesc my_desc{};
    if (have_desc) my_desc = a.plan.d[lane];

    if (tid == 0) {
        mbar_init(bar, 1 + kStepTPB); mbar_init(bar + 2, 1 + kStepTPB);
        *Geo<R>::slot(smem, s_shared_slots, 3 * EC, EC) = Geo<R>::pair(R(0), R(0));  // the zero pair (lives in the shared region)
    }
    int it = 0;  // stage uses so far: stage = it & 1, mbarrier parity = (it >> 1) & 1
    constexpr bool SU = MODE == MODE_STEPSU;
    constexpr bool STEP = MODE == MODE_STEP || SU;  // the explicit step proper
    constexpr int HALO_MODE = SU ? (int)MODE_STEP : MODE;
    [[maybe_unused]] const bool tr_on = STEP;
    int tr_k = 0;
    PFF_TR(a.trace, tr_on, 0);
    unsigned int gb_epoch = 0;  // thread 0: the barrier counter's value before this launch (read early, used at the barrier)
    if (tid == 0 && a.N_sh > 0) gb_epoch = *reinterpret_cast<volatile unsigned int*>(a.gbar + 1);
    // MODE_EQ: the recurrence scalars of this iteration (written by the previous launch, or by the host for the first one)
    // and this thread's share of the seven sums p.q, r.z, r.r, z.q, q.Dinv.q, r.q, q.q (channels of cg scalar step)
    __shared__ DamageCtrl s_eq;
    __shared__ double s_w[(MODE == MODE_EQ || SU) ? kCh * kRedWarps : 1], s_out[kCh];
    double acc[kCh];
    R eq_alpha = R(0), eq_beta = R(0);
    bool eq_first = true;
    if (MODE == MODE_EQ) {
        if (tid == 0) s_eq = *a.eq_ctrl;
        __syncthreads();
        if (s_eq.done) return;  // converged (or broke down) in an earlier launch of this batch: nothing to do
        eq_alpha = R(s_eq.alpha); eq_beta = R(s_eq.beta); eq_first = s_eq.first != 0;
#pragma unroll
        for (int c = 0; c < kCh; ++c) acc[c] = 0.0;
    }
    if (SU) {
#pragma unroll
        for (int c = 0; c < kCh; ++c) acc[c] = 0.0;
        // the CG kernel that follows in stream order counts its grid barriers from zero (as dmg_setup_chunk does)
        if (blockIdx.x == 0 && tid == 0) a.su.ticket[1] = 0u;
    }
    for (int e0 = 0; e0 < n_my; e0 += kMetaCap) {
        const int n_ep = min(kMetaCap, n_my - e0);
        __syncthreads();  // previous epoch fully consumed (also publishes the mbarrier init)
        if (tid < n_ep) s_meta[tid] = a.meta[blockIdx.x + (e0 + tid) * G];
        __syncthreads();
        {   // epoch prologue: chunk 0 of the epoch is loaded with exposed latency (once per kMetaCap chunks)
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
                    step_halo_gather<R, HALO_MODE>(a, L, stg, hb0 + j, j, __ldg(a.halo_ids + cm.halo_off + j));
            }
            cp_async_mbar_arrive(bar + 2 * (it & 1));
        }
        for (int k = 0; k < n_ep; ++k, ++it) {
            const int st = it & 1;
            unsigned char* stg = smem + st * L.stage_bytes;
            const ushort4* s_lconn = reinterpret_cast<const ushort4*>(stg + L.lconn);
            unsigned char* s_geo = stg + L.geo;
            const R* s_area = reinterpret_cast<const R*>(stg + L.area);
            const R* s_H = reinterpret_cast<const R*>(stg + L.H);
            R* s_ux = reinterpret_cast<R*>(stg + L.node[0]);
            R* s_uy = reinterpret_cast<R*>(stg + L.node[1]);
            const R* s_d = reinterpret_cast<const R*>(stg + L.node[2]);
            const R* s_vx = reinterpret_cast<const R*>(stg + L.node[3]);
            const R* s_vy = reinterpret_cast<const R*>(stg + L.node[4]);
            const R* s_ax = reinterpret_cast<const R*>(stg + L.node[5]);
            const R* s_ay = reinterpret_cast<const R*>(stg + L.node[6]);
            const R* s_fex = reinterpret_cast<const R*>(stg + L.node[7]);
            const R* s_fey = reinterpret_cast<const R*>(stg + L.node[8]);
            const R* s_minv = reinterpret_cast<const R*>(stg + L.node[9]);
            // MODE_EQ (layout kind 3): [3],[4] = p, [5],[6] = r, [7],[8] = old q, [9],[10] = 1/D, [11],[12] = du
            R* s_px = reinterpret_cast<R*>(stg + L.node[3]);
            R* s_py = reinterpret_cast<R*>(stg + L.node[4]);
            R* s_rx = reinterpret_cast<R*>(stg + L.node[5]);
            R* s_ry = reinterpret_cast<R*>(stg + L.node[6]);
            const R* s_qx = reinterpret_cast<const R*>(stg + L.node[7]);
            const R* s_qy = reinterpret_cast<const R*>(stg + L.node[8]);
            const R* s_dix = reinterpret_cast<const R*>(stg + L.node[9]);
            const R* s_diy = reinterpret_cast<const R*>(stg + L.node[MODE == MODE_EQ ? 10 : 9]);
            const R* s_ex = reinterpret_cast<const R*>(stg + L.node[MODE == MODE_EQ ? 11 : 9]);
            const R* s_ey = reinterpret_cast<const R*>(stg + L.node[MODE == MODE_EQ ? 12 : 9]);
            const uint8_t* s_flags = stg + L.flags;
            const uint16_t* s_ell = reinterpret_cast<const uint16_t*>(stg + L.ell);
            const ChunkMeta cm = s_meta[k];
            const int nloc = cm.n_int + cm.n_halo;
            const int shift = cm.node_start & (A - 1), hb = (shift + cm.n_int + A - 1) & ~(A - 1), fshift = cm.node_start & 15;
            const int* s_hdst = reinterpret_cast<const int*>(stg + L.hdst) + (cm.halo_off & 3);

            // ---- prefetch chunk k + 1 into the other stage, bulk copies FIRST: they do not depend on this chunk's data, so
            // two stages are in flight whenever the CTA is waiting for memory (the other stage was freed by the barrier that
            // ended the previous chunk)
            if (k + 1 < n_ep && issuer) {
                const ChunkMeta cn = s_meta[k + 1];
                const ChunkRange cr{cn.elem_start, cn.n_elem, a.Ne, cn.node_start, cn.n_int, a.N, cn.ell_off,
                                    cn.ell_w * (cn.n_int + cn.n_halo), (int)a.ell_total, cn.halo_off, cn.n_halo, (int)a.n_entries,
                                    k + 2 < n_ep ? s_meta[k + 2].halo_off : 0, k + 2 < n_ep ? s_meta[k + 2].n_halo : 0};
                fence_proxy_async();
                stage_issue_desc(my_desc, have_desc, smem + (st ^ 1) * L.stage_bytes, bar + 2 * (st ^ 1), lane, cr);
            }
            // bulk copies AND every thread's halo gathers of this chunk (all issued one iteration ago)
            mbar_wait(bar + 2 * st, (it >> 1) & 1);
            PFF_TR(a.trace, tr_on && tr_k < 24, 1 + 4 * tr_k);
            // ---- halo gathers of chunk k + 1 (its halo ids arrived with THIS stage)
            if (k + 1 < n_ep) {
                const ChunkMeta cn = s_meta[k + 1];
                unsigned char* stn = smem + (st ^ 1) * L.stage_bytes;
                if (issuer) {
                    const int hbn = ((cn.node_start & (A - 1)) + cn.n_int + A - 1) & ~(A - 1);
                    const int* ids = reinterpret_cast<const int*>(stg + L.hnext) + (cn.halo_off & 3);
                    for (int j = lane; j < cn.n_halo; j += 32) step_halo_gather<R, HALO_MODE>(a, L, stn, hbn + j, j, ids[j]);
                }
                cp_async_mbar_arrive(bar + 2 * (st ^ 1));
            }
            // ---- phase 1: predictor (Eq. 16) in place, halo nodes by the middle warps, interior by the low warps;
            // Dirichlet dofs hold u_bar already (dirichlet_kernel)
            if (STEP && !issuer) {
                for (int j = (tid + kWorkers / 2) % kWorkers; j < cm.n_halo; j += kWorkers) {
                    const int s = hb + j, gid = reinterpret_cast<const int*>(stg + L.hids)[j];
                    const unsigned fl = reinterpret_cast<const unsigned*>(stg + L.hflag)[j] >> (8 * (gid & 3));
                    const R ux = s_ux[s], uy = s_uy[s];
                    const R px = rfma(a.hdt2, s_ax[s], rfma(a.dt, s_vx[s], ux));
                    const R py = rfma(a.hdt2, s_ay[s], rfma(a.dt, s_vy[s], uy));
                    s_ux[s] = (fl & 1) ? ux : px;
                    s_uy[s] = (fl & 2) ? uy : py;
                }
                for (int i = tid; i < cm.n_int; i += kWorkers) {
                    const int s = shift + i;
                    const uint8_t fl = s_flags[fshift + i];
                    const R ux = s_ux[s], uy = s_uy[s];
                    const R px = rfma(a.hdt2, s_ax[s], rfma(a.dt, s_vx[s], ux));
                    const R py = rfma(a.hdt2, s_ay[s], rfma(a.dt, s_vy[s], uy));
                    s_ux[s] = (fl & 1) ? ux : px;
                    s_uy[s] = (fl & 2) ? uy : py;
                }
            }
            // ---- MODE_EQ phase 1: CG node prologue for every local node (halo nodes redundantly, from gathered values):
            // apply the previous step, form the new direction in the p slots; interior nodes are written back
            if (MODE == MODE_EQ && !issuer) {
                for (int i = tid; i < nloc; i += kWorkers) {
                    const bool interior = i < cm.n_int;
                    const int s = interior ? shift + i : hb + (i - cm.n_int);
                    const R dx = s_dix[s], dy = s_diy[s];  // 0 on constrained dofs: r, p stay 0 there
                    R rx = s_rx[s], ry = s_ry[s], px = s_px[s], py = s_py[s];
                    if (!eq_first) {
                        rx = dx != R(0) ? rfma(-eq_alpha, s_qx[s], rx) : R(0);
                        ry = dy != R(0) ? rfma(-eq_alpha, s_qy[s], ry) : R(0);
                        if (interior) {
                            const int gid = cm.node_start + i;
                            a.ex[gid] = rfma(eq_alpha, px, s_ex[s]); a.ey[gid] = rfma(eq_alpha, py, s_ey[s]);
                            a.rx[gid] = rx; a.ry[gid] = ry;
                        }
                    }
                    const R zx = dx * rx, zy = dy * ry;
                    px = eq_first ? zx : rfma(eq_beta, px, zx);
                    py = eq_first ? zy : rfma(eq_beta, py, zy);
                    s_px[s] = px; s_py[s] = py; s_rx[s] = rx; s_ry[s] = ry;
                    if (interior) {
                        const int gid = cm.node_start + i;
                        a.cpx[gid] = px; a.cpy[gid] = py;
                        acc[1] += double(rx) * double(zx) + double(ry) * double(zy);
                        acc[2] += double(rx) * double(rx) + double(ry) * double(ry);
                    }
                }
            }
            if (!issuer) asm volatile("bar.sync 1, %0;" ::"n"(kWorkers) : "memory");  // workers only
            PFF_TR(a.trace, tr_on && tr_k < 24, 2 + 4 * tr_k);

            // ---- phase 2: fused element pass (workers); nodal force pairs go to the slots corner * EC + e
            for (int e = tid; e < (issuer ? 0 : cm.n_elem); e += kWorkers) {
                const ushort4 c = s_lconn[e];
                R b1, c1, b2, c2;
                Geo<R>::load_smem(s_geo, e, EC, b1, c1, b2, c2);
                R psi_p, f[6];
                element_forces<R, SPLIT>(a.mat, b1, c1, b2, c2, s_area[e], s_ux[c.x], s_uy[c.x], s_ux[c.y], s_uy[c.y], s_ux[c.z],
                                         s_uy[c.z], s_d[c.x] + s_d[c.y] + s_d[c.z], psi_p, f);
                if (MODE == MODE_TANGENT || MODE == MODE_EQ) {  // Eq. 13: f_int(u + p) - f_int(u), element by element (s_vx, s_vy hold p)
                    R f1[6], pp1;
                    element_forces<R, SPLIT>(a.mat, b1, c1, b2, c2, s_area[e], s_ux[c.x] + s_vx[c.x], s_uy[c.x] + s_vy[c.x],
                                             s_ux[c.y] + s_vx[c.y], s_uy[c.y] + s_vy[c.y], s_ux[c.z] + s_vx[c.z],
                                             s_uy[c.z] + s_vy[c.z], s_d[c.x] + s_d[c.y] + s_d[c.z], pp1, f1);
#pragma unroll
                    for (int k = 0; k < 6; ++k) f[k] = f1[k] - f[k];
                }
                *Geo<R>::slot(s_geo, s_shared_slots, e, EC) = Geo<R>::pair(f[0], f[1]);
                *Geo<R>::slot(s_geo, s_shared_slots, EC + e, EC) = Geo<R>::pair(f[2], f[3]);
                *Geo<R>::slot(s_geo, s_shared_slots, 2 * EC + e, EC) = Geo<R>::pair(f[4], f[5]);
                if (STEP) {
                    const R Hold = s_H[e];
                    if (psi_p > Hold) a.H[cm.elem_start + e] = psi_p;  // H <- max(H, psi+)  (L98, L114)
                    if (SU) {  // damage setup for this element with the NEW history value (dmg_setup_chunk's element pass)
                        const R He = psi_p > Hold ? psi_p : Hold, Ar = s_area[e];
                        R q1, q2, q3, cm_, w12, w13, w23;
                        elem_damage_apply<R>(a.mat, b1, c1, b2, c2, Ar, He, s_d[c.x], s_d[c.y], s_d[c.z], q1, q2, q3);
                        elem_coefficients<R>(a.mat, b1, c1, b2, c2, Ar, He, cm_, w12, w13, w23);
                        Geo<R>::store_global(a.su.ca, a.su.cb, cm.elem_start + e, cm_, w12, w13, w23);
                        const R ce = a.mat.c0 + R(2) * He, se = R(2) * He - a.mat.s0;
                        const R m12 = ce * Ar * R(1.0 / 12.0), kA = a.mat.kappa * Ar;
                        const R b3 = -(b1 + b2), c3 = -(c1 + c2);
                        // (q, D) of corners 1, 2 go to the hold region; corner 3's and the element's share of the right-hand
                        // side replace what only this thread needed from the stage: H, the connectivity word, the area
                        Pair* hold = reinterpret_cast<Pair*>(smem + L.hold);
                        hold[e] = Geo<R>::pair(q1, R(2) * m12 + kA * (b1 * b1 + c1 * c1));
                        hold[EC + e] = Geo<R>::pair(q2, R(2) * m12 + kA * (b2 * b2 + c2 * c2));
                        const R D3 = R(2) * m12 + kA * (b3 * b3 + c3 * c3);
                        if (sizeof(R) == 8) { const_cast<R*>(s_H)[e] = q3; reinterpret_cast<R*>(stg + L.lconn)[e] = D3; }
                        else hold[2 * EC + e] = Geo<R>::pair(q3, D3);  // fp32: the hold region has room for all three corners
                        const_cast<R*>(s_area)[e] = se * Ar * R(1.0 / 3.0);
                    }
                } else if (MODE == MODE_FORCE) {
                    if (a.psi_out) a.psi_out[cm.elem_start + e] = psi_p;
                }
            }
            __syncthreads();
            PFF_TR(a.trace, tr_on && tr_k < 24, 3 + 4 * tr_k);

            // ---- phase 3: ordered gather of each node's incident force pairs, then Eq. 17-18 for interior nodes
            for (int i = tid; i < nloc; i += kStepTPB) {
                R fx = R(0), fy = R(0);
                [[maybe_unused]] R qs = R(0), Ds = R(0), bs = R(0);  // MODE_STEPSU: A d_n, diagonal, right-hand side of this node
                const uint16_t* row = s_ell + i;
#pragma unroll 4
                for (int w = 0; w < cm.ell_w; ++w) {
                    const int idx = row[w * nloc];
                    const Pair v = *Geo<R>::slot(s_geo, s_shared_slots, idx, EC);
                    fx += v.x; fy += v.y;
                    if (SU && idx < 3 * EC) {  // same order of sums as dmg_setup_chunk (padding entries add nothing there either)
                        const int kc = (idx >= EC) + (idx >= 2 * EC), e = idx - kc * EC;
                        Pair h;
                        if (kc < 2 || sizeof(R) == 4) h = reinterpret_cast<const Pair*>(smem + L.hold)[idx];
                        else h = Geo<R>::pair(s_H[e], reinterpret_cast<const R*>(stg + L.lconn)[e]);
                        qs += h.x; Ds += h.y; bs += s_area[e];
                    }
                }
                if (i < cm.n_int) {
                    const int gid = cm.node_start + i, s = shift + i;
                    if (MODE == MODE_EQ) {  // q = K p of an interior node and its share of the sums (free dofs: 1/D != 0)
                        const double qx = double(fx), qy = double(fy), dx = double(s_dix[s]), dy = double(s_diy[s]);
                        const double rx = double(s_rx[s]), ry = double(s_ry[s]);
                        acc[0] += double(s_px[s]) * qx + double(s_py[s]) * qy;
                        acc[3] += dx * rx * qx + dy * ry * qy; acc[4] += dx * qx * qx + dy * qy * qy;
                        acc[5] += rx * qx + ry * qy;
                        acc[6] += (dx != 0.0 ? qx * qx : 0.0) + (dy != 0.0 ? qy * qy : 0.0);
                    }
                    if (MODE == MODE_FORCE || MODE == MODE_TANGENT || MODE == MODE_EQ) { a.fx_out[gid] = fx; a.fy_out[gid] = fy; continue; }
                    const uint8_t fl = s_flags[fshift + i];
                    const R minv = s_minv[s];
                    R axn = (a.S * s_fex[s] - fx) * minv;
                    R ayn = (a.S * s_fey[s] - fy) * minv;
                    if (fl & 1) axn = R(0);
                    if (fl & 2) ayn = R(0);
                    if (STEP) {
                        const R vxo = s_vx[s], vyo = s_vy[s];
                        a.ux[gid] = s_ux[s]; a.uy[gid] = s_uy[s];
                        a.vx[gid] = (fl & 1) ? vxo : rfma(a.hdt, s_ax[s] + axn, vxo);
                        a.vy[gid] = (fl & 2) ? vyo : rfma(a.hdt, s_ay[s] + ayn, vyo);
                    }
                    a.ax[gid] = axn; a.ay[gid] = ayn;
                    if (SU) {  // dmg_setup_chunk's node epilogue
                        const bool fixed = (fl & 4) != 0;
                        const R r = bs - qs;
                        reinterpret_cast<R*>(a.su.r)[gid] = r;
                        reinterpret_cast<R*>(a.su.dinv)[gid] = (a.su.zero_dinv_fixed && fixed) ? R(0) : R(1) / Ds;
                        reinterpret_cast<R*>(a.su.lb)[gid] = s_d[s];
                        a.su.mask[gid] = fixed ? 2 : 1;
                        acc[0] += double(bs) * double(bs);
                        if (!fixed) acc[1] += double(r) * double(r);
                        if (!fixed && (a.mat.model != PFF_AT1 || r > R(0))) acc[2] += double(r) * double(r);
                    }
                } else {
                    const int slot = s_hdst[i - cm.n_int];
                    a.halo_part[slot] = fx;
                    a.halo_part[a.n_slots + slot] = fy;
                    if (SU) {
                        R* sp = reinterpret_cast<R*>(a.su.part3);
                        sp[slot] = qs; sp[a.n_slots + slot] = Ds; sp[2 * a.n_slots + slot] = bs;
                    }
                }
            }
            __syncthreads();  // stage st and the slots are free again
            PFF_TR(a.trace, tr_on && tr_k < 24, 4 + 4 * tr_k);
            ++tr_k;
        }
    }
    PFF_TR(a.trace, tr_on, 100);
    // ---- interface nodes (owned by no chunk), after a grid-wide barrier: ordered sum of the per-chunk partials, then the
    // same Eq. 16-18.  Every read of the OLD interface state by the chunk phase (halo gathers) precedes the barrier.
    if (a.N_sh > 0) {
        unsigned int target = gb_epoch;
        grid_barrier(a.gbar, target, (unsigned)G);
        PFF_TR(a.trace, tr_on, 101);
        // every CTA has read the epoch before arriving, and all have arrived: publish the next launch's epoch
        if (blockIdx.x == 0 && tid == 0) a.gbar[1] = target;
        // Equal slice per CTA, TWO nodes per thread and trip: all loads of both nodes are issued before anything is computed
        // or stored, so a trip costs one memory round trip (the slice is ~1.7 nodes per thread at 10^6 nodes).
        struct IfNode { R fx, fy, ux, uy, vx, vy, ax, ay, fex, fey, minv, px, py, rx, ry, qx, qy, dx, dy, ex, ey, sq, sD, sb, sd; uint8_t fl; };
        auto if_load = [&](int s, IfNode& v) {
            const int gid = a.N_int + s;
            v.fx = iface_sum<R>(a.halo_part, s, a.N_sh, a.n_ovf, a.sh_rowptr);
            v.fy = iface_sum<R>(a.halo_part + a.n_slots, s, a.N_sh, a.n_ovf, a.sh_rowptr);
            if (MODE == MODE_EQ) {  // CG state of an interface node (u is not needed: the element pass is over)
                v.px = a.cpx[gid]; v.py = a.cpy[gid]; v.rx = a.rx[gid]; v.ry = a.ry[gid];
                v.dx = a.dix[gid]; v.dy = a.diy[gid];
                if (!eq_first) { v.qx = a.fx_out[gid]; v.qy = a.fy_out[gid]; v.ex = a.ex[gid]; v.ey = a.ey[gid]; }
                return;
            }
            v.ux = a.ux[gid]; v.uy = a.uy[gid];
            if (STEP) { v.vx = a.vx[gid]; v.vy = a.vy[gid]; v.ax = a.ax[gid]; v.ay = a.ay[gid]; }
            if (STEP || MODE == MODE_INIT) { v.fl = a.flags[gid]; v.minv = a.minv[gid]; v.fex = a.fex[gid]; v.fey = a.fey[gid]; }
            if (SU) {  // the three partial planes of the fused damage setup and d_n
                const R* sp = reinterpret_cast<const R*>(a.su.part3);
                v.sq = iface_sum<R>(sp, s, a.N_sh, a.n_ovf, a.sh_rowptr);
                v.sD = iface_sum<R>(sp + a.n_slots, s, a.N_sh, a.n_ovf, a.sh_rowptr);
                v.sb = iface_sum<R>(sp + 2 * a.n_slots, s, a.N_sh, a.n_ovf, a.sh_rowptr);
                v.sd = a.d[gid];
            }
            if (MODE == MODE_TANGENT) { v.px = a.px[gid]; v.py = a.py[gid]; }
        };
        auto if_finish = [&](int s, const IfNode& v) {  // the same Eq. 16-18 as predict() + finish_node(), from the loaded values
            const int gid = a.N_int + s;
            if (MODE == MODE_EQ) {  // the same prologue as in the chunk phase, then q = K p from the ordered partials
                R rx = v.rx, ry = v.ry, px = v.px, py = v.py;
                if (!eq_first) {
                    rx = v.dx != R(0) ? rfma(-eq_alpha, v.qx, rx) : R(0);
                    ry = v.dy != R(0) ? rfma(-eq_alpha, v.qy, ry) : R(0);
                    a.ex[gid] = rfma(eq_alpha, px, v.ex); a.ey[gid] = rfma(eq_alpha, py, v.ey);
                    a.rx[gid] = rx; a.ry[gid] = ry;
                }
                const R zx = v.dx * rx, zy = v.dy * ry;
                px = eq_first ? zx : rfma(eq_beta, px, zx);
                py = eq_first ? zy : rfma(eq_beta, py, zy);
                a.cpx[gid] = px; a.cpy[gid] = py; a.fx_out[gid] = v.fx; a.fy_out[gid] = v.fy;
                const double qx = double(v.fx), qy = double(v.fy), dx = double(v.dx), dy = double(v.dy);
                acc[0] += double(px) * qx + double(py) * qy;
                acc[1] += double(rx) * double(zx) + double(ry) * double(zy);
                acc[2] += double(rx) * double(rx) + double(ry) * double(ry);
                acc[3] += dx * double(rx) * qx + dy * double(ry) * qy; acc[4] += dx * qx * qx + dy * qy * qy;
                acc[5] += double(rx) * qx + double(ry) * qy;
                acc[6] += (dx != 0.0 ? qx * qx : 0.0) + (dy != 0.0 ? qy * qy : 0.0);
                return;
            }
            if (MODE == MODE_FORCE || MODE == MODE_TANGENT) { a.fx_out[gid] = v.fx; a.fy_out[gid] = v.fy; return; }
            R axn = (a.S * v.fex - v.fx) * v.minv;
            R ayn = (a.S * v.fey - v.fy) * v.minv;
            if (v.fl & 1) axn = R(0);
            if (v.fl & 2) ayn = R(0);
            if (STEP) {
                const R px = rfma(a.hdt2, v.ax, rfma(a.dt, v.vx, v.ux));
                const R py = rfma(a.hdt2, v.ay, rfma(a.dt, v.vy, v.uy));
                a.ux[gid] = (v.fl & 1) ? v.ux : px; a.uy[gid] = (v.fl & 2) ? v.uy : py;
                a.vx[gid] = (v.fl & 1) ? v.vx : rfma(a.hdt, v.ax + axn, v.vx);
                a.vy[gid] = (v.fl & 2) ? v.vy : rfma(a.hdt, v.ay + ayn, v.vy);
            }
            a.ax[gid] = axn; a.ay[gid] = ayn;
            if (SU) {  // dmg_setup_chunk's interface epilogue
                const bool fixed = (v.fl & 4) != 0;
                const R r = v.sb - v.sq;
                reinterpret_cast<R*>(a.su.r)[gid] = r;
                reinterpret_cast<R*>(a.su.dinv)[gid] = (a.su.zero_dinv_fixed && fixed) ? R(0) : R(1) / v.sD;
                reinterpret_cast<R*>(a.su.lb)[gid] = v.sd;
                a.su.mask[gid] = fixed ? 2 : 1;
                acc[0] += double(v.sb) * double(v.sb);
                if (!fixed) acc[1] += double(r) * double(r);
                if (!fixed && (a.mat.model != PFF_AT1 || r > R(0))) acc[2] += double(r) * double(r);
            }
        };
        const int per = (a.N_sh + G - 1) / G, end = min(a.N_sh, ((int)blockIdx.x + 1) * per);
        for (int s0 = blockIdx.x * per + tid; s0 < end; s0 += 2 * kStepTPB) {
            const int s1 = s0 + kStepTPB;
            const bool two = s1 < end;
            IfNode n0, n1;
            if_load(s0, n0);
            if (two) if_load(s1, n1);
            if_finish(s0, n0);
            if (two) if_finish(s1, n1);
        }
    }
    PFF_TR(a.trace, tr_on, 102);
    if (SU) {
        // ---- norms of the fused damage setup and the control block of the solve (dmg_setup_chunk's tail): one block
        // reduction per CTA, the last CTA to arrive sums the block partials in a fixed order
        __syncthreads();
        block_reduce_ch(acc, s_w, s_out);
        if (tid < kCh) a.su.part[(int64_t)tid * a.su.part_n + blockIdx.x] = s_out[tid];
        if (last_block(a.su.ticket)) {
            const int w = tid >> 5;
            if (w < 3) {
                double v = 0.0;
                for (int i = lane; i < G; i += 32) v += __ldcg(a.su.part + (int64_t)w * a.su.part_n + i);
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) s_out[w] = v;
            }
            __syncthreads();
            if (tid == 0) {
                DamageCtrl c{};
                c.tol = a.su.tol; c.max_iter = a.su.max_iter; c.first = 1; c.restart = 1; c.status = PFF_ENOCONV;
                c.nb = fmax(fmax(sqrt(s_out[0]), sqrt(s_out[1])), 1e-300);
                if (sqrt(s_out[2]) <= c.tol * c.nb) { c.done = 1; c.status = PFF_OK; c.relres = sqrt(s_out[2]) / c.nb; }
                *a.su.ctrl = c;
            }
        }
    }
    if (MODE == MODE_EQ) {
        // ---- one ordered block reduction per CTA; the LAST CTA to finish sums the block partials in index order and
        // advances the recurrence scalars for the next launch (alpha, predicted beta, convergence: eq_scalar_step)
        acc[kCh - 1] = INFINITY;
        __syncthreads();
        block_reduce_ch(acc, s_w, s_out);
        if (tid < kCh) a.eq_part[(size_t)tid * G + blockIdx.x] = s_out[tid];
        if (last_block(a.eq_ticket)) {
            const int w = tid >> 5;
            if (w < kCh - 1) {
                double v = 0.0;
                for (int i = lane; i < G; i += 32) v += __ldcg(a.eq_part + (size_t)w * G + i);
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) s_out[w] = v;
            }
            __syncthreads();
            if (tid == 0) {
                eq_scalar_step(&s_eq, s_out);
                *a.eq_ctrl = s_eq;
            }
        }
    }
}

// ---- atomic variant: warp-aggregated floating-point atomics -------------------------------------------
// Lanes of a warp that target the same node (frequent after the Morton element order) are matched with
// __match_any_sync, their contributions summed in lane order through shuffles, and ONE atomicAdd per distinct node
// is issued by the lowest matching lane.  Order across warps is still arbitrary: not bit-reproducible.
__device__ __forceinline__ void red_add(double* p, double v) { atomicAdd(p, v); }
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }

template <typename R>
__device__ __forceinline__ void warp_aggregated_add(R* fx, R* fy, int node, R vx, R vy, unsigned active)
{
    const unsigned peers = __match_any_sync(active, node);
    R sx = R(0), sy = R(0);
    for (unsigned m = peers; m; m &= m - 1) {
        const int l = __ffs(m) - 1;
        sx += __shfl_sync(peers, vx, l);
        sy += __shfl_sync(peers, vy, l);
    }
    if ((int)(threadIdx.x & 31) == __ffs(peers) - 1) { red_add(fx + node, sx); red_add(fy + node, sy); }
}

template <typename R, int SPLIT, int MODE>
__global__ void __launch_bounds__(kTPB) elem_atomic_kernel(const StepArgs<R> a)
{
    const int e = blockIdx.x * kTPB + threadIdx.x;
    const bool live = e < a.Ne;
    const unsigned active = __ballot_sync(0xffffffffu, live);
    if (!live) return;
    const int4 c = __ldg(a.conn + e);
    R b1, c1, b2, c2;
    Geo<R>::load(a.ga, a.gb, e, b1, c1, b2, c2);
    const R A = __ldg(a.area + e);
    R u1x, u1y, u2x, u2y, u3x, u3y;
    predict<R, MODE>(a, c.x, u1x, u1y);
    predict<R, MODE>(a, c.y, u2x, u2y);
    predict<R, MODE>(a, c.z, u3x, u3y);
    R psi_p, f[6];
    element_forces<R, SPLIT>(a.mat, b1, c1, b2, c2, A, u1x, u1y, u2x, u2y, u3x, u3y, a.d[c.x] + a.d[c.y] + a.d[c.z],
                             psi_p, f);
    warp_aggregated_add<R>(a.fwx, a.fwy, c.x, f[0], f[1], active);
    warp_aggregated_add<R>(a.fwx, a.fwy, c.y, f[2], f[3], active);
    warp_aggregated_add<R>(a.fwx, a.fwy, c.z, f[4], f[5], active);
    if (MODE == MODE_STEP) {
        const R h = a.H[e];
        if (psi_p > h) a.H[e] = psi_p;
    } else if (MODE == MODE_FORCE) {
        if (a.psi_out) a.psi_out[e] = psi_p;
    }
}

template <typename R, int MODE>
__global__ void __launch_bounds__(kTPB) node_atomic_kernel(const StepArgs<R> a)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= a.N) return;
    R px, py;
    predict<R, MODE>(a, i, px, py);
    const R fx = a.fwx[i], fy = a.fwy[i];
    a.fwx[i] = R(0); a.fwy[i] = R(0);
    finish_node<R, MODE>(a, i, px, py, fx, fy);
}

template <typename R>
__global__ void dirichlet_kernel(int n, const int32_t* dof, const R* du, const R* dv, R* ux, R* uy, R* vx, R* vy)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const int node = dof[k] >> 1, comp = dof[k] & 1;
    if (comp == 0) { ux[node] = du[k]; vx[node] = dv[k]; }
    else { uy[node] = du[k]; vy[node] = dv[k]; }
}

template <typename R, int SPLIT, int MODE>
static pff_status launch_step_t(pff_mesh* m, const StepArgs<R>& a)
{
    const HostMesh& hm = m->hm;
    if (m->opt.scatter == PFF_SCATTER_ATOMIC) {
        if (m->only_kernel != 1) {
            PFF_LAUNCH(m, PFF_K_STEP_CHUNK, (elem_atomic_kernel<R, SPLIT, MODE><<<(unsigned)((hm.Ne + kTPB - 1) / kTPB), kTPB, 0, m->stream>>>(a)));
        }
        if (m->only_kernel != 0) {
            PFF_LAUNCH(m, PFF_K_STEP_SHARED, (node_atomic_kernel<R, MODE><<<(unsigned)((hm.N + kTPB - 1) / kTPB), kTPB, 0, m->stream>>>(a)));
        }
    } else {
        auto kern = step_chunk_kernel<R, SPLIT, MODE>;
        int grid = 0;  // persistent grid: every SM filled with as many CTAs as fit (cached per mesh, with the smem opt-in)
        const size_t smem = MODE == MODE_EQ ? m->lay_eq.total : (MODE == MODE_STEPSU ? m->lay_stepsu.total : m->lay_step.total);
        if (smem + 4096 > kSmemPerSM) { set_error("quasi-static CG: the chunk does not fit shared memory (use a smaller chunk_elems)"); return PFF_EUNSUPPORTED; }
        pff_status st = persistent_config(m, (const void*)kern, (int)smem, &grid, kStepTPB);
        if (st != PFF_OK) return st;
        {   // ONE cooperative launch: chunk phase, grid barrier, interface phase (all CTAs co-resident by construction)
            const unsigned g = (unsigned)std::min<int64_t>(grid, hm.C);
            StepArgs<R> b = a;
            b.gbar = m->d_step_bar;
            void* kargs[] = {(void*)&b};
            prof_mark(m, PFF_K_STEP_CHUNK);
            cudaError_t e = launch_cooperative((const void*)kern, g, kStepTPB, kargs, smem, m->stream);
            prof_mark(m, PFF_K_STEP_CHUNK);
            if (e != cudaSuccess) return cuda_check(e, "explicit step: cooperative launch");
            m->last_step_grid = (int)g;
            ++m->n_launches;
        }
    }
    return cuda_check(cudaGetLastError(), "explicit step launch");
}

template <typename R, int MODE>
static pff_status launch_step_s(pff_mesh* m, const StepArgs<R>& a)
{
    switch (m->mat.split) {
        case PFF_SPLIT_ISOTROPIC: return launch_step_t<R, PFF_SPLIT_ISOTROPIC, MODE>(m, a);
        case PFF_SPLIT_SPECTRAL: return launch_step_t<R, PFF_SPLIT_SPECTRAL, MODE>(m, a);
        case PFF_SPLIT_VOLDEV: return launch_step_t<R, PFF_SPLIT_VOLDEV, MODE>(m, a);
        case PFF_SPLIT_STARCONVEX: return launch_step_t<R, PFF_SPLIT_STARCONVEX, MODE>(m, a);
    }
    return PFF_EINVAL;
}

template <typename R>
static pff_status launch_step_r(pff_mesh* m, pff_state* s, const pff_bc* bc, double dt, int mode, void* fx, void* fy,
                                void* psi, const void* px, const void* py)
{
    const HostMesh& hm = m->hm;
    StepArgs<R> a{};
    a.meta = m->d_meta; a.lconn = (const ushort4*)m->d_lconn; a.conn = (const int4*)m->d_conn;
    a.ga = m->d_ga; a.gb = m->d_gb; a.area = (const R*)m->d_area;
    a.halo_ids = m->d_halo_ids; a.ell = m->d_ell; a.flags = m->d_flags; a.minv = (const R*)m->d_minv;
    a.halo_part = (R*)m->d_halo_part; a.n_slots = m->n_slots;
    a.EC = hm.chunk_elems; a.ell_total = m->ell_total; a.n_entries = m->n_entries; a.C = (int)hm.C; a.N = (int)hm.N; a.Ne = (int)hm.Ne;
    a.N_int = (int)hm.N_int; a.N_sh = (int)hm.N_sh;
    a.sh_rowptr = m->d_sh_rowptr; a.halo_dst = m->d_halo_dst; a.n_ovf = hm.n_ovf;
    a.ux = (R*)s->ux; a.uy = (R*)s->uy; a.vx = (R*)s->vx; a.vy = (R*)s->vy; a.ax = (R*)s->ax; a.ay = (R*)s->ay;
    a.d = (const R*)s->d; a.H = (R*)s->H; a.fex = (const R*)s->fext_x; a.fey = (const R*)s->fext_y;
    a.fx_out = (R*)fx; a.fy_out = (R*)fy; a.psi_out = (R*)psi;
    a.px = (const R*)px; a.py = (const R*)py;
    if (mode == MODE_EQ) {  // CG vectors and control of the quasi-static solve (pff_equilibrium.cu set them up)
        a.ex = (R*)m->eq.ex; a.ey = (R*)m->eq.ey; a.rx = (R*)m->eq.rx; a.ry = (R*)m->eq.ry;
        a.cpx = (R*)const_cast<void*>(px); a.cpy = (R*)const_cast<void*>(py);
        a.dix = (const R*)m->eq.dix; a.diy = (const R*)m->eq.diy;
        a.eq_ctrl = m->d_eq_ctrl; a.eq_part = m->d_eq_part; a.eq_ticket = m->d_eq_ticket;
    }
    a.fwx = (R*)m->d_fwx; a.fwy = (R*)m->d_fwy;
    if (mode == MODE_STEPSU) {  // outputs of the damage setup this launch performs as well (pff_damage.cu fills them in)
        pff_status fst = damage_fused_setup(m, &a.su);
        if (fst != PFF_OK) return fst;
    }
    a.dt = R(dt); a.hdt = R(0.5 * dt); a.hdt2 = R(0.5 * dt * dt);
    a.S = R(bc ? bc->load_scale : 1.0);
    a.mat = make_matc<R>(m->mat);
    a.trace = m->d_trace ? m->d_trace + kTraceStepOffset : nullptr;
    {   // TMA plan: one descriptor per contiguous array the chosen mode reads (kind 0 elements, 1 nodes, 2 gather table)
        const StageLayout& L = mode == MODE_EQ ? m->lay_eq : (mode == MODE_STEPSU ? m->lay_stepsu : m->lay_step);
        a.lay = L;
        StagePlan& P = a.plan;
        P.n = 0;
        const uint16_t lr = sizeof(R) == 8 ? 3 : 2;
        auto add = [&](const void* src, uint32_t off, uint16_t l, uint16_t kind) { P.d[P.n++] = StageDesc{src, off, l, kind}; };
        add(m->d_lconn, L.lconn, 3, 0);
        if (sizeof(R) == 8) { add(m->d_ga, L.geo, 4, 0); add(m->d_gb, L.geo + 16u * (uint32_t)hm.chunk_elems, 4, 0); }
        else add(m->d_ga, L.geo, 4, 0);
        add(m->d_area, L.area, lr, 0);
        const bool step_like = mode == MODE_STEP || mode == MODE_STEPSU;
        if (step_like) add(s->H, L.H, lr, 0);
        add(m->d_ell, L.ell, 1, 2);
        add(m->d_halo_dst, L.hdst, 2, 3);   // partial slots of the chunk's halo nodes
        add(m->d_halo_ids, L.hnext, 2, 4);  // ids of the next chunk's halo nodes
        add(s->ux, L.node[0], lr, 1); add(s->uy, L.node[1], lr, 1); add(s->d, L.node[2], lr, 1);
        if (step_like) {
            add(s->vx, L.node[3], lr, 1); add(s->vy, L.node[4], lr, 1);
            add(s->ax, L.node[5], lr, 1); add(s->ay, L.node[6], lr, 1);
        }
        if (mode == MODE_TANGENT) { add(a.px, L.node[3], lr, 1); add(a.py, L.node[4], lr, 1); }
        if (mode == MODE_EQ) {
            add(a.cpx, L.node[3], lr, 1); add(a.cpy, L.node[4], lr, 1); add(a.rx, L.node[5], lr, 1); add(a.ry, L.node[6], lr, 1);
            add(a.fx_out, L.node[7], lr, 1); add(a.fy_out, L.node[8], lr, 1); add(a.dix, L.node[9], lr, 1); add(a.diy, L.node[10], lr, 1);
            add(a.ex, L.node[11], lr, 1); add(a.ey, L.node[12], lr, 1);
        }
        if (mode != MODE_FORCE && mode != MODE_TANGENT && mode != MODE_EQ) {
            add(s->fext_x, L.node[7], lr, 1); add(s->fext_y, L.node[8], lr, 1); add(m->d_minv, L.node[9], lr, 1);
            add(m->d_flags, L.flags, 0, 1);
        }
    }
    if ((mode == MODE_STEP || mode == MODE_STEPSU) && m->n_dir > 0 && bc && bc->dir_u && bc->dir_v) {
        PFF_LAUNCH(m, PFF_K_OTHER, (dirichlet_kernel<R><<<(unsigned)((m->n_dir + 127) / 128), 128, 0, m->stream>>>(
            (int)m->n_dir, m->d_dir_dof, (const R*)bc->dir_u, (const R*)bc->dir_v, a.ux, a.uy, a.vx, a.vy)));
    }
    switch (mode) {
        case MODE_STEP: return launch_step_s<R, MODE_STEP>(m, a);
        case MODE_INIT: return launch_step_s<R, MODE_INIT>(m, a);
        case MODE_FORCE: return launch_step_s<R, MODE_FORCE>(m, a);
        case MODE_TANGENT:
            if (m->opt.scatter == PFF_SCATTER_ATOMIC) { set_error("stiffness action: gather scatter only"); return PFF_EUNSUPPORTED; }
            return launch_step_s<R, MODE_TANGENT>(m, a);
        case MODE_EQ:
            if (m->opt.scatter == PFF_SCATTER_ATOMIC) { set_error("quasi-static CG: gather scatter only"); return PFF_EUNSUPPORTED; }
            return launch_step_s<R, MODE_EQ>(m, a);
        case MODE_STEPSU:
            if (m->opt.scatter == PFF_SCATTER_ATOMIC) { set_error("fused step + damage setup: gather meshes only"); return PFF_EUNSUPPORTED; }
            return launch_step_s<R, MODE_STEPSU>(m, a);
    }
    return PFF_EINVAL;
}

pff_status launch_step(pff_mesh* m, pff_state* s, const pff_bc* bc, double dt, int mode, void* fx, void* fy, void* psi,
                       const void* px, const void* py)
{
    if (m->opt.precision == PFF_F32) return launch_step_r<float>(m, s, bc, dt, mode, fx, fy, psi, px, py);
    return launch_step_r<double>(m, s, bc, dt, mode, fx, fy, psi, px, py);
}

}  // namespace pff
