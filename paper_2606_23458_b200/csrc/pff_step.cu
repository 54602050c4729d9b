// Explicit step kernels (Eq. 16-18; element math L42, L71-93, L124):
//
//   step_chunk_kernel   one CTA per chunk of elements.  Phase 1 forms the predictor u_{n+1} (Eq. 16) of all
//                       nodes the chunk touches and stages it with d in shared memory; phase 2 is the fused
//                       element pass (strain -> split -> degradation -> stress -> force -> history) writing
//                       element forces to shared-memory slots; phase 3 gathers each node's incident slots
//                       in a fixed order (chunk-local ELL table) and, for interior nodes, completes Eq. 17-18
//                       in the same kernel -- f_int never reaches HBM.  Interface nodes get a partial sum.
//   step_shared_kernel  interface nodes: ordered sum of the per-chunk partials, then the same Eq. 16-18.
//   elem_atomic_kernel / node_atomic_kernel   PFF_SCATTER_ATOMIC variant: thread per element, global
//                       floating-point atomics (the paper's "atomic indexed accumulation", L43, L124).
//   dirichlet_kernel    writes u_bar, v_bar into the Dirichlet dofs before the step (Eq. 5, R8).
#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

enum { MODE_STEP = 0, MODE_INIT = 1, MODE_FORCE = 2 };

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
    int EC, max_nloc, N, Ne, N_int, N_sh;
    const int32_t *sh_rowptr, *sh_slots;
    R *ux, *uy, *vx, *vy, *ax, *ay;
    const R* d;
    R* H;
    const R *fex, *fey;
    R *fx_out, *fy_out, *psi_out;
    R *fwx, *fwy;
    R dt, hdt, hdt2, S;
    MatC<R> mat;
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
    if (MODE == MODE_FORCE) { a.fx_out[gid] = fx; a.fy_out[gid] = fy; return; }
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

template <typename R, int SPLIT, int MODE>
__global__ void __launch_bounds__(kTPB) step_chunk_kernel(const StepArgs<R> a)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    R* s_ux = reinterpret_cast<R*>(smem_raw);
    R* s_uy = s_ux + a.max_nloc;
    R* s_d = s_uy + a.max_nloc;
    R* s_f = s_d + a.max_nloc;  // [6][EC]
    const ChunkMeta cm = a.meta[blockIdx.x];
    const int nloc = cm.n_int + cm.n_halo;
    const int tid = threadIdx.x;

    for (int i = tid; i < nloc; i += kTPB) {
        const int gid = i < cm.n_int ? cm.node_start + i : a.halo_ids[cm.halo_off + i - cm.n_int];
        R px, py;
        predict<R, MODE>(a, gid, px, py);
        s_ux[i] = px; s_uy[i] = py; s_d[i] = a.d[gid];
    }
    __syncthreads();

    for (int e = tid; e < cm.n_elem; e += kTPB) {
        const int ge = cm.elem_start + e;
        const ushort4 c = __ldg(a.lconn + ge);
        R b1, c1, b2, c2;
        Geo<R>::load(a.ga, a.gb, ge, b1, c1, b2, c2);
        const R A = __ldg(a.area + ge);
        R psi_p, f[6];
        element_forces<R, SPLIT>(a.mat, b1, c1, b2, c2, A, s_ux[c.x], s_uy[c.x], s_ux[c.y], s_uy[c.y], s_ux[c.z],
                                 s_uy[c.z], s_d[c.x] + s_d[c.y] + s_d[c.z], psi_p, f);
#pragma unroll
        for (int k = 0; k < 6; ++k) s_f[k * a.EC + e] = f[k];
        if (MODE == MODE_STEP) {
            const R h = a.H[ge];
            if (psi_p > h) a.H[ge] = psi_p;  // H <- max(H, psi+)  (L98, L114)
        } else if (MODE == MODE_FORCE) {
            if (a.psi_out) a.psi_out[ge] = psi_p;
        }
    }
    __syncthreads();

    const uint16_t* ell = a.ell + cm.ell_off;
    for (int i = tid; i < nloc; i += kTPB) {
        R fx = R(0), fy = R(0);
        for (int k = 0; k < cm.ell_w; ++k) {
            const unsigned ent = ell[k * nloc + i];
            if (ent != 0xFFFFu) {
                const int e = ent >> 2, cnr = ent & 3;
                fx += s_f[(2 * cnr) * a.EC + e];
                fy += s_f[(2 * cnr + 1) * a.EC + e];
            }
        }
        if (i < cm.n_int) {
            finish_node<R, MODE>(a, cm.node_start + i, s_ux[i], s_uy[i], fx, fy);
        } else {
            const int64_t slot = cm.halo_off + i - cm.n_int;
            a.halo_part[slot] = fx;
            a.halo_part[a.n_slots + slot] = fy;
        }
    }
}

template <typename R, int MODE>
__global__ void __launch_bounds__(kTPB) step_shared_kernel(const StepArgs<R> a)
{
    const int s = blockIdx.x * kTPB + threadIdx.x;
    if (s >= a.N_sh) return;
    const int gid = a.N_int + s;
    R fx = R(0), fy = R(0);
    for (int k = a.sh_rowptr[s]; k < a.sh_rowptr[s + 1]; ++k) {
        const int slot = a.sh_slots[k];
        fx += a.halo_part[slot];
        fy += a.halo_part[a.n_slots + slot];
    }
    R px, py;
    predict<R, MODE>(a, gid, px, py);
    finish_node<R, MODE>(a, gid, px, py, fx, fy);
}

// ---- atomic variant ------------------------------------------------------------------------
__device__ __forceinline__ void red_add(double* p, double v) { atomicAdd(p, v); }
__device__ __forceinline__ void red_add(float* p, float v) { atomicAdd(p, v); }

template <typename R, int SPLIT, int MODE>
__global__ void __launch_bounds__(kTPB) elem_atomic_kernel(const StepArgs<R> a)
{
    const int e = blockIdx.x * kTPB + threadIdx.x;
    if (e >= a.Ne) return;
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
    red_add(a.fwx + c.x, f[0]); red_add(a.fwy + c.x, f[1]);
    red_add(a.fwx + c.y, f[2]); red_add(a.fwy + c.y, f[3]);
    red_add(a.fwx + c.z, f[4]); red_add(a.fwy + c.z, f[5]);
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
        static int granted = 48 * 1024;  // per instantiation high-water mark of the dynamic smem opt-in
        if (m->smem_step > granted) {
            cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, m->smem_step);
            if (e != cudaSuccess) return cuda_check(e, "cudaFuncSetAttribute(step_chunk_kernel)");
            granted = m->smem_step;
        }
        if (m->only_kernel != 1) {
            PFF_LAUNCH(m, PFF_K_STEP_CHUNK, (kern<<<(unsigned)hm.C, kTPB, m->smem_step, m->stream>>>(a)));
        }
        if (hm.N_sh > 0 && m->only_kernel != 0) {
            PFF_LAUNCH(m, PFF_K_STEP_SHARED, (step_shared_kernel<R, MODE><<<(unsigned)((hm.N_sh + kTPB - 1) / kTPB), kTPB, 0, m->stream>>>(a)));
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
                                void* psi)
{
    const HostMesh& hm = m->hm;
    StepArgs<R> a{};
    a.meta = m->d_meta; a.lconn = (const ushort4*)m->d_lconn; a.conn = (const int4*)m->d_conn;
    a.ga = m->d_ga; a.gb = m->d_gb; a.area = (const R*)m->d_area;
    a.halo_ids = m->d_halo_ids; a.ell = m->d_ell; a.flags = m->d_flags; a.minv = (const R*)m->d_minv;
    a.halo_part = (R*)m->d_halo_part; a.n_slots = m->n_slots;
    a.EC = hm.chunk_elems; a.max_nloc = hm.max_nloc; a.N = (int)hm.N; a.Ne = (int)hm.Ne;
    a.N_int = (int)hm.N_int; a.N_sh = (int)hm.N_sh;
    a.sh_rowptr = m->d_sh_rowptr; a.sh_slots = m->d_sh_slots;
    a.ux = (R*)s->ux; a.uy = (R*)s->uy; a.vx = (R*)s->vx; a.vy = (R*)s->vy; a.ax = (R*)s->ax; a.ay = (R*)s->ay;
    a.d = (const R*)s->d; a.H = (R*)s->H; a.fex = (const R*)s->fext_x; a.fey = (const R*)s->fext_y;
    a.fx_out = (R*)fx; a.fy_out = (R*)fy; a.psi_out = (R*)psi;
    a.fwx = (R*)m->d_fwx; a.fwy = (R*)m->d_fwy;
    a.dt = R(dt); a.hdt = R(0.5 * dt); a.hdt2 = R(0.5 * dt * dt);
    a.S = R(bc ? bc->load_scale : 1.0);
    a.mat = make_matc<R>(m->mat);
    if (mode == MODE_STEP && m->n_dir > 0 && bc && bc->dir_u && bc->dir_v) {
        PFF_LAUNCH(m, PFF_K_OTHER, (dirichlet_kernel<R><<<(unsigned)((m->n_dir + 127) / 128), 128, 0, m->stream>>>(
            (int)m->n_dir, m->d_dir_dof, (const R*)bc->dir_u, (const R*)bc->dir_v, a.ux, a.uy, a.vx, a.vy)));
    }
    switch (mode) {
        case MODE_STEP: return launch_step_s<R, MODE_STEP>(m, a);
        case MODE_INIT: return launch_step_s<R, MODE_INIT>(m, a);
        case MODE_FORCE: return launch_step_s<R, MODE_FORCE>(m, a);
    }
    return PFF_EINVAL;
}

pff_status launch_step(pff_mesh* m, pff_state* s, const pff_bc* bc, double dt, int mode, void* fx, void* fy, void* psi)
{
    if (m->opt.precision == PFF_F32) return launch_step_r<float>(m, s, bc, dt, mode, fx, fy, psi);
    return launch_step_r<double>(m, s, bc, dt, mode, fx, fy, psi);
}

}  // namespace pff
