// Quasi-static mechanics solve by conjugate gradients on the matrix-free stiffness action (Eq. 11-15;
// L337 "staggered quasi-static mode"):
//     K(u_ref) du = S f_ext - f_int(u_ref)   on the free dofs,   u = u_ref + du,
// with K(u_ref) p = f_int(u_ref + p) - f_int(u_ref).  ONE launch of the explicit-step kernel per CG iteration (pff_step.cu,
// MODE_EQ): its node prologue applies the previous step (du += alpha p, r -= alpha q) and forms p = D^-1 r + beta p in the
// stage, the element pass evaluates both forces of Eq. 13, the ordered gather leaves q = K p and the seven sums that give
// alpha and PREDICT r.z after the step (so beta is known without another pass: the recurrence of the damage CG), and the
// last CTA advances the scalars: one pass over HBM per iteration, alpha, beta and the norms never leave the device (the
// host reads the control block once per batch of 25 launches).  Jacobi preconditioner: the diagonal of the ISOTROPIC
// degraded stiffness g(d_e) A_e B^T C B, summed per node over a node -> element table in a fixed order (any SPD diagonal is
// a valid preconditioner for the other splits).  Every reduction is ordered: the solve is bit-reproducible run to run.
#include <algorithm>
#include <vector>

#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

template <typename R>
__global__ void __launch_bounds__(kTPB) eq_dirichlet_kernel(int n, const int32_t* dof, const R* du, R* ux, R* uy)
{
    const int k = blockIdx.x * kTPB + threadIdx.x;
    if (k >= n) return;
    const int node = dof[k] >> 1;
    if (dof[k] & 1) uy[node] = du[k];
    else ux[node] = du[k];
}

// Jacobi diagonal: K_ii of the isotropic degraded stiffness, x and y dof of one node, incident elements in table order
template <typename R>
__global__ void __launch_bounds__(kTPB) eq_diag_kernel(int N, const int32_t* ptr, const int32_t* adj, const int4* conn,
                                                       const void* ga, const void* gb, const R* area, const R* d,
                                                       const uint8_t* flags, MatC<R> mat, R* dix, R* diy)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N) return;
    double sx = 0.0, sy = 0.0;
    for (int k = ptr[i]; k < ptr[i + 1]; ++k) {
        const int e = adj[k] >> 2, corner = adj[k] & 3;
        const int4 c = __ldg(conn + e);
        R b1, c1, b2, c2;
        Geo<R>::load(ga, gb, e, b1, c1, b2, c2);
        const double b = corner == 0 ? double(b1) : (corner == 1 ? double(b2) : -(double(b1) + double(b2)));
        const double cc = corner == 0 ? double(c1) : (corner == 1 ? double(c2) : -(double(c1) + double(c2)));
        const double de = (double(d[c.x]) + double(d[c.y]) + double(d[c.z])) * (1.0 / 3.0);
        const double gA = ((1.0 - de) * (1.0 - de) + double(mat.eta)) * double(area[e]);
        const double l2m = double(mat.lam) + 2.0 * double(mat.mu), mu = double(mat.mu);
        sx += gA * (l2m * b * b + mu * cc * cc);
        sy += gA * (l2m * cc * cc + mu * b * b);
    }
    const uint8_t fl = flags[i];
    dix[i] = (fl & 1) ? R(0) : R(1.0 / sx);
    diy[i] = (fl & 2) ? R(0) : R(1.0 / sy);
}

template <typename R>
struct EqVec {
    R *xx, *xy, *rx, *ry, *px, *py, *qx, *qy, *dix, *diy;
};

// r = S f_ext - f_int(u_ref) on the free dofs (f_int arrives in q), du = 0, p = 0; block 0 writes the control block of the solve
template <typename R>
__global__ void __launch_bounds__(kTPB) eq_init_kernel(int N, const uint8_t* flags, const R* fex, const R* fey, R S, EqVec<R> v,
                                                       DamageCtrl* ctrl, double tol, int max_iter)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i < N) {
        const uint8_t fl = flags[i];
        v.rx[i] = (fl & 1) ? R(0) : S * fex[i] - v.qx[i];
        v.ry[i] = (fl & 2) ? R(0) : S * fey[i] - v.qy[i];
        v.px[i] = R(0); v.py[i] = R(0); v.xx[i] = R(0); v.xy[i] = R(0);
    }
    if (i == 0) {
        DamageCtrl c{};
        c.tol = tol; c.max_iter = max_iter; c.first = 1; c.status = PFF_ENOCONV;
        *ctrl = c;
    }
}

// u <- u_ref + du, with the last step (decided, not yet applied) added first
template <typename R>
__global__ void __launch_bounds__(kTPB) eq_finish_kernel(int N, EqVec<R> v, const DamageCtrl* ctrl, R* ux, R* uy)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N) return;
    R dx = v.xx[i], dy = v.xy[i];
    if (ctrl->pending) { const R alpha = R(ctrl->alpha); dx = rfma(alpha, v.px[i], dx); dy = rfma(alpha, v.py[i], dy); }
    ux[i] += dx; uy[i] += dy;
}

static pff_status ensure_eq_workspace(pff_mesh* m)
{
    if (m->d_eq_ctrl) return PFF_OK;
    const HostMesh& hm = m->hm;
    const size_t N = (size_t)hm.N, Ne = (size_t)hm.Ne;
    pff_status st;
    // node -> (element, corner) table in element order: counting sort over the connectivity
    std::vector<int32_t> ptr(N + 1, 0), adj(3 * Ne);
    for (size_t e = 0; e < Ne; ++e)
        for (int k = 0; k < 3; ++k) ++ptr[hm.conn4[4 * e + k] + 1];
    for (size_t i = 0; i < N; ++i) ptr[i + 1] += ptr[i];
    {
        std::vector<int32_t> fill(ptr.begin(), ptr.end() - 1);
        for (size_t e = 0; e < Ne; ++e)
            for (int k = 0; k < 3; ++k) adj[fill[hm.conn4[4 * e + k]]++] = int32_t(4 * e + k);
    }
    if ((st = cuda_check(cudaMalloc((void**)&m->d_n2e_ptr, sizeof(int32_t) * (N + 1)), "equilibrium: table")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_n2e, sizeof(int32_t) * 3 * Ne), "equilibrium: table")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMemcpy(m->d_n2e_ptr, ptr.data(), sizeof(int32_t) * (N + 1), cudaMemcpyHostToDevice), "equilibrium: table")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMemcpy(m->d_n2e, adj.data(), sizeof(int32_t) * 3 * Ne, cudaMemcpyHostToDevice), "equilibrium: table")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc(&m->d_eq_vec, 10 * ((N + 15) & ~size_t(15)) * m->rb), "equilibrium: vectors")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_eq_part, sizeof(double) * kCh * 2048), "equilibrium: partials")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_eq_ticket, sizeof(unsigned int)), "equilibrium: ticket")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMemset(m->d_eq_ticket, 0, sizeof(unsigned int)), "equilibrium: ticket")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMallocHost((void**)&m->h_eq_ctrl, sizeof(DamageCtrl)), "equilibrium: pinned ctrl")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_eq_ctrl, sizeof(DamageCtrl)), "equilibrium: ctrl")) != PFF_OK) return st;
    return PFF_OK;
}

template <typename R>
static pff_status equilibrium_solve_t(pff_mesh* m, pff_state* s, const pff_bc* bc, double rel_tol, int max_iter, int* iters,
                                      double* relres)
{
    pff_status st = ensure_eq_workspace(m);
    if (st != PFF_OK) return st;
    const int N = (int)m->hm.N;
    const unsigned nb = (unsigned)((N + kTPB - 1) / kTPB);
    cudaStream_t cs = m->stream;
    R* base = (R*)m->d_eq_vec;
    const size_t ld = ((size_t)N + 15) & ~size_t(15);  // every vector 16-byte aligned (sources of bulk copies)
    EqVec<R> v{base, base + ld, base + 2 * ld, base + 3 * ld, base + 4 * ld, base + 5 * ld, base + 6 * ld, base + 7 * ld,
               base + 8 * ld, base + 9 * ld};
    if (m->n_dir > 0 && bc && bc->dir_u) {
        PFF_LAUNCH(m, PFF_K_OTHER, (eq_dirichlet_kernel<R><<<(unsigned)((m->n_dir + kTPB - 1) / kTPB), kTPB, 0, cs>>>(
            (int)m->n_dir, m->d_dir_dof, (const R*)bc->dir_u, (R*)s->ux, (R*)s->uy)));
    }
    // f_int(u_ref) -> q, preconditioner, first residual; the control block of the solve is written on the device
    if ((st = launch_step(m, s, nullptr, 0.0, /*MODE_FORCE*/ 2, v.qx, v.qy, nullptr)) != PFF_OK) return st;
    const MatC<R> mat = make_matc<R>(m->mat);
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_diag_kernel<R><<<nb, kTPB, 0, cs>>>(N, m->d_n2e_ptr, m->d_n2e, (const int4*)m->d_conn, m->d_ga, m->d_gb,
                                                                     (const R*)m->d_area, (const R*)s->d, m->d_flags, mat, v.dix, v.diy)));
    const R S = R(bc ? bc->load_scale : 1.0);
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_init_kernel<R><<<nb, kTPB, 0, cs>>>(N, m->d_flags, (const R*)s->fext_x, (const R*)s->fext_y, S, v,
                                                                     m->d_eq_ctrl, rel_tol, max_iter)));
    m->eq.ex = v.xx; m->eq.ey = v.xy; m->eq.rx = v.rx; m->eq.ry = v.ry; m->eq.dix = v.dix; m->eq.diy = v.diy;
    // One launch per CG iteration (pff_step.cu, MODE_EQ: node prologue with the previous step, fused stiffness action,
    // gather, sums, scalar step by the last CTA); a launch that finds the solve finished returns at once.  The host looks at
    // the control block once per batch.  The pass count exceeds the iteration count by one (the last pass only measures).
    DamageCtrl* h = m->h_eq_ctrl;
    h->done = 0;
    for (int enq = 0; enq <= max_iter && !h->done;) {
        const int batch = std::min(25, max_iter + 1 - enq);
        for (int k = 0; k < batch; ++k)
            if ((st = launch_step(m, s, nullptr, 0.0, /*MODE_EQ*/ 4, v.qx, v.qy, nullptr, v.px, v.py)) != PFF_OK) return st;
        enq += batch;
        if ((st = cuda_check(cudaMemcpyAsync(h, m->d_eq_ctrl, sizeof(DamageCtrl), cudaMemcpyDeviceToHost, cs), "equilibrium: readback")) != PFF_OK) return st;
        if ((st = cuda_check(cudaStreamSynchronize(cs), "equilibrium: sync")) != PFF_OK) return st;
    }
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_finish_kernel<R><<<nb, kTPB, 0, cs>>>(N, v, m->d_eq_ctrl, (R*)s->ux, (R*)s->uy)));
    if ((st = cuda_check(cudaStreamSynchronize(cs), "equilibrium: sync")) != PFF_OK) return st;
    if (iters) *iters = h->iters;
    if (relres) *relres = h->relres;
    if (h->done && h->status == PFF_OK) return PFF_OK;
    if (h->restart)
        set_error("pff_equilibrium_solve: breakdown, p . K p <= 0 (operator not positive definite along the search direction); "
                  "the steps taken so far are applied");
    else
        set_error("pff_equilibrium_solve: max_iter reached");
    return PFF_ENOCONV;
}

pff_status equilibrium_solve(pff_mesh* m, pff_state* s, const pff_bc* bc, double rel_tol, int max_iter, int* iters, double* relres)
{
    if (m->opt.scatter == PFF_SCATTER_ATOMIC) { set_error("pff_equilibrium_solve: gather scatter only"); return PFF_EUNSUPPORTED; }
    if (m->opt.precision == PFF_F32) return equilibrium_solve_t<float>(m, s, bc, rel_tol, max_iter, iters, relres);
    return equilibrium_solve_t<double>(m, s, bc, rel_tol, max_iter, iters, relres);
}

}  // namespace pff
