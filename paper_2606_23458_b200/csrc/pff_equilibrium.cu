// Quasi-static mechanics solve by conjugate gradients on the matrix-free stiffness action (Eq. 11-15;
// L337 "staggered quasi-static mode"):
//     K(u_ref) du = S f_ext - f_int(u_ref)   on the free dofs,   u = u_ref + du,
// with K(u_ref) p = f_int(u_ref + p) - f_int(u_ref) evaluated by ONE fused pass of the explicit-step kernel per
// iteration (pff_step.cu, MODE_TANGENT), which also leaves the block partials of p . q.  The rest of the CG recurrence is a
// handful of small node kernels; alpha, beta and the norms stay on the device (the host reads the scalar block once per
// batch of iterations).  Jacobi preconditioner:
// the diagonal of the ISOTROPIC degraded stiffness g(d_e) A_e B^T C B, summed per node over a node -> element table in a
// fixed order (any SPD diagonal is a valid preconditioner for the other splits).  Every reduction is ordered: the solve
// is bit-reproducible run to run.  First correct path of this NEXT row; the vector kernels are not fused into the
// element pass the way the damage CG is.
#include <algorithm>
#include <vector>

#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

enum { SC_RZ = 0, SC_PQ, SC_ALPHA, SC_BETA, SC_RR, SC_R0, SC_DONE, SC_ITERS, SC_TOL, SC_N };

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

// r = S f_ext - f_int(u_ref) on the free dofs (f_int arrives in q), z = D^-1 r, p = z, du = 0
template <typename R>
__global__ void __launch_bounds__(kTPB) eq_init_kernel(int N, const uint8_t* flags, const R* fex, const R* fey, R S, EqVec<R> v,
                                                       double* part)
{
    __shared__ double s_red[32];
    const int i = blockIdx.x * kTPB + threadIdx.x;
    double rz = 0.0, rr = 0.0;
    if (i < N) {
        const uint8_t fl = flags[i];
        const R rx = (fl & 1) ? R(0) : S * fex[i] - v.qx[i];
        const R ry = (fl & 2) ? R(0) : S * fey[i] - v.qy[i];
        const R zx = v.dix[i] * rx, zy = v.diy[i] * ry;
        v.rx[i] = rx; v.ry[i] = ry; v.px[i] = zx; v.py[i] = zy; v.xx[i] = R(0); v.xy[i] = R(0);
        rz = double(rx) * double(zx) + double(ry) * double(zy);
        rr = double(rx) * double(rx) + double(ry) * double(ry);
    }
    const double t0 = block_sum(rz, s_red);
    const double t1 = block_sum(rr, s_red);
    if (threadIdx.x == 0) { part[blockIdx.x] = t0; part[gridDim.x + blockIdx.x] = t1; }
}

// du += alpha p, r -= alpha q (free dofs), partials of r.z and r.r
template <typename R>
__global__ void __launch_bounds__(kTPB) eq_update_kernel(int N, const uint8_t* flags, EqVec<R> v, const double* sc, double* part)
{
    __shared__ double s_red[32];
    if (sc[SC_DONE] != 0.0) return;
    const R alpha = R(sc[SC_ALPHA]);
    const int i = blockIdx.x * kTPB + threadIdx.x;
    double rz = 0.0, rr = 0.0;
    if (i < N) {
        const uint8_t fl = flags[i];
        v.xx[i] = rfma(alpha, v.px[i], v.xx[i]);
        v.xy[i] = rfma(alpha, v.py[i], v.xy[i]);
        const R rx = (fl & 1) ? R(0) : rfma(-alpha, v.qx[i], v.rx[i]);
        const R ry = (fl & 2) ? R(0) : rfma(-alpha, v.qy[i], v.ry[i]);
        v.rx[i] = rx; v.ry[i] = ry;
        rz = double(rx) * double(rx) * double(v.dix[i]) + double(ry) * double(ry) * double(v.diy[i]);
        rr = double(rx) * double(rx) + double(ry) * double(ry);
    }
    const double t0 = block_sum(rz, s_red);
    const double t1 = block_sum(rr, s_red);
    if (threadIdx.x == 0) { part[blockIdx.x] = t0; part[gridDim.x + blockIdx.x] = t1; }
}

template <typename R>
__global__ void __launch_bounds__(kTPB) eq_dir_kernel(int N, EqVec<R> v, const double* sc)
{
    if (sc[SC_DONE] != 0.0) return;
    const R beta = R(sc[SC_BETA]);
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N) return;
    v.px[i] = rfma(beta, v.px[i], v.dix[i] * v.rx[i]);
    v.py[i] = rfma(beta, v.py[i], v.diy[i] * v.ry[i]);
}

template <typename R>
__global__ void __launch_bounds__(kTPB) eq_finish_kernel(int N, EqVec<R> v, R* ux, R* uy)
{
    const int i = blockIdx.x * kTPB + threadIdx.x;
    if (i >= N) return;
    ux[i] += v.xx[i]; uy[i] += v.xy[i];
}

// single block: fixed-order sums of the block partials, then the scalar step of the recurrence
// MODE 0: after eq_init; 1: after eq_dot (alpha); 2: after eq_update (beta, convergence)
template <int MODE>
__global__ void __launch_bounds__(kTPB) eq_reduce_kernel(const double* part, int nb, double* sc)
{
    __shared__ double s_red[32];
    if (MODE != 0 && sc[SC_DONE] != 0.0) return;
    double a = 0.0, b = 0.0;
    for (int i = threadIdx.x; i < nb; i += kTPB) { a += part[i]; if (MODE != 1) b += part[nb + i]; }
    const double t0 = block_sum(a, s_red);
    const double t1 = block_sum(b, s_red);
    if (threadIdx.x != 0) return;
    if (MODE == 0) {
        sc[SC_RZ] = t0; sc[SC_RR] = t1; sc[SC_R0] = sqrt(t1); sc[SC_ITERS] = 0.0;
        sc[SC_DONE] = (t1 == 0.0) ? 1.0 : 0.0;
    } else if (MODE == 1) {
        // breakdown guard: for the non-isotropic splits the shifted difference need not be positive definite (eta = 0 with
        // fully damaged patches, sign changes of the split): stop without applying a step along this direction
        sc[SC_PQ] = t0;
        if (t0 > 0.0 && isfinite(t0)) sc[SC_ALPHA] = sc[SC_RZ] / t0;
        else { sc[SC_ALPHA] = 0.0; sc[SC_DONE] = 2.0; }
    } else {
        sc[SC_BETA] = t0 / sc[SC_RZ]; sc[SC_RZ] = t0; sc[SC_RR] = t1; sc[SC_ITERS] += 1.0;
        if (sqrt(t1) <= sc[SC_TOL] * sc[SC_R0]) sc[SC_DONE] = 1.0;
    }
}

static pff_status ensure_eq_workspace(pff_mesh* m)
{
    if (m->d_eq_sc) return PFF_OK;
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
    const size_t nb = (N + kTPB - 1) / kTPB;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_eq_part, sizeof(double) * (2 * nb + (size_t)hm.C)), "equilibrium: partials")) != PFF_OK) return st;
    if ((st = cuda_check(cudaMalloc((void**)&m->d_eq_sc, sizeof(double) * SC_N), "equilibrium: scalars")) != PFF_OK) return st;
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
    const size_t ld = ((size_t)N + 15) & ~size_t(15);  // every vector 16-byte aligned (bulk copies of the trial direction)
    EqVec<R> v{base, base + ld, base + 2 * ld, base + 3 * ld, base + 4 * ld, base + 5 * ld, base + 6 * ld, base + 7 * ld,
               base + 8 * ld, base + 9 * ld};
    double* sc = m->d_eq_sc;
    double h_sc[SC_N] = {};
    h_sc[SC_TOL] = rel_tol;
    if ((st = cuda_check(cudaMemcpyAsync(sc, h_sc, sizeof(h_sc), cudaMemcpyHostToDevice, cs), "equilibrium: scalars")) != PFF_OK) return st;
    if (m->n_dir > 0 && bc && bc->dir_u) {
        PFF_LAUNCH(m, PFF_K_OTHER, (eq_dirichlet_kernel<R><<<(unsigned)((m->n_dir + kTPB - 1) / kTPB), kTPB, 0, cs>>>(
            (int)m->n_dir, m->d_dir_dof, (const R*)bc->dir_u, (R*)s->ux, (R*)s->uy)));
    }
    // f_int(u_ref) -> q, preconditioner, first residual and direction
    if ((st = launch_step(m, s, nullptr, 0.0, /*MODE_FORCE*/ 2, v.qx, v.qy, nullptr)) != PFF_OK) return st;
    const MatC<R> mat = make_matc<R>(m->mat);
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_diag_kernel<R><<<nb, kTPB, 0, cs>>>(N, m->d_n2e_ptr, m->d_n2e, (const int4*)m->d_conn, m->d_ga, m->d_gb,
                                                                     (const R*)m->d_area, (const R*)s->d, m->d_flags, mat, v.dix, v.diy)));
    const R S = R(bc ? bc->load_scale : 1.0);
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_init_kernel<R><<<nb, kTPB, 0, cs>>>(N, m->d_flags, (const R*)s->fext_x, (const R*)s->fext_y, S, v, m->d_eq_part)));
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_reduce_kernel<0><<<1, kTPB, 0, cs>>>(m->d_eq_part, (int)nb, sc)));
    int enq = 0;
    while (enq < max_iter) {
        const int batch = std::min(25, max_iter - enq);
        for (int k = 0; k < batch; ++k) {
            // q = K p; the action kernel also leaves the block partials of p . q (p is zero on the constrained dofs)
            m->tangent_pq_part = m->d_eq_part;
            st = launch_step(m, s, nullptr, 0.0, /*MODE_TANGENT*/ 3, v.qx, v.qy, nullptr, v.px, v.py);
            m->tangent_pq_part = nullptr;
            if (st != PFF_OK) return st;
            PFF_LAUNCH(m, PFF_K_OTHER, (eq_reduce_kernel<1><<<1, kTPB, 0, cs>>>(m->d_eq_part, m->last_step_grid, sc)));
            PFF_LAUNCH(m, PFF_K_OTHER, (eq_update_kernel<R><<<nb, kTPB, 0, cs>>>(N, m->d_flags, v, sc, m->d_eq_part)));
            PFF_LAUNCH(m, PFF_K_OTHER, (eq_reduce_kernel<2><<<1, kTPB, 0, cs>>>(m->d_eq_part, (int)nb, sc)));
            PFF_LAUNCH(m, PFF_K_OTHER, (eq_dir_kernel<R><<<nb, kTPB, 0, cs>>>(N, v, sc)));
        }
        enq += batch;
        if ((st = cuda_check(cudaMemcpyAsync(h_sc, sc, sizeof(h_sc), cudaMemcpyDeviceToHost, cs), "equilibrium: readback")) != PFF_OK) return st;
        if ((st = cuda_check(cudaStreamSynchronize(cs), "equilibrium: sync")) != PFF_OK) return st;
        if (h_sc[SC_DONE] != 0.0) break;
    }
    if (enq == 0) {  // max_iter < 1 is rejected by the caller; keep the readback for completeness
        if ((st = cuda_check(cudaMemcpyAsync(h_sc, sc, sizeof(h_sc), cudaMemcpyDeviceToHost, cs), "equilibrium: readback")) != PFF_OK) return st;
        if ((st = cuda_check(cudaStreamSynchronize(cs), "equilibrium: sync")) != PFF_OK) return st;
    }
    PFF_LAUNCH(m, PFF_K_OTHER, (eq_finish_kernel<R><<<nb, kTPB, 0, cs>>>(N, v, (R*)s->ux, (R*)s->uy)));
    if ((st = cuda_check(cudaStreamSynchronize(cs), "equilibrium: sync")) != PFF_OK) return st;
    if (iters) *iters = (int)h_sc[SC_ITERS];
    if (relres) *relres = h_sc[SC_R0] > 0.0 ? sqrt(h_sc[SC_RR]) / h_sc[SC_R0] : 0.0;
    if (h_sc[SC_DONE] == 2.0) {
        set_error("pff_equilibrium_solve: breakdown, p . K p <= 0 (operator not positive definite along the search direction); "
                  "the steps taken so far are applied");
        return PFF_ENOCONV;
    }
    if (h_sc[SC_DONE] == 0.0) {
        set_error("pff_equilibrium_solve: max_iter reached");
        return PFF_ENOCONV;
    }
    return PFF_OK;
}

pff_status equilibrium_solve(pff_mesh* m, pff_state* s, const pff_bc* bc, double rel_tol, int max_iter, int* iters, double* relres)
{
    if (m->opt.scatter == PFF_SCATTER_ATOMIC) { set_error("pff_equilibrium_solve: gather scatter only"); return PFF_EUNSUPPORTED; }
    if (m->opt.precision == PFF_F32) return equilibrium_solve_t<float>(m, s, bc, rel_tol, max_iter, iters, relres);
    return equilibrium_solve_t<double>(m, s, bc, rel_tol, max_iter, iters, relres);
}

}  // namespace pff
