// pff_run_host: the host-buffer path of include/pff.h.  State arrives in USER numbering, fp64, AoS on the
// host; it is uploaded, permuted to internal order / mesh precision by a kernel, stepped, permuted back and
// downloaded.  Every step of the method still runs in the kernels of pff_step.cu / pff_damage.cu.
#include <cmath>

#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

template <typename R>
struct HostIO {
    double *u, *v, *a, *fext, *d, *H;  // staging, user order
    R *ux, *uy, *vx, *vy, *ax, *ay, *dd, *HH, *fex, *fey;
    const int32_t *node_old_of_new, *elem_old_of_new;
    int N, Ne;
};

template <typename R>
__global__ void host_in_kernel(const HostIO<R> io)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < io.N) {
        const int o = io.node_old_of_new[i];
        io.ux[i] = R(io.u[2 * o]); io.uy[i] = R(io.u[2 * o + 1]);
        io.vx[i] = R(io.v[2 * o]); io.vy[i] = R(io.v[2 * o + 1]);
        io.ax[i] = R(io.a[2 * o]); io.ay[i] = R(io.a[2 * o + 1]);
        io.fex[i] = R(io.fext[2 * o]); io.fey[i] = R(io.fext[2 * o + 1]);
        io.dd[i] = R(io.d[o]);
    }
    if (i < io.Ne) io.HH[i] = R(io.H[io.elem_old_of_new[i]]);
}

// parts: 1 = what the explicit step produces (u, v, a, H), 2 = what the damage solve produces (d)
template <typename R>
__global__ void host_out_kernel(const HostIO<R> io, int parts)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < io.N) {
        const int o = io.node_old_of_new[i];
        if (parts & 1) {
            io.u[2 * o] = double(io.ux[i]); io.u[2 * o + 1] = double(io.uy[i]);
            io.v[2 * o] = double(io.vx[i]); io.v[2 * o + 1] = double(io.vy[i]);
            io.a[2 * o] = double(io.ax[i]); io.a[2 * o + 1] = double(io.ay[i]);
        }
        if (parts & 2) io.d[o] = double(io.dd[i]);
    }
    if ((parts & 1) && i < io.Ne) io.H[io.elem_old_of_new[i]] = double(io.HH[i]);
}

template <typename R>
static pff_status run_host_t(pff_mesh* m, pff_host_state* hs, const double* dir_u, const double* dir_v, double S,
                             double dt, int64_t n_steps, int damage_every, double rel_tol, int max_iter)
{
    const int64_t N = m->hm.N, Ne = m->hm.Ne;
    cudaStream_t cs = m->stream;
    pff_status st;
    const size_t stage_doubles = size_t(9) * N + Ne;
    const int64_t Np = (N + 3) / 4 * 4, Nep = (Ne + 3) / 4 * 4;  // every device state array starts 16-byte aligned
    if (!m->d_stage) {
        if ((st = cuda_check(cudaMalloc(&m->d_stage, stage_doubles * sizeof(double)), "run_host: staging")) != PFF_OK) return st;
        if ((st = cuda_check(cudaMalloc(&m->d_hstate, (size_t(9) * Np + Nep) * sizeof(R)), "run_host: state")) != PFF_OK) return st;
    }
    if (m->n_dir > m->hdir_cap) {  // the Dirichlet set may have been replaced by a larger one since the last call
        if ((st = cuda_check(cudaStreamSynchronize(cs), "run_host: sync")) != PFF_OK) return st;
        if (m->d_hdir) { cudaFree(m->d_hdir); m->d_hdir = nullptr; m->hdir_cap = 0; }
        if ((st = cuda_check(cudaMalloc(&m->d_hdir, 2 * size_t(m->n_dir) * sizeof(R)), "run_host: Dirichlet values")) != PFF_OK) return st;
        m->hdir_cap = m->n_dir;
    }
    double* sg = (double*)m->d_stage;
    HostIO<R> io{};
    io.u = sg; io.v = sg + 2 * N; io.a = sg + 4 * N; io.fext = sg + 6 * N; io.d = sg + 8 * N; io.H = sg + 9 * N;
    R* ds = (R*)m->d_hstate;
    io.ux = ds; io.uy = ds + Np; io.vx = ds + 2 * Np; io.vy = ds + 3 * Np; io.ax = ds + 4 * Np; io.ay = ds + 5 * Np;
    io.dd = ds + 6 * Np; io.fex = ds + 7 * Np; io.fey = ds + 8 * Np; io.HH = ds + 9 * Np;
    R* d_du = (R*)m->d_hdir;
    R* d_dv = d_du + m->hdir_cap;
    io.node_old_of_new = m->d_node_old_of_new; io.elem_old_of_new = m->d_elem_old_of_new;
    io.N = (int)N; io.Ne = (int)Ne;
#define CP(dst, src, n, kind) if ((st = cuda_check(cudaMemcpyAsync(dst, src, (n) * sizeof(double), kind, cs), "run_host: copy")) != PFF_OK) return st
    CP(io.u, hs->u, 2 * N, cudaMemcpyHostToDevice); CP(io.v, hs->v, 2 * N, cudaMemcpyHostToDevice);
    CP(io.a, hs->a, 2 * N, cudaMemcpyHostToDevice); CP(io.fext, hs->fext, 2 * N, cudaMemcpyHostToDevice);
    CP(io.d, hs->d, N, cudaMemcpyHostToDevice); CP(io.H, hs->H, Ne, cudaMemcpyHostToDevice);
    const unsigned nb = (unsigned)((std::max(N, Ne) + 255) / 256);
    host_in_kernel<R><<<nb, 256, 0, cs>>>(io);
    m->n_launches += 2;  // host_in + host_out
    pff_bc bc{nullptr, nullptr, S};
    std::vector<R> hu, hv;
    if (m->n_dir > 0 && dir_u && dir_v) {
        hu.assign(dir_u, dir_u + m->n_dir); hv.assign(dir_v, dir_v + m->n_dir);
        if ((st = cuda_check(cudaMemcpyAsync(d_du, hu.data(), m->n_dir * sizeof(R), cudaMemcpyHostToDevice, cs), "run_host: bc")) != PFF_OK) return st;
        if ((st = cuda_check(cudaMemcpyAsync(d_dv, hv.data(), m->n_dir * sizeof(R), cudaMemcpyHostToDevice, cs), "run_host: bc")) != PFF_OK) return st;
        bc.dir_u = d_du; bc.dir_v = d_dv;
    }
    pff_state s{io.ux, io.uy, io.vx, io.vy, io.ax, io.ay, io.dd, io.HH, io.fex, io.fey};
    pff_status worst = PFF_OK;
    // The results of the LAST explicit step (u, v, a, H) are final before its damage solve: they are permuted and copied
    // back on a second stream while the solve runs on the mesh stream; d follows when the solve is done.
    if (!m->copy_stream && (st = cuda_check(cudaStreamCreateWithFlags(&m->copy_stream, cudaStreamNonBlocking), "run_host: stream")) != PFF_OK) return st;
    if (!m->ev_step && (st = cuda_check(cudaEventCreateWithFlags(&m->ev_step, cudaEventDisableTiming), "run_host: event")) != PFF_OK) return st;
    if (!m->ev_out && (st = cuda_check(cudaEventCreateWithFlags(&m->ev_out, cudaEventDisableTiming), "run_host: event")) != PFF_OK) return st;
    cudaStream_t cp = m->copy_stream;
    bool mech_out = false;
    auto mechanics_out = [&]() -> pff_status {
        pff_status e;
        if ((e = cuda_check(cudaEventRecord(m->ev_step, cs), "run_host: record")) != PFF_OK) return e;
        if ((e = cuda_check(cudaStreamWaitEvent(cp, m->ev_step, 0), "run_host: wait")) != PFF_OK) return e;
        host_out_kernel<R><<<nb, 256, 0, cp>>>(io, 1);
        // The mesh stream goes on only when this permutation kernel is done: the persistent CG kernel that may come next
        // fills every SM (3 CTAs of 74 KB each) and would keep the permutation kernel, and with it the copies below, waiting
        // until the whole solve is over (measured: the end-to-end step 0.4 ms longer when the CG kernel follows the step
        // kernel directly, as it does with the fused setup).  The copies themselves then overlap the solve.
        if ((e = cuda_check(cudaEventRecord(m->ev_out, cp), "run_host: record")) != PFF_OK) return e;
        if ((e = cuda_check(cudaStreamWaitEvent(cs, m->ev_out, 0), "run_host: wait")) != PFF_OK) return e;
#define CPC(dst, src, n) if ((e = cuda_check(cudaMemcpyAsync(dst, src, (n) * sizeof(double), cudaMemcpyDeviceToHost, cp), "run_host: copy")) != PFF_OK) return e
        CPC(hs->u, io.u, 2 * N); CPC(hs->v, io.v, 2 * N); CPC(hs->a, io.a, 2 * N); CPC(hs->H, io.H, Ne);
#undef CPC
        mech_out = true;
        return PFF_OK;
    };
    const bool fuse = fused_setup_ok(m);  // the step before a solve performs the solve's setup pass as well (as pff_run_steps)
    for (int64_t k = 1; k <= n_steps; ++k) {
        const bool solve = damage_every > 0 && k % damage_every == 0;
        m->su_tol = rel_tol; m->su_max_iter = max_iter;
        st = launch_step(m, &s, &bc, dt, solve && fuse ? /*MODE_STEPSU*/ 5 : /*MODE_STEP*/ 0, nullptr, nullptr, nullptr);
        if (st != PFF_OK) { m->su_ready = false; return st; }
        if (k == n_steps && (st = mechanics_out()) != PFF_OK) { m->su_ready = false; return st; }
        if (solve) {
            st = damage_solve(m, &s, rel_tol, max_iter, nullptr, nullptr);
            m->su_ready = false;
            if (st == PFF_ENOCONV) worst = st;
            else if (st != PFF_OK) return st;
        }
    }
    if (!mech_out && (st = mechanics_out()) != PFF_OK) return st;  // n_steps == 0
    host_out_kernel<R><<<nb, 256, 0, cs>>>(io, 2);
    CP(hs->d, io.d, N, cudaMemcpyDeviceToHost);
    if ((st = cuda_check(cudaStreamSynchronize(cp), "run_host: copy sync")) != PFF_OK) return st;
#undef CP
    if ((st = cuda_check(cudaStreamSynchronize(cs), "run_host: sync")) != PFF_OK) return st;
    return worst;
}

}  // namespace pff

extern "C" pff_status pff_run_host(pff_mesh* m, pff_host_state* hs, const double* dir_u, const double* dir_v,
                                   double load_scale, double dt, int64_t n_steps, int32_t damage_every,
                                   double rel_tol, int32_t max_iter)
{
    using namespace pff;
    if (!m || !hs || !hs->u || !hs->v || !hs->a || !hs->d || !hs->H || !hs->fext) {
        set_error("pff_run_host: null argument"); return PFF_EINVAL;
    }
    if (!(dt > 0) || !std::isfinite(dt) || n_steps < 0 || damage_every < 0 ||
        (damage_every > 0 && (!(rel_tol > 0) || max_iter < 1))) {
        set_error("pff_run_host: need dt > 0, n_steps >= 0, damage_every >= 0, rel_tol > 0, max_iter >= 1");
        return PFF_EINVAL;
    }
    if (m->n_dir > 0 && ((dir_u == nullptr) != (dir_v == nullptr))) {
        set_error("pff_run_host: dir_u and dir_v must be given together"); return PFF_EINVAL;
    }
    DeviceGuard dg(m);
    if (m->opt.precision == PFF_F32)
        return run_host_t<float>(m, hs, dir_u, dir_v, load_scale, dt, n_steps, damage_every, rel_tol, max_iter);
    return run_host_t<double>(m, hs, dir_u, dir_v, load_scale, dt, n_steps, damage_every, rel_tol, max_iter);
}
