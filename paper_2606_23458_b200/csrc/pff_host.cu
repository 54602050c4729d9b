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

template <typename R>
__global__ void host_out_kernel(const HostIO<R> io)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < io.N) {
        const int o = io.node_old_of_new[i];
        io.u[2 * o] = double(io.ux[i]); io.u[2 * o + 1] = double(io.uy[i]);
        io.v[2 * o] = double(io.vx[i]); io.v[2 * o + 1] = double(io.vy[i]);
        io.a[2 * o] = double(io.ax[i]); io.a[2 * o + 1] = double(io.ay[i]);
        io.d[o] = double(io.dd[i]);
    }
    if (i < io.Ne) io.H[io.elem_old_of_new[i]] = double(io.HH[i]);
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
        if ((st = cuda_check(cudaMalloc(&m->d_hstate, (size_t(9) * Np + Nep) * sizeof(R) + 2 * size_t(std::max<int64_t>(m->n_dir, 1)) * sizeof(R)), "run_host: state")) != PFF_OK) return st;
    }
    double* sg = (double*)m->d_stage;
    HostIO<R> io{};
    io.u = sg; io.v = sg + 2 * N; io.a = sg + 4 * N; io.fext = sg + 6 * N; io.d = sg + 8 * N; io.H = sg + 9 * N;
    R* ds = (R*)m->d_hstate;
    io.ux = ds; io.uy = ds + Np; io.vx = ds + 2 * Np; io.vy = ds + 3 * Np; io.ax = ds + 4 * Np; io.ay = ds + 5 * Np;
    io.dd = ds + 6 * Np; io.fex = ds + 7 * Np; io.fey = ds + 8 * Np; io.HH = ds + 9 * Np;
    R* d_du = ds + 9 * Np + Nep;
    R* d_dv = d_du + std::max<int64_t>(m->n_dir, 1);
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
    for (int64_t k = 1; k <= n_steps; ++k) {
        if ((st = launch_step(m, &s, &bc, dt, 0, nullptr, nullptr, nullptr)) != PFF_OK) return st;
        if (damage_every > 0 && k % damage_every == 0) {
            st = damage_solve(m, &s, rel_tol, max_iter, nullptr, nullptr);
            if (st == PFF_ENOCONV) worst = st;
            else if (st != PFF_OK) return st;
        }
    }
    host_out_kernel<R><<<nb, 256, 0, cs>>>(io);
    CP(hs->u, io.u, 2 * N, cudaMemcpyDeviceToHost); CP(hs->v, io.v, 2 * N, cudaMemcpyDeviceToHost);
    CP(hs->a, io.a, 2 * N, cudaMemcpyDeviceToHost); CP(hs->d, io.d, N, cudaMemcpyDeviceToHost);
    CP(hs->H, io.H, Ne, cudaMemcpyDeviceToHost);
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
    if (m->opt.precision == PFF_F32)
        return run_host_t<float>(m, hs, dir_u, dir_v, load_scale, dt, n_steps, damage_every, rel_tol, max_iter);
    return run_host_t<double>(m, hs, dir_u, dir_v, load_scale, dt, n_steps, damage_every, rel_tol, max_iter);
}
