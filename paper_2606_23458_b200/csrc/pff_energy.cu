// Energies per unit thickness (Eq. 1): E_el, E_kin, E_frac, E_tot.
// One element pass + one node pass writing fp64 block partials, then one fixed-order final sum:
// bit-reproducible run to run.  Diagnostics path (not on the per-step hot loop).
#include <mutex>
#include <string>

#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

template <typename R, int SPLIT>
__global__ void __launch_bounds__(kTPB) energy_elem_kernel(int Ne, const int4* conn, const void* ga, const void* gb,
                                                           const R* area, const R* ux, const R* uy, const R* d,
                                                           MatC<R> mat, double* part /* [2][nblocks] */)
{
    __shared__ double s_red[32];
    const int e = blockIdx.x * kTPB + threadIdx.x;
    double eel = 0.0, efr = 0.0;
    if (e < Ne) {
        const int4 c = __ldg(conn + e);
        R b1, c1, b2, c2;
        Geo<R>::load(ga, gb, e, b1, c1, b2, c2);
        const R A = area[e];
        const R ax = ux[c.x] - ux[c.z], bx = ux[c.y] - ux[c.z], ay = uy[c.x] - uy[c.z], by = uy[c.y] - uy[c.z];
        const R exx = b1 * ax + b2 * bx, eyy = c1 * ay + c2 * by;
        const R exy = R(0.5) * (c1 * ax + c2 * bx + b1 * ay + b2 * by);
        const R d1 = d[c.x], d2 = d[c.y], d3 = d[c.z];
        const R de = (d1 + d2 + d3) * R(1.0 / 3.0);
        const R g = (R(1) - de) * (R(1) - de) + mat.eta;
        R pp, pm, sxx, syy, sxy;
        elem_response<R, SPLIT>(mat, exx, eyy, exy, g, pp, pm, sxx, syy, sxy);
        eel = double(A) * (double(g) * double(pp) + double(pm));
        // grad d_e and the AT1 / AT2 crack surface density (L69); consistent mass for d^2 (L185)
        const double gx = double(b1) * double(d1 - d3) + double(b2) * double(d2 - d3);
        const double gy = double(c1) * double(d1 - d3) + double(c2) * double(d2 - d3);
        const double gg = gx * gx + gy * gy;
        if (mat.model == PFF_AT2) {
            const double s = double(d1) + double(d2) + double(d3);
            const double dMd = double(A) / 12.0 * (double(d1) * d1 + double(d2) * d2 + double(d3) * d3 + s * s);
            efr = double(mat.Gc) * (dMd / (2.0 * double(mat.l0)) + 0.5 * double(mat.l0) * double(A) * gg);
        } else {
            efr = 0.375 * double(mat.Gc) * (double(A) * double(de) / double(mat.l0) + double(mat.l0) * double(A) * gg);
        }
    }
    const double t0 = block_sum(eel, s_red);
    const double t1 = block_sum(efr, s_red);
    if (threadIdx.x == 0) { part[blockIdx.x] = t0; part[gridDim.x + blockIdx.x] = t1; }
}

template <typename R>
__global__ void __launch_bounds__(kTPB) energy_node_kernel(int N, const R* mass, const R* vx, const R* vy, double* part)
{
    __shared__ double s_red[32];
    const int i = blockIdx.x * kTPB + threadIdx.x;
    double ek = 0.0;
    if (i < N) ek = 0.5 * double(mass[i]) * (double(vx[i]) * double(vx[i]) + double(vy[i]) * double(vy[i]));
    const double t = block_sum(ek, s_red);
    if (threadIdx.x == 0) part[blockIdx.x] = t;
}

// out[k] = sum of part_k[0..n_k) in a fixed order (single block)
__global__ void __launch_bounds__(kTPB) energy_final_kernel(const double* p0, int n0, const double* p1, int n1,
                                                            const double* p2, int n2, double* out)
{
    __shared__ double s_red[32];
    const double* ps[3] = {p0, p1, p2};
    const int ns[3] = {n0, n1, n2};
    for (int k = 0; k < 3; ++k) {
        double v = 0.0;
        for (int i = threadIdx.x; i < ns[k]; i += kTPB) v += ps[k][i];
        const double t = block_sum(v, s_red);
        if (threadIdx.x == 0) out[k] = t;
    }
}

template <typename R, int SPLIT>
static void launch_elem(pff_mesh* m, const pff_state* s, double* part, int nbe)
{
    energy_elem_kernel<R, SPLIT><<<nbe, kTPB, 0, m->stream>>>((int)m->hm.Ne, (const int4*)m->d_conn, m->d_ga, m->d_gb,
                                                              (const R*)m->d_area, (const R*)s->ux, (const R*)s->uy,
                                                              (const R*)s->d, make_matc<R>(m->mat), part);
}

template <typename R>
static pff_status energies_r(pff_mesh* m, const pff_state* s, double out[4])
{
    const int nbe = (int)((m->hm.Ne + kTPB - 1) / kTPB), nbn = (int)((m->hm.N + kTPB - 1) / kTPB);
    double* part = nullptr;
    pff_status st = cuda_check(cudaMallocAsync((void**)&part, sizeof(double) * (2 * nbe + nbn + 4), m->stream), "energies: alloc");
    if (st != PFF_OK) return st;
    switch (m->mat.split) {
        case PFF_SPLIT_ISOTROPIC: launch_elem<R, PFF_SPLIT_ISOTROPIC>(m, s, part, nbe); break;
        case PFF_SPLIT_SPECTRAL: launch_elem<R, PFF_SPLIT_SPECTRAL>(m, s, part, nbe); break;
        case PFF_SPLIT_VOLDEV: launch_elem<R, PFF_SPLIT_VOLDEV>(m, s, part, nbe); break;
        default: launch_elem<R, PFF_SPLIT_STARCONVEX>(m, s, part, nbe); break;
    }
    energy_node_kernel<R><<<nbn, kTPB, 0, m->stream>>>((int)m->hm.N, (const R*)m->d_mass, (const R*)s->vx, (const R*)s->vy,
                                                       part + 2 * nbe);
    double* dout = part + 2 * nbe + nbn;
    energy_final_kernel<<<1, kTPB, 0, m->stream>>>(part, nbe, part + 2 * nbe, nbn, part + nbe, nbe, dout);
    m->n_launches += 3;  // diagnostics, not bracketed for profiling
    double h[3];
    st = cuda_check(cudaMemcpyAsync(h, dout, sizeof(h), cudaMemcpyDeviceToHost, m->stream), "energies: copy");
    cudaFreeAsync(part, m->stream);
    if (st == PFF_OK) st = cuda_check(cudaStreamSynchronize(m->stream), "energies: sync");
    if (st != PFF_OK) return st;
    out[0] = h[0]; out[1] = h[1]; out[2] = h[2]; out[3] = h[0] + h[1] + h[2];
    return PFF_OK;
}

// ---- pff_energies_static: the same three kernels with their block partials in a file-scope device array, for callers that
// may not allocate (CUDA graph capture, serving loops).  kEnergyScratchDoubles doubles = 1 MiB on every GPU that loads the
// library, until the process exits.  Every word a call reads it has written itself before (all 2 nbe + nbn partials), so
// nothing has to be cleared between calls; ALL calls share the array, so two calls that overlap on the GPU race.
constexpr int kEnergyScratchDoubles = 1 << 17;
static __device__ __align__(256) double g_energy_scratch[kEnergyScratchDoubles];

// In host code g_energy_scratch is only a stand-in for the symbol: the device address is looked up once per device, with
// that device current (the caller's DeviceGuard), and cached.
constexpr int kMaxDevices = 64;
static std::mutex g_scratch_mutex;
static double* g_scratch_addr[kMaxDevices];

pff_status energy_static_scratch(double** ptr)
{
    int dev = 0;
    pff_status st = cuda_check(cudaGetDevice(&dev), "pff_energies_static: cudaGetDevice");
    if (st != PFF_OK) return st;
    if (dev < 0 || dev >= kMaxDevices) { set_error("pff_energies_static: device ordinal beyond 63"); return PFF_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_scratch_mutex);
    if (!g_scratch_addr[dev]) {
        double* p = nullptr;
        st = cuda_check(cudaGetSymbolAddress((void**)&p, g_energy_scratch), "pff_energies_static: cudaGetSymbolAddress");
        if (st != PFF_OK) return st;
        if (!p) { set_error("pff_energies_static: null scratch address"); return PFF_ECUDA; }
        g_scratch_addr[dev] = p;
    }
    *ptr = g_scratch_addr[dev];
    return PFF_OK;
}

// out[0..2] as energy_final_kernel, out[3] = (out[0] + out[1]) + out[2]: the host sum of energies_r, done on the device
__global__ void __launch_bounds__(kTPB) energy_final4_kernel(const double* p0, int n0, const double* p1, int n1,
                                                             const double* p2, int n2, double* out)
{
    __shared__ double s_red[32];
    const double* ps[3] = {p0, p1, p2};
    const int ns[3] = {n0, n1, n2};
    double r[3] = {0.0, 0.0, 0.0};
    for (int k = 0; k < 3; ++k) {
        double v = 0.0;
        for (int i = threadIdx.x; i < ns[k]; i += kTPB) v += ps[k][i];
        r[k] = block_sum(v, s_red);
    }
    if (threadIdx.x == 0) { out[0] = r[0]; out[1] = r[1]; out[2] = r[2]; out[3] = r[0] + r[1] + r[2]; }
}

template <typename R>
static pff_status energies_static_r(pff_mesh* m, const pff_state* s, double* out_device)
{
    const int64_t nbe = (m->hm.Ne + kTPB - 1) / kTPB, nbn = (m->hm.N + kTPB - 1) / kTPB;
    if (2 * nbe + nbn > kEnergyScratchDoubles) {
        set_error("pff_energies_static: mesh too large for the static scratch array: 2 ceil(n_elems / 256) + ceil(n_nodes / 256) = " +
                  std::to_string(2 * nbe + nbn) + " block partials, the limit is " + std::to_string(kEnergyScratchDoubles) +
                  " (use pff_energies)");
        return PFF_EUNSUPPORTED;
    }
    double* part = nullptr;
    pff_status st = energy_static_scratch(&part);
    if (st != PFF_OK) return st;
    switch (m->mat.split) {
        case PFF_SPLIT_ISOTROPIC: launch_elem<R, PFF_SPLIT_ISOTROPIC>(m, s, part, (int)nbe); break;
        case PFF_SPLIT_SPECTRAL: launch_elem<R, PFF_SPLIT_SPECTRAL>(m, s, part, (int)nbe); break;
        case PFF_SPLIT_VOLDEV: launch_elem<R, PFF_SPLIT_VOLDEV>(m, s, part, (int)nbe); break;
        default: launch_elem<R, PFF_SPLIT_STARCONVEX>(m, s, part, (int)nbe); break;
    }
    energy_node_kernel<R><<<(int)nbn, kTPB, 0, m->stream>>>((int)m->hm.N, (const R*)m->d_mass, (const R*)s->vx, (const R*)s->vy,
                                                            part + 2 * nbe);
    energy_final4_kernel<<<1, kTPB, 0, m->stream>>>(part, (int)nbe, part + 2 * nbe, (int)nbn, part + nbe, (int)nbe, out_device);
    m->n_launches += 3;
    return cuda_check(cudaGetLastError(), "pff_energies_static: launch");
}

pff_status energies_static(pff_mesh* m, const pff_state* s, double* out_device)
{
    return m->opt.precision == PFF_F32 ? energies_static_r<float>(m, s, out_device) : energies_static_r<double>(m, s, out_device);
}

// lambda^T M d and lambda^T K d with the consistent mass M^e = A (1 + delta_ij) / 12 (L185) and the P1 stiffness
// K^e = A grad phi_i . grad phi_j: the two scalars of the (G_c, l0) gradient of Eq. 24.
template <typename R>
__global__ void __launch_bounds__(kTPB) param_terms_kernel(int Ne, const int4* conn, const void* ga, const void* gb,
                                                           const R* area, const R* lam, const R* d, double* part /* [2][nblocks] */)
{
    __shared__ double s_red[32];
    const int e = blockIdx.x * kTPB + threadIdx.x;
    double tM = 0.0, tK = 0.0;
    if (e < Ne) {
        const int4 c = __ldg(conn + e);
        R b1, c1, b2, c2;
        Geo<R>::load(ga, gb, e, b1, c1, b2, c2);
        const double A = double(area[e]);
        const double l1 = lam[c.x], l2 = lam[c.y], l3 = lam[c.z], d1 = d[c.x], d2 = d[c.y], d3 = d[c.z];
        const double ds = d1 + d2 + d3;
        tM = A / 12.0 * (l1 * (d1 + ds) + l2 * (d2 + ds) + l3 * (d3 + ds));
        const double glx = double(b1) * (l1 - l3) + double(b2) * (l2 - l3), gly = double(c1) * (l1 - l3) + double(c2) * (l2 - l3);
        const double gdx = double(b1) * (d1 - d3) + double(b2) * (d2 - d3), gdy = double(c1) * (d1 - d3) + double(c2) * (d2 - d3);
        tK = A * (glx * gdx + gly * gdy);
    }
    const double t0 = block_sum(tM, s_red);
    const double t1 = block_sum(tK, s_red);
    if (threadIdx.x == 0) { part[blockIdx.x] = t0; part[gridDim.x + blockIdx.x] = t1; }
}

template <typename R>
static pff_status param_terms_r(pff_mesh* m, const void* lambda, const void* d, double out[2])
{
    const int nbe = (int)((m->hm.Ne + kTPB - 1) / kTPB);
    double* part = nullptr;
    pff_status st = cuda_check(cudaMallocAsync((void**)&part, sizeof(double) * (2 * nbe + 4), m->stream), "param terms: alloc");
    if (st != PFF_OK) return st;
    param_terms_kernel<R><<<nbe, kTPB, 0, m->stream>>>((int)m->hm.Ne, (const int4*)m->d_conn, m->d_ga, m->d_gb, (const R*)m->d_area,
                                                       (const R*)lambda, (const R*)d, part);
    double* dout = part + 2 * nbe;
    energy_final_kernel<<<1, kTPB, 0, m->stream>>>(part, nbe, part + nbe, nbe, part, 0, dout);
    m->n_launches += 2;
    double h[2];
    st = cuda_check(cudaMemcpyAsync(h, dout, sizeof(h), cudaMemcpyDeviceToHost, m->stream), "param terms: copy");
    cudaFreeAsync(part, m->stream);
    if (st == PFF_OK) st = cuda_check(cudaStreamSynchronize(m->stream), "param terms: sync");
    if (st != PFF_OK) return st;
    out[0] = h[0]; out[1] = h[1];
    return PFF_OK;
}

pff_status damage_param_terms(pff_mesh* m, const void* lambda, const void* d, double out[2])
{
    return m->opt.precision == PFF_F32 ? param_terms_r<float>(m, lambda, d, out) : param_terms_r<double>(m, lambda, d, out);
}

pff_status energies(pff_mesh* m, const pff_state* s, double out[4])
{
    return m->opt.precision == PFF_F32 ? energies_r<float>(m, s, out) : energies_r<double>(m, s, out);
}

}  // namespace pff
