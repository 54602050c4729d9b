// C-ABI entry points of libpff (include/pff.h): argument checking, uploads, dispatch.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <mutex>
#include <new>

#include "pff_device.cuh"
#include "pff_mesh.h"

namespace pff {

static thread_local std::string g_err;
void set_error(const std::string& s) { g_err = s; }

pff_status cuda_check(cudaError_t e, const char* what)
{
    if (e == cudaSuccess) return PFF_OK;
    set_error(std::string(what) + ": " + cudaGetErrorString(e));
    return PFF_ECUDA;
}

#define PFF_CUDA(call)                                                   \
    do {                                                                 \
        pff_status st__ = pff::cuda_check((call), #call);                \
        if (st__ != PFF_OK) return st__;                                 \
    } while (0)

template <typename T>
static pff_status upload(T** dst, const void* src, size_t count, cudaStream_t st)
{
    *dst = nullptr;
    if (count == 0) count = 1;  // keep pointers valid
    PFF_CUDA(cudaMalloc((void**)dst, count * sizeof(T)));
    if (src) PFF_CUDA(cudaMemcpyAsync(*dst, src, count * sizeof(T), cudaMemcpyHostToDevice, st));
    else PFF_CUDA(cudaMemsetAsync(*dst, 0, count * sizeof(T), st));
    return PFF_OK;
}

// upload a fp64 host array narrowed to the mesh precision
static pff_status upload_real(void** dst, const double* src, size_t count, size_t rb, cudaStream_t st)
{
    if (rb == 8) return upload((double**)dst, src, count, st);
    std::vector<float> tmp(count);
    for (size_t i = 0; i < count; ++i) tmp[i] = (float)src[i];
    pff_status s = upload((float**)dst, tmp.data(), count, st);
    if (s == PFF_OK) s = cuda_check(cudaStreamSynchronize(st), "upload sync");  // tmp dies at return
    return s;
}

// The dynamic shared-memory opt-in is an attribute of the FUNCTION on a device, shared by every mesh of the process that
// uses the kernel there: it is only ever raised (a high-water mark per device and kernel, under a mutex), so a mesh with
// small chunks never lowers it under a mesh with large ones.  The persistent grid depends on the mesh's own stage size
// and is cached per mesh.
static std::mutex g_optin_mutex;
static std::map<std::pair<int, const void*>, int> g_optin;  // (device, kernel) -> bytes granted

pff_status persistent_config(pff_mesh* m, const void* kern, int smem_bytes, int* grid, int block)
{
    auto it = m->launch_grid.find(kern);
    if (it != m->launch_grid.end()) { *grid = it->second; return PFF_OK; }
    {
        std::lock_guard<std::mutex> lock(g_optin_mutex);
        int& granted = g_optin[{m->device, kern}];
        if (smem_bytes > granted) {  // static + dynamic shared memory may exceed 48 KB: always opt in
            PFF_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_bytes));
            granted = smem_bytes;
        }
    }
    int per_sm = 0, sms = 0;
    PFF_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, block, (size_t)smem_bytes));
    PFF_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device));
    *grid = (per_sm > 0 ? per_sm : 1) * sms;
    m->launch_grid.emplace(kern, *grid);
    return PFF_OK;
}

// Dirichlet values come as a pair: with a Dirichlet set installed, giving exactly one of dir_u / dir_v is an error
static bool valid_bc(const pff_mesh* m, const pff_bc* bc)
{
    return !(m->n_dir > 0 && bc && ((bc->dir_u == nullptr) != (bc->dir_v == nullptr)));
}

// all ten arrays present and 16-byte aligned (they are streamed with bulk-asynchronous copies)
static bool valid_state(const pff_state* s)
{
    if (!(s && s->ux && s->uy && s->vx && s->vy && s->ax && s->ay && s->d && s->H && s->fext_x && s->fext_y)) return false;
    const void* p[] = {s->ux, s->uy, s->vx, s->vy, s->ax, s->ay, s->d, s->H, s->fext_x, s->fext_y};
    for (const void* q : p) if (reinterpret_cast<uintptr_t>(q) & 15) return false;
    return true;
}

}  // namespace pff

using namespace pff;

extern "C" {

const char* pff_last_error(void) { return g_err.c_str(); }

void pff_mesh_destroy(pff_mesh* m)
{
    if (!m) return;
    DeviceGuard dg(m);
    cudaStreamSynchronize(m->stream);
    mg_free(m);
    void* ptrs[] = {m->d_meta, m->d_lconn, m->d_conn, m->d_ga, m->d_gb, m->d_area, m->d_minv, m->d_mass,
                    m->d_halo_ids, m->d_sh_rowptr, m->d_halo_dst, m->d_ell, m->d_flags, m->d_halo_part,
                    m->d_fwx, m->d_fwy, m->d_dir_dof, m->d_ca, m->d_cb, m->d_lb, m->d_r, m->d_p, m->d_q, m->d_dinv, m->d_mask,
                    m->d_part, m->d_tally, m->d_cg2, m->d_ctrl, m->d_ticket, m->d_step_bar, m->d_stage, m->d_hstate, m->d_hdir, m->d_node_old_of_new,
                    m->d_elem_old_of_new, m->d_n2e_ptr, m->d_n2e, m->d_eq_vec, m->d_eq_part, m->d_eq_ctrl, m->d_eq_ticket, m->d_su_part};
    for (void* p : ptrs) if (p) cudaFree(p);
    if (m->h_ctrl) cudaFreeHost(m->h_ctrl);
    if (m->h_tally) cudaFreeHost(m->h_tally);
    if (m->h_eq_ctrl) cudaFreeHost(m->h_eq_ctrl);
    if (m->graph_exec) cudaGraphExecDestroy(m->graph_exec);
    if (m->copy_stream) { cudaStreamSynchronize(m->copy_stream); cudaStreamDestroy(m->copy_stream); }
    if (m->ev_step) cudaEventDestroy(m->ev_step);
    if (m->ev_out) cudaEventDestroy(m->ev_out);
    for (auto& v : m->prof_ev) for (cudaEvent_t e : v) cudaEventDestroy(e);
    delete m;
}

pff_status pff_mesh_create(int64_t n_nodes, const double* xy, int64_t n_elems, const int32_t* tri,
                           const pff_material* mat, const pff_options* opt_in, void* cuda_stream, pff_mesh** out)
{
    if (out) *out = nullptr;
    if (!xy || !tri || !mat || !out) { set_error("pff_mesh_create: null argument"); return PFF_EINVAL; }
    pff_options opt{PFF_F64, PFF_ORDER_BISECTION, PFF_SCATTER_GATHER, 0};
    if (opt_in) opt = *opt_in;
    if (!(mat->E > 0) || !(mat->rho > 0) || !(mat->Gc > 0) || !(mat->l0 > 0) || !(mat->nu > -1.0) || !(mat->nu < 0.5) ||
        !(mat->eta >= 0) || !std::isfinite(mat->E + mat->rho + mat->Gc + mat->l0 + mat->eta)) {
        set_error("pff_mesh_create: material out of range (need E, rho, Gc, l0 > 0, -1 < nu < 0.5, eta >= 0)");
        return PFF_EINVAL;
    }
    if ((mat->model != PFF_AT1 && mat->model != PFF_AT2) || mat->split < 0 || mat->split > 3 ||
        (mat->plane != PFF_PLANE_STRAIN && mat->plane != PFF_PLANE_STRESS) ||
        (opt.precision != PFF_F64 && opt.precision != PFF_F32) ||
        (opt.order != PFF_ORDER_NONE && opt.order != PFF_ORDER_MORTON && opt.order != PFF_ORDER_BISECTION) ||
        (opt.scatter != PFF_SCATTER_GATHER && opt.scatter != PFF_SCATTER_ATOMIC) || opt.chunk_elems < 0) {
        set_error("pff_mesh_create: bad enum value"); return PFF_EINVAL;
    }
    if (mat->split == PFF_SPLIT_STARCONVEX && !(mat->gamma_star >= -1.0)) {
        set_error("pff_mesh_create: gamma_star must be >= -1"); return PFF_EINVAL;
    }
    pff_mesh* m = new (std::nothrow) pff_mesh;
    if (!m) { set_error("out of host memory"); return PFF_ENOMEM; }
    m->mat = *mat; m->opt = opt; m->stream = (cudaStream_t)cuda_stream;
    m->rb = opt.precision == PFF_F32 ? 4 : 8;
    std::string err;
    pff_status st;
    int sms = 0;  // the persistent CG kernel runs 3 CTAs per SM: the chunk size is balanced for that grid
    if (cudaGetDevice(&m->device) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, m->device);
    try {
        st = build_host_mesh(n_nodes, xy, n_elems, tri, mat->rho, opt.order, opt.chunk_elems, m->rb, m->hm, err, 3 * sms);
    } catch (const std::bad_alloc&) { st = PFF_ENOMEM; err = "out of host memory in mesh setup"; }
    if (st != PFF_OK) { set_error("pff_mesh_create: " + err); delete m; return st; }
    HostMesh& hm = m->hm;
    opt.chunk_elems = m->opt.chunk_elems = hm.chunk_elems;
    {
        const double mu = mat->E / (2 * (1 + mat->nu));
        const double lam = mat->plane == PFF_PLANE_STRESS ? mat->E * mat->nu / (1 - mat->nu * mat->nu)
                                                           : mat->E * mat->nu / ((1 + mat->nu) * (1 - 2 * mat->nu));
        m->dt_crit = hm.hmin / std::sqrt((lam + 2 * mu) / mat->rho);
    }
    m->lay_step = make_stage_layout(0, hm.chunk_elems, hm.node_len, hm.flag_len, hm.ell_len, hm.max_nhalo, m->rb, chunk_kernel_stages(0));
    m->lay_mv = make_stage_layout(1, hm.chunk_elems, hm.node_len, hm.flag_len, hm.ell_len, hm.max_nhalo, m->rb, chunk_kernel_stages(1));
    m->lay_stepsu = make_stage_layout(5, hm.chunk_elems, hm.node_len, hm.flag_len, hm.ell_len, hm.max_nhalo, m->rb, chunk_kernel_stages(0));
    m->lay_eq = make_stage_layout(3, hm.chunk_elems, hm.node_len, hm.flag_len, hm.ell_len, hm.max_nhalo, m->rb, chunk_kernel_stages(0));
    m->lay_su = make_stage_layout(2, hm.chunk_elems, hm.node_len, hm.flag_len, hm.ell_len, hm.max_nhalo, m->rb, chunk_kernel_stages(2));
    m->ell_total = (int64_t)hm.ell.size();
    if (!verify_stage_extents(hm, m->ell_total, (int64_t)hm.halo_ids.size(), m->rb, err)) {
        set_error("pff_mesh_create: " + err); delete m; return PFF_EMESH;
    }

    auto fail = [&](pff_status s) { pff_mesh_destroy(m); return s; };
    cudaStream_t cs = m->stream;
    if ((st = cuda_check(cudaGetDevice(&m->device), "cudaGetDevice")) != PFF_OK) return fail(st);
    {   // set-up: device address of pff_energies_static's scratch array on this GPU (a lookup, nothing is allocated; a
        // failure is reported by pff_energies_static itself, which retries)
        double* scratch = nullptr;
        (void)energy_static_scratch(&scratch);
    }
    const size_t N = hm.N, Ne = hm.Ne;
#define UP(call) if ((st = (call)) != PFF_OK) return fail(st)
    UP(upload(&m->d_meta, hm.meta.data(), hm.meta.size(), cs));
    UP(upload((uint16_t**)&m->d_lconn, hm.lconn4.data(), 4 * Ne, cs));
    UP(upload((int32_t**)&m->d_conn, hm.conn4.data(), 4 * Ne, cs));
    if (m->rb == 8) {
        std::vector<double> ga(2 * Ne), gb(2 * Ne);
        for (size_t e = 0; e < Ne; ++e) {
            ga[2 * e] = hm.g12[4 * e]; ga[2 * e + 1] = hm.g12[4 * e + 1];
            gb[2 * e] = hm.g12[4 * e + 2]; gb[2 * e + 1] = hm.g12[4 * e + 3];
        }
        UP(upload((double**)&m->d_ga, ga.data(), 2 * Ne, cs));
        UP(upload((double**)&m->d_gb, gb.data(), 2 * Ne, cs));
        UP(cuda_check(cudaStreamSynchronize(cs), "sync"));
    } else {
        UP(upload_real(&m->d_ga, hm.g12.data(), 4 * Ne, 4, cs));
    }
    UP(upload_real(&m->d_area, hm.area.data(), Ne, m->rb, cs));
    {
        std::vector<double> minv(N);
        for (size_t i = 0; i < N; ++i) minv[i] = 1.0 / hm.mass[i];
        UP(upload_real(&m->d_minv, minv.data(), N, m->rb, cs));
        UP(upload_real(&m->d_mass, hm.mass.data(), N, m->rb, cs));
        UP(cuda_check(cudaStreamSynchronize(cs), "sync"));
    }
    m->n_entries = (int64_t)hm.halo_ids.size();
    m->n_slots = (int64_t)kIfaceWidth * hm.N_sh + hm.n_ovf;
    UP(upload(&m->d_halo_ids, hm.halo_ids.data(), hm.halo_ids.size(), cs));
    UP(upload(&m->d_sh_rowptr, hm.sh_rowptr.data(), hm.sh_rowptr.size(), cs));
    UP(upload(&m->d_halo_dst, hm.halo_dst.data(), hm.halo_dst.size(), cs));
    UP(upload(&m->d_ell, hm.ell.data(), hm.ell.size(), cs));
    m->h_flags.assign(N, 0);
    UP(upload(&m->d_flags, m->h_flags.data(), N, cs));
    UP(upload((uint8_t**)&m->d_halo_part, nullptr, size_t(3) * std::max<int64_t>(m->n_slots, 1) * m->rb, cs));
    UP(upload((uint8_t**)&m->d_fwx, nullptr, N * m->rb, cs));
    UP(upload((uint8_t**)&m->d_fwy, nullptr, N * m->rb, cs));
    UP(upload((uint8_t**)&m->d_ca, nullptr, (m->rb == 8 ? 2 : 4) * Ne * m->rb, cs));
    if (m->rb == 8) UP(upload((uint8_t**)&m->d_cb, nullptr, 2 * Ne * m->rb, cs));
    UP(upload((uint8_t**)&m->d_lb, nullptr, N * m->rb, cs));
    UP(upload((uint8_t**)&m->d_r, nullptr, N * m->rb, cs));
    UP(upload((uint8_t**)&m->d_p, nullptr, N * m->rb, cs));
    UP(upload((uint8_t**)&m->d_q, nullptr, N * m->rb, cs));
    UP(upload((uint8_t**)&m->d_dinv, nullptr, N * m->rb, cs));
    UP(upload(&m->d_mask, nullptr, 2 * N, cs));
    UP(upload(&m->d_step_bar, nullptr, 2, cs));
    UP(upload(&m->d_node_old_of_new, hm.node_old_of_new.data(), N, cs));
    {
        std::vector<int32_t> eon(Ne);
        for (size_t e = 0; e < Ne; ++e) eon[hm.elem_new_of_old[e]] = (int32_t)e;
        UP(upload(&m->d_elem_old_of_new, eon.data(), Ne, cs));
        UP(cuda_check(cudaStreamSynchronize(cs), "sync"));
    }
#undef UP
    if ((st = cuda_check(cudaStreamSynchronize(cs), "mesh upload")) != PFF_OK) return fail(st);
    // the big host tables are no longer needed
    std::vector<uint16_t>().swap(hm.lconn4); std::vector<uint16_t>().swap(hm.ell);
    std::vector<double>().swap(hm.g12);
    *out = m;
    return PFF_OK;
}

pff_status pff_mesh_plan(int64_t n_nodes, const double* xy, int64_t n_elems, const int32_t* tri, const pff_options* opt_in,
                         int32_t* node_new_of_old, int32_t* elem_new_of_old, int64_t* n_chunks, int64_t* n_shared,
                         int32_t* chunk_elems, int32_t* max_local_nodes, double* h_min)
{
    if (!xy || !tri) { set_error("pff_mesh_plan: null argument"); return PFF_EINVAL; }
    pff_options opt{PFF_F64, PFF_ORDER_BISECTION, PFF_SCATTER_GATHER, 0};
    if (opt_in) opt = *opt_in;
    HostMesh hm;
    std::string err;
    pff_status st;
    try {
        st = build_host_mesh(n_nodes, xy, n_elems, tri, 1.0, opt.order, opt.chunk_elems, opt.precision == PFF_F32 ? 4 : 8,
                             hm, err);
    } catch (const std::bad_alloc&) { st = PFF_ENOMEM; err = "out of host memory in mesh setup"; }
    if (st != PFF_OK) { set_error("pff_mesh_plan: " + err); return st; }
    if (!verify_stage_extents(hm, (int64_t)hm.ell.size(), (int64_t)hm.halo_ids.size(), opt.precision == PFF_F32 ? 4 : 8, err)) {
        set_error("pff_mesh_plan: " + err); return PFF_EMESH;
    }
    if (node_new_of_old) std::memcpy(node_new_of_old, hm.node_new_of_old.data(), sizeof(int32_t) * hm.N);
    if (elem_new_of_old) std::memcpy(elem_new_of_old, hm.elem_new_of_old.data(), sizeof(int32_t) * hm.Ne);
    if (n_chunks) *n_chunks = hm.C;
    if (n_shared) *n_shared = hm.N_sh;
    if (chunk_elems) *chunk_elems = hm.chunk_elems;
    if (max_local_nodes) *max_local_nodes = hm.max_nloc;
    if (h_min) *h_min = hm.hmin;
    return PFF_OK;
}

pff_status pff_mesh_info(const pff_mesh* m, int64_t* n_nodes, int64_t* n_elems, double* h_min, double* dt_crit,
                         int64_t* n_chunks, int64_t* n_shared)
{
    if (!m) { set_error("pff_mesh_info: null mesh"); return PFF_EINVAL; }
    if (n_nodes) *n_nodes = m->hm.N;
    if (n_elems) *n_elems = m->hm.Ne;
    if (h_min) *h_min = m->hm.hmin;
    if (dt_crit) *dt_crit = m->dt_crit;
    if (n_chunks) *n_chunks = m->hm.C;
    if (n_shared) *n_shared = m->hm.N_sh;
    return PFF_OK;
}

pff_status pff_mesh_permutations(const pff_mesh* m, int32_t* node_new_of_old, int32_t* elem_new_of_old)
{
    if (!m) { set_error("pff_mesh_permutations: null mesh"); return PFF_EINVAL; }
    if (node_new_of_old) std::memcpy(node_new_of_old, m->hm.node_new_of_old.data(), sizeof(int32_t) * m->hm.N);
    if (elem_new_of_old) std::memcpy(elem_new_of_old, m->hm.elem_new_of_old.data(), sizeof(int32_t) * m->hm.Ne);
    return PFF_OK;
}

static pff_status push_flags(pff_mesh* m)
{
    ++m->flags_gen;  // invalidates a captured pff_run_steps period (the Dirichlet dof list pointer may have changed)
    PFF_CUDA(cudaMemcpyAsync(m->d_flags, m->h_flags.data(), m->h_flags.size(), cudaMemcpyHostToDevice, m->stream));
    PFF_CUDA(cudaStreamSynchronize(m->stream));
    return PFF_OK;
}

pff_status pff_set_dirichlet(pff_mesh* m, int64_t n_dir, const int32_t* dir_dof)
{
    if (!m || n_dir < 0 || (n_dir > 0 && !dir_dof)) { set_error("pff_set_dirichlet: bad argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    std::vector<int32_t> idof(n_dir);
    for (int64_t k = 0; k < n_dir; ++k) {
        if (dir_dof[k] < 0 || dir_dof[k] >= 2 * m->hm.N) { set_error("pff_set_dirichlet: dof out of range"); return PFF_EINVAL; }
    }
    for (auto& f : m->h_flags) f &= uint8_t(~3);
    for (int64_t k = 0; k < n_dir; ++k) {
        const int32_t node = m->hm.node_new_of_old[dir_dof[k] >> 1], comp = dir_dof[k] & 1;
        idof[k] = 2 * node + comp;
        m->h_flags[node] |= uint8_t(1 << comp);
    }
    PFF_CUDA(cudaStreamSynchronize(m->stream));
    if (m->d_dir_dof) { cudaFree(m->d_dir_dof); m->d_dir_dof = nullptr; }
    m->n_dir = n_dir;
    pff_status st = upload(&m->d_dir_dof, idof.data(), (size_t)n_dir, m->stream);
    if (st != PFF_OK) return st;
    return push_flags(m);
}

pff_status pff_set_damage_dirichlet(pff_mesh* m, int64_t n, const int32_t* nodes)
{
    if (!m || n < 0 || (n > 0 && !nodes)) { set_error("pff_set_damage_dirichlet: bad argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    for (int64_t k = 0; k < n; ++k)
        if (nodes[k] < 0 || nodes[k] >= m->hm.N) { set_error("pff_set_damage_dirichlet: node out of range"); return PFF_EINVAL; }
    for (auto& f : m->h_flags) f &= uint8_t(~4);
    for (int64_t k = 0; k < n; ++k) m->h_flags[m->hm.node_new_of_old[nodes[k]]] |= 4;
    return push_flags(m);
}

pff_status pff_set_traction(pff_mesh* m, pff_state* s, int64_t n_edges, const int32_t* edge_nodes, const double* t)
{
    if (!m || !s || !s->fext_x || !s->fext_y || n_edges < 0 || (n_edges > 0 && (!edge_nodes || !t))) {
        set_error("pff_set_traction: bad argument"); return PFF_EINVAL;
    }
    DeviceGuard dg(m);
    const int64_t N = m->hm.N;
    std::vector<double> fx(N, 0.0), fy(N, 0.0);
    const double* xy = m->hm.xy_user.data();
    for (int64_t k = 0; k < n_edges; ++k) {
        const int32_t a = edge_nodes[2 * k], b = edge_nodes[2 * k + 1];
        if (a < 0 || b < 0 || a >= N || b >= N) { set_error("pff_set_traction: node out of range"); return PFF_EINVAL; }
        const double L = std::hypot(xy[2 * a] - xy[2 * b], xy[2 * a + 1] - xy[2 * b + 1]);
        const int32_t ia = m->hm.node_new_of_old[a], ib = m->hm.node_new_of_old[b];
        fx[ia] += 0.5 * L * t[2 * k]; fx[ib] += 0.5 * L * t[2 * k];
        fy[ia] += 0.5 * L * t[2 * k + 1]; fy[ib] += 0.5 * L * t[2 * k + 1];
    }
    if (m->rb == 8) {
        PFF_CUDA(cudaMemcpyAsync(s->fext_x, fx.data(), N * 8, cudaMemcpyHostToDevice, m->stream));
        PFF_CUDA(cudaMemcpyAsync(s->fext_y, fy.data(), N * 8, cudaMemcpyHostToDevice, m->stream));
    } else {
        std::vector<float> gx(fx.begin(), fx.end()), gy(fy.begin(), fy.end());
        PFF_CUDA(cudaMemcpyAsync(s->fext_x, gx.data(), N * 4, cudaMemcpyHostToDevice, m->stream));
        PFF_CUDA(cudaMemcpyAsync(s->fext_y, gy.data(), N * 4, cudaMemcpyHostToDevice, m->stream));
        PFF_CUDA(cudaStreamSynchronize(m->stream));
    }
    PFF_CUDA(cudaStreamSynchronize(m->stream));
    return PFF_OK;
}

pff_status pff_init_accel(pff_mesh* m, pff_state* s, const pff_bc* bc)
{
    if (!m || !valid_state(s)) { set_error("pff_init_accel: null mesh, null or misaligned (16 B) state pointer"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return launch_step(m, s, bc, 0.0, /*MODE_INIT*/ 1, nullptr, nullptr, nullptr);
}

pff_status pff_explicit_step(pff_mesh* m, pff_state* s, const pff_bc* bc, double dt)
{
    if (!m || !valid_state(s)) { set_error("pff_explicit_step: null mesh, null or misaligned (16 B) state pointer"); return PFF_EINVAL; }
    if (!(dt > 0) || !std::isfinite(dt)) { set_error("pff_explicit_step: dt must be > 0"); return PFF_EINVAL; }
    if (!valid_bc(m, bc)) { set_error("pff_explicit_step: dir_u and dir_v must be given together"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return launch_step(m, s, bc, dt, /*MODE_STEP*/ 0, nullptr, nullptr, nullptr);
}

pff_status pff_internal_force(pff_mesh* m, const pff_state* s, void* fx, void* fy, void* psi_plus)
{
    if (!m || !valid_state(s) || !fx || !fy) { set_error("pff_internal_force: null argument"); return PFF_EINVAL; }
    if (m->opt.scatter == PFF_SCATTER_ATOMIC) { set_error("pff_internal_force: gather meshes only"); return PFF_EUNSUPPORTED; }
    DeviceGuard dg(m);
    return launch_step(m, const_cast<pff_state*>(s), nullptr, 0.0, /*MODE_FORCE*/ 2, fx, fy, psi_plus);
}

pff_status pff_damage_solve(pff_mesh* m, pff_state* s, double rel_tol, int32_t max_iter, int32_t* iters, double* relres)
{
    if (!m || !valid_state(s)) { set_error("pff_damage_solve: null mesh, null or misaligned (16 B) state pointer"); return PFF_EINVAL; }
    if (!(rel_tol > 0) || max_iter < 1) { set_error("pff_damage_solve: need rel_tol > 0, max_iter >= 1"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return damage_solve(m, s, rel_tol, max_iter, iters, relres);
}

pff_status pff_damage_last_stats(const pff_mesh* m, int32_t* restarts, int32_t* truncations)
{
    if (!m) { set_error("pff_damage_last_stats: null mesh"); return PFF_EINVAL; }
    if (restarts) *restarts = m->last_restarts;
    if (truncations) *truncations = m->last_truncs;
    return PFF_OK;
}

pff_status pff_subcycle_limit(const pff_material* mat, int32_t* n_max, double* ratio)
{
    if (!mat || !n_max) { set_error("pff_subcycle_limit: null argument"); return PFF_EINVAL; }
    if (!(mat->E > 0) || !(mat->rho > 0) || !(mat->nu > -1.0) || !(mat->nu < 0.5)) {
        set_error("pff_subcycle_limit: material out of range"); return PFF_EINVAL;
    }
    const double mu = mat->E / (2 * (1 + mat->nu));
    const double lam = mat->plane == PFF_PLANE_STRESS ? mat->E * mat->nu / (1 - mat->nu * mat->nu)
                                                       : mat->E * mat->nu / ((1 + mat->nu) * (1 - 2 * mat->nu));
    const double cp = std::sqrt((lam + 2 * mu) / mat->rho), cs = std::sqrt(mu / mat->rho);
    const double cR = cs * (0.862 + 1.14 * mat->nu) / (1 + mat->nu);
    const double r = cp / (0.6 * cR);
    if (ratio) *ratio = r;
    *n_max = (int32_t)std::floor(r);
    return PFF_OK;
}

pff_status pff_run_steps(pff_mesh* m, pff_state* s, const pff_bc* bc, double dt, int64_t n_steps, int32_t damage_every,
                         double rel_tol, int32_t max_iter, int64_t* cg_iters_total)
{
    if (!m || !valid_state(s)) { set_error("pff_run_steps: null mesh, null or misaligned (16 B) state pointer"); return PFF_EINVAL; }
    if (!(dt > 0) || !std::isfinite(dt) || n_steps < 0 || damage_every < 0 ||
        (damage_every > 0 && (!(rel_tol > 0) || max_iter < 1))) {
        set_error("pff_run_steps: need dt > 0, n_steps >= 0, damage_every >= 0, rel_tol > 0, max_iter >= 1"); return PFF_EINVAL;
    }
    if (!valid_bc(m, bc)) { set_error("pff_run_steps: dir_u and dir_v must be given together"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    // The whole loop is asynchronous: every solve adds its counters to a device-resident tally, which the host reads ONCE at
    // the end, so the GPU never waits for the host between steps.  When the run is long enough, one period of the loop
    // (damage_every explicit steps + one solve; kernels only, no copies) is captured into a CUDA graph after it has run
    // once the ordinary way and replayed for the remaining periods: small meshes, where a step is a handful of
    // microsecond kernels, then pay one graph launch per period instead of a cooperative launch per kernel.
    if (!m->d_tally) {
        PFF_CUDA(cudaMalloc((void**)&m->d_tally, sizeof(RunTally)));
        PFF_CUDA(cudaMallocHost((void**)&m->h_tally, sizeof(RunTally)));
    }
    PFF_CUDA(cudaMemsetAsync(m->d_tally, 0, sizeof(RunTally), m->stream));
    pff_status st = PFF_OK;
    m->defer = true;
    // The explicit step that precedes a damage solve also performs that solve's setup pass where the mesh allows it
    // (pff_step.cu MODE_STEPSU: everything the pass reads is already in the step kernel's shared memory).
    const bool fuse = fused_setup_ok(m);
    m->last_step_fused = fuse && damage_every > 0 ? 1 : 0;
    auto one_step = [&](int64_t k) -> pff_status {
        const bool solve = damage_every > 0 && k % damage_every == 0;
        m->su_tol = rel_tol; m->su_max_iter = max_iter;
        pff_status e = launch_step(m, s, bc, dt, solve && fuse ? /*MODE_STEPSU*/ 5 : /*MODE_STEP*/ 0, nullptr, nullptr, nullptr);
        if (e == PFF_OK && solve) e = damage_solve(m, s, rel_tol, max_iter, nullptr, nullptr);
        m->su_ready = false;
        return e;
    };
    const int64_t period = damage_every > 0 ? damage_every : 1;
    int64_t k = 1;
    // (the multigrid solver tests convergence on the host every iteration: its solves cannot be part of a captured period)
    const bool mg_solver = m->damage_solver == 1 && m->mg && damage_every > 0;
    const bool want_graph = m->graph_mode != 0 && !m->graph_unsupported && !m->prof_on && period <= 64 && n_steps >= 4 * period && !mg_solver;
    if (want_graph) {
        // key of everything a captured period depends on (kernel arguments are frozen at capture time)
        struct Key { pff_state s; pff_bc bc; double dt, tol; int32_t every, max_iter; int64_t n_dir; uint64_t flags_gen; int32_t variant, fuse; } key{};
        key.s = *s; if (bc) key.bc = *bc; else key.bc.load_scale = 1.0;
        key.dt = dt; key.tol = rel_tol; key.every = damage_every; key.max_iter = max_iter; key.n_dir = m->n_dir; key.flags_gen = m->flags_gen;
        key.variant = m->cg_variant;  // decides which CG kernel the frozen period launches
        key.fuse = fuse ? 1 : 0;
        const unsigned char* kb = reinterpret_cast<const unsigned char*>(&key);
        const bool cached = m->graph_exec && m->graph_key.size() == sizeof(Key) && std::memcmp(m->graph_key.data(), kb, sizeof(Key)) == 0;
        if (!cached) {
            if (m->graph_exec) { cudaGraphExecDestroy(m->graph_exec); m->graph_exec = nullptr; }
            for (; k <= period && st == PFF_OK; ++k) st = one_step(k);  // first period the ordinary way (also does every lazy allocation)
            if (st == PFF_OK) {
                const int64_t l0 = m->n_launches;
                cudaGraph_t graph = nullptr;
                // The period is recorded on a stream of the library's own (the caller's may be the legacy default stream,
                // which cannot capture); recording executes nothing, and the replays go to the caller's stream.
                cudaError_t ce = m->copy_stream ? cudaSuccess : cudaStreamCreateWithFlags(&m->copy_stream, cudaStreamNonBlocking);
                pff_status cst = PFF_OK;
                if (ce == cudaSuccess) ce = cudaStreamBeginCapture(m->copy_stream, cudaStreamCaptureModeThreadLocal);
                if (ce == cudaSuccess) {
                    cudaStream_t user = m->stream;
                    m->stream = m->copy_stream;
                    for (int64_t j = 1; j <= period && cst == PFF_OK; ++j) cst = one_step(j);
                    m->stream = user;
                    ce = cudaStreamEndCapture(m->copy_stream, &graph);
                }
                m->graph_launches = (int)(m->n_launches - l0);
                m->n_launches = l0;  // captured, not launched
                if (ce == cudaSuccess && cst == PFF_OK && graph) ce = cudaGraphInstantiate(&m->graph_exec, graph, 0);
                if (graph) cudaGraphDestroy(graph);
                if (ce != cudaSuccess || cst != PFF_OK || !m->graph_exec) {  // not capturable here: plain launches from now on
                    m->graph_refusal = ce != cudaSuccess ? cudaGetErrorString(ce) : pff_last_error();
                    cudaGetLastError();
                    m->graph_exec = nullptr; m->graph_unsupported = true;
                } else {
                    m->graph_key.assign(kb, kb + sizeof(Key));
                }
            }
        }
        if (st == PFF_OK && m->graph_exec) {
            for (; k + period - 1 <= n_steps && st == PFF_OK; k += period) {
                st = cuda_check(cudaGraphLaunch(m->graph_exec, m->stream), "pff_run_steps: graph launch");
                m->n_launches += m->graph_launches;
            }
        }
    }
    for (; k <= n_steps && st == PFF_OK; ++k) st = one_step(k);
    m->defer = false;
    pff_status e = cuda_check(cudaMemcpyAsync(m->h_tally, m->d_tally, sizeof(RunTally), cudaMemcpyDeviceToHost, m->stream), "pff_run_steps: tally");
    if (e == PFF_OK) e = cuda_check(cudaStreamSynchronize(m->stream), "pff_run_steps: sync");
    if (st != PFF_OK) return st;
    if (e != PFF_OK) return e;
    m->last_restarts = m->h_tally->restarts; m->last_truncs = m->h_tally->truncs;
    if (cg_iters_total) *cg_iters_total = m->h_tally->iters;
    if (m->h_tally->noconv > 0) { set_error("pff_run_steps: a damage solve reached max_iter"); return PFF_ENOCONV; }
    return PFF_OK;
}

pff_status pff_trace_set(pff_mesh* m, void* device_words, int32_t cg_iteration)
{
    if (!m) { set_error("pff_trace_set: null mesh"); return PFF_EINVAL; }
#ifdef PFF_TRACE
    m->d_trace = (long long*)device_words; m->trace_iter = cg_iteration;
    return PFF_OK;
#else
    (void)device_words; (void)cg_iteration;
    set_error("pff_trace_set: this build has no phase timestamps (build with python -m paper_2606_23458_b200.build --trace)");
    return PFF_EUNSUPPORTED;
#endif
}

pff_status pff_last_cg_kernel(const pff_mesh* m, int32_t* kernel)
{
    if (!m || !kernel) { set_error("pff_last_cg_kernel: null argument"); return PFF_EINVAL; }
    *kernel = m->last_cg_kernel;
    return PFF_OK;
}

pff_status pff_set_fused_setup(pff_mesh* m, int32_t enable)
{
    if (!m) { set_error("pff_set_fused_setup: null mesh"); return PFF_EINVAL; }
    m->fuse_setup = enable != 0;
    return PFF_OK;
}

pff_status pff_fused_setup_used(const pff_mesh* m, int32_t* used)
{
    if (!m || !used) { set_error("pff_fused_setup_used: null argument"); return PFF_EINVAL; }
    *used = m->last_step_fused;
    return PFF_OK;
}

pff_status pff_set_cg_variant(pff_mesh* m, int32_t variant)
{
    if (!m || variant < 0 || variant > 2) { set_error("pff_set_cg_variant: null mesh or variant not 0 / 1 / 2"); return PFF_EINVAL; }
    m->cg_variant = variant;
    return PFF_OK;
}

pff_status pff_graph_status(const pff_mesh* m, int32_t* captured, int32_t* refused)
{
    if (!m) { set_error("pff_graph_status: null mesh"); return PFF_EINVAL; }
    if (captured) *captured = m->graph_exec != nullptr;
    if (refused) *refused = m->graph_unsupported;
    if (m->graph_unsupported) set_error("graph capture refused: " + m->graph_refusal);  // readable through pff_last_error()
    return PFF_OK;
}

pff_status pff_set_graph_mode(pff_mesh* m, int32_t enable)
{
    if (!m) { set_error("pff_set_graph_mode: null mesh"); return PFF_EINVAL; }
    m->graph_mode = enable != 0;
    return PFF_OK;
}

pff_status pff_stiffness_action(pff_mesh* m, const pff_state* s, const void* px, const void* py, void* qx, void* qy)
{
    if (!m || !valid_state(s) || !px || !py || !qx || !qy) { set_error("pff_stiffness_action: null argument"); return PFF_EINVAL; }
    if ((reinterpret_cast<uintptr_t>(px) | reinterpret_cast<uintptr_t>(py)) & 15) {
        set_error("pff_stiffness_action: px, py must be 16-byte aligned"); return PFF_EINVAL;
    }
    DeviceGuard dg(m);
    return launch_step(m, const_cast<pff_state*>(s), nullptr, 0.0, /*MODE_TANGENT*/ 3, qx, qy, nullptr, px, py);
}

pff_status pff_equilibrium_solve(pff_mesh* m, pff_state* s, const pff_bc* bc, double rel_tol, int32_t max_iter, int32_t* iters,
                                 double* relres)
{
    if (!m || !valid_state(s)) { set_error("pff_equilibrium_solve: null mesh, null or misaligned (16 B) state pointer"); return PFF_EINVAL; }
    if (!(rel_tol > 0) || max_iter < 1) { set_error("pff_equilibrium_solve: need rel_tol > 0, max_iter >= 1"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return equilibrium_solve(m, s, bc, rel_tol, max_iter, iters, relres);
}

pff_status pff_damage_adjoint(pff_mesh* m, const pff_state* s, const void* g, const uint8_t* free_mask, void* lambda, double rel_tol,
                              int32_t max_iter, int32_t* iters, double* relres)
{
    if (!m || !valid_state(s) || !g || !lambda || (reinterpret_cast<uintptr_t>(lambda) & 15)) {
        set_error("pff_damage_adjoint: null mesh / state / g / lambda, or lambda not 16-byte aligned");
        return PFF_EINVAL;
    }
    if (!(rel_tol > 0) || max_iter < 1) { set_error("pff_damage_adjoint: need rel_tol > 0, max_iter >= 1"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return damage_adjoint(m, s, g, free_mask, lambda, rel_tol, max_iter, iters, relres);
}

pff_status pff_damage_param_terms(pff_mesh* m, const void* lambda, const void* d, double out[2])
{
    if (!m || !lambda || !d || !out) { set_error("pff_damage_param_terms: null argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return damage_param_terms(m, lambda, d, out);
}

pff_status pff_damage_matvec(pff_mesh* m, const pff_state* s, const void* p, void* q)
{
    if (!m || !valid_state(s) || !p || !q) { set_error("pff_damage_matvec: null argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return damage_matvec(m, s, p, q);
}

pff_status pff_damage_rhs_diag(pff_mesh* m, const pff_state* s, void* b, void* D)
{
    if (!m || !valid_state(s)) { set_error("pff_damage_rhs_diag: null argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return damage_rhs_diag(m, s, b, D);
}

pff_status pff_mesh_counters(const pff_mesh* m, int64_t* kernel_launches)
{
    if (!m || !kernel_launches) { set_error("pff_mesh_counters: null argument"); return PFF_EINVAL; }
    *kernel_launches = m->n_launches;
    return PFF_OK;
}

pff_status pff_profile_enable(pff_mesh* m, int32_t enable)
{
    if (!m) { set_error("pff_profile_enable: null mesh"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    PFF_CUDA(cudaStreamSynchronize(m->stream));
    m->prof_on = enable != 0;
    for (auto& u : m->prof_used) u = 0;
    return PFF_OK;
}

pff_status pff_profile_read(pff_mesh* m, double* ms_sum, int64_t* launches)
{
    if (!m || !ms_sum || !launches) { set_error("pff_profile_read: null argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    PFF_CUDA(cudaStreamSynchronize(m->stream));
    for (int c = 0; c < PFF_NUM_KERNEL_CLASSES; ++c) {
        double sum = 0.0;
        for (size_t k = 0; k + 1 < m->prof_used[c]; k += 2) {
            float ms = 0.f;
            PFF_CUDA(cudaEventElapsedTime(&ms, m->prof_ev[c][k], m->prof_ev[c][k + 1]));
            sum += ms;
        }
        ms_sum[c] = sum;
        launches[c] = (int64_t)(m->prof_used[c] / 2);
        m->prof_used[c] = 0;
    }
    return PFF_OK;
}

pff_status pff_time_kernel(pff_mesh* m, pff_state* s, int32_t which, int32_t reps, float* ms_per_launch)
{
    if (!m || !valid_state(s) || !ms_per_launch || reps < 1 || which < 0 || which > 3) {
        set_error("pff_time_kernel: bad argument"); return PFF_EINVAL;
    }
    if (m->opt.scatter != PFF_SCATTER_GATHER && which >= 2) { set_error("pff_time_kernel: gather meshes only"); return PFF_EUNSUPPORTED; }
    DeviceGuard dg(m);
    cudaEvent_t e0, e1;
    PFF_CUDA(cudaEventCreate(&e0));
    PFF_CUDA(cudaEventCreate(&e1));
    pff_bc bc{nullptr, nullptr, 1.0};
    pff_status st = PFF_OK;
    m->only_kernel = which;
    // one untimed launch (attribute setup, instruction cache), then the timed train
    for (int pass = 0; pass < 2 && st == PFF_OK; ++pass) {
        const int n = pass == 0 ? 1 : reps;
        if (pass == 1) cudaEventRecord(e0, m->stream);
        for (int k = 0; k < n && st == PFF_OK; ++k) {
            if (which < 2) st = launch_step(m, s, &bc, 1e-12 * m->dt_crit, 0, nullptr, nullptr, nullptr);
            else st = damage_matvec(m, s, s->d, m->d_q);
        }
    }
    cudaEventRecord(e1, m->stream);
    m->only_kernel = -1;
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (st != PFF_OK) return st;
    PFF_CUDA(e);
    *ms_per_launch = ms / float(reps);
    return PFF_OK;
}

pff_status pff_energies(pff_mesh* m, const pff_state* s, double out[4])
{
    if (!m || !valid_state(s) || !out) { set_error("pff_energies: null argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return energies(m, s, out);
}

pff_status pff_mg_attach(pff_mesh* m, int32_t n_coarse, pff_mesh* const* coarse)
{
    if (!m || n_coarse < 0 || n_coarse > 16 || (n_coarse > 0 && !coarse)) { set_error("pff_mg_attach: null mesh or n_coarse outside 0..16"); return PFF_EINVAL; }
    if (m->opt.scatter != PFF_SCATTER_GATHER) { set_error("pff_mg_attach: gather meshes only"); return PFF_EUNSUPPORTED; }
    DeviceGuard dg(m);
    return mg_attach(m, n_coarse, coarse);
}

pff_status pff_set_damage_solver(pff_mesh* m, int32_t solver)
{
    if (!m || solver < 0 || solver > 1) { set_error("pff_set_damage_solver: null mesh or solver not 0 / 1"); return PFF_EINVAL; }
    if (solver == 1 && !m->mg) { set_error("pff_set_damage_solver: no hierarchy attached (pff_mg_attach)"); return PFF_EINVAL; }
    m->damage_solver = solver;
    return PFF_OK;
}

pff_status pff_mg_set_params(pff_mesh* m, double omega, int32_t coarse_sweeps)
{
    if (!m) { set_error("pff_mg_set_params: null mesh"); return PFF_EINVAL; }
    return mg_set_params(m, omega, coarse_sweeps);
}

pff_status pff_mg_apply(pff_mesh* m, const pff_state* s, const void* r, void* z)
{
    if (!m || !valid_state(s) || !r || !z) { set_error("pff_mg_apply: null argument"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return mg_apply(m, s, r, z);
}

pff_status pff_damage_solve_mg(pff_mesh* m, pff_state* s, double rel_tol, int32_t max_iter, int32_t* iters, double* relres)
{
    if (!m || !valid_state(s)) { set_error("pff_damage_solve_mg: null mesh, null or misaligned (16 B) state pointer"); return PFF_EINVAL; }
    if (!(rel_tol > 0) || max_iter < 1) { set_error("pff_damage_solve_mg: need rel_tol > 0, max_iter >= 1"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return mg_solve(m, s, rel_tol, max_iter, iters, relres);
}

pff_status pff_energies_static(pff_mesh* m, const pff_state* s, double* out_device)
{
    if (!m || !valid_state(s) || !out_device) { set_error("pff_energies_static: null argument"); return PFF_EINVAL; }
    if (reinterpret_cast<uintptr_t>(out_device) % 8) { set_error("pff_energies_static: out_device must be 8-byte aligned"); return PFF_EINVAL; }
    DeviceGuard dg(m);
    return energies_static(m, s, out_device);
}

}  // extern "C"
