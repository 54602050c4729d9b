// The opaque pff_mesh object: host tables + device copies + workspaces.
#pragma once
#include <cuda_runtime.h>

#include <string>
#include <unordered_map>
#include <vector>

#include "pff_internal.h"

// device-resident control block of the CG recurrence (pff_damage.cu); one 128-byte read-back per solve
struct DamageCtrl {
    double rz, alpha, beta, amax, nb, tol, relres;
    int iters, max_iter, done, status, first, restart, trunc, pending;
    int restarts;  // AT1: free-set re-derivations after the first (a bound became inactive / a step was truncated, L181)
    int truncs;    // AT1: steps cut short at the first bound hit
};

// counters of all solves of one pff_run_steps call (device-resident, added to by the last phase of the CG kernel)
struct RunTally {
    long long iters;
    int solves, noconv, restarts, truncs;
};
static_assert(sizeof(DamageCtrl) % 8 == 0, "the control block is copied in 8-byte words");

// Outputs of the damage setup pass when the explicit-step kernel performs it as well (pff_step.cu MODE_STEPSU); filled in
// by damage_fused_setup (pff_damage.cu) with exactly the buffers and options the next damage_solve will use.
struct FusedSetup {
    void *ca, *cb;            // operator coefficients of the solve
    void *r, *dinv, *lb;      // first residual, Jacobi diagonal (inverse), lower bound d_n
    uint8_t* mask;
    void* part3;              // [3][n_slots] reals: per (chunk, interface node) partials of A d_n, D, b
    double* part;             // [kCh][part_n] block partials of the norms
    int64_t part_n;
    unsigned int* ticket;     // the damage workspace's tickets ([0] last block, [1] CG barrier counter)
    DamageCtrl* ctrl;
    double tol;
    int max_iter, zero_dinv_fixed;
};

struct pff_mesh {
    pff::HostMesh hm;
    pff_material mat{};
    pff_options opt{};
    cudaStream_t stream = nullptr;
    int device = 0;
    size_t rb = 8;  // bytes per real
    double dt_crit = 0.0;
    pff::StageLayout lay_step{}, lay_stepsu{}, lay_mv{}, lay_su{}, lay_eq{};  // shared-memory stages of the step / CG iteration / setup / quasi-static CG kernels
    int64_t ell_total = 0;                       // entries of d_ell (padded)
    int64_t n_launches = 0;  // kernels launched so far (pff_mesh_counters)
    long long* d_trace = nullptr;  // pff_trace_set (instrumentation build)
    int trace_iter = 3;
    void* mg = nullptr;      // multigrid hierarchy attached to this (finest) mesh: pff_multigrid.cu
    // fused explicit step + damage setup (pff_run_steps): option, the partial planes of the fused setup, and what the last
    // fused launch prepared (consumed by the next damage_solve, which then skips its own setup kernel)
    int fuse_setup = 1;
    void* d_su_part = nullptr;
    bool su_ready = false;
    double su_tol = 0.0;
    int su_max_iter = 0, su_zero_dinv = 0;
    int last_step_fused = 0;
    int damage_solver = 0;   // pff_set_damage_solver: 0 Jacobi-PCG kernels, 1 multigrid-preconditioned CG (AT2, hierarchy attached)
    int only_kernel = -1;    // profiling hook: restrict multi-kernel entry points to one kernel (pff_time_kernel)
    // launch configuration of every persistent chunk kernel this mesh has used, keyed by the kernel's address: the grid
    // (CTAs that fit the mesh's device with this mesh's shared-memory stage).  Presence also means the dynamic
    // shared-memory opt-in was made on that device.  Per mesh, so meshes on different GPUs or with different chunk sizes
    // never see each other's values.  A mesh must not be driven from two host threads at once.
    std::unordered_map<const void*, int> launch_grid;
    // per-kernel-class CUDA-event timing (pff_profile_enable / pff_profile_read)
    bool prof_on = false;
    std::vector<cudaEvent_t> prof_ev[PFF_NUM_KERNEL_CLASSES];  // start/stop pairs
    size_t prof_used[PFF_NUM_KERNEL_CLASSES] = {};

    // device mesh tables
    pff::ChunkMeta* d_meta = nullptr;
    void* d_lconn = nullptr;  // ushort4[Ne]
    void* d_conn = nullptr;   // int4[Ne]
    void *d_ga = nullptr, *d_gb = nullptr, *d_area = nullptr, *d_minv = nullptr, *d_mass = nullptr;
    int32_t *d_halo_ids = nullptr, *d_sh_rowptr = nullptr, *d_halo_dst = nullptr;
    uint16_t* d_ell = nullptr;
    uint8_t* d_flags = nullptr;  // bit0: u_x Dirichlet, bit1: u_y Dirichlet, bit2: damage Dirichlet
    void* d_halo_part = nullptr;  // [3][n_slots] reals: per (chunk, interface node) partial sums
    int64_t n_slots = 0;    // partial slots per plane: kIfaceWidth per interface node + overflow
    int64_t n_entries = 0;  // (chunk, halo node) entries = length of d_halo_ids / d_halo_dst
    void *d_fwx = nullptr, *d_fwy = nullptr;  // atomic-scatter force accumulators (kept zero between steps)

    // Dirichlet set
    int64_t n_dir = 0;
    int32_t* d_dir_dof = nullptr;  // internal node * 2 + comp
    std::vector<uint8_t> h_flags;

    // damage solve workspaces (reals [N] unless noted)
    void *d_lb = nullptr, *d_r = nullptr, *d_p = nullptr, *d_q = nullptr, *d_dinv = nullptr;
    // element operator of the current solve, 4 reals per element (mass coefficient m_e and the three edge weights w_12,
    // w_13, w_23 of the P1 stiffness): fp64 two double2 streams, fp32 one float4 stream (written by the setup pass)
    void *d_ca = nullptr, *d_cb = nullptr;
    void* d_cg2 = nullptr;       // second set of x, r, p, s and both sets of w of the one-rendezvous CG kernel (6 vectors)
    int last_cg_kernel = 0;      // which kernel the last solve launched (1 two-rendezvous, 2 one-rendezvous)
    int cg_variant = 0;          // 0: pick per solve; 1: always the two-rendezvous kernel; 2: the one-rendezvous kernel wherever it applies
    uint8_t* d_mask = nullptr;   // [N] bit0: in the free set, bit1: damage-Dirichlet
    double* d_part = nullptr;    // chunk-kernel block partials [channels][n_part_blocks]
    int64_t n_part_blocks = 0;
    DamageCtrl* d_ctrl = nullptr;  // initialised on the device by the setup kernel of every solve (no host upload)
    DamageCtrl* h_ctrl = nullptr;  // pinned download image of the last synchronous solve
    int last_restarts = 0, last_truncs = 0;  // of the last pff_damage_solve, or summed over the last pff_run_steps
    // pff_run_steps: every solve adds its counters to a device-resident tally instead of being read back (no host round
    // trip per solve, and the launches can be replayed from a CUDA graph); the host reads the tally once at the end
    RunTally* d_tally = nullptr;
    RunTally* h_tally = nullptr;  // pinned
    bool defer = false;           // true inside pff_run_steps: damage_solve tallies on the device and does not synchronise
    // one captured period of pff_run_steps (damage_every explicit steps + one solve) and the arguments it was captured with
    cudaGraphExec_t graph_exec = nullptr;
    std::vector<unsigned char> graph_key;
    uint64_t flags_gen = 0;       // bumped by pff_set_dirichlet / pff_set_damage_dirichlet
    int graph_launches = 0;       // kernel launches one replay stands for
    int graph_mode = 1;           // 0: never capture (pff_set_graph_mode); 1: capture when a run has enough periods
    std::string graph_refusal;    // why
    bool graph_unsupported = false;  // capture of a cooperative launch was refused once on this driver: do not try again
    unsigned int* d_ticket = nullptr;
    // quasi-static mechanics solve (pff_equilibrium.cu), allocated at its first call
    int32_t *d_n2e_ptr = nullptr, *d_n2e = nullptr;  // node -> (4 * element + corner) table
    void* d_eq_vec = nullptr;                        // 10 nodal vectors
    double* d_eq_part = nullptr;                     // block partials [kCh][grid] of the fused CG iteration
    DamageCtrl *d_eq_ctrl = nullptr, *h_eq_ctrl = nullptr;  // its recurrence scalars (device; pinned read-back image)
    unsigned int* d_eq_ticket = nullptr;
    struct { void *ex, *ey, *rx, *ry, *dix, *diy; } eq{};  // CG vectors of the running quasi-static solve (MODE_EQ launches)
    int last_step_grid = 0;             // CTAs of the last step-kernel launch
    unsigned int* d_step_bar = nullptr;  // [0] grid-barrier counter of the step kernel, [1] its epoch (both device-maintained)

    // host-path staging (pff_run_host)
    cudaStream_t copy_stream = nullptr;  // second stream: copies the mechanics results back while the damage solve runs
    cudaEvent_t ev_step = nullptr, ev_out = nullptr;  // pff_run_host: step done (copy stream waits) / permutation done (mesh stream waits)
    void* d_stage = nullptr; size_t stage_bytes = 0;
    void* d_hstate = nullptr;  // device state arrays owned by the library for pff_run_host
    void* d_hdir = nullptr;    // its Dirichlet values (dir_u | dir_v), re-allocated when the Dirichlet set outgrows it
    int64_t hdir_cap = 0;      // entries per half of d_hdir
    int32_t *d_node_old_of_new = nullptr, *d_elem_old_of_new = nullptr;
};

namespace pff {
// Event bracket around one launch of kernel class `cls` (no-ops unless profiling is enabled).
inline void prof_mark(pff_mesh* m, int cls)
{
    if (!m->prof_on) return;
    auto& v = m->prof_ev[cls];
    if (m->prof_used[cls] == v.size()) { cudaEvent_t e; cudaEventCreate(&e); v.push_back(e); }
    cudaEventRecord(v[m->prof_used[cls]++], m->stream);
}
#define PFF_LAUNCH(m, cls, ...)            \
    do {                                   \
        pff::prof_mark((m), (cls));        \
        __VA_ARGS__;                       \
        pff::prof_mark((m), (cls));        \
        ++(m)->n_launches;                 \
    } while (0)
// implemented in pff_step.cu / pff_damage.cu / pff_energy.cu
pff_status launch_step(pff_mesh* m, pff_state* s, const pff_bc* bc, double dt, int mode, void* fx, void* fy, void* psi,
                       const void* px = nullptr, const void* py = nullptr);
pff_status damage_solve(pff_mesh* m, pff_state* s, double rel_tol, int max_iter, int* iters, double* relres);
pff_status damage_matvec(pff_mesh* m, const pff_state* s, const void* p, void* q, bool refresh_coef = true, bool skip_interface = false);
pff_status damage_refresh_coef(pff_mesh* m, const pff_state* s);
pff_status damage_fused_setup(pff_mesh* m, FusedSetup* fs);  // tolerance / iteration cap: m->su_tol, m->su_max_iter
bool fused_setup_ok(const pff_mesh* m);
// pff_multigrid.cu: geometric-multigrid-preconditioned CG for the AT2 damage solve
pff_status mg_attach(pff_mesh* m, int n_coarse, pff_mesh* const* coarse);
pff_status mg_apply(pff_mesh* m, const pff_state* s, const void* r, void* z);
pff_status mg_solve(pff_mesh* m, pff_state* s, double rel_tol, int max_iter, int* iters, double* relres);
pff_status mg_set_params(pff_mesh* m, double omega, int coarse_sweeps);
pff_status mg_adjoint(pff_mesh* m, const pff_state* s, const void* g, const uint8_t* free_mask, void* lambda, double rel_tol,
                      int max_iter, int* iters, double* relres);
void mg_free(pff_mesh* m);
pff_status damage_adjoint(pff_mesh* m, const pff_state* s, const void* g, const uint8_t* free_mask, void* lambda, double rel_tol,
                          int max_iter, int* iters, double* relres);
pff_status damage_param_terms(pff_mesh* m, const void* lambda, const void* d, double out[2]);
pff_status equilibrium_solve(pff_mesh* m, pff_state* s, const pff_bc* bc, double rel_tol, int max_iter, int* iters, double* relres);
pff_status damage_rhs_diag(pff_mesh* m, const pff_state* s, void* b, void* D);
pff_status energies(pff_mesh* m, const pff_state* s, double out[4]);
pff_status energies_static(pff_mesh* m, const pff_state* s, double* out_device);  // block partials in a static device array
pff_status energy_static_scratch(double** ptr);  // device address of that array on the CURRENT device (cached per device)
pff_status cuda_check(cudaError_t e, const char* what);
// Cooperative launch (all CTAs co-resident: the kernels synchronise grid-wide) through the extensible launch API with the
// cooperative attribute: unlike the legacy cooperative-launch entry point it can be captured into a CUDA graph.
inline cudaError_t launch_cooperative(const void* kern, unsigned grid, unsigned block, void** args, size_t smem, cudaStream_t stream)
{
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(block); cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr{};
    attr.id = cudaLaunchAttributeCooperative;
    attr.val.cooperative = 1;
    cfg.attrs = &attr; cfg.numAttrs = 1;
    return cudaLaunchKernelExC(&cfg, kern, args);
}
// dynamic shared-memory opt-in + occupancy-derived persistent grid of `kern` for this mesh (cached in m->launch_grid)
pff_status persistent_config(pff_mesh* m, const void* kern, int smem_bytes, int* grid, int block = 256);

// Makes the mesh's device current for the duration of an entry point (the caller may have switched devices since
// pff_mesh_create) and restores the caller's device afterwards.
struct DeviceGuard {
    int prev = -1;
    bool switched = false;
    explicit DeviceGuard(const pff_mesh* m)
    {
        if (m && cudaGetDevice(&prev) == cudaSuccess && prev != m->device) switched = cudaSetDevice(m->device) == cudaSuccess;
    }
    ~DeviceGuard() { if (switched) cudaSetDevice(prev); }
    DeviceGuard(const DeviceGuard&) = delete;
    DeviceGuard& operator=(const DeviceGuard&) = delete;
};
}  // namespace pff
