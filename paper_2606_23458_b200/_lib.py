"""ctypes loader of libpff.so and the raw C-ABI prototypes of include/pff.h (same names)."""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libpff.so")

PFF_OK, PFF_EINVAL, PFF_EMESH, PFF_ENOMEM, PFF_ECUDA, PFF_ENOCONV, PFF_EUNSUPPORTED = range(7)
PFF_AT1, PFF_AT2 = 1, 2
PFF_SPLIT_ISOTROPIC, PFF_SPLIT_SPECTRAL, PFF_SPLIT_VOLDEV, PFF_SPLIT_STARCONVEX = 0, 1, 2, 3
PFF_PLANE_STRAIN, PFF_PLANE_STRESS = 0, 1
PFF_F64, PFF_F32 = 0, 1
PFF_SCATTER_GATHER, PFF_SCATTER_ATOMIC = 0, 1
PFF_ORDER_NONE, PFF_ORDER_MORTON, PFF_ORDER_BISECTION = 0, 1, 2
KERNEL_CLASSES = ("step_chunk", "step_shared", "matvec_chunk", "matvec_shared", "damage_setup", "other")

# every symbol include/pff.h declares
SYMBOLS = [
    "pff_mesh_create", "pff_mesh_plan", "pff_mesh_destroy", "pff_mesh_info", "pff_mesh_permutations", "pff_set_dirichlet",
    "pff_set_damage_dirichlet", "pff_set_traction", "pff_init_accel", "pff_explicit_step", "pff_damage_solve",
    "pff_energies", "pff_set_fused_setup", "pff_fused_setup_used", "pff_energies_static", "pff_mg_attach", "pff_set_damage_solver", "pff_mg_set_params", "pff_damage_solve_mg", "pff_mg_apply", "pff_set_cg_variant", "pff_last_cg_kernel", "pff_damage_last_stats", "pff_subcycle_limit", "pff_run_steps", "pff_set_graph_mode", "pff_graph_status", "pff_damage_adjoint", "pff_damage_param_terms", "pff_stiffness_action", "pff_equilibrium_solve", "pff_internal_force", "pff_damage_matvec", "pff_damage_rhs_diag", "pff_run_host", "pff_mesh_counters", "pff_time_kernel",
    "pff_profile_enable", "pff_profile_read", "pff_trace_set",
    "pff_last_error",
]


class pff_material(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("E", "nu", "rho", "Gc", "l0", "eta", "gamma_star")] + [
        (k, C.c_int32) for k in ("model", "split", "plane")]


class pff_options(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("precision", "order", "scatter", "chunk_elems")]


class pff_state(C.Structure):
    _fields_ = [(k, C.c_void_p) for k in ("ux", "uy", "vx", "vy", "ax", "ay", "d", "H", "fext_x", "fext_y")]


class pff_bc(C.Structure):
    _fields_ = [("dir_u", C.c_void_p), ("dir_v", C.c_void_p), ("load_scale", C.c_double)]


class pff_host_state(C.Structure):
    _fields_ = [(k, C.POINTER(C.c_double)) for k in ("u", "v", "a", "d", "H", "fext")]


_lib = None


def load() -> C.CDLL:
    """Load libpff.so; there is NO fallback: a missing library is an error.  PFF_LIBRARY in the environment selects another
    build of the same library (the instrumentation build libpff_trace.so)."""
    global _lib, LIB_PATH
    if _lib is not None:
        return _lib
    LIB_PATH = os.environ.get("PFF_LIBRARY", LIB_PATH)
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} not found: build it with `python -m paper_2606_23458_b200.build` "
            "(nvcc, sm_100a). There is no CPU or PyTorch fallback for the pff hot path.")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32 = C.c_void_p, C.c_int64, C.c_int32
    dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
    L.pff_mesh_create.argtypes = [i64, vp, i64, vp, C.POINTER(pff_material), C.POINTER(pff_options), vp, C.POINTER(vp)]
    L.pff_mesh_plan.argtypes = [i64, vp, i64, vp, C.POINTER(pff_options), vp, vp, C.POINTER(i64), C.POINTER(i64), ip, ip, dp]
    L.pff_mesh_destroy.argtypes = [vp]
    L.pff_mesh_destroy.restype = None
    L.pff_mesh_info.argtypes = [vp, C.POINTER(i64), C.POINTER(i64), dp, dp, C.POINTER(i64), C.POINTER(i64)]
    L.pff_mesh_permutations.argtypes = [vp, vp, vp]
    L.pff_set_dirichlet.argtypes = [vp, i64, vp]
    L.pff_set_damage_dirichlet.argtypes = [vp, i64, vp]
    L.pff_set_traction.argtypes = [vp, C.POINTER(pff_state), i64, vp, vp]
    L.pff_init_accel.argtypes = [vp, C.POINTER(pff_state), C.POINTER(pff_bc)]
    L.pff_explicit_step.argtypes = [vp, C.POINTER(pff_state), C.POINTER(pff_bc), C.c_double]
    L.pff_damage_solve.argtypes = [vp, C.POINTER(pff_state), C.c_double, i32, ip, dp]
    L.pff_energies.argtypes = [vp, C.POINTER(pff_state), dp]
    L.pff_energies_static.argtypes = [vp, C.POINTER(pff_state), vp]
    L.pff_mg_attach.argtypes = [vp, i32, C.POINTER(vp)]
    L.pff_mg_set_params.argtypes = [vp, C.c_double, i32]
    L.pff_set_damage_solver.argtypes = [vp, i32]
    L.pff_damage_solve_mg.argtypes = [vp, C.POINTER(pff_state), C.c_double, i32, ip, dp]
    L.pff_mg_apply.argtypes = [vp, C.POINTER(pff_state), vp, vp]
    L.pff_damage_last_stats.argtypes = [vp, ip, ip]
    L.pff_set_cg_variant.argtypes = [vp, i32]
    L.pff_set_fused_setup.argtypes = [vp, i32]
    L.pff_fused_setup_used.argtypes = [vp, C.POINTER(i32)]
    L.pff_last_cg_kernel.argtypes = [vp, ip]
    L.pff_subcycle_limit.argtypes = [C.POINTER(pff_material), ip, dp]
    L.pff_run_steps.argtypes = [vp, C.POINTER(pff_state), C.POINTER(pff_bc), C.c_double, i64, i32, C.c_double, i32, C.POINTER(i64)]
    L.pff_set_graph_mode.argtypes = [vp, i32]
    L.pff_graph_status.argtypes = [vp, ip, ip]
    L.pff_internal_force.argtypes = [vp, C.POINTER(pff_state), vp, vp, vp]
    L.pff_damage_matvec.argtypes = [vp, C.POINTER(pff_state), vp, vp]
    L.pff_damage_adjoint.argtypes = [vp, C.POINTER(pff_state), vp, vp, vp, C.c_double, i32, ip, dp]
    L.pff_damage_param_terms.argtypes = [vp, vp, vp, dp]
    L.pff_stiffness_action.argtypes = [vp, C.POINTER(pff_state), vp, vp, vp, vp]
    L.pff_equilibrium_solve.argtypes = [vp, C.POINTER(pff_state), C.POINTER(pff_bc), C.c_double, i32, ip, dp]
    L.pff_damage_rhs_diag.argtypes = [vp, C.POINTER(pff_state), vp, vp]
    L.pff_run_host.argtypes = [vp, C.POINTER(pff_host_state), vp, vp, C.c_double, C.c_double, i64, i32, C.c_double, i32]
    L.pff_mesh_counters.argtypes = [vp, C.POINTER(i64)]
    L.pff_time_kernel.argtypes = [vp, C.POINTER(pff_state), i32, i32, C.POINTER(C.c_float)]
    L.pff_profile_enable.argtypes = [vp, i32]
    L.pff_profile_read.argtypes = [vp, dp, C.POINTER(i64)]
    L.pff_trace_set.argtypes = [vp, vp, i32]
    L.pff_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        if name not in ("pff_mesh_destroy", "pff_last_error"):
            getattr(L, name).restype = C.c_int
    _lib = L
    return L
