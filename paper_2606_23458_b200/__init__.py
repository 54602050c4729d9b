"""paper_2606_23458_b200 -- B200-native explicit phase-field fracture hot path (arxiv/paper_2606_23458).

Thin Python binding over the C-ABI library libpff.so (include/pff.h).  The methods below have the names
of the C entry points and only marshal arguments: every step of the method runs in the CUDA kernels of
csrc/.  PyTorch is used for device memory and streams only.  There is no CPU fallback: importing works
without a GPU (so the library can be inspected), creating a Mesh does not.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import _lib
from ._lib import (PFF_AT1, PFF_AT2, PFF_ENOCONV, PFF_F32, PFF_F64, PFF_OK, PFF_ORDER_BISECTION, PFF_ORDER_MORTON,  # noqa: F401
                   PFF_ORDER_NONE,
                   PFF_PLANE_STRAIN, PFF_PLANE_STRESS, PFF_SCATTER_ATOMIC, PFF_SCATTER_GATHER,
                   PFF_SPLIT_ISOTROPIC, PFF_SPLIT_SPECTRAL, PFF_SPLIT_STARCONVEX, PFF_SPLIT_VOLDEV)


class PffError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"pff status {status}: {msg}")
        self.status = status


def _check(status: int, allow=()):
    if status != PFF_OK and status not in allow:
        raise PffError(status, _lib.load().pff_last_error().decode())
    return status


class State:
    """Caller-owned device state in INTERNAL order (torch tensors) + the pff_state struct pointing at it."""

    FIELDS = ("ux", "uy", "vx", "vy", "ax", "ay", "d", "H", "fext_x", "fext_y")

    def __init__(self, mesh: "Mesh"):
        import torch
        dt = mesh.dtype
        for k in self.FIELDS:
            n = mesh.n_elems if k == "H" else mesh.n_nodes
            setattr(self, k, torch.zeros(n, dtype=dt, device=mesh.device))
        self.c = _lib.pff_state(*[getattr(self, k).data_ptr() for k in self.FIELDS])


class Mesh:
    """pff_mesh handle.  Host index sets are in USER numbering; device vectors in internal order."""

    def __init__(self, xy, tri, material: dict, precision=PFF_F64, order=PFF_ORDER_BISECTION,
                 scatter=PFF_SCATTER_GATHER, chunk_elems=0, device="cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2606_23458_b200 needs a CUDA device (no CPU fallback)")
        self.L = _lib.load()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.dtype = torch.float32 if precision == PFF_F32 else torch.float64
        self.np_dtype = np.float32 if precision == PFF_F32 else np.float64
        xy = np.ascontiguousarray(xy, dtype=np.float64)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        self.material = _lib.pff_material(**material)
        opt = _lib.pff_options(precision, order, scatter, chunk_elems)
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        _check(self.L.pff_mesh_create(len(xy), xy.ctypes.data, len(tri), tri.ctypes.data, C.byref(self.material),
                                      C.byref(opt), C.c_void_p(self.stream.cuda_stream), C.byref(h)))
        self.h = h
        nn, ne, nc, ns = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int64()
        hm, dtc = C.c_double(), C.c_double()
        _check(self.L.pff_mesh_info(h, C.byref(nn), C.byref(ne), C.byref(hm), C.byref(dtc), C.byref(nc), C.byref(ns)))
        self.n_nodes, self.n_elems, self.h_min, self.dt_crit = nn.value, ne.value, hm.value, dtc.value
        self.n_chunks, self.n_shared = nc.value, ns.value
        self.node_new_of_old = np.empty(self.n_nodes, dtype=np.int32)
        self.elem_new_of_old = np.empty(self.n_elems, dtype=np.int32)
        _check(self.L.pff_mesh_permutations(h, self.node_new_of_old.ctypes.data, self.elem_new_of_old.ctypes.data))
        self.n_dir = 0

    def __del__(self):
        h = getattr(self, "h", None)
        if h:
            self.L.pff_mesh_destroy(h)
            self.h = None

    # -- numbering helpers (pure permutation, no arithmetic) -----------------------------------
    def nodes_to_internal(self, a_user):
        import torch
        a = np.asarray(a_user)
        out = np.empty_like(a, dtype=self.np_dtype)
        out[self.node_new_of_old] = a
        return torch.from_numpy(out).to(self.device)

    def nodes_to_user(self, t):
        return t.detach().cpu().numpy().astype(np.float64)[self.node_new_of_old]

    def elems_to_internal(self, a_user):
        import torch
        out = np.empty(self.n_elems, dtype=self.np_dtype)
        out[self.elem_new_of_old] = np.asarray(a_user)
        return torch.from_numpy(out).to(self.device)

    def elems_to_user(self, t):
        return t.detach().cpu().numpy().astype(np.float64)[self.elem_new_of_old]

    def new_state(self, u=None, v=None, a=None, d=None, H=None, fext=None) -> State:
        s = State(self)
        for name, arr in (("u", u), ("v", v), ("a", a), ("fext_", fext)):
            if arr is not None:
                arr = np.asarray(arr)
                getattr(s, name + "x").copy_(self.nodes_to_internal(arr[:, 0]))
                getattr(s, name + "y").copy_(self.nodes_to_internal(arr[:, 1]))
        if d is not None:
            s.d.copy_(self.nodes_to_internal(d))
        if H is not None:
            s.H.copy_(self.elems_to_internal(H))
        return s

    def bc(self, dir_u=None, dir_v=None, load_scale=1.0):
        """pff_bc from host arrays (ordered like the pff_set_dirichlet dof list); keeps the tensors alive."""
        import torch
        b = _lib.pff_bc(None, None, float(load_scale))
        if dir_u is not None and dir_v is not None and self.n_dir:
            tu = torch.as_tensor(np.asarray(dir_u, dtype=self.np_dtype), device=self.device)
            tv = torch.as_tensor(np.asarray(dir_v, dtype=self.np_dtype), device=self.device)
            b.dir_u, b.dir_v = tu.data_ptr(), tv.data_ptr()
            b._keep = (tu, tv)
        return b

    # -- C entry points ------------------------------------------------------------------------
    def pff_set_dirichlet(self, dir_dof):
        d = np.ascontiguousarray(dir_dof, dtype=np.int32)
        _check(self.L.pff_set_dirichlet(self.h, len(d), d.ctypes.data))
        self.n_dir = len(d)

    def pff_set_damage_dirichlet(self, nodes):
        d = np.ascontiguousarray(nodes, dtype=np.int32)
        _check(self.L.pff_set_damage_dirichlet(self.h, len(d), d.ctypes.data))

    def pff_set_traction(self, state: State, edge_nodes, t):
        e = np.ascontiguousarray(edge_nodes, dtype=np.int32)
        tt = np.ascontiguousarray(t, dtype=np.float64)
        _check(self.L.pff_set_traction(self.h, C.byref(state.c), len(e), e.ctypes.data, tt.ctypes.data))

    def pff_init_accel(self, state: State, bc=None):
        _check(self.L.pff_init_accel(self.h, C.byref(state.c), C.byref(bc) if bc is not None else None))

    def pff_explicit_step(self, state: State, bc, dt: float):
        _check(self.L.pff_explicit_step(self.h, C.byref(state.c), C.byref(bc) if bc is not None else None, dt))

    def pff_damage_solve(self, state: State, rel_tol=1e-8, max_iter=1000, allow_noconv=False):
        it, rr = C.c_int32(0), C.c_double(0.0)
        st = _check(self.L.pff_damage_solve(self.h, C.byref(state.c), rel_tol, max_iter, C.byref(it), C.byref(rr)),
                    allow=(PFF_ENOCONV,) if allow_noconv else ())
        return st, it.value, rr.value

    def pff_set_fused_setup(self, enable: bool):
        _check(self.L.pff_set_fused_setup(self.h, int(bool(enable))))

    def pff_fused_setup_used(self) -> bool:
        k = C.c_int32(0)
        _check(self.L.pff_fused_setup_used(self.h, C.byref(k)))
        return bool(k.value)

    def pff_set_cg_variant(self, variant: int):
        _check(self.L.pff_set_cg_variant(self.h, int(variant)))

    def pff_last_cg_kernel(self) -> int:
        k = C.c_int32(0)
        _check(self.L.pff_last_cg_kernel(self.h, C.byref(k)))
        return k.value

    def pff_damage_last_stats(self):
        """(restarts, truncations) of the projected solver in the last solve / summed over the last pff_run_steps."""
        r, t = C.c_int32(0), C.c_int32(0)
        _check(self.L.pff_damage_last_stats(self.h, C.byref(r), C.byref(t)))
        return r.value, t.value

    def pff_run_steps(self, state: State, bc, dt: float, n_steps: int, damage_every=1, rel_tol=1e-8, max_iter=1000,
                      allow_noconv=False):
        """n_steps staggered steps on the device-resident state, damage solve every damage_every-th step."""
        tot = C.c_int64(0)
        st = _check(self.L.pff_run_steps(self.h, C.byref(state.c), C.byref(bc) if bc is not None else None, dt, n_steps,
                                         damage_every, rel_tol, max_iter, C.byref(tot)),
                    allow=(PFF_ENOCONV,) if allow_noconv else ())
        return st, tot.value

    def pff_set_graph_mode(self, enable: bool):
        _check(self.L.pff_set_graph_mode(self.h, int(enable)))

    def pff_graph_status(self):
        c, r = C.c_int32(0), C.c_int32(0)
        _check(self.L.pff_graph_status(self.h, C.byref(c), C.byref(r)))
        return bool(c.value), bool(r.value)

    def pff_energies(self, state: State):
        out = (C.c_double * 4)()
        _check(self.L.pff_energies(self.h, C.byref(state.c), out))
        return np.array(list(out))

    def pff_mg_attach(self, coarse_meshes):
        """Attach coarser meshes (finest first) as the multigrid hierarchy of this mesh; they are kept alive here."""
        arr = (C.c_void_p * len(coarse_meshes))(*[m.h for m in coarse_meshes])
        _check(self.L.pff_mg_attach(self.h, len(coarse_meshes), arr))
        self._mg_levels = list(coarse_meshes)

    def pff_set_damage_solver(self, solver: str):
        """'jacobi' (default) or 'multigrid' (after pff_mg_attach, AT2) for pff_damage_solve / pff_run_steps."""
        _check(self.L.pff_set_damage_solver(self.h, {"jacobi": 0, "multigrid": 1}[solver]))

    def pff_mg_set_params(self, omega=2.0 / 3.0, coarse_sweeps=4):
        _check(self.L.pff_mg_set_params(self.h, omega, coarse_sweeps))

    def pff_damage_solve_mg(self, state: State, rel_tol=1e-8, max_iter=200, allow_noconv=False):
        it, rr = C.c_int32(0), C.c_double(0.0)
        st = _check(self.L.pff_damage_solve_mg(self.h, C.byref(state.c), rel_tol, max_iter, C.byref(it), C.byref(rr)),
                    allow=(PFF_ENOCONV,) if allow_noconv else ())
        return st, it.value, rr.value

    def pff_mg_apply(self, state: State, r):
        import torch
        z = torch.empty_like(r)
        _check(self.L.pff_mg_apply(self.h, C.byref(state.c), r.data_ptr(), z.data_ptr()))
        return z

    def pff_energies_static(self, state: State, out):
        """pff_energies without any allocation: `out` is a caller-owned device tensor of 4 float64; asynchronous."""
        import torch
        if out.dtype != torch.float64 or out.numel() < 4 or not out.is_cuda or not out.is_contiguous():
            raise ValueError("out: contiguous CUDA tensor of at least 4 float64")
        _check(self.L.pff_energies_static(self.h, C.byref(state.c), out.data_ptr()))
        return out

    def pff_damage_adjoint(self, state: State, g, free_mask=None, rel_tol=1e-8, max_iter=1000, allow_noconv=False):
        """lambda with A_FF lambda_F = g_F (operator of state.H); g, free_mask (uint8) device tensors in internal order."""
        import torch
        lam = torch.empty(self.n_nodes, dtype=self.dtype, device=self.device)
        it, rr = C.c_int32(0), C.c_double(0.0)
        st = _check(self.L.pff_damage_adjoint(self.h, C.byref(state.c), g.data_ptr(),
                                              free_mask.data_ptr() if free_mask is not None else None, lam.data_ptr(),
                                              rel_tol, max_iter, C.byref(it), C.byref(rr)),
                    allow=(PFF_ENOCONV,) if allow_noconv else ())
        return lam, st, it.value, rr.value

    def pff_damage_param_terms(self, lam, d):
        out = (C.c_double * 2)()
        _check(self.L.pff_damage_param_terms(self.h, lam.data_ptr(), d.data_ptr(), out))
        return out[0], out[1]

    def pff_stiffness_action(self, state: State, px, py, qx=None, qy=None):
        """q = f_int(u + p) - f_int(u) (Eq. 13) at the state's u, d; device tensors in internal order."""
        import torch
        if qx is None:
            qx, qy = torch.empty_like(px), torch.empty_like(py)
        _check(self.L.pff_stiffness_action(self.h, C.byref(state.c), px.data_ptr(), py.data_ptr(), qx.data_ptr(), qy.data_ptr()))
        return qx, qy

    def pff_equilibrium_solve(self, state: State, bc=None, rel_tol=1e-8, max_iter=10000, allow_noconv=False):
        it, rr = C.c_int32(0), C.c_double(0.0)
        st = _check(self.L.pff_equilibrium_solve(self.h, C.byref(state.c), C.byref(bc) if bc is not None else None,
                                                 rel_tol, max_iter, C.byref(it), C.byref(rr)),
                    allow=(PFF_ENOCONV,) if allow_noconv else ())
        return st, it.value, rr.value

    def pff_internal_force(self, state: State):
        import torch
        fx = torch.empty(self.n_nodes, dtype=self.dtype, device=self.device)
        fy = torch.empty_like(fx)
        pp = torch.empty(self.n_elems, dtype=self.dtype, device=self.device)
        _check(self.L.pff_internal_force(self.h, C.byref(state.c), fx.data_ptr(), fy.data_ptr(), pp.data_ptr()))
        return fx, fy, pp

    def pff_damage_matvec(self, state: State, p):
        import torch
        q = torch.empty_like(p)
        _check(self.L.pff_damage_matvec(self.h, C.byref(state.c), p.data_ptr(), q.data_ptr()))
        return q

    def pff_damage_rhs_diag(self, state: State):
        import torch
        b = torch.empty(self.n_nodes, dtype=self.dtype, device=self.device)
        D = torch.empty_like(b)
        _check(self.L.pff_damage_rhs_diag(self.h, C.byref(state.c), b.data_ptr(), D.data_ptr()))
        return b, D

    def pff_mesh_counters(self) -> int:
        n = C.c_int64()
        _check(self.L.pff_mesh_counters(self.h, C.byref(n)))
        return n.value

    def pff_time_kernel(self, state: State, which: int, reps: int) -> float:
        ms = C.c_float()
        _check(self.L.pff_time_kernel(self.h, C.byref(state.c), which, reps, C.byref(ms)))
        return ms.value

    def pff_profile_enable(self, enable: bool):
        _check(self.L.pff_profile_enable(self.h, int(enable)))

    def pff_profile_read(self):
        """{kernel class: (summed device ms, launches)} since the last read."""
        n = len(_lib.KERNEL_CLASSES)
        ms, cnt = (C.c_double * n)(), (C.c_int64 * n)()
        _check(self.L.pff_profile_read(self.h, ms, cnt))
        return {k: (ms[i], cnt[i]) for i, k in enumerate(_lib.KERNEL_CLASSES)}

    def pff_run_host(self, u, v, a, d, H, fext, dt, n_steps, damage_every=1, rel_tol=1e-8, max_iter=1000,
                     dir_u=None, dir_v=None, load_scale=1.0, allow_noconv=False):
        """Host-buffer path: numpy fp64 arrays in USER numbering, updated in place."""
        arrs = [u, v, a, d, H, fext]
        for x in arrs:
            assert x.dtype == np.float64 and x.flags.c_contiguous
        dp = C.POINTER(C.c_double)
        hs = _lib.pff_host_state(*[x.ctypes.data_as(dp) for x in arrs])
        ku = np.ascontiguousarray(dir_u, dtype=np.float64) if dir_u is not None else None
        kv = np.ascontiguousarray(dir_v, dtype=np.float64) if dir_v is not None else None
        du = ku.ctypes.data if ku is not None else None
        dv = kv.ctypes.data if kv is not None else None
        return _check(self.L.pff_run_host(self.h, C.byref(hs), du, dv, load_scale, dt, n_steps, damage_every,
                                          rel_tol, max_iter), allow=(PFF_ENOCONV,) if allow_noconv else ())


def pff_subcycle_limit(material: dict):
    """(N_max, continuous ratio c_p / (0.6 c_R)) of PAPER.md L187; host-only."""
    m = _lib.pff_material(**material)
    n, r = C.c_int32(0), C.c_double(0.0)
    _check(_lib.load().pff_subcycle_limit(C.byref(m), C.byref(n), C.byref(r)))
    return n.value, r.value
