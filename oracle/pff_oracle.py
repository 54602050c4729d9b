"""ctypes front end of oracle/pff_oracle.c -- TEST INFRASTRUCTURE ONLY (see the C file's header).

`OracleMesh` keeps the mesh in USER numbering with AoS fields (u[N,2], ...) in fp64 and steps it
with the plain C loops.  No arithmetic of the method lives in this file: it only marshals numpy
arrays into the C functions, each of which cites the PAPER.md passage it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pff_oracle.c")
_SO = os.path.join(_HERE, "libpff_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no OpenMP, no fast-math: plain IEEE fp64)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-o", _SO, _SRC, "-lm"]
        )
    return _SO


class _Mat(C.Structure):
    _fields_ = [(k, C.c_double) for k in ("E", "nu", "rho", "Gc", "l0", "eta", "gamma_star")] + [
        (k, C.c_int) for k in ("model", "split", "plane")
    ]


@dataclass
class Material:
    E: float
    nu: float
    rho: float
    Gc: float
    l0: float
    eta: float = 1e-7
    gamma_star: float = 0.0
    model: int = 2  # 1 AT1, 2 AT2
    split: int = 1  # 0 iso, 1 spectral, 2 vol-dev, 3 star-convex
    plane: int = 0  # 0 plane strain, 1 plane stress

    def c(self) -> _Mat:
        return _Mat(self.E, self.nu, self.rho, self.Gc, self.l0, self.eta, self.gamma_star,
                    self.model, self.split, self.plane)


_D = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")
_I = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_i64 = C.c_int64
_MP = C.POINTER(_Mat)


def _load():
    global _lib
    if _lib is not None:
        return _lib
    L = C.CDLL(build())
    L.orc_geometry.argtypes = [_i64, _D, _i64, _I, _I, _D, _D]
    L.orc_geometry.restype = C.c_int
    L.orc_lumped_mass.argtypes = [_i64, _i64, _I, _D, C.c_double, _D]
    L.orc_hmin.argtypes = [_i64, _I, _D, _D]
    L.orc_hmin.restype = C.c_double
    L.orc_dt_crit.argtypes = [_MP, C.c_double]
    L.orc_dt_crit.restype = C.c_double
    L.orc_element_response.argtypes = [_MP, C.c_double, C.c_double, C.c_double, C.c_double,
                                       C.POINTER(C.c_double), C.POINTER(C.c_double), C.POINTER(C.c_double)]
    L.orc_internal_force.argtypes = [_i64, _i64, _I, _D, _D, _MP, _D, _D, _D, _D]
    L.orc_traction.argtypes = [_i64, _I, _D, _D, _D]
    L.orc_init_accel.argtypes = [_i64, _i64, _I, _D, _D, _D, _MP, _D, _D, _D, C.c_double, _i64, _I, _D]
    L.orc_explicit_step.argtypes = [_i64, _i64, _I, _D, _D, _D, _MP, _D, _D, _D, _D, _D, _D,
                                    C.c_double, C.c_double, _i64, _I, _D, _D]
    L.orc_damage_matvec.argtypes = [_i64, _i64, _I, _D, _D, _MP, _D, _D, _D]
    L.orc_damage_rhs_diag.argtypes = [_i64, _i64, _I, _D, _D, _MP, _D, _D, _D]
    L.orc_damage_solve.argtypes = [_i64, _i64, _I, _D, _D, _MP, _D, _D, _i64, _I, C.c_double, C.c_int,
                                   C.POINTER(C.c_int), C.POINTER(C.c_double)]
    L.orc_damage_solve.restype = C.c_int
    L.orc_energies.argtypes = [_i64, _i64, _I, _D, _D, _D, _MP, _D, _D, _D, _D]
    _lib = L
    return L


def element_response(mat: Material, exx: float, eyy: float, exy: float, g: float = 1.0):
    """(psi+, psi-, [sxx, syy, sxy]) of one strain state; see orc_element_response."""
    L = _load()
    pp, pm = C.c_double(), C.c_double()
    s = (C.c_double * 3)()
    m = mat.c()
    L.orc_element_response(C.byref(m), exx, eyy, exy, g, C.byref(pp), C.byref(pm), s)
    return pp.value, pm.value, np.array(list(s))


class OracleMesh:
    """Mesh + state of the oracle in user numbering."""

    def __init__(self, xy, tri, mat: Material):
        L = _load()
        self.L = L
        self.mat = mat
        self._m = mat.c()
        self.xy = np.ascontiguousarray(xy, dtype=np.float64)
        tri = np.ascontiguousarray(tri, dtype=np.int32)
        self.N, self.Ne = len(self.xy), len(tri)
        self.tri = np.empty_like(tri)
        self.gradphi = np.empty((self.Ne, 3, 2))
        self.area = np.empty(self.Ne)
        rc = L.orc_geometry(self.N, self.xy, self.Ne, tri, self.tri, self.gradphi, self.area)
        if rc:
            raise ValueError(f"degenerate or out-of-range element {rc - 1}")
        self.mass = np.empty(self.N)
        L.orc_lumped_mass(self.N, self.Ne, self.tri, self.area, mat.rho, self.mass)
        self.u = np.zeros((self.N, 2)); self.v = np.zeros((self.N, 2)); self.a = np.zeros((self.N, 2))
        self.d = np.zeros(self.N); self.H = np.zeros(self.Ne); self.fext = np.zeros((self.N, 2))
        self.dir_dof = np.zeros(0, dtype=np.int32)
        self.ddir = np.zeros(0, dtype=np.int32)

    # -- setup helpers ---------------------------------------------------------------
    def hmin(self) -> float:
        return self.L.orc_hmin(self.Ne, self.tri, self.xy, self.area)

    def dt_crit(self) -> float:
        return self.L.orc_dt_crit(C.byref(self._m), self.hmin())

    def add_traction(self, edge_nodes, t):
        e = np.ascontiguousarray(edge_nodes, dtype=np.int32)
        self.L.orc_traction(len(e), e, np.ascontiguousarray(t, dtype=np.float64), self.xy, self.fext)

    def set_dirichlet(self, dir_dof):
        self.dir_dof = np.ascontiguousarray(dir_dof, dtype=np.int32)

    def set_damage_dirichlet(self, nodes):
        self.ddir = np.ascontiguousarray(nodes, dtype=np.int32)

    # -- operators ---------------------------------------------------------------------
    def internal_force(self, u=None, d=None):
        u = self.u if u is None else np.ascontiguousarray(u, dtype=np.float64)
        d = self.d if d is None else np.ascontiguousarray(d, dtype=np.float64)
        f = np.empty((self.N, 2)); pp = np.empty(self.Ne)
        self.L.orc_internal_force(self.N, self.Ne, self.tri, self.gradphi, self.area, C.byref(self._m), u, d, f, pp)
        return f, pp

    def stiffness_action(self, p, u=None, d=None):
        """K(u) p = f_int(u + p) - f_int(u) with d held fixed: PAPER.md Eq. 13 written out with the internal force."""
        u = self.u if u is None else np.ascontiguousarray(u, dtype=np.float64)
        return self.internal_force(u + np.asarray(p, dtype=np.float64), d)[0] - self.internal_force(u, d)[0]

    def init_accel(self, S=1.0):
        self.L.orc_init_accel(self.N, self.Ne, self.tri, self.gradphi, self.area, self.mass, C.byref(self._m),
                              self.u, self.d, self.fext, S, len(self.dir_dof), self.dir_dof, self.a)

    def explicit_step(self, dt, S=1.0, dir_u=None, dir_v=None):
        nd = len(self.dir_dof)
        du = np.zeros(nd) if dir_u is None else np.ascontiguousarray(dir_u, dtype=np.float64)
        dv = np.zeros(nd) if dir_v is None else np.ascontiguousarray(dir_v, dtype=np.float64)
        self.L.orc_explicit_step(self.N, self.Ne, self.tri, self.gradphi, self.area, self.mass, C.byref(self._m),
                                 self.u, self.v, self.a, self.d, self.H, self.fext, S, dt, nd, self.dir_dof, du, dv)

    def damage_matvec(self, p, H=None):
        H = self.H if H is None else np.ascontiguousarray(H, dtype=np.float64)
        q = np.empty(self.N)
        self.L.orc_damage_matvec(self.N, self.Ne, self.tri, self.gradphi, self.area, C.byref(self._m), H,
                                 np.ascontiguousarray(p, dtype=np.float64), q)
        return q

    def damage_rhs_diag(self, H=None):
        H = self.H if H is None else np.ascontiguousarray(H, dtype=np.float64)
        b = np.empty(self.N); D = np.empty(self.N)
        self.L.orc_damage_rhs_diag(self.N, self.Ne, self.tri, self.gradphi, self.area, C.byref(self._m), H, b, D)
        return b, D

    def damage_solve(self, rel_tol=1e-8, max_iter=1000):
        it, rr = C.c_int(0), C.c_double(0.0)
        rc = self.L.orc_damage_solve(self.N, self.Ne, self.tri, self.gradphi, self.area, C.byref(self._m), self.H,
                                     self.d, len(self.ddir), self.ddir, rel_tol, max_iter, C.byref(it), C.byref(rr))
        return rc, it.value, rr.value

    def energies(self):
        out = np.empty(4)
        self.L.orc_energies(self.N, self.Ne, self.tri, self.gradphi, self.area, self.mass, C.byref(self._m),
                            self.u, self.v, self.d, out)
        return out


def oracle_from(cfg) -> OracleMesh:
    """OracleMesh of a pff_inputs.config dictionary (mesh, material, initial fields, tractions, Dirichlet sets):
    marshalling only.  Used by the parity tests and by bench.py's cpu_baseline / --impl reference legs."""
    m = OracleMesh(cfg["xy"], cfg["tri"], Material(**cfg["material"]))
    m.u[:] = cfg["u0"]
    m.d[:] = cfg["d0"]
    if len(cfg["edges"]):
        m.add_traction(cfg["edges"], cfg["traction"])
    if len(cfg["notch"]):
        m.set_damage_dirichlet(cfg["notch"])
    if len(cfg["dir_dof"]):
        m.set_dirichlet(cfg["dir_dof"])
    return m
