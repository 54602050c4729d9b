"""Assembled linear-elastic stiffness of the degraded solid -- TEST INFRASTRUCTURE ONLY.

PAPER.md Eq. 14: K = sum_e P_e^T K^e P_e with K^e = g(d_e) A_e B^T C B (P1 triangle, constant strain), the classical
assembled operator the matrix-free action of Eq. 11-13 is compared with.  Valid for the ISOTROPIC split (psi+ = psi, so
sigma = g(d) C : eps is linear in u).  Written from the textbook definition with scipy.sparse; shares nothing with
oracle/pff_oracle.c (whose internal force defines the action through Eq. 13) nor with the CUDA path.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp

from .pff_adjoint_oracle import element_geometry


def elasticity_matrix(E, nu, plane):
    """Voigt C for (eps_xx, eps_yy, gamma_xy = 2 eps_xy): plane strain (0) or plane stress (1) (L85)."""
    mu = E / (2.0 * (1.0 + nu))
    lam = E * nu / ((1.0 + nu) * (1.0 - 2.0 * nu))
    if plane == 1:
        lam = 2.0 * lam * mu / (lam + 2.0 * mu)
    return np.array([[lam + 2 * mu, lam, 0.0], [lam, lam + 2 * mu, 0.0], [0.0, 0.0, mu]])


def assemble_stiffness(xy, tri, E, nu, plane, d, eta):
    """K [2N x 2N], dof order (node, component); g(d_e) with the centroid damage (R3)."""
    n = len(xy)
    tri_o, area, grad = element_geometry(xy, tri)
    C = elasticity_matrix(E, nu, plane)
    de = np.asarray(d, dtype=np.float64)[tri_o].mean(axis=1)
    g = (1.0 - de) ** 2 + eta
    B = np.zeros((len(tri_o), 3, 6))
    for i in range(3):
        B[:, 0, 2 * i] = grad[:, i, 0]
        B[:, 1, 2 * i + 1] = grad[:, i, 1]
        B[:, 2, 2 * i] = grad[:, i, 1]
        B[:, 2, 2 * i + 1] = grad[:, i, 0]
    Ke = (g * area)[:, None, None] * np.einsum("eki,kl,elj->eij", B, C, B)
    dofs = (2 * tri_o[:, :, None] + np.arange(2)[None, None, :]).reshape(len(tri_o), 6)
    rows = np.repeat(dofs, 6, axis=1).ravel()
    cols = np.tile(dofs, (1, 6)).ravel()
    return sp.coo_matrix((Ke.reshape(-1), (rows, cols)), shape=(2 * n, 2 * n)).tocsr()


def equilibrium_solve(K, u_ref, fext, S, fixed_dofs):
    """u = u_ref + du with K_ff du_f = (S f_ext - K u_ref)_f and du = 0 on the fixed dofs (2 * node + component):
    the quasi-static equilibrium f_int(u) = S f_ext of the linear (isotropic-split) problem, by a direct solve."""
    import scipy.sparse.linalg as spla
    n2 = K.shape[0]
    free = np.ones(n2, dtype=bool)
    free[np.asarray(fixed_dofs, dtype=np.int64)] = False
    u0 = np.asarray(u_ref, dtype=np.float64).ravel()
    r = S * np.asarray(fext, dtype=np.float64).ravel() - K @ u0
    du = np.zeros(n2)
    du[free] = spla.spsolve(K[free][:, free].tocsc(), r[free])
    return (u0 + du).reshape(-1, 2)
