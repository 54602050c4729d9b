"""Oracle for the implicit-differentiation backward of the damage solve -- TEST INFRASTRUCTURE ONLY.

PAPER.md section 4.2 (L426-448): the forward pass solves A(theta) d = b(theta) (Eq. 22); the backward pass solves ONE
adjoint system A^T lambda = g with the same operator (Eq. 23; A is symmetric) and the parameter gradient follows
from the dependence of A and b on the parameters; for AT2 and (G_c, l0) it reduces to element mass and stiffness
terms, e.g. -[l0 lambda^T K d + (1/l0) lambda^T M d] for G_c (Eq. 24).  Irreversibility is handled by active-set
masking (L446): the system is linearised on the free set F realised by the forward solve, lambda = 0 elsewhere.

This oracle is the DEFINITION written out: the operator is ASSEMBLED as a sparse matrix from the element matrices
M^e = A_e (1 + delta_ij) / 12 (L185) and K^e = A_e grad phi_i . grad phi_j (Eq. 9), and the adjoint system is solved
DIRECTLY (scipy.sparse.linalg.spsolve) on the free set.  It shares nothing with oracle/pff_oracle.c (which applies the
operator matrix-free) nor with the CUDA path; tests/test_adjoint_pins.py pins it against the C oracle's operator and
against central finite differences of forward solves.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla


def element_geometry(xy, tri):
    """Positive areas and grad phi_i of every P1 triangle (Eq. 9); nodes 2 and 3 swapped where the signed area is negative."""
    xy = np.asarray(xy, dtype=np.float64)
    tri = np.array(tri, dtype=np.int64, copy=True)
    x, y = xy[tri, 0], xy[tri, 1]
    a2 = (x[:, 1] - x[:, 0]) * (y[:, 2] - y[:, 0]) - (x[:, 2] - x[:, 0]) * (y[:, 1] - y[:, 0])
    flip = a2 < 0
    tri[flip, 1], tri[flip, 2] = tri[flip, 2].copy(), tri[flip, 1].copy()
    x, y = xy[tri, 0], xy[tri, 1]
    a2 = np.abs(a2)
    grad = np.empty((len(tri), 3, 2))
    for i in range(3):
        j, k = (i + 1) % 3, (i + 2) % 3
        grad[:, i, 0] = (y[:, j] - y[:, k]) / a2  # d phi_i / dx
        grad[:, i, 1] = (x[:, k] - x[:, j]) / a2  # d phi_i / dy
    return tri, 0.5 * a2, grad


def _assemble(n_nodes, tri, elem_mats):
    rows = np.repeat(tri, 3, axis=1).ravel()
    cols = np.tile(tri, (1, 3)).ravel()
    return sp.coo_matrix((elem_mats.reshape(-1), (rows, cols)), shape=(n_nodes, n_nodes)).tocsr()


def mass_stiffness(xy, tri, weight=None):
    """Assembled consistent mass M (optionally weighted by a per-element factor) and stiffness K."""
    n = len(xy)
    tri, area, grad = element_geometry(xy, tri)
    w = np.ones(len(tri)) if weight is None else np.asarray(weight, dtype=np.float64)
    Me = (area * w)[:, None, None] / 12.0 * (np.ones((3, 3)) + np.eye(3))[None]
    Ke = area[:, None, None] * np.einsum("eix,ejx->eij", grad, grad)
    return _assemble(n, tri, Me), _assemble(n, tri, Ke)


def damage_system(xy, tri, H, Gc, l0, model):
    """A and b of the damage sub-problem (Eq. 6 AT2 / Eq. 8 AT1; L98-112): A = M[c_e] + kappa K, b_i = sum_e s_e A_e / 3."""
    H = np.asarray(H, dtype=np.float64)
    if model == 2:
        c_e, kappa, s_e = Gc / l0 + 2.0 * H, Gc * l0, 2.0 * H
    else:
        c_e, kappa, s_e = 2.0 * H, 0.75 * Gc * l0, 2.0 * H - 3.0 * Gc / (8.0 * l0)
    Mc, K = mass_stiffness(xy, tri, c_e)
    tri_o, area, _ = element_geometry(xy, tri)
    b = np.zeros(len(xy))
    np.add.at(b, tri_o.ravel(), np.repeat(s_e * area / 3.0, 3))
    return (Mc + kappa * K).tocsr(), b


def forward_solve(A, b, fixed_nodes=(), fixed_values=None):
    """Unconstrained solution of A d = b with d prescribed on fixed_nodes (Eq. 22 on the non-Dirichlet nodes)."""
    n = A.shape[0]
    d = np.zeros(n)
    fixed = np.zeros(n, dtype=bool)
    fixed[np.asarray(fixed_nodes, dtype=np.int64)] = True
    if fixed.any():
        d[fixed] = 1.0 if fixed_values is None else np.asarray(fixed_values, dtype=np.float64)
    F = ~fixed
    rhs = b[F] - A[F][:, ~F] @ d[~F]
    d[F] = spla.spsolve(A[F][:, F].tocsc(), rhs)
    return d


def adjoint_solve(A, g, free):
    """lambda with A_FF lambda_F = g_F on the free set F and lambda = 0 elsewhere (Eq. 23 with active-set masking, L446)."""
    free = np.asarray(free, dtype=bool)
    lam = np.zeros(A.shape[0])
    lam[free] = spla.spsolve(A[free][:, free].tocsc(), np.asarray(g, dtype=np.float64)[free])
    return lam


def param_terms(M, K, lam, d):
    """(lambda^T M d, lambda^T K d): the two scalars every (G_c, l0) gradient of Eq. 24 is built from."""
    return float(lam @ (M @ d)), float(lam @ (K @ d))


def grad_at2(Gc, l0, lMd, lKd):
    """dL/dG_c and dL/dl0 of a loss with dL/dd = g, AT2 (b does not depend on G_c, l0):
    dL/dtheta = -lambda^T (dA/dtheta) d,  A = (G_c / l0) M + 2 M[H] + G_c l0 K   (Eq. 24 for G_c)."""
    return -(lMd / l0 + l0 * lKd), -(-Gc / l0**2 * lMd + Gc * lKd)
