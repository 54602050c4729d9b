"""TEST INFRASTRUCTURE ONLY: dense CPU restatement of the multigrid preconditioner of pff_damage_solve_mg.

Only tests/ may import this (like everything under oracle/).  The product path (csrc/pff_multigrid.cu) shares no code
with it.  The paper only names the class of method (preconditioned CG, a multilevel preconditioner
cutting the iteration count 5-20x on fine meshes); the cycle itself is this repository's design and is defined in
include/pff.h (pff_damage_solve_mg) and DESIGN.md section 5.  It is restated here step by step in that order, with dense
matrices, for meshes of a few hundred nodes:

    level l:   x = w D^-1 b;   r = b - A x;   x += P V_{l+1}(P^T r);   x += w D^-1 (b - A x)
    coarsest:  x = w D^-1 b, then (sweeps - 1) times x += w D^-1 (b - A x)

A_l is the oracle's own damage operator (orc_damage_matvec) on the mesh of level l with the history
field of level l; H_{l+1}[E] = sum over the elements e of level l whose centroid lies in E of area_e H_l[e] / sum area_e;
P_l[i, :] = barycentric coordinates of node i of level l in the triangle of level l + 1 that holds it.  On the finest
level the rows / columns of damage-Dirichlet nodes are removed (D^-1 = 0 there, residual and correction masked).

Pins (tests/test_multigrid.py, -m "not gpu"): interpolation reproduces affine functions exactly (partition of unity and
linear precision); the cycle matrix is symmetric and positive definite; with an exact coarsest solve and one level it is
the textbook two-grid operator S + S^T - S^T A S + (I - S^T A) P A_c^-1 P^T (I - A S) assembled from its factors; PCG
with it reaches the oracle's converged Jacobi solve (the unique minimiser).
"""
from __future__ import annotations

import numpy as np

from .pff_oracle import Material, OracleMesh


def locate(xy_c, tri_c, pts):
    """For every point: (triangle of the coarse mesh that holds it, barycentric coordinates).  Brute force."""
    a, b, c = xy_c[tri_c[:, 0]], xy_c[tri_c[:, 1]], xy_c[tri_c[:, 2]]
    det = (b[:, 0] - a[:, 0]) * (c[:, 1] - a[:, 1]) - (c[:, 0] - a[:, 0]) * (b[:, 1] - a[:, 1])
    elem = np.empty(len(pts), dtype=np.int64)
    w = np.empty((len(pts), 3))
    for k, p in enumerate(pts):
        l1 = ((p[0] - a[:, 0]) * (c[:, 1] - a[:, 1]) - (c[:, 0] - a[:, 0]) * (p[1] - a[:, 1])) / det
        l2 = ((b[:, 0] - a[:, 0]) * (p[1] - a[:, 1]) - (p[0] - a[:, 0]) * (b[:, 1] - a[:, 1])) / det
        l0 = 1.0 - l1 - l2
        mn = np.minimum(l0, np.minimum(l1, l2))
        e = int(np.argmax(mn))
        if mn[e] < -1e-6:
            raise ValueError("point outside the coarse mesh")
        ww = np.array([l0[e], l1[e], l2[e]])
        ww[np.abs(ww) < 1e-12] = 0.0
        ww = np.maximum(ww, 0.0)
        elem[k], w[k] = e, ww / ww.sum()
    return elem, w


def interpolation(fine: OracleMesh, coarse: OracleMesh):
    """Dense P [N_fine, N_coarse]."""
    elem, w = locate(coarse.xy, coarse.tri, fine.xy)
    P = np.zeros((fine.N, coarse.N))
    for i in range(fine.N):
        for k in range(3):
            P[i, coarse.tri[elem[i], k]] += w[i, k]
    return P


def restrict_history(fine: OracleMesh, coarse: OracleMesh, H):
    cen = fine.xy[fine.tri].mean(axis=1)
    parent, _ = locate(coarse.xy, coarse.tri, cen)
    num = np.zeros(coarse.Ne)
    den = np.zeros(coarse.Ne)
    np.add.at(num, parent, fine.area * H)
    np.add.at(den, parent, fine.area)
    return np.where(den > 0, num / np.where(den > 0, den, 1.0), 0.0)


def dense_operator(mesh: OracleMesh, H):
    A = np.empty((mesh.N, mesh.N))
    e = np.zeros(mesh.N)
    for j in range(mesh.N):
        e[j] = 1.0
        A[:, j] = mesh.damage_matvec(e, H=H)
        e[j] = 0.0
    return A


class Hierarchy:
    """levels[0] = finest.  meshes: list of (xy, tri); material: dict as in pff_inputs; fixed: damage-Dirichlet nodes of
    the finest level."""

    def __init__(self, meshes, material: dict, H, fixed=(), omega=2.0 / 3.0, coarse_sweeps=4):
        mat = Material(**material)
        self.m = [OracleMesh(xy, tri, mat) for xy, tri in meshes]
        self.omega, self.coarse_sweeps = omega, coarse_sweeps
        self.H = [np.asarray(H, dtype=np.float64)]
        self.P = []
        for l in range(len(self.m) - 1):
            self.P.append(interpolation(self.m[l], self.m[l + 1]))
            self.H.append(restrict_history(self.m[l], self.m[l + 1], self.H[l]))
        self.A = [dense_operator(m, h) for m, h in zip(self.m, self.H)]
        self.Dinv = [1.0 / np.diag(a) for a in self.A]
        self.free = np.ones(self.m[0].N, dtype=bool)
        self.free[np.asarray(fixed, dtype=np.int64)] = False
        self.Dinv[0] = np.where(self.free, self.Dinv[0], 0.0)

    def vcycle(self, b, l=0):
        A, Di, w = self.A[l], self.Dinv[l], self.omega
        x = w * Di * b
        if l == len(self.m) - 1:
            for _ in range(self.coarse_sweeps - 1):
                x = x + w * Di * (b - A @ x)
            return x
        r = b - A @ x
        if l == 0:
            r = np.where(self.free, r, 0.0)
        c = self.P[l] @ self.vcycle(self.P[l].T @ r, l + 1)
        if l == 0:
            c = np.where(self.free, c, 0.0)
        x = x + c
        return x + w * Di * (b - A @ x)

    def matrix(self):
        n = self.m[0].N
        M = np.empty((n, n))
        e = np.zeros(n)
        for j in range(n):
            e[j] = 1.0
            M[:, j] = self.vcycle(e)
            e[j] = 0.0
        return M

    def pcg(self, b, x0, rel_tol=1e-12, max_iter=200):
        """PCG with the cycle, on the free nodes; x0 holds the fixed values.  Returns (x, iterations)."""
        A = self.A[0]
        x = np.array(x0, dtype=np.float64)
        r = np.where(self.free, b - A @ x, 0.0)
        lim = rel_tol * max(np.linalg.norm(np.where(self.free, b, 0.0)), np.linalg.norm(r))
        p = None
        rz = 0.0
        for it in range(max_iter):
            if np.linalg.norm(r) <= lim:
                return x, it
            z = self.vcycle(r)
            rz_new = r @ z
            p = z if p is None else z + (rz_new / rz) * p
            rz = rz_new
            q = A @ p
            alpha = rz / (p @ q)
            x = x + alpha * p
            r = np.where(self.free, r - alpha * q, 0.0)
        return x, max_iter
