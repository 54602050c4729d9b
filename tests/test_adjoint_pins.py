"""Pins of oracle/pff_adjoint_oracle.py (implicit differentiation of the damage solve, section 4.2, Eq. 22-24)
against things other than itself: the C oracle's matrix-free operator (an independent code), central finite differences
of forward solves done by the C oracle's CG, and the algebra of the adjoint."""
import numpy as np
import pytest

from oracle import Material, OracleMesh
from oracle import pff_adjoint_oracle as adj
from pff_inputs import GLASS, random_mesh


def mat(**kw):
    p = dict(GLASS)
    p.update(kw)
    return Material(**p)


def _problem(seed, model=2, n_side=9, l0=0.15, Gc=3.0):
    """Unit-square jittered mesh with mixed orientations, history field of the size that gives d of order 0.1..0.9."""
    xy, tri = random_mesh(n_side, seed)
    g = np.random.default_rng(100 + seed)
    H = g.uniform(0.2, 3.0, len(tri)) * Gc / l0
    return xy, tri, H, mat(Gc=Gc, l0=l0, model=model)


@pytest.mark.parametrize("model", [1, 2])
def test_assembled_operator_equals_matrix_free_c_oracle(model):
    xy, tri, H, m = _problem(1, model)
    A, b = adj.damage_system(xy, tri, H, m.Gc, m.l0, model)
    orc = OracleMesh(xy, tri, m)
    p = np.random.default_rng(2).standard_normal(len(xy))
    q = orc.damage_matvec(p, H)
    assert np.abs(A @ p - q).max() <= 1e-13 * np.abs(q).max()
    b_c, D_c = orc.damage_rhs_diag(H)
    assert np.abs(b - b_c).max() <= 1e-13 * np.abs(b_c).max()
    assert np.abs(A.diagonal() - D_c).max() <= 1e-13 * np.abs(D_c).max()
    assert abs(A - A.T).max() <= 1e-15 * abs(A).max()  # symmetric: A^T lambda = g is a solve with the same operator (Eq. 23)


def test_mass_and_stiffness_textbook_properties():
    xy, tri, _, _ = _problem(3)
    M, K = adj.mass_stiffness(xy, tri)
    one = np.ones(len(xy))
    assert abs(one @ (M @ one) - 1.0) <= 1e-13          # total area of the unit square
    assert np.abs(K @ one).max() <= 1e-11               # constants are in the kernel of the stiffness
    lin = 2.0 * xy[:, 0] - 3.0 * xy[:, 1]
    assert abs(lin @ (K @ lin) - 13.0) <= 1e-11         # int |grad(2x - 3y)|^2 over the unit square


def _forward_c_oracle(xy, tri, H, m, fixed):
    """Forward solve by the C oracle's Jacobi-PCG from d_n = 0 (converged; the clamp must stay inactive)."""
    orc = OracleMesh(xy, tri, m)
    orc.H[:] = H
    if len(fixed):
        orc.d[fixed] = 1.0
        orc.set_damage_dirichlet(fixed)
    rc, _, rr = orc.damage_solve(rel_tol=1e-14, max_iter=5000)
    assert rc == 0
    return orc.d.copy()


@pytest.mark.parametrize("fixed", [[], [0, 7, 40, 41, 80]])
def test_adjoint_gradient_matches_finite_differences_of_forward_solves(fixed):
    """Eq. 24: dL/dG_c = -[l0 lambda^T K d + (1/l0) lambda^T M d] (and the l0 analogue) for L = g^T d, against central
    differences of the C oracle's forward solve at perturbed G_c / l0; fixed (Dirichlet) nodes carry lambda = 0."""
    xy, tri, H, m = _problem(4)
    fixed = np.asarray(fixed, dtype=np.int32)
    g = np.random.default_rng(5).standard_normal(len(xy))
    d = _forward_c_oracle(xy, tri, H, m, fixed)
    assert d.min() > 0.0 and d.max() <= 1.0  # clamp inactive: d is the solution of the linear system (Eq. 22)
    A, b = adj.damage_system(xy, tri, H, m.Gc, m.l0, 2)
    d_direct = adj.forward_solve(A, b, fixed)
    assert np.abs(d - d_direct).max() <= 1e-11
    free = np.ones(len(xy), dtype=bool)
    free[fixed] = False
    lam = adj.adjoint_solve(A, g, free)
    assert np.all(lam[fixed] == 0.0)
    M, K = adj.mass_stiffness(xy, tri)
    dGc, dl0 = adj.grad_at2(m.Gc, m.l0, *adj.param_terms(M, K, lam, d))
    eps = 1e-5
    for name, ref in (("Gc", dGc), ("l0", dl0)):
        base = getattr(m, name)
        vals = []
        for s in (+1, -1):
            kw = {name: base * (1 + s * eps)}
            vals.append(g @ _forward_c_oracle(xy, tri, H, mat(**{**dict(Gc=m.Gc, l0=m.l0, model=2), **kw}), fixed))
        fd = (vals[0] - vals[1]) / (2 * eps * base)
        assert abs(fd - ref) <= 2e-7 * abs(ref), (name, fd, ref)


def test_adjoint_identity_and_masking():
    """lambda^T b_F = g_F^T d_F when d_F = A_FF^-1 b_F (the defining identity of the adjoint), on a masked free set."""
    xy, tri, H, m = _problem(6, model=1)
    A, b = adj.damage_system(xy, tri, H, m.Gc, m.l0, 1)
    r = np.random.default_rng(7)
    free = r.uniform(size=len(xy)) < 0.7
    g = r.standard_normal(len(xy))
    lam = adj.adjoint_solve(A, g, free)
    dF = np.zeros(len(xy))
    import scipy.sparse.linalg as spla
    dF[free] = spla.spsolve(A[free][:, free].tocsc(), b[free])
    assert abs(lam @ b - g[free] @ dF[free]) <= 1e-11 * abs(lam @ b)
    assert np.all(lam[~free] == 0.0)
    res = (A @ lam - g)[free]
    assert np.abs(res).max() <= 1e-11 * np.abs(g).max()


# ---------------------------------------------------------------- matrix-free stiffness action, Eq. 11-15 (L126-159)
@pytest.mark.parametrize("plane", [0, 1])
def test_stiffness_action_equals_assembled_operator_for_the_isotropic_split(plane):
    """Eq. 13 (difference of the C oracle's internal forces) against Eq. 14 (K assembled from B^T C B in Python)."""
    from oracle import pff_stiffness_oracle as sto
    xy, tri = random_mesh(9, 8)
    m = mat(split=0, plane=plane)
    orc = OracleMesh(xy, tri, m)
    r = np.random.default_rng(9)
    orc.u[:] = 1e-4 * r.standard_normal((len(xy), 2))
    orc.d[:] = r.uniform(0.0, 0.9, len(xy))
    p = 1e-4 * r.standard_normal((len(xy), 2))
    K = sto.assemble_stiffness(xy, tri, m.E, m.nu, plane, orc.d, m.eta)
    q = orc.stiffness_action(p)
    q_ref = (K @ p.ravel()).reshape(-1, 2)
    assert np.abs(q - q_ref).max() <= 1e-10 * np.abs(q_ref).max()  # cancellation in f(u + p) - f(u): ~|u|/|p| ulp
    f, _ = orc.internal_force()
    assert np.abs(f - (K @ orc.u.ravel()).reshape(-1, 2)).max() <= 1e-12 * np.abs(f).max()  # Eq. 10: f_int = K u
    assert abs(K - K.T).max() <= 1e-12 * abs(K).max()
    rigid = np.tile([1.0, 0.0], len(xy))
    assert np.abs(K @ rigid).max() <= 1e-9 * abs(K).max()


def test_stiffness_action_is_the_tangent_when_the_sign_pattern_is_fixed():
    """Spectral split: the shifted difference equals the directional derivative (Eq. 12) for a small p (L140)."""
    xy, tri = random_mesh(7, 10)
    orc = OracleMesh(xy, tri, mat(split=1))
    r = np.random.default_rng(11)
    orc.u[:] = 1e-4 * r.standard_normal((len(xy), 2))
    orc.d[:] = r.uniform(0.0, 0.5, len(xy))
    p = 1e-9 * r.standard_normal((len(xy), 2))
    q = orc.stiffness_action(p)
    eps = 0.5
    fd = (orc.internal_force(orc.u + eps * p)[0] - orc.internal_force(orc.u - eps * p)[0]) / (2 * eps)
    assert np.abs(q - fd).max() <= 1e-4 * np.abs(fd).max()


def _boundary_nodes(n):
    i, j = np.arange(n * n) % n, np.arange(n * n) // n
    return np.nonzero((i == 0) | (i == n - 1) | (j == 0) | (j == n - 1))[0]


def test_equilibrium_oracle_patch_test_and_force_balance():
    """Assembled direct solve: (i) affine Dirichlet data on the whole boundary with uniform damage reproduce the affine
    field in the interior (patch test); (ii) with non-uniform damage and a traction load the C oracle's internal force
    (an independent code) balances S f_ext on every free dof."""
    from oracle import pff_stiffness_oracle as sto
    from pff_inputs import edge_segments
    n = 9
    xy, tri = random_mesh(n, 12)
    m = mat(split=0)
    G = np.array([[1e-4, -2e-4], [3e-4, 0.5e-4]])
    u_aff = xy @ G.T
    bn = _boundary_nodes(n)
    fixed = np.concatenate([2 * bn, 2 * bn + 1])
    u0 = np.zeros_like(u_aff)
    u0[bn] = u_aff[bn]
    K = sto.assemble_stiffness(xy, tri, m.E, m.nu, 0, np.full(len(xy), 0.3), m.eta)
    u = sto.equilibrium_solve(K, u0, np.zeros_like(u0), 1.0, fixed)
    assert np.abs(u - u_aff).max() <= 1e-12 * np.abs(u_aff).max()

    orc = OracleMesh(xy, tri, m)
    orc.d[:] = np.random.default_rng(13).uniform(0.0, 0.9, len(xy))
    top = edge_segments(n, n, "top")
    orc.add_traction(top, np.tile([2e5, 1e6], (len(top), 1)))
    bottom = np.arange(n)
    fixed = np.concatenate([2 * bottom, 2 * bottom + 1])
    K = sto.assemble_stiffness(xy, tri, m.E, m.nu, 0, orc.d, m.eta)
    S = 0.7
    u = sto.equilibrium_solve(K, np.zeros((len(xy), 2)), orc.fext, S, fixed)
    f, _ = orc.internal_force(u)
    res = (f - S * orc.fext).ravel()
    free = np.ones(2 * len(xy), dtype=bool)
    free[fixed] = False
    assert np.abs(res[free]).max() <= 1e-10 * np.abs(orc.fext).max()
    assert np.all(u[bottom] == 0.0)
