"""Pins of the CPU oracle against what the paper and the mathematics fix (run with -m "not gpu").

Each test names the PAPER.md passage / DESIGN.md reading it pins.  Nothing here touches the CUDA path.
"""
import itertools
import os

import numpy as np
import pytest

from oracle import Material, OracleMesh, element_response
from pff_inputs import GLASS, grid_mesh, random_mesh, edge_segments

HERE = os.path.dirname(os.path.abspath(__file__))
SPLITS = [0, 1, 2, 3]
PLANES = [0, 1]


def mat(**kw):
    p = dict(GLASS)
    p.update(kw)
    return Material(**p)


# ---------------------------------------------------------------- geometry, Eq. 9 (L120-124)
def test_reference_triangle_eq9():
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [0.0, 1.0]])
    m = OracleMesh(xy, np.array([[0, 1, 2]], dtype=np.int32), mat())
    assert m.area[0] == 0.5
    np.testing.assert_allclose(m.gradphi[0], [[-1, -1], [1, 0], [0, 1]], atol=0)
    # clockwise input is re-oriented [R1]: same area, gradients follow the swapped nodes
    m2 = OracleMesh(xy, np.array([[0, 2, 1]], dtype=np.int32), mat())
    assert m2.area[0] == 0.5 and list(m2.tri[0]) == [0, 1, 2]


def test_gradients_reproduce_linear_fields():
    xy, tri = random_mesh(7, seed=11)
    m = OracleMesh(xy, tri, mat())
    a, b, c = 0.3, -1.7, 2.1
    f = a + b * xy[:, 0] + c * xy[:, 1]
    g = np.einsum("eid,ei->ed", m.gradphi, f[m.tri])
    np.testing.assert_allclose(g, np.tile([b, c], (m.Ne, 1)), rtol=0, atol=1e-12)
    np.testing.assert_allclose(m.gradphi.sum(axis=1), 0.0, atol=1e-12)  # partition of unity
    assert abs(m.area.sum() - 1.0) < 1e-13  # areas tile the unit square
    assert abs(m.mass.sum() - GLASS["rho"] * 1.0) < 1e-9  # lumped mass conserves total mass (L169)


def test_lumped_mass_per_node_closed_form():
    """m_i = rho sum_{e ni i} A_e / 3 (L169) node by node on a uniform right-triangle grid (quads split along the
    lower-left -> upper-right diagonal): an interior node touches six triangles of area h^2/2 -> rho h^2, an edge node
    three -> rho h^2 / 2, the two corners ON the diagonal (lower-left, upper-right) two -> rho h^2 / 3, the other two
    corners one -> rho h^2 / 6.  A wrong node index in the scatter moves mass between these classes."""
    nx, ny, h = 6, 5, 0.25
    xy, tri = grid_mesh(nx, ny, (nx - 1) * h, (ny - 1) * h)
    rho = 2450.0
    for perm_seed in (None, 3):  # also with flipped orientation and permuted element order
        t = tri.copy()
        if perm_seed is not None:
            g = np.random.default_rng(perm_seed)
            flip = g.uniform(size=len(t)) < 0.5
            t[flip] = t[flip][:, [0, 2, 1]]
            t = np.ascontiguousarray(t[g.permutation(len(t))])
        m = OracleMesh(xy, t, mat(rho=rho))
        i, j = np.arange(nx * ny) % nx, np.arange(nx * ny) // nx
        on_x, on_y = (i == 0) | (i == nx - 1), (j == 0) | (j == ny - 1)
        expect = np.where(on_x & on_y, 0.0, np.where(on_x | on_y, 0.5, 1.0)) * rho * h * h
        diag_corner = ((i == 0) & (j == 0)) | ((i == nx - 1) & (j == ny - 1))
        other_corner = (on_x & on_y) & ~diag_corner
        expect[diag_corner] = rho * h * h / 3.0
        expect[other_corner] = rho * h * h / 6.0
        np.testing.assert_allclose(m.mass, expect, rtol=1e-14, atol=0)


def test_degenerate_element_rejected():
    xy = np.array([[0.0, 0.0], [1.0, 0.0], [2.0, 0.0]])
    with pytest.raises(ValueError):
        OracleMesh(xy, np.array([[0, 1, 2]], dtype=np.int32), mat())


# ---------------------------------------------------------------- material constants and CFL (L85, L169)
def test_cfl_closed_form():
    # glass, plane strain: c_p = sqrt((lambda+2mu)/rho) = 3809.52 m/s; right-isosceles incircle
    # diameter = (2 - sqrt 2) h = 0.585786 h  => dt_crit = 1.53768e-7 s at h = 1 mm (DESIGN R13)
    xy, tri = grid_mesh(11, 5, 0.010, 0.004)
    m = OracleMesh(xy, tri, mat(plane=0))
    h = 1e-3
    assert abs(m.hmin() - (2 - np.sqrt(2)) * h) < 1e-15
    lam = 32e9 * 0.2 / (1.2 * 0.6)
    mu = 32e9 / 2.4
    cp = np.sqrt((lam + 2 * mu) / 2450.0)
    assert abs(cp - 3809.52) < 0.01
    assert abs(m.dt_crit() - (2 - np.sqrt(2)) * h / cp) < 1e-20
    assert abs(0.5 * m.dt_crit() - 7.6884e-8) < 1e-11


# ---------------------------------------------------------------- energy splits, Eq. 2-3 (L71-85)
def test_split_golden_values():
    rows = np.loadtxt(os.path.join(HERE, "golden", "split_energy_values.txt"))
    for exx, eyy, exy, plane, sp, sm, vp, vm, cp_, cm, psi in rows:
        for split, gs, ep, em in [(1, 0.0, sp, sm), (2, 0.0, vp, vm), (3, 2.0, cp_, cm)]:
            pp, pm, _ = element_response(mat(split=split, plane=int(plane), gamma_star=gs), exx, eyy, exy)
            assert abs(pp - ep) < 1e-3 and abs(pm - em) < 1e-3, (split, plane, pp, pm)
            assert abs(pp + pm - psi) < 1e-3
        pp, pm, _ = element_response(mat(split=0, plane=int(plane)), exx, eyy, exy)
        assert abs(pp - psi) < 1e-3 and pm == 0.0


@pytest.mark.parametrize("split,plane", list(itertools.product(SPLITS, PLANES)))
def test_split_identity_psi_plus_plus_psi_minus(split, plane):
    """psi+ + psi- = psi = lambda_eff/2 tr^2 + mu eps:eps for every split (L79, L85)."""
    rng = np.random.default_rng(100 + 10 * split + plane)
    m = mat(split=split, plane=plane, gamma_star=1.3)
    lam = m.E * m.nu / (1 - m.nu**2) if plane else m.E * m.nu / ((1 + m.nu) * (1 - 2 * m.nu))
    mu = m.E / (2 * (1 + m.nu))
    for _ in range(200):
        exx, eyy, exy = rng.normal(0, 1e-3, 3)
        pp, pm, s = element_response(m, exx, eyy, exy)
        psi = 0.5 * lam * (exx + eyy) ** 2 + mu * (exx**2 + eyy**2 + 2 * exy**2)
        assert abs(pp + pm - psi) <= 1e-12 * psi
        assert pp >= 0 and pm >= 0 or split == 3
        # undamaged (g = 1) stress is the linear-elastic stress of the plane assumption
        s_lin = np.array([lam * (exx + eyy) + 2 * mu * exx, lam * (exx + eyy) + 2 * mu * eyy, 2 * mu * exy])
        np.testing.assert_allclose(s, s_lin, rtol=0, atol=1e-9 * np.abs(s_lin).max())


def test_spectral_against_numpy_eigh():
    """Eq. 2 restated with numpy.linalg.eigh (library eigen-decomposition), incl. degraded stress."""
    rng = np.random.default_rng(7)
    m = mat(split=1, plane=0)
    lam = m.E * m.nu / ((1 + m.nu) * (1 - 2 * m.nu))
    mu = m.E / (2 * (1 + m.nu))
    cases = [rng.normal(0, 1e-3, 3) for _ in range(100)]
    cases += [np.array([2e-4, 2e-4, 0.0]), np.array([-3e-4, -3e-4, 0.0]), np.array([0.0, 0.0, 0.0]),
              np.array([1e-4, -1e-4, 0.0]), np.array([0.0, 0.0, 5e-4]), np.array([1e-4, 1e-4, 1e-300])]
    for exx, eyy, exy in cases:
        g = 0.37
        w, V = np.linalg.eigh(np.array([[exx, exy], [exy, eyy]]))
        tr = exx + eyy
        pp_ref = 0.5 * lam * max(tr, 0) ** 2 + mu * sum(max(x, 0) ** 2 for x in w)
        pm_ref = 0.5 * lam * min(tr, 0) ** 2 + mu * sum(min(x, 0) ** 2 for x in w)
        Sp = lam * max(tr, 0) * np.eye(2) + 2 * mu * sum(max(w[a], 0) * np.outer(V[:, a], V[:, a]) for a in range(2))
        Sm = lam * min(tr, 0) * np.eye(2) + 2 * mu * sum(min(w[a], 0) * np.outer(V[:, a], V[:, a]) for a in range(2))
        S = g * Sp + Sm
        pp, pm, s = element_response(m, exx, eyy, exy, g)
        scale = max(pp_ref + pm_ref, 1e-300)
        assert abs(pp - pp_ref) <= 1e-12 * scale and abs(pm - pm_ref) <= 1e-12 * scale
        np.testing.assert_allclose(s, [S[0, 0], S[1, 1], S[0, 1]], rtol=0, atol=1e-12 * max(np.abs(S).max(), 1e-300))


def test_starconvex_limits():
    """[R5] gamma* = 0 is the vol-dev split of Eq. 3; gamma* = -1 degrades everything (isotropic, PE)."""
    rng = np.random.default_rng(3)
    for plane in PLANES:
        for _ in range(50):
            e = rng.normal(0, 1e-3, 3)
            a = element_response(mat(split=3, plane=plane, gamma_star=0.0), *e, 0.4)
            b = element_response(mat(split=2, plane=plane), *e, 0.4)
            assert a[0] == b[0] and a[1] == b[1] and np.array_equal(a[2], b[2])
            c = element_response(mat(split=3, plane=plane, gamma_star=-1.0), *e, 0.4)
            i = element_response(mat(split=0, plane=plane), *e, 0.4)
            assert abs(c[0] - i[0]) <= 1e-12 * i[0] and c[1] == 0.0
            np.testing.assert_allclose(c[2], i[2], rtol=0, atol=1e-9 * np.abs(i[2]).max())


def test_amor_eq3_direct_plane_strain():
    """Eq. 3 typed out for plane strain: tr = exx+eyy, dev of the 3-D strain with ezz = 0."""
    m = mat(split=2, plane=0)
    K, mu = m.E / (3 * (1 - 2 * m.nu)), m.E / (2 * (1 + m.nu))
    for e in ([1e-3, 2e-4, -3e-4], [-1e-3, 2e-4, 3e-4]):
        E3 = np.array([[e[0], e[2], 0], [e[2], e[1], 0], [0, 0, 0]])
        tr = np.trace(E3)
        dev = E3 - tr / 3 * np.eye(3)
        pp, pm, _ = element_response(m, *e)
        assert abs(pp - (K / 2 * max(tr, 0) ** 2 + mu * np.sum(dev * dev))) < 1e-9
        assert abs(pm - K / 2 * min(tr, 0) ** 2) < 1e-9


# ---------------------------------------------------------------- internal force (L42-43, L124)
@pytest.mark.parametrize("split,plane", list(itertools.product(SPLITS, PLANES)))
def test_patch_test_and_rigid_body(split, plane):
    xy, tri = random_mesh(8, seed=5)
    m = OracleMesh(xy, tri, mat(split=split, plane=plane, gamma_star=1.0))
    n = 8
    ii, jj = np.arange(n * n) % n, np.arange(n * n) // n
    interior = (ii > 0) & (ii < n - 1) & (jj > 0) & (jj < n - 1)
    # patch test: affine displacement + uniform damage => zero force at interior nodes
    G = np.array([[1e-3, 4e-4], [-2e-4, -6e-4]])
    u = xy @ G.T + np.array([1e-5, -2e-5])
    f, _ = m.internal_force(u, np.full(m.N, 0.3))
    fscale = np.abs(f).max()
    assert fscale > 0
    assert np.abs(f[interior]).max() <= 1e-12 * fscale
    # rigid translation + infinitesimal rotation => zero force everywhere, zero psi+
    w = 1e-4
    ur = np.array([2e-5, -1e-5]) + np.stack([-w * xy[:, 1], w * xy[:, 0]], axis=1)
    fr, pp = m.internal_force(ur, np.random.default_rng(1).uniform(0, 0.9, m.N))
    assert np.abs(fr).max() <= 1e-12 * fscale
    f0, _ = m.internal_force(np.zeros((m.N, 2)), np.zeros(m.N))
    assert np.all(f0 == 0)  # f_int(0) = 0 (L134)


@pytest.mark.parametrize("split,plane", list(itertools.product(SPLITS, PLANES)))
def test_force_is_fd_gradient_of_elastic_energy(split, plane):
    """f_int = dE_el/du by central finite differences on a <= 50-element mesh (north_star pin);
    this pins the stress formulas of every split incl. the slaved eps_zz of plane stress [R4]."""
    xy, tri = random_mesh(5, seed=21)  # 32 elements
    m = OracleMesh(xy, tri, mat(split=split, plane=plane, gamma_star=0.7))
    rng = np.random.default_rng(split * 2 + plane)
    u = rng.normal(0, 2e-4, (m.N, 2))
    m.d = rng.uniform(0, 0.9, m.N)
    f, _ = m.internal_force(u)
    h = 1e-7 * 0.25
    fd = np.zeros_like(f)
    for i in range(m.N):
        for c in range(2):
            up, um = u.copy(), u.copy()
            up[i, c] += h
            um[i, c] -= h
            m.u = up
            ep = m.energies()[0]
            m.u = um
            em = m.energies()[0]
            fd[i, c] = (ep - em) / (2 * h)
    assert np.abs(f - fd).max() <= 2e-6 * np.abs(f).max()


def test_traction_resultant_and_momentum_balance():
    """Eq. 5 / [R8]: consistent edge load sums to t*L; with lumped mass the total momentum after n
    steps is n*dt*sum(f_ext) because internal forces cancel (L161-169)."""
    nx, ny = 9, 5
    xy, tri = grid_mesh(nx, ny, 0.008, 0.004)
    m = OracleMesh(xy, tri, mat(split=1))
    top = edge_segments(nx, ny, "top")
    m.add_traction(top, np.tile([3e5, 1e6], (len(top), 1)))
    np.testing.assert_allclose(m.fext.sum(axis=0), [3e5 * 0.008, 1e6 * 0.008], rtol=1e-14)
    assert np.all(m.fext[: nx * (ny - 1)] == 0)
    dt = 0.5 * m.dt_crit()
    m.init_accel()
    for _ in range(20):
        m.explicit_step(dt)
    mom = (m.mass[:, None] * m.v).sum(axis=0)
    # v_n = sum of trapezoids of a: a_0 counts half, a_1..a_{n-1} full, a_n half => (n) dt F
    np.testing.assert_allclose(mom, 20 * dt * m.fext.sum(axis=0), rtol=1e-10)


def test_free_flight_and_dirichlet():
    """Eq. 16-18 with zero force: u advances by dt*v exactly; Dirichlet dofs take u_bar, v_bar, a = 0 [R8]."""
    xy, tri = grid_mesh(4, 4, 1.0, 1.0)
    m = OracleMesh(xy, tri, mat(E=1e-30))
    m.v[:] = [2.0, -1.0]
    dof = np.array([0, 1, 7], dtype=np.int32)
    m.set_dirichlet(dof)
    m.init_accel()
    m.explicit_step(0.1, dir_u=[0.5, 0.6, 0.7], dir_v=[1.0, 2.0, 3.0])
    uf, vf, af = m.u.ravel(), m.v.ravel(), m.a.ravel()
    assert list(uf[dof]) == [0.5, 0.6, 0.7] and list(vf[dof]) == [1.0, 2.0, 3.0] and np.all(af[dof] == 0)
    free = np.setdiff1d(np.arange(2 * m.N), dof)
    v0 = np.tile([2.0, -1.0], m.N)
    np.testing.assert_allclose(uf[free], 0.1 * v0[free], rtol=1e-15)
    np.testing.assert_allclose(vf[free], v0[free], rtol=1e-15)


def test_shadow_energy_conservation_1000_steps():
    """Undamaged linear elastic wave, 10^3 steps at 0.5 dt_crit: velocity-Verlet conserves the shadow
    energy E* = E_kin + E_el - dt^2/8 sum m |a|^2 to round-off, plain E to O((w dt)^2) [R15]."""
    xy, tri = random_mesh(9, seed=2, jitter=0.2)
    m = OracleMesh(xy, tri, mat(split=0, eta=0.0))
    rng = np.random.default_rng(4)
    m.u = 1e-5 * np.sin(2 * np.pi * xy) + rng.normal(0, 1e-7, xy.shape)
    dt = 0.5 * m.dt_crit()
    m.init_accel()

    def shadow():
        e = m.energies()
        return e[0] + e[1] - dt**2 / 8 * np.sum(m.mass[:, None] * m.a**2), e[0] + e[1]

    s0, e0 = shadow()
    smax = emax = 0.0
    for _ in range(1000):
        m.explicit_step(dt)
        s, e = shadow()
        smax, emax = max(smax, abs(s - s0) / e0), max(emax, abs(e - e0) / e0)
    assert smax < 1e-10
    assert 1e-6 < emax < 0.2  # plain energy oscillates visibly but stays bounded
    assert np.all(m.H >= 0) and m.H.max() > 0


def test_history_is_running_max():
    xy, tri = random_mesh(6, seed=8)
    m = OracleMesh(xy, tri, mat(split=1))
    m.u = 1e-5 * np.sin(3 * xy)
    dt = 0.5 * m.dt_crit()
    m.init_accel()
    Hprev = m.H.copy()
    run = np.zeros(m.Ne)
    for _ in range(50):
        m.explicit_step(dt)
        _, pp = m.internal_force()
        run = np.maximum(run, pp)
        assert np.all(m.H >= Hprev)
        Hprev = m.H.copy()
    np.testing.assert_array_equal(m.H, run)


# ---------------------------------------------------------------- damage operator (L173, L185)
def dense_operator(m, H=None):
    return np.stack([m.damage_matvec(np.eye(m.N)[i], H) for i in range(m.N)], axis=1)


@pytest.mark.parametrize("model", [1, 2])
def test_damage_operator_textbook_stencils(model):
    """Uniform right-triangle grid: P1 diffusion = 5-point Laplacian (4, -1 x4, 0 on diagonals); the
    consistent mass (L185) row is h^2/12 * (6 centre, 1 for each of the 6 neighbours)."""
    n, h = 6, 0.5
    xy, tri = grid_mesh(n, n, h * (n - 1), h * (n - 1))
    p = dict(Gc=2.0, l0=0.7, model=model)
    m = OracleMesh(xy, tri, mat(**p))
    Hval = 1.3
    A = dense_operator(m, np.full(m.Ne, Hval))
    np.testing.assert_allclose(A, A.T, atol=1e-14)
    c = (p["Gc"] / p["l0"] + 2 * Hval) if model == 2 else 2 * Hval
    kap = p["Gc"] * p["l0"] if model == 2 else 0.75 * p["Gc"] * p["l0"]
    i = 2 + 2 * n  # interior node
    row = A[i].copy()
    expect = {i: c * h * h / 2 + 4 * kap, i + 1: c * h * h / 12 - kap, i - 1: c * h * h / 12 - kap,
              i + n: c * h * h / 12 - kap, i - n: c * h * h / 12 - kap,
              i + n + 1: c * h * h / 12, i - n - 1: c * h * h / 12}
    for j, v in expect.items():
        assert abs(row[j] - v) < 1e-13, (j, row[j], v)
        row[j] = 0
    assert np.abs(row).max() == 0
    b, D = m.damage_rhs_diag(np.full(m.Ne, Hval))
    np.testing.assert_allclose(D, np.diag(A), rtol=1e-14)
    src = 2 * Hval if model == 2 else 2 * Hval - 3 * p["Gc"] / (8 * p["l0"])
    assert abs(b[i] - src * h * h) < 1e-13  # int src phi_i = src * (patch area)/3 = src h^2
    assert abs(b.sum() - src * (h * (n - 1)) ** 2) < 1e-12


def test_damage_operator_general_mesh_properties():
    xy, tri = random_mesh(6, seed=9)
    m = OracleMesh(xy, tri, mat(model=2, Gc=2.0, l0=0.1))
    H = np.random.default_rng(0).uniform(0, 3, m.Ne)
    A = dense_operator(m, H)
    np.testing.assert_allclose(A, A.T, atol=1e-12)
    assert np.linalg.eigvalsh(A).min() > 0  # SPD (L173)
    # A 1 = int c phi_i (constants are in the kernel of the diffusion term): sum_i = sum_e c_e A_e
    c = 2.0 / 0.1 + 2 * H
    assert abs(A.sum() - np.sum(c * m.area)) < 1e-11
    assert np.all(m.damage_matvec(np.zeros(m.N), H) == 0)


def strip(nx, ny, L, W):
    xy, tri = grid_mesh(nx, ny, L, W)
    left = (np.arange(ny) * nx).astype(np.int32)
    return xy, tri, left


def test_at2_profile_cosh_and_convergence():
    """1-D AT2 profile (Fig. 1 caption, L83): H = 0, d = 1 on x = 0, natural BC elsewhere =>
    d = cosh((L-x)/l0)/cosh(L/l0) -> exp(-x/l0); P1 error is O(h^2) (factor ~4 per halving)."""
    l0, L = 1.0, 8.0
    errs = []
    for k in (2, 4, 8):
        nx = 8 * k + 1
        xy, tri, left = strip(nx, 3, L, 2 * L / (nx - 1))
        m = OracleMesh(xy, tri, mat(model=2, Gc=1.0, l0=l0))
        m.d[left] = 1.0
        m.set_damage_dirichlet(left)
        rc, it, rr = m.damage_solve(rel_tol=1e-13, max_iter=5000)
        assert rc == 0
        exact = np.cosh((L - xy[:, 0]) / l0) / np.cosh(L / l0)
        errs.append(np.abs(m.d - exact).max())
        assert np.abs(exact - np.exp(-xy[:, 0] / l0)).max() < 1.01 * np.exp(-L / l0)  # finite-strip tail
    assert errs[0] < 2e-2 and errs[2] < 1.5e-3
    assert 3.3 < errs[0] / errs[1] < 5.5 and 3.3 < errs[1] / errs[2] < 5.5


def test_at1_profile_exact_and_fracture_energy():
    """1-D AT1 profile (L83): d = <1 - x/(2 l0)>_+^2, compact support; with 2 l0/h integer the discrete
    bound-constrained solution is nodally exact [R17]; E_frac ~ Gc * (crack length) * 1/2 (one side)."""
    l0, h = 1.0, 0.25
    nx = int(6 / h) + 1
    xy, tri, left = strip(nx, 3, 6.0, 2 * h)
    m = OracleMesh(xy, tri, mat(model=1, Gc=1.0, l0=l0))
    m.d[left] = 1.0
    m.set_damage_dirichlet(left)
    rc, it, rr = m.damage_solve(rel_tol=1e-14, max_iter=5000)
    assert rc == 0
    exact = np.maximum(1 - xy[:, 0] / (2 * l0), 0) ** 2
    assert np.abs(m.d - exact).max() < 1e-12
    assert np.all(m.d[xy[:, 0] >= 2 * l0] == 0)
    # half of the optimal profile carries Gc/2 per unit crack length (width 2h here): interpolation error O(h^2)
    assert abs(m.energies()[2] - 0.5 * 1.0 * 2 * h) < 0.02 * 2 * h


def test_at2_fracture_energy_of_profile():
    l0, L, h = 1.0, 12.0, 0.125
    nx = int(L / h) + 1
    xy, tri, left = strip(nx, 2, L, h)
    m = OracleMesh(xy, tri, mat(model=2, Gc=3.0, l0=l0))
    m.d = np.exp(-xy[:, 0] / l0)
    # int_0^inf (d^2/(2 l0) + l0/2 d'^2) dx = 1/2 for the exponential profile => Gc * width * 1/2
    assert abs(m.energies()[2] - 3.0 * h * 0.5) < 5e-3 * 3.0 * h


def test_at1_threshold_homogeneous():
    """AT1 elastic threshold H_crit = 3 Gc / (16 l0) (L69): below it d stays 0; above it the
    homogeneous solution of Eq. 8 is d = 1 - 3 Gc / (16 l0 H)."""
    xy, tri = random_mesh(6, seed=3)
    Gc, l0 = 2.0, 0.1
    Hc = 3 * Gc / (16 * l0)
    m = OracleMesh(xy, tri, mat(model=1, Gc=Gc, l0=l0))
    m.H[:] = 0.99 * Hc
    assert m.damage_solve(rel_tol=1e-13)[0] == 0 and np.all(m.d == 0)
    m.H[:] = 2.5 * Hc
    assert m.damage_solve(rel_tol=1e-13, max_iter=5000)[0] == 0
    np.testing.assert_allclose(m.d, 1 - Hc / (2.5 * Hc), atol=1e-11)


def test_at2_homogeneous_closed_form():
    """Eq. 6 with uniform H and no gradient: d = 2H / (Gc/l0 + 2H)."""
    xy, tri = random_mesh(6, seed=4)
    m = OracleMesh(xy, tri, mat(model=2, Gc=2.0, l0=0.1))
    m.H[:] = 7.0
    assert m.damage_solve(rel_tol=1e-13, max_iter=5000)[0] == 0
    np.testing.assert_allclose(m.d, 14.0 / (20.0 + 14.0), atol=1e-11)


def _bruteforce_bound_qp(A, b, lb, fixed_mask, xfixed):
    """Enumerate every active set; return the unique KKT point of min 1/2 x'Ax - b'x s.t. x >= lb."""
    n = len(b)
    free = np.nonzero(~fixed_mask)[0]
    sols = []
    for mask in itertools.product([0, 1], repeat=len(free)):
        act = free[np.array(mask, dtype=bool)]
        ina = free[~np.array(mask, dtype=bool)]
        x = np.where(fixed_mask, xfixed, lb).astype(float)
        if len(ina):
            rhs = b[ina] - A[np.ix_(ina, np.setdiff1d(np.arange(n), ina))] @ x[np.setdiff1d(np.arange(n), ina)]
            x[ina] = np.linalg.solve(A[np.ix_(ina, ina)], rhs)
        r = b - A @ x
        if np.all(x[ina] >= lb[ina] - 1e-13) and np.all(r[act] <= 1e-13):
            sols.append(x)
    return sols


def test_at1_projected_cg_against_bruteforce_active_sets():
    """[R12] the AT1 solve returns the unique minimiser of the bound-constrained quadratic: brute-force
    enumeration of all active sets on a 12-free-node mesh, plus projected Gauss-Seidel."""
    xy, tri = random_mesh(4, seed=13)  # 16 nodes
    Gc, l0 = 1.0, 0.4
    m = OracleMesh(xy, tri, mat(model=1, Gc=Gc, l0=l0))
    rng = np.random.default_rng(5)
    for trial in range(4):
        m.H = rng.uniform(0, 4 * 3 * Gc / (16 * l0), m.Ne) * (rng.uniform(size=m.Ne) < 0.6)
        d0 = np.where(rng.uniform(size=m.N) < 0.3, rng.uniform(0, 0.5, m.N), 0.0)
        fixed = np.zeros(m.N, dtype=bool)
        fixed[[0, 5, 10, 15]] = True
        d0[fixed] = [1.0, 0.0, 0.8, 0.2]
        m.d = d0.copy()
        m.set_damage_dirichlet(np.nonzero(fixed)[0])
        rc, it, rr = m.damage_solve(rel_tol=1e-14, max_iter=2000)
        assert rc == 0
        A = dense_operator(m)
        b, _ = m.damage_rhs_diag()
        sols = _bruteforce_bound_qp(A, b, d0, fixed, d0)
        assert len(sols) >= 1
        for s in sols[1:]:
            np.testing.assert_allclose(s, sols[0], atol=1e-10)
        np.testing.assert_allclose(m.d, np.minimum(sols[0], 1.0), atol=1e-11)
        # projected Gauss-Seidel to the same point
        x = d0.copy()
        for _ in range(4000):
            for i in np.nonzero(~fixed)[0]:
                x[i] = max(d0[i], x[i] + (b[i] - A[i] @ x) / A[i, i])
        np.testing.assert_allclose(m.d, np.minimum(x, 1.0), atol=1e-10)
        assert np.all(m.d >= d0) and np.all(m.d <= 1)


def test_at2_solve_against_dense_and_irreversibility():
    """AT2: unconstrained SPD solve on the free nodes, then clamp to [d_n, 1] (L179)."""
    xy, tri = random_mesh(7, seed=17)
    m = OracleMesh(xy, tri, mat(model=2, Gc=1.0, l0=0.2))
    rng = np.random.default_rng(2)
    m.H = rng.uniform(0, 30, m.Ne)
    d0 = rng.uniform(0, 1, m.N) * (rng.uniform(size=m.N) < 0.5)
    fixed = np.zeros(m.N, dtype=bool)
    fixed[:7] = True
    d0[fixed] = 1.0
    m.d = d0.copy()
    m.set_damage_dirichlet(np.nonzero(fixed)[0])
    assert m.damage_solve(rel_tol=1e-14, max_iter=3000)[0] == 0
    A = dense_operator(m)
    b, _ = m.damage_rhs_diag()
    fr = ~fixed
    x = d0.copy()
    x[fr] = np.linalg.solve(A[np.ix_(fr, fr)], b[fr] - A[np.ix_(fr, fixed)] @ d0[fixed])
    np.testing.assert_allclose(m.d, np.clip(np.maximum(x, d0), 0, 1), atol=1e-11)
    assert np.all(m.d >= d0) and np.all(m.d <= 1) and np.all(m.d >= 0)
    assert np.any(x < d0 - 1e-6)  # the clamp is exercised


@pytest.mark.parametrize("model", [1, 2])
def test_staggered_run_irreversibility_and_range(model):
    """d_{n+1} >= d_n and 0 <= d <= 1 over a loaded staggered run (L114, L179)."""
    nx, ny = 21, 9
    xy, tri = grid_mesh(nx, ny, 0.020, 0.008)
    m = OracleMesh(xy, tri, mat(model=model, split=2 if model == 1 else 1, l0=1e-3))
    notch = (np.arange(nx // 2 + 1) + (ny // 2) * nx).astype(np.int32)
    m.d[notch] = 1.0
    m.set_damage_dirichlet(notch)
    top, bot = edge_segments(nx, ny, "top"), edge_segments(nx, ny, "bottom")
    m.add_traction(top, np.tile([0.0, 6e6], (len(top), 1)))
    m.add_traction(bot, np.tile([0.0, -6e6], (len(bot), 1)))
    dt = 0.5 * m.dt_crit()
    m.init_accel()
    grew = False
    for _ in range(150):
        dprev = m.d.copy()
        m.explicit_step(dt)
        rc, it, rr = m.damage_solve(rel_tol=1e-8)
        assert rc == 0
        assert np.all(m.d >= dprev) and m.d.min() >= 0 and m.d.max() <= 1
        grew |= bool(np.any(m.d > dprev + 1e-6))
    assert grew
    e = m.energies()
    assert e[3] == e[0] + e[1] + e[2] and e[1] > 0


def test_kinetic_energy_closed_form():
    xy, tri = grid_mesh(5, 5, 2.0, 2.0)
    m = OracleMesh(xy, tri, mat())
    m.v[:] = [3.0, 4.0]
    assert abs(m.energies()[1] - 0.5 * GLASS["rho"] * 4.0 * 25.0) < 1e-9
