"""GPU parity of pff_damage_adjoint / pff_damage_param_terms (through the C ABI) against oracle/pff_adjoint_oracle.py
(assembled operator + direct solve): PAPER.md section 4.2, Eq. 22-24; SURVEY.md 8(f) NEXT-2."""
import numpy as np
import pytest

from oracle import pff_adjoint_oracle as adj
from pff_inputs import GLASS, config, random_mesh

pytestmark = pytest.mark.gpu


def _gpu_mesh(xy, tri, material, H, fixed=(), precision=0, chunk_elems=0):
    import paper_2606_23458_b200 as pff
    mesh = pff.Mesh(xy, tri, material, precision=precision, chunk_elems=chunk_elems)
    st = mesh.new_state(H=H)
    if len(fixed):
        mesh.pff_set_damage_dirichlet(np.asarray(fixed, dtype=np.int32))
    return mesh, st


def _mask_tensor(mesh, free_user):
    import torch
    m = np.empty(len(free_user), dtype=np.uint8)
    m[mesh.node_new_of_old] = free_user.astype(np.uint8)
    return torch.from_numpy(m).to(mesh.device)


@pytest.mark.parametrize("model", [1, 2])
@pytest.mark.parametrize("masked", [False, True])
def test_adjoint_solve_matches_direct_solve(model, masked):
    """Several chunks, jittered mesh with mixed orientations, Dirichlet nodes and (masked) a caller-given free set."""
    xy, tri = random_mesh(33, 11)
    r = np.random.default_rng(12)
    Gc, l0 = 3.0, 0.05
    H = r.uniform(0.2, 3.0, len(tri)) * Gc / l0
    material = dict(GLASS, Gc=Gc, l0=l0, model=model, split=1, plane=0)
    fixed = np.array([0, 5, 100, 517, 1088], dtype=np.int32)
    free = np.ones(len(xy), dtype=bool)
    if masked:
        free = r.uniform(size=len(xy)) < 0.8
    g = r.standard_normal(len(xy))
    A, _ = adj.damage_system(xy, tri, H, Gc, l0, model)
    free_o = free.copy()
    free_o[fixed] = False
    lam_o = adj.adjoint_solve(A, g, free_o)

    mesh, st = _gpu_mesh(xy, tri, material, H, fixed, chunk_elems=256)
    lam_t, status, iters, relres = mesh.pff_damage_adjoint(st, mesh.nodes_to_internal(g),
                                                          _mask_tensor(mesh, free) if masked else None,
                                                          rel_tol=1e-13, max_iter=5000)
    assert status == 0 and iters > 0 and relres <= 1e-13
    lam = mesh.nodes_to_user(lam_t)
    assert np.all(lam[~free_o] == 0.0)
    assert np.abs(lam - lam_o).max() <= 1e-10 * np.abs(lam_o).max()

    # the two scalars of Eq. 24 against the assembled M and K
    d = r.uniform(0.0, 1.0, len(xy))
    M, K = adj.mass_stiffness(xy, tri)
    tM, tK = mesh.pff_damage_param_terms(lam_t, mesh.nodes_to_internal(d))
    oM, oK = adj.param_terms(M, K, lam, d)
    assert abs(tM - oM) <= 1e-11 * abs(oM) and abs(tK - oK) <= 1e-11 * abs(oK)


def test_gc_gradient_end_to_end_against_forward_finite_differences():
    """dL/dG_c from the GPU adjoint (Eq. 24) against central differences of GPU FORWARD solves at perturbed G_c."""
    xy, tri = random_mesh(25, 21)
    r = np.random.default_rng(22)
    Gc, l0 = 3.0, 0.06
    H = r.uniform(0.2, 3.0, len(tri)) * Gc / l0
    g = r.standard_normal(len(xy))

    def forward(gc):
        mesh, st = _gpu_mesh(xy, tri, dict(GLASS, Gc=gc, l0=l0, model=2, split=1, plane=0), H)
        status, _, _ = mesh.pff_damage_solve(st, rel_tol=1e-13, max_iter=5000)
        assert status == 0
        return mesh, st

    mesh, st = forward(Gc)
    d = mesh.nodes_to_user(st.d)
    assert d.min() > 0.0 and d.max() < 1.0  # clamp inactive: the forward result solves Eq. 22
    lam_t, status, _, _ = mesh.pff_damage_adjoint(st, mesh.nodes_to_internal(g), None, rel_tol=1e-13, max_iter=5000)
    assert status == 0
    tM, tK = mesh.pff_damage_param_terms(lam_t, st.d)
    dGc = -(tM / l0 + l0 * tK)
    eps = 1e-5
    vals = []
    for s in (+1, -1):
        m2, s2 = forward(Gc * (1 + s * eps))
        vals.append(g @ m2.nodes_to_user(s2.d))
    fd = (vals[0] - vals[1]) / (2 * eps * Gc)
    assert abs(fd - dGc) <= 1e-6 * abs(dGc)


def test_adjoint_fp32_and_config_mesh():
    """Config 1 plate (notch = damage-Dirichlet), both precisions: fp64 to 1e-9, fp32 to the north_star fp32 tolerance."""
    cfg = config(1)
    xy, tri, material = cfg["xy"], cfg["tri"], cfg["material"]
    r = np.random.default_rng(31)
    H = r.uniform(0.0, 2.0, len(tri)) * material["Gc"] / material["l0"]
    g = r.standard_normal(len(xy))
    A, _ = adj.damage_system(xy, tri, H, material["Gc"], material["l0"], material["model"])
    free = np.ones(len(xy), dtype=bool)
    free[cfg["notch"]] = False
    lam_o = adj.adjoint_solve(A, g, free)
    for precision, tol, cg_tol in ((0, 1e-9, 1e-12), (1, 2e-5, 1e-6)):
        mesh, st = _gpu_mesh(xy, tri, material, H, cfg["notch"], precision=precision)
        lam_t, status, _, relres = mesh.pff_damage_adjoint(st, mesh.nodes_to_internal(g), None, rel_tol=cg_tol, max_iter=5000,
                                                           allow_noconv=(precision == 1))
        assert relres <= 10 * cg_tol
        lam = mesh.nodes_to_user(lam_t)
        assert np.abs(lam - lam_o).max() <= tol * np.abs(lam_o).max()


# ---------------------------------------------------------------- matrix-free stiffness action (Eq. 11-15, NEXT-3)
@pytest.mark.parametrize("split", [0, 1, 2, 3])
@pytest.mark.parametrize("plane", [0, 1])
def test_stiffness_action_matches_oracle(split, plane):
    """q = f_int(u + p) - f_int(u) in one fused pass against the C oracle's difference of two internal forces (Eq. 13),
    several chunks with halos, every split; for the isotropic split also against the assembled K (Eq. 14)."""
    from oracle import Material, OracleMesh
    xy, tri = random_mesh(33, 41)
    material = dict(GLASS, model=2, split=split, plane=plane, gamma_star=1.0 if split == 3 else 0.0)
    r = np.random.default_rng(42)
    u = 1e-4 * r.standard_normal((len(xy), 2))
    d = r.uniform(0.0, 0.9, len(xy))
    p = 1e-4 * r.standard_normal((len(xy), 2))
    orc = OracleMesh(xy, tri, Material(**material))
    orc.u[:] = u
    orc.d[:] = d
    q_o = orc.stiffness_action(p)

    import paper_2606_23458_b200 as pff
    mesh = pff.Mesh(xy, tri, material, chunk_elems=256)
    st = mesh.new_state(u=u, d=d)
    qx, qy = mesh.pff_stiffness_action(st, mesh.nodes_to_internal(p[:, 0]), mesh.nodes_to_internal(p[:, 1]))
    q = np.stack([mesh.nodes_to_user(qx), mesh.nodes_to_user(qy)], 1)
    assert np.abs(q - q_o).max() <= 1e-10 * np.abs(q_o).max()
    qx2, qy2 = mesh.pff_stiffness_action(st, mesh.nodes_to_internal(p[:, 0]), mesh.nodes_to_internal(p[:, 1]))
    assert np.array_equal(qx.cpu().numpy(), qx2.cpu().numpy()) and np.array_equal(qy.cpu().numpy(), qy2.cpu().numpy())
    if split == 0:
        from oracle import pff_stiffness_oracle as sto
        K = sto.assemble_stiffness(xy, tri, material["E"], material["nu"], plane, d, material["eta"])
        q_K = (K @ p.ravel()).reshape(-1, 2)
        assert np.abs(q - q_K).max() <= 1e-10 * np.abs(q_K).max()


def test_stiffness_action_full_size():
    """cfg5_1001 (the bench mesh and launch configuration): the action at every node against the oracle."""
    cfg = config(5, n=1001)
    from _harness import gpu_from, oracle_from
    orc = oracle_from(cfg)
    mesh, st = gpu_from(cfg)
    r = np.random.default_rng(43)
    p = 1e-6 * r.standard_normal((len(cfg["xy"]), 2))
    q_o = orc.stiffness_action(p)
    qx, qy = mesh.pff_stiffness_action(st, mesh.nodes_to_internal(p[:, 0]), mesh.nodes_to_internal(p[:, 1]))
    q = np.stack([mesh.nodes_to_user(qx), mesh.nodes_to_user(qy)], 1)
    assert np.abs(q - q_o).max() <= 1e-8 * np.abs(q_o).max()  # cancellation: |u| / |p| ~ 1e2..1e3 ulp amplification


# ---------------------------------------------------------------- quasi-static mechanics solve (L126-159, L337)
def _equilibrium_case(n, seed, split=0):
    from pff_inputs import edge_segments
    xy, tri = random_mesh(n, seed)
    material = dict(GLASS, model=2, split=split, plane=0)
    d = np.random.default_rng(seed + 1).uniform(0.0, 0.9, len(xy))
    top = edge_segments(n, n, "top")
    trac = np.tile([2e5, 1e6], (len(top), 1))
    bottom = np.arange(n)
    dir_dof = np.concatenate([2 * bottom, 2 * bottom + 1]).astype(np.int32)
    return xy, tri, material, d, top, trac, dir_dof


@pytest.mark.parametrize("precision", [0, 1])
def test_equilibrium_solve_matches_assembled_direct_solve(precision):
    """Isotropic split (linear problem): clamped bottom edge with prescribed values, traction on top, damaged solid,
    several chunks; the GPU CG on the matrix-free action against the assembled K + direct solve."""
    from oracle import pff_stiffness_oracle as sto
    import paper_2606_23458_b200 as pff
    n = 33
    xy, tri, material, d, top, trac, dir_dof = _equilibrium_case(n, 51)
    r = np.random.default_rng(52)
    dir_u = 1e-5 * r.standard_normal(len(dir_dof))
    S = 0.7
    mesh = pff.Mesh(xy, tri, material, precision=precision, chunk_elems=256)
    st = mesh.new_state(d=d)
    mesh.pff_set_traction(st, top, trac)
    mesh.pff_set_dirichlet(dir_dof)
    bc = mesh.bc(dir_u=dir_u, dir_v=np.zeros(len(dir_dof)), load_scale=S)
    status, iters, relres = mesh.pff_equilibrium_solve(st, bc, rel_tol=1e-12 if precision == 0 else 1e-6, max_iter=20000,
                                                       allow_noconv=(precision == 1))
    assert iters > 0 and relres <= (1e-12 if precision == 0 else 1e-4)
    u = np.stack([mesh.nodes_to_user(st.ux), mesh.nodes_to_user(st.uy)], 1)

    fext = np.stack([mesh.nodes_to_user(st.fext_x), mesh.nodes_to_user(st.fext_y)], 1)
    K = sto.assemble_stiffness(xy, tri, material["E"], material["nu"], 0, d, material["eta"])
    u0 = np.zeros((len(xy), 2))
    u0.ravel()[dir_dof] = dir_u
    u_o = sto.equilibrium_solve(K, u0, fext, S, dir_dof)
    assert np.abs(u - u_o).max() <= (1e-8 if precision == 0 else 2e-3) * np.abs(u_o).max()
    assert np.abs(u.ravel()[dir_dof] - dir_u).max() <= (0 if precision == 0 else 1e-12)


def test_equilibrium_solve_balances_forces_and_is_reproducible():
    """The solved state satisfies f_int(u) = S f_ext on the free dofs according to the C ORACLE's internal force, and a
    second solve from the same start gives the same bits."""
    from oracle import Material, OracleMesh
    import paper_2606_23458_b200 as pff
    n = 25
    xy, tri, material, d, top, trac, dir_dof = _equilibrium_case(n, 61)
    orc = OracleMesh(xy, tri, Material(**material))
    orc.d[:] = d
    orc.add_traction(top, trac)
    out = []
    for _ in range(2):
        mesh = pff.Mesh(xy, tri, material)
        st = mesh.new_state(d=d)
        mesh.pff_set_traction(st, top, trac)
        mesh.pff_set_dirichlet(dir_dof)
        status, iters, relres = mesh.pff_equilibrium_solve(st, mesh.bc(), rel_tol=1e-12, max_iter=20000)
        assert status == 0
        out.append(np.stack([mesh.nodes_to_user(st.ux), mesh.nodes_to_user(st.uy)], 1))
    assert np.array_equal(out[0], out[1])
    f, _ = orc.internal_force(out[0])
    res = (f - orc.fext).ravel()
    free = np.ones(2 * len(xy), dtype=bool)
    free[dir_dof] = False
    assert np.abs(res[free]).max() <= 1e-9 * np.abs(orc.fext).max()


def test_equilibrium_step_for_the_spectral_split_under_tension():
    """Spectral split with every principal strain positive (biaxial pre-stretch): psi+ = psi, the shifted difference is
    linear and one solve reaches the same equilibrium as the assembled isotropic operator."""
    from oracle import pff_stiffness_oracle as sto
    import paper_2606_23458_b200 as pff
    n = 17
    xy, tri, material, d, top, trac, dir_dof = _equilibrium_case(n, 71, split=1)
    d = 0.2 * d  # mild stiffness contrast: the equilibrium strain field stays tensile in every element
    i, j = np.arange(n * n) % n, np.arange(n * n) // n
    bn = np.nonzero((i == 0) | (i == n - 1) | (j == 0) | (j == n - 1))[0]
    dir_dof = np.concatenate([2 * bn, 2 * bn + 1]).astype(np.int32)
    stretch = 1e-3 * xy                                  # eps = 1e-3 I: both principal strains positive
    u_start = stretch.copy()
    inner = np.setdiff1d(np.arange(n * n), bn)
    u_start[inner] += 1e-7 * np.random.default_rng(72).standard_normal((len(inner), 2))  # off equilibrium, still tensile
    mesh = pff.Mesh(xy, tri, material)
    st = mesh.new_state(u=u_start, d=d)
    mesh.pff_set_dirichlet(dir_dof)
    status, _, _ = mesh.pff_equilibrium_solve(st, mesh.bc(), rel_tol=1e-12, max_iter=20000)
    assert status == 0
    u = np.stack([mesh.nodes_to_user(st.ux), mesh.nodes_to_user(st.uy)], 1)
    K = sto.assemble_stiffness(xy, tri, material["E"], material["nu"], 0, d, material["eta"])
    u0 = np.zeros_like(u)
    u0[bn] = stretch[bn]
    u_o = sto.equilibrium_solve(K, u0, np.zeros_like(u0), 1.0, dir_dof)
    assert np.abs(u - u_o).max() <= 1e-8 * np.abs(u_o).max()
