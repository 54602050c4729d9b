"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

This module holds NO arithmetic of the method (no strains, energies, CFL, mass ...): it only
generates meshes, index sets, material parameter dictionaries and initial nodal fields.  The
recipes are the ones of DESIGN.md "Input recipe" (BASELINE.json `configs` 1-5); they stand in for
the paper's Gmsh benchmark meshes B1-B4, which are not available, keeping the
paper's P1 workload shape Ne/N ~ 2 and nodal valence ~ 6.

Conventions: SI units; grid node id = i + j*nx; each quad (i, j) is split along its lower-left ->
upper-right diagonal into (n00, n10, n11) and (n00, n11, n01), element id = 2*(i + j*(nx-1)) + {0,1}.
"""
from __future__ import annotations

import numpy as np

GLASS = dict(E=32e9, nu=0.2, rho=2450.0, Gc=3.0, l0=5e-4, eta=1e-7, gamma_star=0.0)

AT1, AT2 = 1, 2
ISO, SPECTRAL, VOLDEV, STARCONVEX = 0, 1, 2, 3
PLANE_STRAIN, PLANE_STRESS = 0, 1


def grid_mesh(nx: int, ny: int, Lx: float, Ly: float):
    """Structured nx x ny node grid on [0,Lx]x[0,Ly], 2 triangles per quad."""
    x = np.linspace(0.0, Lx, nx)
    y = np.linspace(0.0, Ly, ny)
    X, Y = np.meshgrid(x, y)  # [ny, nx]
    xy = np.stack([X.ravel(), Y.ravel()], axis=1)
    i, j = np.meshgrid(np.arange(nx - 1), np.arange(ny - 1))
    n00 = (i + j * nx).ravel()
    n10, n01, n11 = n00 + 1, n00 + nx, n00 + nx + 1
    tri = np.empty((2 * len(n00), 3), dtype=np.int32)
    tri[0::2] = np.stack([n00, n10, n11], axis=1)
    tri[1::2] = np.stack([n00, n11, n01], axis=1)
    return np.ascontiguousarray(xy), tri


def edge_segments(nx: int, ny: int, side: str):
    """Boundary edge node pairs of a grid_mesh side ('top' | 'bottom' | 'left' | 'right')."""
    if side == "bottom":
        a = np.arange(nx - 1)
    elif side == "top":
        a = np.arange(nx - 1) + (ny - 1) * nx
    elif side == "left":
        a = np.arange(ny - 1) * nx
    elif side == "right":
        a = np.arange(ny - 1) * nx + nx - 1
    else:
        raise ValueError(side)
    step = 1 if side in ("top", "bottom") else nx
    return np.stack([a, a + step], axis=1).astype(np.int32)


def edge_nodes(nx: int, ny: int, side: str):
    s = edge_segments(nx, ny, side)
    return np.unique(s.ravel()).astype(np.int32)


def _plate(nx, ny, Lx, Ly, notch_j, notch_imax, traction):
    xy, tri = grid_mesh(nx, ny, Lx, Ly)
    notch = (np.arange(notch_imax + 1) + notch_j * nx).astype(np.int32)
    top, bot = edge_segments(nx, ny, "top"), edge_segments(nx, ny, "bottom")
    edges = np.concatenate([top, bot])
    t = np.concatenate([np.tile([0.0, traction], (len(top), 1)), np.tile([0.0, -traction], (len(bot), 1))])
    return xy, tri, notch, edges, t


def config(k: int, scale: float = 1.0, n: int | None = None):
    """BASELINE.json config k (1..5) as a dict of plain arrays.

    scale < 1 shrinks the node counts (for fast tests) while keeping the recipe; `n` selects the
    grid side for config 5.  Keys: xy, tri, material (dict), model/split/plane inside material,
    notch (damage-Dirichlet nodes with d=1), edges + traction (host arrays), dir_dof (+ dir_u,
    dir_v callables of step index) , d0, u0, dt_factor (x CFL), steps, name.
    """
    if k == 1:
        nx, ny = int(round(100 * scale)) + 1, int(round(40 * scale)) + 1
        xy, tri, notch, edges, t = _plate(nx, ny, 0.100, 0.040, (ny - 1) // 2, (nx - 1) // 2, 1e6)
        mat = dict(GLASS, model=AT2, split=VOLDEV, plane=PLANE_STRAIN)
        return _pack("cfg1_plate_101x41_AT2_voldev_PE", xy, tri, mat, notch, edges, t, steps=200)
    if k == 2:
        nx, ny = int(round(400 * scale)) + 1, int(round(160 * scale)) + 1
        xy, tri, notch, edges, t = _plate(nx, ny, 0.100, 0.040, (ny - 1) // 2, (nx - 1) // 2, 1e6)
        h = 0.100 / (nx - 1)
        J = np.random.default_rng(1).uniform(-0.2 * h, 0.2 * h, (nx * ny, 2))
        ii, jj = np.arange(nx * ny) % nx, np.arange(nx * ny) // nx
        interior = (ii > 0) & (ii < nx - 1) & (jj > 0) & (jj < ny - 1)
        xy = xy + J * interior[:, None]
        tri = np.ascontiguousarray(tri[np.random.default_rng(2).permutation(len(tri))])
        mat = dict(GLASS, model=AT2, split=SPECTRAL, plane=PLANE_STRAIN)
        return _pack("cfg2_plate_401x161_AT2_spectral_PE_jitter", xy, tri, mat, notch, edges, t, steps=2000)
    if k == 3:
        nn = int(round(1000 * scale)) + 1
        h = 1.0 / (nn - 1)
        xy, tri = grid_mesh(nn, nn, 1.0, 1.0)
        Cc = np.random.default_rng(3).uniform(0.0, 1.0, (20, 2))
        seed = np.zeros(nn * nn, dtype=bool)
        for c in Cc:
            seed |= (xy[:, 0] - c[0]) ** 2 + (xy[:, 1] - c[1]) ** 2 <= (3.0 * h) ** 2
        notch = np.nonzero(seed)[0].astype(np.int32)
        # nondimensional material (BASELINE.json gives none): E=1, nu=0.3, rho=1, l0=4h, Gc=1e-6
        mat = dict(E=1.0, nu=0.3, rho=1.0, Gc=1e-6, l0=4.0 * h, eta=1e-7, gamma_star=1.0,
                   model=AT1, split=STARCONVEX, plane=PLANE_STRESS)
        bot, top = edge_nodes(nn, nn, "bottom"), edge_nodes(nn, nn, "top")
        dir_dof = np.concatenate([2 * bot, 2 * bot + 1, 2 * top, 2 * top + 1]).astype(np.int32)
        ntop = len(top)
        cfg = _pack("cfg3_square_1001_AT1_starconvex_PS", xy, tri, mat, notch,
                    np.zeros((0, 2), np.int32), np.zeros((0, 2)), steps=500)
        cfg.update(dir_dof=dir_dof, shear=dict(n_fixed=2 * len(bot), n_top=ntop, vbar=6.8e-3, ramp_steps=50))
        return cfg
    if k == 4:
        nx, ny = int(round(2000 * scale)) + 1, int(round(1000 * scale)) + 1
        Lx, Ly = 0.200, 0.100
        xy, tri = grid_mesh(nx, ny, Lx, Ly)
        g = np.random.default_rng(4)
        holes = []
        ny_mid = Ly / 2
        while len(holes) < 40:
            r, cx, cy = g.uniform(2e-3, 6e-3), g.uniform(0.0, Lx), g.uniform(0.0, Ly)
            gap = 1e-3
            if cx - r < gap or cx + r > Lx - gap or cy - r < gap or cy + r > Ly - gap:
                continue
            if any((cx - a) ** 2 + (cy - b) ** 2 < (r + c + gap) ** 2 for a, b, c in holes):
                continue
            # distance to the notch segment y = Ly/2, 0 <= x <= 0.010
            px = min(max(cx, 0.0), 0.010)
            if (cx - px) ** 2 + (cy - ny_mid) ** 2 < (r + gap) ** 2:
                continue
            holes.append((cx, cy, r))
        cen = xy[tri].mean(axis=1)
        keep = np.ones(len(tri), dtype=bool)
        for cx, cy, r in holes:
            keep &= (cen[:, 0] - cx) ** 2 + (cen[:, 1] - cy) ** 2 > r * r
        tri = tri[keep]
        used = np.zeros(nx * ny, dtype=bool)
        used[tri.ravel()] = True
        new_id = np.cumsum(used) - 1
        jn = (ny - 1) // 2
        notch_old = np.arange(nx * ny)[(np.arange(nx * ny) // nx == jn) & (xy[:, 0] <= 0.010 + 1e-12) & used]
        top_s, bot_s = edge_segments(nx, ny, "top"), edge_segments(nx, ny, "bottom")
        edges_old = np.concatenate([top_s, bot_s])
        t = np.concatenate([np.tile([0.0, 2e6], (len(top_s), 1)), np.tile([0.0, -2e6], (len(bot_s), 1))])
        xy = np.ascontiguousarray(xy[used])
        tri = np.ascontiguousarray(new_id[tri].astype(np.int32))
        mat = dict(GLASS, model=AT2, split=VOLDEV, plane=PLANE_STRAIN)
        cfg = _pack("cfg4_perforated_2001x1001_AT2_voldev_PE", xy, tri, mat, new_id[notch_old].astype(np.int32),
                    new_id[edges_old].astype(np.int32), t, steps=500)
        cfg["holes"] = np.array(holes)
        return cfg
    if k == 5:
        nn = n if n is not None else 1001
        h = 1e-3
        L = (nn - 1) * h
        xy, tri = grid_mesh(nn, nn, L, L)
        g = np.random.default_rng(5)
        pq = g.integers(1, 5, size=(8, 2))
        phi = g.uniform(0.0, 2 * np.pi, 8)
        chi = g.uniform(0.0, 2 * np.pi, 8)
        u0 = np.zeros((nn * nn, 2))
        amp = 1e-4 * L / 8
        for kk in range(8):
            arg = 2 * np.pi * (pq[kk, 0] * xy[:, 0] + pq[kk, 1] * xy[:, 1]) / L
            u0[:, 0] += amp * np.sin(arg + phi[kk])
            u0[:, 1] += amp * np.sin(arg + chi[kk])
        d0 = g.uniform(0.0, 0.9, nn * nn)
        mat = dict(GLASS, model=AT2, split=SPECTRAL, plane=PLANE_STRAIN)
        cfg = _pack(f"cfg5_square_{nn}x{nn}_AT2_spectral_PE", xy, tri, mat, np.zeros(0, np.int32),
                    np.zeros((0, 2), np.int32), np.zeros((0, 2)), steps=100)
        cfg.update(u0=u0, d0=d0)
        return cfg
    raise ValueError(k)


def _pack(name, xy, tri, mat, notch, edges, t, steps):
    N = len(xy)
    d0 = np.zeros(N)
    d0[notch] = 1.0
    return dict(name=name, xy=xy, tri=tri, material=mat, notch=notch, edges=edges, traction=t,
                dir_dof=np.zeros(0, np.int32), d0=d0, u0=np.zeros((N, 2)), dt_factor=0.5, steps=steps)


def shear_bc(cfg, step: int, dt: float):
    """Dirichlet values (dir_u, dir_v) of config 3 at the END of step `step` (1-based): bottom fixed,
    top u_y = 0 and u_x driven by the velocity ramp of PAPER.md Eq. 20 (linear 0 -> vbar over
    ramp_steps steps, then held); the displacement is the time integral of that ramp."""
    sh = cfg["shear"]
    nf, nt, vbar, ns = sh["n_fixed"], sh["n_top"], sh["vbar"], sh["ramp_steps"]
    t, tr = step * dt, ns * dt
    vel = vbar * t / tr if t < tr else vbar
    disp = 0.5 * vbar * t * t / tr if t < tr else vbar * (t - 0.5 * tr)
    du = np.zeros(nf + 2 * nt)
    dv = np.zeros(nf + 2 * nt)
    du[nf:nf + nt] = disp
    dv[nf:nf + nt] = vel
    return du, dv


def random_mesh(n_side: int, seed: int, jitter: float = 0.3, flip_fraction: float = 0.5):
    """Small jittered grid with randomly flipped element orientation and permuted element order:
    the generic unstructured stand-in for operator tests."""
    xy, tri = grid_mesh(n_side, n_side, 1.0, 1.0)
    g = np.random.default_rng(seed)
    h = 1.0 / (n_side - 1)
    ii, jj = np.arange(n_side * n_side) % n_side, np.arange(n_side * n_side) // n_side
    interior = (ii > 0) & (ii < n_side - 1) & (jj > 0) & (jj < n_side - 1)
    xy = xy + g.uniform(-jitter * h, jitter * h, xy.shape) * interior[:, None]
    flip = g.uniform(size=len(tri)) < flip_fraction
    tri = tri.copy()
    tri[flip] = tri[flip][:, [0, 2, 1]]
    tri = np.ascontiguousarray(tri[g.permutation(len(tri))])
    return np.ascontiguousarray(xy), tri
