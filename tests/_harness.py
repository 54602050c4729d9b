"""Shared helpers of the GPU parity tests: build the oracle and the CUDA mesh from the SAME seeded
input dictionary (pff_inputs.config) and compare in USER numbering.  No method arithmetic here."""
import numpy as np

from oracle import oracle_from  # noqa: F401  (oracle-side marshalling lives with the oracle)


def gpu_from(cfg, precision=0, scatter=0, chunk_elems=0, order=2):
    """CUDA mesh + state with the LIBRARY DEFAULTS unless a test asks otherwise (order 2 = PFF_ORDER_BISECTION, default
    chunk: the decomposition bench.py times)."""
    import paper_2606_23458_b200 as pff
    mesh = pff.Mesh(cfg["xy"], cfg["tri"], cfg["material"], precision=precision, scatter=scatter,
                    chunk_elems=chunk_elems, order=order)
    st = mesh.new_state(u=cfg["u0"], d=cfg["d0"])
    if len(cfg["edges"]):
        mesh.pff_set_traction(st, cfg["edges"], cfg["traction"])
    if len(cfg["notch"]):
        mesh.pff_set_damage_dirichlet(cfg["notch"])
    if len(cfg["dir_dof"]):
        mesh.pff_set_dirichlet(cfg["dir_dof"])
    return mesh, st


def relmax(a, b):
    """max-norm relative error ||a - b||_inf / ||b||_inf (north_star's measure)."""
    a, b = np.asarray(a, dtype=np.float64), np.asarray(b, dtype=np.float64)
    den = np.abs(b).max()
    return np.abs(a - b).max() / den if den > 0 else np.abs(a).max()


def gpu_fields(mesh, st):
    """(u[N,2], v, a, d, H) in user numbering as fp64 numpy."""
    nu = mesh.nodes_to_user
    return (np.stack([nu(st.ux), nu(st.uy)], 1), np.stack([nu(st.vx), nu(st.vy)], 1),
            np.stack([nu(st.ax), nu(st.ay)], 1), nu(st.d), mesh.elems_to_user(st.H))
