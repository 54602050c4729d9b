"""pff_energies_static (include/pff.h): the energy diagnostics with their block partials in a static device array, for
callers that may not allocate.  Collected last on purpose (the suite runs with pytest -x).

The entry point is checked against the existing path (pff_energies: stream-ordered allocation, host result) on two calls
in a row with a different state each time, so that a partial left over from the first call would show in the second.
Both run the same kernels in the same fixed order: the results must agree to the last bit; the assertion uses the
trajectory-energy tolerance of test_gpu_parity.py (1e-6 of the largest energy) and then the exact comparison.
"""
import numpy as np
import pytest

from pff_inputs import config
from _harness import gpu_from

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("precision", [0, 1])
def test_energies_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row(precision):
    import torch
    cfg = config(1)
    mesh, st = gpu_from(cfg, precision=precision)
    bc = mesh.bc(load_scale=8.0)
    dt = 0.5 * mesh.dt_crit
    mesh.pff_init_accel(st, bc)
    out = torch.full((4,), float("nan"), dtype=torch.float64, device=mesh.device)  # the only allocation, made by the caller
    seen = []
    for call, n_steps in enumerate((20, 15)):
        mesh.pff_run_steps(st, bc, dt, n_steps, damage_every=1, rel_tol=1e-8 if precision == 0 else 1e-5)
        ref = mesh.pff_energies(st)
        got = mesh.pff_energies_static(st, out).cpu().numpy()  # .cpu() synchronises in stream order
        assert np.isfinite(got).all() and got[3] > 0
        assert np.all(np.abs(got - ref) <= 1e-6 * np.abs(ref).max()), (call, got, ref)
        assert np.array_equal(got, ref), (call, got, ref)
        seen.append(got.copy())
    assert not np.array_equal(seen[0], seen[1])  # the two calls saw different states


def test_energies_static_rejects_bad_arguments():
    import torch
    cfg = config(1)
    mesh, st = gpu_from(cfg)
    out = torch.zeros(5, dtype=torch.float64, device=mesh.device)
    import ctypes as C
    assert mesh.L.pff_energies_static(mesh.h, C.byref(st.c), None) == 1                    # PFF_EINVAL: null output
    assert mesh.L.pff_energies_static(mesh.h, C.byref(st.c), out.data_ptr() + 4) == 1      # PFF_EINVAL: misaligned output
    assert mesh.L.pff_energies_static(None, C.byref(st.c), out.data_ptr()) == 1
    with pytest.raises(ValueError):
        mesh.pff_energies_static(st, out.float())
