"""z4c_constraints_static (include/z4c.h): the constraint monitors with their scratch in a file-scope static device
array of the library -- no allocation inside the call. Checked against the existing path (z4c_constraints, partials
in the caller's workspace) on two calls in a row, on states of different sizes so that the second call meets the
first call's rows in the shared scratch. The file name keeps it last in pytest's collection order.

Tolerance: both paths evaluate the same per-cell constraint values (same point function); the max norms must agree
exactly, the rms norms to rounding of a sum of squares grouped differently -- 1e-12 relative, the one-step tolerance
of the parity tests."""
from dataclasses import replace

import numpy as np
import pytest

from paper_2409_10383_b200 import inputs as I

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def Z():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2409_10383_b200 import build, z4c
    build.build()
    return z4c


def agree(static8: np.ndarray, ref8: np.ndarray):
    assert np.all(np.isfinite(static8)) and np.all(static8 >= 0.0)
    assert np.array_equal(static8[1::2], ref8[1::2]), (static8, ref8)                 # max norms: exact
    assert np.allclose(static8[0::2], ref8[0::2], rtol=1e-12, atol=0.0), (static8, ref8)
    assert ref8[0] > 0.0 and ref8[2] > 0.0                                             # the data violate H and M


def test_static_scratch_constraints_match_the_workspace_path_on_two_calls_in_a_row(Z):
    import torch
    # call 1: 27 blocks of 16^3 (27 rows of the scratch), strong-field noise, after two RK4 steps
    p1 = I.params_noise(16, (3, 3, 3), dx=0.1)
    big = Z.Z4c(p1)
    big.set_initial_data(I.smooth_random_data(p1, 11, 0.05))
    big.step(2)
    ref1 = big.constraints()
    out = torch.full((8,), -1.0, dtype=torch.float64, device=big.device)
    l0 = big.launch_count()
    mem0 = torch.cuda.memory_allocated(big.device)
    got = big.constraints_static(out)
    assert got.data_ptr() == out.data_ptr()
    assert big.launch_count() - l0 == 2                      # the per-block pass and the final pass, nothing else
    assert torch.cuda.memory_allocated(big.device) == mem0
    big.sync()
    agree(out.cpu().numpy(), ref1)
    # call 2, straight after: a smaller pack (8 rows) on another context and stream, outflow boundaries, 4 ghosts;
    # the scratch still holds call 1's 27 rows
    p2 = replace(I.params_noise(16, (2, 2, 2), dx=0.1), bc=1, ng=4)
    small = Z.Z4c(p2)
    small.set_initial_data(I.smooth_random_data(p2, 12, 0.05))
    ref2 = small.constraints()
    big.sync()                                               # calls that overlap on the GPU would race on the scratch
    out2 = small.constraints_static()
    small.sync()
    agree(out2.cpu().numpy(), ref2)
    # and the first context again: same bits as its first call (fixed reduction order)
    small.sync()
    again = big.constraints_static()
    big.sync()
    assert np.array_equal(again.cpu().numpy(), out.cpu().numpy())
    big.close()
    small.close()


def test_static_scratch_refuses_packs_beyond_its_rows(Z):
    p = I.params_noise(6, (17, 16, 16), dx=0.1)              # 4352 blocks > Z4C_STATIC_MAX_BLOCKS = 4096
    sim = Z.Z4c(p)
    sim.set_initial_data(I.noise_data(p, 5))
    with pytest.raises(Z.Z4cError, match="4096"):
        sim.constraints_static()
    assert np.all(np.isfinite(sim.constraints()))            # the workspace path takes it
    sim.close()
