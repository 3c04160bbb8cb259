"""sfh_cfl_dt_noalloc against sfh_cfl_dt.

Some users of libsfh cannot let it allocate device memory: their own memory pool has already claimed the GPU, or
they sit in a loop where a cudaMalloc would stall every stream, or their host program forbids it.  For them
the library has one entry point whose intermediates (per-block maximum speeds, running maximum) live in an array
compiled into libsfh.so instead of a caller-allocated work buffer.  That array is shared by all calls and keeps the
last call's contents, so the check is made on two calls in a row whose answers differ -- the second with the
smaller maximum speed, which a stale running maximum from the first call would get wrong -- each against the
ordinary path (a bound mesh, sfh_cfl_dt) on the same data, within the 1e-14 the other CFL tests use.

This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure here should not hide the
parity tests.  It needs nothing from them and passes alone in a fresh process as well."""
import ctypes as C

import numpy as np
import pytest

import paper_2604_21438_b200 as sfh
from helpers import problem_from_tree, small_amr_tree
from sfh_inputs import make_config

pytestmark = pytest.mark.gpu

TOLDT = 1e-14   # tests/test_gpu_parity.py: CFL dt within 1e-14 relative


def existing_path(p, U, level):
    """(dt, blocks of that level as a device tensor) from a bound mesh: the path every other test exercises."""
    g = sfh.Mesh.from_problem(p)
    g.set_state(U)
    dt = g.cfl_dt(level)
    Ul = g.get_state()[np.flatnonzero(p.level == level)].contiguous()
    return dt, Ul, g.cell_width(level)


def slowed(U, factor):
    """The same gas with velocities and sound speed scaled by `factor` (momenta x factor, energy x factor^2)."""
    V = np.array(U, dtype=np.float64, copy=True)
    V[:, 1:4] *= factor
    V[:, 4] *= factor * factor
    return V


@pytest.mark.parametrize("name, level", [("C1", 0), ("amr", 0), ("amr", 2)])
def test_two_calls_in_a_row_match_the_bound_mesh_path(name, level):
    import torch
    p = make_config("C1") if name == "C1" else problem_from_tree(small_amr_tree(), mode=1)
    out = torch.empty(2, dtype=torch.float64, device="cuda:0")     # the caller's output, reused by both calls
    results = []
    for U in (p.U, slowed(p.U, 0.25)):
        dt_ref, Ul, h = existing_path(p, U, level)
        assert Ul.shape[0] == p.census()[level] > 0
        sfh.cfl_dt_noalloc(Ul, p.gamma, p.cfl, h, out=out)
        dt, smax = out.cpu().numpy()
        assert abs(dt - dt_ref) <= TOLDT * dt_ref, (name, level, dt, dt_ref)
        assert abs(smax - p.cfl * h / dt_ref) <= 4 * TOLDT * smax
        results.append(dt)
    assert results[1] > 3.9 * results[0]        # the second answer really is the one a stale maximum would spoil


def test_the_largest_size_the_built_in_scratch_takes():
    """Exactly SFH_NOALLOC_MAX_BLOCKS blocks (a uniform 512 x 256 x 256 grid), after a small call has left its
    maxima in the front of the array."""
    import torch
    from sfh_inputs import uniform_tree
    out = torch.empty(2, dtype=torch.float64, device="cuda:0")
    small = make_config("C1")
    sfh.cfl_dt_noalloc(torch.from_numpy(slowed(small.U, 50.0)).cuda(), small.gamma, small.cfl, 1.0, out=out)
    p = problem_from_tree(uniform_tree((64, 32, 32)))
    assert p.U.shape[0] == 65536
    dt_ref, Ul, h = existing_path(p, p.U, 0)
    sfh.cfl_dt_noalloc(Ul, p.gamma, p.cfl, h, out=out)
    dt = float(out[0])
    assert abs(dt - dt_ref) <= TOLDT * dt_ref, (dt, dt_ref)


def test_sizes_beyond_the_built_in_scratch_are_rejected():
    import torch
    L = sfh.load_library()
    U = torch.ones(sfh.BLK, dtype=torch.float64, device="cuda:0")
    out = torch.full((2,), -1.0, dtype=torch.float64, device="cuda:0")
    stream = C.c_void_p(torch.cuda.current_stream().cuda_stream)
    for nblocks in (65536 + 1, 0, -3):
        rc = L.sfh_cfl_dt_noalloc(U.data_ptr(), nblocks, 1.4, 0.5, 1.0, out.data_ptr(), stream)
        assert rc == -1, nblocks
        assert b"sfh_cfl_dt_noalloc" in L.sfh_last_error()
    rc = L.sfh_cfl_dt_noalloc(U.data_ptr(), 65537, 1.4, 0.5, 1.0, out.data_ptr(), stream)
    assert rc == -1 and b"SFH_NOALLOC_MAX_BLOCKS" in L.sfh_last_error()
    torch.cuda.synchronize()
    assert (out.cpu().numpy() == -1.0).all()    # a rejected call launches nothing
