"""x-slab decomposition ("results identical"): the decomposed run, all slabs in
this process on one GPU and advanced in lockstep (slab.LocalComm; the multi-process transport is tested on CPU in
tests/test_multiprocess.py), must reproduce the single-grid run of the same library BIT FOR BIT -- same kernels, exact
max reductions, halos = the neighbour's interior values -- and hence inherit its parity with the oracle."""
import numpy as np
import pytest

from paper_2504_13750_b200 import inputs as I
from tests.test_gpu_parity import B, TOL100, field_errors  # noqa: F401

pytestmark = pytest.mark.gpu


def single(B, case, nsteps, options=None, **kw):
    s = B.Solver(case.grid, case.mech, options=options)
    s.set_state(case.U, case.T)
    t = s.step(nsteps, **kw)
    U, T = s.get_state()
    assert s.status == 0
    s.close()
    return U, T, t


def slabs(case, world, nsteps, **kw):
    from paper_2504_13750_b200 import slab
    run = slab.SlabRun(case, slab.LocalComm(world))
    run.step(nsteps, **kw)
    U, T = run.assemble()
    dt = run.last_dt()
    run.close()
    return U, T, dt


@pytest.mark.parametrize("world", [2, 3])
def test_slabs_reproduce_the_single_grid_bitwise_2d(B, ref, world):
    # walls / outflow: physical BCs on the end ranks only; the undecomposed run uses materialised ghosts too
    case = I.config2(nx=150, ny=40)
    U1, T1, _ = single(B, case, 6, options={"halo": "ghost"}, cfl=case.cfl)
    U2, T2, _ = slabs(case, world, 6, cfl=case.cfl)
    assert np.array_equal(U1, U2) and np.array_equal(T1, T2)
    # ... and therefore the oracle's answer
    r = ref.RefSolver(case.grid, case.mech); r.set_state(case.U, case.T); r.step(6, cfl=case.cfl); Ur, _ = r.get_state()
    assert field_errors(case, U2, Ur).max() <= TOL100
    # periodic in x: the end slabs are neighbours (world 2: both neighbours are the same slab)
    from tests.test_oracle_pins import _random_smooth_2d
    per = _random_smooth_2d(case.mech, 96, 24, 9, I.BC_PERIODIC)
    U1, T1, _ = single(B, per, 4, options={"halo": "ghost"}, cfl=0.0, dt=1.0e-9, chem=False)
    U2, T2, _ = slabs(per, world, 4, cfl=0.0, dt=1.0e-9, chem=False)
    assert np.array_equal(U1, U2) and np.array_equal(T1, T2)


def test_slabs_reproduce_the_single_grid_bitwise_1d_3d(B):
    c0 = I.config0(n=300)
    U1, _, t1 = single(B, c0, 20, cfl=c0.cfl)
    U2, _, dt = slabs(c0, 4, 20, cfl=c0.cfl)
    assert np.array_equal(U1, U2)
    c4 = I.config4(n=24, nspheres=3, radius=5)          # periodic box, 20 species: role-warp chemistry on every slab
    U1, _, _ = single(B, c4, 2, cfl=c4.cfl)
    U2, _, _ = slabs(c4, 3, 2, cfl=c4.cfl)
    assert np.array_equal(U1, U2)


def test_exchange_faces_are_refused_where_they_make_no_sense(B):
    case = I.config1(nx=32, ny=16)
    g = case.grid
    with pytest.raises(B.JancError):       # exchange on a y side
        B.Solver(I.Grid(2, g.n, g.dx, (g.bc_lo[0], B.BC_EXCHANGE, 0), g.bc_hi), case.mech)
    s = B.Solver(I.Grid(2, g.n, g.dx, (B.BC_EXCHANGE, g.bc_lo[1], 0), g.bc_hi), case.mech)
    s.set_state(case.U, case.T)
    with pytest.raises(B.JancError):       # unknown part
        s.step_part(9)
    s.close()
