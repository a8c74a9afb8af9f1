"""GPU parity at BASELINE.json's full sizes and full step counts, in the launch configuration bench.py times, plus the
cases that put the bench's own kernels on ragged grids and k_ghost on block lists.  Same tolerances as
tests/test_gpu_parity.py (<= 1e-10 relative L-inf per field after one step, <= 1e-6 after the config's step count).
The oracle runs at a few 1e6 cell-updates/s on the box's host cores; the whole file takes a few minutes."""
import numpy as np
import pytest

from paper_2504_13750_b200 import inputs as I
from tests.test_gpu_parity import B, TOL1, TOL100, check, field_errors  # noqa: F401  (B is a fixture)

pytestmark = pytest.mark.gpu


def march(B, ref, case, marks, tols, chem=True, options=None):
    """Advance the CUDA path and the oracle side by side and compare at every mark (cumulative step counts)."""
    g = B.Solver(case.grid, case.mech, case.blocks, options=options)
    g.set_state(case.U, case.T)
    r = ref.RefSolver(case.grid, case.mech, case.blocks)
    r.set_state(case.U, case.T)
    done, out = 0, []
    for mark, tol in zip(marks, tols):
        tg = g.step(mark - done, cfl=case.cfl, chem=chem)
        tr = r.step(mark - done, cfl=case.cfl, chem=chem)
        done = mark
        Ug, Tg = g.get_state(); Ur, Tr = r.get_state()
        assert g.status == 0 and r.status == 0
        assert abs(tg - tr) <= 1e-12 * tr, (mark, tg, tr)
        e = field_errors(case, Ug, Ur)
        assert e.max() <= tol, (case.name, mark, e)
        assert np.abs(Tg - Tr).max() <= max(tol, 1e-11) * np.abs(Tr).max()
        out.append(e.max())
    g.close(); r.close()
    print(case.name, "steps", marks, "worst per-field rel err", out)
    return out


# ------------------------------------------------------------------ BASELINE configs at full size, full step counts
def test_cfg1_full_size_100_steps(B, ref):
    """configs[1] exactly: 1024 x 128, 9 species / 21 reactions, 100 steps."""
    case = I.config1()
    assert case.grid.n[0] == 1024 and case.grid.n[1] == 128
    march(B, ref, case, (1, 100), (TOL1, TOL100))


def test_cfg2_full_size_100_steps(B, ref):
    """configs[2] exactly: 4096 x 512, right side outflow, 100 steps (k_flux_rk2<64,16,8> + k_ghost, as benched)."""
    case = I.config2()
    assert case.cells == 4096 * 512
    march(B, ref, case, (1, 100), (TOL1, TOL100))


def test_cfg3_full_size_50_steps(B, ref):
    """configs[3] exactly: 8192 patches of 16 x 16 on 2 levels, synchronous advance, 50 steps."""
    case = I.config3()
    assert case.grid.n_patches == 8192
    march(B, ref, case, (1, 50), (TOL1, TOL100))


def test_cfg3_full_size_crossover_advance(B, ref):
    """configs[3] at full size with the crossover (sub-cycled) advance, Fig 2a: 1 and 12 level-0 steps
    (the physical time of 24 synchronous steps)."""
    case = I.config3()
    g = B.Solver(case.grid, case.mech, case.blocks)
    g.set_state(case.U, case.T)
    r = ref.RefSolver(case.grid, case.mech, case.blocks)
    r.set_state(case.U, case.T)
    done = 0
    for mark, tol in ((1, TOL1), (12, TOL100)):
        tg = g.step(mark - done, cfl=case.cfl, crossover=True)
        tr = r.step(mark - done, cfl=case.cfl, crossover=True)
        done = mark
        Ug, Tg = g.get_state(); Ur, Tr = r.get_state()
        assert g.status == 0 and r.status == 0 and abs(tg - tr) <= 1e-12 * tr
        e = field_errors(case, Ug, Ur)
        assert e.max() <= tol, (mark, e)
    g.close(); r.close()


def test_cfg4_full_size_flux_path_element_by_element(B, ref):
    """configs[4] at 256^3, 20 species: ONE full RK3 step of the 3-D flux path (cons->prim, ghost fill, k_flux_rk
    <3,16,8,8,8>, three stages) compared with the oracle on all 16.7 M cells x 24 fields.  The oracle's point-implicit
    chemistry of 100 reactions runs at ~2e4 cells/s, so the chemistry of the same step is compared separately
    (next test) on whole planes of cells."""
    case = I.config4()
    assert case.cells == 256 ** 3
    march(B, ref, case, (1,), (TOL1,), chem=False)


def test_cfg4_full_size_chemistry_planes_and_conservation(B, ref, mech20):
    """configs[4] at 256^3 in the launch configuration bench.py times (role-warp kernel, persistent CTAs):
    (a) total mass, momentum, energy and every element conserved to round-off on the periodic box;
    (b) the step is run twice from the same state, without the chemistry (U*) and with it; the flow part is the same
        kernels on the same inputs (checked bitwise), so U1 - U* is the chemistry kernel's increment.  It is compared
        cell by cell with the oracle's update_aux + solve_implicit_rate (jref_chem_cells) on two whole z-planes
        (131 072 cells: the plane with the most hot-sphere cells and plane 0), every cell of them."""
    case = I.config4()
    s = B.Solver(case.grid, case.mech, case.blocks)
    assert s.chem_kernel() == "jit-roles"
    s.set_state(case.U, case.T)
    s.step(1, cfl=case.cfl, chem=False)
    Ustar, Tstar = s.get_state()
    assert s.status == 0
    s.set_state(case.U, case.T)
    dt = s.step(1, cfl=case.cfl)
    U1, T1 = s.get_state()
    assert s.status == 0
    s.close()
    for v in range(5):
        a, b = case.U[0, v].sum(dtype=np.float64), U1[0, v].sum(dtype=np.float64)
        scale = np.abs(case.U[0, v]).sum(dtype=np.float64) if v not in (1, 2, 3) else case.U[0, 0].sum() * 300.0
        assert abs(a - b) <= 1e-11 * scale, (v, a, b)
    el = np.asarray(mech20.elements, dtype=float)

    def moles(Us):
        ry = [Us[0, 5 + k].sum(dtype=np.float64) for k in range(19)]
        ry.append(Us[0, 0].sum(dtype=np.float64) - sum(ry))
        return (np.array(ry) / mech20.W) @ el
    m0, m1 = moles(case.U), moles(U1)
    assert np.abs(m1 - m0).max() <= 1e-11 * np.abs(m0).max()
    assert np.array_equal(U1[0, :5], Ustar[0, :5])
    hot_per_plane = (case.T[0] > 2000.0).sum(axis=(1, 2))
    planes = sorted({int(np.argmax(hot_per_plane)), 0})
    worst = worst_d = 0.0
    active = 0
    for k in planes:
        Uc = np.ascontiguousarray(Ustar[0, :, k].reshape(24, -1).T)          # [cells, nvar]
        rc, d, Tc = ref.chem_cells(mech20, 3, Uc, case.T[0, k].ravel(), dt)
        assert rc == 0
        ry = Uc[:, 5:]
        got = U1[0, 5:, k].reshape(19, -1).T - ry
        scale = np.maximum(np.abs(ry).max(axis=1), 1e-6 * Uc[:, 0])
        worst = max(worst, (np.abs(got - d).max(axis=1) / scale).max())
        act = np.abs(d).max(axis=1) > 1e-9 * np.abs(ry).max(axis=1)
        active += int(act.sum())
        if act.any():
            worst_d = max(worst_d, (np.abs(got - d)[act].max(axis=1) / np.abs(d)[act].max(axis=1)).max())
        assert np.abs(T1[0, k].ravel() - Tc).max() <= 1e-10 * Tc.max()
    assert worst <= 1e-10, worst
    assert active >= 1000 and worst_d <= 1e-6, (active, worst_d)
    print("cfg4 full-size chemistry on planes", planes, ": state rel err", worst, "increment rel err", worst_d, "active cells", active)


def test_cfg4_20_steps_on_56_cubed(B, ref):
    """The config's 20-step count on the largest cube the oracle's 100-reaction chemistry finishes in about a minute:
    56^3 (3.5 x 7 x 7 tiles of 16 x 8 x 8: ragged in x), 6 hot spheres, same recipe."""
    case = I.config4(n=56, nspheres=6, radius=6)
    march(B, ref, case, (1, 20), (TOL1, TOL100))


# ------------------------------------------------------------------ the bench's own kernels on ragged grids
def test_ragged_2d_above_600k_cells_runs_the_benched_kernels(B, ref):
    """1000 x 700 (>= 600 k cells, so k_flux_rk2<64,16,8,false> + k_ghost run, as on cfg 2): both extents ragged
    w.r.t. the 64 x 16 tile (1000 = 15 x 64 + 40, 700 = 43 x 16 + 12), outflow / reflect mix, 1 and 10 steps."""
    case = I.config2(nx=1000, ny=700, seed=77)
    g = case.grid
    case.grid = I.Grid(2, g.n, g.dx, (I.BC_REFLECT, I.BC_OUTFLOW, 0), (I.BC_OUTFLOW, I.BC_REFLECT, 0))
    march(B, ref, case, (1, 10), (TOL1, TOL100))


def test_small_ragged_grids_through_the_big_grid_path(B, ref, mech9):
    """halo = "ghost" sends small grids through k_ghost + the non-gathering flux kernels (64 x 16 tile: 100 x 40 and
    70 x 37 are ragged in both directions; a 30-column grid takes the 32 x 16 tile), periodic / reflect / outflow."""
    opt = {"halo": "ghost"}
    check(B, ref, I.config1(nx=100, ny=40), 1, TOL1, options=opt)
    check(B, ref, I.config1(nx=100, ny=40), 30, TOL100, options=opt)
    check(B, ref, I.config2(nx=70, ny=37), 5, TOL100, options=opt)
    check(B, ref, I.config2(nx=30, ny=50), 5, TOL100, options=opt)
    from tests.test_oracle_pins import _random_smooth_2d
    check(B, ref, _random_smooth_2d(mech9, 72, 40, 3, I.BC_PERIODIC), 5, TOL100, options=opt)


# ------------------------------------------------------------------ k_ghost on block lists (neighbour / coarse / physical)
def test_block_list_ghost_kernel_2d(B, ref):
    """Two-level 2-D block lists through k_ghost's FK_NEIGHBOUR / FK_COARSE / FK_PHYSICAL branches, per-level launch
    order, and k_average_down: (a) config 3 with the in-kernel gather switched off (16 x 16 patches); (b) 32 x 32
    patches on > 600 k cells, where k_ghost is the default path."""
    check(B, ref, I.config3(pcols=16, prows=8, npc=16), 1, TOL1, options={"halo": "ghost"})
    check(B, ref, I.config3(pcols=16, prows=8, npc=16), 10, TOL100, options={"halo": "ghost"})
    big = I.config3(pcols=32, prows=16, npc=32)
    assert big.cells > 600000 and (big.blocks.level == 1).sum() > 0
    march(B, ref, big, (1, 5), (TOL1, TOL100))


def test_block_list_ghost_kernel_1d_and_3d(B, ref):
    """Two-level block lists in 1-D and 3-D (inputs.refine_uniform): k_ghost, k_flux_rk with level > 0, k_average_down
    with 2 and 8 children per coarse cell; periodic wrap links, slip walls and zero-gradient sides on both levels."""
    base = I.config0(n=192)
    base.grid.bc_lo, base.grid.bc_hi = (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0)
    mask = np.zeros(12, bool); mask[4:8] = True; mask[0] = True
    c1 = I.refine_uniform(base, (16,), mask)
    check(B, ref, c1, 1, TOL1)
    check(B, ref, c1, 20, TOL100)
    b3 = I.config4(n=16, nspheres=2, radius=4)
    b3.grid.bc_lo, b3.grid.bc_hi = (I.BC_PERIODIC, I.BC_REFLECT, I.BC_OUTFLOW), (I.BC_PERIODIC, I.BC_OUTFLOW, I.BC_REFLECT)
    m3 = np.zeros((2, 2, 2), bool); m3[0, 1, 0] = m3[1, 1, 0] = m3[1, 0, 1] = True
    c3 = I.refine_uniform(b3, (8, 8, 8), m3)
    check(B, ref, c3, 1, TOL1)
    check(B, ref, c3, 3, TOL1 * 100)
