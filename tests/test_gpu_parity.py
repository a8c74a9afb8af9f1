"""GPU parity: libjanc (through the C ABI binding) vs the CPU oracle, element by element, on the
same seeded inputs.  Tolerances are BASELINE.json's: <= 1e-10 relative L-inf per field after one
step, <= 1e-6 after 100 steps (fp64).  Run with -m gpu on a B200."""
import numpy as np
import pytest

from paper_2504_13750_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL1, TOL100 = 1e-10, 1e-6


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2504_13750_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def field_errors(case, Ug, Ur):
    """relative L-inf per conserved field; momentum components share one scale."""
    nd = case.grid.ndim
    errs = []
    mom_scale = max(np.abs(Ur[:, 1:1 + nd]).max(), 1e-300)
    rho_c = np.abs(Ur[:, 0]).max() * np.sqrt(np.abs(Ur[:, nd + 1]).max() / np.abs(Ur[:, 0]).max())
    mom_scale = max(mom_scale, 1e-3 * rho_c)
    for v in range(Ur.shape[1]):
        if 1 <= v <= nd:
            scale = mom_scale
        elif v > nd + 1:
            scale = max(np.abs(Ur[:, v]).max(), 1e-6 * np.abs(Ur[:, 0]).max())   # species vs density
        else:
            scale = np.abs(Ur[:, v]).max()
        errs.append(np.abs(Ug[:, v] - Ur[:, v]).max() / scale)
    return np.array(errs)


def both(B, ref, case, nsteps, chem=True, cfl=None, dt=0.0, options=None, crossover=False):
    cfl = case.cfl if cfl is None else cfl
    g = B.Solver(case.grid, case.mech, case.blocks, options=options)
    g.set_state(case.U, case.T)
    tg = g.step(nsteps, cfl=cfl, dt=dt, chem=chem, crossover=crossover)
    Ug, Tg = g.get_state()
    assert g.status == 0, "device flag raised"
    g.close()
    r = ref.RefSolver(case.grid, case.mech, case.blocks)
    r.set_state(case.U, case.T)
    tr = r.step(nsteps, cfl=cfl, dt=dt, chem=chem, crossover=crossover)
    Ur, Tr = r.get_state()
    assert r.status == 0
    assert abs(tg - tr) <= 1e-12 * tr, (tg, tr)
    return Ug, Tg, Ur, Tr


def check(B, ref, case, nsteps, tol, **kw):
    Ug, Tg, Ur, Tr = both(B, ref, case, nsteps, **kw)
    e = field_errors(case, Ug, Ur)
    assert e.max() <= tol, (case.name, nsteps, e)
    assert np.abs(Tg - Tr).max() <= max(tol, 1e-11) * np.abs(Tr).max()
    assert np.abs(Ug - case.U).max() > 0          # something happened
    return e


# ------------------------------------------------------------------ cons->prim kernel alone
def test_cons2prim_kernel(B, ref, mech9):
    case = I.config1(nx=70, ny=20)
    g = B.Solver(case.grid, case.mech)
    g.set_state(case.U, np.full_like(case.T, 900.0))
    T, p, c = g.debug_cons2prim()
    g.close()
    for (j, i) in [(0, 0), (3, 2), (19, 69), (7, 33), (12, 5)]:
        rc, out = ref.cons2prim(mech9, 2, case.U[0, :, 0, j, i], 900.0)
        assert rc == 0
        assert abs(T[0, 0, j, i] - out[0]) <= 1e-12 * out[0]
        assert abs(p[0, 0, j, i] - out[1]) <= 1e-12 * out[1]
        assert abs(c[0, 0, j, i] - out[3]) <= 1e-12 * out[3]
    assert np.abs(T - case.T).max() <= 1e-9 * case.T.max()


# ------------------------------------------------------------------ config 0 (1-D, 2 species)
def test_cfg0_one_step(B, ref):
    check(B, ref, I.config0(), 1, TOL1)


def test_cfg0_full_200_steps(B, ref):
    check(B, ref, I.config0(), 200, TOL100)


def test_cfg0_ragged_and_tiny(B, ref):
    check(B, ref, I.config0(n=300), 1, TOL1)      # tile of 256 + ragged tail
    check(B, ref, I.config0(n=7), 3, TOL1 * 10)   # smaller than the stencil's reach into ghosts


def test_sod_inert_single_species(B, ref):
    from tests.test_oracle_pins import _sod_case
    case, x = _sod_case(400)
    check(B, ref, case, 1, TOL1, chem=False)
    check(B, ref, case, 100, TOL100, chem=False)


# ------------------------------------------------------------------ configs 1, 2 (2-D, 9 species)
def test_cfg1_scaled_one_step_and_100(B, ref):
    case = I.config1(nx=100, ny=40)               # 4 x 3 tiles of 32x16, ragged in both directions
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 100, TOL100)


def test_cfg2_scaled_outflow(B, ref):
    case = I.config2(nx=160, ny=48)
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 30, TOL100)


def test_periodic_2d_smooth(B, ref, mech9):
    from tests.test_oracle_pins import _random_smooth_2d
    case = _random_smooth_2d(mech9, 48, 40, 3, I.BC_PERIODIC)
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 10, TOL100)
    check(B, ref, case, 2, TOL1 * 10, cfl=0.0, dt=1.5e-9)     # fixed-dt mode


def test_explicit_variant_no_chem(B, ref):
    case = I.config1(nx=64, ny=32)
    check(B, ref, case, 5, TOL100, chem=False)


# ------------------------------------------------------------------ config 3 (block list, 2 levels)
def test_cfg3_scaled_block_list(B, ref):
    case = I.config3(pcols=16, prows=8, npc=16)
    assert case.blocks.level.sum() > 0
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 10, TOL100)


def test_block_tiling_equals_uniform_on_gpu(B, ref, mech9):
    from tests.test_oracle_pins import _random_smooth_2d
    case = _random_smooth_2d(mech9, 32, 32, 8, I.BC_REFLECT)
    g = B.Solver(case.grid, case.mech); g.set_state(case.U, case.T); g.step(3, cfl=case.cfl); U1, _ = g.get_state(); g.close()
    tiled = I.tile_uniform(case, 16, 16)
    g = B.Solver(tiled.grid, tiled.mech, tiled.blocks); g.set_state(tiled.U, tiled.T); g.step(3, cfl=case.cfl)
    U2, _ = g.get_state(); g.close()
    U2 = I.untile(tiled, U2, 2, 2)
    assert np.abs(U1 - U2).max() <= 1e-12 * np.abs(U1).max()


# ------------------------------------------------------------------ config 4 (3-D, 20 species)
def test_cfg4_scaled_3d(B, ref):
    case = I.config4(n=24, nspheres=3, radius=5)
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 5, TOL100)


def test_3d_ragged_nonperiodic(B, ref):
    c1 = I.config4(n=20, nspheres=2, radius=4)
    g = c1.grid
    U = c1.U[:, :, :18, :13, :].copy(); T = c1.T[:, :18, :13, :].copy()
    g2 = I.Grid(3, (20, 13, 18), g.dx, (I.BC_REFLECT, I.BC_OUTFLOW, I.BC_PERIODIC), (I.BC_OUTFLOW, I.BC_REFLECT, I.BC_PERIODIC))
    case = I.Case("3d_ragged", g2, c1.mech, U, T, 0.2, 2)
    check(B, ref, case, 2, TOL1 * 10)                           # even padded width: the TMA flux kernel
    check(B, ref, case, 2, TOL1 * 10, options={"tma": 0})       # the staged kernel it replaces (still the odd-width path)
    odd = I.Case("3d_ragged_odd", I.Grid(3, (19, 13, 18), g.dx, g2.bc_lo, g2.bc_hi), c1.mech,
                 np.ascontiguousarray(U[..., :19]), np.ascontiguousarray(T[..., :19]), 0.2, 2)
    check(B, ref, odd, 2, TOL1 * 10)                            # odd padded width: TMA not applicable


def test_3d_tma_flux_kernel_is_bitwise_the_staged_one(B):
    """k_flux_rk3_tma does the arithmetic of k_flux_rk<3> in the same order: identical states on ragged grids (tiles that
    stick out in x, y, z; a grid smaller than one tile), with chemistry and over several steps."""
    def run(case, opts):
        s = B.Solver(case.grid, case.mech, case.blocks, options=opts)
        s.set_state(case.U, case.T)
        s.step(3, cfl=case.cfl)
        U, _ = s.get_state()
        assert s.status == 0
        s.close()
        return U
    c = I.config4(n=40, nspheres=3, radius=5)
    for n in ((40, 20, 12), (34, 10, 18), (16, 8, 8), (6, 4, 4)):
        g = I.Grid(3, n, c.grid.dx, c.grid.bc_lo, c.grid.bc_hi)
        sub = I.Case("crop", g, c.mech, np.ascontiguousarray(c.U[:, :, 8:8 + n[2], 8:8 + n[1], :n[0]]),
                     np.ascontiguousarray(c.T[:, 8:8 + n[2], 8:8 + n[1], :n[0]]), c.cfl, 3)
        assert np.array_equal(run(sub, {"tma": 1}), run(sub, {"tma": 0})), n


# ------------------------------------------------------------------ generic species count (run-time ns path)
def test_generic_ns_path(B, ref):
    m2 = I.single_step_mechanism()
    W = np.array([0.029, 0.029, 0.040]); nasa = np.zeros((3, 7)); nasa[:, 0] = [3.5, 3.5, 2.5]; nasa[0, 5] = m2.nasa[0, 5]
    m3 = I.Mechanism(3, 1, W, nasa, np.array([[1, 0, 0]], dtype=np.int32), np.array([[0, 1, 0]], dtype=np.int32),
                     m2.A, m2.b, np.array([8000.0]), np.array([1], dtype=np.int32), np.array([1], dtype=np.int32),
                     np.array([[1.0, 2.0, 0.5]]))
    n = 96
    x = np.arange(n)
    p = np.where(x < 48, 8e5, 1e5); T = np.where(x < 48, 1800.0, 400.0)
    Y = np.zeros((n, 3)); Y[:, 0] = 0.6; Y[:, 1] = 0.1; Y[:, 2] = 0.3
    U = I.prim_to_cons(m3, 1, p, T, Y, [np.zeros(n)])
    g = I.Grid(1, (n, 1, 1), (1e-4, 1, 1), (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0))
    case = I.Case("ns3", g, m3, U.reshape(1, 5, 1, 1, n), T.reshape(1, 1, 1, n).astype(float), 0.3, 10)
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 10, TOL100)


# ------------------------------------------------------------------ invariants on the GPU path itself
def test_uniform_state_bitwise_on_gpu(B, mech9):
    nx, ny = 70, 37
    Y = I.hot_Y(9); z = np.zeros((ny, nx))
    U = I.prim_to_cons(mech9, 2, z + 2.5e5, z + 1234.5, np.broadcast_to(Y, (ny, nx, 9)), [z + 310.0, z - 95.0])
    U = np.broadcast_to(U[:, :1, :1], U.shape).copy()
    g = I.Grid(2, (nx, ny, 1), (1e-4, 2e-4, 1), (0, 0, 0), (0, 0, 0))
    s = B.Solver(g, mech9); s.set_state(U.reshape(1, -1, 1, ny, nx), np.full((1, 1, ny, nx), 1234.5))
    s.step(5, cfl=0.4, chem=False)
    U1, _ = s.get_state(); s.close()
    assert np.array_equal(U1.reshape(U.shape), U)


def test_device_resident_state_and_async(B, ref):
    import torch
    case = I.config1(nx=64, ny=32)
    s = B.Solver(case.grid, case.mech)
    Ud = torch.from_numpy(case.U).cuda(); Td = torch.from_numpy(case.T).cuda()
    s.set_state(Ud, Td)
    s.step(2, cfl=case.cfl, sync=False)
    U1, T1 = s.get_state(device=True)
    s2 = B.Solver(case.grid, case.mech); s2.set_state(case.U, case.T); s2.step(2, cfl=case.cfl); U2, _ = s2.get_state()
    assert np.array_equal(U1.cpu().numpy(), U2)
    assert s.launch_count() >= 16            # 2 steps x (3 prim + dt + 3 flux + chem); small 2-D grids gather their halo in the flux kernel
    s.close(); s2.close()


def test_error_flag_and_arguments(B):
    case = I.config0(n=64)
    s = B.Solver(case.grid, case.mech)
    with pytest.raises(B.JancError):
        s.step(1, cfl=0.0, dt=0.0)                 # neither cfl nor dt
    U = case.U.copy(); U[0, 2, 0, 0, 10] = -1e9    # negative energy => T <= 0 => device flag
    s.set_state(U, case.T)
    s.step(1, cfl=0.4)
    assert s.status == B.JANC_ENONFINITE
    s.set_state(case.U, case.T)                    # flag is cleared by set_state
    s.step(1, cfl=0.4)
    assert s.status == 0
    s.close()
    # fewer cells than ghost layers along a mirrored / periodic direction: refused at creation (janc.h)
    m = I.config1(nx=32, ny=16).mech
    for bc in (I.BC_REFLECT, I.BC_PERIODIC):
        with pytest.raises(B.JancError):
            B.Solver(I.Grid(2, (40, 2, 1), (1e-4, 1e-4, 1), (I.BC_OUTFLOW, bc, 0), (I.BC_OUTFLOW, bc, 0)), m)
    B.Solver(I.Grid(2, (40, 2, 1), (1e-4, 1e-4, 1), (I.BC_OUTFLOW, I.BC_OUTFLOW, 0), (I.BC_OUTFLOW, I.BC_OUTFLOW, 0)), m).close()
    # options: unknown key / value refused; kernel-selection keys refused once the mechanism is set
    with pytest.raises(B.JancError):
        B.Solver(case.grid, case.mech, options={"no_such_key": 1})
    with pytest.raises(B.JancError):
        B.Solver(case.grid, case.mech, options={"halo": "sometimes"})
    s = B.Solver(case.grid, case.mech)
    with pytest.raises(B.JancError) as e:
        s.set_option("jit", 0)
    assert e.value.code == B.JANC_ESTATE
    s.set_option("graph", 0)
    # a rejected mechanism (A <= 0) leaves the context as it was: the old mechanism keeps running
    s.set_state(case.U, case.T); s.step(1, cfl=0.4); U1, _ = s.get_state()
    bad = I.single_step_mechanism(); bad.A = np.array([-1.0])
    m_, keep = B._mech_struct(bad)
    import ctypes
    assert B.lib().janc_set_mechanism(s._h, ctypes.byref(m_)) == B.JANC_EINVAL
    s.set_state(case.U, case.T); s.step(1, cfl=0.4); U2, _ = s.get_state()
    assert s.status == 0 and np.array_equal(U1, U2)
    s.close()


# ------------------------------------------------------------------ chemistry kernel selection
def test_specialised_chemistry_kernel_is_the_one_running(B, mech9, mech20):
    """janc_set_mechanism compiles the mechanism-specialised kernel (chemgen.h) for <= 12 unknowns;
    larger mechanisms (up to 24 species) run the role-warp kernel of chemgen_roles.h."""
    c = I.config1(nx=32, ny=16)
    s = B.Solver(c.grid, mech9)
    assert s.chem_kernel() == "jit", s.jit_log()
    s.close()
    c0 = I.config0(n=64)
    s = B.Solver(c0.grid, c0.mech)
    assert s.chem_kernel() == "jit", s.jit_log()
    s.close()
    c4 = I.config4(n=16, nspheres=2, radius=3)
    s = B.Solver(c4.grid, mech20)
    assert s.chem_kernel() == "jit-roles", s.jit_log()
    s.close()


def big_dt_case(mech, nx, ny, seed):
    """hot gas, random composition, one fixed-dt step of pure chemistry with a dt large enough for real row swaps"""
    ns = mech.ns
    rng = np.random.default_rng(seed)
    z = np.zeros((ny, nx))
    Y = np.broadcast_to(I.hot_Y(ns), (ny, nx, ns)).copy()
    Y[..., :ns - 1] *= rng.uniform(0.2, 1.8, size=(ny, nx, ns - 1)); Y[..., ns - 1] = 1.0 - Y[..., :ns - 1].sum(-1)
    T = 1500.0 + 1500.0 * rng.random((ny, nx))
    U = I.prim_to_cons(mech, 2, z + 2.0e6, T, Y, [z, z])
    g = I.Grid(2, (nx, ny, 1), (1e-3, 1e-3, 1), (0, 0, 0), (0, 0, 0))
    return I.Case("chem_big_dt", g, mech, U.reshape(1, -1, 1, ny, nx), T.reshape(1, 1, ny, nx), 0.2, 1)


def test_role_warp_chemistry_kernel(B, ref, mech9, mech20):
    """chemgen_roles.h: (a) the 20-species mechanism with a large dt (pivoting swaps rows across the roles'
    register columns), ragged cell count; (b) the 9-species mechanism pushed through the same generator
    (2 column slots, a role with no column in slot 1) on configs 1 and 3; (c) the one-thread-per-cell
    shared-memory variant it replaces still agrees."""
    case = big_dt_case(mech20, 37, 11, 11)
    Ug, Tg, Ur, Tr = both(B, ref, case, 1, cfl=0.0, dt=1e-7)
    assert field_errors(case, Ug, Ur).max() <= 1e-8
    small = {"jit_max_unknowns": 4}
    c1 = I.config1(nx=96, ny=40)
    s = B.Solver(c1.grid, c1.mech, options=small)
    assert s.chem_kernel() == "jit-roles", s.jit_log()
    s.close()
    check(B, ref, c1, 1, TOL1, options=small)
    check(B, ref, c1, 20, TOL100, options=small)
    check(B, ref, I.config3(pcols=8, prows=4, npc=16), 2, TOL1 * 10, options=small)
    check(B, ref, I.config3(pcols=8, prows=4, npc=16), 3, TOL100, options=small, crossover=True)   # per-level launches (patch0 / dt scale)
    case9 = big_dt_case(mech9, 40, 24, 7)
    Ug, Tg, Ur, Tr = both(B, ref, case9, 1, cfl=0.0, dt=2e-7, options=small)
    assert field_errors(case9, Ug, Ur).max() <= 1e-8
    r16 = {"roles": 16}                                       # 16 roles x 2 column slots: same generator, other split
    Ug, Tg, Ur, Tr = both(B, ref, case, 1, cfl=0.0, dt=1e-7, options=r16)
    assert field_errors(case, Ug, Ur).max() <= 1e-8
    check(B, ref, I.config4(n=16, nspheres=2, radius=3), 1, TOL1, options=r16)
    c4 = I.config4(n=16, nspheres=2, radius=3)
    s = B.Solver(c4.grid, c4.mech, options={"jit_big": "smem"})
    assert s.chem_kernel() == "jit-smem", s.jit_log()
    s.close()
    check(B, ref, c4, 1, TOL1, options={"jit_big": "smem"})
    # the variants behind the options: Newton iteration inside the kernel, column-distributed Gauss-Jordan
    for opt in ({"roles_newton": "kernel"}, {"roles_lu": "columns"}, {"roles_lu": "columns", "roles_newton": "kernel", "roles": 16}):
        check(B, ref, c4, 2, TOL1 * 10, options=opt)
        Ug, Tg, Ur, Tr = both(B, ref, case, 1, cfl=0.0, dt=1e-7, options=opt)
        assert field_errors(case, Ug, Ur).max() <= 1e-8, opt
    # run-to-run determinism with other kernels in between (a missing barrier between the roles once showed up only as
    # results that changed with what had run before on the SMs)
    def once(case_, opts):
        s_ = B.Solver(case_.grid, case_.mech, case_.blocks, options=opts)
        s_.set_state(case_.U, case_.T); s_.step(1, cfl=case_.cfl)
        U_, _ = s_.get_state(); s_.close()
        return U_
    for opt in ({}, r16):
        first = once(c4, opt)
        for _ in range(3):
            once(c1, small); once(case9, small)
            assert np.array_equal(once(c4, opt), first), opt
    # the default takes T* from a cons->prim launch in front of the kernel: one launch more per step
    a, b = (B.Solver(c4.grid, c4.mech, options={"graph": 0, **o}) for o in ({}, {"roles_newton": "kernel"}))
    for s_ in (a, b):
        s_.set_state(c4.U, c4.T)
    n0 = (a.launch_count(), b.launch_count())
    a.step(1, cfl=c4.cfl); b.step(1, cfl=c4.cfl)
    assert (a.launch_count() - n0[0]) - (b.launch_count() - n0[1]) == 1
    a.close(); b.close()


def test_table_driven_chemistry_fallback_parity(B, ref):
    """Same parity bar with the specialised kernels switched off (janc_set_option "jit" = 0): the table-driven
    kernels of chem.cuh / prim.cuh remain correct; a context on that path and a specialised one may alternate
    (the constant-memory mechanism table is re-uploaded under the library's lock)."""
    nojit = {"jit": 0}
    case = I.config1(nx=96, ny=40)
    s = B.Solver(case.grid, case.mech, options=nojit)
    assert s.chem_kernel() == "reg"
    s.close()
    check(B, ref, case, 1, TOL1, options=nojit)
    check(B, ref, case, 20, TOL100, options=nojit)
    case0 = I.config0(n=130)
    check(B, ref, case0, 5, TOL100, options=nojit)
    # two table-driven contexts with different mechanisms, stepped alternately: each must see its own table
    a = B.Solver(case.grid, case.mech, options=nojit); b = B.Solver(case0.grid, case0.mech, options=nojit)
    a.set_state(case.U, case.T); b.set_state(case0.U, case0.T)
    for _ in range(3):
        a.step(1, cfl=case.cfl); b.step(1, cfl=case0.cfl)
    Ua, _ = a.get_state(); Ub, _ = b.get_state(); a.close(); b.close()
    a = B.Solver(case.grid, case.mech, options=nojit); a.set_state(case.U, case.T); a.step(3, cfl=case.cfl); Ua2, _ = a.get_state(); a.close()
    b = B.Solver(case0.grid, case0.mech, options=nojit); b.set_state(case0.U, case0.T); b.step(3, cfl=case0.cfl); Ub2, _ = b.get_state(); b.close()
    assert np.array_equal(Ua, Ua2) and np.array_equal(Ub, Ub2)


def test_chemistry_pivoting_path(B, ref, mech9):
    """Large dt makes off-diagonal entries of I - dt J dominate, so partial pivoting actually swaps rows
    (the warp-wide skip must not change the answer): one fixed-dt step of pure chemistry on hot gas."""
    nx, ny = 40, 24
    rng = np.random.default_rng(7)
    z = np.zeros((ny, nx))
    Y = np.broadcast_to(I.hot_Y(9), (ny, nx, 9)).copy()
    Y[..., :8] *= rng.uniform(0.2, 1.8, size=(ny, nx, 8)); Y[..., 8] = 1.0 - Y[..., :8].sum(-1)
    T = 1500.0 + 1500.0 * rng.random((ny, nx))
    U = I.prim_to_cons(mech9, 2, z + 2.0e6, T, Y, [z, z])
    g = I.Grid(2, (nx, ny, 1), (1e-3, 1e-3, 1), (0, 0, 0), (0, 0, 0))
    case = I.Case("chem_big_dt", g, mech9, U.reshape(1, -1, 1, ny, nx), T.reshape(1, 1, ny, nx), 0.2, 1)
    Ug, Tg, Ur, Tr = both(B, ref, case, 1, cfl=0.0, dt=2e-7)
    e = field_errors(case, Ug, Ur)
    assert e.max() <= 1e-8, e


def test_gpu_detonation_speed_is_cj(B):
    """Property check of the CUDA path on its own (no oracle): the same 1-D single-step detonation as
    tests/test_oracle_cj.py reaches the closed-form Chapman-Jouguet speed."""
    from tests.test_oracle_cj import d_cj, front_position
    n, dx, ndrv = 1800, 1.0e-4, 10
    mech = I.single_step_mechanism()
    x = np.arange(n); drv = x < ndrv
    p = np.where(drv, 4.0e6, 1.0e5); T = np.where(drv, 2500.0, 300.0)
    Y = np.zeros((n, 2)); Y[:, 0] = 1.0
    U = I.prim_to_cons(mech, 1, p, T, Y, [np.zeros(n)])
    g = I.Grid(1, (n, 1, 1), (dx, 1.0, 1.0), (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0))
    s = B.Solver(g, mech)
    s.set_state(U.reshape(1, 4, 1, 1, n), T.reshape(1, 1, 1, n).astype(float))
    t, marks = 0.0, []
    for target in (4.0e-5, 8.0e-5):
        while t < target:
            t += s.step(50, cfl=0.4)
        Uc, _ = s.get_state()
        marks.append((t, front_position(Uc, dx)))
    assert s.status == 0
    s.close()
    D = (marks[1][1] - marks[0][1]) / (marks[1][0] - marks[0][0])
    assert abs(D - d_cj()) <= 0.004 * d_cj(), (D, d_cj())


def test_graph_replay_is_bitwise_the_eager_path(B):
    """janc_step replays a captured CUDA graph per slot parity (first step eager).  Same kernels, same order:
    the state must be bit-identical to eager launches, across several calls, a cfl change (re-capture) and the
    explicit variant (other flags), in uniform and block-list mode; the launch counter counts graph nodes too."""
    for case in (I.config1(nx=96, ny=40), I.config3(pcols=8, prows=4, npc=16), I.config0(n=130)):
        out = []
        for graph in ("1", "0"):
            s = B.Solver(case.grid, case.mech, case.blocks, options={"graph": graph})
            s.set_state(case.U, case.T)
            t = s.step(3, cfl=case.cfl) + s.step(1, cfl=case.cfl) + s.step(4, cfl=0.5 * case.cfl)
            t += s.step(2, cfl=case.cfl, chem=False) + s.step(3, cfl=case.cfl) + s.step(2, cfl=case.cfl, chem="explicit")
            U, T = s.get_state()
            assert s.status == 0
            out.append((t, U, T, s.launch_count()))
            s.close()
        assert out[0][0] == out[1][0]
        assert np.array_equal(out[0][1], out[1][1]) and np.array_equal(out[0][2], out[1][2])
        assert out[0][3] == out[1][3] > 0


# ------------------------------------------------------------------ explicit source variant
def test_explicit_source_variant_parity(B, ref):
    """the mechanism's source W_k omega_k inside every RK stage, no point-implicit
    step.  Same parity bar against the oracle's explicit variant in 1-D, 2-D, block-list and 3-D / 20-species form."""
    check(B, ref, I.config0(n=130), 5, TOL100, chem="explicit")
    c1 = I.config1(nx=96, ny=40)
    check(B, ref, c1, 1, TOL1, chem="explicit")
    check(B, ref, c1, 20, TOL100, chem="explicit")
    check(B, ref, I.config3(pcols=8, prows=4, npc=16), 2, TOL1 * 10, chem="explicit")
    check(B, ref, I.config4(n=16, nspheres=2, radius=3), 1, TOL1, chem="explicit")


def test_explicit_source_is_the_rk3_polynomial_on_gpu(B):
    """Property of the CUDA path on its own: first-order reaction at constant k in a uniform gas at rest ->
    y (1 - z + z^2/2 - z^3/6)^n, z = k dt (the SSP-RK3 stage recursion on y' = -k y)."""
    W = np.array([0.029, 0.029]); nasa = np.zeros((2, 7)); nasa[:, 0] = 3.5
    k = 4.0e6
    m = I.Mechanism(2, 1, W, nasa, np.array([[1, 0]], dtype=np.int32), np.array([[0, 1]], dtype=np.int32),
                    np.array([k]), np.array([0.0]), np.array([0.0]), np.array([0], dtype=np.int32),
                    np.array([0], dtype=np.int32), np.ones((1, 2)))
    n, dt, nsteps = 37, 1.0e-7, 3
    z = np.zeros(n)
    U = I.prim_to_cons(m, 1, z + 2.0e5, z + 900.0, np.tile([0.7, 0.3], (n, 1)), [z])
    g = I.Grid(1, (n, 1, 1), (1e-3, 1, 1), (I.BC_PERIODIC, 0, 0), (I.BC_PERIODIC, 0, 0))
    s = B.Solver(g, m)
    s.set_state(U.reshape(1, -1, 1, 1, n), (z + 900.0).reshape(1, 1, 1, n))
    s.step(nsteps, dt=dt, chem="explicit")
    Ug, Tg = s.get_state()
    assert s.status == 0
    s.close()
    zz = k * dt
    amp = (1.0 - zz + zz * zz / 2.0 - zz ** 3 / 6.0) ** nsteps
    assert np.abs(Ug[0, 3, 0, 0] - U[3] * amp).max() <= 4e-15 * U[3].max()
    assert np.array_equal(Ug[0, 0, 0, 0], U[0]) and np.abs(Tg - 900.0).max() <= 1e-9


def test_explicit_source_without_nvrtc_fails_loudly(B):
    """No silent fallback: with the run-time specialised kernels switched off the explicit-source variant is
    refused (JANC_ESTATE with a message), while the point-implicit and no-chemistry variants still run."""
    case = I.config1(nx=32, ny=16)
    s = B.Solver(case.grid, case.mech, options={"jit": 0})
    s.set_state(case.U, case.T)
    with pytest.raises(B.JancError) as e:
        s.step(1, cfl=case.cfl, chem="explicit")
    assert "explicit source variant" in str(e.value)
    s.step(1, cfl=case.cfl)
    s.step(1, cfl=case.cfl, chem=False)
    assert s.status == 0
    s.close()


def test_degenerate_mechanisms(B, ref, mech9):
    """Degenerate cases of the method: a mixture with NO reactions (nr = 0: the chemistry step is the identity, the
    specialised cons->prim kernel still runs), explicit-source mode on it (nothing to add), and the thinnest grid the 3-layer mirror admits (3 rows)."""
    m0 = I.Mechanism(9, 0, mech9.W, mech9.nasa, np.zeros((0, 9), dtype=np.int32), np.zeros((0, 9), dtype=np.int32),
                     np.zeros(0), np.zeros(0), np.zeros(0), np.zeros(0, dtype=np.int32), np.zeros(0, dtype=np.int32),
                     np.zeros((0, 9)))
    base = I.config1(nx=48, ny=24)
    case = I.Case("inert9", base.grid, m0, base.U, base.T, base.cfl, 2)
    check(B, ref, case, 2, TOL1 * 10)
    check(B, ref, case, 2, TOL1 * 10, chem="explicit")
    g3 = I.Grid(2, (40, 3, 1), base.grid.dx, base.grid.bc_lo, base.grid.bc_hi)     # three rows of cells in y
    thin = I.Case("three_rows", g3, mech9, base.U[:, :, :, :3, :40].copy(), base.T[:, :, :3, :40].copy(), base.cfl, 2)
    check(B, ref, thin, 2, TOL1 * 10)


# ------------------------------------------------------------------ crossover (sub-cycled) level advance
def test_crossover_advance_parity(B, ref):
    """PAPER.md:186 Fig 2a: two half steps of level 1, then one step of level 0, per janc_step iteration.  Same parity
    bar against the oracle's crossover mode: 2-D block list with the halo gathered in the flux kernel and with k_ghost,
    32 x 32 patches (TMA tiles), 1-D and 3-D two-level lists, the explicit-source variant, fixed dt; a single level
    ignores the flag; patches not ordered by level are refused."""
    c3 = I.config3(pcols=16, prows=8, npc=16)
    check(B, ref, c3, 1, TOL1, crossover=True)
    check(B, ref, c3, 10, TOL100, crossover=True)
    check(B, ref, c3, 4, TOL100, crossover=True, options={"halo": "ghost"})
    check(B, ref, c3, 3, TOL100, crossover=True, cfl=0.0, dt=4.0e-9, chem="explicit")
    check(B, ref, I.config3(pcols=8, prows=4, npc=32), 3, TOL100, crossover=True)
    base = I.config0(n=192)
    base.grid.bc_lo, base.grid.bc_hi = (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0)
    mask = np.zeros(12, bool); mask[4:8] = True; mask[0] = True
    check(B, ref, I.refine_uniform(base, (16,), mask), 10, TOL100, crossover=True)
    b3 = I.config4(n=16, nspheres=2, radius=4)
    m3 = np.zeros((2, 2, 2), bool); m3[0, 1, 0] = m3[1, 1, 0] = m3[1, 0, 1] = True
    check(B, ref, I.refine_uniform(b3, (8, 8, 8), m3), 2, TOL1 * 100, crossover=True)
    # one level: the flag changes nothing
    c1 = I.config1(nx=64, ny=32)
    g = B.Solver(c1.grid, c1.mech); g.set_state(c1.U, c1.T); ta = g.step(3, cfl=c1.cfl); Ua, _ = g.get_state()
    g.set_state(c1.U, c1.T); tb = g.step(3, cfl=c1.cfl, crossover=True); Ub, _ = g.get_state(); g.close()
    assert ta == tb and np.array_equal(Ua, Ub)
    # level order
    perm = np.arange(c3.grid.n_patches)[::-1].copy()
    inv = np.empty_like(perm); inv[perm] = np.arange(len(perm))
    blk = c3.blocks
    nbr = np.where(blk.nbr[perm] >= 0, inv[np.maximum(blk.nbr[perm], 0)], -1)
    par = blk.parent[perm].copy(); par[:, 0] = np.where(par[:, 0] >= 0, inv[np.maximum(par[:, 0], 0)], -1)
    rev = I.Case("rev", c3.grid, c3.mech, c3.U[perm], c3.T[perm], c3.cfl, 1, blocks=I.Blocks(blk.level[perm], nbr.astype(np.int32), par.astype(np.int32)))
    check(B, ref, rev, 2, TOL1 * 10)                                    # the synchronous advance takes any order
    g = B.Solver(rev.grid, rev.mech, rev.blocks); g.set_state(rev.U, rev.T)
    with pytest.raises(B.JancError) as e:
        g.step(1, cfl=rev.cfl, crossover=True)
    assert e.value.code == B.JANC_EINVAL
    g.close()


# ------------------------------------------------------------------ two-range NASA-7 data
def test_two_range_thermo_parity(B, ref, mech9, mech20):
    """Cantera / Chemkin style thermo data: two NASA-7 coefficient sets per species switched at T_mid[k].
    Config-1 flow (300 K ambient next to 3000 K driver gas: cells on both sides of every switch temperature) through
    the specialised kernels, the table-driven ones, the explicit-source variant and a block list; a 20-species
    two-range mechanism runs the shared-memory kernel (the role-warp kernel is single-range only)."""
    m2 = I.two_range(mech9, np.linspace(700.0, 2300.0, 9), 0.5, seed=6)
    c1 = I.config1(nx=96, ny=40, mech=m2)
    s = B.Solver(c1.grid, m2); assert s.chem_kernel() == "jit", s.jit_log(); s.close()
    check(B, ref, c1, 1, TOL1)
    check(B, ref, c1, 30, TOL100)
    check(B, ref, c1, 5, TOL100, options={"jit": 0})
    check(B, ref, c1, 5, TOL100, chem="explicit")
    check(B, ref, I.config3(pcols=8, prows=4, npc=16, mech=m2), 3, TOL100, crossover=True)
    m20 = I.two_range(mech20, 1000.0, 0.5, seed=7)
    c4 = I.config4(n=16, nspheres=2, radius=3, mech=m20)
    s = B.Solver(c4.grid, m20); assert s.chem_kernel() == "jit-smem", s.jit_log(); s.close()
    check(B, ref, c4, 2, TOL1 * 10)
    # identical sets: bitwise the single-range kernels' answer
    same = I.Mechanism(**{**mech9.__dict__}); same.nasa_hi = mech9.nasa.copy(); same.T_mid = np.full(9, 1000.0)
    ca, cb = I.config1(nx=64, ny=32, mech=mech9), I.config1(nx=64, ny=32, mech=same)
    out = []
    for c in (ca, cb):
        g = B.Solver(c.grid, c.mech); g.set_state(c.U, c.T); g.step(3, cfl=c.cfl); out.append(g.get_state()[0]); g.close()
    assert np.array_equal(out[0], out[1])


def test_mechanism_read_from_chemkin_text_runs_on_the_gpu(B, ref, mech9):
    """janc_mech_parse -> janc_set_mechanism: a mechanism that came in as Chemkin-format text (written here from the
    seeded synthetic one, two-range thermo) drives the specialised kernels; parity with the oracle on the same arrays."""
    from tests import chemkin_writer as CW
    m = B.load_chemkin(CW.write(I.two_range(mech9, 1000.0, 0.5, seed=2))[0])
    case = I.config1(nx=96, ny=40, mech=m)
    check(B, ref, case, 1, TOL1)
    check(B, ref, case, 20, TOL100)


# ------------------------------------------------------------------ regridding (rest of SURVEY NEXT-1)
def test_regrid_matches_the_oracle(B, ref, mech9):
    """janc_regrid_plan / janc_regrid_fill (reading B12) against jref_regrid: identical
    block lists (integer work: exact), identical data (copies and injections: bitwise) -- after both sides advanced the
    same list; 2-D with walls (carried / new / dropped blocks), periodic 2-D, 1-D and 3-D; then the regridded list runs
    on the GPU and stays in parity."""
    base = I.config2(nx=128, ny=64)
    base.grid.bc_hi = (I.BC_REFLECT, I.BC_REFLECT, 0)
    m0 = np.zeros((8, 16), bool); m0[:, 0] = True; m0[:, 5] = True
    c2 = I.refine_uniform(base, (8, 8), m0)
    from tests.test_oracle_pins import _random_smooth_2d
    per = _random_smooth_2d(mech9, 64, 32, 17, I.BC_PERIODIC)
    per.U[0, :, 0, :, 60:64] *= 1.6
    cp = I.refine_uniform(per, (8, 8), np.zeros((4, 8), bool)); cp.grid.n_levels = 2
    b1 = I.config0(n=192)
    b1.grid.bc_lo, b1.grid.bc_hi = (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0)
    m1 = np.zeros(12, bool); m1[2] = True
    c1 = I.refine_uniform(b1, (16,), m1)
    b3 = I.config4(n=16, nspheres=2, radius=4)
    m3 = np.zeros((2, 2, 2), bool); m3[0, 1, 0] = True
    c3 = I.refine_uniform(b3, (8, 8, 8), m3)
    for case, nsteps, thr, nbuf in ((c2, 3, 0.05, 2), (c2, 0, 0.2, 0), (cp, 0, 0.1, 3), (c1, 4, 0.02, 2), (c3, 1, 0.05, 1)):
        g = B.Solver(case.grid, case.mech, case.blocks); g.set_state(case.U, case.T)
        r = ref.RefSolver(case.grid, case.mech, case.blocks); r.set_state(case.U, case.T)
        if nsteps:
            g.step(nsteps, cfl=case.cfl); r.step(nsteps, cfl=case.cfl)
            # the criterion is a threshold on data that agree to round-off only: give both sides the same state
            Ur, Tr = r.get_state(); g.set_state(Ur, Tr)
        lg, ng, pg, Ug, Tg = g.regrid(thr, nbuf)
        lr, nr_, pr, Ur2, Tr2 = r.regrid(thr, nbuf)
        assert np.array_equal(lg, lr) and np.array_equal(ng, nr_) and np.array_equal(pg, pr), case.name
        assert np.array_equal(Ug, Ur2) and np.array_equal(Tg, Tr2), case.name
        assert (lg == 1).sum() > 0
        g.close(); r.close()
        new = I.Case(case.name + "_regridded", I.Grid(case.grid.ndim, case.grid.n, case.grid.dx, case.grid.bc_lo, case.grid.bc_hi,
                                                       n_patches=len(lg), n_levels=2, ratio=2),
                     case.mech, Ug, Tg, case.cfl, 2, blocks=I.Blocks(lg, ng, pg))
        check(B, ref, new, 2, TOL1 * 100)


def test_amr_run_cycles_against_the_oracle(B, ref, mech9):
    """amr.AmrRun (advance / regrid cycles, workspace capacity by Algorithm 1 of the paper): four cycles of a driver
    front sweeping over a two-level list.  Per cycle the oracle advances the same list from the same state (parity within
    tolerance), then both regrid the GPU's state: identical lists, bitwise identical data.  The workspace is re-allocated
    only when N_max changes."""
    from paper_2504_13750_b200 import amr
    base = I.config2(nx=128, ny=64, mech=mech9)
    base.grid.bc_hi = (I.BC_REFLECT, I.BC_REFLECT, 0)
    m0 = np.zeros((8, 16), bool); m0[:, 0] = True
    case = I.refine_uniform(base, (8, 8), m0)
    run = amr.AmrRun(case, thr=0.05, nbuf=2, every=10 ** 9, n_max=1)
    assert run.n_max >= run.n_valid + 1 and run.allocations == 1
    seen = set()
    for cycle in range(4):
        U0, T0 = run.state()
        grid = I.Grid(2, case.grid.n, case.grid.dx, case.grid.bc_lo, case.grid.bc_hi, n_patches=len(run.blocks.level), n_levels=2, ratio=2)
        r = ref.RefSolver(grid, case.mech, run.blocks); r.set_state(U0, T0)
        run.step(3, cfl=case.cfl); r.step(3, cfl=case.cfl)
        Ug, Tg = run.state(); Ur, _ = r.get_state()
        assert r.status == 0
        assert field_errors(case, Ug, Ur).max() <= TOL1 * 100, cycle
        r.set_state(Ug, Tg)                                   # the criterion is a threshold: decide on the same data
        lr, nr_, pr, Ur2, Tr2 = r.regrid(0.05, 2)
        n_max_before, alloc_before = run.n_max, run.allocations
        run.regrid()
        assert np.array_equal(run.blocks.level, lr) and np.array_equal(run.blocks.nbr, nr_) and np.array_equal(run.blocks.parent, pr)
        Ug2, Tg2 = run.state()
        assert np.array_equal(Ug2, Ur2) and np.array_equal(Tg2, Tr2)
        assert run.n_max == amr.update_n_max(run.n_valid, n_max_before)
        assert run.allocations == alloc_before + (run.n_max != n_max_before)
        seen.add(run.n_valid)
        r.close()
    assert len(seen) > 1, "the refined region never changed"
    # the loop that regrids by itself: same lists as stepping and regridding by hand (deterministic kernels)
    a = amr.AmrRun(case, thr=0.05, nbuf=2, every=3, n_max=64)
    a.step(12, cfl=case.cfl)
    assert a.regrids == 4 and np.array_equal(a.blocks.level, run.blocks.level) and np.array_equal(a.blocks.parent, run.blocks.parent)
    Ua, _ = a.state(); Ub, _ = run.state()
    assert np.array_equal(Ua, Ub)
    assert a.n_max <= 64 and a.n_max >= a.n_valid + 1
    a.close(); run.close()


def test_amr_run_in_3d_and_1d(B, ref):
    """The same cycle check on a 3-D two-level list (8^3 patches: TMA flux boxes that stick out of the patch, k_ghost with
    coarse parents, 3-D regridding) and on a 1-D one."""
    from paper_2504_13750_b200 import amr
    b3 = I.config4(n=16, nspheres=2, radius=4)
    m3 = np.zeros((2, 2, 2), bool); m3[0, 1, 0] = True
    c3 = I.refine_uniform(b3, (8, 8, 8), m3)
    b1 = I.config0(n=192)
    b1.grid.bc_lo, b1.grid.bc_hi = (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0)
    m1 = np.zeros(12, bool); m1[2] = True
    c1 = I.refine_uniform(b1, (16,), m1)
    for case, thr, nbuf in ((c3, 0.05, 1), (c1, 0.02, 2)):
        run = amr.AmrRun(case, thr=thr, nbuf=nbuf, every=10 ** 9)
        for cycle in range(2):
            U0, T0 = run.state()
            g = case.grid
            grid = I.Grid(g.ndim, g.n, g.dx, g.bc_lo, g.bc_hi, n_patches=len(run.blocks.level), n_levels=2, ratio=2)
            r = ref.RefSolver(grid, case.mech, run.blocks); r.set_state(U0, T0)
            run.step(2, cfl=case.cfl); r.step(2, cfl=case.cfl)
            Ug, Tg = run.state(); Ur, _ = r.get_state()
            assert field_errors(case, Ug, Ur).max() <= TOL1 * 100, (case.name, cycle)
            r.set_state(Ug, Tg)
            lr, nr_, pr, Ur2, Tr2 = r.regrid(thr, nbuf)
            run.regrid()
            assert np.array_equal(run.blocks.level, lr) and np.array_equal(run.blocks.nbr, nr_) and np.array_equal(run.blocks.parent, pr), case.name
            Ug2, Tg2 = run.state()
            assert np.array_equal(Ug2, Ur2) and np.array_equal(Tg2, Tr2), case.name
            r.close()
        assert run.n_max >= run.n_valid + 1
        run.close()
