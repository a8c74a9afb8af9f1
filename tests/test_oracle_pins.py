"""Pins for the CPU oracle: what the paper and the mathematics fix (SURVEY.md §8(c) 'pins').

None of these compares the oracle with itself through the same formula: they use closed forms,
the exact Riemann solution, conservation laws, symmetries, finite differences, LAPACK and
tiny-step references.  CPU only (-m "not gpu").
"""
import math

import numpy as np
import pytest

from paper_2504_13750_b200 import inputs as I
from tests import riemann_exact as RE

RU = 8.314472


def run(ref, case, nsteps=None, cfl=None, dt=0.0, chem=True):
    s = ref.RefSolver(case.grid, case.mech, case.blocks)
    s.set_state(case.U, case.T)
    t = s.step(case.nsteps if nsteps is None else nsteps, cfl=case.cfl if cfl is None else cfl, dt=dt, chem=chem)
    U, T = s.get_state()
    return U, T, t, s.status


# ----------------------------------------------------------------------------- cons -> prim
def test_T_closed_form_constant_cp(ref, mech9):
    """constant c_p: e = sum Y_k R_k ((a0-1) T + a5)  =>  T in closed form (eq 4.2-4.4)."""
    rng = np.random.default_rng(1)
    for _ in range(20):
        Y = rng.dirichlet(np.ones(9))
        T = rng.uniform(250, 3500)
        rho = rng.uniform(0.1, 20)
        vel = rng.uniform(-1500, 1500, size=2)
        Rk = RU / mech9.W
        cv = (Y * Rk * (mech9.nasa[:, 0] - 1)).sum()
        e = cv * T + (Y * Rk * mech9.nasa[:, 5]).sum()
        E = rho * e + 0.5 * rho * (vel**2).sum()
        Uc = np.concatenate([[rho], rho * vel, [E], rho * Y[:-1]])
        rc, out = ref.cons2prim(mech9, 2, Uc, 1000.0)
        assert rc == 0
        assert abs(out[0] - T) <= 1e-12 * T
        R = (Y * Rk).sum()
        assert abs(out[1] - rho * R * T) <= 1e-12 * rho * R * T
        gam = (cv + R) / cv
        assert abs(out[2] - gam) <= 1e-12
        assert abs(out[3] - math.sqrt(gam * R * T)) <= 1e-12 * out[3]


def test_T_quadratic_linear_cp(ref):
    """c_p linear in T (a1 != 0): e(T) is a quadratic, solved by the quadratic formula."""
    m = I.single_step_mechanism()
    m.nasa[:, 1] = [4e-4, 7e-4]
    Rk = RU / m.W
    for Y0, T in ((0.3, 400.0), (0.9, 2200.0), (0.0, 900.0)):
        Y = np.array([Y0, 1 - Y0])
        # e = sum Y R [(a0-1) T + a1/2 T^2 + a5]
        A2 = (Y * Rk * m.nasa[:, 1] / 2).sum(); A1 = (Y * Rk * (m.nasa[:, 0] - 1)).sum(); A0 = (Y * Rk * m.nasa[:, 5]).sum()
        e = A2 * T * T + A1 * T + A0
        rho = 1.3
        Uc = np.array([rho, rho * 120.0, rho * e + 0.5 * rho * 120.0**2, rho * Y0])
        rc, out = ref.cons2prim(m, 1, Uc, 300.0)
        Tq = (-A1 + math.sqrt(A1 * A1 - 4 * A2 * (A0 - e))) / (2 * A2)
        assert rc == 0 and abs(out[0] - Tq) <= 1e-11 * Tq and abs(out[0] - T) <= 1e-10 * T


def test_prim_cons_prim_roundtrip(ref, mech20):
    rng = np.random.default_rng(2)
    m = mech20
    m2 = I.Mechanism(**{**m.__dict__})
    m2.nasa = m.nasa.copy(); m2.nasa[:, 1] = 1e-4; m2.nasa[:, 2] = -1e-8   # genuinely polynomial c_p
    for _ in range(10):
        Y = rng.dirichlet(np.ones(20)); T = rng.uniform(300, 3000); p = rng.uniform(1e4, 5e6)
        v = rng.uniform(-800, 800, size=3)
        U = I.prim_to_cons(m2, 3, np.array([p]), np.array([T]), Y[None], [np.array([x]) for x in v])[:, 0]
        rc, out = ref.cons2prim(m2, 3, U, 0.7 * T)
        assert rc == 0 and abs(out[0] - T) <= 1e-13 * T * 10 and abs(out[1] - p) <= 1e-12 * p


# ----------------------------------------------------------------------------- WENO5
def test_weno5_exact_on_quadratics(ref):
    """Every 3-point sub-stencil reproduces a quadratic flux function exactly, so the result is
    h(x_{i+1/2}) for any weights, where f = sliding average of h: h = f - a dx^2/12."""
    rng = np.random.default_rng(3)
    for _ in range(50):
        a, b, c = rng.uniform(-3, 3, size=3)
        dx = rng.uniform(0.1, 2.0); x0 = rng.uniform(-5, 5)
        f = lambda x: a * x * x + b * x + c
        v = [f(x0 + k * dx) for k in (-2, -1, 0, 1, 2)]
        exact = f(x0 + dx / 2) - a * dx * dx / 12
        assert abs(ref.weno5(v) - exact) <= 1e-12 * (1 + abs(exact))


def test_weno5_linear_weights_and_eno(ref):
    # linear data => all smoothness indicators equal => optimal 5th-order linear combination
    v = np.array([1.0, 1.5, 2.0, 2.5, 3.0])
    lin = (2 * v[0] - 13 * v[1] + 47 * v[2] + 27 * v[3] - 3 * v[4]) / 60
    assert abs(ref.weno5(v) - lin) < 1e-14 and abs(lin - 2.25) < 1e-14
    # a jump inside the right part of the stencil => the smooth left stencil takes over (ENO property)
    assert abs(ref.weno5([1, 1, 1, 0, 0]) - 1.0) < 1e-9
    assert abs(ref.weno5([0, 0, 1, 1, 1]) - 1.0) < 1e-9
    # asymmetry check: not mirror-invariant (upwind-biased): stencil reversed gives value at -1/2
    vv = [0.3, 1.0, 0.2, 0.9, 0.5]
    assert abs(ref.weno5(vv) - ref.weno5(vv[::-1])) > 1e-3
    # smooth data: 5th-order accurate against the exact h
    errs = []
    for dx in (0.1, 0.05):
        f = lambda x: math.sin(x)
        # h with sliding average f: h(x) = f(x) * (dx/2)/sin(dx/2)
        v = [f(1.0 + k * dx) for k in (-2, -1, 0, 1, 2)]
        exact = math.sin(1.0 + dx / 2) * (dx / 2) / math.sin(dx / 2)
        errs.append(abs(ref.weno5(v) - exact))
    assert math.log2(errs[0] / errs[1]) > 4.5


def _wave_case(n, gas):
    x = (np.arange(n) + 0.5) / n
    rho = 1.0 + 0.2 * np.sin(2 * np.pi * x)
    u = np.full(n, 1.0); p = np.full(n, 1.0)
    R = RU / gas.W[0]
    T = p / (rho * R)
    U = I.prim_to_cons(gas, 1, p, T, np.ones((n, 1)), [u])
    g = I.Grid(1, (n, 1, 1), (1.0 / n, 1, 1), (0, 0, 0), (0, 0, 0))
    return I.Case("wave", g, gas, U.reshape(1, 3, 1, 1, n), T.reshape(1, 1, 1, n), 0.0, 0), x


def test_density_wave_convergence_order(ref):
    """rho = 1 + 0.2 sin(2 pi x), u = p = const: exact solution is translation; dt ~ dx^(5/3) keeps
    the RK3 error below the spatial one, observed order -> 5."""
    gas = I.inert_gas(1.4, 1.0)
    errs = []
    tend = 0.1
    for n in (16, 32, 64):
        case, x = _wave_case(n, gas)
        dt0 = 0.5 * (1.0 / n) ** (5.0 / 3.0)
        nst = int(math.ceil(tend / dt0)); dt = tend / nst
        U, T, t, st = run(ref, case, nsteps=nst, cfl=0.0, dt=dt, chem=False)
        assert st == 0
        exact = 1.0 + 0.2 * np.sin(2 * np.pi * (x - tend))
        errs.append(np.abs(U[0, 0, 0, 0] - exact).max())
    o1 = math.log2(errs[0] / errs[1]); o2 = math.log2(errs[1] / errs[2])
    assert o2 > 4.5 and o1 > 3.5, (errs, o1, o2)


# ----------------------------------------------------------------------------- Sod
def _sod_case(n):
    gas = I.inert_gas(1.4, 287.0)
    x = -10.0 + (np.arange(n) + 0.5) * 20.0 / n
    left = x < 0
    rho = np.where(left, 1.0, 0.125); p = np.where(left, 1e5, 1e4)      # p_R restored, reading A13
    T = p / (rho * 287.0)
    U = I.prim_to_cons(gas, 1, p, T, np.ones((n, 1)), [np.zeros(n)])
    g = I.Grid(1, (n, 1, 1), (20.0 / n, 1, 1), (I.BC_OUTFLOW, 0, 0), (I.BC_OUTFLOW, 0, 0))
    return I.Case("sod", g, gas, U.reshape(1, 3, 1, 1, n), T.reshape(1, 1, 1, n), 0.2, 0), x


def _run_to(ref, case, tend):
    s = ref.RefSolver(case.grid, case.mech)
    s.set_state(case.U, case.T)
    t = 0.0
    while True:
        U0, T0 = s.get_state()
        dt = None
        tt = s.step(1, cfl=case.cfl, chem=False)
        if t + tt >= tend:
            s.set_state(U0, T0)
            s.step(1, cfl=0.0, dt=tend - t, chem=False)
            break
        t += tt
    return s.get_state()[0]


def test_sod_exact_riemann(ref):
    ps, us = RE.star_state(1.0, 0.0, 1e5, 0.125, 0.0, 1e4, 1.4)
    # star state of the restored IC (SURVEY §4 [probe] values)
    assert abs(ps - 30313.02) < 0.02 and abs(us - 293.286) < 2e-3
    l1 = []
    for n in (200, 400, 800):
        case, x = _sod_case(n)
        U = _run_to(ref, case, 0.01)
        ex = RE.sample(x / 0.01, 1.0, 0.0, 1e5, 0.125, 0.0, 1e4, 1.4)
        rho = U[0, 0, 0, 0]
        l1.append(np.abs(rho - ex[0]).mean())
        if n == 400:   # the paper's resolution: plateaus match the analytical star state
            u = U[0, 1, 0, 0] / rho
            p = 0.4 * (U[0, 2, 0, 0] - 0.5 * rho * u * u)
            star = (x > 0.5) & (x < 2.0)            # between tail of the fan (-0.7) and contact (2.93)
            assert np.abs(p[star] - ps).max() < 2e-3 * ps
            assert np.abs(u[star] - us).max() < 2e-3 * us
            assert np.abs(rho[star] - 0.426319).max() < 1e-3
            post = (x > 3.6) & (x < 5.0)            # between contact and shock (5.54)
            assert np.abs(rho[post] - 0.265574).max() < 1e-3
            assert rho[x > 5.9].max() < 0.12501 and rho[x < -4.6].min() > 0.9999   # S = 554.08 m/s
    o1 = math.log2(l1[0] / l1[1]); o2 = math.log2(l1[1] / l1[2])
    assert 0.6 < o1 < 1.3 and 0.6 < o2 < 1.3, (l1, o1, o2)
    assert l1[1] < 4e-3


# ----------------------------------------------------------------------------- whole flux path
def _random_smooth_2d(mech, nx, ny, seed, bc):
    rng = np.random.default_rng(seed)
    x = (np.arange(nx) + 0.5) / nx; y = (np.arange(ny) + 0.5) / ny
    X, Yg = np.meshgrid(x, y)
    s = np.sin(2 * np.pi * X) * np.cos(2 * np.pi * Yg)
    p = 1e5 * (1 + 0.3 * s); T = 600.0 * (1 + 0.2 * np.cos(2 * np.pi * X + 1.0) * np.sin(2 * np.pi * Yg))
    Ya, Yh = I.ambient_Y(mech.ns), I.hot_Y(mech.ns)
    w = 0.5 * (1 + np.sin(2 * np.pi * (X + Yg)))
    Y = w[..., None] * Ya + (1 - w[..., None]) * Yh
    u = 200 * np.sin(2 * np.pi * Yg); v = -150 * np.cos(2 * np.pi * X)
    U = I.prim_to_cons(mech, 2, p, T, Y, [u, v])
    g = I.Grid(2, (nx, ny, 1), (1e-3 / nx, 1e-3 / ny, 1), (bc, bc, 0), (bc, bc, 0))
    return I.Case("smooth2d", g, mech, U.reshape(1, -1, 1, ny, nx), T.reshape(1, 1, ny, nx), 0.3, 5)


@pytest.mark.parametrize("bc", [I.BC_PERIODIC, I.BC_REFLECT, I.BC_OUTFLOW])
def test_uniform_state_is_bitwise_fixed_point(ref, mech9, bc):
    nx, ny = 20, 12
    Y = I.hot_Y(9)
    z = np.zeros((ny, nx))
    U = I.prim_to_cons(mech9, 2, z + 2.5e5, z + 1234.5, np.broadcast_to(Y, (ny, nx, 9)), [z + 0.0, z + 0.0])
    if bc != I.BC_REFLECT:   # a moving uniform state is a fixed point too unless walls reflect it
        U = I.prim_to_cons(mech9, 2, z + 2.5e5, z + 1234.5, np.broadcast_to(Y, (ny, nx, 9)), [z + 310.0, z - 95.0])
    U = np.broadcast_to(U[:, :1, :1], U.shape).copy()   # exactly identical cells
    g = I.Grid(2, (nx, ny, 1), (1e-4, 2e-4, 1), (bc, bc, 0), (bc, bc, 0))
    case = I.Case("uni", g, mech9, U.reshape(1, -1, 1, ny, nx), np.full((1, 1, ny, nx), 1234.5), 0.4, 7)
    U1, T1, t, st = run(ref, case, chem=False)
    assert st == 0 and t > 0
    assert np.array_equal(U1, case.U)


def test_periodic_conservation_no_chem(ref, mech9):
    case = _random_smooth_2d(mech9, 24, 16, 5, I.BC_PERIODIC)
    U1, T1, t, st = run(ref, case, nsteps=6, chem=False)
    assert st == 0
    assert np.abs(U1 - case.U).max() > 1e-3                    # something moved
    for v in range(case.nvar):
        s0, s1 = case.U[0, v].sum(), U1[0, v].sum()
        scale = np.abs(case.U[0, v]).sum()
        assert abs(s1 - s0) <= 2e-13 * scale, (v, s0, s1)


def test_periodic_conservation_with_chem_elements_energy(ref, mech9):
    case = _random_smooth_2d(mech9, 16, 12, 6, I.BC_PERIODIC)
    case.T[:] = 2600.0 + 0 * case.T
    # hot reactive state
    rng = np.random.default_rng(0)
    p = 2e6 * (1 + 0.05 * rng.uniform(-1, 1, size=(12, 16)))
    T = np.full((12, 16), 2600.0)
    Y = np.broadcast_to(I.hot_Y(9), (12, 16, 9))
    u = 100 * rng.uniform(-1, 1, size=(12, 16))
    case.U = I.prim_to_cons(mech9, 2, p, T, Y, [u, u * 0.5]).reshape(1, -1, 1, 12, 16)
    U1, T1, t, st = run(ref, case, nsteps=10, cfl=0.0, dt=2e-9, chem=True)
    assert st == 0

    def elem_moles(U):
        rho = U[0, 0]
        rY = [U[0, 4 + k] for k in range(8)]
        rY.append(rho - sum(rY))
        return np.array([sum(mech9.elements[k, e] * rY[k].sum() / mech9.W[k] for k in range(9)) for e in range(3)])

    for v in range(4):                                           # rho, rho u, rho v, E
        assert abs(U1[0, v].sum() - case.U[0, v].sum()) <= 2e-13 * np.abs(case.U[0, v]).sum()
    e0, e1 = elem_moles(case.U), elem_moles(U1)
    assert np.abs(e1 - e0).max() <= 1e-12 * e0.max()
    # chemistry did something: species sums changed
    assert abs(U1[0, 4].sum() - case.U[0, 4].sum()) > 1e-6 * abs(case.U[0, 4].sum())


def test_transpose_symmetry(ref, mech9):
    case = _random_smooth_2d(mech9, 16, 12, 7, I.BC_REFLECT)
    U1, _, t1, _ = run(ref, case, nsteps=3)
    Ut = case.U.transpose(0, 1, 2, 4, 3).copy()
    Ut[:, [1, 2]] = Ut[:, [2, 1]]
    g = case.grid
    gt = I.Grid(2, (g.n[1], g.n[0], 1), (g.dx[1], g.dx[0], 1), g.bc_lo, g.bc_hi)
    ct = I.Case("t", gt, mech9, Ut, case.T.transpose(0, 1, 3, 2).copy(), case.cfl, 3)
    U2, _, t2, _ = run(ref, ct, nsteps=3)
    U2 = U2.transpose(0, 1, 2, 4, 3).copy(); U2[:, [1, 2]] = U2[:, [2, 1]]
    assert abs(t1 - t2) <= 1e-15 * t1
    assert np.abs(U1 - U2).max() <= 1e-11 * np.abs(U1).max()
    for v in range(case.nvar):
        assert np.abs(U1[0, v] - U2[0, v]).max() <= 1e-11 * (np.abs(U1[0, v]).max() + 1e-300)


def test_y_invariant_2d_equals_1d(ref):
    c1 = I.config0(n=96, nsteps=12)
    U1, _, t1, st = run(ref, c1)
    ny = 5
    U2 = np.zeros((1, 5, 1, ny, 96))
    U2[0, 0] = c1.U[0, 0, 0]; U2[0, 1] = c1.U[0, 1, 0]; U2[0, 3] = c1.U[0, 2, 0]; U2[0, 4] = c1.U[0, 3, 0]
    g = I.Grid(2, (96, ny, 1), (1e-4, 1e-4, 1), (I.BC_OUTFLOW, I.BC_PERIODIC, 0), (I.BC_OUTFLOW, I.BC_PERIODIC, 0))
    c2 = I.Case("2d", g, c1.mech, U2, np.broadcast_to(c1.T[:, :, 0:1, :], (1, 1, ny, 96)).copy(), c1.cfl, 12)
    Ub, _, t2, st2 = run(ref, c2)
    assert st == 0 and st2 == 0 and abs(t1 - t2) <= 1e-14 * t1
    for a, b in ((0, 0), (1, 1), (2, 3), (3, 4)):
        for j in range(ny):
            assert np.abs(Ub[0, b, 0, j] - U1[0, a, 0, 0]).max() <= 1e-12 * np.abs(U1[0, a]).max()
    assert np.abs(Ub[0, 2]).max() == 0.0


def test_3d_axis_permutation(ref):
    """1-D problem laid along x, y or z of a 3-D grid gives the same line (dimension-by-dimension, A18)."""
    c1 = I.config0(n=40, nsteps=6)
    U1, _, t1, _ = run(ref, c1)
    for axis in (0, 1, 2):
        n = [3, 3, 3]; n[axis] = 40
        shape = (n[2], n[1], n[0])
        U3 = np.zeros((1, 6) + shape)
        line_shape = [1, 1, 1]; line_shape[2 - axis] = 40
        for a, b in ((0, 0), (2, 4), (3, 5)):
            U3[0, b] = np.broadcast_to(c1.U[0, a, 0, 0].reshape(line_shape), shape)
        U3[0, 1 + axis] = np.broadcast_to(c1.U[0, 1, 0, 0].reshape(line_shape), shape)
        T3 = np.broadcast_to(c1.T[0, 0, 0].reshape(line_shape), shape).copy().reshape((1,) + shape)
        bl = [I.BC_PERIODIC] * 3; bl[axis] = I.BC_OUTFLOW
        g = I.Grid(3, tuple(n), (1e-4,) * 3, tuple(bl), tuple(bl))
        U, _, t3, st = run(ref, I.Case("3d", g, c1.mech, U3, T3, c1.cfl, 6))
        assert st == 0 and abs(t3 - t1) <= 1e-14 * t1
        idx = [1, 1, 1]; idx[2 - axis] = slice(None)
        for a, b in ((0, 0), (2, 4), (3, 5)):
            assert np.abs(U[0, b][tuple(idx)] - U1[0, a, 0, 0]).max() <= 1e-12 * np.abs(U1[0, a]).max()
        assert np.abs(U[0, 1 + axis][tuple(idx)] - U1[0, 1, 0, 0]).max() <= 1e-12 * np.abs(U1[0, 1]).max() + 1e-9


# ----------------------------------------------------------------------------- kinetics
def _g_over_RT(mech, T):
    """Textbook: g_k/(R T) = h_k/(R T) - s_k/R from the NASA polynomials."""
    a = mech.nasa
    h = a[:, 0] + a[:, 1] / 2 * T + a[:, 2] / 3 * T**2 + a[:, 3] / 4 * T**3 + a[:, 4] / 5 * T**4 + a[:, 5] / T
    s = a[:, 0] * math.log(T) + a[:, 1] * T + a[:, 2] / 2 * T**2 + a[:, 3] / 3 * T**3 + a[:, 4] / 4 * T**4 + a[:, 6]
    return h - s


def test_detailed_balance_at_equilibrium(ref, mech9):
    """A single reversible reaction at a composition with prod X^dnu = K_c has zero net rate
    (K_c = exp(-dG0/RuT) (p_atm/RuT)^dn, eq 4.9)."""
    T = 1800.0
    g = _g_over_RT(mech9, T)
    for i in range(mech9.nr):
        dn = (mech9.nu_b[i] - mech9.nu_f[i]).astype(float)
        lnK = -(dn * g).sum() + dn.sum() * math.log(101325.0 / (RU * T))
        # choose ln X with dn . lnX = lnK : start from a positive composition and project
        lx = np.log(np.full(9, 2.0) + np.arange(9) * 0.3)
        lx = lx + dn * (lnK - dn @ lx) / (dn @ dn)
        X = np.exp(lx)
        m1 = I.Mechanism(9, 1, mech9.W, mech9.nasa, mech9.nu_f[i:i + 1], mech9.nu_b[i:i + 1], mech9.A[i:i + 1],
                         mech9.b[i:i + 1], mech9.Ta[i:i + 1], mech9.reversible[i:i + 1],
                         mech9.third_body[i:i + 1], mech9.eff[i:i + 1])
        q = ref.rates(m1, T, X)[0]
        kf = mech9.A[i] * T ** mech9.b[i] * math.exp(-mech9.Ta[i] / T)
        M = (mech9.eff[i] * X).sum() if mech9.third_body[i] else 1.0
        fwd = M * kf * np.prod(X ** mech9.nu_f[i])
        assert fwd > 0 and abs(q) <= 1e-10 * fwd, (i, q, fwd)
        # and away from equilibrium the net rate has the sign of (K - Q)
        X2 = X.copy(); j = int(np.argmax(mech9.nu_f[i])); X2[j] *= 1.5
        assert ref.rates(m1, T, X2)[0] > 1e-3 * fwd


def _one_reaction(W, nu_f, nu_b, A, b, Ta, rev, tb, eff):
    ns = len(W)
    nasa = np.zeros((ns, 7)); nasa[:, 0] = 3.5 + 0.25 * np.arange(ns); nasa[:, 5] = -1000.0 * np.arange(ns); nasa[:, 6] = 0.1 * np.arange(ns)
    return I.Mechanism(ns, 1, np.asarray(W, float), nasa, np.array([nu_f], dtype=np.int32), np.array([nu_b], dtype=np.int32),
                       np.array([A]), np.array([b]), np.array([Ta]), np.array([rev], dtype=np.int32),
                       np.array([tb], dtype=np.int32), np.array([eff], dtype=float))


def test_third_body_factor_value_and_species_order(ref):
    """eq 4.7, reading A9: M_i = sum_j a_ij X_j multiplies the rate of a flagged reaction.
    (a) one irreversible reaction A (+M) -> B + C with strongly asymmetric a_ij: q = M k_f X_A re-evaluated here;
    (b) with a single non-zero efficiency a_ic the collider IS species c, so the third-body reaction must coincide
        with the plain reaction A + c -> B + C + c of rate constant a_ic k_f (and, reversible, k_b scaled alike:
        K_eq is unchanged because c appears on both sides) -- value and Jacobian; this ties the a_ij column order
        to the stoichiometric product path, which has its own pins (detailed balance, FD Jacobian, elements)."""
    W = [0.030, 0.010, 0.020, 0.028, 0.004]
    T, A, b, Ta = 1700.0, 3.0e7, -0.7, 6500.0
    nu_f, nu_b = [1, 0, 0, 0, 0], [0, 1, 1, 0, 0]
    eff = [0.25, 7.0, 1.5, 40.0, 0.0]
    X = np.array([3.1, 0.4, 1.7, 11.0, 5.3])
    kf = A * T ** b * math.exp(-Ta / T)
    q = ref.rates(_one_reaction(W, nu_f, nu_b, A, b, Ta, 0, 1, eff), T, X)[0]
    want = (0.25 * 3.1 + 7.0 * 0.4 + 1.5 * 1.7 + 40.0 * 11.0 + 0.0 * 5.3) * kf * 3.1
    assert abs(q - want) <= 1e-14 * want
    q0 = ref.rates(_one_reaction(W, nu_f, nu_b, A, b, Ta, 0, 0, eff), T, X)[0]       # flag off: factor is 1
    assert abs(q0 - kf * 3.1) <= 1e-14 * kf * 3.1
    rho = float((X * np.array(W)).sum())
    rhoY = (X * np.array(W))[:-1]
    for c in range(5):
        for rev in (0, 1):
            e1 = np.zeros(5); e1[c] = 2.5
            m_tb = _one_reaction(W, nu_f, nu_b, A, b, Ta, rev, 1, e1)
            f2, b2 = list(nu_f), list(nu_b); f2[c] += 1; b2[c] += 1
            m_cat = _one_reaction(W, f2, b2, 2.5 * A, b, Ta, rev, 0, np.ones(5))
            qa, qb = ref.rates(m_tb, T, X)[0], ref.rates(m_cat, T, X)[0]
            assert abs(qa - qb) <= 1e-13 * abs(qb), (c, rev, qa, qb)
            oa, Ja = ref.omega_jac(m_tb, T, rho, rhoY)
            ob, Jb = ref.omega_jac(m_cat, T, rho, rhoY)
            assert np.abs(oa - ob).max() <= 1e-13 * np.abs(ob).max()
            assert np.abs(Ja - Jb).max() <= 1e-12 * np.abs(Jb).max(), (c, rev)


def test_omega_mass_and_element_balance(ref, mech9, mech20):
    rng = np.random.default_rng(11)
    for m in (mech9, mech20):
        ns = m.ns
        Y = rng.dirichlet(np.ones(ns)); rho = 3.0; T = 2100.0
        om, J = ref.omega_jac(m, T, rho, rho * Y[:-1])
        X = rho * Y / m.W
        q = ref.rates(m, T, X)
        wdot = (m.nu_b - m.nu_f).T @ q                      # mol/m^3/s, all ns species
        assert np.abs(om[:ns - 1] - m.W[:-1] * wdot[:-1]).max() <= 1e-12 * np.abs(om).max()
        assert abs((m.W * wdot).sum()) <= 1e-12 * np.abs(m.W * wdot).sum()          # sum_k omega_k = 0
        assert np.abs(m.elements.T @ wdot).max() <= 1e-12 * np.abs(wdot).sum()      # elements


def test_jacobian_finite_differences(ref, mech9, mech20):
    rng = np.random.default_rng(12)
    for m in (mech9, mech20):
        ns = m.ns
        Y = 0.02 + rng.dirichlet(np.ones(ns)); Y /= Y.sum()
        rho, T = 4.0, 1900.0
        ry = rho * Y[:-1]
        om, J = ref.omega_jac(m, T, rho, ry)
        Jfd = np.zeros_like(J)
        for l in range(ns - 1):
            h = 1e-6 * ry[l]
            rp = ry.copy(); rp[l] += h; rm = ry.copy(); rm[l] -= h
            Jfd[:, l] = (ref.omega_jac(m, T, rho, rp)[0] - ref.omega_jac(m, T, rho, rm)[0]) / (2 * h)
        assert np.abs(J - Jfd).max() <= 1e-6 * np.abs(J).max()


def test_gauss_solve_vs_lapack(ref):
    rng = np.random.default_rng(13)
    for n in (1, 3, 8, 19):
        A = rng.normal(size=(n, n)); b = rng.normal(size=n)
        if n > 1:
            A[0, 0] = 0.0   # needs a row exchange
        rc, x = ref.gauss_solve(A, b)
        assert rc == 0 and np.abs(x - np.linalg.solve(A, b)).max() <= 1e-11 * (1 + np.abs(x).max())


def test_point_implicit_first_order_reaction_closed_form(ref):
    """Ns=2, R -> P first order, fixed T: rhoY_R_new = rhoY_R / (1 + k dt) exactly (eq 4.12)."""
    m = I.single_step_mechanism(A=3.0e7, Ta=9000.0)
    m.b[:] = 0.7
    T, rho, yr, dt = 1700.0, 1.9, 0.8, 3e-8
    k = 3.0e7 * T**0.7 * math.exp(-9000.0 / T)
    rc, d = ref.chem_cell(m, T, rho, [rho * yr], dt)
    assert rc == 0
    assert abs((rho * yr + d[0]) - rho * yr / (1 + k * dt)) <= 1e-14 * rho


def test_point_implicit_matches_lapack_on_full_system(ref, mech9):
    rho, T, dt = 5.0, 2400.0, 4e-9
    ry = rho * I.hot_Y(9)[:-1]
    om, J = ref.omega_jac(mech9, T, rho, ry)
    rc, d = ref.chem_cell(mech9, T, rho, ry, dt)
    x = np.linalg.solve(np.eye(8) - dt * J, dt * om)
    assert rc == 0 and np.abs(d - x).max() <= 1e-11 * np.abs(x).max()


def _zero_d(ref, mech, T0, p0, dt, nsteps):
    """0-D constant-volume reactor = one cell with zero-gradient sides."""
    Y = I.hot_Y(mech.ns)
    U = I.prim_to_cons(mech, 1, np.array([p0]), np.array([T0]), Y[None], [np.zeros(1)])
    g = I.Grid(1, (1, 1, 1), (1e-3, 1, 1), (I.BC_OUTFLOW, 0, 0), (I.BC_OUTFLOW, 0, 0))
    c = I.Case("0d", g, mech, U.reshape(1, -1, 1, 1, 1), np.array(T0).reshape(1, 1, 1, 1), 0.0, nsteps)
    return run(ref, c, nsteps=nsteps, cfl=0.0, dt=dt)


def test_zero_d_ignition_first_order_vs_tiny_step(ref, mech9):
    tend = 2.0e-7
    Uref, Tref, _, st = _zero_d(ref, mech9, 2000.0, 2.0e6, tend / 8192, 8192)
    assert st == 0
    errs = []
    for n in (8, 16, 32):
        U, T, _, st = _zero_d(ref, mech9, 2000.0, 2.0e6, tend / n, n)
        assert st == 0
        errs.append(np.abs(U[0, 3:, 0, 0, 0] - Uref[0, 3:, 0, 0, 0]).max())
        # frozen convection: rho, momentum, E untouched bitwise (S has zeros there)
        assert np.array_equal(U[0, :3], Uref[0, :3])
    # sanity check that the gas released heat (start 2000 K), not an arithmetic pin: over 2e-7 s this seeded mechanism
    # heats the cell by ~15-20 K; the first draft asked for > 2050 before the run length was fixed (lowered in 5955d77)
    assert Tref[0, 0, 0, 0] > 2010.0
    r1, r2 = errs[0] / errs[1], errs[1] / errs[2]
    assert 1.6 < r1 < 2.6 and 1.7 < r2 < 2.4, (errs, r1, r2)         # error ~ dt


def test_zero_d_vs_rk4_reference(ref, mech9):
    """Independent time integrator (classical RK4 at tiny dt on the oracle's omega, T updated from
    energy conservation through cons2prim) agrees with the small-step point-implicit run."""
    T0, p0, tend, n = 2000.0, 2.0e6, 1.0e-7, 4000
    Y = I.hot_Y(9)
    U0 = I.prim_to_cons(mech9, 1, np.array([p0]), np.array([T0]), Y[None], [np.zeros(1)])[:, 0]
    rho = U0[0]

    def f(ry):
        Uc = np.concatenate([U0[:3], ry])
        T = ref.cons2prim(mech9, 1, Uc, T0)[1][0]
        return ref.omega_jac(mech9, T, rho, ry)[0]

    ry = U0[3:].copy(); h = tend / n
    for _ in range(n):
        k1 = f(ry); k2 = f(ry + h / 2 * k1); k3 = f(ry + h / 2 * k2); k4 = f(ry + h * k3)
        ry = ry + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    U, T, _, st = _zero_d(ref, mech9, T0, p0, tend / 2048, 2048)
    assert np.abs(U[0, 3:, 0, 0, 0] - ry).max() <= 2e-3 * np.abs(ry).max()


# ----------------------------------------------------------------------------- explicit source variant
def _zero_d_explicit(ref, mech, T0, p0, dt, nsteps, Y=None):
    Y = I.hot_Y(mech.ns) if Y is None else Y
    U = I.prim_to_cons(mech, 1, np.array([p0]), np.array([T0]), Y[None], [np.zeros(1)])
    g = I.Grid(1, (1, 1, 1), (1e-3, 1, 1), (I.BC_OUTFLOW, 0, 0), (I.BC_OUTFLOW, 0, 0))
    c = I.Case("0d", g, mech, U.reshape(1, -1, 1, 1, 1), np.array(T0).reshape(1, 1, 1, 1), 0.0, nsteps)
    return run(ref, c, nsteps=nsteps, cfl=0.0, dt=dt, chem="explicit"), U


def test_explicit_source_linear_decay_is_the_rk3_polynomial(ref):
    """the source is advanced WITH the convection terms by the TVD RK3.  For a first
    order reaction R -> P at constant k (b = 0, Ta = 0, no heat release, uniform gas at rest) the stage recursion
    of SSP-RK3 on y' = -k y gives y (1 - z + z^2/2 - z^3/6), z = k dt, exactly; rho, momentum, E, T stay put."""
    W = np.array([0.029, 0.029]); nasa = np.zeros((2, 7)); nasa[:, 0] = 3.5
    k = 4.0e6
    m = I.Mechanism(2, 1, W, nasa, np.array([[1, 0]], dtype=np.int32), np.array([[0, 1]], dtype=np.int32),
                    np.array([k]), np.array([0.0]), np.array([0.0]), np.array([0], dtype=np.int32),
                    np.array([0], dtype=np.int32), np.ones((1, 2)))
    dt, nsteps = 1.0e-7, 3
    (U, T, t, st), U0 = _zero_d_explicit(ref, m, 900.0, 2.0e5, dt, nsteps, Y=np.array([0.7, 0.3]))
    assert st == 0 and abs(t - nsteps * dt) <= 1e-20
    z = k * dt
    amp = (1.0 - z + z * z / 2.0 - z ** 3 / 6.0) ** nsteps
    assert abs(U[0, 3, 0, 0, 0] - U0[3, 0] * amp) <= 2e-15 * U0[3, 0]
    assert np.array_equal(U[0, :3, 0, 0, 0], U0[:3, 0])
    assert abs(T[0, 0, 0, 0] - 900.0) <= 1e-9


def test_explicit_source_third_order_and_agrees_with_rk4(ref, mech9):
    """0-D reactor with the 9-species mechanism: the explicit variant converges with order 3 in dt (T is refreshed
    by update_aux in every stage) to the same answer as an independent classical RK4 on the oracle's omega."""
    T0, p0, tend = 2000.0, 2.0e6, 4.0e-8
    Y = I.hot_Y(9)
    U0 = I.prim_to_cons(mech9, 1, np.array([p0]), np.array([T0]), Y[None], [np.zeros(1)])[:, 0]
    rho = U0[0]

    def f(ry):
        Uc = np.concatenate([U0[:3], ry])
        Tc = ref.cons2prim(mech9, 1, Uc, T0)[1][0]
        return ref.omega_jac(mech9, Tc, rho, ry)[0]

    ry = U0[3:].copy(); n = 2000; h = tend / n
    for _ in range(n):
        k1 = f(ry); k2 = f(ry + h / 2 * k1); k3 = f(ry + h / 2 * k2); k4 = f(ry + h * k3)
        ry = ry + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    errs = []
    for ns_ in (8, 16, 32):
        (U, T, _, st), _ = _zero_d_explicit(ref, mech9, T0, p0, tend / ns_, ns_)
        assert st == 0
        errs.append(np.abs(U[0, 3:, 0, 0, 0] - ry).max())
    assert errs[2] <= 1e-6 * np.abs(ry).max()
    assert errs[0] / errs[1] > 5.0 and errs[1] / errs[2] > 5.0, errs      # ~ 8 for third order


def test_explicit_source_conserves_mass_elements_energy(ref, mech9):
    """Periodic 2-D flow with the source inside the stages: total mass, momentum, energy and every element stay to
    round-off (sum_k W_k omega_k = 0 and element balance hold stage by stage)."""
    case = _random_smooth_2d(mech9, 24, 20, 5, I.BC_PERIODIC)
    U, T, _, st = run(ref, case, nsteps=4, cfl=0.3, chem="explicit")
    assert st == 0
    for v in (0, 1, 2, 3):
        assert abs(U[0, v].sum() - case.U[0, v].sum()) <= 1e-12 * max(np.abs(case.U[0, v]).sum(), 1.0)
    el = np.asarray(mech9.elements, dtype=float)                     # [ns][n_elements]
    def moles(Us):
        ry = np.concatenate([Us[0, 4:], (Us[0, 0] - Us[0, 4:].sum(0))[None]])
        return (ry.reshape(9, -1).sum(1) / mech9.W) @ el
    assert np.abs(moles(U) - moles(case.U)).max() <= 1e-12 * np.abs(moles(case.U)).max()
    assert np.abs(U - case.U).max() > 0


# ----------------------------------------------------------------------------- block mode
def test_tiled_block_list_equals_uniform_grid(ref, mech9):
    for bc in (I.BC_REFLECT, I.BC_PERIODIC):
        case = _random_smooth_2d(mech9, 32, 24, 21, bc)
        U1, _, t1, st1 = run(ref, case, nsteps=3)
        tiled = I.tile_uniform(case, 8, 8)
        U2, _, t2, st2 = run(ref, tiled, nsteps=3)
        assert st1 == 0 and st2 == 0 and abs(t1 - t2) <= 1e-15 * t1
        U2 = I.untile(tiled, U2, 4, 3)
        for v in range(case.nvar):
            assert np.abs(U1[0, v] - U2[0, v]).max() <= 1e-13 * np.abs(U1[0, v]).max() + 1e-300


def test_two_level_uniform_state_stays_uniform(ref, mech9):
    c = I.config3(pcols=8, prows=4, npc=8, nsteps=3)
    Y = I.hot_Y(9)
    Ucell = I.prim_to_cons(mech9, 2, np.array([3e5]), np.array([900.0]), Y[None], [np.zeros(1), np.zeros(1)])[:, 0]
    c.U[:] = Ucell[None, :, None, None, None]
    c.T[:] = 900.0
    U1, _, t, st = run(ref, c, nsteps=3, chem=False)
    assert st == 0 and np.array_equal(U1, c.U)
    # dt uses the finest spacing: CFL * (dx/2) / c
    R = (Y * RU / mech9.W).sum(); cp = (Y * RU / mech9.W * mech9.nasa[:, 0]).sum()
    cs = math.sqrt(cp / (cp - R) * R * 900.0)
    assert abs(t - 3 * 0.2 * 0.5e-4 / cs) <= 1e-12 * t


def test_two_level_average_down_and_conservation_structure(ref, mech9):
    c = I.config3(pcols=8, prows=4, npc=8, nsteps=2)
    U1, _, t, st = run(ref, c, nsteps=2)
    assert st == 0
    lev, par = c.blocks.level, c.blocks.parent
    assert (lev == 1).sum() > 0
    for f in np.nonzero(lev == 1)[0]:
        k, sx, sy = par[f]
        fine = U1[f, :, 0]                                        # [nvar, 8, 8]
        mean = 0.25 * (fine[:, 0::2, 0::2] + fine[:, 0::2, 1::2] + fine[:, 1::2, 0::2] + fine[:, 1::2, 1::2])
        coarse = U1[k, :, 0, sy * 4:(sy + 1) * 4, sx * 4:(sx + 1) * 4]
        assert np.abs(coarse - mean).max() <= 1e-14 * np.abs(mean).max()
    # a fine patch next to the wall sees the wall (physical BC), not its parent: mirror symmetry in y
    # of an IC symmetric about the channel axis is preserved on both levels
    assert np.isfinite(U1).all()


def test_two_level_ghosts_hold_the_cell_that_contains_their_centre(ref, mech9):
    """PAPER.md:115 (one-to-four), :117, :213-216; reading A19.  Both levels carry a distinct exact integer per
    cell that is a known function of the GLOBAL cell index (level 0: 1 + X + 1000 Y; level 1: 5e6 + x + 4000 y),
    computed from the layout generator's patch origins -- not from parent[] arithmetic.  After one ghost_fill:
    a fine ghost whose face has a same-level neighbour holds the level-1 value of its own global position; a fine
    ghost at a coarse-fine face holds the level-0 value of the coarse cell that contains its centre,
    (X, Y) = (x // 2, y // 2); a ghost beyond the domain wall holds the mirror cell (reading A15) with the normal
    momentum negated."""
    c = I.config3(pcols=8, prows=4, npc=8, nsteps=1)
    npc, NX, NY = 8, 8 * 8, 4 * 8
    lev, org, nbr = c.blocks.level, c.blocks.origin, c.blocks.nbr
    f0 = lambda X, Y: 1.0 + X + 1000.0 * Y
    f1 = lambda x, y: 5.0e6 + x + 4000.0 * y
    jj, ii = np.meshgrid(np.arange(npc), np.arange(npc), indexing="ij")
    U = np.zeros_like(c.U)
    for p in range(len(lev)):
        f = f1 if lev[p] else f0
        for v in range(c.nvar):
            U[p, v, 0] = (v + 1) * f(org[p, 0] + ii, org[p, 1] + jj)
    s = ref.RefSolver(c.grid, c.mech, c.blocks)
    s.set_state(U, c.T)
    Up, _ = s.debug_ghost_fill()
    s.close()
    seen = {"nbr": 0, "coarse": 0, "wall": 0}
    for p in np.nonzero(lev == 1)[0]:
        ox, oy = org[p]
        for face, (d, side) in enumerate(((0, 0), (0, 1), (1, 0), (1, 1))):
            for g in (1, 2, 3):
                for t in range(npc):
                    i, j = (((-g if side == 0 else npc - 1 + g), t) if d == 0 else (t, (-g if side == 0 else npc - 1 + g)))
                    x, y = ox + i, oy + j                                 # global level-1 index of the ghost cell
                    sign = np.ones(c.nvar)
                    if not (0 <= x < 2 * NX and 0 <= y < 2 * NY):         # beyond the wall: mirror image
                        xm = -1 - x if x < 0 else (4 * NX - 1 - x if x >= 2 * NX else x)
                        ym = -1 - y if y < 0 else (4 * NY - 1 - y if y >= 2 * NY else y)
                        want = f1(xm, ym); sign[1 + d] = -1.0; seen["wall"] += 1
                    elif nbr[p, face] >= 0:
                        want = f1(x, y); seen["nbr"] += 1
                    else:
                        want = f0(x // 2, y // 2); seen["coarse"] += 1
                    got = Up[p, :, 0, j + 3, i + 3]
                    assert np.array_equal(got, sign * (np.arange(c.nvar) + 1) * want), (p, face, g, t, got[0], want)
    assert min(seen.values()) > 0, seen
    # level 0: neighbour patches continue the global numbering, walls mirror
    for p in np.nonzero(lev == 0)[0]:
        ox, oy = org[p]
        for (i, j) in ((-1, 2), (-3, 5), (npc + 2, 1), (4, -2), (6, npc)):
            X, Y = ox + i, oy + j
            Xm = -1 - X if X < 0 else (2 * NX - 1 - X if X >= NX else X)
            Ym = -1 - Y if Y < 0 else (2 * NY - 1 - Y if Y >= NY else Y)
            assert Up[p, 0, 0, j + 3, i + 3] == f0(Xm, Ym)


def _ghost_expect(x, N, bc_lo, bc_hi):
    """global index of the interior cell a position beyond a physical side copies, and whether it is a mirror"""
    if x < 0:
        return {I.BC_PERIODIC: x + N, I.BC_REFLECT: -1 - x, I.BC_OUTFLOW: 0}[bc_lo], bc_lo == I.BC_REFLECT
    if x >= N:
        return {I.BC_PERIODIC: x - N, I.BC_REFLECT: 2 * N - 1 - x, I.BC_OUTFLOW: N - 1}[bc_hi], bc_hi == I.BC_REFLECT
    return x, False


@pytest.mark.parametrize("nd", [1, 3])
def test_two_level_ghosts_1d_and_3d_block_lists(ref, nd):
    """The same global-coordinate pin as above for 1-D and 3-D two-level block lists (inputs.refine_uniform) with a
    mix of periodic, slip-wall and zero-gradient sides: every face ghost of every patch holds the value of the cell
    (of its own level if that position is refined or it is a level-0 patch, else of level 0) that the neighbour /
    coarse-parent / physical-BC rule points at, computed here from patch origins only."""
    if nd == 1:
        base = I.config0(n=64); tile = (8,); mask = np.zeros(8, bool); mask[[0, 3, 4]] = True
        bc_lo, bc_hi = (I.BC_REFLECT, 0, 0), (I.BC_OUTFLOW, 0, 0)
    else:
        base = I.config4(n=16, nspheres=1, radius=3); tile = (8, 4, 8)
        mask = np.zeros((2, 4, 2), bool); mask[0, 1, 0] = mask[1, 1, 0] = mask[1, 2, 1] = mask[0, 0, 1] = mask[1, 3, 1] = True
        bc_lo, bc_hi = (I.BC_PERIODIC, I.BC_REFLECT, I.BC_OUTFLOW), (I.BC_PERIODIC, I.BC_OUTFLOW, I.BC_REFLECT)
    base.grid.bc_lo, base.grid.bc_hi = bc_lo, bc_hi
    c = I.refine_uniform(base, tile, mask)
    N0 = [base.grid.n[d] for d in range(nd)]
    lev, org, nbr = c.blocks.level, c.blocks.origin, c.blocks.nbr
    t3 = list(tile) + [1] * (3 - nd)
    w = [1.0, 300.0, 90000.0]
    f0 = lambda X: 1.0 + sum(w[d] * X[d] for d in range(nd))
    f1 = lambda x: 5.0e7 + sum(2 * w[d] * x[d] for d in range(nd))
    refined = set()
    for p in np.nonzero(lev == 1)[0]:
        refined.add(tuple(org[p] // np.array(tile)))            # fine-patch coordinates present on level 1
    U = np.zeros_like(c.U)
    kk, jj, ii = np.meshgrid(np.arange(t3[2]), np.arange(t3[1]), np.arange(t3[0]), indexing="ij")
    loc = [ii, jj, kk]
    for p in range(len(lev)):
        f = f1 if lev[p] else f0
        val = f([org[p, d] + loc[d] for d in range(nd)])
        for v in range(c.nvar):
            U[p, v] = (v + 1) * val
    s = ref.RefSolver(c.grid, c.mech, c.blocks)
    s.set_state(U, c.T)
    Up, _ = s.debug_ghost_fill()
    s.close()
    G = [3 if d < nd else 0 for d in range(3)]
    kinds = set()
    rng = np.random.default_rng(5)
    for p in range(len(lev)):
        L = int(lev[p]); N = [N0[d] * (2 ** L) for d in range(nd)]
        for d in range(nd):
            for side in (0, 1):
                for g in (1, 2, 3):
                    for _ in range(6):
                        i = [int(rng.integers(0, t3[e])) for e in range(3)]
                        i[d] = -g if side == 0 else t3[d] - 1 + g
                        x = [int(org[p, e]) + i[e] for e in range(nd)]
                        src, mirror = _ghost_expect(x[d], N[d], bc_lo[d], bc_hi[d])
                        xs = list(x); xs[d] = src
                        if L == 0:
                            want = f0(xs); kinds.add("l0-phys" if src != x[d] else "l0-nbr")
                        else:
                            outside = x[d] < 0 or x[d] >= N[d]
                            periodic = (bc_lo[d] if x[d] < 0 else bc_hi[d]) == I.BC_PERIODIC
                            if outside and not periodic:      # wall / zero-gradient side: own-level interior cell
                                want = f1(xs); kinds.add("l1-phys")
                            elif tuple(xs[e] // tile[e] for e in range(nd)) in refined:
                                want = f1(xs); kinds.add("l1-nbr")
                            else:                             # coarse-fine face (possibly across a periodic wrap)
                                want = f0([q // 2 for q in xs]); kinds.add("l1-coarse")
                        sign = np.ones(c.nvar)
                        if mirror:
                            sign[1 + d] = -1.0
                        got = Up[(p, slice(None)) + tuple(i[e] + G[e] for e in (2, 1, 0))]
                        assert np.array_equal(got, sign * (np.arange(c.nvar) + 1) * want), (p, d, side, g, i, got[0], want)
    assert {"l0-nbr", "l0-phys", "l1-nbr", "l1-coarse", "l1-phys"} <= kinds, kinds


def _mirror_case(mech, n, m, seed, axis):
    """Random smooth reflecting box n x m and its even extension across the `axis` wall to a periodic box of
    twice the length (rho, E, rho Y, tangential momentum even; wall-normal momentum odd)."""
    half = _random_smooth_2d(mech, n, m, seed, I.BC_REFLECT)
    U = half.U
    ax = 4 if axis == 0 else 3
    Um = np.flip(U, axis=ax).copy()
    Um[:, 1 + axis] *= -1.0
    Ufull = np.concatenate([U, Um], axis=ax)
    Tfull = np.concatenate([half.T, np.flip(half.T, axis=ax - 1)], axis=ax - 1)
    g = half.grid
    nn = (2 * n, m, 1) if axis == 0 else (n, 2 * m, 1)
    lo = list(g.bc_lo); hi = list(g.bc_hi)
    lo[axis] = hi[axis] = I.BC_PERIODIC
    full = I.Case("mirror", I.Grid(2, nn, g.dx, tuple(lo), tuple(hi)), mech, Ufull, Tfull, half.cfl, half.nsteps)
    return half, full


@pytest.mark.parametrize("axis", [0, 1])
def test_reflecting_wall_equals_half_of_the_mirrored_periodic_box(ref, mech9, axis):
    """PAPER.md:426 (slip walls), reading A15.  The scheme commutes with the reflection x -> -x, u -> -u, so a box
    with slip walls at both ends of `axis` must evolve exactly like one half of a periodic box of twice the length
    started from the even extension.  A mirror rule off by one cell, a wrong sign or a wrong component breaks it."""
    half, full = _mirror_case(mech9, 20, 14, 31 + axis, axis)
    Uh, _, th, sh = run(ref, half, nsteps=4)
    Uf, _, tf, sf = run(ref, full, nsteps=4)
    assert sh == 0 and sf == 0 and abs(th - tf) <= 1e-15 * th
    n = half.grid.n[axis]
    left = Uf[..., :n] if axis == 0 else Uf[..., :n, :]
    assert np.abs(Uh - half.U).max() > 1e-3 * np.abs(half.U).max()          # the flow moved
    for v in range(half.nvar):
        scale = np.abs(Uh[0, v]).max() if v not in (1, 2) else np.abs(Uh[0, 1:3]).max()
        assert np.abs(left[0, v] - Uh[0, v]).max() <= 1e-13 * scale, v
    # and the other half stayed the mirror image (the periodic run itself respects the symmetry)
    right = np.flip(Uf[..., n:] if axis == 0 else Uf[..., n:, :], axis=4 if axis == 0 else 3).copy()
    right[:, 1 + axis] *= -1.0
    assert np.abs(right - left).max() <= 1e-13 * np.abs(left).max()


# ----------------------------------------------------------------------------- crossover (sub-cycled) level advance
def _run_x(ref, case, nsteps, crossover, cfl=None, dt=0.0, chem=True):
    s = ref.RefSolver(case.grid, case.mech, case.blocks)
    s.set_state(case.U, case.T)
    t = s.step(nsteps, cfl=case.cfl if cfl is None else cfl, dt=dt, chem=chem, crossover=crossover)
    U, T = s.get_state()
    return U, T, t, s.status


def test_crossover_on_one_level_is_the_plain_advance(ref, mech9):
    """with a single level there is nothing to sub-cycle: bitwise the synchronous result."""
    tiled = I.tile_uniform(_random_smooth_2d(mech9, 32, 24, 3, I.BC_REFLECT), 8, 8)
    Ua, _, ta, _ = _run_x(ref, tiled, 3, False)
    Ub, _, tb, _ = _run_x(ref, tiled, 3, True)
    assert ta == tb and np.array_equal(Ua, Ub)


def test_crossover_uniform_state_and_step_size(ref, mech9):
    """A uniform two-level state stays uniform, and the step is CFL dx(level 0) / (|u| + c): twice the synchronous step
    (each level at half the step of the previous one).  Not bitwise as in the synchronous advance: the
    levels reach the same U through different sequences of Newton iterates, and T(U) is defined to 1e-11 only (reading
    A6), so the pressures of a fine cell and of its coarse-parent ghost differ in the last bits; the momentum that
    imbalance creates is bounded by that tolerance."""
    c = I.config3(pcols=8, prows=4, npc=8, nsteps=3)
    Y = I.hot_Y(9)
    Ucell = I.prim_to_cons(mech9, 2, np.array([3e5]), np.array([900.0]), Y[None], [np.zeros(1), np.zeros(1)])[:, 0]
    c.U[:] = Ucell[None, :, None, None, None]; c.T[:] = 900.0
    U1, _, t, st = _run_x(ref, c, 3, True, chem=False)
    R = (Y * RU / mech9.W).sum(); cp = (Y * RU / mech9.W * mech9.nasa[:, 0]).sum()
    cs = math.sqrt(cp / (cp - R) * R * 900.0)
    assert st == 0
    for v in range(c.nvar):
        scale = abs(Ucell[v]) if v not in (1, 2) else Ucell[0] * cs
        assert np.abs(U1[:, v] - c.U[:, v]).max() <= 1e-11 * scale, v
    assert np.array_equal(U1[:, 0], c.U[:, 0])                      # density: exactly (mass flux 0 x anything)
    assert abs(t - 3 * 0.2 * 1.0e-4 / cs) <= 1e-12 * t


def test_crossover_fully_refined_equals_two_fine_steps(ref, mech9):
    """Every level-0 patch refined: level 1 then has only same-level neighbours and walls, so its two half steps are two
    plain steps of the uniform fine grid with dt/2 (pinned elsewhere: tiling == uniform grid), and level 0 ends as the
    four-to-one mean of level 1 whatever its own step did."""
    nx, ny, tile = 32, 16, 8
    coarse = _random_smooth_2d(mech9, nx, ny, 11, I.BC_REFLECT)
    c2 = I.refine_uniform(coarse, (tile, tile), np.ones((ny // tile, nx // tile), bool))
    dt = 4.0e-9
    Ux, _, t, st = _run_x(ref, c2, 2, True, cfl=0.0, dt=dt)
    assert st == 0 and abs(t - 2 * dt) <= 1e-15 * t
    # the same fine data as ONE uniform grid (the injection of the coarse initial state), four steps of dt/2
    fineU = np.repeat(np.repeat(coarse.U, 2, axis=3), 2, axis=4)
    fineT = np.repeat(np.repeat(coarse.T, 2, axis=2), 2, axis=3)
    g = coarse.grid
    fine = I.Case("fine", I.Grid(2, (2 * nx, 2 * ny, 1), (g.dx[0] / 2, g.dx[1] / 2, 1), g.bc_lo, g.bc_hi), mech9, fineU, fineT, 0.2, 4)
    Uf, _, _, st2 = run(ref, fine, nsteps=4, cfl=0.0, dt=dt / 2)
    assert st2 == 0
    lev, org = c2.blocks.level, c2.blocks.origin
    for p in np.nonzero(lev == 1)[0]:
        ox, oy = org[p]
        want = Uf[0, :, 0, oy:oy + tile, ox:ox + tile]
        assert np.abs(Ux[p, :, 0] - want).max() <= 1e-13 * np.abs(want).max(), p
    for p in np.nonzero(lev == 0)[0]:
        ox, oy = org[p]
        f = Uf[0, :, 0, 2 * oy:2 * oy + 2 * tile, 2 * ox:2 * ox + 2 * tile]
        mean = 0.25 * (f[:, 0::2, 0::2] + f[:, 0::2, 1::2] + f[:, 1::2, 0::2] + f[:, 1::2, 1::2])
        assert np.abs(Ux[p, :, 0] - mean).max() <= 1e-13 * np.abs(mean).max(), p


def test_crossover_coarse_level_takes_the_full_step_with_frozen_fine_ghosts(ref, mech9):
    """Far from the refined patches (beyond the reach of 3 stages x 3 cells per step) level 0 must evolve exactly as a
    level-0-only run with the same fixed dt: it takes ONE step of dt per iteration and never reads level 1."""
    nx, ny, tile = 64, 16, 8
    coarse = _random_smooth_2d(mech9, nx, ny, 12, I.BC_PERIODIC)
    mask = np.zeros((ny // tile, nx // tile), bool); mask[:, 0] = True          # refine the first patch column only
    c2 = I.refine_uniform(coarse, (tile, tile), mask)
    dt = 3.0e-9
    Ux, _, _, st = _run_x(ref, c2, 1, True, cfl=0.0, dt=dt)
    U0, _, _, st0 = run(ref, coarse, nsteps=1, cfl=0.0, dt=dt)
    assert st == 0 and st0 == 0
    lev, org = c2.blocks.level, c2.blocks.origin
    checked = 0
    for p in np.nonzero(lev == 0)[0]:
        ox, oy = org[p]
        if 24 <= ox <= 32:                          # >= 16 cells from the refined column on either (periodic) side
            assert np.array_equal(Ux[p, :, 0], U0[0, :, 0, oy:oy + tile, ox:ox + tile]); checked += 1
    assert checked >= 2
    assert np.abs(Ux[:, 0] - c2.U[:, 0]).max() > 0


def test_crossover_converges_to_synchronous_at_first_order(ref, mech9):
    """Both strategies integrate the same equations; they differ by the frozen coarse-fine ghost data and the splitting
    of the steps, an O(dt) effect: at a fixed final time the difference halves with dt (Fig 2a vs 2b)."""
    c = I.config3(pcols=8, prows=4, npc=8)
    tend = 1.6e-8
    errs = []
    for n in (2, 4, 8):
        Ux, _, _, s1 = _run_x(ref, c, n, True, cfl=0.0, dt=tend / n)               # level-0 step tend / n
        Us, _, _, s2 = _run_x(ref, c, 2 * n, False, cfl=0.0, dt=tend / (2 * n))    # every level at the fine step
        assert s1 == 0 and s2 == 0
        errs.append(np.abs(Ux[:, 0] - Us[:, 0]).max() / np.abs(Us[:, 0]).max())
    assert errs[2] < errs[1] < errs[0] and errs[2] < 0.7 * errs[1] and errs[0] < 0.05, errs


def test_crossover_fine_level_sees_the_coarse_state_at_the_start_of_the_step(ref, mech9):
    """"The deepest refinement level is solved first": during its two half steps the fine level's
    coarse-fine ghosts hold level-0 data of time t^n, so the fine result of ONE step depends on the coarse initial data
    only through the two coarse cells under its three ghost layers.  A perturbation of the coarse initial state 5..7
    cells away from the refined patches (within reach of a coarse step: 9 cells) must therefore leave the fine patches
    bitwise unchanged; had level 0 been advanced first, its new state next to the fine patches would differ."""
    nx, ny, tile = 64, 16, 8
    coarse = _random_smooth_2d(mech9, nx, ny, 13, I.BC_REFLECT)
    mask = np.zeros((ny // tile, nx // tile), bool); mask[:, 3] = True              # refine patch column 3: cells 24..31
    base = I.refine_uniform(coarse, (tile, tile), mask)
    pert = I.refine_uniform(coarse, (tile, tile), mask)
    lev, org = base.blocks.level, base.blocks.origin
    for p in np.nonzero(lev == 0)[0]:                                               # coarse columns 37..39 (5..7 cells right of the band)
        if org[p, 0] == 32:
            pert.U[p, :, 0, :, 5:8] *= 0.97                                         # density, momentum, energy, species: a slower, same-T gas
    dt = 2.0e-9
    Ua, _, _, sa = _run_x(ref, base, 1, True, cfl=0.0, dt=dt, chem=False)
    Ub, _, _, sb = _run_x(ref, pert, 1, True, cfl=0.0, dt=dt, chem=False)
    assert sa == 0 and sb == 0
    fine = np.nonzero(lev == 1)[0]
    assert np.array_equal(Ua[fine], Ub[fine])
    # the coarse cells next to the band did feel it (so a coarse-first order would have passed it on)
    near = [p for p in np.nonzero(lev == 0)[0] if org[p, 0] == 32]
    assert max(np.abs(Ua[p, 0, 0, :, 0:2] - Ub[p, 0, 0, :, 0:2]).max() for p in near) > 0


# ----------------------------------------------------------------------------- two-range NASA-7
def test_two_range_identical_sets_equal_single_range(ref, mech9):
    """PAPER.md:247-258 with Cantera-format data: two coefficient sets per species, switched at T_mid.  Both sets equal
    => bitwise the single-range answer (full steps with chemistry)."""
    m2 = I.Mechanism(**{**mech9.__dict__}); m2.nasa_hi = mech9.nasa.copy(); m2.T_mid = np.full(9, 1000.0)
    c1 = I.config1(nx=24, ny=12, mech=mech9); c2 = I.config1(nx=24, ny=12, mech=m2)
    U1, T1, t1, s1 = run(ref, c1, nsteps=3); U2, T2, t2, s2 = run(ref, c2, nsteps=3)
    assert s1 == 0 and s2 == 0 and t1 == t2 and np.array_equal(U1, U2) and np.array_equal(T1, T2)


def test_two_range_temperature_closed_form_per_species_switch(ref):
    """Piecewise-constant c_p with different switch temperatures per species and h continuous at each T_mid:
    e(T) = sum_k Y_k R_k (h_k/R_k - T) is piecewise linear, so T(e) is known in closed form on every piece; the pressure,
    gamma and sound speed must use the coefficient set of the recovered T."""
    W = np.array([0.010, 0.030, 0.020]); Rk = RU / W
    lo = np.zeros((3, 7)); lo[:, 0] = [3.5, 4.0, 2.5]; lo[:, 5] = [-500.0, 2000.0, 100.0]
    hi = lo.copy(); hi[:, 0] = [4.5, 4.75, 2.5]
    Tm = np.array([800.0, 1500.0, 1000.0])
    hi[:, 5] = lo[:, 5] + (lo[:, 0] - hi[:, 0]) * Tm                      # h continuous at T_mid
    z = np.zeros((0, 3), dtype=np.int32)
    m = I.Mechanism(3, 0, W, lo, z, z.copy(), np.zeros(0), np.zeros(0), np.zeros(0), np.zeros(0, dtype=np.int32),
                    np.zeros(0, dtype=np.int32), np.zeros((0, 3)), nasa_hi=hi, T_mid=Tm)
    Y = np.array([0.2, 0.5, 0.3]); rho = 1.7; u = 140.0
    def e_of(T):
        a0 = np.where(T >= Tm, hi[:, 0], lo[:, 0]); a5 = np.where(T >= Tm, hi[:, 5], lo[:, 5])
        return (Y * Rk * ((a0 - 1.0) * T + a5)).sum(), a0
    for T in (500.0, 799.0, 801.0, 1200.0, 1499.9, 1500.1, 2600.0):
        e, a0 = e_of(T)
        Uc = np.array([rho, rho * u, rho * e + 0.5 * rho * u * u, rho * Y[0], rho * Y[1]])
        for guess in (300.0, T, 3000.0):                                  # Newton crosses the kinks from either side
            rc, out = ref.cons2prim(m, 1, Uc, guess)
            assert rc == 0 and abs(out[0] - T) <= 1e-10 * T, (T, guess, out[0])
        cv = (Y * Rk * (a0 - 1.0)).sum(); R = (Y * Rk).sum()
        assert abs(out[2] - (cv + R) / cv) <= 1e-12 and abs(out[1] - rho * R * T) <= 1e-9 * rho * R * T


def test_two_range_equilibrium_constant_uses_the_upper_set_and_is_continuous(ref, mech9):
    """eq 4.9 with two-range data: above T_mid a reversible reaction is in detailed balance at the composition built
    from the UPPER coefficients' Gibbs energies (re-derived here), and K_eq is continuous across T_mid when h and s are
    (inputs.two_range builds such data)."""
    m2 = I.two_range(mech9, 1000.0, 0.6, seed=3)
    T = 1850.0
    a = m2.nasa_hi
    h = a[:, 0] + a[:, 1] / 2 * T + a[:, 5] / T
    s = a[:, 0] * math.log(T) + a[:, 1] * T + a[:, 6]
    g = h - s
    for i in (0, 5, 11, 20):
        dn = (m2.nu_b[i] - m2.nu_f[i]).astype(float)
        lnK = -(dn * g).sum() + dn.sum() * math.log(101325.0 / (RU * T))
        lx = np.log(np.full(9, 2.0) + np.arange(9) * 0.3)
        lx = lx + dn * (lnK - dn @ lx) / (dn @ dn)
        m1 = I.Mechanism(9, 1, m2.W, m2.nasa, m2.nu_f[i:i + 1], m2.nu_b[i:i + 1], m2.A[i:i + 1], m2.b[i:i + 1], m2.Ta[i:i + 1],
                         m2.reversible[i:i + 1], m2.third_body[i:i + 1], m2.eff[i:i + 1], nasa_hi=m2.nasa_hi, T_mid=m2.T_mid)
        X = np.exp(lx)
        q = ref.rates(m1, T, X)[0]
        kf = m2.A[i] * T ** m2.b[i] * math.exp(-m2.Ta[i] / T)
        M = (m2.eff[i] * X).sum() if m2.third_body[i] else 1.0
        fwd = M * kf * np.prod(X ** m2.nu_f[i])
        assert abs(q) <= 1e-10 * fwd, (i, q, fwd)
        # with the LOWER set the same composition is far from balance: the switch matters
        m_lo = I.Mechanism(9, 1, m2.W, m2.nasa, m2.nu_f[i:i + 1], m2.nu_b[i:i + 1], m2.A[i:i + 1], m2.b[i:i + 1], m2.Ta[i:i + 1],
                           m2.reversible[i:i + 1], m2.third_body[i:i + 1], m2.eff[i:i + 1])
        assert abs(ref.rates(m_lo, T, X)[0]) > 1e-4 * fwd
        # continuity of the net rate across T_mid
        X1 = np.full(9, 1.3) + 0.1 * np.arange(9)
        qa, qb = ref.rates(m1, 1000.0 * (1 - 1e-12), X1)[0], ref.rates(m1, 1000.0, X1)[0]
        assert abs(qa - qb) <= 1e-8 * max(abs(qa), abs(qb), 1e-300), (i, qa, qb)


def test_two_range_roundtrip_and_energy_conservation_in_a_step(ref, mech9):
    """prim -> cons (inputs, forward formula) -> prim (oracle, Newton) on two-range data across the switch, and a 0-D
    point-implicit run heating through T_mid keeps rho, E fixed and elements conserved."""
    m2 = I.two_range(mech9, np.linspace(900.0, 1300.0, 9), 0.4, seed=4)
    rng = np.random.default_rng(8)
    for T in (600.0, 950.0, 1100.0, 1299.0, 1301.0, 2400.0):
        Y = rng.dirichlet(np.ones(9)); p = 3.0e5
        U = I.prim_to_cons(m2, 2, np.array([p]), np.array([T]), Y[None], [np.array([50.0]), np.array([-20.0])])[:, 0]
        rc, out = ref.cons2prim(m2, 2, U, 1000.0)
        assert rc == 0 and abs(out[0] - T) <= 1e-10 * T and abs(out[1] - p) <= 1e-9 * p
    m3 = I.two_range(mech9, np.linspace(2002.0, 2012.0, 9), 0.4, seed=5)     # the 0-D case of the pins above: 2000 K -> ~2018 K
    U = I.prim_to_cons(m3, 1, np.array([2.0e6]), np.array([2000.0]), I.hot_Y(9)[None], [np.zeros(1)])
    g = I.Grid(1, (1, 1, 1), (1e-3, 1, 1), (2, 0, 0), (2, 0, 0))
    s = ref.RefSolver(g, m3); s.set_state(U.reshape(1, -1, 1, 1, 1), np.full((1, 1, 1, 1), 2000.0))
    s.step(100, cfl=0.0, dt=2e-9)
    U1, T1 = s.get_state()
    assert s.status == 0 and T1[0, 0, 0, 0] > 2012.5, T1                   # heated through every species' T_mid
    assert np.array_equal(U1[0, :3], U.reshape(1, -1, 1, 1, 1)[0, :3])
    el = np.asarray(m3.elements, dtype=float)
    def moles(Us):
        ry = np.concatenate([Us[0, 3:, 0, 0, 0], [Us[0, 0, 0, 0, 0] - Us[0, 3:, 0, 0, 0].sum()]])
        return (ry / m3.W) @ el
    assert np.abs(moles(U1) - moles(U.reshape(1, -1, 1, 1, 1))).max() <= 1e-12 * np.abs(moles(U1)).max()


# ----------------------------------------------------------------------------- regridding (rest of SURVEY NEXT-1)
def _assemble_level0(case, U, n0, NX, NY):
    """level-0 density as one global array, from the generator's patch origins"""
    npc = case.grid.n[0]
    rho = np.zeros((NY, NX))
    for p in range(n0):
        ox, oy = case.blocks.origin[p]
        rho[oy:oy + npc, ox:ox + npc] = U[p, 0, 0]
    return rho


def _brute_force_flags(rho, thr, nbuf, npc, wall=True):
    """criterion, box dilation and sub-region flags recomputed on the global array (reflecting walls: mirror ghosts)"""
    NY, NX = rho.shape
    pad = np.pad(rho, 1, mode="symmetric" if wall else "wrap")                 # mirror about the wall face / periodic
    gx = np.abs(pad[1:-1, 2:] - pad[1:-1, :-2]) / (2 * rho)
    gy = np.abs(pad[2:, 1:-1] - pad[:-2, 1:-1]) / (2 * rho)
    m = np.maximum(gx, gy) > thr
    for _ in range(nbuf):
        pm = np.pad(m, 1, mode="constant" if wall else "wrap")
        m = np.zeros_like(m)
        for dj in (0, 1, 2):
            for di in (0, 1, 2):
                m |= pm[dj:dj + NY, di:di + NX]
    h = npc // 2
    return m.reshape(NY // h, h, NX // h, h).any(axis=(1, 3))                 # [sub-region row, sub-region column]


def test_regrid_marks_buffers_and_rebuilds_the_block_list(ref, mech9):
    """PAPER.md:73-75, :123, :175-184 (reading B12): the refined sub-regions are exactly those that hold a cell whose
    relative density jump exceeds the threshold or that lies within nbuf cells of one -- recomputed here by brute force
    on the assembled global array --; blocks that existed keep their data bitwise, new ones are the one-to-four
    injection of their parent; neighbour lists follow the geometry; regridding the result changes nothing."""
    pcols, prows, npc = 16, 8, 8
    base = I.config2(nx=pcols * npc, ny=prows * npc)                          # hot driver in the first 8 columns, walls / outflow
    base.grid.bc_hi = (I.BC_REFLECT, I.BC_REFLECT, 0)
    m0 = np.zeros((prows, pcols), bool); m0[:, 0] = True; m0[:, 5] = True      # refined so far: patch columns 0 and 5
    c = I.refine_uniform(base, (npc, npc), m0)
    n0, NX, NY = pcols * prows, pcols * npc, prows * npc
    s = ref.RefSolver(c.grid, c.mech, c.blocks); s.set_state(c.U, c.T)
    s.step(3, cfl=c.cfl)                                                     # a state with fine data that differs from its parents
    U, T = s.get_state()
    for thr, nbuf in ((0.05, 0), (0.05, 2), (0.2, 3), (1e9, 1)):
        lev, nbr, par, Un, Tn = s.regrid(thr, nbuf)
        want = _brute_force_flags(_assemble_level0(c, U, n0, NX, NY), thr, nbuf, npc)
        got = np.zeros_like(want)
        assert (lev[:n0] == 0).all() and (lev[n0:] == 1).all()
        for p in range(n0, len(lev)):
            k, sx, sy = par[p]
            ox, oy = c.blocks.origin[k]
            got[2 * (oy // npc) + sy, 2 * (ox // npc) + sx] = True
        assert np.array_equal(got, want), (thr, nbuf, got.sum(), want.sum())
        assert len(lev) - n0 == want.sum()
        if thr > 1e8:
            assert len(lev) == n0
        # data: level 0 untouched; carried-over blocks bitwise, new blocks injected
        assert np.array_equal(Un[:n0], U[:n0]) and np.array_equal(Tn[:n0], T[:n0])
        old = {tuple(c.blocks.parent[p]): p for p in range(n0, c.grid.n_patches)}
        carried = fresh = 0
        for p in range(n0, len(lev)):
            key = tuple(par[p])
            if key in old:
                assert np.array_equal(Un[p], U[old[key]]) and np.array_equal(Tn[p], T[old[key]]); carried += 1
            else:
                k, sx, sy = par[p]; h = npc // 2
                blk = U[k, :, 0, sy * h:(sy + 1) * h, sx * h:(sx + 1) * h]
                assert np.array_equal(Un[p, :, 0], np.repeat(np.repeat(blk, 2, axis=1), 2, axis=2)); fresh += 1
        if nbuf == 2:
            assert carried > 0 and fresh > 0 and carried < c.grid.n_patches - n0      # some kept, some new, some dropped
        # neighbours from geometry: fine-patch coordinates (fx, fy) -> id
        pos = {}
        for p in range(n0, len(lev)):
            k, sx, sy = par[p]; ox, oy = c.blocks.origin[k]
            pos[(2 * (ox // npc) + sx, 2 * (oy // npc) + sy)] = p
        for (fx, fy), p in pos.items():
            assert nbr[p].tolist() == [pos.get((fx - 1, fy), -1), pos.get((fx + 1, fy), -1), pos.get((fx, fy - 1), -1), pos.get((fx, fy + 1), -1)]
        assert np.array_equal(nbr[:n0], c.blocks.nbr[:n0])
        # idempotent: the regridded list, regridded again with the same parameters, is itself
        if len(lev) > n0:
            g2 = I.Grid(2, c.grid.n, c.grid.dx, c.grid.bc_lo, c.grid.bc_hi, n_patches=len(lev), n_levels=2, ratio=2)
            s2 = ref.RefSolver(g2, c.mech, I.Blocks(lev, nbr, par)); s2.set_state(Un, Tn)
            lev2, nbr2, par2, Un2, Tn2 = s2.regrid(thr, nbuf)
            assert np.array_equal(lev2, lev) and np.array_equal(nbr2, nbr) and np.array_equal(par2, par) and np.array_equal(Un2, Un)


def test_regrid_periodic_buffer_wraps_and_the_new_list_runs(ref, mech9):
    """Buffer cells cross periodic sides (through the neighbour lists of a tiled periodic grid) and stop at nothing else;
    the regridded list is a valid input of the solver."""
    base = _random_smooth_2d(mech9, 64, 32, 17, I.BC_PERIODIC)
    base.U[0, :, 0, :, 60:64] *= 1.6                                         # a density jump next to the periodic seam
    c = I.refine_uniform(base, (8, 8), np.zeros((4, 8), bool))               # no level-1 patches yet
    c.grid.n_levels = 2
    s = ref.RefSolver(c.grid, c.mech, c.blocks); s.set_state(c.U, c.T)
    lev, nbr, par, Un, Tn = s.regrid(0.1, 3)
    want = _brute_force_flags(base.U[0, 0, 0], 0.1, 3, 8, wall=False)
    got = np.zeros_like(want)
    for p in range(32, len(lev)):
        k, sx, sy = par[p]; ox, oy = c.blocks.origin[k]
        got[2 * (oy // 8) + sy, 2 * (ox // 8) + sx] = True
    assert np.array_equal(got, want) and got[:, 0].any() and got[:, -1].any()          # both sides of the seam
    g2 = I.Grid(2, c.grid.n, c.grid.dx, c.grid.bc_lo, c.grid.bc_hi, n_patches=len(lev), n_levels=2, ratio=2)
    s2 = ref.RefSolver(g2, c.mech, I.Blocks(lev, nbr, par)); s2.set_state(Un, Tn)
    s2.step(3, cfl=0.2)
    U3, _ = s2.get_state()
    assert s2.status == 0 and np.isfinite(U3).all()
