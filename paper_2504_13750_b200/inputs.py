"""Seeded synthetic inputs: mechanisms, initial conditions and patch layouts.

This module serves BOTH the CUDA path and the CPU oracle (tests hand the same
arrays to each).  It holds no part of the method (no Newton, WENO, RK, rates or
solves): only the random draws and the textbook ideal-gas-mixture formulas
needed to turn a stated (p, T, Y, velocity) into the conserved vector U of
PAPER.md:232 (eq. 4.1-4.2).  The recipe is the one in SURVEY.md §8(d), restated
in DESIGN.md "Synthetic inputs"; it stands in for the paper's H2-O2-N2
detonation tube, whose mechanism/thermo files are not
available here and are not reproduced.
"""
from __future__ import annotations

import itertools
import math
from dataclasses import dataclass, field

import numpy as np

RU = 8.314472  # J/(mol K)
NG = 3         # ghost layers

BC_PERIODIC, BC_REFLECT, BC_OUTFLOW = 0, 1, 2

MECH_SEED_9 = 250413750
MECH_SEED_20 = 250413751


# --------------------------------------------------------------------------
# containers
# --------------------------------------------------------------------------
@dataclass
class Mechanism:
    ns: int
    nr: int
    W: np.ndarray            # [ns] kg/mol
    nasa: np.ndarray         # [ns,7] a0..a6 (eq. 4.3-4.5, single range)
    nu_f: np.ndarray         # [nr,ns] int32
    nu_b: np.ndarray         # [nr,ns] int32
    A: np.ndarray            # [nr] SI (mol, m^3, s)
    b: np.ndarray            # [nr]
    Ta: np.ndarray           # [nr] K  (= Ea/Ru)
    reversible: np.ndarray   # [nr] int32
    third_body: np.ndarray   # [nr] int32
    eff: np.ndarray          # [nr,ns] third-body efficiencies a_ij
    elements: np.ndarray = None   # [ns,ne] atoms of element e in species k (tests only)
    names: list = field(default_factory=list)
    nasa_hi: np.ndarray = None    # [ns,7] upper-range coefficients (two-range NASA-7, as in Cantera / Chemkin data); None: single range
    T_mid: np.ndarray = None      # [ns] switch temperature: T >= T_mid[k] uses nasa_hi[k]


@dataclass
class Grid:
    ndim: int
    n: tuple                 # interior cells per direction (per patch in block mode)
    dx: tuple                # level-0 spacing
    bc_lo: tuple
    bc_hi: tuple
    n_patches: int = 0       # 0 => one uniform grid
    n_levels: int = 1
    ratio: int = 2


@dataclass
class Blocks:
    level: np.ndarray        # [np] int32
    nbr: np.ndarray          # [np, 2*ndim] int32 (lo-x, hi-x, lo-y, hi-y, ...), -1 none
    parent: np.ndarray       # [np, 1+ndim] int32 (parent id, sub-region index per dir), -1 on level 0
    origin: np.ndarray = None  # [np, ndim] global index of the patch's cell (0,..,0) in cells of its OWN level
                               # (layout bookkeeping for tests and regridding; the solver never needs it)


@dataclass
class Case:
    name: str
    grid: Grid
    mech: Mechanism
    U: np.ndarray            # [np|1, nvar, nz, ny, nx] interior only, x fastest
    T: np.ndarray            # [np|1, nz, ny, nx] initial temperature (Newton guess)
    cfl: float
    nsteps: int
    blocks: Blocks = None

    @property
    def nvar(self):
        return self.grid.ndim + 2 + self.mech.ns - 1

    @property
    def cells(self):
        return int(np.prod(self.U.shape) // self.nvar)


# --------------------------------------------------------------------------
# ideal-gas mixture bookkeeping for initial conditions (eq. 4.2-4.4)
# --------------------------------------------------------------------------
def _h_over_R(nasa, T, nasa_hi=None, T_mid=None):
    """h_k/(Ru/W_k) of eq. 4.4 for every species; T array broadcast on the right.  Two-range data: the upper set from
    T_mid[k] upwards."""
    T = np.asarray(T, dtype=np.float64)[..., None]
    def poly(a):
        return (a[:, 0] * T + a[:, 1] / 2 * T**2 + a[:, 2] / 3 * T**3
                + a[:, 3] / 4 * T**4 + a[:, 4] / 5 * T**5 + a[:, 5])
    if nasa_hi is None:
        return poly(nasa)
    return np.where(T >= np.asarray(T_mid), poly(np.asarray(nasa_hi)), poly(nasa))


def prim_to_cons(mech: Mechanism, ndim, p, T, Y, vel):
    """(p, T, Y[..., ns], vel[ndim][...]) -> U[nvar, ...] per PAPER.md:232, eq. 4.2."""
    p = np.asarray(p, dtype=np.float64)
    T = np.asarray(T, dtype=np.float64)
    Y = np.asarray(Y, dtype=np.float64)
    Rk = RU / mech.W
    R = (Y * Rk).sum(-1)
    rho = p / (R * T)
    h = (Y * Rk * _h_over_R(mech.nasa, T, getattr(mech, "nasa_hi", None), getattr(mech, "T_mid", None))).sum(-1)
    ke = np.zeros_like(rho)
    for d in range(ndim):
        ke = ke + 0.5 * vel[d] ** 2
    E = rho * h - p + rho * ke
    comps = [rho] + [rho * vel[d] for d in range(ndim)] + [E]
    comps += [rho * Y[..., k] for k in range(mech.ns - 1)]
    return np.stack(comps, axis=0)


# --------------------------------------------------------------------------
# mechanisms
# --------------------------------------------------------------------------
def single_step_mechanism(q=2.0e6, A=1.0e9, Ta=15000.0, W=0.029, gamma=1.4):
    """Config 0: reactant R -> product P, irreversible Arrhenius (BASELINE.json configs[0]).

    Species order: R (carried as rho*Y_1), P (by difference)."""
    a0 = gamma / (gamma - 1.0)
    Rk = RU / W
    nasa = np.zeros((2, 7))
    nasa[:, 0] = a0
    nasa[0, 5] = q / Rk
    return Mechanism(
        ns=2, nr=1, W=np.array([W, W]), nasa=nasa,
        nu_f=np.array([[1, 0]], dtype=np.int32), nu_b=np.array([[0, 1]], dtype=np.int32),
        A=np.array([A]), b=np.array([0.0]), Ta=np.array([Ta]),
        reversible=np.array([0], dtype=np.int32), third_body=np.array([0], dtype=np.int32),
        eff=np.ones((1, 2)), elements=np.array([[1], [1]], dtype=np.int64),
        names=["R", "P"])


def inert_gas(gamma=1.4, R=287.0):
    """Ns=1, Nr=0 ideal gas (Sod tube)."""
    nasa = np.zeros((1, 7))
    nasa[0, 0] = gamma / (gamma - 1.0)
    z = np.zeros((0, 1), dtype=np.int32)
    return Mechanism(ns=1, nr=0, W=np.array([RU / R]), nasa=nasa, nu_f=z, nu_b=z.copy(),
                     A=np.zeros(0), b=np.zeros(0), Ta=np.zeros(0),
                     reversible=np.zeros(0, dtype=np.int32), third_body=np.zeros(0, dtype=np.int32),
                     eff=np.zeros((0, 1)), elements=np.array([[1]], dtype=np.int64), names=["air"])


def _species_set(ns):
    """Composition vectors; returns (comps [ns,ne], element weights, bond energies D_e)."""
    if ns == 9:
        ew = np.array([0.002, 0.016, 0.014])          # a, b, n
        D = np.array([2.18e5, 2.49e5, 0.0])
        fuel, oxid, inert = (2, 0, 0), (0, 2, 0), (0, 0, 2)
        others = [(i, j, 0) for i in range(3) for j in range(3)
                  if (i, j) != (0, 0) and (i, j, 0) not in (fuel, oxid)]
        n_other = 6
    elif ns == 20:
        ew = np.array([0.002, 0.016, 0.012, 0.014])   # a, b, c, n
        D = np.array([2.18e5, 2.49e5, 3.5e5, 0.0])
        fuel, oxid, inert = (2, 0, 0, 0), (0, 2, 0, 0), (0, 0, 0, 2)
        others = []
        for i in range(5):
            for j in range(3):
                for k in range(3):
                    atoms = i + j + k
                    w = 0.002 * i + 0.016 * j + 0.012 * k
                    if 1 <= atoms <= 5 and 0.002 - 1e-12 <= w <= 0.04 + 1e-12:
                        c = (i, j, k, 0)
                        if c not in (fuel, oxid):
                            others.append(c)
        n_other = 17
    else:
        raise ValueError("synthetic mechanisms exist for ns=9 and ns=20")
    others.sort(key=lambda c: (sum(c),) + tuple(-x for x in c))
    comps = [fuel, oxid] + others[:n_other] + [inert]
    return np.array(comps, dtype=np.int64), ew, D


def _candidates(comps):
    """Element-balanced A+B<=>C+D and A(+M)<=>B+C(+M) over the non-inert species."""
    n = comps.shape[0] - 1  # last is inert
    pairs = [(i, j) for i in range(n) for j in range(i, n)]
    cands = []
    for (a, b), (c, d) in itertools.combinations(pairs, 2):
        if np.array_equal(comps[a] + comps[b], comps[c] + comps[d]):
            cands.append(((a, b), (c, d), 0))
    for a in range(n):
        for (b, c) in pairs:
            if np.array_equal(comps[a], comps[b] + comps[c]):
                cands.append(((a,), (b, c), 1))
    return cands


def synthetic_mechanism(ns=9, nr=21, seed=None):
    """Seeded element-balanced mechanism, SURVEY.md §8(d) recipe."""
    if seed is None:
        seed = MECH_SEED_9 if ns == 9 else MECH_SEED_20
    rng = np.random.default_rng(seed)
    comps, ew, D = _species_set(ns)
    atoms = comps.sum(1)
    W = comps @ ew
    # thermo: constant cp
    nasa = np.zeros((ns, 7))
    Hf = np.zeros(ns)
    for k in range(ns):
        a0 = 2.5 + (atoms[k] - 1) + rng.uniform(-0.25, 0.25)
        cp = min(max(a0 * RU / W[k], 900.0), 15000.0)
        a0 = cp * W[k] / RU
        bond = rng.uniform(4.0e5, 5.0e5)
        Hf[k] = float(comps[k] @ D) - (atoms[k] - 1) * bond
        if k in (0, 1, ns - 1):
            Hf[k] = 0.0
        nasa[k, 0] = a0
        nasa[k, 5] = Hf[k] / RU - 298.15 * a0
        nasa[k, 6] = 1.5 * math.log(W[k] / 0.002) + rng.uniform(-1.0, 1.0)
    # reactions
    cands = _candidates(comps)
    perm = rng.permutation(len(cands))
    chosen, covered = [], set()
    for idx in perm:
        lhs, rhs, tb = cands[idx]
        sp = set(lhs) | set(rhs)
        if not sp <= covered:
            chosen.append(idx)
            covered |= sp
        if len(chosen) == nr:
            break
    for idx in perm:
        if len(chosen) == nr:
            break
        if idx not in chosen:
            chosen.append(idx)
    if len(chosen) < nr:
        raise ValueError("not enough balanced candidate reactions")
    nu_f = np.zeros((nr, ns), dtype=np.int32)
    nu_b = np.zeros((nr, ns), dtype=np.int32)
    A = np.zeros(nr); bb = np.zeros(nr); Ta = np.zeros(nr)
    third = np.zeros(nr, dtype=np.int32)
    eff = np.ones((nr, ns))
    for i, idx in enumerate(chosen):
        lhs, rhs, tb = cands[idx]
        if sum(Hf[list(rhs)]) > sum(Hf[list(lhs)]):     # write in the exothermic direction
            lhs, rhs = rhs, lhs
        for s in lhs:
            nu_f[i, s] += 1
        for s in rhs:
            nu_b[i, s] += 1
        third[i] = tb
        bb[i] = rng.uniform(-1.0, 1.0)
        Ta[i] = rng.uniform(0.0, 2.0e4)
        if set(lhs) <= {0, 1} or set(rhs) <= {0, 1}:
            Ta[i] = 2.0e4
        kref = 10.0 ** rng.uniform(8.0, 13.0)
        A_cgs = min(max(kref * 2000.0 ** (-bb[i]) * math.exp(Ta[i] / 2000.0), 1e8), 1e14)
        order = len(lhs) + tb
        A[i] = A_cgs * (1e-6) ** (order - 1)
        eff[i, :] = rng.uniform(0.5, 3.0, size=ns)
    names = ["".join(f"{e}{c}" for e, c in zip("abcn"[:comps.shape[1] - 1] + "n", row) if c)
             for row in comps]
    return Mechanism(ns=ns, nr=nr, W=W, nasa=nasa, nu_f=nu_f, nu_b=nu_b, A=A, b=bb, Ta=Ta,
                     reversible=np.ones(nr, dtype=np.int32), third_body=third, eff=eff,
                     elements=comps, names=names)


def ambient_Y(ns):
    Y = np.zeros(ns)
    Y[0], Y[1], Y[ns - 1] = 0.028, 0.226, 0.746
    return Y


def hot_Y(ns):
    Y = ambient_Y(ns)
    Y[2:ns - 1] = 0.01                               # radical pool taken from the inert share
    Y[ns - 1] -= 0.01 * (ns - 3)
    return Y


# --------------------------------------------------------------------------
# configurations (BASELINE.json configs[0..4]); sizes can be scaled down for parity tests
# --------------------------------------------------------------------------
def config0(n=512, seed=1000, nsteps=200):
    mech = single_step_mechanism()
    rng = np.random.default_rng(seed)
    x = np.arange(n)
    left = x < n // 2
    p = np.where(left, 1.0e6, 1.0e5)
    T = np.where(left, 1500.0, 300.0) * (1.0 + 0.01 * rng.uniform(-1.0, 1.0, size=n))
    Y = np.zeros((n, 2))
    Y[:, 0] = np.where(left, 0.0, 1.0)
    Y[:, 1] = 1.0 - Y[:, 0]
    U = prim_to_cons(mech, 1, p, T, Y, [np.zeros(n)])
    g = Grid(1, (n, 1, 1), (1e-4, 1.0, 1.0), (BC_OUTFLOW, 0, 0), (BC_OUTFLOW, 0, 0))
    return Case("cfg0_1d_shock_tube", g, mech, U.reshape(1, 4, 1, 1, n), T.reshape(1, 1, 1, n), 0.4, nsteps)


def _channel(name, nx, ny, ndrv, seed, bc_lo, bc_hi, nsteps, mech=None):
    mech = mech or synthetic_mechanism(9, 21)
    ns = mech.ns
    rng = np.random.default_rng(seed)
    ii = np.arange(nx)[None, :] + np.zeros((ny, 1), dtype=np.int64)
    hot = ii < ndrv
    T = np.where(hot, 3000.0, 300.0)
    p = np.where(hot, 3.0e6, 1.0e5) * (1.0 + 0.02 * rng.uniform(-1.0, 1.0, size=(ny, nx)))
    Y = np.where(hot[..., None], hot_Y(ns), ambient_Y(ns))
    z = np.zeros((ny, nx))
    U = prim_to_cons(mech, 2, p, T, Y, [z, z])
    g = Grid(2, (nx, ny, 1), (5e-5, 5e-5, 1.0), bc_lo, bc_hi)
    return Case(name, g, mech, U.reshape(1, -1, 1, ny, nx), T.reshape(1, 1, ny, nx).copy(), 0.2, nsteps)


def config1(nx=1024, ny=128, seed=1001, nsteps=100, mech=None):
    r = (BC_REFLECT, BC_REFLECT, 0)
    return _channel("cfg1_2d_channel_1024x128", nx, ny, max(1, nx // 16), seed, r, r, nsteps, mech)


def config2(nx=4096, ny=512, seed=1002, nsteps=100, mech=None):
    return _channel("cfg2_2d_channel_4096x512", nx, ny, max(1, nx // 16), seed,
                    (BC_REFLECT, BC_REFLECT, 0), (BC_OUTFLOW, BC_REFLECT, 0), nsteps, mech)


def config3(pcols=128, prows=32, npc=16, seed=1003, nsteps=50, mech=None):
    """Two-level block list: level 0 = pcols x prows patches of npc x npc; a band of
    level-0 patches around a wavy front is refined 2x2."""
    mech = mech or synthetic_mechanism(9, 21)
    ns = mech.ns
    rng = np.random.default_rng(seed)
    phi = rng.uniform(0.0, 2.0 * math.pi)
    jit = rng.integers(-2, 3, size=prows)
    half = max(1, pcols // 8)
    xf = np.array([int(round(0.375 * pcols + (pcols / 16.0) * math.sin(2 * math.pi * r / prows + phi)))
                   for r in range(prows)]) + jit
    xf = np.clip(xf, half, pcols - half)
    n0 = pcols * prows
    refined = np.zeros((prows, pcols), dtype=bool)
    for r in range(prows):
        refined[r, xf[r] - half: xf[r] + half] = True
    # level-0 fields on the assembled grid
    NX, NY = pcols * npc, prows * npc
    rows = np.arange(NY) // npc
    front_cell = (xf[rows] * npc)[:, None]
    ii = np.arange(NX)[None, :]
    hot = ii < front_cell
    T0 = np.where(hot, 3000.0, 300.0)
    p0 = np.where(hot, 3.0e6, 1.0e5) * (1.0 + 0.02 * rng.uniform(-1.0, 1.0, size=(NY, NX)))
    Y0 = np.where(hot[..., None], hot_Y(ns), ambient_Y(ns))
    z = np.zeros((NY, NX))
    Ug = prim_to_cons(mech, 2, p0, T0, Y0, [z, z])          # [nvar, NY, NX]
    nvar = Ug.shape[0]
    # patch lists
    fine_id = -np.ones((prows, pcols, 2, 2), dtype=np.int64)   # [r, c, sy, sx]
    nxt = n0
    for r in range(prows):
        for c in range(pcols):
            if refined[r, c]:
                for sy in range(2):
                    for sx in range(2):
                        fine_id[r, c, sy, sx] = nxt
                        nxt += 1
    npatch = nxt
    level = np.zeros(npatch, dtype=np.int32)
    nbr = -np.ones((npatch, 4), dtype=np.int32)
    parent = -np.ones((npatch, 3), dtype=np.int32)
    origin = np.zeros((npatch, 2), dtype=np.int64)
    U = np.zeros((npatch, nvar, 1, npc, npc))
    T = np.zeros((npatch, 1, npc, npc))
    for r in range(prows):
        for c in range(pcols):
            k = r * pcols + c
            origin[k] = [c * npc, r * npc]
            nbr[k] = [k - 1 if c > 0 else -1, k + 1 if c < pcols - 1 else -1,
                      k - pcols if r > 0 else -1, k + pcols if r < prows - 1 else -1]
            U[k, :, 0] = Ug[:, r * npc:(r + 1) * npc, c * npc:(c + 1) * npc]
            T[k, 0] = T0[r * npc:(r + 1) * npc, c * npc:(c + 1) * npc]

    def fid(fy, fx):      # fine patch id from fine-patch coordinates, -1 if absent/outside
        if fy < 0 or fx < 0 or fy >= 2 * prows or fx >= 2 * pcols:
            return -1
        return int(fine_id[fy // 2, fx // 2, fy % 2, fx % 2])

    for r in range(prows):
        for c in range(pcols):
            for sy in range(2):
                for sx in range(2):
                    f = fine_id[r, c, sy, sx]
                    if f < 0:
                        continue
                    level[f] = 1
                    parent[f] = [r * pcols + c, sx, sy]
                    fy, fx = 2 * r + sy, 2 * c + sx
                    origin[f] = [fx * npc, fy * npc]
                    nbr[f] = [fid(fy, fx - 1), fid(fy, fx + 1), fid(fy - 1, fx), fid(fy + 1, fx)]
                    h = npc // 2
                    y0, x0 = r * npc + sy * h, c * npc + sx * h
                    sub = Ug[:, y0:y0 + h, x0:x0 + h]
                    U[f, :, 0] = np.repeat(np.repeat(sub, 2, axis=1), 2, axis=2)   # one-to-four
                    T[f, 0] = np.repeat(np.repeat(T0[y0:y0 + h, x0:x0 + h], 2, axis=0), 2, axis=1)
    r_ = (BC_REFLECT, BC_REFLECT, 0)
    g = Grid(2, (npc, npc, 1), (1e-4, 1e-4, 1.0), r_, r_, n_patches=npatch, n_levels=2, ratio=2)
    return Case(f"cfg3_amr_{npatch}x{npc}x{npc}", g, mech, U, T, 0.2, nsteps,
                blocks=Blocks(level, nbr, parent, origin))


def config4(n=256, nspheres=50, radius=8, seed=1004, nsteps=20, mech=None):
    mech = mech or synthetic_mechanism(20, 100)
    ns = mech.ns
    rng = np.random.default_rng(seed)
    centres = rng.uniform(0.0, n, size=(nspheres, 3))
    ax = np.arange(n) + 0.5
    hot = np.zeros((n, n, n), dtype=bool)               # [z, y, x]
    for cx, cy, cz in centres:
        dxp = np.abs(ax - cx); dxp = np.minimum(dxp, n - dxp)
        dyp = np.abs(ax - cy); dyp = np.minimum(dyp, n - dyp)
        dzp = np.abs(ax - cz); dzp = np.minimum(dzp, n - dzp)
        hot |= (dzp[:, None, None] ** 2 + dyp[None, :, None] ** 2 + dxp[None, None, :] ** 2) <= radius ** 2
    T = np.where(hot, 2500.0, 300.0)
    Ya, Yh = ambient_Y(ns), hot_Y(ns)
    # two distinct states only: build them once, then scatter (keeps 256^3 x 24 cheap)
    z1 = np.zeros(1)
    Ua = prim_to_cons(mech, 3, np.array([1e5]), np.array([300.0]), Ya[None, :], [z1, z1, z1])[:, 0]
    Uh = prim_to_cons(mech, 3, np.array([1e5]), np.array([2500.0]), Yh[None, :], [z1, z1, z1])[:, 0]
    nvar = Ua.shape[0]
    U = np.empty((1, nvar, n, n, n))
    for m in range(nvar):
        U[0, m] = np.where(hot, Uh[m], Ua[m])
    p3 = (BC_PERIODIC,) * 3
    g = Grid(3, (n, n, n), (5e-5,) * 3, p3, p3)
    return Case(f"cfg4_3d_{n}cubed", g, mech, U, T.reshape(1, n, n, n).astype(np.float64), 0.2, nsteps)


def tile_uniform(case: Case, tx, ty):
    """Re-express a 2-D uniform-grid case as an all-level-0 block list of tx x ty patches
    (pin: patch tiling == single grid).  Physical BCs stay on outer faces;
    periodic sides become wrap-around neighbour links."""
    g = case.grid
    assert g.ndim == 2 and g.n_patches == 0
    nx, ny = g.n[0], g.n[1]
    assert nx % tx == 0 and ny % ty == 0
    px, py = nx // tx, ny // ty
    npatch = px * py
    nvar = case.nvar
    U = np.zeros((npatch, nvar, 1, ty, tx)); T = np.zeros((npatch, 1, ty, tx))
    nbr = -np.ones((npatch, 4), dtype=np.int32)
    per_x = g.bc_lo[0] == BC_PERIODIC
    per_y = g.bc_lo[1] == BC_PERIODIC
    for r in range(py):
        for c in range(px):
            k = r * px + c
            U[k, :, 0] = case.U[0, :, 0, r * ty:(r + 1) * ty, c * tx:(c + 1) * tx]
            T[k, 0] = case.T[0, 0, r * ty:(r + 1) * ty, c * tx:(c + 1) * tx]
            lo_x = k - 1 if c > 0 else (k + px - 1 if per_x else -1)
            hi_x = k + 1 if c < px - 1 else (k - px + 1 if per_x else -1)
            lo_y = k - px if r > 0 else (k + px * (py - 1) if per_y else -1)
            hi_y = k + px if r < py - 1 else (k - px * (py - 1) if per_y else -1)
            nbr[k] = [lo_x, hi_x, lo_y, hi_y]
    g2 = Grid(2, (tx, ty, 1), g.dx, g.bc_lo, g.bc_hi, n_patches=npatch, n_levels=1, ratio=2)
    blocks = Blocks(np.zeros(npatch, dtype=np.int32), nbr, -np.ones((npatch, 3), dtype=np.int32))
    return Case(case.name + "_tiled", g2, case.mech, U, T, case.cfl, case.nsteps, blocks=blocks)


def untile(case_tiled: Case, U, px, py):
    """Inverse of tile_uniform for a state array U[np, nvar, 1, ty, tx] -> [1, nvar, 1, ny, nx]."""
    npatch, nvar, _, ty, tx = U.shape
    out = np.zeros((1, nvar, 1, py * ty, px * tx))
    for r in range(py):
        for c in range(px):
            out[0, :, 0, r * ty:(r + 1) * ty, c * tx:(c + 1) * tx] = U[r * px + c, :, 0]
    return out


def refine_uniform(case: Case, tile, refine):
    """Re-express a uniform-grid case (ndim 1, 2 or 3) as a two-level block list: the grid is cut into level-0
    patches of `tile` cells and every patch with refine[pz, py, px] True gets 2^ndim level-1 children (its fixed
    sub-regions) holding the one-to-four injection of its data.  Periodic sides
    become wrap-around neighbour links on both levels.  Patch order: level 0 x-fastest, then the children of each
    refined patch, sub-region x-fastest."""
    g = case.grid
    nd = g.ndim
    assert g.n_patches == 0
    n = [g.n[d] if d < nd else 1 for d in range(3)]
    t = [tile[d] if d < nd else 1 for d in range(3)]
    assert all(n[d] % t[d] == 0 and (t[d] % 2 == 0 or d >= nd) for d in range(3))
    pc = [n[d] // t[d] for d in range(3)]
    refine = np.asarray(refine, dtype=bool).reshape(pc[2], pc[1], pc[0])
    per = [d < nd and g.bc_lo[d] == BC_PERIODIC for d in range(3)]
    n0 = pc[0] * pc[1] * pc[2]
    sub = [2 if d < nd else 1 for d in range(3)]
    fine_id = -np.ones((pc[2], pc[1], pc[0], sub[2], sub[1], sub[0]), dtype=np.int64)
    nxt = n0
    for z, y, x in itertools.product(range(pc[2]), range(pc[1]), range(pc[0])):
        if refine[z, y, x]:
            for sz, sy, sx in itertools.product(range(sub[2]), range(sub[1]), range(sub[0])):
                fine_id[z, y, x, sz, sy, sx] = nxt
                nxt += 1
    npatch = nxt
    nvar = case.nvar
    level = np.zeros(npatch, dtype=np.int32)
    nbr = -np.ones((npatch, 2 * nd), dtype=np.int32)
    parent = -np.ones((npatch, 1 + nd), dtype=np.int32)
    origin = np.zeros((npatch, nd), dtype=np.int64)
    U = np.zeros((npatch, nvar, t[2], t[1], t[0]))
    T = np.zeros((npatch, t[2], t[1], t[0]))

    def wrap(c, cnt):
        """patch coordinates -> wrapped coordinates or None when outside a non-periodic side"""
        out = []
        for d in range(3):
            v = c[d]
            if v < 0 or v >= cnt[d]:
                if not per[d]:
                    return None
                v %= cnt[d]
            out.append(v)
        return out

    for z, y, x in itertools.product(range(pc[2]), range(pc[1]), range(pc[0])):
        k = (z * pc[1] + y) * pc[0] + x
        c = [x, y, z]
        origin[k] = [c[d] * t[d] for d in range(nd)]
        for d in range(nd):
            for side in (0, 1):
                cc = list(c); cc[d] += 2 * side - 1
                w = wrap(cc, pc)
                nbr[k, 2 * d + side] = -1 if w is None else (w[2] * pc[1] + w[1]) * pc[0] + w[0]
        sl = (slice(z * t[2], (z + 1) * t[2]), slice(y * t[1], (y + 1) * t[1]), slice(x * t[0], (x + 1) * t[0]))
        U[k] = case.U[0][(slice(None),) + sl]
        T[k] = case.T[0][sl]
    fcnt = [pc[d] * sub[d] for d in range(3)]
    for z, y, x in itertools.product(range(pc[2]), range(pc[1]), range(pc[0])):
        if not refine[z, y, x]:
            continue
        k = (z * pc[1] + y) * pc[0] + x
        for sz, sy, sx in itertools.product(range(sub[2]), range(sub[1]), range(sub[0])):
            f = fine_id[z, y, x, sz, sy, sx]
            s3 = [sx, sy, sz]
            fc = [2 * x + sx if nd > 0 else 0, (2 * y + sy) if nd > 1 else 0, (2 * z + sz) if nd > 2 else 0]
            level[f] = 1
            parent[f] = [k] + s3[:nd]
            origin[f] = [fc[d] * t[d] for d in range(nd)]
            for d in range(nd):
                for side in (0, 1):
                    cc = list(fc); cc[d] += 2 * side - 1
                    w = wrap(cc, fcnt)
                    if w is not None:
                        nbr[f, 2 * d + side] = fine_id[w[2] // sub[2], w[1] // sub[1], w[0] // sub[0],
                                                       w[2] % sub[2], w[1] % sub[1], w[0] % sub[0]]
            h = [t[d] // sub[d] for d in range(3)]
            sl = tuple(slice(s3[d] * h[d], (s3[d] + 1) * h[d]) for d in (2, 1, 0))
            blockU = U[k][(slice(None),) + sl]
            blockT = T[k][sl]
            for ax, d in ((1, 2), (2, 1), (3, 0)):
                blockU = np.repeat(blockU, sub[d], axis=ax)
                blockT = np.repeat(blockT, sub[d], axis=ax - 1)
            U[f] = blockU
            T[f] = blockT
    g2 = Grid(nd, tuple(t), g.dx, g.bc_lo, g.bc_hi, n_patches=npatch, n_levels=2, ratio=2)
    return Case(case.name + "_2lev", g2, case.mech, U, T, case.cfl, case.nsteps,
                blocks=Blocks(level, nbr, parent, origin))


def two_range(mech: Mechanism, T_mid, dcp, seed=0):
    """A two-range version of a single-range mechanism: above T_mid[k] species k has c_p/R = a0 + dcp[k] + a1' T with
    a seeded small slope, and a5', a6' chosen so that h_k and s_k are continuous at T_mid[k] (what fitted NASA data
    satisfy to their fitting accuracy).  Stands in for Cantera-format thermo data."""
    rng = np.random.default_rng(seed)
    T_mid = np.broadcast_to(np.asarray(T_mid, dtype=np.float64), (mech.ns,)).copy()
    lo = mech.nasa
    hi = lo.copy()
    hi[:, 0] = lo[:, 0] + np.broadcast_to(dcp, (mech.ns,))
    hi[:, 1] = lo[:, 1] + rng.uniform(1e-5, 2e-4, size=mech.ns)
    Tm = T_mid
    def h(a): return a[:, 0] * Tm + a[:, 1] / 2 * Tm**2 + a[:, 2] / 3 * Tm**3 + a[:, 3] / 4 * Tm**4 + a[:, 4] / 5 * Tm**5
    def s(a): return a[:, 0] * np.log(Tm) + a[:, 1] * Tm + a[:, 2] / 2 * Tm**2 + a[:, 3] / 3 * Tm**3 + a[:, 4] / 4 * Tm**4
    hi[:, 5] = lo[:, 5] + h(lo) - h(hi)
    hi[:, 6] = lo[:, 6] + s(lo) - s(hi)
    out = Mechanism(**{**mech.__dict__})
    out.nasa_hi, out.T_mid = hi, T_mid
    return out
