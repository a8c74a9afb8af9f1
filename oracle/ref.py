"""ctypes wrapper around oracle/janc_ref.c (the CPU fp64 oracle).

TEST INFRASTRUCTURE ONLY: importable from tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs.  Never imported by paper_2504_13750_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "janc_ref.c")
_LIB = os.path.join(_HERE, "libjanc_ref.so")
_lib = None


def build(force=False):
    """gcc -O2 -ffp-contract=off -fopenmp (no FMA contraction: plain IEEE operations)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                               "-std=c11", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Grid(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("dx", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("n_patches", C.c_int), ("n_levels", C.c_int), ("ratio", C.c_int)]


class _Mech(C.Structure):
    _fields_ = [("ns", C.c_int), ("nr", C.c_int),
                ("W", C.c_void_p), ("nasa", C.c_void_p),
                ("nu_f", C.c_void_p), ("nu_b", C.c_void_p),
                ("A", C.c_void_p), ("b", C.c_void_p), ("Ta", C.c_void_p),
                ("reversible", C.c_void_p), ("third_body", C.c_void_p), ("eff", C.c_void_p),
                ("nasa_hi", C.c_void_p), ("T_mid", C.c_void_p)]


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.jref_weno5.restype = C.c_double
        _lib.jref_last_dt.restype = C.c_double
        _lib.jref_last_dt.argtypes = [C.c_void_p]
        _lib.jref_destroy.argtypes = [C.c_void_p]
        _lib.jref_destroy.restype = None
        if "OMP_NUM_THREADS" not in os.environ:   # cgroup-limited boxes: do not oversubscribe
            _lib.jref_set_threads(len(os.sched_getaffinity(0)))
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


class _MechHolder:
    """Keeps the numpy arrays alive next to the C struct."""

    def __init__(self, mech):
        self.arrs = dict(W=_f64(mech.W), nasa=_f64(mech.nasa), nu_f=_i32(mech.nu_f), nu_b=_i32(mech.nu_b),
                         A=_f64(mech.A), b=_f64(mech.b), Ta=_f64(mech.Ta),
                         reversible=_i32(mech.reversible), third_body=_i32(mech.third_body),
                         eff=_f64(mech.eff))
        two = getattr(mech, "nasa_hi", None) is not None
        if two:
            self.arrs["nasa_hi"] = _f64(mech.nasa_hi); self.arrs["T_mid"] = _f64(mech.T_mid)
        self.c = _Mech(mech.ns, mech.nr, *[_ptr(self.arrs[k]) for k in
                                           ("W", "nasa", "nu_f", "nu_b", "A", "b", "Ta",
                                            "reversible", "third_body", "eff")],
                       _ptr(self.arrs["nasa_hi"]) if two else None, _ptr(self.arrs["T_mid"]) if two else None)


class RefSolver:
    """janc_ref_* context on host memory; same call sequence as the CUDA binding."""

    def __init__(self, grid, mech, blocks=None):
        L = lib()
        g = _Grid(grid.ndim, (C.c_int * 3)(*grid.n), (C.c_double * 3)(*grid.dx),
                  (C.c_int * 3)(*grid.bc_lo), (C.c_int * 3)(*grid.bc_hi),
                  grid.n_patches, grid.n_levels, grid.ratio)
        self._h = C.c_void_p()
        rc = L.jref_create(C.byref(g), C.byref(self._h))
        if rc:
            raise RuntimeError(f"jref_create failed: {rc}")
        self._mh = _MechHolder(mech)
        rc = L.jref_set_mechanism(self._h, C.byref(self._mh.c))
        if rc:
            raise RuntimeError(f"jref_set_mechanism failed: {rc}")
        if blocks is not None:
            rc = L.jref_set_blocks(self._h, _ptr(_i32(blocks.level)), _ptr(_i32(blocks.nbr)),
                                   _ptr(_i32(blocks.parent)))
            if rc:
                raise RuntimeError(f"jref_set_blocks failed: {rc}")
        self.np_ = max(1, grid.n_patches)
        self.ndim = grid.ndim
        self.nvar = grid.ndim + 2 + mech.ns - 1
        self.shape = (self.np_, self.nvar, grid.n[2] if grid.ndim > 2 else 1,
                      grid.n[1] if grid.ndim > 1 else 1, grid.n[0])

    def set_state(self, U, T=None):
        U = _f64(U)
        assert U.size == int(np.prod(self.shape)), (U.shape, self.shape)
        Tp = _ptr(_f64(T)) if T is not None else None
        rc = lib().jref_set_state(self._h, _ptr(U), Tp)
        if rc:
            raise RuntimeError(f"jref_set_state failed: {rc}")

    def step(self, nsteps, cfl=0.0, dt=0.0, chem=True, crossover=False):
        """chem: True point-implicit, False none, "explicit" source inside the RK stages (:351-357);
        crossover: sub-cycled level advance of a two-level block list (Fig 2a)."""
        t = C.c_double(0.0)
        mode = (2 if chem == "explicit" else int(bool(chem))) | (4 if crossover else 0)
        rc = lib().jref_step(self._h, int(nsteps), C.c_double(cfl), C.c_double(dt), mode, C.byref(t))
        self.status = rc
        return t.value

    def last_dt(self):
        return lib().jref_last_dt(self._h)

    def get_state(self):
        U = np.empty(self.shape)
        T = np.empty((self.shape[0],) + self.shape[2:])
        self.status = lib().jref_get_state(self._h, _ptr(U), _ptr(T))
        return U, T

    def debug_ghost_fill(self):
        """Padded U [np, nvar, Pz, Py, Px] and T [np, Pz, Py, Px] right after ghost_fill (pins only)."""
        nd = self.ndim
        pad = lambda n, d: n + 6 if d < nd else 1
        P = (pad(self.shape[2], 2), pad(self.shape[3], 1), pad(self.shape[4], 0))
        U = np.empty((self.np_, self.nvar) + P)
        T = np.empty((self.np_,) + P)
        rc = lib().jref_debug_ghost_fill(self._h, _ptr(U), _ptr(T))
        assert rc == 0, rc
        return U, T

    def regrid(self, thr, nbuf):
        """jref_regrid: (level, nbr, parent, U, T) of the regridded two-level list (level-0 patches first)."""
        n0cap = self.np_ * (1 + (1 << self.ndim))
        nf = 2 * self.ndim
        level = np.zeros(n0cap, np.int32); nbr = np.zeros((n0cap, nf), np.int32); parent = np.zeros((n0cap, 1 + self.ndim), np.int32)
        U = np.zeros((n0cap,) + self.shape[1:]); T = np.zeros((n0cap,) + self.shape[2:])
        n = C.c_int(0)
        rc = lib().jref_regrid(self._h, C.c_double(thr), int(nbuf), C.byref(n), _ptr(level), _ptr(nbr), _ptr(parent), _ptr(U), _ptr(T))
        if rc:
            raise RuntimeError(f"jref_regrid failed: {rc}")
        k = n.value
        return level[:k].copy(), nbr[:k].copy(), parent[:k].copy(), U[:k].copy(), T[:k].copy()

    def close(self):
        if self._h:
            lib().jref_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


# ---- fine-grained entry points used by the pins -------------------------------------------
def weno5(v):
    v = _f64(v)
    assert v.size == 5
    return lib().jref_weno5(_ptr(v))


def cons2prim(mech, ndim, Uc, Tguess):
    mh = _MechHolder(mech)
    out = np.zeros(4)
    rc = lib().jref_cons2prim(C.byref(mh.c), int(ndim), _ptr(_f64(Uc)), C.c_double(Tguess), _ptr(out))
    return rc, out  # T, p, gamma, c


def omega_jac(mech, T, rho, rhoY):
    mh = _MechHolder(mech)
    n1 = mech.ns - 1
    om = np.zeros(max(n1, 1)); J = np.zeros((max(n1, 1), max(n1, 1)))
    lib().jref_omega_jac(C.byref(mh.c), C.c_double(T), C.c_double(rho), _ptr(_f64(rhoY)), _ptr(om), _ptr(J))
    return om, J


def rates(mech, T, X):
    mh = _MechHolder(mech)
    q = np.zeros(max(mech.nr, 1))
    lib().jref_rates(C.byref(mh.c), C.c_double(T), _ptr(_f64(X)), _ptr(q))
    return q[:mech.nr]


def chem_cell(mech, T, rho, rhoY, dt):
    mh = _MechHolder(mech)
    d = np.zeros(max(mech.ns - 1, 1))
    rc = lib().jref_chem_cell(C.byref(mh.c), C.c_double(T), C.c_double(rho), _ptr(_f64(rhoY)), C.c_double(dt), _ptr(d))
    return rc, d


def chem_cells(mech, ndim, Uc, Tguess, dt):
    """Batch of independent cells: Uc [ncell, nvar], Tguess [ncell] -> (rc, delta [ncell, ns-1], T [ncell])."""
    mh = _MechHolder(mech)
    Uc = _f64(Uc); Tg = _f64(Tguess)
    n = Uc.shape[0]
    d = np.zeros((n, max(mech.ns - 1, 1))); T = np.zeros(n)
    fn = lib().jref_chem_cells
    fn.argtypes = [C.c_void_p, C.c_int, C.c_long, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p, C.c_void_p]
    rc = fn(C.byref(mh.c), int(ndim), n, _ptr(Uc), _ptr(Tg), float(dt), _ptr(d), _ptr(T))
    return rc, d, T


def gauss_solve(A, b):
    A = _f64(A).copy(); b = _f64(b).copy()
    rc = lib().jref_gauss_solve(int(b.size), _ptr(A), _ptr(b))
    return rc, b


def threads(n=0):
    """Set (n>0) and return the OpenMP thread count the oracle uses."""
    return lib().jref_set_threads(int(n))
