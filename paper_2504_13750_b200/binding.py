"""Thin ctypes binding of libjanc.so (include/janc.h): argument marshalling only.

PyTorch supplies device memory (the workspace, device-resident state tensors) and the CUDA
stream; every step of the path runs in the library's kernels.  There is no CPU fallback: if the
library is missing, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libjanc.so")
_lib = None

JANC_OK, JANC_EINVAL, JANC_ENOMEM, JANC_ECUDA, JANC_ESTATE, JANC_ENONFINITE = 0, -1, -2, -3, -4, -5
FLAG_NO_CHEM = 1
FLAG_EXPLICIT_SOURCE = 2
FLAG_CROSSOVER = 4
PART_PRIM, PART_DT, PART_GHOST, PART_FLUX, PART_SOURCE = range(5)
BC_EXCHANGE = 3

EXPORTS = ["janc_mech_parse", "janc_mech_file_view", "janc_mech_file_species", "janc_mech_file_free",
           "janc_create", "janc_set_option", "janc_set_mechanism", "janc_workspace_bytes", "janc_bind_workspace",
           "janc_set_blocks", "janc_set_state", "janc_step", "janc_step_part", "janc_halo_doubles", "janc_halo",
           "janc_reduction_slots", "janc_last_dt", "janc_regrid_plan", "janc_regrid_fill", "janc_cfl_dt_static", "janc_get_state",
           "janc_status",
           "janc_launch_count", "janc_debug_cons2prim", "janc_profile_step",
           "janc_measure_dfma_peak", "janc_chem_kernel", "janc_jit_log", "janc_jit_probe",
           "janc_last_error", "janc_destroy"]


class JancError(RuntimeError):
    def __init__(self, code, msg=""):
        super().__init__(f"libjanc error {code}: {msg}")
        self.code = code


class _Grid(C.Structure):
    _fields_ = [("ndim", C.c_int), ("n", C.c_int * 3), ("dx", C.c_double * 3),
                ("bc_lo", C.c_int * 3), ("bc_hi", C.c_int * 3),
                ("n_patches", C.c_int), ("n_levels", C.c_int), ("ratio", C.c_int)]


class _Mech(C.Structure):
    _fields_ = [("ns", C.c_int), ("nr", C.c_int),
                ("W", C.c_void_p), ("nasa", C.c_void_p), ("nu_f", C.c_void_p), ("nu_b", C.c_void_p),
                ("A", C.c_void_p), ("b", C.c_void_p), ("Ta", C.c_void_p),
                ("reversible", C.c_void_p), ("third_body", C.c_void_p), ("eff", C.c_void_p),
                ("nasa_hi", C.c_void_p), ("T_mid", C.c_void_p)]


def lib():
    """Load libjanc.so (built in-tree by paper_2504_13750_b200.build); fail loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not built: run `python -m paper_2504_13750_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.janc_workspace_bytes.restype = C.c_size_t
        L.janc_workspace_bytes.argtypes = [C.c_void_p]
        L.janc_bind_workspace.argtypes = [C.c_void_p, C.c_void_p, C.c_size_t]
        L.janc_create.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p]
        L.janc_set_mechanism.argtypes = [C.c_void_p, C.c_void_p]
        L.janc_set_option.argtypes = [C.c_void_p, C.c_char_p, C.c_char_p]
        L.janc_set_blocks.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.janc_set_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.janc_step.argtypes = [C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int, C.c_void_p]
        L.janc_get_state.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.janc_step_part.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_int]
        L.janc_halo_doubles.argtypes = [C.c_void_p]
        L.janc_halo_doubles.restype = C.c_size_t
        L.janc_halo.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_int]
        L.janc_reduction_slots.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p]
        L.janc_last_dt.argtypes = [C.c_void_p, C.c_void_p]
        L.janc_regrid_plan.argtypes = [C.c_void_p, C.c_double, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
        L.janc_regrid_fill.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.janc_cfl_dt_static.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_void_p]
        L.janc_status.argtypes = [C.c_void_p]
        L.janc_launch_count.argtypes = [C.c_void_p]
        L.janc_launch_count.restype = C.c_longlong
        L.janc_debug_cons2prim.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]
        L.janc_profile_step.argtypes = [C.c_void_p, C.c_double, C.c_double, C.c_void_p, C.c_void_p]
        L.janc_measure_dfma_peak.argtypes = [C.c_int, C.c_void_p, C.c_void_p]
        L.janc_last_error.argtypes = [C.c_void_p]
        L.janc_last_error.restype = C.c_char_p
        L.janc_chem_kernel.argtypes = [C.c_void_p]
        L.janc_chem_kernel.restype = C.c_char_p
        L.janc_jit_log.argtypes = [C.c_void_p]
        L.janc_jit_log.restype = C.c_char_p
        L.janc_jit_probe.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p]
        L.janc_mech_parse.argtypes = [C.c_char_p, C.c_char_p, C.c_void_p, C.c_char_p, C.c_size_t]
        L.janc_mech_file_view.argtypes = [C.c_void_p, C.c_void_p]
        L.janc_mech_file_species.argtypes = [C.c_void_p, C.c_int]
        L.janc_mech_file_species.restype = C.c_char_p
        L.janc_mech_file_free.argtypes = [C.c_void_p]
        L.janc_mech_file_free.restype = None
        L.janc_destroy.argtypes = [C.c_void_p]
        L.janc_destroy.restype = None
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def _mech_struct(mech):
    keep = dict(W=_f64(mech.W), nasa=_f64(mech.nasa), nu_f=_i32(mech.nu_f), nu_b=_i32(mech.nu_b),
                A=_f64(mech.A), b=_f64(mech.b), Ta=_f64(mech.Ta), reversible=_i32(mech.reversible),
                third_body=_i32(mech.third_body), eff=_f64(mech.eff))
    two = getattr(mech, "nasa_hi", None) is not None
    if two:
        keep["nasa_hi"] = _f64(mech.nasa_hi); keep["T_mid"] = _f64(mech.T_mid)
    m = _Mech(mech.ns, mech.nr, *[_ptr(keep[k]) for k in
                                  ("W", "nasa", "nu_f", "nu_b", "A", "b", "Ta", "reversible", "third_body", "eff")],
              _ptr(keep["nasa_hi"]) if two else None, _ptr(keep["T_mid"]) if two else None)
    return m, keep


def jit_probe(mech, ndim, compile=True):
    """janc_jit_probe: (specialised CUDA source, cubin size or None).  Needs no GPU."""
    m, keep = _mech_struct(mech)
    n = C.c_size_t(0)
    rc = lib().janc_jit_probe(C.byref(m), int(ndim), None, 0, C.byref(n), None)
    if rc:
        raise JancError(rc, "janc_jit_probe")
    buf = C.create_string_buffer(n.value + 1)
    nb = C.c_size_t(0)
    rc = lib().janc_jit_probe(C.byref(m), int(ndim), buf, n.value + 1, None, C.byref(nb) if compile else None)
    if rc:
        raise JancError(rc, "janc_jit_probe (NVRTC)")
    return buf.value.decode(), (nb.value if compile else None)


def load_chemkin(mech_text, thermo_text=None):
    """janc_mech_parse: Chemkin-format text(s) -> inputs.Mechanism (SI units, two-range NASA-7).  Needs no GPU."""
    from . import inputs
    h = C.c_void_p()
    err = C.create_string_buffer(512)
    rc = lib().janc_mech_parse(mech_text.encode(), thermo_text.encode() if thermo_text else None, C.byref(h), err, 512)
    if rc:
        raise JancError(rc, "janc_mech_parse: " + err.value.decode())
    try:
        v = _Mech()
        lib().janc_mech_file_view(h, C.byref(v))
        ns, nr = v.ns, v.nr
        def arr(ptr, n, ct, dt):
            return np.ctypeslib.as_array(C.cast(ptr, C.POINTER(ct)), shape=(n,)).astype(dt).copy() if n else np.zeros(0, dt)
        f = lambda ptr, n: arr(ptr, n, C.c_double, np.float64)
        i = lambda ptr, n: arr(ptr, n, C.c_int32, np.int32)
        names = [lib().janc_mech_file_species(h, k).decode() for k in range(ns)]
        return inputs.Mechanism(ns=ns, nr=nr, W=f(v.W, ns), nasa=f(v.nasa, ns * 7).reshape(ns, 7),
                                nu_f=i(v.nu_f, nr * ns).reshape(nr, ns), nu_b=i(v.nu_b, nr * ns).reshape(nr, ns),
                                A=f(v.A, nr), b=f(v.b, nr), Ta=f(v.Ta, nr), reversible=i(v.reversible, nr),
                                third_body=i(v.third_body, nr), eff=f(v.eff, nr * ns).reshape(nr, ns), names=names,
                                nasa_hi=f(v.nasa_hi, ns * 7).reshape(ns, 7), T_mid=f(v.T_mid, ns))
    finally:
        lib().janc_mech_file_free(h)


def measure_dfma_peak(device=0, stream=None):
    out = C.c_double(0.0)
    rc = lib().janc_measure_dfma_peak(int(device), C.c_void_p(stream or 0), C.byref(out))
    if rc:
        raise JancError(rc, "janc_measure_dfma_peak")
    return out.value


def workspace_bytes_for(grid, mech, device=0, options=None):
    """janc_workspace_bytes of a context for `grid` (n_patches taken from it) and `mech`, without allocating anything:
    how the AMR driver sizes the workspace for its block capacity."""
    L = lib()
    g = _Grid(grid.ndim, (C.c_int * 3)(*grid.n), (C.c_double * 3)(*grid.dx), (C.c_int * 3)(*grid.bc_lo), (C.c_int * 3)(*grid.bc_hi),
              grid.n_patches, grid.n_levels, grid.ratio)
    h = C.c_void_p()
    rc = L.janc_create(C.byref(g), int(device), None, C.byref(h))
    if rc:
        raise JancError(rc, "janc_create")
    try:
        for k, v in (options or {}).items():
            if L.janc_set_option(h, str(k).encode(), str(v).encode()):
                raise JancError(JANC_EINVAL, f"janc_set_option({k})")
        m, keep = _mech_struct(mech)
        rc = L.janc_set_mechanism(h, C.byref(m))
        if rc:
            raise JancError(rc, "janc_set_mechanism")
        return int(L.janc_workspace_bytes(h))
    finally:
        L.janc_destroy(h)


class Solver:
    """janc_* context: create -> set_mechanism -> bind_workspace (torch) -> [set_blocks] -> set_state
    -> step -> get_state -> destroy.  Same call names as the C ABI."""

    def __init__(self, grid, mech, blocks=None, device=0, stream=None, options=None, workspace=None):
        """workspace: a uint8 CUDA tensor to bind instead of allocating one (at least workspace_bytes + 256 bytes; the
        AMR driver keeps one sized for its block capacity across regrids)."""
        import torch
        if not torch.cuda.is_available():
            raise JancError(JANC_ECUDA, "no CUDA device (libjanc has no CPU fallback)")
        L = lib()
        self._torch = torch
        self.device = int(device)
        torch.cuda.set_device(self.device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        g = _Grid(grid.ndim, (C.c_int * 3)(*grid.n), (C.c_double * 3)(*grid.dx),
                  (C.c_int * 3)(*grid.bc_lo), (C.c_int * 3)(*grid.bc_hi),
                  grid.n_patches, grid.n_levels, grid.ratio)
        self._h = C.c_void_p()
        rc = L.janc_create(C.byref(g), self.device, C.c_void_p(stream.cuda_stream), C.byref(self._h))
        if rc:
            raise JancError(rc, "janc_create")
        for k, v in (options or {}).items():          # janc_set_option(key, value), see include/janc.h
            self._check(L.janc_set_option(self._h, str(k).encode(), str(v).encode()), f"janc_set_option({k})")
        m, self._keep = _mech_struct(mech)
        self._check(L.janc_set_mechanism(self._h, C.byref(m)), "janc_set_mechanism")
        nbytes = L.janc_workspace_bytes(self._h)
        self.workspace_bytes = nbytes
        if workspace is not None:
            if not (workspace.is_cuda and workspace.dtype == torch.uint8 and workspace.numel() >= nbytes + 256):
                raise JancError(JANC_EINVAL, f"workspace tensor too small: {workspace.numel()} < {nbytes + 256}")
            self.workspace = workspace
        else:
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=f"cuda:{self.device}")
        base = (self.workspace.data_ptr() + 255) // 256 * 256
        self._ws_off = base - self.workspace.data_ptr()
        self._check(L.janc_bind_workspace(self._h, C.c_void_p(base), nbytes), "janc_bind_workspace")
        if blocks is not None:
            self._check(L.janc_set_blocks(self._h, _ptr(_i32(blocks.level)), _ptr(_i32(blocks.nbr)),
                                          _ptr(_i32(blocks.parent))), "janc_set_blocks")
        self.np_ = max(1, grid.n_patches)
        self.nvar = grid.ndim + 2 + mech.ns - 1
        self.shape = (self.np_, self.nvar, grid.n[2] if grid.ndim > 2 else 1,
                      grid.n[1] if grid.ndim > 1 else 1, grid.n[0])
        self.tshape = (self.shape[0],) + self.shape[2:]

    def set_option(self, key, value):
        self._check(lib().janc_set_option(self._h, str(key).encode(), str(value).encode()), f"janc_set_option({key})")

    def chem_kernel(self):
        """'jit' (mechanism-specialised, NVRTC), 'reg' or 'generic' (table-driven kernels)."""
        return lib().janc_chem_kernel(self._h).decode()

    def jit_log(self):
        return lib().janc_jit_log(self._h).decode()

    def _check(self, rc, what):
        if rc:
            msg = lib().janc_last_error(self._h)
            raise JancError(rc, f"{what}: {msg.decode() if msg else ''}")

    # -- state ------------------------------------------------------------------------------
    def set_state(self, U, T=None):
        """U, T: numpy arrays (host) or torch CUDA tensors (device), interior layout."""
        torch = self._torch
        if isinstance(U, torch.Tensor):
            assert U.is_cuda and U.dtype == torch.float64 and U.is_contiguous() and U.numel() == int(np.prod(self.shape))
            Tp = None
            if T is not None:
                assert T.is_cuda and T.dtype == torch.float64 and T.is_contiguous()
                Tp = C.c_void_p(T.data_ptr())
            self._check(lib().janc_set_state(self._h, C.c_void_p(U.data_ptr()), Tp, 1), "janc_set_state")
        else:
            U = _f64(U)
            assert U.size == int(np.prod(self.shape)), (U.shape, self.shape)
            Tn = _f64(T) if T is not None else None
            self._check(lib().janc_set_state(self._h, _ptr(U), _ptr(Tn) if Tn is not None else None, 0),
                        "janc_set_state")

    def step(self, nsteps, cfl=0.0, dt=0.0, chem=True, sync=True, crossover=False):
        """Returns the time advanced (sync=True) or None (asynchronous enqueue).  chem: True = point-implicit after the
        RK3, False = none, "explicit" = source inside every RK stage; crossover:
        sub-cycled level advance of a two-level block list (Fig 2a), dt / cfl then refer to level 0."""
        flags = FLAG_EXPLICIT_SOURCE if chem == "explicit" else (0 if chem else FLAG_NO_CHEM)
        if crossover:
            flags |= FLAG_CROSSOVER
        if sync:
            t = C.c_double(0.0)
            rc = lib().janc_step(self._h, int(nsteps), float(cfl), float(dt), flags, C.byref(t))
            self.status = rc
            if rc not in (JANC_OK, JANC_ENONFINITE):
                self._check(rc, "janc_step")
            return t.value
        self._check(lib().janc_step(self._h, int(nsteps), float(cfl), float(dt), flags, None), "janc_step")
        return None

    # -- x-slab decomposition (janc_step_part / janc_halo / janc_reduction_slots) -------------
    def step_part(self, part, stage=0, cfl=0.0, dt=0.0, chem=True):
        self._check(lib().janc_step_part(self._h, int(part), int(stage), float(cfl), float(dt), 0 if chem else FLAG_NO_CHEM),
                    "janc_step_part")

    def halo_doubles(self):
        return lib().janc_halo_doubles(self._h)

    def halo(self, stage, side, buf, unpack):
        """buf: contiguous float64 CUDA tensor of halo_doubles() elements."""
        assert buf.is_cuda and buf.dtype == self._torch.float64 and buf.is_contiguous() and buf.numel() >= self.halo_doubles()
        self._check(lib().janc_halo(self._h, int(stage), int(side), C.c_void_p(buf.data_ptr()), int(bool(unpack))), "janc_halo")

    def slots_tensor(self):
        """The reduction slots as an int64 view into the workspace (non-negative doubles order like their bit patterns)."""
        off, cnt = C.c_size_t(0), C.c_size_t(0)
        self._check(lib().janc_reduction_slots(self._h, C.byref(off), C.byref(cnt)), "janc_reduction_slots")
        a = self._ws_off + off.value
        return self.workspace[a:a + 8 * cnt.value].view(self._torch.int64)

    def regrid(self, thr, nbuf, device=False):
        """janc_regrid_plan + janc_regrid_fill: (level, nbr, parent, U, T) of the regridded two-level list (lists: host
        arrays; U, T: host arrays, or CUDA tensors with device=True)."""
        nd = 1 + (self.shape[3] > 1) + (self.shape[2] > 1)
        cap = self.np_ * (1 + (1 << nd))
        level = np.zeros(cap, np.int32); nbr = np.zeros((cap, 2 * nd), np.int32); parent = np.zeros((cap, 1 + nd), np.int32)
        n = C.c_int32(0)
        self._check(lib().janc_regrid_plan(self._h, float(thr), int(nbuf), C.byref(n), _ptr(level), _ptr(nbr), _ptr(parent)),
                    "janc_regrid_plan")
        k = n.value
        torch = self._torch
        U = torch.empty((k,) + self.shape[1:], dtype=torch.float64, device=f"cuda:{self.device}")
        T = torch.empty((k,) + self.shape[2:], dtype=torch.float64, device=f"cuda:{self.device}")
        self._check(lib().janc_regrid_fill(self._h, C.c_void_p(U.data_ptr()), C.c_void_p(T.data_ptr()), 1), "janc_regrid_fill")
        if device:
            return level[:k].copy(), nbr[:k].copy(), parent[:k].copy(), U, T
        return level[:k].copy(), nbr[:k].copy(), parent[:k].copy(), U.cpu().numpy(), T.cpu().numpy()

    def last_dt(self):
        """dt of the most recent step (device scalar), synchronising."""
        t = C.c_double(0.0)
        self._check(lib().janc_last_dt(self._h, C.byref(t)), "janc_last_dt")
        return t.value

    def cfl_dt_static(self, U, T, cfl, out):
        """janc_cfl_dt_static: dt and the max(|u_d| + c) of the state U (T = Newton start or None), all CUDA tensors of the
        caller (U, T in the interior layout of set_state; out: 4 doubles), enqueued on the solver's stream; allocates nothing."""
        torch = self._torch
        for t, n in ((U, int(np.prod(self.shape))), (T, int(np.prod(self.tshape))), (out, 4)):
            assert t is None or (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous() and t.numel() == n)
        self._check(lib().janc_cfl_dt_static(self._h, C.c_void_p(U.data_ptr()), C.c_void_p(T.data_ptr()) if T is not None else None,
                                             float(cfl), C.c_void_p(out.data_ptr())), "janc_cfl_dt_static")

    def get_state(self, device=False):
        if device:
            torch = self._torch
            U = torch.empty(self.shape, dtype=torch.float64, device=f"cuda:{self.device}")
            T = torch.empty(self.tshape, dtype=torch.float64, device=f"cuda:{self.device}")
            rc = lib().janc_get_state(self._h, C.c_void_p(U.data_ptr()), C.c_void_p(T.data_ptr()), 1)
        else:
            U = np.empty(self.shape); T = np.empty(self.tshape)
            rc = lib().janc_get_state(self._h, _ptr(U), _ptr(T), 0)
        self.status = rc
        if rc not in (JANC_OK, JANC_ENONFINITE):
            self._check(rc, "janc_get_state")
        return U, T

    def get_state_into(self, U_host):
        """Device -> caller's (pinned) host array; returns status."""
        rc = lib().janc_get_state(self._h, _ptr(U_host), None, 0)
        self.status = rc
        return rc

    def status_sync(self):
        return lib().janc_status(self._h)

    def launch_count(self):
        return lib().janc_launch_count(self._h)

    def debug_cons2prim(self):
        T = np.empty(self.tshape); p = np.empty(self.tshape); c = np.empty(self.tshape)
        rc = lib().janc_debug_cons2prim(self._h, _ptr(T), _ptr(p), _ptr(c), 0)
        if rc not in (JANC_OK, JANC_ENONFINITE):
            self._check(rc, "janc_debug_cons2prim")
        return T, p, c

    def profile_step(self, cfl=0.0, dt=0.0):
        ms = (C.c_float * 6)(); n = (C.c_int * 6)()
        rc = lib().janc_profile_step(self._h, float(cfl), float(dt), ms, n)
        if rc not in (JANC_OK, JANC_ENONFINITE):
            self._check(rc, "janc_profile_step")
        names = ["cons2prim", "ghost", "flux_rk", "chem", "average_down", "step"]
        return {k: (ms[i], n[i]) for i, k in enumerate(names)}

    def close(self):
        if getattr(self, "_h", None):
            lib().janc_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
