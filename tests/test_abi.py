"""CPU-side checks of the boundary: the C-ABI library builds for sm_100a, loads without a GPU and
exports every symbol include/janc.h declares; without a device it refuses to run (no CPU fallback)."""
import ctypes
import os
import re

import pytest

from paper_2504_13750_b200 import inputs as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_2504_13750_b200 import binding, build
    build.build()
    return binding.lib()


def test_exports_match_header(L):
    from paper_2504_13750_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "janc.h")).read()
    declared = set(re.findall(r"\b(janc_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.EXPORTS), declared ^ set(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_no_cpu_fallback_without_device(L):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_2504_13750_b200 import binding
    case = I.config0(n=16)
    with pytest.raises(binding.JancError):
        binding.Solver(case.grid, case.mech)
    # and the raw ABI refuses too
    g = binding._Grid(1, (ctypes.c_int * 3)(16, 1, 1), (ctypes.c_double * 3)(1e-4, 1, 1),
                      (ctypes.c_int * 3)(2, 0, 0), (ctypes.c_int * 3)(2, 0, 0), 0, 1, 2)
    h = ctypes.c_void_p()
    assert L.janc_create(ctypes.byref(g), 0, None, ctypes.byref(h)) == binding.JANC_ECUDA


def test_product_never_imports_oracle():
    pkg = os.path.join(ROOT, "paper_2504_13750_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "janc_ref" not in src and "from oracle" not in src and "import oracle" not in src, f


def test_mechanism_health_of_chosen_seeds(ref, mech9, mech20):
    """0-D run at 3000 K / 30 bar, 200 steps of 4e-9 s stays finite and positive."""
    import numpy as np
    for m in (mech9, mech20):
        U = I.prim_to_cons(m, 1, np.array([3.0e6]), np.array([3000.0]), I.hot_Y(m.ns)[None], [np.zeros(1)])
        g = I.Grid(1, (1, 1, 1), (1e-3, 1, 1), (2, 0, 0), (2, 0, 0))
        s = ref.RefSolver(g, m)
        s.set_state(U.reshape(1, -1, 1, 1, 1), np.full((1, 1, 1, 1), 3000.0))
        s.step(200, cfl=0.0, dt=4e-9)
        U1, T1 = s.get_state()
        assert s.status == 0 and np.isfinite(U1).all() and T1[0, 0, 0, 0] > 0
        rho = U1[0, 0, 0, 0, 0]
        Y = U1[0, 3:, 0, 0, 0] / rho
        assert Y.min() > -1e-12 and 1 - Y.sum() > -1e-12


def test_specialised_chemistry_source_compiles_for_sm100a(L, mech9):
    """janc_set_mechanism's code generator (csrc/chemgen.h): the emitted CUDA C compiles with NVRTC for
    sm_100a without a GPU, for the synthetic 9-species mechanism and the single-step model."""
    from paper_2504_13750_b200 import binding
    for mech, ndim in ((mech9, 2), (I.single_step_mechanism(), 1)):
        src, nbytes = binding.jit_probe(mech, ndim)
        assert "k_chem_jit" in src and "__any_sync" in src or mech.ns == 2
        assert nbytes and nbytes > 1000
        # every reaction and every unknown appears as literals: no table lookups in the kernel
        assert f"// reaction {mech.nr - 1}" in src and f"A{mech.ns - 2}_{mech.ns - 2}" in src
        assert "k_prim_jit" in src and "c_mech" not in src
        assert "__shared__" not in src[src.index("k_chem_jit"):]


def test_role_warp_chemistry_source_compiles_for_sm100a(L, mech20):
    """csrc/chemgen_roles.h (mechanisms with 13..23 unknowns): 8 role-specific literal sections, the system
    columns as named registers, reaction tables in __constant__ memory; compiles for sm_100a without a GPU."""
    from paper_2504_13750_b200 import binding
    src, nbytes = binding.jit_probe(mech20, 3)
    k = src[src.index("k_chem_jit"):]
    assert nbytes and nbytes > 1000
    assert all(f"case {w}:" in k for w in range(8)) and "A2_18" in k and "BAR();" in k and "bar.sync" in src
    assert "__constant__ double g_td[" in src and "barrier.arrive" in src and "c_mech" not in src
