"""janc_cfl_dt_static (include/janc.h): the entry point that allocates nothing -- its scratch is a file-scope
`static __device__` array of the library -- against the existing path (janc_step's cons->prim + max-reduction into the
workspace slots + k_dt), on several calls in a row that share the array.  Collected last on purpose (the suite runs with
pytest -x); passes alone in a fresh process and after the other tests (then another context's species tables sit in
constant memory and the first call re-uploads its own)."""
import ctypes as C
import dataclasses

import numpy as np
import pytest

from paper_2504_13750_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL = 1e-12      # the tolerance the parity tests put on the time advanced; the maxima themselves are exact reductions


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2504_13750_b200 import binding, build
    build.build()
    binding.lib()
    return binding


class BareCtx:
    """janc_create + janc_set_mechanism only: no workspace, no blocks, no state."""

    def __init__(self, B, grid, mech, device=0):
        import torch
        L = B.lib()
        g = B._Grid(grid.ndim, (C.c_int * 3)(*grid.n), (C.c_double * 3)(*grid.dx), (C.c_int * 3)(*grid.bc_lo),
                    (C.c_int * 3)(*grid.bc_hi), grid.n_patches, grid.n_levels, grid.ratio)
        self.B, self.h = B, C.c_void_p()
        stream = torch.cuda.current_stream(device)
        assert L.janc_create(C.byref(g), device, C.c_void_p(stream.cuda_stream), C.byref(self.h)) == 0
        m, self.keep = B._mech_struct(mech)
        assert L.janc_set_mechanism(self.h, C.byref(m)) == 0, L.janc_last_error(self.h)

    def call(self, U, T, cfl, out):
        return self.B.lib().janc_cfl_dt_static(self.h, C.c_void_p(U.data_ptr()), C.c_void_p(T.data_ptr()) if T is not None else None,
                                               float(cfl), C.c_void_p(out.data_ptr()))

    def error(self):
        return self.B.lib().janc_last_error(self.h).decode()

    def close(self):
        self.B.lib().janc_destroy(self.h)


def existing_path(B, case, cfl):
    """dt and the per-direction maxima of the step-start state as janc_step forms them (workspace slots + k_dt)."""
    s = B.Solver(case.grid, case.mech, case.blocks)
    s.set_state(case.U, case.T)
    s.step(1, cfl=cfl, chem=False)
    assert s.status == 0
    dt = s.last_dt()
    slots = s.slots_tensor().cpu().numpy().view(np.float64)      # parity 0, sub-step 0, stage 0: [level][direction]
    smax = np.maximum(slots[0:3], slots[3:6])
    s.close()
    return dt, smax


def evolved(B, case, nsteps=8):
    """The case after a few steps: the seeded initial states are at rest, so that every direction has the same maximum;
    after the driver / spheres have started to expand the three maxima differ."""
    s = B.Solver(case.grid, case.mech, case.blocks)
    s.set_state(case.U, case.T)
    s.step(nsteps, cfl=case.cfl, chem=False)
    U, T = s.get_state()
    assert s.status == 0
    s.close()
    return dataclasses.replace(case, U=U, T=T)


def cases(B, mech9):
    a = evolved(B, I.config1(nx=300, ny=70, mech=mech9))          # 21000 cells: 83 CTAs with a ragged tail
    b = evolved(B, I.config3(pcols=8, prows=4, npc=16, mech=mech9))   # two-level block list: dx_min is the fine spacing
    c = evolved(B, I.config4(n=24, nspheres=3, radius=5, mech=mech9))   # 3-D
    return [a, b, c, a]                                           # ... and the first one again over the others' leftovers


def test_static_scratch_matches_existing_path_on_calls_in_a_row(B, mech9):
    import torch
    todo = cases(B, mech9)
    want = [existing_path(B, cs, cs.cfl) for cs in todo]
    # all calls back to back on one stream, results read afterwards: the shared array is reused without a host sync between
    ctxs, outs = [], []
    for cs in todo:
        ctx = BareCtx(B, cs.grid, cs.mech)
        U = torch.from_numpy(np.ascontiguousarray(cs.U)).cuda()
        T = torch.from_numpy(np.ascontiguousarray(cs.T)).cuda()
        out = torch.full((4,), -1.0, dtype=torch.float64, device="cuda")
        assert ctx.call(U, T, cs.cfl, out) == 0, ctx.error()
        ctxs.append((ctx, U, T)); outs.append(out)
    torch.cuda.synchronize()
    for cs, (dt_ref, smax_ref), out in zip(todo, want, outs):
        got = out.cpu().numpy()
        assert np.isfinite(got).all() and got[0] > 0.0
        assert abs(got[0] - dt_ref) <= TOL * dt_ref, (cs.name, got[0], dt_ref)
        assert np.abs(got[1:] - smax_ref).max() <= TOL * smax_ref.max(), (cs.name, got[1:], smax_ref)
        assert (got[1 + cs.grid.ndim:] == 0.0).all()
    assert len({tuple(np.round(w[1] / w[1].max(), 6)) for w in want}) > 1 and want[0][1][0] != want[0][1][1]
    # free device memory does not move over further calls (everything is loaded by now)
    free0 = torch.cuda.mem_get_info()[0]
    for (ctx, U, T), cs, out in zip(ctxs, todo, outs):
        assert ctx.call(U, T, cs.cfl, out) == 0, ctx.error()
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0, "the calls changed the device's free memory"
    for ctx, _, _ in ctxs:
        ctx.close()


def test_static_scratch_flag_is_cleared_between_calls(B, mech9):
    import torch
    cs = I.config1(nx=96, ny=40, mech=mech9)
    dt_ref, _ = existing_path(B, cs, cs.cfl)
    ctx = BareCtx(B, cs.grid, cs.mech)
    bad = np.ascontiguousarray(cs.U).copy()
    bad[0, cs.grid.ndim + 1].flat[1234] = -1e9                    # negative total energy: the Newton iteration fails there
    out1, out2 = (torch.zeros(4, dtype=torch.float64, device="cuda") for _ in range(2))
    Ub, Ug = torch.from_numpy(bad).cuda(), torch.from_numpy(np.ascontiguousarray(cs.U)).cuda()
    # same context, same stream, no host synchronisation between the two calls
    assert ctx.call(Ub, None, cs.cfl, out1) == 0, ctx.error()     # T_dev = NULL: Newton from 1000 K
    assert ctx.call(Ug, None, cs.cfl, out2) == 0, ctx.error()
    first, second = out1.cpu().numpy(), out2.cpu().numpy()
    assert np.isnan(first[0]) and np.isfinite(first[1:]).all()
    # the existing path started its Newton iteration from the case's T, this one from 1000 K: same root to rounding
    assert abs(second[0] - dt_ref) <= 1e-10 * dt_ref, (second[0], dt_ref)
    ctx.close()


def test_static_scratch_rejects_sizes_beyond_the_maximum(B):
    import torch
    g = I.Grid(2, (8192, 2049, 1), (1e-3, 1e-3, 1.0), (2, 2, 0), (2, 2, 0))      # one column more than 2^24 cells
    ctx = BareCtx(B, g, I.inert_gas())
    dummy = torch.zeros(4, dtype=torch.float64, device="cuda")
    assert ctx.call(dummy, None, 0.5, dummy) == B.JANC_EINVAL
    assert "exceed the static scratch" in ctx.error()
    ok = BareCtx(B, I.Grid(2, (64, 48, 1), (1e-3, 1e-3, 1.0), (2, 2, 0), (2, 2, 0)), I.inert_gas())
    assert ok.call(dummy, None, 0.0, dummy) == B.JANC_EINVAL and "cfl" in ok.error()
    ctx.close(); ok.close()


def test_static_scratch_inside_cuda_graph_capture(B, mech9):
    """The use case the entry point exists for: after one call outside capture (symbol address, species tables), calls
    are captured into a CUDA graph -- where cudaMalloc and synchronisation are not allowed -- and the replay gives the
    result of the workspace path for whatever state is in the caller's buffers at replay time."""
    import torch
    cs = I.config1(nx=96, ny=40, mech=mech9)
    cs2 = evolved(B, cs, 6)
    ref1, ref2 = existing_path(B, cs, cs.cfl), existing_path(B, cs2, cs2.cfl)
    side = torch.cuda.Stream()
    U = torch.from_numpy(np.ascontiguousarray(cs.U)).cuda()
    T = torch.from_numpy(np.ascontiguousarray(cs.T)).cuda()
    out = torch.zeros(4, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        ctx = BareCtx(B, cs.grid, cs.mech)                       # bound to the side stream
        assert ctx.call(U, T, cs.cfl, out) == 0, ctx.error()      # set-up call, outside capture
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            assert ctx.call(U, T, cs.cfl, out) == 0, ctx.error()
    out.zero_()
    g.replay(); torch.cuda.synchronize()
    got1 = out.cpu().numpy().copy()
    U.copy_(torch.from_numpy(np.ascontiguousarray(cs2.U))); T.copy_(torch.from_numpy(np.ascontiguousarray(cs2.T)))
    g.replay(); torch.cuda.synchronize()
    got2 = out.cpu().numpy().copy()
    assert abs(got1[0] - ref1[0]) <= TOL * ref1[0] and np.abs(got1[1:] - ref1[1]).max() <= TOL * ref1[1].max()
    assert abs(got2[0] - ref2[0]) <= TOL * ref2[0] and np.abs(got2[1:] - ref2[1]).max() <= TOL * ref2[1].max()
    assert got1[0] != got2[0]
    ctx.close()
