"""The algebra the flux kernels rely on (csrc/flux.cuh header), checked on the CPU against the oracle's WENO5-JS.

flux.cuh does not evaluate the Jiang-Shu formula (eq 4.11) as written: it
reconstructs 2f+- in difference form, carries the smoothness indicators as 4 beta with eps scaled to match, replaces
the three divisions by products over a common denominator, re-uses t_k in the candidate numerators and joins the two
reconstructions of a face over one reciprocal.  This file restates that regrouping in numpy, step by step as the
header comment gives it, and compares it with `oracle.ref.weno5` (the formula as the paper gives it) on smooth data,
on shocks and on widely scaled data.  It checks the derivation, not the CUDA code: that is what the `-m gpu` parity
tests do.  CPU only.
"""
import numpy as np

EPS16 = 16 * 1e-6        # 16 eps: eps -> 4 eps for 2f, carried x 4 with the indicators


def _num_den(D0, D1, D2, D3):
    """6 (q - v) = num / den for differences D_k = v_{k+1} - v_k about the centre value v = v_0 (flux.cuh weno5_diff)."""
    K = 13.0 / 3.0
    S0 = K * (D1 - D0) ** 2 + EPS16
    S1 = K * (D2 - D1) ** 2 + EPS16
    S2 = K * (D3 - D2) ** 2 + EPS16
    t0, t1, t2 = 3 * D1 - D0, D1 + D2, D3 - 3 * D2
    b0, b1, b2 = (t0 * t0 + S0) ** 2, (t1 * t1 + S1) ** 2, (t2 * t2 + S2) ** 2
    c0, c1, c2 = 2 * t0 - D1, t1 + D2, D2 - t2
    a0, h, w = b1 * b2, 3 * b0, 2 * b2
    return a0 * c0 + h * (w * c1 + b1 * c2), h * (w + b1) + a0


def face_flux_regrouped(fp, fm):
    """Numerical flux at i+1/2 from f+ on cells i-2..i+2 and f- on cells i-1..i+3 (6 template points), via 2f+-."""
    P, M = 2 * np.asarray(fp, float), 2 * np.asarray(fm, float)      # P[k]: cell i-2+k, M[k]: cell i-1+k
    dP, dM = np.diff(P), np.diff(M)
    np_, dp = _num_den(dP[0], dP[1], dP[2], dP[3])                    # centre P[2] = cell i
    nm, dm = _num_den(-dM[3], -dM[2], -dM[1], -dM[0])                 # mirror image, centre M[2] = cell i+1
    twice = (P[2] + M[2]) + (nm * dp + np_ * dm) / (dp * dm) / 6.0
    return 0.5 * twice


def _check(ref, fp, fm, tol):
    want = ref.weno5(list(fp)) + ref.weno5(list(fm[::-1]))            # minus part: the mirrored stencil
    got = face_flux_regrouped(fp, fm)
    scale = max(np.max(np.abs(fp)), np.max(np.abs(fm)), 1e-300)
    assert abs(got - want) <= tol * scale, (got, want)


def test_regrouped_weno_equals_jiang_shu_on_random_data(ref):
    rng = np.random.default_rng(7)
    for _ in range(300):
        _check(ref, rng.normal(size=5), rng.normal(size=5), 2e-14)


def test_regrouped_weno_on_smooth_and_shock_data(ref):
    x = np.arange(-2, 4) * 0.1
    smooth = np.sin(x) + 2.0
    _check(ref, smooth[:5], smooth[1:], 2e-15)
    step = np.array([1.0, 1.0, 1.0, 0.0, 0.0, 0.0])
    for sh in range(4):
        s = np.roll(step, sh - 1)
        _check(ref, s[:5], s[1:], 2e-14)
    # uniform data: the reconstruction returns the cell value exactly (uniform-state preservation, A5)
    assert face_flux_regrouped([3.5] * 5, [1.25] * 5) == 3.5 + 1.25


def test_regrouped_weno_at_flux_magnitudes_of_the_workloads(ref):
    """energy fluxes of a 30 bar detonation are ~1e10, species fluxes ~1e-3: the products of eight factors in the
    common-denominator form must neither overflow nor lose the eps weighting."""
    rng = np.random.default_rng(11)
    for scale in (1e-6, 1e-3, 1.0, 1e5, 1e10, 1e12):
        for _ in range(50):
            base = scale * (1.0 + 0.3 * rng.normal(size=6))
            _check(ref, base[:5], base[1:] * (1 + 0.1 * rng.normal()), 5e-14)
