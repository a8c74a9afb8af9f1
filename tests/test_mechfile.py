"""The Chemkin-format reader of the library (csrc/mechfile.h, janc_mech_parse):
round trip of the seeded synthetic mechanisms through Chemkin text, unit keywords, separate thermo text, and the
refusal of what eq 4.6-4.9 cannot express.  CPU only: the reader is host code."""
import numpy as np
import pytest

from paper_2504_13750_b200 import inputs as I
from tests import chemkin_writer as CW


@pytest.fixture(scope="module")
def B():
    from paper_2504_13750_b200 import binding, build
    build.build()
    binding.lib()
    return binding


def same(a, b, tol):
    a, b = np.asarray(a, float), np.asarray(b, float)
    return a.shape == b.shape and np.abs(a - b).max() <= tol * max(np.abs(a).max(), 1e-300)


@pytest.mark.parametrize("ns,nr", [(9, 21), (20, 100)])
def test_round_trip_through_chemkin_text(B, ns, nr):
    m = I.two_range(I.synthetic_mechanism(ns, nr), np.linspace(800.0, 1400.0, ns), 0.5, seed=ns)
    text, thermo, names = CW.write(m)
    r = B.load_chemkin(text)
    assert r.ns == ns and r.nr == nr and r.names == names
    assert same(r.W, m.W, 1e-9)
    assert np.array_equal(r.nu_f, m.nu_f) and np.array_equal(r.nu_b, m.nu_b)
    assert np.array_equal(r.reversible, m.reversible) and np.array_equal(r.third_body, m.third_body)
    assert same(r.A, m.A, 1e-14) and same(r.b, m.b, 1e-14) and same(r.Ta, m.Ta, 1e-14)
    tb = m.third_body.astype(bool)
    assert same(r.eff[tb], m.eff[tb], 1e-14) and (r.eff[~tb] == 1.0).all()
    for k in range(ns):                       # E15.8 fields: 9 significant digits
        assert same(r.nasa[k], m.nasa[k], 2e-8) and same(r.nasa_hi[k], m.nasa_hi[k], 2e-8), k
    assert same(r.T_mid, m.T_mid, 1e-5)
    # the thermo section as a separate text, another energy unit
    text2, thermo2, _ = CW.write(m, e_unit="KELVINS", inline_thermo=False)
    r2 = B.load_chemkin(text2, thermo2)
    assert same(r2.Ta, m.Ta, 1e-14) and same(r2.nasa_hi, r.nasa_hi, 0.0) and same(r2.A, m.A, 1e-14)
    text3, _, _ = CW.write(m, e_unit="KCAL/MOLE")
    assert same(B.load_chemkin(text3).Ta, m.Ta, 1e-13)


def test_small_hand_written_file(B):
    """Built-in atomic weights, stoichiometric coefficients, '=' / '=>' / '<=>', comments, DUP, default T_mid."""
    text = """
ELEM H O N END
SPECIES
 H2 O2 H2O   ! three reacting species
 N2
END
THERMO
   300.000  1000.000  5000.000
H2                synth H   2               G   300.000  5000.000 1000.00      1
 1.00000000E+00 2.00000000E-03 0.00000000E+00 0.00000000E+00 0.00000000E+00    2
 3.00000000E+00 4.00000000E+00 5.00000000E+00 6.00000000E-03 0.00000000E+00    3
 0.00000000E+00 0.00000000E+00 7.00000000E+00 8.00000000E+00                   4
O2                synth O   2               G   300.000  5000.000              1
 3.50000000E+00 0.00000000E+00 0.00000000E+00 0.00000000E+00 0.00000000E+00    2
 0.00000000E+00 1.00000000E+00 3.40000000E+00 0.00000000E+00 0.00000000E+00    3
 0.00000000E+00 0.00000000E+00 0.00000000E+00 2.00000000E+00                   4
H2O               synth H   2O   1          G   300.000  5000.000 1200.00      1
 4.00000000E+00 0.00000000E+00 0.00000000E+00 0.00000000E+00 0.00000000E+00    2
-3.00000000E+04 1.00000000E+00 3.90000000E+00 0.00000000E+00 0.00000000E+00    3
 0.00000000E+00 0.00000000E+00-3.00000000E+04 2.00000000E+00                   4
N2                synth N   2               G   300.000  5000.000 1000.00      1
 3.50000000E+00 0.00000000E+00 0.00000000E+00 0.00000000E+00 0.00000000E+00    2
 0.00000000E+00 1.00000000E+00 3.50000000E+00 0.00000000E+00 0.00000000E+00    3
 0.00000000E+00 0.00000000E+00 0.00000000E+00 1.00000000E+00                   4
END
REACTIONS
2H2 + O2 => 2H2O        1.0E+13  0.5  1000.0
 DUPLICATE
H2O + M = H2 + O2 + M   2.0E+10  -1.0  0.0     ! unbalanced on purpose: the reader does not check balance
 H2/2.5/ H2O/12/
END
"""
    m = B.load_chemkin(text)
    assert m.names == ["H2", "O2", "H2O", "N2"] and m.nr == 2
    assert same(m.W, [2 * 1.00794e-3, 2 * 15.9994e-3, (2 * 1.00794 + 15.9994) * 1e-3, 2 * 14.0067e-3], 1e-12)
    assert m.nu_f.tolist() == [[2, 1, 0, 0], [0, 0, 1, 0]] and m.nu_b.tolist() == [[0, 0, 2, 0], [1, 1, 0, 0]]
    assert m.reversible.tolist() == [0, 1] and m.third_body.tolist() == [0, 1]
    assert same(m.A, [1.0e13 * 1e-12, 2.0e10 * 1e-6], 1e-14)                 # orders 3 and 2 (with M)
    assert same(m.Ta, [1000.0 * 4.184 / 8.314472, 0.0], 1e-14) and m.b.tolist() == [0.5, -1.0]
    assert m.eff[1].tolist() == [2.5, 1.0, 12.0, 1.0]
    assert m.nasa_hi[0].tolist() == [1.0, 2.0e-3, 0.0, 0.0, 0.0, 3.0, 4.0] and m.nasa[0].tolist() == [5.0, 6.0e-3, 0.0, 0.0, 0.0, 7.0, 8.0]
    assert m.T_mid.tolist() == [1000.0, 1000.0, 1200.0, 1000.0]              # O2: blank field -> the section default


@pytest.mark.parametrize("bad,msg", [
    ("H + O2 (+M) = HO2 (+M)  1e12 0 0", "fall-off"),
    ("H + O2 = HO2  1e12 0 0\n LOW / 1e15 0 0 /", "LOW"),
    ("H + O2 = HO2  1e12 0 0\n REV / 1e15 0 0 /", "REV"),
    ("H + XX = HO2  1e12 0 0", "unknown species"),
    ("H + O2 + M => HO2  1e12 0 0", "third body on one side"),
    ("H + O2 = HO2  1e12 0", "A, b, E"),
])
def test_unsupported_input_is_refused_with_a_message(B, bad, msg):
    head = "ELEM H O END\nSPECIES H O2 HO2 END\nTHERMO\n 300. 1000. 5000.\n"
    for sp, comp in (("H", "H   1"), ("O2", "O   2"), ("HO2", "H   1O   2")):
        l1 = f"{sp:<18s}{'x':<6s}{comp:<20s}G{300.0:>10.3f}{5000.0:>10.3f}{1000.0:>8.2f}".ljust(79) + "1"
        z = "".join(f"{v:15.8E}" for v in (2.5, 0, 0, 0, 0))
        head += l1 + "\n" + z.ljust(79) + "2\n" + z.ljust(79) + "3\n" + "".join(f"{v:15.8E}" for v in (0, 0, 0, 0)).ljust(79) + "4\n"
    head += "END\nREACTIONS\n"
    with pytest.raises(B.JancError) as e:
        B.load_chemkin(head + bad + "\nEND\n")
    assert msg in str(e.value), str(e.value)


def test_loaded_mechanism_drives_the_oracle_like_the_original(B, ref):
    """The arrays that come back are usable as they are: the oracle advanced with the re-read mechanism stays within the
    text's precision of the run with the original arrays."""
    m = I.two_range(I.synthetic_mechanism(9, 21), 1000.0, 0.5, seed=2)
    r = B.load_chemkin(CW.write(m)[0])
    r.elements = m.elements
    ca, cb = I.config1(nx=24, ny=12, mech=m), I.config1(nx=24, ny=12, mech=r)
    out = []
    for c in (ca, cb):
        s = ref.RefSolver(c.grid, c.mech); s.set_state(c.U, c.T); s.step(5, cfl=0.2); out.append(s.get_state()[0]); assert s.status == 0
    assert np.abs(out[0] - out[1]).max() <= 1e-6 * np.abs(out[0]).max()
