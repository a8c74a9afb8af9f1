"""Test helper: write an inputs.Mechanism (synthetic, seeded) as Chemkin-format text, so that the library's reader
(csrc/mechfile.h, janc_mech_parse) can be checked by a round trip without any real mechanism file.  The element symbols
of the synthetic species (a, b, c, n) are not real elements: their atomic weights go into the ELEMENTS section."""
import numpy as np

RU = 8.314472


def write(mech, elem_names=("EA", "EB", "EC", "EN"), elem_w=None, e_unit="CAL/MOLE", inline_thermo=True):
    ns, nr = mech.ns, mech.nr
    comp = np.asarray(mech.elements)
    ne = comp.shape[1]
    names = [f"S{k}" + "".join(f"{elem_names[e][1]}{comp[k, e]}" for e in range(ne) if comp[k, e]) for k in range(ns)]
    if elem_w is None:          # recover atomic weights (g/mol) from W = comp @ w
        elem_w = np.linalg.lstsq(comp.astype(float), mech.W * 1e3, rcond=None)[0]
    out = ["! synthetic mechanism written by tests/chemkin_writer.py", "ELEMENTS"]
    out.append("  " + "  ".join(f"{elem_names[e]} /{elem_w[e]:.10g}/" for e in range(ne)))
    out += ["END", "SPECIES", "  " + " ".join(names), "END"]
    lo = mech.nasa
    hi = mech.nasa_hi if getattr(mech, "nasa_hi", None) is not None else mech.nasa
    tm = mech.T_mid if getattr(mech, "T_mid", None) is not None else np.full(ns, 1000.0)
    th = ["THERMO ALL", "   200.000  1000.000  6000.000"]
    for k in range(ns):
        fields = [(elem_names[e], comp[k, e]) for e in range(ne) if comp[k, e]]
        compstr = "".join(f"{s:<2s}{c:>3d}" for s, c in fields[:4]).ljust(20)
        l1 = f"{names[k]:<18s}{'synth':<6s}{compstr}G{200.0:>10.3f}{6000.0:>10.3f}{tm[k]:>8.2f}"
        l1 = l1.ljust(79) + "1"
        e = lambda v: f"{v:15.8E}"
        l2 = "".join(e(hi[k, q]) for q in range(5)).ljust(79) + "2"
        l3 = (e(hi[k, 5]) + e(hi[k, 6]) + "".join(e(lo[k, q]) for q in range(3))).ljust(79) + "3"
        l4 = "".join(e(lo[k, q]) for q in range(3, 7)).ljust(79) + "4"
        th += [l1, l2, l3, l4]
    th.append("END")
    if inline_thermo:
        out += th
    scale = {"CAL/MOLE": RU / 4.184, "KCAL/MOLE": RU / 4184.0, "JOULES/MOLE": RU, "KELVINS": 1.0}[e_unit]
    out.append(f"REACTIONS {e_unit}")
    for i in range(nr):
        side = lambda nu: " + ".join((f"{int(nu[k])}" if nu[k] > 1 else "") + names[k] for k in range(ns) if nu[k] > 0)
        tb = bool(mech.third_body[i])
        lhs, rhs = side(mech.nu_f[i]), side(mech.nu_b[i])
        if tb:
            lhs += " + M"; rhs += " + M"
        order = int(mech.nu_f[i].sum()) + (1 if tb else 0)
        A_cgs = mech.A[i] / (1e-6) ** (order - 1)
        arrow = "<=>" if mech.reversible[i] and i % 2 else ("=" if mech.reversible[i] else "=>")
        out.append(f"{lhs} {arrow} {rhs}   {A_cgs:.16E}  {mech.b[i]:.16g}  {mech.Ta[i] * scale:.16E}   ! reaction {i}")
        if tb:
            out.append("   " + " ".join(f"{names[k]}/{mech.eff[i, k]:.16g}/" for k in range(ns)))
        if i % 7 == 3:
            out.append("  DUPLICATE")
    out.append("END")
    return "\n".join(out) + "\n", "\n".join(th) + "\n", names
