// mechfile.h -- Chemkin-format mechanism / thermo reader (host only): text -> the arrays of janc_mech.
// PAPER.md:279 ("a chemkin-format reader"), :400 (the H2-O2 mechanism file), :258 (two-range NASA-7 thermo data).
// The paper's solver reads its mechanism from such files; this library takes the mechanism as arrays (janc_set_mechanism)
// and offers this reader so that a user who HAS the files can run them.  No mechanism data ships with the library.
//
// What is read (the CHEMKIN-II input format, restated):
//   ELEMENTS / ELEM ... END      element symbols; "X /w/" gives an atomic weight in g/mol (needed for symbols that are
//                                not in the small built-in table)
//   SPECIES / SPEC ... END       species names, in the order of the state vector (the LAST one is the species carried
//                                by difference)
//   THERMO [ALL] ... END         one line "Tlow Tmid Thigh" (defaults), then 4 fixed-column lines per species:
//                                  1: cols 1-18 name, 25-44 four (2-char element, 3-char count) fields, 46-55 Tlow,
//                                     56-65 Thigh, 66-73 Tmid, 74-78 fifth element field
//                                  2: a1..a5 of the UPPER range (5 x E15.8)      3: a6 a7 upper, a1 a2 a3 lower
//                                  4: a4..a7 lower
//                                (may come as a separate text: "thermo file")
//   REACTIONS [units] ... END    "A + B <=> C + D   A_pre  b  E": "<=>" or "=" reversible, "=>" irreversible; "+ M"
//                                third body with an auxiliary line "SP/eff/ SP/eff/"; DUP lines are skipped.  Units:
//                                A in cm-mol-s, E in cal/mol unless KCAL/MOLE, JOULES/MOLE, KJOULES/MOLE or KELVINS is
//                                given.  Pressure-dependent forms ((+M), LOW, TROE, SRI, PLOG), REV, FORD, ions and
//                                real stoichiometric coefficients are not part of eq 4.6-4.9: rejected with a message.
// '!' starts a comment.  Output in SI: W kg/mol, A in (mol, m^3, s), Ta = E / R_u in K.
#pragma once
#include <cctype>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <sstream>
#include <string>
#include <vector>

#include "../../include/janc.h"

struct janc_mech_file {
  std::vector<std::string> species, elements;
  std::vector<double> W, nasa, nasa_hi, T_mid, A, b, Ta, eff, elem_w;
  std::vector<int32_t> nu_f, nu_b, reversible, third_body, comp;   // comp[ns][ne]
  std::string err;
};

namespace mechfile {

inline std::string upper(std::string s) { for (auto &c : s) c = (char)toupper((unsigned char)c); return s; }
inline std::string strip(const std::string &s) {
  size_t a = 0, b = s.size();
  while (a < b && isspace((unsigned char)s[a])) a++;
  while (b > a && isspace((unsigned char)s[b - 1])) b--;
  return s.substr(a, b - a);
}
inline std::vector<std::string> lines_of(const char *text) {
  std::vector<std::string> out;
  std::string cur;
  for (const char *p = text; *p; p++) {
    if (*p == '\n') { out.push_back(cur); cur.clear(); }
    else if (*p != '\r') cur += *p;
  }
  if (!cur.empty()) out.push_back(cur);
  return out;
}
inline std::string no_comment(const std::string &l) { size_t k = l.find('!'); return k == std::string::npos ? l : l.substr(0, k); }
inline std::vector<std::string> tokens(const std::string &s) {
  std::vector<std::string> t; std::istringstream is(s); std::string w;
  while (is >> w) t.push_back(w);
  return t;
}
inline bool to_double(std::string s, double &v) {
  for (auto &c : s) if (c == 'D' || c == 'd') c = 'E';      // Fortran exponents
  char *end = nullptr;
  v = strtod(s.c_str(), &end);
  return end && *end == 0 && !s.empty();
}
inline double field(const std::string &l, size_t a, size_t n, bool &ok) {
  if (l.size() <= a) { ok = false; return 0.0; }
  double v = 0.0;
  if (!to_double(strip(l.substr(a, n)), v)) ok = false;
  return v;
}
// atomic weights in g/mol for the symbols combustion mechanisms use; anything else must come as "X /w/"
inline double builtin_weight(const std::string &e) {
  static const std::map<std::string, double> w = {{"H", 1.00794}, {"D", 2.014102}, {"HE", 4.002602}, {"C", 12.0107}, {"N", 14.0067},
                                                   {"O", 15.9994}, {"F", 18.9984032}, {"NE", 20.1797}, {"S", 32.065}, {"CL", 35.453},
                                                   {"AR", 39.948}, {"KR", 83.798}, {"XE", 131.293}};
  auto it = w.find(e);
  return it == w.end() ? -1.0 : it->second;
}

}  // namespace mechfile

namespace mechfile {

// one side of a reaction: species counts, whether a third body "M" appears; false + err on anything unsupported
inline bool parse_side(const std::string &side, const std::map<std::string, int> &sp, std::vector<int> &nu, bool &has_M, std::string &err) {
  has_M = false;
  if (side.find("(+") != std::string::npos) { err = "pressure-dependent (fall-off) reactions are not supported"; return false; }
  std::string cur;
  std::vector<std::string> parts;
  for (char c : side) {
    if (c == '+') { parts.push_back(strip(cur)); cur.clear(); }
    else cur += c;
  }
  parts.push_back(strip(cur));
  for (std::string t : parts) {
    if (t.empty()) { err = "empty species in '" + side + "'"; return false; }
    int mult = 1;
    size_t d = 0;
    while (d < t.size() && isdigit((unsigned char)t[d])) d++;
    // a leading integer is a stoichiometric coefficient unless the whole token is a species name
    std::string name = upper(t);
    if (sp.find(name) == sp.end() && d > 0) {
      mult = atoi(t.substr(0, d).c_str());
      name = upper(strip(t.substr(d)));
      if (!name.empty() && name[0] == '.') { err = "real stoichiometric coefficients are not supported"; return false; }
    }
    if (name == "M") { has_M = true; continue; }
    auto it = sp.find(name);
    if (it == sp.end()) { err = "unknown species '" + t + "'"; return false; }
    nu[it->second] += mult;
  }
  return true;
}

inline bool parse(const char *mech_text, const char *thermo_text, janc_mech_file &F) {
  enum { NONE, ELEM, SPEC, THERMO, REAC } sec = NONE;
  std::map<std::string, int> spidx, elidx;
  std::vector<std::string> thermo_lines;
  struct Rx { std::vector<int> f, b; double A, bb, E; bool rev, tb; std::vector<double> eff; };
  std::vector<Rx> rx;
  double e_to_K = 4.184 / 8.314472;          // default cal/mol -> K (E / R_u)
  bool thermo_all_inline = false;
  for (const std::string &raw : lines_of(mech_text)) {
    if (sec == THERMO) {                      // fixed columns: keep the line as it is (comments start at '!' in column 1 only)
      const std::string u = upper(strip(raw));
      if (u.rfind("END", 0) == 0) { sec = NONE; continue; }
      if (u.rfind("REAC", 0) == 0) { sec = REAC; }     // some files omit END before REACTIONS
      else { if (!raw.empty() && raw[0] != '!') thermo_lines.push_back(raw); continue; }
    }
    std::string l = strip(no_comment(raw));
    if (l.empty()) continue;
    std::vector<std::string> t = tokens(l);
    const std::string k0 = upper(t[0]);
    if (k0.rfind("ELEM", 0) == 0) { sec = ELEM; t.erase(t.begin()); }
    else if (k0.rfind("SPEC", 0) == 0) { sec = SPEC; t.erase(t.begin()); }
    else if (k0.rfind("THER", 0) == 0) { sec = THERMO; thermo_all_inline = true; continue; }
    else if (k0.rfind("REAC", 0) == 0) {
      sec = REAC;
      for (size_t q = 1; q < t.size(); q++) {
        const std::string u = upper(t[q]);
        if (u == "CAL/MOLE") e_to_K = 4.184 / 8.314472;
        else if (u == "KCAL/MOLE") e_to_K = 4184.0 / 8.314472;
        else if (u == "JOULES/MOLE") e_to_K = 1.0 / 8.314472;
        else if (u == "KJOULES/MOLE" || u == "KJOU/MOLE") e_to_K = 1000.0 / 8.314472;
        else if (u == "KELVINS" || u == "KELVIN") e_to_K = 1.0;
        else if (u == "MOLES") {}
        else { F.err = "REACTIONS unit keyword '" + t[q] + "' is not supported"; return false; }
      }
      continue;
    }
    if (sec == NONE) { F.err = "text outside a section: '" + l + "'"; return false; }
    if (sec == ELEM || sec == SPEC) {
      // items are NAME or NAME /w/ (atomic weight in g/mol, elements only), blanks optional around the slashes
      std::string joined;
      for (auto &w : t) joined += w + " ";
      size_t q = 0;
      while (q < joined.size()) {
        while (q < joined.size() && isspace((unsigned char)joined[q])) q++;
        if (q >= joined.size()) break;
        size_t e = q;
        while (e < joined.size() && !isspace((unsigned char)joined[e]) && joined[e] != '/') e++;
        const std::string name = upper(joined.substr(q, e - q));
        q = e;
        while (q < joined.size() && isspace((unsigned char)joined[q])) q++;
        std::string wt;
        if (q < joined.size() && joined[q] == '/') {
          size_t e2 = joined.find('/', q + 1);
          if (e2 == std::string::npos) { F.err = "unterminated '/' in '" + l + "'"; return false; }
          wt = strip(joined.substr(q + 1, e2 - q - 1));
          q = e2 + 1;
        }
        if (name.empty()) { F.err = "cannot read '" + l + "'"; return false; }
        if (name == "END") { sec = NONE; break; }
        if (sec == ELEM) {
          double v = builtin_weight(name);
          if (!wt.empty() && (!to_double(wt, v) || !(v > 0))) { F.err = "bad atomic weight for " + name; return false; }
          if (elidx.count(name)) { F.elem_w[elidx[name]] = v; continue; }
          elidx[name] = (int)F.elements.size(); F.elements.push_back(name); F.elem_w.push_back(v);
        } else {
          if (!wt.empty()) { F.err = "'/" + wt + "/' after species " + name; return false; }
          if (spidx.count(name)) { F.err = "species '" + name + "' listed twice"; return false; }
          spidx[name] = (int)F.species.size(); F.species.push_back(name);
        }
      }
      continue;
    }
    // ---- REACTIONS section
    if (k0 == "END") { sec = NONE; continue; }
    if (k0.rfind("DUP", 0) == 0) continue;
    const int ns = (int)F.species.size();
    if (l.find('=') == std::string::npos) {       // auxiliary line of the previous reaction
      if (rx.empty()) { F.err = "auxiliary line before any reaction: '" + l + "'"; return false; }
      const std::string u = upper(l);
      for (const char *kw : {"LOW", "TROE", "SRI", "PLOG", "REV", "FORD", "RORD", "HIGH", "LT", "RLT", "CHEB", "TCHEB", "PCHEB", "UNITS", "EXCI", "XSMI", "MOME", "FIT1", "JAN"})
        if (u.rfind(kw, 0) == 0 && (u.size() == strlen(kw) || !isalnum((unsigned char)u[strlen(kw)]))) { F.err = std::string("auxiliary keyword ") + kw + " is not supported (eq 4.6-4.9 have Arrhenius rates with third-body efficiencies only)"; return false; }
      if (!rx.back().tb) { F.err = "efficiencies given for a reaction without +M: '" + l + "'"; return false; }
      // SP/eff/ SP/eff/ ...
      std::string rest = l;
      while (true) {
        rest = strip(rest);
        if (rest.empty()) break;
        size_t s1 = rest.find('/'); if (s1 == std::string::npos) { F.err = "cannot read efficiencies '" + l + "'"; return false; }
        size_t s2 = rest.find('/', s1 + 1); if (s2 == std::string::npos) { F.err = "cannot read efficiencies '" + l + "'"; return false; }
        const std::string nm = upper(strip(rest.substr(0, s1)));
        double v; if (!to_double(strip(rest.substr(s1 + 1, s2 - s1 - 1)), v)) { F.err = "bad efficiency in '" + l + "'"; return false; }
        auto it = spidx.find(nm); if (it == spidx.end()) { F.err = "efficiency for unknown species '" + nm + "'"; return false; }
        rx.back().eff[it->second] = v;
        rest = rest.substr(s2 + 1);
      }
      continue;
    }
    if (t.size() < 4) { F.err = "reaction line needs an equation and A, b, E: '" + l + "'"; return false; }
    Rx r; r.f.assign(ns, 0); r.b.assign(ns, 0); r.eff.assign(ns, 1.0);
    if (!to_double(t[t.size() - 3], r.A) || !to_double(t[t.size() - 2], r.bb) || !to_double(t[t.size() - 1], r.E)) { F.err = "cannot read A, b, E in '" + l + "'"; return false; }
    std::string eq;
    for (size_t q = 0; q + 3 < t.size(); q++) eq += t[q];
    size_t pos; std::string lhs, rhs;
    if ((pos = eq.find("<=>")) != std::string::npos) { lhs = eq.substr(0, pos); rhs = eq.substr(pos + 3); r.rev = true; }
    else if ((pos = eq.find("=>")) != std::string::npos) { lhs = eq.substr(0, pos); rhs = eq.substr(pos + 2); r.rev = false; }
    else { pos = eq.find('='); lhs = eq.substr(0, pos); rhs = eq.substr(pos + 1); r.rev = true; }
    bool mf = false, mb = false;
    if (!parse_side(lhs, spidx, r.f, mf, F.err) || !parse_side(rhs, spidx, r.b, mb, F.err)) { F.err += " in '" + l + "'"; return false; }
    if (mf != mb) { F.err = "third body on one side only in '" + l + "'"; return false; }
    r.tb = mf;
    rx.push_back(r);
  }
  // ---- THERMO: the mechanism's own section, else the separate thermo text
  if (thermo_text && *thermo_text) {
    bool in = false;
    for (const std::string &raw : lines_of(thermo_text)) {
      const std::string u = upper(strip(raw));
      if (u.rfind("THER", 0) == 0) { in = true; continue; }
      if (u.rfind("END", 0) == 0) { if (in) break; continue; }
      if (!raw.empty() && raw[0] != '!' && !u.empty()) thermo_lines.push_back(raw);
    }
  } else if (!thermo_all_inline) { F.err = "no THERMO section and no thermo text"; return false; }
  const int ns = (int)F.species.size(), ne = (int)F.elements.size(), nr = (int)rx.size();
  if (ns < 1) { F.err = "no species"; return false; }
  F.nasa.assign((size_t)ns * 7, 0.0); F.nasa_hi.assign((size_t)ns * 7, 0.0); F.T_mid.assign(ns, 0.0);
  F.comp.assign((size_t)ns * ne, 0);
  std::vector<char> have(ns, 0);
  double Tmid_default = 1000.0;
  size_t li = 0;
  if (!thermo_lines.empty()) {            // "Tlow Tmid Thigh" line: three numbers and nothing in column 80
    std::vector<std::string> t = tokens(thermo_lines[0]);
    double v0, v1, v2;
    if (t.size() == 3 && to_double(t[0], v0) && to_double(t[1], v1) && to_double(t[2], v2)) { Tmid_default = v1; li = 1; }
  }
  while (li + 3 < thermo_lines.size() + 0 && li < thermo_lines.size()) {
    if (li + 3 >= thermo_lines.size()) break;
    const std::string &l1 = thermo_lines[li], &l2 = thermo_lines[li + 1], &l3 = thermo_lines[li + 2], &l4 = thermo_lines[li + 3];
    li += 4;
    const std::vector<std::string> nt = tokens(l1.substr(0, std::min<size_t>(18, l1.size())));
    if (nt.empty()) { F.err = "thermo entry without a species name: '" + l1 + "'"; return false; }
    auto it = spidx.find(upper(nt[0]));
    if (it == spidx.end()) continue;                                       // data for a species the mechanism does not use
    const int k = it->second;
    bool ok = true;
    double up[7], lo[7];
    for (int q = 0; q < 5; q++) up[q] = field(l2, 15 * q, 15, ok);
    up[5] = field(l3, 0, 15, ok); up[6] = field(l3, 15, 15, ok);
    for (int q = 0; q < 3; q++) lo[q] = field(l3, 30 + 15 * q, 15, ok);
    for (int q = 0; q < 4; q++) lo[3 + q] = field(l4, 15 * q, 15, ok);
    if (!ok) { F.err = "cannot read the NASA coefficients of " + F.species[k]; return false; }
    double tm = Tmid_default;
    if (l1.size() > 65) { double v; if (to_double(strip(l1.substr(65, 8)), v) && v > 0) tm = v; }
    for (int q = 0; q < 7; q++) { F.nasa[(size_t)k * 7 + q] = lo[q]; F.nasa_hi[(size_t)k * 7 + q] = up[q]; }
    F.T_mid[k] = tm;
    // element composition: four 5-column fields from column 25, a fifth at column 74
    for (int fld = 0; fld < 5; fld++) {
      const size_t c0 = fld < 4 ? 24 + 5 * fld : 73;
      if (l1.size() < c0 + 5) continue;
      const std::string sym = upper(strip(l1.substr(c0, 2)));
      double cnt = 0.0;
      if (sym.empty() || !to_double(strip(l1.substr(c0 + 2, 3)), cnt) || cnt == 0.0) continue;
      auto ie = elidx.find(sym);
      if (ie == elidx.end()) { F.err = "species " + F.species[k] + " contains element " + sym + " which is not in ELEMENTS"; return false; }
      F.comp[(size_t)k * ne + ie->second] += (int32_t)llround(cnt);
    }
    have[k] = 1;
  }
  F.W.assign(ns, 0.0);
  for (int k = 0; k < ns; k++) {
    if (!have[k]) { F.err = "no thermo data for species " + F.species[k]; return false; }
    for (int e = 0; e < ne; e++) {
      if (F.comp[(size_t)k * ne + e] && !(F.elem_w[e] > 0)) { F.err = "no atomic weight for element " + F.elements[e] + " (give it as " + F.elements[e] + " /w/)"; return false; }
      F.W[k] += 1e-3 * F.elem_w[e] * F.comp[(size_t)k * ne + e];
    }
    if (!(F.W[k] > 0)) { F.err = "species " + F.species[k] + " has no elements"; return false; }
  }
  // ---- reactions in SI
  F.nu_f.assign((size_t)nr * ns, 0); F.nu_b.assign((size_t)nr * ns, 0);
  F.A.resize(nr); F.b.resize(nr); F.Ta.resize(nr); F.reversible.resize(nr); F.third_body.resize(nr); F.eff.assign((size_t)nr * ns, 1.0);
  for (int i = 0; i < nr; i++) {
    int order = rx[i].tb ? 1 : 0;
    for (int k = 0; k < ns; k++) {
      F.nu_f[(size_t)i * ns + k] = rx[i].f[k]; F.nu_b[(size_t)i * ns + k] = rx[i].b[k];
      F.eff[(size_t)i * ns + k] = rx[i].eff[k];
      order += rx[i].f[k];
    }
    F.A[i] = rx[i].A * pow(1e-6, order - 1);        // cm^3 -> m^3 per mole, (order - 1) times
    F.b[i] = rx[i].bb; F.Ta[i] = rx[i].E * e_to_K;
    F.reversible[i] = rx[i].rev ? 1 : 0; F.third_body[i] = rx[i].tb ? 1 : 0;
  }
  return true;
}

}  // namespace mechfile
