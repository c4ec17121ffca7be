/*
 * ckb_chemkin.cu -- host-side preprocessing (no kernels): a reader for mechanisms in the Chemkin text format and the
 * paper's reversible -> irreversible converter (Appendix A; "we converted all such reversible
 * reactions into two irreversible reactions"; the paper's kernels were generated from such files).
 * Output: the arrays of ckb_mech_desc / ckb_mech_load3, owned by the ckb_chemkin object.  SURVEY 8(f)-f2.
 *
 * Supported: ELEMENTS, SPECIES, THERMO (7-coefficient fits, two ranges), REACTIONS with units CAL/MOLE (default),
 * KCAL/MOLE, JOULES/MOLE, KJOULES/MOLE, KELVINS and MOLES (default) / MOLECULES; "=" / "<=>" reversible and "=>"
 * irreversible reactions; integer stoichiometric coefficients as prefixes or repeated species; "+M" with efficiencies;
 * "(+M)" with LOW and optional TROE; REV; DUPLICATE.  Anything else (SRI, PLOG, CHEB, FORD, specific colliders "(+X)",
 * real coefficients, ...) is refused with CKB_EUNSUPPORTED and a message (ckb_chemkin_error).
 */
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <sstream>
#include <string>
#include <vector>

#include "../../include/ckb.h"

namespace {

constexpr double RU = 8.314462618e7;     /* erg/(mol K), R20 */
constexpr double RC = 1.98720425864;     /* cal/(mol K), R20 */
constexpr double P_ATM = 1.01325e6;      /* dyn/cm^2 */
constexpr double AVOGADRO = 6.02214076e23;

thread_local std::string g_err;

struct Fail {
  int code;
};
[[noreturn]] void fail(int code, const std::string &msg) {
  g_err = msg;
  throw Fail{code};
}

std::string upper(std::string s) {
  for (auto &c : s) c = (char)std::toupper((unsigned char)c);
  return s;
}
std::vector<std::string> tokens(const std::string &s) {
  std::istringstream is(s);
  std::vector<std::string> t;
  std::string w;
  while (is >> w) t.push_back(w);
  return t;
}
bool to_number(const std::string &w, double *out) {
  std::string t = w;
  for (auto &c : t)
    if (c == 'D' || c == 'd') c = 'E'; /* Fortran exponents */
  char *end = nullptr;
  const double v = std::strtod(t.c_str(), &end);
  if (end == t.c_str() || *end != '\0') return false;
  *out = v;
  return true;
}
double field(const std::string &line, size_t pos, size_t len, bool *ok = nullptr) {
  double v = 0.0;
  bool good = false;
  if (pos < line.size()) {
    std::vector<std::string> t = tokens(line.substr(pos, len));
    if (t.size() == 1) good = to_number(t[0], &v);
  }
  if (ok) *ok = good;
  return v;
}

const std::map<std::string, double> &atomic_weights() {
  static const std::map<std::string, double> w = {
      {"H", 1.008},   {"D", 2.014},   {"HE", 4.002602}, {"C", 12.011},  {"N", 14.007},  {"O", 15.999},
      {"F", 18.998},  {"NE", 20.1797}, {"SI", 28.085},  {"S", 32.06},   {"CL", 35.45},  {"AR", 39.948},
      {"KR", 83.798}, {"E", 5.4858e-4}};
  return w;
}

struct Species {
  std::string name;
  std::map<std::string, double> comp;
  double lo[7], hi[7], Tlow, Thigh, Tmid, W;
  bool have_thermo = false;
};

struct Side {
  std::vector<std::pair<int, int>> sp; /* (species, nu) merged */
};

struct Reaction {
  Side reac, prod;
  bool reversible = false, third_body = false, falloff = false, have_rev = false, have_low = false, have_troe = false,
       dup = false;
  double A = 0, b = 0, E = 0, revA = 0, revb = 0, revE = 0, low[3] = {0, 0, 0}, troe[4] = {0, 0, 0, 0};
  int n_troe = 0;
  std::map<int, double> eff;
  int line = 0;
  std::string text;
};

}  // namespace

struct ckb_chemkin {
  std::vector<std::string> elements;
  std::vector<Species> species;
  std::vector<Reaction> input;
  /* the irreversible mechanism */
  std::vector<double> W, nasa, nasa_hi, Tmid, A, beta, E, tb_eff, fo_low, fo_troe;
  std::vector<int32_t> reac_ptr, reac_sp, reac_nu, prod_ptr, prod_sp, prod_nu, tb_reaction, tb_ptr, tb_species, fo_reaction,
      origin, reversed;
};

namespace {

int species_index(const ckb_chemkin &ck, const std::string &name) {
  for (size_t k = 0; k < ck.species.size(); k++)
    if (ck.species[k].name == name) return (int)k;
  return -1;
}

void parse_thermo(ckb_chemkin &ck, const std::vector<std::string> &lines) {
  size_t i = 0;
  double dlo = 300.0, dmid = 1000.0, dhi = 5000.0;
  /* optional line with the three default temperatures */
  if (i < lines.size()) {
    std::vector<std::string> t = tokens(lines[i]);
    double a, b, c;
    if (t.size() == 3 && to_number(t[0], &a) && to_number(t[1], &b) && to_number(t[2], &c)) {
      dlo = a; dmid = b; dhi = c;
      i++;
    }
  }
  while (i + 3 < lines.size()) { /* records of four lines */
    const std::string &l1 = lines[i];
    const std::string name = tokens(l1.substr(0, 18)).empty() ? std::string() : tokens(l1.substr(0, 18))[0];
    const int k = species_index(ck, name);
    if (k >= 0 && !ck.species[k].have_thermo) {
      Species &s = ck.species[k];
      for (int q = 0; q < 4; q++) { /* element fields: 2 characters + 3 for the count */
        const size_t p = 24 + 5 * (size_t)q;
        if (p + 2 > l1.size()) break;
        std::vector<std::string> e = tokens(l1.substr(p, 2));
        if (e.empty() || e[0] == "0") continue;
        bool ok = false;
        const double cnt = field(l1, p + 2, 3, &ok);
        if (ok && cnt != 0.0) s.comp[e[0]] += cnt;
      }
      bool ok;
      s.Tlow = field(l1, 45, 10, &ok); if (!ok) s.Tlow = dlo;
      s.Thigh = field(l1, 55, 10, &ok); if (!ok) s.Thigh = dhi;
      s.Tmid = field(l1, 65, 8, &ok); if (!ok) s.Tmid = dmid;
      double c[15];
      for (int q = 0; q < 15; q++) {
        const std::string &ln = lines[i + 1 + q / 5];
        c[q] = field(ln, 15 * (size_t)(q % 5), 15, &ok);
        if (!ok && q < 14) fail(CKB_EINVAL, "thermo: unreadable coefficient " + std::to_string(q + 1) + " of " + name);
      }
      for (int q = 0; q < 7; q++) { s.hi[q] = c[q]; s.lo[q] = c[7 + q]; }
      s.W = 0.0;
      for (auto &kv : s.comp) {
        auto it = atomic_weights().find(kv.first);
        if (it == atomic_weights().end()) fail(CKB_EUNSUPPORTED, "thermo: no atomic weight for element " + kv.first);
        s.W += kv.second * it->second;
      }
      if (!(s.W > 0.0)) fail(CKB_EINVAL, "thermo: species " + name + " has no composition");
      s.have_thermo = true;
    }
    i += 4;
  }
}

Side parse_side(const ckb_chemkin &ck, std::string s, Reaction &r, const std::string &ctx) {
  size_t p;
  while ((p = s.find("(+M)")) != std::string::npos) { /* fall-off */
    r.falloff = true;
    s.erase(p, 4);
  }
  if (s.find("(+") != std::string::npos) fail(CKB_EUNSUPPORTED, "specific collider in " + ctx);
  std::map<int, int> merged;
  std::vector<int> order;
  size_t start = 0;
  while (start <= s.size()) {
    size_t plus = s.find('+', start);
    /* a '+' that ends the string or is followed by another '+' belongs to an ion name: not supported */
    std::string term = s.substr(start, plus == std::string::npos ? std::string::npos : plus - start);
    if (term.empty()) fail(CKB_EINVAL, "empty term in " + ctx);
    if (term == "M") {
      r.third_body = true;
    } else {
      int nu = 1, k = species_index(ck, term);
      if (k < 0) {
        size_t d = 0;
        while (d < term.size() && std::isdigit((unsigned char)term[d])) d++;
        if (d == 0 || d == term.size()) {
          if (term.find('.') != std::string::npos) fail(CKB_EUNSUPPORTED, "real stoichiometric coefficient in " + ctx);
          fail(CKB_EINVAL, "unknown species " + term + " in " + ctx);
        }
        nu = std::atoi(term.substr(0, d).c_str());
        k = species_index(ck, term.substr(d));
        if (k < 0) fail(CKB_EINVAL, "unknown species " + term.substr(d) + " in " + ctx);
      }
      if (!merged.count(k)) order.push_back(k);
      merged[k] += nu;
    }
    if (plus == std::string::npos) break;
    start = plus + 1;
  }
  Side out;
  for (int k : order) out.sp.push_back({k, merged[k]});
  return out;
}

double energy_to_cal(double E, const std::string &unit) {
  if (unit == "CAL/MOLE") return E;
  if (unit == "KCAL/MOLE") return E * 1000.0;
  if (unit == "JOULES/MOLE") return E / 4.184;
  if (unit == "KJOULES/MOLE" || unit == "KJOU/MOLE") return E * 1000.0 / 4.184;
  if (unit == "KELVINS" || unit == "KELVIN") return E * RC;
  fail(CKB_EUNSUPPORTED, "energy unit " + unit);
}

void parse_reactions(ckb_chemkin &ck, const std::vector<std::pair<int, std::string>> &lines, const std::string &header) {
  std::string eunit = "CAL/MOLE";
  bool molecules = false;
  for (const std::string &t : tokens(header)) {
    if (t == "REACTIONS" || t == "REAC") continue;
    if (t == "MOLES") molecules = false;
    else if (t == "MOLECULES") molecules = true;
    else eunit = t;
  }
  energy_to_cal(0.0, eunit);
  for (auto &ln : lines) {
    const std::string &text = ln.second;
    std::vector<std::string> t = tokens(text);
    if (t.empty()) continue;
    const std::string ctx = "line " + std::to_string(ln.first) + ": " + text;
    const bool aux = text.find('/') != std::string::npos;
    if (!aux && (t[0] == "DUP" || t[0] == "DUPLICATE")) {
      if (ck.input.empty()) fail(CKB_EINVAL, "DUPLICATE before any reaction, " + ctx);
      ck.input.back().dup = true;
      continue;
    }
    if (aux) { /* KEYWORD / values / ... */
      if (ck.input.empty()) fail(CKB_EINVAL, "auxiliary data before any reaction, " + ctx);
      Reaction &r = ck.input.back();
      size_t p = 0;
      while (true) {
        size_t s1 = text.find('/', p);
        if (s1 == std::string::npos) break;
        size_t s2 = text.find('/', s1 + 1);
        if (s2 == std::string::npos) fail(CKB_EINVAL, "unbalanced '/' in " + ctx);
        std::vector<std::string> kw = tokens(text.substr(p, s1 - p));
        std::vector<std::string> vals = tokens(text.substr(s1 + 1, s2 - s1 - 1));
        if (kw.size() != 1) fail(CKB_EINVAL, "bad auxiliary keyword in " + ctx);
        std::vector<double> v(vals.size());
        for (size_t q = 0; q < vals.size(); q++)
          if (!to_number(vals[q], &v[q])) fail(CKB_EINVAL, "bad number in " + ctx);
        if (kw[0] == "LOW") {
          if (v.size() != 3) fail(CKB_EINVAL, "LOW needs three values, " + ctx);
          r.have_low = true;
          for (int q = 0; q < 3; q++) r.low[q] = v[q];
        } else if (kw[0] == "TROE") {
          if (v.size() != 3 && v.size() != 4) fail(CKB_EINVAL, "TROE needs three or four values, " + ctx);
          r.have_troe = true;
          r.n_troe = (int)v.size();
          for (size_t q = 0; q < v.size(); q++) r.troe[q] = v[q];
        } else if (kw[0] == "REV") {
          if (v.size() != 3) fail(CKB_EINVAL, "REV needs three values, " + ctx);
          r.have_rev = true;
          r.revA = v[0]; r.revb = v[1]; r.revE = v[2];
        } else {
          const int k = species_index(ck, kw[0]);
          if (k < 0) fail(CKB_EUNSUPPORTED, "auxiliary keyword " + kw[0] + " in " + ctx);
          if (v.size() != 1) fail(CKB_EINVAL, "efficiency needs one value, " + ctx);
          r.eff[k] = v[0];
        }
        p = s2 + 1;
      }
      continue;
    }
    /* reaction line: equation (may contain blanks) followed by A, beta, E */
    if (t.size() < 4) fail(CKB_EINVAL, "reaction needs an equation and three numbers, " + ctx);
    Reaction r;
    r.line = ln.first;
    double num[3];
    for (int q = 0; q < 3; q++)
      if (!to_number(t[t.size() - 3 + q], &num[q])) fail(CKB_EINVAL, "bad Arrhenius parameter in " + ctx);
    std::string eq;
    for (size_t q = 0; q + 3 < t.size(); q++) eq += t[q];
    r.text = eq;
    size_t pos, len;
    if ((pos = eq.find("<=>")) != std::string::npos) { len = 3; r.reversible = true; }
    else if ((pos = eq.find("=>")) != std::string::npos) { len = 2; r.reversible = false; }
    else if ((pos = eq.find('=')) != std::string::npos) { len = 1; r.reversible = true; }
    else fail(CKB_EINVAL, "no '=' in " + ctx);
    Reaction lhs, rhs;
    r.reac = parse_side(ck, eq.substr(0, pos), lhs, ctx);
    r.prod = parse_side(ck, eq.substr(pos + len), rhs, ctx);
    if (lhs.third_body != rhs.third_body || lhs.falloff != rhs.falloff) fail(CKB_EINVAL, "third body on one side only, " + ctx);
    r.third_body = lhs.third_body;
    r.falloff = lhs.falloff;
    r.A = num[0]; r.b = num[1]; r.E = num[2];
    /* element balance */
    std::map<std::string, double> bal;
    for (auto &e : r.reac.sp) for (auto &kv : ck.species[e.first].comp) bal[kv.first] -= e.second * kv.second;
    for (auto &e : r.prod.sp) for (auto &kv : ck.species[e.first].comp) bal[kv.first] += e.second * kv.second;
    for (auto &kv : bal)
      if (std::fabs(kv.second) > 1e-9) fail(CKB_EINVAL, "element " + kv.first + " not balanced in " + ctx);
    ck.input.push_back(r);
  }
  /* units -> cal/mol, mol-cm-s */
  for (Reaction &r : ck.input) {
    int order_f = (r.third_body ? 1 : 0), order_r = order_f;
    for (auto &e : r.reac.sp) order_f += e.second;
    for (auto &e : r.prod.sp) order_r += e.second;
    r.E = energy_to_cal(r.E, eunit);
    r.revE = energy_to_cal(r.revE, eunit);
    r.low[2] = energy_to_cal(r.low[2], eunit);
    if (molecules) {
      r.A *= std::pow(AVOGADRO, order_f - 1);
      r.revA *= std::pow(AVOGADRO, order_r - 1);
      r.low[0] *= std::pow(AVOGADRO, order_f); /* k_0 carries one more concentration */
    }
    if (r.falloff && !r.have_low) fail(CKB_EINVAL, "(+M) without LOW, reaction " + r.text);
    if (!r.falloff && (r.have_low || r.have_troe)) fail(CKB_EINVAL, "LOW / TROE without (+M), reaction " + r.text);
    if (r.have_rev && !r.reversible) fail(CKB_EINVAL, "REV on an irreversible reaction, " + r.text);
    if (r.have_rev && r.falloff) fail(CKB_EUNSUPPORTED, "REV on a fall-off reaction, " + r.text);
  }
}

/* ln K_c of an input reaction at T: Chemkin form (reading R32) */
double ln_Kc(const ckb_chemkin &ck, const Reaction &r, double T) {
  double dG = 0.0;
  int dnu = 0;
  auto add = [&](const Side &s, int sign) {
    for (auto &e : s.sp) {
      const Species &sp = ck.species[e.first];
      const double *a = T > sp.Tmid ? sp.hi : sp.lo;
      const double sR = a[0] * std::log(T) + T * (a[1] + T * (a[2] / 2.0 + T * (a[3] / 3.0 + T * a[4] / 4.0))) + a[6];
      const double hRT = a[0] + T * (a[1] / 2.0 + T * (a[2] / 3.0 + T * (a[3] / 4.0 + T * a[4] / 5.0))) + a[5] / T;
      dG += sign * e.second * (sR - hRT);
      dnu += sign * e.second;
    }
  };
  add(r.prod, 1);
  add(r.reac, -1);
  return dG + dnu * std::log(P_ATM / (RU * T));
}

/* Appendix A, Eq. A.10-A.12: Arrhenius parameters through three (T, ln k) points */
void fit3(const double *T, const double *a, double *A, double *beta, double *E) {
  const double x1 = std::log(T[0]), x2 = std::log(T[1]), x3 = std::log(T[2]);
  const double T1 = T[0], T2 = T[1], T3 = T[2];
  const double den = x1 * T1 * (T3 - T2) + x2 * T2 * (T1 - T3) + x3 * T3 * (T2 - T1);
  *beta = (a[0] * T1 * (T3 - T2) + a[1] * T2 * (T1 - T3) + a[2] * T3 * (T2 - T1)) / den;
  const double Tar = T1 * T2 * T3 * (a[0] * (x2 - x3) + a[1] * (x3 - x1) + a[2] * (x1 - x2)) / den;
  const double lnA = (a[0] * T1 * (x2 * T2 - x3 * T3) + a[1] * T2 * (x3 * T3 - x1 * T1) + a[2] * T3 * (x1 * T1 - x2 * T2)) / den;
  *A = std::exp(lnA);
  *E = Tar * RC;
}

void emit(ckb_chemkin &ck, const Reaction &r, int origin, bool reverse, double A, double b, double E, const double *low) {
  const int j = (int)ck.A.size();
  const Side &lhs = reverse ? r.prod : r.reac, &rhs = reverse ? r.reac : r.prod;
  for (auto &e : lhs.sp) { ck.reac_sp.push_back(e.first); ck.reac_nu.push_back(e.second); }
  for (auto &e : rhs.sp) { ck.prod_sp.push_back(e.first); ck.prod_nu.push_back(e.second); }
  ck.reac_ptr.push_back((int32_t)ck.reac_sp.size());
  ck.prod_ptr.push_back((int32_t)ck.prod_sp.size());
  ck.A.push_back(A); ck.beta.push_back(b); ck.E.push_back(E);
  ck.origin.push_back(origin);
  ck.reversed.push_back(reverse ? 1 : 0);
  if (r.third_body || (r.falloff && !r.eff.empty())) {
    ck.tb_reaction.push_back(j);
    for (auto &kv : r.eff) { ck.tb_species.push_back(kv.first); ck.tb_eff.push_back(kv.second); }
    ck.tb_ptr.push_back((int32_t)ck.tb_species.size());
  }
  if (r.falloff) {
    ck.fo_reaction.push_back(j);
    for (int q = 0; q < 3; q++) ck.fo_low.push_back(low[q]);
    const double nan = std::numeric_limits<double>::quiet_NaN(), inf = std::numeric_limits<double>::infinity();
    if (r.have_troe) {
      ck.fo_troe.push_back(r.troe[0]);
      ck.fo_troe.push_back(r.troe[1]);
      ck.fo_troe.push_back(r.troe[2]);
      ck.fo_troe.push_back(r.n_troe == 4 ? r.troe[3] : inf);
    } else {
      ck.fo_troe.push_back(nan);
      for (int q = 0; q < 3; q++) ck.fo_troe.push_back(inf);
    }
  }
}

void convert(ckb_chemkin &ck, const double *T3) {
  const int K = (int)ck.species.size();
  for (int k = 0; k < K; k++) {
    const Species &s = ck.species[k];
    if (!s.have_thermo) fail(CKB_EINVAL, "no thermodynamic data for species " + s.name);
    ck.W.push_back(s.W);
    ck.Tmid.push_back(s.Tmid);
    for (int q = 0; q < 7; q++) { ck.nasa.push_back(s.lo[q]); ck.nasa_hi.push_back(s.hi[q]); }
  }
  ck.reac_ptr.push_back(0);
  ck.prod_ptr.push_back(0);
  ck.tb_ptr.push_back(0);
  for (size_t i = 0; i < ck.input.size(); i++) {
    const Reaction &r = ck.input[i];
    emit(ck, r, (int)i, false, r.A, r.b, r.E, r.low);
    if (!r.reversible) continue;
    if (r.have_rev) {
      emit(ck, r, (int)i, true, r.revA, r.revb, r.revE, r.low);
      continue;
    }
    /* Appendix A: k_r = k_f / K_c at three temperatures -> (A_r, beta_r, E_r); a fall-off reaction has both of its
     * limits divided by K_c (P_r = k_0 [M] / k_inf and F are unchanged by that) */
    double a[3], al[3];
    for (int q = 0; q < 3; q++) {
      const double lk = ln_Kc(ck, r, T3[q]);
      a[q] = std::log(r.A) + r.b * std::log(T3[q]) - r.E / (RC * T3[q]) - lk;
      if (r.falloff) al[q] = std::log(r.low[0]) + r.low[1] * std::log(T3[q]) - r.low[2] / (RC * T3[q]) - lk;
    }
    double Ar, br, Er, low_r[3] = {0, 0, 0};
    fit3(T3, a, &Ar, &br, &Er);
    if (r.falloff) fit3(T3, al, &low_r[0], &low_r[1], &low_r[2]);
    emit(ck, r, (int)i, true, Ar, br, Er, low_r);
  }
}

}  // namespace

extern "C" {

int ckb_chemkin_parse(const char *mech_text, const char *thermo_text, const double *fit_T3, ckb_chemkin **out) {
  if (!mech_text || !out) return CKB_EINVAL;
  *out = nullptr;
  static const double T_default[3] = {1000.0, 1500.0, 2000.0};
  const double *T3 = fit_T3 ? fit_T3 : T_default;
  if (!(T3[0] > 0.0) || !(T3[1] > 0.0) || !(T3[2] > 0.0) || T3[0] == T3[1] || T3[1] == T3[2] || T3[0] == T3[2]) return CKB_EINVAL;
  ckb_chemkin *ck = new (std::nothrow) ckb_chemkin();
  if (!ck) return CKB_ENOMEM;
  try {
    /* split into sections; '!' starts a comment; thermo lines keep their columns */
    enum { NONE, ELEM, SPEC, THERMO, REAC } sec = NONE;
    std::vector<std::string> thermo_lines;
    std::vector<std::pair<int, std::string>> reac_lines;
    std::string reac_header;
    for (int pass = 0; pass < 2; pass++) {
      const char *text = pass == 0 ? mech_text : thermo_text;
      if (!text) continue;
      std::istringstream is(text);
      std::string raw;
      int lineno = 0;
      if (pass == 1) sec = THERMO; /* a separate thermodynamic database: THERMO block with or without its keyword */
      while (std::getline(is, raw)) {
        lineno++;
        if (!raw.empty() && raw.back() == '\r') raw.pop_back();
        const size_t bang = raw.find('!');
        std::string line = upper(bang == std::string::npos ? raw : raw.substr(0, bang));
        std::vector<std::string> t = tokens(line);
        if (t.empty()) continue;
        if (t[0] == "ELEMENTS" || t[0] == "ELEM") { sec = ELEM; t.erase(t.begin()); }
        else if (t[0] == "SPECIES" || t[0] == "SPEC") { sec = SPEC; t.erase(t.begin()); }
        else if (t[0] == "THERMO") { sec = THERMO; continue; }
        else if (t[0] == "REACTIONS" || t[0] == "REAC") { sec = REAC; reac_header = line; continue; }
        else if (t[0] == "END") { sec = NONE; continue; }
        if (sec == ELEM || sec == SPEC) {
          for (const std::string &w : t) {
            if (w == "END") { sec = NONE; break; }
            if (w.find('/') != std::string::npos) fail(CKB_EUNSUPPORTED, "isotope weights in the ELEMENTS block");
            if (sec == ELEM) ck->elements.push_back(w);
            else if (species_index(*ck, w) < 0) { Species s; s.name = w; ck->species.push_back(s); }
          }
        } else if (sec == THERMO) {
          thermo_lines.push_back(line);
        } else if (sec == REAC) {
          reac_lines.push_back({lineno, line});
        }
      }
    }
    if (ck->species.empty()) fail(CKB_EINVAL, "no SPECIES block");
    if (ck->species.size() > 254) fail(CKB_EUNSUPPORTED, "more than 254 species");
    parse_thermo(*ck, thermo_lines);
    for (const Species &s : ck->species)
      if (!s.have_thermo) fail(CKB_EINVAL, "no thermodynamic data for species " + s.name);
    parse_reactions(*ck, reac_lines, reac_header);
    convert(*ck, T3);
  } catch (const Fail &f) {
    delete ck;
    return f.code;
  } catch (const std::bad_alloc &) {
    delete ck;
    return CKB_ENOMEM;
  }
  *out = ck;
  return CKB_OK;
}

void ckb_chemkin_free(ckb_chemkin *ck) { delete ck; }

int ckb_chemkin_desc(const ckb_chemkin *ck, ckb_mech_desc *d, const double **nasa_high, const double **T_mid,
                     int32_t *n_falloff, const int32_t **fo_reaction, const double **fo_low, const double **fo_troe) {
  if (!ck || !d) return CKB_EINVAL;
  d->n_species = (int32_t)ck->species.size();
  d->n_reactions = (int32_t)ck->A.size();
  d->mol_weight = ck->W.data();
  d->nasa = ck->nasa.data();
  d->arr_A = ck->A.data();
  d->arr_beta = ck->beta.data();
  d->arr_E = ck->E.data();
  d->reac_ptr = ck->reac_ptr.data();
  d->reac_species = ck->reac_sp.data();
  d->reac_nu = ck->reac_nu.data();
  d->prod_ptr = ck->prod_ptr.data();
  d->prod_species = ck->prod_sp.data();
  d->prod_nu = ck->prod_nu.data();
  d->n_third_body = (int32_t)ck->tb_reaction.size();
  d->tb_reaction = ck->tb_reaction.data();
  d->tb_ptr = ck->tb_ptr.data();
  d->tb_species = ck->tb_species.data();
  d->tb_eff = ck->tb_eff.data();
  if (nasa_high) *nasa_high = ck->nasa_hi.data();
  if (T_mid) *T_mid = ck->Tmid.data();
  if (n_falloff) *n_falloff = (int32_t)ck->fo_reaction.size();
  if (fo_reaction) *fo_reaction = ck->fo_reaction.data();
  if (fo_low) *fo_low = ck->fo_low.data();
  if (fo_troe) *fo_troe = ck->fo_troe.data();
  return CKB_OK;
}

const char *ckb_chemkin_species(const ckb_chemkin *ck, int32_t k) {
  if (!ck || k < 0 || k >= (int32_t)ck->species.size()) return nullptr;
  return ck->species[k].name.c_str();
}

int ckb_chemkin_reaction_origin(const ckb_chemkin *ck, int32_t j, int32_t *input_reaction, int32_t *is_reverse) {
  if (!ck || j < 0 || j >= (int32_t)ck->A.size()) return CKB_EINVAL;
  if (input_reaction) *input_reaction = ck->origin[j];
  if (is_reverse) *is_reverse = ck->reversed[j];
  return CKB_OK;
}

const char *ckb_chemkin_error(void) { return g_err.c_str(); }

} /* extern "C" */
