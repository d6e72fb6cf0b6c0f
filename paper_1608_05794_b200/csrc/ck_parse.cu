// ck_mech_parse: a kinetic model in CHEMKIN-II style text -> ck_mech_desc.  The paper's codes read
// their models through `create_rate_subs`, which interprets such files into a binary database; here the
// text is interpreted into the plain description ck_mech_load takes.  Host code only (no CUDA call).
//
// Supported (the subset the paper's three models need: reversible and irreversible elementary
// reactions, third bodies with efficiencies, Lindemann and Troe falloff, two-range NASA-7 thermo):
//   ELEMENTS ... END        SPECIES ... END
//   THERMO [ALL] / default temperature line / four 80-column cards per species (name in columns 1-18, up to four
//        element fields of 2 + 3 columns from column 25, T_low T_high T_mid in columns 46-75, then 7 high-range and
//        7 low-range coefficients in fields of 15 columns) / END
//   REACTIONS [CAL/MOLE] / one line per reaction "equation  A  beta  Ea" with "<=>" or "=" (reversible) or "=>"
//        (irreversible), "+M" (third body) or "(+M)" (falloff) / auxiliary lines LOW/ A0 beta0 Ea0 /,
//        TROE/ a T*** T* [T**] /, efficiencies NAME/value/ ..., DUPLICATE (ignored) / END
//   '!' starts a comment.  Units: cm-mol-s-K, activation energies in cal/mol (the defaults of the format).
// Molar masses are sums of standard atomic weights over the element fields of the thermo card.
#include <algorithm>
#include <cctype>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <map>
#include <sstream>
#include <string>
#include <vector>

#include "ck_internal.h"

using namespace ck;

struct ck_parsed {
  ck_mech_desc desc;
  std::vector<std::string> elements, species;
  std::vector<double> mol_wt, nasa_lo, nasa_hi, t_mid, A, beta, Ea, A0, beta0, Ea0, troe, eff_val;
  std::vector<int32_t> elem_comp, reac_ptr, reac_spec, reac_nu, prod_ptr, prod_spec, prod_nu, eff_ptr, eff_spec;
  std::vector<uint8_t> reversible, type;
};

namespace {

std::string upper(std::string s) { for (auto& c : s) c = (char)std::toupper((unsigned char)c); return s; }
std::string strip(const std::string& s) {
  size_t b = s.find_first_not_of(" \t\r\n"), e = s.find_last_not_of(" \t\r\n");
  return b == std::string::npos ? std::string() : s.substr(b, e - b + 1);
}
std::vector<std::string> words(const std::string& s) {
  std::istringstream is(s);
  std::vector<std::string> w;
  std::string t;
  while (is >> t) w.push_back(t);
  return w;
}
bool number(const std::string& s, double* v) {
  if (s.empty()) return false;
  std::string t = s;
  for (auto& c : t) if (c == 'D' || c == 'd') c = 'E';   // Fortran exponents
  char* end = nullptr;
  *v = std::strtod(t.c_str(), &end);
  return end && *end == 0;
}
double atomic_weight(const std::string& sym) {
  static const std::map<std::string, double> w = {{"H", 1.008}, {"C", 12.011}, {"O", 15.999}, {"N", 14.007},
                                                   {"AR", 39.948}, {"HE", 4.002602}, {"S", 32.06}, {"CL", 35.45}};
  auto it = w.find(upper(sym));
  return it == w.end() ? -1.0 : it->second;
}

// one side of a reaction equation -> (species, nu) pairs; sets third body / falloff flags
bool parse_side(std::string side, const std::map<std::string, int>& sp_index, std::vector<std::pair<int, int>>* out, bool* third,
                bool* falloff, std::string* why) {
  size_t pos;
  while ((pos = upper(side).find("(+M)")) != std::string::npos) { side.erase(pos, 4); *falloff = true; }
  std::vector<std::string> terms;
  std::string cur;
  for (char c : side) {
    if (c == '+') { terms.push_back(cur); cur.clear(); }
    else if (!std::isspace((unsigned char)c)) cur.push_back(c);
  }
  terms.push_back(cur);
  for (auto& t : terms) {
    if (t.empty()) { *why = "empty term in '" + side + "'"; return false; }
    if (upper(t) == "M") { *third = true; continue; }
    size_t d = 0;
    while (d < t.size() && std::isdigit((unsigned char)t[d])) ++d;
    int nu = d ? std::atoi(t.substr(0, d).c_str()) : 1;
    auto it = sp_index.find(upper(t.substr(d)));
    if (it == sp_index.end() || nu < 1) { *why = "unknown species '" + t + "'"; return false; }
    bool merged = false;
    for (auto& pr : *out) if (pr.first == it->second) { pr.second += nu; merged = true; }
    if (!merged) out->push_back({it->second, nu});
  }
  std::sort(out->begin(), out->end());
  return true;
}

int32_t fail(int line, const std::string& msg) {
  set_error("ck_mech_parse: line %d: %s", line, msg.c_str());
  return CK_EINVAL;
}

}  // namespace

extern "C" int32_t ck_mech_parse(const char* text, ck_parsed** out) {
  if (!text || !out) { set_error("ck_mech_parse: null argument"); return CK_EINVAL; }
  *out = nullptr;
  ck_parsed* P = new ck_parsed;
  struct Guard { ck_parsed* p; ~Guard() { delete p; } } guard{P};
  std::vector<std::string> lines;
  {
    std::istringstream is(text);
    std::string l;
    while (std::getline(is, l)) lines.push_back(l);
  }
  std::map<std::string, int> el_index, sp_index;
  std::map<std::string, std::vector<std::string>> thermo_cards;   // species -> its four cards
  enum { NONE, ELEM, SPEC, THERMO, REAC } sec = NONE;
  double t_default[3] = {300.0, 1000.0, 5000.0};
  bool thermo_default_read = false;
  std::vector<std::string> card;
  struct Rxn { std::vector<std::pair<int, int>> re, pr; double A, b, E, A0 = 0, b0 = 0, E0 = 0, troe[4] = {0, 1, 1, -1}; bool rev, third = false, fall = false, has_low = false, has_troe = false; std::vector<std::pair<int, double>> eff; int line; };
  std::vector<Rxn> rx;
  for (size_t li = 0; li < lines.size(); ++li) {
    const int ln = (int)li + 1;
    std::string raw = lines[li];
    const size_t bang = raw.find('!');
    if (bang != std::string::npos) raw = raw.substr(0, bang);
    std::string l = strip(raw);
    if (l.empty()) continue;
    std::vector<std::string> w = words(l);
    const std::string k0 = upper(w[0]);
    if (sec != THERMO || card.empty()) {
      if (k0.rfind("ELEM", 0) == 0) { sec = ELEM; w.erase(w.begin()); }
      else if (k0.rfind("SPEC", 0) == 0) { sec = SPEC; w.erase(w.begin()); }
      else if (k0.rfind("THER", 0) == 0) { sec = THERMO; thermo_default_read = false; card.clear(); continue; }
      else if (k0.rfind("REAC", 0) == 0) { sec = REAC; continue; }
    }
    if (k0 == "END" && card.empty()) { sec = NONE; continue; }
    if (sec == ELEM || sec == SPEC) {
      for (auto& t : w) {
        if (upper(t) == "END") { sec = NONE; break; }
        auto& idx = (sec == ELEM) ? el_index : sp_index;
        auto& names = (sec == ELEM) ? P->elements : P->species;
        if (idx.count(upper(t))) return fail(ln, "'" + t + "' listed twice");
        idx[upper(t)] = (int)names.size();
        names.push_back(t);
      }
    } else if (sec == THERMO) {
      if (!thermo_default_read && card.empty()) {   // optional line of three default temperatures
        double a, b, c;
        if (w.size() == 3 && number(w[0], &a) && number(w[1], &b) && number(w[2], &c)) { t_default[0] = a; t_default[1] = b; t_default[2] = c; thermo_default_read = true; continue; }
        thermo_default_read = true;
      }
      std::string c80 = raw;
      c80.resize(80, ' ');
      card.push_back(c80);
      if (card.size() == 4) {
        const std::string name = upper(words(card[0].substr(0, 18)).empty() ? std::string() : words(card[0].substr(0, 18))[0]);
        if (name.empty()) return fail(ln, "thermo card without a species name");
        thermo_cards[name] = card;
        card.clear();
      }
    } else if (sec == REAC) {
      const std::string U = upper(l);
      if (U.rfind("DUP", 0) == 0) continue;
      const bool aux = U.find('/') != std::string::npos && U.find('=') == std::string::npos;
      if (aux) {
        if (rx.empty()) return fail(ln, "auxiliary line before any reaction");
        Rxn& r = rx.back();
        // NAME / numbers / groups
        size_t p = 0;
        while (p < l.size()) {
          const size_t s1 = l.find('/', p);
          if (s1 == std::string::npos) break;
          const size_t s2 = l.find('/', s1 + 1);
          if (s2 == std::string::npos) return fail(ln, "unterminated '/'");
          const std::string key = upper(strip(l.substr(p, s1 - p)));
          std::vector<std::string> vals = words(l.substr(s1 + 1, s2 - s1 - 1));
          std::vector<double> v(vals.size());
          for (size_t i = 0; i < vals.size(); ++i) if (!number(vals[i], &v[i])) return fail(ln, "bad number '" + vals[i] + "'");
          if (key == "LOW") { if (v.size() != 3) return fail(ln, "LOW needs three numbers"); r.A0 = v[0]; r.b0 = v[1]; r.E0 = v[2]; r.has_low = true; }
          else if (key == "TROE") { if (v.size() != 3 && v.size() != 4) return fail(ln, "TROE needs three or four numbers"); for (size_t i = 0; i < v.size(); ++i) r.troe[i] = v[i]; if (v.size() == 3) r.troe[3] = -1.0; r.has_troe = true; }
          else {
            auto it = sp_index.find(key);
            if (it == sp_index.end() || v.size() != 1) return fail(ln, "unknown auxiliary keyword or species '" + key + "'");
            r.eff.push_back({it->second, v[0]});
          }
          p = s2 + 1;
        }
        continue;
      }
      if (w.size() < 4) return fail(ln, "reaction line needs an equation and three numbers");
      Rxn r;
      r.line = ln;
      if (!number(w[w.size() - 3], &r.A) || !number(w[w.size() - 2], &r.b) || !number(w[w.size() - 1], &r.E)) return fail(ln, "bad Arrhenius numbers");
      std::string eq;
      for (size_t i = 0; i + 3 < w.size(); ++i) eq += w[i];
      size_t pos;
      std::string lhs, rhs;
      if ((pos = eq.find("<=>")) != std::string::npos) { r.rev = true; lhs = eq.substr(0, pos); rhs = eq.substr(pos + 3); }
      else if ((pos = eq.find("=>")) != std::string::npos) { r.rev = false; lhs = eq.substr(0, pos); rhs = eq.substr(pos + 2); }
      else if ((pos = eq.find('=')) != std::string::npos) { r.rev = true; lhs = eq.substr(0, pos); rhs = eq.substr(pos + 1); }
      else return fail(ln, "no '=' in reaction");
      std::string why;
      bool t1 = false, t2 = false, f1 = false, f2 = false;
      if (!parse_side(lhs, sp_index, &r.re, &t1, &f1, &why) || !parse_side(rhs, sp_index, &r.pr, &t2, &f2, &why)) return fail(ln, why);
      if (t1 != t2 || f1 != f2) return fail(ln, "third body must appear on both sides");
      r.third = t1; r.fall = f1;
      rx.push_back(r);
    }
  }
  const int K = (int)P->species.size(), E = (int)P->elements.size(), R = (int)rx.size();
  if (K < 1) { set_error("ck_mech_parse: no species"); return CK_EINVAL; }
  // ---- thermo cards -> NASA-7, element composition, molar masses
  P->nasa_lo.assign(7 * (size_t)K, 0.0); P->nasa_hi.assign(7 * (size_t)K, 0.0); P->t_mid.assign(K, 0.0);
  P->elem_comp.assign((size_t)K * std::max(E, 1), 0); P->mol_wt.assign(K, 0.0);
  for (int k = 0; k < K; ++k) {
    auto it = thermo_cards.find(upper(P->species[k]));
    if (it == thermo_cards.end()) { set_error("ck_mech_parse: no thermo data for species '%s'", P->species[k].c_str()); return CK_EINVAL; }
    const std::vector<std::string>& c = it->second;
    for (int f = 0; f < 4; ++f) {
      const std::string sym = strip(c[0].substr(24 + 5 * f, 2)), cnt = strip(c[0].substr(26 + 5 * f, 3));
      if (sym.empty() || cnt.empty()) continue;
      double cn;
      if (!number(cnt, &cn) || cn == 0) continue;
      auto ie = el_index.find(upper(sym));
      const double aw = atomic_weight(sym);
      if (ie == el_index.end() || aw < 0) { set_error("ck_mech_parse: species '%s': unknown element '%s'", P->species[k].c_str(), sym.c_str()); return CK_EINVAL; }
      P->elem_comp[(size_t)k * E + ie->second] += (int)cn;
      P->mol_wt[k] += cn * aw;
    }
    double tl, th, tm;
    if (!number(strip(c[0].substr(45, 10)), &tl)) tl = t_default[0];
    if (!number(strip(c[0].substr(55, 10)), &th)) th = t_default[2];
    if (!number(strip(c[0].substr(65, 10)), &tm)) tm = t_default[1];
    P->t_mid[k] = tm;
    double a[14];
    for (int j = 0; j < 14; ++j) {
      const int cardno = 1 + j / 5, field = j % 5;
      if (!number(strip(c[cardno].substr(15 * field, 15)), &a[j])) { set_error("ck_mech_parse: species '%s': bad coefficient %d", P->species[k].c_str(), j + 1); return CK_EINVAL; }
    }
    for (int j = 0; j < 7; ++j) { P->nasa_hi[7 * (size_t)k + j] = a[j]; P->nasa_lo[7 * (size_t)k + j] = a[7 + j]; }
    if (!(P->mol_wt[k] > 0)) { set_error("ck_mech_parse: species '%s' has no element composition", P->species[k].c_str()); return CK_EINVAL; }
  }
  // ---- reactions
  P->reac_ptr.assign(1, 0); P->prod_ptr.assign(1, 0); P->eff_ptr.assign(1, 0);
  for (const Rxn& r : rx) {
    for (auto& pr : r.re) { P->reac_spec.push_back(pr.first); P->reac_nu.push_back(pr.second); }
    for (auto& pr : r.pr) { P->prod_spec.push_back(pr.first); P->prod_nu.push_back(pr.second); }
    P->reac_ptr.push_back((int)P->reac_spec.size()); P->prod_ptr.push_back((int)P->prod_spec.size());
    int type = CK_PLAIN;
    if (r.fall) {
      if (!r.has_low) return fail(r.line, "falloff reaction without LOW/ ... /");
      type = r.has_troe ? CK_TROE : CK_LINDEMANN;
    } else if (r.third) type = CK_THREE_BODY;
    else if (r.has_low || r.has_troe || !r.eff.empty()) return fail(r.line, "auxiliary data on a reaction without third body");
    std::vector<std::pair<int, double>> eff = r.eff;
    std::sort(eff.begin(), eff.end());
    for (auto& e : eff) { P->eff_spec.push_back(e.first); P->eff_val.push_back(e.second); }
    P->eff_ptr.push_back((int)P->eff_spec.size());
    P->A.push_back(r.A); P->beta.push_back(r.b); P->Ea.push_back(r.E);
    P->A0.push_back(r.A0); P->beta0.push_back(r.b0); P->Ea0.push_back(r.E0);
    for (int j = 0; j < 4; ++j) P->troe.push_back(r.troe[j]);
    P->reversible.push_back(r.rev ? 1 : 0); P->type.push_back((uint8_t)type);
  }
  ck_mech_desc& d = P->desc;
  std::memset(&d, 0, sizeof d);
  d.struct_size = (int32_t)sizeof d; d.n_species = K; d.n_reactions = R; d.n_elements = E;
  d.mol_wt = P->mol_wt.data(); d.elem_comp = E ? P->elem_comp.data() : nullptr;
  d.nasa_lo = P->nasa_lo.data(); d.nasa_hi = P->nasa_hi.data(); d.t_mid = P->t_mid.data();
  d.reac_ptr = P->reac_ptr.data(); d.reac_spec = P->reac_spec.data(); d.reac_nu = P->reac_nu.data();
  d.prod_ptr = P->prod_ptr.data(); d.prod_spec = P->prod_spec.data(); d.prod_nu = P->prod_nu.data();
  d.A = P->A.data(); d.beta = P->beta.data(); d.Ea = P->Ea.data(); d.reversible = P->reversible.data(); d.type = P->type.data();
  d.A0 = P->A0.data(); d.beta0 = P->beta0.data(); d.Ea0 = P->Ea0.data(); d.troe = P->troe.data();
  d.eff_ptr = P->eff_ptr.data(); d.eff_spec = P->eff_spec.data(); d.eff_val = P->eff_val.data();
  guard.p = nullptr;
  *out = P;
  return CK_OK;
}

extern "C" const ck_mech_desc* ck_parsed_desc(const ck_parsed* p) { return p ? &p->desc : nullptr; }
extern "C" int32_t ck_parsed_name(const ck_parsed* p, int32_t what, int32_t index, char* buf, int32_t len) {
  if (!p || !buf || len < 1) { set_error("ck_parsed_name: bad argument"); return CK_EINVAL; }
  const std::vector<std::string>& v = what ? p->elements : p->species;
  if (index < 0 || index >= (int)v.size()) { set_error("ck_parsed_name: index out of range"); return CK_EINVAL; }
  std::strncpy(buf, v[index].c_str(), (size_t)len - 1);
  buf[len - 1] = 0;
  return CK_OK;
}
extern "C" int32_t ck_parsed_free(ck_parsed* p) { delete p; return CK_OK; }
