// pd_card.cpp -- detector cards of libpd: built-ins and the text-file loader (host only, no CUDA).
//
// A card is "per-module parameters loaded from the selected detector card"; the paper's
// cards are "ported from their respective Delphes Tcl cards" (L81, L655) which are not available, so
// the three built-ins carry the numbers of BASELINE.json configs[0] (cms_like), [3] (atlas_like) and
// [4] (aleph_like) in the readings A2, A8, A9, A15, A20 of DESIGN.md.  Every number is rounded to
// fp32 first (reading A28); the derived tables the kernels use (sinh of the edges, bin widths, tower
// centres) are then computed in double from those fp32 values and rounded once.
#include <algorithm>
#include <array>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <fstream>
#include <limits>
#include <sstream>

#include "pd_internal.h"

namespace {

struct RawCard {
  std::string name;
  double bz = 0, radius = 0, half_length = 0, kappa = 0.299792458;
  bool theta = false;
  std::vector<double> edges;
  std::vector<long> nphi;
  std::vector<std::array<double, 6>> eff;  // pt_lo, pt_hi, |eta|_lo, |eta|_hi, eps, species (0 all, 1 e, 2 mu, 3 charged hadron)
  bool has_cos = false;
  double cos_max = 0;
  double trk_a = 0.01, trk_b = 1.5e-4;
  bool has_trk_sp[4] = {false, false, false, false};  // per-species track resolution (reading J2)
  double trk_a_sp[4] = {0, 0, 0, 0}, trk_b_sp[4] = {0, 0, 0, 0};
  double ecal[3] = {0, 0, 0}, hcal[3] = {0, 0, 0};
  double thr_ecal = 0.5, thr_hcal = 1.0;
  std::vector<std::array<double, 5>> ecal_eta, hcal_eta;  // reading K1: aeta_lo, aeta_hi, C, S, N
  double nsig_ecal = 0, nsig_hcal = 0;                    // reading K2
  bool smear_center = false;                              // reading K3
  std::vector<std::array<double, 5>> trk_eta;             // reading K4: aeta_lo, aeta_hi, a, b, species
  bool eflow_weighted = false;                            // reading K5
  std::vector<double> hcal_edges;                         // reading K6: the HCAL's own grid
  std::vector<long> hcal_nphi;
};

constexpr double kPi = 3.14159265358979323846;
const double kInf = std::numeric_limits<double>::infinity();

void default_tracking(RawCard &r) {
  // BASELINE.json configs[0], reading A8: ordered rows (pt_lo, pt_hi, |eta|_lo, |eta|_hi, eps)
  r.eff = {{{1.0, kInf, 0.0, 1.5, 0.97, 0.0}}, {{1.0, kInf, 1.5, 2.5, 0.85, 0.0}}, {{0.1, 1.0, 0.0, 2.5, 0.70, 0.0}}};
}

void builtin_cms(RawCard &r) {
  // 0.087-wide eta bins to |eta| = 3 (last one narrower), 0.175-wide to |eta| = 5 (reading A15)
  std::vector<double> pos;  // positive edges, ascending, starting at 0
  for (int k = 0; k <= 34; ++k) pos.push_back(double(k) * 0.087);
  pos.push_back(3.0);
  for (int k = 1; k <= 11; ++k) pos.push_back(3.0 + double(k) * 0.175);
  pos.push_back(5.0);
  for (size_t i = pos.size() - 1; i >= 1; --i) r.edges.push_back(-pos[i]);
  for (double e : pos) r.edges.push_back(e);
  const size_t nb = r.edges.size() - 1;  // 94
  for (size_t i = 0; i < nb; ++i) r.nphi.push_back((i < 12 || i + 12 >= nb) ? 36 : 72);
  r.bz = 3.8, r.radius = 1.29, r.half_length = 3.0;
  default_tracking(r);
  r.ecal[0] = 0.007, r.ecal[1] = 0.07, r.ecal[2] = 0.35;
  r.hcal[0] = 0.05, r.hcal[1] = 1.5, r.hcal[2] = 0.0;
}

void builtin_atlas(RawCard &r) {
  for (int i = 0; i <= 64; ++i) r.edges.push_back(double(i - 32) * 0.1);
  r.nphi.assign(64, 64);
  r.bz = 2.0, r.radius = 1.15, r.half_length = 3.5;
  default_tracking(r);
  r.ecal[0] = 0.0017, r.ecal[1] = 0.101, r.ecal[2] = 0.0;
  r.hcal[0] = 0.0302, r.hcal[1] = 0.5205, r.hcal[2] = 0.0;
}

void builtin_aleph(RawCard &r) {
  r.theta = true;
  r.edges.push_back(std::acos(0.98));
  for (int i = 0; i <= 90; ++i) r.edges.push_back(kPi / 2.0 + double(i - 45) * 0.03);
  r.edges.push_back(std::acos(-0.98));
  r.nphi.assign(92, 210);
  r.bz = 1.5, r.radius = 1.8, r.half_length = 2.5;
  default_tracking(r);
  r.has_cos = true, r.cos_max = 0.98;
  r.ecal[0] = 0.009, r.ecal[1] = 0.18, r.ecal[2] = 0.0;
  r.hcal[0] = 0.0, r.hcal[1] = 0.85, r.hcal[2] = 0.0;
}

std::string trim(const std::string &s) {
  size_t a = s.find_first_not_of(" \t\r\n"), b = s.find_last_not_of(" \t\r\n");
  return a == std::string::npos ? std::string() : s.substr(a, b - a + 1);
}

bool parse_numbers(const std::string &text, std::vector<double> &out) {
  const char *p = text.c_str();
  for (;;) {
    char *end = nullptr;
    double v = std::strtod(p, &end);
    if (end == p) break;
    out.push_back(v);
    p = end;
  }
  while (*p == ' ' || *p == '\t' || *p == '\r' || *p == '\n') ++p;
  return *p == 0;
}

bool from_file(RawCard &r, const char *path) {
  std::ifstream in(path);
  if (!in) return false;
  r.eff.clear();
  std::string line;
  while (std::getline(in, line)) {
    size_t hash = line.find('#');
    if (hash != std::string::npos) line.erase(hash);
    size_t eq = line.find('=');
    if (eq == std::string::npos) continue;
    const std::string key = trim(line.substr(0, eq)), val = trim(line.substr(eq + 1));
    if (key == "name") {
      r.name = val;
      continue;
    }
    if (key == "grid") {
      r.theta = val.compare(0, 5, "theta") == 0;
      continue;
    }
    std::vector<double> v;
    if (!parse_numbers(val, v)) return false;
    if (key == "edges") r.edges.insert(r.edges.end(), v.begin(), v.end());
    else if (key == "hcal_edges") r.hcal_edges.insert(r.hcal_edges.end(), v.begin(), v.end());
    else if (key == "hcal_nphi") for (double x : v) r.hcal_nphi.push_back(long(x));
    else if (key == "nphi") for (double x : v) r.nphi.push_back(long(x));
    else if (key == "bz" && v.size() == 1) r.bz = v[0];
    else if (key == "radius" && v.size() == 1) r.radius = v[0];
    else if (key == "half_length" && v.size() == 1) r.half_length = v[0];
    else if (key == "kappa" && v.size() == 1) r.kappa = v[0];
    else if (key == "abs_costheta_max" && v.size() == 1) r.has_cos = true, r.cos_max = v[0];
    else if (key == "track_res" && v.size() == 2) r.trk_a = v[0], r.trk_b = v[1];
    else if (key == "track_res" && v.size() == 3 && (v[2] == 1.0 || v[2] == 2.0 || v[2] == 3.0))
      r.has_trk_sp[int(v[2])] = true, r.trk_a_sp[int(v[2])] = v[0], r.trk_b_sp[int(v[2])] = v[1];
    else if (key == "ecal_res" && v.size() == 3) std::copy(v.begin(), v.end(), r.ecal);
    else if (key == "hcal_res" && v.size() == 3) std::copy(v.begin(), v.end(), r.hcal);
    else if (key == "ecal_res_eta" && v.size() == 5 && r.ecal_eta.size() < 8) r.ecal_eta.push_back({{v[0], v[1], v[2], v[3], v[4]}});
    else if (key == "hcal_res_eta" && v.size() == 5 && r.hcal_eta.size() < 8) r.hcal_eta.push_back({{v[0], v[1], v[2], v[3], v[4]}});
    else if (key == "track_res_eta" && (v.size() == 4 || (v.size() == 5 && (v[4] == 0.0 || v[4] == 1.0 || v[4] == 2.0 || v[4] == 3.0))) &&
             r.trk_eta.size() < size_t(PD_MAX_TRK_ROWS))
      r.trk_eta.push_back({{v[0], v[1], v[2], v[3], v.size() == 5 ? v[4] : 0.0}});
    else if (key == "ecal_nsigma" && v.size() == 1) r.nsig_ecal = v[0];
    else if (key == "hcal_nsigma" && v.size() == 1) r.nsig_hcal = v[0];
    else if (key == "smear_tower_center" && v.size() == 1) r.smear_center = v[0] != 0.0;
    else if (key == "eflow_weighted" && v.size() == 1) r.eflow_weighted = v[0] != 0.0;
    else if (key == "ecal_thr" && v.size() == 1) r.thr_ecal = v[0];
    else if (key == "hcal_thr" && v.size() == 1) r.thr_hcal = v[0];
    else if (key == "eff" && (v.size() == 5 || (v.size() == 6 && (v[5] == 0.0 || v[5] == 1.0 || v[5] == 2.0 || v[5] == 3.0))) &&
             r.eff.size() < size_t(PD_MAX_EFF))
      r.eff.push_back({{v[0], v[1], v[2], v[3], v[4], v.size() == 6 ? v[5] : 0.0}});
    else return false;
  }
  return true;
}

inline double f32(double x) { return double(float(x)); }

}  // namespace

int pd_card_parse(const char *name_or_path, pd_card *c) {
  RawCard r;
  const std::string key(name_or_path);
  r.name = key;
  if (key == "cms_like") builtin_cms(r);
  else if (key == "atlas_like") builtin_atlas(r);
  else if (key == "aleph_like") builtin_aleph(r);
  else if (!from_file(r, name_or_path)) return PD_ECARD;

  // validation
  const size_t nb = r.edges.size() < 2 ? 0 : r.edges.size() - 1;
  if (nb < 1 || nb > size_t(PD_MAX_BINS) || r.nphi.size() != nb) return PD_ECARD;
  if (!(r.radius > 0 && r.half_length > 0 && r.kappa > 0)) return PD_ECARD;
  for (size_t i = 1; i <= nb; ++i)
    if (!(float(r.edges[i]) > float(r.edges[i - 1]))) return PD_ECARD;
  long total = 0;
  for (long n : r.nphi) {
    if (n < 1) return PD_ECARD;
    total += n;
  }
  // reading K6: a grid of its own for the HCAL
  const bool dual = !r.hcal_edges.empty() || !r.hcal_nphi.empty();
  const size_t nbh = dual && r.hcal_edges.size() >= 2 ? r.hcal_edges.size() - 1 : 0;
  if (dual) {
    if (nbh < 1 || nb + nbh > size_t(PD_MAX_BINS) || r.hcal_nphi.size() != nbh) return PD_ECARD;
    for (size_t i = 1; i <= nbh; ++i)
      if (!(float(r.hcal_edges[i]) > float(r.hcal_edges[i - 1]))) return PD_ECARD;
    for (long n : r.hcal_nphi) {
      if (n < 1) return PD_ECARD;
      total += n;
    }
  }

  if (total > long(PD_MAX_TOWERS)) return PD_ECARD;
  // every number finite and in its range: thresholds and resolutions >= 0 (a negative threshold would let pass W count
  // a neutral that pass O never writes), efficiencies in [0, 1], |cos theta| cut in (0, 1], edges and rows ordered
  {
    auto fin = [](double x) { return std::isfinite(x); };
    auto nonneg = [&](double x) { return fin(x) && x >= 0.0; };
    if (!fin(r.bz) || !fin(r.radius) || !fin(r.half_length) || !fin(r.kappa)) return PD_ECARD;
    if (!nonneg(r.thr_ecal) || !nonneg(r.thr_hcal) || !nonneg(r.trk_a) || !nonneg(r.trk_b)) return PD_ECARD;
    for (int k = 0; k < 3; ++k)
      if (!nonneg(r.ecal[k]) || !nonneg(r.hcal[k])) return PD_ECARD;
    for (int sp = 1; sp <= 3; ++sp)
      if (r.has_trk_sp[sp] && (!nonneg(r.trk_a_sp[sp]) || !nonneg(r.trk_b_sp[sp]))) return PD_ECARD;
    if (r.has_cos && !(fin(r.cos_max) && r.cos_max > 0.0 && r.cos_max <= 1.0)) return PD_ECARD;
    for (double e : r.edges)
      if (!fin(e)) return PD_ECARD;
    for (double e : r.hcal_edges)
      if (!fin(e)) return PD_ECARD;
    if (r.theta && !(r.edges.front() >= 0.0 && r.edges.back() <= kPi)) return PD_ECARD;
    if (r.theta && dual && !(r.hcal_edges.front() >= 0.0 && r.hcal_edges.back() <= kPi)) return PD_ECARD;
    if (!nonneg(r.nsig_ecal) || !nonneg(r.nsig_hcal)) return PD_ECARD;
    for (const auto &row : r.trk_eta)  // aeta_hi may be "inf"
      if (!(nonneg(row[0]) && row[1] > row[0] && nonneg(row[2]) && nonneg(row[3]))) return PD_ECARD;
    for (const auto *rows : {&r.ecal_eta, &r.hcal_eta})
      for (const auto &row : *rows)
        if (!(nonneg(row[0]) && row[1] > row[0] && nonneg(row[2]) && nonneg(row[3]) && nonneg(row[4]))) return PD_ECARD;
    for (const auto &row : r.eff) {
      // pt_lo < pt_hi, |eta|_lo < |eta|_hi (the upper ends may be +inf), 0 <= eps <= 1
      if (!(nonneg(row[0]) && row[1] > row[0] && nonneg(row[2]) && row[3] > row[2])) return PD_ECARD;
      if (!(fin(row[4]) && row[4] >= 0.0 && row[4] <= 1.0)) return PD_ECARD;
    }
  }

  c->name = r.name;
  c->bz = float(r.bz);
  c->n_eff_rows = int(r.eff.size());
  PdCardScalars &s = c->sc;
  const double R = f32(r.radius), L = f32(r.half_length), B = f32(r.bz), kappa = f32(r.kappa);
  s.R = float(R), s.L = float(L), s.R2 = float(R * R), s.inv_R = float(1.0 / R);
  s.kB_d = kappa * std::fabs(B);
  s.kB = float(s.kB_d);
  s.inv_kB = s.kB_d > 0 ? float(1.0 / s.kB_d) : 0.f;
  s.sB = B > 0 ? 1.f : (B < 0 ? -1.f : 0.f);
  s.grid_theta = r.theta ? 1 : 0;
  s.n_bins = int(nb + nbh);  // all bins of the card: the ECAL grid's, then (reading K6) the HCAL grid's
  s.n_towers = int(total);
  s.words_per_event = int((total + 127) / 128) * 4;
  for (int sp = 1; sp <= 3; ++sp) {  // reading J2: the species' own resolution, else the card's common one
    const double a = f32(r.has_trk_sp[sp] ? r.trk_a_sp[sp] : r.trk_a);
    s.trk_a2[sp - 1] = float(a * a);
    s.trk_b[sp - 1] = float(r.has_trk_sp[sp] ? r.trk_b_sp[sp] : r.trk_b);
  }
  s.trk_per_species = (r.has_trk_sp[1] || r.has_trk_sp[2] || r.has_trk_sp[3]) ? 1 : 0;
  for (int k = 0; k < 3; ++k) {
    const double e = f32(r.ecal[k]), h = f32(r.hcal[k]);
    s.ecal2[k] = float(e * e);
    s.hcal2[k] = float(h * h);
  }
  s.thr_ecal = float(r.thr_ecal), s.thr_hcal = float(r.thr_hcal);

  // ---- efficiency table -> grid of cells (reading A8: rows are pt_lo < pT <= pt_hi and
  // |eta|_lo <= |eta| < |eta|_hi, first match wins; A9: eps = 0 for |cos theta| >= cmax).  Every pT
  // edge therefore splits "pT > e", every |eta| edge splits "|eta| >= e", i.e. T = |pz|/pT >= sinh e.
  {
    std::vector<double> pte, te;  // distinct finite edges, ascending (fp32 values)
    auto add = [](std::vector<double> &v, double x) {
      if (!std::isfinite(x)) return;
      for (double y : v)
        if (float(y) == float(x)) return;
      v.push_back(x);
    };
    const double cm = f32(r.cos_max);
    // |cos theta| >= cmax  <=>  |pz|/pT >= cmax / sqrt(1 - cmax^2)
    const double t_cos = r.has_cos ? (cm < 1.0 ? double(float(cm / std::sqrt(1.0 - cm * cm))) : kInf) : kInf;
    struct Row { double lo, hi, tlo, thi, eps; int species; };
    std::vector<Row> rows;
    for (const auto &row : r.eff) {
      Row w;
      w.lo = f32(row[0]), w.hi = std::isinf(row[1]) ? kInf : f32(row[1]);
      const double elo = f32(row[2]), ehi = std::isinf(row[3]) ? kInf : f32(row[3]);
      w.tlo = elo > 0 ? double(float(std::sinh(elo))) : -1.0;
      w.thi = std::isinf(ehi) ? kInf : double(float(std::sinh(ehi)));
      w.eps = f32(row[4]);
      w.species = int(row[5]);
      rows.push_back(w);
      if (w.lo > 0) add(pte, w.lo);
      add(pte, w.hi);
      if (w.tlo > 0) add(te, w.tlo);
      add(te, w.thi);
    }
    if (r.has_cos) add(te, t_cos);
    std::sort(pte.begin(), pte.end());
    std::sort(te.begin(), te.end());
    if (pte.size() > size_t(PD_MAX_EFF_EDGES) || te.size() > size_t(PD_MAX_EFF_EDGES)) return PD_ECARD;
    s.n_pt = int(pte.size()), s.n_T = int(te.size());
    for (int k = 0; k < PD_MAX_EFF_EDGES; ++k) {
      s.pt_edge2_d[k] = k < s.n_pt ? pte[size_t(k)] * pte[size_t(k)] : std::numeric_limits<double>::max();
      s.T_edge[k] = k < s.n_T ? float(te[size_t(k)]) : std::numeric_limits<float>::infinity();
    }
    s.eff_per_species = 0;
    for (int k = 0; k <= PD_MAX_EFF; ++k) s.row_eps[k] = 0.f;
    for (const Row &w : rows) s.eff_per_species |= w.species != 0 ? 1 : 0;
    // one grid per species (reading J1: a row applies to every charged particle or to one species only)
    for (int sp = 1; sp <= 3; ++sp)
      for (int ip = 0; ip <= s.n_pt; ++ip) {
        // representative pT of the interval (e[ip-1], e[ip]]: its closed upper end, or beyond the last edge
        const double pt_rep = ip < s.n_pt ? pte[size_t(ip)] : (s.n_pt ? 2.0 * pte.back() + 1.0 : 1.0);
        for (int it = 0; it <= s.n_T; ++it) {
          // representative T of [t[it-1], t[it]): its closed lower end, or 0
          const double T_rep = it > 0 ? te[size_t(it - 1)] : 0.0;
          float eps = 0.f;
          int rowi = -1;
          if (!(r.has_cos && T_rep >= t_cos)) {
            for (size_t k = 0; k < rows.size(); ++k) {
              const Row &w = rows[k];
              if (w.species != 0 && w.species != sp) continue;
              if (pt_rep > w.lo && pt_rep <= w.hi && (w.tlo <= 0 || T_rep >= w.tlo) && T_rep < w.thi) {
                rowi = int(k), eps = float(w.eps);
                break;
              }
            }
          }
          s.cell_eps[sp - 1][ip * (s.n_T + 1) + it] = eps;
          if (rowi >= 0) s.row_eps[rowi] = eps;
          s.cell_row[sp - 1][ip * (s.n_T + 1) + it] = (signed char)rowi;
        }
      }
  }

  // ---- per-bin tables, grid by grid (one grid, or the ECAL's followed by the HCAL's: reading K6); tower offsets run on
  const size_t nball = nb + nbh;
  c->edges.assign(2 * nball, 0.f);
  c->tb.clear();
  c->nphi.resize(nball);
  c->offset.resize(nball + 1);
  c->inv_w.resize(nball), c->half.resize(nball), c->w.resize(nball), c->eta_c.resize(nball), c->inv_cosh.resize(nball);
  c->lut.clear();
  int acc = 0;
  s.n_grids = dual ? 2 : 1;
  for (int g = 0; g < s.n_grids; ++g) {
    const std::vector<double> &ge = g == 0 ? r.edges : r.hcal_edges;
    const std::vector<long> &gn = g == 0 ? r.nphi : r.hcal_nphi;
    const size_t gnb = ge.size() - 1, b0 = g == 0 ? 0 : nb, t0 = c->tb.size();
    s.g_nb[g] = int(gnb), s.g_bin_off[g] = int(b0), s.g_tb_off[g] = int(t0);
    for (size_t i = 0; i <= gnb; ++i) {
      const double e = f32(ge[i]);
      if (i < gnb) c->edges[2 * (b0 + i)] = float(e);
      if (i > 0) c->edges[2 * (b0 + i - 1) + 1] = float(e);
      // bin test "edge_i <= coord < edge_{i+1}" mapped to u = z/r (eta: u = sinh eta, ascending) or
      // u = -z/r (theta: u = -cot theta, ascending in theta)
      double t;
      if (!r.theta) t = std::sinh(e);
      else if (e <= 0.0) t = -kInf;
      else if (e >= kPi) t = kInf;
      else t = -std::cos(e) / std::sin(e);
      c->tb.push_back(float(t));
    }
    for (size_t i = 0; i < gnb; ++i) {
      const size_t bi = b0 + i;
      const int n = int(gn[i]);
      c->nphi[bi] = n;
      c->offset[bi] = acc;
      acc += n;
      c->inv_w[bi] = float(double(n) / (2.0 * kPi));
      c->w[bi] = float(2.0 * kPi / double(n));
      c->half[bi] = (n & 1) ? 0.5f : 0.f;
      const double mid = 0.5 * (double(c->edges[2 * bi]) + double(c->edges[2 * bi + 1]));
      const double eta = r.theta ? -std::log(std::tan(0.5 * mid)) : mid;
      c->eta_c[bi] = float(eta);
      c->inv_cosh[bi] = float(1.0 / std::cosh(eta));
    }
    s.g_tb_first[g] = c->tb[t0], s.g_tb_last[g] = c->tb[t0 + gnb];
    // ---- eta-bin lookup of the grid: cells of |u| by float bits (2^(23 - PD_LUT_SHIFT) cells per octave, |u| < 2^MIN_EXP
    // in one cell), mirrored for u < 0.  lut[cell] = the bin (relative to the grid) holding the cell's LOWER bound
    // (clamped to the grid); the kernel then steps forward while u >= tb[bin + 1], so any monotone edge list is handled exactly.
    const float *tbg = c->tb.data() + t0;
    float umax = 1.f;
    for (size_t i = 0; i <= gnb; ++i)
      if (std::isfinite(tbg[i])) umax = std::max(umax, std::fabs(tbg[i]));
    auto bits = [](float x) {
      uint32_t b;
      std::memcpy(&b, &x, 4);
      return int(b >> PD_LUT_SHIFT);
    };
    const int lbase = bits(std::ldexp(1.f, PD_LUT_MIN_EXP));
    const int side = bits(umax) - lbase + 2;
    s.g_lut_base[g] = lbase, s.g_lut_side[g] = side, s.g_lut_off[g] = int(c->lut.size());
    const size_t l0 = c->lut.size();
    c->lut.resize(l0 + size_t(2 * side), 0);
    auto cell_lo_abs = [&](int ca) {  // smallest |u| of cell ca on one side
      if (ca <= 0) return 0.f;
      const uint32_t b = uint32_t(ca + lbase) << PD_LUT_SHIFT;
      float x;
      std::memcpy(&x, &b, 4);
      return x;
    };
    auto bin_of = [&](double u) {  // largest b with tb[b] <= u, clamped to [0, gnb-1]
      int b = 0;
      while (b + 1 < int(gnb) && double(tbg[size_t(b + 1)]) <= u) ++b;
      return b;
    };
    for (int ca = 0; ca < side; ++ca) {
      // positive side: u in [lo(ca), lo(ca+1)); cell index side + ca
      c->lut[l0 + size_t(side + ca)] = (unsigned short)bin_of(double(cell_lo_abs(ca)));
      // negative side: u in (-lo(ca+1), -lo(ca)]; lower bound -lo(ca+1) (-inf for the last cell)
      const double lo = ca + 1 < side ? -double(cell_lo_abs(ca + 1)) : -kInf;
      c->lut[l0 + size_t(side - 1 - ca)] = (unsigned short)bin_of(lo);
    }
  }
  c->offset[nball] = acc;
  if (!dual) {  // one grid: both entries describe it, so that the kernels index by section without a branch
    s.g_nb[1] = s.g_nb[0], s.g_bin_off[1] = s.g_bin_off[0], s.g_tb_off[1] = s.g_tb_off[0], s.g_lut_off[1] = s.g_lut_off[0];
    s.g_lut_side[1] = s.g_lut_side[0], s.g_lut_base[1] = s.g_lut_base[0], s.g_tb_first[1] = s.g_tb_first[0], s.g_tb_last[1] = s.g_tb_last[0];
  }
  s.n_tb = int(c->tb.size()), s.lut_cells = int(c->lut.size());
  // readings K1-K3: per-bin resolutions (the first row whose [aeta_lo, aeta_hi) holds |eta| of the bin's tower centres,
  // else the card's common line), significance cut, smeared tower positions
  s.res_per_bin = (!r.ecal_eta.empty() || !r.hcal_eta.empty()) ? 1 : 0;
  c->res2.assign(6 * nball, 0.f);
  for (size_t i = 0; i < nball; ++i) {
    const double mid = 0.5 * (double(c->edges[2 * i]) + double(c->edges[2 * i + 1]));
    const double aeta = std::fabs(r.theta ? -std::log(std::tan(0.5 * mid)) : mid);
    auto pick = [&](const std::vector<std::array<double, 5>> &rows, const double *dflt, float *out) {
      const double *csn = dflt;
      for (const auto &row : rows)
        if (aeta >= f32(row[0]) && aeta < f32(row[1])) {
          csn = row.data() + 2;
          break;
        }
      for (int k = 0; k < 3; ++k) out[k] = float(f32(csn[k]) * f32(csn[k]));
    };
    pick(r.ecal_eta, r.ecal, &c->res2[6 * i]);
    pick(r.hcal_eta, r.hcal, &c->res2[6 * i + 3]);
  }
  s.nsig2_ecal = float(f32(r.nsig_ecal) * f32(r.nsig_ecal));
  s.nsig2_hcal = float(f32(r.nsig_hcal) * f32(r.nsig_hcal));
  s.smear_center = r.smear_center ? 1 : 0;
  s.eflow_weighted = r.eflow_weighted ? 1 : 0;
  // reading K4: the rows' edges as sinh of the fp32-rounded |eta| (fp64, the form the kernel compares |pz| / pT with)
  s.n_trk_rows = int(r.trk_eta.size());
  for (int k = 0; k < PD_MAX_TRK_ROWS; ++k) {
    const bool on = k < s.n_trk_rows;
    s.trk_row_sp[k] = on ? int(r.trk_eta[k][4]) : 0;
    s.trk_row_lo_d[k] = on ? std::sinh(f32(r.trk_eta[k][0])) : 0.0;
    s.trk_row_hi_d[k] = on ? std::sinh(f32(r.trk_eta[k][1])) : 0.0;
    const double a = on ? f32(r.trk_eta[k][2]) : 0.0;
    s.trk_row_a2[k] = float(a * a);
    s.trk_row_b[k] = on ? float(r.trk_eta[k][3]) : 0.f;
  }
  return PD_OK;
}
