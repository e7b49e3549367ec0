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
  std::vector<std::array<double, 5>> eff;
  bool has_cos = false;
  double cos_max = 0;
  double trk_a = 0.01, trk_b = 1.5e-4;
  double ecal[3] = {0, 0, 0}, hcal[3] = {0, 0, 0};
  double thr_ecal = 0.5, thr_hcal = 1.0;
};

constexpr double kPi = 3.14159265358979323846;
const double kInf = std::numeric_limits<double>::infinity();

void default_tracking(RawCard &r) {
  // BASELINE.json configs[0], reading A8: ordered rows (pt_lo, pt_hi, |eta|_lo, |eta|_hi, eps)
  r.eff = {{{1.0, kInf, 0.0, 1.5, 0.97}}, {{1.0, kInf, 1.5, 2.5, 0.85}}, {{0.1, 1.0, 0.0, 2.5, 0.70}}};
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
    else if (key == "nphi") for (double x : v) r.nphi.push_back(long(x));
    else if (key == "bz" && v.size() == 1) r.bz = v[0];
    else if (key == "radius" && v.size() == 1) r.radius = v[0];
    else if (key == "half_length" && v.size() == 1) r.half_length = v[0];
    else if (key == "kappa" && v.size() == 1) r.kappa = v[0];
    else if (key == "abs_costheta_max" && v.size() == 1) r.has_cos = true, r.cos_max = v[0];
    else if (key == "track_res" && v.size() == 2) r.trk_a = v[0], r.trk_b = v[1];
    else if (key == "ecal_res" && v.size() == 3) std::copy(v.begin(), v.end(), r.ecal);
    else if (key == "hcal_res" && v.size() == 3) std::copy(v.begin(), v.end(), r.hcal);
    else if (key == "ecal_thr" && v.size() == 1) r.thr_ecal = v[0];
    else if (key == "hcal_thr" && v.size() == 1) r.thr_hcal = v[0];
    else if (key == "eff" && v.size() == 5 && r.eff.size() < size_t(PD_MAX_EFF))
      r.eff.push_back({{v[0], v[1], v[2], v[3], v[4]}});
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

  c->name = r.name;
  c->bz = float(r.bz);
  PdCardScalars &s = c->sc;
  const double R = f32(r.radius), L = f32(r.half_length), B = f32(r.bz), kappa = f32(r.kappa);
  s.R = float(R), s.L = float(L), s.R2 = float(R * R);
  s.kB_d = kappa * std::fabs(B);
  s.kB = float(s.kB_d);
  s.sB = B > 0 ? 1.f : (B < 0 ? -1.f : 0.f);
  s.grid_theta = r.theta ? 1 : 0;
  s.n_bins = int(nb);
  s.n_towers = int(total);
  {
    long max_n = 1;
    for (long n : r.nphi) max_n = std::max(max_n, n);
    s.j_bits = 0;
    while ((1L << s.j_bits) < max_n) ++s.j_bits;
    int bin_bits = 0;
    while ((size_t(1) << bin_bits) < nb) ++bin_bits;
    s.code_bits = bin_bits + s.j_bits;
    if (s.code_bits < 1) s.code_bits = 1;
    if (s.code_bits > PD_MAX_CODE_BITS) return PD_ECARD;
  }
  s.n_eff = int(r.eff.size());
  s.has_cos = r.has_cos ? 1 : 0;
  {
    // |cos theta| >= cmax  <=>  |pz|/pT >= cmax / sqrt(1 - cmax^2)
    const double cm = f32(r.cos_max);
    s.t_cos = r.has_cos ? (cm < 1.0 ? float(cm / std::sqrt(1.0 - cm * cm)) : std::numeric_limits<float>::infinity()) : 0.f;
  }
  {
    const double a = f32(r.trk_a);
    s.trk_a2 = float(a * a);
    s.trk_b = float(r.trk_b);
  }
  for (int k = 0; k < 3; ++k) {
    const double e = f32(r.ecal[k]), h = f32(r.hcal[k]);
    s.ecal2[k] = float(e * e);
    s.hcal2[k] = float(h * h);
  }
  s.thr_ecal = float(r.thr_ecal), s.thr_hcal = float(r.thr_hcal);
  for (int i = 0; i < s.n_eff; ++i) {
    const auto &row = r.eff[size_t(i)];
    s.eff[i][0] = float(row[0]);
    s.eff[i][1] = float(row[1]);
    const double lo = f32(row[2]), hi = f32(row[3]);
    s.eff[i][2] = lo > 0 ? float(std::sinh(lo)) : -1.f;
    s.eff[i][3] = std::isinf(hi) ? std::numeric_limits<float>::infinity() : float(std::sinh(hi));
    s.eff[i][4] = float(row[4]);
  }

  c->edges.resize(nb + 1);
  c->tb.resize(nb + 1);
  c->nphi.resize(nb);
  c->offset.resize(nb + 1);
  c->inv_w.resize(nb), c->half.resize(nb), c->w.resize(nb), c->eta_c.resize(nb), c->inv_cosh.resize(nb);
  int acc = 0;
  for (size_t i = 0; i <= nb; ++i) {
    const double e = f32(r.edges[i]);
    c->edges[i] = float(e);
    // bin test "edge_i <= coord < edge_{i+1}" mapped to u = z/r (eta: u = sinh eta, ascending) or
    // u = -z/r (theta: u = -cot theta, ascending in theta)
    double t;
    if (!r.theta) t = std::sinh(e);
    else if (e <= 0.0) t = -kInf;
    else if (e >= kPi) t = kInf;
    else t = -std::cos(e) / std::sin(e);
    c->tb[i] = float(t);
  }
  for (size_t i = 0; i < nb; ++i) {
    const int n = int(r.nphi[i]);
    c->nphi[i] = n;
    c->offset[i] = acc;
    acc += n;
    c->inv_w[i] = float(double(n) / (2.0 * kPi));
    c->w[i] = float(2.0 * kPi / double(n));
    c->half[i] = (n & 1) ? 0.5f : 0.f;
    const double mid = 0.5 * (double(c->edges[i]) + double(c->edges[i + 1]));
    const double eta = r.theta ? -std::log(std::tan(0.5 * mid)) : mid;
    c->eta_c[i] = float(eta);
    c->inv_cosh[i] = float(1.0 / std::cosh(eta));
  }
  c->offset[nb] = acc;
  return PD_OK;
}
