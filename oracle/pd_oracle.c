/*
 * pd_oracle.c -- fp64 single-threaded CPU ORACLE (test infrastructure, see pd_oracle.h).
 *
 * Written from SURVEY.md 8c.2 (steps O0..O7) and the readings A1..A32 of DESIGN.md; the steps it
 * follows are the ones the paper names in P:L46 / P:L81 / P:L653-657.  Plain C99, one thread, no
 * blocking, fusion or reordering: every step is the formula of the reading, written out.
 * Build: gcc -O2 -ffp-contract=off -std=c99 -shared -fPIC (oracle/build.py).
 */
#include "pd_oracle.h"

#include <ctype.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#define PDO_MAX_EFF_ROWS 32
#define PDO_PI 3.14159265358979323846
#define PDO_TWO_PI 6.28318530717958647692
#define PDO_MAX_RES_ROWS 8
#define PDO_REL_TOL 1e-6 /* near-edge band of BASELINE.json north_star / SURVEY 8c.4 */

struct pdo_card {
  char name[64];
  double bz, radius, half_length, kappa; /* tesla, metres, metres, GeV/(T m)  (reading A1, A2) */
  int grid_coord;                        /* 0: eta edges, 1: theta edges      (reading A15)    */
  int n_bins;
  double *edges;   /* [n_bins+1], ascending */
  int32_t *nphi;   /* [n_bins]              */
  int32_t *offset; /* [n_bins] exclusive prefix sum of nphi */
  int n_towers;    /* of this grid (for a dual card: of the ECAL grid + of the HCAL grid, see below) */
  /* reading K6: a second grid for the HCAL (hcal_edges / hcal_nphi).  Tower ids: the ECAL grid's towers first, then the HCAL
   * grid's; a particle's tower is looked up in the grid of the section it deposits in.  The two grids are kept as cards of
   * their own (shallow copies that share everything but the grid), so that every grid function below works on either. */
  int dual;
  struct pdo_card *view[2]; /* [0] ECAL grid, [1] HCAL grid (dual cards only) */
  int32_t hcal_base;        /* id of the HCAL grid's first tower */
  int h_n_bins;
  double *h_edges;
  int32_t *h_nphi, *h_offset;
  int n_eff;
  double eff[PDO_MAX_EFF_ROWS][5]; /* pt_lo, pt_hi, aeta_lo, aeta_hi, eps   (reading A8)      */
  int eff_species[PDO_MAX_EFF_ROWS]; /* 0: every charged particle, 1 electrons, 2 muons, 3 charged hadrons (reading J1) */
  int has_cos;
  double abs_costheta_max; /* reading A9 */
  double trk_a, trk_b;     /* sigma_rel = sqrt(a^2 + (b pT)^2) */
  int has_trk_species[4];  /* reading J2: track_res given for species 1..3 */
  double trk_a_species[4], trk_b_species[4];
  double ecal[3], hcal[3]; /* (C, S, N): sigma = sqrt(C^2 E^2 + S^2 E + N^2)  (reading A20)   */
  double thr_ecal, thr_hcal;
  /* higher card fidelity (readings K1-K3 of DESIGN.md section 17) */
  int n_ecal_eta, n_hcal_eta;            /* K1: rows (aeta_lo, aeta_hi, C, S, N) by the tower centre's |eta|  */
  double ecal_eta[PDO_MAX_RES_ROWS][5], hcal_eta[PDO_MAX_RES_ROWS][5];
  /* K4: track resolution rows (aeta_lo, aeta_hi, a, b, species 0..3) by the |eta| of the true momentum; sinh of the edges */
  int n_trk_eta;
  double trk_eta[PDO_MAX_RES_ROWS][5], trk_eta_sinh[PDO_MAX_RES_ROWS][2];
  double nsig_ecal, nsig_hcal;           /* K2: component kept iff also E' > n_sigma sigma(E')                  */
  int smear_center;                      /* K3: reported tower (eta, phi) uniform inside the cell               */
  int eflow_weighted;                    /* K5: tracks of a component without a neutral are rescaled to the weighted mean */
};

/* reading A28: every card number is rounded to fp32 at load; the oracle uses the promoted value */
static double f32(double x) { return (double)(float)x; }

const char *pdo_strerror(int code) {
  switch (code) {
    case PDO_OK: return "ok";
    case PDO_EINVAL: return "invalid argument";
    case PDO_ECARD: return "unknown card name or malformed card file";
    case PDO_ECAPACITY: return "output capacity too small";
    case PDO_EOVERRIDE: return "override outside the near-edge tolerance";
    default: return "unknown error";
  }
}

/* ------------------------------------------------------------------ cards ----------------- */

static int card_alloc_grid(pdo_card *c, int n_bins) {
  c->n_bins = n_bins;
  c->edges = (double *)calloc((size_t)n_bins + 1, sizeof(double));
  c->nphi = (int32_t *)calloc((size_t)n_bins, sizeof(int32_t));
  c->offset = (int32_t *)calloc((size_t)n_bins, sizeof(int32_t));
  return (c->edges && c->nphi && c->offset) ? 0 : -1;
}

static void card_finish(pdo_card *c) {
  int i, acc = 0;
  for (i = 0; i <= c->n_bins; ++i) c->edges[i] = f32(c->edges[i]);
  for (i = 0; i < c->n_bins; ++i) {
    c->offset[i] = acc;
    acc += c->nphi[i];
  }
  c->n_towers = acc;
  if (c->h_edges) {
    int hacc = 0;
    for (i = 0; i <= c->h_n_bins; ++i) c->h_edges[i] = f32(c->h_edges[i]);
    for (i = 0; i < c->h_n_bins; ++i) c->h_offset[i] = hacc, hacc += c->h_nphi[i];
    c->dual = 1, c->hcal_base = acc, c->n_towers = acc + hacc;
  }
  c->bz = f32(c->bz);
  c->radius = f32(c->radius);
  c->half_length = f32(c->half_length);
  c->kappa = f32(c->kappa);
  for (i = 0; i < c->n_eff; ++i) {
    int k;
    for (k = 0; k < 5; ++k) c->eff[i][k] = f32(c->eff[i][k]);
  }
  c->abs_costheta_max = f32(c->abs_costheta_max);
  c->trk_a = f32(c->trk_a);
  c->trk_b = f32(c->trk_b);
  for (i = 1; i < 4; ++i) c->trk_a_species[i] = f32(c->trk_a_species[i]), c->trk_b_species[i] = f32(c->trk_b_species[i]);
  for (i = 0; i < 3; ++i) {
    c->ecal[i] = f32(c->ecal[i]);
    c->hcal[i] = f32(c->hcal[i]);
  }
  c->thr_ecal = f32(c->thr_ecal);
  c->thr_hcal = f32(c->thr_hcal);
  for (i = 0; i < c->n_ecal_eta; ++i) {
    int k;
    for (k = 0; k < 5; ++k) c->ecal_eta[i][k] = f32(c->ecal_eta[i][k]);
  }
  for (i = 0; i < c->n_hcal_eta; ++i) {
    int k;
    for (k = 0; k < 5; ++k) c->hcal_eta[i][k] = f32(c->hcal_eta[i][k]);
  }
  for (i = 0; i < c->n_trk_eta; ++i) {
    int k;
    for (k = 0; k < 4; ++k) c->trk_eta[i][k] = f32(c->trk_eta[i][k]);
    c->trk_eta_sinh[i][0] = sinh(c->trk_eta[i][0]), c->trk_eta_sinh[i][1] = sinh(c->trk_eta[i][1]); /* sinh(inf) = inf */
  }
  c->nsig_ecal = f32(c->nsig_ecal);
  c->nsig_hcal = f32(c->nsig_hcal);
  if (c->dual) {
    /* the two grids as cards of their own: everything shared, only the grid (and its tower count) differs */
    int g;
    for (g = 0; g < 2; ++g) {
      pdo_card *v = (pdo_card *)malloc(sizeof(pdo_card));
      memcpy(v, c, sizeof(pdo_card));
      v->dual = 0, v->view[0] = v->view[1] = NULL;
      if (g == 1) v->n_bins = c->h_n_bins, v->edges = c->h_edges, v->nphi = c->h_nphi, v->offset = c->h_offset;
      v->n_towers = g == 0 ? c->hcal_base : c->n_towers - c->hcal_base;
      c->view[g] = v;
    }
  }
}

/* the three efficiency rows of BASELINE.json configs[0] in reading A8 */
static void card_default_eff(pdo_card *c) {
  static const double rows[3][5] = {{1.0, INFINITY, 0.0, 1.5, 0.97},
                                    {1.0, INFINITY, 1.5, 2.5, 0.85},
                                    {0.1, 1.0, 0.0, 2.5, 0.70}};
  memcpy(c->eff, rows, sizeof(rows));
  c->n_eff = 3;
  c->trk_a = 0.01;
  c->trk_b = 1.5e-4;
  c->thr_ecal = 0.5;
  c->thr_hcal = 1.0;
  c->kappa = 0.299792458;
}

static int card_builtin_cms(pdo_card *c) {
  /* configs[0]: d_eta 0.087, 72 phi bins for |eta|<3; 0.175, 36 phi bins for 3<|eta|<5 (A15) */
  double pos[48];
  int n = 0, k, i;
  for (k = 0; k <= 34; ++k) pos[n++] = (double)k * 0.087;
  pos[n++] = 3.0;
  for (k = 1; k <= 11; ++k) pos[n++] = 3.0 + (double)k * 0.175;
  pos[n++] = 5.0; /* n == 48: 0 plus 47 positive edges */
  if (card_alloc_grid(c, 94)) return -1;
  for (i = 0; i < 47; ++i) c->edges[i] = -pos[47 - i];
  for (i = 0; i <= 47; ++i) c->edges[47 + i] = pos[i];
  for (i = 0; i < 94; ++i) c->nphi[i] = (i < 12 || i >= 82) ? 36 : 72;
  c->bz = 3.8;
  c->radius = 1.29;
  c->half_length = 3.0;
  card_default_eff(c);
  c->ecal[0] = 0.007, c->ecal[1] = 0.07, c->ecal[2] = 0.35;
  c->hcal[0] = 0.05, c->hcal[1] = 1.5, c->hcal[2] = 0.0;
  return 0;
}

static int card_builtin_atlas(pdo_card *c) {
  /* configs[3]: uniform d_eta 0.1 x 64 phi bins for |eta| < 3.2; unspecified fields inherit cfg0 (A9) */
  int i;
  if (card_alloc_grid(c, 64)) return -1;
  for (i = 0; i <= 64; ++i) c->edges[i] = (double)(i - 32) * 0.1;
  for (i = 0; i < 64; ++i) c->nphi[i] = 64;
  c->bz = 2.0;
  c->radius = 1.15;
  c->half_length = 3.5;
  card_default_eff(c);
  c->ecal[0] = 0.0017, c->ecal[1] = 0.101, c->ecal[2] = 0.0;
  c->hcal[0] = 0.0302, c->hcal[1] = 0.5205, c->hcal[2] = 0.0;
  return 0;
}

static int card_builtin_aleph(pdo_card *c) {
  /* configs[4]: towers 0.03 rad in theta x 0.03 rad in phi, |cos theta| < 0.98 (A15) */
  int i;
  if (card_alloc_grid(c, 92)) return -1;
  c->grid_coord = 1;
  c->edges[0] = acos(0.98);
  for (i = 0; i <= 90; ++i) c->edges[1 + i] = PDO_PI / 2.0 + (double)(i - 45) * 0.03;
  c->edges[92] = acos(-0.98);
  for (i = 0; i < 92; ++i) c->nphi[i] = 210;
  c->bz = 1.5;
  c->radius = 1.8;
  c->half_length = 2.5;
  card_default_eff(c);
  c->has_cos = 1;
  c->abs_costheta_max = 0.98;
  c->ecal[0] = 0.009, c->ecal[1] = 0.18, c->ecal[2] = 0.0;
  c->hcal[0] = 0.0, c->hcal[1] = 0.85, c->hcal[2] = 0.0;
  return 0;
}

/* card text file: "key = v v v ..." lines, '#' comments; keys: name bz radius half_length kappa
 * grid(eta|theta) edges(+, may repeat) nphi(+, may repeat) eff(5 numbers, repeat per row)
 * abs_costheta_max track_res(a b) ecal_res(C S N) hcal_res(C S N) ecal_thr hcal_thr */
static int card_from_file(pdo_card *c, const char *path) {
  FILE *f = fopen(path, "r");
  char *line = NULL;
  size_t cap = 1 << 16;
  double *edges = NULL, *nphi = NULL, *hedges = NULL, *hnphi = NULL;
  int n_edges = 0, n_nphi = 0, cap_e = 0, cap_n = 0, n_he = 0, n_hn = 0, cap_he = 0, cap_hn = 0, ok = 1, i;
  if (!f) return -1;
  line = (char *)malloc(cap);
  card_default_eff(c);
  c->n_eff = 0;
  while (ok && fgets(line, (int)cap, f)) {
    char *hash = strchr(line, '#'), *eq, *key, *val, *end;
    double v[64];
    int nv = 0;
    if (hash) *hash = 0;
    eq = strchr(line, '=');
    if (!eq) continue;
    *eq = 0;
    key = line;
    while (isspace((unsigned char)*key)) ++key;
    end = key + strlen(key);
    while (end > key && isspace((unsigned char)end[-1])) *--end = 0;
    val = eq + 1;
    if (!strcmp(key, "name")) {
      while (isspace((unsigned char)*val)) ++val;
      strncpy(c->name, val, sizeof(c->name) - 1);
      end = c->name + strlen(c->name);
      while (end > c->name && isspace((unsigned char)end[-1])) *--end = 0;
      continue;
    }
    if (!strcmp(key, "grid")) {
      while (isspace((unsigned char)*val)) ++val;
      c->grid_coord = !strncmp(val, "theta", 5) ? 1 : 0;
      continue;
    }
    if (!strcmp(key, "edges") || !strcmp(key, "nphi") || !strcmp(key, "hcal_edges") || !strcmp(key, "hcal_nphi")) {
      const int h = !strncmp(key, "hcal_", 5), e = !strcmp(key + (h ? 5 : 0), "edges");
      double **arr = h ? (e ? &hedges : &hnphi) : (e ? &edges : &nphi);
      int *n = h ? (e ? &n_he : &n_hn) : (e ? &n_edges : &n_nphi);
      int *cp = h ? (e ? &cap_he : &cap_hn) : (e ? &cap_e : &cap_n);
      for (;;) {
        double x = strtod(val, &end);
        if (end == val) break;
        if (*n == *cp) {
          *cp = *cp ? 2 * *cp : 256;
          *arr = (double *)realloc(*arr, (size_t)*cp * sizeof(double));
        }
        (*arr)[(*n)++] = x;
        val = end;
      }
      continue;
    }
    for (nv = 0; nv < 64; ++nv) {
      v[nv] = strtod(val, &end);
      if (end == val) break;
      val = end;
    }
    if (!strcmp(key, "bz") && nv == 1) c->bz = v[0];
    else if (!strcmp(key, "radius") && nv == 1) c->radius = v[0];
    else if (!strcmp(key, "half_length") && nv == 1) c->half_length = v[0];
    else if (!strcmp(key, "kappa") && nv == 1) c->kappa = v[0];
    else if (!strcmp(key, "abs_costheta_max") && nv == 1) c->has_cos = 1, c->abs_costheta_max = v[0];
    else if (!strcmp(key, "track_res") && nv == 2) c->trk_a = v[0], c->trk_b = v[1];
    else if (!strcmp(key, "track_res") && nv == 3 && (v[2] == 1.0 || v[2] == 2.0 || v[2] == 3.0))
      c->has_trk_species[(int)v[2]] = 1, c->trk_a_species[(int)v[2]] = v[0], c->trk_b_species[(int)v[2]] = v[1];
    else if (!strcmp(key, "ecal_res") && nv == 3) memcpy(c->ecal, v, 3 * sizeof(double));
    else if (!strcmp(key, "hcal_res") && nv == 3) memcpy(c->hcal, v, 3 * sizeof(double));
    else if (!strcmp(key, "ecal_res_eta") && nv == 5 && c->n_ecal_eta < PDO_MAX_RES_ROWS) memcpy(c->ecal_eta[c->n_ecal_eta++], v, 5 * sizeof(double));
    else if (!strcmp(key, "hcal_res_eta") && nv == 5 && c->n_hcal_eta < PDO_MAX_RES_ROWS) memcpy(c->hcal_eta[c->n_hcal_eta++], v, 5 * sizeof(double));
    else if (!strcmp(key, "track_res_eta") && (nv == 4 || (nv == 5 && (v[4] == 0.0 || v[4] == 1.0 || v[4] == 2.0 || v[4] == 3.0))) &&
             c->n_trk_eta < PDO_MAX_RES_ROWS) {
      if (nv == 4) v[4] = 0.0;
      memcpy(c->trk_eta[c->n_trk_eta++], v, 5 * sizeof(double));
    }
    else if (!strcmp(key, "ecal_nsigma") && nv == 1) c->nsig_ecal = v[0];
    else if (!strcmp(key, "hcal_nsigma") && nv == 1) c->nsig_hcal = v[0];
    else if (!strcmp(key, "smear_tower_center") && nv == 1) c->smear_center = v[0] != 0.0;
    else if (!strcmp(key, "eflow_weighted") && nv == 1) c->eflow_weighted = v[0] != 0.0;
    else if (!strcmp(key, "ecal_thr") && nv == 1) c->thr_ecal = v[0];
    else if (!strcmp(key, "hcal_thr") && nv == 1) c->thr_hcal = v[0];
    else if (!strcmp(key, "eff") && (nv == 5 || (nv == 6 && (v[5] == 0.0 || v[5] == 1.0 || v[5] == 2.0 || v[5] == 3.0))) &&
             c->n_eff < PDO_MAX_EFF_ROWS) {
      c->eff_species[c->n_eff] = nv == 6 ? (int)v[5] : 0;
      memcpy(c->eff[c->n_eff++], v, 5 * sizeof(double));
    }
    else ok = 0;
  }
  fclose(f);
  free(line);
  if (ok && (n_edges < 2 || n_nphi != n_edges - 1)) ok = 0;
  if (ok && !(c->radius > 0 && c->half_length > 0 && c->kappa > 0)) ok = 0;
  if (ok && card_alloc_grid(c, n_edges - 1)) ok = 0;
  if (ok) {
    for (i = 0; i < n_edges; ++i) c->edges[i] = edges[i];
    for (i = 0; i < n_nphi; ++i) {
      c->nphi[i] = (int32_t)nphi[i];
      if (c->nphi[i] < 1) ok = 0;
    }
    for (i = 1; i < n_edges; ++i)
      if (!((float)edges[i] > (float)edges[i - 1])) ok = 0;
  }
  if (ok && (n_he || n_hn)) {
    /* reading K6: the HCAL's own grid */
    if (n_he < 2 || n_hn != n_he - 1) ok = 0;
    if (ok) {
      c->h_n_bins = n_he - 1;
      c->h_edges = (double *)calloc((size_t)n_he, sizeof(double));
      c->h_nphi = (int32_t *)calloc((size_t)n_hn, sizeof(int32_t));
      c->h_offset = (int32_t *)calloc((size_t)n_hn, sizeof(int32_t));
      for (i = 0; i < n_he; ++i) c->h_edges[i] = hedges[i];
      for (i = 0; i < n_hn; ++i) {
        c->h_nphi[i] = (int32_t)hnphi[i];
        if (c->h_nphi[i] < 1) ok = 0;
      }
      for (i = 1; i < n_he; ++i)
        if (!((float)hedges[i] > (float)hedges[i - 1])) ok = 0;
    }
  }
  free(edges);
  free(nphi);
  free(hedges);
  free(hnphi);
  return ok ? 0 : -1;
}

int pdo_load_card(const char *name_or_path, pdo_card **out) {
  pdo_card *c;
  int rc;
  if (!name_or_path || !out) return PDO_EINVAL;
  c = (pdo_card *)calloc(1, sizeof(pdo_card));
  if (!c) return PDO_EINVAL;
  strncpy(c->name, name_or_path, sizeof(c->name) - 1);
  if (!strcmp(name_or_path, "cms_like")) rc = card_builtin_cms(c);
  else if (!strcmp(name_or_path, "atlas_like")) rc = card_builtin_atlas(c);
  else if (!strcmp(name_or_path, "aleph_like")) rc = card_builtin_aleph(c);
  else rc = card_from_file(c, name_or_path);
  if (rc) {
    pdo_free_card(c);
    return PDO_ECARD;
  }
  card_finish(c);
  *out = c;
  return PDO_OK;
}

void pdo_free_card(pdo_card *c) {
  if (!c) return;
  free(c->edges);
  free(c->nphi);
  free(c->offset);
  free(c->h_edges), free(c->h_nphi), free(c->h_offset);
  free(c->view[0]), free(c->view[1]);
  free(c);
}

int pdo_card_info(const pdo_card *c, pdo_card_info_t *out) {
  if (!c || !out) return PDO_EINVAL;
  out->n_towers = c->n_towers;
  out->n_eta_bins = c->n_bins;
  out->grid_coord = c->grid_coord;
  out->bz = (float)c->bz;
  out->radius = (float)c->radius;
  out->half_length = (float)c->half_length;
  out->n_eff_rows = c->n_eff;
  return PDO_OK;
}

int pdo_card_grid(const pdo_card *c, double *edges, int32_t *nphi, int32_t *offset) {
  int i;
  if (!c) return PDO_EINVAL;
  for (i = 0; i <= c->n_bins && edges; ++i) edges[i] = c->edges[i];
  for (i = 0; i < c->n_bins; ++i) {
    if (nphi) nphi[i] = c->nphi[i];
    if (offset) offset[i] = c->offset[i];
  }
  return PDO_OK;
}

int pdo_card_hcal_grid(const pdo_card *c, double *edges, int32_t *nphi, int32_t *base) {
  int i;
  if (!c) return PDO_EINVAL;
  if (!c->dual) return 0;
  for (i = 0; i <= c->h_n_bins && edges; ++i) edges[i] = c->h_edges[i];
  for (i = 0; i < c->h_n_bins && nphi; ++i) nphi[i] = c->h_nphi[i];
  if (base) *base = c->hcal_base;
  return c->h_n_bins;
}

/* ------------------------------------------------------------------ O0: RNG ---------------- */
/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11), as restated in SURVEY 8c.2 O0. */

void pdo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  int r;
  for (r = 0; r < 10; ++r) {
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)p1;
    uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)p0;
    c0 = n0, c1 = n1, c2 = n2, c3 = n3;
    k0 += W0, k1 += W1;
  }
  out[0] = c0, out[1] = c1, out[2] = c2, out[3] = c3;
}

/* reading A26/A27: key = (seed lo, seed hi); counter = (object, event lo, event hi, stream<<16 | block),
 * block = 0.  stream 0: object = particle index within its event; stream 1: object = tower id. */
void pdo_rng_block(uint64_t seed, int64_t event, uint32_t object, uint32_t stream, uint32_t out[4]) {
  uint32_t ctr[4], key[2];
  uint64_t ev = (uint64_t)event;
  ctr[0] = object;
  ctr[1] = (uint32_t)ev;
  ctr[2] = (uint32_t)(ev >> 32);
  ctr[3] = stream << 16;
  key[0] = (uint32_t)seed;
  key[1] = (uint32_t)(seed >> 32);
  pdo_philox4x32_10(ctr, key, out);
}

double pdo_uniform(uint32_t x) { return (double)(x >> 8) * (1.0 / 16777216.0); }
double pdo_uniform_pos(uint32_t x) { return ((double)(x >> 8) + 1.0) * (1.0 / 16777216.0); }

/* z = sqrt(-2 ln u+(xa)) cos(2 pi u(xb)) */
double pdo_normal(uint32_t xa, uint32_t xb) {
  return sqrt(-2.0 * log(pdo_uniform_pos(xa))) * cos(PDO_TWO_PI * pdo_uniform(xb));
}

/* reading A21: log-normal with mean m and standard deviation s driven by a standard normal z */
double pdo_lognormal(double m, double s, double z) {
  double b2;
  if (!(m > 0.0)) return 0.0;
  if (!(s > 0.0)) return m;
  b2 = log(1.0 + (s * s) / (m * m));
  return exp(log(m) - 0.5 * b2 + sqrt(b2) * z);
}

static double resolution(const double csn[3], double E) {
  return sqrt(csn[0] * csn[0] * E * E + csn[1] * csn[1] * E + csn[2] * csn[2]);
}

/* reading K5: the factor on the EFlow entries of the tracks of a tower component whose neutral excess
 * is not emitted: tracks measure T with variance V = sum (sigma_rel,i E_trk,i)^2, the calorimeter E' with variance s2 =
 * sigma(E')^2; the weighted mean (T / V + E' / s2) / (1 / V + 1 / s2) = (T s2 + E' V) / (s2 + V), over T.  No calorimeter
 * information (E' = 0: nothing deposited or the component was cut) or no tracks: 1.  V = s2 = 0: 1. */
double pdo_eflow_weight(double T, double V, double Ec, double sigma_c) {
  const double s2 = sigma_c * sigma_c;
  if (!(T > 0.0) || !(Ec > 0.0) || !(s2 + V > 0.0)) return 1.0;
  return (T * s2 + Ec * V) / ((s2 + V) * T);
}

/* reading K4: (a, b) of step S3 for a track of the given species with true vertex momentum
 * (px, py, pz): the first track_res_eta row, in file order, that names no species or this one and whose
 * [aeta_lo, aeta_hi) holds |eta_mom| -- decided as sinh(aeta_lo) pT <= |pz| < sinh(aeta_hi) pT in fp64 (pT = sqrt(px^2 +
 * py^2), products and sum rounded one by one), the form in which the CUDA path can take the same decision bit for bit;
 * else reading J2: the species' own track_res line, else the card's common one.  Returns the row or -1. */
int pdo_track_resolution(const pdo_card *c, int species, double px, double py, double pz, double *a, double *b) {
  const double pt = sqrt(px * px + py * py), apz = fabs(pz);
  int r;
  if (species < 1 || species > 3) species = PDO_SPECIES_CHHAD;
  for (r = 0; r < c->n_trk_eta; ++r) {
    const int sp = (int)c->trk_eta[r][4];
    if ((sp == 0 || sp == species) && apz >= c->trk_eta_sinh[r][0] * pt && apz < c->trk_eta_sinh[r][1] * pt) {
      *a = c->trk_eta[r][2], *b = c->trk_eta[r][3];
      return r;
    }
  }
  *a = c->has_trk_species[species] ? c->trk_a_species[species] : c->trk_a;
  *b = c->has_trk_species[species] ? c->trk_b_species[species] : c->trk_b;
  return -1;
}

/* reading K1: (C, S, N) of a tower = the first row whose [aeta_lo, aeta_hi) holds the |eta| of the tower CENTRE, else the
 * card's common line */
static const double *resolution_row(const double dflt[3], const double rows[][5], int n_rows, double aeta_c) {
  int r;
  for (r = 0; r < n_rows; ++r)
    if (aeta_c >= rows[r][0] && aeta_c < rows[r][1]) return rows[r] + 2;
  return dflt;
}

/* ------------------------------------------------------------------ grid ------------------- */

static double tol_angle(double edge) { return PDO_REL_TOL * fmax(1.0, fabs(edge)); }

/* bin i with edges[i] <= coord < edges[i+1]; -1 if outside (reading A16) */
static int grid_bin(const pdo_card *c, double coord) {
  int i;
  if (!(coord >= c->edges[0]) || !(coord < c->edges[c->n_bins])) return -1;
  for (i = 0; i < c->n_bins; ++i)
    if (coord < c->edges[i + 1]) return i;
  return -1;
}

static int phi_bin(int n, double phi_pos) {
  int j = (int)floor((phi_pos + PDO_PI) / (PDO_TWO_PI / (double)n));
  if (j < 0) j = 0;
  if (j > n - 1) j = n - 1;
  return j;
}

int32_t pdo_tower_index(const pdo_card *c, double coord, double phi_pos) {
  int i = grid_bin(c, coord);
  if (i < 0) return -1;
  return c->offset[i] + phi_bin(c->nphi[i], phi_pos);
}

/* reading K6: the grid a deposit of section det (0 ECAL, 1 HCAL) is looked up in, and the id of its first tower */
static const pdo_card *grid_of(const pdo_card *c, int det, int32_t *base) {
  *base = (c->dual && det) ? c->hcal_base : 0;
  return c->dual ? c->view[det ? 1 : 0] : c;
}
int32_t pdo_tower_index_det(const pdo_card *c, int det, double coord, double phi_pos) {
  int32_t base, t;
  const pdo_card *g = grid_of(c, det, &base);
  t = pdo_tower_index(g, coord, phi_pos);
  return t < 0 ? t : base + t;
}
/* the grid that holds tower id `tower` of the card, and the id inside it */
static const pdo_card *grid_of_tower(const pdo_card *c, int32_t *tower) {
  if (!c->dual) return c;
  if (*tower >= c->hcal_base) {
    *tower -= c->hcal_base;
    return c->view[1];
  }
  return c->view[0];
}

/* is `tower` an outcome the position (coord, phi) may legitimately take within the tolerance? */
static int tower_allowed(const pdo_card *c, double coord, double phi_pos, int32_t tower) {
  int i, j, n;
  double lo, hi, w, plo, phi_edge_lo, phi_edge_hi, d;
  if (tower < 0) {
    if (!(coord == coord)) return 1;
    return coord < c->edges[0] + tol_angle(c->edges[0]) ||
           coord >= c->edges[c->n_bins] - tol_angle(c->edges[c->n_bins]);
  }
  if (tower >= c->n_towers) return 0;
  for (i = c->n_bins - 1; i > 0; --i)
    if (c->offset[i] <= tower) break;
  j = tower - c->offset[i];
  n = c->nphi[i];
  lo = c->edges[i], hi = c->edges[i + 1];
  if (!(coord >= lo - tol_angle(lo) && coord < hi + tol_angle(hi))) return 0;
  w = PDO_TWO_PI / (double)n;
  phi_edge_lo = -PDO_PI + (double)j * w;
  phi_edge_hi = -PDO_PI + (double)(j + 1) * w;
  if (phi_pos >= phi_edge_lo - tol_angle(phi_edge_lo) && phi_pos < phi_edge_hi + tol_angle(phi_edge_hi))
    return 1;
  /* wrap-around: phi = +pi and phi = -pi are the same direction */
  plo = phi_pos + PDO_TWO_PI;
  d = tol_angle(PDO_PI);
  if (plo >= phi_edge_lo - d && plo < phi_edge_hi + d) return 1;
  plo = phi_pos - PDO_TWO_PI;
  if (plo >= phi_edge_lo - d && plo < phi_edge_hi + d) return 1;
  return 0;
}

/* near-edge bits of the tower decision (D5) */
static uint32_t tower_near(const pdo_card *c, double coord, double phi_pos) {
  uint32_t near = 0;
  int i = grid_bin(c, coord), k, n;
  double x, fr, w, e;
  if (!(coord == coord) || isinf(coord)) return 0;
  for (k = 0; k <= c->n_bins; ++k)
    if (fabs(coord - c->edges[k]) <= tol_angle(c->edges[k])) near |= PDO_NEAR_ETA;
  if (i < 0) {
    /* outside: the phi bin matters only if the eta decision may flip into the grid */
    if (!near) return 0;
    i = coord < c->edges[0] ? 0 : c->n_bins - 1;
  }
  for (k = (i > 0 ? i - 1 : 0); k <= (i + 1 < c->n_bins ? i + 1 : c->n_bins - 1); ++k) {
    if (k != i && !near) continue;
    n = c->nphi[k];
    w = PDO_TWO_PI / (double)n;
    x = (phi_pos + PDO_PI) / w;
    fr = x - floor(x + 0.5); /* signed distance to the nearest boundary, in bins */
    e = -PDO_PI + floor(x + 0.5) * w;
    if (fabs(fr) * w <= tol_angle(e)) near |= PDO_NEAR_PHI;
  }
  return near;
}

int pdo_tower_centre(const pdo_card *c, int32_t tower, double *eta_c, double *phi_c) {
  int i, j;
  double mid;
  if (!c || tower < 0 || tower >= c->n_towers) return PDO_EINVAL;
  if (c->dual) c = grid_of_tower(c, &tower);
  for (i = c->n_bins - 1; i > 0; --i)
    if (c->offset[i] <= tower) break;
  j = tower - c->offset[i];
  mid = 0.5 * (c->edges[i] + c->edges[i + 1]);
  if (eta_c) *eta_c = c->grid_coord ? -log(tan(0.5 * mid)) : mid;
  if (phi_c) *phi_c = -PDO_PI + ((double)j + 0.5) * (PDO_TWO_PI / (double)c->nphi[i]);
  return PDO_OK;
}

/* ------------------------------------------------------------------ O3: efficiency --------- */

/* mode 0: exact; +1: loose (conditions widened by the tolerance); -1: strict (narrowed) */
/* reading J1: a row applies to every charged particle (species 0) or to one species only */
static int species_of(int32_t pid) {
  const int32_t a = pid < 0 ? -pid : pid;
  return a == 11 ? PDO_SPECIES_ELECTRON : (a == 13 ? PDO_SPECIES_MUON : PDO_SPECIES_CHHAD);
}

static int eff_row_match(const pdo_card *c, int r, double pt, double aeta, int mode, int species) {
  const double *row = c->eff[r];
  double m = (double)mode;
  double t0 = m * PDO_REL_TOL * fabs(row[0]), t1 = isinf(row[1]) ? 0.0 : m * PDO_REL_TOL * fabs(row[1]);
  double t2 = m * tol_angle(row[2]), t3 = isinf(row[3]) ? 0.0 : m * tol_angle(row[3]);
  if (c->eff_species[r] != 0 && c->eff_species[r] != species) return 0;
  if (!(pt > row[0] - t0)) return 0;
  if (!(pt <= row[1] + t1)) return 0;
  if (row[2] > 0.0 ? !(aeta >= row[2] - t2) : 0) return 0;
  if (!(aeta < row[3] + t3)) return 0;
  return 1;
}

double pdo_efficiency(const pdo_card *c, double pt, double eta_mom, double abs_costheta, int *row) {
  return pdo_efficiency_species(c, pt, eta_mom, abs_costheta, PDO_SPECIES_CHHAD, row);
}

double pdo_efficiency_species(const pdo_card *c, double pt, double eta_mom, double abs_costheta, int species, int *row) {
  int r;
  double aeta = fabs(eta_mom);
  if (row) *row = -1;
  if (c->has_cos && abs_costheta >= c->abs_costheta_max) return 0.0;
  for (r = 0; r < c->n_eff; ++r)
    if (eff_row_match(c, r, pt, aeta, 0, species)) {
      if (row) *row = r;
      return c->eff[r][4];
    }
  return 0.0;
}

static int eff_row_allowed(const pdo_card *c, double pt, double aeta, double abs_costheta, int row, int species) {
  int r;
  if (row >= c->n_eff) return 0;
  if (c->has_cos) {
    double t = tol_angle(c->abs_costheta_max);
    if (row >= 0 && abs_costheta >= c->abs_costheta_max + t) return 0;
    if (row < 0 && abs_costheta >= c->abs_costheta_max - t) return 1;
  }
  for (r = 0; r < (row < 0 ? c->n_eff : row); ++r)
    if (eff_row_match(c, r, pt, aeta, -1, species)) return 0;
  return row < 0 ? 1 : eff_row_match(c, row, pt, aeta, +1, species);
}

static uint32_t eff_near(const pdo_card *c, double pt, double aeta, double abs_costheta) {
  int r;
  if (c->has_cos && fabs(abs_costheta - c->abs_costheta_max) <= tol_angle(c->abs_costheta_max))
    return PDO_NEAR_EFF;
  for (r = 0; r < c->n_eff; ++r) {
    const double *row = c->eff[r];
    if (fabs(pt - row[0]) <= PDO_REL_TOL * fabs(row[0])) return PDO_NEAR_EFF;
    if (!isinf(row[1]) && fabs(pt - row[1]) <= PDO_REL_TOL * fabs(row[1])) return PDO_NEAR_EFF;
    if (row[2] > 0.0 && fabs(aeta - row[2]) <= tol_angle(row[2])) return PDO_NEAR_EFF;
    if (!isinf(row[3]) && fabs(aeta - row[3]) <= tol_angle(row[3])) return PDO_NEAR_EFF;
  }
  return 0;
}

/* ------------------------------------------------------------------ O2: propagation -------- */

typedef struct {
  int status;           /* face | PDO_LOOPER */
  double x, y, z;       /* hit position, metres */
  double alpha;         /* turning angle (0 for straight lines) */
  double eta_pos, phi_pos, coord; /* coord = eta_pos or theta_pos per the card's grid */
  uint32_t near;        /* PDO_NEAR_VERTEX | PDO_NEAR_FACE | PDO_NEAR_LOWPT */
  int face_ov_bad;      /* a face override was requested outside the tolerance */
} pdo_hit;

static double sgn(double x) { return x > 0.0 ? 1.0 : (x < 0.0 ? -1.0 : 0.0); }

/* ov_face: -1 none, PDO_BARREL / PDO_ENDCAP to force the D2 decision (honoured only when near) */
static void propagate(const pdo_card *c, int q, double px, double py, double pz, double vx,
                      double vy, double vz, int ov_face, pdo_hit *h) {
  const double R = c->radius, L = c->half_length, B = c->bz;
  double pt2 = px * px + py * py, pt = hypot(px, py), r0 = hypot(vx, vy);
  double x = 0, y = 0, z = 0, alpha = 0;
  int face = PDO_DROPPED, looper = 0;
  memset(h, 0, sizeof(*h));
  /* near-edge bookkeeping of D1 and D7 */
  if (fabs(r0 - R) <= PDO_REL_TOL * R || fabs(fabs(vz) - L) <= PDO_REL_TOL * L) h->near |= PDO_NEAR_VERTEX;
  if (fabs(pt2 - 1e-9) <= PDO_REL_TOL * 1e-9) h->near |= PDO_NEAR_LOWPT;
  /* readings A4, A5: born on/outside the cylinder, or (almost) no transverse momentum: dropped */
  if (r0 >= R || fabs(vz) >= L || pt2 < 1e-9) {
    h->status = PDO_DROPPED;
    h->eta_pos = h->phi_pos = h->coord = NAN;
    return;
  }
  if (q == 0 || B == 0.0) {
    /* straight line: |v + t p|_perp = R  or  z = sgn(pz) L, whichever comes first */
    double a = pt2, b = vx * px + vy * py, cc = r0 * r0 - R * R;
    double tR = (-b + sqrt(b * b - a * cc)) / a;
    double tZ = pz != 0.0 ? (sgn(pz) * L - vz) / pz : INFINITY;
    int endcap = tZ < tR;
    if (isfinite(tZ) && fabs(tR - tZ) <= PDO_REL_TOL * fmax(tR, tZ)) {
      h->near |= PDO_NEAR_FACE;
      if (ov_face == PDO_BARREL) endcap = 0;
      if (ov_face == PDO_ENDCAP) endcap = 1;
    } else if (ov_face >= 0 && ov_face != (endcap ? PDO_ENDCAP : PDO_BARREL)) {
      h->face_ov_bad = 1;
    }
    if (endcap) {
      x = vx + tZ * px, y = vy + tZ * py, z = sgn(pz) * L;
      face = PDO_ENDCAP;
    } else {
      x = vx + tR * px, y = vy + tR * py, z = vz + tR * pz;
      face = PDO_BARREL;
    }
  } else {
    /* helix: radius rho, rotation sense s (reading A3: q > 0 in +z field turns clockwise) */
    double aq = fabs((double)q);
    double rho = pt / (c->kappa * aq * fabs(B));
    double s = -sgn((double)q * B);
    double phi0 = atan2(py, px);
    double cx = vx - s * rho * sin(phi0), cy = vy + s * rho * cos(phi0);
    double rc = hypot(cx, cy), dx = vx - cx, dy = vy - cy;
    double aR = INFINITY, aZ = INFINITY, Cs = 2.0, h2;
    int endcap, near_loop = 0, near_corner = 0, reach;
    if (rc > 0.0) Cs = (R * R - rc * rc - rho * rho) / (2.0 * rc * rho);
    reach = rc > 0.0 && Cs <= 1.0;
    if (fabs(rc + rho - R) <= PDO_REL_TOL * R) near_loop = 1;
    if (near_loop && ov_face == PDO_BARREL) reach = rc > 0.0;
    if (near_loop && ov_face == PDO_ENDCAP) reach = 0;
    if (reach) {
      double psis = acos(fmax(fmin(Cs, 1.0), -1.0));
      double psi0 = atan2(cx * dy - cy * dx, cx * dx + cy * dy);
      if (psi0 < 0.0) psi0 += PDO_TWO_PI;
      aR = s > 0.0 ? (PDO_TWO_PI - psis - psi0) : (psi0 - psis);
      if (aR < 0.0) aR = 0.0;
    } else {
      looper = PDO_LOOPER;
    }
    if (pz != 0.0) aZ = (sgn(pz) * L - vz) * pt / (rho * pz);
    if (near_loop) h->near |= PDO_NEAR_FACE;
    if (isinf(aR) && isinf(aZ)) {
      /* trapped: never leaves the tracker volume (reading A6) */
      h->status = PDO_DROPPED | looper;
      h->eta_pos = h->phi_pos = h->coord = NAN;
      if (ov_face >= 0 && !near_loop) h->face_ov_bad = 1;
      return;
    }
    endcap = aZ < aR;
    if (isfinite(aR) && isfinite(aZ) && fabs(aR - aZ) <= PDO_REL_TOL * fmax(aR, aZ)) near_corner = 1;
    if (near_corner) {
      h->near |= PDO_NEAR_FACE;
      if (ov_face == PDO_BARREL) endcap = 0;
      if (ov_face == PDO_ENDCAP) endcap = 1;
    }
    if (ov_face >= 0 && !near_corner && !near_loop && ov_face != (endcap ? PDO_ENDCAP : PDO_BARREL))
      h->face_ov_bad = 1;
    alpha = endcap ? aZ : aR;
    /* chord form: vertex + 2 rho sin(alpha/2) (cos, sin)(phi0 + s alpha/2) */
    h2 = 0.5 * alpha;
    x = vx + 2.0 * rho * sin(h2) * cos(phi0 + s * h2);
    y = vy + 2.0 * rho * sin(h2) * sin(phi0 + s * h2);
    z = endcap ? sgn(pz) * L : vz + rho * alpha * pz / pt;
    face = endcap ? PDO_ENDCAP : PDO_BARREL;
  }
  h->status = face | looper;
  h->x = x, h->y = y, h->z = z, h->alpha = alpha;
  {
    double r = hypot(x, y);
    h->eta_pos = r > 0.0 ? asinh(z / r) : (z > 0 ? INFINITY : -INFINITY);
    h->phi_pos = atan2(y, x);
    h->coord = c->grid_coord ? atan2(r, z) : h->eta_pos;
  }
}

int pdo_propagate(const pdo_card *c, int charge, double px, double py, double pz, double vx,
                  double vy, double vz, double *x, double *y, double *z, double *alpha,
                  double *eta_pos, double *phi_pos) {
  pdo_hit h;
  propagate(c, charge, px, py, pz, vx, vy, vz, -1, &h);
  if (x) *x = h.x;
  if (y) *y = h.y;
  if (z) *z = h.z;
  if (alpha) *alpha = h.alpha;
  if (eta_pos) *eta_pos = h.eta_pos;
  if (phi_pos) *phi_pos = h.phi_pos;
  return h.status;
}

/* ------------------------------------------------------------------ O1..O7: the chain ------ */

/* order of the tower overrides by (event, tower id) */
static const pdo_overrides *g_sort_ov;
static int cmp_ov(const void *a, const void *b) {
  int64_t i = *(const int64_t *)a, j = *(const int64_t *)b;
  if (g_sort_ov->tw_event[i] != g_sort_ov->tw_event[j]) return g_sort_ov->tw_event[i] < g_sort_ov->tw_event[j] ? -1 : 1;
  if (g_sort_ov->tw_id[i] != g_sort_ov->tw_id[j]) return g_sort_ov->tw_id[i] < g_sort_ov->tw_id[j] ? -1 : 1;
  return i < j ? -1 : (i > j ? 1 : 0);
}

static int cmp_i32(const void *a, const void *b) {
  int32_t x = *(const int32_t *)a, y = *(const int32_t *)b;
  return x < y ? -1 : (x > y ? 1 : 0);
}

/* decide "value > thr" with an optional forced outcome; *near receives whether it was near */
static int above_thr(double value, double thr, double scale, int forced, int *near) {
  int res = value > thr;
  *near = fabs(value - thr) <= 1e-5 * scale; /* D6 band: the float tolerance of north_star */
  if (forced >= 0 && *near) res = forced;
  return res;
}

/* reading K2 on top of A22: the smeared component is kept iff E' > thr AND E' > n_sigma sigma(E'), sigma taken at the
 * smeared energy; near if either comparison is (n_sigma = 0 leaves A22 as it was) */
static int component_kept(double Es, double thr, const double csn[3], double nsig, int forced, int *near) {
  const double cut = nsig > 0.0 ? nsig * resolution(csn, Es) : 0.0;
  int res = Es > thr && (nsig <= 0.0 || Es > cut);
  *near = fabs(Es - thr) <= 1e-5 * fmax(thr, Es) || (nsig > 0.0 && Es > 0.0 && fabs(Es - cut) <= 1e-5 * fmax(cut, Es));
  if (forced >= 0 && *near) res = forced;
  return res;
}

/* reading K3: the reported position of a tower, uniform inside its cell (Philox stream 4, object = tower id: word 0 ->
 * eta or theta, word 1 -> phi); smear_center = 0: the cell centre */
int pdo_tower_position(const pdo_card *c, uint64_t seed, int64_t event, int32_t tower, double *eta, double *phi) {
  int i, j;
  uint32_t r[4];
  double x;
  if (!c || tower < 0 || tower >= c->n_towers) return PDO_EINVAL;
  if (!c->smear_center) return pdo_tower_centre(c, tower, eta, phi);
  pdo_rng_block(seed, event, (uint32_t)tower, 4u, r); /* object = the card's tower id */
  if (c->dual) c = grid_of_tower(c, &tower);           /* reading K6: the cell in the tower's own grid */
  for (i = c->n_bins - 1; i > 0; --i)
    if (c->offset[i] <= tower) break;
  j = tower - c->offset[i];
  x = c->edges[i] + pdo_uniform(r[0]) * (c->edges[i + 1] - c->edges[i]);
  if (eta) *eta = c->grid_coord ? -log(tan(0.5 * x)) : x;
  if (phi) *phi = -PDO_PI + ((double)j + pdo_uniform(r[1])) * (PDO_TWO_PI / (double)c->nphi[i]);
  return PDO_OK;
}

int pdo_simulate(const pdo_card *c, const pdo_events *ev, uint64_t seed, int64_t event_base,
                 pdo_tracks *trk, pdo_towers *tow, pdo_eflow *efl, pdo_debug *dbg,
                 const pdo_overrides *ov) {
  double *Eem, *Ehad, *Tem, *Thad, *Vem, *Vhad, *Fem, *Fhad, *ph_E, *nh_E;
  int32_t *wt_tower = NULL; /* K5: per EFlow track entry of the call: tower * 2 + component (1 = HCAL), -1 none */
  uint8_t *touched;
  int32_t *list, *ph_id, *nh_id;
  int64_t e, n_trk = 0, n_tow = 0, n_efl = 0, n_dbg_tw = 0, rejected = 0;
  int64_t *ov_order = NULL, ov_pos = 0;
  int rc = PDO_OK;
  if (!c || !ev || !trk || !tow || !efl || ev->n_events < 0 || ev->n_particles < 0) return PDO_EINVAL;
  if (ev->n_events > 0 && !ev->offsets) return PDO_EINVAL;
  Eem = (double *)calloc((size_t)c->n_towers * 8, sizeof(double));
  touched = (uint8_t *)calloc((size_t)c->n_towers, 1);
  list = (int32_t *)malloc((size_t)c->n_towers * 3 * sizeof(int32_t));
  ph_E = (double *)malloc((size_t)c->n_towers * 2 * sizeof(double));
  if (!Eem || !touched || !list || !ph_E) {
    free(Eem), free(touched), free(list), free(ph_E);
    return PDO_EINVAL;
  }
  if (ov && ov->n_tower_ov > 0) {
    int64_t j;
    ov_order = (int64_t *)malloc((size_t)ov->n_tower_ov * sizeof(int64_t));
    if (!ov_order) {
      free(Eem), free(touched), free(list), free(ph_E);
      return PDO_EINVAL;
    }
    for (j = 0; j < ov->n_tower_ov; ++j) ov_order[j] = j;
    g_sort_ov = ov;
    qsort(ov_order, (size_t)ov->n_tower_ov, sizeof(int64_t), cmp_ov);
  }
  Ehad = Eem + c->n_towers, Tem = Ehad + c->n_towers, Thad = Tem + c->n_towers;
  Vem = Thad + c->n_towers, Vhad = Vem + c->n_towers, Fem = Vhad + c->n_towers, Fhad = Fem + c->n_towers;
  if (c->eflow_weighted) {
    wt_tower = (int32_t *)malloc((size_t)(efl->capacity > 0 ? efl->capacity : 1) * sizeof(int32_t));
    if (!wt_tower) {
      free(Eem), free(touched), free(list), free(ph_E), free(ov_order);
      return PDO_EINVAL;
    }
  }
  ph_id = list + c->n_towers, nh_id = ph_id + c->n_towers;
  nh_E = ph_E + c->n_towers;
  trk->offsets[0] = tow->offsets[0] = efl->offsets[0] = 0;
  if (dbg && dbg->tw_offsets) dbg->tw_offsets[0] = 0;

  for (e = 0; e < ev->n_events && rc == PDO_OK; ++e) {
    int64_t i0 = ev->offsets[e], i1 = ev->offsets[e + 1], i, trk_begin = n_trk, efl_begin = n_efl;
    int n_list = 0, n_ph = 0, n_nh = 0, t;
    int64_t event = event_base + e; /* reading A27 */
    for (i = i0; i < i1; ++i) {
      /* O1 classify (reading A18) */
      int apid = ev->pid[i] < 0 ? -ev->pid[i] : ev->pid[i], q = ev->charge[i];
      int cls = apid == 11 ? PDO_CLS_ELECTRON : (apid == 13 ? PDO_CLS_MUON : PDO_CLS_CHHAD);
      double fe = (apid == 11 || apid == 22) ? 1.0 : 0.0;
      double fh = (apid == 11 || apid == 22 || apid == 13 || apid == 12 || apid == 14 || apid == 16) ? 0.0 : 1.0;
      double px = ev->px[i], py = ev->py[i], pz = ev->pz[i], E = ev->E[i];
      double pt = hypot(px, py), pt_smeared = 0.0, Etrk = 0.0, sigE = 0.0;
      int64_t my_efl = -1;
      int accepted = 0, row = -1;
      int32_t tower;
      uint32_t near;
      pdo_hit h;
      /* O2 propagate */
      propagate(c, q, px, py, pz, ev->vx[i], ev->vy[i], ev->vz[i], (ov && ov->face) ? ov->face[i] : -1, &h);
      if (h.face_ov_bad) ++rejected;
      near = h.near;
      tower = -1;
      if ((h.status & PDO_FACE_MASK) != PDO_DROPPED) {
        /* O3 track: efficiency at the true vertex momentum (A7), accept iff u < eps (A11) */
        if (q != 0) {
          double eta_mom = asinh(pz / pt), p = sqrt(pt * pt + pz * pz), act = fabs(pz) / p;
          const int species = species_of(ev->pid[i]);
          double eps = pdo_efficiency_species(c, pt, eta_mom, act, species, &row);
          uint32_t r[4];
          near |= eff_near(c, pt, fabs(eta_mom), act);
          if (ov && ov->eps_row && ov->eps_row[i] != -2 && ov->eps_row[i] != row) {
            if ((near & PDO_NEAR_EFF) && eff_row_allowed(c, pt, fabs(eta_mom), act, ov->eps_row[i], species)) {
              row = ov->eps_row[i];
              eps = row < 0 ? 0.0 : c->eff[row][4];
            } else {
              ++rejected;
            }
          }
          pdo_rng_block(seed, event, (uint32_t)(i - i0), 0u, r);
          accepted = pdo_uniform(r[0]) < eps;
          if (accepted) {
            /* track smearing (A12, A13): log-normal, mean pT, std sigma_rel pT; eta, phi unchanged */
            /* reading J2: the resolution given for the particle's species, else the card's common one */
            /* reading K4: an eta-dependent row of the card first */
            double ta, tb, srel;
            pdo_track_resolution(c, species, px, py, pz, &ta, &tb);
            srel = sqrt(ta * ta + (tb * pt) * (tb * pt));
            pt_smeared = pdo_lognormal(pt, srel * pt, pdo_normal(r[1], r[2]));
            Etrk = pt_smeared * cosh(eta_mom);
            sigE = srel * Etrk; /* K5: the track's energy resolution */
            if (n_trk >= trk->capacity || n_efl >= efl->capacity) {
              rc = PDO_ECAPACITY;
              break;
            }
            trk->src[n_trk] = (int32_t)i;
            trk->pid[n_trk] = ev->pid[i];
            trk->charge[n_trk] = (int8_t)q;
            trk->pt[n_trk] = pt_smeared;
            trk->eta[n_trk] = eta_mom;
            trk->phi[n_trk] = atan2(py, px);
            trk->E[n_trk] = Etrk;
            trk->eta_out[n_trk] = h.eta_pos;
            trk->phi_out[n_trk] = h.phi_pos;
            /* O7: the event's EFlow list starts with its accepted tracks, in particle order */
            efl->cls[n_efl] = (int8_t)cls;
            efl->src[n_efl] = (int32_t)i;
            efl->pt[n_efl] = pt_smeared;
            efl->eta[n_efl] = eta_mom;
            efl->phi[n_efl] = trk->phi[n_trk];
            efl->E[n_efl] = Etrk;
            my_efl = n_efl;
            if (wt_tower) wt_tower[n_efl] = -1;
            ++n_trk, ++n_efl;
          }
        }
        /* O4 deposit: tower of the hit position; sums in particle order (A17, A19) */
        {
          /* reading K6: a card with a grid of its own for the HCAL: the tower is looked up in the grid of the section the
           * particle deposits in (electrons and photons: ECAL; everything else, also what deposits nothing: HCAL) */
          int32_t base;
          const pdo_card *g = grid_of(c, fe != 0.0 ? 0 : 1, &base);
          tower = pdo_tower_index(g, h.coord, h.phi_pos);
          if (tower >= 0) tower += base;
          near |= tower_near(g, h.coord, h.phi_pos);
          if (ov && ov->tower && ov->tower[i] != -2 && ov->tower[i] != tower) {
            const int32_t want = ov->tower[i];
            const int in_grid = want < 0 || (want >= base && want - base < g->n_towers);
            if (in_grid && tower_allowed(g, h.coord, h.phi_pos, want < 0 ? want : want - base)) tower = want;
            else ++rejected;
          }
        }
        if (tower >= 0 && (fe != 0.0 || fh != 0.0)) {
          if (!touched[tower]) touched[tower] = 1, list[n_list++] = tower;
          Eem[tower] += fe * E;
          Ehad[tower] += fh * E;
          if (accepted) Tem[tower] += fe * Etrk, Thad[tower] += fh * Etrk;
          if (accepted) Vem[tower] += fe * sigE * sigE, Vhad[tower] += fh * sigE * sigE;
          if (accepted && wt_tower) wt_tower[my_efl] = tower * 2 + (fh != 0.0 ? 1 : 0);
        }
      }
      if (dbg) {
        if (dbg->status) dbg->status[i] = (uint8_t)h.status;
        if (dbg->x) dbg->x[i] = h.x;
        if (dbg->y) dbg->y[i] = h.y;
        if (dbg->z) dbg->z[i] = h.z;
        if (dbg->eta_pos) dbg->eta_pos[i] = h.eta_pos;
        if (dbg->phi_pos) dbg->phi_pos[i] = h.phi_pos;
        if (dbg->tower) dbg->tower[i] = tower;
        if (dbg->accepted) dbg->accepted[i] = (uint8_t)accepted;
        if (dbg->eps_row) dbg->eps_row[i] = (int8_t)row;
        if (dbg->pt_smeared) dbg->pt_smeared[i] = pt_smeared;
        if (dbg->near) dbg->near[i] = near;
      }
    }
    if (rc != PDO_OK) break;
    trk->offsets[e + 1] = n_trk;
    (void)trk_begin;

    /* O5 towers, ascending id; O6 EFlow neutrals */
    qsort(list, (size_t)n_list, sizeof(int32_t), cmp_i32);
    for (t = 0; t < n_list; ++t) {
      int32_t id = list[t];
      uint32_t r[4];
      double em_s, had_s, em_f, had_f, n_em, n_had, eta_c, phi_c;
      int forced[4] = {-1, -1, -1, -1}, nr[4], k, is_ph, is_nh;
      uint8_t tw_near = 0;
      if (ov_order) {
        /* tower overrides, visited in (event, id) order alongside the ascending tower loop */
        while (ov_pos < ov->n_tower_ov &&
               (ov->tw_event[ov_order[ov_pos]] < e ||
                (ov->tw_event[ov_order[ov_pos]] == e && ov->tw_id[ov_order[ov_pos]] < id))) {
          ++rejected; /* names a tower that received no deposit */
          ++ov_pos;
        }
        while (ov_pos < ov->n_tower_ov && ov->tw_event[ov_order[ov_pos]] == e &&
               ov->tw_id[ov_order[ov_pos]] == id) {
          int64_t j = ov_order[ov_pos++];
          for (k = 0; k < 4; ++k)
            if (ov->tw_mask[j] & (1 << k)) forced[k] = (ov->tw_value[j] >> k) & 1;
        }
      }
      pdo_rng_block(seed, event, (uint32_t)id, 1u, r);
      pdo_tower_centre(c, id, &eta_c, &phi_c);
      {
        const double *ecal = resolution_row(c->ecal, c->ecal_eta, c->n_ecal_eta, fabs(eta_c));
        const double *hcal = resolution_row(c->hcal, c->hcal_eta, c->n_hcal_eta, fabs(eta_c));
        em_s = pdo_lognormal(Eem[id], resolution(ecal, Eem[id]), pdo_normal(r[0], r[1]));
        had_s = pdo_lognormal(Ehad[id], resolution(hcal, Ehad[id]), pdo_normal(r[2], r[3]));
        /* reading A22 (+ K2): the threshold is applied twice, strictly, per component */
        em_f = component_kept(em_s, c->thr_ecal, ecal, c->nsig_ecal, forced[0], &nr[0]) ? em_s : 0.0;
        had_f = component_kept(had_s, c->thr_hcal, hcal, c->nsig_hcal, forced[1], &nr[1]) ? had_s : 0.0;
      }
      n_em = em_f - Tem[id];
      n_had = had_f - Thad[id];
      is_ph = above_thr(n_em, c->thr_ecal, fmax(c->thr_ecal, fmax(em_f, Tem[id])), forced[2], &nr[2]);
      is_nh = above_thr(n_had, c->thr_hcal, fmax(c->thr_hcal, fmax(had_f, Thad[id])), forced[3], &nr[3]);
      for (k = 0; k < 4; ++k) {
        if (nr[k]) tw_near |= (uint8_t)(1 << k);
        else if (forced[k] >= 0) ++rejected;
      }
      if (dbg && dbg->tw_offsets) {
        if (n_dbg_tw >= dbg->tw_capacity) {
          rc = PDO_ECAPACITY;
          break;
        }
        if (dbg->tw_id) dbg->tw_id[n_dbg_tw] = id;
        if (dbg->Eem_true) dbg->Eem_true[n_dbg_tw] = Eem[id];
        if (dbg->Ehad_true) dbg->Ehad_true[n_dbg_tw] = Ehad[id];
        if (dbg->Tem) dbg->Tem[n_dbg_tw] = Tem[id];
        if (dbg->Thad) dbg->Thad[n_dbg_tw] = Thad[id];
        if (dbg->Eem_smeared) dbg->Eem_smeared[n_dbg_tw] = em_s;
        if (dbg->Ehad_smeared) dbg->Ehad_smeared[n_dbg_tw] = had_s;
        if (dbg->tw_near) dbg->tw_near[n_dbg_tw] = tw_near;
        ++n_dbg_tw;
      }
      pdo_tower_position(c, seed, event, id, &eta_c, &phi_c);
      if (em_f + had_f > 0.0) {
        if (n_tow >= tow->capacity) {
          rc = PDO_ECAPACITY;
          break;
        }
        tow->tower[n_tow] = id;
        tow->eta[n_tow] = eta_c;
        tow->phi[n_tow] = phi_c;
        tow->E[n_tow] = em_f + had_f;
        tow->Eem[n_tow] = em_f;
        tow->Ehad[n_tow] = had_f;
        tow->ET[n_tow] = (em_f + had_f) / cosh(eta_c);
        ++n_tow;
      }
      if (is_ph) ph_id[n_ph] = id, ph_E[n_ph] = n_em, ++n_ph;
      if (is_nh) nh_id[n_nh] = id, nh_E[n_nh] = n_had, ++n_nh;
      /* reading K5: a component with tracks whose neutral excess is not emitted hands its calorimeter measurement to the
       * tracks: their EFlow entries are rescaled to the weighted mean of the two */
      Fem[id] = Fhad[id] = 1.0;
      if (c->eflow_weighted) {
        pdo_tower_centre(c, id, &eta_c, &phi_c);
        if (!is_ph) Fem[id] = pdo_eflow_weight(Tem[id], Vem[id], em_f, resolution(resolution_row(c->ecal, c->ecal_eta, c->n_ecal_eta, fabs(eta_c)), em_f));
        if (!is_nh) Fhad[id] = pdo_eflow_weight(Thad[id], Vhad[id], had_f, resolution(resolution_row(c->hcal, c->hcal_eta, c->n_hcal_eta, fabs(eta_c)), had_f));
      }
      /* reset the dense accumulators for the next event */
      Eem[id] = Ehad[id] = Tem[id] = Thad[id] = Vem[id] = Vhad[id] = 0.0;
      touched[id] = 0;
    }
    if (rc != PDO_OK) break;
    tow->offsets[e + 1] = n_tow;
    if (dbg && dbg->tw_offsets) dbg->tw_offsets[e + 1] = n_dbg_tw;
    if (wt_tower) {
      int64_t k;
      for (k = efl_begin; k < n_efl; ++k)
        if (wt_tower[k] >= 0) {
          const double f = (wt_tower[k] & 1) ? Fhad[wt_tower[k] >> 1] : Fem[wt_tower[k] >> 1];
          efl->pt[k] *= f, efl->E[k] *= f;
        }
    }
    /* O7: EFlow = tracks (already written) ++ photons ascending id ++ neutral hadrons ascending id */
    if (n_efl + n_ph + n_nh > efl->capacity) {
      rc = PDO_ECAPACITY;
      break;
    }
    for (t = 0; t < n_ph + n_nh; ++t) {
      int is_photon = t < n_ph;
      int32_t id = is_photon ? ph_id[t] : nh_id[t - n_ph];
      double En = is_photon ? ph_E[t] : nh_E[t - n_ph], eta_c, phi_c;
      pdo_tower_position(c, seed, event, id, &eta_c, &phi_c);
      efl->cls[n_efl] = (int8_t)(is_photon ? PDO_CLS_PHOTON : PDO_CLS_NEUHAD);
      efl->src[n_efl] = id;
      efl->pt[n_efl] = En / cosh(eta_c);
      efl->eta[n_efl] = eta_c;
      efl->phi[n_efl] = phi_c;
      efl->E[n_efl] = En;
      ++n_efl;
    }
    efl->offsets[e + 1] = n_efl;
  }
  if (rc == PDO_OK && ov_order) rejected += ov->n_tower_ov - ov_pos; /* overrides never reached */
  free(Eem), free(touched), free(list), free(ph_E), free(ov_order), free(wt_tower);
  if (ov && ov->n_rejected) *ov->n_rejected = rejected;
  if (rc == PDO_OK && rejected > 0) rc = PDO_EOVERRIDE;
  return rc;
}

/* ---- event features and lepton isolation: see pd_oracle.h (Eq. 1) ---- */
int pdo_event_features(const pdo_objects *obj, double dr_max, double fsr_dr, double *ht, double *met_x,
                       double *met_y, double *met, double *iso_charged, double *iso_neutral, double *iso_photon,
                       double *r_iso, double *iso_amb) {
  const double PI = 3.14159265358979323846;
  int64_t e, i, j;
  if (!obj || obj->n_events < 0 || !obj->offsets || !ht || !met_x || !met_y || !met) return PDO_EINVAL;
  if (!iso_charged || !iso_neutral || !iso_photon || !r_iso || !(dr_max >= 0.0) || !(fsr_dr >= 0.0)) return PDO_EINVAL;
  for (e = 0; e < obj->n_events; ++e) {
    const int64_t a = obj->offsets[e], b = obj->offsets[e + 1];
    double sum_pt = 0.0, sx = 0.0, sy = 0.0;
    /* H_T and the missing transverse momentum: plain sums in object order */
    for (i = a; i < b; ++i) {
      const double pt = (double)obj->pt[i], phi = (double)obj->phi[i];
      sum_pt += pt;
      sx += pt * cos(phi);
      sy += pt * sin(phi);
    }
    ht[e] = sum_pt;
    met_x[e] = -sx;
    met_y[e] = -sy;
    met[e] = sqrt(sx * sx + sy * sy);
    /* Eq. 1 for every electron / muon of the event */
    for (i = a; i < b; ++i) {
      double s_ch = 0.0, s_nh = 0.0, s_ph = 0.0, amb = 0.0;
      const int is_lepton = obj->cls[i] == PDO_CLS_ELECTRON || obj->cls[i] == PDO_CLS_MUON;
      if (is_lepton) {
        for (j = a; j < b; ++j) {
          double deta, dphi, dr;
          if (j == i) continue; /* "the sums exclude the lepton itself" */
          deta = (double)obj->eta[j] - (double)obj->eta[i];
          dphi = (double)obj->phi[j] - (double)obj->phi[i];
          while (dphi > PI) dphi -= 2.0 * PI;
          while (dphi <= -PI) dphi += 2.0 * PI;
          dr = sqrt(deta * deta + dphi * dphi);
          if (fabs(dr - dr_max) <= 1e-6 || (obj->cls[j] == PDO_CLS_PHOTON && fsr_dr > 0.0 && fabs(dr - fsr_dr) <= 1e-6))
            amb += (double)obj->pt[j];
          if (!(dr < dr_max)) continue;
          if (obj->cls[j] == PDO_CLS_PHOTON) {
            if (!(dr < fsr_dr)) s_ph += (double)obj->pt[j]; /* reading F4 */
          } else if (obj->cls[j] == PDO_CLS_NEUHAD) {
            s_nh += (double)obj->pt[j];
          } else {
            s_ch += (double)obj->pt[j];
          }
        }
      }
      iso_charged[i] = s_ch, iso_neutral[i] = s_nh, iso_photon[i] = s_ph;
      r_iso[i] = is_lepton ? (s_ch + s_nh + s_ph) / (double)obj->pt[i] : 0.0;
      if (iso_amb) iso_amb[i] = amb;
    }
  }
  return PDO_OK;
}

/* ---- particle filter: see pd_oracle.h (Table C.13) ---- */
static int pdo_condition_holds(const pdo_condition *c, float x) {
  int k;
  if (c->use_abs) x = fabsf(x);
  switch (c->op) {
    case PDO_OP_GT: return x > c->value;
    case PDO_OP_GE: return x >= c->value;
    case PDO_OP_LT: return x < c->value;
    case PDO_OP_LE: return x <= c->value;
    case PDO_OP_EQ: return x == c->value;
    case PDO_OP_NE: return x != c->value;
    case PDO_OP_IN:
      for (k = 0; k < c->n_values; ++k)
        if (x == c->values[k]) return 1;
      return 0;
    case PDO_OP_NOT_IN:
      for (k = 0; k < c->n_values; ++k)
        if (x == c->values[k]) return 0;
      return 1;
    default: return 0;
  }
}

int pdo_filter_eflow(int64_t n_events, const int64_t *offsets, const int8_t *cls, const int32_t *src, const float *pt,
                     const float *eta, const float *phi, const float *E, const pdo_condition *conds, int32_t n_conds,
                     int32_t combine_any, int64_t *out_offsets, int8_t *out_cls, int32_t *out_src, float *out_pt,
                     float *out_eta, float *out_phi, float *out_E, uint8_t *keep) {
  int64_t e, i, n_out = 0;
  int32_t k;
  if (n_events < 0 || !offsets || !out_offsets || n_conds < 0 || (n_conds > 0 && !conds)) return PDO_EINVAL;
  for (k = 0; k < n_conds; ++k)
    if (conds[k].field < PDO_FIELD_PT || conds[k].field > PDO_FIELD_CLS || conds[k].op < PDO_OP_GT ||
        conds[k].op > PDO_OP_NOT_IN || conds[k].n_values < 0 || conds[k].n_values > 8)
      return PDO_EINVAL;
  out_offsets[0] = 0;
  for (e = 0; e < n_events; ++e) {
    for (i = offsets[e]; i < offsets[e + 1]; ++i) {
      int n_true = 0, kept;
      for (k = 0; k < n_conds; ++k) {
        const pdo_condition *c = &conds[k];
        const float x = c->field == PDO_FIELD_PT ? pt[i] : c->field == PDO_FIELD_ETA ? eta[i]
                      : c->field == PDO_FIELD_PHI ? phi[i] : c->field == PDO_FIELD_E ? E[i] : (float)cls[i];
        n_true += pdo_condition_holds(c, x);
      }
      kept = n_conds == 0 ? 1 : (combine_any ? n_true > 0 : n_true == n_conds);
      if (keep) keep[i] = (uint8_t)kept;
      if (kept) {
        out_cls[n_out] = cls[i], out_src[n_out] = src[i];
        out_pt[n_out] = pt[i], out_eta[n_out] = eta[i], out_phi[n_out] = phi[i], out_E[n_out] = E[i];
        ++n_out;
      }
    }
    out_offsets[e + 1] = n_out;
  }
  return PDO_OK;
}

/* ---- pile-up merging: see pd_oracle.h (Listing 8, Table C.9) ---- */
static int pdo_poisson_inverse(double mu, double u) {
  /* smallest n with sum_{k<=n} p_k > u; p_0 = exp(-mu), p_k = p_{k-1} mu / k */
  const int n_max = (int)ceil(mu + 10.0 * sqrt(mu) + 20.0);
  double p = exp(-mu), cdf = p;
  int n = 0;
  while (!(cdf > u) && n < n_max) {
    ++n;
    p = p * mu / (double)n;
    cdf = cdf + p;
  }
  return n;
}

/* standard normal quantile for 0 < q <= 1/2 by bisection of Phi(x) = erfc(-x / sqrt(2)) / 2 on [-40, 0] */
static double pdo_norm_quantile_lower(double q) {
  double lo = -40.0, hi = 0.0;
  int it;
  for (it = 0; it < 200; ++it) {
    const double mid = 0.5 * (lo + hi);
    if (0.5 * erfc(-mid / sqrt(2.0)) < q) lo = mid;
    else hi = mid;
  }
  return 0.5 * (lo + hi);
}

/* reading H4: normal of width sigma_z truncated to |z| <= max_z, by inversion of its distribution function with
 * the 24-bit uniform of word r1 (word r2 is not used): u = ((r1 >> 8) + 1/2) 2^-24 in (0, 1); sign = -1 if
 * u < 1/2 else +1; v = |2 u - 1| in (0, 1); |z| = -sigma_z Phi^-1(q), q = Phi(-a) + (1 - v) (1/2 - Phi(-a)),
 * a = max_z / sigma_z.  (Written through the lower tail so that the far tail keeps its relative precision.) */
static double pdo_truncated_z(uint32_t r1, double sigma_z, double max_z) {
  const double u = ((double)(r1 >> 8) + 0.5) * (1.0 / 16777216.0);
  const double sign = u < 0.5 ? -1.0 : 1.0, v = fabs(2.0 * u - 1.0);
  double lo, q;
  if (!(sigma_z > 0.0)) return 0.0;
  lo = 0.5 * erfc((max_z / sigma_z) / sqrt(2.0)); /* Phi(-a) */
  q = lo + (1.0 - v) * (0.5 - lo);
  return -sign * sigma_z * pdo_norm_quantile_lower(q);
}

/* reading H7: with sigma_t > 0 every interaction also gets a time, the same truncated normal (width sigma_t, cut at
 * max_t_spread; Table C.9) from word 2 of its block -- the hard scatter's from block 0 if smear_hs_vertex, else 0 --
 * written per particle to out_vt (seconds; may be NULL) */
int pdo_pileup_merge_t(const pdo_events *hs, const pdo_events *pool, double mean_pileup, double sigma_z,
                       double max_z_spread, double sigma_t, double max_t_spread, int smear_hs_vertex, uint64_t seed,
                       int64_t event_base, int64_t out_capacity, int64_t *out_offsets, int32_t *out_pid, int8_t *out_charge,
                       float *out_px, float *out_py, float *out_pz, float *out_E, float *out_vx, float *out_vy, float *out_vz,
                       uint8_t *is_pu, int32_t *n_pileup, float *out_vt) {
  int64_t e, n_out = 0;
  int rc = PDO_OK;
  if (!hs || !pool || !out_offsets || hs->n_events < 0 || pool->n_events < 1 || !hs->offsets || !pool->offsets) return PDO_EINVAL;
  if (!(mean_pileup >= 0.0) || mean_pileup > 500.0 || !(sigma_z >= 0.0) || !(max_z_spread >= 0.0)) return PDO_EINVAL;
  if (!(sigma_t >= 0.0) || !(max_t_spread >= 0.0)) return PDO_EINVAL;
  out_offsets[0] = 0;
  for (e = 0; e < hs->n_events; ++e) {
    const int64_t event = event_base + e;
    uint32_t r[4];
    int n, k, s;
    double dz_hs, dt_hs;
    pdo_rng_block(seed, event, 0u, 2u, r);
    n = pdo_poisson_inverse(mean_pileup, pdo_uniform(r[0]));
    dz_hs = smear_hs_vertex ? pdo_truncated_z(r[1], sigma_z, max_z_spread) : 0.0;
    dt_hs = smear_hs_vertex ? pdo_truncated_z(r[2], sigma_t, max_t_spread) : 0.0;
    if (n_pileup) n_pileup[e] = n;
    /* sources: s = -1 the hard-scatter event, s = k the k-th pile-up interaction */
    for (s = -1; s < n; ++s) {
      const pdo_events *src = hs;
      int64_t a = hs->offsets[e], b = hs->offsets[e + 1], i;
      double dz = dz_hs, dt = dt_hs;
      k = s;
      if (s >= 0) {
        int64_t j;
        pdo_rng_block(seed, event, (uint32_t)(1 + k), 2u, r);
        j = (int64_t)(((uint64_t)(r[0] >> 8) * (uint64_t)pool->n_events) >> 24);
        dz = pdo_truncated_z(r[1], sigma_z, max_z_spread);
        dt = pdo_truncated_z(r[2], sigma_t, max_t_spread);
        src = pool, a = pool->offsets[j], b = pool->offsets[j + 1];
      }
      for (i = a; i < b; ++i, ++n_out) {
        if (n_out >= out_capacity) {
          rc = PDO_ECAPACITY;
          continue;
        }
        out_pid[n_out] = src->pid[i], out_charge[n_out] = src->charge[i];
        out_px[n_out] = src->px[i], out_py[n_out] = src->py[i], out_pz[n_out] = src->pz[i], out_E[n_out] = src->E[i];
        out_vx[n_out] = src->vx[i], out_vy[n_out] = src->vy[i];
        out_vz[n_out] = (float)((double)src->vz[i] + dz);
        if (is_pu) is_pu[n_out] = (uint8_t)(s >= 0);
        if (out_vt) out_vt[n_out] = (float)dt;
      }
    }
    out_offsets[e + 1] = n_out;
  }
  return rc;
}

int pdo_pileup_merge(const pdo_events *hs, const pdo_events *pool, double mean_pileup, double sigma_z,
                     double max_z_spread, int smear_hs_vertex, uint64_t seed, int64_t event_base, int64_t out_capacity,
                     int64_t *out_offsets, int32_t *out_pid, int8_t *out_charge, float *out_px, float *out_py,
                     float *out_pz, float *out_E, float *out_vx, float *out_vy, float *out_vz, uint8_t *is_pu,
                     int32_t *n_pileup) {
  return pdo_pileup_merge_t(hs, pool, mean_pileup, sigma_z, max_z_spread, 0.0, 0.0, smear_hs_vertex, seed, event_base, out_capacity,
                            out_offsets, out_pid, out_charge, out_px, out_py, out_pz, out_E, out_vx, out_vy, out_vz, is_pu, n_pileup, NULL);
}

/* ---- track impact parameters (Table 2) ----
 * Geometry of one trajectory, written as the definition: the helix of step S1 (reading A3), extended in both
 * directions, or the straight line when q B = 0.  See the header for the conventions. */
int pdo_impact_true(const pdo_card *c, int q, double px, double py, double pz, double vx, double vy, double vz,
                    double *d0, double *z0) {
  const double pt = hypot(px, py), B = c->bz;
  if (!(pt > 0.0)) return PDO_EINVAL;
  if (q == 0 || B == 0.0) {
    /* straight line: closest approach at t = -(v.p)_T / pT^2; the direction of flight is the same everywhere */
    double t = -(vx * px + vy * py) / (pt * pt);
    double xd = vx + t * px, yd = vy + t * py;
    *d0 = (xd * py - yd * px) / pt;
    *z0 = vz + t * pz;
    return PDO_OK;
  }
  {
    /* circle of S1: radius rho, rotation sense s, centre (cx, cy) */
    double rho = pt / (c->kappa * fabs((double)q) * fabs(B));
    double s = -sgn((double)q * B);
    double phi0 = atan2(py, px);
    double cx = vx - s * rho * sin(phi0), cy = vy + s * rho * cos(phi0);
    double rc = hypot(cx, cy);
    double xd, yd, tx, ty, psi_v, psi_d, alpha;
    if (rc == 0.0) {
      /* the circle is centred on the axis: every point is equally close; the vertex itself is taken */
      *d0 = (vx * py - vy * px) / pt;
      *z0 = vz;
      return PDO_OK;
    }
    /* the point of the circle nearest to the axis lies on the line from the centre through the origin */
    xd = cx - rho * cx / rc, yd = cy - rho * cy / rc;
    /* direction of flight there: the radius vector (xd - cx, yd - cy) turned by s * 90 degrees */
    tx = -s * (yd - cy) / rho, ty = s * (xd - cx) / rho;
    *d0 = xd * ty - yd * tx;
    /* turning angle from the vertex to that point, in the sense of rotation, the shorter way round */
    psi_v = atan2(vy - cy, vx - cx), psi_d = atan2(yd - cy, xd - cx);
    alpha = remainder(s * (psi_d - psi_v), PDO_TWO_PI);
    *z0 = vz + rho * alpha * pz / pt;
  }
  return PDO_OK;
}

int pdo_track_impact(const pdo_card *c, const pdo_events *ev, const int64_t *trk_offsets, const int32_t *trk_src,
                     double d0_a, double d0_b, double z0_a, double z0_b, uint64_t seed, int64_t event_base,
                     double *d0_true, double *z0_true, double *d0, double *z0, double *d0_err, double *z0_err) {
  int64_t e, t;
  if (!c || !ev || !trk_offsets || !trk_src || !d0 || !z0 || !d0_err || !z0_err) return PDO_EINVAL;
  if (d0_a < 0 || d0_b < 0 || z0_a < 0 || z0_b < 0) return PDO_EINVAL;
  for (e = 0; e < ev->n_events; ++e) {
    for (t = trk_offsets[e]; t < trk_offsets[e + 1]; ++t) {
      const int64_t i = trk_src[t];
      double dt, zt, pt, sd, sz;
      uint32_t r[4];
      int rc;
      if (i < ev->offsets[e] || i >= ev->offsets[e + 1]) return PDO_EINVAL;
      rc = pdo_impact_true(c, ev->charge[i], ev->px[i], ev->py[i], ev->pz[i], ev->vx[i], ev->vy[i], ev->vz[i], &dt, &zt);
      if (rc != PDO_OK) return rc;
      pt = hypot((double)ev->px[i], (double)ev->py[i]);
      /* reading I2: sigma = a (+) b / pT, Gaussian, independent for d0 and z0; reported as the errors */
      sd = sqrt(d0_a * d0_a + (d0_b / pt) * (d0_b / pt));
      sz = sqrt(z0_a * z0_a + (z0_b / pt) * (z0_b / pt));
      /* reading I3: stream 3 of A26, object = particle index within its event; words 0,1 -> d0, words 2,3 -> z0 */
      pdo_rng_block(seed, event_base + e, (uint32_t)(i - ev->offsets[e]), 3u, r);
      if (d0_true) d0_true[t] = dt;
      if (z0_true) z0_true[t] = zt;
      d0[t] = dt + sd * pdo_normal(r[0], r[1]);
      z0[t] = zt + sz * pdo_normal(r[2], r[3]);
      d0_err[t] = sd, z0_err[t] = sz;
    }
  }
  return PDO_OK;
}

/* ---- truth-level event features (Table 2 "H_T, E_T^miss values for Truth and PFlow collections";
 * P:L398 "Truth HT") -- readings T1, T2 of DESIGN.md section 15 ---- */
int pdo_truth_features(const pdo_events *ev, int skip_neutrinos, double *ht, double *met_x, double *met_y, double *met) {
  int64_t e, i;
  if (!ev || !ht || !met_x || !met_y || !met) return PDO_EINVAL;
  for (e = 0; e < ev->n_events; ++e) {
    double h = 0.0, sx = 0.0, sy = 0.0;
    for (i = ev->offsets[e]; i < ev->offsets[e + 1]; ++i) {
      const int32_t a = ev->pid[i] < 0 ? -ev->pid[i] : ev->pid[i];
      if (skip_neutrinos && (a == 12 || a == 14 || a == 16)) continue; /* T2: invisible particles */
      h += hypot((double)ev->px[i], (double)ev->py[i]);
      sx += (double)ev->px[i], sy += (double)ev->py[i];
    }
    ht[e] = h, met_x[e] = -sx, met_y[e] = -sy, met[e] = hypot(sx, sy);
  }
  return PDO_OK;
}
