/*
 * pd_oracle.h -- fp64, single-threaded CPU ORACLE of the Delphes-style detector response.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing under oracle/ is part of the product path: only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may build, link or
 * call it.  It shares no code, header, table or constant generator with the CUDA path
 * (paper_2606_26089_b200/csrc, include/pd.h); both were written separately from SURVEY.md section 8c.
 *
 * What it computes (citations: P:Lnnn = /root/reference/PAPER.md line nnn):
 *   the TorchDelphes chain named in P:L46 and P:L81 -- "particle propagation through the magnetic
 *   field, tracking efficiency, momentum smearing, calorimeter response, and energy-flow merging,
 *   with per-module parameters loaded from the selected detector card" -- up to "the generation of
 *   calorimeter tower hits (Towers) and reconstructed photons, neutral hadrons, and charged tracks
 *   (EFlowObjects)".  The paper prints no formula for any step; the formulas are the
 *   readings A1..A32 listed in DESIGN.md (from SURVEY.md 8c.2 / 8c.3 and BASELINE.json configs).
 *
 * Parity status: every function below is pinned by tests/test_oracle_*.py (Philox known-answer
 * vectors, RK4 integration of the Lorentz force, closed forms, the worked values of
 * the text fixtures under tests/golden, invariants, a brute-force tiny event; the event features / isolation,
 * the particle filter and the pile-up merging further down by tests/test_oracle_features.py, _filter.py,
 * _pileup.py: hand-worked cases, scipy quantiles, numpy re-derivations).  What stays UNPINNED is the choice of
 * readings versus the paper's own software (not in the container): "parity with the paper's
 * software: unpinned" -- see DESIGN.md.
 *
 * All pointers are HOST pointers owned by the caller.  Nothing is allocated for outputs.
 */
#ifndef PD_ORACLE_H
#define PD_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pdo_card pdo_card;

/* status byte: low two bits = face, bit 2 = looper (charged, cannot reach r = R) */
enum { PDO_DROPPED = 0, PDO_BARREL = 1, PDO_ENDCAP = 2, PDO_FACE_MASK = 3, PDO_LOOPER = 4 };

/* EFlow / particle classes (charged hadron, electron, muon, neutral hadron, photon) */
enum { PDO_CLS_CHHAD = 0, PDO_CLS_ELECTRON = 1, PDO_CLS_MUON = 2, PDO_CLS_NEUHAD = 3, PDO_CLS_PHOTON = 4 };

/* near-edge bits, per particle (SURVEY 8c.4 decisions D1, D2, D3, D5, D7) */
enum {
  PDO_NEAR_VERTEX = 1,   /* D1: r0 vs R or |vz| vs L                         */
  PDO_NEAR_FACE   = 2,   /* D2: looper threshold or barrel/endcap corner     */
  PDO_NEAR_EFF    = 4,   /* D3: a pT / |eta| / |cos theta| edge of the table */
  PDO_NEAR_ETA    = 8,   /* D5: eta (theta) bin edge or grid coverage        */
  PDO_NEAR_PHI    = 16,  /* D5: phi bin edge                                 */
  PDO_NEAR_LOWPT  = 32   /* D7: pT^2 vs 1e-9                                 */
};
/* near-threshold bits, per deposited tower (decision D6) */
enum { PDO_NEAR_EEM = 1, PDO_NEAR_EHAD = 2, PDO_NEAR_NEM = 4, PDO_NEAR_NHAD = 8 };

/* error codes */
enum { PDO_OK = 0, PDO_EINVAL = -1, PDO_ECARD = -2, PDO_ECAPACITY = -3, PDO_EOVERRIDE = -4 };

typedef struct {
  int32_t n_towers, n_eta_bins, grid_coord; /* grid_coord: 0 = eta, 1 = theta */
  float bz, radius, half_length;
  int32_t n_eff_rows;
} pdo_card_info_t;

typedef struct {
  int64_t n_events;
  int64_t n_particles;
  const int64_t *offsets; /* [n_events+1] */
  const int32_t *pid;
  const int8_t *charge;
  const float *px, *py, *pz, *E, *vx, *vy, *vz;
} pdo_events;

typedef struct {
  int64_t capacity;
  int64_t *offsets; /* [n_events+1] */
  int32_t *src, *pid;
  int8_t *charge;
  double *pt, *eta, *phi, *E, *eta_out, *phi_out;
} pdo_tracks;

typedef struct {
  int64_t capacity;
  int64_t *offsets;
  int32_t *tower;
  double *eta, *phi, *E, *Eem, *Ehad, *ET;
} pdo_towers;

typedef struct {
  int64_t capacity;
  int64_t *offsets;
  int8_t *cls;
  int32_t *src;
  double *pt, *eta, *phi, *E;
} pdo_eflow;

/* optional (NULL allowed as a whole; individual arrays may be NULL too) */
typedef struct {
  /* per particle */
  uint8_t *status;
  double *x, *y, *z, *eta_pos, *phi_pos;
  int32_t *tower;       /* geometric tower id of the hit, -1 if none */
  uint8_t *accepted;
  int8_t *eps_row;      /* row of the efficiency table used, -1 none */
  double *pt_smeared;   /* 0 if not an accepted track */
  uint32_t *near;       /* PDO_NEAR_* bits */
  /* per deposited tower (emitted or not), CSR over events */
  int64_t tw_capacity;
  int64_t *tw_offsets;  /* [n_events+1] */
  int32_t *tw_id;
  double *Eem_true, *Ehad_true, *Tem, *Thad, *Eem_smeared, *Ehad_smeared;
  uint8_t *tw_near;     /* PDO_NEAR_E* bits */
} pdo_debug;

/* optional overrides.  An override is honoured only if the oracle itself finds the
 * requested outcome within the near-edge tolerance; otherwise pdo_simulate returns PDO_EOVERRIDE
 * and *n_rejected counts the offenders. */
typedef struct {
  const int8_t *face;     /* per particle: -1 none, PDO_BARREL or PDO_ENDCAP */
  const int32_t *tower;   /* per particle: -2 none, else tower id or -1 (no tower) */
  const int8_t *eps_row;  /* per particle: -2 none, else row index or -1 (no row) */
  int64_t n_tower_ov;     /* tower-level overrides of threshold decisions */
  const int64_t *tw_event;/* event index within the call */
  const int32_t *tw_id;
  const uint8_t *tw_mask; /* which PDO_NEAR_E* decisions to force */
  const uint8_t *tw_value;/* forced outcome bits (1 = "above threshold") */
  int64_t *n_rejected;    /* out, may be NULL */
} pdo_overrides;

int pdo_load_card(const char *name_or_path, pdo_card **out);
void pdo_free_card(pdo_card *card);
int pdo_card_info(const pdo_card *card, pdo_card_info_t *out);
/* copy of the card tables for tests: edges[n_eta_bins+1], nphi[n_eta_bins], offset[n_eta_bins] */
int pdo_card_grid(const pdo_card *card, double *edges, int32_t *nphi, int32_t *offset);
/* tower centre (eta_c, phi_c) of a tower id; returns PDO_EINVAL if out of range */
int pdo_tower_centre(const pdo_card *card, int32_t tower, double *eta_c, double *phi_c);
/* reading K3: the reported position of a tower -- uniform inside the cell if the card says
 * smear_tower_center = 1 (Philox stream 4, object = tower id), else the centre */
int pdo_tower_position(const pdo_card *card, uint64_t seed, int64_t event, int32_t tower, double *eta, double *phi);

int pdo_simulate(const pdo_card *card, const pdo_events *ev, uint64_t seed, int64_t event_base,
                 pdo_tracks *tracks, pdo_towers *towers, pdo_eflow *eflow, pdo_debug *debug,
                 const pdo_overrides *ov);

/* ---- event features and lepton isolation (section 2.4 Eq. 1, Table 2) ----
 * Computed from an EFlow ("PFlow") collection in CSR form, per event:
 *   H_T = sum_i pT_i,   E_T^miss vector = -( sum_i pT_i cos phi_i, sum_i pT_i sin phi_i ),   E_T^miss = its length
 *   (readings F1, F2 of DESIGN.md section 10: the "cached scalar event features (H_T and E_T^miss)" of P:L119,
 *   "H_T, E_T^miss values for ... PFlow collections" of P:L141, taken over every object of the collection);
 * and, for every object of class electron or muon, Eq. 1 of P:L121-127:
 *   R_iso = ( sum_{dR<dr_max} pT^charged + sum_{dR<dr_max} pT^neutral + sum_{dR<dr_max} pT^gamma ) / pT^lepton,
 *   dR = sqrt(d_eta^2 + d_phi^2), d_phi wrapped into (-pi, pi], "where the sums exclude the lepton itself"
 *   (by index), charged = classes 0,1,2, neutral = class 3, gamma = class 4.  "The last term excludes photons
 *   that are candidates for final-state radiation" -- the paper gives no criterion; reading F4: photons with
 *   dR < fsr_dr are left out of the photon term (fsr_dr = 0 keeps them all).  The cone is strict (dR < dr_max).
 *   Objects of the other classes get 0 in all four isolation arrays.
 * Sums are taken in fp64 in object order.  iso_amb[i] (nullable) receives the pT sum of the objects whose dR
 * lies within 1e-6 of dr_max or fsr_dr (near-edge: either outcome is allowed for those). */
typedef struct {
  int64_t n_events;
  const int64_t *offsets; /* [n_events+1] */
  const int8_t *cls;
  const float *pt, *eta, *phi;
} pdo_objects;

int pdo_event_features(const pdo_objects *obj, double dr_max, double fsr_dr,
                       double *ht, double *met_x, double *met_y, double *met, /* [n_events] */
                       double *iso_charged, double *iso_neutral, double *iso_photon, double *r_iso, /* [n_objects] */
                       double *iso_amb /* [n_objects], may be NULL */);

/* ---- particle filter (section 2.4, P:L634-647 Table C.13) ----
 * "Particle filtering drops particles from a target collection in place according to declarative per-field
 * conditions (e.g. pT, eta, or PDG-ID cuts), combined with logical all (AND) or any (OR) semantics."
 * A condition is (field, op, value | set of values, abs): the object's attribute (its magnitude if abs) is
 * compared with `value` by >, >=, <, <=, ==, != or tested for membership in `values` (in, not in).
 * Attributes of an EFlow object: pt, eta, phi, E (fp32) and the class id (int8, compared as a number).
 * All comparisons are made on the fp32 values as they are (no arithmetic), hence exactly.  An object is
 * kept iff all (combine_any = 0) or any (combine_any = 1) of the conditions hold; an empty condition list
 * keeps everything (reading G1 of DESIGN.md section 11).  Survivors keep their order; the output is the
 * compacted CSR collection.  (Event features are then recomputed from the survivors with
 * pdo_event_features -- "update_event_features", Table C.13.) */
enum { PDO_FIELD_PT = 0, PDO_FIELD_ETA = 1, PDO_FIELD_PHI = 2, PDO_FIELD_E = 3, PDO_FIELD_CLS = 4 };
enum { PDO_OP_GT = 0, PDO_OP_GE = 1, PDO_OP_LT = 2, PDO_OP_LE = 3, PDO_OP_EQ = 4, PDO_OP_NE = 5, PDO_OP_IN = 6, PDO_OP_NOT_IN = 7 };
typedef struct {
  int32_t field, op, use_abs, n_values; /* n_values: members of `values` (in / not in), at most 8 */
  float value;                          /* scalar comparisons */
  float values[8];
} pdo_condition;

/* in: offsets [n_events+1], cls, src, pt, eta, phi, E of the collection; out_*: same arrays with room for
 * as many objects; out_offsets [n_events+1].  keep (nullable): per input object 1 / 0. */
int pdo_filter_eflow(int64_t n_events, const int64_t *offsets, const int8_t *cls, const int32_t *src, const float *pt,
                     const float *eta, const float *phi, const float *E, const pdo_condition *conds, int32_t n_conds,
                     int32_t combine_any, int64_t *out_offsets, int8_t *out_cls, int32_t *out_src, float *out_pt,
                     float *out_eta, float *out_phi, float *out_E, uint8_t *keep);

/* ---- pile-up merging ("merges minimum-bias interactions with the hard-scatter event
 * using a Delphes-compatible PileUpMerger before applying the detector card"; Listing 8; Table C.9
 * mean_pileup, sigma_z 0.053 m, max_z_spread 0.25 m, smear_hs_vertex; sigma_t / max_t_spread have no
 * effect here because the chain carries no time coordinate, reading A29).  Readings H1-H6 of DESIGN.md
 * section 12.  For hard-scatter event e (RNG event index E = event_base + e, Philox stream 2):
 *   block 0:  n = Poisson(mean_pileup) by inversion of u(r0): the smallest n with sum_{k<=n} p_k > u,
 *             p_0 = exp(-mu), p_k = p_{k-1} mu / k in fp64, n <= n_max = ceil(mu + 10 sqrt(mu) + 20);
 *             dz_hs = truncated normal from r1 if smear_hs_vertex, else 0;
 *   block 1+k (k = 0..n-1):  pool event j_k = ((r0 >> 8) * n_pool) >> 24;  dz_k = truncated normal from r1;
 *   truncated normal (reading H4): the normal of width sigma_z cut at |z| <= max_z_spread, sampled by inversion
 *             of its distribution function (one uniform, no rejection): u = ((r1 >> 8) + 1/2) 2^-24,
 *             sign = -1 if u < 1/2 else +1, v = |2u - 1|, |z| = -sigma_z Phi^-1(Phi(-a) + (1 - v)(1/2 - Phi(-a))),
 *             a = max_z_spread / sigma_z.
 * Output event e = the hard-scatter particles (vz + dz_hs) followed by the particles of pool events j_0, j_1, ...
 * in draw order (vz + dz_k); every other field is copied.  is_pu marks the pile-up particles.
 * out arrays need room for the total; returns PDO_ECAPACITY if out_capacity is too small (out_offsets is then
 * still complete, so out_offsets[n_events] tells the room needed). */
int pdo_pileup_merge(const pdo_events *hs, const pdo_events *pool, double mean_pileup, double sigma_z,
                     double max_z_spread, int smear_hs_vertex, uint64_t seed, int64_t event_base, int64_t out_capacity,
                     int64_t *out_offsets, int32_t *out_pid, int8_t *out_charge, float *out_px, float *out_py,
                     float *out_pz, float *out_E, float *out_vx, float *out_vy, float *out_vz, uint8_t *is_pu,
                     int32_t *n_pileup /* [n_events], may be NULL */);

/* The same with the time coordinate of Table C.9 (sigma_t, max_t_spread; reading H7 of DESIGN.md section 12): the time
 * of an interaction is the truncated normal of width sigma_t cut at max_t_spread from word 2 of its block (hard scatter:
 * block 0, only if smear_hs_vertex); out_vt [capacity], seconds, may be NULL. */
int pdo_pileup_merge_t(const pdo_events *hs, const pdo_events *pool, double mean_pileup, double sigma_z,
                       double max_z_spread, double sigma_t, double max_t_spread, int smear_hs_vertex, uint64_t seed,
                       int64_t event_base, int64_t out_capacity, int64_t *out_offsets, int32_t *out_pid, int8_t *out_charge,
                       float *out_px, float *out_py, float *out_pz, float *out_E, float *out_vx, float *out_vy, float *out_vz,
                       uint8_t *is_pu, int32_t *n_pileup, float *out_vt);

/* ---- track impact parameters ("where supported, track impact parameters"; P:L138
 * Table 2 "d_0, z_0 and their errors for charged particles"; P:L424-426 PFlow.D0 / PFlow.Z0) ----
 * The paper names the outputs and gives no formula; readings I1..I3 of DESIGN.md section 14:
 *   I1 (geometry, the textbook definition): the trajectory is the helix of S1 (reading A3: q > 0 in a +z field turns
 *      clockwise; radius rho = pT / (kappa |q| |B|)) through the production vertex, extended in BOTH directions
 *      (the straight line through the vertex along the momentum when q B = 0).  (x_d, y_d) is its point nearest to
 *      the beam (z) axis in the transverse plane and t^ the transverse direction of flight there:
 *          d0 = x_d t^_y - y_d t^_x      (metres; sign of the z component of the angular momentum -- for a straight
 *                                         line this is the familiar (vx py - vy px) / pT)
 *          z0 = z of the trajectory at that point (reached from the vertex by the shorter arc, forwards or backwards).
 *      A circle centred exactly on the axis has no nearest point: the vertex itself is taken.  A vertex exactly
 *      half a turn away from the nearest point makes z0 two-valued (+- pi rho pz/pT): not covered by parity.
 *   I2 (resolution): sigma_d0 = sqrt(d0_a^2 + (d0_b / pT)^2), sigma_z0 likewise (pT = truth transverse momentum in
 *      GeV; a in metres, b in metres GeV: the usual a (+) b/pT form); the measured values are the true ones plus
 *      sigma times a standard normal, independently for d0 and z0; the "errors" of Table 2 are the two sigmas.
 *   I3 (random numbers): stream 3 of reading A26, object = index of the particle within its event, block 0;
 *      words 0,1 drive d0 (pdo_normal), words 2,3 drive z0.
 * pdo_impact_true is the geometry alone; pdo_track_impact runs over the tracks of a call (trk_offsets [n_events+1],
 * trk_src = index of the truth particle within the call, both as produced by pdo_simulate).  d0_true / z0_true may
 * be NULL.  Parity status: geometry pinned by RK4 integration of the Lorentz force, worked cases and invariance
 * along the helix (tests/test_oracle_impact.py); the resolution model is a reading (the paper's own: unpinned). */
int pdo_impact_true(const pdo_card *c, int q, double px, double py, double pz, double vx, double vy, double vz,
                    double *d0, double *z0);
int pdo_track_impact(const pdo_card *c, const pdo_events *ev, const int64_t *trk_offsets, const int32_t *trk_src,
                     double d0_a, double d0_b, double z0_a, double z0_b, uint64_t seed, int64_t event_base,
                     double *d0_true, double *z0_true, double *d0, double *z0, double *d0_err, double *z0_err);

/* ---- truth-level event features (Table 2: "Event-level quantities: Event number, H_T, E_T^miss values for
 * Truth and PFlow collections"; P:L398 event.truth_ht) ----
 * The same two quantities as pdo_event_features, taken over the truth collection (readings T1, T2 of DESIGN.md
 * section 15):  T1  H_T = sum of pT = sqrt(px^2 + py^2) over the event's particles; E_T^miss vector = -(sum px, sum py),
 * E_T^miss its length (the truth collection carries Cartesian momenta, so no angle is involved).
 * T2  skip_neutrinos != 0 leaves out |pid| in {12, 14, 16} (the usual generator-level missing energy: the recoil of
 * the visible particles); 0 sums the collection as it is.  Sums in fp64 in particle order. */
int pdo_truth_features(const pdo_events *ev, int skip_neutrinos, double *ht, double *met_x, double *met_y, double *met);

const char *pdo_strerror(int code);

/* ---- building blocks exposed so that tests can pin them one by one ---- */
void pdo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* the RNG layout of reading A26: stream 0 = particle stream, 1 = tower stream */
void pdo_rng_block(uint64_t seed, int64_t event, uint32_t object, uint32_t stream, uint32_t out[4]);
double pdo_uniform(uint32_t x);       /* (x >> 8) * 2^-24          in [0,1) */
double pdo_uniform_pos(uint32_t x);   /* ((x >> 8) + 1) * 2^-24    in (0,1] */
double pdo_normal(uint32_t xa, uint32_t xb); /* Box-Muller, cosine branch */
double pdo_lognormal(double mean, double sigma, double z);
/* one particle through O2; returns the status byte. alpha = turning angle (0 for neutrals) */
int pdo_propagate(const pdo_card *card, int charge, double px, double py, double pz, double vx,
                  double vy, double vz, double *x, double *y, double *z, double *alpha,
                  double *eta_pos, double *phi_pos);
/* tower id (or -1) of a position given as (eta_pos or theta_pos per the card's grid, phi_pos) */
int32_t pdo_tower_index(const pdo_card *card, double coord, double phi_pos);
/* reading K6 (card keys hcal_edges / hcal_nphi: a grid of its own for the HCAL; tower ids: the ECAL grid's towers, then the
 * HCAL grid's): the tower of a hit for a deposit in section det (0 ECAL, 1 HCAL); pdo_tower_index is det = 0.  On a card with
 * one grid det does not matter.  pdo_card_hcal_grid: bins of the HCAL grid (0: the card has one grid) and, if the pointers
 * are not NULL, its edges [n+1] and nphi [n]; *base receives the id of its first tower. */
int32_t pdo_tower_index_det(const pdo_card *card, int det, double coord, double phi_pos);
int pdo_card_hcal_grid(const pdo_card *card, double *edges, int32_t *nphi, int32_t *base);
/* efficiency of O3 for true (pt, eta_mom, |cos theta|); *row receives the row index or -1 */
double pdo_efficiency(const pdo_card *card, double pt, double eta_mom, double abs_costheta,
                      int *row);
/* reading J1 (per-species cards): the same for a particle of the given species; pdo_efficiency is the
 * charged-hadron case (identical for cards whose rows name no species) */
enum { PDO_SPECIES_ALL = 0, PDO_SPECIES_ELECTRON = 1, PDO_SPECIES_MUON = 2, PDO_SPECIES_CHHAD = 3 };
double pdo_efficiency_species(const pdo_card *c, double pt, double eta_mom, double abs_costheta, int species, int *row);
/* reading K4 (eta-dependent track resolution rows, card key track_res_eta = aeta_lo aeta_hi a b [species]): the (a, b) of
 * sigma_rel = sqrt(a^2 + (b pT)^2) for a track of the species with true momentum (px, py, pz); returns the row, -1 = the
 * species' / the card's track_res line (reading J2) */
int pdo_track_resolution(const pdo_card *c, int species, double px, double py, double pz, double *a, double *b);
/* reading K5 (weighted EFlow, card key eflow_weighted = 1): factor on the EFlow entries (pT, E) of the tracks of a tower
 * component whose neutral is not emitted; T, V: sum and variance of the tracks' energies, Ec, sigma_c: the component's kept
 * smeared energy and its resolution there */
double pdo_eflow_weight(double T, double V, double Ec, double sigma_c);

#ifdef __cplusplus
}
#endif
#endif /* PD_ORACLE_H */
