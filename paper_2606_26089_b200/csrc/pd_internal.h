// pd_internal.h -- types shared by the host side (card loader, API) and the kernels of libpd.
// Product code: shares nothing with oracle/ (see DESIGN.md "Independence").
#pragma once

#include <cstdint>
#include <string>
#include <vector>

#include "pd.h"

constexpr int PD_MAX_BINS = 1024;      // eta/theta bins of a card's grid
constexpr int PD_MAX_EFF = 31;         // rows of the efficiency table in a card (kernel P keeps the row in 5 bits, 31 = none)
constexpr int PD_MAX_EFF_EDGES = 8;    // distinct pT edges / distinct |eta| edges of the table
constexpr int PD_MAX_EFF_CELLS = (PD_MAX_EFF_EDGES + 1) * (PD_MAX_EFF_EDGES + 1);
constexpr int PD_MAX_TOWERS = (1 << 15) - 1;  // tower ids are packed into 15 bits on chip, 0x7fff = none
constexpr int PD_PSEG = 192;           // particles per segment (one warp of kernel P): a multiple of 32, <= 255
constexpr int PD_PTILE = 8 * PD_PSEG;         // particles per tile of kernel P (pd_particles.cu): a multiple of 32, <= 2048
constexpr int PD_LUT_SHIFT = 19;       // eta-bin lookup: 16 cells per octave of |u|
constexpr int PD_LUT_MIN_EXP = -8;     // |u| < 2^-8 shares one cell per side

// Scalars of a card as the kernels want them (all derived in double at load, stored as fp32).
constexpr int PD_MAX_TRK_ROWS = 8;
struct PdCardScalars {
  float R, L, R2, inv_R;  // calorimeter radius, half length, R^2, 1/R
  float kB, inv_kB;       // kappa * |B|  [GeV / m] and its inverse
  double kB_d;            // same in double (only used for the endcap turning angle)
  float sB;               // sign of B (0 if B == 0)
  int grid_theta;         // 0: bins in eta, 1: bins in theta
  int n_bins, n_towers;
  int words_per_event;    // tower bitmap: ceil(n_towers / 128) * 4 words of 32 tower bits
  // eta-bin lookup table over the float bits of |u| (see pd_card.cpp): cells per side, bias
  // One grid, or (reading K6) two: [0] the ECAL's, [1] the HCAL's (one grid: both entries describe it).  Per grid g: its
  // bins are g_bin_off[g] .. + g_nb[g] of the per-bin tables (tower offsets run on through both grids), its u thresholds
  // tb[g_tb_off[g] .. + g_nb[g]], its lookup cells lut[g_lut_off[g] .. + 2 g_lut_side[g]) holding bins relative to the grid.
  int n_grids, n_tb, lut_cells;
  int g_nb[2], g_bin_off[2], g_tb_off[2], g_lut_off[2], g_lut_side[2], g_lut_base[2];
  float g_tb_first[2], g_tb_last[2];  // the grid's coverage in u: tb[first] <= u < tb[last]
  // efficiency table resolved into a grid at load (reading A8: first matching row wins):
  // cell = (#pT edges with pT > e) * (n_T + 1) + (#T edges with |pz|/pT >= t)
  int n_pt, n_T;
  double pt_edge2_d[PD_MAX_EFF_EDGES];  // e^2 in double; unused entries are DBL_MAX
  float T_edge[PD_MAX_EFF_EDGES];       // sinh |eta| edges (incl. the |cos theta| cut); unused entries +inf
  // one grid per species (0 electron, 1 muon, 2 charged hadron; reading J1 of DESIGN.md section 13)
  float cell_eps[3][PD_MAX_EFF_CELLS];
  signed char cell_row[3][PD_MAX_EFF_CELLS];  // row of the card's table, -1 none
  float row_eps[PD_MAX_EFF + 1];              // efficiency of a row of the card's table
  float trk_a2[3], trk_b[3];  // sigma_rel^2 = a^2 + (b pT)^2, per species (reading J2)
  int trk_per_species;        // 0: the three entries are equal (pass T then skips the pid lookup)
  int eff_per_species;        // 0: no efficiency row names a species (the three grids are equal)
  float ecal2[3], hcal2[3];  // C^2, S^2, N^2 of sigma^2 = C^2 E^2 + S^2 E + N^2
  float thr_ecal, thr_hcal;
  // higher card fidelity (readings K1-K3)
  int res_per_bin;                // K1: the card has eta-dependent resolution rows: C^2, S^2, N^2 per eta bin (PdCardTables::res2)
  float nsig2_ecal, nsig2_hcal;   // K2: n_sigma^2 of the significance cut (0: none)
  int smear_center;               // K3: reported tower position uniform inside the cell (Philox stream 4)
  int eflow_weighted;             // K5: tracks of a component without a neutral rescaled to the weighted mean of track and calorimeter
  // K4: eta-dependent track resolution rows (first match in file order; species 0 = any, 1 e, 2 mu, 3 charged hadron);
  // a row holds sinh(aeta_lo) pT <= |pz| < sinh(aeta_hi) pT, decided in fp64 exactly as the definition does
  int n_trk_rows;
  int trk_row_sp[PD_MAX_TRK_ROWS];
  double trk_row_lo_d[PD_MAX_TRK_ROWS], trk_row_hi_d[PD_MAX_TRK_ROWS];
  float trk_row_a2[PD_MAX_TRK_ROWS], trk_row_b[PD_MAX_TRK_ROWS];
};

// Per-bin tables, contiguous in one device allocation.
struct PdCardTables {
  const float *tb;        // [n_tb] bin thresholds in u = z/r (eta grid) or -z/r (theta grid): n_bins + 1 per grid
  const int *nphi;        // [n_bins]
  const int *offset;      // [n_bins+1] exclusive prefix sum of nphi
  const float *inv_w;     // [n_bins] nphi / (2 pi)
  const float *half;      // [n_bins] 0.5 if nphi odd else 0
  const float *w;         // [n_bins] 2 pi / nphi
  const float *eta_c;     // [n_bins] tower-centre pseudorapidity
  const float *inv_cosh;  // [n_bins] 1 / cosh(eta_c)
  const unsigned short *lut;  // [lut_cells] first candidate bin of a cell (per grid: 2 * g_lut_side cells)
  const float *edge;      // [n_bins][2] the bins' lower and upper edges (eta or theta), fp32
  const float *res2;      // [n_bins][6] ECAL C^2, S^2, N^2, HCAL C^2, S^2, N^2 of the bin's towers (reading K1)
};

constexpr int PD_MAX_CARD_DEVICES = 16;
struct pd_card {
  std::string name;
  // host copy (rounded to fp32 where the kernels use fp32)
  PdCardScalars sc{};
  std::vector<float> edges;  // [n_bins][2] lower and upper edge of every bin (eta or theta), fp32
  std::vector<float> tb, inv_w, half, w, eta_c, inv_cosh;
  std::vector<int> nphi, offset;
  std::vector<unsigned short> lut;
  std::vector<float> res2;   // [n_bins][6]
  float bz = 0.f;
  int n_eff_rows = 0;
  // device copy, created lazily by the first simulate call
  // the tables on the devices that have used the card (pd_card_to_device): slot k holds device dev_id[k]
  mutable void *dev_blob[PD_MAX_CARD_DEVICES] = {};
  mutable int dev_id[PD_MAX_CARD_DEVICES] = {};
  mutable PdCardTables dev_tab[PD_MAX_CARD_DEVICES] = {};
  mutable int n_dev = 0;
};

// Philox4x32-10 round keys of the call's seed: (seed lo + r W0, seed hi + r W1), r = 0..9
struct PdPhiloxKeys {
  uint32_t k0[10], k1[10];
};

// Shared-memory carve-up of kernel T (byte offsets; pd_towers.cu make_layout)
struct PdTLayout {
  uint32_t offset, w, eta_c, inv_cosh, binlut;  // card tables (what pass O needs)
  uint32_t res2, edge;                          // K1 / K3 tables (size 0 when the card does not use them)
  uint32_t off32, ntrk, ntow, nph, nnh;         // per-event arrays [G+1]
  uint32_t misc;                                // scratch words
  uint32_t seg;                                 // track segments of the tile [3][64]
  uint32_t cnt;                                 // pass W warp counts -> prefixes [2][256]
  uint32_t bitmap, gprefix;                     // per event: tower bits, group prefix
  uint32_t l2p, pool;                           // sparse mode
  uint32_t res, Ev, Et, head, stg, ev;          // per particle / per slot
  uint32_t Es;                                  // K5: per particle, sigma_E of an accepted track (size 0 otherwise)
  uint32_t total;
};

// Kernel parameters (passed by value).
struct PdParams {
  PdCardScalars sc;
  PdCardTables tab;
  // inputs
  long long n_events, n_particles;
  const long long *offsets;
  const int *pid;
  const signed char *charge;
  const float *px, *py, *pz, *E, *vx, *vy, *vz;
  unsigned long long seed;
  PdPhiloxKeys rk;
  long long event_base;
  // outputs
  long long *trk_offsets;
  int *trk_src, *trk_pid;
  signed char *trk_charge;
  float *trk_pt, *trk_eta, *trk_phi, *trk_E, *trk_eta_out, *trk_phi_out;
  long long *tow_offsets;
  int *tow_tower;
  float *tow_eta, *tow_phi, *tow_E, *tow_Eem, *tow_Ehad, *tow_ET;
  long long *efl_offsets;
  signed char *efl_cls;
  int *efl_src;
  float *efl_pt, *efl_eta, *efl_phi, *efl_E;
  // debug (all nullable)
  unsigned char *dbg_status;
  float *dbg_eta_pos, *dbg_phi_pos;
  int *dbg_tower;
  unsigned char *dbg_accepted;
  signed char *dbg_eps_row;
  float *dbg_pt_smeared;
  unsigned char *dbg_tw_first;
  float *dbg_tw[6];
  unsigned char *dbg_tw_dec;
  // tiling / workspace
  int events_per_tile;   // G
  int n_tiles;
  int capacity;          // C: particles a tile may hold on chip
  int sparse;            // 1: two-level tower bitmap (large grids, small events), see make_layout
  PdTLayout lay;         // shared-memory carve-up of kernel T
  unsigned long long *chain;  // [n_tiles] look-back words of kernel T: towers | neutrals
  unsigned int *tile_counter;
  int *status_word;
  long long *big_acc;    // [max_ctas][n_towers][5] exact accumulators of the tiles that do not fit on chip (pd_towers.cu big_event)
  // kernel P (pd_particles.cu): flat tiles of PD_PTILE particles
  long long p_base;              // offsets[0]: first particle of the call in the arrays (0 for a public call)
  int n_ptiles;
  int tma_ok;                    // 1: every input array is 16-byte aligned (bulk copies), 0: plain loads
  unsigned long long *chain_t;   // [n_tiles] look-back words of kernel T: tracks
  // accepted tracks parked by kernel P, compacted within every segment of PD_PSEG consecutive particles
  unsigned int *accmask;         // [n_ptiles * PD_PTILE / 32] accepted bits
  unsigned char *park_idx;       // [n_ptiles * PD_PTILE] index of the track's particle within its segment
  int *park_pid;
  signed char *park_q;
  float *park_f[6];              // pt, eta, phi, E, eta_out, phi_out
  // impact parameters from the chain itself (pd_options.impact): kernel P parks d0, z0, d0_err, z0_err of an accepted track
  // beside its record, kernel T moves them to imp_out[.][track]; imp_on = 0: none of this is touched
  // weighted EFlow (reading K5): kernel P parks sigma_E = sigma_rel E_trk of an accepted track; accumulators of the big-tile
  // path: acc_stride 64-bit words per tower (5, or 7 with the two variance sums)
  float *park_sig;
  int acc_stride;
  int imp_on;
  float imp_d0_a, imp_d0_b, imp_z0_a, imp_z0_b;
  float *park_imp[4];
  float *imp_out[4];
  unsigned int *ptile_counter;
  int *tile_ev;                  // [n_ptiles + 1][2] per tile boundary: first event with offset >= it, last with offset <= it
  unsigned short *key;           // [n_ptiles * PD_PTILE] per particle: tower id | HCAL bit << 15, 0xffff = no deposit
};

// pd_card.cpp
int pd_card_parse(const char *name_or_path, pd_card *c);
// pd_api.cu
int pd_card_to_device(const pd_card *c, const PdCardTables **tab);  // tables on the current device (uploaded once)
// pd_towers.cu
struct PdLaunchPlan {
  int threads;       // 512 (two CTAs per SM) or 1024 (one)
  int capacity;      // C
  int events_per_tile;
  int n_tiles;
  int n_ptiles;      // tiles of kernel P
  int max_ctas;      // upper bound of kernel T's grid (sizes big_acc)
  int sparse;        // two-level tower bitmap
  size_t smem_bytes;
  PdTLayout lay;
};
int pd_plan(const pd_card *c, long long n_events, long long n_particles, int tile_events, PdLaunchPlan *plan);  // tile_events: 0 = automatic
int pd_launch_chain(const PdParams &prm, const PdLaunchPlan &plan, bool debug, void *stream);
// pd_particles.cu
int pd_launch_particles(const PdParams &prm, bool debug, int num_sms, int max_smem_optin, void *stream);

// pd_features.cu: event features + lepton isolation (pd_event_features)
struct PdFeatParams {
  long long n_events;
  const long long *offsets;
  const signed char *cls;
  const float *pt, *eta, *phi;
  float dr_max2, fsr2;  // squared cone radii (rounded to fp32 from double)
  float inv_strip;      // 1 / width of the eta strips that pre-select cone candidates (width >= dr_max)
  float inv_phi_cell;   // n_phi / (2 pi): phi cells of width >= dr_max
  int n_phi;            // 1..12
  float *ht, *met_x, *met_y, *met;
  float *iso_charged, *iso_neutral, *iso_photon, *r_iso;
};
int pd_launch_features(const PdFeatParams &prm, void *stream);

// pd_filter.cu: particle filter = predicated, ordered stream compaction of an EFlow collection
constexpr int PD_FILTER_TILE = 2048;  // objects per tile (256 threads x 8)
struct PdFilterParams {
  long long n_events;
  const long long *offsets;
  const signed char *cls;
  const int *src;
  const float *pt, *eta, *phi, *E;
  long long *out_offsets;
  signed char *out_cls;
  int *out_src;
  float *out_pt, *out_eta, *out_phi, *out_E;
  pd_condition conds[PD_MAX_CONDITIONS];
  int n_conds, combine_any;
  unsigned int *tile_counter;     // workspace: next tile
  unsigned long long *chain;      // workspace: look-back word per tile
  unsigned long long *wordrank;   // workspace, per 32 input positions (0..n): survivor bits | rank of the first << 32
  int aligned16;                  // all six input arrays start at a multiple of 16 bytes (bulk copies)
  unsigned cond_fields;           // bit f: field f (PD_FIELD_*: pt, eta, phi, E, cls) is tested by a condition; bit 5 (src) never
};
int pd_launch_filter(const PdFilterParams &prm, void *stream);

// pd_pileup.cu: pile-up merging (pd_pileup_merge)
constexpr int PD_PILEUP_SCAN_TILE = 1024;  // events per scan tile
struct PdPileupParams {
  long long n_hs, n_pool;
  const long long *hs_off, *pool_off;
  const int *hs_pid, *pool_pid;
  const signed char *hs_charge, *pool_charge;
  const float *hs_f[7], *pool_f[7];  // px, py, pz, E, vx, vy, vz
  double mu, p0;                     // mean, exp(-mean)
  int n_max, smear_hs;
  float sigma_z, phi_lo, half_minus_lo;  // Phi(-a), 1/2 - Phi(-a), a = max_z / sigma_z
  float sigma_t, phi_lo_t, half_minus_lo_t;  // the same for the time of an interaction (reading H7)
  float *out_vt;                         // nullable
  PdPhiloxKeys rk;
  long long event_base;
  long long capacity;
  long long *out_off;
  int *out_pid;
  signed char *out_charge;
  float *out_f[7];
  unsigned char *is_pu;
  int *n_pileup;
  unsigned int *tile_counter;  // workspace
  int *status_word;            // workspace + 4 (same place as pd_simulate's: pd_last_status reads it)
  long long *cnt;              // workspace: particles per merged event
  unsigned long long *chain;   // workspace: one self-flagged look-back word per scan tile
};
int pd_launch_pileup(const PdPileupParams &prm, void *stream);

// pd_impact.cu: track impact parameters (pd_track_impact)
struct PdImpactParams {
  long long n_events, n_particles;
  const long long *ev_off, *trk_off;
  const int *trk_src;
  const signed char *charge;
  const float *px, *py, *pz, *vx, *vy, *vz;
  float inv_kB, sB;                 // 1 / (kappa |B|), sign of B (0: no field)
  float d0_a, d0_b, z0_a, z0_b;     // sigma = a (+) b / pT
  PdPhiloxKeys rk;
  long long event_base;
  float *d0, *z0, *d0_err, *z0_err;
};
int pd_launch_impact(const PdImpactParams &prm, void *stream);

// pd_truth.cu: truth-level event features (pd_truth_features)
struct PdTruthParams {
  long long n_events, n_particles;
  const long long *ev_off;
  const int *pid;
  const float *px, *py;
  int skip_neutrinos;
  unsigned long long *acc;  // workspace: [n_events][3] fixed-point sums (H_T, sum px, sum py)
  float *ht, *met_x, *met_y, *met;
};
int pd_launch_truth(const PdTruthParams &prm, void *stream);
