/*
 * pd.h -- C ABI of the B200-native Delphes-style detector-response hot path ("pd").
 *
 * What the library computes: the TorchDelphes chain of the Parnassus paper (arxiv/paper_2606_26089),
 *   "particle propagation through the magnetic field, tracking efficiency, momentum smearing,
 *    calorimeter response, and energy-flow merging, with per-module parameters loaded from the
 *    selected detector card"                                   (section 1, L81 section 2.2)
 * up to "calorimeter tower hits (Towers) and reconstructed photons, neutral hadrons, and charged
 * tracks (EFlowObjects)" (App. D.1), for a batch of variable-length truth events
 * ("no fixed model limit", Table 1).  The paper prints no formula for any step; the
 * formulas are the readings A1..A32 of DESIGN.md (SURVEY.md section 8c.2/8c.3 + BASELINE.json configs).
 *
 * Conventions
 *   - Plain C.  No exception crosses the boundary.  Every entry point returns 0 (PD_OK) or a negative
 *     pd_status; pd_strerror() turns it into text.
 *   - Units: GeV, metres, tesla (reading A1).  Pseudorapidity / azimuth in radians, phi in [-pi, pi].
 *   - `pd_simulate` takes DEVICE pointers (memory of the current CUDA device, owned by the caller,
 *     typically torch tensors) and a CUDA stream handle; it allocates nothing, launches its kernels
 *     on that stream and returns without synchronising.  `pd_simulate_host` takes HOST pointers and
 *     performs the host<->device copies itself (stream-ordered allocations; batches of more than 4M
 *     particles in pipelined chunks so that the copies in both directions overlap the kernels),
 *     returning after the results are in host memory.
 *   - There is no CPU fallback: with no CUDA device both simulate calls fail with PD_ECUDA.
 */
#ifndef PD_H
#define PD_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  PD_OK = 0,
  PD_EINVAL = -1,     /* null pointer, negative size, inconsistent arguments                 */
  PD_ECARD = -2,      /* unknown card name or malformed card file                             */
  PD_ECAPACITY = -3,  /* an output capacity is below the sufficient bound (see pd_simulate)    */
  PD_EWORKSPACE = -4, /* workspace null or smaller than pd_workspace_bytes()                  */
  PD_ECUDA = -5,      /* a CUDA runtime call failed (no device, launch error, ...)            */
  PD_EEVENTSIZE = -6  /* (not raised any more: events of any size are handled; kept for ABI stability) */
} pd_status;

/* status byte of a propagated particle ("PropagatedParticle"): low two bits = face */
enum { PD_DROPPED = 0, PD_BARREL = 1, PD_ENDCAP = 2, PD_FACE_MASK = 3, PD_LOOPER = 4 };
/* object classes (charged hadron, electron, muon, neutral hadron, photon) */
enum { PD_CLS_CHHAD = 0, PD_CLS_ELECTRON = 1, PD_CLS_MUON = 2, PD_CLS_NEUHAD = 3, PD_CLS_PHOTON = 4 };
/* bits of pd_debug.tw_decisions (threshold decisions of steps S6/S7) */
enum { PD_DEC_EEM = 1, PD_DEC_EHAD = 2, PD_DEC_NEM = 4, PD_DEC_NHAD = 8 };

typedef struct pd_card pd_card; /* opaque, owned by the library; immutable after pd_load_card */

typedef struct {
  int32_t n_towers, n_eta_bins, grid_coord; /* grid_coord: 0 = eta edges, 1 = theta edges */
  float bz, radius, half_length;            /* tesla, metres, metres                      */
  int32_t n_eff_rows;
} pd_card_info_t;

/* Input: truth events in CSR form (BASELINE.json north_star: "events CSR: offsets, pid, charge, px,
 * py, pz, E, vx, vy, vz").  Particle i of event e has index offsets[e] + i.  Non-finite values are
 * undefined behaviour (reading A31). */
typedef struct {
  int64_t n_events;       /* >= 0                                                        */
  int64_t n_particles;    /* == offsets[n_events]; < 2^30                                */
  const int64_t *offsets; /* [n_events+1], offsets[0] == 0, non-decreasing               */
  const int32_t *pid;     /* PDG id                                                      */
  const int8_t *charge;   /* units of e; authoritative for charged/neutral               */
  const float *px, *py, *pz, *E; /* GeV                                                  */
  const float *vx, *vy, *vz;     /* production vertex, metres                            */
} pd_events;

/* Output collections (PAPER.md L329-342 Table A.6: Track, Tower, PFlow), CSR over the call's events.
 * offsets[e] .. offsets[e+1] delimit event e; offsets[n_events] is the total.
 * Order (reading A25): tracks in particle order; towers by ascending tower id; eflow = the event's
 * tracks (particle order), then photons (ascending tower id), then neutral hadrons (ascending id). */
typedef struct {
  int64_t capacity;  /* elements available in every array below; must be >= n_particles   */
  int64_t *offsets;  /* [n_events+1]                                                      */
  int32_t *src;      /* index of the truth particle within the call                       */
  int32_t *pid;
  int8_t *charge;
  float *pt, *eta, *phi, *E; /* smeared pT; direction of the vertex momentum; E = pT cosh(eta) */
  float *eta_out, *phi_out;  /* position on the calorimeter face                          */
} pd_tracks;

typedef struct {
  int64_t capacity; /* >= n_particles */
  int64_t *offsets;
  int32_t *tower;   /* tower id in the card's grid */
  float *eta, *phi; /* tower centre */
  float *E, *Eem, *Ehad, *ET;
} pd_towers;

typedef struct {
  int64_t capacity; /* >= 2 * n_particles */
  int64_t *offsets;
  int8_t *cls;      /* PD_CLS_* */
  int32_t *src;     /* tracks: truth particle index; neutrals: tower id */
  float *pt, *eta, *phi, *E;
} pd_eflow;

/* Optional intermediate products (the paper's `debug` option, PAPER.md L589 / L669).  All arrays have
 * n_particles elements; any pointer may be NULL.  The per-tower fields describe every tower that
 * received a deposit (emitted or not) and are stored at the index of the FIRST particle (in particle
 * order) that deposited into that (event, tower); tw_first marks those indices (the tw_* entries of all other indices
 * are not written). */
typedef struct {
  uint8_t *status;   /* PD_DROPPED / PD_BARREL / PD_ENDCAP | PD_LOOPER                     */
  float *eta_pos, *phi_pos; /* hit position on the calorimeter surface (NaN if dropped)    */
  int32_t *tower;    /* geometric tower id of the hit, -1 if none                          */
  uint8_t *accepted; /* 1 if the particle became a track                                   */
  int8_t *eps_row;   /* row of the efficiency table used, -1 none                          */
  float *pt_smeared; /* 0 if not an accepted track                                         */
  uint8_t *tw_first;
  float *tw_Eem_true, *tw_Ehad_true, *tw_Tem, *tw_Thad, *tw_Eem_smeared, *tw_Ehad_smeared;
  uint8_t *tw_decisions; /* PD_DEC_* bits: 1 = "above threshold"                           */
} pd_debug;

/* Load a detector card: a built-in name ("cms_like" | "atlas_like" | "aleph_like", the parameter
 * sets of BASELINE.json configs[0], [3], [4]) or the path of a card text file ("key = values" lines,
 * '#' comments; keys name, bz, radius, half_length, kappa, grid (eta|theta), edges, nphi, eff,
 * abs_costheta_max, track_res, ecal_res, hcal_res, ecal_thr, hcal_thr; an `eff` row may carry a sixth
 * number and a `track_res` line a third one -- the species it applies to: 1 electrons, 2 muons, 3 charged
 * hadrons, 0 / absent every charged particle -- PAPER.md L653-655).  Pure host work: no CUDA
 * call is made until the card is first used by a simulate call.  Every card number is rounded to
 * fp32 at load (reading A28).  *out is owned by the library until pd_free_card. */
int pd_load_card(const char *name_or_path, pd_card **out);
void pd_free_card(pd_card *card);
int pd_card_info(const pd_card *card, pd_card_info_t *out);

/* Bytes of DEVICE workspace pd_simulate needs for a call of this size: look-back chains, tile counters, status word,
 * and what kernel P leaves for kernel T -- per particle a 16-bit tower key, an accepted bit and room for a parked track
 * record (~32 B per particle in all) -- plus the accumulators of the big-tile path (40 B x towers x resident CTAs).
 * Negative pd_status on invalid arguments. */
int64_t pd_workspace_bytes(const pd_card *card, int64_t n_events, int64_t n_particles);

/* One pass of the whole chain S0..S8 over a batch of events.
 *   events, tracks, towers, eflow, debug (nullable): structs in HOST memory whose pointer members
 *     are DEVICE pointers.  Outputs are fully overwritten up to their totals.
 *   seed, event_base: the Philox4x32-10 key is (seed lo, seed hi); the counter is (object, event lo,
 *     event hi, stream << 16) with event = event_base + index in the call (readings A26, A27), so a
 *     batch split over several calls / GPUs reproduces the single-call result bit for bit.
 *   workspace: >= pd_workspace_bytes() bytes, 16-byte aligned, device memory; contents are scratch.
 *   cuda_stream: a cudaStream_t (NULL = default stream).  Asynchronous: results are valid after the
 *     caller synchronises the stream; pd_last_status() then reports device-side conditions.
 * Errors are detected synchronously (PD_EINVAL, PD_ECAPACITY, PD_EWORKSPACE, PD_ECUDA); there is no
 * device-side overflow path for the outputs because the capacities above are sufficient bounds, and no limit on the
 * number of particles of an event.  Three kernel launches (event windows of the particle tiles; kernel P: particles ->
 * tower keys + parked tracks; kernel T: towers, EFlow, ordered collections) and one memset. */
int pd_simulate(const pd_card *card, const pd_events *events, uint64_t seed, int64_t event_base,
                pd_tracks *tracks, pd_towers *towers, pd_eflow *eflow, pd_debug *debug,
                void *workspace, int64_t workspace_bytes, void *cuda_stream);

/* Reads back (synchronising the stream) the device-side status word a call left in its workspace: PD_OK for
 * pd_simulate (there is no event-size limit: a tile of events that does not fit on chip is processed event by event
 * through exact accumulators in the workspace -- "no fixed model limit"), PD_ECAPACITY for a
 * pd_pileup_merge whose output did not fit. */
int pd_last_status(const void *workspace, void *cuda_stream);

/* ---- Event features and lepton isolation (section 2.4 Eq. 1; L141 Table 2) ----
 * From an EFlow ("PFlow") collection, per event (readings F1, F2 of DESIGN.md section 10):
 *   ht = sum_i pT_i;  (met_x, met_y) = -(sum_i pT_i cos phi_i, sum_i pT_i sin phi_i);  met = its length;
 * and for every object of class PD_CLS_ELECTRON or PD_CLS_MUON, Eq. 1:
 *   r_iso = (iso_charged + iso_neutral + iso_photon) / pT_lepton, the three terms being the pT sums of the event's
 *   other objects of classes {0,1,2}, {3}, {4} with dR = sqrt(d_eta^2 + d_phi^2) < dr_max around the lepton
 *   (d_phi wrapped; the lepton itself excluded; photons with dR < fsr_dr -- final-state-radiation candidates,
 *   reading F4 -- left out of the photon term; fsr_dr = 0 keeps them all).  Objects of other classes get 0.
 * All pointers are DEVICE pointers owned by the caller; per-event arrays have n_events elements, per-object arrays
 * as many as the collection holds (eflow->offsets[n_events], at most eflow->capacity).  Sums are exact
 * fixed-point sums (units of 2^-32 GeV), hence independent of order and bitwise reproducible. */
typedef struct {
  float *ht, *met_x, *met_y, *met;                       /* [n_events]  */
  float *iso_charged, *iso_neutral, *iso_photon, *r_iso; /* [n_objects] */
} pd_features;

/* Asynchronous on cuda_stream; allocates nothing; needs no workspace (events are independent, no output is
 * compacted).  Only eflow->offsets, cls, pt, eta, phi are read.  Errors: PD_EINVAL (null pointers, negative
 * n_events, dr_max or fsr_dr negative or not finite), PD_ECUDA. */
int pd_event_features(const pd_eflow *eflow, int64_t n_events, float dr_max, float fsr_dr, pd_features *out,
                      void *cuda_stream);

/* ---- Particle filter (section 2.4; Table C.13) ----
 * "Particle filtering drops particles from a target collection ... according to declarative per-field conditions
 * (e.g. pT, eta, or PDG-ID cuts), combined with logical all (AND) or any (OR) semantics."  Here: the EFlow
 * ("pflow", the paper's default) collection, as an ordered stream compaction into a second collection.
 * A condition compares an attribute of the object (its magnitude if use_abs) with `value` (ops >, >=, <, <=,
 * ==, !=) or tests it for membership in values[0..n_values) (ops in, not in).  Attributes: pt, eta, phi, E
 * (fp32, compared as they are, hence exactly) and the class id (compared as a number).  An object is kept iff
 * all (combine_any = 0) or any (combine_any != 0) of the conditions hold; no condition keeps everything.
 * Survivors keep their order.  The paper's update_event_features is a pd_event_features call on the output. */
enum { PD_FIELD_PT = 0, PD_FIELD_ETA = 1, PD_FIELD_PHI = 2, PD_FIELD_E = 3, PD_FIELD_CLS = 4 };
enum { PD_OP_GT = 0, PD_OP_GE = 1, PD_OP_LT = 2, PD_OP_LE = 3, PD_OP_EQ = 4, PD_OP_NE = 5, PD_OP_IN = 6, PD_OP_NOT_IN = 7 };
enum { PD_MAX_CONDITIONS = 16, PD_MAX_SET_VALUES = 8 };
typedef struct {
  int32_t field, op, use_abs, n_values;
  float value;
  float values[8];
} pd_condition;

/* Bytes of DEVICE workspace pd_filter_eflow needs for an input collection of this capacity. */
int64_t pd_filter_workspace_bytes(int64_t capacity);

/* in, out: structs in HOST memory whose pointer members are DEVICE pointers (in->offsets [n_events+1]; the number
 * of objects is read on the device).  out->capacity >= in->capacity; out->offsets [n_events+1]; in and out must
 * not overlap.  conds: HOST array.  Asynchronous on cuda_stream, two kernel launches, allocates nothing.
 * The input arrays may start anywhere; when all six start at a multiple of 16 bytes the tiles are staged by bulk copies
 * (the fast path).  A NaN field fails >, >=, <, <=, ==, "in" and passes !=, "not in".
 * Errors: PD_EINVAL (null pointers, bad field / op / counts), PD_ECAPACITY, PD_EWORKSPACE, PD_ECUDA. */
int pd_filter_eflow(const pd_eflow *in, int64_t n_events, const pd_condition *conds, int32_t n_conds, int32_t combine_any,
                    pd_eflow *out, void *workspace, int64_t workspace_bytes, void *cuda_stream);

/* ---- Pile-up merging (Listing 8; Table C.9) ----
 * "When configured with a pile-up block, the parametric path first merges minimum-bias interactions with the
 * hard-scatter event using a Delphes-compatible PileUpMerger before applying the detector card."  Readings H1-H6
 * of DESIGN.md section 12.  For hard-scatter event e (RNG event index event_base + e, Philox stream 2):
 *   block 0: n = Poisson(mean_pileup) by inversion of the 24-bit uniform of word 0 (fp64 recurrence, the same
 *            operations in the same order as the oracle, so n is bit-exact); the hard-scatter vertex shift from
 *            word 1 if smear_hs_vertex;
 *   block 1+k, k < n: pool event ((r0 >> 8) * n_pool) >> 24; its vertex shift from word 1;
 *   vertex shift: normal of width sigma_z truncated to |z| <= max_z_spread, sampled by inversion of its
 *            distribution function (one uniform, no rejection).
 * Output event e = the hard-scatter particles (vz shifted) followed by the particles of the n picked pool
 * events in draw order (vz shifted); every other field is copied.  sigma_t / max_t_spread of Table C.9: every
 * interaction also gets a time, the same truncated normal from word 2 of its block (the hard scatter's from block 0 if
 * smear_hs_vertex, else 0), written per particle to `vt` (reading H7); the detector chain itself carries no time
 * coordinate (reading A29).  The output is a pd_events-shaped CSR batch that pd_simulate takes as it is. */
typedef struct {
  float mean_pileup;  /* 0 <= mean <= 500 */
  float sigma_z;      /* metres, >= 0 (Table C.9 default 0.053) */
  float max_z_spread; /* metres, >= 0 (default 0.25) */
  int32_t smear_hs_vertex;
  float sigma_t;      /* seconds, >= 0 (Table C.9 default 160e-12); 0: every interaction at t = 0 */
  float max_t_spread; /* seconds, >= 0 (default 800e-12) */
} pd_pileup_config;

typedef struct {
  int64_t capacity;  /* particles the arrays below can hold */
  int64_t *offsets;  /* [n_events+1] */
  int32_t *pid;
  int8_t *charge;
  float *px, *py, *pz, *E, *vx, *vy, *vz;
  uint8_t *is_pu;    /* 1 for pile-up particles */
  int32_t *n_pileup; /* [n_events] interactions merged into each event */
  float *vt;         /* time of the particle's interaction, seconds (reading H7); may be NULL */
} pd_merged_events;

/* Bytes of DEVICE workspace pd_pileup_merge needs (status word, per-event counts, scan words). */
int64_t pd_pileup_workspace_bytes(int64_t n_events);

/* hs, pool, out: structs in HOST memory whose pointer members are DEVICE pointers; pool->n_events >= 1.
 * Asynchronous on cuda_stream, three kernel launches, allocates nothing.  The merged size is only known on
 * the device: out->offsets is always complete, and if out->offsets[n_events] exceeds out->capacity nothing else
 * is written and pd_last_status(workspace) reports PD_ECAPACITY (re-run with that much room).
 * Errors: PD_EINVAL, PD_EWORKSPACE, PD_ECUDA. */
int pd_pileup_merge(const pd_events *hs, const pd_events *pool, const pd_pileup_config *cfg, uint64_t seed,
                    int64_t event_base, pd_merged_events *out, void *workspace, int64_t workspace_bytes,
                    void *cuda_stream);

/* ---- Track impact parameters ("where supported, track impact parameters"; L138 Table 2 "d_0, z_0
 * and their errors for charged particles"; L424-426 PFlow.D0 / PFlow.Z0) ----
 * The paper names the outputs and prints no formula; readings I1-I3 of DESIGN.md section 14:
 *   geometry: the trajectory is the helix of step S1 through the production vertex, extended in both directions
 *     (a straight line when q B = 0); (x_d, y_d) is its point nearest to the beam (z) axis and t^ the transverse
 *     direction of flight there: d0 = x_d t^_y - y_d t^_x, z0 = z of the trajectory at that point (metres; the
 *     shorter arc from the vertex).  For a straight line d0 = (vx py - vy px) / pT.
 *   resolution: sigma = sqrt(a^2 + (b / pT)^2) (pT = truth pT in GeV; a metres, b metres GeV) for d0 and for z0;
 *     measured = true + sigma * standard normal, independent for the two; the sigmas are the reported errors.
 *   random numbers: Philox stream 3, object = index of the particle within its event, words 0,1 -> d0, 2,3 -> z0
 *     (same key and event numbering as pd_simulate, so splitting a batch does not change a value).
 * One value per track of `tracks` (the collection a pd_simulate call wrote for `events` on the same stream or
 * after synchronisation): only tracks->offsets and tracks->src are read.  a = b = 0 gives the true values. */
typedef struct pd_impact_config_s {
  float d0_a, d0_b; /* metres, metres GeV; >= 0 */
  float z0_a, z0_b;
} pd_impact_config;

typedef struct pd_impact_s {
  float *d0, *z0, *d0_err, *z0_err; /* DEVICE arrays of at least tracks->capacity (>= n_particles) elements */
} pd_impact;

/* card, events, tracks, out: structs in HOST memory whose pointer members are DEVICE pointers.  Asynchronous on
 * cuda_stream, one kernel launch, no workspace, allocates nothing.  Errors: PD_EINVAL (null pointers, negative
 * sizes or resolutions), PD_ECUDA. */
int pd_track_impact(const pd_card *card, const pd_events *events, const pd_tracks *tracks,
                    const pd_impact_config *cfg, uint64_t seed, int64_t event_base, pd_impact *out,
                    void *cuda_stream);

/* ---- Truth-level event features (Table 2 "Event-level quantities: ... H_T, E_T^miss values for Truth
 * and PFlow collections"; L398 event.truth_ht; readings T1, T2 of DESIGN.md section 15) ----
 * Per event of the truth collection:  ht = sum_i sqrt(px_i^2 + py_i^2);  (met_x, met_y) = -(sum_i px_i, sum_i py_i);
 * met = its length.  skip_neutrinos != 0 leaves out |pid| in {12, 14, 16} (the generator-level missing energy: the
 * recoil of the visible particles); 0 sums the collection as it is.  Exact fixed-point sums (units of 2^-32 GeV):
 * independent of order, bitwise reproducible.  Writes out->ht, met_x, met_y, met ([n_events], DEVICE pointers); the
 * isolation members of pd_features are not touched and may be NULL.  Only events->offsets, pid, px, py are read.
 * workspace: >= pd_truth_workspace_bytes(n_events) bytes of DEVICE memory, 8-byte aligned, scratch.
 * Asynchronous on cuda_stream, two kernel launches, allocates nothing.  Errors: PD_EINVAL, PD_EWORKSPACE, PD_ECUDA. */
int64_t pd_truth_workspace_bytes(int64_t n_events);
int pd_truth_features(const pd_events *events, int32_t skip_neutrinos, pd_features *out, void *workspace,
                      int64_t workspace_bytes, void *cuda_stream);

/* ---- The same, for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): NO workspace argument.  The scratch (the [n_events][3] 64-bit accumulators of
 * pd_truth_features) lives in a fixed array inside the library, 24 * PD_TRUTH_STATIC_MAX_EVENTS bytes = 6 MiB of device
 * memory that every GPU which loads the library holds until the process exits.  Inputs, outputs, results and launches
 * are those of pd_truth_features (bitwise: the sums are exact).  The call makes no cudaMalloc / cudaFree and calls no
 * allocating library routine; the first call on a device looks the array's device address up (cudaGetSymbolAddress, once
 * per device, with that device current) -- a call with events->n_events == 0 does just that and returns PD_OK, which is
 * the way to do the set-up ahead of a capture.
 * Limit: events->n_events <= PD_TRUTH_STATIC_MAX_EVENTS, else PD_EWORKSPACE ("workspace missing or too small": the
 * built-in scratch is; use pd_truth_features with a workspace of your own, or split the batch).
 * The array is SHARED by every call on the device and keeps the last call's contents: each call clears the part it uses
 * on its stream before summing, so calls ordered on one stream are independent, but calls that overlap on the GPU
 * (different streams, different host threads) race on it -- serialise them, or use pd_truth_features.
 * Does not update pd_last_launch_count().  Errors: PD_EINVAL, PD_EWORKSPACE, PD_ECUDA. */
#define PD_TRUTH_STATIC_MAX_EVENTS 262144
int pd_truth_features_static(const pd_events *events, int32_t skip_neutrinos, pd_features *out, void *cuda_stream);

/* Number of kernels the last pd_simulate / pd_simulate_host call on this thread launched. */
int pd_last_launch_count(void);

/* ---- Options, and the set-up that can be done ahead of the first call ----
 * The library keeps no state between calls: what used to be a per-thread setting (the events per tile) is an argument.
 * pd_options: plain data, all zero = the defaults; a NULL pointer means the same.
 *   tile_events: tuning / testing only.  Events per on-chip tile of kernel T: 0 = chosen from the average event size with
 *     head-room for Poisson-like fluctuations; g >= 1 = at most g (<= 256; 1 also selects the one-CTA-per-SM variant).
 *     Results never depend on it, and no setting is ever needed for correctness: tiles that exceed the on-chip capacity
 *     take the (slower) path through the workspace by themselves.  The workspace size depends on it: size the workspace
 *     with pd_workspace_bytes_ex and the same options.
 * pd_workspace_bytes_ex / pd_simulate_ex: pd_workspace_bytes / pd_simulate with options (those two = options NULL). */
typedef struct pd_options {
  int32_t tile_events;
  int32_t reserved[7]; /* must be 0 */
  /* impact parameters of the tracks from the chain itself (see pd_track_impact below for the definition): both NULL = off;
   * both set = kernel P computes d0, z0 and their errors for every track it accepts (the particle is on chip there) and
   * kernel T writes them beside the Track collection, element k for track k: the same values as a pd_track_impact call
   * with this config, seed and event_base after the step, bit for bit, without its gather over the particle arrays.
   * impact->d0, z0, d0_err, z0_err: DEVICE arrays of at least tracks->capacity elements.  The workspace grows by 16 bytes
   * per particle slot (pd_workspace_bytes_ex with the same options). */
  const struct pd_impact_config_s *impact_config;
  struct pd_impact_s *impact;
} pd_options;
int64_t pd_workspace_bytes_ex(const pd_card *card, int64_t n_events, int64_t n_particles, const pd_options *options);
int pd_simulate_ex(const pd_card *card, const pd_events *events, uint64_t seed, int64_t event_base,
                   pd_tracks *tracks, pd_towers *towers, pd_eflow *eflow, pd_debug *debug,
                   void *workspace, int64_t workspace_bytes, const pd_options *options, void *cuda_stream);

/* Copies the card's per-bin tables (a few KB) to the CURRENT device, if they are not there yet: one cudaMalloc and one
 * synchronous copy per (card, device), kept until pd_free_card.  pd_simulate does this by itself on its first call with a
 * card on a device; after pd_card_upload, pd_simulate / pd_simulate_ex allocate nothing and can run where allocation is
 * not allowed.  A card can be resident on up to 16 devices at once.  Errors: PD_EINVAL, PD_ECUDA. */
int pd_card_upload(const pd_card *card);

/* Same computation with HOST pointers everywhere (inputs and outputs in host memory, pinned or
 * pageable).  Copies inputs to the device, runs pd_simulate, copies the three collections back and
 * synchronises.  Output capacities as for pd_simulate; totals are offsets[n_events].  Large batches (>= 4M particles)
 * go through in chunks of consecutive events with the copies of one chunk overlapping the kernel of the next (same
 * results, bit for bit).  Optional layout hint: if the 4-byte arrays of a collection (events: pid, px..vz; tracks: src,
 * pid, pt..phi_out; towers: tower, eta..ET; eflow: src, pt..E; in this order) are equally spaced rows of ONE pinned
 * host allocation, a chunk of all of them moves with one strided copy instead of one copy per array. */
int pd_simulate_host(const pd_card *card, const pd_events *events, uint64_t seed, int64_t event_base,
                     pd_tracks *tracks, pd_towers *towers, pd_eflow *eflow, void *cuda_stream);

const char *pd_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* PD_H */
