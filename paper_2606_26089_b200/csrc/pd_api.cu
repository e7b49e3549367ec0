// pd_api.cu -- the C ABI of libpd (include/pd.h): argument checking, card upload, workspace layout,
// kernel launch, and the host-pointer convenience entry point.  No torch types, no CPU fallback.
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdlib>
#include <vector>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "pd_internal.h"

namespace {

thread_local int t_launches = 0;
thread_local char t_cuda_msg[256] = "";
std::mutex g_card_mutex;

constexpr size_t kWsHeader = 16;  // tile counter of kernel T (u32), status word (i32), tile counter of kernel P (u32), padding

int cuda_fail(cudaError_t e, const char *what) {
  std::snprintf(t_cuda_msg, sizeof(t_cuda_msg), "CUDA error in %s: %s", what, cudaGetErrorString(e));
  return PD_ECUDA;
}

#define PD_CUDA(call)                                   \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
  } while (0)

}  // namespace

// header + the two look-back chains of kernel T, rounded up so that what follows is 256-byte aligned
static size_t ws_chain_bytes(const PdLaunchPlan &plan) {
  const size_t b = kWsHeader + 2 * sizeof(unsigned long long) * (size_t)(plan.n_tiles > 0 ? plan.n_tiles : 1);
  return (b + 255) & ~size_t(255);
}
// What kernel P leaves for kernel T, per particle slot (n_ptiles * PD_PTILE slots): the 16-bit key, the accepted bit,
// and the parked track records (segment index 1 B, charge 1 B, pid 4 B, six floats).  Each array 256-byte aligned.
struct WsLayout {
  size_t tile_ev, key, accmask, idx, q, pid, f[6], imp[4], sig, big_acc, total;
};
static WsLayout ws_layout(const PdLaunchPlan &plan, int n_towers, bool impact = false, bool weighted = false) {
  const size_t slots = (size_t)PD_PTILE * (size_t)(plan.n_ptiles > 0 ? plan.n_ptiles : 1);
  WsLayout l;
  size_t o = ws_chain_bytes(plan);
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = (o + bytes + 255) & ~size_t(255);
    return at;
  };
  l.tile_ev = take(8 * ((size_t)plan.n_ptiles + 1));
  l.key = take(2 * slots);
  l.accmask = take(slots / 8);
  l.idx = take(slots);
  l.q = take(slots);
  l.pid = take(4 * slots);
  for (int k = 0; k < 6; ++k) l.f[k] = take(4 * slots);
  for (int k = 0; k < 4; ++k) l.imp[k] = take(impact ? 4 * slots : 0);  // pd_options.impact
  l.sig = take(weighted ? 4 * slots : 0);                                // reading K5: sigma_E of the parked tracks
  l.big_acc = take(8 * (weighted ? 7 : 5) * (size_t)n_towers * (size_t)plan.max_ctas);  // tiles that do not fit on chip (any event size)
  l.total = o;
  return l;
}

extern "C" {

const char *pd_strerror(int code) {
  switch (code) {
    case PD_OK: return "ok";
    case PD_EINVAL: return "invalid argument";
    case PD_ECARD: return "unknown card name or malformed card file";
    case PD_ECAPACITY: return "output capacity below the sufficient bound";
    case PD_EWORKSPACE: return "workspace missing or too small";
    case PD_ECUDA: return t_cuda_msg[0] ? t_cuda_msg : "CUDA runtime error";
    case PD_EEVENTSIZE: return "a tile of events exceeded the on-chip capacity";
    default: return "unknown error";
  }
}

int pd_load_card(const char *name_or_path, pd_card **out) {
  if (!name_or_path || !out) return PD_EINVAL;
  pd_card *c = new (std::nothrow) pd_card();
  if (!c) return PD_EINVAL;
  const int rc = pd_card_parse(name_or_path, c);
  if (rc != PD_OK) {
    delete c;
    return rc;
  }
  *out = c;
  return PD_OK;
}

void pd_free_card(pd_card *card) {
  if (!card) return;
  for (int k = 0; k < card->n_dev; ++k)
    if (card->dev_blob[k]) cudaFree(card->dev_blob[k]);
  delete card;
}

int pd_card_info(const pd_card *card, pd_card_info_t *out) {
  if (!card || !out) return PD_EINVAL;
  out->n_towers = card->sc.n_towers;
  out->n_eta_bins = card->sc.g_nb[0];  // of the (ECAL) grid; a card with a second grid for the HCAL has more bins in all
  out->grid_coord = card->sc.grid_theta;
  out->bz = card->bz;
  out->radius = card->sc.R;
  out->half_length = card->sc.L;
  out->n_eff_rows = card->n_eff_rows;
  return PD_OK;
}

static int tile_events_of(const pd_options *opt) { return opt ? opt->tile_events : 0; }
static bool impact_of(const pd_options *opt) { return opt && opt->impact_config && opt->impact; }
static bool options_ok(const pd_options *opt) {
  if (!opt) return true;
  if (opt->tile_events < 0) return false;
  for (int k = 0; k < 7; ++k)
    if (opt->reserved[k] != 0) return false;
  if ((opt->impact_config != nullptr) != (opt->impact != nullptr)) return false;  // both or neither
  if (opt->impact_config) {
    const pd_impact_config *c = opt->impact_config;
    for (float v : {c->d0_a, c->d0_b, c->z0_a, c->z0_b})
      if (!(v >= 0.f) || !std::isfinite(v)) return false;
    const pd_impact *o = opt->impact;
    if (!o->d0 || !o->z0 || !o->d0_err || !o->z0_err) return false;
  }
  return true;
}

int64_t pd_workspace_bytes_ex(const pd_card *card, int64_t n_events, int64_t n_particles, const pd_options *opt) {
  if (!card || n_events < 0 || n_particles < 0 || !options_ok(opt)) return PD_EINVAL;
  PdLaunchPlan plan;
  pd_plan(card, n_events, n_particles, tile_events_of(opt), &plan);
  return (int64_t)ws_layout(plan, card->sc.n_towers, impact_of(opt), card->sc.eflow_weighted != 0).total;
}
int64_t pd_workspace_bytes(const pd_card *card, int64_t n_events, int64_t n_particles) {
  return pd_workspace_bytes_ex(card, n_events, n_particles, nullptr);
}

int pd_card_upload(const pd_card *card) {
  if (!card) return PD_EINVAL;
  const PdCardTables *tab = nullptr;
  return pd_card_to_device(card, &tab);
}

int pd_last_launch_count(void) { return t_launches; }

// pile-up workspace: [tile counter, status word, pad] 16 B | scan words, one per 1,024 events | sizes, 8 B per event
static size_t pileup_chain_bytes(int64_t n_events) {
  const size_t tiles = (size_t)((n_events + PD_PILEUP_SCAN_TILE - 1) / PD_PILEUP_SCAN_TILE) + 1;
  return (16 + 8 * tiles + 255) & ~size_t(255);
}

int64_t pd_pileup_workspace_bytes(int64_t n_events) {
  if (n_events < 0) return PD_EINVAL;
  return (int64_t)(pileup_chain_bytes(n_events) + 8 * (size_t)(n_events > 0 ? n_events : 1));
}

int pd_pileup_merge(const pd_events *hs, const pd_events *pool, const pd_pileup_config *cfg, uint64_t seed,
                    int64_t event_base, pd_merged_events *out, void *workspace, int64_t workspace_bytes,
                    void *cuda_stream) {
  t_launches = 0;
  if (!hs || !pool || !cfg || !out || hs->n_events < 0 || pool->n_events < 1 || !hs->offsets || !pool->offsets) return PD_EINVAL;
  if (!(cfg->mean_pileup >= 0.f) || cfg->mean_pileup > 500.f || !(cfg->sigma_z >= 0.f) || !(cfg->max_z_spread >= 0.f)) return PD_EINVAL;
  if (!std::isfinite(cfg->sigma_z) || !std::isfinite(cfg->max_z_spread)) return PD_EINVAL;
  if (!(cfg->sigma_t >= 0.f) || !(cfg->max_t_spread >= 0.f) || !std::isfinite(cfg->sigma_t) || !std::isfinite(cfg->max_t_spread)) return PD_EINVAL;
  if (!out->offsets || out->capacity < 0) return PD_EINVAL;
  if (hs->n_events > 0 && !out->n_pileup) return PD_EINVAL;
  if (out->capacity > 0 && (!out->pid || !out->charge || !out->px || !out->py || !out->pz || !out->E || !out->vx || !out->vy ||
                            !out->vz || !out->is_pu)) return PD_EINVAL;
  if (hs->n_particles > 0 && (!hs->pid || !hs->charge || !hs->px || !hs->py || !hs->pz || !hs->E || !hs->vx || !hs->vy || !hs->vz)) return PD_EINVAL;
  if (pool->n_particles > 0 && (!pool->pid || !pool->charge || !pool->px || !pool->py || !pool->pz || !pool->E || !pool->vx || !pool->vy || !pool->vz)) return PD_EINVAL;
  const int64_t need = pd_pileup_workspace_bytes(hs->n_events);
  if (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 15u)) return PD_EWORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t chain_bytes = pileup_chain_bytes(hs->n_events);
  PD_CUDA(cudaMemsetAsync(workspace, 0, chain_bytes, st));
  if (hs->n_events == 0) {
    PD_CUDA(cudaMemsetAsync(out->offsets, 0, sizeof(int64_t), st));
    return PD_OK;
  }
  PdPileupParams p;
  std::memset(&p, 0, sizeof(p));
  p.n_hs = hs->n_events, p.n_pool = pool->n_events;
  p.hs_off = (const long long *)hs->offsets, p.pool_off = (const long long *)pool->offsets;
  p.hs_pid = hs->pid, p.pool_pid = pool->pid, p.hs_charge = hs->charge, p.pool_charge = pool->charge;
  const float *hf[7] = {hs->px, hs->py, hs->pz, hs->E, hs->vx, hs->vy, hs->vz};
  const float *pf[7] = {pool->px, pool->py, pool->pz, pool->E, pool->vx, pool->vy, pool->vz};
  float *of[7] = {out->px, out->py, out->pz, out->E, out->vx, out->vy, out->vz};
  for (int f = 0; f < 7; ++f) p.hs_f[f] = hf[f], p.pool_f[f] = pf[f], p.out_f[f] = of[f];
  // card-like constants in double on the host, exactly as the definition writes them (readings H3, H4)
  const double mu = (double)cfg->mean_pileup, sz = (double)cfg->sigma_z, zmax = (double)cfg->max_z_spread;
  p.mu = mu, p.p0 = std::exp(-mu);
  p.n_max = (int)std::ceil(mu + 10.0 * std::sqrt(mu) + 20.0);
  p.smear_hs = cfg->smear_hs_vertex ? 1 : 0;
  p.sigma_z = cfg->sigma_z;
  const double lo = sz > 0.0 ? 0.5 * std::erfc((zmax / sz) / std::sqrt(2.0)) : 0.0;
  p.phi_lo = (float)lo, p.half_minus_lo = (float)(0.5 - lo);
  {
    const double st = (double)cfg->sigma_t, tmax = (double)cfg->max_t_spread;
    const double lo_t = st > 0.0 ? 0.5 * std::erfc((tmax / st) / std::sqrt(2.0)) : 0.0;
    p.sigma_t = cfg->sigma_t, p.phi_lo_t = (float)lo_t, p.half_minus_lo_t = (float)(0.5 - lo_t);
    p.out_vt = out->vt;
  }
  for (int r = 0; r < 10; ++r) {
    p.rk.k0[r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
    p.rk.k1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
  }
  p.event_base = event_base, p.capacity = out->capacity;
  p.out_off = (long long *)out->offsets, p.out_pid = out->pid, p.out_charge = out->charge;
  p.is_pu = out->is_pu, p.n_pileup = out->n_pileup;
  unsigned char *ws = (unsigned char *)workspace;
  p.tile_counter = (unsigned int *)ws, p.status_word = (int *)(ws + 4);
  p.chain = (unsigned long long *)(ws + 16);
  p.cnt = (long long *)(ws + chain_bytes);
  const int rc = pd_launch_pileup(p, cuda_stream);
  if (rc != PD_OK) return cuda_fail(cudaGetLastError(), "pile-up kernel launch");
  t_launches = 3;
  return PD_OK;
}

// filter workspace: [tile counter, pad] 16 B | look-back words, one per tile | one 64-bit word per 32 positions 0..capacity
static size_t filter_chain_bytes(int64_t capacity) {
  const size_t tiles = (size_t)((capacity + 1 + PD_FILTER_TILE - 1) / PD_FILTER_TILE);
  return (16 + 8 * tiles + 255) & ~size_t(255);
}

int64_t pd_filter_workspace_bytes(int64_t capacity) {
  if (capacity < 0) return PD_EINVAL;
  return (int64_t)(filter_chain_bytes(capacity) + 8 * (size_t)((capacity + 1 + 31) / 32));
}

int pd_filter_eflow(const pd_eflow *in, int64_t n_events, const pd_condition *conds, int32_t n_conds, int32_t combine_any,
                    pd_eflow *out, void *workspace, int64_t workspace_bytes, void *cuda_stream) {
  t_launches = 0;
  if (!in || !out || n_events < 0 || n_conds < 0 || n_conds > PD_MAX_CONDITIONS || (n_conds > 0 && !conds)) return PD_EINVAL;
  if (in->capacity < 0 || in->capacity >= (int64_t(1) << 31) - 1) return PD_EINVAL;
  if (!in->offsets || !out->offsets) return PD_EINVAL;
  if (in->capacity > 0) {
    if (!in->cls || !in->src || !in->pt || !in->eta || !in->phi || !in->E) return PD_EINVAL;
    if (!out->cls || !out->src || !out->pt || !out->eta || !out->phi || !out->E) return PD_EINVAL;
  }
  for (int k = 0; k < n_conds; ++k) {
    const pd_condition &c = conds[k];
    if (c.field < PD_FIELD_PT || c.field > PD_FIELD_CLS || c.op < PD_OP_GT || c.op > PD_OP_NOT_IN) return PD_EINVAL;
    if (c.n_values < 0 || c.n_values > PD_MAX_SET_VALUES) return PD_EINVAL;
  }
  if (out->capacity < in->capacity) return PD_ECAPACITY;
  const int64_t need = pd_filter_workspace_bytes(in->capacity);
  if (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 15u)) return PD_EWORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t chain_bytes = filter_chain_bytes(in->capacity);
  PD_CUDA(cudaMemsetAsync(workspace, 0, chain_bytes, st));
  PdFilterParams p;
  std::memset(&p, 0, sizeof(p));
  p.n_events = n_events;
  p.offsets = (const long long *)in->offsets;
  p.cls = in->cls, p.src = in->src, p.pt = in->pt, p.eta = in->eta, p.phi = in->phi, p.E = in->E;
  p.out_offsets = (long long *)out->offsets;
  p.out_cls = out->cls, p.out_src = out->src, p.out_pt = out->pt, p.out_eta = out->eta, p.out_phi = out->phi, p.out_E = out->E;
  for (int k = 0; k < n_conds; ++k) p.conds[k] = conds[k], p.cond_fields |= 1u << conds[k].field;
  p.n_conds = n_conds, p.combine_any = combine_any ? 1 : 0;
  unsigned char *ws = (unsigned char *)workspace;
  p.tile_counter = (unsigned int *)ws;
  p.chain = (unsigned long long *)(ws + 16);
  p.wordrank = (unsigned long long *)(ws + chain_bytes);
  uintptr_t bits = 0;
  for (const void *a : {(const void *)in->cls, (const void *)in->src, (const void *)in->pt, (const void *)in->eta, (const void *)in->phi, (const void *)in->E})
    bits |= reinterpret_cast<uintptr_t>(a);
  p.aligned16 = (bits & 15u) == 0;
  const int rc = pd_launch_filter(p, cuda_stream);
  if (rc != PD_OK) return cuda_fail(cudaGetLastError(), "filter kernel launch");
  t_launches = 2;
  return PD_OK;
}

int pd_event_features(const pd_eflow *efl, int64_t n_events, float dr_max, float fsr_dr, pd_features *out,
                      void *cuda_stream) {
  t_launches = 0;
  if (!efl || !out || n_events < 0) return PD_EINVAL;
  if (!(dr_max >= 0.f) || !(fsr_dr >= 0.f) || !std::isfinite(dr_max) || !std::isfinite(fsr_dr)) return PD_EINVAL;
  if (!efl->offsets || !out->ht || !out->met_x || !out->met_y || !out->met) return PD_EINVAL;
  if (n_events == 0) return PD_OK;
  if (!efl->cls || !efl->pt || !efl->eta || !efl->phi) return PD_EINVAL;
  if (!out->iso_charged || !out->iso_neutral || !out->iso_photon || !out->r_iso) return PD_EINVAL;
  PdFeatParams p;
  p.n_events = n_events;
  p.offsets = (const long long *)efl->offsets;
  p.cls = efl->cls, p.pt = efl->pt, p.eta = efl->eta, p.phi = efl->phi;
  p.dr_max2 = (float)((double)dr_max * (double)dr_max), p.fsr2 = (float)((double)fsr_dr * (double)fsr_dr);
  p.inv_strip = 1.f / std::fmax(dr_max * 1.000001f, 0.375f);  // strip width >= dr_max (with a ulp of margin)
  {
    const double two_pi = 6.283185307179586;
    const double cells = dr_max > 0.f ? std::floor(two_pi / ((double)dr_max * 1.000001)) : 12.0;
    p.n_phi = (int)std::fmin(12.0, std::fmax(1.0, cells));
    p.inv_phi_cell = (float)((double)p.n_phi / two_pi);
  }
  p.ht = out->ht, p.met_x = out->met_x, p.met_y = out->met_y, p.met = out->met;
  p.iso_charged = out->iso_charged, p.iso_neutral = out->iso_neutral, p.iso_photon = out->iso_photon, p.r_iso = out->r_iso;
  const int rc = pd_launch_features(p, cuda_stream);
  if (rc != PD_OK) return cuda_fail(cudaGetLastError(), "features kernel launch");
  t_launches = 1;
  return PD_OK;
}

int64_t pd_truth_workspace_bytes(int64_t n_events) {
  if (n_events < 0) return PD_EINVAL;
  return 24 * (n_events > 0 ? n_events : 1);
}

int pd_truth_features(const pd_events *ev, int32_t skip_neutrinos, pd_features *out, void *workspace, int64_t workspace_bytes,
                      void *cuda_stream) {
  t_launches = 0;
  if (!ev || !out || ev->n_events < 0 || ev->n_particles < 0) return PD_EINVAL;
  if (ev->n_events == 0) return PD_OK;
  if (!ev->offsets || !out->ht || !out->met_x || !out->met_y || !out->met) return PD_EINVAL;
  if (ev->n_particles > 0 && (!ev->pid || !ev->px || !ev->py)) return PD_EINVAL;
  if (!workspace || (reinterpret_cast<uintptr_t>(workspace) & 7)) return PD_EINVAL;
  if (workspace_bytes < pd_truth_workspace_bytes(ev->n_events)) return PD_EWORKSPACE;
  PdTruthParams p;
  p.n_events = ev->n_events, p.n_particles = ev->n_particles;
  p.ev_off = (const long long *)ev->offsets, p.pid = ev->pid, p.px = ev->px, p.py = ev->py;
  p.skip_neutrinos = skip_neutrinos != 0;
  p.acc = (unsigned long long *)workspace;
  p.ht = out->ht, p.met_x = out->met_x, p.met_y = out->met_y, p.met = out->met;
  const int rc = pd_launch_truth(p, cuda_stream);
  if (rc != PD_OK) return cuda_fail(cudaGetLastError(), "truth features launch");
  t_launches = ev->n_particles > 0 ? 2 : 1;
  return PD_OK;
}

int pd_track_impact(const pd_card *card, const pd_events *ev, const pd_tracks *trk, const pd_impact_config *cfg,
                    uint64_t seed, int64_t event_base, pd_impact *out, void *cuda_stream) {
  t_launches = 0;
  if (!card || !ev || !trk || !cfg || !out || ev->n_events < 0 || ev->n_particles < 0) return PD_EINVAL;
  if (!(cfg->d0_a >= 0.f) || !(cfg->d0_b >= 0.f) || !(cfg->z0_a >= 0.f) || !(cfg->z0_b >= 0.f)) return PD_EINVAL;
  if (!std::isfinite(cfg->d0_a) || !std::isfinite(cfg->d0_b) || !std::isfinite(cfg->z0_a) || !std::isfinite(cfg->z0_b))
    return PD_EINVAL;
  if (ev->n_events == 0 || ev->n_particles == 0) return PD_OK;
  if (!ev->offsets || !ev->charge || !ev->px || !ev->py || !ev->pz || !ev->vx || !ev->vy || !ev->vz) return PD_EINVAL;
  if (!trk->offsets || !trk->src || !out->d0 || !out->z0 || !out->d0_err || !out->z0_err) return PD_EINVAL;
  PdImpactParams p;
  p.n_events = ev->n_events, p.n_particles = ev->n_particles;
  p.ev_off = (const long long *)ev->offsets, p.trk_off = (const long long *)trk->offsets;
  p.trk_src = trk->src, p.charge = ev->charge;
  p.px = ev->px, p.py = ev->py, p.pz = ev->pz, p.vx = ev->vx, p.vy = ev->vy, p.vz = ev->vz;
  p.inv_kB = card->sc.inv_kB, p.sB = card->sc.sB;
  p.d0_a = cfg->d0_a, p.d0_b = cfg->d0_b, p.z0_a = cfg->z0_a, p.z0_b = cfg->z0_b;
  for (int r = 0; r < 10; ++r) {
    p.rk.k0[r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
    p.rk.k1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
  }
  p.event_base = event_base;
  p.d0 = out->d0, p.z0 = out->z0, p.d0_err = out->d0_err, p.z0_err = out->z0_err;
  const int rc = pd_launch_impact(p, cuda_stream);
  if (rc != PD_OK) return cuda_fail(cudaGetLastError(), "impact kernel launch");
  t_launches = 1;
  return PD_OK;
}

}  // extern "C"

// The per-bin tables of a card on the current device: uploaded on first use, kept per device until pd_free_card.
int pd_card_to_device(const pd_card *c, const PdCardTables **tab) {
  std::lock_guard<std::mutex> lock(g_card_mutex);
  int dev = 0;
  PD_CUDA(cudaGetDevice(&dev));
  for (int k = 0; k < c->n_dev; ++k)
    if (c->dev_id[k] == dev) {
      *tab = &c->dev_tab[k];
      return PD_OK;
    }
  if (c->n_dev >= PD_MAX_CARD_DEVICES) {
    std::snprintf(t_cuda_msg, sizeof(t_cuda_msg), "card already resident on %d devices", PD_MAX_CARD_DEVICES);
    return PD_ECUDA;
  }
  const int slot = c->n_dev;
  const size_t nb = (size_t)c->sc.n_bins;
  const size_t lut_words = (c->lut.size() + 1) / 2;
  const size_t words = c->tb.size() + nb + (nb + 1) + 5 * nb + lut_words + 2 * nb + 6 * nb;
  std::vector<uint32_t> blob(words);
  size_t o = 0;
  auto put = [&](const void *src, size_t n) {
    std::memcpy(blob.data() + o, src, 4 * n);
    size_t at = o;
    o += n;
    return at;
  };
  const size_t o_tb = put(c->tb.data(), c->tb.size()), o_nphi = put(c->nphi.data(), nb), o_off = put(c->offset.data(), nb + 1);
  const size_t o_iw = put(c->inv_w.data(), nb), o_half = put(c->half.data(), nb), o_w = put(c->w.data(), nb);
  const size_t o_eta = put(c->eta_c.data(), nb), o_ic = put(c->inv_cosh.data(), nb);
  const size_t o_lut = o;
  std::memcpy(blob.data() + o, c->lut.data(), 2 * c->lut.size());
  o += lut_words;
  const size_t o_edge = put(c->edges.data(), 2 * nb), o_res2 = put(c->res2.data(), 6 * nb);
  void *d = nullptr;
  PD_CUDA(cudaMalloc(&d, 4 * words));
  cudaError_t e = cudaMemcpy(d, blob.data(), 4 * words, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(d);
    return cuda_fail(e, "cudaMemcpy(card)");
  }
  const uint32_t *base = (const uint32_t *)d;
  c->dev_tab[slot].tb = (const float *)(base + o_tb);
  c->dev_tab[slot].nphi = (const int *)(base + o_nphi);
  c->dev_tab[slot].offset = (const int *)(base + o_off);
  c->dev_tab[slot].inv_w = (const float *)(base + o_iw);
  c->dev_tab[slot].half = (const float *)(base + o_half);
  c->dev_tab[slot].w = (const float *)(base + o_w);
  c->dev_tab[slot].eta_c = (const float *)(base + o_eta);
  c->dev_tab[slot].inv_cosh = (const float *)(base + o_ic);
  c->dev_tab[slot].lut = (const unsigned short *)(base + o_lut);
  c->dev_tab[slot].edge = (const float *)(base + o_edge);
  c->dev_tab[slot].res2 = (const float *)(base + o_res2);
  c->dev_blob[slot] = d;
  c->dev_id[slot] = dev;
  c->n_dev = slot + 1;
  *tab = &c->dev_tab[slot];
  return PD_OK;
}

// particle_base = offsets[0] (device memory; the host must know it): 0 for the public entry, the first particle of the
// chunk for the pipelined host entry, whose chunks keep absolute offsets into the whole-batch arrays
static int simulate_impl(const pd_card *card, const pd_events *ev, uint64_t seed, int64_t event_base, pd_tracks *trk,
                         pd_towers *tow, pd_eflow *efl, pd_debug *dbg, void *workspace, int64_t workspace_bytes,
                         void *cuda_stream, int64_t particle_base, const pd_options *opt = nullptr) {
  t_launches = 0;
  if (!card || !ev || !trk || !tow || !efl || !options_ok(opt)) return PD_EINVAL;
  if (ev->n_events < 0 || ev->n_particles < 0 || ev->n_particles >= (int64_t(1) << 30)) return PD_EINVAL;
  if (!ev->offsets || !trk->offsets || !tow->offsets || !efl->offsets) return PD_EINVAL;
  const int64_t n = ev->n_particles;
  if (n > 0) {
    if (!ev->pid || !ev->charge || !ev->px || !ev->py || !ev->pz || !ev->E || !ev->vx || !ev->vy || !ev->vz) return PD_EINVAL;
    if (!trk->src || !trk->pid || !trk->charge || !trk->pt || !trk->eta || !trk->phi || !trk->E || !trk->eta_out || !trk->phi_out) return PD_EINVAL;
    if (!tow->tower || !tow->eta || !tow->phi || !tow->E || !tow->Eem || !tow->Ehad || !tow->ET) return PD_EINVAL;
    if (!efl->cls || !efl->src || !efl->pt || !efl->eta || !efl->phi || !efl->E) return PD_EINVAL;
  }
  if (trk->capacity < n || tow->capacity < n || efl->capacity < 2 * n) return PD_ECAPACITY;
  const int64_t need = pd_workspace_bytes_ex(card, ev->n_events, n, opt);
  if (!workspace || workspace_bytes < need || (reinterpret_cast<uintptr_t>(workspace) & 15u)) return PD_EWORKSPACE;
  cudaStream_t st = (cudaStream_t)cuda_stream;

  PdLaunchPlan plan;
  pd_plan(card, ev->n_events, n, tile_events_of(opt), &plan);
  PD_CUDA(cudaMemsetAsync(workspace, 0, ws_chain_bytes(plan), st));  // counters + look-back words; the keys need no init
  if (ev->n_events == 0) {
    PD_CUDA(cudaMemsetAsync(trk->offsets, 0, sizeof(int64_t), st));
    PD_CUDA(cudaMemsetAsync(tow->offsets, 0, sizeof(int64_t), st));
    PD_CUDA(cudaMemsetAsync(efl->offsets, 0, sizeof(int64_t), st));
    return PD_OK;
  }
  const PdCardTables *tab = nullptr;
  int rc = pd_card_to_device(card, &tab);
  if (rc != PD_OK) return rc;

  PdParams p;
  std::memset(&p, 0, sizeof(p));
  p.sc = card->sc;
  p.tab = *tab;
  p.n_events = ev->n_events, p.n_particles = n;
  p.offsets = (const long long *)ev->offsets;
  p.pid = ev->pid, p.charge = ev->charge;
  p.px = ev->px, p.py = ev->py, p.pz = ev->pz, p.E = ev->E, p.vx = ev->vx, p.vy = ev->vy, p.vz = ev->vz;
  p.seed = seed, p.event_base = event_base;
  for (int r = 0; r < 10; ++r) {
    p.rk.k0[r] = (uint32_t)seed + (uint32_t)r * 0x9E3779B9u;
    p.rk.k1[r] = (uint32_t)(seed >> 32) + (uint32_t)r * 0xBB67AE85u;
  }
  p.trk_offsets = (long long *)trk->offsets;
  p.trk_src = trk->src, p.trk_pid = trk->pid, p.trk_charge = trk->charge;
  p.trk_pt = trk->pt, p.trk_eta = trk->eta, p.trk_phi = trk->phi, p.trk_E = trk->E;
  p.trk_eta_out = trk->eta_out, p.trk_phi_out = trk->phi_out;
  p.tow_offsets = (long long *)tow->offsets;
  p.tow_tower = tow->tower, p.tow_eta = tow->eta, p.tow_phi = tow->phi, p.tow_E = tow->E;
  p.tow_Eem = tow->Eem, p.tow_Ehad = tow->Ehad, p.tow_ET = tow->ET;
  p.efl_offsets = (long long *)efl->offsets;
  p.efl_cls = efl->cls, p.efl_src = efl->src, p.efl_pt = efl->pt, p.efl_eta = efl->eta, p.efl_phi = efl->phi, p.efl_E = efl->E;
  if (dbg) {
    p.dbg_status = dbg->status, p.dbg_eta_pos = dbg->eta_pos, p.dbg_phi_pos = dbg->phi_pos, p.dbg_tower = dbg->tower;
    p.dbg_accepted = dbg->accepted, p.dbg_eps_row = dbg->eps_row, p.dbg_pt_smeared = dbg->pt_smeared;
    p.dbg_tw_first = dbg->tw_first;
    p.dbg_tw[0] = dbg->tw_Eem_true, p.dbg_tw[1] = dbg->tw_Ehad_true, p.dbg_tw[2] = dbg->tw_Tem, p.dbg_tw[3] = dbg->tw_Thad;
    p.dbg_tw[4] = dbg->tw_Eem_smeared, p.dbg_tw[5] = dbg->tw_Ehad_smeared;
    p.dbg_tw_dec = dbg->tw_decisions;
  }
  p.events_per_tile = plan.events_per_tile;
  p.n_tiles = plan.n_tiles;
  p.capacity = plan.capacity;
  p.sparse = plan.sparse;
  p.lay = plan.lay;
  unsigned char *ws = (unsigned char *)workspace;
  p.tile_counter = (unsigned int *)ws;
  p.status_word = (int *)(ws + 4);
  p.ptile_counter = (unsigned int *)(ws + 8);
  p.chain = (unsigned long long *)(ws + kWsHeader);
  p.chain_t = p.chain + (plan.n_tiles > 0 ? plan.n_tiles : 1);
  {
    const WsLayout wl = ws_layout(plan, card->sc.n_towers, impact_of(opt), card->sc.eflow_weighted != 0);
    p.tile_ev = (int *)(ws + wl.tile_ev);
    p.key = (unsigned short *)(ws + wl.key);
    p.accmask = (unsigned int *)(ws + wl.accmask);
    p.park_idx = ws + wl.idx;
    p.park_q = (signed char *)(ws + wl.q);
    p.park_pid = (int *)(ws + wl.pid);
    p.big_acc = (long long *)(ws + wl.big_acc);
    for (int k = 0; k < 6; ++k) p.park_f[k] = (float *)(ws + wl.f[k]);
    p.acc_stride = card->sc.eflow_weighted ? 7 : 5;
    if (card->sc.eflow_weighted) p.park_sig = (float *)(ws + wl.sig);
    if (impact_of(opt)) {
      p.imp_on = 1;
      p.imp_d0_a = opt->impact_config->d0_a, p.imp_d0_b = opt->impact_config->d0_b;
      p.imp_z0_a = opt->impact_config->z0_a, p.imp_z0_b = opt->impact_config->z0_b;
      for (int k = 0; k < 4; ++k) p.park_imp[k] = (float *)(ws + wl.imp[k]);
      p.imp_out[0] = opt->impact->d0, p.imp_out[1] = opt->impact->z0, p.imp_out[2] = opt->impact->d0_err, p.imp_out[3] = opt->impact->z0_err;
    }
  }
  p.n_ptiles = plan.n_ptiles;
  p.p_base = particle_base;
  {
    // bulk copies (cp.async.bulk) want 16-byte aligned global addresses: tiles start at multiples of PD_PTILE
    // particles, so it is the base pointers that count
    const uintptr_t all = reinterpret_cast<uintptr_t>(ev->pid) | reinterpret_cast<uintptr_t>(ev->charge) | reinterpret_cast<uintptr_t>(ev->px) |
                          reinterpret_cast<uintptr_t>(ev->py) | reinterpret_cast<uintptr_t>(ev->pz) | reinterpret_cast<uintptr_t>(ev->vx) |
                          reinterpret_cast<uintptr_t>(ev->vy) | reinterpret_cast<uintptr_t>(ev->vz) | reinterpret_cast<uintptr_t>(ev->E);
    p.tma_ok = (all & 15u) == 0 ? 1 : 0;
  }

  rc = pd_launch_chain(p, plan, dbg != nullptr, cuda_stream);
  if (rc != PD_OK) return cuda_fail(cudaGetLastError(), "kernel launch");
  t_launches = n > 0 ? 3 : 1;
  return PD_OK;
}

extern "C" {

int pd_simulate(const pd_card *card, const pd_events *ev, uint64_t seed, int64_t event_base, pd_tracks *trk,
                pd_towers *tow, pd_eflow *efl, pd_debug *dbg, void *workspace, int64_t workspace_bytes,
                void *cuda_stream) {
  return simulate_impl(card, ev, seed, event_base, trk, tow, efl, dbg, workspace, workspace_bytes, cuda_stream, 0);
}

int pd_simulate_ex(const pd_card *card, const pd_events *ev, uint64_t seed, int64_t event_base, pd_tracks *trk,
                   pd_towers *tow, pd_eflow *efl, pd_debug *dbg, void *workspace, int64_t workspace_bytes,
                   const pd_options *opt, void *cuda_stream) {
  return simulate_impl(card, ev, seed, event_base, trk, tow, efl, dbg, workspace, workspace_bytes, cuda_stream, 0, opt);
}

int pd_last_status(const void *workspace, void *cuda_stream) {
  if (!workspace) return PD_EINVAL;
  int word = 0;
  PD_CUDA(cudaMemcpyAsync(&word, (const unsigned char *)workspace + 4, sizeof(int), cudaMemcpyDeviceToHost, (cudaStream_t)cuda_stream));
  PD_CUDA(cudaStreamSynchronize((cudaStream_t)cuda_stream));
  return word;
}

}  // extern "C"

// keep freed blocks in the stream-ordered pool between calls (the default threshold releases them at every sync)
static int keep_pool_blocks() {
  static thread_local int pool_dev = -1;
  int dev = 0;
  PD_CUDA(cudaGetDevice(&dev));
  if (pool_dev != dev) {
    cudaMemPool_t pool;
    PD_CUDA(cudaDeviceGetDefaultMemPool(&pool, dev));
    unsigned long long keep = ~0ull;
    PD_CUDA(cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep));
    pool_dev = dev;
  }
  return PD_OK;
}

static int simulate_host_once(const pd_card *card, const pd_events *ev, uint64_t seed, int64_t event_base, pd_tracks *trk,
                              pd_towers *tow, pd_eflow *efl, void *cuda_stream) {
  t_launches = 0;
  if (!card || !ev || !trk || !tow || !efl) return PD_EINVAL;
  if (ev->n_events < 0 || ev->n_particles < 0 || ev->n_particles >= (int64_t(1) << 30)) return PD_EINVAL;
  if (!ev->offsets || !trk->offsets || !tow->offsets || !efl->offsets) return PD_EINVAL;
  const int64_t n = ev->n_particles, ne = ev->n_events;
  if (trk->capacity < n || tow->capacity < n || efl->capacity < 2 * n) return PD_ECAPACITY;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t np = (size_t)(n > 0 ? n : 1);
  const int64_t ws_bytes = pd_workspace_bytes(card, ne, n);
  // one stream-ordered allocation, carved up (256-byte aligned pieces)
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t b_off = up(8 * (size_t)(ne + 1));
  const size_t in_bytes = b_off + up(4 * np) + up(np) + 7 * up(4 * np);
  const size_t trk_bytes = b_off + 2 * up(4 * np) + up(np) + 6 * up(4 * np);
  const size_t tow_bytes = b_off + up(4 * np) + 6 * up(4 * np);
  const size_t efl_bytes = b_off + up(2 * np) + up(8 * np) + 4 * up(8 * np);
  const size_t total = in_bytes + trk_bytes + tow_bytes + efl_bytes + up((size_t)ws_bytes);
  unsigned char *base = nullptr;
  if (int prc = keep_pool_blocks()) return prc;
  PD_CUDA(cudaMallocAsync((void **)&base, total, st));
  size_t o = 0;
  auto take = [&](size_t bytes) {
    unsigned char *ptr = base + o;
    o += up(bytes);
    return ptr;
  };
  int rc = PD_OK;
  pd_events d_ev = *ev;
  pd_tracks d_trk = *trk;
  pd_towers d_tow = *tow;
  pd_eflow d_efl = *efl;
  cudaError_t ce = cudaSuccess;
  auto h2d = [&](const void *src, size_t bytes) {
    unsigned char *dst = take(bytes);
    if (ce == cudaSuccess && bytes > 0 && src) ce = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, st);
    return dst;
  };
  d_ev.offsets = (const int64_t *)h2d(ev->offsets, 8 * (size_t)(ne + 1));
  d_ev.pid = (const int32_t *)h2d(ev->pid, 4 * (size_t)n);
  d_ev.charge = (const int8_t *)h2d(ev->charge, (size_t)n);
  d_ev.px = (const float *)h2d(ev->px, 4 * (size_t)n);
  d_ev.py = (const float *)h2d(ev->py, 4 * (size_t)n);
  d_ev.pz = (const float *)h2d(ev->pz, 4 * (size_t)n);
  d_ev.E = (const float *)h2d(ev->E, 4 * (size_t)n);
  d_ev.vx = (const float *)h2d(ev->vx, 4 * (size_t)n);
  d_ev.vy = (const float *)h2d(ev->vy, 4 * (size_t)n);
  d_ev.vz = (const float *)h2d(ev->vz, 4 * (size_t)n);
  d_trk.offsets = (int64_t *)take(8 * (size_t)(ne + 1));
  d_trk.src = (int32_t *)take(4 * np), d_trk.pid = (int32_t *)take(4 * np), d_trk.charge = (int8_t *)take(np);
  d_trk.pt = (float *)take(4 * np), d_trk.eta = (float *)take(4 * np), d_trk.phi = (float *)take(4 * np);
  d_trk.E = (float *)take(4 * np), d_trk.eta_out = (float *)take(4 * np), d_trk.phi_out = (float *)take(4 * np);
  d_tow.offsets = (int64_t *)take(8 * (size_t)(ne + 1));
  d_tow.tower = (int32_t *)take(4 * np);
  d_tow.eta = (float *)take(4 * np), d_tow.phi = (float *)take(4 * np), d_tow.E = (float *)take(4 * np);
  d_tow.Eem = (float *)take(4 * np), d_tow.Ehad = (float *)take(4 * np), d_tow.ET = (float *)take(4 * np);
  d_efl.offsets = (int64_t *)take(8 * (size_t)(ne + 1));
  d_efl.cls = (int8_t *)take(2 * np), d_efl.src = (int32_t *)take(8 * np);
  d_efl.pt = (float *)take(8 * np), d_efl.eta = (float *)take(8 * np), d_efl.phi = (float *)take(8 * np), d_efl.E = (float *)take(8 * np);
  void *ws = take((size_t)ws_bytes);
  if (ce != cudaSuccess) rc = cuda_fail(ce, "cudaMemcpyAsync(H2D)");
  if (rc == PD_OK) rc = pd_simulate(card, &d_ev, seed, event_base, &d_trk, &d_tow, &d_efl, nullptr, ws, ws_bytes, cuda_stream);
  const int launches = t_launches;
  int64_t tot[3] = {0, 0, 0};
  if (rc == PD_OK) {
    // totals first (three 8-byte reads), then exactly the produced elements
    ce = cudaMemcpyAsync(&tot[0], d_trk.offsets + ne, 8, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(&tot[1], d_tow.offsets + ne, 8, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(&tot[2], d_efl.offsets + ne, 8, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) rc = cuda_fail(ce, "read totals");
  }
  if (rc == PD_OK) {
    auto d2h = [&](void *dst, const void *src, size_t bytes) {
      if (ce == cudaSuccess && bytes > 0 && dst) ce = cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, st);
    };
    const size_t nt = (size_t)tot[0], nw = (size_t)tot[1], nf = (size_t)tot[2], nofs = 8 * (size_t)(ne + 1);
    d2h(trk->offsets, d_trk.offsets, nofs);
    d2h(trk->src, d_trk.src, 4 * nt), d2h(trk->pid, d_trk.pid, 4 * nt), d2h(trk->charge, d_trk.charge, nt);
    d2h(trk->pt, d_trk.pt, 4 * nt), d2h(trk->eta, d_trk.eta, 4 * nt), d2h(trk->phi, d_trk.phi, 4 * nt);
    d2h(trk->E, d_trk.E, 4 * nt), d2h(trk->eta_out, d_trk.eta_out, 4 * nt), d2h(trk->phi_out, d_trk.phi_out, 4 * nt);
    d2h(tow->offsets, d_tow.offsets, nofs);
    d2h(tow->tower, d_tow.tower, 4 * nw), d2h(tow->eta, d_tow.eta, 4 * nw), d2h(tow->phi, d_tow.phi, 4 * nw);
    d2h(tow->E, d_tow.E, 4 * nw), d2h(tow->Eem, d_tow.Eem, 4 * nw), d2h(tow->Ehad, d_tow.Ehad, 4 * nw), d2h(tow->ET, d_tow.ET, 4 * nw);
    d2h(efl->offsets, d_efl.offsets, nofs);
    d2h(efl->cls, d_efl.cls, nf), d2h(efl->src, d_efl.src, 4 * nf), d2h(efl->pt, d_efl.pt, 4 * nf);
    d2h(efl->eta, d_efl.eta, 4 * nf), d2h(efl->phi, d_efl.phi, 4 * nf), d2h(efl->E, d_efl.E, 4 * nf);
    int word = 0;
    if (ce == cudaSuccess) ce = cudaMemcpyAsync(&word, (unsigned char *)ws + 4, 4, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce != cudaSuccess) rc = cuda_fail(ce, "cudaMemcpyAsync(D2H)");
    else if (word != 0) rc = word;
  }
  cudaFreeAsync(base, st);
  cudaStreamSynchronize(st);
  t_launches = launches;
  return rc;
}

// Large batches: the same call in K chunks of consecutive events, pipelined over three streams so that the
// host->device copy of chunk c+1, the kernel of chunk c and the device->host copy of chunk c-1 overlap (the link is
// full duplex).  Events are independent and offsets / particle indices are kept absolute, so the result is
// bit for bit that of the single-shot path.
static int simulate_host_pipelined(const pd_card *card, const pd_events *ev, uint64_t seed, int64_t event_base, pd_tracks *trk,
                                   pd_towers *tow, pd_eflow *efl, void *cuda_stream, int K) {
  t_launches = 0;
  const int64_t n = ev->n_particles, ne = ev->n_events;
  if (trk->capacity < n || tow->capacity < n || efl->capacity < 2 * n) return PD_ECAPACITY;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // chunk boundaries: consecutive events, balanced by particle count (host offsets)
  std::vector<int64_t> eb(K + 1, 0);
  for (int c = 1; c < K; ++c) {
    const int64_t want = n * c / K;
    const int64_t *pos = std::upper_bound(ev->offsets, ev->offsets + ne + 1, want);
    int64_t e = (pos - ev->offsets) - 1;
    eb[c] = std::min(std::max(e, eb[c - 1]), ne);
  }
  eb[K] = ne;
  int64_t ws_bytes = 0, n_max = 0;
  for (int c = 0; c < K; ++c) {
    const int64_t nc = ev->offsets[eb[c + 1]] - ev->offsets[eb[c]];
    ws_bytes = std::max(ws_bytes, pd_workspace_bytes(card, eb[c + 1] - eb[c], nc));
    n_max = std::max(n_max, nc);
  }
  auto up = [](size_t x) { return (x + 255) & ~size_t(255); };
  const size_t np = (size_t)n;
  const size_t b_off = up(8 * (size_t)(ne + 1 + K));
  const size_t total = b_off + up(4 * np) + up(np) + 7 * up(4 * np)            // inputs
                       + b_off + 2 * up(4 * np) + up(np) + 6 * up(4 * np)      // tracks
                       + b_off + 7 * up(4 * np)                                // towers
                       + b_off + up(2 * np) + 5 * up(8 * np)                   // eflow
                       + up((size_t)ws_bytes) + up(64);
  unsigned char *base = nullptr;
  if (int prc = keep_pool_blocks()) return prc;
  PD_CUDA(cudaMallocAsync((void **)&base, total, st));
  size_t o = 0;
  auto take = [&](size_t bytes) {
    unsigned char *ptr = base + o;
    o += up(bytes);
    return ptr;
  };
  int64_t *d_off = (int64_t *)take(8 * (size_t)(ne + 1 + K));
  // within each collection the 4-byte arrays are allocated back to back (equal pitch): when the caller's host arrays
  // are equally spaced too, a chunk's copies collapse into one 2-D copy per group (copy_rows below)
  int8_t *d_q = (int8_t *)take(np);
  int32_t *d_pid = (int32_t *)take(4 * np);
  float *d_in[7];
  for (auto &ptr : d_in) ptr = (float *)take(4 * np);
  int64_t *t_off = (int64_t *)take(8 * (size_t)(ne + 1 + K));
  int8_t *t_q = (int8_t *)take(np);
  int32_t *t_src = (int32_t *)take(4 * np), *t_pid = (int32_t *)take(4 * np);
  float *t_f[6];
  for (auto &ptr : t_f) ptr = (float *)take(4 * np);
  int64_t *w_off = (int64_t *)take(8 * (size_t)(ne + 1 + K));
  int32_t *w_id = (int32_t *)take(4 * np);
  float *w_f[6];
  for (auto &ptr : w_f) ptr = (float *)take(4 * np);
  int64_t *f_off = (int64_t *)take(8 * (size_t)(ne + 1 + K));
  int8_t *f_cls = (int8_t *)take(2 * np);
  int32_t *f_src = (int32_t *)take(8 * np);
  float *f_f[4];
  for (auto &ptr : f_f) ptr = (float *)take(8 * np);
  void *ws = take((size_t)ws_bytes);
  int *d_words = (int *)take(64);  // the chunks' status words, gathered for one read at the end

  cudaStream_t s_in = nullptr, s_out = nullptr;
  std::vector<cudaEvent_t> e_in(K, nullptr), e_k(K, nullptr);
  cudaEvent_t e_start = nullptr;
  cudaError_t ce = cudaStreamCreateWithFlags(&s_in, cudaStreamNonBlocking);
  if (ce == cudaSuccess) ce = cudaStreamCreateWithFlags(&s_out, cudaStreamNonBlocking);
  for (int c = 0; c < K && ce == cudaSuccess; ++c) {
    ce = cudaEventCreateWithFlags(&e_in[c], cudaEventDisableTiming);
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e_k[c], cudaEventDisableTiming);
  }
  if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e_start, cudaEventDisableTiming);
  // the side streams start after the allocation (and whatever precedes the call) on the caller's stream
  if (ce == cudaSuccess) ce = cudaEventRecord(e_start, st);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(s_in, e_start, 0);
  if (ce == cudaSuccess) ce = cudaStreamWaitEvent(s_out, e_start, 0);
  int rc = ce == cudaSuccess ? PD_OK : cuda_fail(ce, "pipeline set-up");

  const float *h_in[7] = {ev->px, ev->py, ev->pz, ev->E, ev->vx, ev->vy, ev->vz};
  float *h_tf[6] = {trk->pt, trk->eta, trk->phi, trk->E, trk->eta_out, trk->phi_out};
  float *h_wf[6] = {tow->eta, tow->phi, tow->E, tow->Eem, tow->Ehad, tow->ET};
  float *h_ff[4] = {efl->pt, efl->eta, efl->phi, efl->E};
  auto cp = [&](void *dst, const void *src, size_t bytes, cudaMemcpyKind kind, cudaStream_t s) {
    if (ce == cudaSuccess && bytes > 0 && dst && src) ce = cudaMemcpyAsync(dst, src, bytes, kind, s);
  };
  // `rows` copies of `bytes` each; one strided copy when source and destination rows are equally spaced
  bool strided_ok = true;
  auto copy_rows = [&](int rows, void *const *dst, const void *const *src, size_t bytes, cudaMemcpyKind kind, cudaStream_t s) {
    if (bytes == 0 || ce != cudaSuccess) return;
    bool strided = rows > 1;
    ptrdiff_t dp = 0, sp = 0;
    if (strided) {
      dp = (const char *)dst[1] - (const char *)dst[0], sp = (const char *)src[1] - (const char *)src[0];
      strided = dp >= (ptrdiff_t)bytes && sp >= (ptrdiff_t)bytes && dp < (ptrdiff_t)0x7fffffff && sp < (ptrdiff_t)0x7fffffff;
      for (int k = 2; k < rows && strided; ++k)
        strided = (const char *)dst[k] - (const char *)dst[k - 1] == dp && (const char *)src[k] - (const char *)src[k - 1] == sp;
    }
    if (strided) {
      // equally spaced rows that belong to SEPARATE host allocations are refused at enqueue time (the strided copy
      // must lie inside one allocation): nothing was queued, fall back to a copy per row from then on
      const cudaError_t e2 = strided_ok ? cudaMemcpy2DAsync(dst[0], (size_t)dp, src[0], (size_t)sp, bytes, (size_t)rows, kind, s)
                                        : cudaErrorInvalidValue;
      if (e2 == cudaSuccess) return;
      if (e2 != cudaErrorInvalidValue) {
        ce = e2;
        return;
      }
      if (strided_ok) cudaGetLastError();
      strided_ok = false;
    }
    for (int k = 0; k < rows; ++k) cp(dst[k], src[k], bytes, kind, s);
  };
  auto upload = [&](int c) {
    const int64_t e0 = eb[c], e1 = eb[c + 1], p0 = ev->offsets[e0], nc = ev->offsets[e1] - p0;
    cp(d_off + e0 + c, ev->offsets + e0, 8 * (size_t)(e1 - e0 + 1), cudaMemcpyHostToDevice, s_in);  // absolute offsets
    cp(d_q + p0, ev->charge + p0, (size_t)nc, cudaMemcpyHostToDevice, s_in);
    void *dd[8] = {d_pid + p0};
    const void *hh[8] = {ev->pid + p0};
    for (int f = 0; f < 7; ++f) dd[1 + f] = d_in[f] + p0, hh[1 + f] = h_in[f] + p0;
    copy_rows(8, dd, hh, 4 * (size_t)nc, cudaMemcpyHostToDevice, s_in);
    if (ce == cudaSuccess) ce = cudaEventRecord(e_in[c], s_in);
  };
  std::vector<int64_t> tot(3 * (size_t)K, 0), basec(3 * (size_t)(K + 1), 0);
  int launches = 0;
  if (rc == PD_OK) upload(0);
  for (int c = 0; c < K && rc == PD_OK; ++c) {
    if (c + 1 < K) upload(c + 1);  // one chunk ahead of the kernel
    const int64_t e0 = eb[c], e1 = eb[c + 1], p0 = ev->offsets[e0], nc = ev->offsets[e1] - p0, nec = e1 - e0;
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(st, e_in[c], 0);
    if (ce != cudaSuccess) {
      rc = cuda_fail(ce, "pipeline H2D");
      break;
    }
    // the chunk as a call of its own: absolute offsets and whole-batch input arrays (particle indices stay those of
    // the full call), outputs at the chunk's slice of the device arrays
    pd_events cev = {nec, nc, d_off + e0 + c, d_pid, d_q, d_in[0], d_in[1], d_in[2], d_in[3], d_in[4], d_in[5], d_in[6]};
    pd_tracks ct = {nc, t_off + e0 + c, t_src + p0, t_pid + p0, t_q + p0, t_f[0] + p0, t_f[1] + p0, t_f[2] + p0, t_f[3] + p0, t_f[4] + p0, t_f[5] + p0};
    pd_towers cw = {nc, w_off + e0 + c, w_id + p0, w_f[0] + p0, w_f[1] + p0, w_f[2] + p0, w_f[3] + p0, w_f[4] + p0, w_f[5] + p0};
    pd_eflow cf = {2 * nc, f_off + e0 + c, f_cls + 2 * p0, f_src + 2 * p0, f_f[0] + 2 * p0, f_f[1] + 2 * p0, f_f[2] + 2 * p0, f_f[3] + 2 * p0};
    rc = simulate_impl(card, &cev, seed, event_base + e0, &ct, &cw, &cf, nullptr, ws, ws_bytes, cuda_stream, p0);
    if (rc != PD_OK) break;
    launches += t_launches;
    cp(&tot[3 * (size_t)c + 0], t_off + e0 + c + nec, 8, cudaMemcpyDeviceToHost, st);
    cp(&tot[3 * (size_t)c + 1], w_off + e0 + c + nec, 8, cudaMemcpyDeviceToHost, st);
    cp(&tot[3 * (size_t)c + 2], f_off + e0 + c + nec, 8, cudaMemcpyDeviceToHost, st);
    cp(d_words + c, (unsigned char *)ws + 4, 4, cudaMemcpyDeviceToDevice, st);
    if (ce == cudaSuccess) ce = cudaEventRecord(e_k[c], st);
    if (ce == cudaSuccess) ce = cudaEventSynchronize(e_k[c]);  // the totals say how much to copy back, and where to
    if (ce != cudaSuccess) {
      rc = cuda_fail(ce, "pipeline kernel");
      break;
    }
    const size_t nt = (size_t)tot[3 * (size_t)c], nw = (size_t)tot[3 * (size_t)c + 1], nf = (size_t)tot[3 * (size_t)c + 2];
    const size_t bt = (size_t)basec[3 * (size_t)c], bw = (size_t)basec[3 * (size_t)c + 1], bf = (size_t)basec[3 * (size_t)c + 2];
    for (int k = 0; k < 3; ++k) basec[3 * (size_t)(c + 1) + k] = basec[3 * (size_t)c + k] + tot[3 * (size_t)c + k];
    if (ce == cudaSuccess) ce = cudaStreamWaitEvent(s_out, e_k[c], 0);
    // chunk-relative offsets land behind the chunk's first entry; rebased on the host at the end
    cp(trk->offsets + e0 + 1, t_off + e0 + c + 1, 8 * (size_t)nec, cudaMemcpyDeviceToHost, s_out);
    cp(tow->offsets + e0 + 1, w_off + e0 + c + 1, 8 * (size_t)nec, cudaMemcpyDeviceToHost, s_out);
    cp(efl->offsets + e0 + 1, f_off + e0 + c + 1, 8 * (size_t)nec, cudaMemcpyDeviceToHost, s_out);
    {
      void *hh[8] = {trk->src + bt, trk->pid + bt};
      const void *dd[8] = {t_src + p0, t_pid + p0};
      for (int f = 0; f < 6; ++f) hh[2 + f] = h_tf[f] + bt, dd[2 + f] = t_f[f] + p0;
      copy_rows(8, hh, dd, 4 * nt, cudaMemcpyDeviceToHost, s_out);
      cp(trk->charge + bt, t_q + p0, nt, cudaMemcpyDeviceToHost, s_out);
    }
    {
      void *hh[7] = {tow->tower + bw};
      const void *dd[7] = {w_id + p0};
      for (int f = 0; f < 6; ++f) hh[1 + f] = h_wf[f] + bw, dd[1 + f] = w_f[f] + p0;
      copy_rows(7, hh, dd, 4 * nw, cudaMemcpyDeviceToHost, s_out);
    }
    {
      void *hh[5] = {efl->src + bf};
      const void *dd[5] = {f_src + 2 * p0};
      for (int f = 0; f < 4; ++f) hh[1 + f] = h_ff[f] + bf, dd[1 + f] = f_f[f] + 2 * p0;
      copy_rows(5, hh, dd, 4 * nf, cudaMemcpyDeviceToHost, s_out);
      cp(efl->cls + bf, f_cls + 2 * p0, nf, cudaMemcpyDeviceToHost, s_out);
    }
  }
  int words[16] = {0};
  if (rc == PD_OK) {
    cp(words, d_words, 4 * (size_t)K, cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(st);
    if (ce == cudaSuccess) ce = cudaStreamSynchronize(s_out);
    if (ce != cudaSuccess) rc = cuda_fail(ce, "pipeline D2H");
  }
  if (rc == PD_OK) {
    trk->offsets[0] = 0, tow->offsets[0] = 0, efl->offsets[0] = 0;
    for (int c = 0; c < K; ++c) {
      if (words[c] != 0) rc = words[c];
      for (int64_t e = eb[c] + 1; e <= eb[c + 1]; ++e) {
        trk->offsets[e] += basec[3 * (size_t)c], tow->offsets[e] += basec[3 * (size_t)c + 1], efl->offsets[e] += basec[3 * (size_t)c + 2];
      }
    }
  }
  cudaStreamSynchronize(s_in), cudaStreamSynchronize(s_out), cudaStreamSynchronize(st);
  for (int c = 0; c < K; ++c) {
    if (e_in[c]) cudaEventDestroy(e_in[c]);
    if (e_k[c]) cudaEventDestroy(e_k[c]);
  }
  if (e_start) cudaEventDestroy(e_start);
  if (s_in) cudaStreamDestroy(s_in);
  if (s_out) cudaStreamDestroy(s_out);
  cudaFreeAsync(base, st);
  cudaStreamSynchronize(st);
  t_launches = launches;
  return rc;
}

extern "C" {

int pd_simulate_host(const pd_card *card, const pd_events *ev, uint64_t seed, int64_t event_base, pd_tracks *trk,
                     pd_towers *tow, pd_eflow *efl, void *cuda_stream) {
  // large batches go through in pipelined chunks (copies in both directions overlap the kernels)
  int K = 1;
  if (card && ev && trk && tow && efl && ev->offsets && trk->offsets && tow->offsets && efl->offsets && ev->n_events >= 1 &&
      ev->n_particles >= 1 && ev->n_particles < (int64_t(1) << 30)) {
    if (ev->n_events >= 64 && ev->n_particles >= (int64_t(1) << 22)) K = (int)std::min<int64_t>(8, ev->n_particles >> 21);
    if (const char *env = std::getenv("PD_HOST_CHUNKS")) K = std::max(1, std::min(16, std::atoi(env)));  // testing / tuning
    K = (int)std::min<int64_t>(K, ev->n_events);
  }
  int rc = K > 1 ? simulate_host_pipelined(card, ev, seed, event_base, trk, tow, efl, cuda_stream, K)
                 : simulate_host_once(card, ev, seed, event_base, trk, tow, efl, cuda_stream);
  return rc;
}

}  // extern "C"
