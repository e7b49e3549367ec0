// pd_towers.cu -- kernel T of the chain: the per-event half (steps S5-S8 of SURVEY.md section 8a).
//
// Kernel P (pd_particles.cu) has left, per particle, a 16-bit key (tower id | HCAL bit, 0xffff = no deposit) and
// the finished Track collection.  Here persistent CTAs (two 512-thread CTAs per SM, or one 1024-thread CTA for
// large events) claim TILES (runs of G whole events, <= C particles) from an atomic counter and take each through
//   pass A'  S5         keys and deposit energies of the tile (coalesced); marks the tower in the event's BITMAP
//   scan 1              popcount prefix of the bitmaps = the rank ("slot") of every occupied tower in
//                       (event, tower id) order -- this replaces a sort of the deposits; meanwhile the energies of
//                       the tile's tracks are scattered to their particles
//   pass B   S5         every deposit pushes itself on its slot's list (one integer atomicExch)
//   pass W   S5-S7      one thread per occupied tower: exact fixed-point sum of its list (order-independent),
//                       Philox tower stream, log-normal smear, thresholds, EFlow subtraction
//   scan W              one scan over the per-warp counts; chain W published and resolved (decoupled look-back)
//   pass O   S8         ordered compaction of towers / photons / neutral hadrons, the EFlow entries of the tracks
//                       (copied from the Track collection), CSR offsets
// Large grids with small events use a two-level bitmap (sparse mode, see make_layout): groups first, then the
// tower bits of the non-empty groups only.
// Sums are order-stable: each tower's deposits are added as 64-bit fixed-point integers (exact, hence independent
// of the order in which the list was built), and the only atomics are integer (bitmap OR, list exchange, counters).
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstdlib>

#include "pd_internal.h"
#include "pd_math.cuh"
#include "pd_scan.cuh"

namespace pdk {

constexpr int G_MAX = 256;         // events per tile (event index of a particle is kept in 8 bits)
constexpr int C_MAX = 8191;        // particles per tile: list links are 13 bits, 0x1fff = end of list
constexpr uint32_t LINK_END = 0x1fffu;
// per-particle result word: tower id (15 bits, 0x7fff none) | flags | link to the next deposit of the tower
constexpr uint32_t RES_TOWER = 0x7fffu, RES_DEP = 1u << 15, RES_HCAL = 1u << 16, RES_ACC = 1u << 17;
constexpr int RES_LINK_SHIFT = 18;
constexpr unsigned long long FIELD_MASK = (1ull << 31) - 1;  // chain W packs towers | neutrals << 31
// per-slot word after pass W: head particle (13 bits) | tower id (15 bits) << 13 | what the slot emits
constexpr uint32_t SLOT_TW = 1u << 28, SLOT_PH = 1u << 29, SLOT_NH = 1u << 30;

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~size_t(15); }

// Shared-memory carve-up of kernel T (PdTLayout, pd_internal.h): computed once on the host and handed to the kernel
// in its parameters, so that an array's address is one constant-bank operand instead of arithmetic on G and C.
using Layout = PdTLayout;

// Dense mode: one bit per tower and event (bitmap), a prefix per 128-tower group (gprefix).
// Sparse mode (large grids, small events: the bitmaps would be almost empty and take most of the shared memory):
// `bitmap` holds one bit per 128-tower GROUP and event, `l2p` the rank of the first non-empty group of each of its
// words, `pool` the tower bits of the non-empty groups only (at most one per deposit), `gprefix` their prefixes.
__host__ __device__ inline Layout make_layout(int n_bins, int n_towers, int words_per_event, int G, int C, int sparse, int res_per_bin = 0,
                                              int smear_center = 0, int weighted = 0) {
  Layout l;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = align16(o + bytes);
    return (uint32_t)at;
  };
  l.offset = take(4 * (n_bins + 1));
  l.w = take(4 * n_bins);
  l.eta_c = take(4 * n_bins);
  l.inv_cosh = take(4 * n_bins);
  l.binlut = take(2 * (size_t)((n_towers >> 5) + 2));
  l.res2 = take(res_per_bin ? 4 * 6 * (size_t)n_bins : 0);
  l.edge = take(smear_center ? 4 * 2 * (size_t)n_bins : 0);
  l.off32 = take(4 * (G + 1));
  l.ntrk = take(4 * (G + 1));
  l.ntow = take(4 * (G + 1));
  l.nph = take(4 * (G + 1));
  l.nnh = take(4 * (G + 1));
  l.misc = take(8 * 64);
  l.seg = take(4 * 3 * 64);
  l.cnt = take(4 * 2 * 256);
  const int gpe = words_per_event / 4, l2w = (gpe + 31) / 32;
  l.l2p = 0, l.pool = 0;
  if (!sparse) {
    l.bitmap = take(4 * (size_t)G * words_per_event);
    l.gprefix = take(2 * ((size_t)G * gpe + 1));
  } else {
    l.bitmap = take(4 * (size_t)G * l2w);
    l.l2p = take(2 * ((size_t)G * l2w + 1));
    l.pool = take(16 * (size_t)C);
    l.gprefix = take(2 * ((size_t)C + 1));
  }
  l.res = take(4 * (size_t)C);
  l.Ev = take(4 * ((size_t)C + 4));   // + 4: the bulk copy of the deposit energies starts at a 16-byte boundary
  l.Et = take(4 * (size_t)C);
  l.head = take(4 * (size_t)C);
  l.stg = take(4 * ((size_t)C + 4));  // first the keys (2 B each, + 8 for the same reason), later one float per slot
  l.ev = take(G > 1 ? (size_t)C : 0);
  l.Es = take(weighted ? 4 * (size_t)C : 0);  // reading K5
  l.total = (uint32_t)o;
  return l;
}
constexpr int T_BYTES_PER_PARTICLE = 20;  // res, Ev, Et, head, stg

// counts a[0..ne) -> exclusive prefix in place, a[ne] = total.  One warp; ne <= G_MAX = 256.
__device__ __forceinline__ void event_scan(int *a, int ne) {
  const int lane = threadIdx.x & 31;
  int v[8], sum = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int idx = lane * 8 + k;
    v[k] = idx < ne ? a[idx] : 0;
    sum += v[k];
  }
  int incl = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  const int total = __shfl_sync(0xffffffffu, incl, 31);
  __syncwarp();
  int run = incl - sum;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int idx = lane * 8 + k;
    if (idx < ne) a[idx] = run;
    run += v[k];
  }
  if (lane == 0) a[ne] = total;
}

// Block-wide exclusive prefix of per-warp totals wtot[W] (REDUX adds): returns the exclusive prefix of this
// thread's WARP and the block total.
template <int W>
__device__ __forceinline__ void warp_totals_scan(const unsigned *wtot, unsigned &excl_warp, unsigned &total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned v = lane < W ? wtot[lane] : 0u;
  total = __reduce_add_sync(0xffffffffu, v);
  excl_warp = __reduce_add_sync(0xffffffffu, lane < wid ? v : 0u);
}

__device__ __forceinline__ int popc4(const uint4 &v) { return __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w); }

// number of set bits of the 128-bit group below bit position pos (0..127)
__device__ __forceinline__ int popc_below(const uint4 &v, int pos) {
  const int w = pos >> 5;
  const uint32_t m = (1u << (pos & 31)) - 1u;
  // branch-free: words below w count in full, word w below the bit, words above not at all
  const uint32_t m0 = w > 0 ? 0xffffffffu : m, m1 = w > 1 ? 0xffffffffu : (w == 1 ? m : 0u),
                 m2 = w > 2 ? 0xffffffffu : (w == 2 ? m : 0u), m3 = w == 3 ? m : 0u;
  return __popc(v.x & m0) + __popc(v.y & m1) + __popc(v.z & m2) + __popc(v.w & m3);
}

// ---- higher card fidelity ----------------------------------------------------------------
// what S6 / S8 need of the card, by value or in shared memory (never a pointer into the kernel parameters)
struct TCard {
  const int *offset;             // [n_bins+1]
  const unsigned short *binlut;  // eta bin of tower ids 0, 32, 64, ...
  const float *w, *eta_c, *inv_cosh;
  const float *res2;             // [n_bins][6] (reading K1), only if sc.res_per_bin
  const float *edge;             // [n_bins][2] (reading K3), only if sc.smear_center
};
__device__ __forceinline__ int tower_bin(const TCard &tc, int tower) {
  int b = (int)tc.binlut[tower >> 5];
  while (tower >= tc.offset[b + 1]) ++b;
  return b;
}
// S6 of one tower with the resolutions of its eta bin (K1) and the significance cut (K2): smeared components and
// whether each is kept (reading A22: > threshold; K2: and > n_sigma sigma(E'), i.e. E'^2 > n_sigma^2 sigma^2(E'))
// var_em / var_had (K5): sigma^2 of the component's resolution at its smeared energy, with the tower's row
template <bool FID>
__device__ __forceinline__ void tower_components(const PdCardScalars &sc, const TCard &tc, int tower, float Eem, float Ehad, const uint32_t (&rn)[4],
                                                 float &em_s, float &had_s, bool &k_em, bool &k_had, float *var_em = nullptr, float *var_had = nullptr) {
  float e2[3] = {sc.ecal2[0], sc.ecal2[1], sc.ecal2[2]}, h2[3] = {sc.hcal2[0], sc.hcal2[1], sc.hcal2[2]};
  if (FID && sc.res_per_bin) {
    const float *r = tc.res2 + 6 * tower_bin(tc, tower);
    e2[0] = r[0], e2[1] = r[1], e2[2] = r[2], h2[0] = r[3], h2[1] = r[4], h2[2] = r[5];
  }
  tower_smear_csn(e2, h2, Eem, Ehad, rn, em_s, had_s);
  k_em = em_s > sc.thr_ecal, k_had = had_s > sc.thr_hcal;
  if (FID && sc.nsig2_ecal > 0.f) k_em = k_em && em_s * em_s > sc.nsig2_ecal * fmaf(e2[0] * em_s, em_s, fmaf(e2[1], em_s, e2[2]));
  if (FID && sc.nsig2_hcal > 0.f) k_had = k_had && had_s * had_s > sc.nsig2_hcal * fmaf(h2[0] * had_s, had_s, fmaf(h2[1], had_s, h2[2]));  if (FID && var_em) *var_em = fmaf(e2[0] * em_s, em_s, fmaf(e2[1], em_s, e2[2])), *var_had = fmaf(h2[0] * had_s, had_s, fmaf(h2[1], had_s, h2[2]));
}
// reading K5: the factor on the EFlow entries of the tracks of a component whose neutral is not emitted: tracks measure T with
// variance V, the calorimeter Ec (kept smeared energy; 0 = no information) with variance s2: weighted mean over T
__device__ __forceinline__ float eflow_weight(float T, float V, float Ec, float s2) {
  const float d = s2 + V;
  if (!(T > 0.f) || !(Ec > 0.f) || !(d > 0.f)) return 1.f;
  return fmaf(T, s2, Ec * V) / (d * T);
}
// exact sums of sigma_E^2: units of 2^-44 GeV^2, terms capped at 2^19 GeV^2
__device__ __forceinline__ long long var_fix(float sig) { return __float2ll_rn(fminf(sig * sig, 524288.f) * 17592186044416.f); }
constexpr float kVarUnit = 5.6843418860808015e-14f;  // 2^-44

// S8: where a tower (and its neutrals) is reported: the cell centre, or (K3) a point uniform inside the cell drawn from
// Philox stream 4 of (seed, event, tower): word 0 -> eta or theta, word 1 -> phi
template <bool FID>
__device__ __forceinline__ void tower_position(const PdCardScalars &sc, const TCard &tc, const PhiloxKeys &rk, long long event, int tower,
                                               float &eta, float &phi, float &inv_cosh) {
  const int b = tower_bin(tc, tower);
  const int j = tower - tc.offset[b];
  if (!FID || !sc.smear_center) {
    eta = tc.eta_c[b], phi = fmaf((float)j + 0.5f, tc.w[b], -kPiF), inv_cosh = tc.inv_cosh[b];
    return;
  }
  uint32_t rn[4];
  rng_block(rk, event, (uint32_t)tower, 4u, rn);
  const float lo = tc.edge[2 * b], x = fmaf(uniform24(rn[0]), tc.edge[2 * b + 1] - lo, lo);
  eta = sc.grid_theta ? -logf(tanf(0.5f * x)) : x;
  phi = fmaf((float)j + uniform24(rn[1]), tc.w[b], -kPiF);
  inv_cosh = 1.0f / coshf(eta);
}

// ---- tiles that do not fit on chip ---------------------------------------------------------------------------
// A tile of the plan (G whole events) whose particles exceed the on-chip capacity C -- one huge event, or a few large
// ones among the small ones the plan was made for -- takes this path: its events one by one, of ANY size ("no fixed
// model limit"), with the per-tower sums in a dense array of exact 64-bit fixed-point accumulators in
// the workspace (global atomics: integer, hence still order-independent and bitwise reproducible) instead of lists in
// shared memory.  Two sweeps over the tile: the first counts what every event emits, so that the tile can take its
// place in the look-back chains like any other; the second writes.  Slow (everything is computed twice, through L2)
// but exact, and it only runs for the tiles that need it.
struct BigCounts {
  int trk, tow, ph, nh;
};

// one event [pa, pb) of a big tile.  write == false: count only.  Shared memory: bmap[wpe] tower bits, wcnt[2 * wpe]
// per-word counts / prefixes, scal[8] scalars.  acc: this CTA's [n_towers][5] accumulators, all zero on entry and exit.
template <int THREADS, bool DEBUG>
__device__ __noinline__ BigCounts big_event(const PdParams &prm, long long ev_index, long long pa, long long pb, bool write,
                                            long long base_trk, long long base_tow, long long base_efl, const TCard &tc, uint32_t *bmap,
                                            unsigned *wcnt, int *scal, long long *acc) {
  constexpr int W = THREADS / 32;
  const PdCardScalars &sc = prm.sc;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  const int wpe = sc.words_per_event;
  const long long p_al = prm.p_base & ~15ll;
  unsigned long long *uacc = (unsigned long long *)acc;
  const size_t AS = (size_t)prm.acc_stride;  // 5, or 7 with the two variance sums of reading K5
  const bool weighted = sc.eflow_weighted != 0;
  for (int k = tid; k < wpe; k += THREADS) bmap[k] = 0u;
  if (tid < 8) scal[tid] = 0;
  __syncthreads();
  // deposits: tower bit + exact sum, by component
  for (long long i = pa + tid; i < pb; i += THREADS) {
    const unsigned key = (unsigned)__ldg(prm.key + (i - p_al));
    if (key != 0xffffu) {
      const int tower = (int)(key & 0x7fffu), hc = (int)(key >> 15);
      atomicOr(&bmap[tower >> 5], 1u << (tower & 31));
      atomicAdd(uacc + AS * (size_t)tower + hc, (unsigned long long)__float2ll_rn(__ldg(prm.E + i) * 4294967296.f));
      if (DEBUG) atomicMin(acc + AS * (size_t)tower + 4, i - pa - (1ll << 40));  // first depositing particle (biased: the slot starts at 0)
    }
  }
  // the event's tracks, segment by segment (warp per segment): energy into the tower's track sums; in the writing sweep
  // also into the Track collection and the EFlow collection (the event's tracks come first in both)
  {
    const long long qa = pa - p_al, qb = pb - p_al;
    const long long gs_lo = qa / PD_PSEG, gs_hi = pb > pa ? (qb - 1) / PD_PSEG : gs_lo - 1;
    int done = 0;  // tracks of earlier segments (all warps walk the segments in the same order, so each keeps the count)
    for (long long gsi = gs_lo; gsi <= gs_hi; ++gsi) {
      const uint32_t w = lane < PD_PSEG / 32 ? __ldg(prm.accmask + gsi * (PD_PSEG / 32) + lane) : 0u;
      const int lo = (int)max(qa - gsi * PD_PSEG, 0ll), hi = (int)min(qb - gsi * PD_PSEG, (long long)PD_PSEG);
      const int nlo = min(max(lo - 32 * lane, 0), 32), nhi = min(max(hi - 32 * lane, 0), 32);
      const uint32_t mlo = nlo == 32 ? 0xffffffffu : (1u << nlo) - 1u, mhi = nhi == 32 ? 0xffffffffu : (1u << nhi) - 1u;
      const int a = (int)__reduce_add_sync(0xffffffffu, (unsigned)__popc(w & mlo));
      const int c = (int)__reduce_add_sync(0xffffffffu, (unsigned)__popc(w & mhi)) - a;
      if ((int)((gsi - gs_lo) % W) == wid) {
        for (int r = lane; r < c; r += 32) {
          const long long g = gsi * PD_PSEG + a + r;
          const long long q = gsi * PD_PSEG + (long long)__ldg(prm.park_idx + g);  // the particle, relative to p_al
          const unsigned key = (unsigned)__ldg(prm.key + q);
          const float Et = __ldg(prm.park_f[3] + g);
          if (key != 0xffffu)
            atomicAdd(uacc + AS * (size_t)(key & 0x7fffu) + 2 + (key >> 15), (unsigned long long)__float2ll_rn(Et * 4294967296.f));
          if (weighted && key != 0xffffu)
            atomicAdd(uacc + AS * (size_t)(key & 0x7fffu) + 5 + (key >> 15), (unsigned long long)var_fix(__ldg(prm.park_sig + g)));
          if (write) {
            const int pid = __ldg(prm.park_pid + g);
            const float pt = __ldg(prm.park_f[0] + g), eta = __ldg(prm.park_f[1] + g), phi = __ldg(prm.park_f[2] + g);
            const unsigned o = (unsigned)base_trk + (unsigned)(done + r);
            prm.trk_src[o] = (int)(p_al + q);
            prm.trk_pid[o] = pid;
            prm.trk_charge[o] = __ldg(prm.park_q + g);
            prm.trk_pt[o] = pt, prm.trk_eta[o] = eta, prm.trk_phi[o] = phi, prm.trk_E[o] = Et;
            prm.trk_eta_out[o] = __ldg(prm.park_f[4] + g), prm.trk_phi_out[o] = __ldg(prm.park_f[5] + g);
            if (prm.imp_on) {
#pragma unroll
              for (int k4 = 0; k4 < 4; ++k4) prm.imp_out[k4][o] = __ldg(prm.park_imp[k4] + g);
            }
            const unsigned at = (unsigned)base_efl + (unsigned)(done + r);
            const int apid = pid < 0 ? -pid : pid;
            prm.efl_cls[at] = (signed char)(apid == 11 ? PD_CLS_ELECTRON : (apid == 13 ? PD_CLS_MUON : PD_CLS_CHHAD));
            prm.efl_src[at] = (int)(p_al + q);
            prm.efl_pt[at] = pt, prm.efl_eta[at] = eta, prm.efl_phi[at] = phi, prm.efl_E[at] = Et;
          }
        }
      }
      done += c;
    }
    if (tid == 0) scal[0] = done;
  }
  __threadfence();
  __syncthreads();
  const int n_trk = scal[0];
  // sweep A over the occupied towers (a thread takes whole bitmap words, ascending ids inside): sums -> smear ->
  // thresholds -> EFlow subtraction, exactly as pass W; the results are stashed in the tower's accumulators
  for (int w = tid; w < wpe; w += THREADS) {
    uint32_t m = bmap[w];
    unsigned c_tw = 0, c_ph = 0, c_nh = 0;
    while (m) {
      const int b = __ffs(m) - 1;
      m &= m - 1;
      const int tower = 32 * w + b;
      long long *a5 = acc + AS * (size_t)tower;
      const long long a_em = __ldcg(a5), a_had = __ldcg(a5 + 1), t_em = __ldcg(a5 + 2), t_had = __ldcg(a5 + 3);
      const float Eem = (float)a_em * 2.3283064365386963e-10f, Ehad = (float)a_had * 2.3283064365386963e-10f;
      const float Tem = (float)t_em * 2.3283064365386963e-10f, Thad = (float)t_had * 2.3283064365386963e-10f;
      uint32_t rn[4];
      rng_block(prm.rk, ev_index, (uint32_t)tower, 1u, rn);
      float em_s, had_s;
      bool k_em, k_had;
      float var_em = 0.f, var_had = 0.f;
      tower_components<true>(sc, tc, tower, Eem, Ehad, rn, em_s, had_s, k_em, k_had, weighted ? &var_em : nullptr, &var_had);
      const float em_f = k_em ? em_s : 0.f, had_f = k_had ? had_s : 0.f;
      float n_em = em_f - Tem, n_had = had_f - Thad;
      const bool f_ph = n_em > sc.thr_ecal, f_nh = n_had > sc.thr_hcal, f_tw = em_f + had_f > 0.f;
      if (weighted) {
        // reading K5: where the neutral is not emitted the stashed value is the factor for the component's tracks
        if (!f_ph) n_em = eflow_weight(Tem, (float)__ldcg(a5 + 5) * kVarUnit, em_f, var_em);
        if (!f_nh) n_had = eflow_weight(Thad, (float)__ldcg(a5 + 6) * kVarUnit, had_f, var_had);
        __stcg(a5 + 5, 0ll), __stcg(a5 + 6, 0ll);
      }
      c_tw += f_tw, c_ph += f_ph, c_nh += f_nh;
      if (DEBUG && write) {
        const long long g = pa + (__ldcg(a5 + 4) + (1ll << 40));
        if (prm.dbg_tw_first) prm.dbg_tw_first[g] = 1;
        if (prm.dbg_tw[0]) prm.dbg_tw[0][g] = Eem;
        if (prm.dbg_tw[1]) prm.dbg_tw[1][g] = Ehad;
        if (prm.dbg_tw[2]) prm.dbg_tw[2][g] = Tem;
        if (prm.dbg_tw[3]) prm.dbg_tw[3][g] = Thad;
        if (prm.dbg_tw[4]) prm.dbg_tw[4][g] = em_s;
        if (prm.dbg_tw[5]) prm.dbg_tw[5][g] = had_s;
        if (prm.dbg_tw_dec)
          prm.dbg_tw_dec[g] = (unsigned char)((k_em ? PD_DEC_EEM : 0) | (k_had ? PD_DEC_EHAD : 0) | (f_ph ? PD_DEC_NEM : 0) | (f_nh ? PD_DEC_NHAD : 0));
      }
      if (write) {
        __stcg(a5, (long long)(((unsigned long long)__float_as_uint(had_f) << 32) | __float_as_uint(em_f)));
        __stcg(a5 + 1, (long long)(((unsigned long long)__float_as_uint(n_had) << 32) | __float_as_uint(n_em)));
        __stcg(a5 + 2, (long long)((f_tw ? 1 : 0) | (f_ph ? 2 : 0) | (f_nh ? 4 : 0)));
      } else {
        __stcg(a5, 0ll), __stcg(a5 + 1, 0ll), __stcg(a5 + 2, 0ll), __stcg(a5 + 3, 0ll), __stcg(a5 + 4, 0ll);
      }
    }
    wcnt[w] = c_tw | (c_ph << 16), wcnt[wpe + w] = c_nh;
    if (c_tw) atomicAdd(&scal[1], (int)c_tw);
    if (c_ph) atomicAdd(&scal[2], (int)c_ph);
    if (c_nh) atomicAdd(&scal[3], (int)c_nh);
  }
  __syncthreads();
  BigCounts out;
  out.trk = n_trk, out.tow = scal[1], out.ph = scal[2], out.nh = scal[3];
  if (!write) return out;
  if (weighted) {
    // reading K5: the EFlow entries of the event's tracks (written above, in track order from base_efl) take the factor of
    // their tower component, stashed by sweep A where the component's neutral is not emitted
    __threadfence();
    const long long qa = pa - p_al, qb = pb - p_al;
    const long long gs_lo = qa / PD_PSEG, gs_hi = pb > pa ? (qb - 1) / PD_PSEG : gs_lo - 1;
    int done = 0;
    for (long long gsi = gs_lo; gsi <= gs_hi; ++gsi) {
      const uint32_t w = lane < PD_PSEG / 32 ? __ldg(prm.accmask + gsi * (PD_PSEG / 32) + lane) : 0u;
      const int lo = (int)max(qa - gsi * PD_PSEG, 0ll), hi = (int)min(qb - gsi * PD_PSEG, (long long)PD_PSEG);
      const int nlo = min(max(lo - 32 * lane, 0), 32), nhi = min(max(hi - 32 * lane, 0), 32);
      const uint32_t mlo = nlo == 32 ? 0xffffffffu : (1u << nlo) - 1u, mhi = nhi == 32 ? 0xffffffffu : (1u << nhi) - 1u;
      const int a = (int)__reduce_add_sync(0xffffffffu, (unsigned)__popc(w & mlo));
      const int c = (int)__reduce_add_sync(0xffffffffu, (unsigned)__popc(w & mhi)) - a;
      if ((int)((gsi - gs_lo) % W) == wid) {
        for (int r = lane; r < c; r += 32) {
          const long long g = gsi * PD_PSEG + a + r;
          const long long q = gsi * PD_PSEG + (long long)__ldg(prm.park_idx + g);
          const unsigned key = (unsigned)__ldg(prm.key + q);
          if (key == 0xffffu) continue;
          const long long *a5 = acc + AS * (size_t)(key & 0x7fffu);
          const unsigned long long v1 = (unsigned long long)__ldcg(a5 + 1);
          const int flags = (int)__ldcg(a5 + 2);
          const float fw = (key & 0x8000u) ? ((flags & 4) ? 1.f : __uint_as_float((unsigned)(v1 >> 32))) : ((flags & 2) ? 1.f : __uint_as_float((unsigned)v1));
          const unsigned at = (unsigned)base_efl + (unsigned)(done + r);
          prm.efl_pt[at] *= fw, prm.efl_E[at] *= fw;
        }
      }
      done += c;
    }
    __threadfence();
    __syncthreads();
  }
  // exclusive prefix of the per-word counts (one warp, a run of words per lane)
  if (wid == 0) {
    const int chunk = (wpe + 31) / 32, lo = min(wpe, lane * chunk), hi = min(wpe, lo + chunk);
    unsigned sa = 0, sb = 0;
    for (int k = lo; k < hi; ++k) sa += wcnt[k], sb += wcnt[wpe + k];
    unsigned ra = warp_incl_scan(sa) - sa, rb = warp_incl_scan(sb) - sb;
    for (int k = lo; k < hi; ++k) {
      const unsigned ta = wcnt[k], tb = wcnt[wpe + k];
      wcnt[k] = ra, wcnt[wpe + k] = rb;
      ra += ta, rb += tb;
    }
  }
  __syncthreads();
  // sweep B: the ordered outputs of the event
  const unsigned b_ph = (unsigned)base_efl + (unsigned)n_trk, b_nh = b_ph + (unsigned)out.ph;
  for (int w = tid; w < wpe; w += THREADS) {
    uint32_t m = bmap[w];
    unsigned k_tw = (unsigned)base_tow + (wcnt[w] & 0xffffu), k_ph = b_ph + (wcnt[w] >> 16), k_nh = b_nh + wcnt[wpe + w];
    while (m) {
      const int b = __ffs(m) - 1;
      m &= m - 1;
      const int tower = 32 * w + b;
      long long *a5 = acc + AS * (size_t)tower;
      const unsigned long long v0 = (unsigned long long)__ldcg(a5), v1 = (unsigned long long)__ldcg(a5 + 1);
      const int flags = (int)__ldcg(a5 + 2);
      __stcg(a5, 0ll), __stcg(a5 + 1, 0ll), __stcg(a5 + 2, 0ll), __stcg(a5 + 3, 0ll), __stcg(a5 + 4, 0ll);
      if (!flags) continue;
      const float em = __uint_as_float((unsigned)v0), had = __uint_as_float((unsigned)(v0 >> 32));
      const float nem = __uint_as_float((unsigned)v1), nhad = __uint_as_float((unsigned)(v1 >> 32));
      float eta_c, phi_c, ic;
      tower_position<true>(sc, tc, prm.rk, ev_index, tower, eta_c, phi_c, ic);
      if (flags & 1) {
        const unsigned at = k_tw++;
        prm.tow_tower[at] = tower, prm.tow_eta[at] = eta_c, prm.tow_phi[at] = phi_c;
        prm.tow_E[at] = em + had, prm.tow_Eem[at] = em, prm.tow_Ehad[at] = had, prm.tow_ET[at] = (em + had) * ic;
      }
      if (flags & 2) {
        const unsigned at = k_ph++;
        prm.efl_cls[at] = (signed char)PD_CLS_PHOTON, prm.efl_src[at] = tower;
        prm.efl_pt[at] = nem * ic, prm.efl_eta[at] = eta_c, prm.efl_phi[at] = phi_c, prm.efl_E[at] = nem;
      }
      if (flags & 4) {
        const unsigned at = k_nh++;
        prm.efl_cls[at] = (signed char)PD_CLS_NEUHAD, prm.efl_src[at] = tower;
        prm.efl_pt[at] = nhad * ic, prm.efl_eta[at] = eta_c, prm.efl_phi[at] = phi_c, prm.efl_E[at] = nhad;
      }
    }
  }
  __threadfence();
  __syncthreads();
  (void)lt_mask;
  return out;
}

// a whole tile through big_event: count sweep, the tile's place in both look-back chains, write sweep
template <int THREADS, bool DEBUG>
__device__ __noinline__ void big_tile(const PdParams &prm, unsigned char *smem, int tile, long long e0, int ne, long long p0, long long p1,
                                      bool acc_ready) {
  const PdCardScalars &sc = prm.sc;
  const PdTLayout &L = prm.lay;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const TCard tc{(const int *)(smem + L.offset), (const unsigned short *)(smem + L.binlut), (const float *)(smem + L.w),
                 (const float *)(smem + L.eta_c), (const float *)(smem + L.inv_cosh), (const float *)(smem + L.res2), (const float *)(smem + L.edge)};
  int *s_ntrk = (int *)(smem + L.ntrk), *s_ntow = (int *)(smem + L.ntow), *s_nph = (int *)(smem + L.nph), *s_nnh = (int *)(smem + L.nnh);
  unsigned long long *s_misc = (unsigned long long *)(smem + L.misc);
  unsigned *s_wtot = (unsigned *)(s_misc + 8);
  uint32_t *s_res = (uint32_t *)(smem + L.res);
  unsigned *s_head = (unsigned *)(smem + L.head);
  {
      uint32_t *bmap = s_res;
      unsigned *wcnt = s_head;
      int *scal = (int *)s_wtot;
      long long *acc = prm.big_acc + (size_t)blockIdx.x * (size_t)prm.acc_stride * (size_t)sc.n_towers;
      if (!acc_ready) {
        for (size_t k = tid; k < (size_t)prm.acc_stride * (size_t)sc.n_towers; k += THREADS) __stcg(acc + k, 0ll);
        __threadfence();
        __syncthreads();
      }
      for (int e = 0; e < ne; ++e) {
        const BigCounts c = big_event<THREADS, DEBUG>(prm, prm.event_base + e0 + e, prm.offsets[e0 + e], prm.offsets[e0 + e + 1], false, 0, 0, 0,
                                                      tc, bmap, wcnt, scal, acc);
        if (tid == 0) s_ntrk[e] = c.trk, s_ntow[e] = c.tow, s_nph[e] = c.ph, s_nnh[e] = c.nh;
        __syncthreads();
      }
      if (wid == 1) event_scan(s_ntrk, ne);
      else if (wid == 2) event_scan(s_ntow, ne);
      else if (wid == 3) event_scan(s_nph, ne);
      else if (wid == 4) event_scan(s_nnh, ne);
      __syncthreads();
      if (wid == 0) {
        const unsigned long long n_t = (unsigned long long)s_ntrk[ne];
        const unsigned long long agg = (unsigned long long)s_ntow[ne] | ((unsigned long long)(s_nph[ne] + s_nnh[ne]) << 31);
        if (lane == 0) chain_publish(prm.chain_t, tile, n_t), chain_publish(prm.chain, tile, agg);
        const unsigned long long ext = chain_resolve<8>(prm.chain_t, tile, n_t);
        const unsigned long long exw = chain_resolve<8>(prm.chain, tile, agg);
        if (lane == 0) s_misc[1] = ext, s_misc[2] = exw;
      }
      __syncthreads();
      const long long bt = (long long)s_misc[1], bw = (long long)(s_misc[2] & FIELD_MASK);
      const long long bf = bt + (long long)((s_misc[2] >> 31) & FIELD_MASK);
      for (int e = tid; e < ne; e += THREADS) {
        prm.trk_offsets[e0 + e + 1] = bt + s_ntrk[e + 1];
        prm.tow_offsets[e0 + e + 1] = bw + s_ntow[e + 1];
        prm.efl_offsets[e0 + e + 1] = bf + s_ntrk[e + 1] + s_nph[e + 1] + s_nnh[e + 1];
      }
      if (tile == 0 && tid == 0) prm.trk_offsets[0] = 0, prm.tow_offsets[0] = 0, prm.efl_offsets[0] = 0;
      if (DEBUG && prm.dbg_tw_first)
        for (long long i = p0 + tid; i < p1; i += THREADS) prm.dbg_tw_first[i] = 0;
      __syncthreads();
      for (int e = 0; e < ne; ++e) {
        const int kt = s_ntrk[e], kw = s_ntow[e], kp = s_nph[e], kn = s_nnh[e];
        __syncthreads();  // the scalars above are read before big_event reuses shared memory next to them
        big_event<THREADS, DEBUG>(prm, prm.event_base + e0 + e, prm.offsets[e0 + e], prm.offsets[e0 + e + 1], true, bt + kt, bw + kw,
                                  bf + kt + kp + kn, tc, bmap, wcnt, scal, acc);
      }
  }
}

template <int THREADS, int CTAS, bool DEBUG, bool SPARSE, bool FID>
__global__ void __launch_bounds__(THREADS, CTAS) pd_tower_kernel(const __grid_constant__ PdParams prm) {
  constexpr int W = THREADS / 32;
  extern __shared__ __align__(16) unsigned char smem[];
  const PdCardScalars &sc = prm.sc;
  const int nb = sc.n_bins;
  const int C = prm.capacity, G = prm.events_per_tile;
  const int wpe = sc.words_per_event, gpe = wpe >> 2;
  constexpr bool sparse = SPARSE;   // two-level tower bitmap, chosen by pd_plan (prm.sparse)
  const int l2w = (gpe + 31) >> 5;  // words of the per-event group bitmap (sparse mode)
  const Layout &L = prm.lay;
  int *s_offset = (int *)(smem + L.offset);
  float *s_w = (float *)(smem + L.w);
  float *s_eta_c = (float *)(smem + L.eta_c);
  float *s_inv_cosh = (float *)(smem + L.inv_cosh);
  unsigned short *s_binlut = (unsigned short *)(smem + L.binlut);
  float *s_res2 = (float *)(smem + L.res2), *s_edge = (float *)(smem + L.edge);
  const TCard tc{s_offset, s_binlut, s_w, s_eta_c, s_inv_cosh, s_res2, s_edge};
  int *s_off32 = (int *)(smem + L.off32);
  int *s_ntrk = (int *)(smem + L.ntrk);  // tracks of the tile before event e
  int *s_ntow = (int *)(smem + L.ntow);
  int *s_nph = (int *)(smem + L.nph);
  int *s_nnh = (int *)(smem + L.nnh);
  unsigned long long *s_misc = (unsigned long long *)(smem + L.misc);
  unsigned *s_wtot = (unsigned *)(s_misc + 8);    // [32] per-warp totals of scan 1
  unsigned *s_preA = (unsigned *)(smem + L.cnt);  // per (iteration, warp) of pass W: towers | photons << 16 ...
  unsigned *s_preB = s_preA + 256;                // ... and neutral hadrons (counts, then exclusive prefixes)
  uint32_t *s_bitmap = (uint32_t *)(smem + L.bitmap);
  unsigned short *s_gp = (unsigned short *)(smem + L.gprefix);
  unsigned short *s_l2p = (unsigned short *)(smem + L.l2p);  // sparse mode: rank of the first non-empty group of a word
  uint4 *s_pool = (uint4 *)(smem + L.pool);                  // sparse mode: tower bits of the non-empty groups
  uint32_t *s_res = (uint32_t *)(smem + L.res);
  float *s_Ev_raw = (float *)(smem + L.Ev);  // deposit energy; after pass W, at the head particle: Ehad''
  float *s_Et = (float *)(smem + L.Et);     // track energy of accepted tracks; after pass W, at the head: photon energy
  unsigned *s_head = (unsigned *)(smem + L.head);  // per slot: last pusher, then head | tower id << 13 | flags
  float *s_stg = (float *)(smem + L.stg);   // per slot after pass W: Eem''  (neutral-hadron energy goes to s_res[head])
  unsigned char *s_ev = smem + L.ev;
  float *s_Es = (float *)(smem + L.Es);     // K5: sigma_E of an accepted track, at its particle
  const bool weighted = FID && sc.eflow_weighted;
  uint64_t *s_bar = (uint64_t *)(s_misc + 4);
  // kernel P parked the accepted tracks compacted within SEGMENTS of PD_PSEG particles; per segment that overlaps the
  // tile: rank of the tile's first track in the segment, number of the tile's tracks in it, their exclusive prefix
  int *s_sega = (int *)(smem + L.seg), *s_segc = s_sega + 64, *s_segp = s_segc + 64;

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;

  for (int i = tid; i <= nb; i += THREADS) s_offset[i] = prm.tab.offset[i];
  for (int i = tid; i < nb; i += THREADS) {
    s_w[i] = prm.tab.w[i];
    s_eta_c[i] = prm.tab.eta_c[i];
    s_inv_cosh[i] = prm.tab.inv_cosh[i];
  }
  if (sc.res_per_bin)
    for (int i = tid; i < 6 * nb; i += THREADS) s_res2[i] = prm.tab.res2[i];
  if (sc.smear_center)
    for (int i = tid; i < 2 * nb; i += THREADS) s_edge[i] = prm.tab.edge[i];
  __syncthreads();
  // eta bin of tower ids 0, 32, 64, ...: start of the short forward search of pass O
  for (int c = tid; c <= (sc.n_towers >> 5); c += THREADS) {
    const int id = c << 5;
    int lo = 0, hi = nb;
    while (hi - lo > 1) {
      const int mid = (lo + hi) >> 1;
      if (s_offset[mid] <= id) lo = mid;
      else hi = mid;
    }
    s_binlut[c] = (unsigned short)lo;
  }
  if (tid == 0) {
    mbar_init(s_bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  uint32_t phase = 0;
  bool acc_ready = false;  // the accumulators of the big-tile path are cleared when a CTA first needs them
  const long long p_al = prm.p_base & ~15ll;  // the key of particle p sits at key[p - p_al]

  for (;;) {
    __syncthreads();  // previous tile fully done with shared memory (and card tables staged)
    if (tid == 0) s_misc[0] = atomicAdd(prm.tile_counter, 1u);
    __syncthreads();
    const int tile = (int)s_misc[0];
    if (tile >= prm.n_tiles) break;
    const long long e0 = (long long)tile * G;
    const int ne = (int)min((long long)G, prm.n_events - e0);
    const bool multi = G > 1;
    const long long p0 = prm.offsets[e0];
    const long long p1 = prm.offsets[e0 + ne];
    if ((p1 - p0) > (long long)C) {
      // the tile does not fit on chip: its events one by one through the accumulators in the workspace
      big_tile<THREADS, DEBUG>(prm, smem, tile, e0, ne, p0, p1, acc_ready);
      acc_ready = true;
      continue;
    }
    const int n = (int)(p1 - p0);
    // the tile's deposit energies and keys arrive by bulk copies (one thread; completion on the mbarrier) while the
    // CTA sets up the tile: 16-byte aligned start, whole 16-byte pieces; the few elements behind them by plain loads
    const int shE = (int)(p0 & 3), shK = (int)((p0 - p_al) & 7);
    const int nbE = prm.tma_ok ? ((shE + n) & ~3) : 0, nbK = prm.tma_ok ? ((shK + n) & ~7) : 0;
    float *s_Ev = s_Ev_raw + shE;
    const unsigned short *s_key = (const unsigned short *)s_stg + shK;
    const bool bulk = nbE > 0 || nbK > 0;
    if (tid == 0 && bulk) {
      fence_async_smem();  // the slots were last written through the generic proxy
      mbar_expect_tx(s_bar, 4u * nbE + 2u * nbK);
      if (nbE > 0) bulk_g2s(s_Ev_raw, prm.E + (p0 - shE), 4u * nbE, s_bar);
      if (nbK > 0) bulk_g2s(s_stg, prm.key + (p0 - p_al - shK), 2u * nbK, s_bar);
    }
    for (int i = nbE - shE + tid; i < n; i += THREADS) s_Ev[i] = __ldg(prm.E + p0 + i);
    for (int i = nbK - shK + tid; i < n; i += THREADS) ((unsigned short *)s_stg)[shK + i] = __ldg(prm.key + (p0 - p_al) + i);
    for (int e = tid; e <= ne; e += THREADS) {
      s_off32[e] = (int)(prm.offsets[e0 + e] - p0);
      s_ntrk[e] = 0, s_ntow[e] = 0, s_nph[e] = 0, s_nnh[e] = 0;
    }
    // the tile's tracks, segment by segment (warp per segment): from the accepted bits kernel P left
    const long long q0 = p0 - p_al;  // the tile's first particle in the parking arrays
    const long long gseg_lo = q0 / PD_PSEG;
    const int n_seg = n > 0 ? (int)((q0 + n - 1) / PD_PSEG - gseg_lo) + 1 : 0;
    for (int k = wid; k < n_seg; k += W) {
      const long long gs = gseg_lo + k;
      const uint32_t w = lane < PD_PSEG / 32 ? __ldg(prm.accmask + gs * (PD_PSEG / 32) + lane) : 0u;
      const int lo = (int)max(q0 - gs * PD_PSEG, 0ll), hi = (int)min(q0 + n - gs * PD_PSEG, (long long)PD_PSEG);
      const int nlo = min(max(lo - 32 * lane, 0), 32), nhi = min(max(hi - 32 * lane, 0), 32);
      const uint32_t mlo = nlo == 32 ? 0xffffffffu : (1u << nlo) - 1u, mhi = nhi == 32 ? 0xffffffffu : (1u << nhi) - 1u;
      const int a = (int)__reduce_add_sync(0xffffffffu, (unsigned)__popc(w & mlo));
      const int b = (int)__reduce_add_sync(0xffffffffu, (unsigned)__popc(w & mhi));
      if (lane == 0) s_sega[k] = a, s_segc[k] = b - a;
    }
    const int NG = ne * gpe;  // 128-tower bitmap groups of the tile
    const int NW = ne * l2w;  // sparse mode: words of the group bitmaps
    if (!sparse) {
      for (int k = tid; k < NG; k += THREADS) ((uint4 *)s_bitmap)[k] = make_uint4(0u, 0u, 0u, 0u);
    } else {
      for (int k = tid; k < NW; k += THREADS) s_bitmap[k] = 0u;
    }
    __syncthreads();
    if (wid == 0) {
      // exclusive prefix of the segments' track counts (<= 64 segments: two per lane); the tile's total goes on chain T
      // at once: nobody will ever wait for it
      const int c0 = 2 * lane < n_seg ? s_segc[2 * lane] : 0, c1 = 2 * lane + 1 < n_seg ? s_segc[2 * lane + 1] : 0;
      const int incl = (int)warp_incl_scan((unsigned)(c0 + c1));
      if (2 * lane < n_seg) s_segp[2 * lane] = incl - c0 - c1;
      if (2 * lane + 1 < n_seg) s_segp[2 * lane + 1] = incl - c1;
      const int total = __shfl_sync(0xffffffffu, incl, 31);
      if (lane == 0) {
        s_misc[5] = (unsigned long long)total;
        chain_publish(prm.chain_t, tile, (unsigned long long)total);
        if (!multi) s_ntrk[1] = total;
      }
    }
    if (multi) {
      // event index of every particle of the tile: warp per event, lanes over its particles
      for (int e = wid; e < ne; e += W)
        for (int i = s_off32[e] + lane; i < s_off32[e + 1]; i += 32) s_ev[i] = (unsigned char)e;
      __syncthreads();
    }

    // ------------------------------------------------------------------ pass A': keys (deposit energies are in place)
    if (bulk) mbar_wait(s_bar, phase), phase ^= 1u;
    for (int i = tid; i < n; i += THREADS) {
      const unsigned key = s_key[i];
      uint32_t res = RES_TOWER | (LINK_END << RES_LINK_SHIFT);
      if (key != 0xffffu) {
        const int tower = (int)(key & 0x7fffu);
        const int e = multi ? (int)s_ev[i] : 0;
        res = (uint32_t)tower | (LINK_END << RES_LINK_SHIFT) | RES_DEP | ((key & 0x8000u) ? RES_HCAL : 0u);
        if (!sparse) atomicOr(&s_bitmap[e * wpe + (tower >> 5)], 1u << (tower & 31));
        else atomicOr(&s_bitmap[e * l2w + (tower >> 12)], 1u << ((tower >> 7) & 31));  // its 128-tower group
      }
      s_res[i] = res;
      s_head[i] = 0xffffffffu;
      if (DEBUG && prm.dbg_tw_first) prm.dbg_tw_first[p0 + i] = 0;
    }
    __syncthreads();

    // ------------------------------------------------------------------ scan 1: tower slots; track energies
    // Each thread owns a contiguous chunk of bitmap groups (odd chunk lengths keep the shared-memory accesses of a
    // warp on distinct banks).
    int n_slots;
    {
      // dense: the groups' tower bits; sparse: the words of the group bitmaps (their bits = non-empty groups)
      const int NS = sparse ? NW : NG;
      const int kg = ((NS + THREADS - 1) / THREADS) | 1;
      const int g0 = min(NS, tid * kg), g1 = min(NS, g0 + kg);
      unsigned cnt_g = 0;
      if (!sparse) {
        for (int g = g0; g < g1; ++g) cnt_g += (unsigned)popc4(((const uint4 *)s_bitmap)[g]);
      } else {
        for (int g = g0; g < g1; ++g) cnt_g += (unsigned)__popc(s_bitmap[g]);
      }
      const unsigned incl = warp_incl_scan(cnt_g);
      if (lane == 31) s_wtot[wid] = incl;
      // the tile's accepted tracks: their energy goes to their particle (pass W subtracts it from the tower)
      for (int k = wid; k < n_seg; k += W) {
        const long long gs = (gseg_lo + k) * PD_PSEG;
        const int a = s_sega[k], c = s_segc[k];
        for (int r = lane; r < c; r += 32) {
          const long long g = gs + a + r;
          const int i = (int)(gs + (long long)__ldg(prm.park_idx + g) - q0);
          s_Et[i] = __ldg(prm.park_f[3] + g);
          if (weighted) s_Es[i] = __ldg(prm.park_sig + g);
          s_res[i] |= RES_ACC;
          if (multi) atomicAdd(&s_ntrk[(int)s_ev[i]], 1);
        }
      }
      __syncthreads();
      unsigned excl_w, tot;
      warp_totals_scan<W>(s_wtot, excl_w, tot);
      int rg = (int)(excl_w + incl - cnt_g);
      if (!sparse) {
        for (int g = g0; g < g1; ++g) {
          s_gp[g] = (unsigned short)rg;
          rg += popc4(((const uint4 *)s_bitmap)[g]);
        }
      } else {
        for (int g = g0; g < g1; ++g) {
          s_l2p[g] = (unsigned short)rg;
          rg += __popc(s_bitmap[g]);
        }
      }
      n_slots = (int)tot;
    }
    __syncthreads();
    if (sparse) {
      // ---- sparse mode: n_slots is so far the number of NON-EMPTY GROUPS (<= deposits <= C).  Their tower bits go
      // into the pool, at the rank of the group in (event, group) order; a second scan turns them into slots.
      const int n_groups = n_slots;
      for (int k = tid; k < n_groups; k += THREADS) s_pool[k] = make_uint4(0u, 0u, 0u, 0u);
      __syncthreads();
      for (int i = tid; i < n; i += THREADS) {
        const uint32_t r = s_res[i];
        if (r & RES_DEP) {
          const int id = (int)(r & RES_TOWER);
          const int w = (multi ? (int)s_ev[i] * l2w : 0) + (id >> 12);
          const int pg = (int)s_l2p[w] + __popc(s_bitmap[w] & ((1u << ((id >> 7) & 31)) - 1u));
          atomicOr(&((uint32_t *)s_pool)[4 * pg + ((id >> 5) & 3)], 1u << (id & 31));
        }
      }
      __syncthreads();
      const int kp = ((n_groups + THREADS - 1) / THREADS) | 1;
      const int q0 = min(n_groups, tid * kp), q1 = min(n_groups, q0 + kp);
      unsigned cnt_p = 0;
      for (int g = q0; g < q1; ++g) cnt_p += (unsigned)popc4(s_pool[g]);
      const unsigned incl_p = warp_incl_scan(cnt_p);
      if (lane == 31) s_wtot[wid] = incl_p;
      __syncthreads();
      unsigned excl_wp, tot_p;
      warp_totals_scan<W>(s_wtot, excl_wp, tot_p);
      int rp = (int)(excl_wp + incl_p - cnt_p);
      for (int g = q0; g < q1; ++g) {
        s_gp[g] = (unsigned short)rp;
        rp += popc4(s_pool[g]);
      }
      n_slots = (int)tot_p;
      __syncthreads();
    }

    // ------------------------------------------------------------------ pass B (S5): every deposit finds its
    // tower's slot and pushes itself on the slot's list
    for (int i = tid; i < n; i += THREADS) {
      const uint32_t r = s_res[i];
      if (r & RES_DEP) {
        const int id = (int)(r & RES_TOWER);
        int g;
        uint4 bits;
        if (!sparse) {
          g = (multi ? (int)s_ev[i] * gpe : 0) + (id >> 7);
          bits = ((const uint4 *)s_bitmap)[g];
        } else {
          const int w = (multi ? (int)s_ev[i] * l2w : 0) + (id >> 12);
          g = (int)s_l2p[w] + __popc(s_bitmap[w] & ((1u << ((id >> 7) & 31)) - 1u));
          bits = s_pool[g];
        }
        const int slot = (int)s_gp[g] + popc_below(bits, id & 127);
        const unsigned prev = atomicExch(&s_head[slot], (unsigned)i);
        s_res[i] = (r & ~(LINK_END << RES_LINK_SHIFT)) | ((prev & LINK_END) << RES_LINK_SHIFT);
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ pass W: S5-S7, one thread per tower
    const int n_it = (n_slots + THREADS - 1) / THREADS;  // <= C_MAX / THREADS + 1, so n_it * W <= 256
    for (int it = 0; it < n_it; ++it) {
      const int d = it * THREADS + tid;
      bool f_tw = false, f_ph = false, f_nh = false;
      if (d < n_slots) {
        const int h = (int)(s_head[d] & LINK_END);
        const uint32_t rh = s_res[h];
        const int tower = (int)(rh & RES_TOWER);
        const int e = multi ? (int)s_ev[h] : 0;
        // S5: exact fixed-point sums (units of 2^-32 GeV, 64-bit integers) over the slot's list.  Integer
        // addition is associative, so the sums do not depend on the order in which the deposits arrived:
        // bitwise reproducible, and closer to the fp64 definition than a sequential fp32 sum.
        long long a_em = 0, a_had = 0, t_em = 0, t_had = 0, v_em = 0, v_had = 0;
        int first = h;
        for (int c = h;;) {
          const uint32_t rc = c == h ? rh : s_res[c];
          const long long Ev = __float2ll_rn(s_Ev[c] * 4294967296.f);
          const long long Tv = (rc & RES_ACC) ? __float2ll_rn(s_Et[c] * 4294967296.f) : 0ll;
          if (rc & RES_HCAL) a_had += Ev, t_had += Tv;
          else a_em += Ev, t_em += Tv;
          if (weighted && (rc & RES_ACC)) {  // K5: the variance of the component's track sum (exact, like the sums)
            if (rc & RES_HCAL) v_had += var_fix(s_Es[c]);
            else v_em += var_fix(s_Es[c]);
          }
          first = min(first, c);
          c = (int)(rc >> RES_LINK_SHIFT);
          if (c == (int)LINK_END) break;
        }
        const float Eem = (float)a_em * 2.3283064365386963e-10f, Ehad = (float)a_had * 2.3283064365386963e-10f;
        const float Tem = (float)t_em * 2.3283064365386963e-10f, Thad = (float)t_had * 2.3283064365386963e-10f;
        uint32_t rn[4];
        rng_block(prm.rk, prm.event_base + e0 + e, (uint32_t)tower, 1u, rn);
        float em_s, had_s;
        bool k_em, k_had;
        // reading A22: the threshold is applied twice, strictly, per component (K1 / K2: per-bin resolutions, significance)
        float var_em = 0.f, var_had = 0.f;
        tower_components<FID>(sc, tc, tower, Eem, Ehad, rn, em_s, had_s, k_em, k_had, weighted ? &var_em : nullptr, &var_had);
        const float em_f = k_em ? em_s : 0.f, had_f = k_had ? had_s : 0.f;
        float n_em = em_f - Tem, n_had = had_f - Thad;
        f_ph = n_em > sc.thr_ecal, f_nh = n_had > sc.thr_hcal;
        if (weighted) {
          // reading K5: where the neutral is not emitted the staged value is the factor for the component's tracks instead
          if (!f_ph) n_em = eflow_weight(Tem, (float)v_em * kVarUnit, em_f, var_em);
          if (!f_nh) n_had = eflow_weight(Thad, (float)v_had * kVarUnit, had_f, var_had);
        }
        f_tw = em_f + had_f > 0.f;
        if (multi) {
          if (f_tw) atomicAdd(&s_ntow[e], 1);
          if (f_ph) atomicAdd(&s_nph[e], 1);
          if (f_nh) atomicAdd(&s_nnh[e], 1);
        }
        // stage the tower: per slot and at its head particle's index (only this thread ever touches that particle
        // again); pass O takes the decisions from the flags, not from the staged values
        s_stg[d] = em_f, s_Ev[h] = had_f, s_Et[h] = n_em;
        s_res[h] = __float_as_uint(n_had);
        s_head[d] = (unsigned)h | ((unsigned)tower << 13) | (f_tw ? SLOT_TW : 0u) | (f_ph ? SLOT_PH : 0u) | (f_nh ? SLOT_NH : 0u);
        if (DEBUG) {
          const long long g = p0 + first;
          if (prm.dbg_tw_first) prm.dbg_tw_first[g] = 1;
          if (prm.dbg_tw[0]) prm.dbg_tw[0][g] = Eem;
          if (prm.dbg_tw[1]) prm.dbg_tw[1][g] = Ehad;
          if (prm.dbg_tw[2]) prm.dbg_tw[2][g] = Tem;
          if (prm.dbg_tw[3]) prm.dbg_tw[3][g] = Thad;
          if (prm.dbg_tw[4]) prm.dbg_tw[4][g] = em_s;
          if (prm.dbg_tw[5]) prm.dbg_tw[5][g] = had_s;
          if (prm.dbg_tw_dec)
            prm.dbg_tw_dec[g] = (unsigned char)((k_em ? PD_DEC_EEM : 0) | (k_had ? PD_DEC_EHAD : 0) |
                                                (f_ph ? PD_DEC_NEM : 0) | (f_nh ? PD_DEC_NHAD : 0));
        }
      }
      // counts of this warp's 32 slots; scanned over all (iteration, warp) pairs below = slot order
      const unsigned m_tw = __ballot_sync(0xffffffffu, f_tw), m_ph = __ballot_sync(0xffffffffu, f_ph),
                     m_nh = __ballot_sync(0xffffffffu, f_nh);
      if (lane == 0) {
        s_preA[it * W + wid] = (unsigned)__popc(m_tw) | ((unsigned)__popc(m_ph) << 16);
        s_preB[it * W + wid] = (unsigned)__popc(m_nh);
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ scan W + chain W (towers | neutrals)
    if (wid == 0) {
      // exclusive prefix over the <= 256 (iteration, warp) counts: eight consecutive entries per lane
      const int n_ent = n_it * W;
      unsigned va[8], vb[8], sa = 0, sb = 0;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const int idx = lane * 8 + k;
        va[k] = idx < n_ent ? s_preA[idx] : 0u;
        vb[k] = idx < n_ent ? s_preB[idx] : 0u;
        sa += va[k], sb += vb[k];
      }
      const unsigned ia = warp_incl_scan(sa), ib = warp_incl_scan(sb);
      const unsigned ta = __shfl_sync(0xffffffffu, ia, 31), tb = __shfl_sync(0xffffffffu, ib, 31);
      unsigned ra = ia - sa, rb = ib - sb;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const int idx = lane * 8 + k;
        if (idx < n_ent) s_preA[idx] = ra, s_preB[idx] = rb;
        ra += va[k], rb += vb[k];
      }
      const int n_tow = (int)(ta & 0xffffu), n_ph = (int)(ta >> 16), n_nh = (int)tb;
      if (!multi && lane == 0) s_ntow[0] = 0, s_ntow[1] = n_tow, s_nph[0] = 0, s_nph[1] = n_ph, s_nnh[0] = 0, s_nnh[1] = n_nh;
      const unsigned long long agg = (unsigned long long)n_tow | ((unsigned long long)(n_ph + n_nh) << 31);
      if (lane == 0) chain_publish(prm.chain, tile, agg), s_misc[3] = agg;  // successors add it up without waiting for this tile's prefix
    } else if (wid == 1) {
      // the track prefix: every predecessor published its count when it started its tile, so this never waits
      if (multi) event_scan(s_ntrk, ne);
      const unsigned long long ex = chain_resolve<8>(prm.chain_t, tile, s_misc[5]);
      if (lane == 0) s_misc[1] = ex;
    } else if (multi) {
      if (wid == 2) event_scan(s_ntow, ne);
      else if (wid == 3) event_scan(s_nph, ne);
      else if (wid == 4) event_scan(s_nnh, ne);
    }
    __syncthreads();
    const long long t0 = (long long)s_misc[1];  // first track of the tile
    // Warp 0 resolves the tower / neutral prefix (the one place a CTA waits for its predecessors); meanwhile the other
    // warps move the tile's tracks from where kernel P parked them into the Track collection, which needs the track
    // prefix only.
    if (wid == 0) {
      const unsigned long long ex = chain_resolve<8>(prm.chain, tile, s_misc[3]);
      if (lane == 0) s_misc[2] = ex;
    } else {
      for (int e = tid - 32; e < ne; e += THREADS - 32) prm.trk_offsets[e0 + e + 1] = t0 + s_ntrk[e + 1];
      if (tile == 0 && tid == 32) prm.trk_offsets[0] = 0;
      for (int k = wid - 1; k < n_seg; k += W - 1) {
        const long long gs = (gseg_lo + k) * PD_PSEG;
        const int a = s_sega[k], c = s_segc[k];
        const unsigned ob = (unsigned)t0 + (unsigned)s_segp[k];
        // two rows of a segment at a time: twenty independent loads in flight per lane before the first store
        for (int r = lane; r < c; r += 64) {
          const bool two = r + 32 < c;
          const long long g = gs + a + r, g2 = two ? g + 32 : g;
          const unsigned o = ob + (unsigned)r;
          const int i0 = (int)__ldg(prm.park_idx + g), i1 = (int)__ldg(prm.park_idx + g2);
          const int d0 = __ldg(prm.park_pid + g), d1 = __ldg(prm.park_pid + g2);
          const signed char q0_ = __ldg(prm.park_q + g), q1_ = __ldg(prm.park_q + g2);
          float f0[6], f1[6];
#pragma unroll
          for (int k6 = 0; k6 < 6; ++k6) f0[k6] = __ldg(prm.park_f[k6] + g), f1[k6] = __ldg(prm.park_f[k6] + g2);
          prm.trk_src[o] = (int)(p_al + gs + i0), prm.trk_pid[o] = d0, prm.trk_charge[o] = q0_;
          prm.trk_pt[o] = f0[0], prm.trk_eta[o] = f0[1], prm.trk_phi[o] = f0[2], prm.trk_E[o] = f0[3];
          prm.trk_eta_out[o] = f0[4], prm.trk_phi_out[o] = f0[5];
          if (two) {
            const unsigned o2 = o + 32u;
            prm.trk_src[o2] = (int)(p_al + gs + i1), prm.trk_pid[o2] = d1, prm.trk_charge[o2] = q1_;
            prm.trk_pt[o2] = f1[0], prm.trk_eta[o2] = f1[1], prm.trk_phi[o2] = f1[2], prm.trk_E[o2] = f1[3];
            prm.trk_eta_out[o2] = f1[4], prm.trk_phi_out[o2] = f1[5];
          }
        }
      }
      if (prm.imp_on) {
        // pd_options.impact: the four values kernel P parked beside each record, in a loop of their own (the common path
        // above stays as it is)
        for (int k = wid - 1; k < n_seg; k += W - 1) {
          const long long gs = (gseg_lo + k) * PD_PSEG;
          const int a = s_sega[k], c = s_segc[k];
          const unsigned ob = (unsigned)t0 + (unsigned)s_segp[k];
          for (int r = lane; r < c; r += 32) {
            const long long g = gs + a + r;
#pragma unroll
            for (int k4 = 0; k4 < 4; ++k4) prm.imp_out[k4][ob + (unsigned)r] = __ldg(prm.park_imp[k4] + g);
          }
        }
      }
    }
    __syncthreads();
    const long long base_tow = (long long)(s_misc[2] & FIELD_MASK);
    const long long base_efl = t0 + (long long)((s_misc[2] >> 31) & FIELD_MASK);

    // ------------------------------------------------------------------ pass O: ordered outputs
    for (int e = tid; e < ne; e += THREADS) {
      prm.tow_offsets[e0 + e + 1] = base_tow + s_ntow[e + 1];
      prm.efl_offsets[e0 + e + 1] = base_efl + s_ntrk[e + 1] + s_nph[e + 1] + s_nnh[e + 1];
    }
    if (tile == 0 && tid == 0) prm.tow_offsets[0] = 0, prm.efl_offsets[0] = 0;
    // the EFlow entries of the tracks, from the parked records (L2 hits)
    for (int k = wid; k < n_seg; k += W) {
      const long long gs = (gseg_lo + k) * PD_PSEG;
      const int a = s_sega[k], c = s_segc[k], sp = s_segp[k];
      for (int r = lane; r < c; r += 32) {
        const long long g = gs + a + r;
        const int il = (int)(gs + (long long)__ldg(prm.park_idx + g) - q0);
        const int pid = __ldg(prm.park_pid + g);
        const int e = multi ? (int)s_ev[il] : 0;
        const unsigned at = (unsigned)base_efl + (unsigned)(sp + r + s_nph[e] + s_nnh[e]);
        const int apid = pid < 0 ? -pid : pid;
        float fw = 1.f;
        if (weighted) {
          // reading K5: the factor of the track's tower component (staged by pass W where its neutral is not emitted); the
          // slot of the tower through the bitmap ranks, as in pass B
          const unsigned key = (unsigned)__ldg(prm.key + (q0 + il));
          if (key != 0xffffu) {
            const int id = (int)(key & 0x7fffu);
            int gi;
            uint4 bits;
            if (!sparse) {
              gi = e * gpe + (id >> 7);
              bits = ((const uint4 *)s_bitmap)[gi];
            } else {
              const int wq = e * l2w + (id >> 12);
              gi = (int)s_l2p[wq] + __popc(s_bitmap[wq] & ((1u << ((id >> 7) & 31)) - 1u));
              bits = s_pool[gi];
            }
            const int slot = (int)s_gp[gi] + popc_below(bits, id & 127);
            const unsigned hv = s_head[slot];
            const int hh = (int)(hv & LINK_END);
            if (key & 0x8000u) fw = (hv & SLOT_NH) ? 1.f : __uint_as_float(s_res[hh]);
            else fw = (hv & SLOT_PH) ? 1.f : s_Et[hh];
          }
        }
        prm.efl_cls[at] = (signed char)(apid == 11 ? PD_CLS_ELECTRON : (apid == 13 ? PD_CLS_MUON : PD_CLS_CHHAD));
        prm.efl_src[at] = (int)(p0 + il);
        prm.efl_pt[at] = __ldg(prm.park_f[0] + g) * fw;
        prm.efl_eta[at] = __ldg(prm.park_f[1] + g);
        prm.efl_phi[at] = __ldg(prm.park_f[2] + g);
        prm.efl_E[at] = __ldg(prm.park_f[3] + g) * fw;
      }
    }
    for (int it = 0; it < n_it; ++it) {
      const int d = it * THREADS + tid;
      const unsigned hv = d < n_slots ? s_head[d] : 0u;
      const bool f_tw = hv & SLOT_TW, f_ph = hv & SLOT_PH, f_nh = hv & SLOT_NH;
      const unsigned m_tw = __ballot_sync(0xffffffffu, f_tw), m_ph = __ballot_sync(0xffffffffu, f_ph),
                     m_nh = __ballot_sync(0xffffffffu, f_nh);
      if (hv & (SLOT_TW | SLOT_PH | SLOT_NH)) {
        const int h = (int)(hv & LINK_END), tower = (int)((hv >> 13) & RES_TOWER);
        const float em = s_stg[d], had = s_Ev[h], nem = s_Et[h], nhad = __uint_as_float(s_res[h]);
        const unsigned pa = s_preA[it * W + wid], pb = s_preB[it * W + wid];
        const int e = multi ? (int)s_ev[h] : 0;
        float eta_c, phi_c, ic;
        tower_position<FID>(sc, tc, prm.rk, prm.event_base + e0 + e, tower, eta_c, phi_c, ic);
        if (f_tw) {
          const unsigned at = (unsigned)base_tow + (pa & 0xffffu) + (unsigned)__popc(m_tw & lt_mask);
          prm.tow_tower[at] = tower;
          prm.tow_eta[at] = eta_c;
          prm.tow_phi[at] = phi_c;
          prm.tow_E[at] = em + had;
          prm.tow_Eem[at] = em;
          prm.tow_Ehad[at] = had;
          prm.tow_ET[at] = (em + had) * ic;
        }
        if (f_ph) {
          const int slot = (int)(pa >> 16) + __popc(m_ph & lt_mask);
          const unsigned at = (unsigned)base_efl + (unsigned)(s_ntrk[e + 1] + s_nnh[e] + slot);
          prm.efl_cls[at] = (signed char)PD_CLS_PHOTON;
          prm.efl_src[at] = tower;
          prm.efl_pt[at] = nem * ic;
          prm.efl_eta[at] = eta_c;
          prm.efl_phi[at] = phi_c;
          prm.efl_E[at] = nem;
        }
        if (f_nh) {
          const int slot = (int)pb + __popc(m_nh & lt_mask);
          const unsigned at = (unsigned)base_efl + (unsigned)(s_ntrk[e + 1] + s_nph[e + 1] + slot);
          prm.efl_cls[at] = (signed char)PD_CLS_NEUHAD;
          prm.efl_src[at] = tower;
          prm.efl_pt[at] = nhad * ic;
          prm.efl_eta[at] = eta_c;
          prm.efl_phi[at] = phi_c;
          prm.efl_E[at] = nhad;
        }
      }
    }
    fence_async_smem();  // generic-proxy writes to slots the next tile's bulk copies overwrite
  }
}

}  // namespace pdk

// ---- host side: plan + launch ------------------------------------------------------------------

static int g_num_sms = 0;
static int g_max_smem_optin = 0;

static int query_device() {
  if (g_num_sms > 0) return PD_OK;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&g_num_sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&g_max_smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return PD_ECUDA;
  return PD_OK;
}

// Tile plan of kernel T from sizes the host knows (n_events, n_particles).  B200: 228 KB of shared memory per SM,
// 1 KB reserved per CTA, 227 KB per CTA at most.  Preferred shape: two 512-thread CTAs per SM (113 KB each), so one
// CTA's barriers and look-back waits are covered by the other; events too large for that get one 1024-thread CTA
// with the whole SM.  G = events per tile: as many as fit the on-chip capacity C with 6 sigma of head-room
// for a Poisson-like sum, but no more than keeps every CTA slot of the GPU busy on small inputs.
// tile_events: the caller's cap on the events per tile (pd_options.tile_events), 0 = automatic
int pd_plan(const pd_card *c, long long n_events, long long n_particles, int tile_events, PdLaunchPlan *plan) {
  const int t_tile_events = tile_events < 0 ? 0 : (tile_events > pdk::G_MAX ? pdk::G_MAX : tile_events);
  const PdCardScalars &sc = c->sc;
  const double avg = n_events > 0 ? double(n_particles) / double(n_events) : 0.0;
  const size_t budget2 = (228 * 1024 - 2 * 1024) / 2, budget1 = 227 * 1024;
  int sparse = 0;
  auto cap_for = [&](int G, size_t budget) {
    const size_t fixed = pdk::make_layout(sc.n_bins, sc.n_towers, sc.words_per_event, G, 0, sparse, sc.res_per_bin, sc.smear_center, sc.eflow_weighted).total;
    const size_t per = pdk::T_BYTES_PER_PARTICLE + (G > 1 ? 1 : 0) + (sparse ? 18 : 0) + (sc.eflow_weighted ? 4 : 0);
    long cap = budget > fixed + 7 * 16 ? long((budget - fixed - 7 * 16) / per) : 0;
    cap &= ~3L;
    return int(cap > pdk::C_MAX ? pdk::C_MAX : cap);
  };
  auto fits = [&](int G, size_t budget) {
    const double C = cap_for(G, budget);
    return double(G) * avg + 6.0 * std::sqrt(double(G) * avg + 1.0) + 16.0 <= C;
  };
  static const int force_threads = std::getenv("PD_THREADS") ? std::atoi(std::getenv("PD_THREADS")) : 0;
  size_t budget = budget2;
  plan->threads = 512;
  // one event per tile on request (pd_options.tile_events = 1): the
  // large variant, so that the only limit left is the capacity of a whole SM
  if (force_threads == 1024 || t_tile_events == 1 || (force_threads == 0 && !fits(1, budget2))) {
    budget = budget1;
    plan->threads = 1024;
  }
  int g = 1;
  while (g < pdk::G_MAX && fits(g + 1, budget)) ++g;
  if (plan->threads == 512) {
    // sparse mode (two-level tower bitmap) when it packs clearly more events into a tile: large grids, small events
    static const int force_sparse = std::getenv("PD_SPARSE") ? std::atoi(std::getenv("PD_SPARSE")) : -1;
    const int g_dense = g;
    sparse = 1;
    int gs = 1;
    while (gs < pdk::G_MAX && fits(gs + 1, budget)) ++gs;
    const bool take = force_sparse >= 0 ? force_sparse != 0 : (g_dense > 1 && 2 * gs >= 3 * g_dense);
    if (take && fits(1, budget)) g = gs;
    else sparse = 0;
  }
  // keep all CTA slots busy: aim for >= 4 tiles per resident CTA when the input is small
  const long slots = 148L * (plan->threads == 512 ? 2 : 1);
  const long g_bal = long((n_events + 4 * slots - 1) / (4 * slots));
  if (g > g_bal) g = int(g_bal < 1 ? 1 : g_bal);
  if (t_tile_events > 0 && g > t_tile_events) g = t_tile_events;
  plan->events_per_tile = g;
  plan->capacity = cap_for(g, budget);
  plan->n_tiles = int((n_events + g - 1) / g);
  plan->n_ptiles = int((n_particles + 15 + PD_PTILE - 1) / PD_PTILE);  // + 15: tiles start at a multiple of 16 particles
  plan->sparse = sparse;
  {
    // grid <= resident CTAs of the device (256 SMs assumed when no device can be queried yet)
    const long sms = query_device() == PD_OK ? g_num_sms : 256;
    plan->max_ctas = int(sms * (plan->threads == 1024 ? 1 : 2));
  }
  plan->lay = pdk::make_layout(sc.n_bins, sc.n_towers, sc.words_per_event, g, plan->capacity, sparse, sc.res_per_bin, sc.smear_center, sc.eflow_weighted);
  plan->smem_bytes = plan->lay.total;
  return PD_OK;
}

template <int THREADS, bool DEBUG, bool SPARSE, bool FID>
static int launch_variant2(const PdParams &prm, const PdLaunchPlan &plan, cudaStream_t stream) {
  constexpr int CTAS = THREADS == 512 ? 2 : 1;
  auto kern = pdk::pd_tower_kernel<THREADS, CTAS, DEBUG, SPARSE, FID>;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, g_max_smem_optin) != cudaSuccess) return PD_ECUDA;
  // persistent CTAs wait on one another through the look-back chain: the grid must be co-resident
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, THREADS, plan.smem_bytes) != cudaSuccess) return PD_ECUDA;
  if (per_sm < 1) return PD_ECUDA;
  if (per_sm > CTAS) per_sm = CTAS;
  if (const char *e = getenv("PD_T_PER_SM")) per_sm = std::min(per_sm, atoi(e));  // experiment
  int grid = g_num_sms * per_sm;
  if (grid > plan.n_tiles) grid = plan.n_tiles;
  if (grid < 1) grid = 1;
  kern<<<grid, THREADS, plan.smem_bytes, stream>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}

// the variant with the higher-fidelity card options (K1-K3) compiled in only for the cards that use them
template <int THREADS, bool DEBUG, bool SPARSE>
static int launch_variant(const PdParams &prm, const PdLaunchPlan &plan, cudaStream_t stream) {
  const bool fid = prm.sc.res_per_bin || prm.sc.smear_center || prm.sc.nsig2_ecal > 0.f || prm.sc.nsig2_hcal > 0.f || prm.sc.eflow_weighted;
  return fid ? launch_variant2<THREADS, DEBUG, SPARSE, true>(prm, plan, stream) : launch_variant2<THREADS, DEBUG, SPARSE, false>(prm, plan, stream);
}

// the two kernels of the chain, back to back on the stream: P (particles -> keys + tracks), then T (towers, EFlow)
int pd_launch_chain(const PdParams &prm, const PdLaunchPlan &plan, bool debug, void *stream) {
  if (query_device() != PD_OK) return PD_ECUDA;
  if (plan.smem_bytes > (size_t)g_max_smem_optin) return PD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  if (prm.n_ptiles > 0) {
    const int rc = pd_launch_particles(prm, debug, g_num_sms, g_max_smem_optin, stream);
    if (rc != PD_OK) return rc;
  }
  if (plan.threads == 1024) {
    if (plan.sparse) return PD_EINVAL;  // pd_plan never pairs the two
    return debug ? launch_variant<1024, true, false>(prm, plan, st) : launch_variant<1024, false, false>(prm, plan, st);
  }
  if (plan.sparse) return debug ? launch_variant<512, true, true>(prm, plan, st) : launch_variant<512, false, true>(prm, plan, st);
  return debug ? launch_variant<512, true, false>(prm, plan, st) : launch_variant<512, false, false>(prm, plan, st);
}
