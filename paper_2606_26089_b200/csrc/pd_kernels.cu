// pd_kernels.cu -- the fused Delphes-chain kernel for sm_100a (steps S0..S8 of SURVEY.md section 8a), v5f.
//
// Persistent CTAs (two 512-thread CTAs per SM, or one 1024-thread CTA for large events); a CTA repeatedly
// claims a TILE (a run of G whole events, <= C particles) from an atomic counter and takes it through
//   pass A   S0-S2, S4  one thread per particle, particle order, inputs prefetched one iteration ahead:
//                       classify, propagate, efficiency, tower id; marks the tower in the event's BITMAP
//   scan 1              one block scan for two things: the ordered list of accepted tracks, and the
//                       popcount prefix of the bitmaps = the rank ("slot") of every occupied tower in
//                       (event, tower id) order -- this replaces a sort of the deposits
//   pass B   S5         every deposit pushes itself on its slot's list (one integer atomicExch); the tile's
//                       track count is published on chain T
//   pass T   S3         one thread per accepted track: pT smear; E_trk stays on chip, the track record is
//                       parked in this CTA's slice of the workspace ring (L2) until its offset is known
//   pass W   S5-S7      one thread per occupied tower: exact fixed-point sum of its list (order-independent),
//                       Philox tower stream, log-normal smear, thresholds, EFlow subtraction
//   scan W              one scan over the per-warp counts; chain W published and resolved (decoupled
//                       look-back), chain T resolved (never waits: published a whole phase ago)
//   pass O   S8         ordered compaction of tracks / towers / photons / neutral hadrons, CSR offsets
// Large grids with small events use a two-level bitmap (sparse mode, see make_layout): groups first, then the
// tower bits of the non-empty groups only.
// Nothing but the inputs, the final collections and the ring touches memory.  Sums are order-stable: each
// tower's deposits are added as 64-bit fixed-point integers (exact, hence independent of the order in which
// the list was built), and the only atomics are integer (bitmap OR, list exchange, counters).
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdlib>

#include "pd_internal.h"
#include "pd_math.cuh"

namespace pdk {

constexpr int G_MAX = 256;         // events per tile (event index of a particle is kept in 8 bits)
constexpr int C_MAX = 8191;        // particles per tile: list links are 13 bits, 0x1fff = end of list
constexpr uint32_t LINK_END = 0x1fffu;
// per-particle result word: tower id (15 bits, 0x7fff none) | flags | link to the next deposit of the tower
constexpr uint32_t RES_TOWER = 0x7fffu, RES_DEP = 1u << 15, RES_HCAL = 1u << 16, RES_ACC = 1u << 17;
constexpr int RES_LINK_SHIFT = 18;
constexpr unsigned long long FLAG_A = 1ull << 62, FLAG_P = 2ull << 62, VAL_MASK = (1ull << 62) - 1;
constexpr unsigned long long FIELD_MASK = (1ull << 31) - 1;  // chain W packs towers | neutrals << 31

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~size_t(15); }

// Shared-memory carve-up, identical on host (size) and device (pointers).
struct Layout {
  size_t tb, nphi, offset, inv_w, half, w, eta_c, inv_cosh, lut, binlut;  // card tables
  size_t off32, ntrk, ntow, nph, nnh;                                     // per-event arrays [G+1]
  size_t misc;                                                            // scratch words
  size_t cnt;                                                             // pass W warp counts -> prefixes [2][256]
  size_t bitmap, gprefix;                                                 // per event: tower bits, group prefix
  size_t l2p, pool;                                                       // sparse mode (see make_layout)
  size_t res, uT, phi, Ev, head, stg, ev;                                 // per particle / per slot
  size_t total;
};

// Dense mode: one bit per tower and event (bitmap), a prefix per 128-tower group (gprefix).
// Sparse mode (large grids, small events: the bitmaps would be almost empty and take most of the shared memory):
// `bitmap` holds one bit per 128-tower GROUP and event, `l2p` the rank of the first non-empty group of each of its
// words, `pool` the tower bits of the non-empty groups only (at most one per deposit), `gprefix` their prefixes.
__host__ __device__ inline Layout make_layout(int n_bins, int lut_cells, int n_towers, int words_per_event, int G,
                                              int C, int sparse) {
  Layout l;
  size_t o = 0;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = align16(o + bytes);
    return at;
  };
  l.tb = take(4 * (n_bins + 1));
  l.nphi = take(4 * n_bins);
  l.offset = take(4 * (n_bins + 1));
  l.inv_w = take(4 * n_bins);
  l.half = take(4 * n_bins);
  l.w = take(4 * n_bins);
  l.eta_c = take(4 * n_bins);
  l.inv_cosh = take(4 * n_bins);
  l.lut = take(2 * (size_t)lut_cells);
  l.binlut = take(2 * (size_t)((n_towers >> 5) + 2));
  l.off32 = take(4 * (G + 1));
  l.ntrk = take(4 * (G + 1));
  l.ntow = take(4 * (G + 1));
  l.nph = take(4 * (G + 1));
  l.nnh = take(4 * (G + 1));
  l.misc = take(8 * 64);
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
  l.uT = take(4 * (size_t)C);
  l.phi = take(4 * (size_t)C);
  l.Ev = take(4 * (size_t)C);
  l.head = take(2 * (size_t)C);
  l.stg = take(4 * (size_t)C);
  l.ev = take(G > 1 ? (size_t)C : 0);
  l.total = o;
  return l;
}

// ---- look-back chain (decoupled look-back, one 64-bit self-flagged word per tile) ---------------
__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_relaxed(unsigned long long *p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ unsigned long long warp_sum_u64(unsigned long long v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// Decoupled look-back, split in two: chain_publish() makes the tile's aggregate visible as soon as it is
// known; chain_resolve() (one full warp, later) returns the exclusive prefix over all earlier tiles to every
// lane and publishes the inclusive prefix.  All resident CTAs run nearly in phase, so the nearest predecessor
// already holding an inclusive prefix is typically a whole grid (~300 tiles) back: the warp looks at
// LB_K * 32 predecessors per round trip to L2 (LB_K independent loads per lane).  Packed fields add independently.
template <int LB_K>
__device__ __forceinline__ unsigned long long chain_resolve(unsigned long long *st, int tile, unsigned long long agg) {
  const int lane = threadIdx.x & 31;
  if (tile == 0) {
    if (lane == 0) st_relaxed(st, FLAG_P | agg);
    return 0;
  }
  unsigned long long excl = 0;
  int pos = tile - 1;
  for (;;) {
    unsigned long long v[LB_K];
#pragma unroll
    for (int k = 0; k < LB_K; ++k) {
      const int idx = pos - (k * 32 + lane);
      v[k] = idx >= 0 ? ld_relaxed(st + idx) : FLAG_P;  // before the first tile: prefix 0
    }
    bool done = false;
#pragma unroll
    for (int k = 0; k < LB_K; ++k) {
      if (done) break;
      const int idx = pos - (k * 32 + lane);
      unsigned long long w = v[k];
      unsigned pm;
      for (;;) {
        pm = __ballot_sync(0xffffffffu, (w >> 62) == 2);
        const unsigned zm = __ballot_sync(0xffffffffu, (w >> 62) == 0);
        // every entry up to and including the nearest inclusive prefix must have been published
        const unsigned upto = pm ? (0xffffffffu >> (32 - __ffs(pm))) : 0xffffffffu;
        if ((zm & upto) == 0u) break;
        if ((w >> 62) == 0) {
          __nanosleep(40);
          w = ld_relaxed(st + idx);
        }
      }
      if (pm) {
        const int first = __ffs(pm) - 1;
        excl += warp_sum_u64(lane <= first ? (w & VAL_MASK) : 0ull);
        done = true;
      } else {
        excl += warp_sum_u64(w & VAL_MASK);
      }
    }
    if (done) break;
    pos -= 32 * LB_K;
  }
  if (lane == 0) st_relaxed(st + tile, FLAG_P | (excl + agg));
  return excl;
}
__device__ __forceinline__ void chain_publish(unsigned long long *st, int tile, unsigned long long agg) {
  if (tile > 0) st_relaxed(st + tile, FLAG_A | agg);
}

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

// Block-wide exclusive prefix of packed per-warp totals wtot[W] (REDUX adds): returns the exclusive
// prefix of this thread's WARP and the block total.  Fields of the packed word must not overflow.
template <int W>
__device__ __forceinline__ void warp_totals_scan(const unsigned *wtot, unsigned &excl_warp, unsigned &total) {
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  const unsigned v = lane < W ? wtot[lane] : 0u;
  total = __reduce_add_sync(0xffffffffu, v);
  excl_warp = __reduce_add_sync(0xffffffffu, lane < wid ? v : 0u);
}

__device__ __forceinline__ unsigned warp_incl_scan(unsigned v) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

struct ParticleIn {
  int pid, q;
  float px, py, pz, E, vx, vy, vz;
};

// input arrays rebased to the first particle of the tile (uniform pointers + a 32-bit particle index)
struct TileIn {
  const int *pid;
  const signed char *charge;
  const float *px, *py, *pz, *E, *vx, *vy, *vz;
};

__device__ __forceinline__ ParticleIn load_particle(const TileIn &t, unsigned i) {
  ParticleIn p;
  p.pid = __ldg(t.pid + i);
  p.q = (int)__ldg(t.charge + i);
  p.px = __ldg(t.px + i), p.py = __ldg(t.py + i), p.pz = __ldg(t.pz + i);
  p.E = __ldg(t.E + i);
  p.vx = __ldg(t.vx + i), p.vy = __ldg(t.vy + i), p.vz = __ldg(t.vz + i);
  return p;
}

__device__ __forceinline__ int popc4(const uint4 &v) { return __popc(v.x) + __popc(v.y) + __popc(v.z) + __popc(v.w); }

// number of set bits of the 128-bit group below bit position pos (0..127)
__device__ __forceinline__ int popc_below(const uint4 &v, int pos) {
  const int w = pos >> 5;
  const uint32_t m = (1u << (pos & 31)) - 1u;
  const uint32_t cur = w == 0 ? v.x : (w == 1 ? v.y : (w == 2 ? v.z : v.w));
  int c = __popc(cur & m);
  c += w > 0 ? __popc(v.x) : 0;
  c += w > 1 ? __popc(v.y) : 0;
  c += w > 2 ? __popc(v.z) : 0;
  return c;
}

template <int THREADS, int CTAS, bool DEBUG, bool SPARSE>
__global__ void __launch_bounds__(THREADS, CTAS) pd_chain_kernel(const __grid_constant__ PdParams prm) {
  constexpr int W = THREADS / 32;
  extern __shared__ __align__(16) unsigned char smem[];
  const PdCardScalars &sc = prm.sc;
  const int nb = sc.n_bins;
  const int C = prm.capacity, G = prm.events_per_tile;
  const int wpe = sc.words_per_event, gpe = wpe >> 2;
  constexpr bool sparse = SPARSE;  // two-level tower bitmap, chosen by pd_plan (prm.sparse)
  const int l2w = (gpe + 31) >> 5;  // words of the per-event group bitmap (sparse mode)
  const Layout L = make_layout(nb, 2 * sc.lut_side, sc.n_towers, wpe, G, C, prm.sparse);
  float *s_tb = (float *)(smem + L.tb);
  int *s_nphi = (int *)(smem + L.nphi);
  int *s_offset = (int *)(smem + L.offset);
  float *s_inv_w = (float *)(smem + L.inv_w);
  float *s_half = (float *)(smem + L.half);
  float *s_w = (float *)(smem + L.w);
  float *s_eta_c = (float *)(smem + L.eta_c);
  float *s_inv_cosh = (float *)(smem + L.inv_cosh);
  unsigned short *s_lut = (unsigned short *)(smem + L.lut);
  unsigned short *s_binlut = (unsigned short *)(smem + L.binlut);
  int *s_off32 = (int *)(smem + L.off32);
  int *s_ntrk = (int *)(smem + L.ntrk);
  int *s_ntow = (int *)(smem + L.ntow);
  int *s_nph = (int *)(smem + L.nph);
  int *s_nnh = (int *)(smem + L.nnh);
  unsigned long long *s_misc = (unsigned long long *)(smem + L.misc);
  unsigned *s_wtot = (unsigned *)(s_misc + 8);   // [32] per-warp totals of scan 1
  unsigned *s_preA = (unsigned *)(smem + L.cnt);  // per (iteration, warp) of pass W: towers | photons << 16 ...
  unsigned *s_preB = s_preA + 256;                // ... and neutral hadrons (counts, then exclusive prefixes)
  uint32_t *s_bitmap = (uint32_t *)(smem + L.bitmap);
  unsigned short *s_gp = (unsigned short *)(smem + L.gprefix);
  unsigned short *s_l2p = (unsigned short *)(smem + L.l2p);  // sparse mode: rank of the first non-empty group of a word
  uint4 *s_pool = (uint4 *)(smem + L.pool);                  // sparse mode: tower bits of the non-empty groups
  uint32_t *s_res = (uint32_t *)(smem + L.res);
  float *s_uT = (float *)(smem + L.uT);    // hit u of accepted tracks, then E_trk, then staged photon energy
  float *s_phi = (float *)(smem + L.phi);  // hit phi of accepted tracks, then staged Eem''
  float *s_Ev = (float *)(smem + L.Ev);    // deposit energy, then staged Ehad''
  unsigned *s_head = (unsigned *)(smem + L.stg);         // per slot: last pusher, then head | tower id << 13
  unsigned short *s_tk = (unsigned short *)(smem + L.head);  // accepted tracks in particle order
  unsigned char *s_ev = smem + L.ev;

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;

  for (int i = tid; i <= nb; i += THREADS) {
    s_tb[i] = prm.tab.tb[i];
    s_offset[i] = prm.tab.offset[i];
  }
  for (int i = tid; i < nb; i += THREADS) {
    s_nphi[i] = prm.tab.nphi[i];
    s_inv_w[i] = prm.tab.inv_w[i];
    s_half[i] = prm.tab.half[i];
    s_w[i] = prm.tab.w[i];
    s_eta_c[i] = prm.tab.eta_c[i];
    s_inv_cosh[i] = prm.tab.inv_cosh[i];
  }
  for (int i = tid; i < 2 * sc.lut_side; i += THREADS) s_lut[i] = prm.tab.lut[i];
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
  SmCard cd{s_tb, s_nphi, s_offset, s_inv_w, s_half, s_w, s_eta_c, s_inv_cosh, s_lut};

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
    int n = (int)min(p1 - p0, (long long)0x7fffffff);
    const bool overflow = (p1 - p0) > (long long)C;
    if (overflow) {
      n = 0;
      if (tid == 0) atomicExch(prm.status_word, (int)PD_EEVENTSIZE);
    }
    for (int e = tid; e <= ne; e += THREADS) {
      s_off32[e] = overflow ? 0 : (int)(prm.offsets[e0 + e] - p0);
      s_ntrk[e] = 0, s_ntow[e] = 0, s_nph[e] = 0, s_nnh[e] = 0;
    }
    const int NG = ne * gpe;  // 128-tower bitmap groups of the tile
    const int NW = ne * l2w;  // sparse mode: words of the group bitmaps
    if (!sparse) {
      for (int k = tid; k < NG; k += THREADS) ((uint4 *)s_bitmap)[k] = make_uint4(0u, 0u, 0u, 0u);
    } else {
      for (int k = tid; k < NW; k += THREADS) s_bitmap[k] = 0u;
    }
    __syncthreads();
    if (multi) {
      // event index of every particle of the tile: warp per event, lanes over its particles
      for (int e = wid; e < ne; e += W)
        for (int i = s_off32[e] + lane; i < s_off32[e + 1]; i += 32) s_ev[i] = (unsigned char)e;
      __syncthreads();
    }

    // ------------------------------------------------------------------ pass A: S0-S2, S4 per particle
    {
      const TileIn tin{prm.pid + p0, prm.charge + p0, prm.px + p0, prm.py + p0, prm.pz + p0, prm.E + p0,
                       prm.vx + p0, prm.vy + p0, prm.vz + p0};
      ParticleIn nxt;
      if (tid < n) nxt = load_particle(tin, (unsigned)tid);
      for (int i = tid; i < n; i += THREADS) {
        const ParticleIn c = nxt;
        if (i + THREADS < n) nxt = load_particle(tin, (unsigned)(i + THREADS));
        const int e = multi ? (int)s_ev[i] : 0;
        ParticleOut o;
        particle_chain(sc, cd, c.q, c.px, c.py, c.pz, c.vx, c.vy, c.vz, prm.rk, prm.event_base + e0 + e,
                       (uint32_t)(i - s_off32[e]), sc.eff_per_species ? species_of(c.pid) : 2, o);
        const int apid = c.pid < 0 ? -c.pid : c.pid;
        const bool to_ecal = apid == 11 || apid == 22;                             // reading A18
        const bool to_none = apid == 13 || apid == 12 || apid == 14 || apid == 16;
        uint32_t res = RES_TOWER | (LINK_END << RES_LINK_SHIFT);
        if (o.tower >= 0) {
          res = (uint32_t)o.tower | (LINK_END << RES_LINK_SHIFT);
          if (!to_none) {
            res |= RES_DEP | (to_ecal ? 0u : RES_HCAL);
            if (!sparse) atomicOr(&s_bitmap[e * wpe + (o.tower >> 5)], 1u << (o.tower & 31));
            else atomicOr(&s_bitmap[e * l2w + (o.tower >> 12)], 1u << ((o.tower >> 7) & 31));  // its 128-tower group
            s_Ev[i] = c.E;
          }
        }
        if (o.accepted) {
          res |= RES_ACC;
          s_uT[i] = o.u, s_phi[i] = o.phi_pos;
          if (multi) atomicAdd(&s_ntrk[e], 1);
        }
        s_res[i] = res;
        s_head[i] = 0xffffffffu;
        if (DEBUG) {
          const long long g = p0 + i;
          if (prm.dbg_status) prm.dbg_status[g] = (unsigned char)o.status;
          if (prm.dbg_eta_pos) prm.dbg_eta_pos[g] = (o.status & PD_FACE_MASK) ? eta_from_u(sc, o.u) : o.u;
          if (prm.dbg_phi_pos) prm.dbg_phi_pos[g] = o.phi_pos;
          if (prm.dbg_tower) prm.dbg_tower[g] = o.tower;
          if (prm.dbg_accepted) prm.dbg_accepted[g] = o.accepted ? 1 : 0;
          if (prm.dbg_eps_row) prm.dbg_eps_row[g] = (signed char)o.eps_row;
          if (prm.dbg_pt_smeared) prm.dbg_pt_smeared[g] = 0.f;
          if (prm.dbg_tw_first) prm.dbg_tw_first[g] = 0;
        }
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ scan 1: tracks in order + tower slots
    // Each thread owns a contiguous chunk of particles and of bitmap groups (odd chunk lengths keep the
    // shared-memory accesses of a warp on distinct banks); one packed block scan serves both.
    int n_trk, n_slots;
    {
      const int ka = ((n + THREADS - 1) / THREADS) | 1;
      const int a0 = min(n, tid * ka), a1 = min(n, a0 + ka);
      unsigned cnt_a = 0;
      for (int i = a0; i < a1; ++i) cnt_a += (s_res[i] >> 17) & 1u;
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
      const unsigned packed = cnt_a | (cnt_g << 16);
      const unsigned incl = warp_incl_scan(packed);
      if (lane == 31) s_wtot[wid] = incl;
      __syncthreads();
      unsigned excl_w, tot;
      warp_totals_scan<W>(s_wtot, excl_w, tot);
      const unsigned excl = excl_w + incl - packed;
      int ra = (int)(excl & 0xffffu), rg = (int)(excl >> 16);
      for (int i = a0; i < a1; ++i)
        if (s_res[i] & RES_ACC) s_tk[ra++] = (unsigned short)i;
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
      n_trk = (int)(tot & 0xffffu), n_slots = (int)(tot >> 16);
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

    // ------------------------------------------------------------------ publish chain T; pass B
    // the track aggregate is published now and its prefix resolved only at the end of the tile (pass O), when
    // the predecessors have long published theirs: no CTA ever waits on the track chain
    if (tid == 0) chain_publish(prm.chain, tile, (unsigned long long)n_trk);
    if (wid == 1) {
      if (multi) event_scan(s_ntrk, ne);
      else if (lane == 0) s_ntrk[0] = 0, s_ntrk[1] = n_trk;
    }
    // pass B (S5): every deposit finds its tower's slot and pushes itself on the slot's list
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
    // (no barrier: pass T touches nothing pass B does -- it reads the track list and (u, phi) of the accepted
    // tracks and replaces u by E_trk; pass W, behind the next barrier, needs both)

    // ------------------------------------------------------------------ pass T: S3 on the accepted tracks
    // (converged: one thread per track).  The smeared record is parked in this CTA's slice of the workspace ring
    // (L2-resident, rewritten every tile) until pass O knows where the tile's tracks go.
    float *ring = prm.ring + (size_t)blockIdx.x * 6u * (size_t)C;
    for (int s = tid; s < n_trk; s += THREADS) {
      const int i = s_tk[s];
      const long long src = p0 + i;
      const float px = __ldg(prm.px + src), py = __ldg(prm.py + src), pz = __ldg(prm.pz + src);
      const int e = multi ? (int)s_ev[i] : 0;
      TrackOut t;
      track_smear(sc, px, py, pz, prm.rk, prm.event_base + e0 + e, (uint32_t)(i - s_off32[e]), sc.trk_per_species ? species_of(__ldg(prm.pid + src)) : 2, t);
      const float u = s_uT[i];
      s_uT[i] = t.E_trk;  // from here on: the track energy that pass W subtracts
      __stcg(ring + s, t.pt_s);
      __stcg(ring + C + s, t.eta_mom);
      __stcg(ring + 2 * C + s, t.phi0);
      __stcg(ring + 3 * C + s, t.E_trk);
      __stcg(ring + 4 * C + s, eta_from_u(sc, u));
      __stcg(ring + 5 * C + s, s_phi[i]);
      if (DEBUG && prm.dbg_pt_smeared) prm.dbg_pt_smeared[src] = t.pt_s;
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
        long long a_em = 0, a_had = 0, t_em = 0, t_had = 0;
        int first = h;
        for (int c = h;;) {
          const uint32_t rc = c == h ? rh : s_res[c];
          const long long Ev = __float2ll_rn(s_Ev[c] * 4294967296.f);
          const long long Tv = (rc & RES_ACC) ? __float2ll_rn(s_uT[c] * 4294967296.f) : 0ll;
          if (rc & RES_HCAL) a_had += Ev, t_had += Tv;
          else a_em += Ev, t_em += Tv;
          first = min(first, c);
          c = (int)(rc >> RES_LINK_SHIFT);
          if (c == (int)LINK_END) break;
        }
        const float Eem = (float)a_em * 2.3283064365386963e-10f, Ehad = (float)a_had * 2.3283064365386963e-10f;
        const float Tem = (float)t_em * 2.3283064365386963e-10f, Thad = (float)t_had * 2.3283064365386963e-10f;
        uint32_t rn[4];
        rng_block(prm.rk, prm.event_base + e0 + e, (uint32_t)tower, 1u, rn);
        float em_s, had_s;
        tower_smear(sc, Eem, Ehad, rn, em_s, had_s);
        // reading A22: the threshold is applied twice, strictly, per component
        const bool k_em = em_s > sc.thr_ecal, k_had = had_s > sc.thr_hcal;
        const float em_f = k_em ? em_s : 0.f, had_f = k_had ? had_s : 0.f;
        const float n_em = em_f - Tem, n_had = had_f - Thad;
        f_ph = n_em > sc.thr_ecal, f_nh = n_had > sc.thr_hcal;
        f_tw = em_f + had_f > 0.f;
        if (multi) {
          if (f_tw) atomicAdd(&s_ntow[e], 1);
          if (f_ph) atomicAdd(&s_nph[e], 1);
          if (f_nh) atomicAdd(&s_nnh[e], 1);
        }
        // stage the tower at its head particle's index (only this thread ever touches that particle again)
        s_phi[h] = em_f, s_Ev[h] = had_f, s_uT[h] = f_ph ? n_em : 0.f;
        s_res[h] = __float_as_uint(f_nh ? n_had : 0.f);
        s_head[d] = (unsigned)h | ((unsigned)tower << 13);
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
      if (lane == 0) chain_publish(prm.chain + prm.n_tiles, tile, agg), s_misc[3] = agg;
    } else if (wid == 1) {
      // the track prefix: published long ago by every predecessor, so this never waits
      const unsigned long long ex = chain_resolve<10>(prm.chain, tile, (unsigned long long)n_trk);
      if (lane == 0) s_misc[1] = ex;
    } else if (multi) {
      if (wid == 2) event_scan(s_ntow, ne);
      else if (wid == 3) event_scan(s_nph, ne);
      else if (wid == 4) event_scan(s_nnh, ne);
    }
    __syncthreads();
    const long long base_trk = (long long)s_misc[1];
    // The track collection needs the track prefix only: it is written between publishing the tower / neutral
    // aggregate and resolving its prefix, which gives the slower predecessors that much time to publish theirs.
    for (int e = tid; e < ne; e += THREADS) prm.trk_offsets[e0 + e + 1] = base_trk + s_ntrk[e + 1];
    for (int s = tid; s < n_trk; s += THREADS) {
      const long long src = p0 + s_tk[s];
      const unsigned g = (unsigned)base_trk + (unsigned)s;  // all output indices fit 32 bits (n_particles < 2^30)
      prm.trk_src[g] = (int)src;
      prm.trk_pid[g] = __ldg(prm.pid + src);
      prm.trk_charge[g] = __ldg(prm.charge + src);
      prm.trk_pt[g] = __ldcg(ring + s);
      prm.trk_eta[g] = __ldcg(ring + C + s);
      prm.trk_phi[g] = __ldcg(ring + 2 * C + s);
      prm.trk_E[g] = __ldcg(ring + 3 * C + s);
      prm.trk_eta_out[g] = __ldcg(ring + 4 * C + s);
      prm.trk_phi_out[g] = __ldcg(ring + 5 * C + s);
    }
    if (wid == 0) {
      const unsigned long long ex = chain_resolve<1>(prm.chain + prm.n_tiles, tile, s_misc[3]);
      if (lane == 0) s_misc[2] = ex;
    }
    __syncthreads();
    const long long base_tow = (long long)(s_misc[2] & FIELD_MASK);
    const long long base_efl = base_trk + (long long)((s_misc[2] >> 31) & FIELD_MASK);

    // ------------------------------------------------------------------ pass O: ordered outputs
    for (int e = tid; e < ne; e += THREADS) {
      prm.tow_offsets[e0 + e + 1] = base_tow + s_ntow[e + 1];
      prm.efl_offsets[e0 + e + 1] = base_efl + s_ntrk[e + 1] + s_nph[e + 1] + s_nnh[e + 1];
    }
    if (tile == 0 && tid == 0) prm.trk_offsets[0] = 0, prm.tow_offsets[0] = 0, prm.efl_offsets[0] = 0;
    // the EFlow entries of the tracks, from the records pass T parked in the ring (L2 hits)
    for (int s = tid; s < n_trk; s += THREADS) {
      const int i = s_tk[s];
      const long long src = p0 + i;
      const float pt = __ldcg(ring + s), eta = __ldcg(ring + C + s), phi = __ldcg(ring + 2 * C + s), Et = __ldcg(ring + 3 * C + s);
      const int pid = __ldg(prm.pid + src);
      const int e = multi ? (int)s_ev[i] : 0;
      const unsigned at = (unsigned)base_efl + (unsigned)(s + s_nph[e] + s_nnh[e]);
      const int apid = pid < 0 ? -pid : pid;
      prm.efl_cls[at] = (signed char)(apid == 11 ? PD_CLS_ELECTRON : (apid == 13 ? PD_CLS_MUON : PD_CLS_CHHAD));
      prm.efl_src[at] = (int)src;
      prm.efl_pt[at] = pt;
      prm.efl_eta[at] = eta;
      prm.efl_phi[at] = phi;
      prm.efl_E[at] = Et;
    }
    for (int it = 0; it < n_it; ++it) {
      const int d = it * THREADS + tid;
      bool f_tw = false, f_ph = false, f_nh = false;
      int h = 0, tower = 0;
      float em = 0.f, had = 0.f, nem = 0.f, nhad = 0.f;
      if (d < n_slots) {
        const unsigned hv = s_head[d];
        h = (int)(hv & LINK_END), tower = (int)(hv >> 13);
        em = s_phi[h], had = s_Ev[h], nem = s_uT[h], nhad = __uint_as_float(s_res[h]);
        f_tw = em + had > 0.f;
        f_ph = nem > 0.f;
        f_nh = nhad > 0.f;
      }
      const unsigned m_tw = __ballot_sync(0xffffffffu, f_tw), m_ph = __ballot_sync(0xffffffffu, f_ph),
                     m_nh = __ballot_sync(0xffffffffu, f_nh);
      if (f_tw || f_ph || f_nh) {
        const unsigned pa = s_preA[it * W + wid], pb = s_preB[it * W + wid];
        const int e = multi ? (int)s_ev[h] : 0;
        int b = (int)s_binlut[tower >> 5];
        while (tower >= s_offset[b + 1]) ++b;
        const int j = tower - s_offset[b];
        const float eta_c = s_eta_c[b];
        const float phi_c = fmaf((float)j + 0.5f, s_w[b], -kPiF);
        const float ic = s_inv_cosh[b];
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

// Tile plan from sizes the host knows (n_events, n_particles).  B200: 228 KB of shared memory per SM, 1 KB
// reserved per CTA, 227 KB per CTA at most.  Preferred shape: two 512-thread CTAs per SM (113 KB each), so one
// CTA's barriers and look-back waits are covered by the other; events too large for that get one 1024-thread CTA
// with the whole SM.  G = events per tile: as many as fit the on-chip capacity C with 6 sigma of head-room
// for a Poisson-like sum, but no more than keeps every CTA slot of the GPU busy on small inputs.
static thread_local int t_tile_events = 0;  // pd_set_tile_events: 0 = automatic
int pd_plan_set_tile_events(int g) {
  const int prev = t_tile_events;
  t_tile_events = g < 0 ? 0 : (g > pdk::G_MAX ? pdk::G_MAX : g);
  return prev;
}

int pd_plan(const pd_card *c, long long n_events, long long n_particles, PdLaunchPlan *plan) {
  const PdCardScalars &sc = c->sc;
  const double avg = n_events > 0 ? double(n_particles) / double(n_events) : 0.0;
  const size_t budget2 = (228 * 1024 - 2 * 1024) / 2, budget1 = 227 * 1024;
  int sparse = 0;
  auto cap_for = [&](int G, size_t budget) {
    const size_t fixed = pdk::make_layout(sc.n_bins, 2 * sc.lut_side, sc.n_towers, sc.words_per_event, G, 0, sparse).total;
    const size_t per = 22 + (G > 1 ? 1 : 0) + (sparse ? 18 : 0);
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
  // one event per tile on request (pd_set_tile_events(1), the fall-back for batches with outlier events): the
  // large variant, so that the only limit left is the capacity of a whole SM
  if (force_threads == 1024 || t_tile_events == 1 || (force_threads == 0 && !fits(1, budget2))) {
    budget = budget1;
    plan->threads = 1024;
  }
  int g = 1;
  while (g < pdk::G_MAX && fits(g + 1, budget)) ++g;
  {
    // sparse mode (two-level tower bitmap) when it packs clearly more events into a tile: large grids, small events
    static const int force_sparse = std::getenv("PD_SPARSE") ? std::atoi(std::getenv("PD_SPARSE")) : -1;
    const int g_dense = g;
    sparse = 1;
    int gs = 1;
    while (gs < pdk::G_MAX && fits(gs + 1, budget)) ++gs;
    const bool take = t_tile_events != 1 && (force_sparse >= 0 ? force_sparse != 0 : (g_dense > 1 && 2 * gs >= 3 * g_dense));
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
  {
    // grid <= resident CTAs of the device (256 SMs assumed when no device can be queried yet)
    const long sms = query_device() == PD_OK ? g_num_sms : 256;
    const long ctas = sms * (plan->threads == 1024 ? 1 : 2);
    plan->max_ctas = int(plan->n_tiles < ctas ? (plan->n_tiles > 0 ? plan->n_tiles : 1) : ctas);
  }
  plan->sparse = sparse;
  plan->smem_bytes = pdk::make_layout(sc.n_bins, 2 * sc.lut_side, sc.n_towers, sc.words_per_event, g, plan->capacity, sparse).total;
  return PD_OK;
}

template <int THREADS, bool DEBUG, bool SPARSE>
static int launch_variant(const PdParams &prm, const PdLaunchPlan &plan, cudaStream_t stream) {
  constexpr int CTAS = THREADS == 512 ? 2 : 1;
  auto kern = pdk::pd_chain_kernel<THREADS, CTAS, DEBUG, SPARSE>;
  static bool configured = false;
  if (!configured) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, g_max_smem_optin) != cudaSuccess) return PD_ECUDA;
    configured = true;
  }
  // persistent CTAs wait on one another through the look-back chains: the grid must be co-resident
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, THREADS, plan.smem_bytes) != cudaSuccess) return PD_ECUDA;
  if (per_sm < 1) return PD_ECUDA;
  if (per_sm > CTAS) per_sm = CTAS;
  int grid = g_num_sms * per_sm;
  if (grid > plan.n_tiles) grid = plan.n_tiles;
  if (grid < 1) grid = 1;
  kern<<<grid, THREADS, plan.smem_bytes, stream>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}

int pd_launch_chain(const PdParams &prm, const PdLaunchPlan &plan, bool debug, void *stream) {
  if (query_device() != PD_OK) return PD_ECUDA;
  if (plan.smem_bytes > (size_t)g_max_smem_optin) return PD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  if (plan.threads == 1024) {
    if (plan.sparse) return PD_EINVAL;  // pd_plan never pairs the two
    return debug ? launch_variant<1024, true, false>(prm, plan, st) : launch_variant<1024, false, false>(prm, plan, st);
  }
  if (plan.sparse) return debug ? launch_variant<512, true, true>(prm, plan, st) : launch_variant<512, false, true>(prm, plan, st);
  return debug ? launch_variant<512, true, false>(prm, plan, st) : launch_variant<512, false, false>(prm, plan, st);
}
