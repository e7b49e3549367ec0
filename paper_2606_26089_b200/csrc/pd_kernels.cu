// pd_kernels.cu -- the fused Delphes-chain kernel for sm_100a (steps S0..S8 of SURVEY.md section 8a).
//
// One persistent CTA per SM slot; a CTA repeatedly claims a TILE (a run of G whole events, <= C
// particles) from an atomic counter and takes it through
//   phase 1   S0-S4  one thread per particle: classify, propagate, efficiency, pT smear, tower key;
//                    accepted tracks and deposits are compacted IN PARTICLE ORDER into shared memory
//   chain T          decoupled look-back over tiles -> global track offset; tracks + track CSR written
//   phase 2a  S5     stable LSD radix sort of the deposits by (local event, tower) in shared memory
//   phase 2b  S5-S7  one thread per distinct (event, tower): sequential sum in particle order,
//                    Philox tower stream, log-normal smear, thresholds, EFlow subtraction
//   chain W          look-back for the tower and eflow offsets
//   phase 3   S8     ordered compaction of towers / photons / neutral hadrons, EFlow track entries,
//                    CSR offsets
// Nothing but the inputs and the final collections touches HBM.  Sums are order-stable: the sort is
// stable, the per-tower sum is sequential, and the only atomics are integer counters.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdint>
#include <cstdlib>

#include "pd_internal.h"
#include "pd_math.cuh"

namespace pdk {

constexpr int G_MAX = 256;     // events per tile (8 event bits)
constexpr int r_max(int threads) { return threads >= 1024 ? 6 : 12; }  // radix-sort rounds per warp: C <= THREADS * r_max
// deposit key = hcal << 31 | local event << code_bits | tower code (eta bin << j_bits | phi bin)
constexpr uint32_t KEY_MASK = 0x7fffffffu;
constexpr unsigned long long FLAG_A = 1ull << 62, FLAG_P = 2ull << 62, VAL_MASK = (1ull << 62) - 1;

__host__ __device__ inline size_t align16(size_t x) { return (x + 15) & ~size_t(15); }

// Shared-memory carve-up, identical on host (size) and device (pointers).
struct Layout {
  size_t tb, nphi, offset, inv_w, half, w, eta_c, inv_cosh;  // card tables
  size_t off32, ntrk, ntow, nph, nnh;                        // per-event arrays [G_MAX+1]
  size_t misc;                                               // 64 x u64 scratch
  size_t cnt;                                                // radix counters u16 [256 * W]
  size_t dep_key, dep_E, dep_T, dep_idx;                     // deposits
  size_t uni;                                                // union: track staging | tower staging
  size_t total;
};

__host__ __device__ inline Layout make_layout(int n_bins, int threads, int C) {
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
  l.off32 = take(4 * (G_MAX + 1));
  l.ntrk = take(4 * (G_MAX + 1));
  l.ntow = take(4 * (G_MAX + 1));
  l.nph = take(4 * (G_MAX + 1));
  l.nnh = take(4 * (G_MAX + 1));
  l.misc = take(8 * 96);
  l.cnt = take(2 * 256 * (threads / 32));
  l.dep_key = take(4 * (size_t)C);
  l.dep_E = take(4 * (size_t)C);
  l.dep_T = take(4 * (size_t)C);
  l.dep_idx = take(2 * (size_t)C);
  l.uni = take(20 * (size_t)C + 16);
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

// Called by one full warp.  Publishes this tile's aggregate, returns the exclusive prefix over all
// earlier tiles to every lane, then publishes the inclusive prefix.
__device__ unsigned long long chain_lookback(unsigned long long *st, int tile, unsigned long long agg) {
  const int lane = threadIdx.x & 31;
  if (tile == 0) {
    if (lane == 0) st_relaxed(st, FLAG_P | agg);
    return 0;
  }
  if (lane == 0) st_relaxed(st + tile, FLAG_A | agg);
  unsigned long long excl = 0;
  int pos = tile - 1;
  for (;;) {
    const int idx = pos - lane;
    unsigned long long v = FLAG_P;  // before the first tile: prefix 0
    if (idx >= 0) {
      do {
        v = ld_relaxed(st + idx);
      } while ((v >> 62) == 0);
    }
    const unsigned pm = __ballot_sync(0xffffffffu, (v >> 62) == 2);
    if (pm) {
      const int first = __ffs(pm) - 1;  // nearest predecessor holding an inclusive prefix
      excl += warp_sum_u64(lane <= first ? (v & VAL_MASK) : 0ull);
      break;
    }
    excl += warp_sum_u64(v & VAL_MASK);
    pos -= 32;
  }
  if (lane == 0) st_relaxed(st + tile, FLAG_P | (excl + agg));
  return excl;
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

// largest e in [0, ne) with off[e] <= i
__device__ __forceinline__ int find_event(const int *off, int ne, int i) {
  int lo = 0, hi = ne;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (off[mid] <= i) lo = mid;
    else hi = mid;
  }
  return lo;
}

// largest b in [0, nb) with offset[b] <= id
__device__ __forceinline__ int find_bin(const int *offset, int nb, int id) {
  int lo = 0, hi = nb;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (offset[mid] <= id) lo = mid;
    else hi = mid;
  }
  return lo;
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

// bits of the per-particle result word written by pass P1
constexpr uint32_t RES_DEP = 1u << 21, RES_HCAL = 1u << 22, RES_ACC = 1u << 23;

template <int THREADS, int CTAS, bool DEBUG>
__global__ void __launch_bounds__(THREADS, CTAS) pd_chain_kernel(const __grid_constant__ PdParams prm) {
  constexpr int W = THREADS / 32;
  constexpr int R_MAX = r_max(THREADS);
  extern __shared__ __align__(16) unsigned char smem[];
  const PdCardScalars &sc = prm.sc;
  const int nb = sc.n_bins;
  const int C = prm.capacity;
  const Layout L = make_layout(nb, THREADS, C);
  float *s_tb = (float *)(smem + L.tb);
  int *s_nphi = (int *)(smem + L.nphi);
  int *s_offset = (int *)(smem + L.offset);
  float *s_inv_w = (float *)(smem + L.inv_w);
  float *s_half = (float *)(smem + L.half);
  float *s_w = (float *)(smem + L.w);
  float *s_eta_c = (float *)(smem + L.eta_c);
  float *s_inv_cosh = (float *)(smem + L.inv_cosh);
  int *s_off32 = (int *)(smem + L.off32);
  int *s_ntrk = (int *)(smem + L.ntrk);
  int *s_ntow = (int *)(smem + L.ntow);
  int *s_nph = (int *)(smem + L.nph);
  int *s_nnh = (int *)(smem + L.nnh);
  unsigned long long *s_misc = (unsigned long long *)(smem + L.misc);
  int *s_ctr = (int *)(s_misc + 4);             // [0] charged count, [1] neutral count
  unsigned *s_wtot = (unsigned *)(s_misc + 8);  // [5][32]
  uint16_t *s_cnt = (uint16_t *)(smem + L.cnt);
  uint32_t *dep_key = (uint32_t *)(smem + L.dep_key);
  float *dep_E = (float *)(smem + L.dep_E);
  float *dep_T = (float *)(smem + L.dep_T);
  uint16_t *dep_idx = (uint16_t *)(smem + L.dep_idx);
  // union region, view A (passes P0..P2): per-particle scratch
  uint32_t *p_res = (uint32_t *)(smem + L.uni);
  float *p_u = (float *)(p_res + C), *p_phi = p_u + C;
  uint16_t *p_perm = (uint16_t *)(p_phi + C), *tk_i = p_perm + C;
  // union region, view B (phase 2b on): per deposited tower
  uint32_t *st_key = (uint32_t *)(smem + L.uni);
  float *st_em = (float *)(st_key + C), *st_had = st_em + C, *st_nem = st_had + C, *st_nhad = st_nem + C;

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
  SmCard cd{s_tb, s_nphi, s_offset, s_inv_w, s_half, s_w, s_eta_c, s_inv_cosh};
  const int G = prm.events_per_tile;
  const int EV_SHIFT = sc.code_bits;
  const int JB = sc.j_bits;
  const uint32_t code_mask = (1u << EV_SHIFT) - 1u, j_mask = (1u << JB) - 1u;

  for (;;) {
    __syncthreads();  // previous tile fully done with shared memory (and card tables staged)
    if (tid == 0) {
      s_misc[0] = atomicAdd(prm.tile_counter, 1u);
      s_ctr[0] = 0, s_ctr[1] = 0;
    }
    __syncthreads();
    const int tile = (int)s_misc[0];
    if (tile >= prm.n_tiles) break;
    const long long e0 = (long long)tile * G;
    const int ne = (int)min((long long)G, prm.n_events - e0);
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

    // ------------------------------------------------------------------ P0: charged-first permutation
    // (the per-particle math is order-independent; grouping by kind keeps its warps converged)
    for (int it = 0; it * THREADS < n; ++it) {
      const int i = it * THREADS + tid;
      const bool valid = i < n;
      const int q = valid ? (int)__ldg(prm.charge + p0 + i) : 0;
      const bool chg = valid && q != 0, neu = valid && q == 0;
      const unsigned cm = __ballot_sync(0xffffffffu, chg), nm = __ballot_sync(0xffffffffu, neu);
      int cb = 0, nbs = 0;
      if (lane == 0) {
        if (cm) cb = atomicAdd(&s_ctr[0], __popc(cm));
        if (nm) nbs = atomicAdd(&s_ctr[1], __popc(nm));
      }
      cb = __shfl_sync(0xffffffffu, cb, 0), nbs = __shfl_sync(0xffffffffu, nbs, 0);
      if (chg) p_perm[cb + __popc(cm & lt_mask)] = (uint16_t)i;
      if (neu) p_perm[n - 1 - (nbs + __popc(nm & lt_mask))] = (uint16_t)i;
    }
    __syncthreads();

    // ------------------------------------------------------------------ P1: S0-S2, S4 per particle (no barriers)
    for (int k = tid; k < n; k += THREADS) {
      const int i = p_perm[k];
      const long long g = p0 + i;
      const int pid = __ldg(prm.pid + g);
      const int q = (int)__ldg(prm.charge + g);
      const float px = __ldg(prm.px + g), py = __ldg(prm.py + g), pz = __ldg(prm.pz + g);
      const float vx = __ldg(prm.vx + g), vy = __ldg(prm.vy + g), vz = __ldg(prm.vz + g);
      const int e = find_event(s_off32, ne, i);
      ParticleOut o;
      particle_chain(sc, cd, pid, q, px, py, pz, vx, vy, vz, prm.seed, prm.event_base + e0 + e, (uint32_t)(i - s_off32[e]), o);
      const int apid = pid < 0 ? -pid : pid;
      const bool to_ecal = apid == 11 || apid == 22;
      const bool to_none = apid == 13 || apid == 12 || apid == 14 || apid == 16;
      uint32_t res = 0;
      if (o.bin >= 0) res = ((uint32_t)o.bin << JB) | (uint32_t)o.j | (to_none ? 0u : RES_DEP) | (to_ecal ? 0u : RES_HCAL);
      if (o.accepted) {
        res |= RES_ACC;
        p_u[i] = o.u, p_phi[i] = o.phi_pos;
        atomicAdd(&s_ntrk[e], 1);
      }
      p_res[i] = res;
      if (DEBUG) {
        if (prm.dbg_status) prm.dbg_status[g] = (unsigned char)o.status;
        if (prm.dbg_eta_pos) prm.dbg_eta_pos[g] = (o.status & PD_FACE_MASK) ? eta_from_u(sc, o.u) : o.u;
        if (prm.dbg_phi_pos) prm.dbg_phi_pos[g] = o.phi_pos;
        if (prm.dbg_tower) prm.dbg_tower[g] = o.bin >= 0 ? s_offset[o.bin] + o.j : -1;
        if (prm.dbg_accepted) prm.dbg_accepted[g] = o.accepted ? 1 : 0;
        if (prm.dbg_eps_row) prm.dbg_eps_row[g] = (signed char)o.eps_row;
        if (prm.dbg_pt_smeared) prm.dbg_pt_smeared[g] = 0.f;
        if (prm.dbg_tw_first) prm.dbg_tw_first[g] = 0;
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ P1b: ordered compaction (particle order)
    int trk_base = 0, dep_base = 0;
    for (int it = 0; it * THREADS < n; ++it) {
      const int i = it * THREADS + tid;
      const uint32_t res = i < n ? p_res[i] : 0u;
      const bool acc = (res & RES_ACC) != 0, dep = (res & RES_DEP) != 0;
      const unsigned am = __ballot_sync(0xffffffffu, acc), dm = __ballot_sync(0xffffffffu, dep);
      if (lane == 0) s_wtot[(it & 1) * 32 + wid] = (unsigned)__popc(am) | ((unsigned)__popc(dm) << 16);
      __syncthreads();
      unsigned excl_w, tot;
      warp_totals_scan<W>(s_wtot + (it & 1) * 32, excl_w, tot);
      if (acc) tk_i[trk_base + (int)(excl_w & 0xffffu) + __popc(am & lt_mask)] = (uint16_t)i;
      if (dep) {
        const int s = dep_base + (int)(excl_w >> 16) + __popc(dm & lt_mask);
        const int e = find_event(s_off32, ne, i);
        dep_key[s] = ((res & RES_HCAL) ? 0x80000000u : 0u) | ((uint32_t)e << EV_SHIFT) | (res & code_mask);
        dep_idx[s] = (uint16_t)i;
        dep_E[i] = __ldg(prm.E + p0 + i);
        dep_T[i] = 0.f;
      }
      trk_base += (int)(tot & 0xffffu);
      dep_base += (int)(tot >> 16);
    }
    const int n_trk = trk_base, m = dep_base;
    __syncthreads();

    // ------------------------------------------------------------------ phase 2a: stable radix sort
    {
      const int nbits = EV_SHIFT + prm.event_bits;
      int n_pass = (nbits + 7) / 8;
      int bits_per = (nbits + n_pass - 1) / n_pass;
      if (bits_per < 5) bits_per = 5;
      const int bins = 1 << bits_per;
      const int ipw = 32 * ((m + 32 * W - 1) / (32 * W));  // items per warp, multiple of 32
      for (int pass = 0; pass < n_pass; ++pass) {
        const int shift = pass * bits_per;
        const uint32_t dmask = (uint32_t)bins - 1u;
        for (int k = tid; k < bins * W / 2; k += THREADS) ((uint32_t *)s_cnt)[k] = 0u;
        __syncthreads();
        uint32_t kreg[R_MAX], ireg[R_MAX];
#pragma unroll
        for (int r = 0; r < R_MAX; ++r) {
          kreg[r] = 0, ireg[r] = 0;
          if (r * 32 < ipw) {  // warp-uniform
            const int pos = wid * ipw + r * 32 + lane;
            const bool valid = pos < m;
            const uint32_t k = valid ? dep_key[pos] : 0u;
            const uint32_t ix = valid ? (uint32_t)dep_idx[pos] : 0u;
            const uint32_t d = valid ? ((k >> shift) & dmask) : 0xffffffffu;
            const unsigned peers = __match_any_sync(0xffffffffu, d);
            const unsigned lower = peers & lt_mask;
            const uint32_t c = valid ? (uint32_t)s_cnt[d * W + wid] : 0u;
            __syncwarp();
            if (valid && lower == 0u) s_cnt[d * W + wid] = (uint16_t)(c + (uint32_t)__popc(peers));
            __syncwarp();
            kreg[r] = k;
            ireg[r] = ix | ((c + (uint32_t)__popc(lower)) << 16);
          }
        }
        __syncthreads();
        // exclusive scan of the bins*W counters (digit-major, warp-minor); bins*W/THREADS = bins/32 per thread
        {
          const int per = bins / 32;
          const int at = tid * per;
          uint32_t loc[8], sum = 0;
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            loc[k] = k < per ? (uint32_t)s_cnt[at + k] : 0u;
            sum += loc[k];
          }
          uint32_t incl = sum;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const uint32_t t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
          }
          if (lane == 31) s_wtot[64 + wid] = incl;
          __syncthreads();
          unsigned excl_w, tot;
          warp_totals_scan<W>(s_wtot + 64, excl_w, tot);
          uint32_t run = excl_w + incl - sum;
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            if (k < per) s_cnt[at + k] = (uint16_t)run;
            run += loc[k];
          }
        }
        __syncthreads();
#pragma unroll
        for (int r = 0; r < R_MAX; ++r) {
          if (r * 32 < ipw) {
            const int pos = wid * ipw + r * 32 + lane;
            if (pos < m) {
              const uint32_t d = (kreg[r] >> shift) & dmask;
              const uint32_t rank = (uint32_t)s_cnt[d * W + wid] + (ireg[r] >> 16);
              dep_key[rank] = kreg[r];
              dep_idx[rank] = (uint16_t)(ireg[r] & 0xffffu);
            }
          }
        }
        __syncthreads();
      }
    }

    // ------------------------------------------------------------------ chain T (tracks)
    if (wid == 0) {
      const unsigned long long ex = chain_lookback(prm.chain, tile, (unsigned long long)n_trk);
      if (lane == 0) s_misc[1] = ex;
    } else if (wid == 1) {
      event_scan(s_ntrk, ne);
    }
    __syncthreads();
    const long long base_trk = (long long)s_misc[1];

    // ------------------------------------------------------------------ P2: S3 on the accepted tracks (converged),
    // written straight to the track collection
    for (int s = tid; s < n_trk; s += THREADS) {
      const int i = tk_i[s];
      const long long src = p0 + i, g = base_trk + s;
      const int pid = __ldg(prm.pid + src);
      const float px = __ldg(prm.px + src), py = __ldg(prm.py + src), pz = __ldg(prm.pz + src);
      const int e = find_event(s_off32, ne, i);
      TrackOut t;
      track_smear(sc, px, py, pz, prm.seed, prm.event_base + e0 + e, (uint32_t)(i - s_off32[e]), t);
      dep_T[i] = t.E_trk;
      prm.trk_src[g] = (int)src;
      prm.trk_pid[g] = pid;
      prm.trk_charge[g] = __ldg(prm.charge + src);
      prm.trk_pt[g] = t.pt_s;
      prm.trk_eta[g] = t.eta_mom;
      prm.trk_phi[g] = t.phi0;
      prm.trk_E[g] = t.E_trk;
      prm.trk_eta_out[g] = eta_from_u(sc, p_u[i]);
      prm.trk_phi_out[g] = p_phi[i];
      if (DEBUG && prm.dbg_pt_smeared) prm.dbg_pt_smeared[src] = t.pt_s;
    }
    for (int e = tid; e < ne; e += THREADS) prm.trk_offsets[e0 + e + 1] = base_trk + s_ntrk[e + 1];
    if (tile == 0 && tid == 0) prm.trk_offsets[0] = 0, prm.tow_offsets[0] = 0, prm.efl_offsets[0] = 0;
    __syncthreads();  // view A of the union region is dead from here on

    // ------------------------------------------------------------------ phase 2b-1: run heads, in order
    int dt_base = 0;
    for (int it = 0; it * THREADS < m; ++it) {
      const int pos = it * THREADS + tid;
      bool head = false;
      if (pos < m) {
        const uint32_t kk = dep_key[pos] & KEY_MASK;
        const uint32_t prev = pos > 0 ? (dep_key[pos - 1] & KEY_MASK) : 0xffffffffu;
        head = kk != prev;
      }
      const unsigned hm = __ballot_sync(0xffffffffu, head);
      if (lane == 0) s_wtot[(it & 1) * 32 + wid] = (unsigned)__popc(hm);
      __syncthreads();
      unsigned excl_w, tot;
      warp_totals_scan<W>(s_wtot + (it & 1) * 32, excl_w, tot);
      if (head) st_key[dt_base + (int)excl_w + __popc(hm & lt_mask)] = (uint32_t)pos;
      dt_base += (int)tot;
    }
    const int n_dt = dt_base;
    __syncthreads();

    // ------------------------------------------------------------------ phase 2b-2: S5-S7, one thread per tower
    for (int d = tid; d < n_dt; d += THREADS) {
      const int pos = (int)st_key[d];
      const uint32_t kk = dep_key[pos] & KEY_MASK;
      float Eem = 0.f, Ehad = 0.f, Tem = 0.f, Thad = 0.f;
      int qpos = pos;
      do {  // sequential sum in particle order (the sort is stable)
        const uint32_t kq = dep_key[qpos];
        if ((kq & KEY_MASK) != kk) break;
        const int pi = dep_idx[qpos];
        const float Ev = dep_E[pi], Tv = dep_T[pi];
        if (kq >> 31) Ehad += Ev, Thad += Tv;
        else Eem += Ev, Tem += Tv;
        ++qpos;
      } while (qpos < m);
      const uint32_t code = kk & code_mask;
      const int e = (int)(kk >> EV_SHIFT);
      const int tower = s_offset[code >> JB] + (int)(code & j_mask);
      uint32_t rn[4];
      rng_block(prm.seed, prm.event_base + e0 + e, (uint32_t)tower, 1u, rn);
      float em_s, had_s;
      tower_smear(sc, Eem, Ehad, rn, em_s, had_s);
      // reading A22: the threshold is applied twice, strictly, per component
      const bool k_em = em_s > sc.thr_ecal, k_had = had_s > sc.thr_hcal;
      const float em_f = k_em ? em_s : 0.f, had_f = k_had ? had_s : 0.f;
      const float n_em = em_f - Tem, n_had = had_f - Thad;
      const bool is_ph = n_em > sc.thr_ecal, is_nh = n_had > sc.thr_hcal;
      if (em_f + had_f > 0.f) atomicAdd(&s_ntow[e], 1);
      if (is_ph) atomicAdd(&s_nph[e], 1);
      if (is_nh) atomicAdd(&s_nnh[e], 1);
      st_key[d] = kk;
      st_em[d] = em_f, st_had[d] = had_f, st_nem[d] = is_ph ? n_em : 0.f, st_nhad[d] = is_nh ? n_had : 0.f;
      if (DEBUG) {
        const long long g = p0 + dep_idx[pos];
        if (prm.dbg_tw_first) prm.dbg_tw_first[g] = 1;
        if (prm.dbg_tw[0]) prm.dbg_tw[0][g] = Eem;
        if (prm.dbg_tw[1]) prm.dbg_tw[1][g] = Ehad;
        if (prm.dbg_tw[2]) prm.dbg_tw[2][g] = Tem;
        if (prm.dbg_tw[3]) prm.dbg_tw[3][g] = Thad;
        if (prm.dbg_tw[4]) prm.dbg_tw[4][g] = em_s;
        if (prm.dbg_tw[5]) prm.dbg_tw[5][g] = had_s;
        if (prm.dbg_tw_dec)
          prm.dbg_tw_dec[g] = (unsigned char)((k_em ? PD_DEC_EEM : 0) | (k_had ? PD_DEC_EHAD : 0) |
                                              (is_ph ? PD_DEC_NEM : 0) | (is_nh ? PD_DEC_NHAD : 0));
      }
    }
    __syncthreads();

    // ------------------------------------------------------------------ chain W (towers, eflow)
    if (wid == 0) event_scan(s_ntow, ne);
    else if (wid == 1) event_scan(s_nph, ne);
    else if (wid == 2) event_scan(s_nnh, ne);
    __syncthreads();
    if (wid == 0) {
      const unsigned long long ex = chain_lookback(prm.chain + prm.n_tiles, tile, (unsigned long long)s_ntow[ne]);
      if (lane == 0) s_misc[2] = ex;
    } else if (wid == 1) {
      const unsigned long long agg = (unsigned long long)n_trk + (unsigned long long)s_nph[ne] + (unsigned long long)s_nnh[ne];
      const unsigned long long ex = chain_lookback(prm.chain + 2 * (size_t)prm.n_tiles, tile, agg);
      if (lane == 0) s_misc[3] = ex;
    }
    __syncthreads();
    const long long base_tow = (long long)s_misc[2], base_efl = (long long)s_misc[3];

    // ------------------------------------------------------------------ phase 3: ordered outputs
    for (int e = tid; e < ne; e += THREADS) {
      prm.tow_offsets[e0 + e + 1] = base_tow + s_ntow[e + 1];
      prm.efl_offsets[e0 + e + 1] = base_efl + s_ntrk[e + 1] + s_nph[e + 1] + s_nnh[e + 1];
    }
    // EFlow entries of the tracks: copied from the track arrays this CTA wrote above (L2 hits)
    for (int s = tid; s < n_trk; s += THREADS) {
      const long long g = base_trk + s;
      const int src = __ldcg(prm.trk_src + g);
      const int e = find_event(s_off32, ne, (int)(src - p0));
      const long long at = base_efl + s + s_nph[e] + s_nnh[e];
      const int pid = __ldcg(prm.trk_pid + g);
      const int apid = pid < 0 ? -pid : pid;
      prm.efl_cls[at] = (signed char)(apid == 11 ? PD_CLS_ELECTRON : (apid == 13 ? PD_CLS_MUON : PD_CLS_CHHAD));
      prm.efl_src[at] = src;
      prm.efl_pt[at] = __ldcg(prm.trk_pt + g);
      prm.efl_eta[at] = __ldcg(prm.trk_eta + g);
      prm.efl_phi[at] = __ldcg(prm.trk_phi + g);
      prm.efl_E[at] = __ldcg(prm.trk_E + g);
    }
    int tw_run = 0, ph_run = 0, nh_run = 0;
    for (int it = 0; it * THREADS < n_dt; ++it) {
      const int d = it * THREADS + tid;
      bool f_tw = false, f_ph = false, f_nh = false;
      uint32_t kk = 0;
      float em = 0.f, had = 0.f, nem = 0.f, nhad = 0.f;
      if (d < n_dt) {
        kk = st_key[d];
        em = st_em[d], had = st_had[d], nem = st_nem[d], nhad = st_nhad[d];
        f_tw = em + had > 0.f;
        f_ph = nem > 0.f;
        f_nh = nhad > 0.f;
      }
      const unsigned m_tw = __ballot_sync(0xffffffffu, f_tw), m_ph = __ballot_sync(0xffffffffu, f_ph),
                     m_nh = __ballot_sync(0xffffffffu, f_nh);
      if (lane == 0) {
        s_wtot[(it & 1) * 32 + wid] = (unsigned)__popc(m_tw) | ((unsigned)__popc(m_ph) << 16);
        s_wtot[96 + (it & 1) * 32 + wid] = (unsigned)__popc(m_nh);
      }
      __syncthreads();
      unsigned excl_w, tot, excl_n, tot_n;
      warp_totals_scan<W>(s_wtot + (it & 1) * 32, excl_w, tot);
      warp_totals_scan<W>(s_wtot + 96 + (it & 1) * 32, excl_n, tot_n);
      if (f_tw || f_ph || f_nh) {
        const uint32_t code = kk & code_mask;
        const int e = (int)(kk >> EV_SHIFT);
        const int b = (int)(code >> JB), j = (int)(code & j_mask);
        const int tower = s_offset[b] + j;
        const float eta_c = s_eta_c[b];
        const float phi_c = fmaf((float)j + 0.5f, s_w[b], -kPiF);
        const float ic = s_inv_cosh[b];
        if (f_tw) {
          const long long at = base_tow + tw_run + (int)(excl_w & 0xffffu) + __popc(m_tw & lt_mask);
          prm.tow_tower[at] = tower;
          prm.tow_eta[at] = eta_c;
          prm.tow_phi[at] = phi_c;
          prm.tow_E[at] = em + had;
          prm.tow_Eem[at] = em;
          prm.tow_Ehad[at] = had;
          prm.tow_ET[at] = (em + had) * ic;
        }
        if (f_ph) {
          const int slot = ph_run + (int)(excl_w >> 16) + __popc(m_ph & lt_mask);
          const long long at = base_efl + s_ntrk[e + 1] + s_nnh[e] + slot;
          prm.efl_cls[at] = (signed char)PD_CLS_PHOTON;
          prm.efl_src[at] = tower;
          prm.efl_pt[at] = nem * ic;
          prm.efl_eta[at] = eta_c;
          prm.efl_phi[at] = phi_c;
          prm.efl_E[at] = nem;
        }
        if (f_nh) {
          const int slot = nh_run + (int)excl_n + __popc(m_nh & lt_mask);
          const long long at = base_efl + s_ntrk[e + 1] + s_nph[e + 1] + slot;
          prm.efl_cls[at] = (signed char)PD_CLS_NEUHAD;
          prm.efl_src[at] = tower;
          prm.efl_pt[at] = nhad * ic;
          prm.efl_eta[at] = eta_c;
          prm.efl_phi[at] = phi_c;
          prm.efl_E[at] = nhad;
        }
      }
      tw_run += (int)(tot & 0xffffu);
      ph_run += (int)(tot >> 16);
      nh_run += (int)tot_n;
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

// Tile plan from sizes the host knows (n_events, n_particles): G events per tile so that an average
// tile fills ~85% of the on-chip capacity C.  Small events -> 256-thread CTAs, two per SM;
// large events -> one 512-thread CTA per SM with the whole shared memory.
int pd_plan(const pd_card *c, long long n_events, long long n_particles, PdLaunchPlan *plan) {
  const int nb = c->sc.n_bins;
  const size_t smem_sm = 227 * 1024;  // B200: 227 KB per CTA (opt-in), 228 KB per SM
  const double avg = n_events > 0 ? double(n_particles) / double(n_events) : 0.0;
  auto cap_for = [&](int threads, size_t budget) {
    const size_t fixed = pdk::make_layout(nb, threads, 0).total;
    long cap = budget > fixed + 64 ? long((budget - fixed - 64) / 34) : 0;
    cap = cap > long(threads) * pdk::r_max(threads) ? long(threads) * pdk::r_max(threads) : cap;
    cap = cap > 65535 ? 65535 : cap;
    return int(cap);
  };
  const int c_small = cap_for(256, (228 * 1024 - 2 * 1024) / 2);
  static const int large_threads = std::getenv("PD_LARGE_THREADS") ? std::atoi(std::getenv("PD_LARGE_THREADS")) : 1024;
  const int c_large = cap_for(large_threads, smem_sm);
  const bool small = avg * 1.3 + 64.0 <= double(c_small) * 0.5;
  plan->threads = small ? 256 : large_threads;
  plan->capacity = small ? c_small : c_large;
  long g = 1;
  if (avg > 0.0) {
    // leave head-room of ~4 sigma of a Poisson-like sum
    const double target = double(plan->capacity) - 4.0 * std::sqrt(double(plan->capacity)) - 2.0 * avg;
    g = long(target / avg);
  } else {
    g = pdk::G_MAX;
  }
  g = g < 1 ? 1 : (g > pdk::G_MAX ? pdk::G_MAX : g);
  plan->events_per_tile = int(g);
  plan->n_tiles = int((n_events + g - 1) / g);
  int eb = 0;
  while ((1 << eb) < g) ++eb;
  plan->event_bits = eb;
  plan->smem_bytes = pdk::make_layout(nb, plan->threads, plan->capacity).total;
  plan->grid = 0;
  return PD_OK;
}

template <int THREADS, bool DEBUG>
static int launch_variant(const PdParams &prm, const PdLaunchPlan &plan, cudaStream_t stream) {
  auto kern = pdk::pd_chain_kernel<THREADS, (THREADS == 256 ? 2 : 1), DEBUG>;
  static bool configured = false;
  if (!configured) {
    if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, g_max_smem_optin) != cudaSuccess) return PD_ECUDA;
    configured = true;
  }
  const int per_sm = THREADS == 256 ? 2 : 1;
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
  if (plan.threads == 256) return debug ? launch_variant<256, true>(prm, plan, st) : launch_variant<256, false>(prm, plan, st);
  if (plan.threads == 1024) return debug ? launch_variant<1024, true>(prm, plan, st) : launch_variant<1024, false>(prm, plan, st);
  return debug ? launch_variant<512, true>(prm, plan, st) : launch_variant<512, false>(prm, plan, st);
}
