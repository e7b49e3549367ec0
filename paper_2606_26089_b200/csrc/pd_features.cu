// pd_features.cu -- event features (H_T, E_T^miss) and lepton isolation (Eq. 1 of the paper) from an EFlow
// collection: the step right after the detector-response chain (
// readings F1-F4 of DESIGN.md section 10).  Product code; shares nothing with oracle/.
//
// Events are independent and nothing is compacted, so there is no chain and no workspace.  A 256-thread CTA
// (four per SM) walks over chunks of consecutive events (static, strided assignment); inside a chunk it takes
// RUNS of whole events whose objects fit its shared-memory cache (pT, eta, phi, class: 13 bytes per object), so
// the O(leptons x objects) cone sums read shared memory only.  An event larger than the cache is streamed from
// global memory through a second instance of the same code.
//   step 1  objects of the run -> shared memory (coalesced); leptons listed; isolation of non-leptons zeroed
//   step 1b a run that is one big event: counting sort of its object indices by (eta strip, phi cell), both at
//           least dr_max wide, so that a lepton only meets the objects of the 3 x 3 cells around it
//   step 2  H_T and E_T^miss: a warp per event (all warps for one big event), exact 64-bit fixed-point sums
//   step 3  isolation: sixteen lanes per lepton over its candidate objects in the cache (a warp per lepton, lanes over the
//           objects, for an event streamed from global memory), three exact fixed-point sums
// Fixed-point sums (units of 2^-32 GeV) are associative: results do not depend on the order of the objects,
// the chunking or the launch shape.
#include <cuda_runtime.h>

#include <cstdint>

#include "pd_internal.h"

namespace pdf {

constexpr int THREADS = 256;
constexpr int W = THREADS / 32;
constexpr int CAP = 3072;         // objects cached per run
constexpr int RUN_EVENTS = 256;   // events per run at most
constexpr int N_STRIPS = 32;      // eta strips of a big event (cone pre-selection)
constexpr int N_PHI_MAX = 12;     // phi cells per strip at most
constexpr int N_CELLS = N_STRIPS * N_PHI_MAX;
constexpr int STRIP_MIN_OBJECTS = 512;
constexpr int SMEM_BYTES = 17 * CAP;  // pT, eta, phi (4 B each), lepton list, strip list (2 B each), class (1 B)
constexpr float kPi = 3.14159265358979323846f;
constexpr float kTwoPi = 6.28318530717958647692f;
constexpr double kInvFix = 2.3283064365386963e-10;  // 2^-32

// Sum of a 64-bit integer over the warp (two's complement, modulo 2^64) with three integer REDUX instructions
// instead of ten dependent shuffles: pieces of 24 + 24 + 16 bits cannot overflow 32 bits when 32 of them are added.
__device__ __forceinline__ long long warp_sum_ll(long long v) {
  const unsigned long long u = (unsigned long long)v;
  const unsigned a = __reduce_add_sync(0xffffffffu, (unsigned)(u & 0xffffffu));
  const unsigned b = __reduce_add_sync(0xffffffffu, (unsigned)((u >> 24) & 0xffffffu));
  const unsigned c = __reduce_add_sync(0xffffffffu, (unsigned)(u >> 48));
  return (long long)((unsigned long long)a + ((unsigned long long)b << 24) + ((unsigned long long)c << 48));
}
__device__ __forceinline__ long long to_fix(float x) { return __float2ll_rn(x * 4294967296.f); }
// eta strip of an object: N_STRIPS strips of width 1 / inv_strip >= dr_max from eta = -6, the outer ones open-ended
__device__ __forceinline__ int eta_strip(float eta, float inv_strip) {
  return min(max((int)floorf((eta + 6.f) * inv_strip), 0), N_STRIPS - 1);
}
// phi cell: n_phi cells of width 2 pi / n_phi >= dr_max over [-pi, pi]
__device__ __forceinline__ int phi_cell(float phi, const PdFeatParams &prm) {
  return min(max((int)floorf((phi + kPi) * prm.inv_phi_cell), 0), prm.n_phi - 1);
}

// Steps 2 and 3 for one run.  Two instances: the objects in shared memory (plain LDS addressing) or, for an event
// larger than the cache, in global memory.
template <typename PF, typename PC>
__device__ __forceinline__ void run_features(const PdFeatParams &prm, PF o_pt, PF o_eta, PF o_phi, PC o_cls, const int *s_off,
                                             unsigned long long *s_acc, const unsigned short *s_lep, int n_lep, const unsigned short *s_idx,
                                             const unsigned short *s_cstart, int ne, int n, long long e0, long long a0) {
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  // ---- step 2: H_T and E_T^miss.  A run that is one big event: all warps share it (integer atomics in
  // shared memory); otherwise a warp per event.
  if (ne == 1 && n > 8 * 32) {
    long long s_ht = 0, s_x = 0, s_y = 0;
    for (int i = tid; i < n; i += THREADS) {
      const float pt = o_pt[i];
      float sn, cs;
      sincosf(o_phi[i], &sn, &cs);
      s_ht += to_fix(pt), s_x += to_fix(pt * cs), s_y += to_fix(pt * sn);
    }
    s_ht = warp_sum_ll(s_ht), s_x = warp_sum_ll(s_x), s_y = warp_sum_ll(s_y);
    if (lane == 0) {
      atomicAdd(&s_acc[0], (unsigned long long)s_ht);
      atomicAdd(&s_acc[1], (unsigned long long)s_x);
      atomicAdd(&s_acc[2], (unsigned long long)s_y);
    }
  } else if (ne >= 8 && n < 48 * ne) {
    // small events: eight lanes per event, four events per warp pass (the lanes stay busy, and the fold and the
    // epilogue in double are shared by four events)
    const int grp = lane >> 3, gl = lane & 7;
    for (int e4 = 4 * wid; e4 < ne; e4 += 4 * W) {
      const int e = e4 + grp;
      long long s_ht = 0, s_x = 0, s_y = 0;
      if (e < ne)
        for (int i = s_off[e] + gl; i < s_off[e + 1]; i += 8) {
          const float pt = o_pt[i];
          float sn, cs;
          sincosf(o_phi[i], &sn, &cs);
          s_ht += to_fix(pt), s_x += to_fix(pt * cs), s_y += to_fix(pt * sn);
        }
      __syncwarp();
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) {
        s_ht += __shfl_xor_sync(0xffffffffu, s_ht, o);
        s_x += __shfl_xor_sync(0xffffffffu, s_x, o);
        s_y += __shfl_xor_sync(0xffffffffu, s_y, o);
      }
      if (e < ne && gl == 0) {
        const double mx = -(double)s_x * kInvFix, my = -(double)s_y * kInvFix;
        prm.ht[e0 + e] = (float)((double)s_ht * kInvFix);
        prm.met_x[e0 + e] = (float)mx, prm.met_y[e0 + e] = (float)my;
        prm.met[e0 + e] = (float)sqrt(mx * mx + my * my);
      }
    }
  } else
  for (int e = wid; e < ne; e += W) {
    long long s_ht = 0, s_x = 0, s_y = 0;
    for (int i = s_off[e] + lane; i < s_off[e + 1]; i += 32) {
      const float pt = o_pt[i];
      float sn, cs;
      sincosf(o_phi[i], &sn, &cs);
      s_ht += to_fix(pt), s_x += to_fix(pt * cs), s_y += to_fix(pt * sn);
    }
    s_ht = warp_sum_ll(s_ht), s_x = warp_sum_ll(s_x), s_y = warp_sum_ll(s_y);
    if (lane == 0) {
      const double mx = -(double)s_x * kInvFix, my = -(double)s_y * kInvFix;
      prm.ht[e0 + e] = (float)((double)s_ht * kInvFix);
      prm.met_x[e0 + e] = (float)mx, prm.met_y[e0 + e] = (float)my;
      prm.met[e0 + e] = (float)sqrt(mx * mx + my * my);
    }
  }

  // ---- step 3: Eq. 1, a warp per lepton, lanes over the objects of its event
  auto isolate = [&](int i, int ea, int eb) {
    const float eta_i = o_eta[i], phi_i = o_phi[i];
    long long s_ch = 0, s_nh = 0, s_ph = 0;
    auto scan = [&](int lo, int hi, bool listed) {
      for (int jj = lo + lane; jj < hi; jj += 32) {
        const int j = listed ? (int)s_idx[jj] : jj;
        const float deta = o_eta[j] - eta_i;
        float dphi = o_phi[j] - phi_i;
        dphi = dphi > kPi ? dphi - kTwoPi : (dphi <= -kPi ? dphi + kTwoPi : dphi);
        const float dr2 = fmaf(deta, deta, dphi * dphi);
        if (dr2 < prm.dr_max2 && j != i) {  // rare (the cone is ~1 % of the acceptance): the sums stay off the common path
          const int cj = (int)o_cls[j];
          const long long fx = to_fix(o_pt[j]);
          if (cj <= PD_CLS_MUON) s_ch += fx;
          else if (cj == PD_CLS_NEUHAD) s_nh += fx;
          else if (!(dr2 < prm.fsr2)) s_ph += fx;
        }
      }
    };
    if (s_idx != nullptr) {
      // one big event, its objects listed by (eta strip, phi cell), strips and cells at least dr_max wide: only the
      // lepton's strip and its two neighbours, and in each its phi cell and the two next to it (cyclically), can hold
      // objects of the cone; the cells of a strip are contiguous in the list
      const int st = eta_strip(eta_i, prm.inv_strip), pc = phi_cell(phi_i, prm), np = prm.n_phi;
      for (int s2 = max(st - 1, 0); s2 <= min(st + 1, N_STRIPS - 1); ++s2) {
        const unsigned short *row = s_cstart + s2 * N_PHI_MAX;  // row[c] = first list position of cell c; row[np] = end of the strip
        if (np <= 3) {
          scan(row[0], row[np], true);
        } else if (pc == 0) {
          scan(row[0], row[2], true), scan(row[np - 1], row[np], true);
        } else if (pc == np - 1) {
          scan(row[0], row[1], true), scan(row[np - 2], row[np], true);
        } else {
          scan(row[pc - 1], row[pc + 2], true);
        }
      }
    } else {
      scan(ea, eb, false);
    }
    s_ch = warp_sum_ll(s_ch), s_nh = warp_sum_ll(s_nh), s_ph = warp_sum_ll(s_ph);
    if (lane == 0) {
      prm.iso_charged[a0 + i] = (float)((double)s_ch * kInvFix);
      prm.iso_neutral[a0 + i] = (float)((double)s_nh * kInvFix);
      prm.iso_photon[a0 + i] = (float)((double)s_ph * kInvFix);
      prm.r_iso[a0 + i] = (float)((double)(s_ch + s_nh + s_ph) * kInvFix / (double)o_pt[i]);
    }
  };
  if (s_lep != nullptr) {
    // cached run: the leptons were listed by step 1.  SIXTEEN LANES per lepton (two leptons per warp pass) walk over the
    // candidates of a big event in shared memory -- the objects of the 3 x 3 cells around it (a hundred or so), as ONE
    // index space over the (up to four) contiguous pieces of the cell list, so that the lanes stay full and the two
    // halves of a warp run the same loop; the three sums are folded with four shuffle steps.  The event of a lepton is
    // found by bisection of the run's offsets.
    // (eight lanes per lepton, four leptons per pass, when the candidates are the few objects of a small event)
    const bool listed = s_idx != nullptr;
    const int GL = listed ? 16 : 8, per_warp = 32 / GL;
    const int grp = lane / GL, gl = lane & (GL - 1);
    for (int k0 = 0; k0 < n_lep; k0 += per_warp * W) {
      const int k = k0 + per_warp * wid + grp;
      const bool active = k < n_lep;
      const int i = active ? (int)s_lep[k] : 0;
      const float eta_i = o_eta[i], phi_i = o_phi[i];
      // pieces [b0, b0 + n0), [b1, ...), ...: positions in s_idx (listed) or object indices (one event of a multi-event run)
      int b0 = 0, n0 = 0, b1 = 0, n1 = 0, b2 = 0, n2 = 0, b3 = 0;
      if (active) {
        if (listed) {
          const int st = eta_strip(eta_i, prm.inv_strip), pc = phi_cell(phi_i, prm), np = prm.n_phi;
          const bool wrap = np > 3 && (pc == 0 || pc == np - 1);
          // per strip: cells [lo, hi) around pc, clipped; a lepton in the first / last phi cell also takes the cell at the
          // other end: since the strips follow one another in the list, that cell of strip s and the first cells of strip s + 1
          // are not adjacent, so it gets a piece of its own only in the lepton's strip... keep it simple: three pieces for the
          // clipped windows, and the wrap-around cells of all three strips scanned as extra pieces one after the other below
          const int s_lo = max(st - 1, 0), s_hi = min(st + 1, N_STRIPS - 1);
          const int c_lo = np <= 3 ? 0 : max(pc - 1, 0), c_hi = np <= 3 ? np : min(pc + 2, np);
          const unsigned short *r0 = s_cstart + s_lo * N_PHI_MAX;
          b0 = r0[c_lo], n0 = r0[c_hi] - b0;
          if (s_lo + 1 <= s_hi) {
            const unsigned short *r1 = r0 + N_PHI_MAX;
            b1 = r1[c_lo], n1 = r1[c_hi] - b1;
          }
          if (s_lo + 2 <= s_hi) {
            const unsigned short *r2 = r0 + 2 * N_PHI_MAX;
            b2 = r2[c_lo], n2 = r2[c_hi] - b2;
          }
          if (wrap) {
            // the cell at the other end of the phi range, strip by strip, through the fourth piece
            const int wc = pc == 0 ? np - 1 : 0;
            b3 = -1 - wc;  // marker: handled by the loop below
          }
        } else {
          int lo = 0, hi = ne;  // s_off[lo] <= i < s_off[hi]
          while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (s_off[mid] <= i) lo = mid;
            else hi = mid;
          }
          b0 = s_off[lo], n0 = s_off[lo + 1] - b0;
        }
      }
      long long s_ch = 0, s_nh = 0, s_ph = 0;
      auto test = [&](int j) {
        const float deta = o_eta[j] - eta_i;
        float dphi = o_phi[j] - phi_i;
        dphi = dphi > kPi ? dphi - kTwoPi : (dphi <= -kPi ? dphi + kTwoPi : dphi);
        const float dr2 = fmaf(deta, deta, dphi * dphi);
        if (dr2 < prm.dr_max2 && j != i) {
          const int cj = (int)o_cls[j];
          const long long fx = to_fix(o_pt[j]);
          if (cj <= PD_CLS_MUON) s_ch += fx;
          else if (cj == PD_CLS_NEUHAD) s_nh += fx;
          else if (!(dr2 < prm.fsr2)) s_ph += fx;
        }
      };
      const int n01 = n0 + n1, n012 = n01 + n2;
      for (int v = gl; v < n012; v += GL) {
        const int pos = v < n0 ? b0 + v : (v < n01 ? b1 + (v - n0) : b2 + (v - n01));
        test(listed ? (int)s_idx[pos] : pos);
      }
      if (b3 < 0) {
        const int wc = -1 - b3;
        const int st = eta_strip(eta_i, prm.inv_strip);
        for (int s2 = max(st - 1, 0); s2 <= min(st + 1, N_STRIPS - 1); ++s2) {
          const unsigned short *row = s_cstart + s2 * N_PHI_MAX;
          for (int pos = row[wc] + gl; pos < row[wc + 1]; pos += 16) test((int)s_idx[pos]);
        }
      }
      __syncwarp();
      if (listed) s_ch += __shfl_xor_sync(0xffffffffu, s_ch, 8), s_nh += __shfl_xor_sync(0xffffffffu, s_nh, 8), s_ph += __shfl_xor_sync(0xffffffffu, s_ph, 8);
#pragma unroll
      for (int o = 4; o > 0; o >>= 1) {
        s_ch += __shfl_xor_sync(0xffffffffu, s_ch, o);
        s_nh += __shfl_xor_sync(0xffffffffu, s_nh, o);
        s_ph += __shfl_xor_sync(0xffffffffu, s_ph, o);
      }
      if (active && gl == 0) {
        prm.iso_charged[a0 + i] = (float)((double)s_ch * kInvFix);
        prm.iso_neutral[a0 + i] = (float)((double)s_nh * kInvFix);
        prm.iso_photon[a0 + i] = (float)((double)s_ph * kInvFix);
        prm.r_iso[a0 + i] = (float)((double)(s_ch + s_nh + s_ph) * kInvFix / (double)o_pt[i]);
      }
    }
  } else {
    // an event larger than the cache: every warp looks for the leptons among its share of the objects
    for (int i = wid; i < n; i += W) {
      const signed char ci = o_cls[i];
      if (ci == PD_CLS_ELECTRON || ci == PD_CLS_MUON) isolate(i, 0, n);
    }
  }
}

__global__ void __launch_bounds__(THREADS, 4) pd_features_kernel(const __grid_constant__ PdFeatParams prm,
                                                                 int events_per_chunk, long long n_chunks) {
  extern __shared__ __align__(16) unsigned char fsm[];
  float *s_pt = (float *)fsm, *s_eta = s_pt + CAP, *s_phi = s_eta + CAP;
  unsigned short *s_lep = (unsigned short *)(s_phi + CAP);  // the run's leptons (indices into the cache), in arrival order
  unsigned short *s_idx = s_lep + CAP;                       // a big event's objects listed by eta strip
  signed char *s_cls = (signed char *)(s_idx + CAP);
  __shared__ int s_off[RUN_EVENTS + 1];
  __shared__ int s_ccnt[N_CELLS];                 // objects per (strip, phi cell), then running write positions
  __shared__ unsigned short s_cstart[N_CELLS + 1];  // first list position of every cell
  __shared__ unsigned s_nlep;
  __shared__ unsigned long long s_acc[3];  // H_T, sum pT cos, sum pT sin of a run that is one big event
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;

  const long long n_total = __ldg(prm.offsets + prm.n_events);
  // bulk prefetches want 16-byte aligned addresses: true for every array of the collection or not used at all
  const bool pf_ok = ((((uintptr_t)prm.pt | (uintptr_t)prm.eta | (uintptr_t)prm.phi | (uintptr_t)prm.cls) & 15) == 0);
  for (long long chunk = blockIdx.x; chunk < n_chunks; chunk += gridDim.x) {
    const long long c0 = chunk * events_per_chunk;
    const long long c1 = min(c0 + (long long)events_per_chunk, prm.n_events);
    long long e0 = c0;
    while (e0 < c1) {
      // ---- the run [e0, e0 + ne): as many whole events as fit the cache (offsets are non-decreasing)
      const long long a0 = __ldg(prm.offsets + e0);
      bool fits_t = false;
      if (e0 + tid + 1 <= c1) fits_t = __ldg(prm.offsets + e0 + tid + 1) - a0 <= (long long)CAP;
      int ne = __syncthreads_count(fits_t);
      const bool cached = ne > 0;  // else: one event larger than the cache, streamed from global memory
      if (!cached) ne = 1;
      if (tid < 3) s_acc[tid] = 0ull;
      if (tid == 3) s_nlep = 0u;
      for (int c = tid; c < N_CELLS; c += THREADS) s_ccnt[c] = 0;
      for (int e = tid; e <= ne; e += THREADS) s_off[e] = (int)min(__ldg(prm.offsets + e0 + e) - a0, (long long)0x7fffffff);
      __syncthreads();
      const int n = s_off[ne];

      // ---- step 1: cache the run; zero the isolation of everything that is not a lepton.  Four objects per thread at a
      // time, all their loads issued before the first store (the stores would otherwise fence the loads of the next
      // iteration: the phase is bound by memory latency)
      if (tid == 0) {
        // the objects that follow (the next run of this chunk, most of the time) towards L2 meanwhile
        const long long nb = a0 + n, ne_ = min(nb + (long long)n, n_total);
        const long long lo4 = (nb + 3) & ~3ll, hi4 = ne_ & ~3ll, lo16 = (nb + 15) & ~15ll, hi16 = ne_ & ~15ll;
        if (pf_ok && hi4 > lo4) {
          const unsigned bytes = (unsigned)(4 * (hi4 - lo4));
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(prm.pt + lo4), "r"(bytes) : "memory");
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(prm.eta + lo4), "r"(bytes) : "memory");
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(prm.phi + lo4), "r"(bytes) : "memory");
        }
        if (pf_ok && hi16 > lo16)
          asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(prm.cls + lo16), "r"((unsigned)(hi16 - lo16)) : "memory");
      }
      for (int i0 = tid; i0 < n; i0 += 4 * THREADS) {
        signed char c[4];
        float vp[4], ve[4], vf[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int i = i0 + u * THREADS;
          c[u] = 0, vp[u] = ve[u] = vf[u] = 0.f;
          if (i < n) {
            c[u] = __ldg(prm.cls + a0 + i);
            if (cached) vp[u] = __ldg(prm.pt + a0 + i), ve[u] = __ldg(prm.eta + a0 + i), vf[u] = __ldg(prm.phi + a0 + i);
          }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int i = i0 + u * THREADS;
          if (i < n) {
            if (cached) s_cls[i] = c[u], s_pt[i] = vp[u], s_eta[i] = ve[u], s_phi[i] = vf[u];
            if (c[u] == PD_CLS_ELECTRON || c[u] == PD_CLS_MUON) {
              if (cached) s_lep[atomicAdd(&s_nlep, 1u)] = (unsigned short)i;
            } else {
              prm.iso_charged[a0 + i] = 0.f, prm.iso_neutral[a0 + i] = 0.f, prm.iso_photon[a0 + i] = 0.f;
              prm.r_iso[a0 + i] = 0.f;
            }
          }
        }
      }
      __syncthreads();
      const bool strips = cached && ne == 1 && n >= STRIP_MIN_OBJECTS;
      if (strips) {
        // counting sort of the event's object indices by (eta strip, phi cell) (integer atomics; the order inside a
        // cell is arbitrary and irrelevant: the cone sums are exact)
        for (int i = tid; i < n; i += THREADS)
          atomicAdd(&s_ccnt[eta_strip(s_eta[i], prm.inv_strip) * N_PHI_MAX + phi_cell(s_phi[i], prm)], 1);
        __syncthreads();
        if (wid == 0) {
          constexpr int PER = N_CELLS / 32;  // 12 consecutive cells per lane
          int v[PER], sum = 0;
#pragma unroll
          for (int k = 0; k < PER; ++k) v[k] = s_ccnt[lane * PER + k], sum += v[k];
          int incl = sum;
#pragma unroll
          for (int o = 1; o < 32; o <<= 1) {
            const int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
          }
          int run = incl - sum;
#pragma unroll
          for (int k = 0; k < PER; ++k) {
            s_cstart[lane * PER + k] = (unsigned short)run, s_ccnt[lane * PER + k] = run;
            run += v[k];
          }
          if (lane == 31) s_cstart[N_CELLS] = (unsigned short)run;
        }
        __syncthreads();
        for (int i = tid; i < n; i += THREADS)
          s_idx[atomicAdd(&s_ccnt[eta_strip(s_eta[i], prm.inv_strip) * N_PHI_MAX + phi_cell(s_phi[i], prm)], 1)] = (unsigned short)i;
        __syncthreads();
      }

      if (cached) run_features(prm, (const float *)s_pt, (const float *)s_eta, (const float *)s_phi, (const signed char *)s_cls, s_off, s_acc, s_lep, (int)s_nlep,
                               strips ? (const unsigned short *)s_idx : (const unsigned short *)nullptr, s_cstart, ne, n, e0, a0);
      else run_features(prm, prm.pt + a0, prm.eta + a0, prm.phi + a0, prm.cls + a0, s_off, s_acc, (const unsigned short *)nullptr, 0, (const unsigned short *)nullptr, s_cstart,
                        ne, n, e0, a0);
      __syncthreads();  // the cache is reused by the next run
      if (ne == 1 && n > 8 * 32 && tid == 0) {
        const double mx = -(double)(long long)s_acc[1] * kInvFix, my = -(double)(long long)s_acc[2] * kInvFix;
        prm.ht[e0] = (float)((double)(long long)s_acc[0] * kInvFix);
        prm.met_x[e0] = (float)mx, prm.met_y[e0] = (float)my;
        prm.met[e0] = (float)sqrt(mx * mx + my * my);
      }
      e0 += ne;
    }
  }
}

}  // namespace pdf

int pd_launch_features(const PdFeatParams &prm, void *stream) {
  if (prm.n_events <= 0) return PD_OK;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  const long long ctas = 4LL * sms;
  // chunks of consecutive events, about eight per resident CTA, at most one run's worth of events each
  long long epc = (prm.n_events + 8 * ctas - 1) / (8 * ctas);
  if (epc < 1) epc = 1;
  if (epc > pdf::RUN_EVENTS) epc = pdf::RUN_EVENTS;
  const long long n_chunks = (prm.n_events + epc - 1) / epc;
  const long long grid = n_chunks < ctas ? n_chunks : ctas;
  // per launch, not once per process: the attribute belongs to the current device's copy of the kernel
  if (cudaFuncSetAttribute(pdf::pd_features_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, pdf::SMEM_BYTES) != cudaSuccess) return PD_ECUDA;
  pdf::pd_features_kernel<<<(unsigned)grid, pdf::THREADS, pdf::SMEM_BYTES, (cudaStream_t)stream>>>(prm, (int)epc, n_chunks);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}
