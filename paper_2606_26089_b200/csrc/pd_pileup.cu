// pd_pileup.cu -- pile-up merging, the step right before the detector-response chain (Listing 8
// L541-567, Table C.9; readings H1-H6 of DESIGN.md section 12).  Product code;
// shares nothing with oracle/.
//   kernel 1 (count)  eight lanes per hard-scatter event: Poisson draw, pool picks, size of the merged event
//   kernel 2 (scan)   exclusive prefix of the sizes = CSR offsets of the output (decoupled look-back over
//                     tiles of 1,024 events claimed from an atomic counter)
//   kernel 3 (fill)   a CTA per event at a time: warp 0 lists the sources (hard scatter, then every picked pool event) and
//                     scans their sizes; the merged event is then written position by position (a position's source by
//                     binary search in the list; coalesced stores), vz shifted by the source's truncated-normal draw,
//                     while warp 0 lists the CTA's next event
// The random numbers are recomputed from their counters where they are needed (Philox4x32-10, stream 2).
#include <cuda_runtime.h>

#include <cstdint>

#include "pd_internal.h"

namespace pdm {

constexpr unsigned long long FLAG_A = 1ull << 62, FLAG_P = 2ull << 62, VAL_MASK = (1ull << 62) - 1;

__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_relaxed(unsigned long long *p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// Philox4x32-10, counter = (block, event lo, event hi, 2 << 16): stream 2 of reading A26
__device__ __forceinline__ void rng_block2(const PdPhiloxKeys &rk, long long event, uint32_t block, uint32_t (&out)[4]) {
  uint32_t c0 = block, c1 = (uint32_t)(unsigned long long)event, c2 = (uint32_t)((unsigned long long)event >> 32), c3 = 2u << 16;
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
    c1 = (uint32_t)p1;
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
    c3 = (uint32_t)p0;
  }
  out[0] = c0, out[1] = c1, out[2] = c2, out[3] = c3;
}

// reading H3: smallest n with sum_{k<=n} p_k > u; explicit round-to-nearest operations in the oracle's order
// (no fused multiply-add), so the integer is the oracle's
__device__ __forceinline__ int poisson_inverse(const PdPileupParams &prm, uint32_t r0) {
  const double u = (double)(r0 >> 8) * (1.0 / 16777216.0);
  double p = prm.p0, cdf = p;
  int n = 0;
  while (!(cdf > u) && n < prm.n_max) {
    ++n;
    p = __ddiv_rn(__dmul_rn(p, prm.mu), (double)n);
    cdf = __dadd_rn(cdf, p);
  }
  return n;
}

// reading H4: truncated normal by inversion, through the lower tail
__device__ __forceinline__ float truncated_normal(float sigma, float phi_lo, float half_minus_lo, uint32_t r1) {
  if (!(sigma > 0.f)) return 0.f;
  // u = (k + 1/2) 2^-24, v = |2u - 1|: 1 - v = (2^24 - |2k + 1 - 2^24|) 2^-24, formed in integers so that the far
  // tail (u next to 0 or 1) keeps its relative precision
  const int k2 = 2 * (int)(r1 >> 8) + 1 - (1 << 24);
  const float t = (float)((1 << 24) - (k2 < 0 ? -k2 : k2)) * 5.9604644775390625e-08f;  // exact
  const float q = fmaf(t, half_minus_lo, phi_lo);
  const float z = -sigma * normcdfinvf(q);
  return k2 < 0 ? -z : z;
}
__device__ __forceinline__ float truncated_z(const PdPileupParams &prm, uint32_t r1) {
  return truncated_normal(prm.sigma_z, prm.phi_lo, prm.half_minus_lo, r1);
}
// reading H7: the time of the interaction, the same way from word 2 (seconds)
__device__ __forceinline__ float truncated_t(const PdPileupParams &prm, uint32_t r2) {
  return truncated_normal(prm.sigma_t, prm.phi_lo_t, prm.half_minus_lo_t, r2);
}

__device__ __forceinline__ long long pool_pick(const PdPileupParams &prm, uint32_t r0) {
  return (long long)(((unsigned long long)(r0 >> 8) * (unsigned long long)prm.n_pool) >> 24);
}

// eight lanes per event: the picks of an event are independent draws, each a chain of dependent loads (pick -> two offsets)
__global__ void __launch_bounds__(256) pd_pileup_count_kernel(const __grid_constant__ PdPileupParams prm) {
  const int sub = threadIdx.x & 7;
  const long long groups = 32LL * gridDim.x;  // groups of eight lanes in the grid
  const long long rounds = (prm.n_hs + groups - 1) / groups;  // the same for every lane: the shuffles below need whole warps
  long long e = blockIdx.x * 32LL + (threadIdx.x >> 3);
  for (long long it = 0; it < rounds; ++it, e += groups) {
    const bool valid = e < prm.n_hs;
    int n = 0;
    long long cnt = 0;
    if (valid) {
      const long long event = prm.event_base + e;
      uint32_t r[4];
      rng_block2(prm.rk, event, 0u, r);
      n = poisson_inverse(prm, r[0]);
      if (sub == 0) cnt = __ldg(prm.hs_off + e + 1) - __ldg(prm.hs_off + e);
      for (int k = sub; k < n; k += 8) {
        rng_block2(prm.rk, event, (uint32_t)(1 + k), r);
        const long long j = pool_pick(prm, r[0]);
        cnt += __ldg(prm.pool_off + j + 1) - __ldg(prm.pool_off + j);
      }
    }
    cnt += __shfl_xor_sync(0xffffffffu, cnt, 1);
    cnt += __shfl_xor_sync(0xffffffffu, cnt, 2);
    cnt += __shfl_xor_sync(0xffffffffu, cnt, 4);
    if (valid && sub == 0) prm.n_pileup[e] = n, prm.cnt[e] = cnt;
  }
}

// exclusive scan of cnt[0..n_hs) into out_off[0..n_hs]
__global__ void __launch_bounds__(256) pd_pileup_scan_kernel(const __grid_constant__ PdPileupParams prm) {
  __shared__ long long s_w[8];
  __shared__ long long s_excl;
  __shared__ unsigned s_tile;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const long long n_tiles = (prm.n_hs + PD_PILEUP_SCAN_TILE - 1) / PD_PILEUP_SCAN_TILE;
  for (;;) {
    __syncthreads();
    if (tid == 0) s_tile = atomicAdd(prm.tile_counter, 1u);
    __syncthreads();
    const long long tile = s_tile;
    if (tile >= n_tiles) break;
    const long long base = tile * PD_PILEUP_SCAN_TILE + 4LL * tid;  // four consecutive events per thread
    long long v[4], sum = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      v[k] = base + k < prm.n_hs ? prm.cnt[base + k] : 0;
      sum += v[k];
    }
    long long incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const long long t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    if (lane == 31) s_w[wid] = incl;
    __syncthreads();
    if (wid == 0) {
      long long w = lane < 8 ? s_w[lane] : 0, wi = w;
#pragma unroll
      for (int o = 1; o < 8; o <<= 1) {
        const long long t = __shfl_up_sync(0xffffffffu, wi, o);
        if (lane >= o) wi += t;
      }
      const long long total = __shfl_sync(0xffffffffu, wi, 7);
      if (lane < 8) s_w[lane] = wi - w;
      unsigned long long excl = 0;
      if (tile == 0) {
        if (lane == 0) st_relaxed(prm.chain, FLAG_P | (unsigned long long)total);
      } else {
        if (lane == 0) st_relaxed(prm.chain + tile, FLAG_A | (unsigned long long)total);
        long long pos = tile - 1;
        for (;;) {
          const long long idx = pos - lane;
          unsigned long long x = FLAG_P;
          if (idx >= 0) {
            x = ld_relaxed(prm.chain + idx);
            while ((x >> 62) == 0) {
              __nanosleep(40);
              x = ld_relaxed(prm.chain + idx);
            }
          }
          const unsigned pm = __ballot_sync(0xffffffffu, (x >> 62) == 2);
          unsigned long long part = x & VAL_MASK;
          if (pm && lane > __ffs(pm) - 1) part = 0;
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
          excl += part;
          if (pm) break;
          pos -= 32;
        }
        if (lane == 0) st_relaxed(prm.chain + tile, FLAG_P | (excl + (unsigned long long)total));
      }
      if (lane == 0) {
        s_excl = (long long)excl;
        if (tile == n_tiles - 1) {
          prm.out_off[prm.n_hs] = (long long)excl + total;
          if ((long long)excl + total > prm.capacity) atomicExch(prm.status_word, (int)PD_ECAPACITY);
        }
      }
    }
    __syncthreads();
    long long run = s_excl + s_w[wid] + incl - sum;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      if (base + k < prm.n_hs) prm.out_off[base + k] = run;
      run += v[k];
    }
  }
}

// A 256-thread CTA per merged event.  Warp 0 lists the event's sources (the hard scatter, then the n picked pool
// events): start and length in their input batch, vertex shift, and -- by a warp scan -- where each lands in the
// output; the warps copy the sources side by side.  The list of a CTA's NEXT event is made (a chain of dependent
// loads: pick -> offsets -> scan, no traffic to speak of) while the other seven warps copy the current one, in a second set
// of list arrays; warp 0 joins the copy when its list is done (sources are handed out by a counter).
constexpr int UNR = 2;            // positions per lane in flight
constexpr int MAX_SOURCES = 768;  // n_max + 1 <= ceil(500 + 10 sqrt(500) + 20) + 1 = 745
struct SourceList {
  long long a[MAX_SOURCES];  // first particle in its input batch
  int ro[MAX_SOURCES];       // first position in the merged event
  float dz[MAX_SOURCES], dt[MAX_SOURCES];
  int total;                 // particles of the merged event
};
__global__ void __launch_bounds__(256) pd_pileup_fill_kernel(const __grid_constant__ PdPileupParams prm) {
  __shared__ SourceList s_list[2];
  __shared__ int s_next[2];  // next source of the list to hand out
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  if (prm.out_off[prm.n_hs] > prm.capacity) return;  // reported by the scan kernel through the status word
  auto list_sources = [&](long long e, SourceList &L) {  // warp 0
    const long long event = prm.event_base + e;
    const int n_src = prm.n_pileup[e] + 1;
    int run = 0;
    for (int s0 = 0; s0 < n_src; s0 += 32) {
      const int s = s0 + lane;  // source s: block s of the event's stream (0 = the hard scatter)
      long long a = 0;
      int len = 0;
      float dz = 0.f, dt = 0.f;
      if (s < n_src) {
        uint32_t r[4];
        rng_block2(prm.rk, event, (uint32_t)s, r);
        if (s == 0) {
          a = __ldg(prm.hs_off + e), len = (int)(__ldg(prm.hs_off + e + 1) - a);
          dz = prm.smear_hs ? truncated_z(prm, r[1]) : 0.f;
          dt = prm.smear_hs ? truncated_t(prm, r[2]) : 0.f;
        } else {
          const long long j = pool_pick(prm, r[0]);
          a = __ldg(prm.pool_off + j), len = (int)(__ldg(prm.pool_off + j + 1) - a);
          dz = truncated_z(prm, r[1]);
          dt = truncated_t(prm, r[2]);
        }
      }
      int incl = len;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      if (s < n_src) L.a[s] = a, L.dz[s] = dz, L.dt[s] = dt, L.ro[s] = run + (incl - len);
      run += __shfl_sync(0xffffffffu, incl, 31);
    }
    if (lane == 0) L.total = run;
  };
  long long e = blockIdx.x;
  if (e >= prm.n_hs) return;
  if (wid == 0) list_sources(e, s_list[0]);
  if (tid == 0) s_next[0] = 0;
  __syncthreads();
  for (int buf = 0; e < prm.n_hs; e += gridDim.x, buf ^= 1) {
    const int n_src = prm.n_pileup[e] + 1;
    const SourceList &L = s_list[buf];
    if (wid == 0) {
      if (e + gridDim.x < prm.n_hs) list_sources(e + gridDim.x, s_list[buf ^ 1]);
      if (lane == 0) s_next[buf ^ 1] = 0;
    }
    // the merged event position by position (every lane busy, stores coalesced), in chunks of 32 * UNR positions handed out by
    // a counter; a position's source is the last one that starts at or before it
    const long long o0 = prm.out_off[e];
    const int total = L.total;
    for (;;) {
      int c = 0;
      if (lane == 0) c = atomicAdd(&s_next[buf], 1);
      c = __shfl_sync(0xffffffffu, c, 0);
      if (c * (32 * UNR) >= total) break;
      int k[UNR], src[UNR];
      long long from[UNR];
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        k[u] = c * (32 * UNR) + u * 32 + lane;
        int lo = 0, hi = n_src;
        const int kk = min(k[u], total - 1);
        while (hi - lo > 1) {
          const int mid = (lo + hi) >> 1;
          if (L.ro[mid] <= kk) lo = mid;
          else hi = mid;
        }
        src[u] = lo, from[u] = L.a[lo] + (kk - L.ro[lo]);
      }
      int v_pid[UNR];
      signed char v_q[UNR];
      float v_f[UNR][7];
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        const bool pu = src[u] > 0;
        v_pid[u] = __ldg((pu ? prm.pool_pid : prm.hs_pid) + from[u]);
        v_q[u] = __ldg((pu ? prm.pool_charge : prm.hs_charge) + from[u]);
#pragma unroll
        for (int f = 0; f < 7; ++f) v_f[u][f] = __ldg((pu ? prm.pool_f[f] : prm.hs_f[f]) + from[u]);
      }
#pragma unroll
      for (int u = 0; u < UNR; ++u) {
        if (k[u] < total) {
          const long long d = o0 + k[u];
          prm.out_pid[d] = v_pid[u];
          prm.out_charge[d] = v_q[u];
#pragma unroll
          for (int f = 0; f < 6; ++f) prm.out_f[f][d] = v_f[u][f];
          prm.out_f[6][d] = v_f[u][6] + L.dz[src[u]];
          prm.is_pu[d] = src[u] > 0 ? 1 : 0;
          if (prm.out_vt) prm.out_vt[d] = L.dt[src[u]];
        }
      }
    }
    __syncthreads();  // the next list is complete, this one no longer read
  }
}

}  // namespace pdm

int pd_launch_pileup(const PdPileupParams &prm, void *stream) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  long long blocks = (prm.n_hs + 31) / 32;  // eight lanes per event
  if (blocks > 8LL * sms) blocks = 8LL * sms;
  if (blocks < 1) blocks = 1;
  pdm::pd_pileup_count_kernel<<<(unsigned)blocks, 256, 0, st>>>(prm);
  if (cudaGetLastError() != cudaSuccess) return PD_ECUDA;
  pdm::pd_pileup_scan_kernel<<<4 * sms, 256, 0, st>>>(prm);
  if (cudaGetLastError() != cudaSuccess) return PD_ECUDA;
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, pdm::pd_pileup_fill_kernel, 256, 0) != cudaSuccess || per_sm < 1) return PD_ECUDA;
  long long fb = prm.n_hs;  // a CTA per event at a time
  if (fb > (long long)per_sm * sms) fb = (long long)per_sm * sms;
  if (fb < 1) fb = 1;
  pdm::pd_pileup_fill_kernel<<<(unsigned)fb, 256, 0, st>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}
