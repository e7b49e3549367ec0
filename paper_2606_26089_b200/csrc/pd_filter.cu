// pd_filter.cu -- the particle filter of the paper's post-processing (Table C.13;
// SURVEY.md 8f NEXT-4) as an ordered stream compaction of an EFlow collection.  Product code; shares nothing
// with oracle/.
//
// Kernel 1 (persistent CTAs, tiles of 2,048 objects claimed from an atomic counter so that a tile's
// predecessors are always running or done): evaluate the conditions (exact fp32 comparisons), rank the
// survivors inside the tile with warp ballots and one 64-entry scan, chain the tiles with a decoupled
// look-back (one self-flagged 64-bit word per tile), scatter the survivors to their final place, and record the
// exclusive rank of EVERY input position -- including the position one past the last object, whose rank is the
// total.  Kernel 2: the CSR offsets of the output are the ranks at the input offsets.
#include <cuda_runtime.h>

#include <cstdint>

#include "pd_internal.h"

namespace pdx {

constexpr int THREADS = 256, W = THREADS / 32, ITEMS = PD_FILTER_TILE / THREADS;
constexpr unsigned long long FLAG_A = 1ull << 62, FLAG_P = 2ull << 62, VAL_MASK = (1ull << 62) - 1;

__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_relaxed(unsigned long long *p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

__device__ __forceinline__ bool holds(const pd_condition &c, float x) {
  if (c.use_abs) x = fabsf(x);
  switch (c.op) {
    case PD_OP_GT: return x > c.value;
    case PD_OP_GE: return x >= c.value;
    case PD_OP_LT: return x < c.value;
    case PD_OP_LE: return x <= c.value;
    case PD_OP_EQ: return x == c.value;
    case PD_OP_NE: return x != c.value;
    default: {
      bool in = false;
      for (int k = 0; k < c.n_values; ++k) in = in || x == c.values[k];
      return c.op == PD_OP_IN ? in : !in;
    }
  }
}

__global__ void __launch_bounds__(THREADS, 3) pd_filter_kernel(const __grid_constant__ PdFilterParams prm) {
  __shared__ unsigned s_w[ITEMS * W];  // survivors per (row, warp), then their exclusive prefix
  __shared__ unsigned long long s_bcast[2];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  const long long n = __ldg(prm.offsets + prm.n_events);          // objects of the input collection
  const long long n_tiles = (n + 1 + PD_FILTER_TILE - 1) / PD_FILTER_TILE;  // positions 0..n inclusive
  for (;;) {
    __syncthreads();
    if (tid == 0) s_bcast[0] = atomicAdd(prm.tile_counter, 1u);
    __syncthreads();
    const long long tile = (long long)s_bcast[0];
    if (tile >= n_tiles) break;
    const long long base = tile * PD_FILTER_TILE;
    // ---- all fields of the tile's objects into registers first (row k = positions base + k * THREADS + tid:
    // coalesced; 48 independent loads in flight per thread), then the predicate, row by row
    float f_pt[ITEMS], f_eta[ITEMS], f_phi[ITEMS], f_E[ITEMS];
    int f_src[ITEMS];
    signed char f_cls[ITEMS];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      const long long p = base + k * THREADS + tid;
      if (p < n) {
        f_pt[k] = __ldg(prm.pt + p), f_eta[k] = __ldg(prm.eta + p), f_phi[k] = __ldg(prm.phi + p), f_E[k] = __ldg(prm.E + p);
        f_src[k] = __ldg(prm.src + p), f_cls[k] = __ldg(prm.cls + p);
      }
    }
    unsigned keep_bits = 0, ballots[ITEMS];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      const long long p = base + k * THREADS + tid;
      bool keep = false;
      if (p < n) {
        int n_true = 0;
        for (int c = 0; c < prm.n_conds; ++c) {
          const pd_condition &cd = prm.conds[c];
          const float x = cd.field == PD_FIELD_PT    ? f_pt[k]
                          : cd.field == PD_FIELD_ETA ? f_eta[k]
                          : cd.field == PD_FIELD_PHI ? f_phi[k]
                          : cd.field == PD_FIELD_E   ? f_E[k]
                                                     : (float)f_cls[k];
          n_true += holds(cd, x) ? 1 : 0;
        }
        keep = prm.n_conds == 0 || (prm.combine_any ? n_true > 0 : n_true == prm.n_conds);
      }
      ballots[k] = __ballot_sync(0xffffffffu, keep);
      keep_bits |= (keep ? 1u : 0u) << k;
      if (lane == 0) s_w[k * W + wid] = (unsigned)__popc(ballots[k]);
    }
    __syncthreads();
    // ---- exclusive scan of the ITEMS * W = 64 (row, warp) counts in position order; tile total; look-back
    if (wid == 0) {
      const unsigned a = s_w[2 * lane], b = s_w[2 * lane + 1];
      unsigned incl = a + b;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
      }
      const unsigned total = __shfl_sync(0xffffffffu, incl, 31);
      s_w[2 * lane] = incl - a - b, s_w[2 * lane + 1] = incl - b;
      unsigned long long excl = 0;
      if (tile == 0) {
        if (lane == 0) st_relaxed(prm.chain, FLAG_P | total);
      } else {
        if (lane == 0) st_relaxed(prm.chain + tile, FLAG_A | total);
        long long pos = tile - 1;
        for (;;) {
          const long long idx = pos - lane;
          unsigned long long v = FLAG_P;  // before the first tile: prefix 0
          if (idx >= 0) {
            v = ld_relaxed(prm.chain + idx);
            while ((v >> 62) == 0) {
              __nanosleep(40);
              v = ld_relaxed(prm.chain + idx);
            }
          }
          const unsigned pm = __ballot_sync(0xffffffffu, (v >> 62) == 2);
          unsigned long long part = v & VAL_MASK;
          if (pm) {
            const int first = __ffs(pm) - 1;  // nearest predecessor holding an inclusive prefix
            if (lane > first) part = 0;
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
          excl += part;
          if (pm) break;
          pos -= 32;
        }
        if (lane == 0) st_relaxed(prm.chain + tile, FLAG_P | (excl + total));
      }
      if (lane == 0) s_bcast[1] = excl;
    }
    __syncthreads();
    const long long tile_excl = (long long)s_bcast[1];
    // ---- ranks of all positions, survivors to their final place
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      const long long p = base + k * THREADS + tid;
      if (p > n) continue;
      const long long r = tile_excl + s_w[k * W + wid] + __popc(ballots[k] & lt_mask);
      prm.rank[p] = (int)r;
      if ((keep_bits >> k) & 1u) {
        prm.out_cls[r] = f_cls[k];
        prm.out_src[r] = f_src[k];
        prm.out_pt[r] = f_pt[k], prm.out_eta[r] = f_eta[k];
        prm.out_phi[r] = f_phi[k], prm.out_E[r] = f_E[k];
      }
    }
  }
}

// out_offsets[e] = rank of input position offsets[e] (the rank of position n is the total)
__global__ void pd_filter_offsets_kernel(const __grid_constant__ PdFilterParams prm) {
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e <= prm.n_events; e += (long long)gridDim.x * blockDim.x)
    prm.out_offsets[e] = (long long)prm.rank[__ldg(prm.offsets + e)];
}

}  // namespace pdx

int pd_launch_filter(const PdFilterParams &prm, void *stream) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  // tiles are claimed dynamically, so any grid works; three CTAs of 256 threads per SM at ~80 registers
  pdx::pd_filter_kernel<<<3 * sms, pdx::THREADS, 0, (cudaStream_t)stream>>>(prm);
  if (cudaGetLastError() != cudaSuccess) return PD_ECUDA;
  long long blocks = (prm.n_events + 1 + 255) / 256;
  if (blocks > 4LL * sms) blocks = 4LL * sms;
  pdx::pd_filter_offsets_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}
