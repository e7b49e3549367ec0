// pd_filter.cu -- the particle filter of the paper's post-processing (Table C.13;
// SURVEY.md 8f NEXT-4) as an ordered stream compaction of an EFlow collection.  Product code; shares nothing
// with oracle/.
//
// Kernel 1 (persistent CTAs, four per SM, tiles of 2,048 objects claimed from an atomic counter so that a tile's
// predecessors are always running or done): the six arrays of the tile come into shared memory by bulk copies
// (cp.async.bulk + mbarrier: no registers held, no load instructions); then: evaluate the conditions (exact fp32
// comparisons, the conditions' constants prepared once per CTA), rank the survivors inside the tile with warp ballots
// and one 64-entry scan, chain the tiles with a decoupled look-back (one self-flagged 64-bit word per tile), scatter
// the survivors from shared memory to their final place, and record, per 32 input positions, the survivor bits and
// the exclusive rank of the first -- including the word of the position one past the last object, whose rank is the
// total.  Kernel 2: the CSR offsets of the output are the ranks at the input offsets (one such word per event).
//
// What bounds it (profiles/r02g_cfg2_filter_full.txt): the wait for the predecessors' counts in the look-back, i.e. the
// spread of the tiles' load latencies -- a tile is resident for ~12 us, 4 x 43 KB per SM.  Tried and slower: a second
// stage per CTA filled ahead (a tile that is claimed but not yet counted holds up every later tile: 0.50-1.0 ms
// against 0.26), wider look-back windows (LB below).
#include <cuda_runtime.h>

#include <cstdint>

#include "pd_internal.h"
#include "pd_scan.cuh"

namespace pdx {

constexpr int THREADS = 256, W = THREADS / 32, ITEMS = PD_FILTER_TILE / THREADS;
static_assert(ITEMS * W == 64, "the scan of the (row, warp) counts takes two per lane");
constexpr unsigned long long FLAG_A = 1ull << 62, FLAG_P = 2ull << 62, VAL_MASK = (1ull << 62) - 1;

__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long *p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_relaxed(unsigned long long *p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}

// A condition in the form the rows are tested in: keep = neg != any_k ((x > v_k && gt) || (x == v_k && eq) || (x < v_k && lt)),
// x the field (its magnitude if use_abs) -- >=, <= are two of the three, != and "not in" the negations of == and "in" (so that a
// NaN fails every ordered comparison and passes != / "not in", as the C operators do)
struct Cond {
  int field, nv;
  unsigned abs_mask;
  bool gt, eq, lt, neg;
  float v[PD_MAX_SET_VALUES];
};
__device__ __forceinline__ void make_cond(const pd_condition &c, Cond &o) {
  o.field = c.field, o.abs_mask = c.use_abs ? 0x7fffffffu : 0xffffffffu;
  const bool set = c.op == PD_OP_IN || c.op == PD_OP_NOT_IN;
  o.nv = set ? c.n_values : 1;
  for (int k = 0; k < PD_MAX_SET_VALUES; ++k) o.v[k] = set ? c.values[k] : c.value;
  o.gt = c.op == PD_OP_GT || c.op == PD_OP_GE;
  o.lt = c.op == PD_OP_LT || c.op == PD_OP_LE;
  o.eq = c.op == PD_OP_GE || c.op == PD_OP_LE || c.op == PD_OP_EQ || c.op == PD_OP_NE || set;
  o.neg = c.op == PD_OP_NE || c.op == PD_OP_NOT_IN;
}

// one stage of shared memory: the six arrays of a tile, each at a multiple of 16 bytes
struct Stage {
  float pt[PD_FILTER_TILE], eta[PD_FILTER_TILE], phi[PD_FILTER_TILE], E[PD_FILTER_TILE];
  int src[PD_FILTER_TILE];
  signed char cls[PD_FILTER_TILE];
};
constexpr int NS = 1;  // stages per CTA
constexpr int LB = 1;  // look-back: chain words per lane and round trip (measured on cfg2's EFlow: 1 / 2 / 4 / 8 -> 0.264 / 0.283 / 0.292 / 0.337 ms)
constexpr unsigned STAGE_BYTES = 21u * PD_FILTER_TILE;
static_assert(sizeof(Stage) == STAGE_BYTES && STAGE_BYTES % 16 == 0 && NS == 1, "stage layout");

__global__ void __launch_bounds__(THREADS, 4) pd_filter_kernel(const __grid_constant__ PdFilterParams prm) {
  extern __shared__ __align__(128) unsigned char smem[];
  Stage *stages = reinterpret_cast<Stage *>(smem);
  __shared__ unsigned s_w[ITEMS * W];  // survivors per (row, warp), then their exclusive prefix
  __shared__ unsigned long long s_bcast;
  __shared__ long long s_tile[NS];
  __shared__ __align__(8) uint64_t s_bar[NS][2];  // [0]: the fields the conditions test (copied first), [1]: the other fields
  __shared__ Cond s_cond[PD_MAX_CONDITIONS];
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  const long long n = __ldg(prm.offsets + prm.n_events);          // objects of the input collection
  const long long n_tiles = (n + 1 + PD_FILTER_TILE - 1) / PD_FILTER_TILE;  // positions 0..n inclusive
  // a tile whose 2,048 positions are all objects comes by bulk copies (if the arrays are 16-byte aligned); the last one or two by plain loads
  auto bulk = [&](long long tile) { return prm.aligned16 && (tile + 1) * PD_FILTER_TILE <= n; };
  auto request = [&](int s) {  // one thread: claim the next tile for stage s and start its copies
    const long long tile = (long long)atomicAdd(prm.tile_counter, 1u);
    s_tile[s] = tile;
    if (tile < n_tiles && bulk(tile)) {
      const long long base = tile * PD_FILTER_TILE;
      Stage &st = stages[s];
      pdk::fence_async_smem();  // the stage was last read through the generic proxy
      // the fields the conditions test first, on a barrier of their own: the tile is counted (and its count published, which is
      // what every later tile waits for) while the other fields are still on their way
      const void *srcs[6] = {prm.pt + base, prm.eta + base, prm.phi + base, prm.E + base, prm.cls + base, prm.src + base};
      void *dsts[6] = {st.pt, st.eta, st.phi, st.E, st.cls, st.src};
      unsigned bytes0 = 0, bytes1 = 0;
#pragma unroll
      for (int f = 0; f < 6; ++f) {
        const unsigned b = f == 4 ? 1u * PD_FILTER_TILE : 4u * PD_FILTER_TILE;
        if ((prm.cond_fields >> f) & 1u) bytes0 += b;
        else bytes1 += b;
      }
      pdk::mbar_expect_tx(&s_bar[s][0], bytes0);
      pdk::mbar_expect_tx(&s_bar[s][1], bytes1);
#pragma unroll
      for (int f = 0; f < 6; ++f)
        if ((prm.cond_fields >> f) & 1u) pdk::bulk_g2s(dsts[f], srcs[f], f == 4 ? 1u * PD_FILTER_TILE : 4u * PD_FILTER_TILE, &s_bar[s][0]);
#pragma unroll
      for (int f = 0; f < 6; ++f)
        if (!((prm.cond_fields >> f) & 1u)) pdk::bulk_g2s(dsts[f], srcs[f], f == 4 ? 1u * PD_FILTER_TILE : 4u * PD_FILTER_TILE, &s_bar[s][1]);
    }
  };
  if (tid >= 32 && tid < 32 + prm.n_conds) make_cond(prm.conds[tid - 32], s_cond[tid - 32]);
  if (tid == 0) {
    for (int s = 0; s < NS; ++s) pdk::mbar_init(&s_bar[s][0], 1), pdk::mbar_init(&s_bar[s][1], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    request(0);
  }
  __syncthreads();
  unsigned phase = 0;  // bit s: parity of the next completion of stage s's barrier
  for (int it = 0;; ++it) {
    const int s = it % NS;
    const long long tile = s_tile[s];
    if (tile >= n_tiles) break;  // claimed in increasing order: the other stages hold later tiles
    const long long base = tile * PD_FILTER_TILE;
    Stage &st = stages[s];
    if (bulk(tile)) {
      pdk::mbar_wait(&s_bar[s][0], (phase >> s) & 1u);
    } else {
      for (int i = tid; i < PD_FILTER_TILE; i += THREADS) {
        const long long p = base + i;
        if (p < n) {
          st.pt[i] = __ldg(prm.pt + p), st.eta[i] = __ldg(prm.eta + p), st.phi[i] = __ldg(prm.phi + p), st.E[i] = __ldg(prm.E + p);
          st.src[i] = __ldg(prm.src + p), st.cls[i] = __ldg(prm.cls + p);
        }
      }
      // (row k of a thread is what the same thread loaded: no barrier needed before the predicate)
    }
    // ---- the predicate: condition by condition (its constants in registers), the thread's ITEMS rows each (row k =
    // positions base + k * THREADS + tid); one bit per row
    unsigned valid = 0;
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) valid |= (base + k * THREADS + tid < n ? 1u : 0u) << k;
    unsigned all_bits = valid, any_bits = 0;
    for (int c = 0; c < prm.n_conds; ++c) {
      const Cond &cd = s_cond[c];
      const int field = cd.field, nv = cd.nv;
      const unsigned abs_mask = cd.abs_mask;
      const bool gt = cd.gt, eq = cd.eq, lt = cd.lt;
      const float *col = st.pt + (field < 4 ? field : 0) * PD_FILTER_TILE;  // pt, eta, phi, E are consecutive
      unsigned bits = 0;
#pragma unroll
      for (int k = 0; k < ITEMS; ++k) {
        const int i = k * THREADS + tid;
        const float x = __uint_as_float(__float_as_uint(field < 4 ? col[i] : (float)st.cls[i]) & abs_mask);
        bool any = false;
        if (nv == 1) {
          const float v = cd.v[0];
          any = (x > v && gt) || (x == v && eq) || (x < v && lt);
        } else {
          for (int j = 0; j < nv; ++j) any = any || x == cd.v[j];
        }
        bits |= (any ? 1u : 0u) << k;
      }
      if (cd.neg) bits = ~bits;
      all_bits &= bits, any_bits |= bits;
    }
    const unsigned keep_bits = prm.n_conds == 0 ? valid : (prm.combine_any ? any_bits & valid : all_bits);
    unsigned ballots[ITEMS];
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      ballots[k] = __ballot_sync(0xffffffffu, (keep_bits >> k) & 1u);
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
      if (lane == 0) {
        st_relaxed(prm.chain + tile, (tile == 0 ? FLAG_P : FLAG_A) | total);
      }
      if (tile != 0) {
        // a window of 32 * LB predecessors per round trip (a lane takes LB consecutive ones, nearest first)
        long long pos = tile - 1;
        for (;;) {
          unsigned long long v[LB];
#pragma unroll
          for (int j = 0; j < LB; ++j) {
            const long long idx = pos - (long long)lane * LB - j;
            v[j] = idx >= 0 ? ld_relaxed(prm.chain + idx) : FLAG_P;  // before the first tile: prefix 0
          }
          unsigned long long part = 0;
          bool found = false;
#pragma unroll
          for (int j = 0; j < LB; ++j) {
            if (!found) {
              const long long idx = pos - (long long)lane * LB - j;
              while ((v[j] >> 62) == 0) {
                __nanosleep(40);
                v[j] = ld_relaxed(prm.chain + idx);
              }
              part += v[j] & VAL_MASK;
              found = (v[j] >> 62) == 2;
            }
          }
          const unsigned pm = __ballot_sync(0xffffffffu, found);
          if (pm) {
            const int first = __ffs(pm) - 1;  // the lane holding the nearest inclusive prefix
            if (lane > first) part = 0;
          }
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
          excl += part;
          if (pm) break;
          pos -= 32 * LB;
        }
        if (lane == 0) st_relaxed(prm.chain + tile, FLAG_P | (excl + total));
      }
      if (lane == 0) s_bcast = excl;
    }
    __syncthreads();
    const long long tile_excl = (long long)s_bcast;
    if (bulk(tile)) {  // the other fields
      pdk::mbar_wait(&s_bar[s][1], (phase >> s) & 1u);
      phase ^= 1u << s;
    }
    // ---- survivors to their final place; per 32 positions: the survivor bits and the rank of the first
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      const int i = k * THREADS + tid;
      const long long p = base + i;
      const long long r0 = tile_excl + s_w[k * W + wid];
      if (lane == 0 && p <= n) prm.wordrank[p >> 5] = ((unsigned long long)r0 << 32) | ballots[k];
      if ((keep_bits >> k) & 1u) {
        const long long r = r0 + __popc(ballots[k] & lt_mask);
        prm.out_cls[r] = st.cls[i];
        prm.out_src[r] = st.src[i];
        prm.out_pt[r] = st.pt[i], prm.out_eta[r] = st.eta[i];
        prm.out_phi[r] = st.phi[i], prm.out_E[r] = st.E[i];
      }
    }
    __syncthreads();  // the stage and s_w are free again
    // (the next tile is claimed only now: a tile that is claimed but not yet counted holds up every later one)
    if (tid == 0) request(0);
    __syncthreads();
  }
}

// out_offsets[e] = rank of input position offsets[e] (the rank of position n is the total): the rank of its word's first
// position plus the survivors before it in the word
__global__ void pd_filter_offsets_kernel(const __grid_constant__ PdFilterParams prm) {
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e <= prm.n_events; e += (long long)gridDim.x * blockDim.x)
  {
    const long long p = __ldg(prm.offsets + e);
    const unsigned long long w = prm.wordrank[p >> 5];
    prm.out_offsets[e] = (long long)(w >> 32) + __popc((unsigned)w & ((1u << (p & 31)) - 1u));
  }
}

}  // namespace pdx

int pd_launch_filter(const PdFilterParams &prm, void *stream) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  // tiles are claimed dynamically, so any grid works: as many CTAs as fit (two per SM with two 42 KB stages each)
  const size_t smem = sizeof(pdx::Stage) * pdx::NS;
  auto kern = pdx::pd_filter_kernel;
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem) != cudaSuccess) return PD_ECUDA;
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, pdx::THREADS, smem) != cudaSuccess || per_sm < 1) return PD_ECUDA;
  kern<<<per_sm * sms, pdx::THREADS, smem, (cudaStream_t)stream>>>(prm);
  if (cudaGetLastError() != cudaSuccess) return PD_ECUDA;
  long long blocks = (prm.n_events + 1 + 255) / 256;
  if (blocks > 4LL * sms) blocks = 4LL * sms;
  pdx::pd_filter_offsets_kernel<<<(unsigned)blocks, 256, 0, (cudaStream_t)stream>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}
