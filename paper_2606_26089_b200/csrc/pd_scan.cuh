// pd_scan.cuh -- warp scans, the decoupled look-back chain, the warp-wide search and the bulk-copy primitives shared by the kernels
// of the chain (pd_particles.cu, pd_towers.cu).  Device only; product code (shares nothing with oracle/).
#pragma once

#include <cstdint>

namespace pdk {

constexpr unsigned long long FLAG_A = 1ull << 62, FLAG_P = 2ull << 62, VAL_MASK = (1ull << 62) - 1;

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

__device__ __forceinline__ unsigned warp_incl_scan(unsigned v) {
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const unsigned t = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

// Decoupled look-back over tiles that are claimed in order from an atomic counter (so every predecessor of a
// running tile is running or done), split in two: chain_publish() makes the tile's aggregate visible as soon as
// it is known; chain_resolve() (one full warp, later) returns the exclusive prefix over all earlier tiles to
// every lane and publishes the inclusive prefix.  One 64-bit self-flagged word per tile (zero = not yet
// published).  All resident CTAs run nearly in phase, so the nearest predecessor already holding an inclusive
// prefix is typically a whole grid back: the warp looks at LB_K * 32 predecessors per round trip to L2.
// Packed fields of the value add independently.
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
          __nanosleep(64);
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

// Number of entries of the non-decreasing array a[0..n) that are < key (lower bound), found by one full warp
// with a 33-ary search: every round the 32 lanes probe 32 equally spaced entries of the current range.
__device__ __forceinline__ long long warp_lower_bound(const long long *a, long long n, long long key) {
  const int lane = threadIdx.x & 31;
  long long lo = 0, hi = n;  // answer in [lo, hi]
  while (hi - lo > 0) {
    const long long span = hi - lo;
    const long long step = (span + 32) / 33;  // >= 1
    const long long idx = lo + (long long)(lane + 1) * step - 1;  // probes lo+step-1, lo+2step-1, ...
    const bool below = idx < hi ? (__ldg(a + idx) < key) : false;
    const unsigned m = __ballot_sync(0xffffffffu, below);  // monotone: a prefix of the lanes
    const int c = __popc(m);
    // entries up to probe c-1 are < key; probe c (if inside) is >= key
    const long long new_lo = lo + (long long)c * step;
    const long long new_hi = c < 32 ? min(hi, lo + (long long)(c + 1) * step - 1) : hi;
    lo = min(new_lo, hi), hi = new_hi;
  }
  return lo;
}

// ---- mbarrier / bulk-copy primitives (PTX; SASS: SYNCS.*, UBLKCP) --------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
// global -> shared, bytes a multiple of 16, both addresses 16-byte aligned; completes on the mbarrier
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}
// global -> L2 only (no destination): bytes a multiple of 16, address 16-byte aligned
__device__ __forceinline__ void l2_prefetch(const void *src, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(bytes) : "memory");
}
// shared -> global (bulk async-group)
__device__ __forceinline__ void bulk_s2g(void *dst, const void *src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(smem_u32(src)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
// orders this thread's generic-proxy accesses to shared memory before later async-proxy (bulk copy) accesses
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

}  // namespace pdk
