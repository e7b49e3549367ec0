// pd_impact.cu -- track impact parameters d0, z0 and their errors (Table 2;
// SURVEY.md 8f NEXT-3; readings I1..I3 of DESIGN.md section 14).  Product code; shares nothing with oracle/.
//
// A thread takes four adjacent output tracks of a pd_simulate call (16-byte loads of trk.src, 16-byte stores of the
// four outputs).  The event of a track (needed for the Philox counter and for the particle's index within its
// event) comes from the track offsets: two warps find the events of the first and the last track of a 1,024-track
// tile by a 33-ary search, the offsets in between are staged in shared memory relative to the tile, and a thread
// bisects them once for its first track and walks forward for the other three.  The truth particle is gathered
// through trk.src (ascending inside an event, so the gathers of a warp fall into a few cache lines); all loads of a
// thread are issued before anything is computed.
//
// Geometry in fp32, arranged so that nothing cancels (frame: p^ along the transverse momentum, n^ to its left):
//   w = v . p^, u = v . n^ (both from error-free products), helix centre c = (w, u + s rho), r_c = |c|,
//   d0 = s (rho - r_c) = -(2 rho u + s r0^2) / (rho + r_c),   alpha_d = atan2(-w, rho + s u),
//   z0 = v_z + rho alpha_d p_z / p_T;     straight line (q B = 0): d0 = -u, z0 = v_z - w p_z / p_T.
#include <cuda_runtime.h>

#include <cstdint>

#include "pd_internal.h"
#include "pd_impact_math.cuh"

namespace pdi {

constexpr int THREADS = 256, ITEMS = 4, TILE = THREADS * ITEMS;  // ITEMS = 4: the 16-byte vectors below
constexpr int OFF_CACHE = 2048;  // staged track offsets per CTA (events touched by a tile, + 1)

// largest e in [lo, hi) with off[e] <= t (off non-decreasing, off[lo] <= t < off[hi])
template <typename P>
__device__ __forceinline__ long long find_event(P off, long long lo, long long hi, long long t) {
  while (hi - lo > 1) {
    const long long mid = (lo + hi) >> 1;
    if ((long long)off[mid] <= t) lo = mid;
    else hi = mid;
  }
  return lo;
}

// the same by a whole warp: 33-ary narrowing (one round trip to L2 per round instead of one per halving)
__device__ __forceinline__ long long find_event_warp(const long long *off, long long lo, long long hi, long long t, int lane) {
  while (hi - lo > 1) {
    const long long span = hi - lo;
    const long long probe = lo + (span * (lane + 1)) / 33;  // lo <= probe < hi, non-decreasing in lane
    const bool le = probe > lo ? (__ldg(off + probe) <= t) : true;
    const unsigned m = __ballot_sync(0xffffffffu, le);  // a prefix of the lanes (off is non-decreasing)
    const int k = __popc(m);                             // >= 0; lanes 0..k-1 hold off[probe] <= t
    const long long new_lo = k > 0 ? __shfl_sync(0xffffffffu, probe, k - 1) : lo;
    const long long new_hi = k < 32 ? __shfl_sync(0xffffffffu, probe, k & 31) : hi;
    if (new_lo == lo && new_hi == hi) break;  // span < 33 and no probe fell strictly inside: finish by halving
    lo = new_lo, hi = new_hi;
  }
  return find_event(off, lo, hi, t);
}

__global__ void __launch_bounds__(THREADS, 4) pd_impact_kernel(const __grid_constant__ PdImpactParams prm) {
  __shared__ int s_off[OFF_CACHE];  // track offsets of the tile's events, relative to the tile's first track
  __shared__ long long s_range[2];
  const int tid = threadIdx.x;
  const long long n_trk = __ldg(prm.trk_off + prm.n_events);
  const long long n_tiles = (n_trk + TILE - 1) / TILE;
  // 16-byte vectors only if the caller's arrays are aligned for them
  const bool vec_ok = ((reinterpret_cast<uintptr_t>(prm.trk_src) | reinterpret_cast<uintptr_t>(prm.d0) | reinterpret_cast<uintptr_t>(prm.z0) |
                        reinterpret_cast<uintptr_t>(prm.d0_err) | reinterpret_cast<uintptr_t>(prm.z0_err)) & 15) == 0;
  for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
    const long long t0 = tile * TILE, t1 = min(t0 + (long long)TILE, n_trk) - 1;
    __syncthreads();
    if (tid < 64) {
      const long long e = find_event_warp(prm.trk_off, 0, prm.n_events, tid < 32 ? t0 : t1, tid & 31);
      if ((tid & 31) == 0) s_range[tid >> 5] = e;
    }
    __syncthreads();
    const long long e_lo = s_range[0], e_hi = s_range[1] + 1;  // events e_lo .. e_hi-1; offsets e_lo .. e_hi
    const int n_ev = (int)min(e_hi - e_lo, (long long)OFF_CACHE);
    const bool staged = e_hi - e_lo + 1 <= OFF_CACHE;
    if (staged)
      for (int k = tid; k <= n_ev; k += THREADS)
        s_off[k] = (int)max(min(__ldg(prm.trk_off + e_lo + k) - t0, (long long)TILE), -1LL);  // only order matters outside [0, TILE)
    __syncthreads();
    // a thread takes ITEMS ADJACENT tracks: one search for the first, a short walk for the others; src and the four
    // outputs move as 16-byte vectors.  All loads are issued before anything is computed.
    const long long tb = t0 + (long long)ITEMS * tid;
    if (tb > t1) continue;
    const bool full = vec_ok && tb + ITEMS - 1 <= t1;
    int i_[ITEMS], ob_[ITEMS], q_[ITEMS];
    long long e_[ITEMS];
    float px_[ITEMS], py_[ITEMS], pz_[ITEMS], vx_[ITEMS], vy_[ITEMS], vz_[ITEMS];
    if (full) {
      const int4 v = __ldg(reinterpret_cast<const int4 *>(prm.trk_src + tb));
      i_[0] = v.x, i_[1] = v.y, i_[2] = v.z, i_[3] = v.w;
    } else {
#pragma unroll
      for (int k = 0; k < ITEMS; ++k) i_[k] = __ldg(prm.trk_src + min(tb + k, t1));
    }
    if (staged) {
      int e = (int)find_event(s_off, 0, (long long)n_ev, (long long)(ITEMS * tid));
#pragma unroll
      for (int k = 0; k < ITEMS; ++k) {
        const int tl = min(ITEMS * tid + k, (int)(t1 - t0));
        while (s_off[e + 1] <= tl) ++e;  // skips empty events; s_off[n_ev] > tl
        e_[k] = e_lo + e;
      }
    } else {
#pragma unroll
      for (int k = 0; k < ITEMS; ++k) e_[k] = find_event(prm.trk_off, e_lo, e_hi, min(tb + k, t1));
    }
#pragma unroll
    for (int k = 0; k < ITEMS; ++k) {
      const int i = i_[k];
      px_[k] = __ldg(prm.px + i), py_[k] = __ldg(prm.py + i), pz_[k] = __ldg(prm.pz + i);
      vx_[k] = __ldg(prm.vx + i), vy_[k] = __ldg(prm.vy + i), vz_[k] = __ldg(prm.vz + i);
      q_[k] = __ldg(prm.charge + i);
      ob_[k] = i - (int)__ldg(prm.ev_off + e_[k]);
    }
    float o_d0[ITEMS], o_z0[ITEMS], o_sd[ITEMS], o_sz[ITEMS];
    const pdk::ImpactCfg cfg{prm.inv_kB, prm.sB, prm.d0_a, prm.d0_b, prm.z0_a, prm.z0_b};
#pragma unroll
    for (int k = 0; k < ITEMS; ++k)
      pdk::track_impact(cfg, prm.rk, prm.event_base + e_[k], (uint32_t)ob_[k], q_[k], px_[k], py_[k], pz_[k], vx_[k], vy_[k], vz_[k], o_d0[k],
                        o_z0[k], o_sd[k], o_sz[k]);
    if (full) {
      *reinterpret_cast<float4 *>(prm.d0 + tb) = make_float4(o_d0[0], o_d0[1], o_d0[2], o_d0[3]);
      *reinterpret_cast<float4 *>(prm.z0 + tb) = make_float4(o_z0[0], o_z0[1], o_z0[2], o_z0[3]);
      *reinterpret_cast<float4 *>(prm.d0_err + tb) = make_float4(o_sd[0], o_sd[1], o_sd[2], o_sd[3]);
      *reinterpret_cast<float4 *>(prm.z0_err + tb) = make_float4(o_sz[0], o_sz[1], o_sz[2], o_sz[3]);
    } else {
#pragma unroll
      for (int k = 0; k < ITEMS; ++k)
        if (tb + k <= t1) prm.d0[tb + k] = o_d0[k], prm.z0[tb + k] = o_z0[k], prm.d0_err[tb + k] = o_sd[k], prm.z0_err[tb + k] = o_sz[k];
    }
  }
}

}  // namespace pdi

int pd_launch_impact(const PdImpactParams &prm, void *stream) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  // tiles are taken round-robin; the track total lives on the device, so the grid is sized by the bound n_particles
  long long blocks = (prm.n_particles + pdi::TILE - 1) / pdi::TILE;
  if (blocks > 8LL * sms) blocks = 8LL * sms;
  if (blocks < 1) blocks = 1;
  pdi::pd_impact_kernel<<<(unsigned)blocks, pdi::THREADS, 0, (cudaStream_t)stream>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}
