// pd_truth.cu -- truth-level event features: H_T and E_T^miss over the truth collection (Table 2
// "H_T, E_T^miss values for Truth and PFlow collections", L398 "Truth HT"; readings T1, T2
// of DESIGN.md section 15).  Product code; shares nothing with oracle/.
//
// A segmented reduction over the CSR particle arrays, reading px, py, pid (12 B per particle).
// Kernel 1: a CTA walks over CONSECUTIVE tiles of 2,048 particles.  16-byte loads (four adjacent particles per
// thread), issued one tile ahead; (pT, px, py) of the visible particles staged in shared memory.  A tile starts in
// the event the previous one ended in, so one window of 257 offsets, loaded together with the particles, normally
// covers the events it touches (otherwise: a warp-wide 33-ary search for its last event, offsets beyond the window
// from global memory).  Three ways to sum, chosen per tile: fewer than 8 events -> every event's segment is cut into
// 8 pieces, one per warp; 8..31 events -> a warp per event; 32 or more -> a thread per event.  Sums are 64-bit fixed
// point (units of 2^-32 GeV: associative, so the result does not depend on tiles, pieces, batching or the order of
// the atomics) and are added to the event's three accumulators in the workspace with 64-bit atomics.  A tile that lies in
// one or two events (events of thousands of particles) skips the staging: sums in registers, a warp sum, atomics.
// Kernel 2: accumulators -> fp32 outputs.
#include <cuda_runtime.h>

#include <cstdint>
#include <mutex>

#include "pd_internal.h"

namespace pdt {

constexpr int THREADS = 256, W = THREADS / 32, ITEMS = 8, TILE = THREADS * ITEMS;  // ITEMS: a multiple of 4
constexpr double kInvFix = 2.3283064365386963e-10;  // 2^-32

__device__ __forceinline__ long long warp_sum_ll(long long v) {
  const unsigned long long u = (unsigned long long)v;  // pieces of 24 + 24 + 16 bits: 32 of them cannot overflow 32 bits
  const unsigned a = __reduce_add_sync(0xffffffffu, (unsigned)(u & 0xffffffu));
  const unsigned b = __reduce_add_sync(0xffffffffu, (unsigned)((u >> 24) & 0xffffffu));
  const unsigned c = __reduce_add_sync(0xffffffffu, (unsigned)(u >> 48));
  return (long long)((unsigned long long)a + ((unsigned long long)b << 24) + ((unsigned long long)c << 48));
}
__device__ __forceinline__ long long to_fix(float x) { return __float2ll_rn(x * 4294967296.f); }
__device__ __forceinline__ float sqrt_approx(float x) {  // 2 ulp; pT only enters sums compared at 1e-5
  float r;
  asm("sqrt.approx.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// largest e in [lo, hi) with off[e] <= t, by a whole warp: 33-ary narrowing, then halving
__device__ __forceinline__ long long find_event_warp(const long long *off, long long lo, long long hi, long long t, int lane) {
  while (hi - lo > 32) {
    const long long probe = lo + ((hi - lo) * (lane + 1)) / 33;  // lo < probe < hi, non-decreasing in lane
    const unsigned m = __ballot_sync(0xffffffffu, __ldg(off + probe) <= t);  // a prefix of the lanes
    const int k = __popc(m);
    const long long new_lo = k > 0 ? __shfl_sync(0xffffffffu, probe, k - 1) : lo;
    const long long new_hi = k < 32 ? __shfl_sync(0xffffffffu, probe, k & 31) : hi;
    lo = new_lo, hi = new_hi;
  }
  while (hi - lo > 1) {
    const long long mid = (lo + hi) >> 1;
    if (__ldg(off + mid) <= t) lo = mid;
    else hi = mid;
  }
  return lo;
}

// FAST: with the register path for tiles that lie in one or two events (chosen by the host for batches of events of thousands
// of particles; compiled out otherwise: batches of small events lose 30 % to its registers and its two extra loads per tile)
template <bool FAST>
__global__ void __launch_bounds__(THREADS, 4) pd_truth_sum_kernel(const __grid_constant__ PdTruthParams prm) {
  __shared__ __align__(16) float s_pt[TILE], s_px[TILE], s_py[TILE];
  __shared__ int s_off[THREADS + 1];  // offsets of the events e_cur .. e_cur + THREADS, relative to the tile, clamped
  __shared__ long long s_first, s_last;
  __shared__ int s_found;
  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const long long n = prm.n_particles, ne = prm.n_events;
  const long long n_tiles = (n + TILE - 1) / TILE;
  // a CTA takes a contiguous range of tiles, so that the first event of a tile is the last one of the tile before
  const long long per = (n_tiles + gridDim.x - 1) / gridDim.x;
  const long long tile_b = blockIdx.x * per, tile_e = min(tile_b + per, n_tiles);
  if (tile_b >= tile_e) return;
  if (wid == 0) {
    const long long e = find_event_warp(prm.ev_off, 0, ne, tile_b * TILE, lane);
    if (lane == 0) s_first = e;
  }
  __syncthreads();
  long long e_cur = s_first;
  // registers of the tile in flight: its particles (a thread takes groups of four adjacent ones: 16-byte loads when
  // the caller's arrays allow it) and a window of THREADS + 1 offsets starting at its first event
  constexpr int GROUPS = ITEMS / 4;
  float4 r_px[GROUPS], r_py[GROUPS];
  int4 r_pid[GROUPS];
  long long w0, w1, wb = 0, wc = 0;  // wb, wc: where the tile's second and third event start (the same for every thread)
  const bool vec_ok = ((reinterpret_cast<uintptr_t>(prm.px) | reinterpret_cast<uintptr_t>(prm.py) | reinterpret_cast<uintptr_t>(prm.pid)) & 15) == 0;
  auto load_tile = [&](long long tile, long long e_first) {
    const long long t0 = tile * TILE;
    const int len = (int)(min(t0 + (long long)TILE, n) - t0);
#pragma unroll
    for (int g = 0; g < GROUPS; ++g) {
      const int j = (g * THREADS + tid) * 4;
      if (vec_ok && j + 3 < len) {
        r_px[g] = __ldg(reinterpret_cast<const float4 *>(prm.px + t0 + j));
        r_py[g] = __ldg(reinterpret_cast<const float4 *>(prm.py + t0 + j));
        r_pid[g] = __ldg(reinterpret_cast<const int4 *>(prm.pid + t0 + j));
      } else {
        float x[4], y[4];
        int q[4];
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const bool in = j + c < len;
          x[c] = in ? __ldg(prm.px + t0 + j + c) : 0.f, y[c] = in ? __ldg(prm.py + t0 + j + c) : 0.f;
          q[c] = in ? __ldg(prm.pid + t0 + j + c) : 0;
        }
        r_px[g] = make_float4(x[0], x[1], x[2], x[3]), r_py[g] = make_float4(y[0], y[1], y[2], y[3]);
        r_pid[g] = make_int4(q[0], q[1], q[2], q[3]);
      }
    }
    const long long ke = min(e_first + tid, ne);
    w0 = __ldg(prm.ev_off + ke), w1 = __ldg(prm.ev_off + min(ke + 1, ne));
    if (FAST) wb = __ldg(prm.ev_off + min(e_first + 1, ne)), wc = __ldg(prm.ev_off + min(e_first + 2, ne));
  };
  // |pid| in {12, 14, 16} as a bit test (bits 12, 14, 16 of the mask; no bits when neutrinos count)
  const unsigned nu_mask = prm.skip_neutrinos ? 0x15000u : 0u;
  auto visible = [&](int pid) {
    const unsigned a = (unsigned)abs(pid);
    return !(a < 32u && ((nu_mask >> a) & 1u));
  };
  load_tile(tile_b, e_cur);
  for (long long tile = tile_b; tile < tile_e; ++tile) {
    const long long t0 = tile * TILE, t1 = min(t0 + (long long)TILE, n) - 1;
    const int len = (int)(t1 - t0 + 1);
    if (FAST && wc > t1) {
      // ---- the tile lies in one or two events (events of thousands of particles): no staging, no barrier -- every thread sums
      // its eight particles in registers, on the side of the boundary they fall on; a warp sum; three atomics per warp and event
      const int bpos = (int)max(min(wb - t0, (long long)len), 0LL);  // first position of the second event
      long long hA = 0, xA = 0, yA = 0, hB = 0, xB = 0, yB = 0;
#pragma unroll
      for (int g = 0; g < GROUPS; ++g) {
        const int j = (g * THREADS + tid) * 4;  // positions >= len hold zeros
        const float px4[4] = {r_px[g].x, r_px[g].y, r_px[g].z, r_px[g].w}, py4[4] = {r_py[g].x, r_py[g].y, r_py[g].z, r_py[g].w};
        const int pid4[4] = {r_pid[g].x, r_pid[g].y, r_pid[g].z, r_pid[g].w};
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const bool vis = visible(pid4[c]);
          const float x = vis ? px4[c] : 0.f, y = vis ? py4[c] : 0.f;
          const long long fh = to_fix(sqrt_approx(fmaf(x, x, y * y))), fx = to_fix(x), fy = to_fix(y);
          if (j + c < bpos) hA += fh, xA += fx, yA += fy;  // (sums per group of four first, one branch per group: slower, spills)
          else hB += fh, xB += fx, yB += fy;
        }
      }
      const long long e_last = wb <= t1 ? e_cur + 1 : e_cur;
      if (tile + 1 < tile_e) load_tile(tile + 1, e_last);  // in flight during the reductions and the next iteration's start
      hA = warp_sum_ll(hA), xA = warp_sum_ll(xA), yA = warp_sum_ll(yA);
      if (lane < 3) {
        const long long v = lane == 0 ? hA : (lane == 1 ? xA : yA);
        if (v != 0) atomicAdd(prm.acc + 3 * e_cur + lane, (unsigned long long)v);
      }
      if (e_last != e_cur) {
        hB = warp_sum_ll(hB), xB = warp_sum_ll(xB), yB = warp_sum_ll(yB);
        if (lane < 3) {
          const long long v = lane == 0 ? hB : (lane == 1 ? xB : yB);
          if (v != 0) atomicAdd(prm.acc + 3 * e_last + lane, (unsigned long long)v);
        }
      }
      e_cur = e_last;
      continue;
    }
    __syncthreads();  // the previous tile's sums are done with the staging arrays
    if (tid == 0) s_found = 0;
#pragma unroll
    for (int g = 0; g < GROUPS; ++g) {
      const int j = (g * THREADS + tid) * 4;  // positions >= len hold zeros and are never read
      float4 x = r_px[g], y = r_py[g], t;
      if (!visible(r_pid[g].x)) x.x = 0.f, y.x = 0.f;
      if (!visible(r_pid[g].y)) x.y = 0.f, y.y = 0.f;
      if (!visible(r_pid[g].z)) x.z = 0.f, y.z = 0.f;
      if (!visible(r_pid[g].w)) x.w = 0.f, y.w = 0.f;
      t.x = sqrt_approx(fmaf(x.x, x.x, y.x * y.x)), t.y = sqrt_approx(fmaf(x.y, x.y, y.y * y.y));
      t.z = sqrt_approx(fmaf(x.z, x.z, y.z * y.z)), t.w = sqrt_approx(fmaf(x.w, x.w, y.w * y.w));
      *reinterpret_cast<float4 *>(s_px + j) = x, *reinterpret_cast<float4 *>(s_py + j) = y, *reinterpret_cast<float4 *>(s_pt + j) = t;
    }
    s_off[tid] = (int)max(min(w0 - t0, (long long)len), 0LL);
    if (tid == THREADS - 1) s_off[THREADS] = (int)max(min(w1 - t0, (long long)len), 0LL);
    __syncthreads();
    // the event that holds the tile's last particle: in the window unless the tile touches more than THREADS events
    if (e_cur + tid < ne && w0 <= t1 && w1 > t1) s_last = e_cur + tid, s_found = 1;
    __syncthreads();
    if (!s_found) {  // CTA-uniform; rare (events of fewer than 8 particles on average, or runs of empty events)
      if (wid == 0) {
        const long long e = find_event_warp(prm.ev_off, e_cur, ne, t1, lane);
        if (lane == 0) s_last = e;
      }
      __syncthreads();
    }
    const long long e_last = s_last;
    const long long n_ev = e_last - e_cur + 1;  // events e_cur .. e_last
    if (tile + 1 < tile_e) load_tile(tile + 1, e_last);  // in flight while this tile is summed
    auto seg_of = [&](long long e, int &a, int &b) {
      if (e < THREADS) {
        a = s_off[e], b = s_off[e + 1];
      } else {
        a = (int)max(min(__ldg(prm.ev_off + e_cur + e) - t0, (long long)len), 0LL);
        b = (int)max(min(__ldg(prm.ev_off + e_cur + e + 1) - t0, (long long)len), 0LL);
      }
    };
    if (n_ev >= 32) {
      // many small events: a thread per event, sequential sums (no cross-lane work)
      for (long long e = tid; e < n_ev; e += THREADS) {
        int a, b;
        seg_of(e, a, b);
        long long h = 0, x = 0, y = 0;
        for (int j = a; j < b; ++j) h += to_fix(s_pt[j]), x += to_fix(s_px[j]), y += to_fix(s_py[j]);
        if (h != 0) atomicAdd(prm.acc + 3 * (e_cur + e), (unsigned long long)h);
        if (x != 0) atomicAdd(prm.acc + 3 * (e_cur + e) + 1, (unsigned long long)x);
        if (y != 0) atomicAdd(prm.acc + 3 * (e_cur + e) + 2, (unsigned long long)y);
      }
    } else {
      // (event, piece) work items per warp; few events in the tile -> every event's segment is cut into W pieces
      const int sh = n_ev < W ? 3 : 0, P = 1 << sh;  // W = 8 pieces
      static_assert(W == 8, "pieces per event");
      for (int item = wid; item < ((int)n_ev << sh); item += W) {
        const int e = item >> sh, piece = item & (P - 1);
        int a, b;
        seg_of(e, a, b);
        const int seg = b - a;
        const int pa = a + ((seg * piece) >> sh), pb = a + ((seg * (piece + 1)) >> sh);
        if (pb <= pa) continue;  // warp-uniform
        long long h = 0, x = 0, y = 0;
        auto add = [&](int j) { h += to_fix(s_pt[j]), x += to_fix(s_px[j]), y += to_fix(s_py[j]); };
        const int ja = (pa + 3) & ~3, jb = pb & ~3;  // the 16-byte aligned middle [ja, jb)
        if (ja < jb) {
          if (lane < ja - pa) add(pa + lane);
          if (lane < pb - jb) add(jb + lane);
          for (int j = ja + 4 * lane; j < jb; j += 128) {
            const float4 vt = *reinterpret_cast<const float4 *>(s_pt + j), vx = *reinterpret_cast<const float4 *>(s_px + j),
                         vy = *reinterpret_cast<const float4 *>(s_py + j);
            h += to_fix(vt.x) + to_fix(vt.y) + to_fix(vt.z) + to_fix(vt.w);
            x += to_fix(vx.x) + to_fix(vx.y) + to_fix(vx.z) + to_fix(vx.w);
            y += to_fix(vy.x) + to_fix(vy.y) + to_fix(vy.z) + to_fix(vy.w);
          }
        } else {
          for (int j = pa + lane; j < pb; j += 32) add(j);
        }
        h = warp_sum_ll(h), x = warp_sum_ll(x), y = warp_sum_ll(y);
        if (lane < 3) {
          const long long v = lane == 0 ? h : (lane == 1 ? x : y);
          if (v != 0) atomicAdd(prm.acc + 3 * (e_cur + e) + lane, (unsigned long long)v);
        }
      }
    }
    e_cur = e_last;  // it may continue in the next tile
  }
}

__global__ void pd_truth_finish_kernel(const __grid_constant__ PdTruthParams prm) {
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < prm.n_events; e += (long long)gridDim.x * blockDim.x) {
    const double h = (double)(long long)prm.acc[3 * e] * kInvFix;
    const double mx = -(double)(long long)prm.acc[3 * e + 1] * kInvFix, my = -(double)(long long)prm.acc[3 * e + 2] * kInvFix;
    prm.ht[e] = (float)h, prm.met_x[e] = (float)mx, prm.met_y[e] = (float)my;
    prm.met[e] = (float)sqrt(mx * mx + my * my);
  }
}

}  // namespace pdt

int pd_launch_truth(const PdTruthParams &prm, void *stream) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PD_ECUDA;
  cudaStream_t st = (cudaStream_t)stream;
  if (cudaMemsetAsync(prm.acc, 0, 24 * (size_t)prm.n_events, st) != cudaSuccess) return PD_ECUDA;
  if (prm.n_particles > 0) {
    long long blocks = (prm.n_particles + pdt::TILE - 1) / pdt::TILE;
    if (blocks > 4LL * sms) blocks = 4LL * sms;
    if (prm.n_particles >= 2048 * prm.n_events) pdt::pd_truth_sum_kernel<true><<<(unsigned)blocks, pdt::THREADS, 0, st>>>(prm);
    else pdt::pd_truth_sum_kernel<false><<<(unsigned)blocks, pdt::THREADS, 0, st>>>(prm);
    if (cudaGetLastError() != cudaSuccess) return PD_ECUDA;
  }
  long long blocks = (prm.n_events + 255) / 256;
  if (blocks > 4LL * sms) blocks = 4LL * sms;
  pdt::pd_truth_finish_kernel<<<(unsigned)blocks, 256, 0, st>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}

// ---- pd_truth_features_static (pd.h): the entry point that allocates nothing ----------------------------------------
// The accumulators live in a file-scope device array instead of a caller's workspace.  In HOST code the array's name is a
// host-side stand-in, not a device address: the address the kernels get is looked up with cudaGetSymbolAddress, once per
// device, with that device current (every device that loads the library has its own copy of the array).
namespace pdt {
static __device__ __align__(256) unsigned long long g_static_acc[3 * (size_t)PD_TRUTH_STATIC_MAX_EVENTS];
}

namespace {
constexpr int kMaxDevices = 64;
std::mutex g_static_mutex;
unsigned long long *g_static_ptr[kMaxDevices] = {};  // device address of pdt::g_static_acc on device d, once known

// device address of the scratch on the current device; no allocation (the array is part of the loaded module)
int static_scratch(unsigned long long **out) {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return PD_ECUDA;
  if (dev < 0 || dev >= kMaxDevices) return PD_ECUDA;
  std::lock_guard<std::mutex> lock(g_static_mutex);
  if (!g_static_ptr[dev]) {
    unsigned long long *ptr = nullptr;
    if (cudaGetSymbolAddress((void **)&ptr, pdt::g_static_acc) != cudaSuccess || !ptr) return PD_ECUDA;
    g_static_ptr[dev] = ptr;
  }
  *out = g_static_ptr[dev];
  return PD_OK;
}
}  // namespace

extern "C" int pd_truth_features_static(const pd_events *ev, int32_t skip_neutrinos, pd_features *out, void *cuda_stream) {
  if (!ev || !out || ev->n_events < 0 || ev->n_particles < 0) return PD_EINVAL;
  if (ev->n_events > (int64_t)PD_TRUTH_STATIC_MAX_EVENTS) return PD_EWORKSPACE;  // the built-in scratch is too small
  unsigned long long *acc = nullptr;
  const int rs = static_scratch(&acc);  // also for an empty batch: the set-up call
  if (rs != PD_OK) return rs;
  if (ev->n_events == 0) return PD_OK;
  if (!ev->offsets || !out->ht || !out->met_x || !out->met_y || !out->met) return PD_EINVAL;
  if (ev->n_particles > 0 && (!ev->pid || !ev->px || !ev->py)) return PD_EINVAL;
  PdTruthParams p;
  p.n_events = ev->n_events, p.n_particles = ev->n_particles;
  p.ev_off = (const long long *)ev->offsets, p.pid = ev->pid, p.px = ev->px, p.py = ev->py;
  p.skip_neutrinos = skip_neutrinos != 0;
  p.acc = acc;
  p.ht = out->ht, p.met_x = out->met_x, p.met_y = out->met_y, p.met = out->met;
  // clears acc[0 .. 3 n_events) on the stream (the array keeps the last call's contents), then the two kernels
  return pd_launch_truth(p, cuda_stream);
}
