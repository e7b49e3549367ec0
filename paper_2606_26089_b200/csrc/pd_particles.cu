// pd_particles.cu -- kernel P of the chain: the per-particle half (steps S0-S4 of SURVEY.md section 8a, and the
// track half of S8), as a FLAT pass over the particle arrays: tiles of PT_TILE consecutive particles, whatever
// events they belong to, so there is no limit on the size of an event.
//
// Why flat: the chain is bound by instruction issue, and with one thread per particle in particle order a warp
// runs the helix, the straight line, the Philox block and the smear for whoever needs them (17.6 of 32 lanes
// active in round 1).  Here a tile's inputs are staged in shared memory by bulk asynchronous copies
// (cp.async.bulk, one elected thread, completion on an mbarrier), the particles are split by CLASS into index
// lists -- A: charged inside the tracker acceptance (efficiency > 0: helix + Philox + accept + smear), B: other
// charged (helix only), N: neutral (straight line) -- and the lists are processed by full warps gathering from
// shared memory.  An accepted track is smeared on the spot (its Philox block is in registers) and its record PARKED at
// once in the workspace, compacted at the start of the warp's segment of PD_PSEG particles in particle order (the rank
// of a track among its segment's tracks is a running count over the rows of list A), with the segment's accepted bits
// beside them.  Nothing here depends on another tile: no chain, no waiting.  Kernel T,
// which works event by event and knows where an event's tracks go, moves them into the Track collection.
//
// What the tower pass (pd_towers.cu) needs besides: a 16-bit key per particle (tower id | HCAL bit, 0xffff = no
// deposit), written to the workspace by the warp that owns the particle.
#include <cuda_runtime.h>

#include <algorithm>
#include <cstdint>
#include <cstdlib>
#include <type_traits>

#include "pd_internal.h"
#include "pd_impact_math.cuh"
#include "pd_math.cuh"
#include "pd_scan.cuh"

namespace pdk {

constexpr int PT_THREADS = 256;
constexpr int PT_WARPS = PT_THREADS / 32;
constexpr int PT_TILE = PD_PTILE;  // particles per tile (pd_internal.h); a multiple of 32
constexpr int PT_WORDS = PT_TILE / 32;
constexpr uint32_t PT_NONE = 0xffffu;
static_assert(PT_TILE % 32 == 0 && PT_TILE <= 2048, "list entries keep the particle in 11 bits");

// Shared-memory carve-up of kernel P: the per-particle arrays sit at compile-time offsets (their addresses fold into
// the instructions), the card tables behind them at offsets that depend on the card.
constexpr int PT_PER_WARP = PT_TILE / PT_WARPS;  // particles a warp owns: a multiple of 32
constexpr int PT_ITERS = PT_PER_WARP / 32;
static_assert(PT_PER_WARP % 32 == 0 && PT_PER_WARP <= 255, "a warp owns whole 32-particle rows; ranks fit 8 bits");
constexpr int PT_WCAP = 384;                                // event offsets of a tile kept on chip (more: looked up in global memory)
constexpr size_t PO_F = 0;                                  // px, py, pz, vx, vy, vz: 6 x 4 B x TILE
constexpr size_t PO_PID = PO_F + 6 * 4 * (size_t)PT_TILE;   // 4 B x TILE
constexpr size_t PO_Q = PO_PID + 4 * (size_t)PT_TILE;       // 1 B x TILE
constexpr size_t PO_KEY = PO_Q + (size_t)PT_TILE;           // 2 B x TILE: the particle's key for the tower pass
constexpr size_t PO_LIST = PO_KEY + 2 * (size_t)PT_TILE;    // 2 B x TILE: class lists (per warp: A | B | N), then its tracks in order
constexpr size_t PO_MASK = PO_LIST + 2 * (size_t)PT_TILE;   // accepted bits
constexpr size_t PO_PRE = PO_MASK + 4 * (size_t)PT_WORDS;   // their prefix per word, within the owning warp
constexpr size_t PO_WOFF = (PO_PRE + 4 * (size_t)PT_WORDS + 15) & ~size_t(15);  // event offsets of the tile, relative to its start
constexpr size_t PO_MISC = PO_WOFF + 4 * (size_t)PT_WCAP;
constexpr size_t PO_TABLES = PO_MISC + 8 * 24;
static_assert(PO_PID % 16 == 0 && PO_Q % 16 == 0 && PO_KEY % 16 == 0 && PO_LIST % 16 == 0, "bulk copies need 16-byte aligned slots");

struct PTables {
  size_t tb, binrec, lut, total;
};
__host__ __device__ inline PTables make_ptables(int n_bins, int n_tb, int lut_cells) {
  PTables l;
  size_t o = PO_TABLES;
  auto take = [&](size_t bytes) {
    size_t at = o;
    o = (o + bytes + 15) & ~size_t(15);
    return at;
  };
  l.tb = take(4 * (size_t)n_tb);
  l.binrec = take(16 * (size_t)n_bins);  // per bin: inv_w, half, offset | nphi << 16, pad
  l.lut = take(2 * (size_t)lut_cells);
  l.total = o;
  return l;
}

// S4 with the per-bin record in one 16-byte load: tower of the hit (u, phi), -1 outside the grid.  g: the grid the deposit is
// looked up in (0 ECAL, 1 HCAL: reading K6; on a card with one grid both describe it)
__device__ __forceinline__ int hit_tower_rec(const PdCardScalars &sc, int g, const float *tb_all, const float4 *rec_all,
                                             const unsigned short *lut_all, float u, float phi) {
  if (!(u >= sc.g_tb_first[g]) || !(u < sc.g_tb_last[g])) return -1;
  const float *tb = tb_all + sc.g_tb_off[g];
  const int side = sc.g_lut_side[g];
  int ca = (__float_as_int(fabsf(u)) >> PD_LUT_SHIFT) - sc.g_lut_base[g];
  ca = min(max(ca, 0), side - 1);
  const int cell = u < 0.f ? side - 1 - ca : side + ca;
  int b = lut_all[sc.g_lut_off[g] + cell];
  while (u >= tb[b + 1]) ++b;  // terminates: u < tb[last]
  const float4 r = rec_all[sc.g_bin_off[g] + b];
  const int on = __float_as_int(r.z);
  const int n = on >> 16;
  int j = (int)floorf(fmaf(phi, r.x, r.y)) + (n >> 1);
  j = j < 0 ? 0 : j;
  j = j > n - 1 ? n - 1 : j;
  return (on & 0xffff) + j;
}

// For every tile boundary j (the first particle of tile j; the call's first particle for j = 0): the first event whose
// offset is >= that particle, and the last one whose offset is <= it (= the event the particle belongs to).
__global__ void pd_tile_events_kernel(const long long *offsets, long long n_events, long long p_base, int n_ptiles, int *out) {
  const int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j > n_ptiles) return;
  const long long s = j == 0 ? p_base : (p_base & ~15ll) + (long long)j * PT_TILE;
  long long lo = 0, hi = n_events + 1;  // first entry >= s
  while (lo < hi) {
    const long long mid = (lo + hi) >> 1;
    if (__ldg(offsets + mid) < s) lo = mid + 1;
    else hi = mid;
  }
  out[2 * j] = (int)lo;
  hi = n_events + 1;  // first entry > s (from lo on)
  while (lo < hi) {
    const long long mid = (lo + hi) >> 1;
    if (__ldg(offsets + mid) <= s) lo = mid + 1;
    else hi = mid;
  }
  out[2 * j + 1] = (int)lo - 1;
}

template <bool DEBUG, bool IMPACT, bool WEIGHTED, bool DUAL>
__global__ void __launch_bounds__(PT_THREADS, 4) pd_particle_kernel(const __grid_constant__ PdParams prm) {
  extern __shared__ __align__(128) unsigned char smem[];
  const PdCardScalars &sc = prm.sc;
  const int nb = sc.n_bins;
  float *s_px = (float *)(smem + PO_F), *s_py = s_px + PT_TILE, *s_pz = s_py + PT_TILE;
  float *s_vx = s_pz + PT_TILE, *s_vy = s_vx + PT_TILE, *s_vz = s_vy + PT_TILE;
  int *s_pid = (int *)(smem + PO_PID);
  signed char *s_q = (signed char *)(smem + PO_Q);
  unsigned short *s_key = (unsigned short *)(smem + PO_KEY);
  unsigned short *s_list = (unsigned short *)(smem + PO_LIST);
  uint32_t *s_accmask = (uint32_t *)(smem + PO_MASK);
  int *s_woff = (int *)(smem + PO_WOFF);
  unsigned long long *s_misc = (unsigned long long *)(smem + PO_MISC);
  uint64_t *s_bar = (uint64_t *)(s_misc + 0);
  int *s_cnt = (int *)(s_misc + 1);               // [2] this tile
  long long *s_win = (long long *)(s_misc + 3);   // [0] e_lo, [1] e_hi
  const PTables TL = make_ptables(nb, sc.n_tb, sc.lut_cells);
  float *s_tb = (float *)(smem + TL.tb);
  float4 *s_rec = (float4 *)(smem + TL.binrec);
  unsigned short *s_lut = (unsigned short *)(smem + TL.lut);

  const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;

  for (int i = tid; i < sc.n_tb; i += PT_THREADS) s_tb[i] = prm.tab.tb[i];
  for (int i = tid; i < nb; i += PT_THREADS)
    s_rec[i] = make_float4(prm.tab.inv_w[i], prm.tab.half[i], __int_as_float(prm.tab.offset[i] | (prm.tab.nphi[i] << 16)), 0.f);
  for (int i = tid; i < sc.lut_cells; i += PT_THREADS) s_lut[i] = prm.tab.lut[i];
  if (tid == 0) {
    mbar_init(s_bar, 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    s_cnt[2] = (int)atomicAdd(prm.ptile_counter, 1u);
  }
  uint32_t phase = 0;
  // the particles of the call are [p_base, p_end) of the arrays (p_base = offsets[0]: 0 for a public call, the chunk's
  // first particle for the pipelined host entry); tiles start at p_al = p_base rounded down to 16 particles, so that
  // every tile start is 16-byte aligned in all arrays; the (< 16) particles in front of p_base are skipped
  const long long p_base = prm.p_base, p_al = p_base & ~15ll, n_all = p_base + prm.n_particles;
  const int wbase = wid * PT_PER_WARP;  // this warp owns particles [wbase, wbase + PT_PER_WARP) of every tile
  const int wword = wid * PT_ITERS;     // ... and these words of the accepted mask

  for (;;) {
    __syncthreads();  // (A) previous tile fully done with shared memory; this tile's index is in s_cnt[2]
    const int tile = s_cnt[2];
    if (tile >= prm.n_ptiles) break;
    const long long s0 = p_al + (long long)tile * PT_TILE;
    const int n = (int)min((long long)PT_TILE, n_all - s0);
    const int lo_skip = (int)max(p_base - s0, 0ll);  // > 0 only in tile 0
    const bool full = n == PT_TILE && prm.tma_ok;

    // ---- stage the tile's inputs: eight bulk copies (one thread), or plain loads for the ragged last tile /
    // unaligned arrays
    if (full) {
      if (tid == 0) {
        fence_async_smem();  // the staging slots were last written through the generic proxy
        mbar_expect_tx(s_bar, 29u * PT_TILE);
        bulk_g2s(s_px, prm.px + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_py, prm.py + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_pz, prm.pz + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_vx, prm.vx + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_vy, prm.vy + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_vz, prm.vz + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_pid, prm.pid + s0, 4u * PT_TILE, s_bar);
        bulk_g2s(s_q, prm.charge + s0, 1u * PT_TILE, s_bar);
      }
    } else {
      for (int i = tid; i < n; i += PT_THREADS) {
        s_px[i] = __ldg(prm.px + s0 + i), s_py[i] = __ldg(prm.py + s0 + i), s_pz[i] = __ldg(prm.pz + s0 + i);
        s_vx[i] = __ldg(prm.vx + s0 + i), s_vy[i] = __ldg(prm.vy + s0 + i), s_vz[i] = __ldg(prm.vz + s0 + i);
        s_pid[i] = __ldg(prm.pid + s0 + i), s_q[i] = __ldg(prm.charge + s0 + i);
      }
    }

    // ---- the events of the tile (while the copies are in flight).  offsets[0..n_events] is non-decreasing:
    // e_lo = the event of particle s_eff, e_hi = the last event with a particle in the tile.  The offsets of
    // e_lo .. e_hi + 1, relative to the tile, go to shared memory: class A looks its event up there.
    if (wid == 0) {
      // found by pd_tile_events_kernel for every tile boundary: first event with offset >= s, last with offset <= s
      const long long e_lo = (long long)__ldg(prm.tile_ev + 2 * tile + 1);
      const long long w3 = s0 + PT_TILE >= n_all ? prm.n_events + 1 : (long long)__ldg(prm.tile_ev + 2 * (tile + 1));
      const long long e_hi = min(w3, prm.n_events) - 1;
      if (lane == 0) s_win[0] = e_lo, s_win[1] = e_hi;
      if (e_hi - e_lo + 2 <= PT_WCAP)
        for (int k = lane; k <= (int)(e_hi - e_lo) + 1; k += 32) s_woff[k] = (int)(__ldg(prm.offsets + e_lo + k) - s0);
    } else if (tid == 32 && prm.tma_ok) {
      // the tile this CTA will most likely take next: towards L2 now, so that its bulk copies find it there
      const long long sn = s0 + (long long)gridDim.x * PT_TILE;
      if (sn + PT_TILE <= n_all) {
        l2_prefetch(prm.px + sn, 4u * PT_TILE), l2_prefetch(prm.py + sn, 4u * PT_TILE), l2_prefetch(prm.pz + sn, 4u * PT_TILE);
        l2_prefetch(prm.vx + sn, 4u * PT_TILE), l2_prefetch(prm.vy + sn, 4u * PT_TILE), l2_prefetch(prm.vz + sn, 4u * PT_TILE);
        l2_prefetch(prm.pid + sn, 4u * PT_TILE), l2_prefetch(prm.charge + sn, 1u * PT_TILE);
      }
    }
    // this warp's words of the accepted mask
    if (lane < PT_ITERS) s_accmask[wword + lane] = 0u;
    __syncthreads();  // (B) events in place; plain loads done
    if (full) mbar_wait(s_bar, phase), phase ^= 1u;
    const long long e_lo = s_win[0], e_hi = s_win[1];
    const int n_win = (int)min(e_hi - e_lo + 1, (long long)PT_WCAP);  // events of the tile
    const bool wide = e_hi - e_lo + 2 > PT_WCAP;                     // only with > 1,000 events in one tile (empty ones)

    // ---- partition of the warp's own particles by class (S0): A charged with efficiency > 0, B other charged,
    // N neutral; dropped particles are finished here.  No other warp is involved: ballots and register counts.
    int nA = 0, nB = 0, nN = 0;
    bool off_axis = false;  // some vertex of the warp's segment is off the beam axis (then the rare double paths are armed)
    uint32_t pk[PT_ITERS];  // per row: entry (i | row << 11) | class << 16 | rank within the class << 18
#pragma unroll
    for (int k = 0; k < PT_ITERS; ++k) {
      const int i = wbase + 32 * k + lane;
      int cls = 3;  // 0 A, 1 B, 2 N, 3 none
      int row = 0;
      if (i < n && i < lo_skip) s_key[i] = (unsigned short)PT_NONE;
      if (i < n && i >= lo_skip) {
        const int q = (int)s_q[i];
        const float px = s_px[i], py = s_py[i];
        float r02;
        const bool dropped = vertex_dropped(sc, px, py, s_vx[i], s_vy[i], s_vz[i], r02);
        off_axis |= r02 > 0.f;
        if (dropped) {
          s_key[i] = (unsigned short)PT_NONE;
          if (DEBUG) {
            const long long g = s0 + i;
            const float nanv = __int_as_float(0x7fc00000);
            if (prm.dbg_status) prm.dbg_status[g] = (unsigned char)PD_DROPPED;
            if (prm.dbg_eta_pos) prm.dbg_eta_pos[g] = nanv;
            if (prm.dbg_phi_pos) prm.dbg_phi_pos[g] = nanv;
            if (prm.dbg_tower) prm.dbg_tower[g] = -1;
            if (prm.dbg_accepted) prm.dbg_accepted[g] = 0;
            if (prm.dbg_eps_row) prm.dbg_eps_row[g] = -1;
            if (prm.dbg_pt_smeared) prm.dbg_pt_smeared[g] = 0.f;
          }
        } else if (q == 0) {
          cls = 2;
        } else {
          const int sp = sc.eff_per_species ? species_of(s_pid[i]) : 2;
          row = (int)sc.cell_row[sp][eff_cell(sc, px, py, s_pz[i])];
          cls = (row >= 0 && sc.row_eps[row] > 0.f) ? 0 : 1;
          row = row < 0 ? 31 : row;  // class B keeps the row for the debug output (31: none; PD_MAX_EFF = 31 rows)
        }
      }
      const unsigned mA = __ballot_sync(0xffffffffu, cls == 0), mB = __ballot_sync(0xffffffffu, cls == 1),
                     mN = __ballot_sync(0xffffffffu, cls == 2);
      const unsigned mine = cls == 0 ? mA : (cls == 1 ? mB : mN);
      const int before = cls == 0 ? nA : (cls == 1 ? nB : nN);
      pk[k] = (uint32_t)(i | (row << 11)) | ((uint32_t)cls << 16) | ((uint32_t)(before + __popc(mine & lt_mask)) << 18);
      nA += __popc(mA), nB += __popc(mB), nN += __popc(mN);
    }
#pragma unroll
    for (int k = 0; k < PT_ITERS; ++k) {
      const int cls = (int)((pk[k] >> 16) & 3u), rank = (int)(pk[k] >> 18);
      if (cls != 3) s_list[wbase + (cls == 0 ? 0 : (cls == 1 ? nA : nA + nB)) + rank] = (unsigned short)pk[k];
    }
    __syncwarp();
    const int n_work = nA + nB + nN;
    off_axis = __any_sync(0xffffffffu, off_axis);

    // ---- S1-S4 on the warp's lists A | B | N: rows of one class (the rows at the two boundaries are mixed).
    // Accepted tracks are smeared on the spot and PARKED at once in the workspace: list A is in particle order and only
    // its entries can be accepted, so the rank of a track among the tracks of the segment -- its place in the parking
    // arrays -- is the number of tracks accepted so far (a ballot per row and a running count).  Kernel T, which knows
    // where an event's tracks go, moves them into the Track collection.
    const long long seg0 = (s0 - p_al) + wbase;  // first slot of the warp's segment in the parking arrays
    int run = 0;                                 // tracks of the segment so far
    // Two copies of the row loop: the one a warp whose vertices all sit on the beam axis takes (every workload of BASELINE.json)
    // has none of the double-precision redos of far-off vertices compiled in (pd_math.cuh), not even their tests
    auto rows = [&](auto off_tag) {
      constexpr bool OFF = decltype(off_tag)::value;
  #pragma unroll 1
      for (int k = 0; k < PT_ITERS; ++k) {
        const int v = 32 * k + lane;
        bool accepted = false;
        int i = 0, pid = 0;
        float px = 0.f, py = 0.f, pz = 0.f, u = 0.f, phi_pos = 0.f;
        uint32_t r1 = 0u, r2 = 0u, pidx_t = 0u;
        long long ev_t = 0;  // (IMPACT: the track's event and index in it, for Philox stream 3)
        if (v < n_work) {
          const int cls = v < nA ? 0 : (v < nA + nB ? 1 : 2);
          const unsigned ent = s_list[wbase + v];
          i = (int)(ent & 0x7ffu);
          px = s_px[i], py = s_py[i], pz = s_pz[i];
          const float vx = s_vx[i], vy = s_vy[i], vz = s_vz[i];
          pid = s_pid[i];
          float x, y, z;
          uint32_t status;
          if (cls == 2 || sc.sB == 0.f) status = line_hit<OFF>(sc, px, py, pz, vx, vy, vz, x, y, z);
          else status = helix_hit<OFF>(sc, (int)s_q[i], px, py, pz, vx, vy, vz, x, y, z);
          const bool live = (status & PD_FACE_MASK) != PD_DROPPED;
          u = __int_as_float(0x7fc00000), phi_pos = u;
          int tower = -1;
          const int apid = pid < 0 ? -pid : pid;
          const bool to_ecal = apid == 11 || apid == 22;  // reading A18
          const bool to_none = apid == 13 || apid == 12 || apid == 14 || apid == 16;
          if (live) {
            hit_coords(sc, status, x, y, z, u, phi_pos);
            tower = hit_tower_rec(sc, DUAL ? (to_ecal ? 0 : 1) : 0, s_tb, s_rec, s_lut, u, phi_pos);  // in the grid of its section (K6)
          }
          if (cls == 0 && live) {
            // S2: accept iff u24 < eps (A11); Philox(seed, event, particle index within the event), stream 0.
            // The event: the last one whose offset is <= i (bisection of the tile's offsets; one step on big events)
            long long ev;
            uint32_t pidx;
            if (!wide) {
              int lo = 0, hi = n_win - 1;
              while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (s_woff[mid] <= i) lo = mid;
                else hi = mid - 1;
              }
              ev = e_lo + lo, pidx = (uint32_t)(i - s_woff[lo]);
            } else {
              long long lo = e_lo, hi = e_hi;
              const long long g = s0 + i;
              while (lo < hi) {
                const long long mid = (lo + hi + 1) >> 1;
                if (__ldg(prm.offsets + mid) <= g) lo = mid;
                else hi = mid - 1;
              }
              ev = lo, pidx = (uint32_t)(g - __ldg(prm.offsets + lo));
            }
            uint32_t rn[4];
            rng_block(prm.rk, prm.event_base + ev, pidx, 0u, rn);
            accepted = uniform24(rn[0]) < sc.row_eps[ent >> 11];
            r1 = rn[1], r2 = rn[2];
            if (IMPACT) ev_t = prm.event_base + ev, pidx_t = pidx;
          }
          // what the tower pass needs: tower | HCAL bit, or "no deposit"
          s_key[i] = (tower >= 0 && !to_none) ? (unsigned short)((unsigned)tower | (to_ecal ? 0u : 0x8000u)) : (unsigned short)PT_NONE;
          if (DEBUG) {
            const long long g = s0 + i;
            const int row = (int)(ent >> 11);
            if (prm.dbg_status) prm.dbg_status[g] = (unsigned char)status;
            if (prm.dbg_eta_pos) prm.dbg_eta_pos[g] = live ? eta_from_u(sc, u) : u;
            if (prm.dbg_phi_pos) prm.dbg_phi_pos[g] = phi_pos;
            if (prm.dbg_tower) prm.dbg_tower[g] = tower;
            if (prm.dbg_accepted) prm.dbg_accepted[g] = accepted ? 1 : 0;
            if (prm.dbg_eps_row) prm.dbg_eps_row[g] = (signed char)((cls == 2 || !live || row == 31) ? -1 : row);
            if (prm.dbg_pt_smeared && !accepted) prm.dbg_pt_smeared[g] = 0.f;
          }
        }
        const unsigned m_acc = __ballot_sync(0xffffffffu, accepted);
        if (accepted) {
          // S3 on the spot (the Philox words are in registers); the record goes straight to its parking slot
          TrackOut t;
          track_smear_words(sc, px, py, pz, r1, r2, (sc.trk_per_species || sc.n_trk_rows > 0) ? species_of(pid) : 2, t);
          const long long g = seg0 + run + __popc(m_acc & lt_mask);
          prm.park_idx[g] = (unsigned char)(i - wbase);
          prm.park_pid[g] = pid;
          prm.park_q[g] = s_q[i];
          prm.park_f[0][g] = t.pt_s, prm.park_f[1][g] = t.eta_mom, prm.park_f[2][g] = t.phi0;
          prm.park_f[3][g] = t.E_trk, prm.park_f[4][g] = eta_from_u(sc, u), prm.park_f[5][g] = phi_pos;
          if (IMPACT) {
            // pd_options.impact: d0, z0 and their errors while the particle is on chip (the stand-alone kernel has to gather it)
            const ImpactCfg ic{sc.inv_kB, sc.sB, prm.imp_d0_a, prm.imp_d0_b, prm.imp_z0_a, prm.imp_z0_b};
            float d0m, z0m, sd, sz;
            track_impact(ic, prm.rk, ev_t, pidx_t, (int)s_q[i], px, py, pz, s_vx[i], s_vy[i], s_vz[i], d0m, z0m, sd, sz);
            prm.park_imp[0][g] = d0m, prm.park_imp[1][g] = z0m, prm.park_imp[2][g] = sd, prm.park_imp[3][g] = sz;
          }
          if (WEIGHTED) prm.park_sig[g] = fast_sqrt(t.rel2) * t.E_trk;  // reading K5 (cards with eflow_weighted only)
          atomicOr(&s_accmask[i >> 5], 1u << (i & 31));
          if (DEBUG && prm.dbg_pt_smeared) prm.dbg_pt_smeared[s0 + i] = t.pt_s;
        }
        run += __popc(m_acc);
      }
    };
    if (off_axis) rows(std::true_type{});
    else rows(std::false_type{});
    // the segment's accepted bits (the warp's own mask words: nobody else sets their bits) go beside the parked tracks
    __syncwarp();
    if (lane < PT_ITERS) prm.accmask[(seg0 >> 5) + lane] = s_accmask[wword + lane];
    // the warp's keys (what the tower pass needs): PT_PER_WARP 16-bit words, stored as 32-bit ones
    {
      const uint32_t *src = (const uint32_t *)(s_key + wbase);
      uint32_t *dst = (uint32_t *)(prm.key + (s0 - p_al) + wbase);
      for (int j = lane; j < PT_PER_WARP / 2; j += 32) dst[j] = src[j];
    }
    if (tid == 0) s_cnt[2] = (int)atomicAdd(prm.ptile_counter, 1u);  // the CTA's next tile
    fence_async_smem();  // the keys and lists were generic-proxy writes; the next tile's bulk copies overwrite the staging slots
  }
}

}  // namespace pdk

size_t pd_particle_smem_bytes(const pd_card *c) { return pdk::make_ptables(c->sc.n_bins, c->sc.n_tb, c->sc.lut_cells).total; }

int pd_launch_particles(const PdParams &prm, bool debug, int num_sms, int max_smem_optin, void *stream) {
  const size_t smem = pdk::make_ptables(prm.sc.n_bins, prm.sc.n_tb, prm.sc.lut_cells).total;
  if (smem > (size_t)max_smem_optin) return PD_ECUDA;
  // variants: debug outputs; impact parameters from the chain (pd_options.impact); weighted EFlow (reading K5); a second grid
  // for the HCAL (reading K6) -- each compiled in only for the calls and cards that use it
  using Kern = void (*)(const PdParams);
#define PD_P4(I, W, D) pdk::pd_particle_kernel<false, I, W, D>, pdk::pd_particle_kernel<true, I, W, D>
  static const Kern kerns[16] = {PD_P4(false, false, false), PD_P4(true, false, false), PD_P4(false, true, false), PD_P4(true, true, false),
                                 PD_P4(false, false, true),  PD_P4(true, false, true),  PD_P4(false, true, true),  PD_P4(true, true, true)};
#undef PD_P4
  const Kern kern = kerns[(debug ? 1 : 0) | (prm.imp_on ? 2 : 0) | (prm.park_sig ? 4 : 0) | (prm.sc.n_grids > 1 ? 8 : 0)];
  if (cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, max_smem_optin) != cudaSuccess) return PD_ECUDA;
  // persistent CTAs that claim their tiles from a counter: as many as fit on the device
  int per_sm = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, pdk::PT_THREADS, smem) != cudaSuccess) return PD_ECUDA;
  if (per_sm < 1) return PD_ECUDA;
  if (const char *e = getenv("PD_P_PER_SM")) per_sm = std::min(per_sm, atoi(e));  // experiment
  int grid = num_sms * per_sm;
  if (grid > prm.n_ptiles) grid = prm.n_ptiles;
  if (grid < 1) grid = 1;
  pdk::pd_tile_events_kernel<<<(prm.n_ptiles + 1 + 255) / 256, 256, 0, (cudaStream_t)stream>>>(prm.offsets, prm.n_events, prm.p_base, prm.n_ptiles, prm.tile_ev);
  kern<<<grid, pdk::PT_THREADS, smem, (cudaStream_t)stream>>>(prm);
  return cudaGetLastError() == cudaSuccess ? PD_OK : PD_ECUDA;
}
