// pd_math.cuh -- per-particle and per-tower arithmetic of the chain (device only, fp32 with a few fp64
// operations where SURVEY.md 7.2-1 shows fp32 cannot hold the 1e-6 band).  Product code; written from
// DESIGN.md readings, shares nothing with oracle/.
#pragma once

#include <cstdint>

#include "pd_internal.h"

namespace pdk {

constexpr float kPiF = 3.14159265358979323846f;
constexpr float kTwoM24 = 5.9604644775390625e-08f;  // 2^-24

// Card tables staged in shared memory (pointers into the CTA's dynamic shared memory).
struct SmCard {
  const float *tb;
  const int *nphi, *offset;
  const float *inv_w, *half, *w, *eta_c, *inv_cosh;
};

// ---- S-RNG: Philox4x32-10 (Salmon et al., SC'11), reading A26: key = (seed lo, seed hi),
// counter = (object, event lo, event hi, stream << 16) -----------------------------------------
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                              uint32_t k1, uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
    c0 = hi1 ^ c1 ^ k0;
    c1 = lo1;
    c2 = hi0 ^ c3 ^ k1;
    c3 = lo0;
    k0 += 0x9E3779B9u;
    k1 += 0xBB67AE85u;
  }
  out[0] = c0, out[1] = c1, out[2] = c2, out[3] = c3;
}

__device__ __forceinline__ void rng_block(unsigned long long seed, long long event, uint32_t object, uint32_t stream,
                                          uint32_t (&out)[4]) {
  const unsigned long long ev = (unsigned long long)event;
  philox4x32_10(object, (uint32_t)ev, (uint32_t)(ev >> 32), stream << 16, (uint32_t)seed, (uint32_t)(seed >> 32), out);
}

// u in [0,1) on the 2^-24 lattice (exact in fp32)
__device__ __forceinline__ float uniform24(uint32_t x) { return (float)(x >> 8) * kTwoM24; }

// Box-Muller, cosine branch: z = sqrt(-2 ln u+) cos(2 pi u), u+ = ((xa>>8)+1) 2^-24, u = (xb>>8) 2^-24
__device__ __forceinline__ float normal_bm(uint32_t xa, uint32_t xb) {
  const float up = (float)((xa >> 8) + 1u) * kTwoM24;   // exact
  const float u2 = (float)(xb >> 8) * (2.0f * kTwoM24);  // 2u, exact
  return sqrtf(-2.0f * logf(up)) * cospif(u2);
}

// log-normal with mean m and relative standard deviation^2 rel2 = (s/m)^2 (reading A21):
// m exp(-b2/2 + b z), b2 = ln(1 + rel2).  Caller guarantees m > 0, rel2 > 0.
__device__ __forceinline__ float lognormal_rel(float m, float rel2, float z) {
  const float b2 = log1pf(rel2);
  return m * expf(fmaf(sqrtf(b2), z, -0.5f * b2));
}

// calorimeter component: E' = LN(E, sigma(E)), sigma^2 = C2 E^2 + S2 E + N2
__device__ __forceinline__ float smear_component(float E, const float (&csn2)[3], uint32_t xa, uint32_t xb) {
  if (!(E > 0.f)) return 0.f;
  const float s2 = fmaf(csn2[0] * E, E, fmaf(csn2[1], E, csn2[2]));
  if (!(s2 > 0.f)) return E;
  return lognormal_rel(E, s2 / (E * E), normal_bm(xa, xb));
}

// ---- S1..S4 for one particle -------------------------------------------------------------------
struct ParticleOut {
  uint32_t status;  // PD_DROPPED / PD_BARREL / PD_ENDCAP | PD_LOOPER
  int bin, j;       // eta/theta bin and phi bin of the hit; bin = -1: outside the grid
  int eps_row;      // -1 none
  bool accepted;
  float u, phi_pos;  // hit: u = z/r (or -z/r for a theta grid), azimuth
};

// smeared track quantities (S3), computed in a separate, converged pass over the accepted tracks
struct TrackOut {
  float pt_s, eta_mom, phi0, E_trk;
};

// bin i with tb[i] <= u < tb[i+1], -1 if outside or NaN
__device__ __forceinline__ int grid_bin(const SmCard &cd, int nb, float u) {
  if (!(u >= cd.tb[0]) || !(u < cd.tb[nb])) return -1;
  int lo = 0, hi = nb;
  while (hi - lo > 1) {
    const int mid = (lo + hi) >> 1;
    if (u >= cd.tb[mid]) lo = mid;
    else hi = mid;
  }
  return lo;
}

__device__ __forceinline__ int phi_bin(const SmCard &cd, int i, float phi) {
  const int n = cd.nphi[i];
  int j = (int)floorf(fmaf(phi, cd.inv_w[i], cd.half[i])) + (n >> 1);
  j = j < 0 ? 0 : j;
  return j > n - 1 ? n - 1 : j;
}

__device__ __forceinline__ void particle_chain(const PdCardScalars &sc, const SmCard &cd, int pid, int q, float px,
                                               float py, float pz, float vx, float vy, float vz,
                                               unsigned long long seed, long long event, uint32_t pidx,
                                               ParticleOut &o) {
  o.status = PD_DROPPED;
  o.bin = -1, o.j = 0;
  o.eps_row = -1;
  o.accepted = false;
  o.u = __int_as_float(0x7fc00000);
  o.phi_pos = o.u;

  const float pt2 = fmaf(px, px, py * py);
  const float r02 = fmaf(vx, vx, vy * vy);
  // readings A4, A5: born on/outside the cylinder, or no transverse momentum -> dropped
  if (r02 >= sc.R2 || fabsf(vz) >= sc.L || pt2 < 1e-9f) return;
  const float pt = sqrtf(pt2);
  const float sgnz = pz > 0.f ? 1.f : (pz < 0.f ? -1.f : 0.f);
  const float D = sc.R2 - r02;  // > 0
  float x, y, z, r;
  uint32_t face, looper = 0;

  if (q == 0 || sc.sB == 0.f) {
    // straight line to r = R or |z| = L, whichever comes first
    const float b = fmaf(vx, px, vy * py);
    const float sq = sqrtf(fmaf(b, b, pt2 * D));
    const float tR = b > 0.f ? D / (b + sq) : (sq - b) / pt2;
    const float tZ = pz != 0.f ? (sgnz * sc.L - vz) / pz : __int_as_float(0x7f800000);
    if (tZ < tR) {
      x = fmaf(tZ, px, vx), y = fmaf(tZ, py, vy), z = sgnz * sc.L;
      r = sqrtf(fmaf(x, x, y * y));
      face = PD_ENDCAP;
    } else {
      x = fmaf(tR, px, vx), y = fmaf(tR, py, vy), z = fmaf(tR, pz, vz);
      r = sc.R;
      face = PD_BARREL;
    }
  } else {
    // helix of radius rho; momentum azimuth phi0 + s alpha (reading A3: q > 0 in +z field turns clockwise)
    const float aq = fabsf((float)q);
    const float kq = sc.kB * aq;
    const float rho = pt / kq;
    const float s = ((q > 0) == (sc.sB > 0.f)) ? -1.f : 1.f;
    const float c0 = px / pt, s0 = py / pt;
    // vertex in the (u0, s n0) frame: a = v.u0, b = s v.n0
    const float a_ = fmaf(vx, c0, vy * s0);
    const float b_ = s * fmaf(vy, c0, -vx * s0);
    // |v + 2 rho sin h u(phi0 + s h)|^2 = R^2 with t = tan h:  Q t^2 + 2 P t - D = 0   (h = alpha/2)
    const float P = 2.f * rho * a_;
    const float Q = fmaf(4.f * rho, rho + b_, -D);
    const float disc = fmaf(P, P, Q * D);
    const float scale = fmaf(P, P, 4.f * rho * rho * D);
    bool reach;
    float cc = 1.f, ss = 0.f;
    if (disc >= 0.f ? disc < 0.08f * scale : -disc < 1e-3f * scale) {
      // grazing the barrel (within a few % of the looper threshold): the crossing angle amplifies the
      // rounding of rho by 1/sqrt(distance to tangency), so this rare case is redone in double
      const double pxd = px, pyd = py, vxd = vx, vyd = vy, Rd = sc.R;
      const double ptd = sqrt(pxd * pxd + pyd * pyd);
      const double rhod = ptd / (sc.kB_d * (double)aq);
      const double ipt = 1.0 / ptd;
      const double ad = (vxd * pxd + vyd * pyd) * ipt;
      const double bd = (double)s * (vyd * pxd - vxd * pyd) * ipt;
      const double Dd = Rd * Rd - (vxd * vxd + vyd * vyd);
      const double Pd = 2.0 * rhod * ad;
      const double Qd = 4.0 * rhod * (rhod + bd) - Dd;
      const double dd = Pd * Pd + Qd * Dd;
      reach = dd >= 0.0;
      if (reach) {
        const double Sd = sqrt(dd);
        if (Pd >= 0.0) cc = (float)(Pd + Sd), ss = (float)Dd;
        else cc = (float)Qd, ss = (float)(Sd - Pd);
      }
    } else {
      reach = disc >= 0.f;
      if (reach) {
        const float S = sqrtf(disc);
        // first crossing: (cos h, sin h) proportional to (P + S, D) if P >= 0 else (Q, S - P)
        if (P >= 0.f) cc = P + S, ss = D;
        else cc = Q, ss = S - P;
      }
    }
    float sh = 0.f, ch = 1.f, hR = 0.f;
    float aR = __int_as_float(0x7f800000), aZ = aR;
    if (reach) {
      const float inv = 1.0f / sqrtf(fmaf(cc, cc, ss * ss));
      ch = cc * inv, sh = ss * inv;
      hR = atan2f(ss, cc);
      aR = 2.f * hR;
    } else {
      looper = PD_LOOPER;
    }
    double hz = 0.0;
    if (pz != 0.f) {
      // alpha_Z / 2 in double: the turning angle of a looper can be ~1e5 rad
      hz = 0.5 * ((double)sc.L - (double)(sgnz * vz)) * (sc.kB_d * (double)aq) / (double)fabsf(pz);
      aZ = (float)(2.0 * hz);
    }
    if (!reach && pz == 0.f) {
      o.status = PD_DROPPED | looper;  // trapped (reading A6)
      return;
    }
    if (aZ < aR) {
      // reduce h modulo pi in double: the chord formulas are pi-periodic in h
      double f = hz * 0.31830988618379067154;
      f -= rint(f);
      sincospif((float)f, &sh, &ch);
      z = sgnz * sc.L;
      face = PD_ENDCAP;
    } else {
      z = fmaf(aR, pz / kq, vz);
      face = PD_BARREL;
    }
    const float l2 = 2.f * rho * sh;
    x = fmaf(l2, fmaf(c0, ch, -s * s0 * sh), vx);
    y = fmaf(l2, fmaf(s0, ch, s * c0 * sh), vy);
    r = face == PD_BARREL ? sc.R : sqrtf(fmaf(x, x, y * y));
  }
  o.status = face | looper;
  const float u = sc.grid_theta ? -z / r : z / r;
  const float phi_pos = atan2f(y, x);
  o.u = u;
  o.phi_pos = phi_pos;

  // S2/S3 track: efficiency at the true vertex momentum (A7); accept iff u24 < eps (A11)
  if (q != 0) {
    const float T = fabsf(pz) / pt;  // sinh |eta_mom|
    float eps = 0.f;
    int row = -1;
    if (!(sc.has_cos && T >= sc.t_cos)) {
      for (int k = 0; k < sc.n_eff; ++k) {
        const float lo = sc.eff[k][0], hi = sc.eff[k][1];
        bool above_lo = pt > lo, below_hi = pt <= hi;
        if (fabsf(pt - lo) <= 2e-6f * lo || fabsf(pt - hi) <= 2e-6f * hi) {
          // pT within rounding of a table edge (e.g. a generator floor at exactly 0.1 GeV): decide on
          // pT^2 in double, where px^2 + py^2 is (almost) exact
          const double p2 = (double)px * (double)px + (double)py * (double)py;
          above_lo = p2 > (double)lo * (double)lo;
          below_hi = p2 <= (double)hi * (double)hi;
        }
        if (above_lo && below_hi && (sc.eff[k][2] <= 0.f || T >= sc.eff[k][2]) && T < sc.eff[k][3]) {
          row = k;
          eps = sc.eff[k][4];
          break;
        }
      }
    }
    o.eps_row = row;
    if (eps > 0.f) {
      uint32_t rn[4];
      rng_block(seed, event, pidx, 0u, rn);
      o.accepted = uniform24(rn[0]) < eps;
    }
  }

  // S4 tower of the hit
  const int i = grid_bin(cd, sc.n_bins, u);
  o.bin = i;
  if (i >= 0) o.j = phi_bin(cd, i, phi_pos);
}

// S3 for one accepted track (A12/A13): log-normal with mean pT and std sigma_rel pT, driven by words
// 1 and 2 of the particle's Philox block; eta, phi unchanged; E = pT' cosh(eta) = pT' |p| / pT.
__device__ __forceinline__ void track_smear(const PdCardScalars &sc, float px, float py, float pz,
                                            unsigned long long seed, long long event, uint32_t pidx, TrackOut &t) {
  const float pt2 = fmaf(px, px, py * py);
  const float pt = sqrtf(pt2);
  uint32_t rn[4];
  rng_block(seed, event, pidx, 0u, rn);
  const float bp = sc.trk_b * pt;
  const float rel2 = fmaf(bp, bp, sc.trk_a2);
  t.pt_s = rel2 > 0.f ? lognormal_rel(pt, rel2, normal_bm(rn[1], rn[2])) : pt;
  t.E_trk = t.pt_s * (sqrtf(fmaf(pz, pz, pt2)) / pt);
  t.eta_mom = asinhf(pz / pt);
  t.phi0 = atan2f(py, px);
}

// per-tower smear of both components (S6): the common case of a single non-zero component runs one
// branch-free log-normal; only towers holding both ECAL and HCAL energy take the second
__device__ __forceinline__ void tower_smear(const PdCardScalars &sc, float Eem, float Ehad, const uint32_t (&rn)[4],
                                            float &em_s, float &had_s) {
  const bool prim_em = Eem > 0.f;
  const float Ep = prim_em ? Eem : Ehad;
  const float c2 = prim_em ? sc.ecal2[0] : sc.hcal2[0], s2c = prim_em ? sc.ecal2[1] : sc.hcal2[1],
              n2 = prim_em ? sc.ecal2[2] : sc.hcal2[2];
  const uint32_t xa = prim_em ? rn[0] : rn[2], xb = prim_em ? rn[1] : rn[3];
  float sp = 0.f;
  if (Ep > 0.f) {
    const float v = fmaf(c2 * Ep, Ep, fmaf(s2c, Ep, n2));
    sp = v > 0.f ? lognormal_rel(Ep, v / (Ep * Ep), normal_bm(xa, xb)) : Ep;
  }
  em_s = prim_em ? sp : 0.f;
  had_s = prim_em ? 0.f : sp;
  if (prim_em && Ehad > 0.f) had_s = smear_component(Ehad, sc.hcal2, rn[2], rn[3]);
}

// eta of a hit from u (only tracks and debug need it as a number)
__device__ __forceinline__ float eta_from_u(const PdCardScalars &sc, float u) { return asinhf(sc.grid_theta ? -u : u); }

}  // namespace pdk
