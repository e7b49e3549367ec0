// pd_impact_math.cuh -- impact parameters of one track (readings I1-I3 of DESIGN.md section 14), shared by the stand-alone
// kernel (pd_impact.cu) and by kernel P of the chain (pd_particles.cu, pd_options.impact).  Device only; product code.
//
// Geometry in fp32, arranged so that nothing cancels (frame: p^ along the transverse momentum, n^ to its left):
//   w = v . p^, u = v . n^ (both from error-free products), helix centre c = (w, u + s rho), r_c = |c|,
//   d0 = s (rho - r_c) = -(2 rho u + s r0^2) / (rho + r_c),   alpha_d = atan2(-w, rho + s u),
//   z0 = v_z + rho alpha_d p_z / p_T;     straight line (q B = 0): d0 = -u, z0 = v_z - w p_z / p_T.
#pragma once

#include <cstdint>

#include "pd_internal.h"
#include "pd_math.cuh"

namespace pdk {

struct ImpactCfg {
  float inv_kB, sB;              // 1 / (kappa |B|), sign of B (0: no field)
  float d0_a, d0_b, z0_a, z0_b;  // sigma = a (+) b / pT
};

// a b - c d with one rounding of the result's leading part (Kahan): exact products via fma
__device__ __forceinline__ float diff_of_products(float a, float b, float c, float d) {
  const float cd = c * d;
  const float err = fmaf(-c, d, cd);
  const float dop = fmaf(a, b, -cd);
  return dop + err;
}

// measured d0, z0 and their errors for the particle (q, p, v) that is object `pidx` of event `event` (Philox stream 3:
// words 0,1 -> d0, 2,3 -> z0)
__device__ __forceinline__ void track_impact(const ImpactCfg &c, const PhiloxKeys &rk, long long event, uint32_t pidx, int q, float px,
                                             float py, float pz, float vx, float vy, float vz, float &d0m, float &z0m, float &sd,
                                             float &sz) {
  const float pt2 = fmaf(px, px, py * py);
  const float ipt = fast_rsqrt(pt2), pt = pt2 * ipt;
  const float u = -diff_of_products(vx, py, vy, px) * ipt;  // v . n^
  const float w = diff_of_products(vx, px, -vy, py) * ipt;  // v . p^
  const float tl = pz * ipt;
  float d0, z0;
  if (q == 0 || c.sB == 0.f) {
    d0 = -u, z0 = fmaf(-w, tl, vz);
  } else {
    const float rho = pt * c.inv_kB * fast_rcp(fabsf((float)q));
    const float s = (q > 0) == (c.sB > 0.f) ? -1.f : 1.f;
    const float cy = fmaf(s, rho, u);  // centre in the (p^, n^) frame: (w, u + s rho)
    const float rc = fast_sqrt(fmaf(w, w, cy * cy));
    const float r02 = fmaf(u, u, w * w);
    d0 = -fmaf(2.f * rho, u, s * r02) * fast_rcp(rho + rc);
    const float alpha = fast_atan2(-w, fmaf(s, u, rho));
    z0 = fmaf(rho * alpha, tl, vz);
  }
  // resolution a (+) b / pT and the two normals of stream 3 (readings I2, I3)
  const float bd = c.d0_b * ipt, bz = c.z0_b * ipt;
  sd = fast_sqrt(fmaf(c.d0_a, c.d0_a, bd * bd)), sz = fast_sqrt(fmaf(c.z0_a, c.z0_a, bz * bz));
  uint32_t r[4];
  rng_block(rk, event, pidx, 3u, r);
  d0m = fmaf(sd, normal_bm(r[0], r[1]), d0);
  z0m = fmaf(sz, normal_bm(r[2], r[3]), z0);
}

}  // namespace pdk
