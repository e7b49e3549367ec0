// pd_math.cuh -- per-particle and per-tower arithmetic of the chain (device only, fp32 with a few fp64
// operations where SURVEY.md 7.2-1 shows fp32 cannot hold the 1e-6 band).  Product code; written from
// the DESIGN.md readings, shares nothing with oracle/.
//
// v3: the instruction count per particle is the binding resource, so the math is
// written for few issue slots: MUFU reciprocals / rsqrt, one polynomial atan2, no binary searches
// (eta bin through a float-bits lookup table, efficiency through a cell grid built at card load), and
// the barrel/endcap decision without an arctangent.
#pragma once

#include <cstdint>

#include "pd_internal.h"

namespace pdk {

constexpr float kPiF = 3.14159265358979323846f;
constexpr float kHalfPiF = 1.57079632679489661923f;
constexpr float kTwoM24 = 5.9604644775390625e-08f;  // 2^-24
constexpr float kInfF = __builtin_huge_valf();

// Card tables staged in shared memory (pointers into the CTA's dynamic shared memory).

// ---- S-RNG: Philox4x32-10 (Salmon et al., SC'11), reading A26: key = (seed lo, seed hi),
// counter = (object, event lo, event hi, stream << 16) -----------------------------------------
// The ten round keys (k0 + r W0, k1 + r W1) are computed once on the host (PdParams::rk): in the kernel
// they are constant-bank operands of the XORs, so a block costs 20 wide multiplies and 20 three-input XORs.
using PhiloxKeys = PdPhiloxKeys;

__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, const PhiloxKeys &rk,
                                              uint32_t (&out)[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)0xD2511F53u * c0;  // one IMAD.WIDE each
    const unsigned long long p1 = (unsigned long long)0xCD9E8D57u * c2;
    c0 = (uint32_t)(p1 >> 32) ^ c1 ^ rk.k0[r];
    c1 = (uint32_t)p1;
    c2 = (uint32_t)(p0 >> 32) ^ c3 ^ rk.k1[r];
    c3 = (uint32_t)p0;
  }
  out[0] = c0, out[1] = c1, out[2] = c2, out[3] = c3;
}

__device__ __forceinline__ void rng_block(const PhiloxKeys &rk, long long event, uint32_t object, uint32_t stream,
                                          uint32_t (&out)[4]) {
  const unsigned long long ev = (unsigned long long)event;
  philox4x32_10(object, (uint32_t)ev, (uint32_t)(ev >> 32), stream << 16, rk, out);
}

// u in [0,1) on the 2^-24 lattice (exact in fp32)
__device__ __forceinline__ float uniform24(uint32_t x) { return (float)(x >> 8) * kTwoM24; }

__device__ __forceinline__ float fast_rcp(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_rsqrt(float x) {
  float r;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_sqrt(float x) {
  float r;
  asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// atan2(y, x) in (-pi, pi]: octant reduction + odd minimax polynomial (|error| < 7e-8 on [0,1] in
// fp32 Horner form, coefficients fitted for t + t s Q(s), s = t^2) + fix-ups.  atan2(0, 0) = 0.
__device__ __forceinline__ float fast_atan2(float y, float x) {
  const float ax = fabsf(x), ay = fabsf(y);
  const float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
  const float t = mn * fast_rcp(fmaxf(mx, 1e-37f));
  const float s = t * t;
  float q = 2.622228581e-03f;
  q = fmaf(q, s, -1.513247099e-02f);
  q = fmaf(q, s, 4.112175107e-02f);
  q = fmaf(q, s, -7.366696745e-02f);
  q = fmaf(q, s, 1.057392731e-01f);
  q = fmaf(q, s, -1.418597400e-01f);
  q = fmaf(q, s, 1.999039650e-01f);
  q = fmaf(q, s, -3.333298564e-01f);
  float r = fmaf(t * s, q, t);
  r = ay > ax ? kHalfPiF - r : r;
  r = x < 0.f ? kPiF - r : r;
  return copysignf(r, y);
}

// (sin, cos)(pi x) for |x| <= 1/2: fold to [0, 1/4] and two short minimax polynomials (|error| < 3e-9
// before rounding); sin takes the sign of x.
__device__ __forceinline__ void sincospi_half(float x, float &sn, float &cs) {
  const float ax = fabsf(x);
  const bool hi = ax > 0.25f;
  const float y = hi ? 0.5f - ax : ax;
  const float t = y * y;
  float sp = fmaf(fmaf(-5.888253450e-01f, t, 2.549749374e+00f), t, -5.167707920e+00f);
  sp = fmaf(y * t, sp, kPiF * y);
  float cp = fmaf(fmaf(fmaf(2.314294875e-01f, t, -1.335058451e+00f), t, 4.058707714e+00f), t, -4.934802055e+00f);
  cp = fmaf(t, cp, 1.f);
  sn = copysignf(hi ? cp : sp, x);
  cs = hi ? sp : cp;
}

__device__ __forceinline__ float fast_lg2(float x) {
  float r;
  asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}
__device__ __forceinline__ float fast_ex2(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// -ln(x) for a normal x in (0, 1] to ~2e-7 relative (also next to x = 1, where lg2.approx is only good to an
// absolute 2^-22): x = m 2^e with m in [sqrt(1/2), sqrt(2)), ln m = f - f^2/2 + f^3 R(f), f = m - 1.
__device__ __forceinline__ float neg_ln01(float x) {
  const int ix = __float_as_int(x);
  const int e = (ix - 0x3f3504f3) >> 23;
  const float f = __int_as_float(ix - (e << 23)) - 1.0f;
  float r = 8.917524944e-02f;
  r = fmaf(r, f, -1.435014855e-01f);
  r = fmaf(r, f, 1.487704477e-01f);
  r = fmaf(r, f, -1.656564099e-01f);
  r = fmaf(r, f, 1.996539170e-01f);
  r = fmaf(r, f, -2.500174683e-01f);
  r = fmaf(r, f, 3.333385820e-01f);
  const float f2 = f * f;
  const float lnm = fmaf(f2, fmaf(f, r, -0.5f), f);
  return -fmaf((float)e, 0.693147180559945f, lnm);
}

// cos(pi v) for v in [0, 2]: fold to [0, 1/2] and one even polynomial (|error| < 3e-10 before rounding)
__device__ __forceinline__ float cospi_02(float v) {
  const float a = fabsf(v - 1.0f);        // cos(pi v) = -cos(pi a), a in [0, 1]
  const bool flip = a > 0.5f;
  const float b = flip ? 1.0f - a : a;    // cos(pi a) = flip ? -cos(pi b) : cos(pi b)
  const float t = b * b;
  float c = -2.439671581e-02f;
  c = fmaf(c, t, 2.349375585e-01f);
  c = fmaf(c, t, -1.335212057e+00f);
  c = fmaf(c, t, 4.058709164e+00f);
  c = fmaf(c, t, -4.934802137e+00f);
  c = fmaf(c, t, 1.0f);
  return flip ? c : -c;
}

// Box-Muller, cosine branch: z = sqrt(-2 ln u+) cos(2 pi u), u+ = ((xa>>8)+1) 2^-24, u = (xb>>8) 2^-24
__device__ __forceinline__ float normal_bm(uint32_t xa, uint32_t xb) {
  const float up = (float)((xa >> 8) + 1u) * kTwoM24;   // exact
  const float u2 = (float)(xb >> 8) * (2.0f * kTwoM24);  // 2u, exact
  return fast_sqrt(2.0f * neg_ln01(up)) * cospi_02(u2);
}

// log-normal with mean m and relative standard deviation^2 rel2 = (s/m)^2 (reading A21):
// m exp(-b2/2 + b z), b2 = ln(1 + rel2), i.e. m (1 + rel2)^(-1/2) exp(b z).  Caller guarantees m > 0, rel2 > 0.
// ln(1 + x): for x < 1/2 the series 2 s (1 + t Q(t)), s = x / (2 + x), t = s^2 (relative error ~1e-8, so that
// b = sqrt(b2) keeps its relative accuracy for the small x of the track smear); lg2.approx above.
__device__ __forceinline__ float lognormal_rel(float m, float rel2, float z) {
  const float y = 1.0f + rel2;
  const float s = rel2 * fast_rcp(2.0f + rel2);
  const float t = s * s;
  const float q = fmaf(fmaf(1.497972671e-01f, t, 1.998943251e-01f), t, 3.333335706e-01f);
  const float s2 = s + s;
  const float b2 = rel2 < 0.5f ? fmaf(s2 * t, q, s2) : 0.693147180559945f * fast_lg2(y);
  const float b = fast_sqrt(b2);
  return m * fast_rsqrt(y) * fast_ex2(1.4426950408889634f * b * z);
}

// asinh(x) to ~2e-7 absolute / relative (outputs only: eta of a track, eta of its calorimeter hit)
__device__ __forceinline__ float fast_asinh(float x) {
  const float ax = fabsf(x);
  const float y = ax + fast_sqrt(fmaf(ax, ax, 1.0f));
  return copysignf(0.693147180559945f * fast_lg2(y), x);
}

// calorimeter component: E' = LN(E, sigma(E)), sigma^2 = C2 E^2 + S2 E + N2
__device__ __forceinline__ float smear_component(float E, const float (&csn2)[3], uint32_t xa, uint32_t xb) {
  if (!(E > 0.f)) return 0.f;
  const float s2 = fmaf(csn2[0] * E, E, fmaf(csn2[1], E, csn2[2]));
  if (!(s2 > 0.f)) return E;
  const float iE = fast_rcp(E);
  return lognormal_rel(E, s2 * iE * iE, normal_bm(xa, xb));
}

__device__ __forceinline__ float eta_from_u(const PdCardScalars &sc, float u) { return fast_asinh(sc.grid_theta ? -u : u); }

// species of a charged particle for the per-species card tables: 0 electron, 1 muon, 2 charged hadron
__device__ __forceinline__ int species_of(int pid) {
  const int a = pid < 0 ? -pid : pid;
  return a == 11 ? 0 : (a == 13 ? 1 : 2);
}

// Rare path: a helix grazing the barrel (within a few % of the looper threshold).  The crossing angle
// amplifies the rounding of rho by 1/sqrt(distance to tangency), so the quadratic is redone in double.
// 1/sqrt(x) and 1/x in double from the fp32 MUFU seed and two Newton steps (relative error ~1e-14): no
// double-precision divide or square-root routine on this path.
__device__ __forceinline__ double rsqrt_d(double x) {
  double y = (double)fast_rsqrt((float)x);
  y = y * fma(-0.5 * x, y * y, 1.5);
  return y * fma(-0.5 * x, y * y, 1.5);
}
__device__ __forceinline__ double rcp_d(double x) {
  double y = (double)fast_rcp((float)x);
  y = y * fma(-x, y, 2.0);
  return y * fma(-x, y, 2.0);
}

static __device__ __noinline__ bool graze_double(const PdCardScalars &sc, float px, float py, float vx, float vy, float aq,
                                          float s, float &cc, float &ss) {
  const double pxd = px, pyd = py, vxd = vx, vyd = vy, Rd = sc.R;
  const double p2 = pxd * pxd + pyd * pyd;
  const double ipt = rsqrt_d(p2);
  const double ptd = p2 * ipt;
  const double rhod = ptd * rcp_d(sc.kB_d * (double)aq);
  const double ad = (vxd * pxd + vyd * pyd) * ipt;
  const double bd = (double)s * (vyd * pxd - vxd * pyd) * ipt;
  const double Dd = Rd * Rd - (vxd * vxd + vyd * vyd);
  const double Pd = 2.0 * rhod * ad;
  const double Qd = 4.0 * rhod * (rhod + bd) - Dd;
  const double dd = Pd * Pd + Qd * Dd;
  if (!(dd >= 0.0)) return false;
  const double Sd = dd > 1e-30 ? dd * rsqrt_d(dd) : 0.0;
  if (Pd >= 0.0) cc = (float)(Pd + Sd), ss = (float)Dd;
  else cc = (float)Qd, ss = (float)(Sd - Pd);
  return true;
}

// Two more rare paths, for vertices far off the axis: the hit is the vertex plus the chord, and where the result is much
// smaller than either (an endcap hit close to the axis from a vertex a metre away; a barrel hit whose z is a small
// difference of the vertex z and the path along z) the fp32 sum keeps fewer digits than the 1e-6 the tower decision
// wants.  Redone in double (CUDA's own double routines: it hardly ever runs; never for vertices on the axis).
static __device__ __noinline__ void endcap_xy_double(const PdCardScalars &sc, float px, float py, float pz, float vx, float vy,
                                                     float vz, float aq, float s, float &x, float &y) {
  const double pxd = px, pyd = py;
  const double pt = sqrt(pxd * pxd + pyd * pyd);
  const double rho = pt / (sc.kB_d * (double)aq);
  const double zd = (double)sc.L - (pz > 0.f ? (double)vz : -(double)vz);
  double sh, ch;
  sincospi(zd * (sc.kB_d * (0.5 * 0.31830988618379067154) * (double)aq) / fabs((double)pz), &sh, &ch);
  const double c0 = pxd / pt, s0 = pyd / pt, l2 = 2.0 * rho * sh;
  x = (float)((double)vx + l2 * (c0 * ch - (double)s * s0 * sh));
  y = (float)((double)vy + l2 * (s0 * ch + (double)s * c0 * sh));
}
static __device__ __noinline__ float barrel_z_double(const PdCardScalars &sc, float px, float py, float pz, float vx, float vy,
                                                     float vz, float aq, float s) {
  float cc = 1.f, ss = 0.f;
  graze_double(sc, px, py, vx, vy, aq, s, cc, ss);
  return (float)((double)vz + 2.0 * atan2((double)ss, (double)cc) * (double)pz / (sc.kB_d * (double)aq));
}

// a barrel hit at the end of a long arc (chord > sqrt(2) R: only from a vertex far off the axis): the chord is good to ~6e-7 of
// its length in fp32, the azimuth of the hit wants 1e-6 R
static __device__ __noinline__ void barrel_xy_double(const PdCardScalars &sc, float px, float py, float vx, float vy, float aq, float s,
                                                     float &x, float &y) {
  float cc = 1.f, ss = 0.f;
  graze_double(sc, px, py, vx, vy, aq, s, cc, ss);
  const double ccd = cc, ssd = ss, nrm = rsqrt_d(ccd * ccd + ssd * ssd), ch = ccd * nrm, sh = ssd * nrm;
  const double pxd = px, pyd = py, p2 = pxd * pxd + pyd * pyd, ipt = rsqrt_d(p2), pt = p2 * ipt;
  const double rho = pt * rcp_d(sc.kB_d * (double)aq), c0 = pxd * ipt, s0 = pyd * ipt, l2 = 2.0 * rho * sh;
  x = (float)((double)vx + l2 * (c0 * ch - (double)s * s0 * sh));
  y = (float)((double)vy + l2 * (s0 * ch + (double)s * c0 * sh));
}

// The straight line's two rare cases (one call site): an endcap hit much closer to the axis than the vertex is (x, y are small
// differences of vertex and path), and a barrel hit whose z is a small difference of the vertex z and a long path.
static __device__ __noinline__ void line_fix_double(const PdCardScalars &sc, bool endcap, float sgnz, float px, float py, float pz, float vx,
                                                    float vy, float vz, float &x, float &y, float &z) {
  const double pxd = px, pyd = py, vxd = vx, vyd = vy;
  if (endcap) {
    const double td = ((double)sc.L - (double)(sgnz * vz)) * rcp_d(fabs((double)pz));
    x = (float)fma(td, pxd, vxd), y = (float)fma(td, pyd, vyd);
  } else {
    const double pt2 = pxd * pxd + pyd * pyd, bb = vxd * pxd + vyd * pyd, Rd = sc.R;
    const double Dd = Rd * Rd - (vxd * vxd + vyd * vyd);
    const double dd = bb * bb + pt2 * Dd, sq = dd * rsqrt_d(dd);
    const double td = bb > 0.0 ? Dd * rcp_d(bb + sq) : (sq - bb) * rcp_d(pt2);
    z = (float)fma(td, (double)pz, (double)vz);
  }
}

// readings A4, A5: born on/outside the cylinder, or no transverse momentum -> dropped
__device__ __forceinline__ bool vertex_dropped(const PdCardScalars &sc, float px, float py, float vx, float vy, float vz, float &r02) {
  const float pt2 = fmaf(px, px, py * py);
  r02 = fmaf(vx, vx, vy * vy);
  return r02 >= sc.R2 || fabsf(vz) >= sc.L || pt2 < 1e-9f;
}

// S2, first half: cell of the efficiency grid at the true vertex momentum (A7, A8).  pT edges are compared on pT^2
// in double (px^2 + py^2 is then exact to ~1e-16, so a generator floor at exactly an edge, e.g. pT = 0.1 GeV, is
// decided like the fp64 definition); |eta| edges as |pz| >= sinh(edge) pT; unused edges are +max / +inf.
__device__ __forceinline__ int eff_cell(const PdCardScalars &sc, float px, float py, float pz) {
  const double p2 = (double)px * (double)px + (double)py * (double)py;
  const float pt2 = fmaf(px, px, py * py);
  const float pt = pt2 * fast_rsqrt(pt2);
  const float apz = fabsf(pz);
  int ip = 0, it = 0;
  // the first two edges of either kind without a branch, the rest (cards with finer tables) in uniform loops
  ip += p2 > sc.pt_edge2_d[0] ? 1 : 0;
  ip += p2 > sc.pt_edge2_d[1] ? 1 : 0;
  for (int k = 2; k < sc.n_pt; ++k) ip += p2 > sc.pt_edge2_d[k] ? 1 : 0;
  it += apz >= sc.T_edge[0] * pt ? 1 : 0;
  it += apz >= sc.T_edge[1] * pt ? 1 : 0;
  for (int k = 2; k < sc.n_T; ++k) it += apz >= sc.T_edge[k] * pt ? 1 : 0;
  return ip * (sc.n_T + 1) + it;
}

// S1 for a neutral particle (or no field): straight line to r = R or |z| = L, whichever comes first.  The caller
// has excluded dropped vertices.  Returns the face; (x, y, z) = the hit.
template <bool OFF_AXIS = true>
__device__ __forceinline__ uint32_t line_hit(const PdCardScalars &sc, float px, float py, float pz, float vx, float vy, float vz,
                                             float &x, float &y, float &z) {
  const float pt2 = fmaf(px, px, py * py);
  const float apz = fabsf(pz);
  const float sgnz = pz > 0.f ? 1.f : (pz < 0.f ? -1.f : 0.f);
  const float zdist = sc.L - sgnz * vz;  // distance to the endcap the particle flies towards (> 0)
  // (OFF_AXIS false: vx = vy = 0 for certain -- the terms that vanish are left out; the results are bit for bit those of the
  // general form)
  const float D = OFF_AXIS ? sc.R2 - fmaf(vx, vx, vy * vy) : sc.R2;  // > 0
  // t_R = num / den, t_Z = zdist / |pz|
  const float b = OFF_AXIS ? fmaf(vx, px, vy * py) : 0.f;
  const float sq = fast_sqrt(OFF_AXIS ? fmaf(b, b, pt2 * D) : pt2 * D);
  const float num = (OFF_AXIS && b > 0.f) ? D : (OFF_AXIS ? sq - b : sq);
  const float den = (OFF_AXIS && b > 0.f) ? b + sq : pt2;
  const bool endcap = apz > 0.f && zdist * den < num * apz;
  const float t = endcap ? zdist * fast_rcp(apz) : num * fast_rcp(den);
  if (OFF_AXIS) x = fmaf(t, px, vx), y = fmaf(t, py, vy);
  else x = t * px, y = t * py;
  z = endcap ? sgnz * sc.L : fmaf(t, pz, vz);
  // rare cases of a vertex far off the axis, redone in double (see line_fix_double); never for vertices on the axis
  if (OFF_AXIS) {
    const float dzp = z - vz;
    if (endcap ? fmaf(x, x, y * y) < 0.09f * (sc.R2 - D) : dzp * dzp > fmaf(z, z, sc.R2)) line_fix_double(sc, endcap, sgnz, px, py, pz, vx, vy, vz, x, y, z);
  }
  return endcap ? PD_ENDCAP : PD_BARREL;
}

// S1 for a charged particle in the field: helix of radius rho; momentum azimuth phi0 + s alpha (reading A3: q > 0
// in +z field turns clockwise).  Returns PD_DROPPED | PD_LOOPER for a trapped looper (reading A6), else the face
// (| PD_LOOPER when the helix never reaches r = R).
template <bool OFF_AXIS = true>
__device__ __forceinline__ uint32_t helix_hit(const PdCardScalars &sc, int q, float px, float py, float pz, float vx, float vy,
                                              float vz, float &x, float &y, float &z) {
  const float pt2 = fmaf(px, px, py * py);
  const float ipt = fast_rsqrt(pt2);
  const float pt = pt2 * ipt;
  const float apz = fabsf(pz);
  const float sgnz = pz > 0.f ? 1.f : (pz < 0.f ? -1.f : 0.f);
  const float D = OFF_AXIS ? sc.R2 - fmaf(vx, vx, vy * vy) : sc.R2;  // > 0  (OFF_AXIS false: vx = vy = 0 for certain, see line_hit)
  uint32_t looper = 0;
  const float aq = fabsf((float)q);
  const float rho = aq == 1.f ? pt * sc.inv_kB : pt * sc.inv_kB * fast_rcp(aq);
  const float s = ((q > 0) == (sc.sB > 0.f)) ? -1.f : 1.f;
  const float c0 = px * ipt, s0 = py * ipt;
  // vertex in the (u0, s n0) frame: a = v.u0, b = s v.n0
  const float a_ = OFF_AXIS ? fmaf(vx, c0, vy * s0) : 0.f;
  const float b_ = OFF_AXIS ? s * fmaf(vy, c0, -vx * s0) : 0.f;
  // |v + 2 rho sin h u(phi0 + s h)|^2 = R^2 with t = tan h:  Q t^2 + 2 P t - D = 0   (h = alpha/2)
  const float P = OFF_AXIS ? 2.f * rho * a_ : 0.f;
  const float Q = fmaf(4.f * rho, OFF_AXIS ? rho + b_ : rho, -D);
  const float disc = OFF_AXIS ? fmaf(P, P, Q * D) : Q * D;
  const float scale = OFF_AXIS ? fmaf(P, P, 4.f * rho * rho * D) : 4.f * rho * rho * D;
  bool reach;
  float cc = 1.f, ss = 0.f;  // (cos, sin) of the barrel half-angle h_R, unnormalised, ss >= 0
  // (The band is what keeps the azimuth of the hit within 1e-6: measured on 5.7 million on-axis particles the largest error is
  // 6.1e-7 at 0.08, 8.5e-7 at 0.04, 1.24e-6 at 0.02.  A narrower band for the on-axis copy would save 0.8 % of the step at 0.05
  // and was not taken: it leaves 15 % of the tolerance and breaks the bit-for-bit identity of the two copies.)
  if (disc >= 0.f ? disc < 0.08f * scale : -disc < 1e-3f * scale) {
    reach = graze_double(sc, px, py, OFF_AXIS ? vx : 0.f, OFF_AXIS ? vy : 0.f, aq, s, cc, ss);
  } else {
    reach = disc >= 0.f;
    const float S = fast_sqrt(fmaxf(disc, 0.f));
    // first crossing: (cos h, sin h) proportional to (P + S, D) if P >= 0 else (Q, S - P)
    cc = (!OFF_AXIS || P >= 0.f) ? (OFF_AXIS ? P + S : S) : Q;
    ss = (!OFF_AXIS || P >= 0.f) ? D : S - P;
  }
  if (!reach) looper = PD_LOOPER;
  if (!reach && apz == 0.f) return PD_DROPPED | looper;  // trapped (reading A6)
  // endcap half-angle h_Z = zdist kappa |q| B / (2 |pz|), as f = h_Z / pi in double: the turning angle of a
  // looper can be ~1e5 rad.  1/|pz| = MUFU seed + one Newton step in double.
  float sh = 0.f, ch = 1.f;
  bool endcap = false;
  if (apz > 0.f) {
    const double pzd = (double)apz;
    const double r0 = (double)fast_rcp(apz);
    const double r1 = fma(r0, fma(-pzd, r0, 1.0), r0);
    const double zd = (double)sc.L - (double)(sgnz * vz);
    const double fd = zd * (sc.kB_d * (0.5 * 0.31830988618379067154) * (double)aq) * r1;
    const double nd = (fd + 6755399441055744.0) - 6755399441055744.0;  // rint
    const float frac = (float)(fd - nd);                                // in [-0.5, 0.5]
    const float ff = (float)fd;
    sincospi_half(frac, sh, ch);  // (sin, cos)(h_Z) up to a common sign (-1)^n
    // h_Z < h_R  <=>  h_Z < pi and sin(h_R - h_Z) > 0   (both half-angles lie in (0, pi))
    const float cross = fmaf(ss, ch, -cc * sh);
    endcap = !reach || (ff < 1.f && (frac < 0.f ? -cross : cross) > 0.f);
  }
  if (endcap) {
    z = sgnz * sc.L;
  } else {
    const float inv = fast_rsqrt(fmaf(cc, cc, ss * ss));
    ch = cc * inv, sh = ss * inv;
    const float hR = fast_atan2(ss, cc);
    z = fmaf(2.f * hR, pz * sc.inv_kB * (aq == 1.f ? 1.f : fast_rcp(aq)), vz);
    // The path along z is good to ~6e-7 of its length, and eta = asinh(z / R) moves by dz / sqrt(z^2 + R^2): against the 1e-6
    // of eta that matters when the path is longer than the hit is far from the centre (a vertex far away in z, the hit back
    // near z = 0), and for a steep track born next to the barrel surface (D << R^2: the half-angle is then a small difference
    // of large terms).  Neither happens for vertices on the axis; redone in double.
    // (see the end of the function)
  }
  // chord form (pi-periodic in h): position = v + 2 rho sin h u(phi0 + s h)
  const float l2 = 2.f * rho * sh;
  if (OFF_AXIS) {
    x = fmaf(l2, fmaf(c0, ch, -s * s0 * sh), vx);
    y = fmaf(l2, fmaf(s0, ch, s * c0 * sh), vy);
  } else {
    x = l2 * fmaf(c0, ch, -s * s0 * sh);
    y = l2 * fmaf(s0, ch, s * c0 * sh);
  }
  // the three rare cases of a vertex far off the axis (OFF_AXIS: false in the copy of the row loop that a warp whose vertices all sit on the
  // axis -- every workload of BASELINE.json -- which then skips the tests as well)
  if (OFF_AXIS) {
    if (endcap) {
      if (fmaf(x, x, y * y) < 0.09f * (sc.R2 - D)) endcap_xy_double(sc, px, py, pz, vx, vy, vz, aq, s, x, y);
    } else {
      const float dzp = z - vz, dx = x - vx, dy = y - vy;
      if (dzp * dzp > fmaf(z, z, sc.R2) || (D < 0.3f * sc.R2 && apz * ipt > 2.f)) z = barrel_z_double(sc, px, py, pz, vx, vy, vz, aq, s);
      if (fmaf(dx, dx, dy * dy) > 2.f * sc.R2) barrel_xy_double(sc, px, py, vx, vy, aq, s, x, y);
    }
  }
  return (endcap ? PD_ENDCAP : PD_BARREL) | looper;
}

// hit (x, y, z) on the face `status` -> grid coordinate u = z/r (or -z/r for a theta grid) and azimuth
__device__ __forceinline__ void hit_coords(const PdCardScalars &sc, uint32_t status, float x, float y, float z, float &u, float &phi_pos) {
  const float ir = (status & PD_ENDCAP) ? fast_rsqrt(fmaf(x, x, y * y)) : sc.inv_R;
  u = (sc.grid_theta ? -z : z) * ir;
  phi_pos = fast_atan2(y, x);
}

// S3 for one accepted track (A12/A13): log-normal with mean pT and std sigma_rel pT, driven by words
// 1 and 2 of the particle's Philox block; eta, phi unchanged; E = pT' cosh(eta) = pT' |p| / pT.
struct TrackOut {
  float pt_s, eta_mom, phi0, E_trk;
  float rel2;  // sigma_rel^2 of the smear (K5: sigma_E = sqrt(rel2) E_trk)
};

// reading K4: the first track-resolution row (species 0 = any, else 1 + the species index used here) that holds the true
// momentum: sinh(lo) pT <= |pz| < sinh(hi) pT, in fp64 with every operation rounded once, as the fp64 definition takes it,
// so that the row -- an integer decision -- is the same on both sides bit for bit.  Off the fast path: cards without rows
// never get here.
static __device__ __noinline__ void track_res_row(const PdCardScalars &sc, float px, float py, float pz, int species, float &a2, float &b) {
  const double pxd = px, pyd = py;
  const double pt = __dsqrt_rn(__dadd_rn(__dmul_rn(pxd, pxd), __dmul_rn(pyd, pyd)));
  const double apz = fabs((double)pz);
  for (int r = 0; r < sc.n_trk_rows; ++r) {
    const int sp = sc.trk_row_sp[r];
    if ((sp == 0 || sp == species + 1) && apz >= __dmul_rn(sc.trk_row_lo_d[r], pt) && apz < __dmul_rn(sc.trk_row_hi_d[r], pt)) {
      a2 = sc.trk_row_a2[r], b = sc.trk_row_b[r];
      return;
    }
  }
}

// r1, r2: words 1 and 2 of the particle's Philox block (stream 0)
__device__ __forceinline__ void track_smear_words(const PdCardScalars &sc, float px, float py, float pz, uint32_t r1, uint32_t r2,
                                                  int species, TrackOut &t) {
  const float pt2 = fmaf(px, px, py * py);
  const float ipt = fast_rsqrt(pt2);
  const float pt = pt2 * ipt;
  float a2 = sc.trk_a2[species], b = sc.trk_b[species];
  if (sc.n_trk_rows > 0) track_res_row(sc, px, py, pz, species, a2, b);  // reading K4 (cards with eta-dependent rows only)
  const float bp = b * pt;
  const float rel2 = fmaf(bp, bp, a2);
  t.rel2 = rel2;
  t.pt_s = rel2 > 0.f ? lognormal_rel(pt, rel2, normal_bm(r1, r2)) : pt;
  t.E_trk = t.pt_s * (fast_sqrt(fmaf(pz, pz, pt2)) * ipt);
  t.eta_mom = fast_asinh(pz * ipt);
  t.phi0 = fast_atan2(py, px);
}

// per-tower smear of both components (S6): the common case of a single non-zero component runs one
// branch-free log-normal; only towers holding both ECAL and HCAL energy take the second
__device__ __forceinline__ void tower_smear_csn(const float (&ecal2)[3], const float (&hcal2)[3], float Eem, float Ehad,
                                                const uint32_t (&rn)[4], float &em_s, float &had_s) {
  const bool prim_em = Eem > 0.f;
  const float Ep = prim_em ? Eem : Ehad;
  const float c2 = prim_em ? ecal2[0] : hcal2[0], s2c = prim_em ? ecal2[1] : hcal2[1], n2 = prim_em ? ecal2[2] : hcal2[2];
  const uint32_t xa = prim_em ? rn[0] : rn[2], xb = prim_em ? rn[1] : rn[3];
  float sp = 0.f;
  if (Ep > 0.f) {
    const float v = fmaf(c2 * Ep, Ep, fmaf(s2c, Ep, n2));
    const float iE = fast_rcp(Ep);
    sp = v > 0.f ? lognormal_rel(Ep, v * iE * iE, normal_bm(xa, xb)) : Ep;
  }
  em_s = prim_em ? sp : 0.f;
  had_s = prim_em ? 0.f : sp;
  if (prim_em && Ehad > 0.f) had_s = smear_component(Ehad, hcal2, rn[2], rn[3]);
}

}  // namespace pdk
