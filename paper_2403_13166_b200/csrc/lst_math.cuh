// lst_math.cuh -- the cut arithmetic of SPEC.md 3-4 for the device.
//
// Every pass/fail decision is evaluated in fp32 with explicitly rounded, never-contracted
// operations (__fadd_rn / __fsub_rn / __fmul_rn / __fdiv_rn / __fsqrt_rn) in the operation order
// SPEC.md writes down, so that object sets are bit-identical to any other IEEE-754 evaluation of
// the same text (BASELINE.json north_star).  Written from SPEC.md; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace lst {

// ---- SPEC.md 3.1 literals
#define LST_KAPPA 0.0114f
#define LST_C_HALF 0.007125f
#define LST_C_MAX105 0.0149625f
#define LST_C_TOL3 0.00285f
#define LST_Z0_MAX 15.0f

__device__ __forceinline__ float fa(float a, float b) { return __fadd_rn(a, b); }
__device__ __forceinline__ float fs(float a, float b) { return __fsub_rn(a, b); }
__device__ __forceinline__ float fm(float a, float b) { return __fmul_rn(a, b); }
__device__ __forceinline__ float fd(float a, float b) { return __fdiv_rn(a, b); }
__device__ __forceinline__ float fq(float a) { return __fsqrt_rn(a); }

// module type code: bit 1 = subdet (0 barrel / 1 endcap), bit 0 = mtype (0 PS / 1 2S)
__device__ __forceinline__ float tol_dt(int mt) { return (mt & 1) ? 0.01102f : 0.01225f; }
__device__ __forceinline__ float tol_dl(int mt) { return (mt & 1) ? 4.330f : 0.1299f; }
__device__ __forceinline__ float tol_dl2(int mt) { return (mt & 1) ? 6.124f : 0.1837f; }
// anchor tolerances: barrel (dz = DL, dr = 0), endcap (dz = 0, dr = DL)
__device__ __forceinline__ float anchor_dz(int mt) { return (mt & 2) ? 0.0f : tol_dl(mt); }
__device__ __forceinline__ float anchor_dr(int mt) { return (mt & 2) ? tol_dl(mt) : 0.0f; }
__device__ __forceinline__ float md_relf(int mt) { return (mt & 2) ? 0.3f : 0.0f; }

// SPEC.md 3.2
__device__ __forceinline__ float arcfac(float u) {
  float p = 0.017352764f;
  p = fa(0.022372159f, fm(u, p));
  p = fa(0.030381944f, fm(u, p));
  p = fa(0.044642857f, fm(u, p));
  p = fa(0.075f, fm(u, p));
  p = fa(0.16666667f, fm(u, p));
  p = fa(1.0f, fm(u, p));
  return p;
}

// SPEC.md 4.1.  p1 = lower hit, p2 = upper hit.  Returns pass; fills r1, c, w.
// r1, r2 = sqrt(x*x + y*y) of the two hits (computed once per hit by a0 with the same operations).
__device__ __forceinline__ bool md_eval(float x1, float y1, float z1, float r1, float x2, float y2, float z2, float r2, int mt,
                                        float& c, float& w) {
  const float dx = fs(x2, x1), dy = fs(y2, y1), dz = fs(z2, z1);
  const float drho = fd(fa(fm(x1, dx), fm(y1, dy)), r1);
  const float dt = fd(fs(fm(x1, dy), fm(y1, dx)), r1);
  const float S = fminf(1.0f, fm(r2, LST_C_HALF));
  const float dtol = tol_dt(mt);
  const float l2tol = tol_dl2(mt);
  float den;
  if (!(mt & 2)) {
    if (!(drho > 0.0f)) return false;                                                    // M1
    const float L = fq(fa(fm(dt, dt), fm(drho, drho)));
    const float lhs2 = fabsf(fs(dz, fd(fm(drho, z1), r1)));
    const float rhs2 = fa(fd(fm(drho, LST_Z0_MAX), r1), l2tol);
    if (!(lhs2 <= rhs2)) return false;                                                   // M2
    if (!(fabsf(dt) <= fa(fm(L, S), dtol))) return false;                                // M3
    den = fm(r2, L);
  } else {
    const float Ls = fd(fm(fabsf(dz), r1), fabsf(z1));
    if (!(fabsf(fs(drho, Ls)) <= fa(fm(0.15f, Ls), l2tol))) return false;                // M2
    if (!(fabsf(dt) <= fa(fm(fm(1.3f, Ls), S), dtol))) return false;                     // M3
    den = fm(r2, Ls);
  }
  c = fd(fm(-2.0f, dt), den);
  w = fd(fm(2.0f, dtol), den);
  return true;
}

// approximate reciprocal / square roots (1-2 ulp, single MUFU instruction) for the prefilters only
__device__ __forceinline__ float rcp_fast(float x) { float r; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float rsqrt_fast(float x) { float r; asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }
__device__ __forceinline__ float sqrt_fast(float x) { float r; asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x)); return r; }

// Conservative prefilter of md_eval: exact pass  =>  prefilter pass (never the other way round is needed).
// The numerators are formed with the same exactly-rounded operations as md_eval, so their cancellation
// is shared; the divisions and the square root are replaced by approximations (a few ulp) and every
// comparison gets a relative margin of 1e-4 plus an absolute one that exceeds the rounding of the exact
// evaluation by >= 20x.  Non-finite intermediates pass (the exact test decides).
__device__ __forceinline__ bool md_prefilter(float x1, float y1, float z1, float r1, float x2, float y2, float z2, float r2, int mt) {
  const float dx = fs(x2, x1), dy = fs(y2, y1), dz = fs(z2, z1);
  const float nrho = fa(fm(x1, dx), fm(y1, dy));
  const float nt = fs(fm(x1, dy), fm(y1, dx));
  const float S = fminf(1.0f, fm(r2, LST_C_HALF));
  const float inv = rcp_fast(r1);
  const float drho = nrho * inv, dt = nt * inv;
  bool ok;
  if (!(mt & 2)) {
    const float t = drho * z1 * inv;
    const float L = sqrt_fast(dt * dt + drho * drho);
    const bool m1 = nrho > 0.0f;
    const bool m2 = fabsf(dz - t) <= (drho * LST_Z0_MAX * inv + tol_dl2(mt)) * 1.0001f + 1.0e-5f * (fabsf(dz) + fabsf(t));
    const bool m3 = fabsf(dt) <= (L * S + tol_dt(mt)) * 1.0001f;
    ok = m1 && m2 && m3;
    if (!(L < 1.0e30f) || !(fabsf(t) < 1.0e30f)) ok = true;
  } else {
    const float Ls = fabsf(dz) * r1 * rcp_fast(fabsf(z1));
    const bool m2 = fabsf(drho - Ls) <= (0.15f * Ls + tol_dl2(mt)) * 1.0001f + 1.0e-5f * (fabsf(drho) + Ls);
    const bool m3 = fabsf(dt) <= (1.3f * Ls * S + tol_dt(mt)) * 1.0001f;
    ok = m2 && m3;
    if (!(Ls < 1.0e30f) || !(fabsf(drho) < 1.0e30f) || !(fabsf(dt) < 1.0e30f)) ok = true;
  }
  return ok;
}

struct Anchor {   // what the later stages need of an MD
  float x, y, z, r, c, w;
  int mt;
};

// SPEC.md 4.2
__device__ __forceinline__ bool ls_eval(const Anchor& A, const Anchor& B, float& c_out) {
  const float dx = fs(B.x, A.x), dy = fs(B.y, A.y);
  const float d = fq(fa(fm(dx, dx), fm(dy, dy)));
  const float cr = fs(fm(A.x, dy), fm(A.y, dx));
  const float c = fd(fm(-2.0f, cr), fm(fm(A.r, B.r), d));
  const float ac = fabsf(c);
  if (!(ac <= LST_C_MAX105)) return false;                                               // L1
  if (!(fabsf(fs(A.c, c)) <= fa(A.w, fm(md_relf(A.mt), ac)))) return false;              // L3 (inner) -- order of
  if (!(fabsf(fs(B.c, c)) <= fa(B.w, fm(md_relf(B.mt), ac)))) return false;              // L3 (outer)    independent cuts is free
  const float ta = fm(fm(A.r, c), 0.5f), tb = fm(fm(B.r, c), 0.5f);
  const float sA = fm(A.r, arcfac(fm(ta, ta)));
  const float sB = fm(B.r, arcfac(fm(tb, tb)));
  const float lhs = fabsf(fs(fm(A.z, sB), fm(B.z, sA)));
  float rhs = fm(LST_Z0_MAX, fabsf(fs(sB, sA)));
  rhs = fa(rhs, fm(anchor_dz(A.mt), sB));
  rhs = fa(rhs, fm(anchor_dz(B.mt), sA));
  rhs = fa(rhs, fm(anchor_dr(A.mt), fabsf(B.z)));
  rhs = fa(rhs, fm(anchor_dr(B.mt), fabsf(A.z)));
  if (!(lhs <= rhs)) return false;                                                       // L2
  c_out = c;
  return true;
}

// Conservative prefilter of ls_eval (L1 and both L3; L2 is left to the exact test): exact pass => prefilter pass.
// c is formed from the same quantities as in ls_eval but with fused / approximate operations: cr by one FMA
// (|error| <= 2^-23 rA d, i.e. < 1e-8 in c), 1/sqrt by MUFU (2 ulp), 1/r precomputed per MD -- in all a few ulp of
// |c| <= 0.015, i.e. < 1e-8 absolute.  Margins: L1 1e-4 relative; L3 1e-4 relative + 3e-7 absolute, folded into the
// per-MD record by md_emit / k_md_finish: *a = (c_md, w*1.0001 + 3e-7, f*1.0001 | module-type bits, 1/r).  Rejections are positive
// comparisons, so a NaN anywhere lets the pair through to the exact test.
// kinvA = -2 / rA.
__device__ __forceinline__ bool ls_prefilter(float4 Ap, float4 Aa, float kinvA, float4 Bp, float4 Ba) {
  const float dx = Bp.x - Ap.x, dy = Bp.y - Ap.y;
  const float cr = fmaf(Ap.x, dy, -(Ap.y * dx));
  const float dd = fmaf(dx, dx, dy * dy);
  const float c = (cr * rsqrt_fast(dd)) * (kinvA * Ba.w);
  const float ac = fabsf(c);
  const bool rej = (ac > LST_C_MAX105 * 1.0001f) | (fabsf(Aa.x - c) > fmaf(Aa.z, ac, Aa.y)) | (fabsf(Ba.x - c) > fmaf(Ba.z, ac, Ba.y));
  return !rej | (dd < 1.0e-30f);      // dd ~ 0: the approximations may overflow where the exact test does not
}

struct Pt {   // anchor position + long-direction tolerances
  float x, y, z, dz, dr;
};
__device__ __forceinline__ Pt make_pt(float4 p, int mt) {
  Pt q; q.x = p.x; q.y = p.y; q.z = p.z; q.dz = anchor_dz(mt); q.dr = anchor_dr(mt);
  return q;
}

// SPEC.md 4.3 `triplet`: Menger curvature (T1/Q1) and r-z linearity (T2/Q2)
__device__ __forceinline__ bool triplet_eval(const Pt& A, const Pt& B, const Pt& C, float& k_out) {
  const float abx = fs(B.x, A.x), aby = fs(B.y, A.y);
  const float acx = fs(C.x, A.x), acy = fs(C.y, A.y);
  const float bcx = fs(C.x, B.x), bcy = fs(C.y, B.y);
  const float dab = fq(fa(fm(abx, abx), fm(aby, aby)));
  const float dbc = fq(fa(fm(bcx, bcx), fm(bcy, bcy)));
  const float dac = fq(fa(fm(acx, acx), fm(acy, acy)));
  const float k = fd(fm(-2.0f, fs(fm(abx, acy), fm(aby, acx))), fm(fm(dab, dbc), dac));
  if (!(fabsf(k) <= LST_C_MAX105)) return false;                                         // T1
  const float tab = fm(fm(dab, k), 0.5f), tbc = fm(fm(dbc, k), 0.5f);
  const float sab = fm(dab, arcfac(fm(tab, tab)));
  const float sbc = fm(dbc, arcfac(fm(tbc, tbc)));
  const float zab = fs(B.z, A.z), zbc = fs(C.z, B.z);
  const float lhs = fabsf(fs(fm(zab, sbc), fm(zbc, sab)));
  float rhs = fm(fa(A.dz, B.dz), sbc);
  rhs = fa(rhs, fm(fa(B.dz, C.dz), sab));
  rhs = fa(rhs, fm(fa(A.dr, B.dr), fabsf(zbc)));
  rhs = fa(rhs, fm(fa(B.dr, C.dr), fabsf(zab)));
  rhs = fa(rhs, fm(0.05f, fa(sab, sbc)));
  if (!(lhs <= rhs)) return false;                                                       // T2
  k_out = k;
  return true;
}

// SPEC.md 4.6: derived pLS helix quantities
struct Pls {
  float cx, cy, h, cot, sec, z0;
};
__device__ __forceinline__ Pls pls_derive(float px, float py, float pz, float z0, int q) {
  Pls p;
  const float pt = fq(fa(fm(px, px), fm(py, py)));
  const float R = fd(pt, LST_KAPPA);
  const float qR = fm((float)q, R);
  p.cx = fd(fm(qR, py), pt);
  p.cy = fd(-fm(qR, px), pt);
  p.h = fd(0.5f, R);
  p.cot = fd(pz, pt);
  p.sec = fq(fa(1.0f, fm(p.cot, p.cot)));
  p.z0 = z0;
  return p;
}
// transverse half of the anchor test (the cheap early-out): returns pass, e and dT
__device__ __forceinline__ bool pls_anchor_t(const Pls& p, float x, float y, float r, float& e, float& dT) {
  const float r2 = fm(r, r);
  const float wv = fa(fm(x, p.cx), fm(y, p.cy));
  e = fm(fs(r2, fm(2.0f, wv)), p.h);
  dT = fa(fa(fm(0.003f, r), fm(0.03f, fm(r2, p.h))), 0.02f);
  return fabsf(e) <= dT;
}
// full anchor test; adds the two chi2 terms when it passes
__device__ __forceinline__ bool pls_anchor(const Pls& p, float4 a, int mt, float& chi2) {
  float e, dT;
  if (!pls_anchor_t(p, a.x, a.y, a.w, e, dT)) return false;
  const float t = fm(a.w, p.h);
  const float s = fm(a.w, arcfac(fm(t, t)));
  const float zres = fs(a.z, fa(p.z0, fm(s, p.cot)));
  float dZ = fa(anchor_dz(mt), fm(anchor_dr(mt), fabsf(p.cot)));
  dZ = fa(dZ, fm(0.003f, fm(s, p.sec)));
  dZ = fa(dZ, 0.05f);
  if (!(fabsf(zres) <= dZ)) return false;
  const float u = fd(e, dT), v = fd(zres, dZ);
  chi2 = fa(chi2, fm(u, u));
  chi2 = fa(chi2, fm(v, v));
  return true;
}

}  // namespace lst
