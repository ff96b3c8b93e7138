// fx_vec2.cuh -- two-wide fp64 value type for the pair kernel: every operation is written for both zones of a thread
// back to back, so that two independent dependency chains sit next to each other in the instruction stream (the fp64
// pipe has 8 cycles of dependent latency and the pair kernel runs three warps per scheduler: one chain per warp leaves
// it idle).  The generic routines below are the a2..a4 arithmetic of fx_physics.cuh (fx_c2p_v2, fx_minmod_sel,
// fx_riemann_v2), written once for T = double and T = d2, with three changes: the HLLC side choice S* >= 0 <=> num <= 0
// is read from the sign bit of num (num = +0 goes right: the star flux is continuous across S* = 0), the floor tests
// x < floor (floor > 0) are signed 64-bit integer compares, and the two HLLC quotients come from two MUFU seeds.
#pragma once
#include "fx_physics.cuh"

namespace fx2 {

struct d2 { double a, b; };
struct m2 { bool a, b; };
#define FX2 __device__ __forceinline__

FX2 d2 mk(double a, double b) { d2 r; r.a = a; r.b = b; return r; }
FX2 d2 operator+(d2 x, d2 y) { return mk(x.a + y.a, x.b + y.b); }
FX2 d2 operator-(d2 x, d2 y) { return mk(x.a - y.a, x.b - y.b); }
FX2 d2 operator*(d2 x, d2 y) { return mk(x.a * y.a, x.b * y.b); }
FX2 d2 operator*(double s, d2 y) { return mk(s * y.a, s * y.b); }
FX2 d2 operator*(d2 x, double s) { return mk(x.a * s, x.b * s); }
FX2 d2 operator+(double s, d2 y) { return mk(s + y.a, s + y.b); }
FX2 d2 operator-(d2 x) { return mk(-x.a, -x.b); }
FX2 d2 vfma(d2 x, d2 y, d2 z) { return mk(fma(x.a, y.a, z.a), fma(x.b, y.b, z.b)); }
FX2 d2 vfma(double s, d2 y, d2 z) { return mk(fma(s, y.a, z.a), fma(s, y.b, z.b)); }
FX2 d2 vfma(d2 x, d2 y, double s) { return mk(fma(x.a, y.a, s), fma(x.b, y.b, s)); }
FX2 d2 vfma(double s, d2 y, double t) { return mk(fma(s, y.a, t), fma(s, y.b, t)); }
FX2 d2 vfma(d2 x, double s, d2 z) { return mk(fma(x.a, s, z.a), fma(x.b, s, z.b)); }
FX2 double vfma(double x, double y, double z) { return fma(x, y, z); }

FX2 d2 rcp_seed(d2 x) {
  d2 y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y.a) : "d"(x.a));
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y.b) : "d"(x.b));
  return y;
}
FX2 double rcp_seed(double x) { double y; asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }
FX2 d2 rsqrt_seed(d2 x) {
  d2 y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y.a) : "d"(x.a));
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y.b) : "d"(x.b));
  return y;
}
FX2 double rsqrt_seed(double x) { double y; asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x)); return y; }

// one cubic Newton step on the MUFU seed (fx_physics.cuh: fx_rcp3, fx_rsqrt3, fx_sqrt3)
template <class T> FX2 T rcp3(T x) {
  const T y = rcp_seed(x);
  const T e = vfma(-x, y, 1.0);
  return vfma(y, vfma(e, e, e), y);
}
template <class T> FX2 T rsqrt3(T x) {
  const T y = rsqrt_seed(x);
  const T e = vfma(-(x * y), y, 1.0);
  return vfma(y * e, vfma(0.375, e, 0.5), y);
}
template <class T> FX2 T sqrt3(T x) {
  const T y = rsqrt_seed(x);
  const T g = x * y;
  const T e = vfma(-g, y, 1.0);
  return vfma(g * e, vfma(0.375, e, 0.5), g);
}

FX2 bool hi_neg(double x) { return __double2hiint(x) < 0; }
FX2 m2 hi_neg(d2 x) { m2 m; m.a = __double2hiint(x.a) < 0; m.b = __double2hiint(x.b) < 0; return m; }
FX2 bool meq(bool p, bool q) { return p == q; }
FX2 m2 meq(m2 p, m2 q) { m2 m; m.a = p.a == q.a; m.b = p.b == q.b; return m; }
FX2 double sel(bool c, double x, double y) { return c ? x : y; }
FX2 d2 sel(m2 c, d2 x, d2 y) { return mk(c.a ? x.a : y.a, c.b ? x.b : y.b); }
FX2 d2 sel(m2 c, d2 x, double y) { return mk(c.a ? x.a : y, c.b ? x.b : y); }
FX2 double min_sel(double a, double b) { return (a < b) ? a : b; }
FX2 double max_sel(double a, double b) { return (a > b) ? a : b; }
FX2 d2 min_sel(d2 x, d2 y) { return mk(x.a < y.a ? x.a : y.a, x.b < y.b ? x.b : y.b); }
FX2 d2 max_sel(d2 x, d2 y) { return mk(x.a > y.a ? x.a : y.a, x.b > y.b ? x.b : y.b); }
FX2 bool ge0(double x) { return x >= 0.0; }
FX2 bool le0(double x) { return x <= 0.0; }
FX2 m2 ge0(d2 x) { m2 m; m.a = x.a >= 0.0; m.b = x.b >= 0.0; return m; }
FX2 m2 le0(d2 x) { m2 m; m.a = x.a <= 0.0; m.b = x.b <= 0.0; return m; }
FX2 d2 vabs(d2 x) { return mk(fabs(x.a), fabs(x.b)); }
FX2 double vabs(double x) { return fabs(x); }

// a3 [O3, A4, B8]: minmod, one fp64 compare + integer selects (fx_minmod_sel)
FX2 double minmod(double a, double b) { return fx_minmod_sel(a, b); }
FX2 d2 minmod(d2 x, d2 y) { return mk(fx_minmod_sel(x.a, y.a), fx_minmod_sel(x.b, y.b)); }

// a2 [O2]: conserved -> primitive with primitive floors [A7]; status bits of either zone are OR-ed
FX2 unsigned c2p(const FxParams &P, const d2 U[5], d2 W[5], d2 *inv_rho = nullptr) {
  unsigned hit = (fx_hi_nonfinite(__double2hiint(U[0].a)) || fx_hi_nonfinite(__double2hiint(U[0].b))) ? FX_STATUS_NONFINITE : 0u;
  d2 rho = U[0];
  if (__double_as_longlong(rho.a) < __double_as_longlong(P.rho_floor)) { rho.a = P.rho_floor; hit |= FX_STATUS_RHO_FLOOR; }
  if (__double_as_longlong(rho.b) < __double_as_longlong(P.rho_floor)) { rho.b = P.rho_floor; hit |= FX_STATUS_RHO_FLOOR; }
  const d2 r = rcp3(rho);
  if (inv_rho) *inv_rho = r;
  const d2 u = U[1] * r, v = U[2] * r, w = U[3] * r;
  d2 p = P.gm1 * vfma(-0.5, vfma(U[3], w, vfma(U[2], v, U[1] * u)), U[4]);
  if (fx_hi_nonfinite(__double2hiint(p.a)) || fx_hi_nonfinite(__double2hiint(p.b))) hit |= FX_STATUS_NONFINITE;
  if (__double_as_longlong(p.a) < __double_as_longlong(P.p_floor)) { p.a = P.p_floor; hit |= FX_STATUS_P_FLOOR; }
  if (__double_as_longlong(p.b) < __double_as_longlong(P.p_floor)) { p.b = P.p_floor; hit |= FX_STATUS_P_FLOOR; }
  W[0] = rho; W[1] = u; W[2] = v; W[3] = w; W[4] = p;
  return hit;
}

// a4 [O4]: HLLC / HLLE flux in the face frame (the formulas and the order of fx_riemann_v2).
template <int RIEMANN, int WS, class T>
FX2 void riemann(const FxParams &P, const T WL[5], const T WR[5], T F[5]) {
  const T rL = WL[0], unL = WL[1], t1L = WL[2], t2L = WL[3], pL = WL[4];
  const T rR = WR[0], unR = WR[1], t1R = WR[2], t2R = WR[3], pR = WR[4];
  const T y = rsqrt3(rL * rR);
  const T gy = P.gamma * (y * y);
  const T c2L = (gy * rR) * pL, c2R = (gy * rL) * pR;
  const T cL = sqrt3(c2L), cR = sqrt3(c2R);
  T SL, SR;
  if (WS == 0) {
    const T t = rR * y;
    const T wl = rcp3(1.0 + t), wr = t * wl;
    const T dun = unR - unL, dt1 = t1R - t1L, dt2 = t2R - t2L;
    const T d2_ = vfma(dt2, dt2, vfma(dt1, dt1, dun * dun));
    const T un = vfma(wr, dun, unL);
    const T c2 = vfma((0.5 * P.gm1) * (wl * wr), d2_, vfma(wr, c2R - c2L, c2L));
    const T c = sqrt3(c2);
    SL = min_sel(unL - cL, un - c);
    SR = max_sel(unR + cR, un + c);
  } else {
    SL = min_sel(unL - cL, unR - cR);
    SR = max_sel(unL + cL, unR + cR);
  }
  if (RIEMANN == FX_RIEMANN_HLLE) {
    const T keL = 0.5 * vfma(t2L, t2L, vfma(t1L, t1L, unL * unL)), keR = 0.5 * vfma(t2R, t2R, vfma(t1R, t1R, unR * unR));
    const T EL = vfma(pL, P.igm1, rL * keL), ER = vfma(pR, P.igm1, rR * keR);
    const T mL = rL * unL, mR = rR * unR;
    const T FL[5] = {mL, vfma(mL, unL, pL), mL * t1L, mL * t2L, unL * (EL + pL)};
    const T FR[5] = {mR, vfma(mR, unR, pR), mR * t1R, mR * t2R, unR * (ER + pR)};
    const T UL[5] = {rL, mL, rL * t1L, rL * t2L, EL};
    const T UR[5] = {rR, mR, rR * t1R, rR * t2R, ER};
    const T iden = rcp3(SR - SL), ss = SL * SR;
    const auto supL = ge0(SL), supR = le0(SR);
#pragma unroll
    for (int v = 0; v < 5; ++v) {
      const T f = (SR * FL[v] - SL * FR[v] + ss * (UR[v] - UL[v])) * iden;
      F[v] = sel(supL, FL[v], sel(supR, FR[v], f));
    }
    return;
  }
  const T aL = rL * (SL - unL), aR = rR * (SR - unR);  // aL < 0 < aR
  const T num = (pR - pL) + vfma(aL, unL, -(aR * unR));
  const T D1 = aL - aR;                                // < 0, so S* = num / D1 >= 0  <=>  num <= 0
  const T Ss = num * rcp3(D1);
  const auto left = hi_neg(num);
  const T rK = sel(left, rL, rR), unK = sel(left, unL, unR), t1K = sel(left, t1L, t1R), t2K = sel(left, t2L, t2R);
  const T pK = sel(left, pL, pR);
  const T Ssel = sel(left, SL, SR);
  const T SK = sel(meq(hi_neg(Ssel), left), Ssel, 0.0);  // S_K clamped to 0 on the supersonic side
  const T dK = SK - unK;
  const T aK = rK * dK;
  const T g = num * rcp3(vfma(SK, D1, -num));          // S* / (S_K - S*)
  const T EK = vfma(0.5 * rK, vfma(t2K, t2K, vfma(t1K, t1K, unK * unK)), pK * P.igm1);
  const T ps = vfma(aK, Ss - unK, pK);                 // p*
  const T f0 = g * aK;                                 // rho* S*
  F[0] = f0;
  F[1] = vfma(f0, Ss, ps);
  F[2] = f0 * t1K;
  F[3] = f0 * t2K;
  F[4] = g * vfma(SK, ps, vfma(EK, dK, -(unK * pK)));
}

#undef FX2
}  // namespace fx2
