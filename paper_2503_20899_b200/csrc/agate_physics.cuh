// agate_physics.cuh — point functions of the AGATE finite-volume step (CUDA path).
//
// Everything here works in the ROTATED frame of one face: a state is
//     w[0]=rho  w[1]=u (normal velocity)  w[2]=v  w[3]=w (transverse, cyclic order)
//     w[4]=p    w[5]=Bn                   w[6]=Bt1 w[7]=Bt2
// and a flux F[8] is ordered the same way (F[1] = normal momentum flux, F[5] = flux of Bn).
// The callers (stage kernel, unit-test kernel) permute variables when they read/write shared or global memory,
// so ONE body of each Riemann solver serves the x, y and z sweeps.
//
// Citations: PAPER.md (P:Lnnn) and the readings Rn of DESIGN.md.
//   cons<->prim            P:L140 (R2: p/(gamma-1))
//   eq.4 limiter           P:L97-102 (R7)
//   fast speed eq.12       P:L148-151 (R3), whistler speed eq.13
//   physical flux eqs.7-10 P:L128-140 with psi == 0 (R12)
//   HLL eq.5 + Davis eq.6  P:L104-116 (R8, R9)
//   HLLD                   R10 (Miyoshi-Kusano five-wave solver; outer speeds from eq.6; Bn = mean; F[Bn] = 0)
//   Hall v_T = v + v_H     P:L140 (R15)
//
// Functions are __host__ __device__ so that the host-only unit test (tests/test_physics_host.py) can compile
// this header with g++ and compare it against the oracle without a GPU.  The file shares nothing with oracle/.
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define AG_HD __host__ __device__ __forceinline__
#else
#define AG_HD inline
#endif

namespace agate {

constexpr double kHlldEps = 1e-12;  // R10 guards
constexpr double kTiny = 1e-280;    // floor of a square-root argument that can be exactly zero

struct Phys {
  double gamma;   // adiabatic index
  double gm1;     // gamma - 1
  double igm1;    // 1 / (gamma - 1)
  double gogm1;   // gamma / (gamma - 1)
  double hgamma;  // gamma / 2
  double d_i;     // Hall: normalised ion inertial length
  double cwk;     // Hall: d_i * pi / (2 dx_min)   (eq.13 with k_max = pi / dx_min, R15)
  int cgl_form;   // CGL: 0 = logarithmic A of eq.18 (eqs.26-27), 1 = A of eq.16 (eqs.24-25)
};

AG_HD Phys make_phys(double gamma, double d_i, double dxmin) {
  Phys ph;
  ph.gamma = gamma;
  ph.gm1 = gamma - 1.0;
  ph.igm1 = 1.0 / (gamma - 1.0);
  ph.gogm1 = gamma / (gamma - 1.0);
  ph.hgamma = 0.5 * gamma;
  ph.d_i = d_i;
  ph.cwk = d_i * 3.14159265358979323846264338327950288 / (2.0 * dxmin);
  ph.cgl_form = 0;
  return ph;
}

// rotated slot r (rho,u,v,w,p,Bn,Bt1,Bt2) -> fixed variable index for face normal n
AG_HD int rot_var(int r, int n) {
  const int base = (r >= 5) ? 5 : 1;
  const int c = (r >= 5) ? r - 5 : r - 1;
  if (r == 0) return 0;
  if (r == 4) return 4;
  int d = n + c;
  d = (d >= 3) ? d - 3 : d;
  return base + d;
}

// rotated flux -> fixed (x,y,z) component order, by selects (no dynamic register indexing)
AG_HD void unrotate(int n, const double r[8], double f[8]) {
  f[0] = r[0];
  f[4] = r[4];
  f[1] = (n == 0) ? r[1] : ((n == 1) ? r[3] : r[2]);
  f[2] = (n == 0) ? r[2] : ((n == 1) ? r[1] : r[3]);
  f[3] = (n == 0) ? r[3] : ((n == 1) ? r[2] : r[1]);
  f[5] = (n == 0) ? r[5] : ((n == 1) ? r[7] : r[6]);
  f[6] = (n == 0) ? r[6] : ((n == 1) ? r[5] : r[7]);
  f[7] = (n == 0) ? r[7] : ((n == 1) ? r[6] : r[5]);
}

// min / max without the NaN-quieting of fmin / fmax (3 instructions instead of 6; the path never compares NaNs
// that it then keeps: an unphysical state is caught by the dt reduction, R14)
AG_HD double dmin(double a, double b) { return (b < a) ? b : a; }
AG_HD double dmax(double a, double b) { return (b > a) ? b : a; }
// Reciprocal, square root, reciprocal square root.  Device: the MUFU seed (rcp/rsqrt.approx.ftz.f64, ~20 bits)
// refined by Newton steps in straight-line DFMA code -- no special-case branch, no call.  Measured on B200 over
// 4M log-uniform inputs in [e^-20, e^20]: rcp and sqrt equal the IEEE results, rsqrt is within 2.7e-16 relative.
// Arguments on the path are positive and far from the denormal / overflow range (densities, pressures, squared
// speeds); a square-root argument that can be exactly zero is floored at kTiny by the caller.
// Host (tests/host_shim): plain IEEE operations.
AG_HD double rcp(double x) {
#if defined(__CUDA_ARCH__)
  double y;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y, 1.0);               // 1 - x y          (~2^-21)
  return fma(y, fma(e, e, e), y);                 // third-order step  y (1 + e + e^2);  the e^3 term is below 2^-60
#else
  return 1.0 / x;
#endif
}
AG_HD double rsq(double x) {
#if defined(__CUDA_ARCH__)
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double t = x * r;
  const double e = fma(-t, r, 1.0);               // 1 - x r^2
  return fma(r * e, fma(0.375, e, 0.5), r);       // third-order step: r (1 + e/2 + 3 e^2 / 8)
#else
  return 1.0 / sqrt(x);
#endif
}
// sqrt of a STRICTLY POSITIVE argument (callers clamp with kTiny where an exact zero can occur: rsqrt(0) = inf).
// Coupled third-order step on s = x r, h = r/2:  e = 1/2 - s h,  sqrt(x) = s (1 + e + 3 e^2 / 2) + O(e^3).
// 6 FP64 instructions after the MUFU seed; within 1-2 ulp of the IEEE result.
AG_HD double sqrt_pos(double x) {
#if defined(__CUDA_ARCH__)
  double r;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
  const double s = x * r;
  const double h = 0.5 * r;
  const double e = fma(-s, h, 0.5);
  return fma(s * e, fma(1.5, e, 1.0), s);
#else
  return sqrt(x);
#endif
}
// x with its sign flipped when m == sign bit (m = 0: unchanged).  One logic op instead of a negate + select.
AG_HD double xorsign(double x, unsigned long long m) {
#if defined(__CUDA_ARCH__)
  return __longlong_as_double(__double_as_longlong(x) ^ (long long)m);
#else
  return m ? -x : x;
#endif
}

// A1 (R2): fixed-frame conserved (rho, m, E, B) -> primitive (rho, v, p, B).  Frame-agnostic.
AG_HD void cons_to_prim(const Phys& ph, const double U[8], double W[8]) {
  const double ir = rcp(U[0]);
  const double vx = U[1] * ir, vy = U[2] * ir, vz = U[3] * ir;
  const double v2 = vx * vx + vy * vy + vz * vz;
  const double b2 = U[5] * U[5] + U[6] * U[6] + U[7] * U[7];
  W[0] = U[0]; W[1] = vx; W[2] = vy; W[3] = vz;
  W[4] = ph.gm1 * (U[4] - 0.5 * U[0] * v2 - 0.5 * b2);
  W[5] = U[5]; W[6] = U[6]; W[7] = U[7];
}

// eq.4 (R7).  dp = W(i+1)-W(i), dm = W(i)-W(i-1).
AG_HD double limited_slope(int limiter, double beta, double dp, double dm) {
  if (limiter == 2) {
    // minmod[beta dp, beta dm, (dp+dm)/2] for dp, dm of one sign:  beta min(|dp|,|dm|) = min(beta|dp|, beta|dm|) and
    // |dp+dm| = |dp|+|dm| exactly, so this is the same value with one multiply and one compare fewer.
    const double a = fabs(dp), b = fabs(dm);
    const double m = dmin(beta * dmin(a, b), 0.5 * (a + b));
#if defined(__CUDA_ARCH__)
    // sign test on the high words (integer pipe); a zero difference gives m == 0 whatever its sign bit
    const int hp = __double2hiint(dp), hm = __double2hiint(dm);
    const int hi = (__double2hiint(m) | (hp & 0x80000000)) & ~((hp ^ hm) >> 31);
    const int lo = __double2loint(m) & ~((hp ^ hm) >> 31);
    return __hiloint2double(hi, lo);
#else
    return (dp * dm > 0.0) ? copysign(m, dp) : 0.0;
#endif
  }
  if (limiter == 1) return 0.5 * (dp + dm);
  return 0.0;
}

// Half of the eq.4 slope (what the face states W -+ dW/2 use), with the factor folded into the constants:
// hbeta = beta / 2.  Scaling by a power of two is exact, so this is 0.5 * limited_slope bit for bit.
// limiter 3 = eq.4 at beta = 1 (minmod): min(|dp|,|dm|)/2 never exceeds (|dp|+|dm|)/4, rounding included (the sum of
// two doubles is at least twice the smaller one), so the third argument of eq.4 drops out bit for bit.
AG_HD double half_slope(int limiter, double hbeta, double dp, double dm) {
  if (limiter >= 2) {
    const double a = fabs(dp), b = fabs(dm);
    const double m = (limiter == 3) ? 0.5 * dmin(a, b) : dmin(hbeta * dmin(a, b), 0.25 * (a + b));
#if defined(__CUDA_ARCH__)
    const int hp = __double2hiint(dp), hm = __double2hiint(dm);
    const int hi = (__double2hiint(m) | (hp & 0x80000000)) & ~((hp ^ hm) >> 31);
    const int lo = __double2loint(m) & ~((hp ^ hm) >> 31);
    return __hiloint2double(hi, lo);
#else
    return (dp * dm > 0.0) ? copysign(m, dp) : 0.0;
#endif
  }
  if (limiter == 1) return 0.25 * (dp + dm);
  return 0.0;
}

// x with its sign flipped when bit 31 of hmask is set (hmask = 0 or 0x80000000): one logic op on the high word
AG_HD double flipsign_hi(double x, int hmask) {
#if defined(__CUDA_ARCH__)
  return __hiloint2double(__double2hiint(x) ^ hmask, __double2loint(x));
#else
  return hmask ? -x : x;
#endif
}
AG_HD int signbit_hi(double x) {
#if defined(__CUDA_ARCH__)
  return __double2hiint(x) & (int)0x80000000;
#else
  return signbit(x) ? (int)0x80000000 : 0;
#endif
}

// A2 in one piece (eqs.2-4, R7): the two face states of cell b with neighbours a (low) and c (high),
//   lo = W - dW/2  (right state of the low face),   hi = W + dW/2  (left state of the high face).
// limiter 2 (eq.4):  dW = minmod[beta dp, beta dm, (dp+dm)/2],  dp = c-b, dm = b-a.  For dp, dm of one sign the
// candidate of smaller magnitude of {dp, dm} is picked WITH its sign, scaled by 2 beta, and compared in magnitude
// with the centred difference c - a (which carries the same sign), so the result needs no sign fix-up; opposite
// signs (or a zero) give 0.  The common factor 1/4 rides in the two fused multiply-adds that form the states:
// 8 FP64-pipe instructions per variable and direction (12 with half_slope and separate adds).  The scalings are by
// powers of two, so the only difference from half_slope is c - a against dp + dm (one rounding of the centred term).
// limiter 3 = eq.4 at beta = 1 (minmod; the centred term never binds, see half_slope).  beta2 = 2 beta.
AG_HD void plm_faces(int limiter, double beta2, double a, double b, double c, double& lo, double& hi) {
  if (limiter >= 2) {
    const double dp = c - b, dm = b - a;
    const double m = (fabs(dp) < fabs(dm)) ? dp : dm;      // smaller magnitude, with its sign
    // the factor of the fused multiply-adds carries the zero for opposite signs: 0.25 (0.5) and 0.0 differ in the
    // high word only, so that is one 32-bit select
#if defined(__CUDA_ARCH__)
    const bool opp = (__double2hiint(dp) ^ __double2hiint(dm)) < 0;
    const double q = __hiloint2double(opp ? 0 : ((limiter == 3) ? 0x3FE00000 : 0x3FD00000), 0);
#else
    const bool opp = signbit(dp) != signbit(dm);
    const double q = opp ? 0.0 : ((limiter == 3) ? 0.5 : 0.25);
#endif
    if (limiter == 3) {
      lo = fma(-q, m, b);
      hi = fma(q, m, b);
    } else {
      const double t = beta2 * m, cen = c - a;
      const double x = (fabs(t) < fabs(cen)) ? t : cen;    // a zero difference of one sign: m = 0 -> t = 0 -> x = 0
      lo = fma(-q, x, b);
      hi = fma(q, x, b);
    }
    return;
  }
  if (limiter == 1) {
    const double cen = c - a;
    lo = fma(-0.25, cen, b);
    hi = fma(0.25, cen, b);
    return;
  }
  lo = b;
  hi = b;
}

// Per-side quantities every solver needs.
struct Side {
  double ir;    // 1/rho
  double B2;    // |B|^2
  double pt;    // p + |B|^2/2
  double cf;    // fast speed along the normal, eq.12 (R3)
};

AG_HD Side side_of(const Phys& ph, const double w[8]) {
  Side s;
  s.ir = rcp(w[0]);
  s.B2 = w[5] * w[5] + w[6] * w[6] + w[7] * w[7];
  s.pt = w[4] + 0.5 * s.B2;
  const double a2 = ph.gamma * w[4] * s.ir;          // v_s^2 = gamma p / rho
  const double b2 = s.B2 * s.ir;                     // v_A^2 = B^2 / rho
  const double sm = a2 + b2;
  const double rad = dmax(sm * sm - 4.0 * a2 * (w[5] * w[5] * s.ir), kTiny);
  s.cf = sqrt_pos(0.5 * (sm + sqrt_pos(rad)));
  return s;
}

// eq.13:  c_w = aw + sqrt(aw^2 + v_A^2),  aw = d_i pi |B| / (2 rho dx_min)
AG_HD double whistler_speed(const Phys& ph, const double w[8], const Side& s) {
  const double aw = ph.cwk * sqrt_pos(dmax(s.B2, kTiny)) * s.ir;
  return aw + sqrt_pos(dmax(aw * aw + s.B2 * s.ir, kTiny));
}

// Total energy density (R2).
AG_HD double energy_of(const Phys& ph, const double w[8], const Side& s) {
  return 0.5 * w[0] * (w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) + 0.5 * s.B2 + w[4] * ph.igm1;
}

// eqs.7-10 with psi == 0 in the rotated frame; vH = Hall velocity (rotated) or nullptr (ideal: v_T = v).
AG_HD void phys_flux(const Phys& ph, const double w[8], const Side& s, const double* vH, double f[8]) {
  const double ru = w[0] * w[1];
  double tn = w[1], t1 = w[2], t2 = w[3];
  if (vH) { tn += vH[0]; t1 += vH[1]; t2 += vH[2]; }
  const double v2 = w[1] * w[1] + w[2] * w[2] + w[3] * w[3];
  const double tB = tn * w[5] + t1 * w[6] + t2 * w[7];
  f[0] = ru;                                                                    // eq.7
  f[1] = ru * w[1] - w[5] * w[5] + s.pt;                                        // eq.8
  f[2] = ru * w[2] - w[5] * w[6];
  f[3] = ru * w[3] - w[5] * w[7];
  f[4] = (0.5 * w[0] * v2 + ph.gogm1 * w[4]) * w[1] + s.B2 * tn - tB * w[5];     // eq.9
  f[5] = 0.0;                                                                   // eq.10, c == n
  f[6] = tn * w[6] - w[5] * t1;
  f[7] = tn * w[7] - w[5] * t2;
}

// HLL, eq.5 with the Davis speeds eq.6; all 8 components through eq.5 (R9).
// Hall (R15): c = max(c_f, c_w) per side, v_H^a = -d_i J / rho^a in phi.  J in the rotated frame.
// Written for the FP64 pipe: the fast speed from rho c_f^2 = N = H + sqrt(H^2 - gamma p Bn^2), H = (gamma p + B^2)/2
// (no reciprocal of rho in ideal MHD: c_f = N rsqrt(N rho)); each side's physical flux and conserved vector share their
// kinetic and magnetic terms; eq.5 as  F = a F_L + b F_R + c (U_R - U_L)  with a = s_R/(s_R-s_L), b = -s_L/(s_R-s_L),
// c = s_L s_R/(s_R-s_L) (three multiplies once instead of one per component).  ~150 FP64 instructions per face
// (ideal), ~205 (Hall), from ~190 / ~235 as eq.5 is printed.
template <bool HALL>
AG_HD void hll_side(const Phys& ph, const double w[8], const double* dJ, double& cout, double f[8], double& E, double& rv,
                    double& rw) {
  const double bn2 = w[5] * w[5];
  const double hB = 0.5 * fma(w[7], w[7], fma(w[6], w[6], bn2));           // |B|^2 / 2
  const double pt = w[4] + hB;
  const double g = ph.hgamma * w[4], H = g + hB;
  const double Q = dmax(fma(H, H, -(g * (bn2 + bn2))), kTiny);
  const double N = H + sqrt_pos(Q);                                         // rho c_f^2 (eq.12, R3)
  double tn = w[1], t1 = w[2], t2 = w[3];
  if (HALL) {
    const double ir = rcp(w[0]);
    const double B2 = hB + hB;
    double c = sqrt_pos(N * ir);
    const double aw = ph.cwk * sqrt_pos(dmax(B2, kTiny)) * ir;              // eq.13
    c = dmax(c, aw + sqrt_pos(dmax(fma(aw, aw, B2 * ir), kTiny)));
    cout = c;
    tn = fma(-dJ[0], ir, tn); t1 = fma(-dJ[1], ir, t1); t2 = fma(-dJ[2], ir, t2);   // v_T = v - d_i J / rho
  } else {
    cout = N * rsq(N * w[0]);
  }
  const double ru = w[0] * w[1];
  const double ke = (0.5 * w[0]) * fma(w[3], w[3], fma(w[2], w[2], w[1] * w[1]));
  E = fma(w[4], ph.igm1, ke + hB);                                          // P:L140, R2
  rv = w[0] * w[2]; rw = w[0] * w[3];
  const double tB = fma(t2, w[7], fma(t1, w[6], tn * w[5]));
  f[0] = ru;                                                                // eq.7
  f[1] = fma(ru, w[1], pt - bn2);                                           // eq.8
  f[2] = fma(ru, w[2], -(w[5] * w[6]));
  f[3] = fma(ru, w[3], -(w[5] * w[7]));
  f[4] = fma(-tB, w[5], fma(hB + hB, tn, fma(ph.gogm1, w[4], ke) * w[1]));  // eq.9
  f[5] = 0.0;                                                               // eq.10, c == n
  f[6] = fma(tn, w[6], -(w[5] * t1));
  f[7] = fma(tn, w[7], -(w[5] * t2));
}

template <bool HALL>
AG_HD void flux_hll(const Phys& ph, const double L[8], const double R[8], const double* J, double F[8]) {
  double dJ[3] = {0.0, 0.0, 0.0};
  if (HALL) { dJ[0] = ph.d_i * J[0]; dJ[1] = ph.d_i * J[1]; dJ[2] = ph.d_i * J[2]; }
  double fl[8], fr[8], cl, cr, El, Er, rvl, rwl, rvr, rwr;
  hll_side<HALL>(ph, L, dJ, cl, fl, El, rvl, rwl);
  hll_side<HALL>(ph, R, dJ, cr, fr, Er, rvr, rwr);
  const double sL = dmin(dmin(L[1] - cl, R[1] - cr), 0.0);       // s'_L = min(s_L, 0)
  const double sR = dmax(dmax(L[1] + cl, R[1] + cr), 0.0);       // s'_R = max(s_R, 0)
  const double iw = rcp(sR - sL);
  const double a = sR * iw, b = -(sL * iw), c = sL * a;
  F[0] = fma(a, fl[0], fma(b, fr[0], c * (R[0] - L[0])));
  F[1] = fma(a, fl[1], fma(b, fr[1], c * (fr[0] - fl[0])));      // U[1] = rho u = F[0] of the side
  F[2] = fma(a, fl[2], fma(b, fr[2], c * (rvr - rvl)));
  F[3] = fma(a, fl[3], fma(b, fr[3], c * (rwr - rwl)));
  F[4] = fma(a, fl[4], fma(b, fr[4], c * (Er - El)));
  F[5] = c * (R[5] - L[5]);                                      // eq.5 on Bn (R9): both physical fluxes are zero
  F[6] = fma(a, fl[6], fma(b, fr[6], c * (R[6] - L[6])));
  F[7] = fma(a, fl[7], fma(b, fr[7], c * (R[7] - L[7])));
}

// Star-state transverse components behind one outer wave (R10):  S = outer speed, m = rho (S - u).
struct Star {
  double rs;          // rho*
  double idS;         // 1 / (S - SM)
  double v, w, b1, b2;
};

AG_HD Star star_of(const double a[8], double S, double m, double SM, double bn, double bn2, double pts) {
  Star st;
  const double dS = S - SM;
  const double den = m * dS - bn2;
  const bool degenerate = fabs(den) < kHlldEps * pts;       // B_t = 0 and c_f = |Bn|/sqrt(rho)
  const double dsafe = degenerate ? 1.0 : den;
  const double r1 = rcp(dS * dsafe);                         // one reciprocal serves 1/dS and 1/den
  st.idS = dsafe * r1;
  const double iden = dS * r1;
  st.rs = m * st.idS;
  const double t = degenerate ? 0.0 : bn * (SM - a[1]) * iden;
  const double f = degenerate ? 1.0 : (m * (S - a[1]) - bn2) * iden;
  st.v = a[2] - a[6] * t;
  st.w = a[3] - a[7] * t;
  st.b1 = a[6] * f;
  st.b2 = a[7] * f;
  return st;
}

// HLLD (R10), straight-line.  The star-state formulas are the same for both sides with the side's own outer speed,
// so nothing is mirrored: both star states are computed (a warp needs both as soon as one lane is in a double-star
// region), the double-star state is symmetric in L and R, and the upwind side alpha (L if S_M >= 0, else R) enters
// through selects of its state and one sign  sigma = +1 (L) / -1 (R).  The double-star and supersonic cases switch
// their terms on and off through the wave speed that multiplies them, so there is no branch and no divergence.
AG_HD double sel(bool c, double a, double b) { return c ? a : b; }

AG_HD void flux_hlld_general(const Phys& ph, const double L[8], const double R[8], double F[8]) {
  const double bn = 0.5 * (L[5] + R[5]);                     // single-valued Bn: arithmetic mean
  const double bn2 = bn * bn;
  // per-side speeds with Bn := bn (the caller's L[5], R[5] are not used below)
  const double irl = rcp(L[0]), irr = rcp(R[0]);
  const double B2l = bn2 + L[6] * L[6] + L[7] * L[7], B2r = bn2 + R[6] * R[6] + R[7] * R[7];
  const double ptl = L[4] + 0.5 * B2l, ptr = R[4] + 0.5 * B2r;
  const double a2l = ph.gamma * L[4] * irl, sml = a2l + B2l * irl;
  const double a2r = ph.gamma * R[4] * irr, smr = a2r + B2r * irr;
  const double radl = dmax(sml * sml - 4.0 * a2l * (bn2 * irl), kTiny);
  const double radr = dmax(smr * smr - 4.0 * a2r * (bn2 * irr), kTiny);
  const double cfl = sqrt_pos(0.5 * (sml + sqrt_pos(radl)));
  const double cfr = sqrt_pos(0.5 * (smr + sqrt_pos(radr)));
  const double SL = dmin(L[1] - cfl, R[1] - cfr);            // eq.6
  const double SR = dmax(L[1] + cfl, R[1] + cfr);
  const double mL = L[0] * (SL - L[1]), mR = R[0] * (SR - R[1]);     // mL < 0 < mR
  const double idm = rcp(mR - mL);
  const double SM = (mR * R[1] - mL * L[1] - ptr + ptl) * idm;
  const double pts = (mR * ptl - mL * ptr + mL * mR * (R[1] - L[1])) * idm;

  const Star l = star_of(L, SL, mL, SM, bn, bn2, pts);
  const Star r = star_of(R, SR, mR, SM, bn, bn2, pts);
  // double-star state (symmetric in L, R)
  const double irsl = rsq(l.rs), irsr = rsq(r.rs);
  const double ql = l.rs * irsl, qr = r.rs * irsr;           // sqrt(rho*)
  const double I = rcp(ql + qr);
  const double sgn = (bn > 0.0) ? 1.0 : -1.0;
  const double qq = ql * qr * sgn;
  const double vss = (ql * l.v + qr * r.v + (r.b1 - l.b1) * sgn) * I;
  const double wss = (ql * l.w + qr * r.w + (r.b2 - l.b2) * sgn) * I;
  const double b1ss = (ql * r.b1 + qr * l.b1 + qq * (r.v - l.v)) * I;
  const double b2ss = (ql * r.b2 + qr * l.b2 + qq * (r.w - l.w)) * I;

  // upwind side
  const bool supL = SL >= 0.0;
  const bool supR = !supL && (SR <= 0.0);
  const bool rt = supL ? false : (supR ? true : (SM < 0.0));
  double A[8];
  A[0] = sel(rt, R[0], L[0]); A[1] = sel(rt, R[1], L[1]); A[2] = sel(rt, R[2], L[2]); A[3] = sel(rt, R[3], L[3]);
  A[4] = sel(rt, R[4], L[4]); A[5] = bn;                  A[6] = sel(rt, R[6], L[6]); A[7] = sel(rt, R[7], L[7]);
  Side sa;
  sa.ir = 0.0; sa.cf = 0.0;
  sa.B2 = sel(rt, B2r, B2l);
  sa.pt = sel(rt, ptr, ptl);
  const double SA = sel(rt, SR, SL);
  Star a;
  a.rs = sel(rt, r.rs, l.rs); a.idS = sel(rt, r.idS, l.idS);
  a.v = sel(rt, r.v, l.v);    a.w = sel(rt, r.w, l.w);
  a.b1 = sel(rt, r.b1, l.b1); a.b2 = sel(rt, r.b2, l.b2);
  const double qa = sel(rt, qr, ql), irsa = sel(rt, irsr, irsl);
  const double sig = rt ? -1.0 : 1.0;

  double fa[8];
  phys_flux(ph, A, sa, nullptr, fa);
  const double EA = energy_of(ph, A, sa);
  const double vBA = A[1] * bn + A[2] * A[6] + A[3] * A[7];
  const double vBsA = SM * bn + a.v * a.b1 + a.w * a.b2;
  const double vBss = SM * bn + vss * b1ss + wss * b2ss;
  const double EsA = ((SA - A[1]) * EA - sa.pt * A[1] + pts * SM + bn * (vBA - vBsA)) * a.idS;

  // S*_alpha = SM - sigma |Bn| / sqrt(rho*_alpha) lies on the far side of zero  <=>  SM^2 rho*_alpha < Bn^2
  const bool sup = supL || supR;
  const bool twostar = (SM * SM * a.rs < bn2) && !(0.5 * bn2 < kHlldEps * pts) && !sup;
  const double SAe = sup ? 0.0 : SA;                          // supersonic: F = F_alpha
  const double Sse = twostar ? (SM - sig * (fabs(bn) * irsa)) : 0.0;   // single-star: no double-star jump
  F[0] = fa[0] + SAe * (a.rs - A[0]);
  F[1] = fa[1] + SAe * (a.rs * SM - A[0] * A[1]);
  F[2] = fa[2] + SAe * (a.rs * a.v - A[0] * A[2]) + Sse * (a.rs * (vss - a.v));
  F[3] = fa[3] + SAe * (a.rs * a.w - A[0] * A[3]) + Sse * (a.rs * (wss - a.w));
  F[4] = fa[4] + SAe * (EsA - EA) - Sse * (qa * (vBsA - vBss) * (sgn * sig));
  F[5] = 0.0;                                                // F[Bn] = 0 in every branch (R10)
  F[6] = fa[6] + SAe * (a.b1 - A[6]) + Sse * (b1ss - a.b1);
  F[7] = fa[7] + SAe * (a.b2 - A[7]) + Sse * (b2ss - a.b2);
}

// HLLD (R10), the common case: a face inside the Riemann fan (S_L < 0 < S_R) whose star states are regular
// (|den| >= eps pt*).  Returns true when the face is NOT of that kind (supersonic or degenerate) -- its F is then
// meaningless and the caller takes flux_hlld_general.  What makes it lean:
//   * 1/rho is only needed inside the fast speed:  c_f = sqrt(N / rho),  N = H + sqrt(H^2 - gamma p Bn^2),
//     H = (gamma p + B^2)/2, evaluated as N * rsqrt(N rho): one root-type Newton chain less per side, no reciprocal.
//   * pt* = pt_L + m_L (S_M - u_L), the Rankine-Hugoniot condition across S_L (equal to the symmetric formula of
//     R10 up to rounding): one FMA.
//   * the star states satisfy the jump conditions, so the flux behind a wave is the physical flux function of the
//     state behind it:  F = (rho* S_M,  rho* S_M^2 + pt* - Bn^2,  rho* S_M v_t - Bn B_t,  (E + pt*) S_M - Bn (v.B),
//     0,  B_t S_M - Bn v_t)  with (v_t, B_t, E) of the single- or double-star state.  No physical flux of the outer
//     state, no jump terms.
//   * star transverse parts from one ratio  g = (S_M - u)/den:  v* = v - Bn B_t g,  B_t* = B_t (1 + m g).
AG_HD bool flux_hlld_fast(const Phys& ph, const double L[8], const double R[8], double F[8]) {
  const double bn = 0.5 * (L[5] + R[5]);                     // single-valued Bn: arithmetic mean
  const double bn2 = bn * bn, bn2x2 = bn2 + bn2, hbn2 = 0.5 * bn2;
  // Davis speeds eq.6 with eq.12 (R3) of the states with Bn := bn
  const double hBl = fma(0.5, fma(L[6], L[6], L[7] * L[7]), hbn2);       // |B|^2 / 2
  const double hBr = fma(0.5, fma(R[6], R[6], R[7] * R[7]), hbn2);
  const double ptl = L[4] + hBl, ptr = R[4] + hBr;
  const double gl = ph.hgamma * L[4], gr = ph.hgamma * R[4];             // gamma p / 2
  const double Hl = gl + hBl, Hr = gr + hBr;
  const double Ql = dmax(fma(Hl, Hl, -(gl * bn2x2)), kTiny), Qr = dmax(fma(Hr, Hr, -(gr * bn2x2)), kTiny);
  const double Nl = Hl + sqrt_pos(Ql), Nr = Hr + sqrt_pos(Qr);           // rho c_f^2
  const double cfl = Nl * rsq(Nl * L[0]), cfr = Nr * rsq(Nr * R[0]);
  const double SL = dmin(L[1] - cfl, R[1] - cfr);
  const double SR = dmax(L[1] + cfl, R[1] + cfr);
  const double dl = SL - L[1], dr = SR - R[1];
  const double mL = L[0] * dl, mR = R[0] * dr;                           // mL < 0 < mR
  const double idm = rcp(mR - mL);
  const double SM = fma(-mL, L[1], fma(mR, R[1], ptl - ptr)) * idm;
  const double eL = SM - L[1], eR = SM - R[1];
  const double pts = fma(mL, eL, ptl);
  const double epts = kHlldEps * pts;
  // star states behind the two outer waves
  const double dSl = SL - SM, dSr = SR - SM;
  const double denl = fma(mL, dSl, -bn2), denr = fma(mR, dSr, -bn2);
  const double r1l = rcp(dSl * denl), r1r = rcp(dSr * denr);             // one reciprocal serves 1/dS and 1/den
  const double idSl = denl * r1l, idSr = denr * r1r;
  const double rsl = mL * idSl, rsr = mR * idSr;                         // rho*
  const double ggl = eL * (dSl * r1l), ggr = eR * (dSr * r1r);
  const double tl = bn * ggl, tr = bn * ggr;
  const double fl = fma(mL, ggl, 1.0), fr = fma(mR, ggr, 1.0);
  const double vl = fma(-L[6], tl, L[2]), wl = fma(-L[7], tl, L[3]), b1l = L[6] * fl, b2l = L[7] * fl;
  const double vr = fma(-R[6], tr, R[2]), wr = fma(-R[7], tr, R[3]), b1r = R[6] * fr, b2r = R[7] * fr;
  const bool slow = !(SL < 0.0) || !(SR > 0.0) || (fabs(denl) < epts) || (fabs(denr) < epts);
  // double-star state (symmetric in L, R)
  const double ql = rsl * rsq(rsl), qr = rsr * rsq(rsr);                 // sqrt(rho*)
  const int sbn = signbit_hi(bn);                                        // sgn(Bn) = -1
  const double I = rcp(ql + qr), sI = flipsign_hi(I, sbn);
  const double qlI = ql * I, qrI = qr * I, qqI = ql * flipsign_hi(qrI, sbn);
  const double vss = fma(qlI, vl, fma(qrI, vr, sI * (b1r - b1l)));
  const double wss = fma(qlI, wl, fma(qrI, wr, sI * (b2r - b2l)));
  const double b1ss = fma(qlI, b1r, fma(qrI, b1l, qqI * (vr - vl)));
  const double b2ss = fma(qlI, b2r, fma(qrI, b2l, qqI * (wr - wl)));
  // upwind side alpha: L if S_M >= 0, else R
  const bool rt = SM < 0.0;
  const double rA = sel(rt, R[0], L[0]), uA = sel(rt, R[1], L[1]), vA = sel(rt, R[2], L[2]), wA = sel(rt, R[3], L[3]);
  const double pA = sel(rt, R[4], L[4]), b1A = sel(rt, R[6], L[6]), b2A = sel(rt, R[7], L[7]);
  const double hBA = sel(rt, hBr, hBl), ptA = sel(rt, ptr, ptl), dA = sel(rt, dr, dl);
  const double rsA = sel(rt, rsr, rsl), idSA = sel(rt, idSr, idSl), qA = sel(rt, qr, ql);
  const double vsA = sel(rt, vr, vl), wsA = sel(rt, wr, wl), b1sA = sel(rt, b1r, b1l), b2sA = sel(rt, b2r, b2l);
  const double EA = fma(pA, ph.igm1, fma(0.5 * rA, fma(uA, uA, fma(vA, vA, wA * wA)), hBA));
  const double SMbn = SM * bn;
  const double vBA = fma(uA, bn, fma(vA, b1A, wA * b2A));
  const double vBsA = fma(vsA, b1sA, fma(wsA, b2sA, SMbn));
  const double EsA = (fma(dA, EA, -(ptA * uA)) + fma(pts, SM, bn * (vBA - vBsA))) * idSA;
  // S*_alpha lies on the far side of zero  <=>  S_M^2 rho*_alpha < Bn^2;  no rotational waves when Bn^2/2 < eps pt*
  const bool twostar = (SM * SM * rsA < bn2) && !(hbn2 < epts);
  const double vBss = fma(vss, b1ss, fma(wss, b2ss, SMbn));
  // E** = E* -+ sqrt(rho*) (v*.B* - v**.B**) sgn(Bn):  - for alpha = L, + for alpha = R
  const double EssA = fma(-flipsign_hi(qA, sbn ^ (rt ? (int)0x80000000 : 0)), vBsA - vBss, EsA);
  const double vf = sel(twostar, vss, vsA), wf = sel(twostar, wss, wsA);
  const double b1f = sel(twostar, b1ss, b1sA), b2f = sel(twostar, b2ss, b2sA);
  const double Ef = sel(twostar, EssA, EsA), vBf = sel(twostar, vBss, vBsA);
  const double rSM = rsA * SM;
  F[0] = rSM;
  F[1] = fma(rSM, SM, pts - bn2);
  F[2] = fma(rSM, vf, -(bn * b1f));
  F[3] = fma(rSM, wf, -(bn * b2f));
  F[4] = fma(Ef + pts, SM, -(bn * vBf));
  F[5] = 0.0;                                                            // F[Bn] = 0 in every branch (R10)
  F[6] = fma(b1f, SM, -(bn * vf));
  F[7] = fma(b2f, SM, -(bn * wf));
  return slow;
}

#if defined(__CUDACC__)
// One out-of-line copy of the general body for all call sites of a kernel: the path is cold, and inlining it at
// every call site would put ~6 KB of never-executed code between the hot loops of the stage kernels.
static __device__ __noinline__ void flux_hlld_general_cold(const Phys* ph, const double* L, const double* R, double* F) {
  double l[8], r[8], f[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) { l[q] = L[q]; r[q] = R[q]; }
  flux_hlld_general(*ph, l, r, f);
#pragma unroll
  for (int q = 0; q < 8; ++q) F[q] = f[q];
}
#endif

// HLLD (R10): the lean form for regular faces inside the fan, the general straight-line form for a warp that holds a
// supersonic or degenerate face (rare: strong shocks, field-aligned states with B_t = 0).  A lane's result depends
// on its own face only, so the grid decomposition does not change the bits.
AG_HD void flux_hlld(const Phys& ph, const double L[8], const double R[8], double F[8]) {
  const bool slow = flux_hlld_fast(ph, L, R, F);
#if defined(__CUDA_ARCH__)
  if (__any_sync(__activemask(), slow)) {
    // copies in local memory for the call, so that L, R, F themselves stay in registers on the hot path
    double Lc[8], Rc[8], G[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) { Lc[q] = L[q]; Rc[q] = R[q]; }
    flux_hlld_general_cold(&ph, Lc, Rc, G);
    if (slow) {
#pragma unroll
      for (int q = 0; q < 8; ++q) F[q] = G[q];
    }
  }
#else
  if (slow) flux_hlld_general(ph, L, R, F);
#endif
}

template <int RIEMANN, bool HALL>
AG_HD void riemann_flux(const Phys& ph, const double L[8], const double R[8], const double* J, double F[8]) {
  if (RIEMANN == 1) flux_hlld(ph, L, R, F);
  else flux_hll<HALL>(ph, L, R, J, F);
}

// A7 per cell (R3, R4): |v|_2 + max(max_d c_f,d , c_w).  Returns a negative value for an unphysical
// cell (rho <= 0, p <= 0 or a non-finite speed) so that the caller can raise the flag (R14).
template <bool HALL>
AG_HD double cell_speed(const Phys& ph, const double U[8]) {
  double W[8];
  cons_to_prim(ph, U, W);
  if (!(W[0] > 0.0) || !(W[4] > 0.0)) return -1.0;
  const double ir = rcp(W[0]);
  const double B2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
  const double a2 = ph.gamma * W[4] * ir, b2 = B2 * ir, sm = a2 + b2;
  // max over d of c_f,d  ==  c_f at the smallest B_d^2 (R4)
  const double bmin2 = fmin(fmin(W[5] * W[5], W[6] * W[6]), W[7] * W[7]);
  const double rad = fmax(sm * sm - 4.0 * a2 * (bmin2 * ir), 0.0);
  double c = sqrt(0.5 * (sm + sqrt(rad)));
  if (HALL) {
    const double aw = ph.cwk * sqrt(B2) * ir;
    c = fmax(c, aw + sqrt(aw * aw + b2));
  }
  const double sp = sqrt(W[1] * W[1] + W[2] * W[2] + W[3] * W[3]) + c;
  return (sp - sp == 0.0) ? sp : -1.0;     // finite test that survives fast-math-free builds
}

// ------------------------------------------------------------------------------------------------------------
// CGL MHD (NEXT-2; R24).  Nine variables per cell:
//   U = (rho, m, E, B, A_log),  E = rho v^2/2 + B^2/2 + p_par/2 + p_perp,  A_log as eq.18
//   W = (rho, v, p_par, B, p_perp): p_par in slot 4, p_perp in slot 8 (slot 8 is not rotated)
// Reciprocals and roots as in the ideal path (MUFU seed + Newton, a few ulp); exp / log from the CUDA math library.
// ------------------------------------------------------------------------------------------------------------
AG_HD void cgl_cons_to_prim(const double U[9], double W[9], int form = 0) {   // eqs.26-27 (form 0), eqs.24-25 (form 1)
  const double ir = rcp(U[0]);
  const double vx = U[1] * ir, vy = U[2] * ir, vz = U[3] * ir;
  const double b2 = U[5] * U[5] + U[6] * U[6] + U[7] * U[7];
  const double eint = U[4] - 0.5 * U[0] * (vx * vx + vy * vy + vz * vz) - 0.5 * b2;
  const double B3 = b2 * sqrt_pos(dmax(b2, kTiny));
  // X : Y = p_par : p_perp;  form 0: rho^2 exp(-A_log / rho) : B^3,  form 1: rho^3 : A B^3   (no exp, no log)
  const double X = (form == 1) ? U[0] * U[0] * U[0] : U[0] * U[0] * exp(-U[8] * ir);
  const double Y = (form == 1) ? U[8] * B3 : B3;
  const double iden = rcp(X + 2.0 * Y);
  W[0] = U[0]; W[1] = vx; W[2] = vy; W[3] = vz;
  W[4] = 2.0 * X * eint * iden;
  W[5] = U[5]; W[6] = U[6]; W[7] = U[7];
  W[8] = 2.0 * Y * eint * iden;
}
// the thermodynamic variable of a primitive state: eq.18 (form 0) or eq.16 (form 1)
AG_HD double cgl_alog(double rho, double b2, double ppar, double pperp, int form = 0) {
  const double ratio = (rho * rho * pperp) * rcp(b2 * sqrt_pos(dmax(b2, kTiny)) * ppar);     // (rho^2 / B^3) (p_perp / p_par)
  return (form == 1) ? rho * ratio : rho * log(ratio);
}
// eq.29, fast branch, along the face normal of a ROTATED state (w[5] = B_n)
AG_HD double cgl_cfast(const double w[9]) {
  const double B2 = w[5] * w[5] + w[6] * w[6] + w[7] * w[7];
  const double cos2 = w[5] * w[5] * rcp(B2);
  const double b1 = B2 + 2.0 * w[8] + cos2 * (2.0 * w[4] - w[8]);
  const double b2 = b1 - 6.0 * cos2 * w[4];
  const double c = 4.0 * w[8] * w[8] * cos2 * (1.0 - cos2);
  return sqrt_pos((b1 + sqrt_pos(dmax(b2 * b2 + c, kTiny))) * (0.5 * rcp(w[0])));
}
// One side of the CGL face problem in the rotated frame: eqs.19-22 (psi == 0) + eq.17, the conserved vector, and the
// fast speed eq.29 -- |B|^2 and its reciprocal are formed once for Theta, cos^2 and the thermodynamic variable.
AG_HD void cgl_side(const double w[9], double f[9], double u[9], double& cfast, int form) {
  const double bn2 = w[5] * w[5];
  const double B2 = fma(w[7], w[7], fma(w[6], w[6], bn2));
  const double iB2 = rcp(B2);
  const double th = fma(-(w[4] - w[8]), iB2, 1.0);                       // Theta = 1 - (p_par - p_perp)/B^2
  const double v2 = fma(w[3], w[3], fma(w[2], w[2], w[1] * w[1]));
  const double vB = fma(w[3], w[7], fma(w[2], w[6], w[1] * w[5]));
  const double ru = w[0] * w[1];
  const double ke = (0.5 * w[0]) * v2;
  u[0] = w[0]; u[1] = ru; u[2] = w[0] * w[2]; u[3] = w[0] * w[3];
  u[4] = fma(0.5, B2 + w[4], ke) + w[8];
  u[5] = w[5]; u[6] = w[6]; u[7] = w[7];
  // (rho^2 / B^3) (p_perp / p_par):  1/B^3 = (1/B^2) rsqrt(B^2)
  const double ratio = (w[0] * w[0] * w[8]) * (iB2 * rsq(dmax(B2, kTiny))) * rcp(w[4]);
  u[8] = (form == 1) ? w[0] * ratio : w[0] * log(ratio);                   // eq.16 / eq.18
  const double tb = th * w[5];
  f[0] = ru;
  f[1] = fma(ru, w[1], fma(-tb, w[5], fma(0.5, B2, w[8])));
  f[2] = fma(ru, w[2], -(tb * w[6]));
  f[3] = fma(ru, w[3], -(tb * w[7]));
  f[4] = fma(-tb, vB, (fma(0.5, w[4], ke) + fma(2.0, w[8], B2)) * w[1]);
  f[5] = 0.0;
  f[6] = fma(w[1], w[6], -(w[5] * w[2]));
  f[7] = fma(w[1], w[7], -(w[5] * w[3]));
  f[8] = u[8] * w[1];
  const double cos2 = bn2 * iB2;
  const double b1 = fma(cos2, fma(2.0, w[4], -w[8]), fma(2.0, w[8], B2));
  const double b2 = fma(-6.0 * cos2, w[4], b1);
  const double c = (4.0 * w[8] * w[8]) * (cos2 * (1.0 - cos2));
  cfast = sqrt_pos((b1 + sqrt_pos(dmax(fma(b2, b2, c), kTiny))) * (0.5 * rcp(w[0])));
}
// HLL eq.5 with the Davis speeds eq.6 and eq.29's fast speed; all nine components through eq.5 (R9), written as
// a F_L + b F_R + c (U_R - U_L)  with a = s_R/(s_R-s_L), b = -s_L/(s_R-s_L), c = s_L s_R/(s_R-s_L)
AG_HD void flux_hll_cgl(const double L[9], const double R[9], double F[9], int form = 0) {
  double fl[9], fr[9], ul[9], ur[9], cl, cr;
  cgl_side(L, fl, ul, cl, form);
  cgl_side(R, fr, ur, cr, form);
  const double sL = dmin(dmin(L[1] - cl, R[1] - cr), 0.0);
  const double sR = dmax(dmax(L[1] + cl, R[1] + cr), 0.0);
  const double iw = rcp(sR - sL);
  const double a = sR * iw, b = -(sL * iw), c = sL * a;
#pragma unroll
  for (int q = 0; q < 9; ++q) F[q] = fma(a, fl[q], fma(b, fr[q], c * (ur[q] - ul[q])));
}
// eqs.31-33 on a conserved cell: relax the anisotropy, keep E, return the new A_log (C1 = 0.3, C2 = 0.5)
AG_HD double cgl_relaxed_alog(double f, const double U[9], int form = 0) {
  double w[9];
  cgl_cons_to_prim(U, w, form);
  const double B2 = w[5] * w[5] + w[6] * w[6] + w[7] * w[7];
  const double dP = w[8] - w[4];
  const double mirror = (w[4] * rcp(w[8])) * (0.5 * B2);
  const double ic = 0.3 * sqrt_pos(dmax(0.5 * B2 * w[4], kTiny));      // C1 p_par (B^2 / 2 p_par)^(1/2) = C1 (p_par B^2 / 2)^(1/2)
  const double dPs = dmax(-B2, dmin(dP, dmin(mirror, ic)));
  const double ppar = w[4] - (2.0 / 3.0) * (dPs - dP) * f;
  const double pperp = w[8] + (1.0 / 3.0) * (dPs - dP) * f;
  return cgl_alog(w[0], B2, ppar, pperp, form);
}
// eq.28 per cell: |v| + max_d c_cgl,d; negative for an unphysical cell
AG_HD double cell_speed_cgl(const double U[9], int form = 0) {
  double w[9], r[9];
  cgl_cons_to_prim(U, w, form);
  if (!(w[0] > 0.0) || !(w[4] > 0.0) || !(w[8] > 0.0)) return -1.0;
  double cm = 0.0;
  for (int d = 0; d < 3; ++d) {
    for (int q = 0; q < 9; ++q) r[q] = w[q];
    r[5] = w[5 + d]; r[5 + d] = w[5];                      // only B_n matters for the speed
    cm = fmax(cm, cgl_cfast(r));
  }
  const double sp = sqrt(w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) + cm;
  return (sp - sp == 0.0) ? sp : -1.0;
}

// A7 inside the stage epilogue (ideal and Hall MHD): the same quantity as cell_speed<HALL> with the straight-line roots of
// this file, evaluated on the conserved values the stage is about to store.
template <bool HALL = false>
AG_HD double cell_speed_inline(const Phys& ph, const double U[8]) {
  const double ir = rcp(U[0]);
  const double v2 = (U[1] * U[1] + U[2] * U[2] + U[3] * U[3]) * (ir * ir);
  const double bx2 = U[5] * U[5], by2 = U[6] * U[6], bz2 = U[7] * U[7];
  const double B2 = bx2 + by2 + bz2;
  const double p = ph.gm1 * (U[4] - 0.5 * U[0] * v2 - 0.5 * B2);
  if (!(U[0] > 0.0) || !(p > 0.0)) return -1.0;
  const double a2 = ph.gamma * p * ir, sm = a2 + B2 * ir;
  const double rad = dmax(sm * sm - 4.0 * a2 * (dmin(dmin(bx2, by2), bz2) * ir), kTiny);
  double c = sqrt_pos(0.5 * (sm + sqrt_pos(rad)));
  if (HALL) {
    // eq.13: c_w = aw + sqrt(aw^2 + v_A^2),  aw = d_i pi |B| / (2 rho dx_min)
    const double aw = ph.cwk * sqrt_pos(dmax(B2, kTiny)) * ir;
    c = dmax(c, aw + sqrt_pos(dmax(aw * aw + B2 * ir, kTiny)));
  }
  const double sp = sqrt_pos(dmax(v2, kTiny)) + c;
  return (sp - sp == 0.0) ? sp : -1.0;
}

}  // namespace agate
