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
  double d_i;     // Hall: normalised ion inertial length
  double cwk;     // Hall: d_i * pi / (2 dx_min)   (eq.13 with k_max = pi / dx_min, R15)
};

AG_HD Phys make_phys(double gamma, double d_i, double dxmin) {
  Phys ph;
  ph.gamma = gamma;
  ph.gm1 = gamma - 1.0;
  ph.igm1 = 1.0 / (gamma - 1.0);
  ph.gogm1 = gamma / (gamma - 1.0);
  ph.d_i = d_i;
  ph.cwk = d_i * 3.14159265358979323846264338327950288 / (2.0 * dxmin);
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
  const double e = fma(-x, y, 1.0);               // 1 - x y          (~2^-22)
  const double y1 = fma(y, e, y);                 // 1 - x y1 = e^2 exactly, so the second step needs no new residual
  return fma(y1, e * e, y1);
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
template <bool HALL>
AG_HD void flux_hll(const Phys& ph, const double L[8], const double R[8], const double* J, double F[8]) {
  const Side sl = side_of(ph, L), sr = side_of(ph, R);
  double cl = sl.cf, cr = sr.cf;
  double vhl[3], vhr[3];
  if (HALL) {
    cl = dmax(cl, whistler_speed(ph, L, sl));
    cr = dmax(cr, whistler_speed(ph, R, sr));
    for (int c = 0; c < 3; ++c) {
      vhl[c] = -(ph.d_i * J[c]) * sl.ir;
      vhr[c] = -(ph.d_i * J[c]) * sr.ir;
    }
  }
  const double sL = dmin(dmin(L[1] - cl, R[1] - cr), 0.0);       // s'_L = min(s_L, 0)
  const double sR = dmax(dmax(L[1] + cl, R[1] + cr), 0.0);       // s'_R = max(s_R, 0)
  double fl[8], fr[8];
  phys_flux(ph, L, sl, HALL ? vhl : nullptr, fl);
  phys_flux(ph, R, sr, HALL ? vhr : nullptr, fr);
  const double ul[8] = {L[0], L[0] * L[1], L[0] * L[2], L[0] * L[3], energy_of(ph, L, sl), L[5], L[6], L[7]};
  const double ur[8] = {R[0], R[0] * R[1], R[0] * R[2], R[0] * R[3], energy_of(ph, R, sr), R[5], R[6], R[7]};
  const double iw = rcp(sR - sL);
  const double ss = sL * sR;
#pragma unroll
  for (int q = 0; q < 8; ++q) F[q] = (sR * fl[q] - sL * fr[q] + ss * (ur[q] - ul[q])) * iw;
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

// HLLD (R10).  The Riemann fan is mirrored (x -> -x: swap sides, negate u and Bn) when the contact moves left,
// so that a single "upwind side = A" code path serves both halves of the fan and lanes of a warp only diverge
// on single-star vs double-star.  Mirror symmetry of the solver is oracle pin P6(v).
AG_HD void flux_hlld(const Phys& ph, const double L[8], const double R[8], double F[8]) {
  const double bn0 = 0.5 * (L[5] + R[5]);                    // single-valued Bn: arithmetic mean
  const double bn2 = bn0 * bn0;
  // per-side speeds with Bn := bn0 (the caller's L[5], R[5] are not used below)
  Side sl, sr;
  {
    sl.ir = rcp(L[0]); sr.ir = rcp(R[0]);
    sl.B2 = bn2 + L[6] * L[6] + L[7] * L[7];
    sr.B2 = bn2 + R[6] * R[6] + R[7] * R[7];
    sl.pt = L[4] + 0.5 * sl.B2; sr.pt = R[4] + 0.5 * sr.B2;
    const double a2l = ph.gamma * L[4] * sl.ir, sml = a2l + sl.B2 * sl.ir;
    const double a2r = ph.gamma * R[4] * sr.ir, smr = a2r + sr.B2 * sr.ir;
    const double radl = dmax(sml * sml - 4.0 * a2l * (bn2 * sl.ir), kTiny);
    const double radr = dmax(smr * smr - 4.0 * a2r * (bn2 * sr.ir), kTiny);
    sl.cf = sqrt_pos(0.5 * (sml + sqrt_pos(radl)));
    sr.cf = sqrt_pos(0.5 * (smr + sqrt_pos(radr)));
  }
  const double SL = dmin(L[1] - sl.cf, R[1] - sr.cf);        // eq.6
  const double SR = dmax(L[1] + sl.cf, R[1] + sr.cf);
  const double mL = L[0] * (SL - L[1]), mR = R[0] * (SR - R[1]);     // mL < 0 < mR
  const double idm = rcp(mR - mL);
  const double SM0 = (mR * R[1] - mL * L[1] - sr.pt + sl.pt) * idm;
  const double pts = (mR * sl.pt - mL * sr.pt + mL * mR * (R[1] - L[1])) * idm;
  const bool supL = SL >= 0.0;
  const bool supR = !supL && (SR <= 0.0);
  const bool flip = supL ? false : (supR ? true : (SM0 < 0.0));
  const unsigned long long sg = flip ? 0x8000000000000000ull : 0ull;

  // mirrored frame: A = upwind side
  double A[8];
  A[0] = flip ? R[0] : L[0];
  A[1] = xorsign(flip ? R[1] : L[1], sg);
  A[2] = flip ? R[2] : L[2];
  A[3] = flip ? R[3] : L[3];
  A[4] = flip ? R[4] : L[4];
  A[6] = flip ? R[6] : L[6];
  A[7] = flip ? R[7] : L[7];
  const double bn = xorsign(bn0, sg);
  A[5] = bn;
  Side sa;
  sa.ir = 0.0; sa.cf = 0.0;
  sa.B2 = flip ? sr.B2 : sl.B2;
  sa.pt = flip ? sr.pt : sl.pt;
  const double SA = xorsign(flip ? SR : SL, sg);
  const double mA = xorsign(flip ? mR : mL, sg);
  const double SM = xorsign(SM0, sg);                        // >= 0 unless supersonic

  double fa[8];
  phys_flux(ph, A, sa, nullptr, fa);
  const double EA = energy_of(ph, A, sa);

  const Star a = star_of(A, SA, mA, SM, bn, bn2, pts);
  const double vBA = A[1] * bn + A[2] * A[6] + A[3] * A[7];
  const double vBsA = SM * bn + a.v * a.b1 + a.w * a.b2;
  const double EsA = ((SA - A[1]) * EA - sa.pt * A[1] + pts * SM + bn * (vBA - vBsA)) * a.idS;

  double Fm[8];
  Fm[0] = fa[0] + SA * (a.rs - A[0]);
  Fm[1] = fa[1] + SA * (a.rs * SM - A[0] * A[1]);
  Fm[2] = fa[2] + SA * (a.rs * a.v - A[0] * A[2]);
  Fm[3] = fa[3] + SA * (a.rs * a.w - A[0] * A[3]);
  Fm[4] = fa[4] + SA * (EsA - EA);
  Fm[6] = fa[6] + SA * (a.b1 - A[6]);
  Fm[7] = fa[7] + SA * (a.b2 - A[7]);

  // S*_A = SM - |Bn|/sqrt(rho*_A) < 0  <=>  SM^2 rho*_A < Bn^2   (SM >= 0): no square root for the decision
  const bool twostar = (SM * SM * a.rs < bn2) && !(0.5 * bn2 < kHlldEps * pts) && !(supL || supR);
  if (twostar) {
    double B[8];
    B[0] = flip ? L[0] : R[0];
    B[1] = xorsign(flip ? L[1] : R[1], sg);
    B[2] = flip ? L[2] : R[2];
    B[3] = flip ? L[3] : R[3];
    B[6] = flip ? L[6] : R[6];
    B[7] = flip ? L[7] : R[7];
    const double SB = xorsign(flip ? SL : SR, sg);
    const double mB = xorsign(flip ? mL : mR, sg);
    const Star b = star_of(B, SB, mB, SM, bn, bn2, pts);
    const double irsA = rsq(a.rs);
    const double SsA = SM - fabs(bn) * irsA;                 // S*_A
    const double qA = a.rs * irsA, qB = sqrt_pos(b.rs);
    const double I = rcp(qA + qB);
    const double sgn = (bn > 0.0) ? 1.0 : -1.0;
    const double vss = (qA * a.v + qB * b.v + (b.b1 - a.b1) * sgn) * I;
    const double wss = (qA * a.w + qB * b.w + (b.b2 - a.b2) * sgn) * I;
    const double b1ss = (qA * b.b1 + qB * a.b1 + qA * qB * (b.v - a.v) * sgn) * I;
    const double b2ss = (qA * b.b2 + qB * a.b2 + qA * qB * (b.w - a.w) * sgn) * I;
    const double vBss = SM * bn + vss * b1ss + wss * b2ss;
    Fm[2] += SsA * (a.rs * (vss - a.v));
    Fm[3] += SsA * (a.rs * (wss - a.w));
    Fm[4] -= SsA * (qA * (vBsA - vBss) * sgn);
    Fm[6] += SsA * (b1ss - a.b1);
    Fm[7] += SsA * (b2ss - a.b2);
  }
  if (supL || supR) {
#pragma unroll
    for (int q = 0; q < 8; ++q) Fm[q] = fa[q];
  }
  F[0] = xorsign(Fm[0], sg);
  F[1] = Fm[1];
  F[2] = xorsign(Fm[2], sg);
  F[3] = xorsign(Fm[3], sg);
  F[4] = xorsign(Fm[4], sg);
  F[5] = 0.0;                                                // F[Bn] = 0 in every branch (R10)
  F[6] = xorsign(Fm[6], sg);
  F[7] = xorsign(Fm[7], sg);
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

}  // namespace agate
