// agate_ref.cpp — CPU ORACLE of the AGATE finite-volume MHD step.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// Plain, slow, obviously-correct restatement of what the hot path computes, following PAPER.md
// (/root/reference/PAPER.md, cited as P:Lnnn) §2.2 and §3.1 step by step, in
// the paper's order and notation, with the readings R1-R21 of SURVEY.md §8(c) / DESIGN.md where the
// paper is silent, garbled or at odds with itself.  No blocking, fusion or reordering: whole-grid
// primitive array, then per direction per grid line: slopes (eq.4), face states (eq.2-3), Riemann
// flux (eq.5-6 / HLLD), flux difference (eq.1); then the Runge-Kutta combine.
//
// Independence: this file shares no code, header, table or helper with the CUDA path
// (paper_2503_20899_b200/csrc).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may load it.
//
// Precision: IEEE fp64; build with  g++ -O2 -ffp-contract=off  (never -ffast-math).
// Threads: single-threaded by default.  The same loops carry `omp parallel for` over independent
// grid lines; each cell's new value depends only on the stage input and L is accumulated per cell in
// the fixed order x, y, z (R21), so the threaded run is bitwise identical (tests/test_oracle_pins.py).
//
// Pins (tests/test_oracle_pins.py, -m "not gpu"): P1 uniform state bitwise fixed; P2 conservation to
// round-off; P3 hand-derived HLL flux on the paper's Brio-Wu states incl. the 4x4 grid; P4
// linear eigenmode amplification factor (closed form); P5 eq.4 beta=1 == minmod; P6 HLLD exactness
// properties (contact, rotational discontinuity, HLLC limit, symmetries); P7 dt closed form; P8
// second-order convergence; P9 whistler dispersion eq.34 + Table 1; P10 2D-in-3D
// embedding; P11 Orszag-Tang half-turn symmetry; P12 brute-force face-scatter evaluation.
// Parity-unpinned conventions (no passage fixes them): R4 (|v| norm and max over all
// three c_f,d in v_max), R6 (primitive-variable reconstruction), R10's B_n = arithmetic mean with
// F[B_n]=0 in HLLD, R11 (dt once per step), R15's rho-side / speed choices in the Hall flux
// (approximately pinned by Table 1).
#include "agate_ref.h"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

int g_threads = 1;

// ------------------------------------------------------------------------------------------------
// Counting scalar: same templates instantiated on this type give the algorithmic operation counts
// (convention of SURVEY.md §8(d): add/sub/mul/compare/min/max = 1, div = 1, sqrt = 1, abs/neg/select = 0).
// ------------------------------------------------------------------------------------------------
struct OpCount { double add = 0, mul = 0, div = 0, sqrt = 0, cmp = 0; };
OpCount g_ops;

struct Counted {
  double v;
  Counted() : v(0) {}
  Counted(double x) : v(x) {}
};
inline Counted operator+(Counted a, Counted b) { g_ops.add++; return Counted(a.v + b.v); }
inline Counted operator-(Counted a, Counted b) { g_ops.add++; return Counted(a.v - b.v); }
inline Counted operator*(Counted a, Counted b) { g_ops.mul++; return Counted(a.v * b.v); }
inline Counted operator/(Counted a, Counted b) { g_ops.div++; return Counted(a.v / b.v); }
inline Counted operator-(Counted a) { return Counted(-a.v); }
inline Counted& operator+=(Counted& a, Counted b) { a = a + b; return a; }
inline Counted& operator-=(Counted& a, Counted b) { a = a - b; return a; }
inline bool operator<(Counted a, Counted b) { g_ops.cmp++; return a.v < b.v; }
inline bool operator>(Counted a, Counted b) { g_ops.cmp++; return a.v > b.v; }
inline bool operator<=(Counted a, Counted b) { g_ops.cmp++; return a.v <= b.v; }
inline bool operator>=(Counted a, Counted b) { g_ops.cmp++; return a.v >= b.v; }

inline double val(double x) { return x; }
inline double val(Counted x) { return x.v; }
inline double tsqrt(double x) { return std::sqrt(x); }
inline Counted tsqrt(Counted x) { g_ops.sqrt++; return Counted(std::sqrt(x.v)); }
inline double texp(double x) { return std::exp(x); }
inline Counted texp(Counted x) { g_ops.sqrt++; return Counted(std::exp(x.v)); }     // transcendental: counted with sqrt
inline double tlog(double x) { return std::log(x); }
inline Counted tlog(Counted x) { g_ops.sqrt++; return Counted(std::log(x.v)); }
inline double tabs(double x) { return std::fabs(x); }
inline Counted tabs(Counted x) { return Counted(std::fabs(x.v)); }
template <class T> inline T tmin(T a, T b) { return (b < a) ? b : a; }
template <class T> inline T tmax(T a, T b) { return (b > a) ? b : a; }

constexpr double PI = 3.14159265358979323846264338327950288;
constexpr double HLLD_EPS = 1e-12;   // R10 guards

// ------------------------------------------------------------------------------------------------
// Point functions
// ------------------------------------------------------------------------------------------------

// A1, P:L140 with R2 (p/(gamma-1)):  v = m/rho ;  p = (gamma-1)(E - rho|v|^2/2 - |B|^2/2)
template <class T> void cons_to_prim(double gamma, const T U[8], T W[8]) {
  T rho = U[0];
  T vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
  T v2 = vx * vx + vy * vy + vz * vz;
  T b2 = U[5] * U[5] + U[6] * U[6] + U[7] * U[7];
  W[0] = rho; W[1] = vx; W[2] = vy; W[3] = vz;
  W[4] = T(gamma - 1.0) * (U[4] - T(0.5) * rho * v2 - T(0.5) * b2);
  W[5] = U[5]; W[6] = U[6]; W[7] = U[7];
}

// cons(W): E = rho|v|^2/2 + |B|^2/2 + p/(gamma-1)   (R2)
template <class T> void prim_to_cons(double gamma, const T W[8], T U[8]) {
  T rho = W[0];
  T v2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  T b2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
  U[0] = rho; U[1] = rho * W[1]; U[2] = rho * W[2]; U[3] = rho * W[3];
  U[4] = T(0.5) * rho * v2 + T(0.5) * b2 + W[4] / T(gamma - 1.0);
  U[5] = W[5]; U[6] = W[6]; U[7] = W[7];
}

// eq.4 with R7.  dp = W(i+1)-W(i), dm = W(i)-W(i-1).
//   limiter 2: 0 if dp*dm <= 0 else sign(dp) * min(beta|dp|, beta|dm|, |dp+dm|/2)
//   limiter 1: (dp+dm)/2      limiter 0: 0
template <class T> T slope(int limiter, double beta, T dp, T dm) {
  if (limiter == 0) return T(0.0);
  if (limiter == 1) return T(0.5) * (dp + dm);
  if (dp * dm <= T(0.0)) return T(0.0);
  T a = T(beta) * tabs(dp);
  T b = T(beta) * tabs(dm);
  T c = T(0.5) * tabs(dp + dm);
  T m = tmin(tmin(a, b), c);
  return (dp > T(0.0)) ? m : -m;
}

// eq.12 with R3:  c_f,d^2 = ( (vA^2+vs^2) + sqrt( max( (vA^2+vs^2)^2 - 4 vs^2 B_d^2/rho , 0 ) ) ) / 2
template <class T> T cfast(int d, double gamma, const T W[8]) {
  T rho = W[0];
  T a2 = T(gamma) * W[4] / rho;                                   // vs^2 = gamma p / rho
  T b2 = (W[5] * W[5] + W[6] * W[6] + W[7] * W[7]) / rho;         // vA^2 = B^2 / rho
  T s = a2 + b2;
  T rad = s * s - T(4.0) * a2 * W[5 + d] * W[5 + d] / rho;
  rad = tmax(rad, T(0.0));
  return tsqrt(T(0.5) * (s + tsqrt(rad)));
}

// eq.13:  c_w = aw + sqrt(aw^2 + vA^2),  aw = d_i pi |B| / (2 rho dx),  dx := dx_min (R15)
template <class T> T cwhistler(double d_i, double dxmin, const T W[8]) {
  T rho = W[0];
  T B2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
  T aw = T(d_i * PI) * tsqrt(B2) / (T(2.0) * rho * T(dxmin));
  return aw + tsqrt(aw * aw + B2 / rho);
}

// eqs.7-10 with psi == 0 (R12); vT = v + vH (vH may be null: ideal MHD).  n = dir.
template <class T> void phys_flux(int n, double gamma, const T W[8], const T* vH, T F[8]) {
  T rho = W[0], p = W[4];
  const T* v = W + 1;
  const T* B = W + 5;
  T vT[3] = {v[0], v[1], v[2]};
  if (vH) { vT[0] = v[0] + vH[0]; vT[1] = v[1] + vH[1]; vT[2] = v[2] + vH[2]; }
  T v2 = v[0] * v[0] + v[1] * v[1] + v[2] * v[2];
  T B2 = B[0] * B[0] + B[1] * B[1] + B[2] * B[2];
  T pt = p + T(0.5) * B2;
  T vTB = vT[0] * B[0] + vT[1] * B[1] + vT[2] * B[2];
  F[0] = rho * v[n];                                                        // eq.7
  for (int c = 0; c < 3; ++c) {
    F[1 + c] = rho * v[n] * v[c] - B[n] * B[c];                             // eq.8
    if (c == n) F[1 + c] = F[1 + c] + pt;
  }
  F[4] = (T(0.5) * rho * v2 + T(gamma / (gamma - 1.0)) * p) * v[n] + B2 * vT[n] - vTB * B[n];   // eq.9
  for (int c = 0; c < 3; ++c) F[5 + c] = vT[n] * B[c] - B[n] * vT[c];       // eq.10 (== 0 for c == n)
  F[5 + n] = T(0.0);
}

// eq.5-6; R8 (normal bulk velocity in eq.6), R9 (all 8 components through eq.5),
// Hall (R15): c = max(c_f,d , c_w) per side, vH^a = -d_i J / rho^a in phi.
template <class T>
void flux_hll(int eqset, int n, double gamma, double d_i, double dxmin,
              const T WL[8], const T WR[8], const T* J, T F[8]) {
  T cL = cfast(n, gamma, WL), cR = cfast(n, gamma, WR);
  T vHL[3], vHR[3];
  const bool hall = (eqset == AGATE_REF_HALL || eqset == AGATE_REF_HALL_GLM);
  if (hall) {
    cL = tmax(cL, cwhistler(d_i, dxmin, WL));
    cR = tmax(cR, cwhistler(d_i, dxmin, WR));
    for (int c = 0; c < 3; ++c) { vHL[c] = -(T(d_i) * J[c]) / WL[0]; vHR[c] = -(T(d_i) * J[c]) / WR[0]; }
  }
  T sL = tmin(WL[1 + n] - cL, WR[1 + n] - cR);          // eq.6
  T sR = tmax(WL[1 + n] + cL, WR[1 + n] + cR);
  T sLp = tmin(sL, T(0.0)), sRp = tmax(sR, T(0.0));
  T fL[8], fR[8], UL[8], UR[8];
  phys_flux(n, gamma, WL, hall ? vHL : nullptr, fL);
  phys_flux(n, gamma, WR, hall ? vHR : nullptr, fR);
  prim_to_cons(gamma, WL, UL);
  prim_to_cons(gamma, WR, UR);
  for (int q = 0; q < 8; ++q)
    F[q] = (sRp * fL[q] - sLp * fR[q] + sLp * sRp * (UR[q] - UL[q])) / (sRp - sLp);      // eq.5
}

// HLLD (R10): five-wave solver (Miyoshi & Kusano 2005 as restated in SURVEY.md §8(c)), outer speeds from
// the paper's eq.6, single B_n = arithmetic mean, F[B_n] = 0.  u = normal velocity, (v,w)/(By,Bz) the
// transverse components in cyclic order.  Returns the branch id (see agate_ref_hlld_branch).
template <class T>
int flux_hlld(int n, double gamma, const T WLin[8], const T WRin[8], T F[8]) {
  const int t1 = (n + 1) % 3, t2 = (n + 2) % 3;
  T WL[8], WR[8];
  for (int q = 0; q < 8; ++q) { WL[q] = WLin[q]; WR[q] = WRin[q]; }
  T Bn = T(0.5) * (WL[5 + n] + WR[5 + n]);
  WL[5 + n] = Bn; WR[5 + n] = Bn;
  T cL = cfast(n, gamma, WL), cR = cfast(n, gamma, WR);
  T uL = WL[1 + n], uR = WR[1 + n];
  T SL = tmin(uL - cL, uR - cR), SR = tmax(uL + cL, uR + cR);
  T fL[8], fR[8], UL[8], UR[8];
  phys_flux<T>(n, gamma, WL, nullptr, fL);
  phys_flux<T>(n, gamma, WR, nullptr, fR);
  if (SL >= T(0.0)) { for (int q = 0; q < 8; ++q) F[q] = fL[q]; return 0; }
  if (SR <= T(0.0)) { for (int q = 0; q < 8; ++q) F[q] = fR[q]; return 5; }
  prim_to_cons(gamma, WL, UL);
  prim_to_cons(gamma, WR, UR);
  T ptL = WL[4] + T(0.5) * (WL[5] * WL[5] + WL[6] * WL[6] + WL[7] * WL[7]);
  T ptR = WR[4] + T(0.5) * (WR[5] * WR[5] + WR[6] * WR[6] + WR[7] * WR[7]);
  T mL = WL[0] * (SL - uL), mR = WR[0] * (SR - uR);
  T SM = (mR * uR - mL * uL - ptR + ptL) / (mR - mL);
  T pts = (mR * ptL - mL * ptR + mL * mR * (uR - uL)) / (mR - mL);
  int degenerate = 0;

  T Us[2][8];       // U*_L, U*_R
  T vs[2], ws[2], Bys[2], Bzs[2], vBs[2], rhos[2];
  for (int a = 0; a < 2; ++a) {
    const T* Wa = a ? WR : WL;
    const T* Ua = a ? UR : UL;
    T S = a ? SR : SL, m = a ? mR : mL, pt = a ? ptR : ptL;
    T u = Wa[1 + n], v = Wa[1 + t1], w = Wa[1 + t2], By = Wa[5 + t1], Bz = Wa[5 + t2];
    T rs = m / (S - SM);
    T den = m * (S - SM) - Bn * Bn;
    T vst, wst, Byst, Bzst;
    if (tabs(den) < T(HLLD_EPS) * pts) {
      vst = v; wst = w; Byst = By; Bzst = Bz; degenerate = 10;
    } else {
      vst = v - Bn * By * (SM - u) / den;
      wst = w - Bn * Bz * (SM - u) / den;
      T f = (m * (S - u) - Bn * Bn) / den;
      Byst = By * f; Bzst = Bz * f;
    }
    T vB = u * Bn + v * By + w * Bz;
    T vBst = SM * Bn + vst * Byst + wst * Bzst;
    T Es = ((S - u) * Ua[4] - pt * u + pts * SM + Bn * (vB - vBst)) / (S - SM);
    Us[a][0] = rs;
    Us[a][1 + n] = rs * SM; Us[a][1 + t1] = rs * vst; Us[a][1 + t2] = rs * wst;
    Us[a][4] = Es;
    Us[a][5 + n] = Bn; Us[a][5 + t1] = Byst; Us[a][5 + t2] = Bzst;
    vs[a] = vst; ws[a] = wst; Bys[a] = Byst; Bzs[a] = Bzst; vBs[a] = vBst; rhos[a] = rs;
  }
  T SsL = SM - tabs(Bn) / tsqrt(rhos[0]);
  T SsR = SM + tabs(Bn) / tsqrt(rhos[1]);
  if (SsL >= T(0.0)) { for (int q = 0; q < 8; ++q) F[q] = fL[q] + SL * (Us[0][q] - UL[q]); F[5 + n] = T(0.0); return 1 + degenerate; }
  if (SsR <= T(0.0)) { for (int q = 0; q < 8; ++q) F[q] = fR[q] + SR * (Us[1][q] - UR[q]); F[5 + n] = T(0.0); return 4 + degenerate; }
  if (T(0.5) * Bn * Bn < T(HLLD_EPS) * pts) {      // no rotational waves
    if (SM >= T(0.0)) { for (int q = 0; q < 8; ++q) F[q] = fL[q] + SL * (Us[0][q] - UL[q]); F[5 + n] = T(0.0); return 1 + 10; }
    for (int q = 0; q < 8; ++q) F[q] = fR[q] + SR * (Us[1][q] - UR[q]);
    F[5 + n] = T(0.0);
    return 4 + 10;
  }
  T sg = (Bn > T(0.0)) ? T(1.0) : T(-1.0);
  T qL = tsqrt(rhos[0]), qR = tsqrt(rhos[1]);
  T I = T(1.0) / (qL + qR);
  T vss = (qL * vs[0] + qR * vs[1] + (Bys[1] - Bys[0]) * sg) * I;
  T wss = (qL * ws[0] + qR * ws[1] + (Bzs[1] - Bzs[0]) * sg) * I;
  T Byss = (qL * Bys[1] + qR * Bys[0] + qL * qR * (vs[1] - vs[0]) * sg) * I;
  T Bzss = (qL * Bzs[1] + qR * Bzs[0] + qL * qR * (ws[1] - ws[0]) * sg) * I;
  T vBss = SM * Bn + vss * Byss + wss * Bzss;
  if (SM >= T(0.0)) {
    T Uss[8];
    Uss[0] = rhos[0]; Uss[1 + n] = rhos[0] * SM; Uss[1 + t1] = rhos[0] * vss; Uss[1 + t2] = rhos[0] * wss;
    Uss[4] = Us[0][4] - qL * (vBs[0] - vBss) * sg;
    Uss[5 + n] = Bn; Uss[5 + t1] = Byss; Uss[5 + t2] = Bzss;
    for (int q = 0; q < 8; ++q) F[q] = fL[q] + SsL * Uss[q] - (SsL - SL) * Us[0][q] - SL * UL[q];
    F[5 + n] = T(0.0);
    return 2 + degenerate;
  }
  T Uss[8];
  Uss[0] = rhos[1]; Uss[1 + n] = rhos[1] * SM; Uss[1 + t1] = rhos[1] * vss; Uss[1 + t2] = rhos[1] * wss;
  Uss[4] = Us[1][4] + qR * (vBs[1] - vBss) * sg;
  Uss[5 + n] = Bn; Uss[5 + t1] = Byss; Uss[5 + t2] = Bzss;
  for (int q = 0; q < 8; ++q) F[q] = fR[q] + SsR * Uss[q] - (SsR - SR) * Us[1][q] - SR * UR[q];
  F[5 + n] = T(0.0);
  return 3 + degenerate;
}

// ------------------------------------------------------------------------------------------------
// CGL MHD (NEXT-2; R24).  Nine variables per cell:
//   U = (rho, m, E, B, A_log)   with  E = rho v^2/2 + B^2/2 + p_par/2 + p_perp  and
//                                     A_log = rho log[(rho^2/B^3)(p_perp/p_par)]      (eq.18)
//   W = (rho, v, p_par, B, p_perp)    (p_par in slot 4, p_perp in slot 8)
// ------------------------------------------------------------------------------------------------
// eqs.26-27 (log form, form = 0):  X = rho^2 exp(-A/rho);  p_par = 2 X e/(X + 2B^3),  p_perp = 2 B^3 e/(X + 2B^3)
// eqs.24-25 (non-log form, form = 1; "AGATE supports both"):  p_par = 2 rho^3 e/(rho^3 + 2 A B^3),
//                                                                    p_perp = 2 A B^3 e/(rho^3 + 2 A B^3)
template <class T> void cgl_cons_to_prim(const T U[9], T W[9], int form = 0) {
  T rho = U[0];
  T vx = U[1] / rho, vy = U[2] / rho, vz = U[3] / rho;
  T v2 = vx * vx + vy * vy + vz * vz;
  T b2 = U[5] * U[5] + U[6] * U[6] + U[7] * U[7];
  T eint = U[4] - T(0.5) * rho * v2 - T(0.5) * b2;
  T B3 = b2 * tsqrt(b2);
  W[0] = rho; W[1] = vx; W[2] = vy; W[3] = vz;
  W[5] = U[5]; W[6] = U[6]; W[7] = U[7];
  if (form == 1) {
    T r3 = rho * rho * rho;
    T AB = U[8] * B3;
    T den = r3 + T(2.0) * AB;
    W[4] = T(2.0) * r3 * eint / den;                  // eq.24
    W[8] = T(2.0) * AB * eint / den;                  // eq.25
    return;
  }
  T X = rho * rho * texp(-U[8] / rho);
  T den = X + T(2.0) * B3;
  W[4] = T(2.0) * X * eint / den;
  W[8] = T(2.0) * B3 * eint / den;
}
// E of P:L166 and the thermodynamic variable: eq.18 (form 0) or eq.16 (form 1)
template <class T> void cgl_prim_to_cons(const T W[9], T U[9], int form = 0) {
  T rho = W[0];
  T v2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  T b2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
  U[0] = rho; U[1] = rho * W[1]; U[2] = rho * W[2]; U[3] = rho * W[3];
  U[4] = T(0.5) * rho * v2 + T(0.5) * b2 + T(0.5) * W[4] + W[8];
  U[5] = W[5]; U[6] = W[6]; U[7] = W[7];
  if (form == 1) U[8] = (rho * rho * rho / (b2 * tsqrt(b2))) * (W[8] / W[4]);       // eq.16
  else U[8] = rho * tlog((rho * rho / (b2 * tsqrt(b2))) * (W[8] / W[4]));             // eq.18
}
// eq.29, fast (+) branch, along direction d:  c^2 = (b1 + sqrt(b2^2 + c)) / (2 rho)
template <class T> T cgl_cfast(int d, const T W[9]) {
  T B2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
  T cos2 = W[5 + d] * W[5 + d] / B2;
  T b1 = B2 + T(2.0) * W[8] + cos2 * (T(2.0) * W[4] - W[8]);
  T b2 = b1 - T(6.0) * cos2 * W[4];
  T c = T(4.0) * W[8] * W[8] * cos2 * (T(1.0) - cos2);
  return tsqrt((b1 + tsqrt(b2 * b2 + c)) / (T(2.0) * W[0]));
}
// eqs.19-22 with psi == 0 and eq.17 for A, along direction n;  Theta = 1 - (p_par - p_perp)/B^2
template <class T> void cgl_phys_flux(int n, const T W[9], const T U[9], T F[9]) {
  T B2 = W[5] * W[5] + W[6] * W[6] + W[7] * W[7];
  T th = T(1.0) - (W[4] - W[8]) / B2;
  T vn = W[1 + n], bn = W[5 + n];
  T v2 = W[1] * W[1] + W[2] * W[2] + W[3] * W[3];
  T vB = W[1] * W[5] + W[2] * W[6] + W[3] * W[7];
  F[0] = W[0] * vn;
  for (int c = 0; c < 3; ++c) F[1 + c] = W[0] * W[1 + c] * vn - th * W[5 + c] * bn;
  F[1 + n] += W[8] + T(0.5) * B2;
  F[4] = (T(0.5) * W[0] * v2 + T(0.5) * W[4] + T(2.0) * W[8] + B2) * vn - th * vB * bn;
  for (int c = 0; c < 3; ++c) F[5 + c] = vn * W[5 + c] - bn * W[1 + c];
  F[5 + n] = T(0.0);
  F[8] = U[8] * vn;
}
// HLL eq.5 with the Davis speeds eq.6 and c = eq.29's fast speed; all nine components through eq.5
template <class T> void cgl_flux_hll(int n, const T WL[9], const T WR[9], T F[9], int form = 0) {
  T UL[9], UR[9], fL[9], fR[9];
  cgl_prim_to_cons(WL, UL, form); cgl_prim_to_cons(WR, UR, form);
  cgl_phys_flux(n, WL, UL, fL); cgl_phys_flux(n, WR, UR, fR);
  T cl = cgl_cfast(n, WL), cr = cgl_cfast(n, WR);
  T sL = tmin(tmin(WL[1 + n] - cl, WR[1 + n] - cr), T(0.0));
  T sR = tmax(tmax(WL[1 + n] + cl, WR[1 + n] + cr), T(0.0));
  for (int q = 0; q < 9; ++q) F[q] = (sR * fL[q] - sL * fR[q] + sL * sR * (UR[q] - UL[q])) / (sR - sL);
}
// eqs.31-33: relaxation of the anisotropy dP = p_perp - p_par towards the stable range, at constant
// (p_par + 2 p_perp)/3; f = dt/(dt + tau) (paper default 0.99), C1 = 0.3, C2 = 0.5
inline void cgl_relax(double f, double B2, double* ppar, double* pperp) {
  const double dP = *pperp - *ppar;
  const double mirror = (*ppar / *pperp) * B2 / 2.0;
  const double ic = 0.3 * *ppar * std::pow(B2 / (2.0 * *ppar), 0.5);
  const double dPs = std::fmax(-B2, std::fmin(dP, std::fmin(mirror, ic)));
  *ppar = *ppar - (2.0 / 3.0) * (dPs - dP) * f;
  *pperp = *pperp + (1.0 / 3.0) * (dPs - dP) * f;
}

// GLM (eqs.10-11; R22).  Along the face normal, (B_n, psi) obey  dB_n/dt + dpsi/dx = 0,
// dpsi/dt + c_h^2 dB_n/dx = 0: characteristic variables B_n -+ psi/c_h move at -+c_h, and the state
// on the face (x/t = 0) is
//   B_n* = (B_nL + B_nR)/2 - (psi_R - psi_L)/(2 c_h),   psi* = (psi_L + psi_R)/2 - c_h (B_nR - B_nL)/2.
template <class T>
void glm_face(double ch, T bnL, T bnR, T psL, T psR, T* bns, T* pss) {
  *bns = T(0.5) * (bnL + bnR) - T(0.5) * (psR - psL) / T(ch);
  *pss = T(0.5) * (psL + psR) - T(0.5) * T(ch) * (bnR - bnL);
}

template <class T>
void face_flux(int eqset, int riemann, int n, double gamma, double d_i, double dxmin,
               const T WL[8], const T WR[8], const T* J, T F[8]) {
  if (riemann == 1) flux_hlld<T>(n, gamma, WL, WR, F);
  else flux_hll<T>(eqset, n, gamma, d_i, dxmin, WL, WR, J, F);
}

// ------------------------------------------------------------------------------------------------
// The grid solver
// ------------------------------------------------------------------------------------------------
template <class T> struct Solver {
  agate_ref_grid g;
  agate_ref_solver s;
  double gamma;
  int eqset;
  int nd[3];            // interior zones per dimension
  int gh[3];            // ghost width per dimension: 2 if active else 0 (R13, R16)
  int np[3];            // padded sizes
  ptrdiff_t st[3];      // padded strides
  size_t ntot, nint;    // padded / interior cell counts
  double h[3];          // spacings
  double dxmin, cfl;
  int nv;               // variables per cell: 8, + CGL's A (index 8), + the GLM scalar psi (the last index, nv-1)
  bool glm;
  bool cgl = false;
  double ch = 0.0;      // GLM: c_h of the step being taken (R22: 0.95 v_max(U^n))
  std::vector<T> Un, U1, U2, U3, W, L;
  double t = 0.0;
  bool have_state = false;

  Solver(const agate_ref_grid& g_, double gamma_, int eqset_, const agate_ref_solver& s_)
      : g(g_), s(s_), gamma(gamma_), eqset(eqset_) {
    nd[0] = g.nx; nd[1] = g.ny; nd[2] = g.nz;
    h[0] = g.dx; h[1] = g.dy; h[2] = g.dz;
    for (int d = 0; d < 3; ++d) { gh[d] = (d < g.ndim) ? 2 : 0; np[d] = nd[d] + 2 * gh[d]; }
    st[0] = 1; st[1] = np[0]; st[2] = (ptrdiff_t)np[0] * np[1];
    ntot = (size_t)np[0] * np[1] * np[2];
    nint = (size_t)nd[0] * nd[1] * nd[2];
    dxmin = h[0];                                              // R5: min over ACTIVE dimensions
    for (int d = 1; d < g.ndim; ++d) dxmin = std::fmin(dxmin, h[d]);
    cfl = s.cfl;
    if (!(cfl > 0.0)) cfl = (g.ndim == 1) ? 0.8 : (g.ndim == 2 ? 0.45 : 0.325);
    glm = (eqset == AGATE_REF_IDEAL_GLM || eqset == AGATE_REF_HALL_GLM || eqset == AGATE_REF_CGL_GLM);
    cgl = (eqset == AGATE_REF_CGL || eqset == AGATE_REF_CGL_GLM);
    nv = 8 + (glm ? 1 : 0) + (cgl ? 1 : 0);          // psi is always the last variable; CGL's A is index 8
    Un.assign(nv * ntot, T(0.0)); U1.assign(nv * ntot, T(0.0)); W.assign(nv * ntot, T(0.0));
    L.assign(nv * nint, T(0.0));
  }
  inline ptrdiff_t pidx(int i, int j, int k) const {
    return (ptrdiff_t)(i + gh[0]) + st[1] * (j + gh[1]) + st[2] * (k + gh[2]);
  }
  inline size_t iidx(int i, int j, int k) const { return ((size_t)k * nd[1] + j) * nd[0] + i; }

  // A0 (R13): every ghost cell (faces, edges, corners) = interior cell at the index wrapped mod n.
  void fill_ghosts(std::vector<T>& U) const {
    for (int q = 0; q < nv; ++q)
#pragma omp parallel for num_threads(g_threads) if (g_threads > 1)
      for (int k = -gh[2]; k < nd[2] + gh[2]; ++k)
        for (int j = -gh[1]; j < nd[1] + gh[1]; ++j)
          for (int i = -gh[0]; i < nd[0] + gh[0]; ++i) {
            // periodic: wrapped index;  zero-gradient (R26): the nearest interior zone
            int iw = s.bc[0] ? std::min(std::max(i, 0), nd[0] - 1) : ((i % nd[0]) + nd[0]) % nd[0];
            int jw = s.bc[1] ? std::min(std::max(j, 0), nd[1] - 1) : ((j % nd[1]) + nd[1]) % nd[1];
            int kw = s.bc[2] ? std::min(std::max(k, 0), nd[2] - 1) : ((k % nd[2]) + nd[2]) % nd[2];
            if (s.bc[1] == 2 && (j < 0 || j >= nd[1])) {
              // sheared zero-gradient ends in y (R28): the ghost zone (i, j) takes the value of zone
              // (i-1, j+2) at the down side and (i+1, j-2) at the up side, x wrapped periodically.  With two
              // ghost layers the source row j+-2 is an interior row.
              const int sh = (j < 0) ? -1 : 1;
              jw = j - 2 * sh;
              iw = (((i + sh) % nd[0]) + nd[0]) % nd[0];
            }
            if (iw != i || jw != j || kw != k) U[q * ntot + pidx(i, j, k)] = U[q * ntot + pidx(iw, jw, kw)];
          }
  }

  // A1 on interior + ghosts.
  void primitives(const std::vector<T>& U) {
#pragma omp parallel for num_threads(g_threads) if (g_threads > 1)
    for (ptrdiff_t c = 0; c < (ptrdiff_t)ntot; ++c) {
      if (cgl) {
        T u9[9], w9[9];
        for (int q = 0; q < 9; ++q) u9[q] = U[q * ntot + c];
        cgl_cons_to_prim(u9, w9, s.cgl_form);
        for (int q = 0; q < 9; ++q) W[q * ntot + c] = w9[q];
        if (glm) W[9 * ntot + c] = U[9 * ntot + c];               // psi is its own primitive
        continue;
      }
      T u[8], w[8];
      for (int q = 0; q < 8; ++q) u[q] = U[q * ntot + c];
      cons_to_prim(gamma, u, w);
      for (int q = 0; q < 8; ++q) W[q * ntot + c] = w[q];
      if (glm) W[8 * ntot + c] = U[8 * ntot + c];                 // psi is its own primitive
    }
  }

  // R15: J = curl B at the face between cell c and c + e_d, from the cell-centred B of the stage input:
  // central difference across the face along d; along t != d the average of the two adjacent cells'
  // central differences; 0 along inactive dimensions.
  void face_current(int d, ptrdiff_t c, T J[3]) const {
    T dB[3][3];   // dB[a][b] = d_a B_b
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        const T* B = &W[(5 + b) * ntot];
        if (a >= g.ndim) { dB[a][b] = T(0.0); continue; }
        if (a == d) dB[a][b] = (B[c + st[d]] - B[c]) / T(h[d]);
        else dB[a][b] = T(0.5) * ((B[c + st[a]] - B[c - st[a]]) + (B[c + st[d] + st[a]] - B[c + st[d] - st[a]])) / T(2.0 * h[a]);
      }
    J[0] = dB[1][2] - dB[2][1];
    J[1] = dB[2][0] - dB[0][2];
    J[2] = dB[0][1] - dB[1][0];
  }

  // One direction of eq.1 for every grid line: slopes (A2), face states (eq.2-3), fluxes (A3/A4), difference (A5).
  void sweep(int d) {
    const int n = nd[d], d1 = (d + 1) % 3, d2 = (d + 2) % 3;
    const ptrdiff_t sd = st[d];
    const bool hall = (eqset == AGATE_REF_HALL || eqset == AGATE_REF_HALL_GLM);
#pragma omp parallel for collapse(2) num_threads(g_threads) if (g_threads > 1)
    for (int a2 = 0; a2 < nd[d2]; ++a2)
      for (int a1 = 0; a1 < nd[d1]; ++a1) {
        int ijk[3]; ijk[d] = 0; ijk[d1] = a1; ijk[d2] = a2;
        const ptrdiff_t base = pidx(ijk[0], ijk[1], ijk[2]);           // cell 0 of this line
        std::vector<T> dW(nv * (n + 2)), F(nv * (n + 1));
        for (int c = -1; c <= n; ++c)                                    // A2: slopes of cells -1..n
          for (int q = 0; q < nv; ++q) {
            const T* Wq = &W[q * ntot + base];
            T dp = Wq[(c + 1) * sd] - Wq[c * sd];
            T dm = Wq[c * sd] - Wq[(c - 1) * sd];
            dW[q * (n + 2) + (c + 1)] = slope<T>(s.limiter, s.beta, dp, dm);
          }
        for (int c = -1; c < n; ++c) {                                   // face c+1/2, between cells c and c+1
          T WL[10], WR[10], Ff[10], J[3];
          for (int q = 0; q < nv; ++q) {
            const T* Wq = &W[q * ntot + base];
            WL[q] = Wq[c * sd] + T(0.5) * dW[q * (n + 2) + (c + 1)];             // eq.2
            WR[q] = Wq[(c + 1) * sd] - T(0.5) * dW[q * (n + 2) + (c + 2)];       // eq.3
          }
          if (hall) face_current(d, base + c * sd, J);
          if (cgl && glm) {
            // eqs.22-23 (R30): the same (B_n, psi) subsystem as eqs.10-11; CGL's flux sees B_n* on both sides
            T bns, pss;
            glm_face<T>(ch, WL[5 + d], WR[5 + d], WL[9], WR[9], &bns, &pss);
            WL[5 + d] = bns; WR[5 + d] = bns;
            cgl_flux_hll<T>(d, WL, WR, Ff, s.cgl_form);
            Ff[5 + d] = pss;
            Ff[9] = T(ch) * T(ch) * bns;
          } else if (cgl) {
            cgl_flux_hll<T>(d, WL, WR, Ff, s.cgl_form);
          } else if (glm) {
            // eqs.10-11 (R22): (B_n, psi) decouple into a 2x2 linear system with speeds -+c_h; its Riemann
            // solution gives the single-valued face values, the MHD solver sees B_n* on both sides, and the two
            // GLM fluxes are  F[B_n] = psi*,  F[psi] = c_h^2 B_n*.
            T bns, pss;
            glm_face<T>(ch, WL[5 + d], WR[5 + d], WL[8], WR[8], &bns, &pss);
            WL[5 + d] = bns; WR[5 + d] = bns;
            // Hall + GLM: the Hall flux of the same face states with B_n* on both sides (R29)
            face_flux<T>(hall ? AGATE_REF_HALL : AGATE_REF_IDEAL, s.riemann, d, gamma, s.d_i, dxmin, WL, WR, hall ? J : nullptr, Ff);
            Ff[5 + d] = pss;
            Ff[8] = T(ch) * T(ch) * bns;
          } else {
            face_flux<T>(eqset, s.riemann, d, gamma, s.d_i, dxmin, WL, WR, hall ? J : nullptr, Ff);
          }
          for (int q = 0; q < nv; ++q) F[q * (n + 1) + (c + 1)] = Ff[q];
        }
        for (int c = 0; c < n; ++c) {                                    // A5
          ijk[d] = c;
          const size_t ii = iidx(ijk[0], ijk[1], ijk[2]);
          for (int q = 0; q < nv; ++q)
            L[q * nint + ii] -= (F[q * (n + 1) + (c + 1)] - F[q * (n + 1) + c]) / T(h[d]);
        }
      }
  }

  // L(U) of eq.1 (R1: dU/dt = -div F).  U must have its ghosts filled.
  void rhs(const std::vector<T>& U) {
    primitives(U);
    std::fill(L.begin(), L.end(), T(0.0));
    for (int d = 0; d < g.ndim; ++d) sweep(d);       // x, then y, then z (R21)
  }

  // A7 (R3, R4, R5).  Returns status; vmax through the pointer.
  int vmax(double* out) {
    T vm = T(0.0);
    bool bad = false;
    for (int k = 0; k < nd[2]; ++k)
      for (int j = 0; j < nd[1]; ++j)
        for (int i = 0; i < nd[0]; ++i) {
          T u[10], w[10];
          const ptrdiff_t c = pidx(i, j, k);
          for (int q = 0; q < nv; ++q) u[q] = Un[q * ntot + c];
          if (cgl) {
            // eq.28: |v| + max_d c_cgl,d
            cgl_cons_to_prim(u, w, s.cgl_form);
            if (!(val(w[0]) > 0.0) || !(val(w[4]) > 0.0) || !(val(w[8]) > 0.0)) { bad = true; continue; }
            T cm = tmax(tmax(cgl_cfast(0, w), cgl_cfast(1, w)), cgl_cfast(2, w));
            T spc = tsqrt(w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) + cm;
            if (!std::isfinite(val(spc))) { bad = true; continue; }
            vm = tmax(vm, spc);
            continue;
          }
          cons_to_prim(gamma, u, w);
          if (!(val(w[0]) > 0.0) || !(val(w[4]) > 0.0)) { bad = true; continue; }
          T cmax = tmax(tmax(cfast(0, gamma, w), cfast(1, gamma, w)), cfast(2, gamma, w));
          if (eqset == AGATE_REF_HALL || eqset == AGATE_REF_HALL_GLM) cmax = tmax(cmax, cwhistler(s.d_i, dxmin, w));
          T sp = tsqrt(w[1] * w[1] + w[2] * w[2] + w[3] * w[3]) + cmax;
          if (!std::isfinite(val(sp))) { bad = true; continue; }
          vm = tmax(vm, sp);
        }
    *out = val(vm);
    return bad ? 3 : 0;
  }
  int compute_dt(double* dt) {
    double vm;
    int rc = vmax(&vm);
    if (rc) return rc;
    *dt = val(T(cfl) * T(dxmin) / T(vm));
    return 0;
  }

  // R11: SSP-RK2 (Heun / Shu-Osher form), dt fixed for both stages; RK11 = forward Euler.
  // GLM (R22): c_h = 0.95 v_max(U^n) for the whole step, whoever chose dt; after the Runge-Kutta update
  // psi <- psi exp(-dt c_h^2 / c_p^2) with c_p^2 = 0.18 c_h, the exact solution of eq.11's source.
  void glm_source(double dt) {
    const T decay = T(std::exp(-dt * ch / 0.18));
    for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
      const size_t p = (size_t)(nv - 1) * ntot + pidx(i, j, k);
      Un[p] = Un[p] * decay;
    }
  }
  // CGL (R24): after the Runge-Kutta update every cell's anisotropy is relaxed (eqs.31-33) with
  // f = dt/(dt+tau) = s.relax (0 = off); the total energy is unchanged, only A_log moves.
  void cgl_source() {
    if (!(s.relax > 0.0)) return;
    for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
      const ptrdiff_t c = pidx(i, j, k);
      T u[9], w[9];
      for (int q = 0; q < 9; ++q) u[q] = Un[q * ntot + c];
      cgl_cons_to_prim(u, w, s.cgl_form);
      double ppar = val(w[4]), pperp = val(w[8]);
      const double B2 = val(w[5] * w[5] + w[6] * w[6] + w[7] * w[7]);
      cgl_relax(s.relax, B2, &ppar, &pperp);
      const double rho = val(w[0]);
      if (s.cgl_form == 1) Un[8 * ntot + c] = T((rho * rho * rho / (B2 * std::sqrt(B2))) * (pperp / ppar));   // eq.16
      else Un[8 * ntot + c] = T(rho * std::log((rho * rho / (B2 * std::sqrt(B2))) * (pperp / ppar)));
    }
  }
  // Uout = a0 Uref + a1 (Uin + c dt L)  on the interior, L = L(Uin) as left by rhs()
  void combine(std::vector<T>& Uout, double a0, const std::vector<T>& Uref, double a1, const std::vector<T>& Uin, double cdt) {
    for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
      const size_t p = q * ntot + pidx(i, j, k);
      const T up = Uin[p] + T(cdt) * L[q * nint + iidx(i, j, k)];
      Uout[p] = (a0 == 0.0) ? up : T(a0) * Uref[p] + T(a1) * up;
    }
  }
  // R27: the higher-order SSP schemes the paper names without a tableau (ref.[25]), in Shu-Osher form; the
  // first stage's L(U^n) has been evaluated by the caller.  dt once per step (R11).
  //   RK43 (4 stages, order 3, c = 1/2):
  //     U1 = Un + c dt L(Un);  U2 = U1 + c dt L(U1);  U3 = 2/3 Un + 1/3 (U2 + c dt L(U2));  Un+1 = U3 + c dt L(U3)
  //   RK53 (5 stages, order 3, Ruuth's form of the optimal scheme, c = 0.377268915331368):
  //     U1 = Un + c dt L(Un);  U2 = U1 + c dt L(U1);
  //     U3 = 0.355909775063327 Un + 0.644090224936674 (U2 + c dt L(U2));
  //     U4 = 0.367933791638137 Un + 0.632066208361863 (U3 + c dt L(U3));
  //     Un+1 = 0.237593836598569 U2 + 0.762406163401431 (U4 + c dt L(U4))
  void step_ssp_high(double dt) {
    if (U2.empty()) U2.assign(nv * ntot, T(0.0));
    if (s.rk == 4) {
      const double c = 0.5;
      combine(U1, 0.0, Un, 1.0, Un, c * dt);                                   // U1
      fill_ghosts(U1); rhs(U1);
      combine(U2, 0.0, Un, 1.0, U1, c * dt);                                   // U2
      fill_ghosts(U2); rhs(U2);
      combine(U1, 2.0 / 3.0, Un, 1.0 / 3.0, U2, c * dt);                       // U3 (over U1)
      fill_ghosts(U1); rhs(U1);
      combine(Un, 0.0, Un, 1.0, U1, c * dt);                                   // Un+1
    } else {
      const double c = 0.377268915331368;
      if (U3.empty()) U3.assign(nv * ntot, T(0.0));
      combine(U1, 0.0, Un, 1.0, Un, c * dt);                                   // U1
      fill_ghosts(U1); rhs(U1);
      combine(U2, 0.0, Un, 1.0, U1, c * dt);                                   // U2 (kept for the last stage)
      fill_ghosts(U2); rhs(U2);
      combine(U1, 0.355909775063327, Un, 0.644090224936674, U2, c * dt);       // U3 (over U1)
      fill_ghosts(U1); rhs(U1);
      combine(U3, 0.367933791638137, Un, 0.632066208361863, U1, c * dt);       // U4
      fill_ghosts(U3); rhs(U3);
      combine(Un, 0.237593836598569, U2, 0.762406163401431, U3, c * dt);       // Un+1
    }
    if (glm) glm_source(dt);
    if (cgl) cgl_source();
    t += dt;
  }
  void step(double dt) {
    if (glm) { double vm = 0.0; vmax(&vm); ch = 0.95 * vm; }
    fill_ghosts(Un);
    rhs(Un);
    if (s.rk == 4 || s.rk == 5) { step_ssp_high(dt); return; }
    if (s.rk == 1) {
      for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
        const size_t p = q * ntot + pidx(i, j, k);
        Un[p] = Un[p] + T(dt) * L[q * nint + iidx(i, j, k)];
      }
      if (glm) glm_source(dt);
      if (cgl) cgl_source();
      t += dt;
      return;
    }
    for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
      const size_t p = q * ntot + pidx(i, j, k);
      U1[p] = Un[p] + T(dt) * L[q * nint + iidx(i, j, k)];                         // stage 1
    }
    fill_ghosts(U1);
    rhs(U1);
    if (s.rk == 3) {
      // R25: SSP-RK33 in Shu-Osher form:  U2 = 3/4 Un + 1/4 (U1 + dt L(U1));  Un+1 = 1/3 Un + 2/3 (U2 + dt L(U2))
      if (U2.empty()) U2.assign(nv * ntot, T(0.0));
      for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
        const size_t p = q * ntot + pidx(i, j, k);
        U2[p] = T(0.75) * Un[p] + T(0.25) * (U1[p] + T(dt) * L[q * nint + iidx(i, j, k)]);
      }
      fill_ghosts(U2);
      rhs(U2);
      for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
        const size_t p = q * ntot + pidx(i, j, k);
        Un[p] = T(1.0 / 3.0) * Un[p] + T(2.0 / 3.0) * (U2[p] + T(dt) * L[q * nint + iidx(i, j, k)]);
      }
      if (glm) glm_source(dt);
      if (cgl) cgl_source();
      t += dt;
      return;
    }
    for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i) {
      const size_t p = q * ntot + pidx(i, j, k);
      Un[p] = T(0.5) * Un[p] + T(0.5) * (U1[p] + T(dt) * L[q * nint + iidx(i, j, k)]);   // stage 2
    }
    if (glm) glm_source(dt);
    if (cgl) cgl_source();
    t += dt;
  }

  void set_state(const double* U, double t0) {
    for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i)
      Un[q * ntot + pidx(i, j, k)] = T(U[q * nint + iidx(i, j, k)]);
    t = t0; have_state = true;
  }
  void get_state(double* U) const {
    for (int q = 0; q < nv; ++q) for (int k = 0; k < nd[2]; ++k) for (int j = 0; j < nd[1]; ++j) for (int i = 0; i < nd[0]; ++i)
      U[q * nint + iidx(i, j, k)] = val(Un[q * ntot + pidx(i, j, k)]);
  }
};

int check_args(const agate_ref_grid* g, double gamma, int eqset, const agate_ref_solver* s) {
  if (!g || !s) return 1;
  if (g->ndim < 1 || g->ndim > 3) return 1;
  if (g->nx < 1 || g->ny < 1 || g->nz < 1) return 1;
  if (g->ndim < 3 && g->nz != 1) return 1;
  if (g->ndim < 2 && g->ny != 1) return 1;
  if (!(g->dx > 0.0) || (g->ndim >= 2 && !(g->dy > 0.0)) || (g->ndim >= 3 && !(g->dz > 0.0))) return 1;
  if (!(gamma > 1.0)) return 1;
  if (eqset != AGATE_REF_IDEAL && eqset != AGATE_REF_HALL && eqset != AGATE_REF_IDEAL_GLM && eqset != AGATE_REF_CGL &&
      eqset != AGATE_REF_HALL_GLM && eqset != AGATE_REF_CGL_GLM) return 1;
  const bool cgl_set = (eqset == AGATE_REF_CGL || eqset == AGATE_REF_CGL_GLM);
  if (cgl_set && s->riemann != 0) return 1;          // the paper's CGL runs use HLL
  if (cgl_set && !(s->relax >= 0.0 && s->relax <= 1.0)) return 1;
  if (s->cgl_form < 0 || s->cgl_form > 1) return 1;
  if (s->riemann < 0 || s->riemann > 1 || s->limiter < 0 || s->limiter > 2 || s->rk < 1 || s->rk > 5) return 1;
  if (s->limiter == 2 && !(s->beta >= 1.0 && s->beta <= 2.0)) return 1;
  for (int d = 0; d < 3; ++d) if (s->bc[d] < 0 || s->bc[d] > ((d == 1) ? 2 : 1)) return 1;
  if (s->bc[1] == 2 && (g->ndim < 2 || s->bc[0] != 0)) return 1;   // sheared ends in y need a periodic x (R28)
  const bool hall_set = (eqset == AGATE_REF_HALL || eqset == AGATE_REF_HALL_GLM);
  if (hall_set && s->riemann == 1) return 1;        // no Hall-HLLD in the paper
  if (hall_set && !(s->d_i >= 0.0)) return 1;
  return 0;
}

}  // namespace

struct agate_ref_ctx { Solver<double>* s; };

extern "C" {

void agate_ref_set_threads(int n) {
#ifdef _OPENMP
  g_threads = n < 1 ? 1 : n;
#else
  (void)n; g_threads = 1;
#endif
}
int agate_ref_get_threads(void) { return g_threads; }

int agate_ref_create(const agate_ref_grid* g, double gamma, int eqset, const agate_ref_solver* s, agate_ref_ctx** out) {
  if (!out) return 1;
  int rc = check_args(g, gamma, eqset, s);
  if (rc) return rc;
  try {
    agate_ref_ctx* c = new agate_ref_ctx;
    c->s = new Solver<double>(*g, gamma, eqset, *s);
    *out = c;
  } catch (const std::bad_alloc&) { return 5; }
  return 0;
}
int agate_ref_set_state(agate_ref_ctx* c, const double* U, double t0) {
  if (!c || !U) return 1;
  c->s->set_state(U, t0);
  return 0;
}
int agate_ref_compute_dt(agate_ref_ctx* c, double* dt) {
  if (!c || !dt) return 1;
  if (!c->s->have_state) return 2;
  double v; int rc = c->s->compute_dt(&v);
  if (rc) return rc;
  *dt = v; return 0;
}
int agate_ref_vmax(agate_ref_ctx* c, double* vm) {
  if (!c || !vm) return 1;
  if (!c->s->have_state) return 2;
  double v; int rc = c->s->vmax(&v);
  if (rc) return rc;
  *vm = v; return 0;
}
int agate_ref_step(agate_ref_ctx* c, double dt, double* dt_used) {
  if (!c) return 1;
  if (!c->s->have_state) return 2;
  if (!(dt > 0.0)) { int rc = c->s->compute_dt(&dt); if (rc) return rc; }
  c->s->step(dt);
  if (dt_used) *dt_used = dt;
  return 0;
}
int agate_ref_advance(agate_ref_ctx* c, int32_t n, double* t_out) {
  if (!c || n < 0) return 1;
  if (!c->s->have_state) return 2;
  for (int i = 0; i < n; ++i) {
    double dt; int rc = c->s->compute_dt(&dt);
    if (rc) return rc;
    c->s->step(dt);
  }
  if (t_out) *t_out = c->s->t;
  return 0;
}
int agate_ref_get_state(agate_ref_ctx* c, double* U, double* t_out) {
  if (!c || !U) return 1;
  if (!c->s->have_state) return 2;
  c->s->get_state(U);
  if (t_out) *t_out = c->s->t;
  return 0;
}
int agate_ref_rhs(agate_ref_ctx* c, double* Lout) {
  if (!c || !Lout) return 1;
  if (!c->s->have_state) return 2;
  if (c->s->glm) { double vm = 0.0; c->s->vmax(&vm); c->s->ch = 0.95 * vm; }
  c->s->fill_ghosts(c->s->Un);
  c->s->rhs(c->s->Un);
  std::memcpy(Lout, c->s->L.data(), sizeof(double) * c->s->nv * c->s->nint);
  return 0;
}
void agate_ref_cgl_cons_to_prim(const double U[9], double W[9]) { cgl_cons_to_prim<double>(U, W); }
void agate_ref_cgl_prim_to_cons(const double W[9], double U[9]) { cgl_prim_to_cons<double>(W, U); }
void agate_ref_cgl_cons_to_prim_form(int form, const double U[9], double W[9]) { cgl_cons_to_prim<double>(U, W, form); }
void agate_ref_cgl_prim_to_cons_form(int form, const double W[9], double U[9]) { cgl_prim_to_cons<double>(W, U, form); }
void agate_ref_cgl_face_flux_form(int form, int dir, const double WL[9], const double WR[9], double F[9]) { cgl_flux_hll<double>(dir, WL, WR, F, form); }
double agate_ref_cgl_cfast(int dir, const double W[9]) { return cgl_cfast<double>(dir, W); }
void agate_ref_cgl_face_flux(int dir, const double WL[9], const double WR[9], double F[9]) { cgl_flux_hll<double>(dir, WL, WR, F); }
void agate_ref_cgl_relax(double f, double B2, double* ppar, double* pperp) { cgl_relax(f, B2, ppar, pperp); }
int agate_ref_nvar(agate_ref_ctx* c) { return c ? c->s->nv : 0; }
int agate_ref_glm_ch(agate_ref_ctx* c, double* ch_out) {
  if (!c || !ch_out) return 1;
  *ch_out = c->s->ch;
  return 0;
}
void agate_ref_glm_face(double ch, double bnL, double bnR, double psL, double psR, double* bns, double* pss) {
  glm_face<double>(ch, bnL, bnR, psL, psR, bns, pss);
}
int agate_ref_destroy(agate_ref_ctx* c) {
  if (!c) return 1;
  delete c->s; delete c;
  return 0;
}

void agate_ref_cons_to_prim(double gamma, const double U[8], double W[8]) { cons_to_prim<double>(gamma, U, W); }
void agate_ref_prim_to_cons(double gamma, const double W[8], double U[8]) { prim_to_cons<double>(gamma, W, U); }
double agate_ref_slope(int limiter, double beta, double dp, double dm) { return slope<double>(limiter, beta, dp, dm); }
double agate_ref_cfast(int dir, double gamma, const double W[8]) { return cfast<double>(dir, gamma, W); }
double agate_ref_cwhistler(double d_i, double dxmin, const double W[8]) { return cwhistler<double>(d_i, dxmin, W); }
void agate_ref_phys_flux(int dir, double gamma, const double W[8], const double vH[3], double F[8]) {
  phys_flux<double>(dir, gamma, W, vH, F);
}
void agate_ref_face_flux(int eqset, int riemann, int dir, double gamma, double d_i, double dxmin,
                         const double WL[8], const double WR[8], const double J[3], double F[8]) {
  face_flux<double>(eqset, riemann, dir, gamma, d_i, dxmin, WL, WR, J, F);
}
int agate_ref_hlld_branch(int dir, double gamma, const double WL[8], const double WR[8]) {
  double F[8];
  return flux_hlld<double>(dir, gamma, WL, WR, F);
}

int agate_ref_count_ops(const agate_ref_grid* g, double gamma, int eqset, const agate_ref_solver* s,
                        const double* U, double out[5]) {
  int rc = check_args(g, gamma, eqset, s);
  if (rc || !U || !out) return rc ? rc : 1;
  const int saved = g_threads;
  g_threads = 1;                       // the counters are global
  try {
    Solver<Counted> sol(*g, gamma, eqset, *s);
    sol.set_state(U, 0.0);
    g_ops = OpCount();
    double dt;
    rc = sol.compute_dt(&dt);
    if (!rc) sol.step(dt);
  } catch (const std::bad_alloc&) { g_threads = saved; return 5; }
  g_threads = saved;
  out[0] = g_ops.add; out[1] = g_ops.mul; out[2] = g_ops.div; out[3] = g_ops.sqrt; out[4] = g_ops.cmp;
  return rc;
}

}  // extern "C"
