// physics_shim.cpp — HOST build of the CUDA path's point functions (paper_2503_20899_b200/csrc/agate_physics.cuh)
// so that `-m "not gpu"` tests can compare them with the oracle without a GPU.  Test infrastructure only:
// compiled by tests/test_physics_host.py with g++; it is not part of the product library.
#include "agate_physics.cuh"

using namespace agate;

extern "C" {

void shim_face_flux(int eqset, int riemann, int dir, double gamma, double d_i, double dxmin, const double* WL,
                    const double* WR, const double* J, double* F) {
  Phys ph = make_phys(gamma, eqset == 1 ? d_i : 0.0, dxmin);
  double L[8], R[8], Jr[3] = {0, 0, 0}, Fr[8];
  for (int r = 0; r < 8; ++r) { L[r] = WL[rot_var(r, dir)]; R[r] = WR[rot_var(r, dir)]; }
  if (J) for (int c = 0; c < 3; ++c) Jr[c] = J[(dir + c) % 3];
  if (eqset == 1) riemann_flux<0, true>(ph, L, R, Jr, Fr);
  else if (riemann == 1) riemann_flux<1, false>(ph, L, R, nullptr, Fr);
  else riemann_flux<0, false>(ph, L, R, nullptr, Fr);
  unrotate(dir, Fr, F);
}

void shim_cons_to_prim(double gamma, const double* U, double* W) {
  Phys ph = make_phys(gamma, 0.0, 1.0);
  cons_to_prim(ph, U, W);
}

double shim_slope(int limiter, double beta, double dp, double dm) { return limited_slope(limiter, beta, dp, dm); }

double shim_half_slope(int limiter, double hbeta, double dp, double dm) { return half_slope(limiter, hbeta, dp, dm); }

// A2 in one piece (limited slope + both face states), and the two HLLD bodies on their own
void shim_plm_faces(int limiter, double beta2, double a, double b, double c, double* lo, double* hi) {
  plm_faces(limiter, beta2, a, b, c, *lo, *hi);
}
int shim_hlld_fast(int dir, double gamma, const double* WL, const double* WR, double* F) {
  Phys ph = make_phys(gamma, 0.0, 1.0);
  double L[8], R[8], Fr[8];
  for (int r = 0; r < 8; ++r) { L[r] = WL[rot_var(r, dir)]; R[r] = WR[rot_var(r, dir)]; }
  const bool slow = flux_hlld_fast(ph, L, R, Fr);
  unrotate(dir, Fr, F);
  return slow ? 1 : 0;
}
void shim_hlld_general(int dir, double gamma, const double* WL, const double* WR, double* F) {
  Phys ph = make_phys(gamma, 0.0, 1.0);
  double L[8], R[8], Fr[8];
  for (int r = 0; r < 8; ++r) { L[r] = WL[rot_var(r, dir)]; R[r] = WR[rot_var(r, dir)]; }
  flux_hlld_general(ph, L, R, Fr);
  unrotate(dir, Fr, F);
}

double shim_cell_speed_inline(int eqset, double gamma, double d_i, double dxmin, const double* U) {
  Phys ph = make_phys(gamma, eqset == 1 ? d_i : 0.0, dxmin);
  return eqset == 1 ? cell_speed_inline<true>(ph, U) : cell_speed_inline<false>(ph, U);
}

// CGL (R24): the kernels' point functions, rotated frame handled here as the kernels do
void shim_cgl_cons_to_prim(const double* U, double* W) { cgl_cons_to_prim(U, W); }
void shim_cgl_face_flux(int dir, const double* WL, const double* WR, double* F) {
  double L[9], R[9], Fr[9];
  for (int r = 0; r < 9; ++r) { const int v = (r < 8) ? rot_var(r, dir) : r; L[r] = WL[v]; R[r] = WR[v]; }
  flux_hll_cgl(L, R, Fr);
  for (int r = 0; r < 9; ++r) F[(r < 8) ? rot_var(r, dir) : r] = Fr[r];
}
double shim_cgl_relaxed_alog(double f, const double* U) { return cgl_relaxed_alog(f, U); }
double shim_cell_speed_cgl(const double* U) { return cell_speed_cgl(U); }
// the same with the thermodynamic variable of eq.16 (form 1)
void shim_cgl_cons_to_prim_form(int form, const double* U, double* W) { cgl_cons_to_prim(U, W, form); }
void shim_cgl_face_flux_form(int form, int dir, const double* WL, const double* WR, double* F) {
  double L[9], R[9], Fr[9];
  for (int r = 0; r < 9; ++r) { const int v = (r < 8) ? rot_var(r, dir) : r; L[r] = WL[v]; R[r] = WR[v]; }
  flux_hll_cgl(L, R, Fr, form);
  for (int r = 0; r < 9; ++r) F[(r < 8) ? rot_var(r, dir) : r] = Fr[r];
}
double shim_cgl_relaxed_form(int form, double f, const double* U) { return cgl_relaxed_alog(f, U, form); }
double shim_cell_speed_cgl_form(int form, const double* U) { return cell_speed_cgl(U, form); }

double shim_cell_speed(int eqset, double gamma, double d_i, double dxmin, const double* U) {
  Phys ph = make_phys(gamma, eqset == 1 ? d_i : 0.0, dxmin);
  return eqset == 1 ? cell_speed<true>(ph, U) : cell_speed<false>(ph, U);
}
}
