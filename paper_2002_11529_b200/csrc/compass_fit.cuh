// compass_fit.cuh -- step 6 of the Compass definition: the
// weighted linear chi2 fit with the VELO pseudo-point, shared by the fused kernel (compass.cu) and the
// paper-literal two-kernel variant (windows.cu).  __f*_rn intrinsics in the written order: bit-exact, no FMA.
#pragma once
#include "common.cuh"

namespace utc {

// Optional position-dependent kick table (include/ut_compass.h ut_geometry.kick_*; A24):
// a track's kappa and z_mag from the cell that holds its straight-line position at z_ref (nearest cell).
struct KickTable {
  uint32_t nx, ny;
  float x_lo, y_lo, inv_dx, inv_dy, z_ref;
  const float *kappa, *z_mag;
};
inline KickTable make_kick_table(const ut_geometry* g) {
  KickTable k;
  k.nx = g->kick_nx; k.ny = g->kick_ny; k.x_lo = g->kick_x_lo; k.y_lo = g->kick_y_lo; k.inv_dx = g->kick_inv_dx;
  k.inv_dy = g->kick_inv_dy; k.z_ref = g->kick_z_ref; k.kappa = g->kick_kappa; k.z_mag = g->kick_z_mag;
  return k;
}
__device__ __forceinline__ int kick_index(float v, float lo, float inv, uint32_t n) {
  const float u = __fmul_rn(__fsub_rn(v, lo), inv);
  if (!(u == u)) return 0;
  const float f = floorf(u);
  if (f < 0.f) return 0;
  if (f > (float)(n - 1)) return (int)n - 1;
  return (int)f;
}
__device__ __forceinline__ void track_kick(const KickTable& k, const compass_config& c, float vx, float vy, float vtx,
                                           float vty, float vz, float& kappa, float& z_mag) {
  kappa = c.kappa;
  z_mag = c.z_mag;
  if (k.nx == 0) return;
  const float dzr = __fsub_rn(k.z_ref, vz);
  const float xk = __fadd_rn(vx, __fmul_rn(vtx, dzr)), yk = __fadd_rn(vy, __fmul_rn(vty, dzr));
  const int cell = kick_index(yk, k.y_lo, k.inv_dy, k.ny) * (int)k.nx + kick_index(xk, k.x_lo, k.inv_dx, k.nx);
  kappa = __ldg(k.kappa + cell);
  z_mag = __ldg(k.z_mag + cell);
}

struct FitResult { float chi2, b; bool valid; };

__device__ __forceinline__ void fit_acc(bool p, float d, float dz, float w, float& S0, float& S1, float& S2,
                                        float& T0, float& T1) {
  if (p) {
    const float wdz = __fmul_rn(w, dz);
    S0 = __fadd_rn(S0, w);
    S1 = __fadd_rn(S1, wdz);
    S2 = __fadd_rn(S2, __fmul_rn(wdz, dz));
    const float wd = __fmul_rn(w, d);
    T0 = __fadd_rn(T0, wd);
    T1 = __fadd_rn(T1, __fmul_rn(wd, dz));
  }
}
__device__ __forceinline__ float fit_res(bool p, float d, float dz, float w, float a, float b, float chi2) {
  if (p) {
    const float r = __fsub_rn(__fsub_rn(d, a), __fmul_rn(b, dz));
    chi2 = __fadd_rn(chi2, __fmul_rn(__fmul_rn(w, r), r));
  }
  return chi2;
}

// Weighted linear LSQ of d vs dz = z - z_mag with the VELO pseudo-point (0, 0, w_velo); hits in layer order.
// (z_mag: the track's kick plane, compass_config.z_mag unless a kick table is in use)
__device__ __forceinline__ FitResult fit_tracklet(const bool (&p)[4], const float (&d)[4], const float (&z)[4],
                                                  const float (&w)[4], int n, const compass_config& c, float z_mag) {
  float dz[4];
#pragma unroll
  for (int l = 0; l < 4; ++l) dz[l] = __fsub_rn(z[l], z_mag);
  float S0 = c.w_velo, S1 = 0.f, S2 = 0.f, T0 = 0.f, T1 = 0.f;
#pragma unroll
  for (int l = 0; l < 4; ++l) fit_acc(p[l], d[l], dz[l], w[l], S0, S1, S2, T0, T1);
  const float det = __fsub_rn(__fmul_rn(S0, S2), __fmul_rn(S1, S1));
  const float a = __fdiv_rn(__fsub_rn(__fmul_rn(T0, S2), __fmul_rn(T1, S1)), det);
  const float b = __fdiv_rn(__fsub_rn(__fmul_rn(T1, S0), __fmul_rn(T0, S1)), det);
  float chi2 = __fmul_rn(__fmul_rn(c.w_velo, a), a);
#pragma unroll
  for (int l = 0; l < 4; ++l) chi2 = fit_res(p[l], d[l], dz[l], w[l], a, b, chi2);
  FitResult r;
  r.chi2 = chi2;
  r.b = b;
  r.valid = chi2 <= __fmul_rn(c.max_chi2_ndf, (float)(n - 1));
  return r;
}

}  // namespace utc
