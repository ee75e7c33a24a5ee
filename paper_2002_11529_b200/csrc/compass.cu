// compass.cu -- Compass tracking (section V, :276-348) as ONE fused kernel.
//
// The paper runs two kernels: "search UT windows" (2-D: 4 panels x tracks) writes
// (first hit, size) ranges to global memory, then "tracklet finding" (thread per track)
// reads them back through a shared-memory cache.  On a B200 the whole event fits in one
// SM's shared memory, so one CTA takes one event:
//
//   stage the event's x / yBegin / yEnd / z / weight arrays in smem (read HBM/L2 once per event)
//   phase 1, lane = (track, layer)  -- the paper's 2-D window kernel shape:
//       straight-line extrapolation, group range by binary search on the group x-bounds, binary
//       search of the first hit with d >= -win, scan while d <= +win with the y test; the accepted
//       hits (closest `max_candidates_per_layer` in |d|) go to a per-(track, layer) list in smem
//   phase 2, the 4 lanes of a track split the seed pairs (a, b): slope + kink cuts, compatible hits
//       in the other two layers as 32-bit masks, every 3/4-hit combination fitted (linear chi2 fit
//       with the VELO pseudo-point), packed (n, chi2, positions) key, min over the quad = the
//       deterministic best tracklet; forward seeds first, backward only if forward found nothing.
//   The candidate lists never leave the SM; the two phases are separated by __syncwarp only.
//
// fp32 arithmetic uses __f*_rn intrinsics in the order of DESIGN.md section 3 (bit-exact, no FMA).
#include <algorithm>
#include <cstdlib>

#include "common.cuh"

namespace utc {

constexpr float kGroupEps = 0.01f;     // slack of the group pre-selection [mm] (A17)
constexpr unsigned long long kNoKey = ~0ull;

struct CompassArgs {
  const float *hx, *hz, *hyb, *hye, *hdxdy, *hw;
  const uint32_t* hit_offsets;
  const float *vx, *vy, *vtx, *vty;
  float vz;
  const uint32_t* velo_offsets;
  int32_t n_events;
  uint32_t n_groups, gpl;
  const float *group_xmin, *group_xmax;
  float layer_z[4], layer_dxdy[4];
  compass_config c;
  int32_t *out_idx, *out_n;
  float *out_qop, *out_chi2;
  uint32_t* status;
  uint32_t hit_stage;     // elements per staged array
};

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
__device__ __forceinline__ FitResult fit_tracklet(bool p0, float d0, float z0, float w0, bool p1, float d1, float z1,
                                                  float w1, bool p2, float d2, float z2, float w2, bool p3, float d3,
                                                  float z3, float w3, int n, const compass_config& c) {
  const float dz0 = __fsub_rn(z0, c.z_mag), dz1 = __fsub_rn(z1, c.z_mag), dz2 = __fsub_rn(z2, c.z_mag),
              dz3 = __fsub_rn(z3, c.z_mag);
  float S0 = c.w_velo, S1 = 0.f, S2 = 0.f, T0 = 0.f, T1 = 0.f;
  fit_acc(p0, d0, dz0, w0, S0, S1, S2, T0, T1);
  fit_acc(p1, d1, dz1, w1, S0, S1, S2, T0, T1);
  fit_acc(p2, d2, dz2, w2, S0, S1, S2, T0, T1);
  fit_acc(p3, d3, dz3, w3, S0, S1, S2, T0, T1);
  const float det = __fsub_rn(__fmul_rn(S0, S2), __fmul_rn(S1, S1));
  const float a = __fdiv_rn(__fsub_rn(__fmul_rn(T0, S2), __fmul_rn(T1, S1)), det);
  const float b = __fdiv_rn(__fsub_rn(__fmul_rn(T1, S0), __fmul_rn(T0, S1)), det);
  float chi2 = __fmul_rn(__fmul_rn(c.w_velo, a), a);
  chi2 = fit_res(p0, d0, dz0, w0, a, b, chi2);
  chi2 = fit_res(p1, d1, dz1, w1, a, b, chi2);
  chi2 = fit_res(p2, d2, dz2, w2, a, b, chi2);
  chi2 = fit_res(p3, d3, dz3, w3, a, b, chi2);
  FitResult r;
  r.chi2 = chi2;
  r.b = b;
  r.valid = chi2 <= __fmul_rn(c.max_chi2_ndf, (float)(n - 1));
  return r;
}

// (n desc, chi2 asc, hit tuple asc): candidate positions are ascending in hit index, none = 63
__device__ __forceinline__ unsigned long long make_key(int n, float chi2, uint32_t p0, uint32_t p1, uint32_t p2,
                                                       uint32_t p3) {
  return ((unsigned long long)(4 - n) << 56) | ((unsigned long long)__float_as_uint(chi2) << 24) |
         (unsigned long long)((p0 << 18) | (p1 << 12) | (p2 << 6) | p3);
}

struct CandView {           // per-(track, layer) candidate lists, entry i of slot s at [i * slots + s]
  float* d;
  uint16_t* h;
  uint32_t slots;
};

// One search direction for the pairs owned by this lane.  DIR 0: seeds (L0, L2), others (L1, L3);
// DIR 1: seeds (L3, L1), others (L2, L0).
template <int DIR>
__device__ __forceinline__ unsigned long long search_direction(const CandView& cv, const float* __restrict__ Z,
                                                               const float* __restrict__ W, uint32_t qslot, int ql,
                                                               const int (&n)[4], const uint32_t (&lf)[4],
                                                               const compass_config& c) {
  constexpr int LA = DIR ? 3 : 0, LB = DIR ? 1 : 2, LC = DIR ? 2 : 1, LD = DIR ? 0 : 3;
  const int nA = n[LA], nB = n[LB], nC = n[LC], nD = n[LD];
  const uint32_t sA = qslot + LA, sB = qslot + LB, sC = qslot + LC, sD = qslot + LD;
  unsigned long long best = kNoKey;
  const int P = nA * nB;
  if (ql >= P) return best;
  int ia = ql / nB, ib = ql - ia * nB;
  for (int p = ql; p < P; p += 4) {
    const float da = cv.d[ia * cv.slots + sA], db = cv.d[ib * cv.slots + sB];
    const uint32_t ha = lf[LA] + cv.h[ia * cv.slots + sA], hb = lf[LB] + cv.h[ib * cv.slots + sB];
    const float za = Z[ha], zb = Z[hb];
    const float bs = __fdiv_rn(__fsub_rn(db, da), __fsub_rn(zb, za));
    const float a0 = __fsub_rn(da, __fmul_rn(bs, __fsub_rn(za, c.z_mag)));
    if (fabsf(bs) <= c.max_slope && fabsf(a0) <= c.kink_tol) {
      uint32_t mC = 0, mD = 0;
      for (int i = 0; i < nC; ++i) {
        const float dc = cv.d[i * cv.slots + sC];
        const float zc = Z[lf[LC] + cv.h[i * cv.slots + sC]];
        const float pred = __fadd_rn(da, __fmul_rn(bs, __fsub_rn(zc, za)));
        if (fabsf(__fsub_rn(dc, pred)) <= c.seed_tol) mC |= 1u << i;
      }
      for (int i = 0; i < nD; ++i) {
        const float dd = cv.d[i * cv.slots + sD];
        const float zd = Z[lf[LD] + cv.h[i * cv.slots + sD]];
        const float pred = __fadd_rn(da, __fmul_rn(bs, __fsub_rn(zd, za)));
        if (fabsf(__fsub_rn(dd, pred)) <= c.seed_tol) mD |= 1u << i;
      }
      const float wa = W[ha], wb = W[hb];
      // every (c or none) x (d or none) with >= min_hits hits in total
      uint32_t remC = mC;
      for (int ci = -1;;) {
        float dc = 0.f, zc = 0.f, wc = 0.f;
        if (ci >= 0) {
          const uint32_t hc = lf[LC] + cv.h[ci * cv.slots + sC];
          dc = cv.d[ci * cv.slots + sC]; zc = Z[hc]; wc = W[hc];
        }
        uint32_t remD = mD;
        for (int di = -1;;) {
          const int nh = 2 + (ci >= 0) + (di >= 0);
          if (nh >= c.min_hits) {
            float dd = 0.f, zd = 0.f, wd = 0.f;
            if (di >= 0) {
              const uint32_t hd = lf[LD] + cv.h[di * cv.slots + sD];
              dd = cv.d[di * cv.slots + sD]; zd = Z[hd]; wd = W[hd];
            }
            const uint32_t pc = ci >= 0 ? (uint32_t)ci : 63u, pd = di >= 0 ? (uint32_t)di : 63u;
            FitResult r;
            unsigned long long key;
            if (DIR == 0) {      // layer order L0 = a, L1 = c, L2 = b, L3 = d
              r = fit_tracklet(true, da, za, wa, ci >= 0, dc, zc, wc, true, db, zb, wb, di >= 0, dd, zd, wd, nh, c);
              key = make_key(nh, r.chi2, (uint32_t)ia, pc, (uint32_t)ib, pd);
            } else {             // layer order L0 = d, L1 = b, L2 = c, L3 = a
              r = fit_tracklet(di >= 0, dd, zd, wd, true, db, zb, wb, ci >= 0, dc, zc, wc, true, da, za, wa, nh, c);
              key = make_key(nh, r.chi2, pd, (uint32_t)ib, pc, (uint32_t)ia);
            }
            if (r.valid && key < best) best = key;
          }
          if (!remD) break;
          di = __ffs(remD) - 1;
          remD &= remD - 1;
        }
        if (!remC) break;
        ci = __ffs(remC) - 1;
        remC &= remC - 1;
      }
    }
    ib += 4;
    while (ib >= nB) { ib -= nB; ++ia; }
  }
  return best;
}

template <bool STAGED>
__device__ __forceinline__ void track_loop(const CompassArgs& a, const float* __restrict__ X,
                                           const float* __restrict__ YB, const float* __restrict__ YE,
                                           const float* __restrict__ Z, const float* __restrict__ W,
                                           const uint32_t* s_goff, const float* s_gdxdy, const float* s_gxmin,
                                           const float* s_gxmax, const CandView cv, uint32_t a0, uint32_t t0,
                                           uint32_t t1, uint32_t T) {
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31;
  const int l = tid & 3;                         // layer of this lane in phase 1, lane-in-quad in phase 2
  const uint32_t qslot = tid & ~3u, slot = tid;
  const unsigned qmask = 0xFu << (lane & ~3);
  const uint32_t gpl = a.gpl;
  const int C = a.c.max_candidates_per_layer;
  uint32_t lf[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) lf[k] = s_goff[k * gpl];
  const uint32_t my_lf = lf[0] * (l == 0) + lf[1] * (l == 1) + lf[2] * (l == 2) + lf[3] * (l == 3);

  for (uint32_t tb = t0; tb < t1; tb += (uint32_t)(nt >> 2)) {
    const uint32_t tg = tb + (uint32_t)(tid >> 2);
    const bool active = tg < t1;
    // ---------------- phase 1: window search, lane = (track, layer) ----------------
    int n_st = 0;
    if (active) {
      const float vx = __ldg(a.vx + tg), vy = __ldg(a.vy + tg), vtx = __ldg(a.vtx + tg), vty = __ldg(a.vty + tg);
      const float dzv = __fsub_rn(a.layer_z[l], a.vz);
      const float x_e = __fadd_rn(vx, __fmul_rn(vtx, dzv));
      const float y_e = __fadd_rn(vy, __fmul_rn(vty, dzv));
      const float D = a.c.win_half[l], negD = -D, y_tol = a.c.y_tol;
      const float ctr = __fsub_rn(x_e, __fmul_rn(a.layer_dxdy[l], y_e));
      const float lo = __fsub_rn(__fsub_rn(ctr, D), kGroupEps), hi = __fadd_rn(__fadd_rn(ctr, D), kGroupEps);
      const uint32_t gend = (l + 1) * gpl;
      uint32_t g = l * gpl;
      for (uint32_t cnt = gpl; cnt > 0;) {            // first group with group_xmax >= lo
        const uint32_t half = cnt >> 1, mid = g + half;
        if (s_gxmax[mid] >= lo) cnt = half; else { g = mid + 1; cnt -= half + 1; }
      }
      int worst = -1;
      float worst_abs = 0.f;
      for (; g < gend && s_gxmin[g] <= hi; ++g) {
        const uint32_t ga = s_goff[g], gb = s_goff[g + 1];
        if (ga == gb) continue;
        const float syg = __fmul_rn(s_gdxdy[g], y_e);
        uint32_t first = ga;
        for (uint32_t cnt = gb - ga; cnt > 0;) {      // first hit with d >= -D
          const uint32_t half = cnt >> 1, mid = first + half;
          const float d = __fsub_rn(__fadd_rn(X[mid], syg), x_e);
          if (d >= negD) cnt = half; else { first = mid + 1; cnt -= half + 1; }
        }
        for (uint32_t h = first; h < gb; ++h) {
          const float d = __fsub_rn(__fadd_rn(X[h], syg), x_e);
          if (!(d <= D)) break;
          if (!(__fsub_rn(YB[h], y_tol) <= y_e && y_e <= __fadd_rn(YE[h], y_tol))) continue;
          if (n_st < C) {
            cv.d[n_st * cv.slots + slot] = d;
            cv.h[n_st * cv.slots + slot] = (uint16_t)(h - my_lf);
            ++n_st;
          } else {                                    // keep the C closest in (|d|, h); list stays ascending in h
            if (worst < 0) {
              worst = 0; worst_abs = fabsf(cv.d[slot]);
              for (int i = 1; i < C; ++i) {
                const float v = fabsf(cv.d[i * cv.slots + slot]);
                if (v >= worst_abs) { worst_abs = v; worst = i; }
              }
            }
            if (fabsf(d) < worst_abs) {
              for (int i = worst; i < C - 1; ++i) {
                cv.d[i * cv.slots + slot] = cv.d[(i + 1) * cv.slots + slot];
                cv.h[i * cv.slots + slot] = cv.h[(i + 1) * cv.slots + slot];
              }
              cv.d[(C - 1) * cv.slots + slot] = d;
              cv.h[(C - 1) * cv.slots + slot] = (uint16_t)(h - my_lf);
              worst = -1;
            }
          }
        }
      }
    }
    __syncwarp();
    // ---------------- phase 2: tracklet finding, 4 lanes per track -----------------
    int n[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) n[k] = __shfl_sync(0xFFFFFFFFu, n_st, (lane & ~3) + k);
    const int nonempty = (n[0] > 0) + (n[1] > 0) + (n[2] > 0) + (n[3] > 0);
    unsigned long long best = kNoKey;
    if (nonempty >= a.c.min_hits) {
      best = search_direction<0>(cv, Z, W, qslot, l, n, lf, a.c);
      best = min(best, __shfl_xor_sync(qmask, best, 1));
      best = min(best, __shfl_xor_sync(qmask, best, 2));
      if (best == kNoKey) {                          // backward only if forward found nothing valid (A11)
        best = search_direction<1>(cv, Z, W, qslot, l, n, lf, a.c);
        best = min(best, __shfl_xor_sync(qmask, best, 1));
        best = min(best, __shfl_xor_sync(qmask, best, 2));
      }
    }
    if (active) {
      int nh = 0, hidx = -1;
      float qop = 0.f, chi2 = 0.f;
      if (best != kNoKey) {
        nh = 4 - (int)(best >> 56);
        chi2 = __uint_as_float((uint32_t)(best >> 24));
        const uint32_t pp[4] = {(uint32_t)(best >> 18) & 63u, (uint32_t)(best >> 12) & 63u,
                                (uint32_t)(best >> 6) & 63u, (uint32_t)best & 63u};
        float d[4], z[4], w[4];
        bool pr[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          pr[k] = pp[k] != 63u;
          d[k] = z[k] = w[k] = 0.f;
          if (pr[k]) {
            const uint32_t hh = lf[k] + cv.h[pp[k] * cv.slots + qslot + k];
            d[k] = cv.d[pp[k] * cv.slots + qslot + k]; z[k] = Z[hh]; w[k] = W[hh];
            if (k == l) hidx = (int)(a0 + hh);
          }
        }
        const FitResult r = fit_tracklet(pr[0], d[0], z[0], w[0], pr[1], d[1], z[1], w[1], pr[2], d[2], z[2], w[2],
                                         pr[3], d[3], z[3], w[3], nh, a.c);
        qop = __fdiv_rn(r.b, a.c.kappa);
      }
      a.out_idx[(size_t)l * T + tg] = hidx;
      if (l == 0) { a.out_n[tg] = nh; a.out_qop[tg] = qop; a.out_chi2[tg] = chi2; }
    }
    __syncwarp();
  }
}

__global__ void __launch_bounds__(512) compass_kernel(const CompassArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, nt = blockDim.x;
  const uint32_t ng = a.n_groups;
  Carver cvr(smem_raw);
  float* s_x = cvr.take<float>(a.hit_stage);
  float* s_yb = cvr.take<float>(a.hit_stage);
  float* s_ye = cvr.take<float>(a.hit_stage);
  float* s_z = cvr.take<float>(a.hit_stage);
  float* s_w = cvr.take<float>(a.hit_stage);
  CandView cv;
  cv.slots = (uint32_t)nt;
  cv.d = cvr.take<float>((size_t)a.c.max_candidates_per_layer * nt);
  cv.h = cvr.take<uint16_t>((size_t)a.c.max_candidates_per_layer * nt);
  uint32_t* s_goff = cvr.take<uint32_t>(ng + 1);
  float* s_gdxdy = cvr.take<float>(ng);
  float* s_gxmin = cvr.take<float>(ng);
  float* s_gxmax = cvr.take<float>(ng);

  const int e = blockIdx.x;
  const uint32_t T = __ldg(a.velo_offsets + a.n_events);
  const uint32_t t0 = __ldg(a.velo_offsets + e), t1 = __ldg(a.velo_offsets + e + 1);
  const uint32_t* go = a.hit_offsets + (size_t)e * ng;
  const uint32_t h0 = __ldg(go), h1 = __ldg(go + ng);
  if (t1 < t0 || t1 > T) {                         // inconsistent VELO offsets: nothing can be written safely
    if (tid == 0) atomicOr(a.status, (uint32_t)UT_STATUS_BAD_OFFSETS);
    return;
  }
  const uint32_t a0 = h0 & ~3u;                    // staged arrays start at a 16-byte aligned element
  bool bad = h1 < h0;
  for (uint32_t g = tid; g <= ng; g += nt) {
    const uint32_t o = __ldg(go + g);
    s_goff[g] = o - a0;
    if (g < ng) {
      const uint32_t o1 = __ldg(go + g + 1);
      bad |= o1 < o;
      s_gdxdy[g] = (o1 > o) ? __ldg(a.hdxdy + o) : 0.f;
      s_gxmin[g] = __ldg(a.group_xmin + g);
      s_gxmax[g] = __ldg(a.group_xmax + g);
    }
  }
  uint32_t too_large = 0;
  if (tid < 4 && !bad) too_large = (__ldg(go + (tid + 1) * a.gpl) - __ldg(go + tid * a.gpl)) > 65535u;
  const int flag = __syncthreads_or((bad ? 1 : 0) | (too_large ? 2 : 0));
  if (flag) {                                      // uniform: report and emit "no tracklet" for every track
    if (tid == 0) atomicOr(a.status, (flag & 1 ? (uint32_t)UT_STATUS_BAD_OFFSETS : 0u) |
                                         (flag & 2 ? (uint32_t)UT_STATUS_EVENT_TOO_LARGE : 0u));
    for (uint32_t t = t0 + tid; t < t1; t += nt) {
      for (int k = 0; k < 4; ++k) a.out_idx[(size_t)k * T + t] = -1;
      a.out_n[t] = 0; a.out_qop[t] = 0.f; a.out_chi2[t] = 0.f;
    }
    return;
  }
  const uint32_t n_al = h1 - a0;
  if (n_al <= a.hit_stage) {
    for (uint32_t i = tid; i < n_al; i += nt) {
      s_x[i] = __ldg(a.hx + a0 + i); s_yb[i] = __ldg(a.hyb + a0 + i); s_ye[i] = __ldg(a.hye + a0 + i);
      s_z[i] = __ldg(a.hz + a0 + i); s_w[i] = __ldg(a.hw + a0 + i);
    }
    __syncthreads();
    track_loop<true>(a, s_x, s_yb, s_ye, s_z, s_w, s_goff, s_gdxdy, s_gxmin, s_gxmax, cv, a0, t0, t1, T);
  } else {                                         // event larger than the staging size: same code on global memory
    track_loop<false>(a, a.hx + a0, a.hyb + a0, a.hye + a0, a.hz + a0, a.hw + a0, s_goff, s_gdxdy, s_gxmin, s_gxmax,
                      cv, a0, t0, t1, T);
  }
}

static int env_int(const char* name, int dflt) {
  const char* v = getenv(name);
  return v && *v ? atoi(v) : dflt;
}

static size_t compass_smem_bytes(uint32_t ng, uint32_t hit_stage, int C, int block) {
  size_t b = 5 * align16((size_t)hit_stage * 4);
  b += align16((size_t)C * block * 4) + align16((size_t)C * block * 2);
  b += align16((ng + 1) * 4) + 3 * align16(ng * 4);
  return b;
}

int32_t launch_compass(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                       const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, ut_tracks* out,
                       cudaStream_t stream) {
  static int max_smem = 0;               // largest dynamic size this kernel may ask for
  if (!max_smem) {
    int dev = 0, optin = 0;
    UTC_CUDA(cudaGetDevice(&dev));
    UTC_CUDA(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    cudaFuncAttributes fa;
    UTC_CUDA(cudaFuncGetAttributes(&fa, compass_kernel));
    const int dyn = optin - (int)fa.sharedSizeBytes;
    UTC_CUDA(cudaFuncSetAttribute(compass_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn));
    max_smem = dyn;
  }
  const ut_geometry* geom = hits->geom;
  CompassArgs a;
  a.hx = hits->x_at_y0; a.hz = hits->z_at_y0; a.hyb = hits->y_begin; a.hye = hits->y_end; a.hdxdy = hits->dxdy;
  a.hw = hits->weight; a.hit_offsets = hit_offsets;
  a.vx = velo->x; a.vy = velo->y; a.vtx = velo->tx; a.vty = velo->ty; a.vz = velo->z;
  a.velo_offsets = velo_offsets; a.n_events = n_events;
  a.n_groups = geom->n_groups; a.gpl = geom->n_groups / UT_N_LAYERS;
  a.group_xmin = geom->group_xmin; a.group_xmax = geom->group_xmax;
  for (int l = 0; l < 4; ++l) { a.layer_z[l] = geom->layer_z[l]; a.layer_dxdy[l] = geom->layer_dxdy[l]; }
  a.c = *cfg;
  a.out_idx = out->hit_idx; a.out_n = out->n_hits; a.out_qop = out->qop; a.out_chi2 = out->chi2; a.status = out->status;

  int block = env_int("UT_COMPASS_BLOCK", 256);
  block = std::max(32, std::min(512, (block / 32) * 32));
  const unsigned long long avg = hits->capacity / (unsigned long long)n_events + 1;
  uint32_t hit_stage = (uint32_t)std::min<unsigned long long>(((avg + 127) / 128) * 128 + 128, 1u << 16);
  hit_stage = (uint32_t)env_int("UT_COMPASS_HIT_STAGE", (int)hit_stage);
  const size_t budget = (size_t)max_smem;
  size_t smem = compass_smem_bytes(geom->n_groups, hit_stage, cfg->max_candidates_per_layer, block);
  while (smem > budget && block > 128) {            // fewer tracks in flight before giving up staging
    block -= 64;
    smem = compass_smem_bytes(geom->n_groups, hit_stage, cfg->max_candidates_per_layer, block);
  }
  while (smem > budget && hit_stage > 0) {
    hit_stage = hit_stage > 1024 ? hit_stage - 1024 : 0;
    smem = compass_smem_bytes(geom->n_groups, hit_stage, cfg->max_candidates_per_layer, block);
  }
  if (smem > budget) return UT_ERR_LIMIT;
  a.hit_stage = hit_stage;
  compass_kernel<<<n_events, block, smem, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  ut_launch_info& li = launch_info();
  li.kernels_launched = 1; li.compass_grid = n_events; li.compass_block = block; li.compass_smem_bytes = (int)smem;
  li.compass_hit_stage = (int)hit_stage;
  return UT_OK;
}

}  // namespace utc
