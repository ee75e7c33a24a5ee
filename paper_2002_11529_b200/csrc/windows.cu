// windows.cu -- the paper's own two-kernel Compass (section V-A / V-B, :286-348), SURVEY.md 8(f) row 2.
//
// Kept beside the fused kernel (compass.cu) as an A/B measurement of the paper's layout claims (PAPER.md:448:
// "+15 % windows SoA"), not as the product path:
//
//   search_windows_kernel   "search UT windows": a two-dimensional kernel, first dimension the
//                           four UT panels, second the VELO tracks of an event; per (track, panel) the sector group
//                           the extrapolation points to and its neighbours (1, 3 or 5 groups: central, -1, +1, -2,
//                           +2), in each two searches on the x-sorted group give the window range, stored as Fig. 7
//                           draws it: per track, per panel, W begin indices then W sizes, signed 16-bit, begin
//                           relative to the event's first hit, (-1, -1) = no hits.  Tracks outside the acceptance
//                           are dropped first through a shared-memory array of valid tracks.
//   tracklets_kernel        "tracklet finding": thread per VELO track, window
//                           ranges cached in shared memory as num_threads x num_panels x 2W shorts,
//                           valid tracks (enough panels with a range) compacted through shared memory; the thread
//                           walks its ranges, repeats the tolerance + y test per hit, keeps the
//                           max_candidates_per_layer closest hits, and runs the seed / compatible-hit / fit /
//                           best-tracklet loops of DESIGN.md section 3 on its own.
//
// Results are those of oracle_search_windows / oracle_compass_from_windows bit for bit; with 5 sector groups they
// equal compass_track's on the synthetic workloads (every group a window can touch is searched).
#include <algorithm>

#include "common.cuh"
#include "compass_fit.cuh"

namespace utc {

constexpr int kWinTracks = 64;         // tracks per block in both kernels (second kernel dimension)
constexpr int kMaxC = UT_MAX_CANDIDATES;

struct WindowArgs {
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
  KickTable kick;
  int32_t W;
  int16_t* windows;            // [T][4][2W]
  unsigned long long capacity;
  uint32_t* status;
  int32_t *out_idx, *out_n;
  float *out_qop, *out_chi2;
};

__device__ __forceinline__ int slot_group(int l, int gpl, int central, int k) {     // 0, -1, +1, -2, +2
  const int off = k == 0 ? 0 : ((k & 1) ? -((k + 1) >> 1) : (k >> 1));
  const int gi = central + off;
  return (gi < l * gpl || gi >= (l + 1) * gpl) ? -1 : gi;
}

__device__ __forceinline__ float resid_at(const float* X, uint32_t h, float syg, float x_e) {
  return __fsub_rn(__fadd_rn(__ldg(X + h), syg), x_e);
}

// ---- kernel 1: search UT windows --------------------------------------------------------------
__global__ void __launch_bounds__(4 * kWinTracks) search_windows_kernel(const WindowArgs a) {
  __shared__ float s_xmax[UT_MAX_GROUPS], s_xmin[UT_MAX_GROUPS];
  __shared__ uint32_t s_goff[UT_MAX_GROUPS + 1];
  __shared__ uint32_t s_valid[kWinTracks];                  // the array of valid tracks
  __shared__ uint32_t s_nvalid;
  const int l = threadIdx.x, ty = threadIdx.y, tid = ty * 4 + l, nt = 4 * kWinTracks;
  const int e = blockIdx.x, W = a.W, gpl = (int)a.gpl;
  const uint32_t ng = a.n_groups;
  for (uint32_t g = tid; g < ng; g += nt) { s_xmax[g] = __ldg(a.group_xmax + g); s_xmin[g] = __ldg(a.group_xmin + g); }
  const uint32_t* go = a.hit_offsets + (size_t)e * ng;
  for (uint32_t g = tid; g <= ng; g += nt) s_goff[g] = __ldg(go + g);
  __syncthreads();
  const uint32_t h0 = s_goff[0], h1 = s_goff[ng];
  const uint32_t t0 = __ldg(a.velo_offsets + e), t1 = __ldg(a.velo_offsets + e + 1);
  // an event that shorts cannot index, or that the decode did not write: every range empty, status says why
  const bool unusable = h1 < h0 || h1 - h0 > 32767u || (unsigned long long)h1 > a.capacity;
  if (unusable && tid == 0 && t1 > t0)
    atomicOr(a.status, h1 < h0 ? (uint32_t)UT_STATUS_BAD_OFFSETS
                               : ((unsigned long long)h1 > a.capacity ? (uint32_t)UT_STATUS_CAPACITY : (uint32_t)UT_STATUS_EVENT_TOO_LARGE));
  const float zl = a.layer_z[l], sl = a.layer_dxdy[l], D = a.c.win_half[l];
  const float lay_lo = s_xmin[l * gpl], lay_hi = s_xmax[l * gpl + gpl - 1];
  for (uint32_t tb = t0; tb < t1; tb += kWinTracks) {
    // ---- valid-track array: tracks whose window meets the panel in at least one layer ------------------------
    if (tid == 0) s_nvalid = 0;
    __syncthreads();
    const uint32_t t = tb + ty;
    bool hit_layer = false;
    if (t < t1 && !unusable) {
      const float dzv = __fsub_rn(zl, a.vz);
      const float x_e = __fadd_rn(__ldg(a.vx + t), __fmul_rn(__ldg(a.vtx + t), dzv));
      const float y_e = __fadd_rn(__ldg(a.vy + t), __fmul_rn(__ldg(a.vty + t), dzv));
      const float c = __fsub_rn(x_e, __fmul_rn(sl, y_e));
      hit_layer = c + D + 0.01f >= lay_lo && c - D - 0.01f <= lay_hi;     // (slack >> fp32 rounding; NaN: dropped)
    }
    // the 4 panel threads of a track are 4 consecutive lanes
    const unsigned m4 = __ballot_sync(0xFFFFFFFFu, hit_layer) >> ((tid & 31) & ~3) & 0xFu;
    if (t < t1) {
      if (m4 != 0 && l == 0) s_valid[atomicAdd(&s_nvalid, 1u)] = t;
      if (m4 == 0) {                                           // outside every panel: empty ranges, written here
        int16_t* w = a.windows + ((size_t)t * 4 + l) * 2 * W;
        for (int k = 0; k < 2 * W; ++k) w[k] = -1;
      }
    }
    __syncthreads();
    // ---- the window search proper, parallel over (panel, valid track) -----------------------------------------
    if ((uint32_t)ty < s_nvalid) {
      const uint32_t tv = s_valid[ty];
      const float dzv = __fsub_rn(zl, a.vz);
      const float x_e = __fadd_rn(__ldg(a.vx + tv), __fmul_rn(__ldg(a.vtx + tv), dzv));
      const float y_e = __fadd_rn(__ldg(a.vy + tv), __fmul_rn(__ldg(a.vty + tv), dzv));
      const float syg = __fmul_rn(sl, y_e);
      const float c = __fsub_rn(x_e, syg);
      // the region the extrapolation points to: binary search over the groups of the panel
      int lo = 0, n = gpl;
      while (n > 0) {
        const int half = n >> 1;
        if (s_xmax[l * gpl + lo + half] >= c) n = half; else { lo += half + 1; n -= half + 1; }
      }
      const int central = l * gpl + min(lo, gpl - 1);
      int16_t* w = a.windows + ((size_t)tv * 4 + l) * 2 * W;
      for (int k = 0; k < W; ++k) {
        const int gi = slot_group(l, gpl, central, k);
        int16_t begin = -1, size = -1;
        if (gi >= 0) {
          uint32_t first = s_goff[gi];
          for (uint32_t cnt = s_goff[gi + 1] - first; cnt > 0;) {          // first hit with d >= -D
            const uint32_t half = cnt >> 1, mid = first + half;
            if (resid_at(a.hx, mid, syg, x_e) >= -D) cnt = half; else { first = mid + 1; cnt -= half + 1; }
          }
          uint32_t last = first;
          for (uint32_t cnt = s_goff[gi + 1] - last; cnt > 0;) {           // first hit with d > D
            const uint32_t half = cnt >> 1, mid = last + half;
            if (resid_at(a.hx, mid, syg, x_e) > D) cnt = half; else { last = mid + 1; cnt -= half + 1; }
          }
          if (last > first) { begin = (int16_t)(first - h0); size = (int16_t)(last - first); }
        }
        w[k] = begin;
        w[W + k] = size;
      }
    }
    __syncthreads();
  }
}

// ---- kernel 2: tracklet finding, thread per track ----------------------------------------------
struct LocalCand {            // per-thread candidate lists (local memory; the paper iterates its ranges in place)
  float d[4][kMaxC], z[4][kMaxC], w[4][kMaxC];
  int h[4][kMaxC];
  int n[4];
};

struct BestT { int n; float chi2; int h[4]; bool valid; };

__device__ __forceinline__ bool better_t(int n, float chi2, const int (&h)[4], const BestT& b) {
  if (n != b.n) return n > b.n;
  if (chi2 != b.chi2) return chi2 < b.chi2;
#pragma unroll
  for (int l = 0; l < 4; ++l) {
    const int x = h[l] < 0 ? 0x7FFFFFFF : h[l], y = b.h[l] < 0 ? 0x7FFFFFFF : b.h[l];
    if (x != y) return x < y;
  }
  return false;
}

__device__ void search_direction_t(const WindowArgs& a, const LocalCand& L, float z_mag, int LA, int LB, int LC, int LD,
                                   BestT& best) {
  const compass_config& c = a.c;
  for (int ia = 0; ia < L.n[LA]; ++ia) {
    for (int ib = 0; ib < L.n[LB]; ++ib) {
      const float da = L.d[LA][ia], za = L.z[LA][ia];
      const float bs = __fdiv_rn(__fsub_rn(L.d[LB][ib], da), __fsub_rn(L.z[LB][ib], za));
      const float a0 = __fsub_rn(da, __fmul_rn(bs, __fsub_rn(za, z_mag)));
      if (!(fabsf(bs) <= c.max_slope && fabsf(a0) <= c.kink_tol)) continue;
      uint32_t mC = 0, mD = 0;
      for (int i = 0; i < L.n[LC]; ++i)
        if (fabsf(__fsub_rn(L.d[LC][i], __fadd_rn(da, __fmul_rn(bs, __fsub_rn(L.z[LC][i], za))))) <= c.seed_tol) mC |= 1u << i;
      for (int i = 0; i < L.n[LD]; ++i)
        if (fabsf(__fsub_rn(L.d[LD][i], __fadd_rn(da, __fmul_rn(bs, __fsub_rn(L.z[LD][i], za))))) <= c.seed_tol) mD |= 1u << i;
      // (c or none) x (d or none) with >= min_hits hits in total
      int ic = -1;
      for (uint32_t rc = mC;; ic = __ffs(rc) - 1, rc &= rc - 1) {          // none, then every compatible hit of C
        int id = -1;
        for (uint32_t rd = mD;; id = __ffs(rd) - 1, rd &= rd - 1) {        // none, then every compatible hit of D
          const int nh = 2 + (ic >= 0) + (id >= 0);
          if (nh >= c.min_hits) {
          int pos[4];
          pos[LA] = ia; pos[LB] = ib; pos[LC] = ic; pos[LD] = id;
          bool pr[4];
          float d[4], z[4], w[4];
          int h[4];
#pragma unroll
          for (int l = 0; l < 4; ++l) {
            pr[l] = pos[l] >= 0;
            const int q = pr[l] ? pos[l] : 0;
            d[l] = pr[l] ? L.d[l][q] : 0.f; z[l] = pr[l] ? L.z[l][q] : 0.f; w[l] = pr[l] ? L.w[l][q] : 0.f;
            h[l] = pr[l] ? L.h[l][q] : -1;
          }
          const FitResult fr = fit_tracklet(pr, d, z, w, nh, c, z_mag);
          if (fr.valid && (!best.valid || better_t(nh, fr.chi2, h, best))) {
            best.valid = true; best.n = nh; best.chi2 = fr.chi2;
#pragma unroll
            for (int l = 0; l < 4; ++l) best.h[l] = h[l];
          }
          }
          if (!rd) break;
        }
        if (!rc) break;
      }
    }
  }
}

__global__ void __launch_bounds__(kWinTracks) tracklets_kernel(const WindowArgs a) {
  extern __shared__ __align__(16) int16_t s_win[];          // [kWinTracks][4][2W]: the window-range cache
  __shared__ uint32_t s_valid[kWinTracks];
  __shared__ uint32_t s_nvalid;
  const int tid = threadIdx.x, e = blockIdx.x, W = a.W, rowlen = 4 * 2 * W;
  const uint32_t t0 = __ldg(a.velo_offsets + e), t1 = __ldg(a.velo_offsets + e + 1);
  const uint32_t T = __ldg(a.velo_offsets + a.n_events);
  const uint32_t h0 = __ldg(a.hit_offsets + (size_t)e * a.n_groups);
  const compass_config& c = a.c;
  for (uint32_t tb = t0; tb < t1; tb += kWinTracks) {
    const uint32_t nchunk = min((uint32_t)kWinTracks, t1 - tb);
    if (tid == 0) s_nvalid = 0;
    // the chunk's window ranges, contiguous in global memory -> shared memory
    for (uint32_t i = tid; i < nchunk * rowlen; i += kWinTracks) s_win[i] = a.windows[(size_t)tb * rowlen + i];
    __syncthreads();
    // valid tracks: enough panels with a range ("at least one valid window range"; fewer than min_hits
    // panels with a range cannot give a tracklet) -> compacted; the others get "no tracklet" right away
    if ((uint32_t)tid < nchunk) {
      const int16_t* w = s_win + tid * rowlen;
      int panels = 0;
      for (int l = 0; l < 4; ++l) {
        bool any = false;
        for (int k = 0; k < W; ++k) any |= w[l * 2 * W + W + k] > 0;
        panels += any;
      }
      const uint32_t t = tb + tid;
      if (panels >= c.min_hits) s_valid[atomicAdd(&s_nvalid, 1u)] = (uint32_t)tid;
      else {
        for (int l = 0; l < 4; ++l) a.out_idx[(size_t)l * T + t] = -1;
        a.out_n[t] = 0; a.out_qop[t] = 0.f; a.out_chi2[t] = 0.f;
      }
    }
    __syncthreads();
    if ((uint32_t)tid < s_nvalid) {
      const uint32_t ti = s_valid[tid], t = tb + ti;
      const int16_t* w = s_win + ti * rowlen;
      LocalCand L;
      int nonempty = 0;
      const float vx = __ldg(a.vx + t), vy = __ldg(a.vy + t), vtx = __ldg(a.vtx + t), vty = __ldg(a.vty + t);
      for (int l = 0; l < 4; ++l) {
        const float dzv = __fsub_rn(a.layer_z[l], a.vz);
        const float x_e = __fadd_rn(vx, __fmul_rn(vtx, dzv));
        const float y_e = __fadd_rn(vy, __fmul_rn(vty, dzv));
        const float D = c.win_half[l];
        const int C = c.max_candidates_per_layer;
        int n = 0;
        int prev = -1;
        for (int pass = 0; pass < W; ++pass) {               // the ranges in ascending hit order (= ascending group)
          int k = -1, kb = 0x7FFFFFFF;
          for (int q = 0; q < W; ++q) {
            const int b = w[l * 2 * W + q];
            if (w[l * 2 * W + W + q] > 0 && b > prev && b < kb) { kb = b; k = q; }
          }
          if (k < 0) break;
          prev = kb;
          const uint32_t hb = h0 + (uint32_t)kb, he = hb + (uint32_t)w[l * 2 * W + W + k];
          for (uint32_t h = hb; h < he; ++h) {
            // the tolerance test again, and the y test that the unsorted sector group needs
            const float d = __fsub_rn(__fadd_rn(__ldg(a.hx + h), __fmul_rn(__ldg(a.hdxdy + h), y_e)), x_e);
            if (!(fabsf(d) <= D)) continue;
            if (!(__fsub_rn(__ldg(a.hyb + h), c.y_tol) <= y_e && y_e <= __fadd_rn(__ldg(a.hye + h), c.y_tol))) continue;
            if (n == C) {                                     // keep the C closest in (|d|, h)
              int worst = 0;
              for (int i = 1; i < C; ++i)
                if (fabsf(L.d[l][i]) > fabsf(L.d[l][worst]) ||
                    (fabsf(L.d[l][i]) == fabsf(L.d[l][worst]) && L.h[l][i] > L.h[l][worst])) worst = i;
              if (!(fabsf(d) < fabsf(L.d[l][worst]))) continue;                // (h is larger than every kept index)
              for (int i = worst; i < C - 1; ++i) {
                L.d[l][i] = L.d[l][i + 1]; L.z[l][i] = L.z[l][i + 1]; L.w[l][i] = L.w[l][i + 1]; L.h[l][i] = L.h[l][i + 1];
              }
              n = C - 1;
            }
            L.d[l][n] = d; L.z[l][n] = __ldg(a.hz + h); L.w[l][n] = __ldg(a.hw + h); L.h[l][n] = (int)h;
            ++n;
          }
        }
        L.n[l] = n;
        nonempty += n > 0;
      }
      BestT best;
      best.valid = false; best.n = 0; best.chi2 = 0.f;
      for (int l = 0; l < 4; ++l) best.h[l] = -1;
      float kappa, z_mag;                                     // the track's kick (table cell or the config's constants)
      track_kick(a.kick, c, vx, vy, vtx, vty, a.vz, kappa, z_mag);
      if (nonempty >= c.min_hits) {
        search_direction_t(a, L, z_mag, 0, 2, 1, 3, best);                    // forward seeds (L0, L2)
        if (c.both_directions || !best.valid) search_direction_t(a, L, z_mag, 3, 1, 2, 0, best);   // backward (L3, L1)
      }
      float qop = 0.f;
      if (best.valid) {                                       // q/p of the winner: its fit again (step 6)
        bool pr[4];
        float d[4], z[4], wv[4];
        for (int l = 0; l < 4; ++l) {
          pr[l] = best.h[l] >= 0;
          d[l] = z[l] = wv[l] = 0.f;
          if (pr[l])
            for (int i = 0; i < L.n[l]; ++i)
              if (L.h[l][i] == best.h[l]) { d[l] = L.d[l][i]; z[l] = L.z[l][i]; wv[l] = L.w[l][i]; }
        }
        qop = __fdiv_rn(fit_tracklet(pr, d, z, wv, best.n, c, z_mag).b, kappa);
      }
      for (int l = 0; l < 4; ++l) a.out_idx[(size_t)l * T + t] = best.valid ? best.h[l] : -1;
      a.out_n[t] = best.valid ? best.n : 0;
      a.out_qop[t] = qop;
      a.out_chi2[t] = best.valid ? best.chi2 : 0.f;
    }
    __syncthreads();
  }
}

static void fill_args(WindowArgs& a, const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                      const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, int32_t W) {
  const ut_geometry* geom = hits->geom;
  a.hx = hits->x_at_y0; a.hz = hits->z_at_y0; a.hyb = hits->y_begin; a.hye = hits->y_end; a.hdxdy = hits->dxdy;
  a.hw = hits->weight; a.hit_offsets = hit_offsets;
  a.vx = velo->x; a.vy = velo->y; a.vtx = velo->tx; a.vty = velo->ty; a.vz = velo->z;
  a.velo_offsets = velo_offsets; a.n_events = n_events;
  a.n_groups = geom->n_groups; a.gpl = geom->n_groups / UT_N_LAYERS;
  a.group_xmin = geom->group_xmin; a.group_xmax = geom->group_xmax;
  for (int l = 0; l < 4; ++l) { a.layer_z[l] = geom->layer_z[l]; a.layer_dxdy[l] = geom->layer_dxdy[l]; }
  a.c = *cfg; a.kick = make_kick_table(geom); a.W = W; a.capacity = hits->capacity;
  a.windows = nullptr; a.status = nullptr; a.out_idx = nullptr; a.out_n = nullptr; a.out_qop = nullptr; a.out_chi2 = nullptr;
}

int32_t launch_search_windows(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                              const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, int32_t W,
                              int16_t* windows, uint32_t* status, cudaStream_t stream) {
  WindowArgs a;
  fill_args(a, hits, hit_offsets, velo, velo_offsets, n_events, cfg, W);
  a.windows = windows; a.status = status;
  search_windows_kernel<<<n_events, dim3(4, kWinTracks), 0, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  launch_info().kernels_launched = 1;
  return UT_OK;
}

int32_t launch_tracklets(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                         const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, int32_t W,
                         const int16_t* windows, ut_tracks* out, cudaStream_t stream) {
  WindowArgs a;
  fill_args(a, hits, hit_offsets, velo, velo_offsets, n_events, cfg, W);
  a.windows = const_cast<int16_t*>(windows); a.status = out->status;
  a.out_idx = out->hit_idx; a.out_n = out->n_hits; a.out_qop = out->qop; a.out_chi2 = out->chi2;
  const size_t smem = (size_t)kWinTracks * 4 * 2 * W * sizeof(int16_t);
  tracklets_kernel<<<n_events, kWinTracks, smem, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  launch_info().kernels_launched = 1;
  return UT_OK;
}

}  // namespace utc
