// compass.cu -- Compass tracking (section V, :276-348) as ONE fused kernel.
//
// The paper runs two kernels: "search UT windows" (2-D: 4 panels x tracks) writes
// (first hit, size) ranges to global memory, then "tracklet finding" (thread per track)
// reads them back through a shared-memory cache.  That shape leaves a B200 warp at
// 7 of 32 lanes (profiles/r1a_first_path.md).  Here a CTA takes one work item = (event, part k of K) by an
// atomic ticket and keeps the event on chip (K = 1, 2 or 4 CTAs share the tracks of an event: track i belongs
// to part i mod K; K > 1 only for batches of fewer events than resident CTAs):
//
//   stage    the event's window-search data is its per-sector view: x and the container index bucketed per
//            dense sector plus the sector offsets.  When ut_decode wrote the view (ut_hits.x_by_sector ...) it
//            arrives by three TMA bulk copies and no thread touches it; otherwise a warp per sector group
//            re-buckets the group-sorted arrays in shared memory (match.any ranks, per-sector counts, warp
//            scan).  A sector's y range, stereo slope, z and weight are rows of the geometry table, so the y
//            test of the window search is a per-sector test: the scan touches the hits of the one sector row
//            the track crosses instead of all rows of the column.
//   order    the tracks of the item are binned by their radius at the first layer (counting sort over
//            logarithmic bins, O(n)): a batch costs what its heaviest track costs and the inner tracks cross
//            the busy sectors, so like goes with like and the heavy batches start first.  Results do not
//            depend on the order.
//   phase 1  lane = (track, layer), 8 tracks per warp (the paper's 2-D window kernel shape):
//            straight-line extrapolation, column groups and sector row from a linear guess corrected against
//            the tables (y ranges from L1), lower-bound search in busy sectors, |d| <= win test with early exit;
//            accepted hits go to the (track, layer) candidate list in shared memory, kept sorted by hit index
//            and capped to the `max_candidates_per_layer` closest in |d| (a run longer than the cap starts at
//            the zero crossing minus the cap and ends at the first hit the full list rejects).
//   phase 2  the nested loops of the tracklet search are spread over the 32 lanes of the warp:
//            (a) seed rows (track, hit a) of the 8 tracks, one row per lane walking the partner hits b with a
//                cheap conservative filter of the slope + kink cuts (reciprocal instead of the division, a
//                margin of 2e-6 relative: it never drops a pair the exact cuts keep); survivors are compacted
//                (ballot) into a per-warp seed queue;
//            (b) the queued seeds, 4 lanes per seed: the exact slope and kink cuts in the order of DESIGN.md
//                section 3, then the compatible hits in the other two layers as 32-bit masks, giving the
//                number of 3/4-hit combinations of the seed;
//            (c) all combinations of those seeds, one fit per lane (linear chi2 fit with the VELO pseudo-point),
//                packed (n, chi2, positions) key, atomicMin into the track's best key.
//            Forward seeds first, backward only for tracks where forward found nothing valid (A11), or both
//            directions for every track (compass_config.both_directions).
//            When every candidate list of the batch has one z and one weight (always in a layer-uniform
//            geometry) those come from two per-slot words instead of a table look-up per candidate.
//   Candidate lists, queues and best keys never leave the SM; the phases of a warp are separated by
//   __syncwarp only, and the warps of a CTA pull 8-track batches from a shared-memory ticket.
//
// Events that do not fit the staging buffer take the same phases with a group-level binary search on the
// global x-sorted arrays (the plain definition of the window, per-hit y test).
// fp32 arithmetic uses __f*_rn intrinsics in the order of DESIGN.md section 3 (bit-exact, no FMA).
#include <algorithm>
#include <cstdio>
#include <cstdlib>

#include "common.cuh"
#include "compass_fit.cuh"

namespace utc {

constexpr float kGroupEps = 0.01f;     // slack of the group pre-selection [mm] (A17)
constexpr unsigned long long kNoKey = ~0ull;
constexpr int kTPW = 8;                // tracks per warp batch (x 4 layers = 32 lanes)
constexpr int kSeedQ = 64;             // per-warp seed ring (<= 31 left over + <= 32 new)
constexpr int kBins = 128;             // radius bins of the batch order
constexpr float kFilterEps = 2e-6f;    // relative margin of the seed pre-filter (>= 16 roundings of 6e-8)

struct CompassArgs {
  const float* hx;
  const uint32_t* hid;
  const float *hyb, *hye;              // per-hit y range: only the global (unstaged) path reads them
  const uint32_t* hit_offsets;
  const float* sx;                     // per-sector view written by ut_decode (or null)
  const uint16_t* si;
  const uint16_t* soff;
  uint32_t soff_stride;
  const float *vx, *vy, *vtx, *vty;
  float vz;
  const uint32_t* velo_offsets;
  int32_t n_events;
  uint32_t n_sectors, n_groups, gpl, id_table_size, rows_sorted;
  uint32_t rows_uniform;               // rows per group when every group of a layer has the same y rows, else 0
  uint32_t order_y;                    // the container's groups are in (y_begin, x) order (UT_ORDER_Y), not x order
  const uint32_t *id_to_sector, *group_first_sector;
  const float *group_xmin, *group_xmax, *sec_yb, *sec_ye, *sec_dxdy, *sec_z, *sec_w;
  float layer_z[4], layer_dxdy[4];
  float layer_w[4];                    // UT_GEOM_LAYER_UNIFORM: the one weight of the layer's sectors (LU kernels)
  compass_config c;
  int32_t *out_idx, *out_n;
  float *out_qop, *out_chi2;
  uint32_t* status;                    // [0] status word
  uint32_t* ticket;                    // [0] next work item, [1] CTAs done (one pair per launch that may run at a time)
  uint32_t hit_stage;                  // elements of the staged (bucketed) arrays
  uint32_t trk_stage;                  // tracks of an item that can be ordered by radius (0: never)
  uint32_t ev_stage;                   // events of a batch that can be handed out heaviest first (0: never)
  unsigned long long capacity;         // elements of the hit arrays (bulk copies never read past it)
  uint32_t bulk_ok;                    // hit arrays are 16-byte aligned: the event's x and id ranges come by TMA
  uint32_t idx_stride;                 // row stride of out_idx (0: velo_offsets[n_events])
  uint32_t split;                      // K: CTAs sharing the tracks of one event
  KickTable kick;                      // optional per-track kappa / z_mag (kick.nx == 0: the config's constants)
  float slope_lim;                     // max_slope * (1 + kFilterEps): pre-filter limit
  int32_t interval_min;                // seed partner lists longer than this are searched, not walked
};

// (n desc, chi2 asc, hit tuple asc): candidate positions are ascending in hit index, none = 63
__device__ __forceinline__ unsigned long long make_key(int n, float chi2, uint32_t p0, uint32_t p1, uint32_t p2,
                                                       uint32_t p3) {
  return ((unsigned long long)(4 - n) << 56) | ((unsigned long long)__float_as_uint(chi2) << 24) |
         (unsigned long long)((p0 << 18) | (p1 << 12) | (p2 << 6) | p3);
}

__device__ __forceinline__ float rcp_approx(float x) {
  float r;
  asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// n / d for the small counts of the combination index (n < 2^16, d <= 64): (n + 0.5) / d is at least 0.5 / d away from
// an integer, far more than the error of the approximate reciprocal, so the truncation is the exact quotient -- five
// instructions instead of the ~20 of an integer division.
__device__ __forceinline__ uint32_t small_div(uint32_t n, uint32_t d) {
  return (uint32_t)(((float)n + 0.5f) * rcp_approx((float)d));
}

// Per-warp working set in shared memory.  Candidate i of lane-slot s (= track-in-batch * 4 + layer) lives at
// [s * CS + i] with CS odd: the rows (track, hit) and the 4 lanes of a seed in phase 2 read consecutive banks.
struct WarpArea {
  float* cd;                   // [32 * CS] residual d of the candidate
  uint32_t* chs;               // [32 * CS] (hit index relative to the event) << 16 | dense sector
  uint32_t* seedq;             // [kSeedQ] track << 10 | ia << 5 | ib
  unsigned long long* best;    // [kTPW]
  int* n;                      // [32] candidates per slot
  float* zs;                   // [32] z of the slot's candidates when they all share one
  float* ws;                   // [32] weight, likewise
  float* tzm;                  // [kTPW] kick plane z_mag of the track
  float* tkap;                 // [kTPW] kick strength kappa of the track
  int* srt;                    // [32] 1: the slot's residuals ascend with the position (kernels with INTERVAL only)
  int CS;
};

__host__ __device__ inline int cand_stride(int C) { return C | 1; }
// CC: max_candidates_per_layer as a compile-time constant (0: the run-time value): strides and caps fold into the code;
// kernels with CC are for row-uniform geometries (UT_GEOM_ROWS_UNIFORM), whose per-sector y search they leave out
template <int CC>
__device__ __forceinline__ int stride_of(const WarpArea& wa) { return CC ? (CC | 1) : wa.CS; }
// (zs / ws exist in the kernels that are not for layer-uniform geometries, srt in those with the interval search, tzm / tkap
//  in those with a kick table: at 4 CTAs per SM every byte of the 7 warp areas counts)
__host__ __device__ inline size_t warp_area_bytes(int C, bool lu, bool interval, bool kick) {
  return (size_t)cand_stride(C) * 32 * 8 + kSeedQ * 4 + kTPW * 8 + 32 * 4 + (lu ? 0 : 32 * 4 * 2) + (interval ? 32 * 4 : 0) +
         (kick ? kTPW * 4 * 2 : 0);
}

// Sorted insert by hit index with the cap rule of step 3: keep the C smallest in (|d|, h).
// Returns false when the list is full and the new hit is not closer than its worst entry.
template <int CC>
__device__ __forceinline__ bool cand_insert(const WarpArea& wa, int slot, int& n, int C, float d, uint32_t hs) {
  float* cd = wa.cd + slot * stride_of<CC>(wa);
  uint32_t* chs = wa.chs + slot * stride_of<CC>(wa);
  if (n == C) {
    int worst = 0;
    float wabs = fabsf(cd[0]);
    uint32_t whs = chs[0];
    // In the kernels with a compile-time cap the compiler would unroll these loops C times; full lists are rare at
    // their settings and the kernel's code size matters more (config 3: 109.0 -> 106.2 us), so they stay rolled there.
    // The general kernels serve the long lists of C = 32, where the unrolled loops are the faster ones.
    if (CC != 0) {
#pragma unroll 1
      for (int i = 1; i < C; ++i) {
        const float v = fabsf(cd[i]);
        const uint32_t k = chs[i];
        if (v > wabs || (v == wabs && k > whs)) { wabs = v; whs = k; worst = i; }
      }
    } else {
      for (int i = 1; i < C; ++i) {
        const float v = fabsf(cd[i]);
        const uint32_t k = chs[i];
        if (v > wabs || (v == wabs && k > whs)) { wabs = v; whs = k; worst = i; }
      }
    }
    const float nabs = fabsf(d);
    if (!(nabs < wabs || (nabs == wabs && hs < whs))) return false;
    if (CC != 0) {
#pragma unroll 1
      for (int i = worst; i < C - 1; ++i) { cd[i] = cd[i + 1]; chs[i] = chs[i + 1]; }
    } else {
      for (int i = worst; i < C - 1; ++i) { cd[i] = cd[i + 1]; chs[i] = chs[i + 1]; }
    }
    n = C - 1;
  }
  int i = n;
  while (i > 0) {
    const uint32_t k = chs[i - 1];
    if (k < hs) break;
    chs[i] = k;
    cd[i] = cd[i - 1];
    --i;
  }
  cd[i] = d;
  chs[i] = hs;
  ++n;
  return true;
}

// Shared-memory view of one CTA: geometry tables (staged once per CTA) and the current event's hits.
// (group tables are indexed by g + 2 * layer: the 4 lanes of a track read 4 different bank groups)
struct SmemView {
  const float4* gA;      // [ng + 8]  group: xmin, xmax, dxdy, row-hint base (y_hi of the first sector)
  const uint2* gB;       // [ng + 8]  group: row-hint scale (float bits), first sector | end sector << 16
  const float2* lay;     // [4]   layer: group-hint base (xmax of the first group), scale
  const float2* yr;      // [4][rows] toleranced y range of a row of the layer (rows_uniform geometries)
  const uint32_t* goff;  // [ng + 1] group offsets relative to the event's first hit
  const uint16_t* off;   // [ns + 1] bucketed position of every sector's first hit
  const float* hx;       // x_at_y0, bucketed per sector, x-sorted inside the sector (indexed by `off` positions)
  const uint16_t* hh;    // hit index relative to the event
};

// y range of a sector widened by y_tol (same two roundings wherever it is evaluated)
__device__ __forceinline__ float yr_hi(const CompassArgs& a, int s) {
  return __fadd_rn(__ldg(a.sec_ye + s), a.c.y_tol);
}
__device__ __forceinline__ float2 yr_of(const CompassArgs& a, int s) {
  return make_float2(__fsub_rn(__ldg(a.sec_yb + s), a.c.y_tol), __fadd_rn(__ldg(a.sec_ye + s), a.c.y_tol));
}

// z / weight of the slot's candidates: remembered while they all agree (zu = NaN once they do not)
__device__ __forceinline__ void note_zw(const CompassArgs& a, int s, bool first, float& zu, float& wu) {
  const float z = __ldg(a.sec_z + s), w = __ldg(a.sec_w + s);
  if (first) { zu = z; wu = w; }
  else if (!(z == zu && w == wu)) zu = __int_as_float(0x7FC00000);
}

// ---- phase 1: candidate list of one (track, layer) -------------------------------------
// Group and sector row are found from a linear guess corrected against the tables (exact lower bound of
// the same predicates the oracle's search uses; O(1) on a regular layout, any sorted layout works).
// LU: layer-uniform geometry (UT_GEOM_LAYER_UNIFORM): z and weight of a candidate are its layer's, nothing to note
template <bool BUCKETED, bool LU, int CC>
__device__ __forceinline__ int collect_window(const CompassArgs& a, const WarpArea& wa, const SmemView& S, int slot,
                                              int l, float x_e, float y_e, uint32_t h0, float& zu, float& wu) {
  const int C = CC ? CC : a.c.max_candidates_per_layer;
  float D = a.c.win_half[l];
  asm volatile("" : "+f"(D));                     // keep D in a register: the indexed constant load is not redone per hit
  const float negD = -D;
  const float ctr = __fsub_rn(x_e, __fmul_rn(a.layer_dxdy[l], y_e));
  const float lo = __fsub_rn(__fsub_rn(ctr, D), kGroupEps), hi = __fadd_rn(__fadd_rn(ctr, D), kGroupEps);
  const int g0 = l * (int)a.gpl, g1 = g0 + (int)a.gpl;
  float* cd = wa.cd + slot * stride_of<CC>(wa);
  uint32_t* chs = wa.chs + slot * stride_of<CC>(wa);
  const int pad = 2 * l;                            // bank padding of the group tables
  int g;
  {                                                 // first group with group_xmax >= lo
    const float2 hint = S.lay[l];
    const int guess = (int)ceilf((lo - hint.x) * hint.y);
    g = g0 + max(0, min(guess, (int)a.gpl - 1));
    while (g > g0 && lo <= S.gA[g - 1 + pad].y) --g;
    while (g < g1 && !(lo <= S.gA[g + pad].y)) ++g;
  }
  // rows_uniform: the sector rows the track crosses, once for all groups of the layer (rows r0 .. r0 + nr - 1)
  int r0 = 0, nr = 0;
  if (BUCKETED && (CC || a.rows_uniform)) {       // (CC kernels are chosen for row-uniform geometries only)
    const int R = (int)a.rows_uniform;
    const float2* yr = S.yr + l * R;
    const float4 grp0 = S.gA[g0 + pad];
    const int guess = (int)ceilf((y_e - grp0.w) * __uint_as_float(S.gB[g0 + pad].x));
    r0 = max(0, min(guess, R - 1));
    while (r0 > 0 && y_e <= yr[r0 - 1].y) --r0;     // first row with y_e <= y_end + y_tol
    while (r0 < R && !(y_e <= yr[r0].y)) ++r0;
    while (r0 + nr < R && yr[r0 + nr].x <= y_e) ++nr;
    if (nr == 0) return 0;                          // outside every row of the layer
  }
  int n = 0;
  uint32_t last = 0;
  for (; g < g1; ++g) {
    const float4 grp = S.gA[g + pad];
    if (!(grp.x <= hi)) break;
    const uint32_t ga = S.goff[g], gb = S.goff[g + 1];
    if (ga == gb) continue;
    const float syg = __fmul_rn(grp.z, y_e);        // one stereo angle per group (container contract)
    if (BUCKETED) {
      const uint2 gi = S.gB[g + pad];
      const int sa = (int)(gi.y & 0xFFFFu);
      int s = sa, sb = (int)(gi.y >> 16);
      const bool per_sector_y = CC ? false : a.rows_uniform == 0;
      if (!per_sector_y) {
        s = sa + r0;
        sb = s + nr;
      } else if (a.rows_sorted) {                   // first sector row with y_e <= y_end + y_tol
        const int guess = (int)ceilf((y_e - grp.w) * __uint_as_float(gi.x));
        s = sa + max(0, min(guess, sb - sa - 1));
        while (s > sa && y_e <= yr_hi(a, s - 1)) --s;
        while (s < sb && !(y_e <= yr_hi(a, s))) ++s;
      }
      for (; s < sb; ++s) {
        if (per_sector_y) {
          const float2 yr = yr_of(a, s);
          if (!(yr.x <= y_e)) { if (a.rows_sorted) break; continue; }
          if (!(y_e <= yr.y)) continue;
        }
        uint32_t p1 = S.off[s + 1];
        uint32_t p = S.off[s];
        if (p1 - p > 6u) {                          // busy sector: lower bound of d >= -D
          for (uint32_t cnt = p1 - p; cnt > 0;) {
            const uint32_t half = cnt >> 1, mid = p + half;
            if (__fsub_rn(__fadd_rn(S.hx[mid], syg), x_e) >= negD) cnt = half; else { p = mid + 1; cnt -= half + 1; }
          }
          if (__builtin_expect(n == 0 && p1 - p > (uint32_t)C, 0)) {
            // the slot's first run may overflow the cap by itself: of a run that is sorted in d the C closest in
            // (|d|, index) are a contiguous stretch around the zero crossing.  Find the end of the window, then
            // grow the stretch from the zero crossing one hit at a time (ties go to the left: lower index), and
            // let the scan below append exactly that stretch -- no eviction.
            uint32_t ub = p;
            for (uint32_t cnt = p1 - p; cnt > 0;) {           // first hit with d > D
              const uint32_t half = cnt >> 1, mid = ub + half;
              if (__fsub_rn(__fadd_rn(S.hx[mid], syg), x_e) > D) cnt = half; else { ub = mid + 1; cnt -= half + 1; }
            }
            p1 = ub;
            if (ub - p > (uint32_t)C) {
              uint32_t zc = p;
              for (uint32_t cnt = ub - p; cnt > 0;) {         // first hit with d >= 0
                const uint32_t half = cnt >> 1, mid = zc + half;
                if (__fsub_rn(__fadd_rn(S.hx[mid], syg), x_e) >= 0.f) cnt = half; else { zc = mid + 1; cnt -= half + 1; }
              }
              uint32_t L = zc, R = zc;                        // the stretch is [L, R)
              float dl = L > p ? fabsf(__fsub_rn(__fadd_rn(S.hx[L - 1], syg), x_e)) : 0.f;
              float dr = R < ub ? fabsf(__fsub_rn(__fadd_rn(S.hx[R], syg), x_e)) : 0.f;
#pragma unroll 1                                     // (rare, and C may be a compile-time constant: keep the code small)
              for (int k = 0; k < C; ++k) {
                const bool left = L > p && (R >= ub || dl <= dr);
                if (left) { --L; dl = L > p ? fabsf(__fsub_rn(__fadd_rn(S.hx[L - 1], syg), x_e)) : 0.f; }
                else { ++R; dr = R < ub ? fabsf(__fsub_rn(__fadd_rn(S.hx[R], syg), x_e)) : 0.f; }
              }
              // (equal x across the left cut: the lower index beats the kept one, the C closest are not one
              //  stretch -- leave the run to the eviction path below)
              if (!(L > p && S.hx[L - 1] == S.hx[L])) {
                p = L;
                p1 = R;
              }
            }
          } else if (__builtin_expect(p1 - p > (uint32_t)C, 0)) {
            // a run that can overflow the cap: of the hits on the negative side only the C next to the zero
            // crossing can be among the C closest (each one further out has C closer hits of this very run in
            // front of it), so the scan starts there instead of evicting its way through the run
            uint32_t zc = p;
            for (uint32_t cnt = p1 - p; cnt > 0;) {
              const uint32_t half = cnt >> 1, mid = zc + half;
              if (__fsub_rn(__fadd_rn(S.hx[mid], syg), x_e) >= 0.f) cnt = half; else { zc = mid + 1; cnt -= half + 1; }
            }
            if (zc - p > (uint32_t)C) {
              uint32_t q = zc - (uint32_t)C;
              while (q > p && S.hx[q - 1] == S.hx[q]) --q;     // equal x: equal |d|, the lower index wins the tie
              p = q;
            }
          }
        }
        const int n_before = n;
        bool took_any = false;
        for (; p < p1; ++p) {
          const float d = __fsub_rn(__fadd_rn(S.hx[p], syg), x_e);
          if (d > D) break;                         // x-sorted inside the sector: d only grows
          const bool acc = d >= negD;
          const uint32_t hs = ((uint32_t)S.hh[p] << 16) | (uint32_t)s;
          if (acc && (n >= C || (n > 0 && hs <= last))) {   // rare: cap reached or out of hit order
            const bool took = cand_insert<CC>(wa, slot, n, C, d, hs);
            took_any |= took;
            last = chs[n - 1];
            if (!took && d >= 0.f) break;           // full list, positive side: every later hit is further still
            continue;
          }
          if (acc) {                                // hits arrive in ascending index almost always: append
            cd[n] = d;
            chs[n] = hs;
            last = hs;
            ++n;
          }
        }
        if (!LU && (n != n_before || took_any)) note_zw(a, s, n_before == 0, zu, wu);
      }
    } else if (a.order_y) {
      // Y-sorted group: "two binary searches over the Y axis, one to delimit the beginning of the
      // region and another to delimit the end of it", then "the window range is refined by checking the hits"
      const float* X = a.hx + h0;
      uint32_t first = ga, lastp = ga;
      for (uint32_t cnt = gb - ga; cnt > 0;) {      // first hit with y_e <= y_end + y_tol
        const uint32_t half = cnt >> 1, mid = first + half;
        if (y_e <= __fadd_rn(__ldg(a.hye + h0 + mid), a.c.y_tol)) cnt = half; else { first = mid + 1; cnt -= half + 1; }
      }
      lastp = first;
      for (uint32_t cnt = gb - first; cnt > 0;) {   // first hit with y_begin - y_tol > y_e
        const uint32_t half = cnt >> 1, mid = lastp + half;
        if (__fsub_rn(__ldg(a.hyb + h0 + mid), a.c.y_tol) > y_e) cnt = half; else { lastp = mid + 1; cnt -= half + 1; }
      }
      for (uint32_t h = first; h < lastp; ++h) {
        const float d = __fsub_rn(__fadd_rn(__ldg(X + h), syg), x_e);
        if (!(fabsf(d) <= D)) continue;
        if (!(__fsub_rn(__ldg(a.hyb + h0 + h), a.c.y_tol) <= y_e && y_e <= __fadd_rn(__ldg(a.hye + h0 + h), a.c.y_tol)))
          continue;
        const uint32_t rid = __ldg(a.hid + h0 + h) >> 9;
        const uint32_t s = rid < a.id_table_size ? __ldg(a.id_to_sector + rid) : kInvalid;
        if (s >= a.n_sectors) continue;
        const bool first_cand = n == 0;
        if (cand_insert<CC>(wa, slot, n, C, d, (h << 16) | s) && !LU) note_zw(a, (int)s, first_cand, zu, wu);
      }
    } else {
      const float* X = a.hx + h0;
      uint32_t first = ga;
      for (uint32_t cnt = gb - ga; cnt > 0;) {      // first hit with d >= -D
        const uint32_t half = cnt >> 1, mid = first + half;
        const float d = __fsub_rn(__fadd_rn(__ldg(X + mid), syg), x_e);
        if (d >= negD) cnt = half; else { first = mid + 1; cnt -= half + 1; }
      }
      for (uint32_t h = first; h < gb; ++h) {
        const float d = __fsub_rn(__fadd_rn(__ldg(X + h), syg), x_e);
        if (!(d <= D)) break;
        if (!(__fsub_rn(__ldg(a.hyb + h0 + h), a.c.y_tol) <= y_e && y_e <= __fadd_rn(__ldg(a.hye + h0 + h), a.c.y_tol)))
          continue;
        const uint32_t rid = __ldg(a.hid + h0 + h) >> 9;
        const uint32_t s = rid < a.id_table_size ? __ldg(a.id_to_sector + rid) : kInvalid;
        if (s >= a.n_sectors) continue;             // reported by the staging pass of the bucketed path only
        const bool first_cand = n == 0;
        if (cand_insert<CC>(wa, slot, n, C, d, (h << 16) | s) && !LU) note_zw(a, (int)s, first_cand, zu, wu);
      }
    }
  }
  return n;
}

// z of candidate `i` of `slot` (UNI: every list of the batch has one z, kept per slot)
// (LU: layer-uniform geometry, the z of slot's layer straight from the kernel parameters)
template <bool UNI, bool LU = false, int CC = 0>
__device__ __forceinline__ float cand_z(const CompassArgs& a, const WarpArea& wa, int slot, int i) {
  return LU ? a.layer_z[slot & 3] : (UNI ? wa.zs[slot] : __ldg(a.sec_z + (wa.chs[slot * stride_of<CC>(wa) + i] & 0xFFFFu)));
}

// ---- phase 2 (b) + (c): `cnt` queued seeds, one per lane, then all their 3/4-hit combinations --------------
template <bool UNI, bool KICK, bool LU, int CC>
__device__ __forceinline__ void process_seeds(const CompassArgs& a, const WarpArea& wa, int lane, int cnt, int qhead,
                                              int dir) {
  const int LA = dir ? 3 : 0, LB = dir ? 1 : 2, LC = dir ? 2 : 1, LD = dir ? 0 : 3;
  const int CS = stride_of<CC>(wa);
  const bool min3 = a.c.min_hits == 3;
  // (b) 4 lanes share one seed (8 seeds per round): the exact cuts of step 5, then every 4th hit of the two
  //     other layers per lane; the masks of compatible hits end up in lane = seed index
  uint32_t pk = 0, mC = 0, mD = 0, k = 0;
  bool alive = false;                                // the seed of this lane passed the exact cuts
  if (lane < cnt) pk = wa.seedq[(qhead + lane) & (kSeedQ - 1)];
  const int sub = lane & 3;
  for (int r0 = 0; r0 < cnt; r0 += 8) {
    const int q = r0 + (lane >> 2);
    uint32_t pC = 0, pD = 0;
    bool ok = false;
    if (q < cnt) {
      const uint32_t sd = wa.seedq[(qhead + q) & (kSeedQ - 1)];
      const int j4 = (int)(sd >> 10) * 4, ia = (sd >> 5) & 31, ib = sd & 31;
      const float da = wa.cd[(j4 + LA) * CS + ia], db = wa.cd[(j4 + LB) * CS + ib];
      const float za = cand_z<UNI, LU, CC>(a, wa, j4 + LA, ia), zb = cand_z<UNI, LU, CC>(a, wa, j4 + LB, ib);
      const float bs = __fdiv_rn(__fsub_rn(db, da), __fsub_rn(zb, za));
      const float a0 = __fsub_rn(da, __fmul_rn(bs, __fsub_rn(za, KICK ? wa.tzm[sd >> 10] : a.c.z_mag)));
      ok = fabsf(bs) <= a.c.max_slope && fabsf(a0) <= a.c.kink_tol;
      if (ok) {
        const int nC = wa.n[j4 + LC], nD = wa.n[j4 + LD];
        const float* cC = wa.cd + (j4 + LC) * CS;
        const float* cDl = wa.cd + (j4 + LD) * CS;
        if (UNI) {
          const float predC = __fadd_rn(da, __fmul_rn(bs, __fsub_rn(LU ? a.layer_z[LC] : wa.zs[j4 + LC], za)));
          const float predD = __fadd_rn(da, __fmul_rn(bs, __fsub_rn(LU ? a.layer_z[LD] : wa.zs[j4 + LD], za)));
#pragma unroll 1
          for (int i = sub; i < nC; i += 4)
            if (fabsf(__fsub_rn(cC[i], predC)) <= a.c.seed_tol) pC |= 1u << i;
#pragma unroll 1
          for (int i = sub; i < nD; i += 4)
            if (fabsf(__fsub_rn(cDl[i], predD)) <= a.c.seed_tol) pD |= 1u << i;
        } else {
          for (int i = sub; i < nC; i += 4) {
            const float zc = cand_z<false, false, CC>(a, wa, j4 + LC, i);
            const float pred = __fadd_rn(da, __fmul_rn(bs, __fsub_rn(zc, za)));
            if (fabsf(__fsub_rn(cC[i], pred)) <= a.c.seed_tol) pC |= 1u << i;
          }
          for (int i = sub; i < nD; i += 4) {
            const float zd = cand_z<false, false, CC>(a, wa, j4 + LD, i);
            const float pred = __fadd_rn(da, __fmul_rn(bs, __fsub_rn(zd, za)));
            if (fabsf(__fsub_rn(cDl[i], pred)) <= a.c.seed_tol) pD |= 1u << i;
          }
        }
      }
    }
    pC |= __shfl_xor_sync(0xFFFFFFFFu, pC, 1); pC |= __shfl_xor_sync(0xFFFFFFFFu, pC, 2);
    pD |= __shfl_xor_sync(0xFFFFFFFFu, pD, 1); pD |= __shfl_xor_sync(0xFFFFFFFFu, pD, 2);
    const int src = ((lane - r0) & 7) * 4;               // lanes r0 .. r0+7 pick up the masks of their seed
    const uint32_t gC = __shfl_sync(0xFFFFFFFFu, pC, src), gD = __shfl_sync(0xFFFFFFFFu, pD, src);
    const bool gok = __shfl_sync(0xFFFFFFFFu, ok ? 1 : 0, src) != 0;
    if (lane >= r0 && lane < r0 + 8) { mC = gC; mD = gD; alive = gok; }
  }
  if (lane < cnt && alive) {
    const uint32_t pc = __popc(mC), pd = __popc(mD);
    k = min3 ? (pc + 1) * (pd + 1) - 1 : pc * pd;   // (c or none) x (d or none) with >= min_hits hits in total
  }
  const uint32_t incl = warp_incl_scan(k, lane), excl = incl - k;
  const uint32_t K = __shfl_sync(0xFFFFFFFFu, incl, 31);
  for (uint32_t base = 0; base < K; base += 32) {
    const uint32_t i = base + lane;
    int q = 0;                                       // owner seed: largest q with excl[q] <= i
#pragma unroll
    for (int step = 16; step > 0; step >>= 1) {
      const uint32_t e = __shfl_sync(0xFFFFFFFFu, excl, q + step);
      if (e <= i) q += step;
    }
    const uint32_t r = i - __shfl_sync(0xFFFFFFFFu, excl, q);
    const uint32_t pkq = __shfl_sync(0xFFFFFFFFu, pk, q);
    const uint32_t mCq = __shfl_sync(0xFFFFFFFFu, mC, q), mDq = __shfl_sync(0xFFFFFFFFu, mD, q);
    if (i < K) {
      const uint32_t pc = __popc(mCq);
      uint32_t selC, selD;                           // 0 = none, else 1-based ordinal of the set bit
      if (min3) { const uint32_t r1 = r + 1, w = pc + 1; selD = small_div(r1, w); selC = r1 - selD * w; }
      else { selD = small_div(r, pc); selC = r - selD * pc + 1; selD += 1; }
      int ci = -1, di = -1;
      if (selC) { uint32_t m = mCq; for (uint32_t t = 1; t < selC; ++t) m &= m - 1; ci = __ffs(m) - 1; }
      if (selD) { uint32_t m = mDq; for (uint32_t t = 1; t < selD; ++t) m &= m - 1; di = __ffs(m) - 1; }
      const int j = (int)(pkq >> 10), ia = (pkq >> 5) & 31, ib = pkq & 31;
      int pos[4];                                    // candidate position per layer, -1 = none
      if (dir == 0) { pos[0] = ia; pos[1] = ci; pos[2] = ib; pos[3] = di; }
      else { pos[0] = di; pos[1] = ib; pos[2] = ci; pos[3] = ia; }
      bool pr[4];
      float d[4], z[4], w[4];
      int nh = 0;
#pragma unroll
      for (int l = 0; l < 4; ++l) {
        pr[l] = pos[l] >= 0;
        d[l] = z[l] = w[l] = 0.f;
        if (pr[l]) {
          const int slot = j * 4 + l;
          d[l] = wa.cd[slot * CS + pos[l]];
          if (LU) { z[l] = a.layer_z[l]; w[l] = a.layer_w[l]; }
          else if (UNI) { z[l] = wa.zs[slot]; w[l] = wa.ws[slot]; }
          else {
            const uint32_t s = wa.chs[slot * CS + pos[l]] & 0xFFFFu;
            z[l] = __ldg(a.sec_z + s);
            w[l] = __ldg(a.sec_w + s);
          }
          ++nh;
        }
      }
      const FitResult fr = fit_tracklet(pr, d, z, w, nh, a.c, KICK ? wa.tzm[j] : a.c.z_mag);
      if (fr.valid)
        atomicMin(&wa.best[j], make_key(nh, fr.chi2, (uint32_t)pos[0] & 63u, (uint32_t)pos[1] & 63u,
                                        (uint32_t)pos[2] & 63u, (uint32_t)pos[3] & 63u));
    }
  }
}

// ---- phase 2 (a): seed rows of the batch, conservative filter of the slope + kink cuts, seed queue -----------
// (process_seeds has ONE call site per variant: the kernel's code size decides how well it stays in the
//  instruction cache)
template <bool UNI, bool INTERVAL, bool KICK, bool LU, int CC>
__device__ __forceinline__ void find_tracklets(const CompassArgs& a, const WarpArea& wa, int lane, uint32_t todo) {
  const int j = lane & 7;
  const int CS = stride_of<CC>(wa);
  const uint32_t lt_mask = (1u << lane) - 1u;
  for (int dir = 0; dir < 2 && todo; ++dir) {     // forward seeds (L0, L2), then backward (L3, L1)
    const int LA = dir ? 3 : 0, LB = dir ? 1 : 2;
    const uint32_t nA = wa.n[4 * j + LA], nB = wa.n[4 * j + LB];
    // rows (track, hit a) of the batch, one per lane; the lane walks the partner hits b of its row
    const uint32_t P = (lane < kTPW && ((todo >> j) & 1u) && nB > 0u) ? nA : 0u;
    const uint32_t incl = warp_incl_scan(P, lane), excl = incl - P;
    const uint32_t total = __shfl_sync(0xFFFFFFFFu, incl, 31);
    int qn = 0, qhead = 0;
    for (uint32_t base = 0; base < total; base += 32) {
      const uint32_t i = base + lane;
      int jj = 0;                               // owner track: largest jj < 8 with excl[jj] <= i
#pragma unroll
      for (int step = 4; step > 0; step >>= 1) {
        const uint32_t e = __shfl_sync(0xFFFFFFFFu, excl, jj + step);
        if (e <= i) jj += step;
      }
      const uint32_t ia = i - __shfl_sync(0xFFFFFFFFu, excl, jj);
      int nBj = (int)__shfl_sync(0xFFFFFFFFu, nB, jj);
      const int sA = jj * 4 + LA, sB = jj * 4 + LB;
      const float* cB = wa.cd + sB * CS;
      float da = 0.f, za = 0.f, zam = 0.f, rinv = 0.f, lim0 = 0.f;
      if (i < total) {
        da = wa.cd[sA * CS + ia];
        za = cand_z<UNI, LU, CC>(a, wa, sA, (int)ia);
        zam = za - (KICK ? wa.tzm[jj] : a.c.z_mag);
        if (UNI) rinv = rcp_approx((LU ? a.layer_z[LB] : wa.zs[sB]) - za);
        lim0 = a.c.kink_tol + kFilterEps * (a.c.kink_tol + fabsf(da));
      } else {
        nBj = 0;
      }
      int maxB = __reduce_max_sync(0xFFFFFFFFu, nBj);
      int ib0 = 0;
      if (INTERVAL && maxB > a.interval_min && __all_sync(0xFFFFFFFFu, nBj == 0 || wa.srt[sB] != 0)) {
        // long partner lists that ascend in d (one x-sorted run, or runs of x-disjoint sectors): the partners that
        // can pass the slope and kink cuts are an interval of d, found by two searches instead of a walk over the
        // whole list.  [lo, hi] contains every db the cuts accept (real arithmetic widened by 1e-5 relative; a NaN
        // bound opens the interval), the filter below and the exact cuts still decide.
        const float dz = (LU ? a.layer_z[LB] : wa.zs[sB]) - za, sdz = a.slope_lim * fabsf(dz);
        const float rho = zam * rinv, rr = rcp_approx(rho);
        const float k1 = a.c.kink_tol * (1.f + 1e-5f);
        const float qa = (da - k1) * rr, qb = (da + k1) * rr;
        float lo = fmaxf(da - sdz, da + fminf(qa, qb)), hi = fminf(da + sdz, da + fmaxf(qa, qb));
        const float mg = 1e-5f * (fabsf(da) + fabsf(lo) + fabsf(hi)) + 1e-6f;
        lo -= mg; hi += mg;
        if (!(fabsf(rho) > 1e-12f) || !(lo == lo) || !(hi == hi)) { lo = -__int_as_float(0x7F800000); hi = -lo; }
        int plo = 0, phi = 0;
#pragma unroll
        for (int step = 32; step > 0; step >>= 1) {
          const int q1 = plo + step, q2 = phi + step;
          if (q1 <= nBj && cB[q1 - 1] < lo) plo = q1;           // first partner with d >= lo
          if (q2 <= nBj && cB[q2 - 1] <= hi) phi = q2;          // first partner with d > hi
        }
        ib0 = plo;
        nBj = max(phi - plo, 0);
        maxB = __reduce_max_sync(0xFFFFFFFFu, nBj);
      }
      const bool last_chunk = base + 32 >= total;
      for (int ik = 0; ik < (INTERVAL ? max(maxB, last_chunk ? 1 : 0) : maxB); ++ik) {
        // conservative filter: bs and a0 through a reciprocal, accepted with a relative margin that covers the
        // roundings of both evaluations; the exact cuts follow in process_seeds
        bool pass = false;
        const int ib = INTERVAL ? ib0 + ik : ik;
        if (ik < nBj) {
          if (!UNI) rinv = rcp_approx(cand_z<false, false, CC>(a, wa, sB, ib) - za);
          const float bsa = (cB[ib] - da) * rinv;
          const float t = bsa * zam;
          pass = fabsf(bsa) <= a.slope_lim && fabsf(da - t) <= __fmaf_rn(kFilterEps, fabsf(t), lim0);
        }
        const uint32_t m = __ballot_sync(0xFFFFFFFFu, pass);
        const bool last = last_chunk && ik + 1 >= maxB;
        if (m == 0u && !last) continue;
        if (pass)
          wa.seedq[(qhead + qn + __popc(m & lt_mask)) & (kSeedQ - 1)] = ((uint32_t)jj << 10) | (ia << 5) | (uint32_t)ib;
        qn += __popc(m);
        while (qn >= 32 || (last && qn > 0)) {  // a full queue, or the rest after the last pair
          __syncwarp();
          const int cnt = min(qn, 32);
          process_seeds<UNI, KICK, LU, CC>(a, wa, lane, cnt, qhead, dir);
          qhead += cnt;
          qn -= cnt;
          __syncwarp();
        }
      }
    }
    if (!a.c.both_directions)                   // backward only if nothing valid (A11); else best of both
      todo &= ~__ballot_sync(0xFFFFFFFFu, lane < kTPW && wa.best[j] != kNoKey);
  }
}

// The warps of the CTA pull 8-track batches of the item: track m of the item is VELO track t0 + m * K + part.
template <bool BUCKETED, bool INTERVAL, bool KICK, bool LU, int CC>
__device__ __forceinline__ void track_loop(const CompassArgs& a, const WarpArea& wa, const SmemView& S, int* s_ticket,
                                           uint32_t h0, uint32_t t0, uint32_t nTk, uint32_t part, uint32_t T,
                                           const uint16_t* perm) {
  const int lane = threadIdx.x & 31;
  const int l = lane & 3;                         // layer of this lane in phase 1 and in the output
  const int j = lane & 7;                         // track-in-batch this lane does the bookkeeping for (lanes 0..7)
  const int CS = stride_of<CC>(wa);
  for (;;) {
    int batch = 0;
    if (lane == 0) batch = atomicAdd(s_ticket, 1);
    batch = __shfl_sync(0xFFFFFFFFu, batch, 0);
    const uint32_t ti = (uint32_t)batch * kTPW + (uint32_t)(lane >> 2);      // track of the item, in batch order
    if ((uint32_t)batch * kTPW >= nTk) break;
    const bool active = ti < nTk;
    const uint32_t tg = t0 + (active ? (perm ? (uint32_t)perm[ti] : ti) * a.split + part : 0u);
    // ---------------- phase 1: window search, lane = (track, layer) ---------------------------------------
    int n_st = 0;
    float zu = LU ? a.layer_z[l] : 0.f, wu = LU ? a.layer_w[l] : 0.f;
    if (active) {
      const float vx = __ldg(a.vx + tg), vy = __ldg(a.vy + tg), vtx = __ldg(a.vtx + tg), vty = __ldg(a.vty + tg);
      const float dzv = __fsub_rn(a.layer_z[l], a.vz);
      const float x_e = __fadd_rn(vx, __fmul_rn(vtx, dzv));
      const float y_e = __fadd_rn(vy, __fmul_rn(vty, dzv));
      n_st = collect_window<BUCKETED, LU, CC>(a, wa, S, lane, l, x_e, y_e, h0, zu, wu);
      if (KICK && l == 0) track_kick(a.kick, a.c, vx, vy, vtx, vty, a.vz, wa.tkap[lane >> 2], wa.tzm[lane >> 2]);
    } else if (KICK && l == 0) {
      wa.tkap[lane >> 2] = a.c.kappa;
      wa.tzm[lane >> 2] = a.c.z_mag;
    }
    wa.n[lane] = n_st;
    if (!LU) { wa.zs[lane] = zu; wa.ws[lane] = wu; }
    // long lists that ascend in d (one x-sorted run, or runs of x-disjoint sectors) are searched, not walked
    if (INTERVAL && __any_sync(0xFFFFFFFFu, n_st > a.interval_min)) {
      int srt = 1;
      const float* cdl = wa.cd + lane * CS;
      for (int i = 1; i < n_st; ++i) srt &= cdl[i] >= cdl[i - 1] ? 1 : 0;
      wa.srt[lane] = srt;
    }
    if (lane < kTPW) wa.best[lane] = kNoKey;
    const bool uni = LU || __all_sync(0xFFFFFFFFu, zu == zu);      // every list of the batch has one z and one weight
    __syncwarp();
    // ---------------- phase 2: tracklet finding, flattened over the warp ---------------
    const int nonempty = (wa.n[4 * j] > 0) + (wa.n[4 * j + 1] > 0) + (wa.n[4 * j + 2] > 0) + (wa.n[4 * j + 3] > 0);
    const uint32_t todo = __ballot_sync(0xFFFFFFFFu, lane < kTPW && nonempty >= a.c.min_hits);
    if (LU || uni) find_tracklets<true, INTERVAL, KICK, LU, CC>(a, wa, lane, todo);
    else find_tracklets<false, false, KICK, false, CC>(a, wa, lane, todo);
    // ---------------- output: the 4 lanes of a track write one layer each ----------------------------------
    if (active) {
      const int q4 = lane & ~3;
      const unsigned long long best = wa.best[lane >> 2];
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
            const uint32_t hs = wa.chs[(q4 + k) * CS + pp[k]];
            d[k] = wa.cd[(q4 + k) * CS + pp[k]];
            z[k] = LU ? a.layer_z[k] : __ldg(a.sec_z + (hs & 0xFFFFu));
            w[k] = LU ? a.layer_w[k] : __ldg(a.sec_w + (hs & 0xFFFFu));
            if (k == l) hidx = (int)(h0 + (hs >> 16));
          }
        }
        const FitResult r = fit_tracklet(pr, d, z, w, nh, a.c, KICK ? wa.tzm[lane >> 2] : a.c.z_mag);
        qop = __fdiv_rn(r.b, KICK ? wa.tkap[lane >> 2] : a.c.kappa);
      }
      a.out_idx[(size_t)l * T + tg] = hidx;
      if (l == 0) { a.out_n[tg] = nh; a.out_qop[tg] = qop; a.out_chi2[tg] = chi2; }
    }
    __syncwarp();                                 // the batch is consumed before its lists are overwritten
  }
}

// Geometry tables of a CTA, staged once.  (Not inlined, and its arguments are scalars: the kernel's register allocation
// is tight, and a call with the parameter struct by reference would copy the struct to local memory.)
__device__ __noinline__ void stage_tables(const uint32_t* group_first_sector, const float* sec_ye, const float* sec_yb,
                                          const float* sec_dxdy, const float* group_xmin, const float* group_xmax, uint32_t gpl,
                                          uint32_t rows_uniform, float y_tol, uint32_t ng, float4* s_gA, uint2* s_gB,
                                          float2* s_yr, float2* s_lay) {
  const int tid = threadIdx.x, nt = blockDim.x;
  for (uint32_t g = tid; g < ng; g += nt) {
    const uint32_t sa = __ldg(group_first_sector + g), sb = __ldg(group_first_sector + g + 1);
    const float y0 = __fadd_rn(__ldg(sec_ye + sa), y_tol), y1 = __fadd_rn(__ldg(sec_ye + sb - 1), y_tol);
    const float inv = (sb - sa > 1 && y1 > y0) ? (float)(sb - sa - 1) / (y1 - y0) : 0.f;
    const uint32_t gp = g + 2 * (g / gpl);
    s_gA[gp] = make_float4(__ldg(group_xmin + g), __ldg(group_xmax + g), __ldg(sec_dxdy + sa), y0);
    s_gB[gp] = make_uint2(__float_as_uint(inv), sa | (sb << 16));
  }
  for (uint32_t i = tid; i < 4 * rows_uniform; i += nt) {       // y rows of a layer = those of its first group
    const uint32_t s = __ldg(group_first_sector + (i / rows_uniform) * gpl) + i % rows_uniform;
    s_yr[i] = make_float2(__fsub_rn(__ldg(sec_yb + s), y_tol), __fadd_rn(__ldg(sec_ye + s), y_tol));
  }
  if (tid < 4) {
    const uint32_t ga = tid * gpl, gb = ga + gpl;
    const float x0 = __ldg(group_xmax + ga), x1 = __ldg(group_xmax + gb - 1);
    s_lay[tid] = make_float2(x0, (gpl > 1 && x1 > x0) ? (float)(gpl - 1) / (x1 - x0) : 0.f);
  }
}

// Event order of a batch: the events with the most VELO tracks first.
// A batch of more events than resident CTAs ends with CTAs that find no work while others still hold a whole event
// (config 3: 1000 events on 592 CTAs).  Handing the heavy events out first leaves the light ones for the end (events
// sorted like this on the host: Compass 101.8 -> 97 us).  Every CTA computes the same order itself: a stable counting
// sort of the events by track count relative to the batch mean (32 bins of 1/32 of the mean, heaviest bin first; events
// of a bin keep their order) -- each warp owns a contiguous range of events, counts per (warp, bin), a scan, then the
// same walk again.  Results do not depend on the order.  perm == nullptr: no order for this launch.
// The small kernels (72 registers at 4 CTAs per SM) pay for the code: however it is placed, inlined or not, the track
// loop spills a little more (24 -> 40 bytes of stack in this form, called unconditionally; 56-88 in the others tried).
// Config 3: Compass timed alone 102.0 -> 105.1 us (103.4 with the order off: the order's own prologue, two round trips
// to the VELO offsets, is exposed there), but the two calls back to back 152.6 -> 149.3 us -- behind ut_decode the
// prologue runs while the decode's last CTAs finish, and the shorter tail is what remains.
// scratch: 128 bytes per warp + n_events bytes.
__device__ __noinline__ void order_events(const uint32_t* velo_offsets, uint32_t ne, unsigned char* scratch, uint16_t* perm) {
  if (perm == nullptr) return;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  uint32_t* cnt = reinterpret_cast<uint32_t*>(scratch);               // [nwarps][32]
  unsigned char* ebin = scratch + (size_t)nwarps * 128;               // [ne] bin of every event
  // (4 events per thread and round, their loads and the one of the total in flight together: one round trip to the
  //  offsets for a batch of up to 4 x blockDim events)
  for (uint32_t e0 = tid; e0 < ne; e0 += 4u * (uint32_t)nt) {
    uint32_t v0[4], v1[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const uint32_t e = e0 + (uint32_t)q * (uint32_t)nt;
      v0[q] = v1[q] = 0u;
      if (e < ne) { v0[q] = __ldg(velo_offsets + e); v1[q] = __ldg(velo_offsets + e + 1); }
    }
    // bin = 16 + 32 * (tracks - mean) / mean, in fp32 (the same instructions on the same numbers in every CTA)
    const float mean = fmaxf((float)__ldg(velo_offsets + ne) / (float)ne, 1.f), scale = 32.f / mean;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const uint32_t e = e0 + (uint32_t)q * (uint32_t)nt;
      const float nTe = v1[q] >= v0[q] ? (float)min(v1[q] - v0[q], 0x3FFFFFu) : 0.f;
      const int b = __float2int_rd(fminf(fmaxf(__fmul_rn(__fsub_rn(nTe, mean), scale), -16.f), 15.f));     // -16 .. 15
      if (e < ne) ebin[e] = (unsigned char)(15 - b);                                                          // heavy first
    }
  }
  const uint32_t per_warp = ((ne + (uint32_t)nwarps - 1u) / (uint32_t)nwarps + 31u) & ~31u;
  const uint32_t eb = min((uint32_t)warp * per_warp, ne), ee = min(eb + per_warp, ne);
  cnt[warp * 32 + lane] = 0;
  __syncthreads();
  for (int pass = 0; pass < 2; ++pass) {
    for (uint32_t e0 = eb; e0 < ee; e0 += 32u) {
      const uint32_t e = e0 + (uint32_t)lane;
      const uint32_t b = e < ee ? (uint32_t)ebin[e] : 32u;            // 32: no event in this lane
      const uint32_t m = __match_any_sync(0xFFFFFFFFu, b);
      if (pass == 1 && b < 32u) perm[cnt[warp * 32 + b] + __popc(m & lt_mask)] = (uint16_t)e;
      __syncwarp();
      if (b < 32u && (m & lt_mask) == 0u) cnt[warp * 32 + b] += __popc(m);
      __syncwarp();
    }
    if (pass == 0) {
      __syncthreads();
      // first slot of (warp, bin): the events of the heavier bins, then those of the same bin in earlier warps
      uint32_t col = 0, before = 0;
      for (int w = 0; w < nwarps; ++w) {
        const uint32_t c = cnt[w * 32 + lane];
        if (w < warp) before += c;
        col += c;
      }
      const uint32_t base = warp_incl_scan(col, lane) - col;
      __syncthreads();                                                // every warp has read the counts
      cnt[warp * 32 + lane] = base + before;
      __syncwarp();
    }
  }
}

// One CTA works through work items (event, part) handed out by the ticket.  Geometry tables are staged once.
// INTERVAL: the seed search of long, d-sorted partner lists by interval (worth its code only when
// max_candidates_per_layer allows long lists; the kernel without it is the faster one for short lists).
// KICK: per-track kappa / z_mag from the kick table (ut_geometry.kick_*); without it the config's constants come
// straight from the kernel parameters.
template <int MAXT, int MINB, bool INTERVAL, bool KICK, bool LU, int CC = 0>
__global__ void __launch_bounds__(MAXT, MINB) compass_kernel(const CompassArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;
  const uint32_t ng = a.n_groups, ns = a.n_sectors;
  const int C = a.c.max_candidates_per_layer;
  Carver cvr(smem_raw);
  cvr.take<uint16_t>(a.ev_stage);       // event of every ticket (thread 0 reads it), at offset 0 of the dynamic array
  float4* s_gA = cvr.take<float4>(ng + 8);
  uint2* s_gB = cvr.take<uint2>(ng + 8);
  float2* s_yr = cvr.take<float2>(4 * a.rows_uniform);
  uint32_t* s_goff = cvr.take<uint32_t>(ng + 1);
  uint16_t* s_off = cvr.take<uint16_t>(a.soff_stride);
  float* s_hx = cvr.take<float>(a.hit_stage + 8);
  uint16_t* s_hh = cvr.take<uint16_t>(a.hit_stage + 16);
  uint16_t* s_perm = cvr.take<uint16_t>(a.trk_stage);
  unsigned char* s_warp_areas = cvr.take<unsigned char>(1);  // nwarps x warp_area_bytes(C); aliased by the scratch below
  // scratch while no warp is in the track loop: radius bins + per-track (bin, position); re-bucketing counters and
  // the event's id and x ranges (two bulk copies) when the container carries no per-sector view
  uint32_t* s_bins = reinterpret_cast<uint32_t*>(s_warp_areas);
  uint32_t* s_binpos = s_bins + kBins;
  uint32_t* s_cnt = reinterpret_cast<uint32_t*>(s_warp_areas);
  uint32_t* s_tmp_id = reinterpret_cast<uint32_t*>(s_warp_areas + align16((size_t)ns * 8));
  float* s_tmp_x = reinterpret_cast<float*>(s_warp_areas + align16((size_t)ns * 8) + align16((size_t)(a.hit_stage + 8) * 4));
  __shared__ float2 s_lay[4];
  __shared__ int s_ticket;
  __shared__ uint64_t s_bar;
  uint32_t bar_phase = 0;
  if (tid == 0) { mbar_init(&s_bar, 1); fence_mbar_init(); }
  const uint32_t lt_mask = (1u << lane) - 1u;

  // ---- event order: the events with the most VELO tracks first (order_events above; ev_stage != 0: the launch found room
  // for the table and one CTA per event, K == 1).  Only the VELO offsets are read: none of it waits for ut_decode.
  order_events(a.velo_offsets, (uint32_t)a.n_events, s_warp_areas,
               a.ev_stage != 0u ? reinterpret_cast<uint16_t*>(smem_raw) : nullptr);
  // ---- geometry tables, once per CTA

  stage_tables(a.group_first_sector, a.sec_ye, a.sec_yb, a.sec_dxdy, a.group_xmin, a.group_xmax, a.gpl, a.rows_uniform,
               a.c.y_tol, ng, s_gA, s_gB, s_yr, s_lay);
  SmemView S;
  S.gA = s_gA; S.gB = s_gB; S.yr = s_yr; S.lay = s_lay; S.goff = s_goff; S.off = s_off; S.hx = s_hx; S.hh = s_hh;
  WarpArea wa;
  {
    const int CS = cand_stride(C);
    unsigned char* p = s_warp_areas + (size_t)warp * warp_area_bytes(C, LU, INTERVAL, KICK);
    wa.CS = CS;
    wa.cd = reinterpret_cast<float*>(p);
    wa.chs = reinterpret_cast<uint32_t*>(p + (size_t)CS * 32 * 4);
    p += (size_t)CS * 32 * 8;
    wa.best = reinterpret_cast<unsigned long long*>(p);
    wa.seedq = reinterpret_cast<uint32_t*>(p + kTPW * 8);
    wa.n = reinterpret_cast<int*>(p + kTPW * 8 + kSeedQ * 4);
    p += kTPW * 8 + kSeedQ * 4 + 32 * 4;
    wa.zs = reinterpret_cast<float*>(p);               // (arrays a kernel variant does not use take no room: their
    wa.ws = reinterpret_cast<float*>(p + 32 * 4);      //  pointers are never dereferenced there)
    if (!LU) p += 32 * 8;
    wa.srt = reinterpret_cast<int*>(p);
    if (INTERVAL) p += 32 * 4;
    wa.tzm = reinterpret_cast<float*>(p);
    wa.tkap = wa.tzm + kTPW;
  }
  const uint32_t Tend = __ldg(a.velo_offsets + a.n_events);
  const uint32_t T = a.idx_stride ? a.idx_stride : Tend;
  const uint32_t K = a.split;
  const uint32_t n_items = (uint32_t)a.n_events * K;

  // Launched with programmatic stream serialization the CTAs may be resident, with their tables staged, while the
  // preceding kernel of the stream (ut_decode) still runs on other SMs: everything it wrote is read after this point.
  asm volatile("griddepcontrol.wait;" ::: "memory");
  __shared__ uint32_t s_item[2];                   // double-buffered: a slow thread still reads the previous ticket
  for (int k = 0;; ++k) {
    // work items are dealt out dynamically: CTAs that finish early take more
    if (tid == 0) {                                // (ev_stage != 0: K == 1, the item is the event the order gives the ticket)
      const uint32_t t = atomicAdd(a.ticket, 1u);
      s_item[k & 1] = (a.ev_stage != 0u && t < n_items) ? (uint32_t)reinterpret_cast<const uint16_t*>(smem_raw)[t] : t;
    }
    __syncthreads();                               // tables staged, event order written / previous item fully consumed
    const uint32_t item = s_item[k & 1];
    if (item >= n_items) break;
    const int e = (int)(item / K);
    const uint32_t part = item - (uint32_t)e * K;
    const uint32_t t0 = __ldg(a.velo_offsets + e), t1 = __ldg(a.velo_offsets + e + 1);
    const uint32_t* go = a.hit_offsets + (size_t)e * ng;
    const uint32_t h0 = __ldg(go), h1 = __ldg(go + ng);
    if (t1 < t0 || t1 > Tend) {                       // inconsistent VELO offsets: nothing can be written safely
      if (tid == 0) atomicOr(a.status, (uint32_t)UT_STATUS_BAD_OFFSETS);
      continue;
    }
    bool bad = h1 < h0;
    for (uint32_t g = tid; g <= ng; g += nt) {
      const uint32_t o = __ldg(go + g);
      s_goff[g] = o - h0;
      if (g < ng) bad |= __ldg(go + g + 1) < o;
    }
    if (tid == 0) s_ticket = 0;
    const uint32_t n = h1 - h0;
    const uint32_t nT = t1 - t0;
    const uint32_t nTk = nT > part ? (nT - part + K - 1) / K : 0u;      // tracks t0 + part, t0 + part + K, ...
    // an event whose hits end past `capacity` was not written by the decode (UT_STATUS_CAPACITY there): its range of
    // the hit arrays must not be read
    // (__syncthreads_or returns a truth value, not the OR of the arguments; n is the same in every thread)
    const int flag = __syncthreads_or(bad ? 1 : 0) ? 1 : ((unsigned long long)h1 > a.capacity ? 4 : (n > 65535u ? 2 : 0));
    if (flag) {                                    // uniform: report and emit "no tracklet" for every track of the part
      if (tid == 0) atomicOr(a.status, (flag & 1 ? (uint32_t)UT_STATUS_BAD_OFFSETS : 0u) |
                                           (flag & 2 ? (uint32_t)UT_STATUS_EVENT_TOO_LARGE : 0u) |
                                           (flag & 4 ? (uint32_t)UT_STATUS_CAPACITY : 0u));
      for (uint32_t m = tid; m < nTk; m += nt) {
        const uint32_t t = t0 + m * K + part;
        for (int q = 0; q < 4; ++q) a.out_idx[(size_t)q * T + t] = -1;
        a.out_n[t] = 0; a.out_qop[t] = 0.f; a.out_chi2[t] = 0.f;
      }
      continue;
    }
    if (nTk == 0) continue;
    const bool staged = n <= a.hit_stage;
    // the per-sector view of the event as ut_decode left it: three bulk copies, nothing to compute
    const bool view = staged && a.soff != nullptr &&
                      __ldg(a.soff + (size_t)e * a.soff_stride + ns + 1) == (uint16_t)UT_SECTOR_INDEX_VALID;
    if (view) {
      const uint32_t cx0 = h0 & ~3u, cx1 = (h1 + 3u) & ~3u, ci0 = h0 & ~7u, ci1 = (h1 + 7u) & ~7u;
      if (tid == 0) {
        fence_proxy_async();                 // earlier generic-proxy accesses of the staging arrays are done (barrier above)
        mbar_expect_tx(&s_bar, (n > 0 ? (cx1 - cx0) * 4u + (ci1 - ci0) * 2u : 0u) + a.soff_stride * 2u);
        bulk_g2s(s_off, a.soff + (size_t)e * a.soff_stride, a.soff_stride * 2u, &s_bar);
        if (n > 0) {
          bulk_g2s(s_hx, a.sx + cx0, (cx1 - cx0) * 4u, &s_bar);
          bulk_g2s(s_hh, a.si + ci0, (ci1 - ci0) * 2u, &s_bar);
        }
      }
      S.hx = s_hx + (h0 - cx0);
      S.hh = s_hh + (h0 - ci0);
    } else if (staged) {
      S.hx = s_hx;
      S.hh = s_hh;
      // ---- stage: a warp re-buckets one sector group at a time, per sector, keeping the x order -----------
      // (count -> warp scan over the group's sectors -> ordered scatter with match.any; no block barrier)
      bool bad_id = false;
      // the event's ids and x by two bulk copies over the 16-byte aligned superset of [h0, h1)
      const uint32_t c0 = h0 & ~3u, c1 = (h1 + 3u) & ~3u;
      const bool bulk = a.bulk_ok && (unsigned long long)c1 <= a.capacity && n > 0;
      const uint32_t* idp = a.hid + h0;
      const float* xp = a.hx + h0;
      if (bulk) {
        if (tid == 0) {
          fence_proxy_async();               // earlier generic-proxy accesses of the region are done (barrier above)
          mbar_expect_tx(&s_bar, 2u * (c1 - c0) * 4u);
          bulk_g2s(s_tmp_id, a.hid + c0, (c1 - c0) * 4u, &s_bar);
          bulk_g2s(s_tmp_x, a.hx + c0, (c1 - c0) * 4u, &s_bar);
        }
        mbar_wait(&s_bar, bar_phase);
        bar_phase ^= 1u;
        idp = s_tmp_id + (h0 - c0);
        xp = s_tmp_x + (h0 - c0);
      }
      for (uint32_t g = warp; g < ng; g += nwarps) {
        const uint32_t ga = s_goff[g], gb = s_goff[g + 1];
        const uint32_t gp = g + 2 * (g / a.gpl);
        const uint32_t sa = s_gB[gp].y & 0xFFFFu, sb = s_gB[gp].y >> 16;
        if (g == ng - 1 && lane == 0) s_off[ns] = (uint16_t)n;
        if (gb - ga <= 64u && sb - sa <= 32u) {
          // one pass, <= 2 hits per lane: rank among the lanes of the same sector (match.any keeps the x
          // order), per-sector counts through shared memory, exclusive scan over the group's sectors
          uint32_t* cntA = s_cnt;
          uint32_t* cntB = s_cnt + ns;
          if (sa + lane < sb) { cntA[sa + lane] = 0; cntB[sa + lane] = 0; }
          const uint32_t i0 = ga + lane, i1 = i0 + 32u;
          uint32_t sec0 = kInvalid, sec1 = kInvalid;
          float x0 = 0.f, x1 = 0.f;
          if (i0 < gb) {
            const uint32_t rid = idp[i0] >> 9;
            sec0 = rid < a.id_table_size ? __ldg(a.id_to_sector + rid) : kInvalid;
            if (!(sec0 >= sa && sec0 < sb)) { sec0 = kInvalid; bad_id = true; }
            x0 = xp[i0];
          }
          if (i1 < gb) {
            const uint32_t rid = idp[i1] >> 9;
            sec1 = rid < a.id_table_size ? __ldg(a.id_to_sector + rid) : kInvalid;
            if (!(sec1 >= sa && sec1 < sb)) { sec1 = kInvalid; bad_id = true; }
            x1 = xp[i1];
          }
          const uint32_t peers0 = __match_any_sync(0xFFFFFFFFu, sec0);
          const uint32_t rank0 = __popc(peers0 & lt_mask);
          const bool two = gb - ga > 32u;                       // warp-uniform
          uint32_t peers1 = 0, rank1 = 0;
          if (two) { peers1 = __match_any_sync(0xFFFFFFFFu, sec1); rank1 = __popc(peers1 & lt_mask); }
          __syncwarp();
          if (sec0 != kInvalid && rank0 == 0) cntA[sec0] = __popc(peers0);
          if (sec1 != kInvalid && rank1 == 0) cntB[sec1] = __popc(peers1);
          __syncwarp();
          const uint32_t cA = sa + lane < sb ? cntA[sa + lane] : 0u;
          const uint32_t cB = sa + lane < sb ? cntB[sa + lane] : 0u;
          const uint32_t excl = warp_incl_scan(cA + cB, lane) - (cA + cB);
          if (sa + lane < sb) s_off[sa + lane] = (uint16_t)(ga + excl);
          const uint32_t b0 = __shfl_sync(0xFFFFFFFFu, excl, sec0 == kInvalid ? 0 : (int)(sec0 - sa));
          const int src1 = sec1 == kInvalid ? 0 : (int)(sec1 - sa);
          const uint32_t b1 = __shfl_sync(0xFFFFFFFFu, excl, src1) + __shfl_sync(0xFFFFFFFFu, cA, src1);
          if (sec0 != kInvalid) { s_hx[ga + b0 + rank0] = x0; s_hh[ga + b0 + rank0] = (uint16_t)i0; }
          if (sec1 != kInvalid) { s_hx[ga + b1 + rank1] = x1; s_hh[ga + b1 + rank1] = (uint16_t)i1; }
          __syncwarp();                                          // cntA / cntB are reused by the next group
          continue;
        }
        for (uint32_t s = sa + lane; s < sb; s += 32) s_cnt[s] = 0;
        __syncwarp();
        for (uint32_t i = ga + lane; i < gb; i += 32) {
          const uint32_t rid = idp[i] >> 9;
          const uint32_t s = rid < a.id_table_size ? __ldg(a.id_to_sector + rid) : kInvalid;
          if (s >= sa && s < sb) atomicAdd(&s_cnt[s], 1u); else bad_id = true;
        }
        __syncwarp();
        uint32_t run = ga;
        for (uint32_t s0 = sa; s0 < sb; s0 += 32) {
          const uint32_t s = s0 + lane;
          const uint32_t c = s < sb ? s_cnt[s] : 0u;
          const uint32_t incl = warp_incl_scan(c, lane);
          if (s < sb) { s_off[s] = (uint16_t)(run + incl - c); s_cnt[s] = run + incl - c; }
          run += __shfl_sync(0xFFFFFFFFu, incl, 31);
        }
        __syncwarp();
        for (uint32_t i0 = ga; i0 < gb; i0 += 32) {
          const uint32_t i = i0 + lane;
          uint32_t s = kInvalid;
          float x = 0.f;
          if (i < gb) {
            const uint32_t rid = idp[i] >> 9;
            s = rid < a.id_table_size ? __ldg(a.id_to_sector + rid) : kInvalid;
            if (!(s >= sa && s < sb)) s = kInvalid;
            x = xp[i];
          }
          const uint32_t peers = __match_any_sync(0xFFFFFFFFu, s);
          const uint32_t rank = __popc(peers & lt_mask);
          if (s != kInvalid) {
            const uint32_t p = s_cnt[s] + rank;
            s_hx[p] = x;
            s_hh[p] = (uint16_t)i;
          }
          __syncwarp();
          if (s != kInvalid && rank == 0) s_cnt[s] += __popc(peers);
          __syncwarp();
        }
      }
      if (bad_id) atomicOr(a.status, (uint32_t)UT_STATUS_BAD_HIT_ID);
      __syncthreads();                             // s_cnt is dead from here on: the bins / warp areas take its place
    }
    // ---- batch order: the tracks of the item binned by radius at the first layer, inner tracks first -----------
    // Inner tracks cross the busy sectors and have the long candidate lists; a batch costs what its heaviest
    // track costs, so like goes with like and the heavy batches start first.  Results do not depend on the order
    // (the order inside a bin is whatever the atomics make it).  Bin = exponent and 3 mantissa bits of r^2.
    const uint16_t* perm = nullptr;
    if (nTk > (uint32_t)kTPW && nTk <= a.trk_stage) {
      for (uint32_t i = tid; i < (uint32_t)kBins; i += nt) s_bins[i] = 0;
      __syncthreads();
      const float dz0 = __fsub_rn(a.layer_z[0], a.vz);
      for (uint32_t m = tid; m < nTk; m += nt) {
        const uint32_t t = t0 + m * K + part;
        const float x = __ldg(a.vx + t) + __ldg(a.vtx + t) * dz0, y = __ldg(a.vy + t) + __ldg(a.vty + t) * dz0;
        const float r2 = x * x + y * y;
        int b = (int)(__float_as_uint(r2) >> 20) - 0x418;        // r = 4 mm -> bin 0, r = 1 m -> bin 127
        b = r2 == r2 ? max(0, min(kBins - 1, b)) : kBins - 1;    // NaN state: last
        s_binpos[m] = ((uint32_t)b << 16) | atomicAdd(&s_bins[b], 1u);
      }
      __syncthreads();
      if (warp == 0) {
        uint32_t c[kBins / 32], run = 0;
#pragma unroll
        for (int q = 0; q < kBins / 32; ++q) { c[q] = s_bins[lane * (kBins / 32) + q]; run += c[q]; }
        uint32_t ex = warp_incl_scan(run, lane) - run;
#pragma unroll
        for (int q = 0; q < kBins / 32; ++q) { s_bins[lane * (kBins / 32) + q] = ex; ex += c[q]; }
      }
      __syncthreads();
      for (uint32_t m = tid; m < nTk; m += nt) {
        const uint32_t bp = s_binpos[m];
        s_perm[s_bins[bp >> 16] + (bp & 0xFFFFu)] = (uint16_t)m;
      }
      perm = s_perm;
    }
    if (view) {
      mbar_wait(&s_bar, bar_phase);
      bar_phase ^= 1u;
    }
    __syncthreads();                               // order and staged data visible; scratch is dead from here on
    if (staged) {
      track_loop<true, INTERVAL, KICK, LU, CC>(a, wa, S, &s_ticket, h0, t0, nTk, part, T, perm);
    } else {                                       // event larger than the staging size: window search on global memory
      track_loop<false, INTERVAL, KICK, LU, CC>(a, wa, S, &s_ticket, h0, t0, nTk, part, T, perm);
    }
  }
  if (tid == 0) {                             // last CTA out re-arms the ticket for the next call
    __threadfence();
    if (atomicAdd(a.ticket + 1, 1u) == gridDim.x - 1) { a.ticket[0] = 0; a.ticket[1] = 0; __threadfence(); }
  }
}

static size_t compass_smem_bytes(uint32_t ns, uint32_t ng, uint32_t rows, uint32_t soff_stride, uint32_t hit_stage, int C,
                                 int block, int variant, uint32_t trk_stage = 0, uint32_t ev_stage = 0) {
  const bool lu = (variant & 3) == 1, kick = (variant & 3) == 2, interval = (variant & 4) != 0;   // kk | iv << 2
  size_t b = align16((size_t)(ng + 8) * 16) + align16((size_t)(ng + 8) * 8) + align16((size_t)rows * 32);
  b += align16((ng + 1) * 4) + align16((size_t)soff_stride * 2);
  b += align16((size_t)(hit_stage + 8) * 4) + align16((size_t)(hit_stage + 16) * 2) + align16((size_t)trk_stage * 2);
  b += align16((size_t)ev_stage * 2);
  b += std::max({align16((size_t)(block / 32) * warp_area_bytes(C, lu, interval, kick)),
                 align16((size_t)ns * 8) + 2 * align16((size_t)(hit_stage + 8) * 4),   // re-bucketing scratch aliases the warp areas
                 align16((size_t)(kBins + trk_stage) * 4),                              // and so do the radius bins
                 align16((size_t)(block / 32) * 128 + ev_stage)});                      // and the scratch of the event order
  return b;
}

// Two register budgets: CTAs of <= 224 threads at 4 per SM (72 registers), and larger CTAs (big events / C = 32,
// where shared memory allows one CTA per SM and only more warps per CTA raise the occupancy).
constexpr int kSmallBlock = 224;
constexpr int kLargeBlock = 640;             // (a 768-thread bound caps the kernel at 80 registers and it spills; 640: 84-88, none)
#define UTC_K(T, B, I, K, U) reinterpret_cast<const void*>(&compass_kernel<T, B, I, K, U>)
// [large CTAs][interval search][2: kick table, 1: layer-uniform geometry (UT_GEOM_LAYER_UNIFORM) without kick table, 0: neither]
static const void* const kKernels[2][2][3] = {
    {{UTC_K(kSmallBlock, 4, false, false, false), UTC_K(kSmallBlock, 4, false, false, true), UTC_K(kSmallBlock, 4, false, true, false)},
     {UTC_K(kSmallBlock, 4, true, false, false), UTC_K(kSmallBlock, 4, true, false, true), UTC_K(kSmallBlock, 4, true, true, false)}},
    {{UTC_K(kLargeBlock, 1, false, false, false), UTC_K(kLargeBlock, 1, false, false, true), UTC_K(kLargeBlock, 1, false, true, false)},
     {UTC_K(kLargeBlock, 1, true, false, false), UTC_K(kLargeBlock, 1, true, false, true), UTC_K(kLargeBlock, 1, true, true, false)}}};
#undef UTC_K
// the metric's configuration (small CTAs, layer-uniform geometry, C = 16) with the cap compiled in
static const void* const kKernelC16 = reinterpret_cast<const void*>(&compass_kernel<kSmallBlock, 4, false, false, true, 16>);

int32_t launch_compass(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                       const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, ut_tracks* out,
                       cudaStream_t stream, uint32_t idx_stride, unsigned long long hits_hint, uint32_t* ticket) {
  DeviceInfo dev;
  int max_smem = 0, max_smem_large = 0;               // largest dynamic size a CTA may ask for on this device
  if (const int32_t rc = device_info(&dev)) return rc;
  const ut_tuning tune = tuning_snapshot();
  const int interval_min = tuned(tune.compass_interval_min, 16);
  const int iv = cfg->max_candidates_per_layer > interval_min ? 1 : 0;    // long partner lists are possible
  // kernel variant: 2 = per-track kick from the table, 1 = layer-uniform geometry (z and weight of a candidate are its
  // layer's), 0 = the general kernel
  const int kk = hits->geom->kick_nx != 0 ? 2 : ((hits->geom->flags & UT_GEOM_LAYER_UNIFORM) ? 1 : 0);
  if (const int32_t rc = kernel_max_dynamic_smem(kKernels[0][iv][kk], kSlotCompassSmall + 3 * iv + kk, &max_smem)) return rc;
  if (const int32_t rc = kernel_max_dynamic_smem(kKernels[1][iv][kk], kSlotCompassLarge + 3 * iv + kk, &max_smem_large)) return rc;
  max_smem = std::min(max_smem, max_smem_large);
  const int n_sm = dev.n_sm, sm_smem = dev.smem_per_sm;
  const ut_geometry* geom = hits->geom;
  CompassArgs a;
  a.hx = hits->x_at_y0; a.hid = hits->id; a.hyb = hits->y_begin; a.hye = hits->y_end;
  a.hit_offsets = hit_offsets;
  a.soff_stride = (geom->n_sectors + 2u + 7u) & ~7u;
  // the per-sector view is used when all three arrays are there and 16-byte aligned (bulk copies)
  const bool view_ok = hits->x_by_sector && hits->idx_by_sector && hits->sector_offsets &&
                       ((reinterpret_cast<uintptr_t>(hits->x_by_sector) | reinterpret_cast<uintptr_t>(hits->idx_by_sector) |
                         reinterpret_cast<uintptr_t>(hits->sector_offsets)) & 15u) == 0;
  a.sx = view_ok ? hits->x_by_sector : nullptr;
  a.si = view_ok ? hits->idx_by_sector : nullptr;
  a.soff = view_ok ? hits->sector_offsets : nullptr;
  a.vx = velo->x; a.vy = velo->y; a.vtx = velo->tx; a.vty = velo->ty; a.vz = velo->z;
  a.velo_offsets = velo_offsets; a.n_events = n_events;
  a.n_sectors = geom->n_sectors; a.n_groups = geom->n_groups; a.gpl = geom->n_groups / UT_N_LAYERS;
  a.id_table_size = geom->id_table_size; a.rows_sorted = (geom->flags & UT_GEOM_ROWS_SORTED) ? 1u : 0u;
  a.rows_uniform = (geom->flags & UT_GEOM_ROWS_UNIFORM) ? geom->n_sectors / geom->n_groups : 0u;
  a.order_y = hits->order == UT_ORDER_Y ? 1u : 0u;
  a.id_to_sector = geom->id_to_sector; a.group_first_sector = geom->group_first_sector;
  a.group_xmin = geom->group_xmin; a.group_xmax = geom->group_xmax;
  a.sec_yb = geom->y_begin; a.sec_ye = geom->y_end; a.sec_dxdy = geom->dxdy; a.sec_z = geom->z; a.sec_w = geom->weight;
  for (int l = 0; l < 4; ++l) { a.layer_z[l] = geom->layer_z[l]; a.layer_dxdy[l] = geom->layer_dxdy[l]; a.layer_w[l] = geom->layer_weight[l]; }
  a.c = *cfg;
  a.kick = make_kick_table(geom);
  a.slope_lim = cfg->max_slope * (1.0f + kFilterEps);
  a.interval_min = iv ? std::min(interval_min, 8) : interval_min;     // inside the interval kernel the search pays from ~8 partners
  a.idx_stride = idx_stride;
  a.capacity = hits->capacity;
  a.bulk_ok = ((reinterpret_cast<uintptr_t>(hits->x_at_y0) | reinterpret_cast<uintptr_t>(hits->id)) & 15u) == 0 ? 1u : 0u;
  a.out_idx = out->hit_idx; a.out_n = out->n_hits; a.out_qop = out->qop; a.out_chi2 = out->chi2; a.status = out->status;
  a.ticket = ticket ? ticket : out->status + 1;      // (ut_tracks.status is 4 words: status, ticket pair, spare)

  const int C = cfg->max_candidates_per_layer;
  const uint32_t ns = geom->n_sectors, ng = geom->n_groups;
  // hits per event as far as the host can tell without a sync: capacity (or the caller's bound for this call) / events
  const unsigned long long avg = (hits_hint ? hits_hint : hits->capacity) / (unsigned long long)n_events + 1;
  // the capacity bound counts the pad half-word of every odd bank as a hit: about n_sectors / 2 per event
  const unsigned long long est = avg > ns ? avg - ns / 2 : avg;
  uint32_t hit_stage = (uint32_t)std::min<unsigned long long>(((est + est / 8 + 127) / 128) * 128 + 128, 65536ull);
  hit_stage = (uint32_t)tuned(tune.compass_hit_stage, (int)hit_stage);
  const size_t budget = (size_t)max_smem;
  // Block size: the one that keeps the most warps resident per SM (shared memory is the limit; about 24
  // warps per SM is what the register budget of the small variant allows).
  int block = tuned(tune.compass_block, 0);
  // the event order: a batch of more events than SMs and at most 4096 -- beyond that the tail of the launch is a small
  // part of it
  const uint32_t ev_fit = (n_events > n_sm && n_events <= 4096 && tune.compass_event_order != 0) ? ((uint32_t)n_events + 7u) & ~7u : 0u;
  if (block <= 0) {
    int best_warps = -1;
    for (int b = 192; b <= kLargeBlock; b += 32) {
      // (with room for the radius order of 512 tracks per item and for the event order: a block size
      //  that squeezes them out loses more than its extra warp wins -- config 4, 608 threads without the event order against
      //  576 with it: 1.300 against 1.306 ms for the 1000 events at once, but 2.31 against 2.07 ms through the host pipeline,
      //  whose chunks of 100-400 events are 1-3 waves of 148 CTAs)
      const size_t sm = compass_smem_bytes(ns, ng, a.rows_uniform, a.soff_stride, hit_stage, C, b, kk | iv << 2, 512,
                                           ev_fit) + 1024;
      if (sm > budget) continue;
      const int regs_warps = b <= kSmallBlock ? 28 : 21;       // 72 registers per thread: 4 CTAs of up to 7 warps
      const int ctas = std::min<int>((int)((size_t)sm_smem / sm), std::max(1, regs_warps / (b / 32)));
      const int warps = ctas * (b / 32);
      if (warps > best_warps) { best_warps = warps; block = b; }
    }
    if (block <= 0) block = 192;
  }
  block = std::max(32, std::min(kLargeBlock, (block / 32) * 32));
  size_t smem = compass_smem_bytes(ns, ng, a.rows_uniform, a.soff_stride, hit_stage, C, block, kk | iv << 2);
  while (smem > budget && block > 64) {             // fewer warps before giving up staging
    block -= 32;
    smem = compass_smem_bytes(ns, ng, a.rows_uniform, a.soff_stride, hit_stage, C, block, kk | iv << 2);
  }
  while (smem > budget && hit_stage > 0) {
    hit_stage = hit_stage > 1024 ? hit_stage - 1024 : 0;
    smem = compass_smem_bytes(ns, ng, a.rows_uniform, a.soff_stride, hit_stage, C, block, kk | iv << 2);
  }
  if (smem > budget) return UT_ERR_LIMIT;
  a.hit_stage = hit_stage;
  // room for ordering up to 2048 (else 1024, 512) tracks per item and, first, the events of the batch, if it costs no
  // resident CTA
  a.trk_stage = 0;
  a.ev_stage = 0;
  // (the order only matters when the batch is more than one wave of CTAs: 4 small CTAs per SM at best, one large one)
  const bool ev_useful = ev_fit != 0u && n_events > n_sm * (block <= kSmallBlock ? 4 : 1);
  for (int with_ev = ev_useful ? 1 : 0; with_ev >= 0 && a.trk_stage == 0; --with_ev) {
    for (uint32_t want = (uint32_t)tuned(tune.compass_trk_stage, 2048); want >= 512; want /= 2) {
      const uint32_t evs = with_ev ? ev_fit : 0u;
      const size_t with = compass_smem_bytes(ns, ng, a.rows_uniform, a.soff_stride, hit_stage, C, block, kk | iv << 2, want, evs);
      if (with <= budget && (size_t)sm_smem / (with + 1024) == (size_t)sm_smem / (smem + 1024)) {
        a.trk_stage = want;
        a.ev_stage = evs;
        smem = with;
        break;
      }
    }
  }
  const void* kernel = kKernels[block <= kSmallBlock ? 0 : 1][iv][kk];
  if (block <= kSmallBlock && iv == 0 && kk == 1 && C == 16 && a.rows_uniform != 0) {
    int dummy = 0;
    if (const int32_t rc = kernel_max_dynamic_smem(kKernelC16, kSlotCompassC16, &dummy)) return rc;
    kernel = kKernelC16;
  }
  int per_sm = 0;
  UTC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kernel, block, smem));
  if (per_sm < 1) return cuda_fail("compass kernel does not fit on an SM", cudaErrorInvalidConfiguration);
  // K CTAs share the tracks of an event only while whole events would leave resident CTAs idle (a 100-event batch
  // on 592 CTA slots).  Measured on a B200, config 3: K = 1 127 us, K = 2 145 us, K = 4 182 us -- a part pays the
  // event's fixed cost again (ticket, offsets, staging wait, order) and its last round of batches is emptier.
  const int resident = n_sm * per_sm;
  int split = tuned(tune.compass_split, 0);
  if (split <= 0) {
    split = 1;
    while (split < 4 && (long long)n_events * split * 2 <= resident && avg >= 256) split *= 2;
  }
  split = split >= 4 ? 4 : (split >= 2 ? 2 : 1);
  a.split = (uint32_t)split;
  if (split != 1) a.ev_stage = 0;            // (the room stays allocated, the kernel leaves the order out)
  const int grid = std::max(1, (int)std::min<long long>((long long)n_events * split, resident));
  void* params[] = {&a};
  {
    cudaLaunchConfig_t lc = {};
    lc.gridDim = dim3(grid); lc.blockDim = dim3(block); lc.dynamicSmemBytes = smem; lc.stream = stream;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    lc.attrs = at; lc.numAttrs = 1;
    UTC_CUDA(cudaLaunchKernelExC(&lc, kernel, params));
  }
  ut_launch_info& li = launch_info();
  li.kernels_launched = 1; li.compass_grid = grid; li.compass_block = block; li.compass_smem_bytes = (int)smem;
  li.compass_hit_stage = (int)hit_stage; li.compass_split = split; li.compass_view = view_ok ? 1 : 0;
  li.compass_event_order = (int)a.ev_stage;
  return UT_OK;
}

}  // namespace utc
