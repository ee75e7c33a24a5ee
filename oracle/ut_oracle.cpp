// ut_oracle.cpp -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
// A plain, slow, single-threaded C++17 implementation of what the hot path of
// arxiv/paper_2002_11529 computes: UT raw-bank decoding into an x-sorted SoA hit
// container (section IV, :235-274) and Compass tracking (section V,
// :276-348), in the reading fixed by SURVEY.md section 8(c) / DESIGN.md section 3.
//
//   * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
//     reference legs may call this.  The product (paper_2002_11529_b200/) never does.
//   * Shares no code, header, table generator or helper with the CUDA path.
//   * Arithmetic: fp32, round-to-nearest, operations in exactly the written order,
//     no FMA contraction (build with -ffp-contract=off), IEEE division (A14;
//     PAPER.md:444 "single precision").  Decode = the plain definition; Compass = the
//     algorithm step by step.
//   * Pins (tests/, -m "not gpu"): raw-format round trip, count invariants, closed-form
//     x for X layers, sort invariants, windowed == linear-scan candidate lists (BF-1),
//     seeded search == exhaustive enumeration (BF-2), fit == weighted lstsq in double,
//     collinear chi2 = 0, q/p sign == generated charge, truth recovery on isolated
//     noise-free tracks, monotonicity in C / min_hits, permutation equivariance.
//     Absolute efficiency values against the paper's Table 3 are "parity unpinned"
//     (they need the LHCb Monte-Carlo).
//
// Build: g++ -std=c++17 -O2 -ffp-contract=off -fPIC -shared ut_oracle.cpp -o liboracle.so

#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>

extern "C" {

// Host-resident geometry tables (the synthetic stand-in for PAPER.md:274 "geometry and
// panel information from the subdetector").
struct oracle_geometry {
  uint32_t n_layers, n_sectors, n_groups, id_table_size;
  const uint32_t* id_to_sector;     // [id_table_size], 0xFFFFFFFF = invalid
  const uint32_t* sector_raw_id;    // [n_sectors]
  const uint32_t* sector_group;     // [n_sectors], non-decreasing
  const float *x0, *pitch, *dxdy, *z, *y_begin, *y_end, *weight;   // [n_sectors]
  const float *group_xmin, *group_xmax;                            // [n_groups]
  float layer_z[4], layer_dxdy[4];
  // optional position-dependent kick table; kick_nx == 0: constant kick
  uint32_t kick_nx, kick_ny;
  float kick_x_lo, kick_y_lo, kick_inv_dx, kick_inv_dy, kick_z_ref;
  const float *kick_kappa, *kick_z_mag;                            // [kick_ny * kick_nx]
};

struct oracle_hits {                // SoA container of PAPER.md:243-254
  float *x_at_y0, *z_at_y0, *y_begin, *y_end, *dxdy, *weight;
  uint32_t* id;
  uint64_t capacity;
};

struct oracle_config {              // same fields as synth.CompassParams
  float win_half[4];
  float y_tol, max_slope, kink_tol, seed_tol, w_velo, max_chi2_ndf, kappa, z_mag;
  int32_t min_hits, max_candidates_per_layer;
  int32_t both_directions;          // 0: backward only if forward found nothing (A11); 1: best of forward and backward
};

// status bits (data-dependent errors), same meaning as include/ut_compass.h
enum : uint32_t {
  ST_UNKNOWN_SECTOR = 1u, ST_DUPLICATE_SECTOR = 2u, ST_BAD_BANK_SIZE = 4u, ST_CAPACITY = 8u,
};

static inline uint16_t rd16(const uint8_t* p) { return (uint16_t)(p[0] | (p[1] << 8)); }
static inline uint32_t rd32(const uint8_t* p) {
  return (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24);
}

// ---------------------------------------------------------------------------------------
// Decode: the plain definition.
// For event e, every bank, every word k -> one hit
//   strip = w & 0x1FF, frac = (w >> 9) & 1                       (ADC = w >> 10 ignored)
//   x   = x0[s] + ((2*strip + frac) * 0.5 + 0.25) * pitch[s]     (fp32, RN, no FMA; A3)
//   z, y_begin, y_end, dxdy, weight copied from the sector row   (A5)
//   id  = (raw_sector_id << 9) | strip                           (LHCbID)
// Output order: events ascending; groups ascending; inside a group ascending x, ties by
// (dense sector, k) (stable sort of the fill order).  hit_offsets = exclusive prefix of
// group sizes, n_events*n_groups + 1 entries.
// ---------------------------------------------------------------------------------------
// order = 1 ("sort the hits by Y coordinate ... within the sector group";
// DESIGN.md A1/A25): inside a group ascending y_begin, then ascending x, ties still in fill order.
int32_t oracle_decode(const uint8_t* raw, const uint32_t* bank_offsets, int32_t n_events,
                      const oracle_geometry* g, oracle_hits* out, uint32_t* hit_offsets,
                      uint32_t* status, int32_t order) {
  if (!bank_offsets || !g || !out || !hit_offsets || n_events < 0) return -1;
  const uint32_t ns = g->n_sectors, ng = g->n_groups;
  uint32_t st = 0;
  uint64_t total = 0;
  struct Bank { const uint8_t* words; uint32_t count; bool seen; };
  struct Hit { float x; uint32_t s; uint32_t strip; };
  std::vector<Bank> banks(ns);
  std::vector<Hit> grp;
  for (int32_t e = 0; e < n_events; ++e) {
    for (auto& b : banks) b = Bank{nullptr, 0, false};
    // the event's byte range: from its first bank offset to the first offset of the next event (or the end)
    const uint64_t ev_begin = bank_offsets[(uint64_t)e * ns], ev_end = bank_offsets[(uint64_t)(e + 1) * ns];
    for (uint32_t j = 0; j < ns; ++j) {
      const uint64_t o0 = bank_offsets[(uint64_t)e * ns + j], o1 = bank_offsets[(uint64_t)e * ns + j + 1];
      // DESIGN.md A22 (raw format of BASELINE.json configs[0] / SURVEY.md 8(d): banks are padded to 4 bytes and the
      // banks of an event are contiguous): a bank that does not start on a 4-byte boundary, is shorter than its
      // 6-byte header or does not lie inside [ev_begin, ev_end) is malformed -> ignored and flagged
      if ((o0 & 3u) != 0 || o1 < o0 + 6 || o0 < ev_begin || o1 > ev_end) { st |= ST_BAD_BANK_SIZE; continue; }
      const uint32_t rid = rd32(raw + o0);
      const uint32_t cnt = rd16(raw + o0 + 4);
      const uint32_t s = rid < g->id_table_size ? g->id_to_sector[rid] : 0xFFFFFFFFu;
      if (s >= ns) { st |= ST_UNKNOWN_SECTOR; continue; }
      if (o1 - o0 != ((6ull + 2ull * cnt + 3ull) & ~3ull)) { st |= ST_BAD_BANK_SIZE; continue; }
      if (banks[s].seen) { st |= ST_DUPLICATE_SECTOR; continue; }
      banks[s] = Bank{raw + o0 + 6, cnt, true};
    }
    uint64_t ev_total = 0;
    for (uint32_t s = 0; s < ns; ++s) ev_total += banks[s].count;
    const bool fits = total + ev_total <= out->capacity;
    if (!fits) st |= ST_CAPACITY;
    uint32_t s = 0;
    for (uint32_t grp_i = 0; grp_i < ng; ++grp_i) {
      hit_offsets[(uint64_t)e * ng + grp_i] = (uint32_t)total;
      grp.clear();
      for (; s < ns && g->sector_group[s] == grp_i; ++s) {
        for (uint32_t k = 0; k < banks[s].count; ++k) {
          const uint32_t w = rd16(banks[s].words + 2 * k);
          const uint32_t strip = w & 0x1FFu, frac = (w >> 9) & 1u;
          const float t = (float)(2 * strip + frac) * 0.5f + 0.25f;
          const float tp = t * g->pitch[s];
          const float x = g->x0[s] + tp;
          grp.push_back(Hit{x, s, strip});
        }
      }
      if (order == 1)
        std::stable_sort(grp.begin(), grp.end(), [g](const Hit& a, const Hit& b) {
          const float ya = g->y_begin[a.s], yb = g->y_begin[b.s];
          return ya < yb || (ya == yb && a.x < b.x);
        });
      else
        std::stable_sort(grp.begin(), grp.end(), [](const Hit& a, const Hit& b) { return a.x < b.x; });
      if (fits) {
        for (size_t i = 0; i < grp.size(); ++i) {
          const uint64_t p = total + i;
          const uint32_t sc = grp[i].s;
          out->x_at_y0[p] = grp[i].x;
          out->z_at_y0[p] = g->z[sc];
          out->y_begin[p] = g->y_begin[sc];
          out->y_end[p] = g->y_end[sc];
          out->dxdy[p] = g->dxdy[sc];
          out->weight[p] = g->weight[sc];
          out->id[p] = (g->sector_raw_id[sc] << 9) | grp[i].strip;
        }
      }
      total += grp.size();
    }
  }
  hit_offsets[(uint64_t)n_events * ng] = (uint32_t)total;
  if (status) *status = st;
  return 0;
}

// ---------------------------------------------------------------------------------------
// Compass.
// ---------------------------------------------------------------------------------------
struct Cand { int32_t h; float d, z, w; };

static const float GROUP_EPS = 0.01f;   // mm, slack of the group pre-selection (A17)

struct HitsView {
  const float *x, *z, *yb, *ye, *dxdy, *w;
};

static inline float resid(const HitsView& H, int64_t h, float x_e, float y_e) {
  const float sy = H.dxdy[h] * y_e;          // d_h = (x_at_y0[h] + dxdy[h]*y_e) - x_e
  const float xh = H.x[h] + sy;
  return xh - x_e;
}
static inline bool y_ok(const HitsView& H, int64_t h, float y_e, float y_tol) {
  return (H.yb[h] - y_tol <= y_e) && (y_e <= H.ye[h] + y_tol);
}

// SURVEY.md 8(f) row 4 / DESIGN.md A24 ("look-up tables ... the influence of the magnetic field"):
// the track's kick strength and kick plane from the table cell that holds its straight-line position at z_ref
// (nearest cell, no interpolation; a NaN coordinate takes cell 0).  Without a table: the config's constants.
static inline int lut_index(float v, float lo, float inv, uint32_t n) {
  const float u = (v - lo) * inv;
  if (!(u == u)) return 0;
  const float f = std::floor(u);
  if (f < 0.f) return 0;
  if (f > (float)(n - 1)) return (int)n - 1;
  return (int)f;
}
static oracle_config track_config(const oracle_geometry* g, const oracle_config* c, float vx, float vy, float vtx,
                                  float vty, float vz) {
  oracle_config ct = *c;
  if (g->kick_nx == 0) return ct;
  const float dzr = g->kick_z_ref - vz;
  const float xk = vx + vtx * dzr, yk = vy + vty * dzr;
  const int cell = lut_index(yk, g->kick_y_lo, g->kick_inv_dy, g->kick_ny) * (int)g->kick_nx +
                   lut_index(xk, g->kick_x_lo, g->kick_inv_dx, g->kick_nx);
  ct.kappa = g->kick_kappa[cell];
  ct.z_mag = g->kick_z_mag[cell];
  return ct;
}

// step 2 (+3): candidate list of one layer.  mode 0 = windowed (group pre-selection + binary
// search on the monotone predicate), mode 1 = linear scan of the whole layer.
static void layer_candidates(int mode, const HitsView& H, const uint32_t* goff /* event's group offsets */,
                             const oracle_geometry* g, int l, float x_e, float y_e,
                             const oracle_config* c, std::vector<Cand>& out, int32_t* n_before_cap) {
  out.clear();
  const float D = c->win_half[l];
  const uint32_t gpl = g->n_groups / g->n_layers;
  if (mode == 0) {
    const float sy = g->layer_dxdy[l] * y_e;
    const float ctr = x_e - sy;
    const float lo = (ctr - D) - GROUP_EPS, hi = (ctr + D) + GROUP_EPS;
    for (uint32_t gi = l * gpl; gi < (l + 1) * gpl; ++gi) {
      if (!(g->group_xmax[gi] >= lo && g->group_xmin[gi] <= hi)) continue;
      int64_t a = goff[gi], b = goff[gi + 1];
      int64_t first = a, n = b - a;                 // lower bound of "d >= -D"
      while (n > 0) {
        const int64_t half = n / 2, mid = first + half;
        if (resid(H, mid, x_e, y_e) >= -D) n = half; else { first = mid + 1; n -= half + 1; }
      }
      for (int64_t h = first; h < b; ++h) {
        const float d = resid(H, h, x_e, y_e);
        if (!(d <= D)) break;
        if (y_ok(H, h, y_e, c->y_tol)) out.push_back(Cand{(int32_t)h, d, H.z[h], H.w[h]});
      }
    }
  } else if (mode == 3) {
    // Y-sorted groups: the groups the x window can touch, in each "two binary searches over the Y
    // axis, one to delimit the beginning of the region and another to delimit the end of it", then "the window
    // range is refined by checking the hits".  The searches need y_begin and y_end non-decreasing along the group,
    // which the (y_begin, x) order gives when the sector rows do not nest.
    const float sy = g->layer_dxdy[l] * y_e;
    const float ctr = x_e - sy;
    const float lo = (ctr - D) - GROUP_EPS, hi = (ctr + D) + GROUP_EPS;
    for (uint32_t gi = l * gpl; gi < (l + 1) * gpl; ++gi) {
      if (!(g->group_xmax[gi] >= lo && g->group_xmin[gi] <= hi)) continue;
      int64_t first = goff[gi], n = (int64_t)goff[gi + 1] - first;      // first hit with y_e <= y_end + y_tol
      while (n > 0) {
        const int64_t half = n / 2, mid = first + half;
        if (y_e <= H.ye[mid] + c->y_tol) n = half; else { first = mid + 1; n -= half + 1; }
      }
      int64_t last = first;                                              // first hit with y_begin - y_tol > y_e
      n = (int64_t)goff[gi + 1] - last;
      while (n > 0) {
        const int64_t half = n / 2, mid = last + half;
        if (H.yb[mid] - c->y_tol > y_e) n = half; else { last = mid + 1; n -= half + 1; }
      }
      for (int64_t h = first; h < last; ++h) {
        const float d = resid(H, h, x_e, y_e);
        if (std::fabs(d) <= D && y_ok(H, h, y_e, c->y_tol)) out.push_back(Cand{(int32_t)h, d, H.z[h], H.w[h]});
      }
    }
  } else {
    for (int64_t h = goff[l * gpl]; h < (int64_t)goff[(l + 1) * gpl]; ++h) {
      const float d = resid(H, h, x_e, y_e);
      if (std::fabs(d) <= D && y_ok(H, h, y_e, c->y_tol)) out.push_back(Cand{(int32_t)h, d, H.z[h], H.w[h]});
    }
  }
  if (n_before_cap) *n_before_cap = (int32_t)out.size();
  const size_t C = (size_t)c->max_candidates_per_layer;
  if (out.size() > C) {                             // step 3: keep the C closest in (|d|, h)
    std::sort(out.begin(), out.end(), [](const Cand& a, const Cand& b) {
      const float fa = std::fabs(a.d), fb = std::fabs(b.d);
      return fa < fb || (fa == fb && a.h < b.h);
    });
    out.resize(C);
    std::sort(out.begin(), out.end(), [](const Cand& a, const Cand& b) { return a.h < b.h; });
  }
}

struct Tracklet {
  int n = 0;
  float chi2 = 0.f, qop = 0.f;
  int32_t h[4] = {-1, -1, -1, -1};
  bool valid = false;
};

// step 6: weighted linear LSQ of d vs dz = z - z_mag with a VELO pseudo-point (0, 0, w_velo).
static Tracklet fit(const Cand* const hit[4] /* per layer, null = none */, const oracle_config* c) {
  Tracklet t;
  float S0 = c->w_velo, S1 = 0.f, S2 = 0.f, T0 = 0.f, T1 = 0.f;
  for (int l = 0; l < 4; ++l) {
    if (!hit[l]) continue;
    const float w = hit[l]->w, d = hit[l]->d;
    const float dz = hit[l]->z - c->z_mag;
    const float wdz = w * dz;
    S0 = S0 + w;
    S1 = S1 + wdz;
    S2 = S2 + wdz * dz;
    const float wd = w * d;
    T0 = T0 + wd;
    T1 = T1 + wd * dz;
    t.h[l] = hit[l]->h;
    ++t.n;
  }
  const float det = S0 * S2 - S1 * S1;
  const float a = (T0 * S2 - T1 * S1) / det;
  const float b = (T1 * S0 - T0 * S1) / det;
  float chi2 = (c->w_velo * a) * a;
  for (int l = 0; l < 4; ++l) {
    if (!hit[l]) continue;
    const float dz = hit[l]->z - c->z_mag;
    const float r = (hit[l]->d - a) - b * dz;
    chi2 = chi2 + (hit[l]->w * r) * r;
  }
  t.chi2 = chi2;
  t.qop = b / c->kappa;
  t.valid = chi2 <= c->max_chi2_ndf * (float)(t.n - 1);
  return t;
}

// step 7 ordering: n desc, chi2 asc, (h0,h1,h2,h3) asc with none = INT32_MAX
static bool better(const Tracklet& a, const Tracklet& b) {
  if (a.n != b.n) return a.n > b.n;
  if (a.chi2 != b.chi2) return a.chi2 < b.chi2;
  for (int l = 0; l < 4; ++l) {
    const int32_t x = a.h[l] < 0 ? std::numeric_limits<int32_t>::max() : a.h[l];
    const int32_t y = b.h[l] < 0 ? std::numeric_limits<int32_t>::max() : b.h[l];
    if (x != y) return x < y;
  }
  return false;
}

struct Best {
  Tracklet best;
  float runner_chi2 = std::numeric_limits<float>::infinity();   // 2nd lowest chi2 among valid with same n
  int n_fits = 0;
  void offer(const Tracklet& t) {
    ++n_fits;
    if (!t.valid) return;
    if (!best.valid) { best = t; return; }
    if (better(t, best)) {
      if (t.n == best.n) runner_chi2 = best.chi2; else runner_chi2 = std::numeric_limits<float>::infinity();
      best = t;
    } else if (t.n == best.n && t.chi2 < runner_chi2) {
      runner_chi2 = t.chi2;
    }
  }
};

// step 7, choice between the directions.  Paper reading A11 (both == 0): forward's result if it has one, else
// backward's.  SURVEY.md 8(f) row 4 (both == 1): the better of the two in the same total order; a tracklet both
// directions found (same hits, same fit) counts once.
static Best combine_directions(const Best& fwd, const Best& bwd, bool both) {
  if (!both) { Best r = fwd.best.valid ? fwd : bwd; r.n_fits = fwd.n_fits + bwd.n_fits; return r; }
  Best r;
  if (!fwd.best.valid) r = bwd;
  else if (!bwd.best.valid) r = fwd;
  else {
    bool same = true;
    for (int l = 0; l < 4; ++l) same = same && fwd.best.h[l] == bwd.best.h[l];
    const bool take_bwd = !same && better(bwd.best, fwd.best);
    r = take_bwd ? bwd : fwd;
    const Best& other = take_bwd ? fwd : bwd;
    if (same) r.runner_chi2 = std::min(fwd.runner_chi2, bwd.runner_chi2);
    else if (other.best.n == r.best.n) r.runner_chi2 = std::min(r.runner_chi2, other.best.chi2);
  }
  r.n_fits = fwd.n_fits + bwd.n_fits;
  return r;
}

// seed predicates of step 5
static inline bool seed_ok(const Cand& a, const Cand& b, const oracle_config* c, float* bs_out) {
  const float bs = (b.d - a.d) / (b.z - a.z);
  const float a0 = a.d - bs * (a.z - c->z_mag);
  *bs_out = bs;
  return std::fabs(bs) <= c->max_slope && std::fabs(a0) <= c->kink_tol;
}
static inline bool compat(const Cand& a, float bs, const Cand& x, const oracle_config* c) {
  const float pred = a.d + bs * (x.z - a.z);
  return std::fabs(x.d - pred) <= c->seed_tol;
}

// step 5: one direction.  LA, LB = seed layers, LC, LD = the other two.
static void search_direction(const std::vector<Cand> cand[4], int LA, int LB, int LC, int LD,
                             const oracle_config* c, Best& best) {
  std::vector<const Cand*> cc, dd;
  for (const Cand& a : cand[LA]) {
    for (const Cand& b : cand[LB]) {
      float bs;
      if (!seed_ok(a, b, c, &bs)) continue;
      cc.clear(); dd.clear();
      cc.push_back(nullptr); dd.push_back(nullptr);       // "none"
      for (const Cand& x : cand[LC]) if (compat(a, bs, x, c)) cc.push_back(&x);
      for (const Cand& x : cand[LD]) if (compat(a, bs, x, c)) dd.push_back(&x);
      for (const Cand* pc : cc) {
        for (const Cand* pd : dd) {
          const int n = 2 + (pc ? 1 : 0) + (pd ? 1 : 0);
          if (n < c->min_hits) continue;
          const Cand* hit[4] = {nullptr, nullptr, nullptr, nullptr};
          hit[LA] = &a; hit[LB] = &b; hit[LC] = pc; hit[LD] = pd;
          best.offer(fit(hit, c));
        }
      }
    }
  }
}

// mode 0: windowed candidates + seeded search (the algorithm, x-sorted groups);
// mode 3: the same on Y-sorted groups (binary searches over Y);
// mode 1: linear-scan candidates + seeded search (BF-1; any order inside the groups);
// mode 2: linear-scan candidates, NO cap, exhaustive loop over every (h0|none, h1|none, h2|none,
//         h3|none) combination under the same predicates (BF-2; tiny events only).
// Optional outputs (may be null): runner_chi2 [T], cand_n [T*4] pre-cap counts,
// cand_list [T*4*C] post-cap candidate hit indices padded with -1, n_fits [T].
int32_t oracle_compass(int32_t mode, const oracle_hits* hits, const uint32_t* hit_offsets,
                       const float* vx, const float* vy, const float* vtx, const float* vty, float vz,
                       const uint32_t* velo_offsets, int32_t n_events, const oracle_geometry* g,
                       const oracle_config* c, int32_t* out_hit_idx /* [4][T] */, int32_t* out_n_hits,
                       float* out_qop, float* out_chi2, float* runner_chi2, int32_t* cand_n,
                       int32_t* cand_list, int32_t* n_fits, int64_t out_stride /* T of out_hit_idx rows; <=0: velo_offsets[n_events] */) {
  if (!hits || !hit_offsets || !velo_offsets || !g || !c || n_events < 0) return -1;
  if (g->n_layers != 4 || (c->min_hits != 3 && c->min_hits != 4) || c->max_candidates_per_layer < 1) return -2;
  const HitsView H{hits->x_at_y0, hits->z_at_y0, hits->y_begin, hits->y_end, hits->dxdy, hits->weight};
  const int64_t T = out_stride > 0 ? out_stride : (int64_t)velo_offsets[n_events];
  const int C = c->max_candidates_per_layer;
  std::vector<Cand> cand[4];
  for (int32_t e = 0; e < n_events; ++e) {
    const uint32_t* goff = hit_offsets + (uint64_t)e * g->n_groups;
    for (int64_t t = velo_offsets[e]; t < (int64_t)velo_offsets[e + 1]; ++t) {
      int nonempty = 0;
      for (int l = 0; l < 4; ++l) {
        const float dzv = g->layer_z[l] - vz;              // step 1: straight-line extrapolation
        const float x_e = vx[t] + vtx[t] * dzv;
        const float y_e = vy[t] + vty[t] * dzv;
        int32_t nb = 0;
        if (mode == 2) {
          oracle_config nocap = *c;
          nocap.max_candidates_per_layer = std::numeric_limits<int32_t>::max();
          layer_candidates(1, H, goff, g, l, x_e, y_e, &nocap, cand[l], &nb);
        } else {
          layer_candidates(mode, H, goff, g, l, x_e, y_e, c, cand[l], &nb);
        }
        if (!cand[l].empty()) ++nonempty;
        if (cand_n) cand_n[t * 4 + l] = nb;
        if (cand_list && mode != 2)
          for (int i = 0; i < C; ++i)
            cand_list[(t * 4 + l) * C + i] = i < (int)cand[l].size() ? cand[l][i].h : -1;
      }
      Best result;
      int fits = 0;
      const oracle_config ct = track_config(g, c, vx[t], vy[t], vtx[t], vty[t], vz);   // kick of THIS track (A24)
      if (nonempty >= c->min_hits) {                        // step 4
        if (mode != 2) {
          Best fwd, bwd;
          search_direction(cand, 0, 2, 1, 3, &ct, fwd);     // forward seeds (L0, L2)
          if (c->both_directions || !fwd.best.valid)        // A11: backward only if forward found nothing valid
            search_direction(cand, 3, 1, 2, 0, &ct, bwd);
          result = combine_directions(fwd, bwd, c->both_directions != 0);
          fits = result.n_fits;
        } else {
          // exhaustive: every combination, each tested against the predicates of its direction
          Best dir[2];
          const int LA[2] = {0, 3}, LB[2] = {2, 1}, LC[2] = {1, 2}, LD[2] = {3, 0};
          int64_t idx[4];
          for (idx[0] = -1; idx[0] < (int64_t)cand[0].size(); ++idx[0])
            for (idx[1] = -1; idx[1] < (int64_t)cand[1].size(); ++idx[1])
              for (idx[2] = -1; idx[2] < (int64_t)cand[2].size(); ++idx[2])
                for (idx[3] = -1; idx[3] < (int64_t)cand[3].size(); ++idx[3]) {
                  const Cand* hit[4];
                  int n = 0;
                  for (int l = 0; l < 4; ++l) { hit[l] = idx[l] < 0 ? nullptr : &cand[l][idx[l]]; n += hit[l] != nullptr; }
                  if (n < c->min_hits) continue;
                  for (int dct = 0; dct < 2; ++dct) {
                    const Cand *a = hit[LA[dct]], *b = hit[LB[dct]];
                    if (!a || !b) continue;
                    float bs;
                    if (!seed_ok(*a, *b, &ct, &bs)) continue;
                    if (hit[LC[dct]] && !compat(*a, bs, *hit[LC[dct]], &ct)) continue;
                    if (hit[LD[dct]] && !compat(*a, bs, *hit[LD[dct]], &ct)) continue;
                    dir[dct].offer(fit(hit, &ct));
                  }
                }
          result = combine_directions(dir[0], dir[1], c->both_directions != 0);
          fits = result.n_fits;
        }
      }
      const Tracklet& b = result.best;
      for (int l = 0; l < 4; ++l) out_hit_idx[(int64_t)l * T + t] = b.valid ? b.h[l] : -1;
      out_n_hits[t] = b.valid ? b.n : 0;
      out_qop[t] = b.valid ? b.qop : 0.f;
      out_chi2[t] = b.valid ? b.chi2 : 0.f;
      if (runner_chi2) runner_chi2[t] = b.valid ? result.runner_chi2 : std::numeric_limits<float>::infinity();
      if (n_fits) n_fits[t] = fits;
    }
  }
  return 0;
}

// ---------------------------------------------------------------------------------------
// the paper's two-kernel layout (Fig. 7) as plain definitions.
//
// "Search UT windows": per VELO track and panel (layer), the sector group the extrapolation
// points to and its neighbours (W = 1, 3 or 5 groups in all: the central one, then -1, +1, -2, +2; PAPER.md:300,
// :332); in each the window range = the hits of the group's x-sorted run with |d| <= win_half[l], found by two
// searches on the monotone residual and nothing else ("only two pointers to the hits").  The y
// test is left to the tracklet step ("has to still be performed again in the tracking kernel").
// Stored as Fig. 7 draws it: per track, per panel, W begin indices then W sizes, signed 16-bit, the begin
// relative to the first hit of the track's event; an empty or missing range is (-1, -1).
// Central group (A23): the first group of the layer with group_xmax >= c, c = x_e - layer_dxdy*y_e
// (the last group if there is none).  Events of more than 32767 hits cannot be indexed by a short: all their
// ranges are (-1, -1) and status bit 32 is set.
// ---------------------------------------------------------------------------------------
static int central_group(const oracle_geometry* g, int l, float c) {
  const int gpl = (int)(g->n_groups / g->n_layers);
  for (int k = 0; k < gpl; ++k)
    if (g->group_xmax[l * gpl + k] >= c) return l * gpl + k;
  return l * gpl + gpl - 1;
}
static int slot_group(const oracle_geometry* g, int l, int central, int k) {      // k-th range: 0, -1, +1, -2, +2
  const int gpl = (int)(g->n_groups / g->n_layers);
  const int off = k == 0 ? 0 : (k % 2 == 1 ? -((k + 1) / 2) : k / 2);
  const int gi = central + off;
  return (gi < l * gpl || gi >= (l + 1) * gpl) ? -1 : gi;
}

int32_t oracle_search_windows(const oracle_hits* hits, const uint32_t* hit_offsets, const float* vx, const float* vy,
                              const float* vtx, const float* vty, float vz, const uint32_t* velo_offsets,
                              int32_t n_events, const oracle_geometry* g, const oracle_config* c, int32_t W,
                              int16_t* windows /* [T][4][2W] */, uint32_t* status) {
  if (!hits || !hit_offsets || !velo_offsets || !g || !c || !windows || n_events < 0) return -1;
  if (W != 1 && W != 3 && W != 5) return -2;
  const HitsView H{hits->x_at_y0, hits->z_at_y0, hits->y_begin, hits->y_end, hits->dxdy, hits->weight};
  uint32_t st = 0;
  for (int32_t e = 0; e < n_events; ++e) {
    const uint32_t* goff = hit_offsets + (uint64_t)e * g->n_groups;
    const int64_t ev0 = goff[0], ev1 = goff[g->n_groups];
    const bool too_large = ev1 - ev0 > 32767;
    if (too_large) st |= 32u;
    for (int64_t t = velo_offsets[e]; t < (int64_t)velo_offsets[e + 1]; ++t) {
      for (int l = 0; l < 4; ++l) {
        int16_t* w = windows + (t * 4 + l) * 2 * W;
        const float dzv = g->layer_z[l] - vz;
        const float x_e = vx[t] + vtx[t] * dzv;
        const float y_e = vy[t] + vty[t] * dzv;
        const float D = c->win_half[l];
        const float sy = g->layer_dxdy[l] * y_e;
        const int central = central_group(g, l, x_e - sy);
        for (int k = 0; k < W; ++k) {
          w[k] = -1; w[W + k] = -1;
          const int gi = slot_group(g, l, central, k);
          if (gi < 0 || too_large) continue;
          int64_t first = goff[gi], n = (int64_t)goff[gi + 1] - first;        // first hit with d >= -D
          while (n > 0) {
            const int64_t half = n / 2, mid = first + half;
            if (resid(H, mid, x_e, y_e) >= -D) n = half; else { first = mid + 1; n -= half + 1; }
          }
          int64_t last = first;                                                // first hit with d > D
          n = (int64_t)goff[gi + 1] - last;
          while (n > 0) {
            const int64_t half = n / 2, mid = last + half;
            if (resid(H, mid, x_e, y_e) > D) n = half; else { last = mid + 1; n -= half + 1; }
          }
          if (last > first) { w[k] = (int16_t)(first - ev0); w[W + k] = (int16_t)(last - first); }
        }
      }
    }
  }
  if (status) *status = st;
  return 0;
}

// "Tracklet finding" from stored window ranges: the candidates of a layer are the hits of its
// W ranges that pass the y test, capped and ordered as step 3; steps 4-7 as oracle_compass.
int32_t oracle_compass_from_windows(const oracle_hits* hits, const uint32_t* hit_offsets, const float* vx,
                                    const float* vy, const float* vtx, const float* vty, float vz,
                                    const uint32_t* velo_offsets, int32_t n_events, const oracle_geometry* g,
                                    const oracle_config* c, int32_t W, const int16_t* windows, int32_t* out_hit_idx,
                                    int32_t* out_n_hits, float* out_qop, float* out_chi2, int32_t* cand_n /* [T][4] or null */) {
  if (!hits || !hit_offsets || !velo_offsets || !g || !c || !windows || n_events < 0) return -1;
  if ((W != 1 && W != 3 && W != 5) || (c->min_hits != 3 && c->min_hits != 4) || c->max_candidates_per_layer < 1) return -2;
  const HitsView H{hits->x_at_y0, hits->z_at_y0, hits->y_begin, hits->y_end, hits->dxdy, hits->weight};
  const int64_t T = velo_offsets[n_events];
  std::vector<Cand> cand[4];
  for (int32_t e = 0; e < n_events; ++e) {
    const int64_t ev0 = hit_offsets[(uint64_t)e * g->n_groups];
    for (int64_t t = velo_offsets[e]; t < (int64_t)velo_offsets[e + 1]; ++t) {
      int nonempty = 0;
      for (int l = 0; l < 4; ++l) {
        const int16_t* w = windows + (t * 4 + l) * 2 * W;
        const float dzv = g->layer_z[l] - vz;
        const float x_e = vx[t] + vtx[t] * dzv;
        const float y_e = vy[t] + vty[t] * dzv;
        cand[l].clear();
        for (int k = 0; k < W; ++k) {
          if (w[W + k] <= 0) continue;                                       // (-1, -1): no hits
          for (int64_t h = ev0 + w[k]; h < ev0 + w[k] + w[W + k]; ++h) {
            const float d = resid(H, h, x_e, y_e);
            if (std::fabs(d) <= c->win_half[l] && y_ok(H, h, y_e, c->y_tol)) cand[l].push_back(Cand{(int32_t)h, d, H.z[h], H.w[h]});
          }
        }
        std::sort(cand[l].begin(), cand[l].end(), [](const Cand& a, const Cand& b) { return a.h < b.h; });
        if (cand_n) cand_n[t * 4 + l] = (int32_t)cand[l].size();
        const size_t C = (size_t)c->max_candidates_per_layer;
        if (cand[l].size() > C) {                                           // step 3
          std::sort(cand[l].begin(), cand[l].end(), [](const Cand& a, const Cand& b) {
            const float fa = std::fabs(a.d), fb = std::fabs(b.d);
            return fa < fb || (fa == fb && a.h < b.h);
          });
          cand[l].resize(C);
          std::sort(cand[l].begin(), cand[l].end(), [](const Cand& a, const Cand& b) { return a.h < b.h; });
        }
        if (!cand[l].empty()) ++nonempty;
      }
      Best result;
      const oracle_config ct = track_config(g, c, vx[t], vy[t], vtx[t], vty[t], vz);
      if (nonempty >= c->min_hits) {
        Best fwd, bwd;
        search_direction(cand, 0, 2, 1, 3, &ct, fwd);
        if (c->both_directions || !fwd.best.valid) search_direction(cand, 3, 1, 2, 0, &ct, bwd);
        result = combine_directions(fwd, bwd, c->both_directions != 0);
      }
      const Tracklet& b = result.best;
      for (int l = 0; l < 4; ++l) out_hit_idx[(int64_t)l * T + t] = b.valid ? b.h[l] : -1;
      out_n_hits[t] = b.valid ? b.n : 0;
      out_qop[t] = b.valid ? b.qop : 0.f;
      out_chi2[t] = b.valid ? b.chi2 : 0.f;
    }
  }
  return 0;
}

// The fit alone, for the lstsq / collinear pins: n points (layer order), returns a, b, chi2.
int32_t oracle_fit(int32_t n, const float* d, const float* z, const float* w, const oracle_config* c,
                   float* a_out, float* b_out, float* chi2_out, float* qop_out) {
  if (n < 1 || n > 4) return -1;
  Cand cs[4];
  const Cand* hit[4] = {nullptr, nullptr, nullptr, nullptr};
  for (int i = 0; i < n; ++i) { cs[i] = Cand{i, d[i], z[i], w[i]}; hit[i] = &cs[i]; }
  const Tracklet t = fit(hit, c);
  // recompute a, b the same way for reporting
  float S0 = c->w_velo, S1 = 0.f, S2 = 0.f, T0 = 0.f, T1 = 0.f;
  for (int i = 0; i < n; ++i) {
    const float dz = z[i] - c->z_mag, wdz = w[i] * dz, wd = w[i] * d[i];
    S0 = S0 + w[i]; S1 = S1 + wdz; S2 = S2 + wdz * dz; T0 = T0 + wd; T1 = T1 + wd * dz;
  }
  const float det = S0 * S2 - S1 * S1;
  *a_out = (T0 * S2 - T1 * S1) / det;
  *b_out = (T1 * S0 - T0 * S1) / det;
  *chi2_out = t.chi2;
  *qop_out = t.qop;
  return 0;
}

// Compacted VELO+UT tracks: the plain definition.  Walk the events in
// order and the VELO tracks of each event in order; every track with a tracklet (n_hits > 0) is appended.
// track_offsets[e] = number of tracklets in front of event e.  Nothing past `capacity` is written (status 8),
// the offsets stay exact.  hit_idx in has row stride T, hit_idx_out row stride `capacity`.
int32_t oracle_consolidate(const int32_t* hit_idx, const int32_t* n_hits, const float* qop, const float* chi2,
                           const uint32_t* velo_offsets, int32_t n_events, uint32_t* velo_index_out,
                           int32_t* hit_idx_out, int32_t* n_hits_out, float* qop_out, float* chi2_out,
                           uint64_t capacity, uint32_t* track_offsets, uint32_t* status) {
  const uint64_t T = velo_offsets[n_events];
  uint64_t k = 0;
  for (int32_t e = 0; e < n_events; ++e) {
    track_offsets[e] = (uint32_t)k;
    for (uint64_t t = velo_offsets[e]; t < velo_offsets[e + 1]; ++t) {
      if (n_hits[t] <= 0) continue;
      if (k < capacity) {
        velo_index_out[k] = (uint32_t)t;
        for (int l = 0; l < 4; ++l) hit_idx_out[(uint64_t)l * capacity + k] = hit_idx[(uint64_t)l * T + t];
        n_hits_out[k] = n_hits[t];
        qop_out[k] = qop[t];
        chi2_out[k] = chi2[t];
      } else {
        *status |= 8u;
      }
      ++k;
    }
  }
  track_offsets[n_events] = (uint32_t)k;
  return 0;
}

}  // extern "C"
