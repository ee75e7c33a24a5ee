// ut_decode.cu -- UT raw-bank decoding (section IV, :235-274) as ONE persistent kernel.
//
// The paper splits decoding into 7 launches (Table 1: count, 3-kernel Blelloch
// scan with a host read-back of the total, pre-decode, find permutation, decode in order).  That
// shape was made for sm_61/sm_70 and a batch of events that is tiny for a B200.
// Here one CTA owns one event at a time (dynamic ticket), keeps the event on chip and touches HBM
// once per byte:
//
//   ticket -> bank offsets (coalesced, requested before the copy below is awaited) -> raw banks of the
//      event by ONE TMA bulk copy into shared memory
//   -> thread per bank: header check, sector claim, count            (paper: "calculate number of hits")
//   -> CTA-wide exclusive prefix of the counts in dense sector order, in place: the fill order of the
//      event is (sector, word), so a group's start and size and every bank's offset fall out; the
//      event total is published at once for the chained exclusive prefix over events (decoupled
//      look-back by warp 0; paper: prefix sum + host sync; here no sync, no second launch)
//   -> while warp 0 resolves the look-back, the other warps (named barrier 1):
//        fill   thread per bank: x and (sector, word) of its words at their place in the PADDED fill
//               order (every group starts at a multiple of 4, pad slots hold +inf)   (paper: "pre-decode")
//        rank   thread per hit: one sweep over its group's x (128-bit shared loads, one FSET.BF + one
//               FADD per comparison) counts the hits with smaller x; atomicMin of the fill index into
//               slot [group start + count] of the sorted order.  Hits with equal x collide there: the
//               first in fill order keeps the slot, each later one is moved once to slot + (equal hits
//               in front of it) -- so the result is the stable sort by x         (paper: "find permutation")
//   -> output, all warps: a warp takes one sector group at a time and walks its slots of the sorted order,
//      the 7 SoA arrays by fully coalesced stores (32 consecutive elements of each array per step)
//                                                                     (paper: "decode raw banks in order")
//      and the hit's entry in the per-sector view for compass_track (ut_hits.x_by_sector ...): the fill
//      order is sector-major, so a sector's entries are a contiguous run; a hit goes behind the hits of its
//      sector that came earlier in the sorted order (running count per sector + match.any among the lanes)
//
// Events whose padded fill order does not fit the buffers, and UT_ORDER_Y containers, are ordered warp per
// sector group instead (ticket inside the CTA): gather into the warp's slice of the same buffers, rank per
// chunk of 32 hits (<= for earlier chunks, < for the rest, ties inside the chunk by match.any), groups larger
// than the slice by recomputation.  Same results on every path (tests/test_gpu_parity.py::test_decode_data_paths).
// Arithmetic of x follows include/ut_compass.h exactly (__fmul_rn/__fadd_rn, never fused).
#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <mutex>

#include "common.cuh"

namespace utc {

struct DecodeArgs {
  const uint8_t* raw;
  const uint32_t* bank_offsets;
  int32_t n_events;
  GeomDev g;
  float *x, *z, *yb, *ye, *dxdy, *w;
  uint32_t* id;
  unsigned long long capacity;
  uint32_t* status;
  uint32_t* hit_offsets;
  uint32_t* ctrl;               // [0] ticket, [1] CTAs done, [2] epoch   ([4], [5]: compass_track's event ticket)
  unsigned long long* flags;    // [n_events] look-back words: epoch:30 | state:2 | value:32
  uint32_t raw_stage_bytes;     // multiple of 16
  uint32_t hit_stage;           // largest padded event the CTA orders as a whole (0: always warp per group)
  uint32_t buf_elems;           // elements of the x / word buffers: max(hit_stage, warps * sort_buf)
  uint32_t sort_buf;            // elements of a warp's slice of those buffers on the warp-per-group path (multiple of 32)
  const uint32_t* carry_in;     // hits in front of event 0 (chunked pipeline) or null
  float* sx;                    // per-sector view (ut_hits.x_by_sector / idx_by_sector / sector_offsets) or null
  uint16_t* si;
  uint16_t* soff;
  uint32_t soff_stride;
  uint32_t order_y;             // 1: inside a group ascending (y_begin, x) -- the paper's literal order (UT_ORDER_Y)
  uint32_t view_ok;             // the per-sector view can describe this container (UT_ORDER_Y: only if a group's
                                // sectors ascend in y_begin in dense order, else its sector runs are not in dense order)
};

__device__ __forceinline__ float decode_x(uint32_t word, float x0, float pitch) {
  const uint32_t u = ((word & 0x1FFu) << 1) | ((word >> 9) & 1u);   // 2*strip + frac
  const float t = __fadd_rn(__fmul_rn((float)u, 0.5f), 0.25f);
  return __fadd_rn(x0, __fmul_rn(t, pitch));
}

__device__ __forceinline__ uint32_t ld_volatile_shared_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(smem_u32(p)) : "memory");
  return v;
}

// 1.0f when a < b (a <= b, a == b), else 0.0f: one FSET.BF, and one FADD to count it (exact below 2^24; the compiler's
// `n += a < b ? 1 : 0` is three instructions)
__device__ __forceinline__ float lt(float a, float b) {
  float d;
  asm("set.lt.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}
__device__ __forceinline__ float le(float a, float b) {
  float d;
  asm("set.le.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}
__device__ __forceinline__ float eq(float a, float b) {
  float d;
  asm("set.eq.f32.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b));
  return d;
}

// stable order of the fill sequence: (x, position in the fill order)
__device__ __forceinline__ uint32_t before(float xj, uint32_t j, float x, uint32_t i) {
  return (xj < x || (xj == x && j < i)) ? 1u : 0u;
}

__global__ void __launch_bounds__(512, 3) ut_decode_kernel(const DecodeArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t ns = a.g.n_sectors, ng = a.g.n_groups;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;

  // a dependent launch (compass_track with programmatic stream serialization) may be scheduled onto free SMs from now
  // on; it waits for this grid's completion before it reads anything written here
  asm volatile("griddepcontrol.launch_dependents;");
  Carver cv(smem_raw);
  // raw banks of the event; once every word is decoded the same bytes hold the sorted order (s_perm)
  unsigned char* s_rawstage = cv.take<unsigned char>(max(a.raw_stage_bytes, 4u * a.hit_stage));
  uint32_t* s_perm = reinterpret_cast<uint32_t*>(s_rawstage);
  uint16_t* g_gfirst = cv.take<uint16_t>(ng + 1);
  uint32_t* s_pstart = cv.take<uint32_t>(ng + 1); // start of every group in the padded fill order (multiples of 4)
  uint8_t* g_sgrp = cv.take<uint8_t>(ns);         // dense sector -> group (n_groups <= 128)
  uint32_t* s_cnt = cv.take<uint32_t>(ns + 1);    // bank word counts, then their exclusive prefix in dense sector order
  uint32_t* s_wpos = cv.take<uint32_t>(ns);
  float* s_xbuf = cv.take<float>(a.buf_elems);    // x of the event's hits in padded fill order (warp slices on the group path)
  uint32_t* s_wbuf = cv.take<uint32_t>(a.buf_elems);   // (dense sector << 16) | raw word, likewise

  __shared__ uint64_t s_bar;
  __shared__ int s_event;
  __shared__ uint32_t s_epoch, s_status, s_base, s_ready, s_gticket;
  __shared__ uint32_t s_warp[32];

  // geometry tables: staged once per CTA, reused for every event this CTA takes
  for (uint32_t i = tid; i <= ng; i += nt) g_gfirst[i] = (uint16_t)a.g.group_first_sector[i];
  for (uint32_t i = tid; i < ns; i += nt) g_sgrp[i] = (uint8_t)a.g.sector_group[i];
  if (tid == 0) {
    mbar_init(&s_bar, 1);
    fence_mbar_init();
    s_epoch = ld_volatile_u32(a.ctrl + 2);
    s_status = 0;
  }
  __syncthreads();
  uint32_t bar_phase = 0;
  const uint32_t lt_mask = (1u << lane) - 1u;
  float* xbuf = s_xbuf + (size_t)warp * a.sort_buf;
  uint32_t* wbuf = s_wbuf + (size_t)warp * a.sort_buf;

  for (;;) {
    // (drawing the ticket one event ahead was measured: 59 -> 71 us on config 3.  A CTA that holds its next event
    //  while it is still busy keeps faster CTAs from taking it.)
    if (tid == 0) s_event = (int)atomicAdd(a.ctrl, 1u);
    __syncthreads();                     // also: every warp is done with the previous event's tables
    const int e = s_event;
    if (e >= a.n_events) break;

    // ---- bank offsets of the event, table reset -------------------------------------------------------
    const uint32_t* bo = a.bank_offsets + (size_t)e * ns;
    const uint32_t b0 = __ldg(bo), b1 = __ldg(bo + ns);          // first byte and end of the event's banks
    // this thread's bank offsets are requested now and used after the raw copy has landed
    constexpr int kPre = 3;
    uint32_t o0r[kPre], o1r[kPre];
#pragma unroll
    for (int k = 0; k < kPre; ++k) {
      const uint32_t j = (uint32_t)tid + (uint32_t)k * (uint32_t)nt;
      o0r[k] = j < ns ? __ldg(bo + j) : 0u;
      o1r[k] = j < ns ? __ldg(bo + j + 1) : 0u;
    }
    for (uint32_t i = tid; i < ns; i += nt) { s_cnt[i] = 0; s_wpos[i] = kInvalid; }
    if (tid == 0) { s_ready = 0; s_gticket = 0; }
    __syncthreads();

    const uint32_t b0a = b0 & ~15u;
    const bool range_ok = b1 >= b0;
    const uint32_t span = range_ok ? (((b1 + 15u) & ~15u) - b0a) : 0u;
    const bool raw_staged = span > 0 && span <= a.raw_stage_bytes;
    const uint8_t* rawp = raw_staged ? s_rawstage : a.raw + b0a;   // rawp + (o - b0a) is byte o
    if (raw_staged) {
      if (tid == 0) {
        fence_proxy_async();                 // earlier generic-proxy reads of the stage are done (barrier above)
        mbar_expect_tx(&s_bar, span);
        bulk_g2s(s_rawstage, a.raw + b0a, span, &s_bar);
      }
      mbar_wait(&s_bar, bar_phase);
      bar_phase ^= 1u;
    }

    // ---- per bank: header check, sector claim, count ---------------------------------
    uint32_t st = range_ok ? 0u : (uint32_t)UT_STATUS_BAD_BANK_SIZE;
    if (range_ok) {
      auto bank = [&](uint32_t o0, uint32_t o1) {
        if ((o0 & 3u) || o1 < o0 + 6u || o0 < b0 || o1 > b1) { st |= UT_STATUS_BAD_BANK_SIZE; return; }
        const uint32_t rel = o0 - b0a;
        const uint32_t rid = *reinterpret_cast<const uint32_t*>(rawp + rel);
        const uint32_t cnt = *reinterpret_cast<const uint32_t*>(rawp + rel + 4) & 0xFFFFu;
        uint32_t s = kInvalid;
        if (rid < a.g.id_table_size) s = __ldg(a.g.id_to_sector + rid);   // 4 KB table, L1 / L2 resident
        if (s >= ns) { st |= UT_STATUS_UNKNOWN_SECTOR; return; }
        if (o1 - o0 != ((6u + 2u * cnt + 3u) & ~3u)) { st |= UT_STATUS_BAD_BANK_SIZE; return; }
        if (atomicCAS(&s_wpos[s], kInvalid, rel + 6u) != kInvalid) { st |= UT_STATUS_DUPLICATE_SECTOR; return; }
        s_cnt[s] = cnt;
      };
#pragma unroll
      for (int k = 0; k < kPre; ++k)
        if ((uint32_t)tid + (uint32_t)k * (uint32_t)nt < ns) bank(o0r[k], o1r[k]);
      for (uint32_t j = (uint32_t)tid + (uint32_t)kPre * (uint32_t)nt; j < ns; j += nt) bank(__ldg(bo + j), __ldg(bo + j + 1));
    }
    if (st) atomicOr(&s_status, st);
    __syncthreads();

    // ---- exclusive prefix of the bank counts in dense sector order, in place -----------------
    // The fill order of the event is (dense sector, word), so s_cnt[s] becomes the place of sector s's first word in
    // it; a group's sectors are contiguous: its start and size, and every bank's offset inside it, fall out.
    uint32_t tot;
    {
      const uint32_t per = ((ns + (uint32_t)nt - 1u) / (uint32_t)nt) | 1u;     // odd: conflict-free strided rows
      const uint32_t s0 = min((uint32_t)tid * per, ns), s1 = min(s0 + per, ns);
      uint32_t sum = 0;
      for (uint32_t q = s0; q < s1; ++q) sum += s_cnt[q];
      const uint32_t incl = warp_incl_scan(sum, lane);
      if (lane == 31) s_warp[warp] = incl;
      __syncthreads();
      const uint32_t wv = lane < nwarps ? s_warp[lane] : 0u;
      const uint32_t wi = warp_incl_scan(wv, lane);
      tot = __shfl_sync(0xFFFFFFFFu, wi, 31);
      uint32_t run = __shfl_sync(0xFFFFFFFFu, wi - wv, warp) + incl - sum;
      for (uint32_t q = s0; q < s1; ++q) { const uint32_t c = s_cnt[q]; s_cnt[q] = run; run += c; }
      if (tid == 0) s_cnt[ns] = tot;
    }
    __syncthreads();                     // last block barrier of the event: warps run on their own from here
    const uint32_t* s_start = s_cnt;

    // ---- padded fill order: every group starts at a multiple of 4 so that the rank sweep reads whole float4 rows ----
    if (warp == nwarps - 1) {
      uint32_t gp[4], run = 0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t g = lane * 4 + q;
        gp[q] = g < ng ? (s_start[g_gfirst[g + 1]] - s_start[g_gfirst[g]] + 3u) & ~3u : 0u;
        run += gp[q];
      }
      const uint32_t incl = warp_incl_scan(run, lane);
      uint32_t ex = incl - run;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t g = lane * 4 + q;
        if (g < ng) s_pstart[g] = ex;
        ex += gp[q];
      }
      if (lane == 31) s_pstart[ng] = incl;
    }
    __syncthreads();
    const uint32_t ptot = s_pstart[ng];
    // The whole event is ordered by the CTA when its padded fill order fits the buffers; otherwise (and for
    // UT_ORDER_Y) a warp takes one sector group at a time further down.
    const bool cta_path = !a.order_y && nwarps > 1 && ptot <= a.hit_stage;

    // ---- event base: warp 0 publishes the total and resolves the chained prefix over events -----------
    uint32_t base = 0;
    bool have_base = false;
    // per-sector view: usable by compass_track iff the event fits u16 positions and no group takes the generic path
    bool big = false;
    if (!cta_path)
      for (uint32_t g = lane; g < ng; g += 32u) big |= s_start[g_gfirst[g + 1]] - s_start[g_gfirst[g]] > a.sort_buf;
    const bool view = a.soff != nullptr && a.view_ok && tot <= 65535u && !__any_sync(0xFFFFFFFFu, big);
    uint16_t* soff = a.soff ? a.soff + (size_t)e * a.soff_stride : nullptr;
    if (warp == 0) {
      base = event_base_lookback(a.flags, e, tot, s_epoch, lane, a.carry_in);
      have_base = true;
      if (lane == 0) {
        s_base = base;
        __threadfence_block();
        *reinterpret_cast<volatile uint32_t*>(&s_ready) = 1u;
        if ((unsigned long long)base + tot > a.capacity) atomicOr(&s_status, (uint32_t)UT_STATUS_CAPACITY);
        if (e == a.n_events - 1) a.hit_offsets[(size_t)a.n_events * ng] = base + tot;
        if (soff) {
          soff[ns] = (uint16_t)tot;
          soff[ns + 1] = (view && (unsigned long long)base + tot <= a.capacity) ? (uint16_t)UT_SECTOR_INDEX_VALID : (uint16_t)0;
        }
      }
      for (uint32_t g = lane; g < ng; g += 32u) a.hit_offsets[(size_t)e * ng + g] = base + s_start[g_gfirst[g]];
    }
    if (tot == 0 && !view) continue;

    if (cta_path) {
      // Warp 0 is busy with the look-back; the other warps ("workers", named barrier 1) fill, clear and rank.
      const uint32_t nw = (uint32_t)nt - 32u;
      if (warp != 0) {
        const uint32_t wt = (uint32_t)tid - 32u;
        // x order: a sector's run of the view starts where its words start in the fill order
        if (view)
          for (uint32_t q = wt; q < ns; q += nw) soff[q] = (uint16_t)s_start[q];
        // ---- fill: thread per bank, x and (sector, word) of its words at their place in the padded fill order
        //      (paper: "pre-decode")
        for (uint32_t sct = wt; sct < ns; sct += nw) {
          const uint32_t es = s_start[sct], c = s_start[sct + 1] - es;
          if (c == 0) continue;
          const uint32_t g = g_sgrp[sct];
          const uint32_t p0 = s_pstart[g] + (es - s_start[g_gfirst[g]]);
          const float2 xp = __ldg(reinterpret_cast<const float2*>(a.g.sector_rows + 2 * sct + 1) + 1);      // {x0, pitch}
          const uint16_t* wd = reinterpret_cast<const uint16_t*>(rawp + s_wpos[sct]);
          for (uint32_t k = 0; k < c; ++k) {
            const uint32_t word = wd[k];
            s_xbuf[p0 + k] = decode_x(word, xp.x, xp.y);
            s_wbuf[p0 + k] = (sct << 16) | word;
          }
        }
        for (uint32_t g = wt; g < ng; g += nw) {          // pad slots: +inf is never "smaller", kInvalid marks them
          const uint32_t n = s_start[g_gfirst[g + 1]] - s_start[g_gfirst[g]];
          for (uint32_t q = s_pstart[g] + n; q < s_pstart[g + 1]; ++q) { s_xbuf[q] = __int_as_float(0x7F800000); s_wbuf[q] = kInvalid; }
        }
        asm volatile("bar.sync 1, %0;" ::"r"(nw) : "memory");      // every word is decoded: the raw bytes are dead
        for (uint32_t q = wt; q < ptot; q += nw) s_perm[q] = kInvalid;
        for (uint32_t q = wt; q < ns; q += nw) s_wpos[q] = 0;       // (word positions are dead too: per-sector counters of the output)
        asm volatile("bar.sync 1, %0;" ::"r"(nw) : "memory");
        // ---- rank: thread per hit, one sweep over its group counts the hits with smaller x ("find permutation",
        //      PAPER.md:273).  Hits with equal x get the same count: the first of them in fill order keeps the slot
        //      (atomicMin), each of the others is moved once to slot + (equal hits in front of it).
        for (uint32_t pi = wt; pi < ptot; pi += nw) {
          const uint32_t rw = s_wbuf[pi];
          if (rw == kInvalid) continue;
          const float x = s_xbuf[pi];
          const uint32_t g = g_sgrp[rw >> 16];
          const uint32_t pga = s_pstart[g], pge = s_pstart[g + 1];
          float r0 = 0.f, r1 = 0.f;
#pragma unroll 2                                     // (measured: 4 as the compiler picks 58.0 us, 2: 57.0, 1: 57.3; config 4 same at 2)
          for (uint32_t j = pga; j < pge; j += 4u) {
            const float4 v = *reinterpret_cast<const float4*>(s_xbuf + j);
            r0 += lt(v.x, x); r1 += lt(v.y, x);
            r0 += lt(v.z, x); r1 += lt(v.w, x);
          }
          const uint32_t rank = (uint32_t)(r0 + r1);
          const uint32_t old = atomicMin(&s_perm[pga + rank], pi);
          if (old != kInvalid) {                            // equal x: re-home the later one of the two
            const uint32_t later = max(old, pi);
            float o0 = 0.f, o1 = 0.f;
            uint32_t j = pga;
            for (; j + 4u <= later; j += 4u) {
              const float4 v = *reinterpret_cast<const float4*>(s_xbuf + j);
              o0 += eq(v.x, x); o1 += eq(v.y, x);
              o0 += eq(v.z, x); o1 += eq(v.w, x);
            }
            for (; j < later; ++j) o0 += eq(s_xbuf[j], x);
            s_perm[pga + rank + (uint32_t)(o0 + o1)] = later;
          }
        }
      }
      __syncthreads();                                       // order complete, base known
      base = s_base;
      if ((unsigned long long)base + tot > a.capacity) continue;        // flagged by warp 0; offsets stay exact
      // ---- output: a warp takes one sector group at a time (ticket) and walks its slots of the sorted order, 32 per
      //      step: coalesced SoA stores ("decode raw banks in order").  The per-sector view entry of a hit
      //      goes behind the hits of its sector that came earlier in the sorted order: a running count per sector
      //      (s_wpos, zeroed above) plus the rank among the lanes of the same sector (match.any).
      for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = atomicAdd(&s_gticket, 1u);
        g = __shfl_sync(0xFFFFFFFFu, g, 0);
        if (g >= ng) break;
        const uint32_t pga = s_pstart[g], gfs = s_start[g_gfirst[g]], n = s_start[g_gfirst[g + 1]] - gfs;
        for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
          const bool valid = c0 + lane < n;
          const uint32_t pi = valid ? s_perm[pga + c0 + lane] : 0u;
          const uint32_t rw = valid ? s_wbuf[pi] : 0xFFFFFFFFu, sct = rw >> 16;
          const uint32_t peers = __match_any_sync(0xFFFFFFFFu, sct);
          const uint32_t ahead = __popc(peers & lt_mask);
          if (valid) {
            const float x = s_xbuf[pi];
            const uint32_t hpos = gfs + c0 + lane;             // place in the event's part of the container
            const float4 A = __ldg(a.g.sector_rows + 2 * sct), B = __ldg(a.g.sector_rows + 2 * sct + 1);
            const size_t P = (size_t)base + hpos;
            a.x[P] = x; a.z[P] = A.x; a.yb[P] = A.y; a.ye[P] = A.z; a.dxdy[P] = A.w; a.w[P] = B.x;
            a.id[P] = (__float_as_uint(B.y) << 9) | (rw & 0x1FFu);
            if (view) {
              const uint32_t seen = s_wpos[sct];
              const size_t Q = (size_t)base + s_start[sct] + seen + ahead;
              a.sx[Q] = x;
              a.si[Q] = (uint16_t)hpos;
              if (n > 32u) {                                   // (a one-step group never reads the count again)
                __syncwarp(peers);
                if (ahead == 0) s_wpos[sct] = seen + __popc(peers);
              }
            }
          }
          __syncwarp();
        }
      }
      continue;
    }
    // x order: a sector's run of the view starts where its words start in the fill order
    if (view && !a.order_y)
      for (uint32_t q = tid; q < ns; q += nt) soff[q] = (uint16_t)s_start[q];

    // ---- warp per sector group (ticket inside the CTA) --------------------------------------------------
    for (;;) {
      uint32_t g = 0;
      if (lane == 0) g = atomicAdd(&s_gticket, 1u);
      g = __shfl_sync(0xFFFFFFFFu, g, 0);
      if (g >= ng) break;
      const uint32_t sa = g_gfirst[g], sb = g_gfirst[g + 1], nsec = sb - sa;   // nsec <= 32 (ut_geometry_upload)
      const uint32_t gstart = s_start[sa], n = s_start[sb] - gstart;
      if (n == 0) {
        if (view && a.order_y && (uint32_t)lane < nsec) soff[sa + lane] = (uint16_t)gstart;
        continue;
      }
      // the group's banks: word position, word count and offset inside the group's fill order, one bank per lane
      const uint32_t wpos_r = (uint32_t)lane < nsec ? s_wpos[sa + lane] : 0u;
      const uint32_t e_r = (uint32_t)lane < nsec ? s_start[sa + lane] - gstart : n;   // lanes past the group: never selected
      const uint32_t cnt_r = (uint32_t)lane < nsec ? s_start[sa + lane + 1] - gstart - e_r : 0u;
      if (a.order_y) {
        // ---- UT_ORDER_Y: sectors in (y_begin, dense index) order, x-sorted inside a sector.  A hit's
        // place = its sector's start in that order + its rank among the words of its own bank: no group-wide rank.
        const uint32_t yo = (uint32_t)lane < nsec ? __ldg(a.g.sector_yorder + sa + lane) : 0u;
        const uint32_t cnt_y = __shfl_sync(0xFFFFFFFFu, cnt_r, (int)((yo >> 8) & 31u));     // count of the lane-th sector in y order
        const uint32_t cy = (uint32_t)lane < nsec ? cnt_y : 0u;
        const uint32_t ey_k = warp_incl_scan(cy, lane) - cy;
        const uint32_t ey_r = __shfl_sync(0xFFFFFFFFu, ey_k, (int)(yo & 31u));               // start of THIS lane's sector
        if (view && (uint32_t)lane < nsec) soff[sa + lane] = (uint16_t)(gstart + ey_r);
        if (!have_base) {
          while (ld_volatile_shared_u32(&s_ready) == 0u) {}
          __threadfence_block();
          base = *reinterpret_cast<volatile uint32_t*>(&s_base);
          have_base = true;
        }
        if ((unsigned long long)base + tot > a.capacity) continue;
        const size_t P0 = (size_t)base + gstart;
        for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
          const uint32_t i = c0 + lane;
          int r = 0;                                    // largest r with e_r <= i (fill order -> sector, word)
#pragma unroll
          for (int step = 16; step > 0; step >>= 1) {
            const uint32_t ev = __shfl_sync(0xFFFFFFFFu, e_r, r + step);
            if (ev <= i) r += step;
          }
          const uint32_t k = i - __shfl_sync(0xFFFFFFFFu, e_r, r);
          const uint32_t wp = __shfl_sync(0xFFFFFFFFu, wpos_r, r);
          const uint32_t cs = __shfl_sync(0xFFFFFFFFu, cnt_r, r);
          const uint32_t ey = __shfl_sync(0xFFFFFFFFu, ey_r, r);
          if (i < n) {
            const uint32_t s = sa + (uint32_t)r;
            const float4 A = __ldg(a.g.sector_rows + 2 * s), B = __ldg(a.g.sector_rows + 2 * s + 1);
            const uint32_t word = *reinterpret_cast<const uint16_t*>(rawp + wp + 2u * k);
            const float x = decode_x(word, B.z, B.w);
            uint32_t pos = 0;
            for (uint32_t k2 = 0; k2 < cs; ++k2)
              pos += before(decode_x(*reinterpret_cast<const uint16_t*>(rawp + wp + 2u * k2), B.z, B.w), k2, x, k);
            const size_t Q = P0 + ey + pos;
            a.x[Q] = x; a.z[Q] = A.x; a.yb[Q] = A.y; a.ye[Q] = A.z; a.dxdy[Q] = A.w; a.w[Q] = B.x;
            a.id[Q] = (__float_as_uint(B.y) << 9) | (word & 0x1FFu);
            if (view) { a.sx[Q] = x; a.si[Q] = (uint16_t)(gstart + ey + pos); }
          }
        }
        continue;
      }
      if (n <= a.sort_buf) {
        // ---- gather: element i of the fill order -> (sector r, word k); x and the word go to the warp's buffer ----
        for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
          const uint32_t i = c0 + lane;
          int r = 0;                                    // largest r with e_r <= i
#pragma unroll
          for (int step = 16; step > 0; step >>= 1) {
            const uint32_t ev = __shfl_sync(0xFFFFFFFFu, e_r, r + step);
            if (ev <= i) r += step;
          }
          const uint32_t k = i - __shfl_sync(0xFFFFFFFFu, e_r, r);
          const uint32_t wp = __shfl_sync(0xFFFFFFFFu, wpos_r, r);
          if (i < n) {
            const uint32_t word = *reinterpret_cast<const uint16_t*>(rawp + wp + 2u * k);
            const float2 xp = __ldg(reinterpret_cast<const float2*>(a.g.sector_rows + 2 * (sa + r) + 1) + 1);   // {x0, pitch}
            xbuf[i] = decode_x(word, xp.x, xp.y);
            wbuf[i] = ((uint32_t)r << 16) | word;       // (sector in group, raw word)
          }
        }
        const uint32_t npad = (n + 3u) & ~3u;           // pad the tail of the buffer with +inf (never "smaller")
        if (n + lane < npad) xbuf[n + lane] = __int_as_float(0x7F800000);
        __syncwarp();
        if (!have_base) {                               // the event's base is needed from here on
          while (ld_volatile_shared_u32(&s_ready) == 0u) {}
          __threadfence_block();
          base = *reinterpret_cast<volatile uint32_t*>(&s_base);
          have_base = true;
        }
        if ((unsigned long long)base + tot > a.capacity) continue;      // flagged by warp 0; offsets stay exact
        const size_t P0 = (size_t)base + gstart;
        // ---- rank = place in the stable order (x, fill index): one sweep over the buffer per chunk of 32 hits.
        // Earlier chunks win ties (<=), the own and later chunks never (<); ties inside the chunk by one match.any.
        for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
          const uint32_t i = c0 + lane;
          const bool valid = i < n;
          const float xi = valid ? xbuf[i] : __int_as_float(0x7F800000);
          float r0 = 0.f, r1 = 0.f;
          for (uint32_t j = 0; j < c0; j += 4u) {
            const float4 v = *reinterpret_cast<const float4*>(xbuf + j);
            r0 += le(v.x, xi); r1 += le(v.y, xi);
            r0 += le(v.z, xi); r1 += le(v.w, xi);
          }
          for (uint32_t j = c0; j < npad; j += 4u) {
            const float4 v = *reinterpret_cast<const float4*>(xbuf + j);
            r0 += lt(v.x, xi); r1 += lt(v.y, xi);
            r0 += lt(v.z, xi); r1 += lt(v.w, xi);
          }
          const uint32_t ties = __match_any_sync(0xFFFFFFFFu, __float_as_uint(xi + 0.0f));      // -0 == +0
          const uint32_t rank = (uint32_t)(r0 + r1) + __popc(ties & lt_mask);
          const uint32_t rwi = valid ? wbuf[i] : 0u;
          const uint32_t es = __shfl_sync(0xFFFFFFFFu, e_r, (int)(rwi >> 16));
          const uint32_t cs = __shfl_sync(0xFFFFFFFFu, cnt_r, (int)(rwi >> 16));
          if (valid) {
            const uint32_t s = sa + (rwi >> 16);
            const float4 A = __ldg(a.g.sector_rows + 2 * s), B = __ldg(a.g.sector_rows + 2 * s + 1);
            const size_t P = P0 + rank;
            a.x[P] = xi; a.z[P] = A.x; a.yb[P] = A.y; a.ye[P] = A.z; a.dxdy[P] = A.w; a.w[P] = B.x;
            a.id[P] = (__float_as_uint(B.y) << 9) | (rwi & 0x1FFu);
            if (view) {
              // per-sector view: the fill order is sector-major, so the sector's words are elements [es, es + cs) of
              // the buffer; the place inside the sector's run is the rank among them
              uint32_t pos = 0;
              for (uint32_t j = es; j < es + cs; ++j) pos += before(xbuf[j], j, xi, i);
              const size_t Q = P0 + es + pos;
              a.sx[Q] = xi;
              a.si[Q] = (uint16_t)(gstart + rank);
            }
          }
        }
        __syncwarp();                                   // the buffer is reused by the warp's next group
      } else {
        // ---- generic path (group larger than the sort buffer): rank by recomputation, O(n^2) --------------
        if (!have_base) {
          while (ld_volatile_shared_u32(&s_ready) == 0u) {}
          __threadfence_block();
          base = *reinterpret_cast<volatile uint32_t*>(&s_base);
          have_base = true;
        }
        if ((unsigned long long)base + tot > a.capacity) continue;
        const size_t P0 = (size_t)base + gstart;
        for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
          const uint32_t i = c0 + lane;
          int r = 0;
#pragma unroll
          for (int step = 16; step > 0; step >>= 1) {
            const uint32_t ev = __shfl_sync(0xFFFFFFFFu, e_r, r + step);
            if (ev <= i) r += step;
          }
          const uint32_t k = i - __shfl_sync(0xFFFFFFFFu, e_r, r);
          const uint32_t wp = __shfl_sync(0xFFFFFFFFu, wpos_r, r);
          const bool valid = i < n;
          uint32_t word = 0;
          float xi = 0.f;
          if (valid) {
            word = *reinterpret_cast<const uint16_t*>(rawp + wp + 2u * k);
            const float4 Bx = __ldg(a.g.sector_rows + 2 * (sa + r) + 1);
            xi = decode_x(word, Bx.z, Bx.w);
          }
          uint32_t rank = 0, j = 0;
          for (uint32_t r2 = 0; r2 < nsec; ++r2) {      // warp-uniform walk over the fill order
            const uint32_t c2 = __shfl_sync(0xFFFFFFFFu, cnt_r, (int)r2);
            const uint32_t w2 = __shfl_sync(0xFFFFFFFFu, wpos_r, (int)r2);
            const float4 Bx2 = __ldg(a.g.sector_rows + 2 * (sa + r2) + 1);
            const float2 xp2 = make_float2(Bx2.z, Bx2.w);
            for (uint32_t k2 = 0; k2 < c2; ++k2, ++j)
              rank += before(decode_x(*reinterpret_cast<const uint16_t*>(rawp + w2 + 2u * k2), xp2.x, xp2.y), j, xi, i);
          }
          if (valid) {
            const uint32_t s = sa + (uint32_t)r;
            const float4 A = __ldg(a.g.sector_rows + 2 * s), B = __ldg(a.g.sector_rows + 2 * s + 1);
            const size_t P = P0 + rank;
            a.x[P] = xi; a.z[P] = A.x; a.yb[P] = A.y; a.ye[P] = A.z; a.dxdy[P] = A.w; a.w[P] = B.x;
            a.id[P] = (__float_as_uint(B.y) << 9) | (word & 0x1FFu);
          }
        }
      }
    }
  }

  if (tid == 0) {
    if (s_status) atomicOr(a.status, s_status);
    __threadfence();
    const uint32_t done = atomicAdd(a.ctrl + 1, 1u);
    if (done == gridDim.x - 1) {          // last CTA out re-arms the workspace for the next call
      a.ctrl[0] = 0;
      a.ctrl[1] = 0;
      __threadfence();
      a.ctrl[2] = s_epoch + 1u;
    }
  }
}

static size_t decode_smem_bytes(uint32_t ns, uint32_t ng, uint32_t raw_stage, uint32_t hit_stage, uint32_t buf_elems) {
  size_t b = align16(std::max<size_t>(raw_stage, 4 * (size_t)hit_stage));
  b += align16((size_t)(ng + 1) * 2) + align16((size_t)(ng + 1) * 4) + align16((size_t)ns);
  b += align16((size_t)(ns + 1) * 4) + align16((size_t)ns * 4);
  b += 2 * align16((size_t)buf_elems * 4);
  return b;
}

int32_t launch_decode(const uint8_t* raw, const uint32_t* bank_offsets, int32_t n_events, const ut_geometry* geom,
                      ut_hits* hits, uint32_t* hit_offsets, cudaStream_t stream, const uint32_t* carry_in,
                      unsigned long long hits_hint) {
  DeviceInfo dev;
  int max_smem = 0;                      // largest dynamic size this kernel may ask for on this device
  if (const int32_t rc = device_info(&dev)) return rc;
  if (const int32_t rc = kernel_max_dynamic_smem(reinterpret_cast<const void*>(&ut_decode_kernel), kSlotDecode, &max_smem))
    return rc;
  const int n_sm = dev.n_sm;
  const ut_tuning tune = tuning_snapshot();
  DecodeArgs a;
  a.raw = raw; a.bank_offsets = bank_offsets; a.n_events = n_events; a.g = make_geom_dev(geom);
  a.x = hits->x_at_y0; a.z = hits->z_at_y0; a.yb = hits->y_begin; a.ye = hits->y_end; a.dxdy = hits->dxdy;
  a.w = hits->weight; a.id = hits->id; a.capacity = hits->capacity; a.status = hits->status;
  a.hit_offsets = hit_offsets;
  a.carry_in = carry_in;
  a.sx = hits->x_by_sector; a.si = hits->idx_by_sector; a.soff = hits->sector_offsets;
  a.soff_stride = (geom->n_sectors + 2u + 7u) & ~7u;
  a.order_y = hits->order == UT_ORDER_Y ? 1u : 0u;
  a.view_ok = (!a.order_y || (geom->flags & UT_GEOM_ROWS_SORTED)) ? 1u : 0u;
  a.ctrl = reinterpret_cast<uint32_t*>(hits->workspace);
  a.flags = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(hits->workspace) + 32);

  // staging sizes from the only size the host knows without a sync: capacity / n_events
  const uint32_t ns = geom->n_sectors, ng = geom->n_groups;
  const unsigned long long avg = (hits_hint ? hits_hint : hits->capacity) / (unsigned long long)n_events + 1;
  const unsigned long long stage_hits = std::min<unsigned long long>(((avg + 255) / 256) * 256 + 256, 1u << 16);
  uint32_t raw_stage = (uint32_t)align16(8u * ns + 2u * stage_hits + 32u);
  raw_stage = (uint32_t)tuned(tune.decode_raw_stage_bytes, (int)raw_stage) & ~15u;
  // the capacity bound counts the pad half-word of every odd bank as a hit: about n_sectors / 2 per event
  const unsigned long long est = avg > ns ? avg - ns / 2 : avg;
  // 12 warps order an event together (measured on config 3: 256 threads 72 us, 384 59 us, 512 63 us); busy events get 16
  int block = tuned(tune.decode_block, avg > 4096 ? 512 : 384);
  block = std::max(64, std::min(512, (block / 32) * 32));
  const uint32_t nwarps = (uint32_t)block / 32u;
  // the warp-per-group path (UT_ORDER_Y, oversize events) slices the same buffers: twice the mean group, at least 64
  uint32_t sort_buf = (uint32_t)std::min<unsigned long long>(((2 * avg / ng + 31) / 32) * 32 + 32, 1024);
  sort_buf = std::max(64u, sort_buf);
  sort_buf = ((uint32_t)tuned(tune.decode_sort_buf, (int)sort_buf) + 31u) & ~31u;
  const size_t budget = (size_t)max_smem;
  // CTA-wide order: the event's padded fill order (<= 3 pad slots per group) with 1/8 (else 1/16) of slack; the smaller
  // slack is taken when it lets one more CTA stay resident
  auto stage_for = [&](unsigned long long slack_div, unsigned long long slack_min) {
    return (uint32_t)std::min<unsigned long long>(((est + est / slack_div + slack_min + 3ull * ng + 31) / 32) * 32, 1u << 16);
  };
  uint32_t hit_stage = stage_for(8, 128);
  if (hits->order == UT_ORDER_Y) hit_stage = 0;
  else if (tune.decode_hit_stage >= 0) hit_stage = ((uint32_t)tune.decode_hit_stage + 31u) & ~31u;
  else {
    const uint32_t tight = stage_for(16, 64);
    const size_t s8 = decode_smem_bytes(ns, ng, raw_stage, hit_stage, std::max(hit_stage, nwarps * sort_buf)) + 1024;
    const size_t s16 = decode_smem_bytes(ns, ng, raw_stage, tight, std::max(tight, nwarps * sort_buf)) + 1024;
    if ((size_t)dev.smem_per_sm / s16 > (size_t)dev.smem_per_sm / s8 || s8 - 1024 > budget) hit_stage = tight;
  }
  auto smem_of = [&]() { return decode_smem_bytes(ns, ng, raw_stage, hit_stage, std::max(hit_stage, nwarps * sort_buf)); };
  size_t smem = smem_of();
  if (smem > budget && tune.decode_hit_stage < 0) { hit_stage = 0; smem = smem_of(); }   // events too large to order as a whole
  while (smem > budget && raw_stage > 4096) {            // oversize events read their banks from global memory
    raw_stage = (raw_stage / 2) & ~15u;
    smem = smem_of();
  }
  while (smem > budget && sort_buf > 32) {
    sort_buf -= 32;
    smem = smem_of();
  }
  while (smem > budget && hit_stage > 0) {
    hit_stage = hit_stage > 1024 ? hit_stage - 1024 : 0;
    smem = smem_of();
  }
  if (smem > budget) return UT_ERR_LIMIT;
  a.raw_stage_bytes = raw_stage; a.hit_stage = hit_stage;
  a.buf_elems = std::max(hit_stage, nwarps * sort_buf);
  if (tune.decode_sort_buf < 0) sort_buf = std::min(1024u, (a.buf_elems / nwarps) & ~31u);   // the slices take what is there
  a.sort_buf = sort_buf;

  int per_sm = 0;
  UTC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ut_decode_kernel, block, smem));
  if (per_sm < 1) return cuda_fail("decode kernel does not fit on an SM", cudaErrorInvalidConfiguration);
  per_sm = std::min(per_sm, std::max(1, tuned(tune.decode_max_ctas_per_sm, 8)));
  const int grid = std::max(1, std::min(n_events, n_sm * per_sm));
  ut_decode_kernel<<<grid, block, smem, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  ut_launch_info& li = launch_info();
  li.kernels_launched = 1; li.decode_grid = grid; li.decode_block = block; li.decode_smem_bytes = (int)smem;
  li.decode_raw_stage_bytes = (int)raw_stage; li.decode_sort_buf = (int)sort_buf; li.decode_hit_stage = (int)hit_stage;
  return UT_OK;
}

// ---- ut_decode_static: the decode kernel's workspace in a file-scope device array (include/ut_compass.h) ----------
// Layout as ut_decode_workspace_bytes(): 8 control words, one look-back word per event, 8 spare bytes.  Zero at module
// load, which is the state ut_decode_workspace_init() produces.  One instance per GPU that loads the library.
constexpr size_t kStaticWorkspaceBytes = (32 + 8 * (size_t)UT_DECODE_STATIC_MAX_EVENTS + 8 + 255) / 256 * 256;
static __device__ __align__(256) unsigned char g_static_workspace[kStaticWorkspaceBytes];

// In host code `g_static_workspace` is only a handle for the runtime, never a device address: the address of this
// device's instance comes from cudaGetSymbolAddress, asked once per device with that device current.
static int32_t static_workspace(void** out) {
  constexpr int kMaxDev = 64;
  static std::mutex mu;
  static void* ptrs[kMaxDev] = {};
  int dev = -1;
  UTC_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) return fail_with(UT_ERR_LIMIT, "ut_decode_static: device ordinal above 63");
  std::lock_guard<std::mutex> lock(mu);
  if (!ptrs[dev]) {
    void* p = nullptr;
    UTC_CUDA(cudaGetSymbolAddress(&p, g_static_workspace));
    if (!p) return fail_with(UT_ERR_CUDA, "ut_decode_static: cudaGetSymbolAddress returned a null address");
    ptrs[dev] = p;
  }
  *out = ptrs[dev];
  return UT_OK;
}

}  // namespace utc

extern "C" int32_t ut_decode_static(const uint8_t* raw_banks, const uint32_t* bank_offsets, int32_t n_events,
                                    const ut_geometry* geometry, ut_hits* hits_out, uint32_t* hit_offsets_out,
                                    ut_stream_t stream) {
  if (!hits_out) return UT_ERR_NULL;
  if (n_events > UT_DECODE_STATIC_MAX_EVENTS) {
    char text[160];
    snprintf(text, sizeof(text), "ut_decode_static: n_events = %d exceeds UT_DECODE_STATIC_MAX_EVENTS = %d (use ut_decode "
             "with a caller-owned workspace)", (int)n_events, (int)UT_DECODE_STATIC_MAX_EVENTS);
    return utc::fail_with(UT_ERR_LIMIT, text);
  }
  void* ws = nullptr;
  if (const int32_t rc = utc::static_workspace(&ws)) return rc;
  // The array keeps what the last call left in it.  [0] ticket and [1] CTAs done must start at zero (the kernel's last
  // CTA re-arms them, a call that was cut short would not have); [2], the epoch, is kept: it tags the look-back words,
  // so those of earlier calls read as "not written yet".
  if (n_events > 0) UTC_CUDA(cudaMemsetAsync(ws, 0, 8, (cudaStream_t)stream));
  ut_hits h = *hits_out;                       // the caller's container with the built-in workspace in place of its own
  h.workspace = ws;
  const int32_t rc = ut_decode(raw_banks, bank_offsets, n_events, geometry, &h, hit_offsets_out, stream);
  if (rc == UT_OK) hits_out->geom = h.geom;    // (what ut_decode records in the container)
  return rc;
}
