// ut_decode.cu -- UT raw-bank decoding (section IV, :235-274) as ONE persistent kernel.
//
// The paper splits decoding into 7 launches (Table 1: count, 3-kernel Blelloch
// scan with a host read-back of the total, pre-decode, find permutation, decode in order).  That
// shape was made for sm_61/sm_70 and a batch of events that is tiny for a B200.
// Here one CTA owns one event at a time (dynamic ticket), keeps the event on chip and touches HBM
// once per byte:
//
//   ticket -> bank offsets (coalesced) -> raw banks of the event by ONE TMA bulk copy into smem
//   -> thread per bank: header check, sector claim, count   (paper: "calculate number of hits")
//   -> event total published at once for the chained exclusive prefix over events (decoupled
//      look-back by warp 0; paper: prefix sum + host sync; here no sync, no second launch); the
//      event's base is only awaited in front of the first store
//   -> warp per sector group (dynamic ticket inside the CTA): the lanes gather the group's words
//      from its banks in fill order (sector, word), decode x, and rank them -- for <= 32 hits in
//      registers with shuffles, else through a per-warp shared-memory buffer.  Lane order is the
//      tie-break order, so the rank IS the stable sort by x   (paper: pre-decode + find permutation)
//   -> SoA store at base + group start + rank; a group is one contiguous window of every array
//                                                            (paper: decode raw banks in order)
//   -> optional per-sector view for compass_track (ut_hits.x_by_sector ...): the same warp re-emits the group's x
//      and container index bucketed per sector (the fill order IS sector-major, so a sector's entries are a
//      contiguous run and the position inside the run is the rank among the sector's own hits)
//
// There is no block barrier after the count: warps run independently through the groups.
// Events or groups that do not fit the staging sizes take slower generic code with the same results.
// Arithmetic of x follows include/ut_compass.h exactly (__fmul_rn/__fadd_rn, never fused).
#include <algorithm>
#include <cstdio>
#include <cstdlib>

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
  uint32_t sort_buf;            // elements of the per-warp sort buffer (multiple of 32)
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

// stable order of the fill sequence: (x, position in the fill order)
__device__ __forceinline__ uint32_t before(float xj, uint32_t j, float x, uint32_t i) {
  return (xj < x || (xj == x && j < i)) ? 1u : 0u;
}

// Rank of this lane's x among the 32 lanes of the warp in the stable order (x, lane): lanes that hold no
// element pass +inf and are never counted.  32 unrolled shuffles for "smaller", one match.any for the ties.
__device__ __forceinline__ uint32_t warp_rank(float x, uint32_t lt_mask) {
  uint32_t rank = 0;
#pragma unroll
  for (int j = 0; j < 32; ++j) rank += __shfl_sync(0xFFFFFFFFu, x, j) < x ? 1u : 0u;
  const uint32_t ties = __match_any_sync(0xFFFFFFFFu, __float_as_uint(x + 0.0f));      // -0 == +0
  return rank + __popc(ties & lt_mask);
}

__global__ void __launch_bounds__(512) ut_decode_kernel(const DecodeArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t ns = a.g.n_sectors, ng = a.g.n_groups;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;

  Carver cv(smem_raw);
  unsigned char* s_rawstage = cv.take<unsigned char>(a.raw_stage_bytes);
  uint16_t* g_gfirst = cv.take<uint16_t>(ng + 1);
  uint32_t* s_cnt = cv.take<uint32_t>(ns);
  uint32_t* s_wpos = cv.take<uint32_t>(ns);
  uint32_t* s_gcnt = cv.take<uint32_t>(ng);
  float* s_xbuf = cv.take<float>((size_t)nwarps * a.sort_buf);
  uint32_t* s_wbuf = cv.take<uint32_t>((size_t)nwarps * a.sort_buf);

  __shared__ uint64_t s_bar;
  __shared__ int s_event;
  __shared__ uint32_t s_epoch, s_status, s_base, s_ready, s_gticket;
  __shared__ uint32_t s_warp[32];

  // geometry tables: staged once per CTA, reused for every event this CTA takes
  for (uint32_t i = tid; i <= ng; i += nt) g_gfirst[i] = (uint16_t)a.g.group_first_sector[i];
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
    if (tid == 0) s_event = (int)atomicAdd(a.ctrl, 1u);
    __syncthreads();                     // also: every warp is done with the previous event's tables
    const int e = s_event;
    if (e >= a.n_events) break;

    // ---- bank offsets of the event, table reset -------------------------------------------------------
    const uint32_t* bo = a.bank_offsets + (size_t)e * ns;
    const uint32_t b0 = __ldg(bo), b1 = __ldg(bo + ns);          // first byte and end of the event's banks
    for (uint32_t i = tid; i < ns; i += nt) { s_cnt[i] = 0; s_wpos[i] = kInvalid; }
    for (uint32_t i = tid; i < ng; i += nt) s_gcnt[i] = 0;
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
    uint32_t local = 0, st = range_ok ? 0u : (uint32_t)UT_STATUS_BAD_BANK_SIZE;
    if (range_ok) {
      for (uint32_t j = tid; j < ns; j += nt) {
        const uint32_t o0 = __ldg(bo + j), o1 = __ldg(bo + j + 1);
        if ((o0 & 3u) || o1 < o0 + 6u || o0 < b0 || o1 > b1) { st |= UT_STATUS_BAD_BANK_SIZE; continue; }
        const uint32_t rel = o0 - b0a;
        const uint32_t rid = *reinterpret_cast<const uint32_t*>(rawp + rel);
        const uint32_t cnt = *reinterpret_cast<const uint32_t*>(rawp + rel + 4) & 0xFFFFu;
        uint32_t s = kInvalid;
        if (rid < a.g.id_table_size) s = __ldg(a.g.id_to_sector + rid);   // 4 KB table, L1 / L2 resident
        if (s >= ns) { st |= UT_STATUS_UNKNOWN_SECTOR; continue; }
        if (o1 - o0 != ((6u + 2u * cnt + 3u) & ~3u)) { st |= UT_STATUS_BAD_BANK_SIZE; continue; }
        if (atomicCAS(&s_wpos[s], kInvalid, rel + 6u) != kInvalid) { st |= UT_STATUS_DUPLICATE_SECTOR; continue; }
        s_cnt[s] = cnt;
        if (cnt) atomicAdd(&s_gcnt[__ldg(a.g.sector_group + s)], cnt);
        local += cnt;
      }
    }
    if (st) atomicOr(&s_status, st);
    local = warp_sum(local);
    if (lane == 0) s_warp[warp] = local;
    __syncthreads();                     // last block barrier of the event: warps run on their own from here

    uint32_t tot = warp_sum(lane < nwarps ? s_warp[lane] : 0u);
    // exclusive scan of the group counts, 4 groups per lane (ng <= 128), kept in registers by every warp
    uint32_t gc[4], gs[4];
    {
      uint32_t run = 0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t g = lane * 4 + q;
        gc[q] = g < ng ? s_gcnt[g] : 0u;
        run += gc[q];
      }
      uint32_t ex = warp_incl_scan(run, lane) - run;
#pragma unroll
      for (int q = 0; q < 4; ++q) { gs[q] = ex; ex += gc[q]; }
    }

    // ---- event base: warp 0 publishes the total and resolves the chained prefix over events -----------
    uint32_t base = 0;
    bool have_base = false;
    if (warp == 0) {
      base = event_base_lookback(a.flags, e, tot, s_epoch, lane, a.carry_in);
      have_base = true;
      if (lane == 0) {
        s_base = base;
        __threadfence_block();
        *reinterpret_cast<volatile uint32_t*>(&s_ready) = 1u;
        if ((unsigned long long)base + tot > a.capacity) atomicOr(&s_status, (uint32_t)UT_STATUS_CAPACITY);
        if (e == a.n_events - 1) a.hit_offsets[(size_t)a.n_events * ng] = base + tot;
      }
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t g = lane * 4 + q;
        if (g < ng) a.hit_offsets[(size_t)e * ng + g] = base + gs[q];
      }
    }
    // per-sector view: usable by compass_track iff the event fits u16 positions and no group takes the generic path
    const bool view = a.soff != nullptr && a.view_ok && tot <= 65535u &&
                      !__any_sync(0xFFFFFFFFu, gc[0] > a.sort_buf || gc[1] > a.sort_buf || gc[2] > a.sort_buf || gc[3] > a.sort_buf);
    uint16_t* soff = a.soff ? a.soff + (size_t)e * a.soff_stride : nullptr;
    if (warp == 0 && lane == 0 && soff) {
      soff[ns] = (uint16_t)tot;
      soff[ns + 1] = (view && (unsigned long long)base + tot <= a.capacity) ? (uint16_t)UT_SECTOR_INDEX_VALID : (uint16_t)0;
    }
    if (tot == 0 && !view) continue;

    // ---- warp per sector group (ticket inside the CTA) --------------------------------------------------
    for (;;) {
      uint32_t g = 0;
      if (lane == 0) g = atomicAdd(&s_gticket, 1u);
      g = __shfl_sync(0xFFFFFFFFu, g, 0);
      if (g >= ng) break;
      const uint32_t q4 = g & 3u;                       // warp-uniform: pick the register, then the lane
      const uint32_t n = __shfl_sync(0xFFFFFFFFu, q4 == 0 ? gc[0] : q4 == 1 ? gc[1] : q4 == 2 ? gc[2] : gc[3], (int)(g >> 2));
      const uint32_t gstart =
          __shfl_sync(0xFFFFFFFFu, q4 == 0 ? gs[0] : q4 == 1 ? gs[1] : q4 == 2 ? gs[2] : gs[3], (int)(g >> 2));
      const uint32_t sa = g_gfirst[g], nsec = g_gfirst[g + 1] - sa;      // nsec <= 32 (ut_geometry_upload)
      if (n == 0) {
        if (view && (uint32_t)lane < nsec) soff[sa + lane] = (uint16_t)gstart;
        continue;
      }
      // the group's banks: word count and word position per sector, exclusive prefix = fill order
      const uint32_t cnt_r = (uint32_t)lane < nsec ? s_cnt[sa + lane] : 0u;
      const uint32_t wpos_r = (uint32_t)lane < nsec ? s_wpos[sa + lane] : 0u;
      const uint32_t e_incl = warp_incl_scan(cnt_r, lane);
      const uint32_t e_r = (uint32_t)lane < nsec ? e_incl - cnt_r : n;   // lanes past the group: never selected
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
      if (view && (uint32_t)lane < nsec) soff[sa + lane] = (uint16_t)(gstart + e_r);
      const bool in_regs = n <= 32u, in_buf = n <= a.sort_buf;

      // gather: element i of the fill order -> (sector r, word k), decode x
      float x = 0.f;
      uint32_t rw = 0;                                  // (sector-in-group << 16) | raw word
      float4 Brow = make_float4(0.f, 0.f, 0.f, 0.f);
      for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
        const uint32_t i = c0 + lane;
        int r = 0;                                      // largest r with e_r <= i
#pragma unroll
        for (int step = 16; step > 0; step >>= 1) {
          const uint32_t ev = __shfl_sync(0xFFFFFFFFu, e_r, r + step);
          if (ev <= i) r += step;
        }
        const uint32_t k = i - __shfl_sync(0xFFFFFFFFu, e_r, r);
        const uint32_t wp = __shfl_sync(0xFFFFFFFFu, wpos_r, r);
        if (i < n) {
          const uint32_t word = *reinterpret_cast<const uint16_t*>(rawp + wp + 2u * k);
          Brow = __ldg(a.g.sector_rows + 2 * (sa + r) + 1);            // {weight, raw id, x0, pitch}
          x = decode_x(word, Brow.z, Brow.w);
          rw = ((uint32_t)r << 16) | word;
          if (!in_regs && in_buf) { xbuf[i] = x; wbuf[i] = rw; }
        }
        if (!in_buf) break;                             // generic path gathers again below
      }

      if (!have_base) {                                 // the event's base is needed from here on
        while (ld_volatile_shared_u32(&s_ready) == 0u) {}
        __threadfence_block();
        base = *reinterpret_cast<volatile uint32_t*>(&s_base);
        have_base = true;
      }
      if ((unsigned long long)base + tot > a.capacity) continue;        // flagged by warp 0; offsets stay exact
      const size_t P0 = (size_t)base + gstart;

      if (in_regs) {
        // ---- <= 32 hits: rank in registers, lane order = fill order --------------------------------------
        const uint32_t rank = warp_rank((uint32_t)lane < n ? x : __int_as_float(0x7F800000), lt_mask);
        if ((uint32_t)lane < n) {
          const uint32_t s = sa + (rw >> 16);
          const float4 A = __ldg(a.g.sector_rows + 2 * s), B = Brow;
          const size_t P = P0 + rank;
          a.x[P] = x; a.z[P] = A.x; a.yb[P] = A.y; a.ye[P] = A.z; a.dxdy[P] = A.w; a.w[P] = B.x;
          a.id[P] = (__float_as_uint(B.y) << 9) | (rw & 0x1FFu);
        }
        if (view) {
          // per-sector view: lane r takes the hit of rank r (container order); its position inside its sector's run
          // is its rank among the lanes of the same sector
          if ((uint32_t)lane < n) { xbuf[rank] = x; wbuf[rank] = rw >> 16; }
          __syncwarp();
          const float xs = (uint32_t)lane < n ? xbuf[lane] : 0.f;
          const uint32_t ss = (uint32_t)lane < n ? wbuf[lane] : 0xFFFFu;
          const uint32_t peers = __match_any_sync(0xFFFFFFFFu, ss);
          const uint32_t es = __shfl_sync(0xFFFFFFFFu, e_r, (int)(ss & 31u));
          if ((uint32_t)lane < n) {
            const size_t Q = P0 + es + __popc(peers & lt_mask);
            a.sx[Q] = xs;
            a.si[Q] = (uint16_t)(gstart + lane);
          }
          __syncwarp();                                 // the buffers are reused by the warp's next group
        }
      } else if (in_buf) {
        // ---- <= sort_buf hits: rank against the warp's shared-memory copy -----------------------------------
        const uint32_t npad = (n + 3u) & ~3u;          // pad the tail of the buffer with +inf (never "smaller")
        if (n + lane < npad) xbuf[n + lane] = __int_as_float(0x7F800000);
        __syncwarp();
        for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
          const uint32_t i = c0 + lane;
          const bool valid = i < n;
          const float xi = valid ? xbuf[i] : __int_as_float(0x7F800000);
          // elements of earlier chunks come first on ties, later chunks never; this chunk: warp_rank
          uint32_t rank = warp_rank(xi, lt_mask);
          for (uint32_t j = 0; j < c0; j += 4u) {
            const float4 v = *reinterpret_cast<const float4*>(xbuf + j);
            rank += (v.x <= xi ? 1u : 0u) + (v.y <= xi ? 1u : 0u) + (v.z <= xi ? 1u : 0u) + (v.w <= xi ? 1u : 0u);
          }
          for (uint32_t j = c0 + 32u; j < npad; j += 4u) {
            const float4 v = *reinterpret_cast<const float4*>(xbuf + j);
            rank += (v.x < xi ? 1u : 0u) + (v.y < xi ? 1u : 0u) + (v.z < xi ? 1u : 0u) + (v.w < xi ? 1u : 0u);
          }
          if (valid) {
            const uint32_t rwi = wbuf[i];
            const uint32_t s = sa + (rwi >> 16);
            const float4 A = __ldg(a.g.sector_rows + 2 * s), B = __ldg(a.g.sector_rows + 2 * s + 1);
            const size_t P = P0 + rank;
            a.x[P] = xi; a.z[P] = A.x; a.yb[P] = A.y; a.ye[P] = A.z; a.dxdy[P] = A.w; a.w[P] = B.x;
            a.id[P] = (__float_as_uint(B.y) << 9) | (rwi & 0x1FFu);
            if (view) wbuf[i] = (rwi & 0xFFFF0000u) | rank;          // (sector in group, rank) for the view below
          }
        }
        if (view) {
          // per-sector view: the fill order is sector-major, so the entries of sector r are elements
          // [e_r, e_r + cnt_r) of the buffer; the position inside the run is the rank among them
          __syncwarp();
          for (uint32_t c0 = 0; c0 < n; c0 += 32u) {
            const uint32_t i = c0 + lane;
            const bool valid = i < n;
            const uint32_t rwi = valid ? wbuf[i] : 0u;
            const uint32_t rank = rwi & 0xFFFFu;
            const uint32_t es = __shfl_sync(0xFFFFFFFFu, e_r, (int)(rwi >> 16));
            const uint32_t cs = __shfl_sync(0xFFFFFFFFu, cnt_r, (int)(rwi >> 16));
            if (valid) {
              uint32_t pos = 0;
              for (uint32_t j = es; j < es + cs; ++j) pos += (wbuf[j] & 0xFFFFu) < rank ? 1u : 0u;
              const size_t Q = P0 + es + pos;
              a.sx[Q] = xbuf[i];
              a.si[Q] = (uint16_t)(gstart + rank);
            }
          }
        }
        __syncwarp();                                   // the buffer is reused by the warp's next group
      } else {
        // ---- generic path (group larger than the sort buffer): rank by recomputation, O(n^2) --------------
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

static size_t decode_smem_bytes(uint32_t ns, uint32_t ng, uint32_t raw_stage, uint32_t sort_buf, int block) {
  size_t b = align16(raw_stage);
  b += align16((size_t)(ng + 1) * 2);
  b += 2 * align16((size_t)ns * 4) + align16((size_t)ng * 4);
  b += 2 * align16((size_t)(block / 32) * sort_buf * 4);
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
  // per-warp sort buffer: twice the mean group size, at least 64, a multiple of 32
  uint32_t sort_buf = (uint32_t)std::min<unsigned long long>(((2 * avg / ng + 31) / 32) * 32 + 32, 1024);
  sort_buf = std::max(64u, sort_buf);
  sort_buf = ((uint32_t)tuned(tune.decode_sort_buf, (int)sort_buf) + 31u) & ~31u;
  // 5-warp CTAs keep a 1000-event batch resident at once (7 per SM); busy events get 8 warps per event
  int block = tuned(tune.decode_block, avg > 4096 ? 256 : 160);
  block = std::max(64, std::min(512, (block / 32) * 32));
  size_t smem = decode_smem_bytes(ns, ng, raw_stage, sort_buf, block);
  const size_t budget = (size_t)max_smem;
  while (smem > budget && raw_stage > 4096) {            // oversize events read their banks from global memory
    raw_stage = (raw_stage / 2) & ~15u;
    smem = decode_smem_bytes(ns, ng, raw_stage, sort_buf, block);
  }
  while (smem > budget && sort_buf > 32) {
    sort_buf -= 32;
    smem = decode_smem_bytes(ns, ng, raw_stage, sort_buf, block);
  }
  if (smem > budget) return UT_ERR_LIMIT;
  a.raw_stage_bytes = raw_stage; a.sort_buf = sort_buf;

  int per_sm = 0;
  UTC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ut_decode_kernel, block, smem));
  if (per_sm < 1) return cuda_fail("decode kernel does not fit on an SM", cudaErrorInvalidConfiguration);
  per_sm = std::min(per_sm, std::max(1, tuned(tune.decode_max_ctas_per_sm, 8)));
  const int grid = std::max(1, std::min(n_events, n_sm * per_sm));
  ut_decode_kernel<<<grid, block, smem, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  ut_launch_info& li = launch_info();
  li.kernels_launched = 1; li.decode_grid = grid; li.decode_block = block; li.decode_smem_bytes = (int)smem;
  li.decode_raw_stage_bytes = (int)raw_stage; li.decode_sort_buf = (int)sort_buf;
  return UT_OK;
}

}  // namespace utc
