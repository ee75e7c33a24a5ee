// ut_decode.cu -- UT raw-bank decoding (section IV, :235-274) as ONE persistent kernel.
//
// The paper splits decoding into 7 launches (Table 1: count, 3-kernel Blelloch
// scan with a host read-back of the total, pre-decode, find permutation, decode in order).  That
// shape was made for sm_61/sm_70 and a batch of events that is tiny for a B200.
// Here one CTA owns one event at a time (dynamic ticket), keeps the event on chip and touches HBM
// once per byte:
//
//   ticket -> bank offsets (coalesced) -> raw banks of the event by ONE TMA bulk copy into smem
//   -> per-bank header check, sector claim, count          (paper: "calculate number of hits")
//   -> event total -> chained exclusive prefix over events by decoupled look-back (paper: prefix sum
//      + host sync; here no sync, no second launch)
//   -> bucket histogram of x inside every sector group (monotone fp32 -> bucket map), block scan,
//      scatter, in-bucket rank by (x, sector, word)         (paper: pre-decode + find permutation)
//   -> coalesced SoA store at base + rank                   (paper: decode raw banks in order)
//
// The bucket pass makes the stable in-group sort O(n) instead of the paper's insertion sort.
// Events that do not fit the shared-memory staging sizes take a slower generic path with the same
// results.  Arithmetic of x follows include/ut_compass.h exactly (__fmul_rn/__fadd_rn, never fused).
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
  uint32_t* ctrl;               // [0] ticket, [1] CTAs done, [2] epoch
  unsigned long long* flags;    // [n_events] look-back words: epoch:30 | state:2 | value:32
  uint32_t raw_stage_bytes;     // multiple of 16
  uint32_t hit_stage;           // elements
  uint32_t log2_buckets;        // buckets per group = 1 << log2_buckets
};

__device__ __forceinline__ float decode_x(uint32_t word, float x0, float pitch) {
  const uint32_t u = ((word & 0x1FFu) << 1) | ((word >> 9) & 1u);   // 2*strip + frac
  const float t = __fadd_rn(__fmul_rn((float)u, 0.5f), 0.25f);
  return __fadd_rn(x0, __fmul_rn(t, pitch));
}

// monotone non-decreasing map x -> bucket inside a group (equal x -> equal bucket)
__device__ __forceinline__ uint32_t bucket_of(float x, float xmin, float inv_span, uint32_t nb) {
  const float f = __fmul_rn(__fmul_rn(__fsub_rn(x, xmin), inv_span), (float)nb);
  int b = (int)f;                                         // cvt.rzi saturates, NaN -> 0
  b = b < 0 ? 0 : b;
  return (uint32_t)b < nb ? (uint32_t)b : nb - 1;
}

__device__ __forceinline__ bool key_less(float xa, uint32_t ka, float xb, uint32_t kb) {
  return xa < xb || (xa == xb && ka < kb);
}

// Chained exclusive prefix over events (decoupled look-back).  Called by warp 0.  Event e only waits
// for events with a smaller ticket, which are running or finished, so it always makes progress.
__device__ uint32_t event_base_lookback(unsigned long long* flags, int e, uint32_t tot, uint32_t epoch, int lane) {
  const unsigned long long tag = (unsigned long long)(epoch & 0x3FFFFFFFu) << 34;
  if (e == 0) {
    if (lane == 0) st_volatile_u64(&flags[0], tag | (2ull << 32) | tot);
    return 0;
  }
  if (lane == 0) st_volatile_u64(&flags[e], tag | (1ull << 32) | tot);
  uint32_t base = 0;
  int idx = e - 1 - lane;
  for (;;) {
    unsigned long long v = 0;
    if (idx >= 0) {
      do { v = ld_volatile_u64(&flags[idx]); } while ((v >> 34) != (tag >> 34) || ((v >> 32) & 3ull) == 0ull);
    }
    const bool incl = idx >= 0 && ((v >> 32) & 3ull) == 2ull;
    const unsigned m = __ballot_sync(0xFFFFFFFFu, incl);
    uint32_t val = idx >= 0 ? (uint32_t)v : 0u;
    if (m) {
      const int first = __ffs(m) - 1;                    // closest predecessor with an inclusive prefix
      base += warp_sum(lane <= first ? val : 0u);
      break;
    }
    base += warp_sum(val);
    idx -= 32;
  }
  if (lane == 0) st_volatile_u64(&flags[e], tag | (2ull << 32) | (unsigned long long)(base + tot));
  return base;
}

__global__ void __launch_bounds__(1024) ut_decode_kernel(const DecodeArgs a) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const uint32_t ns = a.g.n_sectors, ng = a.g.n_groups;
  const uint32_t nbk = 1u << a.log2_buckets, NB = ng << a.log2_buckets;
  const int tid = threadIdx.x, nt = blockDim.x, lane = tid & 31, warp = tid >> 5, nwarps = nt >> 5;

  Carver cv(smem_raw);
  unsigned char* s_rawstage = cv.take<unsigned char>(a.raw_stage_bytes);
  float* g_x0 = cv.take<float>(ns);
  float* g_pitch = cv.take<float>(ns);
  float* g_z = cv.take<float>(ns);
  float* g_yb = cv.take<float>(ns);
  float* g_ye = cv.take<float>(ns);
  float* g_dxdy = cv.take<float>(ns);
  float* g_w = cv.take<float>(ns);
  uint32_t* g_rawid = cv.take<uint32_t>(ns);
  uint16_t* g_group = cv.take<uint16_t>(ns);
  float* g_gxmin = cv.take<float>(ng);
  float* g_ginv = cv.take<float>(ng);
  uint32_t* g_gfirst = cv.take<uint32_t>(ng + 1);
  uint32_t* s_off = cv.take<uint32_t>(ns + 4);
  uint32_t* s_cnt = cv.take<uint32_t>(ns);
  uint32_t* s_wpos = cv.take<uint32_t>(ns);
  uint32_t* s_gstart = cv.take<uint32_t>(ng + 1);
  uint32_t* s_bucket = cv.take<uint32_t>(NB);
  float* t_x = cv.take<float>(a.hit_stage);
  uint32_t* t_key = cv.take<uint32_t>(a.hit_stage);

  __shared__ uint64_t s_bar;
  __shared__ int s_event;
  __shared__ uint32_t s_epoch, s_status, s_base, s_tot;
  __shared__ uint32_t s_warp[32];

  // geometry tables: staged once per CTA, reused for every event this CTA takes
  for (uint32_t i = tid; i < ns; i += nt) {
    g_x0[i] = a.g.x0[i]; g_pitch[i] = a.g.pitch[i]; g_z[i] = a.g.z[i]; g_yb[i] = a.g.y_begin[i];
    g_ye[i] = a.g.y_end[i]; g_dxdy[i] = a.g.dxdy[i]; g_w[i] = a.g.weight[i];
    g_rawid[i] = a.g.sector_raw_id[i]; g_group[i] = (uint16_t)a.g.sector_group[i];
  }
  for (uint32_t i = tid; i < ng; i += nt) { g_gxmin[i] = a.g.group_xmin[i]; g_ginv[i] = a.g.group_inv_span[i]; }
  for (uint32_t i = tid; i <= ng; i += nt) g_gfirst[i] = a.g.group_first_sector[i];
  if (tid == 0) {
    mbar_init(&s_bar, 1);
    fence_mbar_init();
    s_epoch = ld_volatile_u32(a.ctrl + 2);
    s_status = 0;
  }
  __syncthreads();
  uint32_t bar_phase = 0;

  for (;;) {
    if (tid == 0) s_event = (int)atomicAdd(a.ctrl, 1u);
    __syncthreads();
    const int e = s_event;
    if (e >= a.n_events) break;

    // ---- bank offsets of the event, table reset -------------------------------------------------------
    const uint32_t* bo = a.bank_offsets + (size_t)e * ns;
    for (uint32_t i = tid; i <= ns; i += nt) s_off[i] = __ldg(bo + i);
    for (uint32_t i = tid; i < ns; i += nt) { s_cnt[i] = 0; s_wpos[i] = kInvalid; }
    for (uint32_t i = tid; i < NB; i += nt) s_bucket[i] = 0;
    __syncthreads();

    const uint32_t b0 = s_off[0], b1 = s_off[ns];
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
        const uint32_t o0 = s_off[j], o1 = s_off[j + 1];
        if ((o0 & 3u) || o1 < o0 + 6u || o0 < b0 || o1 > b1) { st |= UT_STATUS_BAD_BANK_SIZE; continue; }
        const uint32_t rel = o0 - b0a;
        const uint32_t rid = *reinterpret_cast<const uint32_t*>(rawp + rel);
        const uint32_t cnt = *reinterpret_cast<const uint32_t*>(rawp + rel + 4) & 0xFFFFu;
        const uint32_t s = rid < a.g.id_table_size ? __ldg(a.g.id_to_sector + rid) : kInvalid;
        if (s >= ns) { st |= UT_STATUS_UNKNOWN_SECTOR; continue; }
        if (o1 - o0 != ((6u + 2u * cnt + 3u) & ~3u)) { st |= UT_STATUS_BAD_BANK_SIZE; continue; }
        if (atomicCAS(&s_wpos[s], kInvalid, rel + 6u) != kInvalid) { st |= UT_STATUS_DUPLICATE_SECTOR; continue; }
        s_cnt[s] = cnt;
        local += cnt;
      }
    }
    if (st) atomicOr(&s_status, st);
    local = warp_sum(local);
    if (lane == 0) s_warp[warp] = local;
    __syncthreads();

    // ---- event total, chained prefix over events, group starts ---------------------------------------
    if (warp == 0) {
      uint32_t v = lane < nwarps ? s_warp[lane] : 0u;
      v = warp_sum(v);
      const uint32_t base = event_base_lookback(a.flags, e, v, s_epoch, lane);
      if (lane == 0) { s_tot = v; s_base = base; }
    } else if (warp == 1) {
      // exclusive scan of the per-group counts (groups = runs of sectors), ng <= 128
      uint32_t c[4], run = 0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t g = lane * 4 + q;
        uint32_t v = 0;
        if (g < ng) for (uint32_t s = g_gfirst[g]; s < g_gfirst[g + 1]; ++s) v += s_cnt[s];
        c[q] = v; run += v;
      }
      const uint32_t incl = warp_incl_scan(run, lane);
      uint32_t ex = incl - run;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        const uint32_t g = lane * 4 + q;
        if (g < ng) s_gstart[g] = ex;
        ex += c[q];
      }
      if (lane == 31) s_gstart[ng] = incl;
    }
    __syncthreads();
    const uint32_t tot = s_tot, base = s_base;
    for (uint32_t g = tid; g < ng; g += nt) a.hit_offsets[(size_t)e * ng + g] = base + s_gstart[g];
    if (e == a.n_events - 1 && tid == 0) a.hit_offsets[(size_t)a.n_events * ng] = base + tot;
    const bool fits = (unsigned long long)base + tot <= a.capacity;
    if (!fits && tid == 0) atomicOr(&s_status, (uint32_t)UT_STATUS_CAPACITY);

    if (fits && tot > 0 && tot <= a.hit_stage) {
      // ---- fast path: O(n) bucket ordering on chip ----------------------------------------------------
      for (uint32_t s = tid; s < ns; s += nt) {                      // pass 1: bucket histogram
        const uint32_t cnt = s_cnt[s];
        if (!cnt) continue;
        const uint16_t* w16 = reinterpret_cast<const uint16_t*>(rawp + s_wpos[s]);
        const uint32_t g = g_group[s];
        const float x0 = g_x0[s], pitch = g_pitch[s], xmin = g_gxmin[g], inv = g_ginv[g];
        for (uint32_t k = 0; k < cnt; ++k) {
          const float x = decode_x(w16[k], x0, pitch);
          atomicAdd(&s_bucket[(g << a.log2_buckets) + bucket_of(x, xmin, inv, nbk)], 1u);
        }
      }
      __syncthreads();
      {                                                               // exclusive scan over NB buckets
        const uint32_t ipt = (NB + nt - 1) / nt;
        const uint32_t c0 = min(NB, tid * ipt), c1 = min(NB, c0 + ipt);
        uint32_t sum = 0;
        for (uint32_t i = c0; i < c1; ++i) sum += s_bucket[i];
        const uint32_t incl = warp_incl_scan(sum, lane);
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
          const uint32_t v = lane < nwarps ? s_warp[lane] : 0u;
          const uint32_t iv = warp_incl_scan(v, lane);
          s_warp[lane] = iv - v;
        }
        __syncthreads();
        uint32_t ex = s_warp[warp] + incl - sum;
        for (uint32_t i = c0; i < c1; ++i) { const uint32_t v = s_bucket[i]; s_bucket[i] = ex; ex += v; }
      }
      __syncthreads();
      for (uint32_t s = tid; s < ns; s += nt) {                      // pass 2: scatter into buckets
        const uint32_t cnt = s_cnt[s];
        if (!cnt) continue;
        const uint16_t* w16 = reinterpret_cast<const uint16_t*>(rawp + s_wpos[s]);
        const uint32_t g = g_group[s];
        const float x0 = g_x0[s], pitch = g_pitch[s], xmin = g_gxmin[g], inv = g_ginv[g];
        for (uint32_t k = 0; k < cnt; ++k) {
          const float x = decode_x(w16[k], x0, pitch);
          const uint32_t pos = atomicAdd(&s_bucket[(g << a.log2_buckets) + bucket_of(x, xmin, inv, nbk)], 1u);
          t_x[pos] = x;
          t_key[pos] = (s << 16) | k;
        }
      }
      __syncthreads();                                               // now s_bucket[b] = end of bucket b
      for (uint32_t q = tid; q < tot; q += nt) {                     // pass 3: rank inside bucket, store
        const float x = t_x[q];
        const uint32_t key = t_key[q];
        const uint32_t s = key >> 16, k = key & 0xFFFFu;
        const uint32_t g = g_group[s];
        const uint32_t gb = (g << a.log2_buckets) + bucket_of(x, g_gxmin[g], g_ginv[g], nbk);
        const uint32_t lo = gb ? s_bucket[gb - 1] : 0u, hi = s_bucket[gb];
        uint32_t rank = lo;
        for (uint32_t j = lo; j < hi; ++j) rank += key_less(t_x[j], t_key[j], x, key) ? 1u : 0u;
        const uint32_t word = reinterpret_cast<const uint16_t*>(rawp + s_wpos[s])[k];
        const size_t P = (size_t)base + rank;
        a.x[P] = x; a.z[P] = g_z[s]; a.yb[P] = g_yb[s]; a.ye[P] = g_ye[s];
        a.dxdy[P] = g_dxdy[s]; a.w[P] = g_w[s]; a.id[P] = (g_rawid[s] << 9) | (word & 0x1FFu);
      }
    } else if (fits && tot > 0) {
      // ---- generic path (event larger than the staging sizes): rank by recomputation, O(n^2) per group ----
      for (uint32_t s = 0; s < ns; ++s) {
        const uint32_t cnt = s_cnt[s];
        if (!cnt) continue;
        const uint32_t g = g_group[s];
        const uint16_t* w16 = reinterpret_cast<const uint16_t*>(rawp + s_wpos[s]);
        for (uint32_t k = tid; k < cnt; k += nt) {
          const uint32_t word = w16[k];
          const float x = decode_x(word, g_x0[s], g_pitch[s]);
          const uint32_t key = (s << 16) | k;
          uint32_t rank = 0;
          for (uint32_t s2 = g_gfirst[g]; s2 < g_gfirst[g + 1]; ++s2) {
            const uint32_t c2 = s_cnt[s2];
            if (!c2) continue;
            const uint16_t* v16 = reinterpret_cast<const uint16_t*>(rawp + s_wpos[s2]);
            const float x02 = g_x0[s2], p2 = g_pitch[s2];
            for (uint32_t k2 = 0; k2 < c2; ++k2)
              rank += key_less(decode_x(v16[k2], x02, p2), (s2 << 16) | k2, x, key) ? 1u : 0u;
          }
          const size_t P = (size_t)base + s_gstart[g] + rank;
          a.x[P] = x; a.z[P] = g_z[s]; a.yb[P] = g_yb[s]; a.ye[P] = g_ye[s];
          a.dxdy[P] = g_dxdy[s]; a.w[P] = g_w[s]; a.id[P] = (g_rawid[s] << 9) | (word & 0x1FFu);
        }
      }
    }
    __syncthreads();      // everything of this event is consumed before the tables are reset
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

static int env_int(const char* name, int dflt) {
  const char* v = getenv(name);
  return v && *v ? atoi(v) : dflt;
}

size_t decode_smem_bytes(uint32_t ns, uint32_t ng, uint32_t raw_stage, uint32_t hit_stage, uint32_t log2b) {
  size_t b = align16(raw_stage);
  b += 8 * align16(ns * 4) + align16(ns * 2);
  b += 2 * align16(ng * 4) + align16((ng + 1) * 4);
  b += align16((ns + 4) * 4) + 2 * align16(ns * 4) + align16((ng + 1) * 4);
  b += align16((size_t)(ng << log2b) * 4);
  b += 2 * align16((size_t)hit_stage * 4);
  return b;
}

int32_t launch_decode(const uint8_t* raw, const uint32_t* bank_offsets, int32_t n_events, const ut_geometry* geom,
                      ut_hits* hits, uint32_t* hit_offsets, cudaStream_t stream) {
  static int n_sm = 0, max_smem = 0;     // max_smem = largest dynamic size this kernel may ask for
  if (!n_sm) {
    int dev = 0, optin = 0;
    UTC_CUDA(cudaGetDevice(&dev));
    UTC_CUDA(cudaDeviceGetAttribute(&optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    cudaFuncAttributes fa;
    UTC_CUDA(cudaFuncGetAttributes(&fa, ut_decode_kernel));
    const int dyn = optin - (int)fa.sharedSizeBytes;
    UTC_CUDA(cudaFuncSetAttribute(ut_decode_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn));
    UTC_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev));
    max_smem = dyn;
  }
  DecodeArgs a;
  a.raw = raw; a.bank_offsets = bank_offsets; a.n_events = n_events; a.g = make_geom_dev(geom);
  a.x = hits->x_at_y0; a.z = hits->z_at_y0; a.yb = hits->y_begin; a.ye = hits->y_end; a.dxdy = hits->dxdy;
  a.w = hits->weight; a.id = hits->id; a.capacity = hits->capacity; a.status = hits->status;
  a.hit_offsets = hit_offsets;
  a.ctrl = reinterpret_cast<uint32_t*>(hits->workspace);
  a.flags = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(hits->workspace) + 16);

  // staging sizes from the only size the host knows without a sync: capacity / n_events
  const uint32_t ns = geom->n_sectors, ng = geom->n_groups;
  const unsigned long long avg = hits->capacity / (unsigned long long)n_events + 1;
  uint32_t hit_stage = (uint32_t)std::min<unsigned long long>(((avg + 255) / 256) * 256 + 256, 1u << 16);
  hit_stage = (uint32_t)env_int("UT_DECODE_HIT_STAGE", (int)hit_stage);
  uint32_t log2b = 3;
  while (log2b < 8 && (1.4142f * (float)(1u << log2b)) < (float)avg / (float)ng) ++log2b;
  log2b = (uint32_t)env_int("UT_DECODE_LOG2_BUCKETS", (int)log2b);
  uint32_t raw_stage = (uint32_t)align16(8u * ns + 2u * hit_stage + 32u);
  raw_stage = (uint32_t)env_int("UT_DECODE_RAW_STAGE", (int)raw_stage) & ~15u;
  size_t smem = decode_smem_bytes(ns, ng, raw_stage, hit_stage, log2b);
  const size_t budget = (size_t)max_smem;
  while (smem > budget && hit_stage > 256) {           // shrink until it fits; oversize events take the generic path
    hit_stage /= 2;
    raw_stage = (uint32_t)align16(8u * ns + 2u * hit_stage + 32u);
    if (log2b > 3) --log2b;
    smem = decode_smem_bytes(ns, ng, raw_stage, hit_stage, log2b);
  }
  if (smem > budget) return UT_ERR_LIMIT;
  a.raw_stage_bytes = raw_stage; a.hit_stage = hit_stage; a.log2_buckets = log2b;

  int block = env_int("UT_DECODE_BLOCK", 512);
  block = std::max(64, std::min(1024, (block / 32) * 32));
  int per_sm = 0;
  UTC_CUDA(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, ut_decode_kernel, block, smem));
  if (per_sm < 1) return cuda_fail("decode kernel does not fit on an SM", cudaErrorInvalidConfiguration);
  per_sm = std::min(per_sm, env_int("UT_DECODE_MAX_CTAS_PER_SM", 8));
  const int grid = std::max(1, std::min(n_events, n_sm * per_sm));
  ut_decode_kernel<<<grid, block, smem, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  ut_launch_info& li = launch_info();
  li.kernels_launched = 1; li.decode_grid = grid; li.decode_block = block; li.decode_smem_bytes = (int)smem;
  li.decode_buckets_per_group = 1 << log2b; li.decode_hit_stage = (int)hit_stage;
  return UT_OK;
}

}  // namespace utc
