// consolidate.cu -- compacted VELO+UT track output, SURVEY.md 8(f) row 1.
//
// The paper's tracklet kernel reserves output slots with one atomicAdd per event and a later
// "prefix sum and consolidation" leaves the tracks coalesced for the next algorithm.  Here the
// Compass kernel writes one dense slot per VELO track (deterministic, A13) and this kernel compacts:
// tiles of kTile VELO tracks are handed out by an atomic ticket; a CTA scans the "has a tracklet" flags of
// its tile, publishes the tile total for the chained exclusive prefix over tiles (decoupled look-back, the same
// helper the decode uses over events) and stores the kept tracks at base + rank.  Event boundaries that fall
// inside the tile get their compact offset from the same scan.  One pass over the 28 B / track of input.
#include <algorithm>

#include "common.cuh"

namespace utc {

constexpr int kTile = 1024;            // VELO tracks per tile
constexpr int kThreads = 256;          // 4 tracks per thread
constexpr int kPer = kTile / kThreads;

struct ConsolidateArgs {
  const int32_t *idx, *n;
  const float *qop, *chi2;
  const uint32_t* velo_offsets;
  int32_t n_events;
  uint32_t* o_velo;
  int32_t *o_idx, *o_n;
  float *o_qop, *o_chi2;
  unsigned long long capacity;
  uint32_t max_velo;
  uint32_t* status;
  uint32_t* track_offsets;
  uint32_t* ctrl;               // [0] ticket, [1] CTAs done, [2] epoch
  unsigned long long* flags;    // one look-back word per tile
};

__global__ void __launch_bounds__(kThreads) consolidate_kernel(const ConsolidateArgs a) {
  __shared__ uint32_t s_warp[kThreads / 32], s_base, s_epoch;
  __shared__ int s_tile;
  __shared__ uint32_t s_excl[kTile + 1];           // exclusive rank of every track of the tile (+ the tile total)
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const uint32_t T = __ldg(a.velo_offsets + a.n_events);
  const bool too_many = T > a.max_velo;            // the look-back words would not cover the tiles
  const int n_tiles = too_many ? 0 : (int)((T + kTile - 1) / kTile);
  if (tid == 0) s_epoch = ld_volatile_u32(a.ctrl + 2);
  uint32_t st = too_many ? (uint32_t)UT_STATUS_BAD_OFFSETS : 0u;
  if (n_tiles == 0 && !too_many && blockIdx.x == 0)   // no VELO track at all: every event owns the empty range
    for (int e = tid; e <= a.n_events; e += kThreads) a.track_offsets[e] = 0;
  for (;;) {
    __syncthreads();                               // previous tile fully consumed
    if (tid == 0) s_tile = (int)atomicAdd(a.ctrl, 1u);
    __syncthreads();
    const int tile = s_tile;
    if (tile >= n_tiles) break;
    const uint32_t t0 = (uint32_t)tile * kTile;
    // flags of kPer consecutive tracks per thread, block-wide exclusive scan
    uint32_t keep = 0, cnt = 0;
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
      const uint32_t t = t0 + (uint32_t)(tid * kPer + k);
      if (t < T && __ldg(a.n + t) > 0) { keep |= 1u << k; ++cnt; }
    }
    const uint32_t incl = warp_incl_scan(cnt, lane);
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) {
      const uint32_t v = s_warp[w];
      if (w < warp) wbase += v;
      total += v;
    }
    uint32_t ex = wbase + incl - cnt;
    if (warp == 0) {
      const uint32_t base = event_base_lookback(a.flags, tile, total, s_epoch, lane, nullptr);
      if (lane == 0) s_base = base;
    }
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
      s_excl[tid * kPer + k] = ex;
      ex += (keep >> k) & 1u;
    }
    if (tid == kThreads - 1) s_excl[kTile] = ex;
    __syncthreads();
    const uint32_t base = s_base;
    // kept tracks, coalesced over consecutive threads
    for (int q = tid; q < kTile; q += kThreads) {
      const uint32_t t = t0 + (uint32_t)q;
      if (t >= T) break;
      const uint32_t r = s_excl[q];
      if (s_excl[q + 1] == r) continue;            // no tracklet
      const unsigned long long P = (unsigned long long)base + r;
      if (P >= a.capacity) { st |= UT_STATUS_CAPACITY; continue; }
      a.o_velo[P] = t;
#pragma unroll
      for (int l = 0; l < 4; ++l) a.o_idx[(size_t)l * a.capacity + P] = __ldg(a.idx + (size_t)l * T + t);
      a.o_n[P] = __ldg(a.n + t);
      a.o_qop[P] = __ldg(a.qop + t);
      a.o_chi2[P] = __ldg(a.chi2 + t);
    }
    // event boundaries inside [t0, t0 + kTile) (the last tile also owns the boundary T)
    {
      const uint32_t hi = min(t0 + (uint32_t)kTile, T);
      int lo_e = 0, hi_e = a.n_events + 1;           // first event with velo_offsets[e] >= t0
      while (lo_e < hi_e) {
        const int mid = (lo_e + hi_e) >> 1;
        if (__ldg(a.velo_offsets + mid) >= t0) hi_e = mid; else lo_e = mid + 1;
      }
      for (int e = lo_e + tid; e <= a.n_events; e += kThreads) {
        const uint32_t b = __ldg(a.velo_offsets + e);
        if (b > hi || (b == hi && hi != T)) break;   // boundary belongs to a later tile
        if (b < t0) { st |= UT_STATUS_BAD_OFFSETS; continue; }   // offsets run backwards: nothing to look up
        a.track_offsets[e] = base + s_excl[b - t0];
      }
    }
  }
  if (st) atomicOr(a.status, st);
  if (tid == 0) {
    __threadfence();
    if (atomicAdd(a.ctrl + 1, 1u) == gridDim.x - 1) {       // last CTA out re-arms the workspace
      a.ctrl[0] = 0; a.ctrl[1] = 0;
      __threadfence();
      a.ctrl[2] = s_epoch + 1u;
    }
  }
}

size_t consolidate_workspace_bytes(uint32_t max_velo) {
  return 16 + 8 * ((size_t)max_velo / kTile + 2);
}

int32_t launch_consolidate(const ut_tracks* tracks, const uint32_t* velo_offsets, int32_t n_events, uint32_t n_velo_hint,
                           ut_compact_tracks* out, uint32_t* track_offsets, cudaStream_t stream) {
  DeviceInfo dev;
  if (const int32_t rc = device_info(&dev)) return rc;
  const int n_sm = dev.n_sm;
  ConsolidateArgs a;
  a.idx = tracks->hit_idx; a.n = tracks->n_hits; a.qop = tracks->qop; a.chi2 = tracks->chi2;
  a.velo_offsets = velo_offsets; a.n_events = n_events;
  a.o_velo = out->velo_index; a.o_idx = out->hit_idx; a.o_n = out->n_hits; a.o_qop = out->qop; a.o_chi2 = out->chi2;
  a.capacity = out->capacity; a.max_velo = out->max_velo_total; a.status = out->status; a.track_offsets = track_offsets;
  a.ctrl = reinterpret_cast<uint32_t*>(out->workspace);
  a.flags = reinterpret_cast<unsigned long long*>(reinterpret_cast<unsigned char*>(out->workspace) + 16);
  // the grid only needs to cover the tiles; capacity bounds n_velo_total when the caller sized it that way
  const unsigned long long tiles = (std::max<unsigned long long>(n_velo_hint, 1) + kTile - 1) / kTile;
  const int grid = (int)std::max<unsigned long long>(1, std::min<unsigned long long>(tiles, (unsigned long long)n_sm * 8));
  consolidate_kernel<<<grid, kThreads, 0, stream>>>(a);
  UTC_CUDA(cudaGetLastError());
  launch_info().kernels_launched = 1;
  return UT_OK;
}

}  // namespace utc
