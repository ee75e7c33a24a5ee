// api.cu -- the extern "C" surface of libutcompass (include/ut_compass.h): argument checks on the
// host, geometry upload, workspace, the two hot-path launches and the host-buffer pipeline.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "common.cuh"

namespace utc {
int32_t launch_decode(const uint8_t* raw, const uint32_t* bank_offsets, int32_t n_events, const ut_geometry* geom,
                      ut_hits* hits, uint32_t* hit_offsets, cudaStream_t stream, const uint32_t* carry_in,
                      unsigned long long hits_hint);
int32_t launch_compass(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                       const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, ut_tracks* out,
                       cudaStream_t stream, uint32_t idx_stride, unsigned long long hits_hint, uint32_t* ticket = nullptr);

size_t consolidate_workspace_bytes(uint32_t max_velo);
int32_t launch_consolidate(const ut_tracks* tracks, const uint32_t* velo_offsets, int32_t n_events, uint32_t n_velo_hint,
                           ut_compact_tracks* out, uint32_t* track_offsets, cudaStream_t stream);

int32_t launch_search_windows(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                              const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, int32_t W,
                              int16_t* windows, uint32_t* status, cudaStream_t stream);
int32_t launch_tracklets(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                         const uint32_t* velo_offsets, int32_t n_events, const compass_config* cfg, int32_t W,
                         const int16_t* windows, ut_tracks* out, cudaStream_t stream);

ut_launch_info& launch_info() {
  static thread_local ut_launch_info info = {};
  return info;
}

static thread_local char g_last_error[256] = "";
int32_t cuda_fail(const char* what, cudaError_t err) {
  snprintf(g_last_error, sizeof(g_last_error), "%s: %s", what, cudaGetErrorString(err));
  return UT_ERR_CUDA;
}
int32_t fail_with(int32_t code, const char* text) {
  snprintf(g_last_error, sizeof(g_last_error), "%s", text);
  return code;
}

namespace {
constexpr int kMaxDevices = 64;
struct DeviceEntry {
  bool init = false;
  DeviceInfo info = {};
  bool opted[kNumKernelSlots] = {};
  int max_dyn[kNumKernelSlots] = {};
};
std::mutex g_device_mu;
DeviceEntry g_devices[kMaxDevices];

std::mutex g_tuning_mu;
bool g_tuning_init = false;
ut_tuning g_tuning;

int env_int(const char* name) {
  const char* v = getenv(name);
  return v && *v ? atoi(v) : -1;
}
void tuning_from_env(ut_tuning* t) {
  for (int32_t* p = &t->decode_block; p <= &t->reserved[2]; ++p) *p = -1;
  t->decode_block = env_int("UT_DECODE_BLOCK");
  t->decode_raw_stage_bytes = env_int("UT_DECODE_RAW_STAGE");
  t->decode_sort_buf = env_int("UT_DECODE_SORT_BUF");
  t->decode_max_ctas_per_sm = env_int("UT_DECODE_MAX_CTAS_PER_SM");
  t->compass_block = env_int("UT_COMPASS_BLOCK");
  t->compass_hit_stage = env_int("UT_COMPASS_HIT_STAGE");
  t->compass_trk_stage = env_int("UT_COMPASS_TRK_STAGE");
  t->compass_split = env_int("UT_COMPASS_SPLIT");
  t->pipeline_chunk_events = env_int("UT_PIPELINE_CHUNK_EVENTS");
  t->compass_interval_min = env_int("UT_COMPASS_INTERVAL_MIN");
  t->pipeline_zero_copy = env_int("UT_PIPELINE_ZERO_COPY");
  t->decode_hit_stage = env_int("UT_DECODE_HIT_STAGE");
  t->compass_event_order = env_int("UT_COMPASS_EVENT_ORDER");
}
}  // namespace

ut_tuning tuning_snapshot() {
  std::lock_guard<std::mutex> lock(g_tuning_mu);
  if (!g_tuning_init) { tuning_from_env(&g_tuning); g_tuning_init = true; }
  return g_tuning;
}

static int32_t device_entry(DeviceEntry** out) {
  int dev = 0;
  UTC_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return cuda_fail("device index above the library's table", cudaErrorInvalidDevice);
  DeviceEntry& d = g_devices[dev];
  if (!d.init) {
    d.info.device = dev;
    UTC_CUDA(cudaDeviceGetAttribute(&d.info.n_sm, cudaDevAttrMultiProcessorCount, dev));
    UTC_CUDA(cudaDeviceGetAttribute(&d.info.smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    UTC_CUDA(cudaDeviceGetAttribute(&d.info.smem_per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev));
    d.init = true;
  }
  *out = &d;
  return UT_OK;
}

int32_t device_info(DeviceInfo* out) {
  std::lock_guard<std::mutex> lock(g_device_mu);
  DeviceEntry* d = nullptr;
  if (const int32_t rc = device_entry(&d)) return rc;
  *out = d->info;
  return UT_OK;
}

int32_t kernel_max_dynamic_smem(const void* kernel, int slot, int* max_dyn) {
  std::lock_guard<std::mutex> lock(g_device_mu);
  DeviceEntry* d = nullptr;
  if (const int32_t rc = device_entry(&d)) return rc;
  if (!d->opted[slot]) {
    cudaFuncAttributes fa;
    UTC_CUDA(cudaFuncGetAttributes(&fa, kernel));
    const int dyn = d->info.smem_optin - (int)fa.sharedSizeBytes;
    UTC_CUDA(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, dyn));
    d->max_dyn[slot] = dyn;
    d->opted[slot] = true;
  }
  *max_dyn = d->max_dyn[slot];
  return UT_OK;
}

struct GeomOwner {
  void* block = nullptr;     // one device allocation holding every table
};

static bool geometry_ok(const ut_geometry* g) {
  return g && g->n_layers == UT_N_LAYERS && g->n_groups >= 4 && g->n_groups % 4 == 0 && g->n_sectors >= g->n_groups &&
         g->id_to_sector && g->sector_raw_id && g->sector_group && g->x0 && g->pitch && g->dxdy && g->z &&
         g->y_begin && g->y_end && g->weight && g->group_xmin && g->group_xmax;
}
}  // namespace utc

using namespace utc;

extern "C" {

const char* ut_version(void) { return "ut-compass-b200 0.1 (sm_100a)"; }

const char* ut_last_error(void) { return g_last_error; }

void ut_last_launch_info(ut_launch_info* out) {
  if (out) *out = launch_info();
}

int32_t ut_tuning_get(ut_tuning* out) {
  if (!out) return UT_ERR_NULL;
  *out = tuning_snapshot();
  return UT_OK;
}

int32_t ut_tuning_set(const ut_tuning* in) {
  std::lock_guard<std::mutex> lock(g_tuning_mu);
  if (in) g_tuning = *in; else tuning_from_env(&g_tuning);
  g_tuning_init = true;
  return UT_OK;
}

int32_t ut_geometry_upload(const ut_geometry* h, ut_geometry* out) {
  if (!h || !out) return UT_ERR_NULL;
  if (!geometry_ok(h)) return UT_ERR_GEOMETRY;
  const uint32_t ns = h->n_sectors, ng = h->n_groups, gpl = ng / UT_N_LAYERS;
  if (ns > UT_MAX_SECTORS || ng > UT_MAX_GROUPS || h->id_table_size == 0) return UT_ERR_LIMIT;
  // ---- container contract (include/ut_compass.h) ----
  std::vector<uint32_t> first(ng + 1, 0);
  bool rows_sorted = true;
  {
    uint32_t prev = 0;
    std::vector<uint32_t> cnt(ng, 0);
    for (uint32_t s = 0; s < ns; ++s) {
      const uint32_t g = h->sector_group[s];
      if (g >= ng || g < prev) return UT_ERR_GEOMETRY;
      prev = g;
      ++cnt[g];
      if (!(h->pitch[s] > 0.f) || h->sector_raw_id[s] >= h->id_table_size) return UT_ERR_GEOMETRY;
      if (h->id_to_sector[h->sector_raw_id[s]] != s) return UT_ERR_GEOMETRY;
    }
    for (uint32_t g = 0; g < ng; ++g) {
      if (cnt[g] == 0) return UT_ERR_GEOMETRY;
      if (cnt[g] > 32) return UT_ERR_LIMIT;                                // a warp holds a group's sector table
      first[g + 1] = first[g] + cnt[g];
      for (uint32_t s = first[g]; s < first[g + 1]; ++s) {
        if (h->dxdy[s] != h->dxdy[first[g]]) return UT_ERR_GEOMETRY;      // one stereo angle per group
        if (s > first[g] && (h->y_begin[s] < h->y_begin[s - 1] || h->y_end[s] < h->y_end[s - 1])) rows_sorted = false;
      }
      const float span = h->group_xmax[g] - h->group_xmin[g];
      if (!(span > 0.f)) return UT_ERR_GEOMETRY;
      if (g % gpl != 0 && (h->group_xmin[g] < h->group_xmin[g - 1] || h->group_xmax[g] < h->group_xmax[g - 1]))
        return UT_ERR_GEOMETRY;                                           // bounds monotone inside a layer
    }
  }
  bool rows_uniform = rows_sorted;
  for (uint32_t g = 0; g < ng && rows_uniform; ++g) {
    const uint32_t gl = (g / gpl) * gpl;                                  // first group of the layer
    if (first[g + 1] - first[g] != first[gl + 1] - first[gl]) { rows_uniform = false; break; }
    for (uint32_t r = 0; r < first[g + 1] - first[g]; ++r)
      if (h->y_begin[first[g] + r] != h->y_begin[first[gl] + r] || h->y_end[first[g] + r] != h->y_end[first[gl] + r])
        rows_uniform = false;
  }
  // ---- one device block, 256-byte aligned sub-tables ----
  auto up = [](size_t v) { return (v + 255) & ~size_t(255); };
  const size_t sz_id = up(h->id_table_size * 4), sz_s = up(ns * 4), sz_g = up((ng + 1) * 4);
  const size_t sz_rows = up((size_t)ns * 32);
  const uint32_t n_cells = h->kick_nx * h->kick_ny;
  if (h->kick_nx != 0 && (n_cells == 0 || n_cells > 4096 || !h->kick_kappa || !h->kick_z_mag)) return UT_ERR_GEOMETRY;
  const size_t sz_k = up((size_t)n_cells * 4);
  const size_t total = sz_id + 10 * sz_s + 3 * sz_g + sz_rows + 2 * sz_k;
  unsigned char* dev = nullptr;
  if (cudaMalloc(&dev, total) != cudaSuccess) return UT_ERR_CUDA;
  std::vector<unsigned char> host(total, 0);
  size_t off = 0;
  auto put = [&](const void* src, size_t bytes, size_t slot) {
    const void* d = dev + off;
    memcpy(host.data() + off, src, bytes);
    off += slot;
    return d;
  };
  *out = *h;
  bool layer_uniform = true;                 // every sector of a layer at the layer's z, with one weight
  for (uint32_t g = 0; g < ng; ++g)
    for (uint32_t s2 = first[g]; s2 < first[g + 1]; ++s2)
      if (h->z[s2] != h->layer_z[g / gpl] || h->weight[s2] != h->weight[first[(g / gpl) * gpl]]) layer_uniform = false;
  out->flags = (rows_sorted ? UT_GEOM_ROWS_SORTED : 0u) | (rows_uniform ? UT_GEOM_ROWS_UNIFORM : 0u) |
               (layer_uniform ? UT_GEOM_LAYER_UNIFORM : 0u);
  for (uint32_t l = 0; l < UT_N_LAYERS; ++l) out->layer_weight[l] = layer_uniform ? h->weight[first[l * gpl]] : 0.f;
  out->id_to_sector = (const uint32_t*)put(h->id_to_sector, h->id_table_size * 4, sz_id);
  out->sector_raw_id = (const uint32_t*)put(h->sector_raw_id, ns * 4, sz_s);
  out->sector_group = (const uint32_t*)put(h->sector_group, ns * 4, sz_s);
  out->x0 = (const float*)put(h->x0, ns * 4, sz_s);
  out->pitch = (const float*)put(h->pitch, ns * 4, sz_s);
  out->dxdy = (const float*)put(h->dxdy, ns * 4, sz_s);
  out->z = (const float*)put(h->z, ns * 4, sz_s);
  out->y_begin = (const float*)put(h->y_begin, ns * 4, sz_s);
  out->y_end = (const float*)put(h->y_end, ns * 4, sz_s);
  out->weight = (const float*)put(h->weight, ns * 4, sz_s);
  out->group_xmin = (const float*)put(h->group_xmin, ng * 4, sz_g);
  out->group_xmax = (const float*)put(h->group_xmax, ng * 4, sz_g);
  out->group_first_sector = (const uint32_t*)put(first.data(), (ng + 1) * 4, sz_g);
  {
    std::vector<float> rows((size_t)ns * 8);
    for (uint32_t s = 0; s < ns; ++s) {
      float* r = rows.data() + (size_t)s * 8;
      r[0] = h->z[s]; r[1] = h->y_begin[s]; r[2] = h->y_end[s]; r[3] = h->dxdy[s];
      r[4] = h->weight[s]; memcpy(&r[5], &h->sector_raw_id[s], 4); r[6] = h->x0[s]; r[7] = h->pitch[s];
    }
    out->sector_rows = put(rows.data(), (size_t)ns * 32, sz_rows);
  }
  {
    // order of a group's sectors by (y_begin, dense index): what the Y order of the container follows
    std::vector<uint32_t> yo(ns, 0);
    for (uint32_t g = 0; g < ng; ++g) {
      const uint32_t sa = first[g], n = first[g + 1] - first[g];
      for (uint32_t r = 0; r < n; ++r) {
        uint32_t rank = 0;
        for (uint32_t q = 0; q < n; ++q)
          rank += h->y_begin[sa + q] < h->y_begin[sa + r] || (h->y_begin[sa + q] == h->y_begin[sa + r] && q < r);
        yo[sa + r] |= rank;
        yo[sa + rank] |= r << 8;
      }
    }
    out->sector_yorder = (const uint32_t*)put(yo.data(), ns * 4, sz_s);
  }
  if (n_cells) {
    out->kick_kappa = (const float*)put(h->kick_kappa, (size_t)n_cells * 4, sz_k);
    out->kick_z_mag = (const float*)put(h->kick_z_mag, (size_t)n_cells * 4, sz_k);
  } else {
    out->kick_nx = out->kick_ny = 0;
    out->kick_kappa = out->kick_z_mag = nullptr;
  }
  if (cudaMemcpy(dev, host.data(), total, cudaMemcpyHostToDevice) != cudaSuccess) {
    cudaFree(dev);
    return UT_ERR_CUDA;
  }
  GeomOwner* own = new (std::nothrow) GeomOwner;
  if (!own) { cudaFree(dev); return UT_ERR_CUDA; }
  own->block = dev;
  out->owner = own;
  return UT_OK;
}

int32_t ut_geometry_free(ut_geometry* g) {
  if (!g) return UT_ERR_NULL;
  if (g->owner) {
    GeomOwner* own = static_cast<GeomOwner*>(g->owner);
    cudaFree(own->block);
    delete own;
    g->owner = nullptr;
  }
  return UT_OK;
}

uint32_t ut_sector_offsets_stride(const ut_geometry* geometry) {
  return geometry ? (geometry->n_sectors + 2u + 7u) & ~7u : 0u;
}

size_t ut_decode_workspace_bytes(int32_t max_events, const ut_geometry* /*geometry*/) {
  return 32 + 8 * (size_t)(max_events > 0 ? max_events : 0) + 8;   // 8 control words, then one look-back word per event
}

int32_t ut_decode_workspace_init(void* workspace, int32_t max_events, ut_stream_t stream) {
  if (!workspace) return UT_ERR_NULL;
  if (max_events < 0) return UT_ERR_ARG;
  return cudaMemsetAsync(workspace, 0, ut_decode_workspace_bytes(max_events, nullptr), (cudaStream_t)stream) == cudaSuccess
             ? UT_OK : UT_ERR_CUDA;
}

int32_t ut_decode(const uint8_t* raw_banks, const uint32_t* bank_offsets, int32_t n_events,
                  const ut_geometry* geometry, ut_hits* hits_out, uint32_t* hit_offsets_out, ut_stream_t stream) {
  launch_info().kernels_launched = 0;
  if (!bank_offsets || !geometry || !hits_out || !hit_offsets_out) return UT_ERR_NULL;
  if (n_events < 0) return UT_ERR_ARG;
  if (!geometry->group_first_sector || !geometry->sector_rows || !geometry->sector_yorder)
    return UT_ERR_GEOMETRY;                                                                  // not uploaded
  if (hits_out->order != UT_ORDER_X && hits_out->order != UT_ORDER_Y) return UT_ERR_ARG;
  if (geometry->n_sectors > UT_MAX_SECTORS || geometry->n_groups > UT_MAX_GROUPS) return UT_ERR_LIMIT;
  if (!hits_out->x_at_y0 || !hits_out->z_at_y0 || !hits_out->y_begin || !hits_out->y_end || !hits_out->dxdy ||
      !hits_out->weight || !hits_out->id)
    if (hits_out->capacity > 0) return UT_ERR_NULL;
  if (!hits_out->status || !hits_out->workspace) return UT_ERR_NULL;
  if ((reinterpret_cast<uintptr_t>(raw_banks) & 15u) || (reinterpret_cast<uintptr_t>(bank_offsets) & 15u) ||
      (reinterpret_cast<uintptr_t>(hits_out->workspace) & 15u))
    return UT_ERR_ARG;
  {                                   // the per-sector view: all three arrays or none
    const int have = (hits_out->x_by_sector != nullptr) + (hits_out->idx_by_sector != nullptr) + (hits_out->sector_offsets != nullptr);
    if (have != 0 && have != 3) return UT_ERR_ARG;
  }
  hits_out->geom = geometry;
  if (n_events == 0)      // the offsets array still has its single entry
    return cudaMemsetAsync(hit_offsets_out, 0, 4, (cudaStream_t)stream) == cudaSuccess ? UT_OK : UT_ERR_CUDA;
  if (!raw_banks) return UT_ERR_NULL;
  return launch_decode(raw_banks, bank_offsets, n_events, geometry, hits_out, hit_offsets_out, (cudaStream_t)stream,
                       nullptr, 0ull);
}

int32_t compass_config_default(float p_min_mev, float window_scale, int32_t min_hits, int32_t max_candidates_per_layer,
                               const ut_geometry* geometry, compass_config* out) {
  if (!geometry || !out) return UT_ERR_NULL;
  if (!(p_min_mev > 0.f) || !(window_scale > 0.f)) return UT_ERR_ARG;
  const double kappa = 60.0, z_mag = 1750.0;
  const double kick = (double)window_scale * kappa / (double)p_min_mev;
  for (int l = 0; l < UT_N_LAYERS; ++l) out->win_half[l] = (float)(kick * ((double)geometry->layer_z[l] - z_mag) + 0.5);
  out->y_tol = 0.5f; out->max_slope = (float)(kick + 0.0015); out->kink_tol = 1.5f; out->seed_tol = 0.5f;
  out->w_velo = 100.0f; out->max_chi2_ndf = 9.0f; out->kappa = (float)kappa; out->z_mag = (float)z_mag;
  out->min_hits = min_hits; out->max_candidates_per_layer = max_candidates_per_layer;
  out->both_directions = 0;
  return UT_OK;
}

static int32_t check_config(const compass_config* c) {
  if (c->min_hits != 3 && c->min_hits != 4) return UT_ERR_ARG;
  if (c->max_candidates_per_layer < 1 || c->max_candidates_per_layer > UT_MAX_CANDIDATES) return UT_ERR_ARG;
  if (c->both_directions != 0 && c->both_directions != 1) return UT_ERR_ARG;
  for (int l = 0; l < UT_N_LAYERS; ++l) if (!(c->win_half[l] >= 0.f)) return UT_ERR_ARG;
  return UT_OK;
}

int32_t compass_track(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                      const uint32_t* velo_offsets, int32_t n_events, const compass_config* config,
                      ut_tracks* tracks_out, ut_stream_t stream) {
  launch_info().kernels_launched = 0;
  if (!hits || !hit_offsets || !velo || !velo_offsets || !config || !tracks_out || !hits->geom) return UT_ERR_NULL;
  if (n_events < 0) return UT_ERR_ARG;
  if (const int32_t rc = check_config(config)) return rc;
  if (!tracks_out->status) return UT_ERR_NULL;
  if (n_events == 0) return UT_OK;
  if (!tracks_out->hit_idx || !tracks_out->n_hits || !tracks_out->qop || !tracks_out->chi2 || !velo->x || !velo->y ||
      !velo->tx || !velo->ty)
    return UT_ERR_NULL;
  if (hits->geom->n_layers != UT_N_LAYERS || hits->geom->n_groups > UT_MAX_GROUPS) return UT_ERR_GEOMETRY;
  return launch_compass(hits, hit_offsets, velo, velo_offsets, n_events, config, tracks_out, (cudaStream_t)stream, 0u, 0ull);
}

int32_t compass_search_windows(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                               const uint32_t* velo_offsets, int32_t n_events, const compass_config* config,
                               int32_t n_sectors_search, int16_t* windows_out, uint32_t* status, ut_stream_t stream) {
  launch_info().kernels_launched = 0;
  if (!hits || !hit_offsets || !velo || !velo_offsets || !config || !status || !hits->geom) return UT_ERR_NULL;
  if (n_events < 0 || (n_sectors_search != 1 && n_sectors_search != 3 && n_sectors_search != 5)) return UT_ERR_ARG;
  if (const int32_t rc = check_config(config)) return rc;
  if (n_events == 0) return UT_OK;
  if (!windows_out || !velo->x || !velo->y || !velo->tx || !velo->ty) return UT_ERR_NULL;
  if (hits->geom->n_layers != UT_N_LAYERS || hits->geom->n_groups > UT_MAX_GROUPS) return UT_ERR_GEOMETRY;
  if (hits->order != UT_ORDER_X) return UT_ERR_ARG;                    // the group-wide binary search needs x order
  return launch_search_windows(hits, hit_offsets, velo, velo_offsets, n_events, config, n_sectors_search, windows_out,
                               status, (cudaStream_t)stream);
}

int32_t compass_tracklets_from_windows(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                                       const uint32_t* velo_offsets, int32_t n_events, const compass_config* config,
                                       int32_t n_sectors_search, const int16_t* windows, ut_tracks* tracks_out,
                                       ut_stream_t stream) {
  launch_info().kernels_launched = 0;
  if (!hits || !hit_offsets || !velo || !velo_offsets || !config || !tracks_out || !hits->geom) return UT_ERR_NULL;
  if (n_events < 0 || (n_sectors_search != 1 && n_sectors_search != 3 && n_sectors_search != 5)) return UT_ERR_ARG;
  if (const int32_t rc = check_config(config)) return rc;
  if (!tracks_out->status) return UT_ERR_NULL;
  if (n_events == 0) return UT_OK;
  if (!windows || !tracks_out->hit_idx || !tracks_out->n_hits || !tracks_out->qop || !tracks_out->chi2 || !velo->x ||
      !velo->y || !velo->tx || !velo->ty)
    return UT_ERR_NULL;
  if (hits->geom->n_layers != UT_N_LAYERS || hits->geom->n_groups > UT_MAX_GROUPS) return UT_ERR_GEOMETRY;
  if (hits->order != UT_ORDER_X) return UT_ERR_ARG;
  return launch_tracklets(hits, hit_offsets, velo, velo_offsets, n_events, config, n_sectors_search, windows, tracks_out,
                          (cudaStream_t)stream);
}

// ---------------------------------------------------------------------------------------------------
// Host-buffer pipeline (bench.py "e2e"): one arena of device buffers, async copies around the two calls.
// ---------------------------------------------------------------------------------------------------
size_t compass_consolidate_workspace_bytes(uint32_t max_velo_total) { return consolidate_workspace_bytes(max_velo_total); }

int32_t compass_consolidate(const ut_tracks* tracks, const uint32_t* velo_offsets, int32_t n_events,
                            ut_compact_tracks* out, uint32_t* track_offsets_out, ut_stream_t stream) {
  launch_info().kernels_launched = 0;
  if (!tracks || !velo_offsets || !out || !track_offsets_out) return UT_ERR_NULL;
  if (n_events < 0) return UT_ERR_ARG;
  if (!out->status || !out->workspace) return UT_ERR_NULL;
  if (reinterpret_cast<uintptr_t>(out->workspace) & 15u) return UT_ERR_ARG;
  if (n_events == 0) return cudaMemsetAsync(track_offsets_out, 0, 4, (cudaStream_t)stream) == cudaSuccess ? UT_OK : UT_ERR_CUDA;
  if (out->capacity > 0 && (!out->velo_index || !out->hit_idx || !out->n_hits || !out->qop || !out->chi2)) return UT_ERR_NULL;
  if (out->max_velo_total > 0 && (!tracks->hit_idx || !tracks->n_hits || !tracks->qop || !tracks->chi2)) return UT_ERR_NULL;
  return launch_consolidate(tracks, velo_offsets, n_events, out->max_velo_total, out, track_offsets_out, (cudaStream_t)stream);
}

struct ut_pipeline {
  ut_geometry geom;
  int32_t max_events;
  size_t max_raw;
  uint64_t max_hits;
  uint32_t max_velo;
  unsigned char* block;
  uint8_t* raw;
  uint32_t *bank_offsets, *hit_offsets, *velo_offsets, *status /* [2] */;
  float *vx, *vy, *vtx, *vty;
  ut_hits hits;
  ut_tracks tracks;
  // chunked overlap of copies and kernels: copy-in stream, copy-out stream, per-chunk events
  cudaStream_t s_in, s_in2, s_out, s_cmp, s_cmp2;
  cudaEvent_t ev_start, ev_out, ev_in[4], ev_velo[4], ev_done[4], ev_dec[4], ev_d2h[4];
  int last_chunks;               // chunks of the most recent run (ut_pipeline_timeline)
  bool last_zero_copy;
};

int32_t ut_pipeline_create(const ut_geometry* g, int32_t max_events, size_t max_raw_bytes, uint64_t max_hits,
                           uint32_t max_velo, ut_pipeline** out) {
  if (!g || !out) return UT_ERR_NULL;
  if (max_events < 1) return UT_ERR_ARG;
  ut_pipeline* p = new (std::nothrow) ut_pipeline;
  if (!p) return UT_ERR_CUDA;
  memset(p, 0, sizeof(*p));
  p->geom = *g; p->geom.owner = nullptr;
  p->max_events = max_events; p->max_raw = max_raw_bytes; p->max_hits = max_hits; p->max_velo = max_velo;
  auto up = [](size_t v) { return (v + 255) & ~size_t(255); };
  const size_t s_raw = up(max_raw_bytes + 16), s_bo = up(((size_t)max_events * g->n_sectors + 1) * 4),
               s_ho = up(((size_t)max_events * g->n_groups + 1) * 4), s_vo = up(((size_t)max_events + 1) * 4),
               s_st = 256, s_v = up((size_t)max_velo * 4), s_h = up((size_t)max_hits * 4 + 32),
               s_ws = up(ut_decode_workspace_bytes(max_events, g)), s_ti = 4 * s_v,
               s_so = up((size_t)max_events * ut_sector_offsets_stride(g) * 2);
  const size_t total = s_raw + s_bo + s_ho + s_vo + s_st + 4 * s_v + 9 * s_h + s_ws + s_ti + 3 * s_v + s_so;
  if (cudaMalloc(&p->block, total) != cudaSuccess) { delete p; return UT_ERR_CUDA; }
  unsigned char* q = p->block;
  auto take = [&](size_t n) { unsigned char* r = q; q += n; return r; };
  p->raw = take(s_raw);
  p->bank_offsets = (uint32_t*)take(s_bo); p->hit_offsets = (uint32_t*)take(s_ho);
  p->velo_offsets = (uint32_t*)take(s_vo); p->status = (uint32_t*)take(s_st);
  p->vx = (float*)take(s_v); p->vy = (float*)take(s_v); p->vtx = (float*)take(s_v); p->vty = (float*)take(s_v);
  p->hits.x_at_y0 = (float*)take(s_h); p->hits.z_at_y0 = (float*)take(s_h); p->hits.y_begin = (float*)take(s_h);
  p->hits.y_end = (float*)take(s_h); p->hits.dxdy = (float*)take(s_h); p->hits.weight = (float*)take(s_h);
  p->hits.id = (uint32_t*)take(s_h);
  p->hits.capacity = max_hits; p->hits.geom = &p->geom; p->hits.status = p->status;
  p->hits.workspace = take(s_ws);
  p->hits.x_by_sector = (float*)take(s_h); p->hits.idx_by_sector = (uint16_t*)take(s_h);   // (half of the slot used)
  p->hits.sector_offsets = (uint16_t*)take(s_so);
  // the track SoA is 7 rows s_v bytes apart (4 of hit_idx, n_hits, qop, chi2): one strided copy takes a range of tracks out
  p->tracks.hit_idx = (int32_t*)take(s_ti);
  p->tracks.n_hits = (int32_t*)take(s_v); p->tracks.qop = (float*)take(s_v); p->tracks.chi2 = (float*)take(s_v);
  p->tracks.status = p->status + 4;                    // 4 words: status + the kernel's work ticket
  if (cudaMemset(p->block, 0, total) != cudaSuccess) { cudaFree(p->block); delete p; return UT_ERR_CUDA; }
  bool ok = cudaStreamCreateWithFlags(&p->s_in, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&p->s_in2, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&p->s_out, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&p->s_cmp, cudaStreamNonBlocking) == cudaSuccess &&
            cudaStreamCreateWithFlags(&p->s_cmp2, cudaStreamNonBlocking) == cudaSuccess &&
            cudaEventCreate(&p->ev_start) == cudaSuccess && cudaEventCreate(&p->ev_out) == cudaSuccess;
  for (int k = 0; k < 4 && ok; ++k)         // (timing events: ut_pipeline_timeline reads them)
    ok = cudaEventCreate(&p->ev_in[k]) == cudaSuccess && cudaEventCreate(&p->ev_velo[k]) == cudaSuccess &&
         cudaEventCreate(&p->ev_done[k]) == cudaSuccess && cudaEventCreate(&p->ev_dec[k]) == cudaSuccess &&
         cudaEventCreate(&p->ev_d2h[k]) == cudaSuccess;
  if (!ok) { cudaFree(p->block); delete p; return UT_ERR_CUDA; }
  *out = p;
  return UT_OK;
}

int32_t ut_pipeline_destroy(ut_pipeline* p) {
  if (!p) return UT_ERR_NULL;
  cudaStreamSynchronize(p->s_in);
  cudaStreamSynchronize(p->s_in2);
  cudaStreamSynchronize(p->s_out);
  cudaStreamSynchronize(p->s_cmp);
  cudaStreamSynchronize(p->s_cmp2);
  for (int k = 0; k < 4; ++k) {
    cudaEventDestroy(p->ev_in[k]); cudaEventDestroy(p->ev_velo[k]); cudaEventDestroy(p->ev_done[k]); cudaEventDestroy(p->ev_dec[k]);
    cudaEventDestroy(p->ev_d2h[k]);
  }
  cudaEventDestroy(p->ev_start); cudaEventDestroy(p->ev_out);
  cudaStreamDestroy(p->s_in); cudaStreamDestroy(p->s_in2); cudaStreamDestroy(p->s_out); cudaStreamDestroy(p->s_cmp); cudaStreamDestroy(p->s_cmp2);
  cudaFree(p->block);
  delete p;
  return UT_OK;
}

int32_t ut_pipeline_run_host(ut_pipeline* p, const uint8_t* raw_h, size_t raw_bytes, const uint32_t* bo_h,
                             const velo_states* velo_h, const uint32_t* vo_h, uint32_t n_velo, int32_t n_events,
                             const compass_config* config, ut_tracks* tracks_h, uint32_t* status_h, uint32_t* n_hits_h,
                             ut_stream_t stream_) {
  if (!p || !bo_h || !velo_h || !vo_h || !config || !tracks_h) return UT_ERR_NULL;
  if (n_events < 0 || n_events > p->max_events || raw_bytes > p->max_raw || n_velo > p->max_velo) return UT_ERR_ARG;
  if (n_events > 0 && !raw_h) return UT_ERR_NULL;
  cudaStream_t s = (cudaStream_t)stream_;
  const ut_geometry* g = &p->geom;
  const uint32_t ns = g->n_sectors, ng = g->n_groups;
  // The batch is cut into up to 4 chunks of events: chunk k+1 is copied in while chunk k is decoded and
  // tracked, and the tracks of chunk k go out while chunk k+1 is computed.  Results are those of one call:
  // the decode of chunk k starts its hit prefix from the total chunk k-1 left in hit_offsets.
  const int kChunkEvents = tuned(tuning_snapshot().pipeline_chunk_events, 333);
  int K = n_events / (kChunkEvents > 0 ? kChunkEvents : 333);
  K = K < 1 ? 1 : (K > 4 ? 4 : K);
  // busy events (config 4: ~8000 hits each) make the call compute-bound: Compass of chunk k holds every SM while chunk
  // k + 1 waits decoded-or-not, so what counts is an early start -- 4 chunks, the first copy-in 40 % of the bytes
  // instead of 50 % (config 4: 2.22 -> 2.07 ms per call)
  if (tuning_snapshot().pipeline_chunk_events < 0 && K == 3 && raw_bytes / (size_t)n_events > 6 * (size_t)ns + 2 * 4096) K = 4;
  bool ok = cudaMemsetAsync(p->status, 0, 64, s) == cudaSuccess && cudaEventRecord(p->ev_start, s) == cudaSuccess &&
            cudaStreamWaitEvent(p->s_in, p->ev_start, 0) == cudaSuccess &&
            cudaStreamWaitEvent(p->s_in2, p->ev_start, 0) == cudaSuccess &&
            cudaStreamWaitEvent(p->s_out, p->ev_start, 0) == cudaSuccess &&
            cudaStreamWaitEvent(p->s_cmp, p->ev_start, 0) == cudaSuccess &&
            cudaStreamWaitEvent(p->s_cmp2, p->ev_start, 0) == cudaSuccess;
  if (!ok) return cuda_fail("ut_pipeline_run_host", cudaGetLastError());
  // Zero copy (ut_tuning.pipeline_zero_copy = 1, off by default): when the raw banks and their offsets sit in mapped
  // pinned host memory the decode kernel reads them over PCIe itself (bulk copies and coalesced loads straight from
  // the host buffer, no staging copy) and Compass runs on a second stream, so that chunk k is tracked while chunk
  // k + 1 streams in.  Measured on a B200 (config 3): SM-issued reads reach ~28 GB/s against ~53 GB/s of the copy
  // engine, 0.70 ms per call against 0.54-0.57 ms staged -- kept as an option, not the default.
  const uint8_t* raw_z = nullptr;
  const uint32_t* bo_z = nullptr;
  if (tuned(tuning_snapshot().pipeline_zero_copy, 0) != 0 && n_events > 0) {
    void *d1 = nullptr, *d2 = nullptr;
    if (cudaHostGetDevicePointer(&d1, const_cast<uint8_t*>(raw_h), 0) == cudaSuccess &&
        cudaHostGetDevicePointer(&d2, const_cast<uint32_t*>(bo_h), 0) == cudaSuccess &&
        ((reinterpret_cast<uintptr_t>(d1) | reinterpret_cast<uintptr_t>(d2)) & 15u) == 0) {
      raw_z = static_cast<const uint8_t*>(d1);
      bo_z = static_cast<const uint32_t*>(d2);
    } else {
      cudaGetLastError();                          // not mapped pinned memory: staged copies
    }
  }
  p->last_zero_copy = raw_z != nullptr;
  if (n_events == 0) {
    ok = cudaMemsetAsync(p->hit_offsets, 0, 4, s) == cudaSuccess;
    if (status_h) ok = ok && cudaMemcpyAsync(status_h, p->status, 4, cudaMemcpyDeviceToHost, s) == cudaSuccess &&
                     cudaMemcpyAsync(status_h + 1, p->status + 4, 4, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    if (n_hits_h) ok = ok && cudaMemcpyAsync(n_hits_h, p->hit_offsets, 4, cudaMemcpyDeviceToHost, s) == cudaSuccess;
    return ok ? UT_OK : UT_ERR_CUDA;
  }
  if (!p->hits.geom->group_first_sector || !p->hits.geom->sector_rows) return UT_ERR_GEOMETRY;
  if (const int32_t rc = check_config(config)) return rc;
  auto h2d = [&](void* d, const void* h, size_t n) {
    return n == 0 || cudaMemcpyAsync(d, h, n, cudaMemcpyHostToDevice, p->s_in) == cudaSuccess;
  };
  auto d2h = [&](void* h, const void* d, size_t n) {
    return n == 0 || cudaMemcpyAsync(h, d, n, cudaMemcpyDeviceToHost, p->s_out) == cudaSuccess;
  };
  // `rows` arrays of `n` bytes each, `hpitch` / `dpitch` bytes apart: one strided copy when the host arrays are evenly
  // spaced (every copy costs ~10 us of engine latency on top of its bytes), else one copy per array
  auto rows_copy = [&](void* const* hp, ptrdiff_t hpitch, unsigned char* d, size_t dpitch, size_t n, int rows, bool to_host,
                       cudaStream_t st) {
    if (n == 0) return true;
    if (hpitch >= (ptrdiff_t)n) {
      if ((to_host ? cudaMemcpy2DAsync(hp[0], (size_t)hpitch, d, dpitch, n, (size_t)rows, cudaMemcpyDeviceToHost, st)
                   : cudaMemcpy2DAsync(d, dpitch, hp[0], (size_t)hpitch, n, (size_t)rows, cudaMemcpyHostToDevice, st)) == cudaSuccess)
        return true;
      cudaGetLastError();          // evenly spaced, but not rows of ONE page-locked allocation: the call refuses; copy per array
    }
    bool good = true;
    for (int r = 0; r < rows && good; ++r)
      good = (to_host ? cudaMemcpyAsync(hp[r], d + (size_t)r * dpitch, n, cudaMemcpyDeviceToHost, st)
                      : cudaMemcpyAsync(d + (size_t)r * dpitch, hp[r], n, cudaMemcpyHostToDevice, st)) == cudaSuccess;
    return good;
  };
  // spacing of evenly spaced host arrays (0: not evenly spaced)
  auto pitch_of = [](const void* a0, const void* a1, const void* a2, const void* a3) -> ptrdiff_t {
    const ptrdiff_t d = (const unsigned char*)a1 - (const unsigned char*)a0;
    if (d <= 0 || (const unsigned char*)a2 - (const unsigned char*)a1 != d) return 0;
    if (a3 && (const unsigned char*)a3 - (const unsigned char*)a2 != d) return 0;
    return d;
  };
  velo_states vd = {p->vx, p->vy, p->vtx, p->vty, velo_h->z};
  const size_t dv_pitch = (size_t)((unsigned char*)p->vy - (unsigned char*)p->vx);
  // The VELO states and their offsets (15 % of the input bytes) go in at once, in FRONT of the first chunk's banks on the
  // one copy-in stream.  On a second stream beside the banks the two copies took the link in either order from call to
  // call: states first 0.47-0.49 ms per call on config 3 (device timeline), states last 0.52-0.54 ms, as every Compass
  // launch waits for them.  The states of each chunk in front of that chunk's banks cost three more copies: 0.50 ms.
  {
    void* const hv[4] = {const_cast<float*>(velo_h->x), const_cast<float*>(velo_h->y), const_cast<float*>(velo_h->tx),
                         const_cast<float*>(velo_h->ty)};
    cudaStream_t sv = p->s_in;
    ok = cudaMemcpyAsync(p->velo_offsets, vo_h, ((size_t)n_events + 1) * 4, cudaMemcpyHostToDevice, sv) == cudaSuccess &&
         rows_copy(hv, pitch_of(hv[0], hv[1], hv[2], hv[3]), (unsigned char*)p->vx, dv_pitch, (size_t)n_velo * 4, 4, false, sv) &&
         cudaEventRecord(p->ev_velo[0], sv) == cudaSuccess && cudaStreamWaitEvent(p->s_cmp, p->ev_velo[0], 0) == cudaSuccess &&
         cudaStreamWaitEvent(p->s_cmp2, p->ev_velo[0], 0) == cudaSuccess;
    if (!ok) return cuda_fail("ut_pipeline_run_host", cudaGetLastError());
  }
  const ptrdiff_t ht_pitch = pitch_of(tracks_h->n_hits, tracks_h->qop, tracks_h->chi2, nullptr);
  const size_t dt_pitch = (size_t)((unsigned char*)p->tracks.qop - (unsigned char*)p->tracks.n_hits);   // all 7 device rows
  // host track arrays that form one [7][n_velo] block (hit_idx rows, n_hits, qop, chi2 back to back) leave by ONE copy
  const bool one_block = (const void*)tracks_h->n_hits == (const void*)(tracks_h->hit_idx + 4 * (size_t)n_velo) &&
                         ht_pitch == (ptrdiff_t)((size_t)n_velo * 4);
  int launched = 0;
  // Chunk sizes fall linearly (K = 4: 40 / 30 / 20 / 10 % of the events).  The copy-in is the longest stage (PCIe), every
  // chunk's kernels hide behind the next chunk's copy, and what remains exposed at the end is the last chunk's decode +
  // Compass + copy-out: the smaller that chunk, the shorter the call.
  auto chunk_begin = [&](int k) { return (int)((long long)n_events * k * (2 * K - k + 1) / ((long long)K * (K + 1))); };
  for (int k = 0; k < K; ++k) {
    const int e0 = chunk_begin(k), e1 = k == K - 1 ? n_events : chunk_begin(k + 1), ne = e1 - e0;
    const size_t r0 = k == 0 ? 0 : bo_h[(size_t)e0 * ns], r1 = k == K - 1 ? raw_bytes : bo_h[(size_t)e1 * ns];
    const uint32_t v0 = vo_h[e0], v1 = vo_h[e1];
    if (r1 < r0 || r1 > raw_bytes || v1 < v0 || v1 > n_velo) return UT_ERR_ARG;
    ok = raw_z != nullptr ||
         (h2d(p->raw + r0, raw_h + r0, r1 - r0) &&
          h2d(p->bank_offsets + (size_t)e0 * ns, bo_h + (size_t)e0 * ns, ((size_t)ne * ns + 1) * 4) &&
          cudaEventRecord(p->ev_in[k], p->s_in) == cudaSuccess && cudaStreamWaitEvent(s, p->ev_in[k], 0) == cudaSuccess);
    if (!ok) return cuda_fail("ut_pipeline_run_host", cudaGetLastError());
    uint32_t* ho = p->hit_offsets + (size_t)e0 * ng;
    // upper bound of this chunk's hits from its raw size alone (sizes the on-chip staging like a whole call)
    const size_t hdr = 6 * (size_t)ne * ns;
    const unsigned long long hint = r1 - r0 > hdr ? (r1 - r0 - hdr) / 2 : 1;
    ut_hits hc = p->hits;                              // this chunk's rows of the per-sector view
    hc.sector_offsets = p->hits.sector_offsets + (size_t)e0 * ut_sector_offsets_stride(g);
    int32_t rc = launch_decode(raw_z ? raw_z : p->raw, (raw_z ? bo_z : p->bank_offsets) + (size_t)e0 * ns, ne, g, &hc, ho, s,
                               k == 0 ? nullptr : ho, hint);
    if (rc) return rc;
    launched += launch_info().kernels_launched;
    // Compass runs beside the decode stream, chunks alternating between two streams (each launch with its own work
    // ticket): chunk k is tracked while chunk k + 1 is decoded and chunk k + 2 streams in, and the short last chunks,
    // which cost one event's latency whatever their size, overlap each other.  Both kernels leave issue slots idle alone.
    // The last chunk has no decode behind it: its Compass and its copy-out stay on the decode's stream (no event hops
    // between streams in the exposed tail of the call, and the launch overlaps the decode's end like two plain calls).
    const bool tail = k == K - 1;
    cudaStream_t sc = tail ? s : ((k & 1) ? p->s_cmp2 : p->s_cmp);
    cudaStream_t so = tail ? s : p->s_out;
    if (tail && cudaStreamWaitEvent(s, p->ev_velo[0], 0) != cudaSuccess)
      return cuda_fail("ut_pipeline_run_host (events)", cudaGetLastError());
    if (cudaEventRecord(p->ev_dec[k], s) != cudaSuccess || (!tail && cudaStreamWaitEvent(sc, p->ev_dec[k], 0) != cudaSuccess))
      return cuda_fail("ut_pipeline_run_host (events)", cudaGetLastError());
    rc = launch_compass(&hc, ho, &vd, p->velo_offsets + e0, ne, config, &p->tracks, sc, (uint32_t)(dt_pitch / 4), hint,
                        p->status + 8 + (tail ? 4 : 2 * (k & 1)));   // (a ticket pair per stream: launches that may overlap never share one)
    if (rc) return rc;
    launched += launch_info().kernels_launched;
    // (the hit total is final once the last chunk is decoded: it leaves while that chunk is tracked, not behind its tracks)
    if (k == K - 1 && n_hits_h &&
        !(cudaStreamWaitEvent(p->s_out, p->ev_dec[k], 0) == cudaSuccess && d2h(n_hits_h, p->hit_offsets + (size_t)n_events * ng, 4)))
      return cuda_fail("ut_pipeline_run_host", cudaGetLastError());
    ok = cudaEventRecord(p->ev_done[k], sc) == cudaSuccess && (tail || cudaStreamWaitEvent(p->s_out, p->ev_done[k], 0) == cudaSuccess);
    {
      void* const hi[4] = {tracks_h->hit_idx + v0, tracks_h->hit_idx + (size_t)n_velo + v0, tracks_h->hit_idx + 2 * (size_t)n_velo + v0,
                           tracks_h->hit_idx + 3 * (size_t)n_velo + v0};
      void* const hr[3] = {tracks_h->n_hits + v0, tracks_h->qop + v0, tracks_h->chi2 + v0};
      if (one_block) {
        void* const h7[7] = {hi[0], hi[1], hi[2], hi[3], hr[0], hr[1], hr[2]};
        ok = ok && rows_copy(h7, (ptrdiff_t)n_velo * 4, (unsigned char*)(p->tracks.hit_idx + v0), dt_pitch, (size_t)(v1 - v0) * 4, 7,
                             true, so);
      } else {
        ok = ok && rows_copy(hi, (ptrdiff_t)n_velo * 4, (unsigned char*)(p->tracks.hit_idx + v0), dt_pitch, (size_t)(v1 - v0) * 4, 4,
                             true, so) &&
             rows_copy(hr, ht_pitch, (unsigned char*)(p->tracks.n_hits + v0), dt_pitch, (size_t)(v1 - v0) * 4, 3, true, so);
      }
      ok = ok && cudaEventRecord(p->ev_d2h[k], so) == cudaSuccess;
    }
    if (!ok) return cuda_fail("ut_pipeline_run_host", cudaGetLastError());
  }
  p->last_chunks = K;
  launch_info().kernels_launched = launched;
  // the decode's and Compass's status words (16 bytes apart) by one strided copy, behind everything: the caller's stream
  // joins the copy-out stream first (the last chunk's Compass ran on the caller's stream itself)
  void* const hs[2] = {status_h, status_h + 1};
  ok = ok && cudaEventRecord(p->ev_out, p->s_out) == cudaSuccess && cudaStreamWaitEvent(s, p->ev_out, 0) == cudaSuccess;
  if (status_h) ok = ok && rows_copy(hs, 4, (unsigned char*)p->status, 16, 4, 2, true, s);
  return ok ? UT_OK : cuda_fail("ut_pipeline_run_host (copy out)", cudaGetLastError());
}

int32_t ut_pipeline_timeline(ut_pipeline* p, float* ms_out, int32_t* n_chunks_out) {
  if (!p || !ms_out || !n_chunks_out) return UT_ERR_NULL;
  *n_chunks_out = p->last_chunks;
  for (int k = 0; k < p->last_chunks; ++k) {
    cudaEvent_t ev[5] = {p->ev_in[k], p->ev_velo[0], p->ev_dec[k], p->ev_done[k], p->ev_d2h[k]};   // (VELO states: one copy per call)
    for (int q = 0; q < 5; ++q) {
      float ms = -1.f;
      if (q == 0 && p->last_zero_copy) { ms_out[k * 5] = -1.f; continue; }
      if (cudaEventElapsedTime(&ms, p->ev_start, ev[q]) != cudaSuccess) { cudaGetLastError(); ms = -1.f; }
      ms_out[k * 5 + q] = ms;
    }
  }
  return UT_OK;
}

int32_t ut_host_alloc(void** out, size_t bytes) {
  if (!out) return UT_ERR_NULL;
  *out = nullptr;
  const cudaError_t err = cudaHostAlloc(out, bytes ? bytes : 1, cudaHostAllocPortable | cudaHostAllocMapped);
  return err == cudaSuccess ? UT_OK : cuda_fail("cudaHostAlloc", err);
}

int32_t ut_host_free(void* p) {
  if (!p) return UT_OK;
  const cudaError_t err = cudaFreeHost(p);
  return err == cudaSuccess ? UT_OK : cuda_fail("cudaFreeHost", err);
}

int32_t ut_pipeline_device_hits(ut_pipeline* p, ut_hits* hits_out, const uint32_t** hit_offsets_out) {
  if (!p || !hits_out || !hit_offsets_out) return UT_ERR_NULL;
  *hits_out = p->hits;
  *hit_offsets_out = p->hit_offsets;
  return UT_OK;
}

}  // extern "C"
