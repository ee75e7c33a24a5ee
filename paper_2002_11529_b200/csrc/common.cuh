// common.cuh -- device helpers shared by the decode and Compass kernels (sm_100a).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/ut_compass.h"

namespace utc {

constexpr uint32_t kInvalid = 0xFFFFFFFFu;
constexpr int kWarp = 32;

// Device-side view of the geometry tables (passed by value in kernel parameters).
struct GeomDev {
  uint32_t n_sectors, n_groups, id_table_size, groups_per_layer;
  const uint32_t *id_to_sector, *sector_raw_id, *sector_group, *group_first_sector, *sector_yorder;
  const float *x0, *pitch, *dxdy, *z, *y_begin, *y_end, *weight;
  const float *group_xmin, *group_xmax;
  const float4* sector_rows;
  float layer_z[4], layer_dxdy[4];
};

inline GeomDev make_geom_dev(const ut_geometry* g) {
  GeomDev d;
  d.n_sectors = g->n_sectors; d.n_groups = g->n_groups; d.id_table_size = g->id_table_size;
  d.groups_per_layer = g->n_groups / UT_N_LAYERS;
  d.id_to_sector = g->id_to_sector; d.sector_raw_id = g->sector_raw_id; d.sector_group = g->sector_group;
  d.group_first_sector = g->group_first_sector; d.sector_yorder = g->sector_yorder;
  d.x0 = g->x0; d.pitch = g->pitch; d.dxdy = g->dxdy; d.z = g->z; d.y_begin = g->y_begin; d.y_end = g->y_end;
  d.weight = g->weight; d.group_xmin = g->group_xmin; d.group_xmax = g->group_xmax;
  d.sector_rows = reinterpret_cast<const float4*>(g->sector_rows);
  for (int l = 0; l < 4; ++l) { d.layer_z[l] = g->layer_z[l]; d.layer_dxdy[l] = g->layer_dxdy[l]; }
  return d;
}

// thread-local record of the last launches (ut_last_launch_info)
ut_launch_info& launch_info();
// records "<what>: <cuda error string>" for ut_last_error(); returns UT_ERR_CUDA
int32_t cuda_fail(const char* what, cudaError_t err);
// records `text` for ut_last_error(); returns `code`
int32_t fail_with(int32_t code, const char* text);

// Per-device facts and the dynamic shared-memory opt-in of the kernels.  cudaFuncAttributeMaxDynamicSharedMemorySize
// is a per-DEVICE attribute: the table is keyed by the current device and filled under a mutex, so any number of
// devices and host threads may call into the library.
struct DeviceInfo { int device, n_sm, smem_optin, smem_per_sm; };
enum KernelSlot { kSlotDecode = 0, kSlotCompassSmall = 1, kSlotCompassLarge = 7, kSlotWindows = 13, kSlotTracklets = 14,
                  kSlotCompassC16 = 15, kNumKernelSlots = 16 };     // (6 Compass slots each: interval search x {general, layer-uniform, kick table})
int32_t device_info(DeviceInfo* out);
// largest dynamic shared-memory size `kernel` may ask for on the current device (opted in on its first use there)
int32_t kernel_max_dynamic_smem(const void* kernel, int slot, int* max_dyn);
// the process-wide tuning values (ut_tuning_get / ut_tuning_set), read from the environment once
ut_tuning tuning_snapshot();
inline int tuned(int32_t v, int dflt) { return v >= 0 ? (int)v : dflt; }

#define UTC_CUDA(call)                                              \
  do {                                                              \
    const cudaError_t utc_err__ = (call);                           \
    if (utc_err__ != cudaSuccess) return utc::cuda_fail(#call, utc_err__); \
  } while (0)

#ifdef __CUDACC__

__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// ---- mbarrier + 1-D bulk copy (TMA unit, SASS UBLKCP) ----------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_u32(dst_smem)), "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}

// ---- single-word flags in global memory --------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_volatile_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_volatile_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}

// ---- warp helpers -------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t warp_sum(uint32_t v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
  return v;
}
__device__ __forceinline__ uint32_t warp_incl_scan(uint32_t v, int lane) {
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xFFFFFFFFu, v, o);
    if (lane >= o) v += t;
  }
  return v;
}

// Chained exclusive prefix over work items handed out by an atomic ticket (decoupled look-back; the decode
// chains events, the track consolidation chains tiles).  Called by one warp.  Item e only waits for items with a
// smaller ticket, which are running or finished, so it always makes progress.  flags[e] = epoch:30 | state:2 |
// value:32 with state 1 = the item's own total, 2 = inclusive prefix; the epoch makes the words reusable.
__device__ inline uint32_t event_base_lookback(unsigned long long* flags, int e, uint32_t tot, uint32_t epoch, int lane,
                                        const uint32_t* carry_in) {
  const unsigned long long tag = (unsigned long long)(epoch & 0x3FFFFFFFu) << 34;
  if (e == 0) {
    const uint32_t carry = carry_in ? ld_volatile_u32(carry_in) : 0u;
    if (lane == 0) st_volatile_u64(&flags[0], tag | (2ull << 32) | (unsigned long long)(carry + tot));
    return carry;
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

// bump allocator over dynamic shared memory, 16-byte granules
struct Carver {
  unsigned char* p;
  __device__ explicit Carver(unsigned char* base) : p(base) {}
  template <typename T>
  __device__ T* take(size_t n) {
    T* r = reinterpret_cast<T*>(p);
    p += (n * sizeof(T) + 15) & ~size_t(15);
    return r;
  }
};

#endif  // __CUDACC__

#ifdef __CUDACC__
__host__ __device__
#endif
inline size_t align16(size_t v) { return (v + 15) & ~size_t(15); }

}  // namespace utc
