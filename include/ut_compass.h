/* ut_compass.h -- C ABI of libutcompass: UT raw-bank decoding and Compass tracking on one B200.
 *
 * The two hot-path calls follow the problem statement of arxiv/paper_2002_11529
 * ("A parallel-computing algorithm for high-energy physics particle tracking and decoding
 * using GPU architectures"; citations are lines of the paper text, PAPER.md):
 *
 *   ut_decode      section IV: UT raw banks -> SoA hit container
 *                  {LHCbID, zAtYEq0, xAtYEq0, yBegin, yEnd, weight} (+ dxdy) grouped into sector
 *                  groups and sorted inside each group, plus the offsets array.
 *   compass_track  section V: every VELO track is extrapolated to the four UT
 *                  layers, window hits are collected per layer, 3/4-hit tracklets are enumerated from
 *                  seed pairs, fitted (chi2, q/p) and the best one is kept.
 *
 * Conventions
 *   - Plain C, no CUDA or torch types.  `ut_stream_t` is a cudaStream_t / CUstream handle (0 = default).
 *   - Unless a comment says HOST, every data pointer is a DEVICE pointer owned by the caller; the
 *     library never frees or reallocates it.  The descriptor structs themselves live in HOST memory.
 *   - Hot-path calls are asynchronous on `stream`, perform no host synchronisation and no allocation,
 *     and are CUDA-graph capturable.
 *   - Return value: 0 = launched; < 0 = invalid argument detected on the host (UT_ERR_*).
 *     Data-dependent errors set bits in the device `status` word of the output struct (UT_STATUS_*);
 *     kernels never write past `capacity`.
 *   - Arithmetic: IEEE fp32, round-to-nearest, no FMA contraction, operations in the order written
 *     in DESIGN.md section 3, so results are bit-identical to the reference definition.
 */
#ifndef UT_COMPASS_H
#define UT_COMPASS_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef void* ut_stream_t;

#define UT_N_LAYERS 4

/* host-detected errors */
#define UT_OK 0
#define UT_ERR_NULL (-1)        /* required pointer is null */
#define UT_ERR_ARG (-2)         /* negative size, bad config value, misaligned buffer */
#define UT_ERR_GEOMETRY (-3)    /* geometry table violates the container contract */
#define UT_ERR_CUDA (-4)        /* CUDA runtime error (allocation, launch) */
#define UT_ERR_LIMIT (-5)       /* table larger than the compiled limits (UT_MAX_*) */

/* data-dependent status bits (device word) */
#define UT_STATUS_UNKNOWN_SECTOR 1u    /* raw sector id not in id_to_sector            (bank ignored)   */
#define UT_STATUS_DUPLICATE_SECTOR 2u  /* two banks of one event name the same sector  (one ignored)    */
#define UT_STATUS_BAD_BANK_SIZE 4u     /* bank bytes != round4(6 + 2*count) or misaligned (bank ignored) */
#define UT_STATUS_CAPACITY 8u          /* hits would exceed `capacity`; that event's hits are not written */
#define UT_STATUS_BAD_OFFSETS 16u      /* compass_track: offsets not monotone / inconsistent            */
#define UT_STATUS_EVENT_TOO_LARGE 32u  /* compass_track: > 65535 hits in one event; no tracks for that event */
#define UT_STATUS_BAD_HIT_ID 64u       /* compass_track: a hit id names no sector of the geometry (hit ignored) */

#define UT_MAX_SECTORS 1024
#define UT_MAX_GROUPS 128
#define UT_MAX_CANDIDATES 32

/* Geometry tables (stand-in for the detector conditions of PAPER.md:231, :274).
 * Dense sector index s in [0, n_sectors): the sectors of one group are contiguous and groups are
 * numbered layer-major, so `sector_group` is non-decreasing; group g belongs to layer
 * g / (n_groups / n_layers).  A sector group is a region of unique X.
 * Contract checked by ut_geometry_upload: n_layers == 4; n_groups % 4 == 0; every group non-empty;
 * at most 32 sectors per group; dxdy constant inside a group; group_xmin and group_xmax
 * non-decreasing inside a layer;
 * pitch > 0; every x a sector can produce lies in [group_xmin, group_xmax] of its group. */
typedef struct {
  uint32_t n_layers, n_sectors, n_groups;
  uint32_t id_table_size;
  const uint32_t* id_to_sector;   /* [id_table_size] raw id -> dense s, 0xFFFFFFFF = invalid */
  const uint32_t* sector_raw_id;  /* [n_sectors] */
  const uint32_t* sector_group;   /* [n_sectors] */
  const float *x0, *pitch, *dxdy, *z, *y_begin, *y_end, *weight; /* [n_sectors] */
  const float *group_xmin, *group_xmax;                          /* [n_groups] bounds of xAtYEq0 */
  float layer_z[UT_N_LAYERS], layer_dxdy[UT_N_LAYERS];           /* HOST values inside the struct */
  /* filled by ut_geometry_upload (device, library-owned until ut_geometry_free) */
  const uint32_t* group_first_sector; /* [n_groups + 1] */
  const void* sector_rows;            /* [n_sectors] 32-byte rows {z, y_begin, y_end, dxdy | weight, raw id, x0,
                                         pitch}: the table row a decoded hit copies, packed for 128-bit loads */
  const uint32_t* sector_yorder;      /* [n_sectors] rank of the sector inside its group by (y_begin, dense index)
                                         | (sector-in-group index of the sector with that rank) << 8 */
  uint32_t flags;                     /* UT_GEOM_* properties found by ut_geometry_upload */
  void* owner;                        /* opaque allocation handle, NULL for caller-owned tables */
  /* Optional position-dependent kick table ("look-up tables are used, which give quick access to the
   * influence of the magnetic field", A24).  kick_nx == 0: the constants
   * compass_config.kappa / z_mag apply to every track.  Otherwise every VELO track takes its kappa and z_mag from the
   * cell that holds its straight-line position at kick_z_ref (nearest cell, no interpolation):
   *   x_k = x + tx*(kick_z_ref - z0), y_k likewise (fp32);  ix = clamp(floor((x_k - kick_x_lo)*kick_inv_dx), 0, nx-1),
   *   iy likewise (a NaN coordinate takes index 0);  cell = iy*kick_nx + ix.
   * HOST arrays on input to ut_geometry_upload, device arrays in its output; at most 4096 cells. */
  uint32_t kick_nx, kick_ny;
  float kick_x_lo, kick_y_lo, kick_inv_dx, kick_inv_dy, kick_z_ref;
  const float *kick_kappa, *kick_z_mag;   /* [kick_ny * kick_nx] */
  float layer_weight[UT_N_LAYERS];        /* filled by ut_geometry_upload: the one weight of the layer's sectors when
                                             UT_GEOM_LAYER_UNIFORM is set (HOST values inside the struct) */
} ut_geometry;

/* y_begin and y_end are non-decreasing over the sectors of every group: the sector row a track crosses
 * can be found by binary search (else compass_track scans the group's sectors). */
#define UT_GEOM_ROWS_SORTED 1u
/* every group of a layer has the same number of sectors with the same y ranges, row by row: compass_track finds the
 * sector row a track crosses once per layer instead of once per group */
#define UT_GEOM_ROWS_UNIFORM 2u
/* every sector of layer l has z == layer_z[l] and the same weight (layer_weight[l]): compass_track takes the z and the
 * weight of a candidate from the layer instead of from the sector rows (its own kernel variant) */
#define UT_GEOM_LAYER_UNIFORM 4u

/* Copies HOST tables (`host_tables` holds HOST pointers in the array fields) to the device, checks
 * the contract above and fills `device_out` with device pointers.  Synchronous; call once at set-up. */
int32_t ut_geometry_upload(const ut_geometry* host_tables, ut_geometry* device_out);
int32_t ut_geometry_free(ut_geometry* device_geometry);

/* SoA hit container.  All arrays have `capacity` elements.
 * Order: events ascending; inside an event sector groups ascending; inside a group ascending
 * x_at_y0, ties in fill order (dense sector, then word order in the bank).
 *   x_at_y0 = x0[s] + ((2*strip + frac)*0.5f + 0.25f) * pitch[s]     (fp32, two roundings)
 *   z_at_y0, y_begin, y_end, dxdy, weight = the sector's table row;  id = (raw_id << 9) | strip. */
typedef struct {
  float *x_at_y0, *z_at_y0, *y_begin, *y_end, *dxdy, *weight;
  uint32_t* id;
  uint64_t capacity;          /* (total_raw_bytes - 6*n_banks)/2 is always enough */
  const ut_geometry* geom;    /* HOST pointer to the device-table descriptor used to decode */
  uint32_t* status;           /* device word, OR-ed with UT_STATUS_* (caller zeroes it) */
  void* workspace;            /* device, ut_decode_workspace_bytes() bytes, zeroed once by
                                 ut_decode_workspace_init(); reusable across calls on one stream.
                                 Only ut_decode uses it: may be NULL for a container filled otherwise. */
  /* Optional per-sector view of the same hits (the "layer / sector / x-sorted" order of the problem statement;
   * PAPER.md:288-290 searches sector by sector): every dense sector's hits contiguous, in container order inside
   * the sector.  All three pointers or none (NULL).  ut_decode fills it in the same launch; compass_track stages
   * an event's window-search data from it with three bulk copies instead of re-bucketing the group-sorted arrays
   * (same results either way).  Entry k of sector s of event e sits at hit_offsets[n_groups*e] + sector_offsets
   * [e][s] + k. */
  float* x_by_sector;         /* [capacity rounded up to a multiple of 8] x_at_y0 */
  uint16_t* idx_by_sector;    /* [same] container index of the entry, relative to the event's first hit */
  uint16_t* sector_offsets;   /* [max_events][ut_sector_offsets_stride(geometry)]: n_sectors + 1 offsets relative to
                                 the event's first hit, then a word that is UT_SECTOR_INDEX_VALID if the row may be
                                 used (an event of > 65535 hits, a group larger than the decode's sort buffer or a
                                 capacity overflow leaves it 0 and compass_track re-buckets that event itself) */
  uint32_t order;             /* order inside a sector group, set by the caller before ut_decode: UT_ORDER_X (default)
                                 ascending x_at_y0; UT_ORDER_Y the paper's literal order (SURVEY.md
                                 8(f) row 3): ascending y_begin, then ascending x_at_y0.  Ties in fill order either way.
                                 compass_track reads it (window look-up by binary searches over Y, when
                                 it has to search global memory); the two-kernel variant takes UT_ORDER_X only. */
} ut_hits;
#define UT_ORDER_X 0u
#define UT_ORDER_Y 1u
#define UT_SECTOR_INDEX_VALID 0xA5A5u
uint32_t ut_sector_offsets_stride(const ut_geometry* geometry);   /* u16 elements per event, a multiple of 8 */

/* Bytes of `workspace` for batches of up to `max_events` events decoded with `geometry` (control words and one
 * look-back word per event; `geometry` may be NULL: the size does not depend on the tables today, the argument
 * is SURVEY.md 8(b)'s and keeps the call stable if per-sector scratch moves here). */
size_t ut_decode_workspace_bytes(int32_t max_events, const ut_geometry* geometry);
int32_t ut_decode_workspace_init(void* workspace, int32_t max_events, ut_stream_t stream);

/* ut_decode -- PAPER.md section IV.
 * raw_banks    : device bytes, 16-byte aligned, readable up to the next multiple of 16 past the end.
 *                Bank = u32 raw sector id | u16 count | count x u16 word | zero pad to 4 bytes;
 *                word = 9-bit strip | frac << 9 | ADC << 10 (ADC ignored).  Little endian.
 * bank_offsets : device u32 [n_events*n_sectors + 1], 16-byte aligned: byte offset of every bank and the
 *                end; the banks of an event are contiguous, one per sector, in any order.
 * hit_offsets_out : device u32 [n_events*n_groups + 1]: global exclusive prefix of group sizes; event e
 *                owns hits [off[n_groups*e], off[n_groups*(e+1)]).  Always exact, even on CAPACITY.
 * One kernel launch: per-sector count -> event total -> chained exclusive prefix over events
 * (decoupled look-back, no host sync; the paper reads the total back) -> bucketed fill
 * -> stable in-group ordering -> coalesced SoA store. */
int32_t ut_decode(const uint8_t* raw_banks, const uint32_t* bank_offsets, int32_t n_events,
                  const ut_geometry* geometry, ut_hits* hits_out, uint32_t* hit_offsets_out,
                  ut_stream_t stream);

/* ut_decode_static -- ut_decode for callers that cannot allocate device memory (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc).  Same kernel, same arguments, same results as ut_decode; the one
 * difference is where the kernel's scratch lives: the control words and the per-event look-back words that ut_decode
 * keeps in hits_out->workspace sit in ONE array built into the library (a file-scope __device__ array of
 * 32 + 8 * UT_DECODE_STATIC_MAX_EVENTS + 8 bytes rounded up to 256, about 128 KB, held by every GPU that loads the
 * library until the process exits).  hits_out->workspace is not read and may be NULL; no ut_decode_workspace_bytes /
 * ut_decode_workspace_init call is needed.  The call itself performs no cudaMalloc, cudaFree or other allocating
 * routine; inputs and outputs are the caller's as for ut_decode.
 *   - n_events > UT_DECODE_STATIC_MAX_EVENTS returns UT_ERR_LIMIT (ut_last_error() says so); nothing is launched.
 *   - Every call on a device shares the array and finds the previous call's contents in it: the call clears the two
 *     counters that must start at zero (stream-ordered, in front of the kernel) and keeps the epoch word, which makes
 *     the previous call's look-back words recognisable as stale.
 *   - Calls that OVERLAP on one GPU (two streams, two host threads, ut_decode_static inside concurrently replayed
 *     graphs) race on that array and produce wrong offsets or hang: serialise them (one stream, or events between
 *     streams).  ut_decode with one workspace per container has no such limit. */
#define UT_DECODE_STATIC_MAX_EVENTS 16384
int32_t ut_decode_static(const uint8_t* raw_banks, const uint32_t* bank_offsets, int32_t n_events,
                         const ut_geometry* geometry, ut_hits* hits_out, uint32_t* hit_offsets_out,
                         ut_stream_t stream);

/* VELO states: straight lines x(z) = x + tx*(z - z0), same for y, SoA. */
typedef struct {
  const float *x, *y, *tx, *ty; /* [n_velo_total] */
  float z;                      /* z0 of all states (770 mm in the synthetic workloads) */
} velo_states;

/* Compass configuration.  Derived fields are computed on the host once (double, rounded once).
 * The paper's two knobs -- sectors searched {1,3,5} and hit candidates {1..16} --
 * appear as the window half-widths and max_candidates_per_layer (readings A6, A7). */
typedef struct {
  float win_half[UT_N_LAYERS]; /* |d| <= win_half[l] selects window hits of layer l [mm] */
  float y_tol;                 /* y_begin - y_tol <= y_e <= y_end + y_tol [mm] */
  float max_slope;             /* |seed slope in residual space| limit */
  float kink_tol;              /* |seed-line intercept at z_mag| limit [mm] */
  float seed_tol;              /* |residual to the seed line| limit in the other two layers [mm] */
  float w_velo;                /* weight of the VELO pseudo-point (dz = 0, d = 0) in the fit */
  float max_chi2_ndf;          /* valid iff chi2 <= max_chi2_ndf * (n_hits - 1) */
  float kappa;                 /* q/p = slope / kappa  [MeV] */
  float z_mag;                 /* kick plane [mm] */
  int32_t min_hits;            /* 3 or 4 */
  int32_t max_candidates_per_layer; /* 1 .. UT_MAX_CANDIDATES, closest-first in |d| */
  int32_t both_directions;     /* 0: backward seeds (L3, L1) only for tracks where the forward seeds (L0, L2) gave no
                                  valid tracklet (A11); 1: best of both directions */
} compass_config;

/* win_half[l] = window_scale * (kappa/p_min_mev) * (layer_z[l] - z_mag) + 0.5,
 * max_slope = window_scale * kappa / p_min_mev + 0.0015, other fields DESIGN.md A8 defaults. */
int32_t compass_config_default(float p_min_mev, float window_scale, int32_t min_hits,
                               int32_t max_candidates_per_layer, const ut_geometry* geometry,
                               compass_config* out /* HOST */);

/* Track output: dense, one slot per VELO track (PAPER.md:348 without the atomicAdd; A13). */
typedef struct {
  int32_t* hit_idx;  /* [4][n_velo_total], row l = global hit index in layer l or -1 */
  int32_t* n_hits;   /* [n_velo_total] 0 (no tracklet), 3 or 4 */
  float* qop;        /* [n_velo_total] q/p in 1/MeV, sign = charge; 0 if none */
  float* chi2;       /* [n_velo_total] 0 if none */
  uint32_t* status;  /* device u32[4]: [0] status word (OR-ed with UT_STATUS_*, caller zeroes it); [1..3] scratch of
                        compass_track (its work ticket: zero once, the kernel re-arms it), so that calls with
                        different outputs may run at the same time on any streams */
} ut_tracks;

/* compass_track -- PAPER.md section V, fused (window search + tracklet finding in one kernel; the
 * paper's CPU port does the same).
 * hits, hit_offsets : as produced by ut_decode (hits->geom gives the group tables).
 * velo_offsets      : device u32 [n_events + 1]; n_velo_total = velo_offsets[n_events] (read on device).
 * The kernel is launched with programmatic stream serialization: when the preceding operation of `stream` is the
 * ut_decode kernel its CTAs may become resident on SMs that kernel has left and stage their geometry tables, and they
 * wait for its completion (griddepcontrol.wait) before they read hits, offsets or the per-sector view.  Stream order
 * is otherwise unchanged; behind any other operation the launch is an ordinary one. */
int32_t compass_track(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                      const uint32_t* velo_offsets, int32_t n_events, const compass_config* config,
                      ut_tracks* tracks_out, ut_stream_t stream);

/* Compacted VELO+UT track container ("a prefix sum and a consolidation of the tracks", which
 * replaces the atomicAdd slot allocation of PAPER.md:348): only the VELO tracks that got a tracklet, events
 * ascending and the VELO order inside an event kept, so the result is unique.  Arrays have `capacity`
 * elements (n_velo_total is always enough); hit_idx has row stride `capacity`. */
typedef struct {
  uint32_t* velo_index; /* [capacity] global VELO track index of the tracklet */
  int32_t* hit_idx;     /* [4][capacity] */
  int32_t* n_hits;      /* [capacity] 3 or 4 */
  float* qop;           /* [capacity] */
  float* chi2;          /* [capacity] */
  uint64_t capacity;
  uint32_t* status;     /* device word; UT_STATUS_CAPACITY if the tracklets do not fit (nothing past capacity
                           is written, track_offsets_out stays exact) */
  void* workspace;      /* device, compass_consolidate_workspace_bytes(max_velo_total) bytes, zeroed once;
                           reusable across calls on one stream */
  uint32_t max_velo_total; /* what the workspace was sized for; n_velo_total above it sets UT_STATUS_BAD_OFFSETS
                              and nothing is written */
} ut_compact_tracks;

size_t compass_consolidate_workspace_bytes(uint32_t max_velo_total);

/* compass_consolidate -- PAPER.md:460.  One launch: tiles of 1024 VELO tracks by atomic ticket, block scan of
 * the "has a tracklet" flags, chained exclusive prefix over tiles (decoupled look-back), coalesced stores.
 * tracks, velo_offsets : as given to / filled by compass_track (n_velo_total = velo_offsets[n_events], read on
 *                        the device; the row stride of tracks->hit_idx is n_velo_total).
 * track_offsets_out    : device u32 [n_events + 1]: event e owns compact tracks [off[e], off[e+1]). */
int32_t compass_consolidate(const ut_tracks* tracks, const uint32_t* velo_offsets, int32_t n_events,
                            ut_compact_tracks* out, uint32_t* track_offsets_out, ut_stream_t stream);

/* The paper's own two-kernel layout (section V-A / V-B): kept beside the fused
 * compass_track as an A/B measurement of the paper's layout claims, not as the product path.
 *
 * compass_search_windows -- "search UT windows": a 2-D kernel (4 panels x VELO tracks); per
 *   (track, panel) the sector group the extrapolation points to and its neighbours, n_sectors_search = 1, 3 or 5
 *   groups in all (central, -1, +1, -2, +2); per group the window range = the hits of the
 *   group's x-sorted run with |d| <= win_half[l] (two searches, nothing else: the y test is repeated by the tracklet
 *   kernel).  windows_out: device int16 [n_velo_total][4][2 * n_sectors_search] in the layout of
 *   Fig. 7 -- per track, per panel, W begin indices then W sizes; begin relative to the first hit of the track's
 *   event; (-1, -1) = no hits or no such group.  Events of more than 32767 hits cannot be
 *   indexed by shorts: UT_STATUS_EVENT_TOO_LARGE in *status, their ranges empty.  status: device u32 word.
 * compass_tracklets_from_windows -- "tracklet finding": thread per VELO track, window ranges
 *   cached in shared memory (num_threads x num_panels x 2W shorts), valid tracks compacted through
 *   shared memory; same predicates, cap, fit and selection as compass_track.
 * With 5 sector groups every group a window of the synthetic workloads can touch is searched and tracks_out equals
 * compass_track's bit for bit; 1 and 3 groups search less (the paper's physics / speed trade-off, Table 3). */
int32_t compass_search_windows(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                               const uint32_t* velo_offsets, int32_t n_events, const compass_config* config,
                               int32_t n_sectors_search, int16_t* windows_out, uint32_t* status, ut_stream_t stream);
int32_t compass_tracklets_from_windows(const ut_hits* hits, const uint32_t* hit_offsets, const velo_states* velo,
                                       const uint32_t* velo_offsets, int32_t n_events, const compass_config* config,
                                       int32_t n_sectors_search, const int16_t* windows, ut_tracks* tracks_out,
                                       ut_stream_t stream);

/* End-to-end convenience for HOST buffers (bench.py "e2e"): H2D of raw banks, offsets and VELO
 * states, ut_decode, compass_track, D2H of the track SoA, all asynchronous on `stream`.
 * The arena holds the device staging buffers (library-owned). Host buffers should be pinned. */
typedef struct ut_pipeline ut_pipeline;
int32_t ut_pipeline_create(const ut_geometry* device_geometry, int32_t max_events, size_t max_raw_bytes,
                           uint64_t max_hits, uint32_t max_velo, ut_pipeline** out);
int32_t ut_pipeline_destroy(ut_pipeline* p);
/* All pointers HOST.  tracks_host receives hit_idx/n_hits/qop/chi2; status_host[0] the decode's status word and
 * status_host[1] Compass's; *n_hits_host the total decoded hits.  Returns after enqueueing; sync the stream to read.
 * Any host pointers work.  Every copy costs ~10 us of engine latency on top of its bytes, so layouts that let several
 * arrays travel as ONE strided copy are the fast ones: the four VELO arrays evenly spaced inside one page-locked
 * allocation (x, y, tx, ty rows of one block), and the track SoA as one [7][n_velo_total] block -- hit_idx (4 rows),
 * then n_hits, qop, chi2 back to back (n_hits == hit_idx + 4*n_velo_total ...), which leaves by a single copy per
 * chunk; n_hits/qop/chi2 evenly spaced but apart from hit_idx take two.  The call recognises these layouts itself. */
int32_t ut_pipeline_run_host(ut_pipeline* p, const uint8_t* raw_banks_host, size_t raw_bytes,
                             const uint32_t* bank_offsets_host, const velo_states* velo_host,
                             const uint32_t* velo_offsets_host, uint32_t n_velo_total, int32_t n_events,
                             const compass_config* config, ut_tracks* tracks_host, uint32_t* status_host,
                             uint32_t* n_hits_host, ut_stream_t stream);
/* Device-side timeline of the most recent ut_pipeline_run_host on `p`, read after the stream was synchronised
 * (tracing aid; bench.py reports it): ms_out[k*5 + q] = milliseconds from the start of the call to the point where
 * chunk k had q = 0: its raw banks and offsets on the device, 1: its VELO states, 2: been decoded, 3: been tracked,
 * 4: its tracks on the host; *n_chunks_out = chunks the call used (<= 4; ms_out holds 20 floats); -1 = not recorded
 * (zero-copy runs record no copy-in point). */
int32_t ut_pipeline_timeline(ut_pipeline* p, float* ms_out, int32_t* n_chunks_out);
/* Page-locked HOST memory for the buffers handed to ut_pipeline_run_host (cudaHostAlloc, portable and mapped; 256-byte
 * aligned).  Any pinned memory works; this is the allocation the copy engines were measured at full PCIe rate with
 * on the bench box (other pinned allocations of the same size copied at a quarter of it in some processes).
 * ut_host_free releases it (never free() it).  Returns UT_ERR_CUDA when the allocation fails. */
int32_t ut_host_alloc(void** out, size_t bytes);
int32_t ut_host_free(void* p);
/* Device views of the arena (valid after a run): decoded hits and offsets, for inspection. */
int32_t ut_pipeline_device_hits(ut_pipeline* p, ut_hits* hits_out, const uint32_t** hit_offsets_out);

/* Launch statistics of the most recent call on this thread (host side, no sync). */
typedef struct {
  int32_t kernels_launched;     /* kernels enqueued by the last hot-path call */
  int32_t decode_grid, decode_block, decode_smem_bytes;
  int32_t decode_raw_stage_bytes;   /* shared-memory staging of one event's raw banks (larger events read global memory) */
  int32_t decode_sort_buf;          /* per-warp sort buffer, in hits (larger groups rank by recomputation) */
  int32_t compass_grid, compass_block, compass_smem_bytes, compass_hit_stage;
  int32_t compass_split;            /* CTAs sharing the tracks of one event (1, 2 or 4) */
  int32_t compass_view;             /* 1: the container's per-sector view was offered to the kernel */
  int32_t decode_hit_stage;         /* hits (padded fill order) of an event the decode CTA orders as a whole; larger events
                                       and UT_ORDER_Y containers are ordered warp per sector group */
  int32_t compass_event_order;      /* events the Compass CTAs hand out heaviest first (0: in batch order) */
} ut_launch_info;
void ut_last_launch_info(ut_launch_info* out);

/* Launch tuning, process-wide (HOST).  -1 = automatic.  The values are read ONCE from the environment when the
 * library is first used (UT_DECODE_BLOCK, UT_DECODE_RAW_STAGE, UT_DECODE_SORT_BUF, UT_DECODE_MAX_CTAS_PER_SM,
 * UT_COMPASS_BLOCK, UT_COMPASS_HIT_STAGE, UT_COMPASS_TRK_STAGE, UT_COMPASS_SPLIT, UT_COMPASS_INTERVAL_MIN,
 * UT_PIPELINE_CHUNK_EVENTS, UT_PIPELINE_ZERO_COPY, UT_DECODE_HIT_STAGE, UT_COMPASS_EVENT_ORDER); the
 * hot-path calls never touch the environment.  ut_tuning_set replaces them (NULL: back to the environment's).
 * Results never depend on these values, only launch shapes and which of the equivalent code paths run. */
typedef struct {
  int32_t decode_block;             /* threads per decode CTA */
  int32_t decode_raw_stage_bytes;   /* shared-memory staging of an event's raw banks */
  int32_t decode_sort_buf;          /* per-warp sort buffer of the warp-per-group path, in hits */
  int32_t decode_max_ctas_per_sm;
  int32_t compass_block;            /* threads per Compass CTA */
  int32_t compass_hit_stage;        /* hits of an event staged in shared memory; 0: window search on global memory */
  int32_t compass_trk_stage;        /* tracks of an event that can be ordered by radius */
  int32_t compass_split;            /* CTAs sharing one event's track batches (1, 2 or 4) */
  int32_t pipeline_chunk_events;    /* ut_pipeline_run_host: events per overlapped chunk */
  int32_t compass_interval_min;     /* seed partner lists longer than this are searched (interval of d), not walked */
  int32_t pipeline_zero_copy;       /* ut_pipeline_run_host: 0 = always stage the raw banks with copies; else the decode
                                       reads mapped pinned host buffers directly over PCIe */
  int32_t decode_hit_stage;         /* largest event (hits) a decode CTA orders as a whole; 0: always warp per sector group */
  int32_t compass_event_order;      /* 0: Compass hands the events of a batch out in batch order; else (default) by descending
                                       track count when the batch is 149-4096 events and shared memory has room for the table */
  int32_t reserved[3];
} ut_tuning;
int32_t ut_tuning_get(ut_tuning* out);
int32_t ut_tuning_set(const ut_tuning* in);

const char* ut_version(void);
/* Text of the last UT_ERR_CUDA on this thread ("<call>: <cuda error string>") or of the last UT_ERR_LIMIT of
 * ut_decode_static, "" if none. */
const char* ut_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* UT_COMPASS_H */
