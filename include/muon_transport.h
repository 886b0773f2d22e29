/* muon_transport.h — C ABI of the B200-native muon transport library (libmuon_transport.so).
 *
 * The library implements the per-muon transport step loop of "Ultra-Fast Muon Transport via Histogram
 * Sampling on GPUs" (arxiv 2512.10520): Algorithm 1 (§4) with the sampling of §2-§3
 * (L51-53, L73-77), the rotation of §4.2 (L124-129, Eq. 3) and the RK4 Lorentz push of §4.3 (L133-137,
 * Eq. 4).  The exact arithmetic is DESIGN.md §3.  Call order follows the paper's statement of the problem
 * (Alg. 1 "Input", L144-146; static data resident in GPU global memory, L174):
 *
 *     mt_create -> mt_load_histograms -> mt_build_alias -> mt_set_geometry -> mt_transport (any number)
 *
 * Conventions.  Units: metres, GeV/c, tesla.  Every function returns an int status: MT_OK (0) or a
 * negative MT_ERR_* code; nothing throws or aborts across this boundary; mt_last_error() gives a text for
 * the last failure on a context.  A context belongs to one CUDA device and is not thread-safe; its transports share
 * library-owned scratch, so successive mt_transport calls on one context must be ordered on the device (same stream, or
 * streams synchronised by the caller).  "HOST"
 * pointers are ordinary host memory, read during the call and never retained.  "DEVICE" pointers are
 * CUDA device memory on the context's device; the caller owns them (the library never frees them), and
 * those marked "borrowed" must stay valid and unchanged until the context is destroyed or the geometry is
 * replaced.  There is no CPU implementation behind these calls: without a CUDA device they fail.
 */
#ifndef MUON_TRANSPORT_H_
#define MUON_TRANSPORT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mt_ctx mt_ctx;

enum {
  MT_OK = 0,
  MT_ERR_INVALID_ARG = -1, /* null pointer, non-positive size, unsorted regions, ...                      */
  MT_ERR_STATE = -2,       /* call order violated (e.g. mt_transport before mt_set_geometry)               */
  MT_ERR_EMPTY_HIST = -3,  /* a (material, bin) histogram sums to 0 or holds a negative / non-finite count */
  MT_ERR_UNSUPPORTED = -4, /* a size beyond what the kernels support (see each call)                       */
  MT_ERR_CUDA = -5,        /* a CUDA runtime call failed; mt_last_error() has the CUDA message             */
  MT_ERR_NOMEM = -6
};

/* termination flags written to the outputs (Alg. 1 l.2-4, L148-151) */
enum { MT_FLAG_STOPPED = 1, MT_FLAG_EXITED = 2, MT_FLAG_ESCAPED = 3, MT_FLAG_MAXSTEPS = 4 };

enum {
  MT_GEOM_REGIONS = 0,     /* axis-aligned boxes found through a sorted z-interval table (BASELINE.json configs[0-2])      */
  MT_GEOM_VOXEL = 1,       /* uint8 material grid + float32x3 field grid (configs[3-4])                                    */
  MT_GEOM_POLY = 2         /* the paper's own: convex polyhedra, slice + Eq. 2 sign test, spatial-hash pruning (L109-120)  */
};

/* what the histograms hold (mt_hist_desc.hist_mode) */
enum {
  MT_HIST_MARGINAL = 0,    /* BASELINE.json configs: one Dp/p and one polar-angle histogram per (material, bin)    */
  MT_HIST_JOINT = 1        /* the paper's own (L77, Fig. 3): ONE 2D histogram per (material, bin) over             */
};                         /* (log2 of -dPz/|P|, log2 of dPt/|P|), sampled through one alias table*/

/* field lookup (mt_geometry.field_mode): interpolation, optionally | MT_FIELD_PER_STAGE */
enum {
  MT_FIELD_TRILINEAR = 0,  /* trilinear over cell centres (BASELINE.json configs[3]); regions: the region's B     */
  MT_FIELD_NEAREST = 1,    /* VOXEL mode: the value of the cell that contains the point (the paper's own, L133)   */
  MT_FIELD_PER_STAGE = 2   /* flag: B looked up at every Runge-Kutta stage position instead of once per step       */
};

/* where the compact exit list records an EXITED muon (mt_geometry.exit_mode) */
enum {
  MT_EXIT_AT_BREAK = 0,    /* its state at the break of Algorithm 1: up to one step length behind the exit plane (default) */
  MT_EXIT_PROJECT = 1      /* moved back onto the plane z = z_exit along its final direction; momentum unchanged.  The  */
};                         /* dense outputs pos_flag / mom_steps are never changed by this                              */

/* alias-table placement (north_star subsystem 1): gathered through L1 / L2, which is what AUTO picks (the field grid does
 * not allocate in L1, so the tables have it to themselves), or the longest prefix of whole materials that fits
 * staged in shared memory by every CTA */
enum { MT_PLACE_AUTO = 0, MT_PLACE_SMEM = 1, MT_PLACE_L2 = 2 };

/* scheduling of muons onto lanes (north_star subsystem 4); results never depend on it */
enum {
  MT_SCHED_AUTO = 0,
  MT_SCHED_STATIC = 1,     /* one lane per muon for its whole life (the paper's mapping, L59, L174)        */
  MT_SCHED_REFILL = 2,     /* persistent warps; idle lanes refill from a global work counter               */
  MT_SCHED_WAVEFRONT = 3   /* z-slab passes over a compacted live list (field working set stays in L2/L1)  */
};

/* integer options for mt_set_option */
enum {
  MT_OPT_SCHEDULE = 1,       /* MT_SCHED_*                                                                 */
  MT_OPT_BLOCK_THREADS = 2,  /* 0 = library default; else a multiple of 32 in [32, 768] (the largest block  */
                             /* the transport kernels are compiled for)                                    */
  MT_OPT_BLOCKS_PER_SM = 3,  /* 0 = library default (persistent kernels)                                   */
  MT_OPT_SLAB_CELLS = 4,     /* wavefront: slab thickness along z, in units of 1 cm; 0 = default (by geometry */
                             /* and call size: voxel grids 96 for a full batch, thicker for small calls)      */
  MT_OPT_REFILL_MIN_IDLE = 5,/* refill: lanes of a warp that must be idle before it refills; 0 = default   */
  MT_OPT_KEY_LOOKAHEAD = 6,  /* wavefront: the sort key is the xy cell a muon reaches after this many percent */
                             /* of a slab on a straight line; -1 = default (50), 0 = its current cell         */
  MT_OPT_HASH_NXY = 7,       /* POLY: cells of the spatial hash along x and along y; 0 = default (16); 1..256 */
  MT_OPT_HASH_NZ = 8,        /* POLY: cells of the spatial hash along z; 0 = default (256); 1..4096.  Both    */
                             /* take effect at the next mt_set_geometry; results never depend on them         */
  MT_OPT_NO_LEAN = 9,        /* 1: never take the kernel variants that drop operations the host has proven to  */
                             /* be identities for the loaded tables and geometry; for testing    */
  MT_OPT_LANES = 10,         /* concurrent lanes a call is split into (contiguous id ranges on library-owned    */
                             /* streams, joined on the caller's stream); 0 = default (by n), 1..16             */
  MT_OPT_PASS_MODE = 12,     /* WAVEFRONT passes: 1 = persistent CTAs pulling 32-muon items from a counter; 2 = one  */
                             /* item per warp, CTAs exit with their items (lanes interleave); 0 = default          */
  MT_OPT_LANE_PRIORITY = 13, /* lane streams: 1 = priorities descending with the lane index; 2 = equal; 0 = default  */
  MT_OPT_SORT_EVERY = 14,    /* WAVEFRONT: the live list is re-sorted by xy cell after every k-th pass; 0 = default (1) */
  MT_OPT_CHECK_SELFTEST = 11 /* checked build only (MT_INFO_CHECK_ERRORS): 1 hands the kernels a wrong table size */
                             /* so that the bounds checks must fire; MT_ERR_UNSUPPORTED in the normal build     */
};

const char* mt_strerror(int code);
const char* mt_last_error(const mt_ctx* ctx);

/* Create / destroy a context on CUDA device `cuda_device`.  MT_ERR_CUDA if there is no such device. */
int mt_create(mt_ctx** out, int cuda_device);
int mt_destroy(mt_ctx* ctx);
int mt_set_option(mt_ctx* ctx, int option, int64_t value);

/* Histograms H_{M,i} (BASELINE.json configs[0]: one Dp/p and one polar-angle
 * histogram per material and momentum bin, on log2 axes).  All arrays HOST, row-major, copied. */
typedef struct {
  int32_t n_materials;     /* material ids 1..n_materials; id 0 = vacuum, never sampled (L155); <= 255     */
  int32_t n_pbins;         /* log-spaced momentum bins over [p_lo, p_hi] GeV/c (L99); 1..4096              */
  float p_lo, p_hi;
  int32_t n_dp, n_th;      /* cells per Dp/p and per theta histogram; 1..65536                             */
  const float* counts_dp;  /* [n_materials][n_pbins][n_dp] non-negative weights                            */
  const float* counts_th;  /* [n_materials][n_pbins][n_th]                                                 */
  const float* axis_dp;    /* [n_materials][n_pbins][2] = {log2 of the lower edge, log2 width of a cell}   */
  const float* axis_th;    /* same for theta (radians)                                                     */
  const float* step_m;     /* [n_materials + 1] path length per step in material id (index 0 = vacuum)     */
  int32_t hist_mode;       /* MT_HIST_MARGINAL | MT_HIST_JOINT.  JOINT: counts_dp is [n_materials][n_pbins][n_dp][n_th]*/
                           /* (axis a = longitudinal loss, n_dp cells, axis_dp; axis b = transverse kick, n_th     */
                           /* cells, axis_th), counts_th is ignored, and n_dp * n_th <= 2^24, n_dp * n_th^2 < 2^32  */
} mt_hist_desc;
int mt_load_histograms(mt_ctx* ctx, const mt_hist_desc* desc);

/* Build the alias tables (Walker/Vose; construction order DESIGN.md §3.9), pack them
 * and upload them.  MT_ERR_EMPTY_HIST names the offending table in mt_last_error().  A failed call leaves the context
 * without tables (the previous ones are not kept): MT_ERR_STATE from mt_set_geometry / mt_transport until it succeeds. */
int mt_build_alias(mt_ctx* ctx, int placement);

/* Test export of the tables as built: HOST outputs shaped like counts_dp / counts_th.  JOINT mode: prob_dp / alias_dp
 * are [n_materials][n_pbins][n_dp * n_th]; prob_th / alias_th are not written and may be NULL. */
int mt_get_alias(const mt_ctx* ctx, float* prob_dp, uint32_t* alias_dp, float* prob_th, uint32_t* alias_th);

/* Geometry G and field map (Alg. 1 "Input", L144-146; L61-63; §4.3).  Regions: axis-aligned boxes,
 * half-open on every axis, sorted by z_lo and disjoint in z.  Voxel: cell (ix,iy,iz) spans
 * [o + i*cell, o + (i+1)*cell); field values sit at cell centres and are interpolated trilinearly. */
typedef struct {
  float z_lo, z_hi, x_lo, x_hi, y_lo, y_hi;
  int32_t material;
  float bx, by, bz;        /* uniform field inside the box                                                 */
} mt_region;

/* One convex block of MT_GEOM_POLY (§4.1): the solid between a lower
 * quadrilateral face at z_lo and an upper one at z_hi, vertex i of one joined to vertex i of the other.  The four
 * vertices go round the face in either orientation (the same for both faces); each face must be convex; a
 * repeated vertex gives a triangle, four equal vertices an apex.  A point is inside if z_lo <= z < z_hi and the
 * cross products S_i of Eq. 2 against the four edges of the slice interpolated at its z have one sign (zeros
 * allowed, not all zero).  Where blocks overlap the one with the lowest index wins. */
typedef struct {
  float z_lo, z_hi;
  float xy_lo[4][2];       /* (x, y) of the lower face's vertices                                          */
  float xy_hi[4][2];       /* (x, y) of the upper face's vertices                                          */
  int32_t material;
  float bx, by, bz;        /* uniform field inside the block                                               */
} mt_poly_block;

typedef struct {
  int32_t mode;            /* MT_GEOM_REGIONS | MT_GEOM_VOXEL | MT_GEOM_POLY                               */
  float x_min, x_max, y_min, y_max, z_min, z_exit; /* world box; z >= z_exit -> EXITED                    */
  float p_min;             /* |p| < p_min -> STOPPED                                                       */
  int32_t max_steps;       /* step cap -> MAXSTEPS                                                         */
  int32_t world_material;  /* material outside every region / outside the voxel grid                       */
  int32_t n_regions;       /* REGIONS mode: 0..1024                                                        */
  const mt_region* regions;/* HOST, copied                                                                 */
  int32_t nx, ny, nz;      /* VOXEL mode                                                                   */
  float ox, oy, oz, cell;
  const uint8_t* d_material; /* DEVICE [nz][ny][nx], read during the call only                            */
  const float* d_field;      /* DEVICE [nz][ny][nx][3], read during the call only                         */
  int32_t field_mode;        /* MT_FIELD_TRILINEAR | MT_FIELD_NEAREST, optionally | MT_FIELD_PER_STAGE             */
  int32_t n_blocks;          /* POLY mode: 0..1024                                                           */
  const mt_poly_block* blocks; /* HOST, copied.  The library bins their bounding boxes into a uniform grid  */
                             /* over the world box (the spatial hash of L120) and tests only a cell's candidates */
  int32_t exit_mode;         /* MT_EXIT_AT_BREAK | MT_EXIT_PROJECT: what mt_muons_out.exit_rec holds         */
} mt_geometry;
/* VOXEL mode repacks both grids into one library-owned grid of 32-byte records (field and material of a cell, and the
 * field difference to its +x neighbour), so the caller may free d_material / d_field after the call
 * returns.  The library's copy takes 32 bytes per cell of the grid padded by one cell on every side.
 * On failure: an argument error found before anything is touched leaves the previous geometry in place; a failure
 * after the library's grid has been overwritten (a material id above n_materials in d_material, a CUDA error) leaves
 * the context WITHOUT a geometry, and mt_transport then returns MT_ERR_STATE until mt_set_geometry succeeds.  If the
 * failure is a CUDA error while the tables are re-uploaded in the new geometry's material order, the tables are gone as
 * well (mt_build_alias, then mt_set_geometry).
 * mt_load_histograms invalidates the tables and the geometry; mt_build_alias keeps a geometry that is set. */
int mt_set_geometry(mt_ctx* ctx, const mt_geometry* geom);

/* Muon state, SoA of 16-byte records (north_star subsystem 3). */
typedef struct {
  const float* pos_q;      /* [n][4] = x, y, z, charge (+1.f / -1.f)                                       */
  const float* mom;        /* [n][4] = px, py, pz, unused                                                  */
} mt_muons_in;

typedef struct {
  float* pos_flag;         /* [n][4] = final x, y, z, flag (int32 bits in the 4th float)                   */
  float* mom_steps;        /* [n][4] = final px, py, pz, step count (int32 bits)                           */
  float* exit_rec;         /* optional [exit_capacity][8]: x,y,z,index(uint32 bits),px,py,pz,steps(int32);  */
                           /* x,y,z per mt_geometry.exit_mode                                              */
  uint32_t* exit_count;    /* optional, one counter; ADDED to (caller zeroes it): one per EXITED muon, so it */
                           /* may exceed the capacity; may be given WITHOUT exit_rec to count hits only     */
  uint32_t exit_capacity;
  uint64_t* counters;      /* optional [8], ADDED to: [0] total steps, [1..4] muons per flag; [5..7] stay  */
                           /* untouched (a -DMT_SLOT_STATS diagnostic build counts lane-slots there)       */
} mt_muons_out;

/* Transport n muons (ids id_base .. id_base+n-1) until each meets a break condition.  All buffers DEVICE.
 * Asynchronous: kernels are enqueued on `cuda_stream` (a cudaStream_t; NULL = default stream) and the call
 * returns; outputs are complete when the stream reaches that point.  Outputs are a function of (inputs,
 * seed, id) only — not of launch shape, schedule, batch split or refill order.  The library's scratch grows to the
 * largest batch seen: the first call at a larger n than any before it allocates (cudaMalloc, which synchronises the
 * device) before it enqueues; calls at the same or a smaller n do not.  MT_ERR_STATE unless mt_build_alias and
 * mt_set_geometry have both succeeded since the last mt_load_histograms. */
int mt_transport(mt_ctx* ctx, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                 const mt_muons_out* out, void* cuda_stream);

/* Same with HOST buffers: copies in, transports, copies out, then synchronises `cuda_stream`; returns when the outputs
 * are in host memory.  Large calls are cut into lanes (MT_OPT_LANES) so that one lane computes while others copy; pinned
 * (page-locked) buffers are what makes those copies asynchronous — pageable buffers work, serially.
 * exit_rec / exit_count / counters (if non-NULL) are HOST too; exit_count and counters are overwritten. */
int mt_transport_host(mt_ctx* ctx, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                      const mt_muons_out* out, void* cuda_stream);

/* mt_transport for callers that must not allocate device memory while they transport.
 *
 * Who that is: code that runs after another component has claimed the device's memory for itself (a framework's caching
 * pool, a memory budget fixed at start-up, a partition with a hard cap), where a cudaMalloc may fail at any moment; and
 * code inside a latency-bound loop (a trigger-level or online simulation step, a service answering requests), where
 * cudaMalloc / cudaFree stall every stream of the device while they run.  mt_transport cannot serve them: its z-slab
 * passes park the muons still in flight, their sort keys and the pass counters in library scratch that it cudaMallocs
 * whenever a call is larger than any before it, and it creates streams and events for its lanes.
 *
 * This call computes exactly what mt_transport computes (same arguments, all buffers DEVICE and the caller's; same
 * outputs bit for bit; same schedule: MT_OPT_SCHEDULE, or the library's choice by geometry and n) but keeps all of that
 * scratch in ONE array that is part of the library's image: MT_STATIC_SCRATCH_BYTES (9 MiB) of device memory that every
 * GPU holds from the moment it loads the library until the process exits, whether this call is ever used or not.  It
 * runs as a single lane on `cuda_stream` itself, and it never calls cudaMalloc, cudaFree, a stream / event constructor
 * or any other routine that allocates.  The price is the size limit: n <= MT_STATIC_SCRATCH_MAX_MUONS (65 536; the
 * array is sized so that every geometry and option setting fits at that n).  A larger n returns MT_ERR_UNSUPPORTED
 * with the limit in mt_last_error() and enqueues nothing; cut the batch into calls of at most that size with their own
 * id_base — results do not depend on the split.
 *
 * First call on a device: the library asks the runtime where that device's copy of the array lives (once per device and
 * process, remembered), and CUDA loads the kernels the call launches.  Make one call — any n >= 1 — during your own
 * set-up, before the phase that must not allocate and before you begin capturing a stream.  The tables and the geometry
 * of the context are device memory too: mt_build_alias / mt_set_geometry allocate them and belong in that set-up as well.
 *
 * The array is shared by every call of this entry point on the device, from every context and thread, and nothing
 * remembers who used it last: each call clears the counters it needs on `cuda_stream` before its kernels, so the
 * previous call's leftovers are harmless, but two calls whose work overlaps on the GPU (different streams without an
 * event between them, two host threads) overwrite each other's in-flight muons.  Order them on one stream, or make the
 * second stream wait for the first.  Calls of mt_transport itself use other memory and may overlap with this one.
 * Errors otherwise as mt_transport: MT_ERR_STATE / MT_ERR_INVALID_ARG before anything is enqueued, MT_ERR_CUDA with the
 * runtime's message. */
enum { MT_STATIC_SCRATCH_MAX_MUONS = 65536, MT_STATIC_SCRATCH_BYTES = 9 * 1024 * 1024 };
int mt_transport_static_scratch(mt_ctx* ctx, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                                const mt_muons_out* out, void* cuda_stream);

/* Number of kernel launches made by this context so far (bench.py's gpu_launches). */
int64_t mt_launch_count(const mt_ctx* ctx);

/* Introspection for tests and bench.py: *value = the item `what` of the context. */
enum {
  MT_INFO_LEAN_FACTS = 1,  /* bit 0: table axes proven inside the clamps; bit 1: world box proven inside the voxel grid   */
  MT_INFO_LAST_LEAN = 2,   /* 1 if the last mt_transport call ran the lean kernel variant                                */
  MT_INFO_LAST_SCHEDULE = 3,/* MT_SCHED_* the last mt_transport call ran under                                           */
  MT_INFO_LAST_LANES = 4,  /* number of concurrent lanes the last mt_transport call was split into                        */
  MT_INFO_CHECK_ERRORS = 5 /* -1 in the normal build.  Checked build (libmuon_transport_checked.so, compiled with           */
                           /* -DMT_CHECKED: every index into a global array is bounds-checked in the kernels instead of       */
                           /* dereferenced): low 32 bits = violations so far, high 32 bits = highest violation code;         */
                           /* synchronises the device                                                                       */
};
int mt_get_info(const mt_ctx* ctx, int what, int64_t* value);

/* Test hooks (DEVICE buffers, asynchronous on the stream).
 * mt_debug_sample: cell_out[i] = alias draw from table `which` (0 = Dp/p, 1 = theta) of
 * (material, pbin) with word d_words[i].  JOINT mode (which = 0): d_words holds 2n words, the select word of draw i
 * at [i] and its accept word at [n + i]; cell_out[i] is the flat cell index.
 * mt_debug_philox: out[i][0..3] = Philox4x32-10 block for (seed, id_base + i, step), computed by the
 * step loop's own routine (host-made round keys) and cross-checked on the device against the form with the key
 * schedule inline. */
int mt_debug_sample(mt_ctx* ctx, int material, int pbin, int which, const uint32_t* d_words, uint64_t n,
                    uint32_t* d_cell_out, void* cuda_stream);
int mt_debug_philox(mt_ctx* ctx, uint64_t seed, uint64_t id_base, uint32_t step, uint64_t n,
                    uint32_t* d_out, void* cuda_stream);
/* mt_debug_lookup: material_out[i] and field_out[i][0..2] = the material id and the field the step loop sees at the
 * point d_xyz[i][0..2] in the geometry that is set — regions, voxel (trilinear or
 * nearest per field_mode) or polyhedra (through the spatial hash). */
int mt_debug_lookup(mt_ctx* ctx, const float* d_xyz, uint64_t n, int32_t* d_material_out, float* d_field_out,
                    void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* MUON_TRANSPORT_H_ */
