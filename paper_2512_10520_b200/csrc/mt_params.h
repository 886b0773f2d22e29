// mt_params.h — plain structs shared by the host side (mt_lib.cu) and the kernels (mt_kernels.cu).
// Part of the CUDA path; shares nothing with oracle/.
#pragma once
#include <stdint.h>

// Region record as staged in shared memory: mt_region's ten words in three 16-byte groups, so that a
// lookup is three 128-bit shared-memory loads instead of ten scalar ones.
struct __align__(16) MtRegionDev {
  float z_lo, z_hi, x_lo, x_hi;
  float y_lo, y_hi;
  int32_t material;
  float bx;
  float by, bz, pad0, pad1;
};

// The "const blob": small read-only arrays every CTA stages into shared memory at start.
//   [0, n_pbins]                         momentum-bin edges, float32
//   [off_edges_open + 0 .. n_pbins]      the same edges with the first replaced by -inf and the last by +inf
//   [off_steps + 4*m .. +3]              h, h/2, h/6 of material m, m = 0..n_materials, and the
//                                        first cell of the material's tables in the packed array (int bits)
//   [off_axes + 4*t .. +3]               lo_dp, d_dp * 2^-16, lo_th, d_th * 2^-16 (log2) of table t = (m-1)*n_pbins + i
//   [off_zlo  + j]                       z_lo of region j (search array)
//   [off_regions + 12*j ..]              MtRegionDev j
//   [off_blocks + 24*j ..]               MtBlockDev j (POLY mode)
//   [off_binlut ..]                      uint16 momentum-bin table (two per word), see MtParams::bin_shift
//   [off_zlut ..]                        int16 z-interval table (two per word), see MtParams::zlut_n; the z_lo array is
//                                        followed by two +inf entries so that the table's two fix-ups need no bound
#ifndef MT_AXES_GLOBAL
#define MT_AXES_GLOBAL 1     // per-table axes read from global memory (L1) instead of a shared-memory copy
#endif
// Words of the blob a CTA stages: everything, or everything but the axes (which then take no shared memory either: the
// arrays behind them move down by the axes' length)
#define MT_STAGED_WORDS(bl) (MT_AXES_GLOBAL ? (bl).n_words - ((bl).off_zlo - (bl).off_axes) : (bl).n_words)
struct MtBlobLayout {
  int32_t off_edges_open, off_steps, off_axes, off_zlo, off_regions, off_blocks, off_binlut, off_zlut, n_words;
};

// Polyhedra block as staged in shared memory: six float4.  inv_dz = 1 / (z_hi - z_lo), dx_i = xh_i - xl_i and
// dy_i = yh_i - yl_i are the float32 operations of DESIGN.md §3.12, done once on the host.
struct __align__(16) MtBlockDev {
  float z_lo, z_hi, inv_dz;
  int32_t material;
  float bx, by, bz, pad;
  float xl[4], yl[4], dx[4], dy[4];
};

// Two x-neighbours of the padded field grid in one 32-byte record, so that the x-pair of a trilinear corner set
// is one 256-bit load.  a = field of cell x; b = field of cell x+1 MINUS that of cell x, each component
// rounded once (the subtraction of §3.3's x-lerp, precomputed); .w = material id of cell x / x+1 (int bits).
struct __align__(32) MtCellPair {
  float4 a, b;
};

// Facts the host proves about a (tables, geometry) pair; when all hold, the LEAN kernel variant drops the operations
// that they turn into identities (results unchanged):
//   MT_LEAN_AXES    every table axis keeps y = fma(cell.jitter, d, lo) inside [-120, 120] (exp2c's clamps), every Dp/p axis
//                   ends below log2(0.999) with a margin of 2^-9 (the cap on f) and every theta axis below log2(0.78)
//                   (theta < pi/4: the cap at pi and the quadrant reduction of its sine and cosine); JOINT tables: the
//                   transverse axis ends at or below 0 (ft <= 1: the new |p| stays in the fast sqrt / rcp range)
//                   and the momentum-bin table exists (bin_shift != 0): the bin is read from it instead of being seeded
//                   with a logarithm
//   MT_LEAN_INSIDE  lean_{x,y,z}_{lo,hi} bound the part of the world box whose every float32 position maps to a cell of
//                   the voxel grid (the whole box but for a few floats next to a face, which take the general code)
//   MT_LEAN_ZTABLE  (regions) the z-interval table exists (zlut_n != 0) or there is at most one region: the region lookup
//                   needs no binary search
enum { MT_LEAN_AXES = 1, MT_LEAN_INSIDE = 2, MT_LEAN_ALL = 3, MT_LEAN_ZTABLE = 4 };

// Checked build (-DMT_CHECKED, `python -m paper_2512_10520_b200.build --checked` -> libmuon_transport_checked.so): every
// index the kernels form into a global array is compared with the array's size first, and a violation is counted in
// MtParams::check instead of being dereferenced.  compute-sanitizer is not available on the GPU pool this was developed on
// (profiles/r2_sanitizers.md); this is the bounds check of our own that stands in for memcheck.  In the normal build the
// macro expands to nothing.
enum {
  MT_CHK_INPUT = 1, MT_CHK_PERM = 2, MT_CHK_RECORD = 3, MT_CHK_PARK_SLOT = 4, MT_CHK_SORT_KEY = 5, MT_CHK_TABLE = 6,
  MT_CHK_GRID = 7, MT_CHK_HASH = 8, MT_CHK_PBIN = 9, MT_CHK_MATERIAL = 10, MT_CHK_PERM_SLOT = 11, MT_CHK_OUTPUT = 12
};
#ifdef MT_CHECKED
#define MT_CHECK(P, cond, code)                                    \
  do {                                                             \
    if (!(cond)) { atomicAdd((P).check, 1u); atomicMax((P).check + 1, (unsigned)(code)); } \
  } while (0)
#define MT_CHECKED_BUILD 1
#else
#define MT_CHECK(P, cond, code) ((void)0)
#define MT_CHECKED_BUILD 0
#endif

#define MT_COUNTER_SLOTS 64

struct MtParams {
  // ---- checked build: {violations, highest MT_CHK_* code seen}, and the sizes the indices are held to
  unsigned* check;
  uint32_t n_tab_cells;          // cells of the packed alias tables
  uint64_t n_grid_cells;         // records of the padded field grid
  uint32_t n_keys;               // WAVEFRONT sort keys
  uint32_t n_hash_cells, n_hash_list;
  // ---- geometry
  int32_t mode;
  float x_min, x_max, y_min, y_max, z_min, z_exit, p_min;
  int32_t max_steps, world_material, n_regions;
  int32_t nx, ny, nz;
  float ox, oy, oz, inv_cell;
  const MtCellPair* grid;        // [nz+2][ny+2][nx+2] pairs {cell x, cell x+1} of {Bx, By, Bz, material}: the caller's grids
                                 // with a one-cell clamp-replicated border, library-owned
  uint32_t gsy, gsz;             // grid strides in cells: nx+2 and (nx+2)(ny+2)
  uint64_t gsy_bytes, gsz_bytes, gsyz_bytes;   // the same in bytes (32 per cell), and their sum
  float fnx, fny, fnz;           // (float)nx, ny, nz for the inside test
  uint32_t grid_k;               // (0x4B400000 - 1) * (gsz + gsy + 1) mod 2^32: see lookup_voxel
  uint32_t lean;                 // MT_LEAN_* facts proven on the host that let a kernel variant skip work
  float lean_x_lo, lean_x_hi, lean_y_lo, lean_y_hi, lean_z_lo;
  float lean_z_hi;               // per pass: also capped by the end of the slab
  // ---- tables
  int32_t n_materials, n_pbins, n_dp, n_th;
  float inv_p_lo, bin_scale;     // bin guess: floor(log2(P * inv_p_lo) * bin_scale), then fixed on the edges
  // Momentum-bin table (LEAN kernels): key = (bits(P) >> bin_shift) - bin_key_lo, clamped to
  // [0, bin_key_max], names a run of consecutive floats; binlut[key] is the bin (§3.4) of the run's smallest float and the
  // host has checked that no run holds more than one edge, so the bin of P is binlut[key] or the next one: ONE comparison
  // with the float32 edge decides, as §3.4 demands, and no logarithm is taken.  bin_shift = 0: no table (bins too narrow).
  int32_t bin_shift, bin_key_lo, bin_key_max;
  // z-interval table (REGIONS): §3.2 asks for the greatest j with z_lo[j] <= z.  The z range
  // [zlut_g0, zlut_g0 + zlut_n / zlut_inv] that covers the world box and every z_lo is cut into zlut_n cells; zlut[k] is
  // that j for a point just below cell k (-1 if none) and the host has checked that no cell holds more than two z_lo, so
  // two exact comparisons with the next z_lo finish the search — no 5-level binary search per step.  zlut_n = 0: no table.
  int32_t zlut_n;
  float zlut_g0, zlut_inv, zlut_max;
  const uint32_t* tab32;         // pack32: [material block][pbin][n_dp + n_th] = threshold24 << 8 | alias8; the blocks are
  const uint2* tab64;            // ordered most-used material first.  pack64: same shape, {threshold (<= 2^24), alias}
  const float* blob;             // const blob (global copy)
  MtBlobLayout bl;
  uint32_t hot_cells;            // the first hot_cells cells of the packed tables are staged in shared memory
                                 // (whole material blocks; 0 = none)
  uint32_t cells_per_bin;        // cells of one (material, momentum bin): n_dp + n_th, or n_dp * n_th in JOINT mode
  uint32_t n_joint;              // JOINT mode: n_dp * n_th cells per table, pack64 cells
  uint32_t nth_magic;            // ceil(2^32 / n_th): cell / n_th == umulhi(cell, nth_magic) for cell * n_th < 2^32
  int32_t field_mode;            // MT_FIELD_*
  int32_t exit_mode;             // MT_EXIT_* (DESIGN.md §3.13): what the compact exit list records
  // ---- POLY mode: spatial hash over the world box; a cell lists, in ascending order, the blocks whose
  //      padded bounding box meets it
  int32_t n_blocks;
  const uint2* hash_cells;       // [hnz][hny][hnx] = {first entry in hash_list, number of candidates}
  const uint16_t* hash_list;     // block indices
  int32_t hnx, hny, hnz;
  float h_inv_x, h_inv_y, h_inv_z;   // cells per metre along each axis
  float h_max_x, h_max_y, h_max_z;   // (float)(hnx - 1), ...: the last cell along each axis
  // ---- this call
  uint64_t n, id_base;           // this lane's muons: n of them, the first with id id_base (= the call's id_base + idx_base)
  uint32_t idx_base;             // index of this lane's first muon within the call (exit records carry call indices)
  uint32_t key0, key1;           // Philox key = seed lo, hi
  uint32_t rk[20];               // the ten round keys (key + r * Weyl), precomputed on the host
  const float4* in_pos_q;
  const float4* in_mom;
  float4* out_pos_flag;
  float4* out_mom_steps;
  float4* exit_rec;
  uint32_t* exit_count;
  uint32_t exit_capacity;
  unsigned long long* counters;  // optional [8]
  unsigned long long* counters_spread;  // item-mode kernels: [MT_COUNTER_SLOTS][8] library scratch summed into `counters`
  int32_t persistent;            // WAVEFRONT passes: 1 = persistent CTAs that pull 32-muon items from work_counter; 0 = one
                                 // item per warp, the CTA exits with its items (lanes interleave at CTA granularity)
  unsigned long long* work_counter;   // refill scheduler
  int32_t refill_min_idle;
  // ---- wavefront scheduler (mt_kernels.cu): one pass per z-slab.  In-flight muons live in library
  //      scratch as 48-byte records {x,y,z,q | px,py,pz,step | index,-,-,-} in the order in which a pass parked them;
  //      the next pass reads them THROUGH a permutation (perm[sorted position] = record), so sorting moves 4 bytes
  //      per muon instead of the records.  Two record buffers alternate between passes.
  const uint32_t* live_in_count; // device count of the records a pass reads
  uint32_t* live_out_count;      // device count of the records it parks (zero on entry)
  float slab_z_end;              // a pass advances each muon until z >= slab_z_end (or it terminates)
  int32_t first_pass;            // 1: the records are the caller's input arrays (step 0, index = position)
  int32_t sorted_in, sort_out;   // this pass reads its records through `perm` / parks them with sort keys for the next sort
                                 // (the live list is re-sorted every MT_OPT_SORT_EVERY-th pass; in between, a pass reads
                                 // the records in the order in which the previous one parked them)
  const float4* rec_in;          // [live][3]
  float4* rec_out;               // [parked][3]
  uint2* sort_key;               // [parked] {sort key, rank within key} of the records just parked / of the inputs
  uint32_t* perm;                // [live] record of each position of the sorted order
  uint32_t* hist;                // [n_keys] muons parked per sort key (zero on entry; the scan zeroes it again)
  uint32_t* key_offset;          // [n_keys] exclusive scan of hist
  float key_x0, key_y0, key_inv; // sort key = iy * key_nx + ix, ix = clamp((int)((x - key_x0) * key_inv), 0, key_nx-1)
  int32_t key_nx, key_ny;
  float key_look;                // the key uses the position extrapolated this far along z (metres)
};
