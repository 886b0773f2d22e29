// mt_lib.cu — host side of the C ABI in include/muon_transport.h: context, alias-table construction and
// packing, geometry upload, schedule selection and the transport launch sequences.
// No transport arithmetic runs on the host; there is no CPU fallback.
#include <cuda_runtime.h>
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "../../include/muon_transport.h"
#include "mt_launch.h"

namespace {

struct DevBuf {
  void* p = nullptr;
  size_t bytes = 0;
  cudaError_t reserve(size_t want) {
    if (want <= bytes) return cudaSuccess;
    if (p) cudaFree(p);
    p = nullptr; bytes = 0;
    cudaError_t e = cudaMalloc(&p, want);
    if (e == cudaSuccess) bytes = want;
    return e;
  }
  void release() { if (p) cudaFree(p); p = nullptr; bytes = 0; }
};

// a lane of concurrent transport work inside one call (run_transport): own stream, own scratch
struct Lane {
  cudaStream_t stream = nullptr;                 // priority descending with the lane index
  cudaStream_t stream_eq = nullptr;              // default priority: lanes that should advance side by side
  cudaEvent_t done = nullptr, ready = nullptr;   // its kernels (and copies out) are done / its inputs have landed
  DevBuf scratch, wave;
  size_t zero_bytes = 0;
};

}  // namespace

struct mt_ctx {
  int device = 0;
  int sm_count = 0;
  size_t smem_optin = 0;
  std::string last_error;
  // options
  int opt_sched = MT_SCHED_AUTO, opt_block = 0, opt_blocks_per_sm = 0, opt_slab_cells = 0, opt_min_idle = 0, opt_key_look = -1;
  // histograms (host copies)
  bool have_hist = false, have_tables = false, have_geom = false;
  int32_t n_materials = 0, n_pbins = 0, n_dp = 0, n_th = 0;
  int hist_mode = MT_HIST_MARGINAL;      // MT_HIST_JOINT: counts_dp / prob_dp / alias_dp hold n_dp * n_th cells per table
  float p_lo = 0, p_hi = 0;
  std::vector<float> counts_dp, counts_th, axis_dp, axis_th, step_m;
  // built tables (host, for mt_get_alias) and packed device copies
  std::vector<float> prob_dp, prob_th;
  std::vector<uint32_t> alias_dp, alias_th;
  int pack = 32;
  int placement = MT_PLACE_AUTO;
  size_t table_bytes = 0;
  std::vector<int> mat_order;        // material ids, most-used first: the order of their blocks in the packed tables
  std::vector<uint32_t> mat_cell0;   // [n_materials + 1] first cell of material m's block in the packed tables
  DevBuf d_tab, d_blob, d_grid, d_scratch, d_check, d_stage_in, d_stage_out, d_stage_misc, d_hash;
  int opt_hash_nxy = 0, opt_hash_nz = 0, opt_no_lean = 0;
  float lean_box[6] = {0, 0, 0, 0, 0, 0};        // x_lo, x_hi, y_lo, y_hi, z_lo, z_hi of MT_LEAN_INSIDE
  bool lean_axes = false, lean_inside = false;   // MT_LEAN_* facts (mt_params.h), proven in rebuild_blob / mt_set_geometry
  // geometry
  mt_geometry geom{};
  std::vector<mt_region> regions;
  std::vector<mt_poly_block> blocks;     // POLY mode
  int hnx = 0, hny = 0, hnz = 0;         // spatial hash
  float h_inv[3] = {0, 0, 0};
  size_t hash_list_off = 0;              // byte offset of the candidate lists inside d_hash
  uint32_t n_hash_list = 0;              // entries of the candidate lists
  int bin_shift = 0, bin_key_lo = 0, bin_key_max = 0;   // momentum-bin table (mt_params.h)
  int zlut_n = 0;                        // z-interval table (mt_params.h)
  float zlut_g0 = 0, zlut_inv = 0;
  int selftest_bad_bounds = 0;           // checked build: hand the kernels a wrong table size (MT_OPT_CHECK_SELFTEST)
  MtBlobLayout bl{};
  int64_t launches = 0;
  int last_lean = 0, last_sched = 0, last_lanes = 0;
  int opt_lanes = 0, opt_pass_mode = 0, opt_lane_prio = 0, opt_sort_every = 0;
  std::vector<Lane> lanes;
  cudaEvent_t ev_fork = nullptr;
  cudaStream_t copy_in = nullptr;
};

namespace {

struct DeviceGuard {
  int prev = -1;
  explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
  ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int fail(mt_ctx* c, int code, const char* fmt, ...) {
  if (c) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    c->last_error = buf;
  }
  return code;
}

#define MT_CUDA(c, expr)                                                                             \
  do {                                                                                               \
    cudaError_t e_ = (expr);                                                                         \
    if (e_ != cudaSuccess)                                                                           \
      return fail((c), e_ == cudaErrorMemoryAllocation ? MT_ERR_NOMEM : MT_ERR_CUDA, "%s: %s", #expr, \
                  cudaGetErrorString(e_));                                                           \
  } while (0)

// Walker/Vose construction with a pinned pairing order.  Returns false on an empty or
// invalid histogram.
bool build_one_alias(const float* counts, int N, float* prob, uint32_t* alias) {
  double total = 0.0;
  for (int j = 0; j < N; ++j) {
    const float v = counts[j];
    if (!(v >= 0.0f) || isinf(v)) return false;
    total += (double)v;
  }
  if (!(total > 0.0)) return false;
  std::vector<double> scaled(N);
  std::vector<int> below, above;           // stacks of cells with scaled mass < 1 and >= 1
  below.reserve(N); above.reserve(N);
  for (int j = 0; j < N; ++j) {
    scaled[j] = ((double)counts[j] * (double)N) / total;
    (scaled[j] < 1.0 ? below : above).push_back(j);
  }
  while (!below.empty() && !above.empty()) {
    const int s = below.back(), l = above.back();
    below.pop_back(); above.pop_back();
    prob[s] = (float)scaled[s];
    alias[s] = (uint32_t)l;
    scaled[l] = (scaled[l] + scaled[s]) - 1.0;
    (scaled[l] < 1.0 ? below : above).push_back(l);
  }
  for (int j : above) { prob[j] = 1.0f; alias[j] = (uint32_t)j; }
  for (int j : below) { prob[j] = 1.0f; alias[j] = (uint32_t)j; }
  return true;
}

// integer acceptance threshold: a24 < T  <=>  (float)a24 * 2^-24 < prob
uint32_t threshold24(float prob) {
  const double t = ceil((double)prob * 16777216.0);
  return t <= 0.0 ? 0u : (t >= 16777216.0 ? 16777216u : (uint32_t)t);
}

size_t blob_bytes(const mt_ctx* c) { return (size_t)MT_STAGED_WORDS(c->bl) * sizeof(float); }   // shared memory a CTA stages

int rebuild_blob(mt_ctx* c) {
  // [edges][steps x4][axes x4][z_lo][regions]; see mt_params.h
  const int n_edges = c->n_pbins + 1;
  const int n_reg = c->have_geom ? (int)c->regions.size() : 0;
  const int nt = c->n_materials * c->n_pbins;
  MtBlobLayout bl;
  bl.off_edges_open = (n_edges + 3) & ~3;
  bl.off_steps = (bl.off_edges_open + n_edges + 3) & ~3;
  bl.off_axes = bl.off_steps + 4 * (c->n_materials + 1);
  bl.off_zlo = bl.off_axes + 4 * nt;
  bl.off_regions = (bl.off_zlo + n_reg + 2 + 3) & ~3;         // two +inf entries follow the z_lo array
  const int n_blk = c->have_geom ? (int)c->blocks.size() : 0;
  bl.off_blocks = (bl.off_regions + 12 * n_reg + 3) & ~3;
  bl.off_binlut = bl.off_blocks + 24 * n_blk;
  const double lo = (double)c->p_lo, hi = (double)c->p_hi;
  std::vector<float> edges(n_edges);
  for (int j = 0; j <= c->n_pbins; ++j)
    edges[j] = (float)(lo * pow(hi / lo, (double)j / (double)c->n_pbins));                // §3.4
  // Momentum-bin table (mt_params.h: bin_shift).  A key names the 2^shift consecutive floats that share their top bits;
  // the coarsest keys under which no run of floats holds more than one edge are taken, so that one comparison with the
  // edge above the tabulated bin settles §3.4's decision.  Runs are looked at over [p_lo, p_hi] (keys are clamped there).
  auto bits_of = [](float v) { uint32_t u; memcpy(&u, &v, 4); return u; };
  auto float_of = [](uint32_t u) { float v; memcpy(&v, &u, 4); return v; };
  auto bin_of = [&](float Pv) {                              // greatest j in [0, n-1] with edges[j] <= P, 0 if none
    int b = (int)(std::upper_bound(edges.begin(), edges.end() - 1, Pv) - edges.begin()) - 1;
    return std::max(b, 0);
  };
  std::vector<uint16_t> binlut;
  c->bin_shift = 0; c->bin_key_lo = 0; c->bin_key_max = 0;
  for (int m = 3; m <= 12 && c->n_pbins <= 65535; ++m) {
    const int shift = 23 - m;
    const uint32_t k_lo = bits_of(c->p_lo) >> shift, k_hi = bits_of(c->p_hi) >> shift;
    if (k_hi - k_lo + 1 > 16384) break;
    std::vector<uint16_t> lut(k_hi - k_lo + 1);
    bool ok = true;
    for (uint32_t k = k_lo; k <= k_hi && ok; ++k) {
      const int b_first = bin_of(float_of(k << shift)), b_last = bin_of(float_of(((k + 1) << shift) - 1));
      ok = (b_last - b_first) <= 1;
      lut[k - k_lo] = (uint16_t)b_first;
    }
    if (ok) { binlut.swap(lut); c->bin_shift = shift; c->bin_key_lo = (int)k_lo; c->bin_key_max = (int)(k_hi - k_lo); break; }
  }
  bl.off_zlut = bl.off_binlut + (int)((binlut.size() + 1) / 2);
  // z-interval table (mt_params.h: zlut_n): cells fine enough that at most two z_lo fall into one, bounds taken with a
  // margin of 1 % of a cell, which dwarfs the float32 rounding of the device's cell index (below 2^-11 of a cell here)
  std::vector<int16_t> zlut;
  c->zlut_n = 0; c->zlut_g0 = 0.0f; c->zlut_inv = 0.0f;
  // (one region needs neither: a single comparison; the lean kernels take no geometry that would need the search)
  if (n_reg >= 2 && c->geom.mode == MT_GEOM_REGIONS) {
    const double g0 = std::min((double)c->geom.z_min, (double)c->regions[0].z_lo);
    const double g1 = std::max((double)c->geom.z_exit, (double)c->regions[n_reg - 1].z_lo);
    for (int nzc = 1024; nzc <= 4096 && std::isfinite(g0) && std::isfinite(g1) && g1 > g0 && zlut.empty(); nzc *= 2) {
      const float inv = (float)((double)nzc / (g1 - g0));
      const double cell = 1.0 / (double)inv;
      std::vector<int16_t> lut(nzc);
      bool ok = true;
      int j = -1;                                            // greatest j with z_lo[j] <= lower bound of the cell
      for (int k = 0; k < nzc && ok; ++k) {
        const double zb = (double)(float)g0 + ((double)k - 0.01) * cell, zu = (double)(float)g0 + ((double)k + 1.01) * cell;
        while (j + 1 < n_reg && (double)c->regions[j + 1].z_lo <= zb) ++j;
        int inside = 0;
        for (int q = j + 1; q < n_reg && (double)c->regions[q].z_lo <= zu; ++q) ++inside;
        if (k == nzc - 1) inside = n_reg - 1 - j;            // the last cell also serves every z beyond the table
        ok = inside <= 2;
        lut[k] = (int16_t)j;
      }
      if (ok) { zlut.swap(lut); c->zlut_n = nzc; c->zlut_g0 = (float)g0; c->zlut_inv = inv; }
    }
  }
  bl.n_words = bl.off_zlut + (int)((zlut.size() + 1) / 2);
  std::vector<float> blob((size_t)bl.n_words + 4, 0.0f);
  if (!zlut.empty()) memcpy(&blob[bl.off_zlut], zlut.data(), zlut.size() * sizeof(int16_t));
  for (int j = 0; j <= c->n_pbins; ++j) blob[j] = edges[j];
  if (!binlut.empty()) memcpy(&blob[bl.off_binlut], binlut.data(), binlut.size() * sizeof(uint16_t));
  for (int j = 0; j <= c->n_pbins; ++j)
    blob[bl.off_edges_open + j] = (j == 0) ? -INFINITY : (j == c->n_pbins) ? INFINITY : blob[j];
  for (int m = 0; m <= c->n_materials; ++m) {
    const float h = c->step_m[m];
    blob[bl.off_steps + 4 * m + 0] = h;
    blob[bl.off_steps + 4 * m + 1] = h * 0.5f;
    blob[bl.off_steps + 4 * m + 2] = (float)((double)h / 6.0);                           // §3.2
    const int32_t cell0 = (int32_t)c->mat_cell0[m];
    memcpy(&blob[bl.off_steps + 4 * m + 3], &cell0, sizeof cell0);
  }
  const bool joint_axes = (c->hist_mode == MT_HIST_JOINT);   // axis b is then the transverse fraction ft: proven <= 1
  bool axes_ok = true;
  for (int t = 0; t < nt; ++t) {
    // cell widths carry the jitter's 2^-16 (exact: a power of two; mt_step.cuh decode)
    float* ax = &blob[bl.off_axes + 4 * t];
    ax[0] = c->axis_dp[2 * t]; ax[1] = c->axis_dp[2 * t + 1] * 0x1p-16f;
    ax[2] = c->axis_th[2 * t]; ax[3] = c->axis_th[2 * t + 1] * 0x1p-16f;
    // MT_LEAN_AXES: y = fma(v, d, lo) is monotone in v for d >= 0 and v runs over [0, n * 2^16), so the ends bound it.
    // exp2c's polynomial is within 1e-6 relative of 2^y: 2^-0.0034 = 0.99765 < 0.999 and 2^-0.36 = 0.7792 < pi/4 = 0.7854
    // (theta * 2/pi < 0.4961 rounds to quadrant 0).
    const float v_dp = (float)((uint32_t)c->n_dp * 65536u - 1u), v_th = (float)((uint32_t)c->n_th * 65536u - 1u);
    const float hi_dp = fmaf(v_dp, ax[1], ax[0]), hi_th = fmaf(v_th, ax[3], ax[2]);
    axes_ok = axes_ok && ax[1] >= 0.0f && ax[3] >= 0.0f && ax[0] >= -120.0f && ax[2] >= -120.0f &&
              hi_dp <= -0.0034f && hi_th <= (joint_axes ? 0.0f : -0.36f);
  }
  c->lean_axes = axes_ok && c->bin_shift != 0;               // the lean kernels read the bin from the table
  blob[bl.off_zlo + n_reg] = blob[bl.off_zlo + n_reg + 1] = INFINITY;
  for (int j = 0; j < n_reg; ++j) {
    blob[bl.off_zlo + j] = c->regions[j].z_lo;
    static_assert(sizeof(mt_region) == 40 && sizeof(MtRegionDev) == 48, "region layout");
    memcpy(&blob[bl.off_regions + 12 * j], &c->regions[j], sizeof(mt_region));      // same field order; two pad words follow
  }
  for (int j = 0; j < n_blk; ++j) {
    // §3.12: the per-block constants of the slice interpolation, each ONE float32 operation
    static_assert(sizeof(MtBlockDev) == 96, "block layout");
    const mt_poly_block& b = c->blocks[j];
    MtBlockDev d;
    d.z_lo = b.z_lo; d.z_hi = b.z_hi;
    const volatile float dz = b.z_hi - b.z_lo;
    d.inv_dz = 1.0f / dz;
    d.material = b.material; d.bx = b.bx; d.by = b.by; d.bz = b.bz; d.pad = 0.0f;
    for (int i = 0; i < 4; ++i) {
      d.xl[i] = b.xy_lo[i][0]; d.yl[i] = b.xy_lo[i][1];
      const volatile float dx = b.xy_hi[i][0] - b.xy_lo[i][0], dy = b.xy_hi[i][1] - b.xy_lo[i][1];
      d.dx[i] = dx; d.dy[i] = dy;
    }
    memcpy(&blob[bl.off_blocks + 24 * j], &d, sizeof d);
  }
  c->bl = bl;
  MT_CUDA(c, c->d_blob.reserve(blob.size() * sizeof(float)));
  MT_CUDA(c, cudaMemcpy(c->d_blob.p, blob.data(), blob.size() * sizeof(float), cudaMemcpyHostToDevice));
  return MT_OK;
}

// Pack the host tables (per (material, pbin): the Dp/p cells followed by the theta cells) with the material
// blocks in the order c->mat_order, upload them, and record where each block starts.
int upload_tables(mt_ctx* c) {
  const bool joint = (c->hist_mode == MT_HIST_JOINT);
  const int n_dp = joint ? c->n_dp * c->n_th : c->n_dp, n_th = joint ? 0 : c->n_th, n_cells = n_dp + n_th;
  const size_t nt = (size_t)c->n_materials * c->n_pbins;
  const int wpc = (c->pack == 32) ? 1 : 2;                 // 32-bit words per cell
  std::vector<uint32_t> packed(nt * n_cells * wpc + 8, 0u);
  c->mat_cell0.assign(c->n_materials + 1, 0u);
  size_t block = 0;
  for (int m : c->mat_order) {
    c->mat_cell0[m] = (uint32_t)(block * c->n_pbins * n_cells);
    for (int i = 0; i < c->n_pbins; ++i) {
      const size_t t = (size_t)(m - 1) * c->n_pbins + i;                        // table in caller order
      const size_t dst = (block * c->n_pbins + i) * n_cells;                    // first cell in packed order
      for (int k = 0; k < n_cells; ++k) {
        const bool is_dp = k < n_dp;
        const float pr = is_dp ? c->prob_dp[t * n_dp + k] : c->prob_th[t * n_th + (k - n_dp)];
        uint32_t al = is_dp ? c->alias_dp[t * n_dp + k] : c->alias_th[t * n_th + (k - n_dp)];
        uint32_t T = threshold24(pr);
        const uint32_t self = (uint32_t)(is_dp ? k : k - n_dp);
        if (c->pack == 32) {
          if (T >= 16777216u) { T = 16777215u; al = self; }     // prob == 1: the alias is never taken
          packed[dst + k] = (T << 8) | al;
        } else {
          packed[2 * (dst + k)] = T;
          packed[2 * (dst + k) + 1] = al;
        }
      }
    }
    ++block;
  }
  c->table_bytes = nt * n_cells * wpc * sizeof(uint32_t);
  MT_CUDA(c, c->d_tab.reserve(packed.size() * sizeof(uint32_t)));               // padded: staged in 16-byte units
  MT_CUDA(c, cudaMemcpy(c->d_tab.p, packed.data(), packed.size() * sizeof(uint32_t), cudaMemcpyHostToDevice));
  return MT_OK;
}

// order the material blocks by weight (cells or volume per material), heaviest first
void order_materials(mt_ctx* c, const std::vector<double>& weight) {
  c->mat_order.resize(c->n_materials);
  for (int m = 1; m <= c->n_materials; ++m) c->mat_order[m - 1] = m;
  std::stable_sort(c->mat_order.begin(), c->mat_order.end(), [&](int a, int b) { return weight[a] > weight[b]; });
}

// POLY mode: validate the blocks and bin their padded bounding boxes into a uniform grid over the
// world box — the spatial hash of PAPER.md L120.  The hash only prunes: a point's cell (computed on the device in
// float32, clamped into the grid) must list every block that the float32 containment test could accept for that
// point, so each box is grown by a pad that dwarfs float32 rounding (1e-4 of the largest coordinate + 0.1 mm, against
// 2^-22 relative) and cell ranges are taken with the device's own float32 scale factors.
int build_hash(mt_ctx* c, const mt_geometry* gm, const std::vector<mt_poly_block>& blks, std::vector<double>& weight) {
  const int hnx = c->opt_hash_nxy ? c->opt_hash_nxy : 16, hny = hnx, hnz = c->opt_hash_nz ? c->opt_hash_nz : 256;
  const double w_lo[3] = {gm->x_min, gm->y_min, gm->z_min};
  const double w_ext[3] = {(double)gm->x_max - gm->x_min, (double)gm->y_max - gm->y_min, (double)gm->z_exit - gm->z_min};
  const int hn[3] = {hnx, hny, hnz};
  if ((uint64_t)hnx * hny * hnz > ((uint64_t)1 << 24))
    return fail(c, MT_ERR_UNSUPPORTED, "spatial hash of %d x %d x %d cells: at most 2^24 cells", hnx, hny, hnz);
  float inv[3];
  for (int a = 0; a < 3; ++a) inv[a] = (float)((double)hn[a] / w_ext[a]);
  double world = w_ext[0] * w_ext[1] * w_ext[2];
  auto area2 = [](const double q[4][2]) {                   // twice the signed area (shoelace)
    double s = 0.0;
    for (int i = 0; i < 4; ++i) { const int j = (i + 1) & 3; s += q[i][0] * q[j][1] - q[j][0] * q[i][1]; }
    return s;
  };
  std::vector<int> range(blks.size() * 6);
  std::vector<uint32_t> count((size_t)hnx * hny * hnz + 1, 0u);
  for (size_t j = 0; j < blks.size(); ++j) {
    const mt_poly_block& b = blks[j];
    if (!(b.z_lo < b.z_hi) || !std::isfinite(b.z_lo) || !std::isfinite(b.z_hi)) return fail(c, MT_ERR_INVALID_ARG, "block %zu: empty z range", j);
    if (b.material < 0 || b.material > c->n_materials) return fail(c, MT_ERR_INVALID_ARG, "block %zu: bad material", j);
    double lo[3] = {INFINITY, INFINITY, b.z_lo}, hi[3] = {-INFINITY, -INFINITY, b.z_hi}, big = std::max(fabs(b.z_lo), fabs(b.z_hi));
    double face[3][4][2];                                   // lower, upper, middle
    int orient = 0;
    for (int f = 0; f < 2; ++f) {
      const float (*v)[2] = f ? b.xy_hi : b.xy_lo;
      for (int i = 0; i < 4; ++i) {
        if (!std::isfinite(v[i][0]) || !std::isfinite(v[i][1])) return fail(c, MT_ERR_INVALID_ARG, "block %zu: non-finite vertex", j);
        face[f][i][0] = v[i][0]; face[f][i][1] = v[i][1];
        lo[0] = std::min(lo[0], (double)v[i][0]); hi[0] = std::max(hi[0], (double)v[i][0]);
        lo[1] = std::min(lo[1], (double)v[i][1]); hi[1] = std::max(hi[1], (double)v[i][1]);
      }
      // convex: the turns at the four corners have one sign; both faces go round the same way
      int pos = 0, neg = 0;
      for (int i = 0; i < 4; ++i) {
        const int i1 = (i + 1) & 3, i2 = (i + 2) & 3;
        const double ax = face[f][i1][0] - face[f][i][0], ay = face[f][i1][1] - face[f][i][1];
        const double bx = face[f][i2][0] - face[f][i1][0], by = face[f][i2][1] - face[f][i1][1];
        const double cr = ax * by - ay * bx;
        pos += cr > 0; neg += cr < 0;
      }
      if (pos && neg) return fail(c, MT_ERR_INVALID_ARG, "block %zu: %s face is not convex", j, f ? "upper" : "lower");
      const int o = pos ? 1 : (neg ? -1 : 0);
      if (o && orient && o != orient) return fail(c, MT_ERR_INVALID_ARG, "block %zu: faces listed in opposite orientations", j);
      if (o) orient = o;
    }
    for (int a = 0; a < 2; ++a) big = std::max(big, std::max(fabs(lo[a]), fabs(hi[a])));
    for (int a = 0; a < 3; ++a) big = std::max(big, std::max(fabs(w_lo[a]), fabs(w_lo[a] + w_ext[a])));
    const double pad = 1e-4 * big + 1e-4;
    for (int a = 0; a < 3; ++a) {
      const double c_lo = floor((lo[a] - pad - w_lo[a]) * (double)inv[a]), c_hi = floor((hi[a] + pad - w_lo[a]) * (double)inv[a]);
      range[6 * j + 2 * a] = (int)std::min(std::max(c_lo, 0.0), (double)(hn[a] - 1));
      range[6 * j + 2 * a + 1] = (int)std::min(std::max(c_hi, 0.0), (double)(hn[a] - 1));
    }
    for (int z = range[6 * j + 4]; z <= range[6 * j + 5]; ++z)
      for (int y = range[6 * j + 2]; y <= range[6 * j + 3]; ++y)
        for (int x = range[6 * j]; x <= range[6 * j + 1]; ++x) count[((size_t)z * hny + y) * hnx + x] += 1;
    // volume (Simpson over z is exact for linearly moving vertices), for the table order only
    for (int i = 0; i < 4; ++i) for (int k = 0; k < 2; ++k) face[2][i][k] = 0.5 * (face[0][i][k] + face[1][i][k]);
    const double vol = ((double)b.z_hi - b.z_lo) / 12.0 * (fabs(area2(face[0])) + 4.0 * fabs(area2(face[2])) + fabs(area2(face[1])));
    weight[b.material] += vol;
    world -= vol;
  }
  weight[gm->world_material] += std::max(world, 0.0);
  const size_t n_cells = (size_t)hnx * hny * hnz;
  uint64_t n_list64 = 0;                                     // 2^24 cells x 1024 blocks does not fit 32 bits
  for (size_t k = 0; k < n_cells; ++k) n_list64 += count[k];
  if (n_list64 >= ((uint64_t)1 << 28))
    return fail(c, MT_ERR_UNSUPPORTED, "spatial hash candidate lists hold %llu entries (limit 2^28): use a coarser hash",
                (unsigned long long)n_list64);
  std::vector<uint32_t> first(n_cells + 1, 0u);
  for (size_t k = 0; k < n_cells; ++k) first[k + 1] = first[k] + count[k];
  const size_t n_list = first[n_cells];
  std::vector<uint16_t> list(n_list + 8, 0);
  std::vector<uint32_t> fill(first.begin(), first.end() - 1);
  for (size_t j = 0; j < blks.size(); ++j)                   // ascending j: every list ends up in index order
    for (int z = range[6 * j + 4]; z <= range[6 * j + 5]; ++z)
      for (int y = range[6 * j + 2]; y <= range[6 * j + 3]; ++y)
        for (int x = range[6 * j]; x <= range[6 * j + 1]; ++x) list[fill[((size_t)z * hny + y) * hnx + x]++] = (uint16_t)j;
  std::vector<uint2> cells(n_cells);
  for (size_t k = 0; k < n_cells; ++k) cells[k] = make_uint2(first[k], count[k]);
  const size_t list_off = (n_cells * sizeof(uint2) + 255) & ~(size_t)255;
  MT_CUDA(c, c->d_hash.reserve(list_off + list.size() * sizeof(uint16_t)));
  MT_CUDA(c, cudaMemcpy(c->d_hash.p, cells.data(), n_cells * sizeof(uint2), cudaMemcpyHostToDevice));
  MT_CUDA(c, cudaMemcpy((char*)c->d_hash.p + list_off, list.data(), list.size() * sizeof(uint16_t), cudaMemcpyHostToDevice));
  c->hnx = hnx; c->hny = hny; c->hnz = hnz;
  c->h_inv[0] = inv[0]; c->h_inv[1] = inv[1]; c->h_inv[2] = inv[2];
  c->hash_list_off = list_off;
  c->n_hash_list = (uint32_t)n_list;
  return MT_OK;
}

// the header promises that nothing throws across the C boundary: host allocations of the setup calls (std::vector,
// std::string) are the only throwing code in this file
template <class F> int guarded(mt_ctx* c, F&& body) {
  try {
    return body();
  } catch (const std::bad_alloc&) {
    if (c) { try { c->last_error = "host allocation failed"; } catch (...) {} }
    return MT_ERR_NOMEM;
  } catch (...) {
    return MT_ERR_INVALID_ARG;
  }
}

}  // namespace

extern "C" {

const char* mt_strerror(int code) {
  switch (code) {
    case MT_OK: return "ok";
    case MT_ERR_INVALID_ARG: return "invalid argument";
    case MT_ERR_STATE: return "call order violated";
    case MT_ERR_EMPTY_HIST: return "empty or invalid histogram";
    case MT_ERR_UNSUPPORTED: return "unsupported size or mode";
    case MT_ERR_CUDA: return "CUDA error";
    case MT_ERR_NOMEM: return "out of memory";
    default: return "unknown error";
  }
}

const char* mt_last_error(const mt_ctx* ctx) { return ctx ? ctx->last_error.c_str() : "null context"; }

int mt_create(mt_ctx** out, int cuda_device) {
  if (!out) return MT_ERR_INVALID_ARG;
  *out = nullptr;
  int n_dev = 0;
  if (cudaGetDeviceCount(&n_dev) != cudaSuccess || cuda_device < 0 || cuda_device >= n_dev) {
    cudaGetLastError();
    return MT_ERR_CUDA;
  }
  mt_ctx* c = new (std::nothrow) mt_ctx;
  if (!c) return MT_ERR_NOMEM;
  c->device = cuda_device;
  DeviceGuard g(cuda_device);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) { delete c; return MT_ERR_CUDA; }
  c->sm_count = prop.multiProcessorCount;
  c->smem_optin = prop.sharedMemPerBlockOptin;
  if (MT_CHECKED_BUILD) {                // {violations, highest code}: see MT_CHECK in mt_params.h
    if (c->d_check.reserve(256) != cudaSuccess || cudaMemset(c->d_check.p, 0, 256) != cudaSuccess) { delete c; return MT_ERR_CUDA; }
  }
  *out = c;
  return MT_OK;
}

int mt_destroy(mt_ctx* c) {
  if (!c) return MT_OK;
  DeviceGuard g(c->device);
  DevBuf* bufs[] = {&c->d_tab, &c->d_blob, &c->d_grid, &c->d_scratch, &c->d_check,
                    &c->d_stage_in, &c->d_stage_out, &c->d_stage_misc, &c->d_hash};
  for (DevBuf* b : bufs) b->release();
  for (Lane& L : c->lanes) {
    if (L.stream) { cudaStreamSynchronize(L.stream); cudaStreamDestroy(L.stream); }
    if (L.stream_eq) { cudaStreamSynchronize(L.stream_eq); cudaStreamDestroy(L.stream_eq); }
    if (L.done) cudaEventDestroy(L.done);
    if (L.ready) cudaEventDestroy(L.ready);
    L.scratch.release(); L.wave.release();
  }
  if (c->copy_in) { cudaStreamSynchronize(c->copy_in); cudaStreamDestroy(c->copy_in); }
  if (c->ev_fork) cudaEventDestroy(c->ev_fork);
  delete c;
  return MT_OK;
}

int mt_set_option(mt_ctx* c, int option, int64_t value) {
  if (!c) return MT_ERR_INVALID_ARG;
  switch (option) {
    case MT_OPT_SCHEDULE:
      if (value < MT_SCHED_AUTO || value > MT_SCHED_WAVEFRONT) return fail(c, MT_ERR_INVALID_ARG, "bad schedule %lld", (long long)value);
      c->opt_sched = (int)value; return MT_OK;
    case MT_OPT_BLOCK_THREADS:
      if (value != 0 && (value < 32 || value > MT_MAX_THREADS || value % 32))
        return fail(c, MT_ERR_INVALID_ARG, "block threads must be a multiple of 32 in [32, %d]", MT_MAX_THREADS);
      c->opt_block = (int)value; return MT_OK;
    case MT_OPT_BLOCKS_PER_SM:
      if (value < 0 || value > 32) return fail(c, MT_ERR_INVALID_ARG, "bad blocks per SM");
      c->opt_blocks_per_sm = (int)value; return MT_OK;
    case MT_OPT_SLAB_CELLS:
      if (value < 0 || value > 1000000) return fail(c, MT_ERR_INVALID_ARG, "bad slab thickness");
      c->opt_slab_cells = (int)value; return MT_OK;
    case MT_OPT_KEY_LOOKAHEAD:
      if (value < -1 || value > 400) return fail(c, MT_ERR_INVALID_ARG, "bad key lookahead");
      c->opt_key_look = (int)value; return MT_OK;
    case MT_OPT_REFILL_MIN_IDLE:
      if (value < 0 || value > 32) return fail(c, MT_ERR_INVALID_ARG, "bad refill threshold");
      c->opt_min_idle = (int)value; return MT_OK;
    case MT_OPT_NO_LEAN:
      c->opt_no_lean = value != 0; return MT_OK;
    case MT_OPT_CHECK_SELFTEST:
      if (!MT_CHECKED_BUILD) return fail(c, MT_ERR_UNSUPPORTED, "not a checked build");
      c->selftest_bad_bounds = value != 0; return MT_OK;
    case MT_OPT_PASS_MODE:
      if (value < 0 || value > 2) return fail(c, MT_ERR_INVALID_ARG, "bad pass mode");
      c->opt_pass_mode = (int)value; return MT_OK;
    case MT_OPT_LANE_PRIORITY:
      if (value < 0 || value > 2) return fail(c, MT_ERR_INVALID_ARG, "bad lane priority mode");
      c->opt_lane_prio = (int)value; return MT_OK;
    case MT_OPT_SORT_EVERY:
      if (value < 0 || value > 64) return fail(c, MT_ERR_INVALID_ARG, "bad sort interval");
      c->opt_sort_every = (int)value; return MT_OK;
    case MT_OPT_LANES:
      if (value < 0 || value > 16) return fail(c, MT_ERR_INVALID_ARG, "bad lane count");
      c->opt_lanes = (int)value; return MT_OK;
    case MT_OPT_HASH_NXY:
      if (value < 0 || value > 256) return fail(c, MT_ERR_INVALID_ARG, "bad hash resolution");
      c->opt_hash_nxy = (int)value; return MT_OK;
    case MT_OPT_HASH_NZ:
      if (value < 0 || value > 4096) return fail(c, MT_ERR_INVALID_ARG, "bad hash resolution");
      c->opt_hash_nz = (int)value; return MT_OK;
    default: return fail(c, MT_ERR_INVALID_ARG, "unknown option %d", option);
  }
}

static int load_histograms_impl(mt_ctx* c, const mt_hist_desc* d) {
  if (!c || !d) return MT_ERR_INVALID_ARG;
  if (d->hist_mode != MT_HIST_MARGINAL && d->hist_mode != MT_HIST_JOINT) return fail(c, MT_ERR_INVALID_ARG, "bad hist_mode");
  const bool joint = (d->hist_mode == MT_HIST_JOINT);
  if (!d->counts_dp || (!joint && !d->counts_th) || !d->axis_dp || !d->axis_th || !d->step_m)
    return fail(c, MT_ERR_INVALID_ARG, "null histogram array");
  if (d->n_materials < 1 || d->n_materials > 255 || d->n_pbins < 1 || d->n_pbins > 4096 || d->n_dp < 1 ||
      d->n_dp > 65536 || d->n_th < 1 || d->n_th > 65536)
    return fail(c, MT_ERR_UNSUPPORTED, "histogram shape out of range");
  const uint64_t cells_per_table = joint ? (uint64_t)d->n_dp * d->n_th : (uint64_t)d->n_dp + d->n_th;
  if ((uint64_t)d->n_materials * d->n_pbins * cells_per_table >= ((uint64_t)1 << 31))
    return fail(c, MT_ERR_UNSUPPORTED, "more than 2^31 table cells");
  // JOINT: 24-bit cell indices, and the kernel's exact cell / n_th by a 32-bit reciprocal needs cell * n_th < 2^32
  if (joint && (cells_per_table > ((uint64_t)1 << 24) || cells_per_table * (uint64_t)d->n_th >= ((uint64_t)1 << 32)))
    return fail(c, MT_ERR_UNSUPPORTED, "joint tables need n_dp * n_th <= 2^24 and n_dp * n_th^2 < 2^32");
  if ((uint64_t)d->n_materials * d->n_pbins > 4096)        // edges and axes live in shared memory (<= 80 KB)
    return fail(c, MT_ERR_UNSUPPORTED, "more than 4096 (material, momentum bin) tables");
  if (!(d->p_lo > 0.0f) || !(d->p_hi > d->p_lo) || isinf(d->p_hi))
    return fail(c, MT_ERR_INVALID_ARG, "need 0 < p_lo < p_hi");
  // the momentum-bin guess of the kernel (a logarithm, then one comparison against the float32 edges) needs bins
  // wider than 2^-16 in log2(p); the jitter scale 2^-16 is folded into the axis steps, which must stay normal
  if ((double)d->n_pbins / log2((double)d->p_hi / (double)d->p_lo) > 65536.0)
    return fail(c, MT_ERR_UNSUPPORTED, "momentum bins narrower than 2^-16 in log2(p)");
  for (size_t t = 0; t < (size_t)d->n_materials * d->n_pbins; ++t)
    for (const float* ax : {d->axis_dp, d->axis_th}) {
      const float w = ax[2 * t + 1];
      if (!isfinite(ax[2 * t]) || !isfinite(w) || (w != 0.0f && fabsf(w) < 0x1p-100f))
        return fail(c, MT_ERR_INVALID_ARG, "axis of table %zu is not finite or its cell width is below 2^-100", t);
    }
  for (int m = 0; m <= d->n_materials; ++m)
    if (!(d->step_m[m] > 0.0f) || isinf(d->step_m[m])) return fail(c, MT_ERR_INVALID_ARG, "step_m[%d] must be positive", m);
  const size_t nt = (size_t)d->n_materials * d->n_pbins;
  c->n_materials = d->n_materials; c->n_pbins = d->n_pbins; c->n_dp = d->n_dp; c->n_th = d->n_th;
  c->p_lo = d->p_lo; c->p_hi = d->p_hi;
  c->hist_mode = d->hist_mode;
  c->counts_dp.assign(d->counts_dp, d->counts_dp + nt * (joint ? cells_per_table : (uint64_t)d->n_dp));
  if (joint) c->counts_th.clear();
  else c->counts_th.assign(d->counts_th, d->counts_th + nt * d->n_th);
  c->axis_dp.assign(d->axis_dp, d->axis_dp + nt * 2);
  c->axis_th.assign(d->axis_th, d->axis_th + nt * 2);
  c->step_m.assign(d->step_m, d->step_m + d->n_materials + 1);
  c->have_hist = true;
  c->have_tables = false;        // the tables AND the geometry (its material ids, table offsets and shared-memory blob
  c->have_geom = false;          // follow the histogram shape) must be set again: anything else is MT_ERR_STATE
  return MT_OK;
}

static int build_alias_impl(mt_ctx* c, int placement) {
  if (!c) return MT_ERR_INVALID_ARG;
  if (!c->have_hist) return fail(c, MT_ERR_STATE, "mt_build_alias before mt_load_histograms");
  if (placement < MT_PLACE_AUTO || placement > MT_PLACE_L2) return fail(c, MT_ERR_INVALID_ARG, "bad placement");
  DeviceGuard g(c->device);
  const size_t nt = (size_t)c->n_materials * c->n_pbins;
  const bool joint = (c->hist_mode == MT_HIST_JOINT);
  const int n_dp = joint ? c->n_dp * c->n_th : c->n_dp, n_th = joint ? 0 : c->n_th;   // JOINT: one table of n_dp * n_th cells
  // From here on the host copies, the packed device tables and the blob are rewritten one after the other: until all three
  // are done the context has NO tables (a failure on the way must not leave mt_transport running new sizes over old data)
  c->have_tables = false;
  c->prob_dp.assign(nt * n_dp, 0.0f); c->alias_dp.assign(nt * n_dp, 0u);
  c->prob_th.assign(nt * n_th, 0.0f); c->alias_th.assign(nt * n_th, 0u);
  for (size_t t = 0; t < nt; ++t) {
    if (!build_one_alias(&c->counts_dp[t * n_dp], n_dp, &c->prob_dp[t * n_dp], &c->alias_dp[t * n_dp]))
      return fail(c, MT_ERR_EMPTY_HIST, "%s histogram of material %d, momentum bin %d is empty or invalid",
                  joint ? "joint" : "Dp/p", (int)(t / c->n_pbins) + 1, (int)(t % c->n_pbins));
    if (!joint && !build_one_alias(&c->counts_th[t * n_th], n_th, &c->prob_th[t * n_th], &c->alias_th[t * n_th]))
      return fail(c, MT_ERR_EMPTY_HIST, "theta histogram of material %d, momentum bin %d is empty or invalid",
                  (int)(t / c->n_pbins) + 1, (int)(t % c->n_pbins));
  }
  c->pack = (!joint && std::max(n_dp, n_th) <= 256) ? 32 : 64;
  order_materials(c, std::vector<double>(c->n_materials + 1, 0.0));       // caller order until a geometry says otherwise
  int rc = upload_tables(c);
  if (rc != MT_OK) return rc;
  c->placement = placement;
  rc = rebuild_blob(c);
  c->have_tables = (rc == MT_OK);
  return rc;
}

int mt_get_alias(const mt_ctx* c, float* prob_dp, uint32_t* alias_dp, float* prob_th, uint32_t* alias_th) {
  if (!c || !prob_dp || !alias_dp) return MT_ERR_INVALID_ARG;
  if (!c->have_tables) return MT_ERR_STATE;
  const bool joint = (c->hist_mode == MT_HIST_JOINT);
  if (!joint && (!prob_th || !alias_th)) return MT_ERR_INVALID_ARG;
  memcpy(prob_dp, c->prob_dp.data(), c->prob_dp.size() * sizeof(float));
  memcpy(alias_dp, c->alias_dp.data(), c->alias_dp.size() * sizeof(uint32_t));
  if (!joint) {
    memcpy(prob_th, c->prob_th.data(), c->prob_th.size() * sizeof(float));
    memcpy(alias_th, c->alias_th.data(), c->alias_th.size() * sizeof(uint32_t));
  }
  return MT_OK;
}

static int set_geometry_impl(mt_ctx* c, const mt_geometry* gm) {
  if (!c || !gm) return MT_ERR_INVALID_ARG;
  if (!c->have_tables) return fail(c, MT_ERR_STATE, "mt_set_geometry before mt_build_alias");
  if (gm->mode != MT_GEOM_REGIONS && gm->mode != MT_GEOM_VOXEL && gm->mode != MT_GEOM_POLY)
    return fail(c, MT_ERR_INVALID_ARG, "bad geometry mode");
  if (!(gm->x_min < gm->x_max) || !(gm->y_min < gm->y_max) || !(gm->z_min < gm->z_exit))
    return fail(c, MT_ERR_INVALID_ARG, "empty world box");
  if (gm->max_steps < 0 || gm->world_material < 0 || gm->world_material > c->n_materials)
    return fail(c, MT_ERR_INVALID_ARG, "bad max_steps or world_material");
  if (gm->exit_mode != MT_EXIT_AT_BREAK && gm->exit_mode != MT_EXIT_PROJECT) return fail(c, MT_ERR_INVALID_ARG, "bad exit_mode");
  if (gm->field_mode < 0 || gm->field_mode > (MT_FIELD_NEAREST | MT_FIELD_PER_STAGE))
    return fail(c, MT_ERR_INVALID_ARG, "bad field_mode");
  if ((gm->field_mode & MT_FIELD_NEAREST) && gm->mode != MT_GEOM_VOXEL)
    return fail(c, MT_ERR_INVALID_ARG, "MT_FIELD_NEAREST needs a voxel geometry");
  DeviceGuard g(c->device);
  std::vector<mt_region> regs;
  std::vector<mt_poly_block> blks;
  std::vector<double> weight(256, 0.0);                     // how much of the geometry each material fills
  if (gm->mode == MT_GEOM_POLY) {
    if (gm->n_blocks < 0 || gm->n_blocks > 1024) return fail(c, MT_ERR_UNSUPPORTED, "0..1024 blocks supported");
    if (gm->n_blocks > 0 && !gm->blocks) return fail(c, MT_ERR_INVALID_ARG, "null block array");
    blks.assign(gm->blocks, gm->blocks + gm->n_blocks);
    const int rc = build_hash(c, gm, blks, weight);
    if (rc != MT_OK) return rc;
  } else if (gm->mode == MT_GEOM_REGIONS) {
    if (gm->n_regions < 0 || gm->n_regions > 1024) return fail(c, MT_ERR_UNSUPPORTED, "0..1024 regions supported");
    if (gm->n_regions > 0 && !gm->regions) return fail(c, MT_ERR_INVALID_ARG, "null region array");
    regs.assign(gm->regions, gm->regions + gm->n_regions);
    double world = ((double)gm->x_max - gm->x_min) * ((double)gm->y_max - gm->y_min) * ((double)gm->z_exit - gm->z_min);
    for (size_t j = 0; j < regs.size(); ++j) {
      const mt_region& r = regs[j];
      if (!(r.z_lo < r.z_hi) || !(r.x_lo < r.x_hi) || !(r.y_lo < r.y_hi))
        return fail(c, MT_ERR_INVALID_ARG, "region %zu is empty", j);
      if (r.material < 0 || r.material > c->n_materials) return fail(c, MT_ERR_INVALID_ARG, "region %zu: bad material", j);
      if (j > 0 && !(regs[j - 1].z_hi <= r.z_lo))
        return fail(c, MT_ERR_INVALID_ARG, "regions must be sorted by z_lo and disjoint in z (region %zu)", j);
      const double dx = std::min(r.x_hi, gm->x_max) - std::max(r.x_lo, gm->x_min);
      const double dy = std::min(r.y_hi, gm->y_max) - std::max(r.y_lo, gm->y_min);
      const double dz = std::min(r.z_hi, gm->z_exit) - std::max(r.z_lo, gm->z_min);
      const double vol = std::max(dx, 0.0) * std::max(dy, 0.0) * std::max(dz, 0.0);
      weight[r.material] += vol;
      world -= vol;
    }
    weight[gm->world_material] += std::max(world, 0.0);
  } else {
    if (gm->nx < 1 || gm->ny < 1 || gm->nz < 1 || !(gm->cell > 0.0f) || !gm->d_material || !gm->d_field)
      return fail(c, MT_ERR_INVALID_ARG, "bad voxel grid");
    if (gm->nx > (1 << 20) || gm->ny > (1 << 20) || gm->nz > (1 << 20))
      return fail(c, MT_ERR_UNSUPPORTED, "voxel grid above 2^20 cells along an axis");
    const size_t n_cells = (size_t)(gm->nx + 2) * (gm->ny + 2) * (gm->nz + 2);       // with the replicated border
    if (n_cells >= ((size_t)1 << 31)) return fail(c, MT_ERR_UNSUPPORTED, "voxel grid above 2^31 cells");
    // from here on the library's grid is overwritten: a failure below leaves the context WITHOUT a geometry (never with
    // the previous geometry's parameters over the new grid's data)
    c->have_geom = false;
    MT_CUDA(c, c->d_grid.reserve(n_cells * sizeof(MtCellPair)));
    MT_CUDA(c, c->d_scratch.reserve(4096));
    MT_CUDA(c, cudaMemset(c->d_scratch.p, 0, 256 * sizeof(unsigned long long)));
    MT_CUDA(c, mt_launch_repack(gm->d_material, gm->d_field, (MtCellPair*)c->d_grid.p, gm->nx, gm->ny, gm->nz,
                                (unsigned long long*)c->d_scratch.p, 0));
    c->launches += 1;
    unsigned long long cells[256];
    MT_CUDA(c, cudaMemcpy(cells, c->d_scratch.p, sizeof cells, cudaMemcpyDeviceToHost));
    for (int m = 0; m < 256; ++m) {
      if (cells[m] && m > c->n_materials) return fail(c, MT_ERR_INVALID_ARG, "voxel grid holds material %d > n_materials", m);
      weight[m] = (double)cells[m];
    }
  }
  // MT_LEAN_INSIDE: g(x) = fl(fl(x - o) * inv_cell) is monotone in x, so the floats of the world box's half-open range
  // that map into [0, n) form an interval [lo, hi); it is the whole range but for a few floats next to a face (on
  // config 3, x = 1 - 2^-24 gives g = 200 = nx).  Found by stepping inward from each end.
  c->lean_inside = false;
  if (gm->mode == MT_GEOM_VOXEL) {
    const float inv_cell = 1.0f / gm->cell;
    auto g_of = [&](float x, float o) { const volatile float d = x - o; const volatile float g = d * inv_cell; return (float)g; };
    auto interval = [&](float lo, float hi, float o, int n, float* out) {
      float a = lo, b = nextafterf(hi, -INFINITY);                   // first and last float of [lo, hi)
      int k = 0;
      while (!(g_of(a, o) >= 0.0f) && k++ < 64) a = nextafterf(a, INFINITY);
      while (!(g_of(b, o) < (float)n) && k++ < 128) b = nextafterf(b, -INFINITY);
      out[0] = a; out[1] = nextafterf(b, INFINITY);
      return g_of(a, o) >= 0.0f && g_of(b, o) < (float)n && a <= b;
    };
    c->lean_inside = interval(gm->x_min, gm->x_max, gm->ox, gm->nx, c->lean_box) &&
                     interval(gm->y_min, gm->y_max, gm->oy, gm->ny, c->lean_box + 2) &&
                     interval(gm->z_min, gm->z_exit, gm->oz, gm->nz, c->lean_box + 4);
  }
  c->geom = *gm;
  c->geom.regions = nullptr; c->geom.d_material = nullptr; c->geom.d_field = nullptr;
  c->geom.blocks = nullptr;
  c->regions.swap(regs);
  c->blocks.swap(blks);
  c->geom.n_regions = (int32_t)c->regions.size();
  c->geom.n_blocks = (int32_t)c->blocks.size();
  c->have_geom = true;                     // (rebuild_blob stages the regions / blocks of a geometry that is set)
  // the most-used materials come first in the packed tables, so that a shared-memory prefix holds them
  order_materials(c, weight);
  int rc = upload_tables(c);
  if (rc == MT_OK) rc = rebuild_blob(c);
  // the header's promise: a failure after the swap leaves the context without a geometry (and, the tables having been
  // reordered for it, without tables), never with the new region / block counts over the old device blob
  if (rc != MT_OK) c->have_geom = c->have_tables = false;
  return rc;
}

int mt_load_histograms(mt_ctx* c, const mt_hist_desc* d) { return guarded(c, [&] { return load_histograms_impl(c, d); }); }
int mt_build_alias(mt_ctx* c, int placement) { return guarded(c, [&] { return build_alias_impl(c, placement); }); }
int mt_set_geometry(mt_ctx* c, const mt_geometry* gm) { return guarded(c, [&] { return set_geometry_impl(c, gm); }); }
int64_t mt_launch_count(const mt_ctx* c) { return c ? c->launches : 0; }

int mt_get_info(const mt_ctx* c, int what, int64_t* value) {
  if (!c || !value) return MT_ERR_INVALID_ARG;
  switch (what) {
    case MT_INFO_LEAN_FACTS: *value = (c->lean_axes ? 1 : 0) | (c->lean_inside ? 2 : 0); return MT_OK;
    case MT_INFO_LAST_LEAN: *value = c->last_lean; return MT_OK;
    case MT_INFO_LAST_SCHEDULE: *value = c->last_sched; return MT_OK;
    case MT_INFO_LAST_LANES: *value = c->last_lanes; return MT_OK;
    case MT_INFO_CHECK_ERRORS: {
      if (!MT_CHECKED_BUILD) { *value = -1; return MT_OK; }
      unsigned v[2] = {0, 0};
      DeviceGuard g(c->device);
      if (cudaDeviceSynchronize() != cudaSuccess || cudaMemcpy(v, c->d_check.p, sizeof v, cudaMemcpyDeviceToHost) != cudaSuccess)
        return MT_ERR_CUDA;
      *value = (int64_t)v[0] | ((int64_t)v[1] << 32);
      return MT_OK;
    }
    default: return MT_ERR_INVALID_ARG;
  }
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// transport
// ------------------------------------------------------------------------------------------------
namespace {

void fill_params(const mt_ctx* c, MtParams& P) {
  memset(&P, 0, sizeof P);
  const mt_geometry& g = c->geom;
  P.check = (unsigned*)c->d_check.p;
  P.n_tab_cells = c->selftest_bad_bounds ? 1u : (uint32_t)(c->table_bytes / (c->pack == 32 ? 4 : 8));
  P.n_grid_cells = (g.mode == MT_GEOM_VOXEL) ? (uint64_t)(g.nx + 2) * (g.ny + 2) * (g.nz + 2) : 0;
  P.n_hash_cells = (uint32_t)((size_t)c->hnx * c->hny * c->hnz);
  P.n_hash_list = c->n_hash_list;
  P.mode = g.mode;
  P.x_min = g.x_min; P.x_max = g.x_max; P.y_min = g.y_min; P.y_max = g.y_max; P.z_min = g.z_min; P.z_exit = g.z_exit;
  P.p_min = g.p_min; P.max_steps = g.max_steps; P.world_material = g.world_material;
  P.n_regions = g.n_regions;
  P.nx = g.nx; P.ny = g.ny; P.nz = g.nz; P.ox = g.ox; P.oy = g.oy; P.oz = g.oz;
  P.inv_cell = (g.mode == MT_GEOM_VOXEL) ? 1.0f / g.cell : 0.0f;          // IEEE float32 division (§3.2)
  P.grid = (const MtCellPair*)c->d_grid.p;
  P.gsy = g.nx + 2; P.gsz = (g.nx + 2) * (g.ny + 2);
  P.fnx = (float)g.nx; P.fny = (float)g.ny; P.fnz = (float)g.nz;
  P.grid_k = (0x4B400000u - 1u) * (uint32_t)(P.gsz + P.gsy + 1);
  P.gsy_bytes = (uint64_t)P.gsy * sizeof(MtCellPair); P.gsz_bytes = (uint64_t)P.gsz * sizeof(MtCellPair);
  P.gsyz_bytes = P.gsy_bytes + P.gsz_bytes;
  P.lean = (c->lean_axes ? MT_LEAN_AXES : 0) | (c->lean_inside ? MT_LEAN_INSIDE : 0) |
           ((c->zlut_n != 0 || g.n_regions <= 1) ? MT_LEAN_ZTABLE : 0);
  P.lean_x_lo = c->lean_box[0]; P.lean_x_hi = c->lean_box[1]; P.lean_y_lo = c->lean_box[2]; P.lean_y_hi = c->lean_box[3];
  P.lean_z_lo = c->lean_box[4]; P.lean_z_hi = c->lean_box[5];
  P.n_materials = c->n_materials; P.n_pbins = c->n_pbins; P.n_dp = c->n_dp; P.n_th = c->n_th;
  const bool joint = (c->hist_mode == MT_HIST_JOINT);
  P.n_joint = joint ? (uint32_t)(c->n_dp * c->n_th) : 0u;
  P.cells_per_bin = joint ? P.n_joint : (uint32_t)(c->n_dp + c->n_th);
  P.nth_magic = (uint32_t)((((uint64_t)1 << 32) + (uint64_t)c->n_th - 1) / (uint64_t)c->n_th);   // n_th = 1 wraps to 0: unused then
  P.field_mode = g.field_mode;
  P.exit_mode = g.exit_mode;
  P.n_blocks = g.n_blocks;
  P.hash_cells = (const uint2*)c->d_hash.p;
  P.hash_list = (const uint16_t*)((const char*)c->d_hash.p + c->hash_list_off);
  P.hnx = c->hnx; P.hny = c->hny; P.hnz = c->hnz;
  P.h_inv_x = c->h_inv[0]; P.h_inv_y = c->h_inv[1]; P.h_inv_z = c->h_inv[2];
  P.h_max_x = (float)(c->hnx - 1); P.h_max_y = (float)(c->hny - 1); P.h_max_z = (float)(c->hnz - 1);
  P.bin_shift = c->bin_shift; P.bin_key_lo = c->bin_key_lo; P.bin_key_max = c->bin_key_max;
  P.zlut_n = c->zlut_n; P.zlut_g0 = c->zlut_g0; P.zlut_inv = c->zlut_inv; P.zlut_max = (float)(c->zlut_n - 1);
  P.inv_p_lo = 1.0f / c->p_lo;
  P.bin_scale = (float)((double)c->n_pbins / log2((double)c->p_hi / (double)c->p_lo));
  P.tab32 = (c->pack == 32) ? (const uint32_t*)c->d_tab.p : nullptr;
  P.tab64 = (c->pack == 64) ? (const uint2*)c->d_tab.p : nullptr;
  P.blob = (const float*)c->d_blob.p;
  P.bl = c->bl;
}

// Everything about a call that does not depend on which muons a lane holds: the launch configuration, the schedule and,
// for WAVEFRONT, the slab and sort-key geometry.
struct Plan {
  MtParams P;                  // geometry, tables, Philox keys, output pointers of the WHOLE call
  MtLaunchCfg cfg;
  int sched = 0;
  unsigned persistent_grid = 0;
  double slab = 0.0;           // WAVEFRONT: slab thickness (m), passes, sort keys
  int n_pass = 0, n_keys = 0;
};

// One lane = one contiguous range of the call's muons with its own stream and scratch (DESIGN.md §7 "lanes").  The
// lanes of a call run concurrently: lane 0 on the highest-priority stream, the next ones filling the SMs that its
// z-slab passes leave idle in their tails (and, for the host-buffer call, computing while other lanes copy).
struct LaneWork {
  uint64_t off = 0, n = 0;     // muons [off, off + n) of the call
  MtParams P;                  // the plan's parameters narrowed to this range
  unsigned long long* work = nullptr;
  uint32_t* counts = nullptr;
  float4* rec[2] = {nullptr, nullptr};
  unsigned aux_grid = 0, grid = 0;
};

int ensure_lanes(mt_ctx* c, int K) {
  if (!c->ev_fork) MT_CUDA(c, cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
  if (!c->copy_in) MT_CUDA(c, cudaStreamCreateWithFlags(&c->copy_in, cudaStreamNonBlocking));
  int least = 0, greatest = 0;
  MT_CUDA(c, cudaDeviceGetStreamPriorityRange(&least, &greatest));      // greatest = numerically lowest = most urgent
  while ((int)c->lanes.size() < K) {
    Lane L;
    const int prio = std::min(least, greatest + (int)c->lanes.size());
    MT_CUDA(c, cudaStreamCreateWithPriority(&L.stream, cudaStreamNonBlocking, prio));
    MT_CUDA(c, cudaStreamCreateWithPriority(&L.stream_eq, cudaStreamNonBlocking, least));
    MT_CUDA(c, cudaEventCreateWithFlags(&L.done, cudaEventDisableTiming));
    MT_CUDA(c, cudaEventCreateWithFlags(&L.ready, cudaEventDisableTiming));
    c->lanes.push_back(L);
  }
  return MT_OK;
}

int make_plan(mt_ctx* c, uint64_t n, uint64_t seed, const mt_muons_out* out, Plan& pl) {
  MtParams& P = pl.P;
  fill_params(c, P);
  P.key0 = (uint32_t)seed; P.key1 = (uint32_t)(seed >> 32);
  for (uint32_t r = 0; r < 10; ++r) {                       // Philox round keys
    P.rk[2 * r] = P.key0 + r * 0x9E3779B9u;
    P.rk[2 * r + 1] = P.key1 + r * 0xBB67AE85u;
  }
  P.exit_rec = (float4*)out->exit_rec; P.exit_count = out->exit_count; P.exit_capacity = out->exit_capacity;
  P.counters = (unsigned long long*)out->counters;

  int sched = c->opt_sched;
  // POLY: muons sorted by xy cell and advanced slab by slab share a hash cell and its candidate blocks, so a warp's
  // containment tests stay convergent: 53.0 against 42.0 G muon-steps/s under REFILL (profiles/r1g_poly.md)
  // REGIONS: persistent-warp REFILL for small calls (one launch; a 65 536-muon config-1 call is bound by the latency of
  // one muon's history either way: 0.40 ms against 0.53 ms in slab passes), slab passes from 2^18 muons on, where
  // same-z warps look up one region and the passes of two lanes overlap (config 2 at 10^6 muons: 12.99 -> 10.9 ms,
  // profiles/r2b_lanes.md)
  if (sched == MT_SCHED_AUTO)
    sched = (c->geom.mode == MT_GEOM_REGIONS && n < ((uint64_t)1 << 18)) ? MT_SCHED_REFILL : MT_SCHED_WAVEFRONT;
  pl.sched = sched;
  P.refill_min_idle = c->opt_min_idle ? c->opt_min_idle : 1;

  // Table placement (north_star subsystem 1).  The packed tables start with the most-used material; shared
  // memory takes the longest prefix of whole material blocks that fits.  MT_PLACE_SMEM stages as many materials as fit;
  // AUTO: see below.
  MtLaunchCfg& cfg = pl.cfg;
  cfg.pack = c->pack;
  cfg.sched = sched;
  cfg.joint = (c->hist_mode == MT_HIST_JOINT);
  cfg.field = c->geom.field_mode;
  cfg.lean = false;
  const size_t blob_b = ((blob_bytes(c) + 15) & ~(size_t)15);
  const size_t smem_budget = c->smem_optin;
  if (blob_b + 16 > smem_budget) return fail(c, MT_ERR_UNSUPPORTED, "edges, axes and regions (%zu B) do not fit in shared memory", blob_b);
  const size_t cell_b = (c->pack == 32) ? 4 : 8;
  const size_t block_cells = (size_t)c->n_pbins * P.cells_per_bin;                    // cells per material
  const size_t fit_blocks = std::min<size_t>((smem_budget - blob_b - 16) / (block_cells * cell_b), c->n_materials);
  size_t hot_blocks = 0;
  if (cfg.joint) {                                           // joint tables are MBs per material: always gathered from L2
    if (c->placement == MT_PLACE_SMEM) return fail(c, MT_ERR_UNSUPPORTED, "joint tables are not staged in shared memory");
  } else if (c->placement == MT_PLACE_SMEM) {
    if (fit_blocks == 0) return fail(c, MT_ERR_UNSUPPORTED, "no material's tables (%zu B) fit in shared memory", block_cells * cell_b);
    hot_blocks = fit_blocks;
  } else if (c->placement == MT_PLACE_AUTO) {
    // AUTO gathers from L1 / L2.  Since the field-grid loads stopped allocating in L1 (mt_step.cuh: MT_GRID_HINT) the tables
    // have it to themselves and staging loses for every shape: config 4's 50x128x64 (115 KB, all three materials in one
    // 768-thread CTA) 0.773 staged against 0.789 from L1 / L2, 100x256x128 (iron only) 0.711 against 0.775
    // (profiles/r2c_summary.md; in round 2, with the grid allocating, the smallest shape still gained 2 % from staging).
    hot_blocks = 0;
  }
  P.hot_cells = (uint32_t)(hot_blocks * block_cells);
  cfg.tab_smem = hot_blocks > 0;
  // voxel grids need both facts (the lean kernel has no inside-grid test), regions and polyhedra the axes fact only
  const bool facts = (c->geom.mode == MT_GEOM_VOXEL) ? ((P.lean & MT_LEAN_ALL) == MT_LEAN_ALL)
                     : (c->geom.mode == MT_GEOM_REGIONS) ? ((P.lean & (MT_LEAN_AXES | MT_LEAN_ZTABLE)) == (MT_LEAN_AXES | MT_LEAN_ZTABLE))
                     : ((P.lean & MT_LEAN_AXES) != 0);
  cfg.lean = !c->opt_no_lean && facts && mt_has_lean(c->geom.mode, cfg);
  c->last_lean = cfg.lean; c->last_sched = sched;
  cfg.smem_bytes = blob_b + ((hot_blocks * block_cells * cell_b + 15) & ~(size_t)15) + 16;

  // Block size.  A call that fills the machine takes the block that keeps the most threads resident; ties go to the smaller
  // block, except for the persistent CTAs of a z-slab pass, where fewer and larger CTAs are faster for the same 24 resident
  // warps (10^7 muons: 6 x 128 threads 143.6 ms, 3 x 256 142.4, 2 x 384 141.5, 1 x 768 139.2; from 2^21 muons on — a 2^17-muon
  // call is faster with 256-thread CTAs, 4.80 against 5.28 ms; profiles/r2c_summary.md).  A STATIC / REFILL call small enough to be resident all at once is spread as evenly as the block granularity
  // allows instead: its time is that of the fullest SM, so the block that minimises ceil(CTAs / SMs) x block wins
  // (config 1, 65 536 muons: 2 x 256 threads on most SMs but 3 x 128 = 384 at most -> 0.49 -> 0.37 ms, profiles/r2b_lanes.md).
  int occ = 0;
  cfg.block = 0;
  uint64_t best_load = ~(uint64_t)0;
  const bool one_launch = (sched != MT_SCHED_WAVEFRONT);
  for (unsigned cand : {128u, 256u, 384u, 512u, 768u}) {
    if (c->opt_block && cand != 256u) continue;
    const unsigned blk = c->opt_block ? (unsigned)c->opt_block : cand;
    MtLaunchCfg probe = cfg;
    probe.block = blk;
    int o = 0;
    MT_CUDA(c, mt_occupancy(P, probe, &o));
    if (c->opt_blocks_per_sm) o = std::min(o, c->opt_blocks_per_sm);
    if (o < 1) continue;
    const uint64_t ctas = (n + blk - 1) / blk;
    if (one_launch && ctas <= (uint64_t)o * c->sm_count) {
      const uint64_t load = ((ctas + c->sm_count - 1) / c->sm_count) * blk;
      if (load < best_load) { best_load = load; occ = o; cfg.block = blk; }
    } else if (best_load == ~(uint64_t)0 && cand >= 256u &&
               ((size_t)o * blk > (size_t)occ * cfg.block ||
                (!one_launch && n >= ((uint64_t)1 << 21) && (size_t)o * blk == (size_t)occ * cfg.block))) {
      occ = o; cfg.block = blk;                     // (WAVEFRONT: ties -> the LARGER block, see above)
    }
  }
  if (occ < 1) return fail(c, MT_ERR_UNSUPPORTED, "kernel does not fit on an SM with %zu B shared memory", cfg.smem_bytes);
  pl.persistent_grid = (unsigned)(c->sm_count * occ);

  if (sched == MT_SCHED_WAVEFRONT) {
    // one pass per z-slab; between passes the live muons are counting-sorted by xy cell
    const bool voxel = (c->geom.mode == MT_GEOM_VOXEL);
    const double unit = voxel ? (double)c->geom.cell : 0.01;
    // default slab (units of 1 cm).  Voxel grids: 96 cells for a full batch (the slab's field layers stay L2-resident;
    // 64 ... 128 cells are within 0.4 % of each other at 10^7 muons); smaller calls are bound more and more by the latency
    // of one muon's ~2600 dependent steps and by the tails of their passes, and want fewer, thicker ones: 128 cells below
    // 2^22 muons, 512 below 2^18, and a single pass over the whole path below 2^15 (2^14 muons: 4.15 -> 3.13 ms, 2^16:
    // 4.20 -> 3.67, 2^19: 10.2 -> 9.8, 2^21: 33.3 -> 32.5; profiles/r2c_summary.md).  Region and polyhedra geometries
    // have no field working set to bound: 256 (profiles/r2b_lanes.md)
    // A trilinear field evaluated at every Runge-Kutta stage reads four times the grid records per step: its full
    // batches want the slab well inside L2 (32 cells 296 ms, 64 cells 309, 96 cells 328 per 10^7 muons).
    const bool stage_trilinear = voxel && (c->geom.field_mode & 3) == MT_FIELD_PER_STAGE;
    const double auto_slab = !voxel ? 256.0
                             : n < ((uint64_t)1 << 15) ? 1e9
                             : n < ((uint64_t)1 << 18) ? 512.0
                             : n < ((uint64_t)1 << 22) ? 128.0
                             : stage_trilinear ? 32.0 : 96.0;
    const double span = (double)c->geom.z_exit - (double)c->geom.z_min;
    pl.slab = (c->opt_slab_cells ? (double)c->opt_slab_cells : auto_slab) * unit;
    if (span > 0.0 && std::isfinite(span)) pl.slab = std::min(pl.slab, span);      // (one pass: the slab is the whole path)
    pl.n_pass = (int)std::max(1.0, std::min(ceil(span / pl.slab), 4096.0));
    // sort key: the voxel column (coarsened until there are at most 2^18 keys), or a 128 x 128 grid over the world box
    int key_nx, key_ny;
    if (voxel) {
      int coarse = 1;
      while ((size_t)((c->geom.nx + coarse - 1) / coarse) * ((c->geom.ny + coarse - 1) / coarse) > ((size_t)1 << 18)) coarse *= 2;
      key_nx = (c->geom.nx + coarse - 1) / coarse; key_ny = (c->geom.ny + coarse - 1) / coarse;
      P.key_x0 = c->geom.ox; P.key_y0 = c->geom.oy; P.key_inv = 1.0f / (c->geom.cell * (float)coarse);
    } else {
      key_nx = key_ny = 128;
      const float ext = std::max(c->geom.x_max - c->geom.x_min, c->geom.y_max - c->geom.y_min);
      P.key_x0 = c->geom.x_min; P.key_y0 = c->geom.y_min; P.key_inv = 128.0f / ext;
    }
    P.key_nx = key_nx; P.key_ny = key_ny;
    P.key_look = (float)(pl.slab * 0.01 * (c->opt_key_look >= 0 ? (double)c->opt_key_look : 50.0));
    pl.n_keys = key_nx * key_ny;
    P.n_keys = (uint32_t)pl.n_keys;
  }
  return MT_OK;
}

// HOST buffers of mt_transport_host (null for the device call): each lane copies its own range in and out
struct HostIO {
  const float* pos_q; const float* mom;
  float* pos_flag; float* mom_steps;
};

int choose_lanes(const mt_ctx* c, uint64_t n, int sched, bool host_call) {
  if (c->opt_lanes > 0) return (int)std::min<uint64_t>((uint64_t)c->opt_lanes, std::max<uint64_t>(n / 32, 1));
  // Measured on config 3 and config 2 (profiles/r2b_lanes.md).  Host-buffer calls: with four lanes the copy in of lanes
  // 1-3 hides under lane 0's first passes and the copy out of lanes 0-2 under lane 3's last ones (the lanes' passes
  // alternate on the SMs, so all four finish within the last 15 % of the call): 159.4 -> 155 ms per 10^7 muons; each
  // further lane costs ~1.3 ms of pass start-up and tails.  Device calls: two lanes let one lane's
  // passes fill the tails of the other's between 2^18 and 2^21 muons (+1 to +6 % with item-mode passes); above that a single lane's passes
  // are long enough that their tails do not matter (one lane is 1 % faster), below it there is nothing to overlap.
  // REFILL and STATIC kernels run a muon's whole history in one launch: on a device call lanes only serialise them.  On
  // a host-buffer call that is what is wanted under every schedule: the lanes' kernels run one after the other in stream-
  // priority order (each sized for the whole machine), lane k + 1's inputs land while lane k computes and lane k's results
  // leave while lane k + 1 computes.
  if (host_call && n >= ((uint64_t)1 << 21)) return 4;
  if (sched == MT_SCHED_WAVEFRONT && n >= ((uint64_t)1 << 18) && n < ((uint64_t)1 << 21)) return 2;
  return 1;
}

int run_transport(mt_ctx* c, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                  const mt_muons_out* out, cudaStream_t stream, const HostIO* host) {
  if (!c->have_tables || !c->have_geom)
    return fail(c, MT_ERR_STATE, "mt_transport needs mt_build_alias and mt_set_geometry after the last mt_load_histograms");
  if (n == 0) return MT_OK;
  if (!in->pos_q || !in->mom || !out->pos_flag || !out->mom_steps) return fail(c, MT_ERR_INVALID_ARG, "null muon buffer");
  if (n >= ((uint64_t)1 << 32)) return fail(c, MT_ERR_UNSUPPORTED, "at most 2^32 - 1 muons per call");
  if (out->exit_rec && !out->exit_count) return fail(c, MT_ERR_INVALID_ARG, "exit_rec without exit_count");

  Plan pl;
  int rc = make_plan(c, n, seed, out, pl);
  if (rc != MT_OK) return rc;
  const int K = choose_lanes(c, n, pl.sched, host != nullptr);
  rc = ensure_lanes(c, K);
  if (rc != MT_OK) return rc;
  c->last_lanes = K;
  // WAVEFRONT pass mode (profiles/r2b_lanes.md).  Persistent CTAs pulling 32-muon items from a counter are the fastest way
  // through one lane's pass (10^7 muons: 148.2 against 149.0 ms).  With two lanes of a device call, one item per warp and
  // CTAs that exit with their items let the hardware interleave the lanes' CTAs, so each lane's tail and sort are filled
  // by the other's pass: 2^18 muons 6.89 -> 6.31 ms, 2^20 muons 18.74 -> 17.84 ms; those lanes run on equal-priority
  // streams (they should advance side by side).  Host-buffer calls keep persistent passes (item mode: 157.4 against 155 ms).
  // 256-thread CTAs in both modes: smaller ones lose more to CTA start-up than they gain in granularity (64 threads: -6 %).
  const bool item_mode = pl.sched == MT_SCHED_WAVEFRONT &&
                         (c->opt_pass_mode == 2 || (c->opt_pass_mode == 0 && K > 1 && host == nullptr));
  const bool equal_prio = c->opt_lane_prio == 2 || (c->opt_lane_prio == 0 && item_mode);
  // (staged tables: the block the occupancy search chose — one big CTA per SM holds the copy)
  const unsigned item_block = c->opt_block ? (unsigned)c->opt_block : (pl.cfg.tab_smem ? pl.cfg.block : 256u);
  if (item_mode) pl.cfg.block = item_block;
  auto lane_stream = [&](int k) { return equal_prio ? c->lanes[k].stream_eq : c->lanes[k].stream; };
  // Lane boundaries (multiples of 32 muons).  Device calls: equal shares.  Host-buffer calls: the first and the last lane
  // take half a share — what stays exposed of the copies is the first lane's way in and the last lane's way out
  // (1:3:3:1 measured 154.3 against 155.3 ms for equal lanes, profiles/r2b_lanes.md).
  std::vector<uint64_t> bounds(K + 1, n);
  {
    const bool taper = host != nullptr && K >= 3;
    const double total = taper ? (double)(K - 1) : (double)K;
    double acc = 0.0;
    bounds[0] = 0;
    for (int k = 0; k < K; ++k) {
      acc += (taper && (k == 0 || k == K - 1)) ? 0.5 : 1.0;
      const uint64_t b = (uint64_t)((double)n * acc / total);
      bounds[k + 1] = (k == K - 1) ? n : std::max(bounds[k], std::min<uint64_t>(n, (b + 31) & ~(uint64_t)31));
    }
  }

  // ---- per-lane parameters and scratch
  std::vector<LaneWork> W(K);
  const int n_pass = pl.n_pass, n_keys = pl.n_keys;
  for (int k = 0; k < K; ++k) {
    LaneWork& w = W[k];
    Lane& L = c->lanes[k];
    w.off = bounds[k];
    w.n = bounds[k + 1] - bounds[k];
    w.P = pl.P;
    MtParams& P = w.P;
    P.n = w.n; P.id_base = id_base + w.off; P.idx_base = (uint32_t)w.off;
    P.in_pos_q = (const float4*)in->pos_q + w.off; P.in_mom = (const float4*)in->mom + w.off;
    P.out_pos_flag = (float4*)out->pos_flag + w.off; P.out_mom_steps = (float4*)out->mom_steps + w.off;
    if (w.n == 0) continue;
    w.grid = (unsigned)std::min<uint64_t>(pl.persistent_grid, (w.n + pl.cfg.block - 1) / pl.cfg.block);
    if (item_mode) w.grid = (unsigned)((w.n + pl.cfg.block - 1) / pl.cfg.block);      // one muon per thread, 32 per warp-item
    if (pl.sched == MT_SCHED_STATIC) {
      w.grid = (unsigned)((w.n + pl.cfg.block - 1) / pl.cfg.block);
    } else if (pl.sched == MT_SCHED_REFILL) {
      MT_CUDA(c, L.scratch.reserve(4096));
      P.work_counter = (unsigned long long*)L.scratch.p;
    } else {
      // scratch: [n_pass + 1] work counters (u64), [n_pass + 1] live counts (u32), histogram and offsets [n_keys] (u32)
      // (item mode: MT_COUNTER_SLOTS x 8 spread tallies in front)
      const size_t off_work = (size_t)MT_COUNTER_SLOTS * 64;
      const size_t off_counts = off_work + (size_t)(n_pass + 1) * 8, off_hist = (off_counts + (size_t)(n_pass + 1) * 4 + 255) & ~(size_t)255;
      const size_t zero_b = off_hist + (size_t)n_keys * 4, scratch_b = zero_b + (size_t)n_keys * 4;
      MT_CUDA(c, L.scratch.reserve(std::max<size_t>(scratch_b, 4096)));
      P.counters_spread = P.counters ? (unsigned long long*)L.scratch.p : nullptr;
      P.persistent = item_mode ? 0 : 1;
      w.work = (unsigned long long*)((char*)L.scratch.p + off_work);
      w.counts = (uint32_t*)((char*)L.scratch.p + off_counts);
      P.hist = (uint32_t*)((char*)L.scratch.p + off_hist);
      P.key_offset = P.hist + n_keys;
      L.zero_bytes = zero_b;
      // in-flight state: two buffers of 48-byte records (read by a pass / parked by it), {key, rank} 8 B and the
      // permutation 4 B per muon
      const size_t n48 = ((size_t)w.n * 48 + 255) & ~(size_t)255, n8 = ((size_t)w.n * 8 + 255) & ~(size_t)255,
                   n4 = ((size_t)w.n * 4 + 255) & ~(size_t)255;
      MT_CUDA(c, L.wave.reserve(2 * n48 + n8 + n4));
      char* wb = (char*)L.wave.p;
      w.rec[0] = (float4*)wb; w.rec[1] = (float4*)(wb + n48);
      P.sort_key = (uint2*)(wb + 2 * n48);
      P.perm = (uint32_t*)(wb + 2 * n48 + n8);
      w.aux_grid = (unsigned)std::min<uint64_t>((uint64_t)c->sm_count * 8, (w.n + 255) / 256);
    }
  }

  // From the fork on, library streams hold work that the caller's stream has not been told to wait for: the fork, the
  // launches and the join run inside `enqueue`, and if any of it fails the lanes are drained on the host before the error
  // goes back (so a failed call never leaves kernels or copies running behind the caller's back on buffers it owns).
  auto enqueue = [&]() -> int {
  // ---- fork: every lane (and the copy-in stream) starts where the caller's stream stands
  MT_CUDA(c, cudaEventRecord(c->ev_fork, stream));
  if (host) MT_CUDA(c, cudaStreamWaitEvent(c->copy_in, c->ev_fork, 0));
  for (int k = 0; k < K; ++k) {
    if (W[k].n == 0) continue;
    Lane& L = c->lanes[k];
    cudaStream_t LS = lane_stream(k);
    MT_CUDA(c, cudaStreamWaitEvent(LS, c->ev_fork, 0));
    if (host) {
      // inputs arrive lane by lane on ONE stream (in order, each at full link bandwidth); a lane starts when its own have landed
      const size_t b = (size_t)W[k].n * 16, o = (size_t)W[k].off * 4;
      MT_CUDA(c, cudaMemcpyAsync((float*)in->pos_q + o, host->pos_q + o, b, cudaMemcpyHostToDevice, c->copy_in));
      MT_CUDA(c, cudaMemcpyAsync((float*)in->mom + o, host->mom + o, b, cudaMemcpyHostToDevice, c->copy_in));
      MT_CUDA(c, cudaEventRecord(L.ready, c->copy_in));
      MT_CUDA(c, cudaStreamWaitEvent(LS, L.ready, 0));
    }
  }

  // ---- enqueue: prologues, then pass by pass across the lanes
  for (int k = 0; k < K; ++k) {
    LaneWork& w = W[k];
    if (w.n == 0) continue;
    Lane& L = c->lanes[k];
    cudaStream_t LS = lane_stream(k);
    MtLaunchCfg cfg = pl.cfg;
    cfg.grid = w.grid;
    if (pl.sched == MT_SCHED_STATIC) {
      MT_CUDA(c, mt_launch_transport(w.P, cfg, LS));
      c->launches += 1;
    } else if (pl.sched == MT_SCHED_REFILL) {
      MT_CUDA(c, cudaMemsetAsync(L.scratch.p, 0, 8, LS));
      MT_CUDA(c, mt_launch_transport(w.P, cfg, LS));
      c->launches += 1;
    } else {
      MT_CUDA(c, cudaMemsetAsync(L.scratch.p, 0, L.zero_bytes, LS));
      w.P.live_out_count = w.counts;                             // counts[s] = muons entering pass s
      MT_CUDA(c, mt_launch_wave_bin(w.P, w.aux_grid, LS));
      MT_CUDA(c, mt_launch_wave_sort(w.P, n_keys, w.aux_grid, LS));
      c->launches += 3;
    }
  }
  if (pl.sched == MT_SCHED_WAVEFRONT) {
    for (int s = 0; s < n_pass; ++s) {
      for (int k = 0; k < K; ++k) {
        LaneWork& w = W[k];
        if (w.n == 0) continue;
        cudaStream_t LS = lane_stream(k);
        MtLaunchCfg cfg = pl.cfg;
        cfg.grid = w.grid;
        MtParams& P = w.P;
        P.live_in_count = w.counts + s;
        P.live_out_count = w.counts + s + 1;
        P.work_counter = w.work + s;
        P.first_pass = (s == 0);
        // the live list is sorted before pass 0 and after every sort_every-th pass
        const int sort_every = c->opt_sort_every > 0 ? c->opt_sort_every : 1;
        P.sorted_in = (s % sort_every) == 0;
        P.sort_out = (s < n_pass - 1) && ((s + 1) % sort_every) == 0;
        P.rec_in = w.rec[(s + 1) & 1];
        P.rec_out = w.rec[s & 1];
        P.slab_z_end = (s == n_pass - 1) ? INFINITY : (float)((double)c->geom.z_min + (double)(s + 1) * pl.slab);
        P.lean_z_hi = std::min(c->lean_box[5], P.slab_z_end);
        MT_CUDA(c, mt_launch_transport(P, cfg, LS));
        c->launches += 1;
        if (P.sort_out) {
          MT_CUDA(c, mt_launch_wave_sort(P, n_keys, w.aux_grid, LS));
          c->launches += 2;
        } else if (item_mode && P.counters) {
          MT_CUDA(c, mt_launch_reduce_counters(P.counters_spread, P.counters, LS));
          c->launches += 1;
        }
      }
    }
  }

  // ---- join: results out (host call), and the caller's stream waits for every lane
  for (int k = 0; k < K; ++k) {
    if (W[k].n == 0) continue;
    Lane& L = c->lanes[k];
    cudaStream_t LS = lane_stream(k);
    if (host) {
      const size_t b = (size_t)W[k].n * 16, o = (size_t)W[k].off * 4;
      MT_CUDA(c, cudaMemcpyAsync(host->pos_flag + o, out->pos_flag + o, b, cudaMemcpyDeviceToHost, LS));
      MT_CUDA(c, cudaMemcpyAsync(host->mom_steps + o, out->mom_steps + o, b, cudaMemcpyDeviceToHost, LS));
    }
    MT_CUDA(c, cudaEventRecord(L.done, LS));
    MT_CUDA(c, cudaStreamWaitEvent(stream, L.done, 0));
  }
  return MT_OK;
  };
  rc = enqueue();
  if (rc != MT_OK) {
    if (host) cudaStreamSynchronize(c->copy_in);
    for (int k = 0; k < K; ++k) cudaStreamSynchronize(lane_stream(k));
    cudaGetLastError();                          // (the failure is already in last_error; leave no sticky-less error behind)
  }
  return rc;
}

}  // namespace

extern "C" {

int mt_transport(mt_ctx* c, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                 const mt_muons_out* out, void* cuda_stream) {
  if (!c || !in || !out) return MT_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  return guarded(c, [&] { return run_transport(c, in, n, id_base, seed, out, (cudaStream_t)cuda_stream, nullptr); });
}

static int transport_host_impl(mt_ctx* c, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                               const mt_muons_out* out, cudaStream_t stream) {
  if (n == 0) return MT_OK;
  if (!in->pos_q || !in->mom || !out->pos_flag || !out->mom_steps) return fail(c, MT_ERR_INVALID_ARG, "null muon buffer");
  if (out->exit_rec && !out->exit_count) return fail(c, MT_ERR_INVALID_ARG, "exit_rec without exit_count");
  if (!c->have_tables || !c->have_geom)
    return fail(c, MT_ERR_STATE, "mt_transport needs mt_build_alias and mt_set_geometry after the last mt_load_histograms");
  const size_t rec = n * 4 * sizeof(float);
  MT_CUDA(c, c->d_stage_in.reserve(2 * rec));
  MT_CUDA(c, c->d_stage_out.reserve(2 * rec));
  const size_t exit_b = out->exit_rec ? (size_t)out->exit_capacity * 8 * sizeof(float) : 0;
  MT_CUDA(c, c->d_stage_misc.reserve(exit_b + 128));
  char* d_in = (char*)c->d_stage_in.p;
  char* d_out = (char*)c->d_stage_out.p;
  char* d_misc = (char*)c->d_stage_misc.p;
  MT_CUDA(c, cudaMemsetAsync(d_misc, 0, 128, stream));
  mt_muons_in din = {(const float*)d_in, (const float*)(d_in + rec)};
  mt_muons_out dout;
  memset(&dout, 0, sizeof dout);
  dout.pos_flag = (float*)d_out;
  dout.mom_steps = (float*)(d_out + rec);
  dout.counters = out->counters ? (uint64_t*)d_misc : nullptr;            // 8 x u64 at offset 0
  if (out->exit_count) dout.exit_count = (uint32_t*)(d_misc + 64);
  if (out->exit_rec) {
    dout.exit_rec = (float*)(d_misc + 128);
    dout.exit_capacity = out->exit_capacity;
  }
  // the muon state is copied lane by lane inside run_transport, so that one lane computes while others copy
  const HostIO io = {in->pos_q, in->mom, out->pos_flag, out->mom_steps};
  const int rc = run_transport(c, &din, n, id_base, seed, &dout, stream, &io);
  if (rc != MT_OK) return rc;
  if (out->counters) MT_CUDA(c, cudaMemcpyAsync(out->counters, d_misc, 64, cudaMemcpyDeviceToHost, stream));
  if (out->exit_count) MT_CUDA(c, cudaMemcpyAsync(out->exit_count, d_misc + 64, sizeof(uint32_t), cudaMemcpyDeviceToHost, stream));
  if (out->exit_rec) MT_CUDA(c, cudaMemcpyAsync(out->exit_rec, d_misc + 128, exit_b, cudaMemcpyDeviceToHost, stream));
  MT_CUDA(c, cudaStreamSynchronize(stream));
  return MT_OK;
}

int mt_transport_host(mt_ctx* c, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                      const mt_muons_out* out, void* cuda_stream) {
  if (!c || !in || !out) return MT_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  return guarded(c, [&] { return transport_host_impl(c, in, n, id_base, seed, out, (cudaStream_t)cuda_stream); });
}

int mt_debug_sample(mt_ctx* c, int material, int pbin, int which, const uint32_t* d_words, uint64_t n,
                    uint32_t* d_cell_out, void* cuda_stream) {
  if (!c || !d_words || !d_cell_out) return MT_ERR_INVALID_ARG;
  if (!c->have_tables) return fail(c, MT_ERR_STATE, "mt_debug_sample before mt_build_alias");
  if (material < 1 || material > c->n_materials || pbin < 0 || pbin >= c->n_pbins || which < 0 || which > 1)
    return fail(c, MT_ERR_INVALID_ARG, "bad table selector");
  DeviceGuard g(c->device);
  const bool joint = (c->hist_mode == MT_HIST_JOINT);
  if (joint && which != 0) return fail(c, MT_ERR_INVALID_ARG, "joint tables have one table per (material, bin)");
  const size_t per_bin = joint ? (size_t)c->n_dp * c->n_th : (size_t)(c->n_dp + c->n_th);
  const size_t cell = (size_t)c->mat_cell0[material] + (size_t)pbin * per_bin + (which ? c->n_dp : 0);
  const char* tab = (const char*)c->d_tab.p + cell * (c->pack == 32 ? 4 : 8);
  const uint32_t N = joint ? (uint32_t)per_bin : (uint32_t)(which ? c->n_th : c->n_dp);
  MT_CUDA(c, mt_launch_debug_sample(c->pack, joint, tab, N, d_words, n, d_cell_out, (cudaStream_t)cuda_stream));
  c->launches += 1;
  return MT_OK;
}

int mt_debug_lookup(mt_ctx* c, const float* d_xyz, uint64_t n, int32_t* d_material_out, float* d_field_out,
                    void* cuda_stream) {
  if (!c || !d_xyz || !d_material_out || !d_field_out) return MT_ERR_INVALID_ARG;
  if (!c->have_tables || !c->have_geom) return fail(c, MT_ERR_STATE, "mt_debug_lookup before mt_set_geometry");
  DeviceGuard g(c->device);
  MtParams P;
  fill_params(c, P);
  const size_t smem = ((blob_bytes(c) + 15) & ~(size_t)15) + 16;
  if (smem > c->smem_optin) return fail(c, MT_ERR_UNSUPPORTED, "const blob (%zu B) does not fit in shared memory", smem);
  MT_CUDA(c, mt_launch_debug_lookup(P, smem, d_xyz, n, d_material_out, d_field_out, (cudaStream_t)cuda_stream));
  c->launches += 1;
  return MT_OK;
}

int mt_debug_philox(mt_ctx* c, uint64_t seed, uint64_t id_base, uint32_t step, uint64_t n, uint32_t* d_out,
                    void* cuda_stream) {
  if (!c || !d_out) return MT_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  MT_CUDA(c, mt_launch_debug_philox((uint32_t)seed, (uint32_t)(seed >> 32), id_base, step, n, d_out,
                                    (cudaStream_t)cuda_stream));
  c->launches += 1;
  return MT_OK;
}

}  // extern "C"

// ------------------------------------------------------------------------------------------------
// mt_transport_static_scratch: the transport call for callers that may not allocate (include/muon_transport.h)
// ------------------------------------------------------------------------------------------------
// All the scratch of one single-lane call, as a file-scope device array: part of the library's image, so each GPU that
// loads the library sets these 9 MiB aside until the process ends and no call ever has to ask the allocator for them.
// Sized for MT_STATIC_SCRATCH_MAX_MUONS muons under the largest bookkeeping a plan can ask for (4096 passes, 2^18 sort
// keys): 2.05 MiB of counters, histogram and offsets + 108 B per muon in flight = 8.80 MiB.
static __device__ __align__(256) unsigned char mt_static_scratch[MT_STATIC_SCRATCH_BYTES];

namespace {

// In host code the name `mt_static_scratch` is only a handle that the runtime can look the array up by; it is not where
// the array lives on the GPU, and a kernel handed `mt_static_scratch` itself from the host would read and write through a
// host address.  The device address comes from cudaGetSymbolAddress, asked once per device with that device current (each
// GPU has its own copy of the array) and kept for the rest of the process.
int static_scratch_base(mt_ctx* c, unsigned char** base) {
  enum { kMaxDevices = 64 };
  static unsigned char* known[kMaxDevices];      // zero-initialised; written once per device
  if (c->device < 0 || c->device >= kMaxDevices)
    return fail(c, MT_ERR_UNSUPPORTED, "mt_transport_static_scratch serves CUDA devices 0..%d", kMaxDevices - 1);
  unsigned char* p = __atomic_load_n(&known[c->device], __ATOMIC_ACQUIRE);
  if (!p) {
    void* sym = nullptr;
    MT_CUDA(c, cudaGetSymbolAddress(&sym, mt_static_scratch));      // (the caller's DeviceGuard made c->device current)
    if (!sym) return fail(c, MT_ERR_CUDA, "cudaGetSymbolAddress returned no address for the static scratch");
    p = (unsigned char*)sym;
    __atomic_store_n(&known[c->device], p, __ATOMIC_RELEASE);       // (two threads racing here store the same value)
  }
  *base = p;
  return MT_OK;
}

// One lane of run_transport on the caller's own stream, with the lane's two scratch buffers carved out of the static
// array instead of reserved from the allocator.  Nothing here may allocate: no DevBuf::reserve, no ensure_lanes (streams
// and events), no std::vector.
int run_transport_static_scratch(mt_ctx* c, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                                 const mt_muons_out* out, cudaStream_t stream) {
  if (!c->have_tables || !c->have_geom)
    return fail(c, MT_ERR_STATE, "mt_transport_static_scratch needs mt_build_alias and mt_set_geometry after the last mt_load_histograms");
  if (n == 0) return MT_OK;
  if (!in->pos_q || !in->mom || !out->pos_flag || !out->mom_steps) return fail(c, MT_ERR_INVALID_ARG, "null muon buffer");
  if (out->exit_rec && !out->exit_count) return fail(c, MT_ERR_INVALID_ARG, "exit_rec without exit_count");
  if (n > (uint64_t)MT_STATIC_SCRATCH_MAX_MUONS)
    return fail(c, MT_ERR_UNSUPPORTED,
                "mt_transport_static_scratch takes at most %d muons per call (%llu given): its scratch is a fixed %d-byte "
                "array; split the batch, or use mt_transport", (int)MT_STATIC_SCRATCH_MAX_MUONS, (unsigned long long)n,
                (int)MT_STATIC_SCRATCH_BYTES);
  unsigned char* base = nullptr;
  int rc = static_scratch_base(c, &base);
  if (rc != MT_OK) return rc;

  Plan pl;
  rc = make_plan(c, n, seed, out, pl);
  if (rc != MT_OK) return rc;
  c->last_lanes = 1;
  MtParams P = pl.P;
  P.n = n; P.id_base = id_base; P.idx_base = 0u;
  P.in_pos_q = (const float4*)in->pos_q; P.in_mom = (const float4*)in->mom;
  P.out_pos_flag = (float4*)out->pos_flag; P.out_mom_steps = (float4*)out->mom_steps;
  MtLaunchCfg cfg = pl.cfg;
  const uint64_t ctas = (n + cfg.block - 1) / cfg.block;

  if (pl.sched == MT_SCHED_STATIC) {                       // one lane per muon: no scratch at all
    cfg.grid = (unsigned)ctas;
    MT_CUDA(c, mt_launch_transport(P, cfg, stream));
    c->launches += 1;
    return MT_OK;
  }
  if (pl.sched == MT_SCHED_REFILL) {                       // the work counter idle lanes refill from
    cfg.grid = (unsigned)std::min<uint64_t>(pl.persistent_grid, ctas);
    P.work_counter = (unsigned long long*)base;
    MT_CUDA(c, cudaMemsetAsync(base, 0, 8, stream));       // (it still holds the last call's final value)
    MT_CUDA(c, mt_launch_transport(P, cfg, stream));
    c->launches += 1;
    return MT_OK;
  }

  // WAVEFRONT.  Bookkeeping first, as in run_transport: [MT_COUNTER_SLOTS x 8] spread tallies (unused here: persistent
  // passes add to the caller's counters directly), [n_pass + 1] work counters (u64), [n_pass + 1] live counts (u32), then
  // the key histogram and its scan [n_keys] (u32) each; then the state in flight: two buffers of 48-byte records, {key,
  // rank} 8 B and the permutation 4 B per muon.
  const int n_pass = pl.n_pass, n_keys = pl.n_keys;
  const size_t off_work = (size_t)MT_COUNTER_SLOTS * 64;
  const size_t off_counts = off_work + (size_t)(n_pass + 1) * 8;
  const size_t off_hist = (off_counts + (size_t)(n_pass + 1) * 4 + 255) & ~(size_t)255;
  const size_t zero_b = off_hist + (size_t)n_keys * 4;     // everything up to and including the histogram starts at zero
  const size_t off_wave = (zero_b + (size_t)n_keys * 4 + 255) & ~(size_t)255;
  const size_t n48 = ((size_t)n * 48 + 255) & ~(size_t)255, n8 = ((size_t)n * 8 + 255) & ~(size_t)255,
               n4 = ((size_t)n * 4 + 255) & ~(size_t)255;
  const size_t need = off_wave + 2 * n48 + n8 + n4;
  if (need > (size_t)MT_STATIC_SCRATCH_BYTES)              // (cannot happen for n <= the maximum; kept as the last line of defence)
    return fail(c, MT_ERR_UNSUPPORTED, "mt_transport_static_scratch: this call needs %zu bytes of scratch, the static array holds %d",
                need, (int)MT_STATIC_SCRATCH_BYTES);
  unsigned long long* work = (unsigned long long*)(base + off_work);
  uint32_t* counts = (uint32_t*)(base + off_counts);
  P.counters_spread = nullptr;
  P.persistent = 1;
  P.hist = (uint32_t*)(base + off_hist);
  P.key_offset = P.hist + n_keys;
  float4* rec[2] = {(float4*)(base + off_wave), (float4*)(base + off_wave + n48)};
  P.sort_key = (uint2*)(base + off_wave + 2 * n48);
  P.perm = (uint32_t*)(base + off_wave + 2 * n48 + n8);
  cfg.grid = (unsigned)std::min<uint64_t>(pl.persistent_grid, ctas);
  const unsigned aux_grid = (unsigned)std::min<uint64_t>((uint64_t)c->sm_count * 8, (n + 255) / 256);

  // The array keeps whatever the last call (of any context) left in it.  Counters and histogram must start at zero; the
  // records, keys and permutation are written before they are read.
  MT_CUDA(c, cudaMemsetAsync(base, 0, zero_b, stream));
  P.live_out_count = counts;                               // counts[s] = muons entering pass s
  MT_CUDA(c, mt_launch_wave_bin(P, aux_grid, stream));
  MT_CUDA(c, mt_launch_wave_sort(P, n_keys, aux_grid, stream));
  c->launches += 3;
  const int sort_every = c->opt_sort_every > 0 ? c->opt_sort_every : 1;
  for (int s = 0; s < n_pass; ++s) {
    P.live_in_count = counts + s;
    P.live_out_count = counts + s + 1;
    P.work_counter = work + s;
    P.first_pass = (s == 0);
    P.sorted_in = (s % sort_every) == 0;
    P.sort_out = (s < n_pass - 1) && ((s + 1) % sort_every) == 0;
    P.rec_in = rec[(s + 1) & 1];
    P.rec_out = rec[s & 1];
    P.slab_z_end = (s == n_pass - 1) ? INFINITY : (float)((double)c->geom.z_min + (double)(s + 1) * pl.slab);
    P.lean_z_hi = std::min(c->lean_box[5], P.slab_z_end);
    MT_CUDA(c, mt_launch_transport(P, cfg, stream));
    c->launches += 1;
    if (P.sort_out) {
      MT_CUDA(c, mt_launch_wave_sort(P, n_keys, aux_grid, stream));
      c->launches += 2;
    }
  }
  return MT_OK;
}

}  // namespace

extern "C" int mt_transport_static_scratch(mt_ctx* c, const mt_muons_in* in, uint64_t n, uint64_t id_base, uint64_t seed,
                                           const mt_muons_out* out, void* cuda_stream) {
  if (!c || !in || !out) return MT_ERR_INVALID_ARG;
  DeviceGuard g(c->device);
  return guarded(c, [&] { return run_transport_static_scratch(c, in, n, id_base, seed, out, (cudaStream_t)cuda_stream); });
}
