// oracle/muon_oracle.cpp
//
// TEST INFRASTRUCTURE ONLY.  Plain, slow, single-purpose CPU restatement of the per-muon transport
// loop of "Ultra-Fast Muon Transport via Histogram Sampling on GPUs" (arxiv 2512.10520), written
// from /root/reference/PAPER.md and the arithmetic contract in DESIGN.md §3.  Only tests/,
// __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load this file.
// It shares no code, header, table or constant generator with paper_2512_10520_b200/csrc/.
//
// What follows what (PAPER.md line, section):
//   transport loop ............ Algorithm 1, L141-172 (§4); iteration order of §2
//   alias sampling ............ L53 (§2 "The Alias Method"), L124 (§4.2)
//   alias construction ........ L53, L77 (Walker 1977 / Vose pairing; DESIGN.md §3.9 fixes the order)
//   log momentum bins ......... L99 (§3.1), L178 (§5: 95 bins, 0.18-400 GeV)
//   jitter, log axes .......... L75 (§3)
//   azimuth, kick, rotation ... L124-129, Eq. 3; L161-165
//   field lookup .............. L133 (§4.3; BASELINE.json configs[3] asks for trilinear)
//   RK4 Lorentz push .......... L135-137 Eq. 4; L168-170 (one GetField per step, then RK4Step)
//   termination ............... L65, L149
//   joint 2D histogram mode ... L77 (§3), Fig. 3 L95, L163
//   nearest-neighbour field ... L133 (§4.3); per-stage field evaluation: Eq. 4 integrated by RK4 proper
//   exit record on the plane .. L182: straight-line projection of an EXITED muon back onto z_exit
//   convex-polyhedra lookup ... L109-120 (§4.1), Eq. 2; the spatial hash of L120 only prunes, so the
//                               oracle scans every block
//
// Two modes from one templated source: Real=float is the parity reference (every + - * is one
// IEEE binary32 operation in the written order, fma where DESIGN.md says fma; compile with
// -ffp-contract=off); Real=double is the physics mode used by the closed-form pins (straight line,
// helix, RK4 order).  Per-muon code is single-threaded; OpenMP only spreads independent muons.
//
// Parity pins (tests/test_oracle_*.py): Philox vs cuRAND / Triton's interpreter; alias build vs
// the mass-conservation identity; alias sampling vs exact enumeration and chi-square; bin edges vs
// the paper's worked example (118.47-128.48 GeV); straight line; helix; RK4 h^4 convergence;
// Rodrigues (Eq. 3) in double; trilinear on affine fields; region lookup vs brute force;
// exp2/sin/cos polynomials vs libm; two-word alias draw vs the exact pmf of the table; joint-mode kick vs its
// geometry; nearest field vs the stored cell values; per-stage push vs h^4 convergence in a field gradient;
// polyhedra containment vs scipy's convex hull of the eight vertices, the prismatoid volume, and the box regions;
// exit projection vs the exact plane crossing of a straight line and the sagitta bound in a uniform field; the break
// tests of Algorithm 1 l.2-4 vs hand-worked literals for every bound, NaN and the priority order (test_oracle_breaks.py);
// the whole loop vs its own libm witness (ELEM_LIBM below) at north_star's tolerance (test_oracle_witness.py).
// Physics fidelity vs Geant4 (Figs. 5, 7): parity unpinned
// (needs Geant4 histograms, not available).

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

// ------------------------------------------------------------------------------------------------
// Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11).  DESIGN.md §3.0.
// ------------------------------------------------------------------------------------------------
void philox4x32_10(const uint32_t ctr_in[4], const uint32_t key_in[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;   // round multipliers
  const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;   // Weyl key increments
  uint32_t c0 = ctr_in[0], c1 = ctr_in[1], c2 = ctr_in[2], c3 = ctr_in[3];
  uint32_t k0 = key_in[0], k1 = key_in[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    const uint64_t p0 = (uint64_t)M0 * c0;
    const uint64_t p1 = (uint64_t)M1 * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// one block per (seed, muon id, step).
void muon_words(uint64_t seed, uint64_t id, uint32_t step, uint32_t w[4]) {
  const uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  const uint32_t ctr[4] = {(uint32_t)id, (uint32_t)(id >> 32), step, 0u};
  philox4x32_10(ctr, key, w);
}

// ------------------------------------------------------------------------------------------------
// Alias tables.  DESIGN.md §3.9 (build) and §3.5 (draw).
// ------------------------------------------------------------------------------------------------
// returns 0, or -1 when the histogram is empty / has a negative or non-finite weight
int build_alias(const float* counts, int N, float* prob, uint32_t* alias) {
  double sum = 0.0;
  for (int j = 0; j < N; ++j) {
    if (!(counts[j] >= 0.0f) || std::isinf(counts[j])) return -1;
    sum += (double)counts[j];
  }
  if (!(sum > 0.0)) return -1;
  std::vector<double> q(N);
  std::vector<int> small_, large_;
  for (int j = 0; j < N; ++j) {
    q[j] = ((double)counts[j] * (double)N) / sum;
    if (q[j] < 1.0) small_.push_back(j); else large_.push_back(j);
  }
  while (!small_.empty() && !large_.empty()) {
    const int s = small_.back(); small_.pop_back();
    const int l = large_.back(); large_.pop_back();
    prob[s] = (float)q[s];
    alias[s] = (uint32_t)l;
    q[l] = (q[l] + q[s]) - 1.0;
    if (q[l] < 1.0) small_.push_back(l); else large_.push_back(l);
  }
  for (int j : large_) { prob[j] = 1.0f; alias[j] = (uint32_t)j; }
  for (int j : small_) { prob[j] = 1.0f; alias[j] = (uint32_t)j; }   // only through rounding
  return 0;
}

// one 32-bit word selects the cell (high part of w*N) and decides primary/alias (low part)
inline uint32_t alias_draw(const float* prob, const uint32_t* alias, int N, uint32_t w) {
  const uint64_t m = (uint64_t)w * (uint64_t)(uint32_t)N;
  const uint32_t k = (uint32_t)(m >> 32);
  const uint32_t a24 = ((uint32_t)m) >> 8;
  const float u = (float)a24 * 0x1p-24f;            // exact, in [0,1)
  return (u < prob[k]) ? k : alias[k];
}

// joint tables have up to 2^24 cells, so one word selects and a second one accepts
inline uint32_t alias_draw2(const float* prob, const uint32_t* alias, uint32_t N, uint32_t w_sel, uint32_t w_acc) {
  const uint32_t k = (uint32_t)(((uint64_t)w_sel * (uint64_t)N) >> 32);
  const float u = (float)(w_acc >> 8) * 0x1p-24f;    // exact, in [0,1)
  return (u < prob[k]) ? k : alias[k];
}

// ------------------------------------------------------------------------------------------------
// Momentum bins.  DESIGN.md §3.4.
// ------------------------------------------------------------------------------------------------
void make_edges(double p_lo, double p_hi, int n, float* edges /* n+1 */) {
  for (int j = 0; j <= n; ++j)
    edges[j] = (float)(p_lo * std::pow(p_hi / p_lo, (double)j / (double)n));
}

int momentum_bin(const float* edges, int n, float P) {
  // greatest j in [0, n-1] with edges[j] <= P; 0 when P is below the first edge
  int lo = 0, hi = n - 1;
  while (lo < hi) {
    const int mid = (lo + hi + 1) / 2;
    if (edges[mid] <= P) lo = mid; else hi = mid - 1;
  }
  return lo;
}

// ------------------------------------------------------------------------------------------------
// Real-number helpers: every operation is one rounding in Real.
// ------------------------------------------------------------------------------------------------
template <class R> inline R rfma(R a, R b, R c) { return std::fma(a, b, c); }
template <class R> inline R rrcp(R a) { return (R)1 / a; }

// 2^y by rint split + degree-7 Taylor polynomial in r = y - rint(y).
template <class R> R exp2c(R y) {
  const R E1 = (R)0x1.62e430p-1f, E2 = (R)0x1.ebfbe0p-3f, E3 = (R)0x1.c6b08ep-5f,
          E4 = (R)0x1.3b2ab6p-7f, E5 = (R)0x1.5d87fep-10f, E6 = (R)0x1.430912p-13f,
          E7 = (R)0x1.ffcbfcp-17f;
  y = std::min(std::max(y, (R)-120), (R)120);
  const R n = std::nearbyint(y);                     // round-to-nearest-even
  const R r = y - n;                                 // exact
  R p = rfma(r, E7, E6);
  p = rfma(r, p, E5);
  p = rfma(r, p, E4);
  p = rfma(r, p, E3);
  p = rfma(r, p, E2);
  p = rfma(r, p, E1);
  p = rfma(r, p, (R)1);
  return std::ldexp(p, (int)n);                      // exact scaling by 2^n
}

// sine and cosine of (q + r) * pi/2, |r| <= 1/2, q an integer.
template <class R> void sincos_quadrant(int q, R r, R* sn, R* cs) {
  const R S1 = (R)0x1.921fb6p+0f, S3 = (R)-0x1.4abbcep-1f, S5 = (R)0x1.466bc6p-4f,
          S7 = (R)-0x1.32d2ccp-8f, S9 = (R)0x1.507834p-13f;
  const R C2 = (R)-0x1.3bd3ccp+0f, C4 = (R)0x1.03c1f0p-2f, C6 = (R)-0x1.55d3c8p-6f,
          C8 = (R)0x1.e1f506p-11f, C10 = (R)-0x1.a6d1f2p-16f;
  const R r2 = r * r;
  R ps = rfma(r2, S9, S7);
  ps = rfma(r2, ps, S5);
  ps = rfma(r2, ps, S3);
  ps = rfma(r2, ps, S1);
  const R s = r * ps;
  R pc = rfma(r2, C10, C8);
  pc = rfma(r2, pc, C6);
  pc = rfma(r2, pc, C4);
  pc = rfma(r2, pc, C2);
  const R c = rfma(r2, pc, (R)1);
  switch (q & 3) {
    case 0: *sn = s;  *cs = c;  break;
    case 1: *sn = c;  *cs = -s; break;
    case 2: *sn = -s; *cs = -c; break;
    default: *sn = -c; *cs = s; break;
  }
}

// azimuth phi = 2 pi k24 / 2^24 from the 24-bit integer k24
template <class R> void sincos_azimuth(uint32_t k24, R* sn, R* cs) {
  const uint32_t q = (k24 + (1u << 21)) >> 22;                       // 0..4
  const int32_t ri = (int32_t)k24 - (int32_t)(q << 22);              // [-2^21, 2^21)
  const R r = (R)ri * (R)0x1p-22f;                                   // exact
  sincos_quadrant<R>((int)q, r, sn, cs);
}

// polar angle theta in radians
template <class R> void sincos_polar(R theta, R* sn, R* cs) {
  const R PI_F = (R)0x1.921fb6p+1f, TWO_OVER_PI = (R)0x1.45f306p-1f;
  theta = std::min(theta, PI_F);
  const R t = theta * TWO_OVER_PI;
  const R qf = std::nearbyint(t);
  const R r = t - qf;                                                // exact
  sincos_quadrant<R>((int)qf, r, sn, cs);
}

// ------------------------------------------------------------------------------------------------
// The libm witness (R-21, §9): the plain definitions that the fixed polynomials of §3.6 stand for —
// 2^y, sin and cos from the C library in Real, the azimuth as phi = 2 pi u.  ELEM_LIBM runs Algorithm 1 with these in
// place of exp2c / sincos_polar / sincos_azimuth and nothing else changed; it is not the parity reference (its last
// bits are the C library's), it is the second witness against which north_star's real tolerance (>= 99.9 % of muons
// within 1e-5 relative in |p| and 1e-5 m, KS on the rest) is exercised.
// ------------------------------------------------------------------------------------------------
enum { ELEM_CONTRACT = 0, ELEM_LIBM = 1 };
template <class R> R exp2_libm(R y) { return std::exp2(y); }
template <class R> void sincos_polar_libm(R theta, R* sn, R* cs) {
  theta = std::min(theta, (R)0x1.921fb6p+1f);          // the same cap at pi as §3.6c
  *sn = std::sin(theta); *cs = std::cos(theta);
}
template <class R> void sincos_azimuth_libm(uint32_t k24, R* sn, R* cs) {
  const R phi = (R)6.283185307179586 * ((R)k24 * (R)0x1p-24f);       // phi = 2 pi u (L161)
  *sn = std::sin(phi); *cs = std::cos(phi);
}

// ------------------------------------------------------------------------------------------------
// Geometry.  DESIGN.md §3.2, §3.8.
// ------------------------------------------------------------------------------------------------
struct Region { float z_lo, z_hi, x_lo, x_hi, y_lo, y_hi; int32_t material; float bx, by, bz; };

// the solid between two quadrilateral faces, vertex i of the lower face joined to vertex i of the upper
struct PolyBlock { float z_lo, z_hi; float xy_lo[4][2]; float xy_hi[4][2]; int32_t material; float bx, by, bz; };

struct Geometry {
  int32_t mode;                 // 0 = regions, 1 = voxel, 2 = convex polyhedra
  float x_min, x_max, y_min, y_max, z_min, z_exit;
  float p_min; int32_t max_steps; int32_t world_material;
  int32_t n_regions; const Region* regions;
  int32_t nx, ny, nz; float ox, oy, oz, cell;
  const uint8_t* material;      // [nz][ny][nx]
  const float* field;           // [nz][ny][nx][3]
  int32_t field_mode;           // bit 0: nearest-neighbour instead of trilinear; bit 1: field at every RK4 stage
  int32_t n_blocks; const PolyBlock* blocks;   // mode 2
};
enum { FIELD_NEAREST = 1, FIELD_PER_STAGE = 2 };

struct Tables {
  int32_t n_materials, n_pbins, n_dp, n_th;
  double p_lo, p_hi;
  const float* prob_dp; const uint32_t* alias_dp;    // [n_materials][n_pbins][n_dp]
  const float* prob_th; const uint32_t* alias_th;    // [n_materials][n_pbins][n_th]
  const float* axis_dp; const float* axis_th;        // [n_materials][n_pbins][2] = {lo_log2, dlog2}
  const float* step_m;                               // [n_materials + 1]
  int32_t joint;   // 1: prob_dp / alias_dp are joint tables [n_materials][n_pbins][n_dp * n_th]
};

// regions: greatest j with z_lo[j] <= z (binary search), then the half-open box test
template <class R>
void region_lookup(const Geometry& g, R x, R y, R z, int* material, R B[3]) {
  *material = g.world_material; B[0] = B[1] = B[2] = (R)0;
  int lo = -1, hi = g.n_regions - 1;                 // invariant: regions[lo].z_lo <= z (or lo == -1)
  while (lo < hi) {
    const int mid = (lo + hi + 1) / 2;
    if ((R)g.regions[mid].z_lo <= z) lo = mid; else hi = mid - 1;
  }
  if (lo < 0) return;
  const Region& r = g.regions[lo];
  if (z < (R)r.z_hi && (R)r.x_lo <= x && x < (R)r.x_hi && (R)r.y_lo <= y && y < (R)r.y_hi) {
    *material = r.material; B[0] = (R)r.bx; B[1] = (R)r.by; B[2] = (R)r.bz;
  }
}

// voxel: containing cell for the material; returns false when outside the grid
template <class R>
bool voxel_cell(const Geometry& g, R x, R y, R z, int* ix, int* iy, int* iz) {
  const R inv_cell = rrcp<R>((R)g.cell);
  const R gx = (x - (R)g.ox) * inv_cell, gy = (y - (R)g.oy) * inv_cell, gz = (z - (R)g.oz) * inv_cell;
  const R fx = std::floor(gx), fy = std::floor(gy), fz = std::floor(gz);
  if (!(fx >= 0 && fx < (R)g.nx && fy >= 0 && fy < (R)g.ny && fz >= 0 && fz < (R)g.nz)) return false;
  *ix = (int)fx; *iy = (int)fy; *iz = (int)fz;
  return true;
}

// trilinear over cell centres, indices clamped at the faces; lerp x, then y, then z
template <class R>
void trilinear(const Geometry& g, R x, R y, R z, R B[3]) {
  const R inv_cell = rrcp<R>((R)g.cell);
  const R gx = rfma<R>(x - (R)g.ox, inv_cell, (R)-0.5);
  const R gy = rfma<R>(y - (R)g.oy, inv_cell, (R)-0.5);
  const R gz = rfma<R>(z - (R)g.oz, inv_cell, (R)-0.5);
  const R fx = std::floor(gx), fy = std::floor(gy), fz = std::floor(gz);
  const R tx = gx - fx, ty = gy - fy, tz = gz - fz;
  auto clampi = [](R f, int n) { int i = (int)f; return i < 0 ? 0 : (i > n - 1 ? n - 1 : i); };
  const int x0 = clampi(fx, g.nx), x1 = clampi(fx + 1, g.nx);
  const int y0 = clampi(fy, g.ny), y1 = clampi(fy + 1, g.ny);
  const int z0 = clampi(fz, g.nz), z1 = clampi(fz + 1, g.nz);
  auto at = [&](int iz, int iy, int ix, int c) -> R {
    return (R)g.field[(((size_t)iz * g.ny + iy) * g.nx + ix) * 3 + c];
  };
  for (int c = 0; c < 3; ++c) {
    const R v000 = at(z0, y0, x0, c), v001 = at(z0, y0, x1, c);
    const R v010 = at(z0, y1, x0, c), v011 = at(z0, y1, x1, c);
    const R v100 = at(z1, y0, x0, c), v101 = at(z1, y0, x1, c);
    const R v110 = at(z1, y1, x0, c), v111 = at(z1, y1, x1, c);
    const R a00 = rfma<R>(tx, v001 - v000, v000);
    const R a01 = rfma<R>(tx, v011 - v010, v010);
    const R a10 = rfma<R>(tx, v101 - v100, v100);
    const R a11 = rfma<R>(tx, v111 - v110, v110);
    const R b0 = rfma<R>(ty, a01 - a00, a00);
    const R b1 = rfma<R>(ty, a11 - a10, a10);
    B[c] = rfma<R>(tz, b1 - b0, b0);
  }
}

// PAPER.md L111-120, Eq. 2; DESIGN.md §3.12.  The quadrilateral slice of the block at height z, then the sign of
// S_i = (e_i x (p - v_i))_z for each of its four edges.
template <class R>
bool poly_contains(const PolyBlock& b, R x, R y, R z) {
  if (!((R)b.z_lo <= z && z < (R)b.z_hi)) return false;
  const R inv_dz = rrcp<R>((R)b.z_hi - (R)b.z_lo);
  const R t = (z - (R)b.z_lo) * inv_dz;
  R vx[4], vy[4];
  for (int i = 0; i < 4; ++i) {
    vx[i] = rfma<R>(t, (R)b.xy_hi[i][0] - (R)b.xy_lo[i][0], (R)b.xy_lo[i][0]);
    vy[i] = rfma<R>(t, (R)b.xy_hi[i][1] - (R)b.xy_lo[i][1], (R)b.xy_lo[i][1]);
  }
  bool all_ge = true, all_le = true, any_gt = false, any_lt = false;
  for (int i = 0; i < 4; ++i) {
    const int j = (i + 1) % 4;
    const R ex = vx[j] - vx[i], ey = vy[j] - vy[i];
    const R S = rfma<R>(ex, y - vy[i], -(ey * (x - vx[i])));
    all_ge = all_ge && (S >= (R)0);
    all_le = all_le && (S <= (R)0);
    any_gt = any_gt || (S > (R)0);
    any_lt = any_lt || (S < (R)0);
  }
  return (all_ge && any_gt) || (all_le && any_lt);
}

// first block, in index order, that contains the point (no pruning: L120's spatial hash only saves time)
template <class R>
void poly_lookup(const Geometry& g, R x, R y, R z, int* material, R B[3]) {
  *material = g.world_material; B[0] = B[1] = B[2] = (R)0;
  for (int j = 0; j < g.n_blocks; ++j) {
    if (poly_contains<R>(g.blocks[j], x, y, z)) {
      const PolyBlock& b = g.blocks[j];
      *material = b.material; B[0] = (R)b.bx; B[1] = (R)b.by; B[2] = (R)b.bz;
      return;
    }
  }
}

// material and field at a position (Alg. 1 l.5 and l.12 both use r before the move).  Field of a voxel grid:
// trilinear (BASELINE configs[3]) or, the stored value of the containing cell.
template <class R>
void material_and_field(const Geometry& g, R x, R y, R z, int* material, R B[3]) {
  if (g.mode == 0) { region_lookup<R>(g, x, y, z, material, B); return; }
  if (g.mode == 2) { poly_lookup<R>(g, x, y, z, material, B); return; }
  int ix, iy, iz;
  if (!voxel_cell<R>(g, x, y, z, &ix, &iy, &iz)) {
    *material = g.world_material; B[0] = B[1] = B[2] = (R)0; return;
  }
  const size_t cell = ((size_t)iz * g.ny + iy) * g.nx + ix;
  *material = g.material[cell];
  if (g.field_mode & FIELD_NEAREST) {
    for (int c = 0; c < 3; ++c) B[c] = (R)g.field[cell * 3 + c];
  } else {
    trilinear<R>(g, x, y, z, B);
  }
}

// ------------------------------------------------------------------------------------------------
// Kick + rotation (Eq. 3) and RK4 (Eq. 4).
// ------------------------------------------------------------------------------------------------
// orthonormal frame (e1, e2, d) with zhat -> d: the rotation of Eq. 3 about k = zhat x d
template <class R> void frame(R a, R b, R c, R e1[3], R e2[3]) {
  const R s = std::copysign((R)1, c);
  const R A = -rrcp<R>(s + c);
  const R Bq = (a * b) * A;
  const R sa = s * a;
  e1[0] = rfma<R>(sa * a, A, (R)1); e1[1] = s * Bq;                e1[2] = -sa;
  e2[0] = Bq;                       e2[1] = rfma<R>(b * b, A, s);  e2[2] = -b;
}

// p <- (P - P f) * [ sin(th) cos(phi) e1 + sin(th) sin(phi) e2 + cos(th) d ];  returns Pn
template <class R>
R kick(R p[3], R P, R f, R sin_t, R cos_t, R sin_phi, R cos_phi) {
  const R inv = rrcp<R>(P);
  const R a = p[0] * inv, b = p[1] * inv, c = p[2] * inv;
  R e1[3], e2[3];
  frame<R>(a, b, c, e1, e2);
  const R Pn = rfma<R>(-P, f, P);
  const R tx = sin_t * cos_phi, ty = sin_t * sin_phi;
  const R d[3] = {a, b, c};
  for (int i = 0; i < 3; ++i) p[i] = Pn * rfma<R>(tx, e1[i], rfma<R>(ty, e2[i], cos_t * d[i]));
  return Pn;
}

// classical RK4 over path length h of dr/ds = p/Pn, dp/ds = kappa q (p x B)/Pn, B frozen
template <class R>
void rk4_step(R r[3], R p[3], R Pn, R q, const R B[3], R h, R h2, R h6) {
  const R KAPPA = (R)0.299792458f;
  const R invP = rrcp<R>(Pn);
  const R c1 = (KAPPA * q) * invP;
  const R bx = c1 * B[0], by = c1 * B[1], bz = c1 * B[2];
  auto D = [&](const R v[3], R k[3]) {
    k[0] = rfma<R>(v[1], bz, -(v[2] * by));
    k[1] = rfma<R>(v[2], bx, -(v[0] * bz));
    k[2] = rfma<R>(v[0], by, -(v[1] * bx));
  };
  R k1[3], k2[3], k3[3], k4[3], p2[3], p3[3], p4[3];
  D(p, k1);
  for (int i = 0; i < 3; ++i) p2[i] = rfma<R>(h2, k1[i], p[i]);
  D(p2, k2);
  for (int i = 0; i < 3; ++i) p3[i] = rfma<R>(h2, k2[i], p[i]);
  D(p3, k3);
  for (int i = 0; i < 3; ++i) p4[i] = rfma<R>(h, k3[i], p[i]);
  D(p4, k4);
  const R w = h6 * invP;
  for (int i = 0; i < 3; ++i) {
    const R sp = rfma<R>((R)2, p2[i] + p3[i], p[i] + p4[i]);
    const R sk = rfma<R>((R)2, k2[i] + k3[i], k1[i] + k4[i]);
    r[i] = rfma<R>(w, sp, r[i]);
    p[i] = rfma<R>(h6, sk, p[i]);
  }
}

// kick of the joint mode, dp = P [ft cos(phi), ft sin(phi), -fz] in the muon's frame (L163),
// rotated by Eq. 3;  p <- P * [ ft cos(phi) e1 + ft sin(phi) e2 + (1 - fz) d ];  returns the new |p|
template <class R>
R kick_joint(R p[3], R P, R fz, R ft, R sin_phi, R cos_phi) {
  const R inv = rrcp<R>(P);
  const R a = p[0] * inv, b = p[1] * inv, c = p[2] * inv;
  R e1[3], e2[3];
  frame<R>(a, b, c, e1, e2);
  const R tx = ft * cos_phi, ty = ft * sin_phi;
  const R g = (R)1 - fz;
  const R d[3] = {a, b, c};
  for (int i = 0; i < 3; ++i) p[i] = P * rfma<R>(tx, e1[i], rfma<R>(ty, e2[i], g * d[i]));
  return std::sqrt(rfma<R>(p[2], p[2], rfma<R>(p[1], p[1], p[0] * p[0])));
}

// RK4 of the coupled system (r, p) with the field looked up at every stage position
template <class R>
void rk4_step_per_stage(const Geometry& g, R r[3], R p[3], R Pn, R q, R h, R h2, R h6) {
  const R KAPPA = (R)0.299792458f;
  const R invP = rrcp<R>(Pn);
  const R c1 = (KAPPA * q) * invP;
  auto D = [&](const R at[3], const R v[3], R k[3]) {
    int unused; R B[3];
    material_and_field<R>(g, at[0], at[1], at[2], &unused, B);
    const R bx = c1 * B[0], by = c1 * B[1], bz = c1 * B[2];
    k[0] = rfma<R>(v[1], bz, -(v[2] * by));
    k[1] = rfma<R>(v[2], bx, -(v[0] * bz));
    k[2] = rfma<R>(v[0], by, -(v[1] * bx));
  };
  const R u = h2 * invP, v = h * invP;
  R k1[3], k2[3], k3[3], k4[3], p2[3], p3[3], p4[3], r2[3], r3[3], r4[3];
  D(r, p, k1);
  for (int i = 0; i < 3; ++i) { p2[i] = rfma<R>(h2, k1[i], p[i]); r2[i] = rfma<R>(u, p[i], r[i]); }
  D(r2, p2, k2);
  for (int i = 0; i < 3; ++i) { p3[i] = rfma<R>(h2, k2[i], p[i]); r3[i] = rfma<R>(u, p2[i], r[i]); }
  D(r3, p3, k3);
  for (int i = 0; i < 3; ++i) { p4[i] = rfma<R>(h, k3[i], p[i]); r4[i] = rfma<R>(v, p3[i], r[i]); }
  D(r4, p4, k4);
  const R w = h6 * invP;
  for (int i = 0; i < 3; ++i) {
    const R sp = rfma<R>((R)2, p2[i] + p3[i], p[i] + p4[i]);
    const R sk = rfma<R>((R)2, k2[i] + k3[i], k1[i] + k4[i]);
    r[i] = rfma<R>(w, sp, r[i]);
    p[i] = rfma<R>(h6, sk, p[i]);
  }
}

// ------------------------------------------------------------------------------------------------
// Algorithm 1, one muon.
// ------------------------------------------------------------------------------------------------
enum { FLAG_STOPPED = 1, FLAG_EXITED = 2, FLAG_ESCAPED = 3, FLAG_MAXSTEPS = 4 };

struct StepTrace { int32_t material, pbin, cell_dp, cell_th; };

template <class R, int ELEM = ELEM_CONTRACT>
void transport_one(const Tables& T, const float* edges, const Geometry& g, uint64_t seed, uint64_t id,
                   R r[3], R p[3], R q, int32_t* flag_out, int32_t* steps_out,
                   StepTrace* trace, int32_t trace_cap) {
  const R F_MAX = (R)0.999f;
  int32_t step = 0;
  for (;;) {
    // l.2-4: break conditions
    const R P = std::sqrt(rfma<R>(p[2], p[2], rfma<R>(p[1], p[1], p[0] * p[0])));
    if (!(P >= (R)g.p_min)) { *flag_out = FLAG_STOPPED; break; }
    if (r[2] >= (R)g.z_exit) { *flag_out = FLAG_EXITED; break; }
    if (r[0] < (R)g.x_min || r[0] >= (R)g.x_max || r[1] < (R)g.y_min || r[1] >= (R)g.y_max ||
        r[2] < (R)g.z_min) { *flag_out = FLAG_ESCAPED; break; }
    if (step == g.max_steps) { *flag_out = FLAG_MAXSTEPS; break; }

    // l.5 GetMaterial and l.12 GetField, both at the start-of-step position
    int material; R B[3];
    material_and_field<R>(g, r[0], r[1], r[2], &material, B);
    const float hf = T.step_m[material];
    const R h = (R)hf, h2 = h * (R)0.5, h6 = (R)(float)((double)hf / 6.0);

    R Pn = P;
    StepTrace tr = {material, -1, -1, -1};
    if (material != 0) {
      // l.7 momentum bin
      const int i = momentum_bin(edges, T.n_pbins, (float)P);
      const size_t t = (size_t)(material - 1) * T.n_pbins + i;
      // l.8 alias draws + jitter, l.9 azimuth
      uint32_t w[4];
      muon_words(seed, id, (uint32_t)step, w);
      const R ud = (R)(w[2] >> 16) * (R)0x1p-16f, ut = (R)(w[2] & 0xFFFFu) * (R)0x1p-16f;
      uint32_t cd, ct;
      if (T.joint) {
        // the paper's own histogram (L77): one draw over the flattened (loss, kick) cells
        const uint32_t N = (uint32_t)T.n_dp * (uint32_t)T.n_th;
        const uint32_t cell = alias_draw2(T.prob_dp + t * N, T.alias_dp + t * N, N, w[0], w[1]);
        cd = cell / (uint32_t)T.n_th;
        ct = cell - cd * (uint32_t)T.n_th;
      } else {
        cd = alias_draw(T.prob_dp + t * T.n_dp, T.alias_dp + t * T.n_dp, T.n_dp, w[0]);
        ct = alias_draw(T.prob_th + t * T.n_th, T.alias_th + t * T.n_th, T.n_th, w[1]);
      }
      const R yd = rfma<R>((R)cd + ud, (R)T.axis_dp[2 * t + 1], (R)T.axis_dp[2 * t]);
      const R yt = rfma<R>((R)ct + ut, (R)T.axis_th[2 * t + 1], (R)T.axis_th[2 * t]);
      R sphi, cphi;
      if (ELEM == ELEM_LIBM) sincos_azimuth_libm<R>(w[3] >> 8, &sphi, &cphi);
      else sincos_azimuth<R>(w[3] >> 8, &sphi, &cphi);
      const R vd = (ELEM == ELEM_LIBM) ? exp2_libm<R>(yd) : exp2c<R>(yd);
      const R vt = (ELEM == ELEM_LIBM) ? exp2_libm<R>(yt) : exp2c<R>(yt);
      if (T.joint) {
        const R fz = std::min(vd, F_MAX);
        const R ft = vt;
        Pn = kick_joint<R>(p, P, fz, ft, sphi, cphi);
      } else {
        const R f = std::min(vd, F_MAX);
        const R theta = vt;
        R st, ctv;
        if (ELEM == ELEM_LIBM) sincos_polar_libm<R>(theta, &st, &ctv);
        else sincos_polar<R>(theta, &st, &ctv);
        // l.10-11 kick in the muon's frame, rotated to the lab (Eq. 3)
        Pn = kick<R>(p, P, f, st, ctv, sphi, cphi);
      }
      tr.pbin = i; tr.cell_dp = (int32_t)cd; tr.cell_th = (int32_t)ct;
    }
    if (trace && step < trace_cap) trace[step] = tr;
    // l.13 RK4: field frozen over the step (paper-literal) or looked up at every stage
    if (g.field_mode & FIELD_PER_STAGE) rk4_step_per_stage<R>(g, r, p, Pn, q, h, h2, h6);
    else rk4_step<R>(r, p, Pn, q, B, h, h2, h6);
    ++step;
  }
  *steps_out = step;
}

template <class R, int ELEM = ELEM_CONTRACT>
int transport_many(const Tables& T, const Geometry& g, uint64_t seed, uint64_t id_base,
                   const uint64_t* ids, uint64_t n, const R* pos_q, const R* mom,
                   R* out_pos, R* out_mom, int32_t* out_flag, int32_t* out_steps, int threads) {
  std::vector<float> edges(T.n_pbins + 1);
  make_edges(T.p_lo, T.p_hi, T.n_pbins, edges.data());
  (void)threads;
#ifdef _OPENMP
#pragma omp parallel for schedule(dynamic, 64) num_threads(threads > 0 ? threads : 1)
#endif
  for (int64_t k = 0; k < (int64_t)n; ++k) {
    R r[3] = {pos_q[4 * k], pos_q[4 * k + 1], pos_q[4 * k + 2]};
    R p[3] = {mom[4 * k], mom[4 * k + 1], mom[4 * k + 2]};
    const R q = pos_q[4 * k + 3];
    const uint64_t id = ids ? ids[k] : id_base + (uint64_t)k;
    transport_one<R, ELEM>(T, edges.data(), g, seed, id, r, p, q, &out_flag[k], &out_steps[k], nullptr, 0);
    for (int i = 0; i < 3; ++i) { out_pos[3 * k + i] = r[i]; out_mom[3 * k + i] = p[i]; }
  }
  return 0;
}

// the exit record of an EXITED muon moved back onto the plane z = z_exit along its final direction
template <class R> void exit_project(R r[3], const R p[3], R z_exit) {
  if (!(p[2] > (R)0)) return;
  const R s = (r[2] - z_exit) / p[2];
  r[0] = std::fma(-s, p[0], r[0]);
  r[1] = std::fma(-s, p[1], r[1]);
  r[2] = z_exit;
}

}  // namespace

// ------------------------------------------------------------------------------------------------
// C entry points for the ctypes wrapper in oracle/__init__.py
// ------------------------------------------------------------------------------------------------
extern "C" {

void orc_philox4x32_10(const uint32_t* ctr, const uint32_t* key, uint32_t* out, uint64_t n) {
  for (uint64_t i = 0; i < n; ++i) philox4x32_10(ctr + 4 * i, key, out + 4 * i);
}

void orc_muon_words(uint64_t seed, uint64_t id, uint32_t step, uint32_t* w) { muon_words(seed, id, step, w); }

int orc_build_alias(const float* counts, int n_tables, int N, float* prob, uint32_t* alias) {
  for (int t = 0; t < n_tables; ++t)
    if (build_alias(counts + (size_t)t * N, N, prob + (size_t)t * N, alias + (size_t)t * N)) return -(t + 1);
  return 0;
}

void orc_alias_draw(const float* prob, const uint32_t* alias, int N, const uint32_t* w, uint64_t n,
                    uint32_t* cell) {
  for (uint64_t i = 0; i < n; ++i) cell[i] = alias_draw(prob, alias, N, w[i]);
}

// exact outcome counts over all 2^32 words, for small N (brute force)
void orc_alias_enumerate(const float* prob, const uint32_t* alias, int N, uint64_t* counts) {
  for (int j = 0; j < N; ++j) counts[j] = 0;
  for (uint64_t w = 0; w < (1ull << 32); ++w) counts[alias_draw(prob, alias, N, (uint32_t)w)]++;
}

void orc_alias_draw2(const float* prob, const uint32_t* alias, uint32_t N, const uint32_t* w_sel,
                     const uint32_t* w_acc, uint64_t n, uint32_t* cell) {
  for (uint64_t i = 0; i < n; ++i) cell[i] = alias_draw2(prob, alias, N, w_sel[i], w_acc[i]);
}

double orc_kick_joint_f64(double* p, double P, double fz, double ft, uint32_t k24) {
  double sp, cp;
  sincos_azimuth<double>(k24, &sp, &cp);
  return kick_joint<double>(p, P, fz, ft, sp, cp);
}
float orc_kick_joint_f32(float* p, float P, float fz, float ft, uint32_t k24) {
  float sp, cp;
  sincos_azimuth<float>(k24, &sp, &cp);
  return kick_joint<float>(p, P, fz, ft, sp, cp);
}

void orc_make_edges(double p_lo, double p_hi, int n, float* edges) { make_edges(p_lo, p_hi, n, edges); }

void orc_momentum_bin(const float* edges, int n, const float* P, uint64_t m, int32_t* bin) {
  for (uint64_t i = 0; i < m; ++i) bin[i] = momentum_bin(edges, n, P[i]);
}

void orc_exp2c_f32(const float* y, uint64_t n, float* out) { for (uint64_t i = 0; i < n; ++i) out[i] = exp2c<float>(y[i]); }
void orc_sincos_polar_f32(const float* th, uint64_t n, float* s, float* c) {
  for (uint64_t i = 0; i < n; ++i) sincos_polar<float>(th[i], &s[i], &c[i]);
}
void orc_sincos_azimuth_f32(const uint32_t* k24, uint64_t n, float* s, float* c) {
  for (uint64_t i = 0; i < n; ++i) sincos_azimuth<float>(k24[i], &s[i], &c[i]);
}

void orc_frame_f64(const double* d, double* e1, double* e2) { frame<double>(d[0], d[1], d[2], e1, e2); }
void orc_frame_f32(const float* d, float* e1, float* e2) { frame<float>(d[0], d[1], d[2], e1, e2); }

double orc_kick_f64(double* p, double P, double f, double theta, uint32_t k24) {
  double st, ct, sp, cp;
  sincos_polar<double>(theta, &st, &ct); sincos_azimuth<double>(k24, &sp, &cp);
  return kick<double>(p, P, f, st, ct, sp, cp);
}
float orc_kick_f32(float* p, float P, float f, float theta, uint32_t k24) {
  float st, ct, sp, cp;
  sincos_polar<float>(theta, &st, &ct); sincos_azimuth<float>(k24, &sp, &cp);
  return kick<float>(p, P, f, st, ct, sp, cp);
}

void orc_rk4_f64(double* r, double* p, double q, const double* B, double h, int n_steps) {
  for (int s = 0; s < n_steps; ++s) {
    const double P = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]);
    rk4_step<double>(r, p, P, q, B, h, h * 0.5, h / 6.0);
  }
}
void orc_rk4_f32(float* r, float* p, float q, const float* B, float h, int n_steps) {
  for (int s = 0; s < n_steps; ++s) {
    const float P = std::sqrt(std::fma(p[2], p[2], std::fma(p[1], p[1], p[0] * p[0])));
    rk4_step<float>(r, p, P, q, B, h, h * 0.5f, (float)((double)h / 6.0));
  }
}

void orc_material_and_field_f32(const Geometry* g, const float* xyz, uint64_t n, int32_t* material, float* B) {
  for (uint64_t i = 0; i < n; ++i) {
    int m; material_and_field<float>(*g, xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], &m, B + 3 * i);
    material[i] = m;
  }
}
void orc_material_and_field_f64(const Geometry* g, const double* xyz, uint64_t n, int32_t* material, double* B) {
  for (uint64_t i = 0; i < n; ++i) {
    int m; material_and_field<double>(*g, xyz[3 * i], xyz[3 * i + 1], xyz[3 * i + 2], &m, B + 3 * i);
    material[i] = m;
  }
}

int orc_transport_f32(const Tables* T, const Geometry* g, uint64_t seed, uint64_t id_base, const uint64_t* ids,
                      uint64_t n, const float* pos_q, const float* mom, float* out_pos, float* out_mom,
                      int32_t* out_flag, int32_t* out_steps, int threads) {
  return transport_many<float>(*T, *g, seed, id_base, ids, n, pos_q, mom, out_pos, out_mom, out_flag, out_steps, threads);
}
int orc_transport_f64(const Tables* T, const Geometry* g, uint64_t seed, uint64_t id_base, const uint64_t* ids,
                      uint64_t n, const double* pos_q, const double* mom, double* out_pos, double* out_mom,
                      int32_t* out_flag, int32_t* out_steps, int threads) {
  return transport_many<double>(*T, *g, seed, id_base, ids, n, pos_q, mom, out_pos, out_mom, out_flag, out_steps, threads);
}

// the libm witness (ELEM_LIBM): same loop, C-library 2^y / sin / cos instead of the polynomials of DESIGN.md §3.6
int orc_transport_libm_f32(const Tables* T, const Geometry* g, uint64_t seed, uint64_t id_base, const uint64_t* ids,
                           uint64_t n, const float* pos_q, const float* mom, float* out_pos, float* out_mom,
                           int32_t* out_flag, int32_t* out_steps, int threads) {
  return transport_many<float, ELEM_LIBM>(*T, *g, seed, id_base, ids, n, pos_q, mom, out_pos, out_mom, out_flag, out_steps, threads);
}
int orc_transport_libm_f64(const Tables* T, const Geometry* g, uint64_t seed, uint64_t id_base, const uint64_t* ids,
                           uint64_t n, const double* pos_q, const double* mom, double* out_pos, double* out_mom,
                           int32_t* out_flag, int32_t* out_steps, int threads) {
  return transport_many<double, ELEM_LIBM>(*T, *g, seed, id_base, ids, n, pos_q, mom, out_pos, out_mom, out_flag, out_steps, threads);
}

// one muon, float32, with the per-step (material, pbin, cells) record
int orc_trace_f32(const Tables* T, const Geometry* g, uint64_t seed, uint64_t id, const float* pos_q,
                  const float* mom, float* out_pos, float* out_mom, int32_t* out_flag, int32_t* out_steps,
                  int32_t* trace /* [cap][4] */, int32_t cap) {
  std::vector<float> edges(T->n_pbins + 1);
  make_edges(T->p_lo, T->p_hi, T->n_pbins, edges.data());
  float r[3] = {pos_q[0], pos_q[1], pos_q[2]}, p[3] = {mom[0], mom[1], mom[2]};
  transport_one<float>(*T, edges.data(), *g, seed, id, r, p, pos_q[3], out_flag, out_steps,
                       reinterpret_cast<StepTrace*>(trace), cap);
  for (int i = 0; i < 3; ++i) { out_pos[i] = r[i]; out_mom[i] = p[i]; }
  return 0;
}

void orc_exit_project_f32(float* pos, const float* mom, uint64_t n, float z_exit) {
  for (uint64_t i = 0; i < n; ++i) exit_project<float>(pos + 3 * i, mom + 3 * i, z_exit);
}
void orc_exit_project_f64(double* pos, const double* mom, uint64_t n, double z_exit) {
  for (uint64_t i = 0; i < n; ++i) exit_project<double>(pos + 3 * i, mom + 3 * i, z_exit);
}

int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
