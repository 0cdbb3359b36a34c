// md_neighbor.cu — device-side system partitioning and neighbour-list build.
//
// Paper: section 3.2 and Fig.3.  The paper computes only the
// cell index on the GPU (G1-G3) and builds linked lists, sorts atoms by cell and re-sorts velocities
// on the HOST ("due to its sequential nature").  Here the whole chain runs on the
// device: histogram -> scan -> scatter -> per-cell ordering -> re-order -> list.  Whether a rebuild is due is decided on
// the device (decide_rebuild, md_internal.cuh): inside md_step's CUDA graphs the chain is the body of a conditional node;
// launched plainly, every kernel of the chain returns at once unless DevState says a rebuild is due.  Either way md_step
// never needs the host to look at the displacement flag.
#include <type_traits>

#include "md_internal.cuh"

namespace md {

__device__ __forceinline__ double wrap_coord(double x, double L) {
  // x - L*floor(x/L), each operation rounded once (same expression as the oracle's wrap)
  return __dsub_rn(x, __dmul_rn(L, floor(__ddiv_rn(x, L))));
}

__device__ __forceinline__ int cell_coord(double x, double scale, int nc) {
  int c = (int)(x * scale);
  return max(0, min(c, nc - 1));
}

// ---- K0: decision (one thread), then clear the cell counters -------------------------------------
// decide_rebuild (md_internal.cuh) as a kernel of its own: explicit builds and force evaluations outside md_step.
// Inside md_step the last block of the kernel that ends a drift takes the decision (finish_displacement).
__global__ void k_decide(const __grid_constant__ DevSys s, unsigned long long thr2_bits, cudaGraphConditionalHandle cond, int use_cond) {
  decide_rebuild(s, s.st->maxd2_bits > thr2_bits, cond, use_cond);
}

__global__ void k_clear_cells(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  if (blockIdx.x == 0 && threadIdx.x == 0) s.st->maxd2_bits = 0ull;      // x_ref <- x below: the displacement starts from 0 again
  for (int c = blockIdx.x * blockDim.x + threadIdx.x; c <= s.ncell; c += gridDim.x * blockDim.x) { s.cell_count[c] = 0; s.cell_fill[c] = 0; }
}

// ---- K1: wrap, cell index (paper's dIC, G1-G3), histogram (paper's hNAC) ---------------------
__global__ void k_bin(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  double4 p = s.pos[i];
  if (!(isfinite(p.x) && isfinite(p.y) && isfinite(p.z))) {
    atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
    p.x = p.y = p.z = 0.0;
  }
  const double L0 = box_edge(s, 0), L1 = box_edge(s, 1), L2 = box_edge(s, 2);
  p.x = wrap_coord(p.x, L0);
  p.y = wrap_coord(p.y, L1);
  p.z = wrap_coord(p.z, L2);
  s.pos[i] = p;
  const int cx = cell_coord(p.x, s.nc[0] / L0, s.nc[0]);
  const int cy = cell_coord(p.y, s.nc[1] / L1, s.nc[1]);
  const int cz = cell_coord(p.z, s.nc[2] / L2, s.nc[2]);
  // multiple boxes: cell ids of box I shifted by I*TNC
  const int cid = (i / s.npb) * s.tnc + (cx * s.nc[1] + cy) * s.nc[2] + cz;
  s.cell_id[i] = cid;
  atomicAdd(&s.cell_count[cid], 1);
}

// ---- K2-K4: exclusive scan of cell_count[0..ncell] -> cell_start (paper's hFA) ---------------
constexpr int kScanThreads = 1024, kScanItems = 4, kScanTile = kScanThreads * kScanItems;

__device__ __forceinline__ int block_exclusive_scan(int v, int *total) {
  __shared__ int warp_sum[32];
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) warp_sum[wid] = inc;
  __syncthreads();
  if (wid == 0) {
    int w = warp_sum[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int t = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += t;
    }
    warp_sum[lane] = winc - w;          // exclusive prefix of warp totals
    if (lane == 31) *total = winc;
  }
  __syncthreads();
  return warp_sum[wid] + inc - v;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_local(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  __shared__ int total;
  const int n = s.ncell + 1, base = blockIdx.x * kScanTile + threadIdx.x * kScanItems;
  int v[kScanItems], sum = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) { v[k] = (base + k < n) ? s.cell_count[base + k] : 0; sum += v[k]; }
  int ex = block_exclusive_scan(sum, &total);
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) { if (base + k < n) s.cell_start[base + k] = ex; ex += v[k]; }
  if (threadIdx.x == 0) s.scan_block[blockIdx.x] = total;
}

__global__ void __launch_bounds__(kScanThreads) k_scan_blocks(const __grid_constant__ DevSys s, int nblk) {
  if (!s.st->do_rebuild) return;
  __shared__ int total;
  const int base = threadIdx.x * kScanItems;
  int v[kScanItems], sum = 0;
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) { v[k] = (base + k < nblk) ? s.scan_block[base + k] : 0; sum += v[k]; }
  int ex = block_exclusive_scan(sum, &total);
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) { if (base + k < nblk) s.scan_block[base + k] = ex; ex += v[k]; }
}

__global__ void __launch_bounds__(kScanThreads) k_scan_add(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int n = s.ncell + 1, base = blockIdx.x * kScanTile + threadIdx.x * kScanItems, off = s.scan_block[blockIdx.x];
#pragma unroll
  for (int k = 0; k < kScanItems; ++k) if (base + k < n) s.cell_start[base + k] += off;
}

// ---- K5: scatter slot indices into their cell segment (order inside a cell not yet defined) ----
__global__ void k_scatter(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const int c = s.cell_id[i];
  s.perm[s.cell_start[c] + atomicAdd(&s.cell_fill[c], 1)] = i;
}

// ---- K6: make the order inside every cell deterministic: ascending caller index -----------------
__global__ void k_cell_sort(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= s.ncell) return;
  int *seg = s.perm + s.cell_start[c];
  const int n = s.cell_count[c];
  for (int a = 1; a < n; ++a) {
    const int v = seg[a], key = s.orig[v];
    int b = a - 1;
    while (b >= 0 && s.orig[seg[b]] > key) { seg[b + 1] = seg[b]; --b; }
    seg[b + 1] = v;
  }
}

// ---- K7/K8: move every per-atom array into cell order (paper's H9-H28, on the host there) ------
__global__ void k_reorder(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const int src = s.perm[i];
  s.pos_tmp[i] = s.pos[src];
#pragma unroll
  for (int c = 0; c < 3; ++c) s.vel_tmp[(size_t)c * s.N + i] = s.vel[(size_t)c * s.N + src];
  s.type_tmp[i] = s.type[src];
  s.orig_tmp[i] = s.orig[src];
}

__global__ void k_copyback(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const double4 p = s.pos_tmp[i];
  s.pos[i] = p;
  s.pos32[i] = make_float4((float)p.x, (float)p.y, (float)p.z, 0.f);                     // the list build's first look at a candidate
  s.xref[i] = p.x; s.xref[(size_t)s.N + i] = p.y; s.xref[2 * (size_t)s.N + i] = p.z;   // x_ref <- x
#pragma unroll
  for (int c = 0; c < 3; ++c) s.vel[(size_t)c * s.N + i] = s.vel_tmp[(size_t)c * s.N + i];
  s.type[i] = s.type_tmp[i];
  s.orig[i] = s.orig_tmp[i];
}

#ifndef MD_LIST_MINB
#define MD_LIST_MINB 7                           // measured on B200: 6 / 7 / 8 blocks per SM (80 / 72 / 64 registers): 0.814 / 0.784 / 0.795 ms per step on cfg4
#endif

// ---- K9: the neighbour list (paper's G6, Fig.3) ---------------------------------------------------
// One thread per atom (as G6), but no shared-memory tiles: atoms are already in cell order, so the
// candidates of the three z-adjacent cells of one (x,y) column are one contiguous run of slots.
// The pair test is the canonical minimum image + non-contracted r2, so the sets are bit-exact.
// Each entry records which image was taken (2 bits per axis) so that the density and force passes
// can form the SAME d = (x_j - x_i) -/+ L without re-deciding.
__device__ __forceinline__ double4 ld_pos(const double4 *p) {        // one 256-bit load on the read-only path
  double4 v;
  asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
  return v;
}

// The canonical double-precision test of one candidate against r_l, with the shift of its run (d + 0.0 == d).  Out of line
// on purpose: the float classification of k_build_list calls it for about one candidate in 10^4, and inlined it would be
// if-converted into the candidate loop.
__device__ __noinline__ bool exact_within(const double4 *pj_ptr, double4 pi, double sx, double sy, double sz, double rl2) {
  const double4 pj = ld_pos(pj_ptr);
  const double dx = __dadd_rn(__dsub_rn(pj.x, pi.x), sx), dy = __dadd_rn(__dsub_rn(pj.y, pi.y), sy), dz = __dadd_rn(__dsub_rn(pj.z, pi.z), sz);
  return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz)) < rl2;
}

// The stencil is 3 x 3 columns of cells (cell side >= r_l in x and y), each column ONE contiguous run of slots:
// ZWIN = false: cubic cells, three cells of z per column; ZWIN = true (small boxes, DevSys::zfine > 1): thinner cells in z
// and per atom and column the z window that r_l can reach.
// The periodic image is decided per RUN of candidates, not per pair: a run that lies across the box boundary carries the
// shift (-L or +L per axis) and its image code, and d = (x_j - x_i) + shift.  For every pair that can be accepted this is
// the canonical minimum image of reading A3, bit for bit (d + 0.0 == d, d + (-L) == d - L): an accepted pair has
// |d_a + shift_a| < r_l <= L/3 on every axis, so that image IS the one the canonical rule picks; and a candidate whose
// canonical image differs from its run's has |d_a + shift_a| > L/2 there and, since the two cells are neighbours (at most
// two cell widths apart), its canonical component is longer than L - 2 L/nc >= one cell width >= r_l: rejected either way
// (every edge holds at least three cells, MD_EBOX otherwise).  This takes the compares and selects of the minimum image
// out of the candidate loop.  (Up to round 2 boxes with fewer than five cells per edge took the minimum image per pair,
// behind a single-precision filter and a second phase over the survivors; the per-run form with the float
// classification below replaced it: cfg2 list build 0.0827 -> 0.0806 ms per step, cfg0 0.0084 -> 0.0079.)
template <bool ZWIN, bool F32CLS>
__global__ void __launch_bounds__(kForceBlock, F32CLS ? MD_LIST_MINB : 0) k_build_list(const __grid_constant__ DevSys s) {
  if (!s.st->do_rebuild) return;
  const int bpb = (s.npb + blockDim.x - 1) / blockDim.x;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * blockDim.x + threadIdx.x;
  if (local >= s.npb) return;
  const int i = box * s.npb + local;
  const size_t tile = (size_t)box * s.tiles_per_box + (local >> 5);
  unsigned *row = s.nbr + nbr_row_offset(tile, s.cap, local & 31);
  const double4 pi = s.pos[i];
  const double L[3] = {box_edge(s, 0), box_edge(s, 1), box_edge(s, 2)};
  const float4 q32 = s.pos32[i];
  // F32CLS: a candidate is classified on the float copies of the coordinates wherever that is unambiguous.  With u = 2^-24,
  // |x| <= L and the shift rounded to float, each component of d = x_j - x_i (+ shift) is off by at most u (4 L + |d|), and
  // r2 = fma(dz, dz, fma(dy, dy, dx dx)) by at most E(r) = 2 sqrt(3) u r (4 L + r) + 4 u r^2 < u (14 L r + 7.5 r^2);
  // r^2 - E(r) grows with r, so a float r2 outside the band [r_l^2 - eps, r_l^2 + eps), eps = u (32 L r_l + 24 r_l^2) >=
  // 2 E(r_l) plus the rounding of the bounds themselves, is on the same side of r_l^2 as the canonical double-precision r2
  // of reading A3.  Inside the band (about one candidate in 10^4) the canonical test decides: the list is bit-exact either
  // way.  The split of a row at r_in only orders it (both parts of a row are tested against r_c by the passes): it is taken
  // from the float.
  const double eps32 = 5.9604644775390625e-8 * (32.0 * fmax(fmax(L[0], L[1]), L[2]) * s.rl + 24.0 * s.rl2);
  const float rl2_lo = (float)(s.rl2 - eps32), rl2_hi = (float)(s.rl2 + eps32), rl2_below = __int_as_float(__float_as_int(rl2_lo) - 1);
  const float rin2f = fminf((float)s.rin2, rl2_below);
  const int cx = cell_coord(pi.x, s.nc[0] / L[0], s.nc[0]);
  const int cy = cell_coord(pi.y, s.nc[1] / L[1], s.nc[1]);
  const int cz = cell_coord(pi.z, s.nc[2] / L[2], s.nc[2]);
  const int ncx = s.nc[0], ncy = s.nc[1], ncz = s.nc[2];
  constexpr int R = 1;
  const double ax = L[0] / ncx, ay = L[1] / ncy, az = L[2] / ncz;
  int n_all = 0;
  // pairs inside r_in (= r_c) now go to the front of the row (k = 0, 1, ...), skin pairs to the back (k = cap-1, cap-2, ...):
  // the two passes run the full pair evaluation only over the front part (md_force.cu)
  int n_in = 0, n_out = 0;
  // branch-free append (one predicated store): almost every trip has SOME lane that accepts its candidate, so a branchy
  // append would run for the whole warp on nearly every candidate
  int n_lost = 0;                                                 // accepted but not stored (row full)
  int m_out = s.cap - 1;                                          // next free entry from the back (n_out = cap - 1 - m_out)
  // keep(j, inside r_l, inside r_in, image code): the append; test_keep: the canonical double-precision decision first
  auto keep = [&](int j, bool within, bool in, unsigned code) {
    const bool acc = within && j != i;
    const bool put = acc && n_in <= m_out;                        // room: n_in + n_out < cap
    const int k = in ? n_in : m_out;
    // one predicated store, no branch: address = row + 4 * offset by one 32 x 32 -> 64 bit multiply-add
    asm volatile("{\n\t.reg .pred p;\n\t.reg .u64 a;\n\tsetp.ne.u32 p, %3, 0;\n\tmad.wide.u32 a, %1, 4, %0;\n\t@p st.global.u32 [a], %2;\n\t}"
                 :: "l"((unsigned long long)row), "r"(nbr_entry(k)), "r"((unsigned)j | (code << kIdxBits)), "r"((unsigned)put) : "memory");
    n_in += (put && in) ? 1 : 0;
    m_out -= (put && !in) ? 1 : 0;
    n_lost += (acc && !put) ? 1 : 0;
  };
  auto test_keep = [&](int j, double r2, unsigned code) { keep(j, r2 < s.rl2, r2 < s.rin2, code); };
  // candidates of the slot range [jbeg, jend), all with the same periodic shift (sx, sy, sz) / image code
  auto scan_range = [&](int jbeg, int jend, double sx, double sy, double sz, unsigned code) {
    {
      // four candidates per trip: the four loads are issued together (read-only path, so the list stores
      // in between cannot hold them back), then the four tests
      // runs across the box boundary add the shift (d + (-L) == d - L bit for bit); the others (95 % in a large box) do not
      auto scan = [&](auto shifted) {
        auto dist2 = [&](const double4 &pj, double &r2) {
          double dx = __dsub_rn(pj.x, pi.x), dy = __dsub_rn(pj.y, pi.y), dz = __dsub_rn(pj.z, pi.z);
          if (decltype(shifted)::value) { dx = __dadd_rn(dx, sx); dy = __dadd_rn(dy, sy); dz = __dadd_rn(dz, sz); }
          r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
        };
        int j = jbeg;
        for (; j + 4 <= jend; j += 4) {
          const double4 p0 = ld_pos(s.pos + j), p1 = ld_pos(s.pos + j + 1), p2 = ld_pos(s.pos + j + 2), p3 = ld_pos(s.pos + j + 3);
          double r0, r1, r2, r3;
          dist2(p0, r0); dist2(p1, r1); dist2(p2, r2); dist2(p3, r3);
          test_keep(j, r0, code); test_keep(j + 1, r1, code); test_keep(j + 2, r2, code); test_keep(j + 3, r3, code);
        }
        for (; j < jend; ++j) {
          double r2;
          dist2(ld_pos(s.pos + j), r2);
          test_keep(j, r2, code);
        }
      };
      // the same runs on the float copies (16 bytes per candidate instead of 32, no FP64 instruction outside the band)
      auto scan32 = [&](auto shifted) {
        const float fx = (float)sx, fy = (float)sy, fz = (float)sz;
        auto ld32 = [&](int j) {
          float4 v;
          asm("ld.global.nc.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w) : "l"(s.pos32 + j));
          return v;
        };
        auto dist2f = [&](const float4 &a) {
          float dx = a.x - q32.x, dy = a.y - q32.y, dz = a.z - q32.z;
          if (decltype(shifted)::value) { dx += fx; dy += fy; dz += fz; }
          return fmaf(dz, dz, fmaf(dy, dy, dx * dx));
        };
        auto in_band = [&](float r2) { return !(r2 < rl2_lo) && r2 < rl2_hi; };
        // a candidate in the band gets the canonical test (reading A3) and leaves with an r2 outside the band, on the side
        // that test found: the decision below is then taken from the float alone, for every candidate alike
        auto settle = [&](int j, float &r2) {
          if (in_band(r2)) r2 = exact_within(s.pos + j, pi, sx, sy, sz, s.rl2) ? rl2_below : rl2_hi;
        };
        int j = jbeg;
        for (; j + 4 <= jend; j += 4) {
          const float4 a0 = ld32(j), a1 = ld32(j + 1), a2 = ld32(j + 2), a3 = ld32(j + 3);
          float r0 = dist2f(a0), r1 = dist2f(a1), r2 = dist2f(a2), r3 = dist2f(a3);
          if (in_band(r0) | in_band(r1) | in_band(r2) | in_band(r3)) { settle(j, r0); settle(j + 1, r1); settle(j + 2, r2); settle(j + 3, r3); }
          keep(j, r0 < rl2_lo, r0 < rin2f, code); keep(j + 1, r1 < rl2_lo, r1 < rin2f, code);
          keep(j + 2, r2 < rl2_lo, r2 < rin2f, code); keep(j + 3, r3 < rl2_lo, r3 < rin2f, code);
        }
        for (; j < jend; ++j) {
          float r2 = dist2f(ld32(j));
          settle(j, r2);
          keep(j, r2 < rl2_lo, r2 < rin2f, code);
        }
      };
      if constexpr (F32CLS) { if (code) scan32(std::true_type{}); else scan32(std::false_type{}); }
      else { if (code) scan(std::true_type{}); else scan(std::false_type{}); }
    }
  };
  // One (x, y) column of the stencil: up to three runs of slots: the in-range z cells (contiguous), plus the wrapped cell
  // on either side.  part 0: all of it; part 1 / 2 (the atom's own column): the slots ABOVE / BELOW the atom's own.
  auto column = [&](int ox, int oy, int part, auto &&range) {
    int jx = cx + ox, jy = cy + oy;
    double sx = 0.0, sy = 0.0; unsigned kx = 0, ky = 0;
    if (jx < 0) { jx += ncx; sx = -L[0]; kx = 2; } else if (jx >= ncx) { jx -= ncx; sx = L[0]; kx = 1; }
    if (jy < 0) { jy += ncy; sy = -L[1]; ky = 2; } else if (jy >= ncy) { jy -= ncy; sy = L[1]; ky = 1; }
    const int col = box * s.tnc + (jx * ncy + jy) * ncz;
    const unsigned kxy = kx | (ky << 2);
    int klo = cz - R, khi = cz + R;
    if constexpr (ZWIN) {
      // the z window of this column: every atom of it is at least (gx, gy) away laterally (the gaps to the column's faces),
      // so only z within w = sqrt(r_l^2 - gx^2 - gy^2) of z_i can be inside r_l; the margins cover the rounding of the
      // binning (an atom may sit 1e-13 outside the cell it was counted in); L >= 3 r_l: the window never meets itself
      const double gx = fmax(ox > 0 ? (cx + ox) * ax - pi.x : (ox < 0 ? pi.x - (cx + ox + 1) * ax : 0.0), 0.0);
      const double gy = fmax(oy > 0 ? (cy + oy) * ay - pi.y : (oy < 0 ? pi.y - (cy + oy + 1) * ay : 0.0), 0.0);
      const double w2 = s.rl2 * (1.0 + 1e-9) - gx * gx - gy * gy;
      if (!(w2 > 0.0)) return;
      const double w = sqrt(w2) + 1e-9;
      klo = (int)floor((pi.z - w) / az); khi = (int)floor((pi.z + w) / az);
      khi = min(khi, klo + ncz - 1);
    }
    const int zlo = max(klo, 0), zhi = min(khi, ncz - 1);
    for (int run = 0; run < 3; ++run) {                                       // one copy of the candidate loop
      int jbeg, jend;
      double sz = 0.0; unsigned kz = 0;
      if (run == 0) {                                                         // wrapped cells above: 0 .. khi - ncz
        if (part == 2 || khi <= ncz - 1) continue;
        jbeg = s.cell_start[col]; jend = s.cell_start[col + khi - ncz + 1]; sz = L[2]; kz = 1;
      } else if (run == 1) {                                                  // the in-range z cells
        jbeg = s.cell_start[col + zlo]; jend = s.cell_start[col + zhi + 1];
        if (part == 1) jbeg = max(jbeg, i + 1);
        if (part == 2) jend = min(jend, i);
      } else {                                                                // wrapped cells below: ncz + klo .. ncz - 1
        if (part == 1 || klo >= 0) continue;
        jbeg = s.cell_start[col + ncz + klo]; jend = s.cell_start[col + ncz]; sz = -L[2]; kz = 2;
      }
      range(jbeg, jend, sx, sy, sz, kxy | (kz << 4));
    }
  };
  // Scan order = ownership order (row f2, Newton's third law): first the half of the stencil whose pairs THIS atom owns
  // (columns (ox > 0, *), (0, oy > 0), and the slots above its own in its own column), then the other half.  Seen from
  // the partner the offsets are negated, so exactly one atom of every pair owns it, and a row holds its owned pairs first
  // in both of its parts without any sorting: at_switch() notes the fill levels between the two halves.
  auto stencil = [&](auto &&range, auto &&at_switch) {
    constexpr int W = 2 * R + 1, kCentre = (W * W) / 2;
#pragma unroll 1
    for (int c = 0; c <= W * W; ++c) {                                        // (ox, oy) in descending lexicographic order, the centre twice
      const int q = c <= kCentre ? c : c - 1;
      if (c == kCentre + 1) at_switch();
      column(R - q / W, R - q % W, c == kCentre ? 1 : (c == kCentre + 1 ? 2 : 0), range);   // ONE call site: one copy of the candidate loop
    }
  };
  int n_own_in = 0, n_own_out = 0;

  stencil(scan_range, [&]() { n_own_in = n_in; n_own_out = s.cap - 1 - m_out; });
  n_out = s.cap - 1 - m_out;
  n_all += n_in + n_out + n_lost;
  if (n_lost > 0) atomicOr(&s.st->error_flags, MD_FLAG_OVERFLOW);
  // the passes read whole groups of four: zero the unused entries of the two partly filled groups
  const int first_out = s.cap - n_out;
  for (int k = n_in; k < min((n_in + 3) & ~3, first_out); ++k) row[nbr_entry(k)] = 0u;
  for (int k = max(first_out & ~3, n_in); k < first_out; ++k) row[nbr_entry(k)] = 0u;
  s.ncount[i] = n_in | (n_out << 16);
  s.nown[i] = n_own_in | (n_own_out << 16);
  // statistics: one atomic per warp
  const unsigned act = __activemask();
  const int wsum = __reduce_add_sync(act, n_in + n_out), wmax = __reduce_max_sync(act, n_all);
  if ((threadIdx.x & 31) == __ffs(act) - 1) {
    atomicAdd(&s.st->list_entries, (unsigned long long)wsum);
    atomicMax(&s.st->max_neighbors, wmax);
  }
}

StepCtl make_ctl(const md_system *sys, double dt, cudaGraphConditionalHandle cond, bool use_cond, bool chain, int guard) {
  StepCtl c;
  c.dt = dt; c.thr2_bits = (unsigned long long)__builtin_bit_cast(long long, sys->d.thr2);
  c.cond = cond; c.use_cond = use_cond ? 1 : 0; c.chain = chain ? 1 : 0; c.guard = guard;
  return c;
}

// ---- loop graphs (md_api.cu): the one-thread kernels around the steps of a WHILE body -----------------------------------
__global__ void k_loop_head(const __grid_constant__ DevSys s) {
  DevState *st = s.st;
  st->loop_iters += 1;
  st->iters_this_launch += 1;
}
__global__ void k_rebuild_done(const __grid_constant__ DevSys s) { s.st->do_rebuild = 0; }      // last kernel of the rebuild chain in a loop graph
__global__ void k_loop_tail(const __grid_constant__ DevSys s, cudaGraphConditionalHandle loop_cond, int nsteps) {
  // every iteration completes at least one step (a pending rebuild is done first), so nsteps iterations always suffice
  DevState *st = s.st;
  const bool stuck = st->k_done < nsteps && st->iters_this_launch > nsteps + 1;
  if (stuck) st->error_flags |= 1 << 29;
  cudaGraphSetConditional(loop_cond, (st->k_done < nsteps && !stuck) ? 1u : 0u);
}
int launch_loop_head(md_system *sys) {
  ++sys->launches, k_loop_head<<<1, 1, 0, sys->stream>>>(sys->d);
  return (int)cudaGetLastError();
}
int launch_rebuild_done(md_system *sys) {
  ++sys->launches, k_rebuild_done<<<1, 1, 0, sys->stream>>>(sys->d);
  return (int)cudaGetLastError();
}
int launch_loop_tail(md_system *sys, cudaGraphConditionalHandle loop_cond, int nsteps) {
  ++sys->launches, k_loop_tail<<<1, 1, 0, sys->stream>>>(sys->d, loop_cond, nsteps);
  return (int)cudaGetLastError();
}

int launch_decide(md_system *sys, cudaGraphConditionalHandle cond, bool use_cond) {
  const StepCtl c = make_ctl(sys, 0.0, cond, use_cond, false);
  ProfScope p(sys, MD_K_BIN);
  ++sys->launches, k_decide<<<1, 1, 0, sys->stream>>>(sys->d, c.thr2_bits, cond, c.use_cond);
  return (int)cudaGetLastError();
}

// wrap, bin, scan, scatter, per-cell order, re-order, list: every kernel returns at once unless do_rebuild is set
int launch_rebuild_body(md_system *sys) {
  const DevSys &d = sys->d;
  cudaStream_t st = sys->stream;
  const int N = d.N, tb = 256, gN = (N + tb - 1) / tb;
  const int nscan = (d.ncell + 1 + kScanTile - 1) / kScanTile;
  {
    ProfScope p(sys, MD_K_BIN);
    int g0 = (d.ncell + 1 + tb - 1) / tb; if (g0 > 1184) g0 = 1184;
    ++sys->launches, k_clear_cells<<<g0, tb, 0, st>>>(d);
    ++sys->launches, k_bin<<<gN, tb, 0, st>>>(d);
  }
  {
    ProfScope p(sys, MD_K_SCAN);
    ++sys->launches, k_scan_local<<<nscan, kScanThreads, 0, st>>>(d);
    ++sys->launches, k_scan_blocks<<<1, kScanThreads, 0, st>>>(d, nscan);
    ++sys->launches, k_scan_add<<<nscan, kScanThreads, 0, st>>>(d);
  }
  {
    ProfScope p(sys, MD_K_SORT);
    ++sys->launches, k_scatter<<<gN, tb, 0, st>>>(d);
    ++sys->launches, k_cell_sort<<<(d.ncell + 127) / 128, 128, 0, st>>>(d);
  }
  {
    ProfScope p(sys, MD_K_REORDER);
    ++sys->launches, k_reorder<<<gN, tb, 0, st>>>(d);
    ++sys->launches, k_copyback<<<gN, tb, 0, st>>>(d);
  }
  if (sys->integrator == MD_INT_GEAR5 && launch_gear_reorder(sys) != 0) return 1;
  {
    ProfScope p(sys, MD_K_LIST);
    const int gl = d.nb * blocks_per_box(d.npb, kForceBlock);
    // MD_LIST_F64: every candidate tested in double precision (for the measurement in DESIGN.md section 6)
    const bool f64 = getenv("MD_LIST_F64") != nullptr;
    ++sys->launches;
    if (d.zfine > 1) {
      if (f64) k_build_list<true, false><<<gl, kForceBlock, 0, st>>>(d); else k_build_list<true, true><<<gl, kForceBlock, 0, st>>>(d);
    } else {
      if (f64) k_build_list<false, false><<<gl, kForceBlock, 0, st>>>(d); else k_build_list<false, true><<<gl, kForceBlock, 0, st>>>(d);
    }
  }
  return (int)cudaGetLastError();
}

int launch_rebuild_chain(md_system *sys) {
  cudaGraphConditionalHandle none{};
  int rc = launch_decide(sys, none, false);
  if (rc != 0) return rc;
  return launch_rebuild_body(sys);
}

}  // namespace md
