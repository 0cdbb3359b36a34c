// md_force.cu — density pass (paper's G18, Fig.5) and force pass with
// energy and virial (paper's G22, Fig.6), FP64, one thread per atom.
//
// Differences from the paper's kernels:
//  - atoms are in cell order and the list is a blocked-ELL array, so the list reads are coalesced and the
//    neighbour gathers hit L1/L2; the list entry and the gathered position of the NEXT pair are in flight while
//    the current pair is evaluated;
//  - the periodic image of each listed pair is recorded at build time, so there is no min/max logic in
//    the inner loop and r2 is bit-identical to the canonical expression;
//  - pairs that were inside r_c at build time come first in every row: that part of the loop is branch-free
//    (the switch function is clamped, so a pair that has drifted out contributes exactly 0); the skin pairs
//    behind them only get the 9-instruction distance test, and the few that have drifted inside r_c are
//    parked and evaluated together, so a warp does not run the heavy body for one lane at a time;
//  - r and 1/r come from one MUFU.RSQ64H seed + one cubic Newton step; exp() has no slow path (its argument
//    is bounded) and uses a 64-entry 2^(j/64) table in shared memory with a degree-5 polynomial;
//  - F'(rho_j) travels in the w component of the gathered position (one 32-byte sector per neighbour);
//  - energy and virial are reduced by warp shuffles into per-block partials and a second deterministic
//    pass, instead of shared-memory partials summed on the host.
#include "md_internal.cuh"

namespace md {

// ------------------------------------------------------------------------------------------------
// arithmetic helpers
// ------------------------------------------------------------------------------------------------

// d = (x_j - x_i) with the image recorded at build time: code 0: none, 1: +L, 2: -L.
__device__ __forceinline__ double image_delta(double xj, double xi, unsigned code, double L) {
  double d = __dsub_rn(xj, xi);
  if (code) d = (code == 2) ? __dsub_rn(d, L) : __dadd_rn(d, L);
  return d;
}

__device__ __forceinline__ double pair_r2(const double4 &pj, const double4 &pi, unsigned e, const DevSys &s,
                                          double &dx, double &dy, double &dz) {
  const unsigned code = e >> kIdxBits;
  if (code == 0) {
    dx = __dsub_rn(pj.x, pi.x); dy = __dsub_rn(pj.y, pi.y); dz = __dsub_rn(pj.z, pi.z);
  } else {
    dx = image_delta(pj.x, pi.x, code & 3u, s.L[0]);
    dy = image_delta(pj.y, pi.y, (code >> 2) & 3u, s.L[1]);
    dz = image_delta(pj.z, pi.z, (code >> 4) & 3u, s.L[2]);
  }
  return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
}

// 1/sqrt(x), x > 0 finite and normal: hardware seed (relative error ~2^-22) and one cubic Newton step
//   y1 = y (1 + e/2 + 3 e^2/8),  e = 1 - x y^2        (relative error 2.5 delta^3 ~ 2^-64 plus rounding)
__device__ __forceinline__ double rsqrt_fast(double x) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y * y, 1.0);
  const double p = fma(e, 0.375, 0.5);
  return fma(p, y * e, y);
}

// exp(x) for |x| < 690, no special cases.  n = rint(64 x / ln 2); r = x - n ln2/64, |r| <= 0.00542;
// exp(x) = 2^(n >> 6) tab[n & 63] (1 + r + r^2/2 + r^3/6 + r^4/24 + r^5/120); remainder r^6/720 < 3.5e-17.
__device__ __forceinline__ double exp_tab(double x, const double *__restrict__ tab) {
  constexpr double kMagic = 6755399441055744.0;                 // 1.5 * 2^52: the low word of t holds n
  const double t = fma(x, 0x1.71547652b82fep+6, kMagic);
  const double n = t - kMagic;
  double r = fma(n, -0x1.62e42fee00000p-7, x);                  // ln2/64, high 32 bits: n * hi is exact
  r = fma(n, -0x1.a39ef35793c76p-39, r);
  const int ni = __double2loint(t);
  const double T = tab[ni & 63];
  double p = fma(r, 1.0 / 120.0, 1.0 / 24.0);
  p = fma(p, r, 1.0 / 6.0);
  p = fma(p, r, 0.5);
  p = fma(p * r, r, r);
  const double v = fma(T, p, T);
  return __hiloint2double(__double2hiint(v) + ((ni >> 6) << 20), __double2loint(v));
}

// quintic switch on t in [0,1] (clamped): S = 1 - t^3 (10 - 15 t + 6 t^2), dS/dr = -30 t^2 (1-t)^2 inv_w.
// t <= 0 gives S = 1, dS = 0 and t >= 1 gives S = 0, dS = 0 exactly.
__device__ __forceinline__ double switch_t(double r, const TbsmaParams &tb) {
  return fmin(fmax(fma(r, tb.inv_w, tb.t0), 0.0), 1.0);
}
__device__ __forceinline__ double switch_S(double t) {
  const double t2 = t * t;
  return fma(-(t2 * t), fma(t, fma(t, 6.0, -15.0), 10.0), 1.0);
}
__device__ __forceinline__ double switch_dS(double t, double inv_w) {
  const double u = 1.0 - t, tu = t * u;
  return (-30.0 * inv_w) * (tu * tu);
}

// cubic Hermite from NODE data (embedding function only: once per atom)
__device__ __forceinline__ void hermite_nodes(const double *__restrict__ val, const double *__restrict__ der, int n, double h,
                                              double inv_h, double x, double &H, double &dH) {
  const double u = x * inv_h;
  int k = (int)u;
  k = max(0, min(k, n - 2));
  const double t = u - (double)k;
  const double y0 = __ldg(val + k), y1 = __ldg(val + k + 1), d0 = h * __ldg(der + k), d1 = h * __ldg(der + k + 1);
  const double D = y1 - y0;
  const double c2 = 3.0 * D - (2.0 * d0 + d1);
  const double c3 = (d0 + d1) - 2.0 * D;
  H = y0 + t * (d0 + t * (c2 + t * c3));
  dH = (d0 + t * (2.0 * c2 + 3.0 * t * c3)) * inv_h;
}

__device__ __forceinline__ double4 ldg4(const double4 *p) {
  const double2 a = __ldg((const double2 *)p), b = __ldg((const double2 *)p + 1);
  return make_double4(a.x, a.y, b.x, b.y);
}

// interval index and fractional coordinate on the r grid
__device__ __forceinline__ int table_index(const TableParams &tp, double r, double &t) {
  const double u = r * tp.inv_dr;
  const int k = max(0, min(__double2int_rz(u), tp.nr - 2));
  t = u - (double)k;
  return k;
}

template <int KIND>
__device__ __forceinline__ void embed(const DevSys &s, int ti, double rho, double &F, double &Fp) {
  if (KIND == MD_POT_TBSMA) {
    if (rho > 0.0) { const double sq = sqrt(rho); F = -sq; Fp = -0.5 / sq; }
    else { F = 0.0; Fp = (rho == rho) ? 0.0 : rho; }           // NaN propagates so that it is flagged
  } else {
    const TableParams &t = s.tab;
    const double *val = t.F_val + (size_t)ti * t.nrho, *der = t.F_der + (size_t)ti * t.nrho;
    if (rho >= t.rho_max) {
      Fp = der[t.nrho - 1];
      F = val[t.nrho - 1] + Fp * (rho - t.rho_max);
    } else {
      hermite_nodes(val, der, t.nrho, t.drho, t.inv_drho, rho, F, Fp);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// list row walkers.  Row of the atom in (tile, lane): entry k at row[k*32].  Entries 0 .. n_in-1 were inside
// r_c at build time ("main"), entries cap-n_out .. cap-1 were in the skin ("tail").  Both walkers keep the
// entry of pair k+2 and the gathered position of pair k+1 in flight while pair k is evaluated.
// ------------------------------------------------------------------------------------------------
template <class Body>
__device__ __forceinline__ void walk_main(const unsigned *__restrict__ row, int n, const double4 *__restrict__ pos, Body body) {
  unsigned e_nx = n > 0 ? row[0] : 0u;
  unsigned e_n2 = n > 1 ? row[32] : 0u;
  double4 p_nx = pos[e_nx & kIdxMask];
  for (int k = 0; k < n; ++k) {
    const unsigned e = e_nx;
    const double4 pj = p_nx;
    e_nx = e_n2;
    p_nx = pos[e_nx & kIdxMask];                               // slot 0 when there is no next pair: harmless
    e_n2 = (k + 2 < n) ? row[(size_t)(k + 2) * 32] : 0u;
    body(e, pj);
  }
}

// m = warp-uniform trip count (max of n over the warp); body(e, pj, active) is called by all 32 lanes
template <class Body>
__device__ __forceinline__ void walk_tail(const unsigned *__restrict__ row, int n, int m, const double4 *__restrict__ pos, Body body) {
  unsigned e_nx = n > 0 ? row[0] : 0u;
  unsigned e_n2 = n > 1 ? row[32] : 0u;
  double4 p_nx = pos[e_nx & kIdxMask];
  for (int k = 0; k < m; ++k) {
    const unsigned e = e_nx;
    const double4 pj = p_nx;
    e_nx = e_n2;
    p_nx = pos[e_nx & kIdxMask];
    e_n2 = (k + 2 < n) ? row[(size_t)(k + 2) * 32] : 0u;
    body(e, pj, k < n);
  }
}

struct AtomRow { const unsigned *main, *tail; int n_in, n_out; };

__device__ __forceinline__ AtomRow atom_row(const DevSys &s, int box, int local, int i, bool valid) {
  AtomRow r;
  const size_t tile = (size_t)box * s.tiles_per_box + (local >> 5);
  r.main = s.nbr + tile * s.cap * 32 + (local & 31);
  const int c = valid ? s.ncount[i] : 0;
  r.n_in = c & 0xffff; r.n_out = c >> 16;
  r.tail = r.main + (size_t)(s.cap - r.n_out) * 32;
  return r;
}

__device__ __forceinline__ void stage_exp_table(const DevSys &s, double *tab) {
  if (threadIdx.x < 64) tab[threadIdx.x] = s.exp_tab[threadIdx.x];
  __syncthreads();
}

// ------------------------------------------------------------------------------------------------
// Density pass: rho_i = sum_{j in list, r2 < rc2} rho(r_ij); F(rho_i), F'(rho_i).
// ------------------------------------------------------------------------------------------------
template <int KIND, bool FOLD>
__device__ __forceinline__ double density_term(const DevSys &s, const double *tab, int tp, double r2) {
  const double r = r2 * rsqrt_fast(r2);
  if (KIND == MD_POT_TBSMA) {
    const TbsmaParams &tb = s.tb;
    const double S = switch_S(switch_t(r, tb));
    double e = exp_tab(fma(-tb.b_rho[tp], r, tb.a_rho[tp]), tab);
    if (!FOLD) e *= tb.pre_rho[tp];
    return e * S;
  } else {
    double t;
    const int k = table_index(s.tab, r, t);
    const double4 c = ldg4(s.tab.f_c + (size_t)tp * (s.tab.nr - 1) + k);
    return fma(t, fma(t, fma(t, c.w, c.z), c.y), c.x);
  }
}

template <int KIND, bool MULTI, bool FOLD>
__global__ void __launch_bounds__(kForceBlock) k_density(const __grid_constant__ DevSys s) {
  __shared__ double tab[64];
  if (KIND == MD_POT_TBSMA) stage_exp_table(s, tab);
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  const bool valid = local < s.npb;
  const int i = box * s.npb + (valid ? local : 0);
  const AtomRow row = atom_row(s, box, local, i, valid);
  const double4 pi = s.pos[i];
  const int ti = MULTI ? (int)pi.w : 0;
  double rho = 0.0;

  // main part: branch-free.  TB-SMA: the clamped switch makes a pair beyond r_c contribute exactly 0;
  // tables (no switch, reading A9): the strict test r2 < rc2 selects the term.
  walk_main(row.main, row.n_in, s.pos, [&](unsigned e, const double4 &pj) {
    double dx, dy, dz;
    const double r2 = pair_r2(pj, pi, e, s, dx, dy, dz);
    const int tp = MULTI ? ti * s.nt + (int)pj.w : 0;
    const double term = density_term<KIND, FOLD>(s, tab, tp, r2);
    if (KIND == MD_POT_TBSMA) rho += term;
    else rho += (r2 < s.rc2) ? term : 0.0;
  });

  // skin part: distance test only; a pair found inside r_c is parked (one slot per lane) and the warp evaluates
  // the parked pairs together when some lane needs its slot again, and once at the end
  const int m = __reduce_max_sync(0xffffffffu, row.n_out);
  double park_r2 = 0.0; int park_tp = 0; bool parked = false;
  walk_tail(row.tail, row.n_out, m, s.pos, [&](unsigned e, const double4 &pj, bool active) {
    double dx, dy, dz;
    const double r2 = pair_r2(pj, pi, e, s, dx, dy, dz);
    const bool hit = active && r2 < s.rc2;
    if (__any_sync(0xffffffffu, hit && parked)) {
      if (parked) { rho += density_term<KIND, FOLD>(s, tab, park_tp, park_r2); parked = false; }
    }
    if (hit) { park_r2 = r2; park_tp = MULTI ? ti * s.nt + (int)pj.w : 0; parked = true; }
  });
  if (__any_sync(0xffffffffu, parked)) {
    if (parked) rho += density_term<KIND, FOLD>(s, tab, park_tp, park_r2);
  }

  if (!valid) return;
  double F, Fp;
  embed<KIND>(s, ti, rho, F, Fp);
  if (!(fabs(Fp) <= 1.79e308) || !(fabs(rho) <= 1.79e308)) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);   // r = 0 or overflow
  s.rho[i] = rho;
  s.eemb[i] = F;
  s.posf[i] = make_double4(pi.x, pi.y, pi.z, Fp);
}

// ------------------------------------------------------------------------------------------------
// Force pass: f_i = sum_j s_ij d/r, s_ij = V'(r) + (F'_i + F'_j) rho'(r), d = x_j - x_i   [eq.(3)]
// OBS: also E_i = F(rho_i) + 1/2 sum_j V(r) [eq.(1)] and W^{ab} = -1/2 sum_j s_ij d^a d^b / r.
// kick.h[type] != 0: second half-kick v += (dt/2m) f fused into the epilogue.
// ------------------------------------------------------------------------------------------------
struct KickParams { double h[MD_MAX_TYPES]; };

template <bool OBS> struct ForceAcc;
template <> struct ForceAcc<false> { double fx = 0.0, fy = 0.0, fz = 0.0; };
template <> struct ForceAcc<true> { double fx = 0.0, fy = 0.0, fz = 0.0, ev = 0.0, w0 = 0.0, w1 = 0.0, w2 = 0.0, w3 = 0.0, w4 = 0.0, w5 = 0.0; };

// g = s_ij / r and V for one pair; `in` = the pair is inside r_c (only consulted for the tables)
template <int KIND, bool OBS, bool FOLD>
__device__ __forceinline__ void force_term(const DevSys &s, const double *tab, int tp, double r2, double fp_sum, double &g, double &V) {
  const double rinv = rsqrt_fast(r2), r = r2 * rinv;
  if (KIND == MD_POT_TBSMA) {
    const TbsmaParams &tb = s.tb;
    const double t = switch_t(r, tb);
    const double S = switch_S(t), dS = switch_dS(t, tb.inv_w);
    double eh = exp_tab(fma(-tb.b_rho[tp], r, tb.a_rho[tp]), tab);
    double er = exp_tab(fma(-tb.b_rep[tp], r, tb.a_rep[tp]), tab);
    if (!FOLD) { eh *= tb.pre_rho[tp]; er *= tb.pre_rep[tp]; }
    const double df = eh * fma(-tb.b_rho[tp], S, dS);
    const double dV = er * fma(-tb.b_rep[tp], S, dS);
    g = fma(fp_sum, df, dV) * rinv;
    if (OBS) V = er * S;
  } else {
    double t;
    const int k = table_index(s.tab, r, t);
    const size_t o = (size_t)tp * (s.tab.nr - 1) + k;
    const double4 cf = ldg4(s.tab.der_c + 2 * o), cp = ldg4(s.tab.der_c + 2 * o + 1);
    const double df = fma(t, fma(t, cf.z, cf.y), cf.x);
    const double dV = fma(t, fma(t, cp.z, cp.y), cp.x);
    g = fma(fp_sum, df, dV) * rinv;
    if (OBS) { const double4 c = ldg4(s.tab.phi_c + o); V = fma(t, fma(t, fma(t, c.w, c.z), c.y), c.x); }
  }
}

template <bool OBS>
__device__ __forceinline__ void force_accumulate(ForceAcc<OBS> &a, double g, double V, double dx, double dy, double dz) {
  a.fx = fma(g, dx, a.fx); a.fy = fma(g, dy, a.fy); a.fz = fma(g, dz, a.fz);
  if constexpr (OBS) {
    a.ev += V;
    const double gx = g * dx, gy = g * dy;
    a.w0 = fma(-gx, dx, a.w0); a.w1 = fma(-gy, dy, a.w1); a.w2 = fma(-(g * dz), dz, a.w2);
    a.w3 = fma(-gx, dy, a.w3); a.w4 = fma(-gx, dz, a.w4); a.w5 = fma(-gy, dz, a.w5);
  }
}

template <int KIND, bool MULTI, bool OBS, bool FOLD>
__global__ void __launch_bounds__(kForceBlock) k_force(const __grid_constant__ DevSys s, const KickParams kick) {
  __shared__ double tab[64];
  __shared__ double sm[kForceBlock / 32][8];
  if (KIND == MD_POT_TBSMA) stage_exp_table(s, tab);
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  const bool valid = local < s.npb;
  const int i = box * s.npb + (valid ? local : 0);
  const AtomRow row = atom_row(s, box, local, i, valid);
  const double4 pi = s.posf[i];
  const int ti = MULTI ? s.type[i] : 0;
  ForceAcc<OBS> acc;

  walk_main(row.main, row.n_in, s.posf, [&](unsigned e, const double4 &pj) {
    double dx, dy, dz, g, V = 0.0;
    const double r2 = pair_r2(pj, pi, e, s, dx, dy, dz);
    const int tp = MULTI ? ti * s.nt + s.type[e & kIdxMask] : 0;
    force_term<KIND, OBS, FOLD>(s, tab, tp, r2, pi.w + pj.w, g, V);
    if (KIND != MD_POT_TBSMA && !(r2 < s.rc2)) { g = 0.0; V = 0.0; }   // tables: strict cut-off, no switch (reading A9)
    force_accumulate<OBS>(acc, g, V, dx, dy, dz);
  });

  const int m = __reduce_max_sync(0xffffffffu, row.n_out);
  double pk_dx = 0.0, pk_dy = 0.0, pk_dz = 0.0, pk_r2 = 1.0, pk_fp = 0.0; int pk_tp = 0; bool parked = false;
  auto flush = [&]() {
    double g, V = 0.0;
    force_term<KIND, OBS, FOLD>(s, tab, pk_tp, pk_r2, pk_fp, g, V);
    force_accumulate<OBS>(acc, g, V, pk_dx, pk_dy, pk_dz);
    parked = false;
  };
  walk_tail(row.tail, row.n_out, m, s.posf, [&](unsigned e, const double4 &pj, bool active) {
    double dx, dy, dz;
    const double r2 = pair_r2(pj, pi, e, s, dx, dy, dz);
    const bool hit = active && r2 < s.rc2;
    if (__any_sync(0xffffffffu, hit && parked)) {
      if (parked) flush();
    }
    if (hit) {
      pk_dx = dx; pk_dy = dy; pk_dz = dz; pk_r2 = r2; pk_fp = pi.w + pj.w;
      pk_tp = MULTI ? ti * s.nt + s.type[e & kIdxMask] : 0;
      parked = true;
    }
  });
  if (__any_sync(0xffffffffu, parked)) {
    if (parked) flush();
  }

  if (valid) {
    const size_t N = (size_t)s.N;
    s.frc[i] = acc.fx; s.frc[N + i] = acc.fy; s.frc[2 * N + i] = acc.fz;
    const double h = kick.h[ti];
    if (h != 0.0) { s.vel[i] += h * acc.fx; s.vel[N + i] += h * acc.fy; s.vel[2 * N + i] += h * acc.fz; }
    if (!(fabs(acc.fx) + fabs(acc.fy) + fabs(acc.fz) <= 1.79e308)) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
  }
  if constexpr (OBS) {
    double e_i = 0.0;
    if (valid) { e_i = s.eemb[i] + 0.5 * acc.ev; s.eatom[i] = e_i; }
    // warp-shuffle reduction (fixed butterfly order => deterministic), then across the 4 warps
    double v[7] = {e_i, 0.5 * acc.w0, 0.5 * acc.w1, 0.5 * acc.w2, 0.5 * acc.w3, 0.5 * acc.w4, 0.5 * acc.w5};
    if (!valid) {
#pragma unroll
      for (int c = 0; c < 7; ++c) v[c] = 0.0;
    }
#pragma unroll
    for (int c = 0; c < 7; ++c)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0)
#pragma unroll
      for (int c = 0; c < 7; ++c) sm[wid][c] = v[c];
    __syncthreads();
    if (threadIdx.x < 7) {
      double a = 0.0;
#pragma unroll
      for (int w = 0; w < kForceBlock / 32; ++w) a += sm[w][threadIdx.x];
      s.partial[(size_t)blockIdx.x * 8 + threadIdx.x] = a;
    }
  }
}

// per box: sum the block partials in a fixed order
__global__ void __launch_bounds__(256) k_reduce_boxes(const __grid_constant__ DevSys s, int bpb) {
  __shared__ double sm[256];
  const int box = blockIdx.x;
  for (int c = 0; c < 7; ++c) {
    double a = 0.0;
    for (int b = threadIdx.x; b < bpb; b += 256) a += s.partial[((size_t)box * bpb + b) * 8 + c];
    sm[threadIdx.x] = a;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
      __syncthreads();
    }
    if (threadIdx.x == 0) {
      if (c == 0) s.box_epot[box] = sm[0]; else s.box_virial[box * 6 + c - 1] = sm[0];
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------------
// md_create: node data -> per-interval polynomial coefficients (TableParams); one thread per (type pair, interval)
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double4 hermite_coeffs(const double *__restrict__ val, const double *__restrict__ der, int k, double h) {
  const double y0 = val[k], y1 = val[k + 1], d0 = __dmul_rn(h, der[k]), d1 = __dmul_rn(h, der[k + 1]);
  const double D = __dsub_rn(y1, y0);
  const double c2 = __dsub_rn(__dmul_rn(3.0, D), __dadd_rn(__dmul_rn(2.0, d0), d1));
  const double c3 = __dsub_rn(__dadd_rn(d0, d1), __dmul_rn(2.0, D));
  return make_double4(y0, d0, c2, c3);
}

__global__ void k_prepare_tables(const __grid_constant__ DevSys s, double4 *f_c, double4 *phi_c, double4 *der_c) {
  const int per = s.tab.nr - 1;
  const size_t g = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (g >= (size_t)s.nt * s.nt * per) return;
  const int tp = (int)(g / per), k = (int)(g - (size_t)tp * per);
  const size_t off = (size_t)tp * s.tab.nr;
  const double4 cf = hermite_coeffs(s.tab.f_val + off, s.tab.f_der + off, k, s.tab.dr);
  const double4 cp = hermite_coeffs(s.tab.phi_val + off, s.tab.phi_der + off, k, s.tab.dr);
  const double ih = s.tab.inv_dr;
  f_c[g] = cf;
  phi_c[g] = cp;
  der_c[2 * g] = make_double4(cf.y * ih, 2.0 * cf.z * ih, 3.0 * cf.w * ih, 0.0);
  der_c[2 * g + 1] = make_double4(cp.y * ih, 2.0 * cp.z * ih, 3.0 * cp.w * ih, 0.0);
}

int launch_prepare_tables(md_system *sys) {
  const DevSys &d = sys->d;
  const size_t n = (size_t)d.nt * d.nt * (d.tab.nr - 1);
  ++sys->launches, k_prepare_tables<<<(unsigned)((n + 255) / 256), 256, 0, sys->stream>>>(d, (double4 *)d.tab.f_c, (double4 *)d.tab.phi_c,
                                                                                          (double4 *)d.tab.der_c);
  return (int)cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------------
template <int KIND, bool FOLD>
static void launch_density_k(md_system *sys, int grid) {
  if (sys->d.nt > 1) ++sys->launches, k_density<KIND, true, FOLD><<<grid, kForceBlock, 0, sys->stream>>>(sys->d);
  else ++sys->launches, k_density<KIND, false, FOLD><<<grid, kForceBlock, 0, sys->stream>>>(sys->d);
}

int launch_density(md_system *sys) {
  ProfScope p(sys, MD_K_DENSITY);
  const int grid = sys->d.nb * blocks_per_box(sys->d.npb, kForceBlock);
  if (sys->d.kind == MD_POT_TBSMA) {
    if (sys->d.tb.fold) launch_density_k<MD_POT_TBSMA, true>(sys, grid);
    else launch_density_k<MD_POT_TBSMA, false>(sys, grid);
  } else launch_density_k<MD_POT_EAM_TABLE, true>(sys, grid);
  return (int)cudaGetLastError();
}

template <int KIND, bool FOLD>
static void launch_force_k(md_system *sys, int grid, bool obs, const KickParams &kp) {
  const bool multi = sys->d.nt > 1;
  cudaStream_t st = sys->stream;
  ++sys->launches;
  if (multi) {
    if (obs) k_force<KIND, true, true, FOLD><<<grid, kForceBlock, 0, st>>>(sys->d, kp);
    else k_force<KIND, true, false, FOLD><<<grid, kForceBlock, 0, st>>>(sys->d, kp);
  } else {
    if (obs) k_force<KIND, false, true, FOLD><<<grid, kForceBlock, 0, st>>>(sys->d, kp);
    else k_force<KIND, false, false, FOLD><<<grid, kForceBlock, 0, st>>>(sys->d, kp);
  }
}

int launch_force(md_system *sys, bool observables, double half_dt) {
  KickParams kp;
  for (int t = 0; t < MD_MAX_TYPES; ++t) kp.h[t] = (t < sys->d.nt) ? half_dt / sys->mass_ev[t] : 0.0;
  const int grid = sys->d.nb * blocks_per_box(sys->d.npb, kForceBlock);
  {
    ProfScope p(sys, MD_K_FORCE);
    if (sys->d.kind == MD_POT_TBSMA) {
      if (sys->d.tb.fold) launch_force_k<MD_POT_TBSMA, true>(sys, grid, observables, kp);
      else launch_force_k<MD_POT_TBSMA, false>(sys, grid, observables, kp);
    } else launch_force_k<MD_POT_EAM_TABLE, true>(sys, grid, observables, kp);
  }
  if (observables) {
    ProfScope p(sys, MD_K_REDUCE);
    ++sys->launches, k_reduce_boxes<<<sys->d.nb, 256, 0, sys->stream>>>(sys->d, blocks_per_box(sys->d.npb, kForceBlock));
  }
  return (int)cudaGetLastError();
}

}  // namespace md
