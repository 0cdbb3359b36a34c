// md_force.cu — density pass (paper's G18, Fig.5) and force pass with
// energy and virial (paper's G22, Fig.6), FP64; one thread per atom, or 4 / 8 / 32 lanes per
// atom for small systems (k_*_sub); optionally as Newton's-third-law passes (HALF).
// Inside md_step the force pass also performs both half-kicks, the next step's drift and the displacement check, and
// its last block takes the rebuild decision (force_finish, finish_displacement).
//
// Differences from the paper's kernels:
//  - atoms are in cell order and the list is a blocked-ELL array in 16-byte groups of four entries, so one LDG.128
//    brings four pairs and the neighbour gathers (one 256-bit load each) hit L1/L2;
//  - the periodic image of each listed pair is recorded at build time, so there is no min/max logic in
//    the inner loop;
//  - pairs that were inside r_c at build time come first in every row: that part of the loop is branch-free
//    (the switch function is clamped, so a pair that has drifted out contributes exactly 0) and evaluates two pairs
//    per step; the skin pairs behind them only get the distance test, and the few that have drifted inside r_c are
//    parked and evaluated together, so a warp does not run the heavy body for one lane at a time;
//  - r and 1/r come from one MUFU.RSQ64H seed + one cubic Newton step; exp() has no slow path (its argument
//    is bounded): 2^(j/64) table + degree-5 polynomial in the force pass, conflict-free 2^(j/16) table + degree-7
//    polynomial in the L1-bound density pass;
//  - F'(rho_j) travels in the w component of the gathered position (one 32-byte sector per neighbour);
//  - energy and virial are reduced by warp shuffles into per-block partials and a second deterministic
//    pass, instead of shared-memory partials summed on the host.
// What bounds these kernels on B200, and what was tried: DESIGN.md section 6.
#include "md_internal.cuh"

namespace md {

#ifndef MD_FORCE_MINB
#define MD_FORCE_MINB 5
#endif
#ifndef MD_DENS_MINB
#define MD_DENS_MINB 6
#endif
constexpr int kForceMinBlocks = MD_FORCE_MINB, kDensityMinBlocks = MD_DENS_MINB;

// ------------------------------------------------------------------------------------------------
// arithmetic helpers
// ------------------------------------------------------------------------------------------------

// d = (x_j - x_i) with the image recorded at build time: code 0: none, 1: +L, 2: -L.
__device__ __forceinline__ double image_delta(double xj, double xi, unsigned code, double L) {
  // branch-free: d + (-L) is bit-identical to d - L and d + 0.0 to d (up to the sign of a zero)
  const double shift = (code & 1u) ? L : ((code & 2u) ? -L : 0.0);
  return __dadd_rn(__dsub_rn(xj, xi), shift);
}

// CANON: r2 = (dx*dx + dy*dy) + dz*dz with every operation rounded once (reading A3), needed where r2 < rc2 decides a
// discontinuous term (tables, reading A9).  Otherwise (TB-SMA: the clamped switch makes the term continuous and exactly 0
// beyond r_c) two of the five operations are contracted into FMAs.
// DYN: the box edges are device state (a barostat is or was on); otherwise they are kernel parameters
template <bool CANON, bool DYN = true>
__device__ __forceinline__ double pair_r2(const double4 &pj, const double4 &pi, unsigned e, const DevSys &s,
                                          double &dx, double &dy, double &dz) {
  const unsigned code = e >> kIdxBits;
  if (code == 0) {
    dx = __dsub_rn(pj.x, pi.x); dy = __dsub_rn(pj.y, pi.y); dz = __dsub_rn(pj.z, pi.z);
  } else {
    dx = image_delta(pj.x, pi.x, code & 3u, DYN ? s.st->box[0] : s.L0[0]);
    dy = image_delta(pj.y, pi.y, (code >> 2) & 3u, DYN ? s.st->box[1] : s.L0[1]);
    dz = image_delta(pj.z, pi.z, (code >> 4) & 3u, DYN ? s.st->box[2] : s.L0[2]);
  }
  if (CANON) return __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
  return fma(dz, dz, fma(dy, dy, dx * dx));
}

// An FP64 instruction takes at most ONE operand that is not a register (an immediate with a zero low word, or a
// constant-bank address).  Constants that meet another constant in the same FMA are therefore read from MEMORY into
// registers before the loop (LoopConsts): ptxas cannot rematerialise a global load, so they stay in registers instead
// of being rebuilt by MOV / LDC pairs for every pair.  The others sit in the constant bank and are used in place.
__constant__ double kLn2_64 = 0x1.62e42fefa39efp-7;           // ln2/64
__constant__ double kC3 = 1.0 / 6.0, kC4 = 1.0 / 24.0, kC5 = 1.0 / 120.0, kC6 = 1.0 / 720.0;
__constant__ double kLn2_16 = 0x1.62e42fefa39efp-5;           // ln2/16

struct LoopConsts { double c5, c375, six, inv_w, bk_rho, bk_rep, c7, bk16_rho; };

__device__ __forceinline__ double lds_opaque(unsigned addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ LoopConsts load_loop_consts(unsigned tab) {   // tab = shared-space address of the staged exp_tab
  LoopConsts c;
  c.c5 = lds_opaque(tab + 512); c.c375 = lds_opaque(tab + 520); c.six = lds_opaque(tab + 528);
  c.inv_w = lds_opaque(tab + 536); c.bk_rho = lds_opaque(tab + 544); c.bk_rep = lds_opaque(tab + 552);
  c.c7 = lds_opaque(tab + 560); c.bk16_rho = lds_opaque(tab + 568);
  return c;
}

// 1/sqrt(x), x > 0 finite and normal: hardware seed (relative error ~2^-22) and one cubic Newton step
//   y1 = y (1 + e/2 + 3 e^2/8),  e = 1 - x y^2        (relative error 2.5 delta^3 ~ 2^-64 plus rounding)
__device__ __forceinline__ double rsqrt_fast(double x, double c375) {
  double y;
  asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
  const double e = fma(-x, y * y, 1.0);
  const double p = fma(e, c375, 0.5);
  return fma(p, y * e, y);
}

// exp(xk ln2/64) for |xk ln2/64| < 690, no special cases; xk is the exponent in units of ln2/64.
// n = rint(xk) (magic-number rounding); d = xk - n exactly, |d| <= 1/2; r = d ln2/64, |r| <= 0.00542;
// result = 2^(n >> 6) tab[n & 63] (1 + r + r^2/2 + r^3/6 + r^4/24 + r^5/120); remainder r^6/720 < 3.5e-17.
__device__ __forceinline__ double exp_scaled(double xk, unsigned tab, double c5) {   // tab = shared-space address of the table
  constexpr double kMagic = 6755399441055744.0;                 // 1.5 * 2^52: the low word of t holds n
  const double t = xk + kMagic;
  const double n = t - kMagic;
  const double r = (xk - n) * kLn2_64;
  const int ni = __double2loint(t);
  double T;
  asm("ld.shared.f64 %0, [%1];" : "=d"(T) : "r"(tab + ((unsigned)(ni & 63) << 3)));
  double p = fma(r, c5, kC4);
  p = fma(p, r, kC3);
  p = fma(p, r, 0.5);
  p = fma(p * r, r, r);
  const double v = fma(T, p, T);
  return __hiloint2double(__double2hiint(v) + ((ni >> 6) << 20), __double2loint(v));
}

// The same arithmetic for NP pairs at once, written step by step across the pairs: ptxas keeps roughly the source order,
// so the NP dependency chains end up interleaved in the instruction stream (rsqrt_fast / exp_scaled / switch_* above
// are the single-pair forms of exactly these steps).
#define MD_EACH for (int q = 0; q < NP; ++q)
template <int NP>
__device__ __forceinline__ void rsqrt_fast_n(const double (&x)[NP], double c375, double (&y)[NP]) {
  double e[NP], p[NP], ye[NP];
#pragma unroll
  MD_EACH asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y[q]) : "d"(x[q]));
#pragma unroll
  MD_EACH e[q] = y[q] * y[q];
#pragma unroll
  MD_EACH e[q] = fma(-x[q], e[q], 1.0);
#pragma unroll
  MD_EACH p[q] = fma(e[q], c375, 0.5);
#pragma unroll
  MD_EACH ye[q] = y[q] * e[q];
#pragma unroll
  MD_EACH y[q] = fma(p[q], ye[q], y[q]);
}

template <int NP>
__device__ __forceinline__ void exp_scaled_n(const double (&xk)[NP], unsigned tab, double c5, double (&out)[NP]) {
  constexpr double kMagic = 6755399441055744.0;
  double t[NP], n[NP], r[NP], T[NP], p[NP];
  int ni[NP];
#pragma unroll
  MD_EACH t[q] = xk[q] + kMagic;
#pragma unroll
  MD_EACH { n[q] = t[q] - kMagic; ni[q] = __double2loint(t[q]); }
#pragma unroll
  MD_EACH {
    asm("ld.shared.f64 %0, [%1];" : "=d"(T[q]) : "r"(tab + ((unsigned)(ni[q] & 63) << 3)));
  }
#pragma unroll
  MD_EACH r[q] = (xk[q] - n[q]) * kLn2_64;
#pragma unroll
  MD_EACH p[q] = fma(r[q], c5, kC4);
#pragma unroll
  MD_EACH p[q] = fma(p[q], r[q], kC3);
#pragma unroll
  MD_EACH p[q] = fma(p[q], r[q], 0.5);
#pragma unroll
  MD_EACH p[q] = fma(p[q] * r[q], r[q], r[q]);
#pragma unroll
  MD_EACH {
    const double v = fma(T[q], p[q], T[q]);
    out[q] = __hiloint2double(__double2hiint(v) + ((ni[q] >> 6) << 20), __double2loint(v));
  }
}

// The density pass is bound by the L1 data pipe, where a 64-entry look-up at random indices costs ~5 wavefronts (bank
// conflicts).  Its exp therefore uses a 16-entry table 2^(j/16): 16 entries lie in 16 distinct bank pairs, so the
// look-up is conflict-free (2 wavefronts), and the polynomial goes to degree 7: |r| <= ln2/32, r^8/40320 < 1.3e-18.
// xk is the exponent in units of ln2/16; tab16 = shared-space address of the 16-entry table; c7 = 1/5040 in a register.
__device__ __forceinline__ double exp_scaled16(double xk, unsigned tab16, double c7) {
  constexpr double kMagic = 6755399441055744.0;
  const double t = xk + kMagic;
  const double n = t - kMagic;
  const double r = (xk - n) * kLn2_16;
  const int ni = __double2loint(t);
  double T;
  asm("ld.shared.f64 %0, [%1];" : "=d"(T) : "r"(tab16 + ((unsigned)(ni & 15) << 3)));
  double p = fma(r, c7, kC6);
  p = fma(p, r, kC5);
  p = fma(p, r, kC4);
  p = fma(p, r, kC3);
  p = fma(p, r, 0.5);
  p = fma(p * r, r, r);
  const double v = fma(T, p, T);
  return __hiloint2double(__double2hiint(v) + ((ni >> 4) << 20), __double2loint(v));
}

template <int NP>
__device__ __forceinline__ void exp_scaled16_n(const double (&xk)[NP], unsigned tab16, double c7, double (&out)[NP]) {
  constexpr double kMagic = 6755399441055744.0;
  double t[NP], n[NP], r[NP], T[NP], p[NP];
  int ni[NP];
#pragma unroll
  MD_EACH t[q] = xk[q] + kMagic;
#pragma unroll
  MD_EACH { n[q] = t[q] - kMagic; ni[q] = __double2loint(t[q]); }
#pragma unroll
  MD_EACH asm("ld.shared.f64 %0, [%1];" : "=d"(T[q]) : "r"(tab16 + ((unsigned)(ni[q] & 15) << 3)));
#pragma unroll
  MD_EACH r[q] = (xk[q] - n[q]) * kLn2_16;
#pragma unroll
  MD_EACH p[q] = fma(r[q], c7, kC6);
#pragma unroll
  MD_EACH p[q] = fma(p[q], r[q], kC5);
#pragma unroll
  MD_EACH p[q] = fma(p[q], r[q], kC4);
#pragma unroll
  MD_EACH p[q] = fma(p[q], r[q], kC3);
#pragma unroll
  MD_EACH p[q] = fma(p[q], r[q], 0.5);
#pragma unroll
  MD_EACH p[q] = fma(p[q] * r[q], r[q], r[q]);
#pragma unroll
  MD_EACH {
    const double v = fma(T[q], p[q], T[q]);
    out[q] = __hiloint2double(__double2hiint(v) + ((ni[q] >> 4) << 20), __double2loint(v));
  }
}

// quintic switch on t in [0,1]: S = 1 - t^3 (10 - 15 t + 6 t^2), dS/dr = -30 t^2 (1-t)^2 inv_w.
// switch_t clamps on the high word with integer min/max (no FP64-pipe instruction): t <= 0 gives t = 0 (S = 1,
// dS = 0 exactly) and t >= 1 gives t = 1 (S = 0, dS = 0 exactly).
__device__ __forceinline__ double switch_t(double r, double inv_w, double t0) {
  const double t = fma(r, inv_w, t0);
  const int hi = __double2hiint(t);
  const int hc = min(max(hi, 0), 0x3ff00000);
  return __hiloint2double(hc, (unsigned)hi < 0x3ff00000u ? __double2loint(t) : 0);
}
__device__ __forceinline__ double switch_S(double t, double six) {
  const double t2 = t * t;
  return fma(-(t2 * t), fma(t, fma(t, six, -15.0), 10.0), 1.0);
}
__device__ __forceinline__ double switch_dS(double t, double m30_inv_w) {
  const double u = 1.0 - t, tu = t * u;
  return m30_inv_w * (tu * tu);
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

__device__ __forceinline__ double4 ldg4(const double4 *p) {       // one 256-bit load (LDG.E.256) on the read-only path
  double4 v;
  asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
  return v;
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
// list row walkers.  The row of the atom in (tile, lane) is a sequence of 16-byte groups of four entries, group g
// at row[g * 32] (uint4 units).  Entries 0 .. n_in-1 were inside r_c at build time ("main"), entries cap-n_out ..
// cap-1 were in the skin ("tail").
//
// Software pipeline.  prep(e, pj) turns a gathered neighbour into a PairD (d = x_j - x_i with its image, r2, w);
// eval2 / eval1 run the potential on one or two PairDs.  In the source, the gathers of pairs k+2, k+3 and the entries
// of the group after next are issued before pairs k, k+1 are evaluated; ptxas places them where it likes (it gives
// every global load of the loop ONE scoreboard and keeps the loads of a trip close to their first use; forcing them
// earlier through artificial address dependencies was measured and cost 3 %).
// ------------------------------------------------------------------------------------------------
struct PairD { double dx, dy, dz, r2, w; unsigned e; };

// the list is streamed once per pass: it is read past L1 (no allocation), so that L1 keeps the gathered positions
__device__ __forceinline__ uint4 ldg_group(const uint4 *p) {
  uint4 v;
  asm("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
#define MD_GIDX(e) ((e) & kIdxMask)

// One 256-bit load per gathered neighbour (LDG.E.256, sm_100) instead of two 128-bit loads.
__device__ __forceinline__ double4 gather32(const double4 *p) {
  double4 v;
  asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
  return v;
}
// base + 32 * idx with one 32 x 32 -> 64 bit multiply-add (the compiler's own sequence is shift, mask, add, add-with-carry)
__device__ __forceinline__ const double4 *slot_ptr(const double4 *base, unsigned idx) {
  unsigned long long a;
  asm("mad.wide.u32 %0, %1, 32, %2;" : "=l"(a) : "r"(idx), "l"((unsigned long long)base));
  return (const double4 *)a;
}

// Half passes (MD_OPT_HALF_LIST): the partner's share of a pair term, as a 64-bit integer reduction in units of 2^-43.
// The result of the atomic is not used, so it is a fire-and-forget RED.E.ADD.64; integer sums are order-independent.
__device__ __forceinline__ void red_fix(long long *p, double v) {
  const long long q = __double2ll_rn(v * kFixScale);
  if (q) atomicAdd(reinterpret_cast<unsigned long long *>(p), (unsigned long long)q);
}
__device__ __forceinline__ double fix_take(long long *p) {        // read a received sum and clear it for the next pass
  const long long q = *p;
  if (q) *p = 0;
  return (double)q * kFixInv;
}

// eval2 evaluates two pairs at once: their dependency chains are independent (measured on B200: one dependent DFMA
// chain per warp tops out at 64 % of the FP64 pipe, two at 77 %, four at 90 %).
template <class Prep, class Eval2, class Eval1>
__device__ __forceinline__ void walk_main(const uint4 *__restrict__ row, int n, const double4 *__restrict__ pos, Prep prep, Eval2 eval2,
                                          Eval1 eval1) {
  const uint4 none = make_uint4(0u, 0u, 0u, 0u);
  const int ng = (n + 3) >> 2, nfull = n >> 2;
  uint4 E = ng > 0 ? ldg_group(row) : none;
  double4 pA = gather32(slot_ptr(pos, MD_GIDX(E.x)));                      // slot 0 when there is no such pair: harmless
  double4 pB = gather32(slot_ptr(pos, MD_GIDX(E.y)));
  for (int g = 0; g < nfull; ++g) {
    const uint4 En = (g + 1 < ng) ? ldg_group(row + (size_t)(g + 1) * 32) : none;   // a whole trip (four pairs) ahead
    const PairD a = prep(E.x, pA), b = prep(E.y, pB);
    const double4 pC = gather32(slot_ptr(pos, MD_GIDX(E.z)));
    const double4 pD = gather32(slot_ptr(pos, MD_GIDX(E.w)));
    eval2(a, b);
    const PairD c = prep(E.z, pC), d = prep(E.w, pD);
    pA = gather32(slot_ptr(pos, MD_GIDX(En.x)));
    pB = gather32(slot_ptr(pos, MD_GIDX(En.y)));
    eval2(c, d);
    E = En;
  }
  const int rem = n & 3;                                          // the partly filled last group
  if (rem >= 2) {
    const PairD a = prep(E.x, pA), b = prep(E.y, pB);
    const double4 pC = gather32(slot_ptr(pos, MD_GIDX(E.z)));
    eval2(a, b);
    if (rem == 3) eval1(prep(E.z, pC));
  } else if (rem == 1) {
    eval1(prep(E.x, pA));
  }
}

// Tail: walked from the END of the row (entry cap-1-j, j = 0 .. n-1), so that every lane starts on a group boundary.
// last = the last group of the row; mg = warp-uniform number of groups (max over the warp of ceil(n/4));
// body(PairD, active) is called by all 32 lanes.
template <class Prep, class Body>
__device__ __forceinline__ void walk_tail(const uint4 *__restrict__ last, int n, int mg, const double4 *__restrict__ pos, Prep prep, Body body) {
  const uint4 none = make_uint4(0u, 0u, 0u, 0u);
  const int ng = (n + 3) >> 2;
  uint4 E = ng > 0 ? ldg_group(last) : none;
  double4 pA = gather32(slot_ptr(pos, MD_GIDX(E.w)));
  double4 pB = gather32(slot_ptr(pos, MD_GIDX(E.z)));
  for (int g = 0; g < mg; ++g) {
    const int j = g * 4;
    const uint4 En = (g + 1 < ng) ? ldg_group(last - (size_t)(g + 1) * 32) : none;
    const PairD a = prep(E.w, pA), b = prep(E.z, pB);
    const double4 pC = gather32(slot_ptr(pos, MD_GIDX(E.y)));
    const double4 pD = gather32(slot_ptr(pos, MD_GIDX(E.x)));
    body(a, j < n);
    body(b, j + 1 < n);
    const PairD c = prep(E.y, pC), d = prep(E.x, pD);
    pA = gather32(slot_ptr(pos, MD_GIDX(En.w)));
    pB = gather32(slot_ptr(pos, MD_GIDX(En.z)));
    body(c, j + 2 < n);
    body(d, j + 3 < n);
    E = En;
  }
}

struct AtomRow { const uint4 *main, *last; int n_in, n_out; };

__device__ __forceinline__ AtomRow atom_row(const DevSys &s, int box, int local, int i, bool valid) {
  AtomRow r;
  const size_t tile = (size_t)box * s.tiles_per_box + (local >> 5);
  r.main = (const uint4 *)(s.nbr + nbr_row_offset(tile, s.cap, local & 31));
  const int c = valid ? s.ncount[i] : 0;
  r.n_in = c & 0xffff; r.n_out = c >> 16;
  r.last = r.main + (size_t)((s.cap >> 2) - 1) * 32;
  return r;
}

__device__ __forceinline__ unsigned stage_exp_table(const DevSys &s, double *tab) {
  if (threadIdx.x < kExpTabLen && threadIdx.x != kExpAddrSlot) tab[threadIdx.x] = s.exp_tab[threadIdx.x];
  const unsigned a = (unsigned)__cvta_generic_to_shared(tab);
  if (threadIdx.x == kExpAddrSlot) reinterpret_cast<unsigned *>(tab + kExpAddrSlot)[0] = a;
  __syncthreads();
  // read the address back through an opaque load: ptxas would otherwise recompute it (S2UR + ULEA + MOV) at every use
  unsigned t;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(t) : "r"(a + 8u * kExpAddrSlot));
  return t;
}

// ------------------------------------------------------------------------------------------------
// Density pass: rho_i = sum_{j in list, r2 < rc2} rho(r_ij); F(rho_i), F'(rho_i).
// ------------------------------------------------------------------------------------------------
template <int KIND, bool MULTI, bool FOLD>
__device__ __forceinline__ double density_term(const DevSys &s, const LoopConsts &lc, unsigned tab, int tp, double r2) {
  if (KIND == MD_POT_TBSMA) {
    const TbsmaParams &tb = s.tb;
    const double r = r2 * rsqrt_fast(r2, lc.c375);
    const double S = switch_S(switch_t(r, MULTI ? tb.inv_w[tp] : lc.inv_w, tb.t0[tp]), lc.six);
    double e = exp_scaled16(fma(-(MULTI ? tb.bk16_rho[tp] : lc.bk16_rho), r, tb.ak16_rho[tp]), tab + 8u * kExp16Off, lc.c7);
    if (!FOLD) e *= tb.pre_rho[tp];
    return e * S;
  } else {
    const double r = r2 * rsqrt_fast(r2, 0.375);
    double t;
    const int k = table_index(s.tab, r, t);
    const double4 c = ldg4(s.tab.f_c + (size_t)tp * (s.tab.nr - 1) + k);
    return fma(t, fma(t, fma(t, c.w, c.z), c.y), c.x);
  }
}

template <bool FOLD, int NP>
__device__ __forceinline__ void density_term_n(const DevSys &s, const LoopConsts &lc, unsigned tab, const double (&r2)[NP], double (&term)[NP]) {
  const TbsmaParams &tb = s.tb;
  double rinv[NP], r[NP], t[NP], xh[NP], eh[NP];
  rsqrt_fast_n<NP>(r2, lc.c375, rinv);
#pragma unroll
  MD_EACH r[q] = r2[q] * rinv[q];
#pragma unroll
  MD_EACH { xh[q] = fma(-lc.bk16_rho, r[q], tb.ak16_rho[0]); t[q] = switch_t(r[q], lc.inv_w, tb.t0[0]); }
  exp_scaled16_n<NP>(xh, tab + 8u * kExp16Off, lc.c7, eh);
#pragma unroll
  MD_EACH {
    if (!FOLD) eh[q] *= tb.pre_rho[0];
    term[q] = eh[q] * switch_S(t[q], lc.six);
  }
}

template <int KIND, bool MULTI, bool FOLD, bool DYN, bool HALF = false>
__global__ void __launch_bounds__(kForceBlock, kDensityMinBlocks) k_density(const __grid_constant__ DevSys s, const int guard) {
  __shared__ double tab_sm[kExpTabLen];
  const bool go = step_guard(s, guard);
  // the atom's own loads are issued BEFORE the table staging and its barrier, so that their latency overlaps it
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  const bool valid = local < s.npb;
  const int i = box * s.npb + (valid ? local : 0);
  const AtomRow row = atom_row(s, box, local, i, valid);
  const double4 pi = s.pos[i];
  if (!go) return;
  unsigned tab = 0;
  LoopConsts lc = {};
  if (KIND == MD_POT_TBSMA) { tab = stage_exp_table(s, tab_sm); lc = load_loop_consts(tab); }
  const int ti = MULTI ? (int)pi.w : 0;
  double rho = 0.0, rho2 = 0.0;
  // HALF: only the pairs this atom owns (they come first in the row); the partner gets its share by red_fix
  const int own = HALF && valid ? s.nown[i] : 0;
  const int n_main = HALF ? (own & 0xffff) : row.n_in, n_tail = HALF ? (own >> 16) : row.n_out;

  // main part: branch-free.  TB-SMA: the clamped switch makes a pair beyond r_c contribute exactly 0;
  // tables (no switch, reading A9): the strict test r2 < rc2 selects the term.
  auto prep = [&](unsigned e, const double4 &pj) {
    PairD d;
    d.r2 = pair_r2<KIND != MD_POT_TBSMA, DYN>(pj, pi, e, s, d.dx, d.dy, d.dz);
    d.w = pj.w; d.e = e;
    return d;
  };
  auto term1 = [&](const PairD &d) {
    double term = density_term<KIND, MULTI, FOLD>(s, lc, tab, MULTI ? ti * s.nt + (int)d.w : 0, d.r2);
    term = (KIND == MD_POT_TBSMA || d.r2 < (MULTI ? s.rc2p[ti * s.nt + (int)d.w] : s.rc2)) ? term : 0.0;
    if (HALF) red_fix(s.rho_fix + MD_GIDX(d.e), term);              // rho^(ab) is symmetric in (a, b)
    return term;
  };
  walk_main(row.main, n_main, s.pos, prep,
            [&](const PairD &a, const PairD &b) {
              if constexpr (KIND == MD_POT_TBSMA && !MULTI) {
                const double r2v[2] = {a.r2, b.r2};
                double tv[2];
                density_term_n<FOLD, 2>(s, lc, tab, r2v, tv);
                rho += tv[0]; rho2 += tv[1];
                if (HALF) { red_fix(s.rho_fix + MD_GIDX(a.e), tv[0]); red_fix(s.rho_fix + MD_GIDX(b.e), tv[1]); }
              } else {
                rho += term1(a); rho2 += term1(b);
              }
            },
            [&](const PairD &a) { rho += term1(a); });
  rho += rho2;

  // skin part: distance test only; a pair found inside r_c is parked (one slot per lane) and the warp evaluates
  // the parked pairs together when some lane needs its slot again, and once at the end
  const int mg = (__reduce_max_sync(0xffffffffu, n_tail) + 3) >> 2;
  // only the ENTRY is parked (one register); the rare evaluation gathers and prepares the pair again
  unsigned park = 0u;
  bool parked = false;
  auto flush = [&]() { rho += term1(prep(park, gather32(slot_ptr(s.pos, MD_GIDX(park))))); parked = false; };
  walk_tail(row.last, n_tail, mg, s.pos, prep, [&](const PairD &d, bool active) {
    const bool hit = active && d.r2 < s.rc2;
    if (__any_sync(0xffffffffu, hit && parked)) {
      if (parked) flush();
    }
    if (hit) { park = d.e; parked = true; }
  });
  if (__any_sync(0xffffffffu, parked)) {
    if (parked) flush();
  }

  if (!valid) return;
  if (HALF) { s.rho[i] = rho; return; }                            // the owned part; k_embed adds what the partners sent
  double F, Fp;
  embed<KIND>(s, ti, rho, F, Fp);
  if (!(fabs(Fp) <= 1.79e308) || !(fabs(rho) <= 1.79e308)) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);   // r = 0 or overflow
  s.rho[i] = rho;
  s.eemb[i] = F;
  s.posf[i] = make_double4(pi.x, pi.y, pi.z, Fp);
}

// Second kernel of a half density pass: rho_i = owned part + received part; F(rho_i), F'(rho_i)
template <int KIND>
__global__ void __launch_bounds__(256) k_embed(const __grid_constant__ DevSys s, const int guard) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N || !step_guard(s, guard)) return;
  const double4 pi = s.pos[i];
  const double rho = s.rho[i] + fix_take(s.rho_fix + i);
  double F, Fp;
  embed<KIND>(s, s.nt > 1 ? (int)pi.w : 0, rho, F, Fp);
  if (!(fabs(Fp) <= 1.79e308) || !(fabs(rho) <= 1.79e308)) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
  s.rho[i] = rho;
  s.eemb[i] = F;
  s.posf[i] = make_double4(pi.x, pi.y, pi.z, Fp);
}

// ------------------------------------------------------------------------------------------------
// Force pass: f_i = sum_j s_ij d/r, s_ij = V'(r) + (F'_i + F'_j) rho'(r), d = x_j - x_i   [eq.(3)]
// OBS: also E_i = F(rho_i) + 1/2 sum_j V(r) [eq.(1)] and W^{ab} = -1/2 sum_j s_ij d^a d^b / r.
// kick.h[type] != 0: second half-kick v += (dt/2m) f fused into the epilogue.
// ------------------------------------------------------------------------------------------------

template <bool OBS> struct ForceAcc;
template <> struct ForceAcc<false> { double fx = 0.0, fy = 0.0, fz = 0.0; };
template <> struct ForceAcc<true> { double fx = 0.0, fy = 0.0, fz = 0.0, ev = 0.0, w0 = 0.0, w1 = 0.0, w2 = 0.0, w3 = 0.0, w4 = 0.0, w5 = 0.0; };

// g = s_ij / r and V for one pair; `in` = the pair is inside r_c (only consulted for the tables)
template <int KIND, bool MULTI, bool OBS, bool FOLD>
__device__ __forceinline__ void force_term(const DevSys &s, const LoopConsts &lc, unsigned tab, int tp, double r2, double fp_sum,
                                           double &g, double &V) {
  if (KIND == MD_POT_TBSMA) {
    const TbsmaParams &tb = s.tb;
    const double rinv = rsqrt_fast(r2, lc.c375), r = r2 * rinv;
    const double t = switch_t(r, MULTI ? tb.inv_w[tp] : lc.inv_w, tb.t0[tp]);
    const double S = switch_S(t, lc.six), dS = switch_dS(t, tb.m30_inv_w[tp]);
    double eh = exp_scaled(fma(-(MULTI ? tb.bk_rho[tp] : lc.bk_rho), r, tb.ak_rho[tp]), tab, lc.c5);
    double er = exp_scaled(fma(-(MULTI ? tb.bk_rep[tp] : lc.bk_rep), r, tb.ak_rep[tp]), tab, lc.c5);
    if (!FOLD) { eh *= tb.pre_rho[tp]; er *= tb.pre_rep[tp]; }
    const double df = eh * fma(-tb.b_rho[tp], S, dS);
    const double dV = er * fma(-tb.b_rep[tp], S, dS);
    g = fma(fp_sum, df, dV) * rinv;
    if (OBS) V = er * S;
  } else {
    const double rinv = rsqrt_fast(r2, 0.375), r = r2 * rinv;
    double t;
    const int k = table_index(s.tab, r, t);
    const size_t o = (size_t)tp * (s.tab.nr - 1) + k;
    // The derivative of the interpolant on interval k is the quadratic y'_k + a_k t + b_k t^2 with b_k = y'_{k+1} - y'_k - a_k
    // (the interpolant is C1: the quadratic ends at the next node's slope).  Records (y'_k of f, y'_k of phi, a_k of f,
    // a_k of phi), 32 bytes per interval: one 32-byte load here and the first 16 bytes of the next record, 48 bytes per
    // pair from a table of 32 bytes per interval.  Both count on B200 (L1 data pipe): padded 2 x 32-byte records of a
    // 64-byte-per-interval table 2.25 ms, 48 bytes of a 48-byte table 1.75 ms, 64 bytes of a 32-byte node table 1.92 ms
    // (force pass, 4.2 M atoms).
    const double4 *rec = s.tab.der_c + (size_t)tp * s.tab.nr + k;
    const double4 q = ldg4(rec);
    double2 n;
    asm("ld.global.nc.v2.f64 {%0,%1}, [%2];" : "=d"(n.x), "=d"(n.y) : "l"(rec + 1));
    const double df = fma(t, fma(t, (n.x - q.x) - q.z, q.z), q.x);
    const double dV = fma(t, fma(t, (n.y - q.y) - q.w, q.w), q.y);
    g = fma(fp_sum, df, dV) * rinv;
    if (OBS) { const double4 c = ldg4(s.tab.phi_c + o); V = fma(t, fma(t, fma(t, c.w, c.z), c.y), c.x); }
  }
}

// NP pairs at once (TB-SMA, one type pair): the steps of force_term, interleaved across the pairs
template <bool OBS, bool FOLD, int NP>
__device__ __forceinline__ void force_term_n(const DevSys &s, const LoopConsts &lc, unsigned tab, const double (&r2)[NP],
                                             const double (&fp_sum)[NP], double (&g)[NP], double (&V)[NP]) {
  const TbsmaParams &tb = s.tb;
  double rinv[NP], r[NP], t[NP], S[NP], dS[NP], xh[NP], xr[NP], eh[NP], er[NP];
  rsqrt_fast_n<NP>(r2, lc.c375, rinv);
#pragma unroll
  MD_EACH r[q] = r2[q] * rinv[q];
#pragma unroll
  MD_EACH { xh[q] = fma(-lc.bk_rho, r[q], tb.ak_rho[0]); xr[q] = fma(-lc.bk_rep, r[q], tb.ak_rep[0]); t[q] = switch_t(r[q], lc.inv_w, tb.t0[0]); }
  exp_scaled_n<NP>(xh, tab, lc.c5, eh);
  exp_scaled_n<NP>(xr, tab, lc.c5, er);
#pragma unroll
  MD_EACH { S[q] = switch_S(t[q], lc.six); dS[q] = switch_dS(t[q], tb.m30_inv_w[0]); }
#pragma unroll
  MD_EACH {
    if (!FOLD) { eh[q] *= tb.pre_rho[0]; er[q] *= tb.pre_rep[0]; }
    const double df = eh[q] * fma(-tb.b_rho[0], S[q], dS[q]);
    const double dV = er[q] * fma(-tb.b_rep[0], S[q], dS[q]);
    g[q] = fma(fp_sum[q], df, dV) * rinv[q];
    if (OBS) V[q] = er[q] * S[q];
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

template <bool OBS>
__device__ __forceinline__ void force_merge(ForceAcc<OBS> &a, const ForceAcc<OBS> &b) {
  a.fx += b.fx; a.fy += b.fy; a.fz += b.fz;
  if constexpr (OBS) { a.ev += b.ev; a.w0 += b.w0; a.w1 += b.w1; a.w2 += b.w2; a.w3 += b.w3; a.w4 += b.w4; a.w5 += b.w5; }
}

// Epilogue of the force pass, in three pieces (a half pass runs them in two kernels).
// (1) the atom: store the force, second half-kick, non-finite flag.  ctl.chain: the same thread goes on with the NEXT
// step's first half-kick and drift (the new position goes to `pos`, which this pass does not read: it gathers from
// `posf`), so that a step inside md_step costs two kernels (density, force) instead of four.
// Returns the squared displacement from x_ref after that drift (0 otherwise).
__device__ __forceinline__ double atom_update(const DevSys &s, const KickParams &kick, const StepCtl &ctl, int i, int ti, const double4 &pi,
                                              double fx, double fy, double fz) {
  const size_t N = (size_t)s.N;
  double d2 = 0.0;
  if (kick.h[ti] != 0.0) {
    // every load of the epilogue is issued before anything waits for one of them
    double vx = s.vel[i], vy = s.vel[N + i], vz = s.vel[2 * N + i];
    double rx = 0.0, ry = 0.0, rz = 0.0;
    if (ctl.chain) { rx = s.xref[i]; ry = s.xref[N + i]; rz = s.xref[2 * N + i]; }
    s.frc[i] = fx; s.frc[N + i] = fy; s.frc[2 * N + i] = fz;
    half_kick(kick, ti, fx, fy, fz, vx, vy, vz);
    if (ctl.chain) {
      half_kick(kick, ti, fx, fy, fz, vx, vy, vz);
      double4 x = make_double4(pi.x, pi.y, pi.z, (double)ti);
      d2 = drift_atom(ctl.dt, x, vx, vy, vz, rx, ry, rz);
      s.pos[i] = x;
    }
    s.vel[i] = vx; s.vel[N + i] = vy; s.vel[2 * N + i] = vz;
  } else {
    s.frc[i] = fx; s.frc[N + i] = fy; s.frc[2 * N + i] = fz;
  }
  if (!(fabs(fx) + fabs(fy) + fabs(fz) <= 1.79e308)) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
  return d2;
}

// (2) observables: components [C0, C1) of this block's partial sums (0: energy, 1..6: virial), by warp shuffles in a
// fixed butterfly order and then across the 4 warps (deterministic).  Called by every thread of the block.
template <int C0, int C1>
__device__ __forceinline__ void block_partials(const DevSys &s, double (&v)[7], double (*sm)[8]) {
#pragma unroll
  for (int c = C0; c < C1; ++c)
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  if (lane == 0)
#pragma unroll
    for (int c = C0; c < C1; ++c) sm[wid][c] = v[c];
  __syncthreads();
  if ((int)threadIdx.x >= C0 && (int)threadIdx.x < C1) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < kForceBlock / 32; ++w) a += sm[w][threadIdx.x];
    s.partial[(size_t)blockIdx.x * 8 + threadIdx.x] = a;
  }
}

// (1) + (2) + (3: the displacement check of a chained step) for the thread that holds the totals of atom i (valid) or
// nothing (!valid)
template <bool OBS>
__device__ __forceinline__ void force_finish(const DevSys &s, const KickParams &kick, const StepCtl &ctl, int i, bool valid, int ti,
                                             const double4 &pi, const ForceAcc<OBS> &acc, double (*sm)[8], unsigned long long *smd) {
  const double d2 = valid ? atom_update(s, kick, ctl, i, ti, pi, acc.fx, acc.fy, acc.fz) : 0.0;
  if constexpr (OBS) {
    double e_i = 0.0;
    if (valid) { e_i = s.eemb[i] + 0.5 * acc.ev; s.eatom[i] = e_i; }
    double v[7] = {e_i, 0.5 * acc.w0, 0.5 * acc.w1, 0.5 * acc.w2, 0.5 * acc.w3, 0.5 * acc.w4, 0.5 * acc.w5};
    if (!valid) {
#pragma unroll
      for (int c = 0; c < 7; ++c) v[c] = 0.0;
    }
    block_partials<0, 7>(s, v, sm);
  }
  if (ctl.chain || ctl.guard >= 0) finish_displacement(s, ctl, d2, smd);
}

// Half pass, first kernel: the owned part of the force (and of sum V) goes to frc / eatom as it is, the virial partials
// are complete (every undirected pair was evaluated exactly once: weight 1 where the full pass has 1/2 twice)
template <bool OBS>
__device__ __forceinline__ void force_park_half(const DevSys &s, int i, bool valid, const ForceAcc<OBS> &acc, double (*sm)[8]) {
  if (valid) {
    const size_t N = (size_t)s.N;
    s.frc[i] = acc.fx; s.frc[N + i] = acc.fy; s.frc[2 * N + i] = acc.fz;
  }
  if constexpr (OBS) {
    if (valid) s.eatom[i] = acc.ev;
    double v[7] = {0.0, acc.w0, acc.w1, acc.w2, acc.w3, acc.w4, acc.w5};
    if (!valid) {
#pragma unroll
      for (int c = 0; c < 7; ++c) v[c] = 0.0;
    }
    block_partials<1, 7>(s, v, sm);
  }
}

template <int KIND, bool MULTI, bool OBS, bool FOLD, bool DYN, bool HALF = false>
__global__ void __launch_bounds__(kForceBlock, kForceMinBlocks) k_force(const __grid_constant__ DevSys s, const KickParams kick, const StepCtl ctl) {
  __shared__ double tab_sm[kExpTabLen];
  __shared__ double sm[kForceBlock / 32][8];
  __shared__ unsigned long long smd[kForceBlock / 32];
  const bool go = step_guard(s, ctl.guard);
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  const bool valid = local < s.npb;
  const int i = box * s.npb + (valid ? local : 0);
  const AtomRow row = atom_row(s, box, local, i, valid);
  const double4 pi = s.posf[i];
  if (!go) return;
  if (!HALF && kick.h[0] != 0.0) {
    // the epilogue's velocity (and, chained, x_ref) loads come from DRAM at the very end of the block, when nothing is
    // left to hide them: ask L2 for their lines now (one line per warp and array)
    const size_t N = (size_t)s.N;
    if ((threadIdx.x & 15) == 0) {
#pragma unroll
      for (int c = 0; c < 3; ++c) {
        asm volatile("prefetch.global.L2 [%0];" :: "l"(s.vel + c * N + i));
        if (ctl.chain) asm volatile("prefetch.global.L2 [%0];" :: "l"(s.xref + c * N + i));
      }
    }
  }
  unsigned tab = 0;
  LoopConsts lc = {};
  if (KIND == MD_POT_TBSMA) { tab = stage_exp_table(s, tab_sm); lc = load_loop_consts(tab); }
  const int ti = MULTI ? s.type[i] : 0;
  ForceAcc<OBS> acc, acc2;
  // HALF: only the pairs this atom owns (first in the row); the partner's share (-g d, and V) goes out by red_fix
  const int own = HALF && valid ? s.nown[i] : 0;
  const int n_main = HALF ? (own & 0xffff) : row.n_in, n_tail = HALF ? (own >> 16) : row.n_out;
  auto send = [&](const PairD &d, double g, double V) {
    const size_t N = (size_t)s.N;
    long long *f = s.frc_fix + MD_GIDX(d.e);
    red_fix(f, -g * d.dx); red_fix(f + N, -g * d.dy); red_fix(f + 2 * N, -g * d.dz);
    if (OBS) red_fix(f + 3 * N, V);
  };

  auto prep = [&](unsigned e, const double4 &pj) {
    PairD d;
    d.r2 = pair_r2<KIND != MD_POT_TBSMA, DYN>(pj, pi, e, s, d.dx, d.dy, d.dz);
    d.w = pj.w; d.e = e;
    return d;
  };
  auto eval1 = [&](const PairD &d, ForceAcc<OBS> &to) {
    double g, V = 0.0;
    const int tp = MULTI ? ti * s.nt + s.type[d.e & kIdxMask] : 0;
    force_term<KIND, MULTI, OBS, FOLD>(s, lc, tab, tp, d.r2, pi.w + d.w, g, V);
    if (KIND != MD_POT_TBSMA && !(d.r2 < (MULTI ? s.rc2p[tp] : s.rc2))) { g = 0.0; V = 0.0; }   // tables: strict cut-off (A9)
    force_accumulate<OBS>(to, g, V, d.dx, d.dy, d.dz);
    if (HALF) send(d, g, V);
  };
  walk_main(row.main, n_main, s.posf, prep,
            [&](const PairD &a, const PairD &b) {
              if constexpr (KIND == MD_POT_TBSMA && !MULTI) {
                const double r2v[2] = {a.r2, b.r2}, fpv[2] = {pi.w + a.w, pi.w + b.w};
                double gv[2], Vv[2] = {0.0, 0.0};
                force_term_n<OBS, FOLD, 2>(s, lc, tab, r2v, fpv, gv, Vv);
                force_accumulate<OBS>(acc, gv[0], Vv[0], a.dx, a.dy, a.dz);
                force_accumulate<OBS>(acc2, gv[1], Vv[1], b.dx, b.dy, b.dz);
                if (HALF) { send(a, gv[0], Vv[0]); send(b, gv[1], Vv[1]); }
              } else {
                eval1(a, acc); eval1(b, acc2);
              }
            },
            [&](const PairD &a) { eval1(a, acc); });
  force_merge<OBS>(acc, acc2);

  // skin part: distance test only; pairs found inside r_c are parked and evaluated together (see k_density)
  const int mg = (__reduce_max_sync(0xffffffffu, n_tail) + 3) >> 2;
  unsigned park = 0u;
  bool parked = false;
  auto flush = [&]() { eval1(prep(park, gather32(slot_ptr(s.posf, MD_GIDX(park)))), acc); parked = false; };
  walk_tail(row.last, n_tail, mg, s.posf, prep, [&](const PairD &d, bool active) {
    const bool hit = active && d.r2 < s.rc2;
    if (__any_sync(0xffffffffu, hit && parked)) {
      if (parked) flush();
    }
    if (hit) { park = d.e; parked = true; }
  });
  if (__any_sync(0xffffffffu, parked)) {
    if (parked) flush();
  }

  if constexpr (HALF) force_park_half<OBS>(s, i, valid, acc, sm);
  else force_finish<OBS>(s, kick, ctl, i, valid, ti, pi, acc, sm, smd);
}

// Half pass, second kernel (same block-to-atom mapping as k_force): total force = owned part + what the partners sent,
// then the epilogue of the full pass (E_i = F(rho_i) + 1/2 (owned + received sum of V); its block partial is component 0)
template <bool OBS>
__global__ void __launch_bounds__(kForceBlock) k_force_half_finish(const __grid_constant__ DevSys s, const KickParams kick, const StepCtl ctl) {
  __shared__ double sm[kForceBlock / 32][8];
  __shared__ unsigned long long smd[kForceBlock / 32];
  if (!step_guard(s, ctl.guard)) return;
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  const bool valid = local < s.npb;
  const int i = box * s.npb + (valid ? local : 0);
  const size_t N = (size_t)s.N;
  double d2 = 0.0, e_i = 0.0;
  if (valid) {
    const double4 pi = s.posf[i];
    const int ti = s.nt > 1 ? s.type[i] : 0;
    long long *f = s.frc_fix + i;
    const double fx = s.frc[i] + fix_take(f), fy = s.frc[N + i] + fix_take(f + N), fz = s.frc[2 * N + i] + fix_take(f + 2 * N);
    d2 = atom_update(s, kick, ctl, i, ti, pi, fx, fy, fz);
    if (OBS) { e_i = s.eemb[i] + 0.5 * (s.eatom[i] + fix_take(f + 3 * N)); s.eatom[i] = e_i; }
  }
  if constexpr (OBS) {
    double v[7] = {e_i, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    block_partials<0, 1>(s, v, sm);
  }
  if (ctl.chain || ctl.guard >= 0) finish_displacement(s, ctl, d2, smd);
}



// ------------------------------------------------------------------------------------------------
// Small systems: kSub lanes per atom.  With one thread per atom a system of a few thousand atoms fills a fraction of
// the SMs and every thread walks its ~50 pairs one after the other (tens of microseconds of pure latency).  Here the
// kSub lanes of an atom take the 16-byte groups of its row round-robin and their partial sums are combined by
// shuffles in a fixed order (deterministic).  Same arithmetic per pair as the kernels above.
// ------------------------------------------------------------------------------------------------
struct SubMap { int box, local, i, sl; bool valid; };
template <int SUB>
__device__ __forceinline__ SubMap sub_map(const DevSys &s) {
  constexpr int kSubAtoms = kForceBlock / SUB;
  SubMap m;
  const int bpb = (s.npb + kSubAtoms - 1) / kSubAtoms;
  m.box = blockIdx.x / bpb;
  m.local = (blockIdx.x - m.box * bpb) * kSubAtoms + (threadIdx.x / SUB);
  m.sl = threadIdx.x % SUB;
  m.valid = m.local < s.npb;
  m.i = m.box * s.npb + (m.valid ? m.local : 0);
  return m;
}

// calls body(entry, gathered neighbour, in_main) for the entries of the row that this sub-lane owns: whole 16-byte groups
// round-robin, or (SUB >= 16: rows of a few tens of entries would leave most lanes idle) single entries round-robin.
// Software pipeline: the entries are loaded two turns ahead and the neighbours of the next turn are gathered before the
// current turn is evaluated, so that a lane waits for memory once per row, not once per pair.
template <int SUB, class Body>
__device__ __forceinline__ void walk_sub(const AtomRow &row, int sl, const double4 *__restrict__ pos, Body body) {
  if constexpr (SUB >= 16) {
    auto part = [&](const unsigned *base, int n, bool in_main, auto at) {
      int k = sl;
      if (k >= n) return;
      unsigned e = __ldg(base + at(k));
      double4 p = gather32(slot_ptr(pos, MD_GIDX(e)));
      for (;;) {
        const int kn = k + SUB;
        unsigned en = 0u;
        double4 pn = p;
        if (kn < n) { en = __ldg(base + at(kn)); pn = gather32(slot_ptr(pos, MD_GIDX(en))); }
        body(e, p, in_main);
        if (kn >= n) break;
        e = en; p = pn; k = kn;
      }
    };
    part(reinterpret_cast<const unsigned *>(row.main), row.n_in, true, [](int k) { return (int)nbr_entry(k); });
    part(reinterpret_cast<const unsigned *>(row.last), row.n_out, false, [](int k) { return 3 - (int)nbr_entry(k); });   // entry cap-1-k
    return;
  } else {
    // dir = +1: groups from the front (main part), -1: from the end of the row (skin part, entries in reverse inside a group)
    auto part = [&](const uint4 *base, int n, bool in_main, int dir) {
      const int ng = (n + 3) >> 2;
      int g = sl;
      if (g >= ng) return;
      const uint4 none = make_uint4(0u, 0u, 0u, 0u);
      auto order = [&](const uint4 &E, unsigned (&e)[4]) {
        if (dir > 0) { e[0] = E.x; e[1] = E.y; e[2] = E.z; e[3] = E.w; } else { e[0] = E.w; e[1] = E.z; e[2] = E.y; e[3] = E.x; }
      };
      unsigned e[4], en[4];
      double4 p[4], pn[4];
      order(ldg_group(base + (ptrdiff_t)dir * g * 32), e);
      uint4 En = (g + SUB < ng) ? ldg_group(base + (ptrdiff_t)dir * (g + SUB) * 32) : none;
#pragma unroll
      for (int c = 0; c < 4; ++c) p[c] = gather32(slot_ptr(pos, MD_GIDX(e[c])));           // slot 0 for the padding of a partly filled group: harmless
      for (;;) {
        const int gn = g + SUB;
        const bool more = gn < ng;
        order(En, en);
        En = (gn + SUB < ng) ? ldg_group(base + (ptrdiff_t)dir * (gn + SUB) * 32) : none;
        if (more) {
#pragma unroll
          for (int c = 0; c < 4; ++c) pn[c] = gather32(slot_ptr(pos, MD_GIDX(en[c])));
        }
#pragma unroll
        for (int c = 0; c < 4; ++c)
          if (g * 4 + c < n) body(e[c], p[c], in_main);
        if (!more) break;
#pragma unroll
        for (int c = 0; c < 4; ++c) { e[c] = en[c]; p[c] = pn[c]; }
        g = gn;
      }
    };
    part(row.main, row.n_in, true, 1);
    part(row.last, row.n_out, false, -1);
  }
}

template <int KIND, bool MULTI, bool FOLD, int SUB>
__global__ void __launch_bounds__(kForceBlock) k_density_sub(const __grid_constant__ DevSys s, const int guard) {
  constexpr int kSub = SUB;
  __shared__ double tab_sm[kExpTabLen];
  if (!step_guard(s, guard)) return;
  unsigned tab = 0;
  LoopConsts lc = {};
  if (KIND == MD_POT_TBSMA) { tab = stage_exp_table(s, tab_sm); lc = load_loop_consts(tab); }
  const SubMap m = sub_map<SUB>(s);
  const AtomRow row = atom_row(s, m.box, m.local, m.i, m.valid);
  const double4 pi = s.pos[m.i];
  const int ti = MULTI ? (int)pi.w : 0;
  double rho = 0.0;
  walk_sub<SUB>(row, m.sl, s.pos, [&](unsigned e, const double4 &pj, bool in_main) {
    double dx, dy, dz;
    const double r2 = pair_r2<KIND != MD_POT_TBSMA>(pj, pi, e, s, dx, dy, dz);
    // main: TB-SMA is switched off continuously beyond r_c, tables need the strict test; skin: only pairs now inside r_c
    const int tp = MULTI ? ti * s.nt + (int)pj.w : 0;
    if ((in_main && KIND == MD_POT_TBSMA) || r2 < (MULTI && KIND != MD_POT_TBSMA ? s.rc2p[tp] : s.rc2))
      rho += density_term<KIND, MULTI, FOLD>(s, lc, tab, tp, r2);
  });
#pragma unroll
  for (int o = 1; o < kSub; o <<= 1) rho += __shfl_xor_sync(0xffffffffu, rho, o);
  if (!m.valid || m.sl != 0) return;
  double F, Fp;
  embed<KIND>(s, ti, rho, F, Fp);
  if (!(fabs(Fp) <= 1.79e308) || !(fabs(rho) <= 1.79e308)) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
  s.rho[m.i] = rho;
  s.eemb[m.i] = F;
  s.posf[m.i] = make_double4(pi.x, pi.y, pi.z, Fp);
}

template <int KIND, bool MULTI, bool OBS, bool FOLD, int SUB>
__global__ void __launch_bounds__(kForceBlock) k_force_sub(const __grid_constant__ DevSys s, const KickParams kick, const StepCtl ctl) {
  constexpr int kSub = SUB;
  __shared__ double tab_sm[kExpTabLen];
  __shared__ double sm[kForceBlock / 32][8];
  __shared__ unsigned long long smd[kForceBlock / 32];
  if (!step_guard(s, ctl.guard)) return;
  unsigned tab = 0;
  LoopConsts lc = {};
  if (KIND == MD_POT_TBSMA) { tab = stage_exp_table(s, tab_sm); lc = load_loop_consts(tab); }
  const SubMap m = sub_map<SUB>(s);
  const AtomRow row = atom_row(s, m.box, m.local, m.i, m.valid);
  const double4 pi = s.posf[m.i];
  const int ti = MULTI ? s.type[m.i] : 0;
  ForceAcc<OBS> acc;
  walk_sub<SUB>(row, m.sl, s.posf, [&](unsigned e, const double4 &pj, bool in_main) {
    double dx, dy, dz, g, V = 0.0;
    const double r2 = pair_r2<KIND != MD_POT_TBSMA>(pj, pi, e, s, dx, dy, dz);
    const int tp = MULTI ? ti * s.nt + s.type[e & kIdxMask] : 0;
    if ((in_main && KIND == MD_POT_TBSMA) || r2 < (MULTI && KIND != MD_POT_TBSMA ? s.rc2p[tp] : s.rc2)) {
      force_term<KIND, MULTI, OBS, FOLD>(s, lc, tab, tp, r2, pi.w + pj.w, g, V);
      force_accumulate<OBS>(acc, g, V, dx, dy, dz);
    }
  });
#pragma unroll
  for (int o = 1; o < kSub; o <<= 1) {
    acc.fx += __shfl_xor_sync(0xffffffffu, acc.fx, o); acc.fy += __shfl_xor_sync(0xffffffffu, acc.fy, o);
    acc.fz += __shfl_xor_sync(0xffffffffu, acc.fz, o);
    if constexpr (OBS) {
      acc.ev += __shfl_xor_sync(0xffffffffu, acc.ev, o);
      acc.w0 += __shfl_xor_sync(0xffffffffu, acc.w0, o); acc.w1 += __shfl_xor_sync(0xffffffffu, acc.w1, o);
      acc.w2 += __shfl_xor_sync(0xffffffffu, acc.w2, o); acc.w3 += __shfl_xor_sync(0xffffffffu, acc.w3, o);
      acc.w4 += __shfl_xor_sync(0xffffffffu, acc.w4, o); acc.w5 += __shfl_xor_sync(0xffffffffu, acc.w5, o);
    }
  }
  force_finish<OBS>(s, kick, ctl, m.i, m.valid && m.sl == 0, ti, pi, acc, sm, smd);
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
  // (y'_k, a_k = 2 c2 / h) of both functions; the last node's record only serves as "next record" of the last interval
  der_c[off + k] = make_double4(cf.y * ih, cp.y * ih, 2.0 * cf.z * ih, 2.0 * cp.z * ih);
  if (k == per - 1) {
    const double df1 = (cf.y + 2.0 * cf.z + 3.0 * cf.w) * ih, dp1 = (cp.y + 2.0 * cp.z + 3.0 * cp.w) * ih;   // the quadratic's value at t = 1
    der_c[off + k + 1] = make_double4(df1, dp1, 0.0, 0.0);
  }
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
// variant of the two passes: lanes per atom.  One thread per atom fills the GPU from ~25 k atoms on; below that the
// lanes of an atom share its row (8 lanes, or 32 for a few thousand atoms, where a step is pure latency).
int sub_lanes(const md_system *sys) {
  switch (sys->opt_force_variant) {
    case 1: return 1;
    case 2: return 8;
    case 3: return sys->d.N <= kSub32Limit ? 32 : 8;
    case 4: return 4;
  }
  if (sys->d.N <= kSub32MaxAtoms) return 32;
  return sys->d.N <= kSubMaxAtoms ? 8 : 1;
}
// passes that run as half passes (MD_OPT_HALF_LIST): only with one thread per atom and a static box
// opt_half < 0 (default): chosen by what was measured on B200: the table passes are bound by the
// L1 data pipe (two gathered sectors per pair in the density pass), where one reduction per pair is cheaper than the
// second evaluation; the TB-SMA passes are bound by FP64 issue and the force pass sends three reductions per pair: full.
int half_mask(const md_system *sys) {
  if (sub_lanes(sys) != 1 || sys->d.dyn_box) return 0;
  if (sys->opt_half >= 0) return sys->opt_half;
  return sys->d.kind == MD_POT_EAM_TABLE ? 1 : 0;
}
int force_blocks(const md_system *sys) {
  return sys->d.nb * blocks_per_box(sys->d.npb, kForceBlock / sub_lanes(sys));
}

template <int KIND, bool FOLD, int SUB>
static void launch_density_sub(md_system *sys, int grid, int guard) {
  if (sys->d.nt > 1) k_density_sub<KIND, true, FOLD, SUB><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
  else k_density_sub<KIND, false, FOLD, SUB><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
}

template <int KIND, bool FOLD>
static void launch_density_k(md_system *sys, int grid, int guard) {
  ++sys->launches;
  switch (sub_lanes(sys)) {
    case 32: launch_density_sub<KIND, FOLD, 32>(sys, grid, guard); return;
    case 8: launch_density_sub<KIND, FOLD, 8>(sys, grid, guard); return;
    case 4: launch_density_sub<KIND, FOLD, 4>(sys, grid, guard); return;
  }
  if (sys->d.half & 1) {
    if (sys->d.nt > 1) k_density<KIND, true, FOLD, false, true><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
    else k_density<KIND, false, FOLD, false, true><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
    ++sys->launches, k_embed<KIND><<<(sys->d.N + 255) / 256, 256, 0, sys->stream>>>(sys->d, guard);
    return;
  }
  if (sys->d.dyn_box) {
    if (sys->d.nt > 1) k_density<KIND, true, FOLD, true><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
    else k_density<KIND, false, FOLD, true><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
  } else {
    if (sys->d.nt > 1) k_density<KIND, true, FOLD, false><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
    else k_density<KIND, false, FOLD, false><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, guard);
  }
}

int launch_density(md_system *sys, int guard) {
  ProfScope p(sys, MD_K_DENSITY);
  const int grid = force_blocks(sys);
  if (sys->d.kind == MD_POT_TBSMA) {
    if (sys->d.tb.fold) launch_density_k<MD_POT_TBSMA, true>(sys, grid, guard);
    else launch_density_k<MD_POT_TBSMA, false>(sys, grid, guard);
  } else launch_density_k<MD_POT_EAM_TABLE, true>(sys, grid, guard);
  return (int)cudaGetLastError();
}

template <int KIND, bool FOLD, int SUB>
static void launch_force_sub(md_system *sys, int grid, bool obs, const KickParams &kp, const StepCtl &ctl) {
  cudaStream_t st = sys->stream;
  if (sys->d.nt > 1) {
    if (obs) k_force_sub<KIND, true, true, FOLD, SUB><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    else k_force_sub<KIND, true, false, FOLD, SUB><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
  } else {
    if (obs) k_force_sub<KIND, false, true, FOLD, SUB><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    else k_force_sub<KIND, false, false, FOLD, SUB><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
  }
}

template <int KIND, bool FOLD>
static void launch_force_k(md_system *sys, int grid, bool obs, const KickParams &kp, const StepCtl &ctl) {
  const bool multi = sys->d.nt > 1;
  cudaStream_t st = sys->stream;
  ++sys->launches;
  switch (sub_lanes(sys)) {
    case 32: launch_force_sub<KIND, FOLD, 32>(sys, grid, obs, kp, ctl); return;
    case 8: launch_force_sub<KIND, FOLD, 8>(sys, grid, obs, kp, ctl); return;
    case 4: launch_force_sub<KIND, FOLD, 4>(sys, grid, obs, kp, ctl); return;
  }
  if (sys->d.half & 2) {
    if (multi) {
      if (obs) k_force<KIND, true, true, FOLD, false, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
      else k_force<KIND, true, false, FOLD, false, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    } else {
      if (obs) k_force<KIND, false, true, FOLD, false, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
      else k_force<KIND, false, false, FOLD, false, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    }
    ++sys->launches;
    if (obs) k_force_half_finish<true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    else k_force_half_finish<false><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    return;
  }
  if (multi) {
    if (sys->d.dyn_box) {
      if (obs) k_force<KIND, true, true, FOLD, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
      else k_force<KIND, true, false, FOLD, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    } else {
      if (obs) k_force<KIND, true, true, FOLD, false><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
      else k_force<KIND, true, false, FOLD, false><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    }
  } else {
    if (sys->d.dyn_box) {
      if (obs) k_force<KIND, false, true, FOLD, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
      else k_force<KIND, false, false, FOLD, true><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    } else {
      if (obs) k_force<KIND, false, true, FOLD, false><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
      else k_force<KIND, false, false, FOLD, false><<<grid, kForceBlock, 0, st>>>(sys->d, kp, ctl);
    }
  }
}

int launch_force(md_system *sys, bool observables, double half_dt, const StepCtl *ctlp) {
  const KickParams kp = make_kick(sys, half_dt);
  cudaGraphConditionalHandle none{};
  const StepCtl ctl = ctlp ? *ctlp : make_ctl(sys, 0.0, none, false, false);
  const int grid = force_blocks(sys);
  {
    ProfScope p(sys, ctl.chain ? MD_K_FORCE_CHAINED : MD_K_FORCE);
    if (sys->d.kind == MD_POT_TBSMA) {
      if (sys->d.tb.fold) launch_force_k<MD_POT_TBSMA, true>(sys, grid, observables, kp, ctl);
      else launch_force_k<MD_POT_TBSMA, false>(sys, grid, observables, kp, ctl);
    } else launch_force_k<MD_POT_EAM_TABLE, true>(sys, grid, observables, kp, ctl);
  }
  if (observables) {
    ProfScope p(sys, MD_K_REDUCE);
    ++sys->launches, k_reduce_boxes<<<sys->d.nb, 256, 0, sys->stream>>>(sys->d, force_blocks(sys) / sys->d.nb);
  }
  return (int)cudaGetLastError();
}

}  // namespace md
