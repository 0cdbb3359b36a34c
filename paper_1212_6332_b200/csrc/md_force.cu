// md_force.cu — density pass (paper's G18, Fig.5) and force pass with
// energy and virial (paper's G22, Fig.6), FP64, one thread per atom.
//
// Differences from the paper's kernels:
//  - atoms are in cell order and the list is a blocked-ELL array, so the list reads are coalesced and the
//    neighbour gathers hit L1/L2;
//  - the periodic image of each listed pair is recorded at build time, so there is no min/max logic in
//    the inner loop and r2 is bit-identical to the canonical expression;
//  - F'(rho_j) travels in the w component of the gathered position (one 32-byte sector per neighbour);
//  - energy and virial are reduced by warp shuffles into per-block partials and a second deterministic
//    pass, instead of shared-memory partials summed on the host.
#include "md_internal.cuh"

namespace md {

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

// quintic switch S and S' on [r_on, r_c]
__device__ __forceinline__ void taper(double r, const TbsmaParams &tb, double &S, double &dS) {
  if (r > tb.r_on) {
    const double t = (r - tb.r_on) * tb.inv_w, u = 1.0 - t, t2 = t * t;
    S = 1.0 - t2 * t * (10.0 + t * (-15.0 + 6.0 * t));
    dS = -30.0 * t2 * u * u * tb.inv_w;
  } else { S = 1.0; dS = 0.0; }
}

// cubic Hermite on a uniform grid from node values and node slopes (value and derivative of the SAME interpolant)
__device__ __forceinline__ void hermite(const double *__restrict__ val, const double *__restrict__ der, int n, double h,
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

template <int KIND>
__device__ __forceinline__ void embed(const DevSys &s, int ti, double rho, double &F, double &Fp) {
  if (KIND == MD_POT_TBSMA) {
    if (rho > 0.0) { const double sq = sqrt(rho); F = -sq; Fp = -0.5 / sq; }
    else { F = 0.0; Fp = 0.0; }
  } else {
    const TableParams &t = s.tab;
    const double *val = t.F_val + (size_t)ti * t.nrho, *der = t.F_der + (size_t)ti * t.nrho;
    if (rho >= t.rho_max) {
      Fp = der[t.nrho - 1];
      F = val[t.nrho - 1] + Fp * (rho - t.rho_max);
    } else {
      hermite(val, der, t.nrho, t.drho, t.inv_drho, rho, F, Fp);
    }
  }
}

// ------------------------------------------------------------------------------------------------
// Density pass: rho_i = sum_{j in list, r2 < rc2} f(r_ij); F(rho_i), F'(rho_i).
// ------------------------------------------------------------------------------------------------
template <int KIND, bool MULTI>
__global__ void __launch_bounds__(kForceBlock) k_density(const __grid_constant__ DevSys s) {
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  if (local >= s.npb) return;
  const int i = box * s.npb + local;
  const size_t tile = (size_t)box * s.tiles_per_box + (local >> 5);
  const unsigned *__restrict__ row = s.nbr + tile * s.cap * 32 + (local & 31);
  const double4 pi = s.pos[i];
  const int ti = MULTI ? (int)pi.w : 0;
  const int n = s.ncount[i];
  double rho = 0.0;
  bool bad = false;
  for (int k = 0; k < n; ++k) {
    const unsigned e = row[(size_t)k * 32];
    const double4 pj = s.pos[e & kIdxMask];
    double dx, dy, dz;
    const double r2 = pair_r2(pj, pi, e, s, dx, dy, dz);
    if (r2 < s.rc2) {
      if (!(r2 > 0.0)) { bad = true; continue; }
      const double r = sqrt(r2);
      const int tp = MULTI ? ti * s.nt + (int)pj.w : 0;
      if (KIND == MD_POT_TBSMA) {
        double S, dS;
        taper(r, s.tb, S, dS);
        rho += s.tb.xi2[tp] * exp(s.tb.q2[tp] - s.tb.q2_r0[tp] * r) * S;
      } else {
        double f, df;
        hermite(s.tab.f_val + (size_t)tp * s.tab.nr, s.tab.f_der + (size_t)tp * s.tab.nr, s.tab.nr, s.tab.dr,
                s.tab.inv_dr, r, f, df);
        rho += f;
      }
    }
  }
  if (bad) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
  double F, Fp;
  embed<KIND>(s, ti, rho, F, Fp);
  s.rho[i] = rho;
  s.eemb[i] = F;
  s.posf[i] = make_double4(pi.x, pi.y, pi.z, Fp);
}

// ------------------------------------------------------------------------------------------------
// Force pass: f_i = sum_j s_ij d/r, s_ij = V'(r) + (F'_i + F'_j) f'(r), d = x_j - x_i   [eq.(3)]
// OBS: also E_i = F(rho_i) + 1/2 sum_j V(r) [eq.(1)] and W^{ab} = -1/2 sum_j s_ij d^a d^b / r.
// half_dt_over_m[type] != 0: second half-kick v += (dt/2m) f fused into the epilogue.
// ------------------------------------------------------------------------------------------------
struct KickParams { double h[MD_MAX_TYPES]; };

template <int KIND, bool MULTI, bool OBS>
__global__ void __launch_bounds__(kForceBlock) k_force(const __grid_constant__ DevSys s, const KickParams kick) {
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  const bool valid = local < s.npb;
  double fx = 0.0, fy = 0.0, fz = 0.0, ev = 0.0;
  double w0 = 0.0, w1 = 0.0, w2 = 0.0, w3 = 0.0, w4 = 0.0, w5 = 0.0;
  const int i = box * s.npb + local;
  if (valid) {
    const size_t tile = (size_t)box * s.tiles_per_box + (local >> 5);
    const unsigned *__restrict__ row = s.nbr + tile * s.cap * 32 + (local & 31);
    const double4 pi = s.posf[i];
    const int ti = MULTI ? s.type[i] : 0;
    const int n = s.ncount[i];
    for (int k = 0; k < n; ++k) {
      const unsigned e = row[(size_t)k * 32];
      const int j = (int)(e & kIdxMask);
      const double4 pj = s.posf[j];
      double dx, dy, dz;
      const double r2 = pair_r2(pj, pi, e, s, dx, dy, dz);
      if (r2 < s.rc2 && r2 > 0.0) {
        const double r = sqrt(r2);
        const int tp = MULTI ? ti * s.nt + s.type[j] : 0;
        double df, V, dV;
        if (KIND == MD_POT_TBSMA) {
          double S, dS;
          taper(r, s.tb, S, dS);
          const double eh = s.tb.xi2[tp] * exp(s.tb.q2[tp] - s.tb.q2_r0[tp] * r);
          const double er = s.tb.A2[tp] * exp(s.tb.p[tp] - s.tb.p_r0[tp] * r);
          df = eh * (dS - s.tb.q2_r0[tp] * S);
          dV = er * (dS - s.tb.p_r0[tp] * S);
          V = er * S;
        } else {
          double f;
          const size_t off = (size_t)tp * s.tab.nr;
          hermite(s.tab.f_val + off, s.tab.f_der + off, s.tab.nr, s.tab.dr, s.tab.inv_dr, r, f, df);
          hermite(s.tab.phi_val + off, s.tab.phi_der + off, s.tab.nr, s.tab.dr, s.tab.inv_dr, r, V, dV);
        }
        const double g = (dV + (pi.w + pj.w) * df) / r;
        fx += g * dx; fy += g * dy; fz += g * dz;
        if (OBS) {
          ev += V;
          const double gx = g * dx, gy = g * dy;
          w0 -= gx * dx; w1 -= gy * dy; w2 -= g * dz * dz;
          w3 -= gx * dy; w4 -= gx * dz; w5 -= gy * dz;
        }
      }
    }
    s.frc[i] = fx; s.frc[(size_t)s.N + i] = fy; s.frc[2 * (size_t)s.N + i] = fz;
    const double h = kick.h[ti];
    if (h != 0.0) {
      s.vel[i] += h * fx; s.vel[(size_t)s.N + i] += h * fy; s.vel[2 * (size_t)s.N + i] += h * fz;
    }
    if (!(isfinite(fx) && isfinite(fy) && isfinite(fz))) atomicOr(&s.st->error_flags, MD_FLAG_NONFINITE);
  }
  if (OBS) {
    double e_i = 0.0;
    if (valid) { e_i = s.eemb[i] + 0.5 * ev; s.eatom[i] = e_i; }
    // warp-shuffle reduction (fixed butterfly order => deterministic), then across the 4 warps
    double v[7] = {e_i, 0.5 * w0, 0.5 * w1, 0.5 * w2, 0.5 * w3, 0.5 * w4, 0.5 * w5};
#pragma unroll
    for (int c = 0; c < 7; ++c)
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) v[c] += __shfl_xor_sync(0xffffffffu, v[c], o);
    __shared__ double sm[kForceBlock / 32][8];
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

template <int KIND>
static void launch_density_k(md_system *sys, int grid) {
  if (sys->d.nt > 1) ++sys->launches, k_density<KIND, true><<<grid, kForceBlock, 0, sys->stream>>>(sys->d);
  else ++sys->launches, k_density<KIND, false><<<grid, kForceBlock, 0, sys->stream>>>(sys->d);
}

int launch_density(md_system *sys) {
  ProfScope p(sys, MD_K_DENSITY);
  const int grid = sys->d.nb * blocks_per_box(sys->d.npb, kForceBlock);
  if (sys->d.kind == MD_POT_TBSMA) launch_density_k<MD_POT_TBSMA>(sys, grid);
  else launch_density_k<MD_POT_EAM_TABLE>(sys, grid);
  return (int)cudaGetLastError();
}

template <int KIND, bool MULTI>
static void launch_force_k(md_system *sys, int grid, bool obs, const KickParams &kp) {
  if (obs) ++sys->launches, k_force<KIND, MULTI, true><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, kp);
  else ++sys->launches, k_force<KIND, MULTI, false><<<grid, kForceBlock, 0, sys->stream>>>(sys->d, kp);
}

int launch_force(md_system *sys, bool observables, double half_dt) {
  KickParams kp;
  for (int t = 0; t < MD_MAX_TYPES; ++t) kp.h[t] = (t < sys->d.nt) ? half_dt / sys->mass_ev[t] : 0.0;
  const int grid = sys->d.nb * blocks_per_box(sys->d.npb, kForceBlock);
  {
    ProfScope p(sys, MD_K_FORCE);
    const bool multi = sys->d.nt > 1;
    if (sys->d.kind == MD_POT_TBSMA) {
      if (multi) launch_force_k<MD_POT_TBSMA, true>(sys, grid, observables, kp);
      else launch_force_k<MD_POT_TBSMA, false>(sys, grid, observables, kp);
    } else {
      if (multi) launch_force_k<MD_POT_EAM_TABLE, true>(sys, grid, observables, kp);
      else launch_force_k<MD_POT_EAM_TABLE, false>(sys, grid, observables, kp);
    }
  }
  if (observables) {
    ProfScope p(sys, MD_K_REDUCE);
    ++sys->launches, k_reduce_boxes<<<sys->d.nb, 256, 0, sys->stream>>>(sys->d, blocks_per_box(sys->d.npb, kForceBlock));
  }
  return (int)cudaGetLastError();
}

}  // namespace md
