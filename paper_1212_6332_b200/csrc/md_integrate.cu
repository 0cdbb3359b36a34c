// md_integrate.cu — velocity-Verlet half-kick + drift fused with the displacement check, kinetic energy,
// and the FP64 issue-rate diagnostic.
//
// Paper: section 3.3 (G8-G14): "each thread predicts the position and the velocity of
// one atom".  The paper's scheme is a predictor-corrector with a fixed 10-step rebuild interval
// (PAPER.md:199); BASELINE.json's north_star fixes velocity-Verlet and a skin/2 displacement trigger.
#include "md_internal.cuh"

namespace md {


// v += (dt/2m) f;  x += dt v;  d2 = |x - x_ref|^2  -> block max -> atomicMax on the bit pattern; the last block decides
// whether the list is rebuilt (finish_displacement).  drift_atom is shared with the chained epilogue of the force pass
// (md_force.cu), so that a step gives the same bits whichever kernel performs its drift.
__global__ void __launch_bounds__(256) k_kick_drift(const __grid_constant__ DevSys s, const KickParams p, const StepCtl ctl) {
  __shared__ unsigned long long sm[8];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const size_t N = (size_t)s.N;
  double d2 = 0.0;
  if (i < s.N) {
    double4 x = s.pos[i];
    double vx = s.vel[i], vy = s.vel[N + i], vz = s.vel[2 * N + i];
    const double rx = s.xref[i], ry = s.xref[N + i], rz = s.xref[2 * N + i];
    half_kick(p, s.nt > 1 ? (int)x.w : 0, s.frc[i], s.frc[N + i], s.frc[2 * N + i], vx, vy, vz);
    d2 = drift_atom(ctl.dt, x, vx, vy, vz, rx, ry, rz);
    s.vel[i] = vx; s.vel[N + i] = vy; s.vel[2 * N + i] = vz;
    s.pos[i] = x;
  }
  finish_displacement(s, ctl, d2, sm);
}

KickParams make_kick(const md_system *sys, double half_dt) {
  KickParams k;
  const bool on = sys->thermo_tau > 0.0 && half_dt != 0.0;
  k.gdt = on ? half_dt / sys->thermo_tau : 0.0;
  for (int t = 0; t < MD_MAX_TYPES; ++t) {
    const bool used = t < sys->d.nt;
    k.h[t] = used ? half_dt / sys->mass_ev[t] : 0.0;
    k.c2[t] = used ? 3.0 * kBoltzmannEv * sys->thermo_Te / sys->mass_ev[t] : 0.0;
  }
  return k;
}

int launch_kick_drift(md_system *sys, double dt, const StepCtl &ctl) {
  ProfScope p(sys, MD_K_INTEGRATE);
  const KickParams kp = make_kick(sys, 0.5 * dt);
  ++sys->launches, k_kick_drift<<<(sys->d.N + 255) / 256, 256, 0, sys->stream>>>(sys->d, kp, ctl);
  return (int)cudaGetLastError();
}

// kinetic energy per box: block partials (tile mapping, one box per block) then a fixed-order sum
struct MassParams { double m[MD_MAX_TYPES]; };

__global__ void __launch_bounds__(kForceBlock) k_ekin_partial(const __grid_constant__ DevSys s, const MassParams mp) {
  const int bpb = (s.npb + kForceBlock - 1) / kForceBlock;
  const int box = blockIdx.x / bpb, local = (blockIdx.x - box * bpb) * kForceBlock + threadIdx.x;
  double e = 0.0;
  if (local < s.npb) {
    const int i = box * s.npb + local;
    const size_t N = (size_t)s.N;
    const double vx = s.vel[i], vy = s.vel[N + i], vz = s.vel[2 * N + i];
    e = 0.5 * mp.m[s.nt > 1 ? s.type[i] : 0] * (vx * vx + vy * vy + vz * vz);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) e += __shfl_xor_sync(0xffffffffu, e, o);
  __shared__ double sm[kForceBlock / 32];
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = e;
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0;
#pragma unroll
    for (int w = 0; w < kForceBlock / 32; ++w) a += sm[w];
    s.partial[(size_t)blockIdx.x * 8 + 7] = a;
  }
}

__global__ void __launch_bounds__(256) k_ekin_boxes(const __grid_constant__ DevSys s, int bpb) {
  __shared__ double sm[256];
  const int box = blockIdx.x;
  double a = 0.0;
  for (int b = threadIdx.x; b < bpb; b += 256) a += s.partial[((size_t)box * bpb + b) * 8 + 7];
  sm[threadIdx.x] = a;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if (threadIdx.x < o) sm[threadIdx.x] += sm[threadIdx.x + o];
    __syncthreads();
  }
  if (threadIdx.x == 0) s.box_ekin[box] = sm[0];
}

int launch_ekin(md_system *sys) {
  ProfScope p(sys, MD_K_REDUCE);
  MassParams mp;
  for (int t = 0; t < MD_MAX_TYPES; ++t) mp.m[t] = (t < sys->d.nt) ? sys->mass_ev[t] : 0.0;
  const int bpb = blocks_per_box(sys->d.npb, kForceBlock);
  ++sys->launches, k_ekin_partial<<<sys->d.nb * bpb, kForceBlock, 0, sys->stream>>>(sys->d, mp);
  ++sys->launches, k_ekin_boxes<<<sys->d.nb, 256, 0, sys->stream>>>(sys->d, bpb);
  return (int)cudaGetLastError();
}

// ---- Berendsen barostat, eq.(5)-(6) ---------------------------------------------------
// P = (2/3 E_kin + 1/3 tr W) / V of box 0 (one box only); dt_over_tau < 0: pressure only, no scaling.
__global__ void k_pressure_mu(const __grid_constant__ DevSys s, double dt_over_tau, double P0) {
  DevState *st = s.st;
  const double trw = (s.box_virial[0] + s.box_virial[1]) + s.box_virial[2];
  const double V = st->box[0] * st->box[1] * st->box[2];
  const double P = ((2.0 / 3.0) * s.box_ekin[0] + trw / 3.0) / V;
  st->pressure = P;
  if (dt_over_tau < 0.0) return;
  const double mu = cbrt(1.0 - dt_over_tau * (P0 - P));
  st->mu = mu;
  st->box[0] *= mu; st->box[1] *= mu; st->box[2] *= mu;
}

__global__ void __launch_bounds__(256) k_scale_positions(const __grid_constant__ DevSys s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const double mu = s.st->mu;
  double4 p = s.pos[i];
  p.x *= mu; p.y *= mu; p.z *= mu;
  s.pos[i] = p;
}

int launch_pressure(md_system *sys) {
  if (launch_ekin(sys) != 0) return 1;
  ProfScope p(sys, MD_K_REDUCE);
  ++sys->launches, k_pressure_mu<<<1, 1, 0, sys->stream>>>(sys->d, -1.0, 0.0);
  return (int)cudaGetLastError();
}

int launch_barostat(md_system *sys, double dt) {
  if (launch_ekin(sys) != 0) return 1;
  ProfScope p(sys, MD_K_INTEGRATE);
  ++sys->launches, k_pressure_mu<<<1, 1, 0, sys->stream>>>(sys->d, dt / sys->baro_tau, sys->baro_P0);
  ++sys->launches, k_scale_positions<<<(sys->d.N + 255) / 256, 256, 0, sys->stream>>>(sys->d);
  return (int)cudaGetLastError();
}

// ---- FP64 issue-rate diagnostic: 8 independent DFMA chains per thread, register resident ---------
__global__ void __launch_bounds__(256) k_dfma_chains(double *out, int iters, double a, double b, long long *clocks) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0, x6 = x0 + 6.0,
         x7 = x0 + 7.0;
  unsigned long long g0, g1;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g0));
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 8; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  const long long t1 = clock64();
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(g1));
  const double r = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (r == 123.456) out[0] = r;        // keep the chains alive
  if (threadIdx.x == 0 && blockIdx.x == 0) { clocks[0] = t1 - t0; clocks[1] = (long long)(g1 - g0); }
}

}  // namespace md

extern "C" int md_fp64_dfma_rate(void *stream, double *dfma_per_s, double *sm_clock_mhz) {
  using namespace md;
  cudaStream_t st = (cudaStream_t)stream;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess)
    return MD_ECUDA;
  double *out = nullptr;
  long long *clk = nullptr;
  if (cudaMalloc(&out, sizeof(double)) != cudaSuccess) return MD_ECUDA;   // diagnostic only: the MD path never allocates
  if (cudaMalloc(&clk, 2 * sizeof(long long)) != cudaSuccess) { cudaFree(out); return MD_ECUDA; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 4096, blocks = sms * 8, threads = 256;
  k_dfma_chains<<<blocks, threads, 0, st>>>(out, 64, 0.999999, 1e-6, clk);   // warm-up
  float best = 1e30f;
  long long cyc[2] = {0, 1};
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, st);
    k_dfma_chains<<<blocks, threads, 0, st>>>(out, iters, 0.999999, 1e-6, clk);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { cudaFree(out); cudaFree(clk); return MD_ECUDA; }
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) { best = ms; cudaMemcpy(cyc, clk, sizeof(cyc), cudaMemcpyDeviceToHost); }
  }
  const double n = (double)blocks * threads * (double)iters * 64.0;
  if (dfma_per_s) *dfma_per_s = n / (best * 1e-3);
  // SM clock under this load: cycles / nanoseconds that block 0 spent in the loop
  if (sm_clock_mhz) *sm_clock_mhz = cyc[1] > 0 ? 1e3 * (double)cyc[0] / (double)cyc[1] : 0.0;
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(out); cudaFree(clk);
  return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ECUDA;
}
