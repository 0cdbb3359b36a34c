// md_gear.cu — the paper's predictor-corrector integration (sec. 3.3: "A predictor-corrector scheme is
// used for the stepwise integration ... Each thread predicts the position and the velocity of one atom"; PAPER.md:165-167:
// the velocities are corrected after the force calculation), as an alternative to velocity-Verlet (md_set_integrator).
// The paper gives neither order nor coefficients (reading G1): the five-value Gear scheme for m x'' = f(x) of
// Allen & Tildesley, sec. 3.2: state x, v, a, j, s (the first four time derivatives), Taylor predictor, forces at the
// predicted positions, corrector with (19/120, 3/4, 1, 1/2, 1/12).  One thread per atom, as in the paper; the skin/2
// rule acts on the predicted positions and the last block of the predictor takes the rebuild decision.
#include "md_internal.cuh"

namespace md {

struct InvMass { double im[MD_MAX_TYPES]; };

static InvMass inv_mass(const md_system *sys) {
  InvMass m;
  for (int t = 0; t < MD_MAX_TYPES; ++t) m.im[t] = t < sys->d.nt ? 1.0 / sys->mass_ev[t] : 0.0;
  return m;
}

// dst = f / m  (a(x) at the start-up, a(+tau) parked in gjrk)
__global__ void __launch_bounds__(256) k_gear_accel(const __grid_constant__ DevSys s, const InvMass im, double *__restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t N = (size_t)s.N;
  const double w = im.im[s.nt > 1 ? s.type[i] : 0];
#pragma unroll
  for (int c = 0; c < 3; ++c) dst[c * N + i] = s.frc[c * N + i] * w;
}

// start-up: x <- x0 + sign tau v + tau^2/2 a   (x0 is kept in pos_tmp, free outside the rebuild chain)
__global__ void __launch_bounds__(256) k_gear_shift(const __grid_constant__ DevSys s, double stau, double tau) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t N = (size_t)s.N;
  double4 p = s.pos_tmp[i];
  const double h2 = 0.5 * tau * tau;
  p.x = p.x + stau * s.vel[i] + h2 * s.gacc[i];
  p.y = p.y + stau * s.vel[N + i] + h2 * s.gacc[N + i];
  p.z = p.z + stau * s.vel[2 * N + i] + h2 * s.gacc[2 * N + i];
  s.pos[i] = p;
}

// start-up, last kernel: j = (a(+tau) - a(-tau)) / 2 tau,  s = (a(+tau) - 2 a + a(-tau)) / tau^2,  x <- x0
__global__ void __launch_bounds__(256) k_gear_start(const __grid_constant__ DevSys s, const InvMass im, double tau) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t N = (size_t)s.N;
  const double w = im.im[s.nt > 1 ? s.type[i] : 0];
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const double ap = s.gjrk[c * N + i], am = s.frc[c * N + i] * w, a = s.gacc[c * N + i];
    s.gjrk[c * N + i] = (ap - am) / (2.0 * tau);
    s.gsnp[c * N + i] = ((ap - a) + (am - a)) / (tau * tau);
  }
  s.pos[i] = s.pos_tmp[i];
}

// predictor (Taylor series in dt) + displacement check of the predicted positions
__global__ void __launch_bounds__(256) k_gear_predict(const __grid_constant__ DevSys s, const StepCtl ctl) {
  __shared__ unsigned long long sm[8];
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  const size_t N = (size_t)s.N;
  const double h1 = ctl.dt, h2 = ctl.dt * ctl.dt / 2.0, h3 = ctl.dt * ctl.dt * ctl.dt / 6.0, h4 = ctl.dt * ctl.dt * ctl.dt * ctl.dt / 24.0;
  double d2 = 0.0;
  if (i < s.N) {
    double4 p = s.pos[i];
    double x[3] = {p.x, p.y, p.z};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const size_t k = c * N + i;
      const double v = s.vel[k], a = s.gacc[k], j = s.gjrk[k], q = s.gsnp[k];
      x[c] = x[c] + h1 * v + h2 * a + h3 * j + h4 * q;
      s.vel[k] = v + h1 * a + h2 * j + h3 * q;
      s.gacc[k] = a + h1 * j + h2 * q;
      s.gjrk[k] = j + h1 * q;
      const double u = x[c] - s.xref[k];
      d2 += u * u;
    }
    p.x = x[0]; p.y = x[1]; p.z = x[2];
    s.pos[i] = p;
  }
  finish_displacement(s, ctl, d2, sm);
}

// corrector: D = dt^2/2 (f(x_p)/m - a_p), then every derivative gets its share of D
__global__ void __launch_bounds__(256) k_gear_correct(const __grid_constant__ DevSys s, const InvMass im, double dt) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t N = (size_t)s.N;
  const double c0 = 19.0 / 120.0, c1 = 3.0 / 4.0, c3 = 1.0 / 2.0, c4 = 1.0 / 12.0;
  const double h1 = dt, h2 = dt * dt / 2.0, h3 = dt * dt * dt / 6.0, h4 = dt * dt * dt * dt / 24.0;
  const double w = im.im[s.nt > 1 ? s.type[i] : 0];
  double4 p = s.pos[i];
  double x[3] = {p.x, p.y, p.z};
#pragma unroll
  for (int c = 0; c < 3; ++c) {
    const size_t k = c * N + i;
    const double D = h2 * (s.frc[k] * w - s.gacc[k]);
    x[c] += c0 * D;
    s.vel[k] += c1 * D / h1;
    s.gacc[k] += D / h2;
    s.gjrk[k] += c3 * D / h3;
    s.gsnp[k] += c4 * D / h4;
  }
  p.x = x[0]; p.y = x[1]; p.z = x[2];
  s.pos[i] = p;
}

// re-order: the three derivative arrays follow the atoms into cell order (perm of the rebuild chain, through vel_tmp)
__global__ void __launch_bounds__(256) k_gear_permute(const __grid_constant__ DevSys s, const double *__restrict__ src) {
  if (!s.st->do_rebuild) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t N = (size_t)s.N;
  const int from = s.perm[i];
#pragma unroll
  for (int c = 0; c < 3; ++c) s.vel_tmp[c * N + i] = src[c * N + from];
}
__global__ void __launch_bounds__(256) k_gear_copy(const __grid_constant__ DevSys s, double *__restrict__ dst) {
  if (!s.st->do_rebuild) return;
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t N = (size_t)s.N;
#pragma unroll
  for (int c = 0; c < 3; ++c) dst[c * N + i] = s.vel_tmp[c * N + i];
}

int launch_gear_reorder(md_system *sys) {
  const DevSys &d = sys->d;
  const int g = (d.N + 255) / 256;
  ProfScope p(sys, MD_K_REORDER);
  double *arr[3] = {d.gacc, d.gjrk, d.gsnp};
  for (double *a : arr) {
    ++sys->launches, k_gear_permute<<<g, 256, 0, sys->stream>>>(d, a);
    ++sys->launches, k_gear_copy<<<g, 256, 0, sys->stream>>>(d, a);
  }
  return (int)cudaGetLastError();
}

// a = f(x)/m and, by central differences of a along the Taylor path x(+-tau), tau = dt/10, the third and fourth derivative
// (with j = s = 0 the first predicted velocity would be off by dt^2/2 j and the scheme would stay second order).
// Expects a valid list and frc = f(x).
int launch_gear_start(md_system *sys, double dt) {
  const DevSys &d = sys->d;
  const int g = (d.N + 255) / 256;
  const InvMass im = inv_mass(sys);
  const double tau = 0.1 * dt;
  cudaStream_t st = sys->stream;
  ProfScope p(sys, MD_K_INTEGRATE);
  ++sys->launches, k_gear_accel<<<g, 256, 0, st>>>(d, im, d.gacc);
  if (cudaMemcpyAsync(d.pos_tmp, d.pos, (size_t)d.N * sizeof(double4), cudaMemcpyDeviceToDevice, st) != cudaSuccess) return 1;
  ++sys->launches, k_gear_shift<<<g, 256, 0, st>>>(d, tau, tau);
  if (launch_density(sys) != 0 || launch_force(sys, false, 0.0) != 0) return 1;
  ++sys->launches, k_gear_accel<<<g, 256, 0, st>>>(d, im, d.gjrk);
  ++sys->launches, k_gear_shift<<<g, 256, 0, st>>>(d, -tau, tau);
  if (launch_density(sys) != 0 || launch_force(sys, false, 0.0) != 0) return 1;
  ++sys->launches, k_gear_start<<<g, 256, 0, st>>>(d, im, tau);
  return (int)cudaGetLastError();
}

int launch_gear_predict(md_system *sys, double dt) {
  cudaGraphConditionalHandle none{};
  ProfScope p(sys, MD_K_INTEGRATE);
  ++sys->launches, k_gear_predict<<<(sys->d.N + 255) / 256, 256, 0, sys->stream>>>(sys->d, make_ctl(sys, dt, none, false, false));
  return (int)cudaGetLastError();
}

int launch_gear_correct(md_system *sys, double dt) {
  ProfScope p(sys, MD_K_INTEGRATE);
  ++sys->launches, k_gear_correct<<<(sys->d.N + 255) / 256, 256, 0, sys->stream>>>(sys->d, inv_mass(sys), dt);
  return (int)cudaGetLastError();
}

}  // namespace md
