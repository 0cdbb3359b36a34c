// md_internal.cuh — internal types shared by the translation units of libmd_b200.so.
// Nothing here is visible across the C ABI (include/md.h) and nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/md.h"

namespace md {

constexpr int kIdxBits = 26;                       // neighbour entry = index | (image code << 26)
constexpr unsigned kIdxMask = (1u << kIdxBits) - 1u;
constexpr int kMaxAtoms = 1 << kIdxBits;
constexpr int kPairs = MD_MAX_TYPES * MD_MAX_TYPES;
// exp_scaled() of md_force.cu: [0,64) 2^(j/64) (force pass, degree-5 polynomial), [64,80) the loop constants of the
// passes, [80,96) 2^(j/16) (density pass, degree-7 polynomial: 16 entries sit in 16 distinct bank pairs, so the
// look-up is free of bank conflicts; the density pass is bound by the L1 data pipe, the force pass is not)
constexpr int kExpTabLen = 64 + 16 + 16, kExp16Off = 80, kExpAddrSlot = 79;   // [64,80): constants; slot 79: the table's shared address
constexpr double kAmuToEvFs2PerA2 = 103.642696526805;  // 1 amu (A/fs)^2 in eV

// Device-resident mutable state (one per system).
struct DevState {
  unsigned long long maxd2_bits;   // bit pattern of max_i |x_i - x_ref,i|^2 since the last BUILD (>=0 doubles order as u64)
  double last_maxd2;               // its value at the last rebuild decision
  int force_rebuild;               // host request: rebuild at the next decision point
  int do_rebuild;                  // decision of the current rebuild chain
  int error_flags;                 // MD_FLAG_* (sticky)
  int max_neighbors;               // of the last build
  unsigned long long rebuilds;
  unsigned long long list_entries; // sum of list lengths of the last build
  double box[3];                   // CURRENT box edges (md_create's, then scaled by the barostat): every kernel reads them here
  double mu, pressure;             // last barostat step
  unsigned long long graph_body_runs; // rebuild bodies that ran inside a CUDA-graph step (for the launch count)
  unsigned long long step_word;    // running drift / chained force kernel: blocks arrived (low half) | blocks with an atom beyond skin/2 (high half)
  int k_done;                      // loop graphs (md_api.cu): steps of the current graph launch that are complete
  int iters_this_launch;           // ... and iterations of its WHILE node (bounded: a loop that makes no progress ends with MD_FLAG_LOOP)
  unsigned long long loop_iters;   // loop graphs: iterations of their WHILE nodes so far (for the launch count)
};

struct TbsmaParams {               // per type pair, pre-combined on the host
  // rho(r) = pre_rho exp(a_rho - b_rho r) S(r),  V(r) = pre_rep exp(a_rep - b_rep r) S(r)
  // fold != 0: ln(xi^2) and ln(2A) are folded into a_rho / a_rep and pre_* = 1 (all prefactors > 0)
  // ak_* = a_* 64/ln2 and bk_* = b_* 64/ln2: the exponent in units of ln2/64, as exp_scaled() takes it
  double ak_rho[kPairs], bk_rho[kPairs], b_rho[kPairs], pre_rho[kPairs];
  double ak16_rho[kPairs], bk16_rho[kPairs];   // the same in units of ln2/16 (density pass)
  double ak_rep[kPairs], bk_rep[kPairs], b_rep[kPairs], pre_rep[kPairs];
  // per type pair: switch variable t = clamp(r inv_w + t0, 0, 1), inv_w = 1/(r_c - r_on), t0 = -r_on inv_w;
  // m30_inv_w = -30 inv_w (dS/dr prefactor)
  double m30_inv_w[kPairs], inv_w[kPairs], t0[kPairs];
  int fold;
};

// Cubic-Hermite tables re-expressed per INTERVAL k (r in [k dr, (k+1) dr), t = r/dr - k) at md_create:
//   value      c0 + t (c1 + t (c2 + t c3))            c0 = y_k, c1 = h y'_k, c2 = 3D - h(2 y'_k + y'_{k+1}), c3 = h(y'_k + y'_{k+1}) - 2D
//   derivative (c1 + t (2 c2 + 3 c3 t)) / h  =  d1 + t (d2 + t d3)
struct TableParams {
  int nr, nrho;
  double dr, inv_dr, drho, inv_drho, rho_max;
  const double *f_val, *f_der, *phi_val, *phi_der;   // [nt*nt][nr]   node data as given (kept for the embedding and as the source)
  const double *F_val, *F_der;                       // [nt][nrho]
  const double4 *f_c;                                // [nt*nt][nr-1]  (c0,c1,c2,c3) of rho(r): density pass
  const double4 *phi_c;                              // [nt*nt][nr-1]  (c0,c1,c2,c3) of V(r): force pass with observables
  const double4 *der_c;                              // [nt*nt][nr]  (f'_k, phi'_k, a_k of f, a_k of phi): node slopes and linear coefficients of the
                                                     // derivative quadratics; the quadratic coefficient follows from the next record (md_force.cu): force pass
};

// Everything a kernel needs, passed by value as a __grid_constant__ parameter.
struct DevSys {
  int N, nb, npb, nt;
  double rl;                       // cutoff + skin
  double L0[3]; int dyn_box;       // box edges: L0 while no barostat has touched them, else DevState::box (box_edge())
  double rc2p[kPairs];             // per-pair cut-off squared (the paper's RCUT(ity,jty)); rc2 is their maximum
  double rc2, rl2, thr2, rin2;     // rin2: build-time split of a list row (pairs with r2 < rin2 first)
  int nc[3], tnc, ncell;           // cells per box (per dim, total) and cells of all boxes
  int zfine;                       // 1: cubic cells of side >= r_l, 27-cell stencil.  2, 4 (small boxes): cells thinner in z by that
                                   // factor; the candidates of a column of cells are then a z window around the atom (md_neighbor.cu)
  int cap;                         // neighbour capacity per atom
  int tiles_per_box;               // 32-atom tiles per box
  int kind;
  // per-atom state, CELL ORDER (index = "slot")
  double4 *pos;                    // x,y,z, w = type as double
  double4 *posf;                   // x,y,z, w = F'(rho): written by the density pass, gathered by the force pass
  float4 *pos32;                   // x,y,z rounded to float at the last re-order: the list build classifies its candidates on these
  double *vel, *frc, *xref;        // SoA, component c at [c*N + i]
  double *gacc, *gjrk, *gsnp;      // Gear predictor-corrector (md_gear.cu): second, third and fourth time derivative of x, SoA
  int *type, *orig;                // orig = caller index of the atom in this slot (paper's hGID)
  // re-order scratch
  double4 *pos_tmp; double *vel_tmp; int *type_tmp, *orig_tmp;
  int *cell_id, *cell_count, *cell_start, *cell_fill, *perm, *scan_block;
  // neighbour list, blocked ELL in groups of four: entries 4g .. 4g+3 of the atom in (tile, lane) are the 16 bytes at
  // nbr[((tile*cap/4 + g)*32 + lane)*4] (cap is a multiple of 4), so a warp reads 512 contiguous bytes per group.
  // Entries that were inside r_c at build time are at k = 0 .. n_in-1, the others at k = cap-n_out .. cap-1;
  // the unused entries of a partly filled group are 0; ncount = n_in | n_out << 16
  unsigned *nbr; int *ncount;
  // Newton's-third-law variant (MD_OPT_HALF_LIST, row f2): `half` bit 0: density pass, bit 1: force pass.  The list build
  // scans the half of the stencil whose pairs the atom OWNS first, so both parts of a row start with the owned pairs:
  // nown = n_own_in | n_own_out << 16.  A half pass evaluates only those and sends the partner's share to rho_fix /
  // frc_fix by 64-bit integer reductions in units of 2^-43 (integer addition is associative: the sums do not depend
  // on the order of arrival)
  int half; int *nown;
  long long *rho_fix;              // [N]
  long long *frc_fix;              // [4][N]: fx, fy, fz, sum of V (observables)
  const double *exp_tab;           // [kExpTabLen] 2^(j/64), correctly rounded (staged into shared memory by the passes), then LoopConsts
  // per-atom results
  double *rho, *eemb, *eatom;
  double *partial;                 // [n_blocks][8] block partial sums: E, Wxx,Wyy,Wzz,Wxy,Wxz,Wyz, (pad)
  double *box_epot, *box_virial, *box_ekin;
  DevState *st;
  TbsmaParams tb;
  TableParams tab;
};

// What the kernel that ends a drift needs for the rebuild decision (taken by its last block, decide_rebuild below):
// chain != 0 (force pass only): the epilogue also does the NEXT step's first half-kick, drift and displacement check.
// guard (loop graphs, md_api.cu): >= 0: this kernel belongs to step `guard` of a graph whose steps all sit in the body of
// ONE loop: it runs only if no rebuild is pending and exactly `guard` steps are complete (step_guard below), and the force
// pass that completes the step says so; kGuardReset (the drift at the head of such a graph): zero steps are complete.
struct StepCtl { double dt; unsigned long long thr2_bits; cudaGraphConditionalHandle cond; int use_cond; int chain; int guard; };
constexpr int kGuardNone = -1, kGuardReset = -2;

constexpr double kFixScale = 8796093022208.0, kFixInv = 1.0 / 8796093022208.0;   // 2^43: one unit = 1.1e-13 (eV/A, eV, density), range +-1.0e6

// first entry of the list row of the atom in (tile, lane); entry k is at row[(k >> 2) * 128 + (k & 3)]
__host__ __device__ inline size_t nbr_row_offset(size_t tile, int cap, int lane) { return (tile * (size_t)(cap >> 2) * 32 + lane) * 4; }
__host__ __device__ inline unsigned nbr_entry(int k) { return ((unsigned)k >> 2) * 128u + ((unsigned)k & 3u); }   // 32-bit: one IMAD.WIDE per store

// current box edge a: a kernel parameter until a barostat is switched on, device state from then on
__device__ __forceinline__ double box_edge(const DevSys &s, int a) { return s.dyn_box ? s.st->box[a] : s.L0[a]; }

// The rebuild decision, on the device (one thread): rebuild if the host asked for it or if some atom has moved more
// than skin/2 since the last build (`exceeded`: strict >, reading A11).  Inside a CUDA-graph step `cond` is the handle of
// the conditional node whose body is the rebuild chain; otherwise every kernel of the chain is launched and returns at
// once unless do_rebuild is set.
__device__ __forceinline__ void decide_rebuild(const DevSys &s, bool exceeded, cudaGraphConditionalHandle cond, int use_cond) {
  DevState *st = s.st;
  const bool go = *(volatile int *)&st->force_rebuild != 0 || exceeded;
  st->do_rebuild = go ? 1 : 0;
  st->last_maxd2 = __longlong_as_double((long long)*(volatile unsigned long long *)&st->maxd2_bits);
  st->force_rebuild = 0;
  if (go) {
    st->max_neighbors = 0; st->list_entries = 0ull; st->rebuilds += 1;
    for (int a = 0; a < 3; ++a)                        // the cell grid is fixed at md_create; a barostat may have shrunk the box
      if (!(a == 2 && s.zfine > 1) && !(box_edge(s, a) >= s.nc[a] * s.rl)) st->error_flags |= MD_FLAG_BOX;   // (a z window adapts to the box)
  }
  if (use_cond) { cudaGraphSetConditional(cond, go ? 1u : 0u); if (go) st->graph_body_runs += 1; }
}

// End of a drift (k_kick_drift, or the chained epilogue of the force pass): d2 = |x - x_ref|^2 of this thread's atom
// (0 for a thread without one).  Thread 0 of every block adds ONE word to DevState::step_word: the low half counts the
// blocks that have arrived, the high half those in which some atom exceeded skin/2.  The block that completes the count
// reads the decision off the value the atomic returns, so no fence, no second round trip and no separate decision
// kernel is needed; a block's resources are held for one L2 round trip after its last warp has finished.
// maxd2_bits (bit pattern of the largest d2 since the last build: non-negative doubles order like their bit patterns)
// is kept for md_stats and for md_set_positions; nothing waits for that reduction.
// Called by every thread of the block; sm holds blockDim.x / 32 entries.
__device__ __forceinline__ void finish_displacement(const DevSys &s, const StepCtl &c, double d2, unsigned long long *sm) {
  if (!(d2 == d2)) d2 = __longlong_as_double(0x7ff0000000000000ll);   // NaN -> +inf: forces a rebuild, which flags it
  unsigned long long b = (unsigned long long)__double_as_longlong(d2);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { const unsigned long long t = __shfl_xor_sync(0xffffffffu, b, o); b = t > b ? t : b; }
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = b;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < (int)(blockDim.x >> 5); ++w) b = sm[w] > b ? sm[w] : b;
    DevState *st = s.st;
    if (b) atomicMax(&st->maxd2_bits, b);
    const unsigned long long inc = 1ull | (b > c.thr2_bits ? (1ull << 32) : 0ull);
    const unsigned long long w = atomicAdd(&st->step_word, inc) + inc;
    if ((unsigned)(w & 0xffffffffull) == gridDim.x) {
      st->step_word = 0ull;                              // for the next kernel that ends a drift
      if (c.chain || c.guard == kGuardReset || c.guard == kGuardNone) decide_rebuild(s, (w >> 32) != 0ull, c.cond, c.use_cond);
      if (c.guard >= 0) st->k_done = c.guard + 1;        // (a step's last force pass without a drift only reports the step complete)
      if (c.guard == kGuardReset) { st->k_done = 0; st->iters_this_launch = 0; }
    }
  }
}

// Loop graphs: does this kernel of step `guard` run?  Every block asks (one L2 read, issued before the block's own loads).
__device__ __forceinline__ bool step_guard(const DevSys &s, int guard) {
  if (guard < 0) return true;
  const volatile DevState *st = s.st;
  return st->do_rebuild == 0 && st->k_done == guard;
}

struct ProfClass { std::vector<cudaEvent_t> ev; size_t used = 0; long dropped = 0; };

}  // namespace md

struct md_system {
  md::DevSys d;
  cudaStream_t stream;
  double mass_ev[MD_MAX_TYPES];    // eV fs^2 / A^2
  double cutoff, skin;
  double thermo_Te, thermo_tau;    // eq.(4) thermostat; tau <= 0: off
  double baro_P0, baro_tau;        // eq.(5) barostat; tau <= 0: off
  bool have_list, forces_valid, observables_valid;
  bool opt_step_obs, opt_profile, opt_graph;
  // one velocity-Verlet step as a CUDA graph: kick+drift, decision, IF(rebuild body), density, force (md_api.cu)
  // [0]: kStepUnroll steps, [1]: the remainder.  loop: the steps are the body of ONE while node (small systems); kernels:
  // launches per replay (loop: with one iteration); iter_kernels: launches of every further iteration
  struct StepGraph { cudaGraph_t graph; cudaGraphExec_t exec; double dt; bool obs, loop; int nsteps, kernels, iter_kernels; } sg[2];
  int body_kernels;
  int graph_error;                 // cudaError_t of a failed step-graph build (0: none); md_step then uses plain launches
  bool last_step_graph;            // the last md_step replayed the graph
  bool frc_keep;                   // frc holds the forces of the coordinates BEFORE the barostat scaled them: queries must not replace them
  int opt_force_variant, opt_half;
  int integrator; bool gear_ready; // MD_INT_*; the derivative arrays of the Gear scheme belong to the current x, v
  long steps, launches;
  double exp_tab_host[md::kExpTabLen];
  void *stage; size_t stage_bytes; // staging area for host<->device copies (inside the workspace)
  // md_step_get_state: a second stream (highest priority) and two events, created at its first call, so that the download of the
  // positions runs beside the two passes of the last step
  cudaStream_t side; cudaEvent_t ev_fork, ev_join; bool side_ready;
  md::ProfClass prof[MD_K_COUNT];
};

namespace md {
constexpr double kBoltzmannEv = 8.617333262e-5;     // eV/K
// half-kick parameters: h[t] = dt/(2 m_t); thermostat (eq.4): gdt = dt/(2 tau) (0: off), c2[t] = 3 k_B T_e / m_t
struct KickParams { double h[MD_MAX_TYPES]; double c2[MD_MAX_TYPES]; double gdt; };
KickParams make_kick(const md_system *s, double half_dt);
// v <- v + h f - gdt (1 - c2/|v|^2) v   (the second term only with the thermostat on; 0 for an atom at rest)
__device__ __forceinline__ void half_kick(const KickParams &k, int t, double fx, double fy, double fz, double &vx, double &vy, double &vz) {
  double g = 0.0;
  if (k.gdt != 0.0) {
    const double v2 = fma(vz, vz, fma(vy, vy, vx * vx));
    if (v2 > 0.0) g = k.gdt * (1.0 - k.c2[t] / v2);
  }
  const double h = k.h[t];
  // explicit FMAs: the same bits from every kernel that inlines this, whatever else it does with h, f or v
  vx = fma(-g, vx, fma(h, fx, vx)); vy = fma(-g, vy, fma(h, fy, vy)); vz = fma(-g, vz, fma(h, fz, vz));
}
// x += dt v and the squared displacement from x_ref = (rx, ry, rz) (explicit FMAs: the same bits from every kernel that inlines this)
__device__ __forceinline__ double drift_atom(double dt, double4 &x, double vx, double vy, double vz, double rx, double ry, double rz) {
  x.x = fma(dt, vx, x.x); x.y = fma(dt, vy, x.y); x.z = fma(dt, vz, x.z);
  const double ux = x.x - rx, uy = x.y - ry, uz = x.z - rz;
  return fma(uz, uz, fma(uy, uy, ux * ux));
}
// launch geometry of the per-atom kernels that use the tile mapping
constexpr int kForceBlock = 128;
constexpr int kSubMaxAtoms = 24576;                // at or below this many atoms the passes use 8 lanes per atom (md_force.cu)
constexpr int kSub32MaxAtoms = 4096;               // ... and 32 lanes per atom at or below this many
constexpr int kSub32Limit = 32768;                 // largest system the 32-lane variant may be forced on (sizes the block partials)
constexpr int kStepUnroll = 8;                     // time steps per CUDA graph of md_step (md_api.cu)
constexpr int kLoopGraphMaxAtoms = 4096;           // up to this many atoms the steps of a graph share ONE loop node instead of an IF node each
                                                   // (measured: 864 atoms 21.9 -> 17.5 us/step; 16,384 and 65,536 atoms: no gain; rebuilds every other step: a loss)
int sub_lanes(const md_system *s);                 // lanes per atom of the two passes: 1, 2, 4, 8 or 32
int force_blocks(const md_system *s);              // grid of the two passes (and number of block partials)
inline int blocks_per_box(int npb, int block) { return (npb + block - 1) / block; }

// launchers (each enqueues on s->stream; returns cudaError_t of the launch)
int launch_rebuild_chain(md_system *s);                       // decision + body, conditional on DevState (force_rebuild / maxd2)
int launch_decide(md_system *s, cudaGraphConditionalHandle cond, bool use_cond);
StepCtl make_ctl(const md_system *s, double dt, cudaGraphConditionalHandle cond, bool use_cond, bool chain, int guard = kGuardNone);
int launch_rebuild_body(md_system *s);
int launch_density(md_system *s, int guard = kGuardNone);
int launch_loop_head(md_system *s);                                            // loop graphs: one-thread kernels around the steps
int launch_loop_tail(md_system *s, cudaGraphConditionalHandle loop_cond, int nsteps);
int launch_rebuild_done(md_system *s);
int half_mask(const md_system *s);                            // passes that run as half passes now (0 unless one thread per atom, static box)
int launch_prepare_tables(md_system *s);                      // md_create, MD_POT_EAM_TABLE: per-interval coefficients
int launch_force(md_system *s, bool observables, double half_dt, const StepCtl *ctl = nullptr); // half_dt = dt/2 (0: no velocity update); ctl->chain: + next drift
int launch_kick_drift(md_system *s, double dt, const StepCtl &ctl);
int launch_ekin(md_system *s);
int launch_gear_start(md_system *s, double dt);               // md_gear.cu: the paper's predictor-corrector (five-value Gear scheme)
int launch_gear_predict(md_system *s, double dt);
int launch_gear_correct(md_system *s, double dt);
int launch_gear_reorder(md_system *s);
int launch_barostat(md_system *s, double dt);                 // ekin, mu and box update, scale positions (end of a step)
int launch_pressure(md_system *s);                            // ekin + eq.(6) into DevState::pressure

struct ProfScope {                 // brackets launches of one kernel class with events when profiling is on
  md_system *s; int cls; cudaEvent_t stop = nullptr;
  ProfScope(md_system *s, int cls);
  ~ProfScope();
};
}  // namespace md
