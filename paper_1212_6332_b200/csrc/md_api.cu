// md_api.cu — the C ABI of include/md.h: argument checking, workspace layout, host/device staging,
// and the call sequences of md_build_neighbors / md_compute_forces / md_step.
#include <math.h>
#include <string.h>

#include <new>

#include <cstdio>
#include <cstdlib>

#include "md_internal.cuh"

using namespace md;

namespace md {

// ------------------------------------------------------------------------------------------------
// profiling scopes
// ------------------------------------------------------------------------------------------------
ProfScope::ProfScope(md_system *sys, int c) : s(sys), cls(c) {
  if (!s->opt_profile) return;
  ProfClass &p = s->prof[cls];
  if (p.used + 2 > p.ev.size()) {
    if (p.ev.size() >= 2 * 65536) { p.dropped++; return; }
    cudaEvent_t a, b;
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { p.dropped++; return; }
    p.ev.push_back(a); p.ev.push_back(b);
  }
  cudaEventRecord(p.ev[p.used], s->stream);
  stop = p.ev[p.used + 1];
  p.used += 2;
}
ProfScope::~ProfScope() { if (stop) cudaEventRecord(stop, s->stream); }

// ------------------------------------------------------------------------------------------------
// workspace layout: one bump allocation, 256-byte aligned pieces
// ------------------------------------------------------------------------------------------------
struct Bump {
  char *base; size_t off = 0;
  explicit Bump(void *b) : base((char *)b) {}
  template <class T> T *take(size_t n) {
    off = (off + 255) & ~(size_t)255;
    T *p = base ? (T *)(base + off) : nullptr;
    off += n * sizeof(T);
    return p;
  }
};

struct Geometry { int nc[3], zfine, tnc, ncell, cap, tiles_per_box, n_blocks, npb; size_t stage_bytes; };

// check_pairs: also validate the optional per-pair host arrays (md_create); the size query reads no pointer of *d
static int geometry(const md_desc *d, Geometry &g, bool check_pairs) {
  if (!d || d->n_atoms <= 0 || d->n_boxes <= 0 || d->n_types <= 0 || d->n_types > MD_MAX_TYPES) return MD_EINVAL;
  if (d->n_atoms % d->n_boxes || d->n_atoms > kMaxAtoms) return MD_EINVAL;
  if (!(d->cutoff > 0.0) || !(d->skin >= 0.0) || !isfinite(d->cutoff) || !isfinite(d->skin)) return MD_EINVAL;
  if (d->pot_kind != MD_POT_TBSMA && d->pot_kind != MD_POT_EAM_TABLE) return MD_EINVAL;
  if (d->pot_kind == MD_POT_EAM_TABLE && (d->nr < 2 || d->nrho < 2 || !(d->dr > 0.0) || !(d->drho > 0.0))) return MD_EINVAL;
  if (d->pot_kind == MD_POT_EAM_TABLE && (double)(d->nr - 1) * d->dr < d->cutoff * (1.0 - 1e-12)) return MD_EINVAL;
  if (d->pot_kind == MD_POT_TBSMA && !(d->taper_on < d->cutoff)) return MD_EINVAL;
  if (d->max_neighbors < 0) return MD_EINVAL;
  for (int a = 0; check_pairs && a < d->n_types; ++a)
    for (int b = 0; b < d->n_types; ++b) {
      const int k = a * d->n_types + b, kt = b * d->n_types + a;
      const double rc = d->pair_cutoff ? d->pair_cutoff[k] : d->cutoff;
      if (!(rc > 0.0) || !(rc <= d->cutoff) || (d->pair_cutoff && d->pair_cutoff[kt] != rc)) return MD_EINVAL;
      if (d->pot_kind == MD_POT_TBSMA) {
        const double ron = d->pair_taper_on ? d->pair_taper_on[k] : d->taper_on;
        if (!(ron < rc) || (d->pair_taper_on && d->pair_taper_on[kt] != ron)) return MD_EINVAL;
      }
    }
  const double rl = d->cutoff + d->skin;
  g.npb = d->n_atoms / d->n_boxes;
  double vol = 1.0;
  for (int a = 0; a < 3; ++a) {
    if (!(d->box[a] > 0.0) || !isfinite(d->box[a])) return MD_EINVAL;
    g.nc[a] = (int)floor(d->box[a] / rl);
    if (g.nc[a] < 3) return MD_EBOX;                 // 26 distinct neighbour cells
    vol *= d->box[a];
  }
  // Small boxes (some edge shorter than 5 r_l): cells four times thinner in z (the fastest cell index: a column of cells is
  // one contiguous run of slots).  The candidates of a column are then the z window [z_i - w, z_i + w], w^2 = r_l^2 -
  // (lateral gap to the column)^2, instead of three whole cells: cfg2 list build 0.097 (cubic cells) / 0.088 (half) / 0.081
  // (quarter cells) ms per step with the list kernel of md_neighbor.cu.  Large boxes keep cubic cells: there the
  // lanes of a warp that share a cell scan the SAME slots (their loads are broadcasts), and per-atom windows cost more in
  // L1 wavefronts than they save in tests (measured: 0.58 -> 0.70 ms per 1 M atoms with quarter cells, 0.61 with half).
  // Also measured and dropped: cells of half the cut-off in all three directions with a 5 x 5 x 5 stencil (0.76 ms).
  const bool large = g.nc[0] >= 5 && g.nc[1] >= 5 && g.nc[2] >= 5;
  g.zfine = large ? 1 : 4;
  if (const char *e = getenv("MD_CELL_ZFINE")) { const int v = atoi(e); if (v == 1 || v == 2 || v == 4) g.zfine = v; }   // for the measurements above
  while (g.zfine > 1 && (double)g.nc[0] * g.nc[1] * floor(g.zfine * d->box[2] / rl) * d->n_boxes > 1.6e7) g.zfine /= 2;
  g.nc[2] = (int)floor(g.zfine * d->box[2] / rl);
  const double cells = (double)g.nc[0] * g.nc[1] * g.nc[2];
  if (cells * d->n_boxes > 1.6e7) return MD_EINVAL;  // two-level scan limit (4096 * 4096 cells)
  g.tnc = g.nc[0] * g.nc[1] * g.nc[2];
  g.ncell = g.tnc * d->n_boxes;
  if (d->max_neighbors > 0) g.cap = d->max_neighbors;
  else {
    // MN "adjusted according to the particle density of the system and the cut-off"
    const double expect = 4.18879020478639 * rl * rl * rl * (double)g.npb / vol;
    g.cap = (int)(1.5 * expect) + 16;
  }
  if (g.cap > g.npb - 1) g.cap = g.npb - 1;
  if (g.cap < 4) g.cap = 4;
  if (g.cap > 0xfff0) return MD_EINVAL;               // ncount packs two 16-bit counts
  g.cap = (g.cap + 3) & ~3;
  g.tiles_per_box = (g.npb + 31) / 32;
  // block partials: enough for the 8-lanes-per-atom variant, and for 32 lanes per atom where that variant is allowed
  g.n_blocks = d->n_boxes * blocks_per_box(g.npb, kForceBlock / (d->n_atoms <= kSub32Limit ? 32 : 8));
  g.stage_bytes = (size_t)d->n_atoms * 6 * sizeof(double);        // positions and velocities of one md_set_state / md_get_state
  if (g.stage_bytes < (1u << 20)) g.stage_bytes = 1u << 20;
  return MD_OK;
}

static size_t layout(const md_desc *d, const Geometry &g, void *base, md_system *sys) {
  Bump b(base);
  DevSys t;  // filled only when sys != nullptr
  const size_t N = (size_t)d->n_atoms, nt2 = (size_t)d->n_types * d->n_types;
  t.st = b.take<DevState>(1);
  t.pos = b.take<double4>(N); t.posf = b.take<double4>(N); t.pos_tmp = b.take<double4>(N); t.pos32 = b.take<float4>(N);
  t.vel = b.take<double>(3 * N); t.vel_tmp = b.take<double>(3 * N);
  t.frc = b.take<double>(3 * N); t.xref = b.take<double>(3 * N);
  t.gacc = b.take<double>(3 * N); t.gjrk = b.take<double>(3 * N); t.gsnp = b.take<double>(3 * N);
  t.type = b.take<int>(N); t.type_tmp = b.take<int>(N); t.orig = b.take<int>(N); t.orig_tmp = b.take<int>(N);
  t.cell_id = b.take<int>(N); t.perm = b.take<int>(N);
  t.cell_count = b.take<int>((size_t)g.ncell + 1); t.cell_start = b.take<int>((size_t)g.ncell + 1);
  t.cell_fill = b.take<int>((size_t)g.ncell + 1);
  t.scan_block = b.take<int>(4096);
  t.nbr = b.take<unsigned>((size_t)d->n_boxes * g.tiles_per_box * g.cap * 32);
  t.ncount = b.take<int>(N);
  t.nown = b.take<int>(N); t.rho_fix = b.take<long long>(N); t.frc_fix = b.take<long long>(4 * N);
  t.rho = b.take<double>(N); t.eemb = b.take<double>(N); t.eatom = b.take<double>(N);
  t.partial = b.take<double>((size_t)g.n_blocks * 8);
  t.box_epot = b.take<double>(d->n_boxes); t.box_virial = b.take<double>((size_t)d->n_boxes * 6);
  t.box_ekin = b.take<double>(d->n_boxes);
  double *tabs[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
  double4 *coef[3] = {nullptr, nullptr, nullptr};
  if (d->pot_kind == MD_POT_EAM_TABLE) {
    for (int k = 0; k < 4; ++k) tabs[k] = b.take<double>(nt2 * d->nr);
    for (int k = 4; k < 6; ++k) tabs[k] = b.take<double>((size_t)d->n_types * d->nrho);
    coef[0] = b.take<double4>(nt2 * (d->nr - 1)); coef[1] = b.take<double4>(nt2 * (d->nr - 1));
    coef[2] = b.take<double4>(2 * nt2 * (d->nr - 1));
  }
  double *exp_tab = b.take<double>(kExpTabLen);
  void *stage = b.take<char>(g.stage_bytes);
  if (sys) {
    DevSys &o = sys->d;
    o.st = t.st; o.pos = t.pos; o.posf = t.posf; o.pos_tmp = t.pos_tmp; o.pos32 = t.pos32; o.vel = t.vel; o.vel_tmp = t.vel_tmp;
    o.frc = t.frc; o.xref = t.xref; o.gacc = t.gacc; o.gjrk = t.gjrk; o.gsnp = t.gsnp; o.type = t.type; o.type_tmp = t.type_tmp; o.orig = t.orig; o.orig_tmp = t.orig_tmp;
    o.cell_id = t.cell_id; o.perm = t.perm; o.cell_count = t.cell_count; o.cell_start = t.cell_start;
    o.cell_fill = t.cell_fill; o.scan_block = t.scan_block; o.nbr = t.nbr; o.ncount = t.ncount; o.rho = t.rho;
    o.nown = t.nown; o.rho_fix = t.rho_fix; o.frc_fix = t.frc_fix;
    o.eemb = t.eemb; o.eatom = t.eatom; o.partial = t.partial; o.box_epot = t.box_epot; o.box_virial = t.box_virial;
    o.box_ekin = t.box_ekin;
    o.tab.f_val = tabs[0]; o.tab.f_der = tabs[1]; o.tab.phi_val = tabs[2]; o.tab.phi_der = tabs[3];
    o.tab.F_val = tabs[4]; o.tab.F_der = tabs[5];
    o.tab.f_c = coef[0]; o.tab.phi_c = coef[1]; o.tab.der_c = coef[2]; o.exp_tab = exp_tab;
    sys->stage = stage; sys->stage_bytes = g.stage_bytes;
  }
  return (b.off + 255) & ~(size_t)255;
}

// ------------------------------------------------------------------------------------------------
// host / device pointer handling
// ------------------------------------------------------------------------------------------------
static bool on_device(const void *p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

// ---- conversion kernels between caller order (AoS [N][3]) and cell order ------------------------
__global__ void k_init_atoms(const __grid_constant__ DevSys s, const double *__restrict__ x, const int *__restrict__ types) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const int t = types[i];
  if (t < 0 || t >= s.nt) atomicOr(&s.st->error_flags, 1 << 30);
  s.pos[i] = make_double4(x[3 * (size_t)i], x[3 * (size_t)i + 1], x[3 * (size_t)i + 2], (double)t);
  s.type[i] = t;
  s.orig[i] = i;
}

__global__ void k_set_vec(const __grid_constant__ DevSys s, double *__restrict__ dst, const double *__restrict__ src) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;   // slot
  if (i >= s.N) return;
  const size_t o = 3 * (size_t)s.orig[i];
  dst[i] = src ? src[o] : 0.0; dst[(size_t)s.N + i] = src ? src[o + 1] : 0.0; dst[2 * (size_t)s.N + i] = src ? src[o + 2] : 0.0;
}

__global__ void k_get_vec(const __grid_constant__ DevSys s, const double *__restrict__ src, double *__restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t o = 3 * (size_t)s.orig[i];
  dst[o] = src[i]; dst[o + 1] = src[(size_t)s.N + i]; dst[o + 2] = src[2 * (size_t)s.N + i];
}

__global__ void k_get_scalar(const __grid_constant__ DevSys s, const double *__restrict__ src, double *__restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < s.N) dst[s.orig[i]] = src[i];
}

__global__ void k_get_fprime(const __grid_constant__ DevSys s, double *__restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < s.N) dst[s.orig[i]] = s.posf[i].w;
}

__global__ void k_get_pos(const __grid_constant__ DevSys s, double *__restrict__ dst) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const double4 p = s.pos[i];
  const size_t o = 3 * (size_t)s.orig[i];
  dst[o] = p.x; dst[o + 1] = p.y; dst[o + 2] = p.z;
}

// new positions: take the periodic image nearest x_ref (so that x - x_ref needs no image logic later) and
// fold the displacement into the rebuild decision
__global__ void k_set_pos(const __grid_constant__ DevSys s, const double *__restrict__ src, int have_ref) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t o = 3 * (size_t)s.orig[i], N = (size_t)s.N;
  double4 p = s.pos[i];
  double x[3] = {src[o], src[o + 1], src[o + 2]};
  if (have_ref) {
    double d2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double ref = s.xref[c * N + i];
      double u = x[c] - ref;
      const double Lc = box_edge(s, c);
      u -= Lc * rint(u / Lc);
      x[c] = ref + u;
      d2 += u * u;
    }
    if (!(d2 == d2)) d2 = __longlong_as_double(0x7ff0000000000000ll);
    atomicMax(&s.st->maxd2_bits, (unsigned long long)__double_as_longlong(d2));
  }
  p.x = x[0]; p.y = x[1]; p.z = x[2];
  s.pos[i] = p;
}

// md_set_state: positions (as k_set_pos, but an atom whose uploaded coordinates are bit-identical to the resident ones is
// left alone and does not count as moved) and velocities in one kernel; *changed is set if some position differs.
__global__ void k_set_state(const __grid_constant__ DevSys s, const double *__restrict__ x, const double *__restrict__ v, int have_ref,
                            int *changed) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= s.N) return;
  const size_t o = 3 * (size_t)s.orig[i], N = (size_t)s.N;
  if (v) { s.vel[i] = v[o]; s.vel[N + i] = v[o + 1]; s.vel[2 * N + i] = v[o + 2]; }
  if (!x) return;
  double4 p = s.pos[i];
  double q[3] = {x[o], x[o + 1], x[o + 2]};
  if (q[0] == p.x && q[1] == p.y && q[2] == p.z) return;
  *changed = 1;
  if (have_ref) {
    double d2 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
      const double ref = s.xref[c * N + i];
      double u = q[c] - ref;
      const double Lc = box_edge(s, c);
      u -= Lc * rint(u / Lc);
      q[c] = ref + u;
      d2 += u * u;
    }
    if (!(d2 == d2)) d2 = __longlong_as_double(0x7ff0000000000000ll);
    atomicMax(&s.st->maxd2_bits, (unsigned long long)__double_as_longlong(d2));
  }
  p.x = q[0]; p.y = q[1]; p.z = q[2];
  s.pos[i] = p;
}

// neighbour list as caller indices, ascending per atom (test hook).  perm[] (free outside the rebuild chain)
// is first filled with the inverse of orig[]; then one thread per CALLER atom in [first, first+natoms)
// writes its count and its row (insertion sort in place) at chunk-relative position a.
__global__ void k_invert_orig(const __grid_constant__ DevSys s) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < s.N) s.perm[s.orig[i]] = i;
}

__global__ void k_export_neighbors(const __grid_constant__ DevSys s, int first, int natoms, int *__restrict__ count,
                                   int *__restrict__ list, int stride, int *overflow) {
  const int a = blockIdx.x * blockDim.x + threadIdx.x;
  if (a >= natoms) return;
  const int i = s.perm[first + a];
  const int box = i / s.npb, local = i - box * s.npb;
  const size_t tile = (size_t)box * s.tiles_per_box + (local >> 5);
  const unsigned *row = s.nbr + nbr_row_offset(tile, s.cap, local & 31);
  const int c = s.ncount[i], n_in = c & 0xffff, n = n_in + (c >> 16);
  count[a] = n;
  if (n > stride) { atomicOr(overflow, 1); return; }
  int *out = list + (size_t)a * stride;
  for (int k = 0; k < n; ++k) {
    const int kk = k < n_in ? k : s.cap - 1 - (k - n_in);        // front part, then the skin part stored from the back
    const int v = s.orig[row[nbr_entry(kk)] & kIdxMask];
    int b = k - 1;
    while (b >= 0 && out[b] > v) { out[b + 1] = out[b]; --b; }
    out[b + 1] = v;
  }
  for (int k = n; k < stride; ++k) out[k] = -1;      // rows are padded with -1
}

static inline int grid_for(int n, int tb = 256) { return (n + tb - 1) / tb; }

static int check_cuda(cudaError_t e) { return e == cudaSuccess ? MD_OK : MD_ECUDA; }

static int sync_and_flags(md_system *s, int *flags_out = nullptr) {
  DevState st;
  if (cudaMemcpyAsync(&st, s->d.st, sizeof(st), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA;
  if (cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
  if (flags_out) *flags_out = st.error_flags;
  if (st.error_flags & (1 << 29)) return MD_ESTATE;                  // a loop graph that made no progress (internal error)
  if (st.error_flags & MD_FLAG_BOX) return MD_EBOX;                 // first: an over-compressed box also overflows the lists
  if (st.error_flags & MD_FLAG_NONFINITE) return MD_ENONFINITE;
  if (st.error_flags & MD_FLAG_OVERFLOW) return MD_EOVERFLOW;
  return MD_OK;
}

// copy `bytes` from a device scratch/result buffer to a user pointer (host or device)
static int deliver(md_system *s, void *user, const void *dev, size_t bytes, bool *was_host) {
  const bool dev_ptr = on_device(user);
  if (was_host) *was_host = !dev_ptr;
  return check_cuda(cudaMemcpyAsync(user, dev, bytes, dev_ptr ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, s->stream));
}

static int forces_sequence(md_system *s, bool observables, double half_dt) {
  if (launch_rebuild_chain(s) != 0 || launch_density(s) != 0 || launch_force(s, observables, half_dt) != 0) return MD_ECUDA;
  s->have_list = true;
  s->forces_valid = true;
  s->observables_valid = observables;
  return MD_OK;
}

// Force evaluation on behalf of a QUERY (md_compute_forces, md_get_energies, md_get_pressure between steps).  After a
// barostat step the observables belong to the SCALED coordinates, while the next first half-kick must use the forces of
// the unscaled ones whether or not anybody asked in between (reading B1): frc is stashed in vel_tmp (free
// outside the rebuild chain; a query cannot trigger a rebuild, the step's own decision consumed the displacement) and
// put back by query_restore() once the caller has read what it wanted from frc.
static int query_forces(md_system *s, bool *stashed) {
  const size_t bytes = 3 * (size_t)s->d.N * sizeof(double);
  *stashed = s->frc_keep && s->forces_valid;
  if (*stashed && cudaMemcpyAsync(s->d.vel_tmp, s->d.frc, bytes, cudaMemcpyDeviceToDevice, s->stream) != cudaSuccess) return MD_ECUDA;
  return forces_sequence(s, true, 0.0);
}
static int query_restore(md_system *s, bool stashed) {
  if (!stashed) return MD_OK;
  return check_cuda(cudaMemcpyAsync(s->d.frc, s->d.vel_tmp, 3 * (size_t)s->d.N * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
}

static void drop_step_graph(md_system *s) {
  for (auto &g : s->sg) {
    if (g.exec) cudaGraphExecDestroy(g.exec);
    if (g.graph) cudaGraphDestroy(g.graph);
    g.exec = nullptr; g.graph = nullptr; g.nsteps = 0;
  }
}

// `nsteps` time steps as ONE CUDA graph (built once per (dt, observables, nsteps), replayed by md_step):
//   k_kick_drift -> { IF(do_rebuild){ clear, bin, 3 x scan, scatter, cell order, re-order, copy back, list } -> k_density -> k_force [-> k_reduce_boxes] } x nsteps
// The force pass of every step but the last also performs the next step's first half-kick, drift and displacement
// check (StepCtl::chain), and the last block of the kernel that ends a drift takes the rebuild decision and sets the
// handle of the following conditional node: a step without a rebuild is two kernel launches, the host never
// synchronises, and the launch latency of a small system is paid once per graph instead of once per step.
// With a barostat (scaling between the steps) nsteps is 1 and nothing is chained.
static int build_step_graph(md_system *s, md_system::StepGraph &sg, double dt, bool obs, int nsteps) {
  // Small systems: a conditional node costs 11-20 us on B200 whether or not its body runs (measured on 864 atoms: 21.8 us
  // per step with an IF node per step, 10.3 us for the same kernels without), more than the two passes together.  There
  // a graph is
  //   k_kick_drift -> { k_density, k_force } x nsteps -> tail -> WHILE(steps left){ head, rebuild chain, done, { k_density, k_force } x nsteps, tail }
  // and every pass is guarded (StepCtl::guard): it runs only if no rebuild is pending and exactly its number of steps
  // is complete, otherwise its blocks return at once.  A graph without a rebuild pays ONE conditional node (not entered);
  // a rebuild makes the remaining passes return at once, and the loop body rebuilds and resumes (a pending rebuild is
  // the only way to have steps left).  Same kernels, same order, same bits as the per-step IF nodes.  Large systems keep
  // those: a skipped pass of 8192 blocks costs 8 us.
  const bool loop = s->d.N <= kLoopGraphMaxAtoms && !obs && !(s->baro_tau > 0.0) && nsteps >= 2 && !getenv("MD_NO_LOOP_GRAPH");
  if (sg.exec && sg.dt == dt && sg.obs == obs && sg.nsteps == nsteps && sg.loop == loop) return MD_OK;
  if (sg.exec) cudaGraphExecDestroy(sg.exec);
  if (sg.graph) cudaGraphDestroy(sg.graph);
  sg.exec = nullptr; sg.graph = nullptr; sg.nsteps = 0;
  const long launches0 = s->launches;
  // captured on a stream of the library's own (the caller's may be the legacy default stream, which cannot capture);
  // nothing executes during capture, and the graph is launched on the caller's stream
  cudaStream_t user = s->stream, st = nullptr;
  if (cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking) != cudaSuccess) {
    const cudaError_t err = cudaGetLastError();
    s->graph_error = err != cudaSuccess ? (int)err : (int)cudaErrorUnknown; s->opt_graph = false;
    return MD_ECUDA;
  }
  s->stream = st;
  cudaGraph_t g = nullptr;
  std::vector<cudaGraphConditionalHandle> cond((size_t)nsteps);
  cudaGraphConditionalHandle loop_cond{};
  bool ok = cudaGraphCreate(&g, 0) == cudaSuccess;
  for (int k = 0; ok && !loop && k < nsteps; ++k) ok = cudaGraphConditionalHandleCreate(&cond[k], g, 0, cudaGraphCondAssignDefault) == cudaSuccess;
  if (ok && loop) ok = cudaGraphConditionalHandleCreate(&loop_cond, g, 0, cudaGraphCondAssignDefault) == cudaSuccess;
  long iter = 0;
  const cudaGraphNode_t *deps = nullptr;
  size_t ndeps = 0;
  cudaGraphNode_t last = nullptr, cnode = nullptr;
  cudaGraph_t tmp = nullptr;
  long fixed = 0, body = 0;
  // the node the stream's next captured work would depend on; ends the capture
  auto end_capture = [&](bool okin) {
    bool o = okin;
    cudaStreamCaptureStatus cs;
#if CUDART_VERSION >= 13000
    if (o) o = cudaStreamGetCaptureInfo(st, &cs, nullptr, nullptr, &deps, nullptr, &ndeps) == cudaSuccess && ndeps == 1;   // + edge data
#else
    if (o) o = cudaStreamGetCaptureInfo(st, &cs, nullptr, nullptr, &deps, &ndeps) == cudaSuccess && ndeps == 1;
#endif
    if (o) last = deps[0];
    return (cudaStreamEndCapture(st, &tmp) == cudaSuccess) && o;
  };
  if (ok) ok = cudaStreamBeginCaptureToGraph(st, g, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    const long l0 = s->launches;
    ok = launch_kick_drift(s, dt, loop ? make_ctl(s, dt, loop_cond, false, false, kGuardReset) : make_ctl(s, dt, cond[0], true, false)) == 0;
    fixed += s->launches - l0;
    ok = end_capture(ok);
  }
  if (ok && loop) {
    // the guarded passes of all steps, then the tail that sets the loop handle, then the while node; its body: head, the
    // rebuild chain, done, the guarded passes again, tail
    auto passes = [&](bool in_body) {
      bool o = true;
      const long l0 = s->launches;
      if (in_body) o = launch_loop_head(s) == 0 && launch_rebuild_body(s) == 0 && launch_rebuild_done(s) == 0;
      for (int k = 0; o && k < nsteps; ++k) {
        const StepCtl ctl = make_ctl(s, dt, loop_cond, false, k + 1 < nsteps, k);
        o = launch_density(s, k) == 0 && launch_force(s, obs, 0.5 * dt, &ctl) == 0;
      }
      if (o) o = launch_loop_tail(s, loop_cond, nsteps) == 0;
      (in_body ? iter : fixed) += s->launches - l0;
      return o;
    };
    ok = cudaStreamBeginCaptureToGraph(st, g, &last, nullptr, 1, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) ok = end_capture(passes(false));
    cudaGraphNodeParams wp = {};
    wp.type = cudaGraphNodeTypeConditional;
    wp.conditional.handle = loop_cond;
    wp.conditional.type = cudaGraphCondTypeWhile;
    wp.conditional.size = 1;
    cudaGraphNode_t wnode = nullptr;
#if CUDART_VERSION >= 13000
    if (ok) ok = cudaGraphAddNode(&wnode, g, &last, nullptr, 1, &wp) == cudaSuccess;
#else
    if (ok) ok = cudaGraphAddNode(&wnode, g, &last, 1, &wp) == cudaSuccess;
#endif
    if (ok) ok = cudaStreamBeginCaptureToGraph(st, wp.conditional.phGraph_out[0], nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) { ok = passes(true); ok = (cudaStreamEndCapture(st, &tmp) == cudaSuccess) && ok; }
    body = 0;
  }
  for (int k = 0; ok && !loop && k < nsteps; ++k) {
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = cond[k];
    cp.conditional.type = cudaGraphCondTypeIf;
    cp.conditional.size = 1;
#if CUDART_VERSION >= 13000
    ok = cudaGraphAddNode(&cnode, g, &last, nullptr, 1, &cp) == cudaSuccess;     // + dependency edge data
#else
    ok = cudaGraphAddNode(&cnode, g, &last, 1, &cp) == cudaSuccess;
#endif
    if (ok) {
      cudaGraph_t bodyg = cp.conditional.phGraph_out[0];
      ok = cudaStreamBeginCaptureToGraph(st, bodyg, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
      if (ok) {
        const long l0 = s->launches;
        ok = launch_rebuild_body(s) == 0;
        body = s->launches - l0;
        ok = (cudaStreamEndCapture(st, &tmp) == cudaSuccess) && ok;
      }
    }
    if (ok) ok = cudaStreamBeginCaptureToGraph(st, g, &cnode, nullptr, 1, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
      const long l0 = s->launches;
      const bool chain = k + 1 < nsteps;
      const StepCtl ctl = make_ctl(s, dt, chain ? cond[k + 1] : cond[k], chain, chain);
      ok = launch_density(s) == 0 && launch_force(s, obs, 0.5 * dt, &ctl) == 0;
      if (ok && s->baro_tau > 0.0) ok = launch_barostat(s, dt) == 0;
      fixed += s->launches - l0;
      ok = end_capture(ok);
    }
  }
  cudaGraphExec_t exec = nullptr;
  if (ok) ok = cudaGraphInstantiate(&exec, g, 0) == cudaSuccess;
  s->launches = launches0;
  s->stream = user;
  cudaStreamDestroy(st);
  if (!ok) {
    // fall back to plain launches (e.g. a driver without conditional nodes): same kernels, same results; the fallback is
    // visible to the caller as md_stats.graph_error != 0 and md_stats.graph_active == 0
    const cudaError_t err = cudaGetLastError();
    s->graph_error = err != cudaSuccess ? (int)err : (int)cudaErrorUnknown;
    if (getenv("MD_DEBUG")) fprintf(stderr, "md: step graph unavailable (%s; %d steps, fixed %ld body %ld, deps %zu)\n", cudaGetErrorString(err), nsteps, fixed, body, ndeps);
    if (g) cudaGraphDestroy(g);
    s->opt_graph = false;
    return MD_ECUDA;
  }
  sg.graph = g; sg.exec = exec; sg.dt = dt; sg.obs = obs; sg.nsteps = nsteps; sg.kernels = (int)fixed; sg.loop = loop; sg.iter_kernels = (int)iter;
  if (!loop) s->body_kernels = (int)body;
  return MD_OK;
}

// The passes that run as half passes depend on three settings (MD_OPT_HALF_LIST, the lanes per atom, the barostat);
// every row holds its owned pairs first whatever the setting, so a change only invalidates the forces.
static void refresh_half(md_system *s) {
  const int h = half_mask(s);
  if (h == s->d.half) return;
  s->d.half = h;
  drop_step_graph(s);
  s->forces_valid = false; s->observables_valid = false; s->frc_keep = false;
}

static int request_rebuild(md_system *s) {
  const int one = 1;
  return check_cuda(cudaMemcpyAsync(&s->d.st->force_rebuild, &one, sizeof(int), cudaMemcpyHostToDevice, s->stream));
}

}  // namespace md

// ================================================================================================
// C ABI
// ================================================================================================
extern "C" {

const char *md_strerror(int e) {
  switch (e) {
    case MD_OK: return "ok";
    case MD_EINVAL: return "invalid argument";
    case MD_EBOX: return "box edge shorter than 3 (cutoff + skin)";
    case MD_EOVERFLOW: return "neighbour-list capacity exceeded";
    case MD_ENONFINITE: return "non-finite coordinate or coincident atoms";
    case MD_ECUDA: return "CUDA error or no device";
    case MD_ESTATE: return "call out of order";
  }
  return "unknown status";
}

const char *md_version(void) { return "paper_1212_6332_b200 0.1 (sm_100a)"; }

const char *md_kernel_name(int c) {
  static const char *names[MD_K_COUNT] = {"bin", "scan", "sort", "reorder", "list", "density", "force", "integrate", "reduce", "force_chained"};
  return (c >= 0 && c < MD_K_COUNT) ? names[c] : "?";
}

int md_workspace_bytes(const md_desc *d, size_t *bytes) {
  Geometry g;
  int rc = geometry(d, g, false);
  if (rc != MD_OK) return rc;
  if (!bytes) return MD_EINVAL;
  *bytes = layout(d, g, nullptr, nullptr);
  return MD_OK;
}

int md_create(const md_desc *d, void *workspace, size_t bytes, md_system **out) {
  Geometry g;
  int rc = geometry(d, g, true);
  if (rc != MD_OK) return rc;
  if (!out || !workspace || !d->positions || !d->types || !d->mass) return MD_EINVAL;
  if (((uintptr_t)workspace & 255) || bytes < layout(d, g, nullptr, nullptr)) return MD_EINVAL;
  if (!on_device(workspace)) return cudaGetLastError() == cudaSuccess ? MD_EINVAL : MD_ECUDA;
  if (d->pot_kind == MD_POT_TBSMA && (!d->A || !d->xi || !d->p || !d->q || !d->r0)) return MD_EINVAL;
  if (d->pot_kind == MD_POT_EAM_TABLE && (!d->f_val || !d->f_der || !d->phi_val || !d->phi_der || !d->F_val || !d->F_der))
    return MD_EINVAL;
  for (int t = 0; t < d->n_types; ++t) if (!(d->mass[t] > 0.0) || !isfinite(d->mass[t])) return MD_EINVAL;

  md_system *s = new (std::nothrow) md_system();
  if (!s) return MD_EINVAL;
  memset(&s->d, 0, sizeof(s->d));
  s->stream = (cudaStream_t)d->stream;
  s->cutoff = d->cutoff; s->skin = d->skin;
  s->have_list = s->forces_valid = s->observables_valid = false;
  s->opt_step_obs = s->opt_profile = false; s->opt_graph = true; s->opt_force_variant = 0; s->opt_half = -1; s->integrator = MD_INT_VERLET; s->gear_ready = false; s->steps = 0; s->launches = 0;
  s->thermo_Te = 0.0; s->thermo_tau = 0.0; s->baro_P0 = 0.0; s->baro_tau = 0.0;
  for (auto &g : s->sg) { g.graph = nullptr; g.exec = nullptr; g.dt = 0.0; g.obs = false; g.loop = false; g.nsteps = 0; g.kernels = 0; g.iter_kernels = 0; }
  s->body_kernels = 0;
  s->graph_error = 0; s->last_step_graph = false; s->frc_keep = false;
  s->side = nullptr; s->ev_fork = nullptr; s->ev_join = nullptr; s->side_ready = false;
  layout(d, g, workspace, s);
  DevSys &o = s->d;
  o.N = d->n_atoms; o.nb = d->n_boxes; o.npb = g.npb; o.nt = d->n_types; o.kind = d->pot_kind;
  const double rl = d->cutoff + d->skin;
  for (int a = 0; a < 3; ++a) {
    o.nc[a] = g.nc[a]; o.L0[a] = d->box[a];
    o.zfine = g.zfine;
  }
  o.rl = rl; o.dyn_box = 0;
  for (int k = 0; k < o.nt * o.nt; ++k) { const double rc = d->pair_cutoff ? d->pair_cutoff[k] : d->cutoff; o.rc2p[k] = rc * rc; }
  o.rc2 = d->cutoff * d->cutoff; o.rin2 = o.rc2; o.rl2 = rl * rl; o.thr2 = (0.5 * d->skin) * (0.5 * d->skin);
  o.tnc = g.tnc; o.ncell = g.ncell; o.cap = g.cap; o.tiles_per_box = g.tiles_per_box;
  for (int t = 0; t < d->n_types; ++t) s->mass_ev[t] = d->mass[t] * kAmuToEvFs2PerA2;
  const size_t N = (size_t)o.N, nt2 = (size_t)o.nt * o.nt;
  cudaStream_t st = s->stream;
  cudaError_t e = cudaMemsetAsync(o.st, 0, sizeof(DevState), st);
  if (e == cudaSuccess) e = cudaMemcpyAsync(o.st->box, d->box, 3 * sizeof(double), cudaMemcpyHostToDevice, st);
  {
    // 2^(j/64), j = 0..63, rounded from long double (64-bit mantissa): the table of exp_scaled() in md_force.cu
    for (int j = 0; j < 64; ++j) s->exp_tab_host[j] = (double)exp2l((long double)j / 64.0L);
    for (int j = 64; j < kExpTabLen; ++j) s->exp_tab_host[j] = 0.0;
    for (int j = 0; j < 16; ++j) s->exp_tab_host[kExp16Off + j] = (double)exp2l((long double)j / 16.0L);
  }
  if (d->pot_kind == MD_POT_TBSMA) {
    bool fold = true;
    for (size_t k = 0; k < nt2; ++k) {
      if (!(d->r0[k] > 0.0)) { delete s; return MD_EINVAL; }
      if (!(d->A[k] > 0.0) || !(d->xi[k] != 0.0)) fold = false;
    }
    o.tb.fold = fold ? 1 : 0;
    for (size_t k = 0; k < nt2; ++k) {
      const double pre_rho = d->xi[k] * d->xi[k], pre_rep = 2.0 * d->A[k];
      const long double K = 64.0L / logl(2.0L);       // exp_scaled() takes its argument in units of ln2/64
      const long double a_rho = 2.0L * d->q[k] + (fold ? logl((long double)pre_rho) : 0.0L), a_rep = (long double)d->p[k] + (fold ? logl((long double)pre_rep) : 0.0L);
      o.tb.b_rho[k] = 2.0 * d->q[k] / d->r0[k]; o.tb.b_rep[k] = d->p[k] / d->r0[k];
      o.tb.ak_rho[k] = (double)(a_rho * K); o.tb.bk_rho[k] = (double)((long double)o.tb.b_rho[k] * K);
      o.tb.ak16_rho[k] = (double)(a_rho * K / 4.0L); o.tb.bk16_rho[k] = (double)((long double)o.tb.b_rho[k] * K / 4.0L);
      o.tb.ak_rep[k] = (double)(a_rep * K); o.tb.bk_rep[k] = (double)((long double)o.tb.b_rep[k] * K);
      o.tb.pre_rho[k] = fold ? 1.0 : pre_rho; o.tb.pre_rep[k] = fold ? 1.0 : pre_rep;
      // exp_scaled() has no overflow handling: its argument must stay well inside +-690 for 0 <= r <= r_c + skin
      const double rmax = d->cutoff + d->skin;
      if (!(fabsl(a_rho) + fabs(o.tb.b_rho[k]) * rmax < 600.0) || !(fabsl(a_rep) + fabs(o.tb.b_rep[k]) * rmax < 600.0)) {
        delete s; return MD_EINVAL;
      }
    }
    for (size_t k = 0; k < nt2; ++k) {
      const double rc = d->pair_cutoff ? d->pair_cutoff[k] : d->cutoff, ron = d->pair_taper_on ? d->pair_taper_on[k] : d->taper_on;
      o.tb.inv_w[k] = 1.0 / (rc - ron); o.tb.t0[k] = -ron * o.tb.inv_w[k]; o.tb.m30_inv_w[k] = -30.0 * o.tb.inv_w[k];
    }
    // loop constants that the passes read from memory into registers (md_force.cu, LoopConsts)
    double *lc = s->exp_tab_host + 64;
    lc[0] = 1.0 / 120.0; lc[1] = 0.375; lc[2] = 6.0; lc[3] = o.tb.inv_w[0]; lc[4] = o.tb.bk_rho[0]; lc[5] = o.tb.bk_rep[0]; lc[6] = 1.0 / 5040.0; lc[7] = o.tb.bk16_rho[0];
  } else {
    TableParams &t = o.tab;
    t.nr = d->nr; t.nrho = d->nrho; t.dr = d->dr; t.inv_dr = 1.0 / d->dr; t.drho = d->drho; t.inv_drho = 1.0 / d->drho;
    t.rho_max = (double)(d->nrho - 1) * d->drho;
    const void *src[6] = {d->f_val, d->f_der, d->phi_val, d->phi_der, d->F_val, d->F_der};
    void *dst[6] = {(void *)t.f_val, (void *)t.f_der, (void *)t.phi_val, (void *)t.phi_der, (void *)t.F_val, (void *)t.F_der};
    for (int k = 0; k < 6 && e == cudaSuccess; ++k)
      e = cudaMemcpyAsync(dst[k], src[k], (k < 4 ? nt2 * d->nr : (size_t)o.nt * d->nrho) * sizeof(double), cudaMemcpyDefault, st);
    if (e == cudaSuccess && launch_prepare_tables(s) != 0) e = cudaErrorUnknown;
  }
  if (e == cudaSuccess) e = cudaMemcpyAsync((void *)o.exp_tab, s->exp_tab_host, sizeof(s->exp_tab_host), cudaMemcpyHostToDevice, st);
  // positions + types (through the staging area when they live on the host)
  const double *xdev = d->positions;
  const int *tdev = d->types;
  if (e == cudaSuccess && !on_device(d->positions)) {
    e = cudaMemcpyAsync(s->stage, d->positions, 3 * N * sizeof(double), cudaMemcpyHostToDevice, st);
    xdev = (const double *)s->stage;
  }
  if (e == cudaSuccess && !on_device(d->types)) {
    e = cudaMemcpyAsync(o.cell_id, d->types, N * sizeof(int), cudaMemcpyHostToDevice, st);   // cell_id is free before the first build
    tdev = o.cell_id;
  }
  if (e == cudaSuccess) {
    ++s->launches, k_init_atoms<<<grid_for(o.N), 256, 0, st>>>(o, xdev, tdev);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) {
    const double *vdev = d->velocities;
    if (vdev && !on_device(vdev)) {
      e = cudaMemcpyAsync(s->stage, vdev, 3 * N * sizeof(double), cudaMemcpyHostToDevice, st);   // stream order: after k_init_atoms
      vdev = (const double *)s->stage;
    }
    if (e == cudaSuccess) { ++s->launches, k_set_vec<<<grid_for(o.N), 256, 0, st>>>(o, o.vel, vdev); e = cudaGetLastError(); }
  }
  if (e == cudaSuccess) e = cudaMemsetAsync(o.frc, 0, 3 * N * sizeof(double), st);
  if (e == cudaSuccess) e = cudaMemsetAsync(o.rho_fix, 0, N * sizeof(long long), st);      // the half passes leave them zero
  if (e == cudaSuccess) e = cudaMemsetAsync(o.frc_fix, 0, 4 * N * sizeof(long long), st);
  int flags = 0;
  if (e != cudaSuccess || sync_and_flags(s, &flags) == MD_ECUDA) { delete s; cudaGetLastError(); return MD_ECUDA; }
  if (flags & (1 << 30)) { delete s; return MD_EINVAL; }   // a type out of range
  s->d.half = half_mask(s);
  *out = s;
  return MD_OK;
}

int md_destroy(md_system *s) {
  if (!s) return MD_OK;
  cudaStreamSynchronize(s->stream);
  for (auto &p : s->prof) for (cudaEvent_t ev : p.ev) cudaEventDestroy(ev);
  if (s->side_ready) { cudaStreamSynchronize(s->side); cudaEventDestroy(s->ev_fork); cudaEventDestroy(s->ev_join); cudaStreamDestroy(s->side); }
  drop_step_graph(s);
  delete s;
  return MD_OK;
}

int md_set_option(md_system *s, int option, int value) {
  if (!s) return MD_EINVAL;
  switch (option) {
    case MD_OPT_STEP_OBSERVABLES: s->opt_step_obs = value != 0; return MD_OK;
    case MD_OPT_PROFILE: s->opt_profile = value != 0; return MD_OK;
    case MD_OPT_GRAPH: s->opt_graph = value != 0; if (value) s->graph_error = 0; return MD_OK;   // switching it on retries a failed build
    case MD_OPT_FORCE_VARIANT:
      if (value < 0 || value > 4 || (value == 3 && s->d.N > kSub32Limit)) return MD_EINVAL;
      s->opt_force_variant = value; drop_step_graph(s); refresh_half(s); return MD_OK;
    case MD_OPT_HALF_LIST:
      if (value < -1 || value > 3) return MD_EINVAL;
      s->opt_half = value; refresh_half(s); return MD_OK;
  }
  return MD_EINVAL;
}

int md_set_integrator(md_system *s, int integrator) {
  if (!s || (integrator != MD_INT_VERLET && integrator != MD_INT_GEAR5)) return MD_EINVAL;
  if (integrator == MD_INT_GEAR5 && (s->thermo_tau > 0.0 || s->baro_tau > 0.0)) return MD_EINVAL;
  if (integrator != s->integrator) { s->integrator = integrator; s->gear_ready = false; s->forces_valid = false; s->observables_valid = false; }
  return MD_OK;
}

int md_set_thermostat(md_system *s, double T_e, double tau) {
  if (!s || !(T_e >= 0.0) || !isfinite(T_e) || !isfinite(tau) || (tau > 0.0 && s->integrator == MD_INT_GEAR5)) return MD_EINVAL;
  s->thermo_Te = T_e; s->thermo_tau = tau;
  drop_step_graph(s);                                // the half-kick parameters are baked into the graph's nodes
  return MD_OK;
}

int md_set_barostat(md_system *s, double P0, double tau_p) {
  if (!s || !isfinite(P0) || !isfinite(tau_p) || (tau_p > 0.0 && (s->d.nb != 1 || s->integrator == MD_INT_GEAR5))) return MD_EINVAL;
  s->baro_P0 = P0; s->baro_tau = tau_p;
  drop_step_graph(s);                                // parameters are baked into the graph's nodes
  if (tau_p > 0.0) s->d.dyn_box = 1;                 // kernels read the box edges from device state from now on
  else if (s->d.dyn_box) {                           // switched off: the current edges become kernel parameters again
    if (cudaMemcpyAsync(s->d.L0, s->d.st->box, 3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
        cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
    s->d.dyn_box = 0;
  }
  refresh_half(s);
  return MD_OK;
}

int md_get_box(md_system *s, double *box) {
  if (!s || !box) return MD_EINVAL;
  if (cudaMemcpyAsync(box, s->d.st->box, 3 * sizeof(double), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA;
  return sync_and_flags(s);
}

int md_get_pressure(md_system *s, double *P) {
  if (!s || !P) return MD_EINVAL;
  int rc;
  if (!s->have_list && (rc = request_rebuild(s)) != MD_OK) return rc;
  bool stashed = false;
  if (!(s->forces_valid && s->observables_valid) && ((rc = query_forces(s, &stashed)) != MD_OK || (rc = query_restore(s, stashed)) != MD_OK)) return rc;
  if (launch_pressure(s) != 0) return MD_ECUDA;
  if (cudaMemcpyAsync(P, &s->d.st->pressure, sizeof(double), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA;
  return sync_and_flags(s);
}

int md_build_neighbors(md_system *s) {
  if (!s) return MD_EINVAL;
  int rc = request_rebuild(s);
  if (rc != MD_OK) return rc;
  if (launch_rebuild_chain(s) != 0) return MD_ECUDA;
  s->have_list = true; s->forces_valid = false; s->observables_valid = false; s->frc_keep = false;
  return MD_OK;
}

int md_compute_forces(md_system *s, double *forces, double *e_atom, double *virial) {
  if (!s) return MD_EINVAL;
  int rc;
  if (!s->have_list && (rc = request_rebuild(s)) != MD_OK) return rc;
  bool stashed = false;
  if ((rc = query_forces(s, &stashed)) != MD_OK) return rc;
  const DevSys &o = s->d;
  bool any_host = false, h;
  double *scratch = (double *)s->stage;
  if (forces) {
    if (on_device(forces)) ++s->launches, k_get_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.frc, forces);
    else {
      ++s->launches, k_get_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.frc, scratch);
      if ((rc = deliver(s, forces, scratch, 3 * (size_t)o.N * sizeof(double), &h)) != MD_OK) return rc;
      any_host = true;
    }
  }
  if ((rc = query_restore(s, stashed)) != MD_OK) return rc;
  if (e_atom) {
    if (on_device(e_atom)) ++s->launches, k_get_scalar<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.eatom, e_atom);
    else {
      ++s->launches, k_get_scalar<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.eatom, scratch);   // stream order: after the copy above
      if ((rc = deliver(s, e_atom, scratch, (size_t)o.N * sizeof(double), &h)) != MD_OK) return rc;
      any_host = true;
    }
  }
  if (virial) {
    if ((rc = deliver(s, virial, o.box_virial, 6 * (size_t)o.nb * sizeof(double), &h)) != MD_OK) return rc;
    any_host |= h;
  }
  if (cudaGetLastError() != cudaSuccess) return MD_ECUDA;
  return any_host ? sync_and_flags(s) : MD_OK;
}

int md_prepare_step(md_system *s, int n, double dt) {
  if (!s || n < 0 || !isfinite(dt)) return MD_EINVAL;
  if (n == 0 || !s->opt_graph || s->opt_profile || s->integrator != MD_INT_VERLET) return MD_OK;
  const bool baro = s->baro_tau > 0.0, obs = s->opt_step_obs || baro;
  const int unroll = baro ? 1 : kStepUnroll, q = n / unroll, r = n % unroll;
  if ((q > 0 && build_step_graph(s, s->sg[0], dt, obs, unroll) != MD_OK) || (r > 0 && build_step_graph(s, s->sg[1], dt, obs, r) != MD_OK))
    return MD_OK;                                      // md_step will run the same kernels as plain launches (md_stats.graph_error says why)
  if (q > 0) cudaGraphUpload(s->sg[0].exec, s->stream);
  if (r > 0) cudaGraphUpload(s->sg[1].exec, s->stream);
  return cudaGetLastError() == cudaSuccess ? MD_OK : MD_ECUDA;
}

int md_step(md_system *s, int n, double dt) {
  if (!s || n < 0 || !isfinite(dt)) return MD_EINVAL;
  int rc;
  if (n == 0) return MD_OK;
  if (!s->have_list && (rc = request_rebuild(s)) != MD_OK) return rc;
  if (s->integrator == MD_INT_GEAR5) {
    // the paper's predictor-corrector (md_gear.cu): predict + displacement check, conditional rebuild, density, force at the
    // predicted positions, correct; plain launches
    if (!s->gear_ready) {
      if ((rc = forces_sequence(s, false, 0.0)) != MD_OK) return rc;
      if (launch_gear_start(s, dt) != 0) return MD_ECUDA;
      s->gear_ready = true;
    }
    for (int k = 0; k < n; ++k)
      if (launch_gear_predict(s, dt) != 0 || launch_rebuild_body(s) != 0 || launch_density(s) != 0 || launch_force(s, s->opt_step_obs, 0.0) != 0 ||
          launch_gear_correct(s, dt) != 0) return MD_ECUDA;
    s->last_step_graph = false;
    s->forces_valid = false; s->observables_valid = false; s->frc_keep = false;   // frc belongs to the predicted positions: queries evaluate the corrected ones
    s->steps += n;
    return MD_OK;
  }
  if (!s->forces_valid && (rc = forces_sequence(s, s->opt_step_obs, 0.0)) != MD_OK) return rc;
  const bool baro = s->baro_tau > 0.0;
  const bool obs = s->opt_step_obs || baro;          // the barostat needs the virial of every step
  const int unroll = baro ? 1 : kStepUnroll;         // steps per graph launch (chained: no scaling in between)
  const int q = n / unroll, r = n % unroll;
  cudaGraphConditionalHandle none{};
  if (s->opt_graph && !s->opt_profile && (q == 0 || build_step_graph(s, s->sg[0], dt, obs, unroll) == MD_OK) &&
      (r == 0 || build_step_graph(s, s->sg[1], dt, obs, r) == MD_OK)) {
    for (int k = 0; k < q; ++k)
      if (cudaGraphLaunch(s->sg[0].exec, s->stream) != cudaSuccess) return MD_ECUDA;
    if (r && cudaGraphLaunch(s->sg[1].exec, s->stream) != cudaSuccess) return MD_ECUDA;
    s->launches += (long)q * s->sg[0].kernels + (r ? s->sg[1].kernels : 0);
    s->have_list = true; s->forces_valid = true; s->observables_valid = obs && !baro;
    s->last_step_graph = true;
  } else {
    // the same kernels in the same order as plain launches: every kernel of the rebuild chain is launched in every step
    // and returns at once unless the decision (taken by the last block of the preceding drift) says otherwise
    s->last_step_graph = false;
    for (int k0 = 0; k0 < n; k0 += unroll) {
      const int m = n - k0 < unroll ? n - k0 : unroll;
      if (launch_kick_drift(s, dt, make_ctl(s, dt, none, false, false)) != 0) return MD_ECUDA;
      for (int j = 0; j < m; ++j) {
        const StepCtl ctl = make_ctl(s, dt, none, false, j + 1 < m);
        if (launch_rebuild_body(s) != 0 || launch_density(s) != 0 || launch_force(s, obs, 0.5 * dt, &ctl) != 0) return MD_ECUDA;
        if (baro && launch_barostat(s, dt) != 0) return MD_ECUDA;
      }
    }
    s->have_list = true; s->forces_valid = true; s->observables_valid = obs && !baro;   // with a barostat: energies and virial on request belong to the scaled positions
  }
  s->frc_keep = baro;
  s->steps += n;
  return MD_OK;
}

int md_get_positions(md_system *s, double *x) {
  if (!s || !x) return MD_EINVAL;
  const DevSys &o = s->d;
  if (on_device(x)) { ++s->launches, k_get_pos<<<grid_for(o.N), 256, 0, s->stream>>>(o, x); return check_cuda(cudaGetLastError()); }
  ++s->launches, k_get_pos<<<grid_for(o.N), 256, 0, s->stream>>>(o, (double *)s->stage);
  int rc = deliver(s, x, s->stage, 3 * (size_t)o.N * sizeof(double), nullptr);
  return rc != MD_OK ? rc : sync_and_flags(s);
}

int md_get_velocities(md_system *s, double *v) {
  if (!s || !v) return MD_EINVAL;
  const DevSys &o = s->d;
  if (on_device(v)) { ++s->launches, k_get_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.vel, v); return check_cuda(cudaGetLastError()); }
  ++s->launches, k_get_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.vel, (double *)s->stage);
  int rc = deliver(s, v, s->stage, 3 * (size_t)o.N * sizeof(double), nullptr);
  return rc != MD_OK ? rc : sync_and_flags(s);
}

int md_set_positions(md_system *s, const double *x) {
  if (!s || !x) return MD_EINVAL;
  const DevSys &o = s->d;
  const double *src = x;
  if (!on_device(x)) {
    if (cudaMemcpyAsync(s->stage, x, 3 * (size_t)o.N * sizeof(double), cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return MD_ECUDA;
    src = (const double *)s->stage;
  }
  ++s->launches, k_set_pos<<<grid_for(o.N), 256, 0, s->stream>>>(o, src, s->have_list ? 1 : 0);
  s->forces_valid = false; s->observables_valid = false; s->frc_keep = false; s->gear_ready = false;
  if (src != x && cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;   // the host buffer may be reused
  return check_cuda(cudaGetLastError());
}

int md_set_state(md_system *s, const double *x, const double *v) {
  if (!s || (!x && !v)) return MD_EINVAL;
  const DevSys &o = s->d;
  const size_t bytes = 3 * (size_t)o.N * sizeof(double);
  const double *xs = x, *vs = v;
  bool host = false;
  if (x && !on_device(x)) {
    if (cudaMemcpyAsync(s->stage, x, bytes, cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return MD_ECUDA;
    xs = (const double *)s->stage; host = true;
  }
  if (v && !on_device(v)) {
    if (cudaMemcpyAsync((char *)s->stage + bytes, v, bytes, cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return MD_ECUDA;
    vs = (const double *)((char *)s->stage + bytes); host = true;
  }
  int *flag = o.scan_block;                            // free outside the rebuild chain
  s->gear_ready = false;
  if (cudaMemsetAsync(flag, 0, sizeof(int), s->stream) != cudaSuccess) return MD_ECUDA;
  ++s->launches, k_set_state<<<grid_for(o.N), 256, 0, s->stream>>>(o, xs, vs, s->have_list ? 1 : 0, flag);
  if (cudaGetLastError() != cudaSuccess) return MD_ECUDA;
  if (!x) return host && cudaStreamSynchronize(s->stream) != cudaSuccess ? MD_ECUDA : MD_OK;
  // the forces stay valid if no coordinate changed: that takes one look at the flag (and the host buffers may be reused)
  int changed = 1;
  if (cudaMemcpyAsync(&changed, flag, sizeof(int), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
      cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
  if (changed) { s->forces_valid = false; s->observables_valid = false; s->frc_keep = false; }
  return MD_OK;
}

int md_get_state(md_system *s, double *x, double *v) {
  if (!s || (!x && !v)) return MD_EINVAL;
  const DevSys &o = s->d;
  const size_t bytes = 3 * (size_t)o.N * sizeof(double);
  bool host = false;
  if (x) {
    const bool dev = on_device(x);
    double *dst = dev ? x : (double *)s->stage;
    ++s->launches, k_get_pos<<<grid_for(o.N), 256, 0, s->stream>>>(o, dst);
    if (!dev) { host = true; if (cudaMemcpyAsync(x, dst, bytes, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA; }
  }
  if (v) {
    const bool dev = on_device(v);
    double *dst = dev ? v : (double *)((char *)s->stage + bytes);
    ++s->launches, k_get_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.vel, dst);
    if (!dev) { host = true; if (cudaMemcpyAsync(v, dst, bytes, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA; }
  }
  if (cudaGetLastError() != cudaSuccess) return MD_ECUDA;
  return host ? sync_and_flags(s) : MD_OK;
}

// n steps and the state after them in one call.  The positions of step n are final after its drift (and the rebuild, which
// re-orders them), while its two passes only produce the forces for the second half-kick: their gather into caller order
// and their copy to the host run on a second stream BESIDE the density and the force pass of the last step (25 MB and
// ~0.47 ms each for 1,048,576 atoms: the download of x disappears behind the passes).  Same kernels, same order, same bits as
// md_step(n) followed by md_get_state; the last step is launched plainly (the fork sits between two kernels of a step).
int md_step_get_state(md_system *s, int n, double dt, double *x, double *v) {
  if (!s || n < 1 || !isfinite(dt) || (!x && !v)) return MD_EINVAL;
  int rc;
  // below ~0.26 M atoms the copy is shorter than what the plainly launched step costs more than its CUDA graph (864 atoms: 0.124
  // against 0.101 ms per step end to end); MD_FORK_MIN_ATOMS overrides the threshold (tests)
  const char *env = getenv("MD_FORK_MIN_ATOMS");
  const long fork_min = env ? atol(env) : 262144;
  const bool fork = x && !on_device(x) && s->integrator == MD_INT_VERLET && !(s->baro_tau > 0.0) && !s->opt_profile && s->d.N >= fork_min;
  if (!fork) return (rc = md_step(s, n, dt)) != MD_OK ? rc : md_get_state(s, x, v);
  if (n > 1 && (rc = md_step(s, n - 1, dt)) != MD_OK) return rc;
  if (!s->have_list && (rc = request_rebuild(s)) != MD_OK) return rc;
  if (!s->forces_valid && (rc = forces_sequence(s, s->opt_step_obs, 0.0)) != MD_OK) return rc;
  if (!s->side_ready) {
    int lo = 0, hi = 0;
    if (cudaDeviceGetStreamPriorityRange(&lo, &hi) != cudaSuccess || cudaStreamCreateWithPriority(&s->side, cudaStreamNonBlocking, hi) != cudaSuccess)
      return MD_ECUDA;
    if (cudaEventCreateWithFlags(&s->ev_fork, cudaEventDisableTiming) != cudaSuccess || cudaEventCreateWithFlags(&s->ev_join, cudaEventDisableTiming) != cudaSuccess)
      return MD_ECUDA;
    s->side_ready = true;
  }
  const DevSys &o = s->d;
  const size_t bytes = 3 * (size_t)o.N * sizeof(double);
  const bool obs = s->opt_step_obs;
  cudaGraphConditionalHandle none{};
  const StepCtl ctl = make_ctl(s, dt, none, false, false);
  if (launch_kick_drift(s, dt, ctl) != 0 || launch_rebuild_body(s) != 0) return MD_ECUDA;
  if (cudaEventRecord(s->ev_fork, s->stream) != cudaSuccess || cudaStreamWaitEvent(s->side, s->ev_fork, 0) != cudaSuccess) return MD_ECUDA;
  ++s->launches, k_get_pos<<<grid_for(o.N), 256, 0, s->side>>>(o, (double *)s->stage);
  if (cudaMemcpyAsync(x, s->stage, bytes, cudaMemcpyDeviceToHost, s->side) != cudaSuccess || cudaEventRecord(s->ev_join, s->side) != cudaSuccess) return MD_ECUDA;
  if (launch_density(s) != 0 || launch_force(s, obs, 0.5 * dt, &ctl) != 0) return MD_ECUDA;
  s->have_list = true; s->forces_valid = true; s->observables_valid = obs; s->last_step_graph = false; s->frc_keep = false;
  s->steps += 1;
  if (v) {
    const bool dev = on_device(v);
    double *dst = dev ? v : (double *)((char *)s->stage + bytes);
    ++s->launches, k_get_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.vel, dst);
    if (!dev && cudaMemcpyAsync(v, dst, bytes, cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA;
  }
  if (cudaStreamWaitEvent(s->stream, s->ev_join, 0) != cudaSuccess || cudaGetLastError() != cudaSuccess) return MD_ECUDA;
  return sync_and_flags(s);
}

int md_set_velocities(md_system *s, const double *v) {
  if (!s || !v) return MD_EINVAL;
  const DevSys &o = s->d;
  const double *src = v;
  if (!on_device(v)) {
    if (cudaMemcpyAsync(s->stage, v, 3 * (size_t)o.N * sizeof(double), cudaMemcpyHostToDevice, s->stream) != cudaSuccess) return MD_ECUDA;
    src = (const double *)s->stage;
  }
  ++s->launches, k_set_vec<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.vel, src);
  s->gear_ready = false;
  if (src != v && cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
  return check_cuda(cudaGetLastError());
}

int md_get_neighbors(md_system *s, int *count, int *list, int stride) {
  if (!s || !count || !list || stride <= 0) return MD_EINVAL;
  if (!s->have_list) return MD_ESTATE;
  const DevSys &o = s->d;
  const bool dev = on_device(list);
  if (dev != on_device(count)) return MD_EINVAL;       // both on the same side
  int *flag = o.scan_block;                            // free outside the rebuild chain
  if (cudaMemsetAsync(flag, 0, sizeof(int), s->stream) != cudaSuccess) return MD_ECUDA;
  ++s->launches, k_invert_orig<<<grid_for(o.N), 256, 0, s->stream>>>(o);
  if (dev) {
    ++s->launches, k_export_neighbors<<<grid_for(o.N, 128), 128, 0, s->stream>>>(o, 0, o.N, count, list, stride, flag);
  } else {
    // chunks of caller atoms that fit the staging area: [chunk] counts followed by [chunk][stride] rows
    const size_t per_atom = ((size_t)stride + 1) * sizeof(int);
    const int chunk = (int)(s->stage_bytes / per_atom < (size_t)o.N ? s->stage_bytes / per_atom : (size_t)o.N);
    if (chunk < 1) return MD_EINVAL;
    int *dcount = (int *)s->stage, *dlist = dcount + chunk;
    for (int first = 0; first < o.N; first += chunk) {
      const int na = o.N - first < chunk ? o.N - first : chunk;
      ++s->launches, k_export_neighbors<<<grid_for(na, 128), 128, 0, s->stream>>>(o, first, na, dcount, dlist, stride, flag);
      if (cudaMemcpyAsync(count + first, dcount, (size_t)na * sizeof(int), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess ||
          cudaMemcpyAsync(list + (size_t)first * stride, dlist, (size_t)na * stride * sizeof(int), cudaMemcpyDeviceToHost,
                          s->stream) != cudaSuccess)
        return MD_ECUDA;
    }
  }
  int over = 0;
  if (cudaMemcpyAsync(&over, flag, sizeof(int), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA;
  int rc = sync_and_flags(s);
  if (rc != MD_OK) return rc;
  return over ? MD_EOVERFLOW : MD_OK;
}

int md_get_densities(md_system *s, double *rho, double *fprime) {
  if (!s) return MD_EINVAL;
  if (!s->forces_valid) return MD_ESTATE;
  const DevSys &o = s->d;
  int rc;
  bool any_host = false;
  double *scratch = (double *)s->stage;
  if (rho) {
    if (on_device(rho)) ++s->launches, k_get_scalar<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.rho, rho);
    else {
      ++s->launches, k_get_scalar<<<grid_for(o.N), 256, 0, s->stream>>>(o, o.rho, scratch);
      if ((rc = deliver(s, rho, scratch, (size_t)o.N * sizeof(double), nullptr)) != MD_OK) return rc;
      any_host = true;
    }
  }
  if (fprime) {
    if (on_device(fprime)) ++s->launches, k_get_fprime<<<grid_for(o.N), 256, 0, s->stream>>>(o, fprime);
    else {
      ++s->launches, k_get_fprime<<<grid_for(o.N), 256, 0, s->stream>>>(o, scratch);
      if ((rc = deliver(s, fprime, scratch, (size_t)o.N * sizeof(double), nullptr)) != MD_OK) return rc;
      any_host = true;
    }
  }
  if (cudaGetLastError() != cudaSuccess) return MD_ECUDA;
  return any_host ? sync_and_flags(s) : MD_OK;
}

int md_get_energies(md_system *s, double *epot, double *ekin) {
  if (!s) return MD_EINVAL;
  int rc;
  const DevSys &o = s->d;
  if (epot) {
    if (!s->have_list && (rc = request_rebuild(s)) != MD_OK) return rc;
    bool stashed = false;
    if (!(s->forces_valid && s->observables_valid) && ((rc = query_forces(s, &stashed)) != MD_OK || (rc = query_restore(s, stashed)) != MD_OK)) return rc;
    if ((rc = deliver(s, epot, o.box_epot, (size_t)o.nb * sizeof(double), nullptr)) != MD_OK) return rc;
  }
  if (ekin) {
    if (launch_ekin(s) != 0) return MD_ECUDA;
    if ((rc = deliver(s, ekin, o.box_ekin, (size_t)o.nb * sizeof(double), nullptr)) != MD_OK) return rc;
  }
  return sync_and_flags(s);
}

int md_get_stats(md_system *s, md_stats *out) {
  if (!s || !out) return MD_EINVAL;
  DevState st;
  if (cudaMemcpyAsync(&st, s->d.st, sizeof(st), cudaMemcpyDeviceToHost, s->stream) != cudaSuccess) return MD_ECUDA;
  if (cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
  out->steps = s->steps; out->rebuilds = (long)st.rebuilds; out->max_neighbors = st.max_neighbors;
  out->error_flags = st.error_flags; out->last_max_disp2 = st.last_maxd2; out->neighbor_capacity = s->d.cap; out->kernel_launches = s->launches + (long)st.graph_body_runs * s->body_kernels +
                                                                                                                                           (long)st.loop_iters * (s->sg[0].loop ? s->sg[0].iter_kernels : s->sg[1].iter_kernels); out->list_entries = (long)st.list_entries;
  out->graph_active = s->last_step_graph ? 1 : 0; out->graph_error = s->graph_error;
  return MD_OK;
}

int md_profile_reset(md_system *s) {
  if (!s) return MD_EINVAL;
  if (cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
  for (auto &p : s->prof) { p.used = 0; p.dropped = 0; }
  return MD_OK;
}

int md_profile_read(md_system *s, int cls, long *launches, double *total_ms) {
  if (!s || cls < 0 || cls >= MD_K_COUNT) return MD_EINVAL;
  if (cudaStreamSynchronize(s->stream) != cudaSuccess) return MD_ECUDA;
  const ProfClass &p = s->prof[cls];
  double tot = 0.0;
  for (size_t k = 0; k + 1 < p.used; k += 2) {
    float ms = 0.f;
    if (cudaEventElapsedTime(&ms, p.ev[k], p.ev[k + 1]) != cudaSuccess) return MD_ECUDA;
    tot += ms;
  }
  if (launches) *launches = (long)(p.used / 2);
  if (total_ms) *total_ms = tot;
  return MD_OK;
}

}  // extern "C"
