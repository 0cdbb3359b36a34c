/* md.h — C ABI of the B200-native EAM / TB-SMA molecular-dynamics hot path.
 *
 * Method: Hou et al., "Molecular dynamics simulations with many-body potentials on multiple
 * GPUs - the implementation, package and performance", arxiv 1212.6332.  Citations below are
 * PAPER.md:<line> of the extracted text plus the section / equation / figure.
 *
 *   E_i = F(sum_j rho(r_ij)) + 1/2 sum_j V(r_ij)                          eq.(1)
 *   f_i = -sum_j [F'(rho_i)+F'(rho_j)] rho'(r_ij) r_ij/r_ij - sum_j V'(r_ij) r_ij/r_ij   eq.(3)
 *
 * evaluated on one GPU by: cell binning + re-ordering into cell order (sec. 3.2, PAPER.md:137-145,
 * done there on the host, here on the device), a full Verlet neighbour list over the 27-cell
 * stencil (Fig.3), a density pass (Fig.5), a
 * force pass with virial (Fig.6) and a time integrator (sec. 3.3; here
 * velocity-Verlet with a skin/2 displacement-triggered rebuild instead of the paper's fixed
 * 10-step interval), optionally for many independent periodic boxes packed into
 * one system (sec. 4.4).
 *
 * GENERAL CONVENTIONS
 *  - Units: eV, Angstrom, fs, amu.  All floating point is IEEE double, all indices int32.
 *  - Every function returns an int status: MD_OK (0) or a negative MD_E* code.  Nothing
 *    throws or aborts across this boundary.  md_strerror() gives text.
 *  - POINTERS.  Every array argument may be a DEVICE pointer (e.g. a torch CUDA tensor's
 *    data_ptr()) or a HOST pointer (pageable or pinned); the library asks the CUDA runtime
 *    which (cudaPointerGetAttributes) and stages host buffers through its workspace with
 *    cudaMemcpyAsync on the system's stream.  Calls that take a host pointer synchronise the
 *    stream before returning; calls with device pointers only enqueue work.  md_desc.mass and the
 *    TB-SMA parameter arrays are always HOST (a few doubles).
 *  - OWNERSHIP.  md_create copies every input; the caller keeps its buffers.  Outputs are
 *    written into caller-provided buffers; any output pointer may be NULL (= skip).
 *    The library never allocates device memory: the caller provides ONE workspace allocation
 *    of md_workspace_bytes() bytes (256-byte aligned) that must outlive the system.
 *  - ORDER.  Inputs and outputs are in CALLER atom order, AoS [n_atoms][3]; internally atoms
 *    are kept in cell order (the paper's hGID map).  With n_boxes > 1, box b owns
 *    atoms [b*n_atoms/n_boxes, (b+1)*n_atoms/n_boxes).
 *  - STREAM.  All work is enqueued on md_desc.stream (a cudaStream_t; NULL = legacy default).
 *  - ERRORS found on the device (neighbour overflow, non-finite coordinate, coincident atoms)
 *    are sticky flags returned by the next call that synchronises: md_get_stats, any getter
 *    into host memory, md_get_energies.
 *  - There is no CPU fallback: without a CUDA device every compute entry point returns MD_ECUDA.
 */
#ifndef PAPER_1212_6332_B200_MD_H
#define PAPER_1212_6332_B200_MD_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

enum {
  MD_OK = 0,
  MD_EINVAL = -1,      /* bad argument (NULL, size <= 0, type out of range, workspace too small ...) */
  MD_EBOX = -2,        /* some L_a < 3 (cutoff+skin): the 27-cell stencil would alias */
  MD_EOVERFLOW = -3,   /* an atom has more neighbours than the list capacity (the paper's MN) */
  MD_ENONFINITE = -4,  /* NaN/Inf coordinate, or two atoms at the same point */
  MD_ECUDA = -5,       /* CUDA runtime error, or no device */
  MD_ESTATE = -6       /* call out of order (e.g. md_get_neighbors before any build) */
};

/* bits of md_stats.error_flags */
enum { MD_FLAG_OVERFLOW = 1, MD_FLAG_NONFINITE = 2, MD_FLAG_BOX = 4 /* barostat shrank a cell below cutoff + skin */ };

enum { MD_POT_TBSMA = 0, MD_POT_EAM_TABLE = 1 };
enum { MD_MAX_TYPES = 4 };

typedef struct md_system md_system; /* opaque; lives in host memory, owned by the library */

typedef struct {
  int n_atoms, n_boxes, n_types;  /* n_boxes = 1: one box.  > 1: batched mode, n_atoms = total, equal
                                     atoms per box.  1 <= n_types <= MD_MAX_TYPES.  n_atoms <= 2^26. */
  double box[3];                  /* orthorhombic edge lengths, all periodic; the same for every box of a batch */
  double cutoff, skin;            /* r_c and the Verlet skin; the list holds pairs with r < r_c + skin */
  const double *positions;        /* [n_atoms][3]; any real values (wrapped into the box at every build) */
  const double *velocities;       /* [n_atoms][3] Angstrom/fs, or NULL (= 0) */
  const int *types;               /* [n_atoms], each in [0, n_types) */
  const double *mass;             /* [n_types] amu, HOST */
  int pot_kind;                   /* MD_POT_TBSMA or MD_POT_EAM_TABLE */
  /* MD_POT_TBSMA: second-moment tight binding, F(rho) = -sqrt(rho), per type pair
   * [n_types*n_types], HOST:  rho(r) = xi^2 exp(-2q(r/r0-1)) S(r),  V(r) = 2A exp(-p(r/r0-1)) S(r),
   * S = quintic switch from 1 at taper_on to 0 at cutoff (taper_on < cutoff). */
  const double *A, *xi, *p, *q, *r0;
  double taper_on;
  /* MD_POT_EAM_TABLE: look-up tables "created once on a CPU and copied to the device".
   * Uniform grids, node VALUES and node SLOPES; evaluation is the cubic Hermite interpolant and, for the
   * force, the derivative of that same interpolant.  r_k = k*dr, k < nr, r_{nr-1} >= cutoff;
   * rho_k = k*drho, k < nrho; above rho_{nrho-1} F continues linearly. */
  int nr;
  double dr;
  const double *f_val, *f_der, *phi_val, *phi_der; /* [n_types*n_types][nr]: rho(r) and V(r) per type pair */
  int nrho;
  double drho;
  const double *F_val, *F_der;                     /* [n_types][nrho] */
  int max_neighbors;              /* list capacity per atom (the paper's MN); 0 = chosen from the number density */
  void *stream;                   /* cudaStream_t */
  /* Optional per-pair cut-offs, the paper's RCUT(ity,jty), [n_types*n_types], HOST, symmetric,
   * NULL = `cutoff` / `taper_on` for every pair.  pair_cutoff[ab] <= cutoff: a pair of types (a,b) contributes only
   * for r < pair_cutoff[ab] (the list still holds every pair within cutoff + skin).  MD_POT_TBSMA: the switch of
   * pair (a,b) runs from pair_taper_on[ab] (< pair_cutoff[ab]) to pair_cutoff[ab]. */
  const double *pair_cutoff, *pair_taper_on;
} md_desc;

typedef struct {
  long steps, rebuilds;           /* time steps taken; neighbour builds done (explicit and displacement-triggered) */
  int max_neighbors;              /* largest list length seen at the last build */
  int error_flags;                /* MD_FLAG_* bits, sticky */
  double last_max_disp2;          /* max_i |x_i - x_ref,i|^2 at the last displacement check (Angstrom^2) */
  int neighbor_capacity;          /* list capacity per atom in use */
  long kernel_launches;           /* CUDA kernels this system has enqueued since md_create (host-side count) */
  long list_entries;              /* sum over atoms of the list lengths of the last build (directed pairs) */
  int graph_active;               /* 1: the last md_step replayed its CUDA graphs (MD_OPT_GRAPH); 0: plain launches */
  int graph_error;                /* cudaError_t of a failed graph build (0: none).  md_step then runs the same kernels as
                                     plain launches for the life of the system (or until MD_OPT_GRAPH is set to 1 again) */
} md_stats;

/* Bytes of device workspace md_create needs for this description.  No pointer in *d is read (they may be NULL or
 * not yet valid); the per-pair arrays pair_cutoff / pair_taper_on are validated by md_create. */
int md_workspace_bytes(const md_desc *d, size_t *bytes);

/* Build a system: copies positions/velocities/types/potential into the workspace (device pointer,
 * 256-byte aligned, `bytes` >= md_workspace_bytes).  No neighbour list exists yet.  *out is set only on MD_OK.
 * Errors: MD_EINVAL, MD_EBOX (some L_a < 3 (cutoff+skin)), MD_ECUDA. */
int md_create(const md_desc *d, void *workspace, size_t bytes, md_system **out);
int md_destroy(md_system *s);

/* Sec. 3.2 / Fig.3 on the device: wrap into the box, cell index, histogram, scan, scatter into cell order
 * (deterministic: ties inside a cell ordered by caller index), re-order positions/velocities/types, build
 * the full neighbour list { j != i, same box : |r_ij|^2 < (cutoff+skin)^2 } with the minimum image
 * d = x_j - x_i; if (d > L/2) d -= L; else if (d < -L/2) d += L; r2 = (dx*dx + dy*dy) + dz*dz, every
 * operation rounded once (no FMA), and record x_ref <- x.  Invalidates forces. */
int md_build_neighbors(md_system *s);

/* Fig.5 then Fig.6: densities rho_i and F'(rho_i), then forces (eq.3), per-atom energies (eq.1) and the
 * virial W^{ab} = 1/2 sum_i sum_j (r_i - r_j)^a f_ij^b per box, components xx,yy,zz,xy,xz,yz.
 * Builds the list first if there is none or if some atom moved more than skin/2 since the last build.
 *   forces [n_atoms][3] eV/A, e_atom [n_atoms] eV, virial [n_boxes][6] eV; each may be NULL. */
int md_compute_forces(md_system *s, double *forces, double *e_atom, double *virial);

/* n velocity-Verlet steps of dt fs:  v += (dt/2m) f;  x += dt v;  if max_i |x_i - x_ref,i|^2 > (skin/2)^2
 * rebuild (one flag for the whole batch);  f = force(x);  v += (dt/2m) f.  Forces are evaluated once before
 * the first step if they are stale.  Nothing crosses the host/device boundary inside the call; the rebuild
 * decision is taken on the device. */
int md_step(md_system *s, int n, double dt);
/* Optional: build, instantiate and upload the CUDA graphs that md_step(n, dt) will replay, without taking a step (set-up
 * work of a few milliseconds that md_step otherwise does on the first call with a new (n mod 8, dt)).  No effect with
 * MD_OPT_GRAPH 0, MD_OPT_PROFILE 1 or MD_INT_GEAR5. */
int md_prepare_step(md_system *s, int n, double dt);

/* Integrator.  MD_INT_VERLET (default): velocity-Verlet as described at md_step.  MD_INT_GEAR5: the paper's
 * predictor-corrector scheme (sec. 3.3), taken as the five-value Gear scheme (the paper gives
 * neither order nor coefficients): per step  predict x, v, a, j, s by their Taylor series;  skin/2 rule on the predicted
 * positions;  f = force(x_p);  D = dt^2/2 (f/m - a_p);  x += 19/120 D, v += 3/4 D/dt, a += D 2/dt^2, j += 1/2 D 6/dt^3,
 * s += 1/12 D 24/dt^4.  The first step after md_create / md_set_* takes a = f(x)/m and j, s from central differences of
 * a along x(+-dt/10) (two more force evaluations).  Positions returned are the corrected ones.  No thermostat and no
 * barostat with MD_INT_GEAR5 (MD_EINVAL either way round); its steps are plain kernel launches. */
enum { MD_INT_VERLET = 0, MD_INT_GEAR5 = 1 };
int md_set_integrator(md_system *s, int integrator);

/* Electron-bath thermostat of eq.(4) (Finnis et al.):  m dv/dt = f - (m/tau)((T_i - T_e)/T_i) v  with the
 * per-atom instantaneous temperature T_i = m |v|^2 / (3 k_B).  T_e in K, tau in fs (a time: the printed 1/tau_T stands
 * for m_i/tau_T); tau <= 0 switches it off (default).  Inside md_step each half-kick becomes
 * v += (dt/2)(f/m - (1/tau)(1 - 3 k_B T_e/(m |v|^2)) v), the damping taken from the velocity the half-kick starts from,
 * and 0 for an atom at rest.  Returns MD_EINVAL for T_e < 0 or non-finite arguments. */
int md_set_thermostat(md_system *s, double T_e, double tau);

/* Berendsen barostat of eq.(5)-(6): at the end of every step of md_step the coordinates and the box
 * edges are scaled by mu = [1 - (dt/tau_p)(P0 - P)]^(1/3), P = (2/3 E_kin + 1/3 (W_xx + W_yy + W_zz)) / V from the force
 * evaluation of that step (which then always computes the observables).  P0 in eV/A^3, tau_p in fs eV/A^3 (it absorbs
 * the compressibility); tau_p <= 0 switches it off (default).  One box only (MD_EINVAL for n_boxes > 1).  The cell grid
 * keeps the number of cells chosen at md_create: if the box shrinks until a cell is thinner than cutoff + skin the
 * sticky flag MD_FLAG_BOX is raised and the next synchronising call returns MD_EBOX.  x_ref is not scaled, so the
 * skin/2 rebuild rule also sees the displacement caused by the scaling. */
int md_set_barostat(md_system *s, double P0, double tau_p);
int md_get_box(md_system *s, double *box /* [3] host */);                /* current box edges; synchronises */
int md_get_pressure(md_system *s, double *P /* host, eV/A^3 */);         /* eq.(6) for the current state; synchronises */

int md_get_positions(md_system *s, double *x);        /* [n_atoms][3]; as wrapped at the last build plus drift since */
int md_get_velocities(md_system *s, double *v);       /* [n_atoms][3] */
int md_set_positions(md_system *s, const double *x);  /* keeps the list if no atom is farther than skin/2 from x_ref */
int md_set_velocities(md_system *s, const double *v);
/* Positions and velocities in one call (either may be NULL = skip): one kernel, and for host buffers one
 * synchronisation instead of two.  md_set_state leaves an atom whose uploaded coordinates are bit-identical to the
 * resident ones untouched, and keeps the forces valid if NO coordinate changed (so a caller that only edits
 * velocities, or echoes a state back, does not pay for a force evaluation); it synchronises even for device pointers
 * when x is given (it reads that flag). */
int md_set_state(md_system *s, const double *x, const double *v);
int md_get_state(md_system *s, double *x, double *v);
/* md_step(n, dt) and md_get_state(x, v) in one call (sec. 3.3; n >= 1, x or v may be NULL): the same
 * kernels in the same order and the same results, bit for bit.  When x is a host buffer (pinned, for the copy to be
 * asynchronous) the positions of the last step are gathered and copied on a second stream right after its drift and
 * rebuild, beside its density and force pass, which only the velocities wait for; below 262,144 atoms (where the copy is
 * shorter than the launch overhead it hides behind; environment variable MD_FORK_MIN_ATOMS), with a barostat, the
 * predictor-corrector integrator or MD_OPT_PROFILE it is md_step followed by md_get_state.  Creates one stream and two
 * events at its first forked call (no device memory); synchronises. */
int md_step_get_state(md_system *s, int n, double dt, double *x, double *v);
/* Test hook: the list as ORIGINAL (caller) indices, ascending per atom.  count [n_atoms], list [n_atoms][stride]
 * (each row padded with -1); MD_ESTATE before the first build, MD_EOVERFLOW if some count exceeds stride. */
int md_get_neighbors(md_system *s, int *count, int *list, int stride);
/* Test hook: rho_i and F'(rho_i) of the last force evaluation, [n_atoms] each (either may be NULL). */
int md_get_densities(md_system *s, double *rho, double *fprime);
/* Potential and kinetic energy per box, [n_boxes] each (either may be NULL); evaluates forces if stale. Synchronises. */
int md_get_energies(md_system *s, double *epot, double *ekin);
int md_get_stats(md_system *s, md_stats *st);         /* synchronises */

/* Options (all default 0):
 *  MD_OPT_STEP_OBSERVABLES  1: every force evaluation inside md_step also accumulates per-atom energy and the
 *                              virial (the paper's force kernel with pressure); 0: forces only
 *                              (the paper's full-MD runs).  md_compute_forces always computes them.
 *  MD_OPT_PROFILE           1: bracket every kernel launch with CUDA events on the system's stream so that
 *                              md_profile_read can report per-kernel device time.
 *  MD_OPT_FORCE_VARIANT     lanes per atom in the two passes.  0: chosen by system size (32 lanes up to 4,096 atoms,
 *                           8 lanes up to 24,576 atoms, else one thread per atom); 1: one thread per atom; 2: 8 lanes;
 *                           3: 32 lanes (MD_EINVAL above 32,768 atoms); 4: 4 lanes.
 *  MD_OPT_GRAPH             1 (default): md_step replays CUDA graphs of up to 8 time steps each; the neighbour rebuild
 *                           of every step is the body of a conditional node, the force pass of a step also performs
 *                           the next step's first half-kick, drift and displacement check, and the last block of that
 *                           kernel takes the rebuild decision (2 kernel launches per step when no rebuild is due);
 *                           up to 4,096 atoms (where a conditional node costs more than the two passes) all steps of
 *                           a graph share ONE loop node that is entered only when a rebuild is due, and the passes
 *                           are guarded instead (they return at once while a rebuild is pending);
 *                           0: the same kernels as plain launches (every kernel of the rebuild chain is launched and
 *                           returns at once unless a rebuild is due).  MD_OPT_PROFILE implies plain launches.
 *  MD_OPT_HALF_LIST         Newton's third law (the paper's CPU code uses it, its GPU kernels do not).  Bit 0:
 *                           the density pass, bit 1: the force pass evaluates every undirected pair ONCE, on the atom
 *                           that owns it, and sends the partner's share by 64-bit integer reductions in units of
 *                           2^-43 (deterministic: integer sums do not depend on the order of arrival; each received
 *                           contribution is rounded to 1.1e-13 eV/A, eV or density units, sums must stay below 1e6).  Takes effect for systems
 *                           that run one thread per atom with a static box (every row of the list holds the pairs
 *                           its atom owns first, so no rebuild is needed).  -1 (default): the library's choice from
 *                           its measurements on B200: 1 for MD_POT_EAM_TABLE (the table passes are bound by the
 *                           gathers, not by arithmetic), 0 for MD_POT_TBSMA (full lists, as the paper's GPU kernels). */
enum { MD_OPT_STEP_OBSERVABLES = 1, MD_OPT_PROFILE = 2, MD_OPT_FORCE_VARIANT = 3, MD_OPT_GRAPH = 4, MD_OPT_HALF_LIST = 5 };
/* Three environment variables select variants that DESIGN.md section 6 measures against the defaults (read by md_create /
 * at the first md_step / at the first list build; results do not depend on them): MD_LIST_F64 (the list build tests every
 * candidate in double precision instead of classifying it on float copies of the coordinates first), MD_CELL_ZFINE = 1, 2, 4 (cells thinner in z by that factor and a z
 * window per column in the list build; default 4 in boxes with an edge shorter than 5 (cutoff + skin), else 1) and
 * MD_NO_LOOP_GRAPH (per-step IF nodes also for small systems).  MD_DEBUG prints why a CUDA graph could not be built. */
int md_set_option(md_system *s, int option, int value);

/* Kernel classes for md_profile_read */
enum { MD_K_BIN = 0, MD_K_SCAN, MD_K_SORT, MD_K_REORDER, MD_K_LIST, MD_K_DENSITY, MD_K_FORCE, MD_K_INTEGRATE,
       MD_K_REDUCE, MD_K_FORCE_CHAINED /* force passes that also perform the next step's drift (inside md_step) */, MD_K_COUNT };
/* Sum of CUDA-event elapsed time (ms) and number of launches of one kernel class since the last
 * md_profile_reset; synchronises.  Needs MD_OPT_PROFILE. */
int md_profile_read(md_system *s, int kernel_class, long *launches, double *total_ms);
int md_profile_reset(md_system *s);
const char *md_kernel_name(int kernel_class);

/* Diagnostic: measured FP64 issue rate of this device, in DFMA thread-instructions per second, from a
 * register-resident kernel of independent DFMA chains on every SM (the ALU roofline denominator).  Not part of the
 * MD path: it needs no md_system and is the one entry point that allocates (16 bytes, cudaMalloc / cudaFree inside
 * the call) and synchronises the device. */
int md_fp64_dfma_rate(void *stream, double *dfma_per_s, double *sm_clock_mhz);

/* Diagnostic: time per warp-wide gather of 32-byte table records (ns, one SM serving 32 resident warps), the access that
 * binds the table passes, in four forms: [0] table in global memory through L1, indices distributed as the passes see
 * them (what the passes do); [1] the reachable window of the table staged in shared memory, same indices; [2], [3] the
 * same two with interval-sorted indices (32 adjacent records per warp).  Not part of the MD path; allocates 160 KB
 * (cudaMalloc / cudaFree inside the call) and synchronises the stream. */
int md_probe_table_gather(void *stream, double ns_per_warp_gather[4]);

/* For callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): E_kin = sum_i 1/2 m_i |v_i|^2 (the kinetic term of eq.(6); what md_get_energies reports per
 * box) of n_atoms atoms, with NO workspace and NO allocation: the block partials of the reduction live in a file-scope
 * device array of the library (33,024 bytes, held by every device that loads the library until the process exits), which
 * bounds n_atoms by MD_NOALLOC_MAX_ATOMS.  Enqueues one 8-byte memset and one kernel on `stream`; calls no cudaMalloc,
 * cudaFree or allocating library routine; does not synchronise.
 *   stream   cudaStream_t of the CURRENT device (the scratch address is looked up per device, for the device that is
 *            current at the call)
 *   v        DEVICE, [n_atoms][3] A/fs (the layout of md_get_velocities)
 *   types    DEVICE, [n_atoms] in 0..n_types-1; may be NULL when n_types == 1
 *   mass     HOST, [n_types] amu (read during the call)
 *   ekin     DEVICE, one double, eV: written by the kernel (n_atoms == 0 gives 0)
 *   err      HOST, optional buffer of err_len bytes that receives a one-line message when the call fails ("" on MD_OK)
 * Returns MD_EINVAL (NULL pointer, n_types outside 1..MD_MAX_TYPES, a mass that is not positive and finite, n_atoms < 0 or
 * n_atoms > MD_NOALLOC_MAX_ATOMS: the message names the limit), MD_ECUDA.  The sum is deterministic (fixed order for a
 * given n_atoms).  ALL calls on one device share the scratch array and it keeps the last call's contents (the call clears
 * the one word that must start at zero): two calls that overlap on the GPU (different streams, or one process's threads
 * without ordering between them) race; calls ordered on one stream do not. */
#define MD_NOALLOC_MAX_ATOMS 4194304
int md_kinetic_energy_noalloc(void *stream, const double *v, const int *types, const double *mass, int n_types, int n_atoms,
                              double *ekin, char *err, int err_len);

const char *md_strerror(int status);
const char *md_version(void);

#ifdef __cplusplus
}
#endif
#endif
