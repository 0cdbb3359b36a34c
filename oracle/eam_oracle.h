/* eam_oracle.h — CPU oracle for the EAM / TB-SMA molecular-dynamics hot path.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may call this.  It shares no code,
 * header, table or constant generator with the CUDA library under paper_1212_6332_b200/.
 *
 * What it computes (arxiv 1212.6332, Hou et al., file /root/reference/PAPER.md):
 *   eq.(1)  E_i = F(sum_j rho(r_ij)) + 1/2 sum_j V(r_ij)
 *   eq.(2)  E_T = sum_i E_i
 *   eq.(3)  f_i = -sum_j [F'(rho_i)+F'(rho_j)] rho'(r_ij) r_ij/r_ij
 *                 -sum_j V'(r_ij) r_ij/r_ij
 *   neighbour list over the 27-cell stencil, test r < RCUT               PAPER.md:137,147,288-336 (Fig.3)
 *   density pass then force pass                                         PAPER.md:159-163,342-409 (Fig.5,6)
 *   virial partial sums                                                  PAPER.md:163 (G22-19)
 *   many independent boxes in one system
 * The integrator is velocity-Verlet with a skin/2 rebuild rule (BASELINE.json north_star;
 * the paper's own predictor-corrector order is not stated).
 *
 * All arithmetic is IEEE double, compiled with -ffp-contract=off (no FMA contraction).
 * All pointers are HOST pointers.  Every call returns 0 on success, <0 on error.
 * Pins: see tests/test_oracle_*.py and DESIGN.md section 3; "parity unpinned" items: the
 * values of a thermal trajectory themselves (only invariants of it are pinned).
 */
#ifndef EAM_ORACLE_H
#define EAM_ORACLE_H
#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_EBOX = -2, ORACLE_EOVERFLOW = -3, ORACLE_ENONFINITE = -4,
       ORACLE_ESTATE = -6 };

typedef struct oracle_system oracle_system;

typedef struct {
  int n_atoms, n_boxes, n_types;        /* n_atoms = total; equal atoms per box; box b owns [b*n, (b+1)*n) */
  double box[3];                        /* orthorhombic, fully periodic, same for all boxes */
  double cutoff, skin;
  const double *positions;              /* [n_atoms][3] */
  const double *velocities;             /* [n_atoms][3] or NULL */
  const int *types;                     /* [n_atoms] */
  const double *mass;                   /* [n_types] amu */
  int pot_kind;                         /* 0 TB-SMA analytic, 1 cubic-Hermite tables */
  const double *A, *xi, *p, *q, *r0;    /* [n_types*n_types] */
  double taper_on;
  int nr; double dr;
  const double *f_val, *f_der, *phi_val, *phi_der;   /* [n_types*n_types][nr] */
  int nrho; double drho;
  const double *F_val, *F_der;          /* [n_types][nrho] */
  int max_neighbors;                    /* list stride; 0 = choose */
  /* optional per-pair cut-offs, the paper's RCUT(ity,jty): [n_types*n_types], symmetric,
   * <= cutoff; NULL = cutoff / taper_on for every pair */
  const double *pair_cutoff, *pair_taper_on;
} oracle_desc;

typedef struct { long steps, rebuilds; int max_neighbors, error_flags; double last_max_disp2; } oracle_stats;

int oracle_create(const oracle_desc *d, oracle_system **out);
int oracle_destroy(oracle_system *s);
int oracle_set_threads(int n);                           /* OpenMP threads; returns the count in use */
/* mode 0: cell list (27-cell stencil); mode 1: brute force over all atoms of the same box */
int oracle_build_neighbors(oracle_system *s, int mode);
int oracle_compute_forces(oracle_system *s, double *forces, double *e_atom, double *virial /*[n_boxes][6]*/);
int oracle_step(oracle_system *s, int n, double dt);
int oracle_set_integrator(oracle_system *s, int kind);   /* 0: velocity-Verlet (default); 1: five-value Gear predictor-corrector */
/* eq.(4): electron-bath thermostat at temperature T_e (K) with time constant tau (fs); tau <= 0: off */
int oracle_set_thermostat(oracle_system *s, double T_e, double tau);
/* eq.(5)-(6): Berendsen barostat, P0 in eV/A^3, tau_p in fs eV/A^3; tau_p <= 0: off; one box only */
int oracle_set_barostat(oracle_system *s, double P0, double tau_p);
int oracle_get_box(oracle_system *s, double *box);
int oracle_get_pressure(oracle_system *s, double *P);   /* eq.(6) for the current state, eV/A^3 */
int oracle_get_positions(oracle_system *s, double *x);
int oracle_get_velocities(oracle_system *s, double *v);
int oracle_set_positions(oracle_system *s, const double *x);
int oracle_set_velocities(oracle_system *s, const double *v);
int oracle_get_neighbors(oracle_system *s, int *count, int *list, int stride);   /* ascending ids per atom */
int oracle_get_densities(oracle_system *s, double *rho, double *fp);              /* after compute_forces */
int oracle_get_energies(oracle_system *s, double *epot, double *ekin);            /* [n_boxes] each */
int oracle_get_stats(oracle_system *s, oracle_stats *st);
/* debug: 1 if every pair with r < cutoff at the CURRENT positions is in the CURRENT list */
int oracle_list_covers_cutoff(oracle_system *s);

/* single-function probes for the pins */
void oracle_min_image(const double xi[3], const double xj[3], const double box[3], double d[3], double *r2);
void oracle_tbsma_eval(double r, double A, double xi, double p, double q, double r0, double r_on, double r_c,
                       double out[6] /* f, f', V, V', S, S' */);
void oracle_hermite_eval(const double *val, const double *der, int n, double h, double x, double *H, double *dH);
const char *oracle_strerror(int);
#ifdef __cplusplus
}
#endif
#endif
