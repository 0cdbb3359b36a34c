/* eam_oracle.c — plain, slow, obviously-correct CPU implementation of the EAM / TB-SMA
 * force path of arxiv 1212.6332 (see eam_oracle.h for the scope and the citations).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT: shares nothing with the CUDA library.
 * Build: gcc -O2 -std=c11 -ffp-contract=off -fopenmp -fPIC -shared (see oracle/build.py).
 *
 * Conventions ("readings"):
 *  - units eV / Angstrom / fs / amu; m[eV fs^2/A^2] = amu * 103.642696526805
 *  - atoms stay in CALLER order; no re-ordering anywhere in the oracle
 *  - full (directed) neighbour lists, as in the paper's GPU kernels (only the
 *    paper's CPU comparator used Newton's third law)
 *  - d = x_j - x_i with the branch minimum image; r2 = (dx*dx + dy*dy) + dz*dz
 *  - strict tests r2 < r_l^2 (list) and r2 < r_c^2 (passes)
 */
#include "eam_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define AMU_EV 103.642696526805

struct oracle_system {
  int N, nb, npb, nt;
  double L[3], rc, skin, rl, rc2, rl2;
  double thermo_Te, thermo_tau;          /* electron-bath thermostat, eq.(4); tau <= 0: off */
  double baro_P0, baro_tau;              /* Berendsen barostat, eq.(5); tau <= 0: off */
  int obs_stale;                         /* the barostat scaled x after the last force evaluation */
  int f_prescale;                        /* f holds the forces of the coordinates before that scaling: queries keep them */
  double *x, *v, *f, *xref, *m;          /* m: per type, eV fs^2/A^2 */
  int *type;
  int kind;
  double *A, *xi, *p, *q, *r0, r_on;     /* [nt*nt] */
  double *rc_p, *rc2_p, *ron_p;          /* per type pair: cut-off, its square, taper start (RCUT(ity,jty)) */
  int nr, nrho; double dr, drho;
  double *f_val, *f_der, *phi_val, *phi_der, *F_val, *F_der;
  int stride, *ncount, *nlist, have_list, forces_valid;
  double *rho, *fp, *eemb, *eatom, *wat; /* wat: per-atom virial [N][6] */
  double *virial;                        /* [nb][6] */
  int integrator, gear_ready;            /* 0: velocity-Verlet; 1: five-value Gear predictor-corrector (its derivatives below) */
  double *ga, *gj, *gs;                  /* [N][3] acceleration, third and fourth time derivative of x */
  oracle_stats st;
};

const char *oracle_strerror(int e) {
  switch (e) {
    case ORACLE_OK: return "ok";
    case ORACLE_EINVAL: return "invalid argument";
    case ORACLE_EBOX: return "box too small for the cut-off";
    case ORACLE_EOVERFLOW: return "neighbour capacity exceeded";
    case ORACLE_ENONFINITE: return "coincident atoms or non-finite value";
    case ORACLE_ESTATE: return "call out of order";
  }
  return "unknown";
}

int oracle_set_threads(int n) {
#ifdef _OPENMP
  if (n > 0) omp_set_num_threads(n);
  return omp_get_max_threads();
#else
  (void)n; return 1;
#endif
}

static double *dup_d(const double *src, size_t n) {
  double *p = (double *)malloc((n ? n : 1) * sizeof(double));
  if (src) memcpy(p, src, n * sizeof(double)); else memset(p, 0, n * sizeof(double));
  return p;
}

/* ---- minimum image, canonical form (reading A3; the paper's line G6-20 is garbled) ---- */
void oracle_min_image(const double xi[3], const double xj[3], const double box[3], double d[3], double *r2) {
  for (int a = 0; a < 3; ++a) {
    double t = xj[a] - xi[a];
    if (t > 0.5 * box[a]) t -= box[a];
    else if (t < -0.5 * box[a]) t += box[a];
    d[a] = t;
  }
  *r2 = (d[0] * d[0] + d[1] * d[1]) + d[2] * d[2];
}

/* ---- TB-SMA radial functions (BASELINE.json configs[0]; Cleri-Rosato form) ----
 * x = r/r0 - 1; f = xi^2 e^{-2qx} S; V = 2A e^{-px} S (factor 2: eq.(1) carries the 1/2);
 * S = quintic switch on [r_on, r_c]: 1 - t^3 (10 - 15 t + 6 t^2), S' = -30 t^2 (1-t)^2 / (r_c - r_on). */
void oracle_tbsma_eval(double r, double A, double xi, double p, double q, double r0, double r_on, double r_c,
                       double out[6]) {
  double S, dS;
  if (r <= r_on) { S = 1.0; dS = 0.0; }
  else if (r >= r_c) { S = 0.0; dS = 0.0; }
  else {
    double w = r_c - r_on, t = (r - r_on) / w;
    S = 1.0 - t * t * t * (10.0 - 15.0 * t + 6.0 * t * t);
    dS = -30.0 * t * t * (1.0 - t) * (1.0 - t) / w;
  }
  double x = r / r0 - 1.0;
  double eh = xi * xi * exp(-2.0 * q * x);     /* hopping integral squared */
  double er = 2.0 * A * exp(-p * x);           /* pair repulsion */
  out[0] = eh * S;
  out[1] = eh * (dS - (2.0 * q / r0) * S);
  out[2] = er * S;
  out[3] = er * (dS - (p / r0) * S);
  out[4] = S;
  out[5] = dS;
}

/* ---- cubic Hermite on a uniform grid x_k = k h (reading A6): value and derivative of the
 * SAME interpolant, so the tabulated force is exactly -grad of the tabulated energy ---- */
void oracle_hermite_eval(const double *val, const double *der, int n, double h, double x, double *H, double *dH) {
  double u = x * (1.0 / h);
  int k = (int)u;
  if (k > n - 2) k = n - 2;
  if (k < 0) k = 0;
  double t = u - (double)k;
  double y0 = val[k], y1 = val[k + 1], d0 = der[k], d1 = der[k + 1];
  double D = y1 - y0;
  double c2 = 3.0 * D - h * (2.0 * d0 + d1);
  double c3 = -2.0 * D + h * (d0 + d1);
  *H = y0 + t * (h * d0 + t * (c2 + t * c3));
  *dH = (h * d0 + t * (2.0 * c2 + 3.0 * t * c3)) / h;
}

/* embedding: analytic -sqrt(rho) for TB-SMA, table with linear continuation
 * above the last node for EAM (reading A8) */
static void embed(const oracle_system *s, int ti, double rho, double *F, double *Fp) {
  if (s->kind == 0) {
    if (rho > 0.0) { double sq = sqrt(rho); *F = -sq; *Fp = -1.0 / (2.0 * sq); }
    else { *F = 0.0; *Fp = 0.0; }
    return;
  }
  const double *val = s->F_val + (size_t)ti * s->nrho, *der = s->F_der + (size_t)ti * s->nrho;
  double rho_max = (double)(s->nrho - 1) * s->drho;
  if (rho >= rho_max) {
    *F = val[s->nrho - 1] + der[s->nrho - 1] * (rho - rho_max);
    *Fp = der[s->nrho - 1];
  } else {
    oracle_hermite_eval(val, der, s->nrho, s->drho, rho, F, Fp);
  }
}

/* pair functions at distance r for type pair (ti,tj): f, f', V, V' */
static void radial(const oracle_system *s, int ti, int tj, double r, double *f, double *df, double *V, double *dV) {
  int tp = ti * s->nt + tj;
  if (s->kind == 0) {
    double o[6];
    oracle_tbsma_eval(r, s->A[tp], s->xi[tp], s->p[tp], s->q[tp], s->r0[tp], s->ron_p[tp], s->rc_p[tp], o);
    *f = o[0]; *df = o[1]; *V = o[2]; *dV = o[3];
  } else {
    size_t off = (size_t)tp * s->nr;
    oracle_hermite_eval(s->f_val + off, s->f_der + off, s->nr, s->dr, r, f, df);
    oracle_hermite_eval(s->phi_val + off, s->phi_der + off, s->nr, s->dr, r, V, dV);
  }
}

int oracle_create(const oracle_desc *d, oracle_system **out) {
  if (!d || !out || d->n_atoms <= 0 || d->n_boxes <= 0 || d->n_types <= 0 || !d->positions || !d->types || !d->mass)
    return ORACLE_EINVAL;
  if (d->n_atoms % d->n_boxes) return ORACLE_EINVAL;
  if (!(d->cutoff > 0.0) || !(d->skin >= 0.0)) return ORACLE_EINVAL;
  double rl = d->cutoff + d->skin;
  for (int a = 0; a < 3; ++a) {
    if (!(d->box[a] > 0.0)) return ORACLE_EINVAL;
    if (!(d->box[a] > 2.0 * rl)) return ORACLE_EBOX;   /* minimum image must be unique */
  }
  for (int i = 0; i < d->n_atoms; ++i)
    if (d->types[i] < 0 || d->types[i] >= d->n_types) return ORACLE_EINVAL;
  oracle_system *s = (oracle_system *)calloc(1, sizeof(*s));
  s->N = d->n_atoms; s->nb = d->n_boxes; s->npb = s->N / s->nb; s->nt = d->n_types;
  memcpy(s->L, d->box, sizeof(s->L));
  s->rc = d->cutoff; s->skin = d->skin; s->rl = rl; s->rc2 = s->rc * s->rc; s->rl2 = rl * rl;
  size_t N = (size_t)s->N, nt2 = (size_t)s->nt * s->nt;
  s->x = dup_d(d->positions, 3 * N);
  s->v = dup_d(d->velocities, 3 * N);
  s->f = dup_d(NULL, 3 * N);
  s->xref = dup_d(NULL, 3 * N);
  s->type = (int *)malloc(N * sizeof(int)); memcpy(s->type, d->types, N * sizeof(int));
  s->m = dup_d(d->mass, s->nt);
  for (int t = 0; t < s->nt; ++t) { if (!(s->m[t] > 0.0)) { oracle_destroy(s); return ORACLE_EINVAL; } s->m[t] *= AMU_EV; }
  s->kind = d->pot_kind;
  /* per-pair cut-offs (RCUT(ity,jty)); default: the global ones */
  s->rc_p = dup_d(NULL, nt2); s->rc2_p = dup_d(NULL, nt2); s->ron_p = dup_d(NULL, nt2);
  for (int a = 0; a < s->nt; ++a)
    for (int b = 0; b < s->nt; ++b) {
      const int k = a * s->nt + b, kt = b * s->nt + a;
      const double rc = d->pair_cutoff ? d->pair_cutoff[k] : d->cutoff, ron = d->pair_taper_on ? d->pair_taper_on[k] : d->taper_on;
      if (!(rc > 0.0) || !(rc <= d->cutoff) || (d->pair_cutoff && d->pair_cutoff[kt] != rc) ||
          (d->pot_kind == 0 && (!(ron < rc) || (d->pair_taper_on && d->pair_taper_on[kt] != ron)))) { oracle_destroy(s); return ORACLE_EINVAL; }
      s->rc_p[k] = rc; s->rc2_p[k] = rc * rc; s->ron_p[k] = ron;
    }
  if (s->kind == 0) {
    if (!d->A || !d->xi || !d->p || !d->q || !d->r0 || !(d->taper_on < d->cutoff)) { oracle_destroy(s); return ORACLE_EINVAL; }
    s->A = dup_d(d->A, nt2); s->xi = dup_d(d->xi, nt2); s->p = dup_d(d->p, nt2); s->q = dup_d(d->q, nt2);
    s->r0 = dup_d(d->r0, nt2); s->r_on = d->taper_on;
  } else if (s->kind == 1) {
    if (!d->f_val || !d->f_der || !d->phi_val || !d->phi_der || !d->F_val || !d->F_der || d->nr < 2 || d->nrho < 2 ||
        !(d->dr > 0.0) || !(d->drho > 0.0)) { oracle_destroy(s); return ORACLE_EINVAL; }
    s->nr = d->nr; s->dr = d->dr; s->nrho = d->nrho; s->drho = d->drho;
    s->f_val = dup_d(d->f_val, nt2 * s->nr); s->f_der = dup_d(d->f_der, nt2 * s->nr);
    s->phi_val = dup_d(d->phi_val, nt2 * s->nr); s->phi_der = dup_d(d->phi_der, nt2 * s->nr);
    s->F_val = dup_d(d->F_val, (size_t)s->nt * s->nrho); s->F_der = dup_d(d->F_der, (size_t)s->nt * s->nrho);
  } else { oracle_destroy(s); return ORACLE_EINVAL; }
  if (d->max_neighbors > 0) s->stride = d->max_neighbors;
  else {
    /* MN "adjusted according to the particle density and the cut-off" */
    double dens = (double)s->npb / (s->L[0] * s->L[1] * s->L[2]);
    s->stride = (int)(1.6 * 4.18879020478639 * rl * rl * rl * dens) + 24;
  }
  if (s->stride > s->npb - 1) s->stride = s->npb > 1 ? s->npb - 1 : 1;
  s->ncount = (int *)calloc(N, sizeof(int));
  s->nlist = (int *)malloc(N * (size_t)s->stride * sizeof(int));
  s->rho = dup_d(NULL, N); s->fp = dup_d(NULL, N); s->eemb = dup_d(NULL, N); s->eatom = dup_d(NULL, N);
  s->wat = dup_d(NULL, 6 * N); s->virial = dup_d(NULL, 6 * (size_t)s->nb);
  *out = s;
  return ORACLE_OK;
}

int oracle_destroy(oracle_system *s) {
  if (!s) return ORACLE_OK;
  free(s->x); free(s->v); free(s->f); free(s->xref); free(s->m); free(s->type);
  free(s->A); free(s->xi); free(s->p); free(s->q); free(s->r0);
  free(s->f_val); free(s->f_der); free(s->phi_val); free(s->phi_der); free(s->F_val); free(s->F_der);
  free(s->rc_p); free(s->rc2_p); free(s->ron_p);
  free(s->ncount); free(s->nlist); free(s->rho); free(s->fp); free(s->eemb); free(s->eatom); free(s->wat);
  free(s->virial); free(s->ga); free(s->gj); free(s->gs); free(s);
  return ORACLE_OK;
}

static int cmp_int(const void *a, const void *b) { int x = *(const int *)a, y = *(const int *)b; return (x > y) - (x < y); }

/* Neighbour list N_l(i) = { j != i, same box : r_ij^2 < r_l^2 } (Fig.3 G6-9..G6-27;
 * self-exclusion and tail guards per reading A4).  Positions are wrapped into [0,L) first and
 * x_ref <- x.  mode 0 = linked cells + 27-cell stencil ("normative [1]"),
 * mode 1 = all atoms of the same box (the definition). */
int oracle_build_neighbors(oracle_system *s, int mode) {
  const int N = s->N, npb = s->npb;
  for (int i = 0; i < N; ++i)
    for (int a = 0; a < 3; ++a) {
      double x = s->x[3 * i + a];
      if (!isfinite(x)) { s->st.error_flags |= 2; return ORACLE_ENONFINITE; }
      s->x[3 * i + a] = x - s->L[a] * floor(x / s->L[a]);
    }
  memcpy(s->xref, s->x, 3 * (size_t)N * sizeof(double));
  int nc[3] = {1, 1, 1}, tnc = 1;
  int *head = NULL, *next = NULL, *cell = NULL;
  if (mode == 0) {
    for (int a = 0; a < 3; ++a) {
      nc[a] = (int)floor(s->L[a] / s->rl);
      if (nc[a] < 3) return ORACLE_EBOX;       /* 26 distinct neighbour cells */
    }
    tnc = nc[0] * nc[1] * nc[2];
    /* multiple boxes: cell ids of box I shifted by I*TNC */
    head = (int *)malloc((size_t)tnc * s->nb * sizeof(int));
    next = (int *)malloc((size_t)N * sizeof(int));
    cell = (int *)malloc((size_t)N * sizeof(int));
    for (int c = 0; c < tnc * s->nb; ++c) head[c] = -1;
    for (int i = N - 1; i >= 0; --i) {
      int c[3];
      for (int a = 0; a < 3; ++a) {
        c[a] = (int)(s->x[3 * i + a] * nc[a] / s->L[a]);
        if (c[a] > nc[a] - 1) c[a] = nc[a] - 1;
        if (c[a] < 0) c[a] = 0;
      }
      int cid = (i / npb) * tnc + (c[0] * nc[1] + c[1]) * nc[2] + c[2];
      cell[i] = cid; next[i] = head[cid]; head[cid] = i;
    }
  }
  int overflow = 0, maxn = 0;
#pragma omp parallel for schedule(static) reduction(| : overflow) reduction(max : maxn)
  for (int i = 0; i < N; ++i) {
    int n = 0, *li = s->nlist + (size_t)i * s->stride, b = i / npb;
    double d[3], r2;
    if (mode == 1) {
      for (int j = b * npb; j < (b + 1) * npb; ++j) {
        if (j == i) continue;
        oracle_min_image(s->x + 3 * i, s->x + 3 * j, s->L, d, &r2);
        if (r2 < s->rl2) { if (n < s->stride) li[n] = j; ++n; }
      }
    } else {
      int cl = cell[i] - b * tnc;
      int cz = cl % nc[2], cy = (cl / nc[2]) % nc[1], cx = cl / (nc[2] * nc[1]);
      for (int ox = -1; ox <= 1; ++ox) for (int oy = -1; oy <= 1; ++oy) for (int oz = -1; oz <= 1; ++oz) {
        int jx = (cx + ox + nc[0]) % nc[0], jy = (cy + oy + nc[1]) % nc[1], jz = (cz + oz + nc[2]) % nc[2];
        for (int j = head[b * tnc + (jx * nc[1] + jy) * nc[2] + jz]; j >= 0; j = next[j]) {
          if (j == i) continue;
          oracle_min_image(s->x + 3 * i, s->x + 3 * j, s->L, d, &r2);
          if (r2 < s->rl2) { if (n < s->stride) li[n] = j; ++n; }
        }
      }
    }
    if (n > s->stride) { overflow |= 1; n = s->stride; }
    qsort(li, (size_t)n, sizeof(int), cmp_int);
    s->ncount[i] = n;
    if (n > maxn) maxn = n;
  }
  free(head); free(next); free(cell);
  s->st.max_neighbors = maxn;
  s->st.rebuilds += 1;
  s->have_list = 1; s->forces_valid = 0;
  if (overflow) { s->st.error_flags |= 1; return ORACLE_EOVERFLOW; }
  return ORACLE_OK;
}

/* Density pass (Fig.5 G18) then force pass (Fig.6 G22). */
static int forces_internal(oracle_system *s) {
  s->obs_stale = 0;
  const int N = s->N;
  int bad = 0;
  /* G18: rho_i = sum_{j in list, r < r_c} f(r_ij); then F(rho_i), F'(rho_i) */
#pragma omp parallel for schedule(static) reduction(| : bad)
  for (int i = 0; i < N; ++i) {
    const int *li = s->nlist + (size_t)i * s->stride;
    double rho = 0.0, d[3], r2, f, df, V, dV;
    for (int k = 0; k < s->ncount[i]; ++k) {
      int j = li[k];
      oracle_min_image(s->x + 3 * i, s->x + 3 * j, s->L, d, &r2);
      if (r2 < s->rc2_p[s->type[i] * s->nt + s->type[j]]) {
        if (!(r2 > 0.0)) { bad |= 1; continue; }
        double r = sqrt(r2);
        radial(s, s->type[i], s->type[j], r, &f, &df, &V, &dV);
        rho += f;
      }
    }
    s->rho[i] = rho;
    embed(s, s->type[i], rho, &s->eemb[i], &s->fp[i]);
  }
  if (bad) { s->st.error_flags |= 2; return ORACLE_ENONFINITE; }
  /* G22: f_i = sum_j s_ij d/r with d = x_j - x_i, s_ij = V'(r) + (F'_i + F'_j) f'(r)   [eq.(3)]
   * E_i = F(rho_i) + 1/2 sum_j V(r)                                                  [eq.(1)]
   * W^{ab} = 1/2 sum_i sum_j (r_i - r_j)^a f_ij^b, f_ij = s_ij d / r                  [G22-19, reading A5] */
#pragma omp parallel for schedule(static)
  for (int i = 0; i < N; ++i) {
    const int *li = s->nlist + (size_t)i * s->stride;
    double fx = 0.0, fy = 0.0, fz = 0.0, ev = 0.0, w[6] = {0, 0, 0, 0, 0, 0}, d[3], r2, f, df, V, dV;
    for (int k = 0; k < s->ncount[i]; ++k) {
      int j = li[k];
      oracle_min_image(s->x + 3 * i, s->x + 3 * j, s->L, d, &r2);
      if (r2 < s->rc2_p[s->type[i] * s->nt + s->type[j]]) {
        double r = sqrt(r2);
        radial(s, s->type[i], s->type[j], r, &f, &df, &V, &dV);
        double sij = dV + (s->fp[i] + s->fp[j]) * df;
        double gx = sij * d[0] / r, gy = sij * d[1] / r, gz = sij * d[2] / r;   /* force on i from j */
        fx += gx; fy += gy; fz += gz;
        ev += V;
        w[0] += 0.5 * (-d[0]) * gx; w[1] += 0.5 * (-d[1]) * gy; w[2] += 0.5 * (-d[2]) * gz;
        w[3] += 0.5 * (-d[0]) * gy; w[4] += 0.5 * (-d[0]) * gz; w[5] += 0.5 * (-d[1]) * gz;
      }
    }
    s->f[3 * i] = fx; s->f[3 * i + 1] = fy; s->f[3 * i + 2] = fz;
    s->eatom[i] = s->eemb[i] + 0.5 * ev;
    for (int c = 0; c < 6; ++c) s->wat[6 * (size_t)i + c] = w[c];
  }
  for (int b = 0; b < s->nb; ++b) {
    long double acc[6] = {0, 0, 0, 0, 0, 0};
    for (int i = b * s->npb; i < (b + 1) * s->npb; ++i)
      for (int c = 0; c < 6; ++c) acc[c] += s->wat[6 * (size_t)i + c];
    for (int c = 0; c < 6; ++c) s->virial[6 * b + c] = (double)acc[c];
  }
  for (int i = 0; i < 3 * N; ++i) if (!isfinite(s->f[i])) { s->st.error_flags |= 2; return ORACLE_ENONFINITE; }
  s->forces_valid = 1;
  return ORACLE_OK;
}

/* Force evaluation on behalf of a QUERY (forces, energies, pressure asked for between steps).  After a barostat step
 * (reading B1) the observables belong to the scaled coordinates, while the next first half-kick uses the forces
 * of the unscaled ones: a query must not change the trajectory, so s->f is put back after the evaluation. */
static int forces_for_query(oracle_system *s, double *forces_out) {
  const size_t n3 = 3 * (size_t)s->N;
  double *keep = (s->forces_valid && s->f_prescale) ? dup_d(s->f, n3) : NULL;
  int rc = forces_internal(s);
  if (rc == ORACLE_OK && forces_out) memcpy(forces_out, s->f, n3 * sizeof(double));
  if (keep) { if (rc == ORACLE_OK) memcpy(s->f, keep, n3 * sizeof(double)); free(keep); }
  return rc;
}

int oracle_compute_forces(oracle_system *s, double *forces, double *e_atom, double *virial) {
  int rc;
  if (!s) return ORACLE_EINVAL;
  if (!s->have_list && (rc = oracle_build_neighbors(s, 0)) != ORACLE_OK) return rc;
  if ((rc = forces_for_query(s, forces)) != ORACLE_OK) return rc;
  if (e_atom) memcpy(e_atom, s->eatom, (size_t)s->N * sizeof(double));
  if (virial) memcpy(virial, s->virial, 6 * (size_t)s->nb * sizeof(double));
  return ORACLE_OK;
}

/* Electron-bath thermostat, eq.(4):  m dv/dt = f - (m/tau_T) ((T_i - T_e)/T_i) v,  with the per-atom
 * instantaneous temperature T_i = m |v|^2 / (3 k_B).  Reading (T1): tau_T is a time, so the printed 1/tau_T
 * stands for m_i/tau_T; the damping acceleration is -(1/tau_T)(1 - c2/|v|^2) v with c2 = 3 k_B T_e / m_i, and 0 for an
 * atom at rest.  Each half-kick of the velocity-Verlet step uses the damping of the velocity it starts from. */
#define KB_EV 8.617333262e-5
int oracle_set_thermostat(oracle_system *s, double T_e, double tau) {
  if (!s || !(T_e >= 0.0) || (tau > 0.0 && s->integrator == 1)) return ORACLE_EINVAL;
  s->thermo_Te = T_e; s->thermo_tau = tau;
  return ORACLE_OK;
}

/* Berendsen barostat, eq.(5)-(6): at the end of every step the coordinates and the box edges are
 * scaled by mu = [1 - (dt/tau_p)(P_0 - P)]^(1/3), with P = (N k_B T + 1/3 sum_i f_i.r_i)/V.  Readings (B1):
 * N k_B T = 2/3 E_kin (velocities after the second half-kick), the virial sum is the pairwise trace W_xx+W_yy+W_zz of
 * the force evaluation of this step, V = Lx Ly Lz; pressures in eV/A^3, tau_p in fs eV/A^3 (it absorbs the
 * compressibility); x_ref is NOT scaled, so the skin/2 rule also sees the displacement that the scaling causes. */
int oracle_set_barostat(oracle_system *s, double P0, double tau_p) {
  if (!s || (tau_p > 0.0 && (s->nb != 1 || s->integrator == 1))) return ORACLE_EINVAL;
  s->baro_P0 = P0; s->baro_tau = tau_p;
  return ORACLE_OK;
}
int oracle_get_box(oracle_system *s, double *box) { for (int a = 0; a < 3; ++a) box[a] = s->L[a]; return ORACLE_OK; }

static double pressure_now(const oracle_system *s) {
  long double ek = 0;
  for (int i = 0; i < s->N; ++i) {
    const double *v = s->v + 3 * i;
    ek += 0.5 * s->m[s->type[i]] * ((v[0] * v[0] + v[1] * v[1]) + v[2] * v[2]);
  }
  const double trw = (s->virial[0] + s->virial[1]) + s->virial[2];
  return ((2.0 / 3.0) * (double)ek + trw / 3.0) / (s->L[0] * s->L[1] * s->L[2]);
}
int oracle_get_pressure(oracle_system *s, double *P) {
  int rc;
  if (!s->have_list && (rc = oracle_build_neighbors(s, 0)) != ORACLE_OK) return rc;
  if ((!s->forces_valid || s->obs_stale) && (rc = forces_for_query(s, NULL)) != ORACLE_OK) return rc;
  *P = pressure_now(s);
  return ORACLE_OK;
}

static void half_kick(oracle_system *s, int i, double dt) {
  const double m = s->m[s->type[i]], h = 0.5 * dt / m;
  double *v = s->v + 3 * i;
  const double *f = s->f + 3 * i;
  double g = 0.0;
  if (s->thermo_tau > 0.0) {
    const double v2 = (v[0] * v[0] + v[1] * v[1]) + v[2] * v[2];
    if (v2 > 0.0) g = (1.0 / s->thermo_tau) * (1.0 - (3.0 * KB_EV * s->thermo_Te / m) / v2);
  }
  for (int a = 0; a < 3; ++a) v[a] = v[a] + h * f[a] - (0.5 * dt * g) * v[a];
}

/* Predictor-corrector integration (sec. 3.3: "A predictor-corrector scheme is used for the stepwise
 * integration [1] ... Each thread predicts the position and the velocity of one atom"; the velocities
 * are corrected after the force calculation).  The paper states neither the order nor the coefficients (DESIGN.md
 * reading G1): taken here as the five-value Gear scheme for m x'' = f(x) in the form of Allen & Tildesley, "Computer
 * Simulation of Liquids", sec. 3.2 / appendix E: the state is x and its first four time derivatives (v, a, j, s);
 *   predictor (Taylor):  x_p = x + dt v + dt^2/2 a + dt^3/6 j + dt^4/24 s,   v_p = v + dt a + dt^2/2 j + dt^3/6 s,
 *                        a_p = a + dt j + dt^2/2 s,   j_p = j + dt s,   s_p = s;
 *   skin/2 rule on x_p (readings A10, A11), forces at x_p;
 *   corrector:  D = dt^2/2 (f(x_p)/m - a_p);  x = x_p + c0 D,  v = v_p + c1 D/dt,  a = a_p + c2 D 2/dt^2,
 *               j = j_p + c3 D 6/dt^3,  s = s_p + c4 D 24/dt^4,   (c0 .. c4) = (19/120, 3/4, 1, 1/2, 1/12).
 * Start-up: below.  No thermostat, no barostat (velocity-Verlet only). */
int oracle_set_integrator(oracle_system *s, int kind) {
  if (!s || (kind != 0 && kind != 1)) return ORACLE_EINVAL;
  if (kind == 1 && (s->thermo_tau > 0.0 || s->baro_tau > 0.0)) return ORACLE_EINVAL;
  if (kind == 1 && !s->ga) {
    s->ga = (double *)calloc(3 * (size_t)s->N, sizeof(double));
    s->gj = (double *)calloc(3 * (size_t)s->N, sizeof(double));
    s->gs = (double *)calloc(3 * (size_t)s->N, sizeof(double));
    if (!s->ga || !s->gj || !s->gs) return ORACLE_EINVAL;
  }
  s->integrator = kind; s->gear_ready = 0;
  return ORACLE_OK;
}

static int gear_steps(oracle_system *s, int n, double dt) {
  static const double c0 = 19.0 / 120.0, c1 = 3.0 / 4.0, c2 = 1.0, c3 = 1.0 / 2.0, c4 = 1.0 / 12.0;
  int rc;
  const int N = s->N;
  const double thr = (0.5 * s->skin) * (0.5 * s->skin);
  const double h1 = dt, h2 = dt * dt / 2.0, h3 = dt * dt * dt / 6.0, h4 = dt * dt * dt * dt / 24.0;
  if (!s->gear_ready) {
    /* start-up: a = f(x)/m, and j, s by central differences of a along the Taylor path x(+-tau) = x +- tau v + tau^2/2 a,
     * tau = dt/10 (with j = s = 0 the first predicted velocity is off by dt^2/2 j and the scheme stays second order) */
    const double tau = 0.1 * dt;
    double *x0 = (double *)malloc(3 * (size_t)N * sizeof(double));
    if (!x0) return ORACLE_EINVAL;
    memcpy(x0, s->x, 3 * (size_t)N * sizeof(double));
    if ((rc = forces_internal(s)) != ORACLE_OK) { free(x0); return rc; }
    for (int i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) s->ga[3 * i + a] = s->f[3 * i + a] / s->m[s->type[i]];
    for (int k = 0; k < 3 * N; ++k) s->x[k] = x0[k] + tau * s->v[k] + 0.5 * tau * tau * s->ga[k];
    if ((rc = forces_internal(s)) != ORACLE_OK) { free(x0); return rc; }
    for (int i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) s->gj[3 * i + a] = s->f[3 * i + a] / s->m[s->type[i]];          /* a(+tau), for now */
    for (int k = 0; k < 3 * N; ++k) s->x[k] = x0[k] - tau * s->v[k] + 0.5 * tau * tau * s->ga[k];
    if ((rc = forces_internal(s)) != ORACLE_OK) { free(x0); return rc; }
    for (int i = 0; i < N; ++i)
      for (int a = 0; a < 3; ++a) {
        const int k = 3 * i + a;
        const double ap = s->gj[k], am = s->f[k] / s->m[s->type[i]];
        s->gj[k] = (ap - am) / (2.0 * tau);
        s->gs[k] = ((ap - s->ga[k]) + (am - s->ga[k])) / (tau * tau);
      }
    memcpy(s->x, x0, 3 * (size_t)N * sizeof(double));
    free(x0);
    s->gear_ready = 1;
  }
  for (int step = 0; step < n; ++step) {
    double maxd2 = 0.0;
    for (int i = 0; i < N; ++i) {
      double d2 = 0.0;
      for (int a = 0; a < 3; ++a) {
        const int k = 3 * i + a;
        const double x = s->x[k], v = s->v[k], ac = s->ga[k], j = s->gj[k], q = s->gs[k];
        s->x[k] = x + h1 * v + h2 * ac + h3 * j + h4 * q;
        s->v[k] = v + h1 * ac + h2 * j + h3 * q;
        s->ga[k] = ac + h1 * j + h2 * q;
        s->gj[k] = j + h1 * q;
        const double u = s->x[k] - s->xref[k];
        d2 += u * u;
      }
      if (d2 > maxd2) maxd2 = d2;
      if (!(d2 == d2)) maxd2 = INFINITY;
    }
    s->st.last_max_disp2 = maxd2;
    if (maxd2 > thr && (rc = oracle_build_neighbors(s, 0)) != ORACLE_OK) return rc;
    if ((rc = forces_internal(s)) != ORACLE_OK) return rc;
    for (int i = 0; i < N; ++i) {
      const double m = s->m[s->type[i]];
      for (int a = 0; a < 3; ++a) {
        const int k = 3 * i + a;
        const double D = h2 * (s->f[k] / m - s->ga[k]);
        s->x[k] += c0 * D;
        s->v[k] += c1 * D / h1;
        s->ga[k] += c2 * D / h2;
        s->gj[k] += c3 * D / h3;
        s->gs[k] += c4 * D / h4;
      }
    }
    s->forces_valid = 0;       /* f belongs to the predicted coordinates: a query evaluates the corrected ones */
    s->st.steps += 1;
  }
  return ORACLE_OK;
}

/* Velocity-Verlet (BASELINE.json north_star) with the skin/2 rule (readings A10, A11):
 *   v += (dt/2)(f/m + a_fric(v)); x += dt v; if max_i |x_i - x_ref,i|^2 > (skin/2)^2: rebuild;
 *   f <- force(x); v += (dt/2)(f/m + a_fric(v)). */
int oracle_step(oracle_system *s, int n, double dt) {
  int rc;
  if (!s || n < 0) return ORACLE_EINVAL;
  if (!s->have_list && (rc = oracle_build_neighbors(s, 0)) != ORACLE_OK) return rc;
  if (s->integrator == 1) return gear_steps(s, n, dt);
  if (!s->forces_valid && (rc = forces_internal(s)) != ORACLE_OK) return rc;
  const int N = s->N;
  const double thr = (0.5 * s->skin) * (0.5 * s->skin);
  for (int step = 0; step < n; ++step) {
    double maxd2 = 0.0;
    for (int i = 0; i < N; ++i) {
      double d2 = 0.0;
      half_kick(s, i, dt);
      for (int a = 0; a < 3; ++a) {
        s->x[3 * i + a] += dt * s->v[3 * i + a];
        double u = s->x[3 * i + a] - s->xref[3 * i + a];
        d2 += u * u;
      }
      if (d2 > maxd2) maxd2 = d2;
      if (!(d2 == d2)) maxd2 = INFINITY;
    }
    s->st.last_max_disp2 = maxd2;
    if (maxd2 > thr && (rc = oracle_build_neighbors(s, 0)) != ORACLE_OK) return rc;
    if ((rc = forces_internal(s)) != ORACLE_OK) return rc;
    s->f_prescale = 0;
    for (int i = 0; i < N; ++i) half_kick(s, i, dt);
    if (s->baro_tau > 0.0) {
      const double mu = cbrt(1.0 - (dt / s->baro_tau) * (s->baro_P0 - pressure_now(s)));
      for (int i = 0; i < 3 * N; ++i) s->x[i] *= mu;
      for (int a = 0; a < 3; ++a) s->L[a] *= mu;
      s->obs_stale = 1;     /* energies / pressure on request are re-evaluated; the next half-kick keeps these forces */
      s->f_prescale = 1;
    }
    s->st.steps += 1;
  }
  return ORACLE_OK;
}

int oracle_get_positions(oracle_system *s, double *x) { memcpy(x, s->x, 3 * (size_t)s->N * sizeof(double)); return ORACLE_OK; }
int oracle_get_velocities(oracle_system *s, double *v) { memcpy(v, s->v, 3 * (size_t)s->N * sizeof(double)); return ORACLE_OK; }
int oracle_set_positions(oracle_system *s, const double *x) {
  memcpy(s->x, x, 3 * (size_t)s->N * sizeof(double)); s->have_list = 0; s->forces_valid = 0; s->f_prescale = 0; s->gear_ready = 0; return ORACLE_OK;
}
int oracle_set_velocities(oracle_system *s, const double *v) { memcpy(s->v, v, 3 * (size_t)s->N * sizeof(double)); s->gear_ready = 0; return ORACLE_OK; }

int oracle_get_neighbors(oracle_system *s, int *count, int *list, int stride) {
  if (!s->have_list) return ORACLE_ESTATE;
  for (int i = 0; i < s->N; ++i) {
    if (s->ncount[i] > stride) return ORACLE_EOVERFLOW;
    count[i] = s->ncount[i];
    memcpy(list + (size_t)i * stride, s->nlist + (size_t)i * s->stride, (size_t)s->ncount[i] * sizeof(int));
  }
  return ORACLE_OK;
}

int oracle_get_densities(oracle_system *s, double *rho, double *fp) {
  if (!s->forces_valid) return ORACLE_ESTATE;
  if (rho) memcpy(rho, s->rho, (size_t)s->N * sizeof(double));
  if (fp) memcpy(fp, s->fp, (size_t)s->N * sizeof(double));
  return ORACLE_OK;
}

int oracle_get_energies(oracle_system *s, double *epot, double *ekin) {
  int rc;
  if (!s->have_list && (rc = oracle_build_neighbors(s, 0)) != ORACLE_OK) return rc;
  if ((!s->forces_valid || s->obs_stale) && (rc = forces_for_query(s, NULL)) != ORACLE_OK) return rc;
  for (int b = 0; b < s->nb; ++b) {
    long double ep = 0, ek = 0;
    for (int i = b * s->npb; i < (b + 1) * s->npb; ++i) {
      ep += s->eatom[i];
      double v2 = (s->v[3 * i] * s->v[3 * i] + s->v[3 * i + 1] * s->v[3 * i + 1]) + s->v[3 * i + 2] * s->v[3 * i + 2];
      ek += 0.5 * s->m[s->type[i]] * v2;
    }
    if (epot) epot[b] = (double)ep;
    if (ekin) ekin[b] = (double)ek;
  }
  return ORACLE_OK;
}

int oracle_get_stats(oracle_system *s, oracle_stats *st) { *st = s->st; return ORACLE_OK; }

int oracle_list_covers_cutoff(oracle_system *s) {
  if (!s->have_list) return ORACLE_ESTATE;
  int ok = 1;
#pragma omp parallel for schedule(static) reduction(& : ok)
  for (int i = 0; i < s->N; ++i) {
    int b = i / s->npb;
    const int *li = s->nlist + (size_t)i * s->stride;
    double d[3], r2;
    for (int j = b * s->npb; j < (b + 1) * s->npb; ++j) {
      if (j == i) continue;
      oracle_min_image(s->x + 3 * i, s->x + 3 * j, s->L, d, &r2);
      if (r2 < s->rc2) {
        int found = 0;
        for (int k = 0; k < s->ncount[i]; ++k) if (li[k] == j) { found = 1; break; }
        ok &= found;
      }
    }
  }
  return ok;
}
