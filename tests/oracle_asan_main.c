/* oracle_asan_main.c — drives oracle/eam_oracle.c under -fsanitize=address,undefined
 * (tests/test_oracle_pins.py::test_oracle_under_address_and_undefined_sanitizers).
 * Test infrastructure: small seeded systems built here in C, every entry point of eam_oracle.h called once. */
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "eam_oracle.h"

static unsigned long long lcg_state = 12126332ull;
static double lcg_uniform(void) {             /* (0,1) */
  lcg_state = lcg_state * 6364136223846793005ull + 1442695040888963407ull;
  return ((double)(lcg_state >> 11) + 0.5) / 9007199254740992.0;
}
static double lcg_normal(void) { return sqrt(-2.0 * log(lcg_uniform())) * cos(6.283185307179586 * lcg_uniform()); }

#define CHECK(call) do { int rc_ = (call); if (rc_ != 0) { fprintf(stderr, "%s -> %d (%s)\n", #call, rc_, oracle_strerror(rc_)); return 1; } } while (0)

/* crystal of nc^3 cells with `nbasis` basis atoms, jittered; nb boxes one after the other */
static int lattice(int nc, double a, const double (*basis)[3], int nbasis, int nb, double sigma, double **x, double **v, int **type, int nt) {
  const int n = nc * nc * nc * nbasis * nb;
  *x = (double *)malloc(3 * (size_t)n * sizeof(double));
  *v = (double *)malloc(3 * (size_t)n * sizeof(double));
  *type = (int *)malloc((size_t)n * sizeof(int));
  int k = 0;
  for (int b = 0; b < nb; ++b)
    for (int ix = 0; ix < nc; ++ix) for (int iy = 0; iy < nc; ++iy) for (int iz = 0; iz < nc; ++iz)
      for (int s = 0; s < nbasis; ++s, ++k) {
        const double c[3] = {ix + basis[s][0], iy + basis[s][1], iz + basis[s][2]};
        for (int d = 0; d < 3; ++d) {
          (*x)[3 * k + d] = a * c[d] + sigma * lcg_normal() + (d == 1 ? -7.0 * a * nc : 0.0);   /* far outside the box along y */
          (*v)[3 * k + d] = 0.003 * lcg_normal();
        }
        (*type)[k] = (int)(lcg_uniform() * nt) % nt;
      }
  return n;
}

static int exercise(oracle_system *s, int n, int nb, int with_controls) {
  double *f = (double *)malloc(3 * (size_t)n * sizeof(double)), *e = (double *)malloc((size_t)n * sizeof(double));
  double *w = (double *)malloc(6 * (size_t)nb * sizeof(double)), *x = (double *)malloc(3 * (size_t)n * sizeof(double));
  double *ep = (double *)malloc((size_t)nb * sizeof(double)), *ek = (double *)malloc((size_t)nb * sizeof(double));
  int *cnt = (int *)malloc((size_t)n * sizeof(int)), *lst = (int *)malloc((size_t)n * 256 * sizeof(int));
  oracle_stats st;
  CHECK(oracle_build_neighbors(s, 1));
  CHECK(oracle_get_neighbors(s, cnt, lst, 256));
  CHECK(oracle_build_neighbors(s, 0));
  CHECK(oracle_compute_forces(s, f, e, w));
  CHECK(oracle_get_densities(s, e, e));
  CHECK(oracle_step(s, 25, 1.0));
  if (!oracle_list_covers_cutoff(s)) { fprintf(stderr, "list does not cover the cut-off\n"); return 1; }
  if (with_controls) {
    double P, box[3];
    CHECK(oracle_set_thermostat(s, 600.0, 50.0));
    if (nb == 1) CHECK(oracle_set_barostat(s, 0.0, 25.0));
    CHECK(oracle_step(s, 10, 1.0));
    CHECK(oracle_get_pressure(s, &P));
    CHECK(oracle_get_box(s, box));
  }
  CHECK(oracle_get_positions(s, x));
  CHECK(oracle_set_positions(s, x));
  CHECK(oracle_get_velocities(s, x));
  CHECK(oracle_set_velocities(s, x));
  CHECK(oracle_step(s, 3, 0.5));
  CHECK(oracle_get_energies(s, ep, ek));
  CHECK(oracle_get_stats(s, &st));
  printf("  n=%d boxes=%d epot[0]=%.12g ekin[0]=%.6g rebuilds=%ld maxn=%d\n", n, nb, ep[0], ek[0], st.rebuilds, st.max_neighbors);
  free(f); free(e); free(w); free(x); free(ep); free(ek); free(cnt); free(lst);
  return st.error_flags != 0;
}

int main(void) {
  static const double fcc[4][3] = {{0, 0, 0}, {0, .5, .5}, {.5, 0, .5}, {.5, .5, 0}}, bcc[2][3] = {{0, 0, 0}, {.5, .5, .5}};
  oracle_set_threads(2);
  /* 1. TB-SMA Cu-like, three species with per-pair cut-offs, three boxes of 5^3 cells */
  {
    double *x, *v; int *type;
    const int nt = 3, nb = 3, n = lattice(5, 3.615, fcc, 4, nb, 0.05, &x, &v, &type, nt);
    double A[9], xi[9], p[9], q[9], r0[9], rcp[9], ron[9], mass[3] = {63.546, 108.0, 82.6};
    for (int s = 0; s < nt; ++s) for (int t = 0; t < nt; ++t) {
      const int k = s * nt + t; const double u = 0.02 * (s + t) + 0.01 * s * t;
      A[k] = 0.0855 * (1 + u); xi[k] = 1.224 * (1 - 0.5 * u); p[k] = 10.96; q[k] = 2.278 * (1 + 2 * u); r0[k] = 2.5562 * (1 + 0.5 * u);
      rcp[k] = 4.9 - 0.1 * (s + t); ron[k] = rcp[k] - 0.5;
    }
    oracle_desc d; memset(&d, 0, sizeof d);
    d.n_atoms = n; d.n_boxes = nb; d.n_types = nt; d.box[0] = d.box[1] = d.box[2] = 5 * 3.615; d.cutoff = 4.9; d.skin = 0.3;
    d.positions = x; d.velocities = v; d.types = type; d.mass = mass; d.pot_kind = 0;
    d.A = A; d.xi = xi; d.p = p; d.q = q; d.r0 = r0; d.taper_on = 4.4; d.pair_cutoff = rcp; d.pair_taper_on = ron;
    oracle_system *s = NULL;
    CHECK(oracle_create(&d, &s));
    if (exercise(s, n, nb, 1)) return 1;
    CHECK(oracle_destroy(s));
    free(x); free(v); free(type);
  }
  /* 2. tabulated EAM (Fe-form), two species, one box of 6^3 bcc cells, rho_max below the lattice density */
  {
    double *x, *v; int *type;
    const int nt = 2, nr = 800, nrho = 300, n = lattice(6, 2.855, bcc, 2, 1, 0.05, &x, &v, &type, nt);
    const double rc = 5.0, dr = rc / (nr - 1), rho_max = 9.0, drho = rho_max / (nrho - 1), re = 2.4725;
    double *fv = (double *)malloc(4 * nr * sizeof(double)), *fd = (double *)malloc(4 * nr * sizeof(double));
    double *pv = (double *)malloc(4 * nr * sizeof(double)), *pd = (double *)malloc(4 * nr * sizeof(double));
    double *Fv = (double *)malloc(2 * nrho * sizeof(double)), *Fd = (double *)malloc(2 * nrho * sizeof(double));
    for (int tp = 0; tp < 4; ++tp) for (int k = 0; k < nr; ++k) {
      const double sc = 1.0 + 0.02 * ((tp >> 1) + (tp & 1)), xx = k * dr / (re * sc) - 1.0;
      fv[tp * nr + k] = exp(-6.0 * xx); fd[tp * nr + k] = -(6.0 / (re * sc)) * fv[tp * nr + k];
      pv[tp * nr + k] = 0.4 * exp(-8.0 * xx) - 0.6 * exp(-4.0 * xx);
      pd[tp * nr + k] = -(8.0 / (re * sc)) * 0.4 * exp(-8.0 * xx) + (4.0 / (re * sc)) * 0.6 * exp(-4.0 * xx);
    }
    for (int t = 0; t < 2; ++t) for (int k = 0; k < nrho; ++k) {
      const double rho = k * drho, F0 = 2.5 + 0.4 * t;
      Fv[t * nrho + k] = -F0 * sqrt(rho / 20.0);
      Fd[t * nrho + k] = k ? -F0 / (2.0 * sqrt(rho * 20.0)) : -F0 * sqrt(drho / 20.0) / drho;
    }
    double mass[2] = {55.845, 94.9};
    oracle_desc d; memset(&d, 0, sizeof d);
    d.n_atoms = n; d.n_boxes = 1; d.n_types = nt; d.box[0] = d.box[1] = d.box[2] = 6 * 2.855; d.cutoff = rc; d.skin = 0.3;
    d.positions = x; d.velocities = v; d.types = type; d.mass = mass; d.pot_kind = 1;
    d.nr = nr; d.dr = dr; d.f_val = fv; d.f_der = fd; d.phi_val = pv; d.phi_der = pd; d.nrho = nrho; d.drho = drho; d.F_val = Fv; d.F_der = Fd;
    oracle_system *s = NULL;
    CHECK(oracle_create(&d, &s));
    if (exercise(s, n, 1, 1)) return 1;
    CHECK(oracle_destroy(s));
    /* error paths free what they allocated */
    d.box[0] = 9.0;
    if (oracle_create(&d, &s) != ORACLE_EBOX) return 1;
    d.box[0] = 6 * 2.855; type[3] = 7;
    if (oracle_create(&d, &s) != ORACLE_EINVAL) return 1;
    type[3] = 0; mass[1] = -1.0;
    if (oracle_create(&d, &s) != ORACLE_EINVAL) return 1;
    free(x); free(v); free(type); free(fv); free(fd); free(pv); free(pd); free(Fv); free(Fd);
  }
  printf("asan-main ok\n");
  return 0;
}
