/*
 * oracle/psc_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the explicit electromagnetic particle-in-cell step of
 * arXiv:1310.7866 (Germaschewski et al., "The Plasma Simulation Code"), written from the
 * paper's equations.  It shares no code, headers, tables or helpers with the CUDA path under
 * paper_1310_7866_b200/ and may be imported / linked / executed only by tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg.
 *
 * This file is the "T1 stencil oracle" (O(N_p) per step).  The definition-level brute force
 * ("T0", loops over all grid points, Eq. 29-31 evaluated directly, flux definition by time
 * quadrature) lives in oracle/brute_force.py and is used to pin this file on 1-8 particles.
 *
 * Conventions:
 *   - units c = eps0 = mu0 = 1; u = p/(m c) is stored in the momentum columns; qw = q_s * w.
 *   - grid indices (i,j,k) <-> (x,y,z); a direction with n[d] == 1 is invariant.
 *   - fields are stored WITHOUT ghosts, periodic by modular indexing:
 *       F[c][k][j][i] at  ((c*nz + k)*ny + j)*nx + i
 *     Yee staggering (Eq. 20-21):
 *       E[0]=E_x(i+1/2,j,k) E[1]=E_y(i,j+1/2,k) E[2]=E_z(i,j,k+1/2)
 *       B[0]=B_x(i,j+1/2,k+1/2) B[1]=B_y(i+1/2,j,k+1/2) B[2]=B_z(i+1/2,j+1/2,k)
 *     J is co-located with E, rho sits on nodes (i,j,k).
 *   - state at step entry: E^{n+1/2}, B^n, x^{n+1/2}, u^n; one step is Fig. 8
 *     (PAPER.md:390-412).
 *
 * Every function is pinned by tests/test_oracle_*.py (closed forms, invariants, brute force);
 * nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
  int32_t n[3];      /* interior cells x,y,z; 1 = invariant direction */
  int32_t order;     /* 1: b1 gather + Villasenor-Buneman; 2: b2 gather + Esirkepov */
  int32_t n_species; /* <= 8 */
  int32_t block[3];  /* sort block (supercell) size in cells; divides n[d] */
  double dx[3];
  double dt;
  double q[8], m[8];
  int32_t scheme;    /* 0: every weight of the gather has the order above; 1: alternating order
                        ([22]; A29): along a direction in which a field
                        component is half-staggered its gather weight is one order LOWER
                        (order 1: b0 instead of b1; order 2: b1 instead of b2) */
} orc_params;

/* ------------------------------------------------------------------------------------------ */
/* indexing                                                                                    */

static inline int wrapi(int i, int n) {
  int r = i % n;
  return r < 0 ? r + n : r;
}

static inline int64_t fidx(const orc_params *p, int c, int i, int j, int k) {
  const int nx = p->n[0], ny = p->n[1], nz = p->n[2];
  return (((int64_t)c * nz + wrapi(k, nz)) * ny + wrapi(j, ny)) * nx + wrapi(i, nx);
}

static inline int64_t ncells(const orc_params *p) {
  return (int64_t)p->n[0] * p->n[1] * p->n[2];
}

int orc_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

void orc_set_num_threads(int n) {
#ifdef _OPENMP
  omp_set_num_threads(n);
#else
  (void)n;
#endif
}

static inline int team_size(void) { /* threads of the enclosing parallel region */
#ifdef _OPENMP
  return omp_get_num_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------------------------------ */
/* discrete operators, PAPER.md:100-118 (Eq. 12-16)                                            */

/* (curl+ F)_c: forward differences; takes an E-staggered field to the B-staggered locations.
 * Eq. 12: (curl+ E)_x,i,j+1/2,k+1/2 = (E_z[i,j+1,k]-E_z[i,j,k])/dy - (E_y[i,j,k+1]-E_y[i,j,k])/dz,
 * y and z components by cyclic permutation. */
void orc_curl_plus(const orc_params *p, const double *F, double *out) {
  const int nx = p->n[0], ny = p->n[1], nz = p->n[2];
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        out[fidx(p, 0, i, j, k)] = (F[fidx(p, 2, i, j + 1, k)] - F[fidx(p, 2, i, j, k)]) / p->dx[1] -
                                   (F[fidx(p, 1, i, j, k + 1)] - F[fidx(p, 1, i, j, k)]) / p->dx[2];
        out[fidx(p, 1, i, j, k)] = (F[fidx(p, 0, i, j, k + 1)] - F[fidx(p, 0, i, j, k)]) / p->dx[2] -
                                   (F[fidx(p, 2, i + 1, j, k)] - F[fidx(p, 2, i, j, k)]) / p->dx[0];
        out[fidx(p, 2, i, j, k)] = (F[fidx(p, 1, i + 1, j, k)] - F[fidx(p, 1, i, j, k)]) / p->dx[0] -
                                   (F[fidx(p, 0, i, j + 1, k)] - F[fidx(p, 0, i, j, k)]) / p->dx[1];
      }
}

/* (curl- F)_c: backward differences; takes a B-staggered field to the E-staggered locations.
 * Eq. 13: (curl- B)_x,i+1/2,j,k = (B_z[i,j,k]-B_z[i,j-1,k])/dy - (B_y[i,j,k]-B_y[i,j,k-1])/dz. */
void orc_curl_minus(const orc_params *p, const double *F, double *out) {
  const int nx = p->n[0], ny = p->n[1], nz = p->n[2];
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++) {
        out[fidx(p, 0, i, j, k)] = (F[fidx(p, 2, i, j, k)] - F[fidx(p, 2, i, j - 1, k)]) / p->dx[1] -
                                   (F[fidx(p, 1, i, j, k)] - F[fidx(p, 1, i, j, k - 1)]) / p->dx[2];
        out[fidx(p, 1, i, j, k)] = (F[fidx(p, 0, i, j, k)] - F[fidx(p, 0, i, j, k - 1)]) / p->dx[2] -
                                   (F[fidx(p, 2, i, j, k)] - F[fidx(p, 2, i - 1, j, k)]) / p->dx[0];
        out[fidx(p, 2, i, j, k)] = (F[fidx(p, 1, i, j, k)] - F[fidx(p, 1, i - 1, j, k)]) / p->dx[0] -
                                   (F[fidx(p, 0, i, j, k)] - F[fidx(p, 0, i, j - 1, k)]) / p->dx[1];
      }
}

/* Eq. 15: (div+ B) at cell centres (i+1/2,j+1/2,k+1/2); forward differences of a B-staggered
 * field (the last term is read as (B_z[k+1]-B_z[k])/dz, forced by Eq. 23; A3). */
void orc_div_plus(const orc_params *p, const double *F, double *out) {
  const int nx = p->n[0], ny = p->n[1], nz = p->n[2];
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++)
        out[fidx(p, 0, i, j, k)] = (F[fidx(p, 0, i + 1, j, k)] - F[fidx(p, 0, i, j, k)]) / p->dx[0] +
                                   (F[fidx(p, 1, i, j + 1, k)] - F[fidx(p, 1, i, j, k)]) / p->dx[1] +
                                   (F[fidx(p, 2, i, j, k + 1)] - F[fidx(p, 2, i, j, k)]) / p->dx[2];
}

/* Eq. 16: (div- E) at nodes (i,j,k); backward differences of an E-staggered field (first term
 * read as (E_x[i]-E_x[i-1])/dx; A3). */
void orc_div_minus(const orc_params *p, const double *F, double *out) {
  const int nx = p->n[0], ny = p->n[1], nz = p->n[2];
  for (int k = 0; k < nz; k++)
    for (int j = 0; j < ny; j++)
      for (int i = 0; i < nx; i++)
        out[fidx(p, 0, i, j, k)] = (F[fidx(p, 0, i, j, k)] - F[fidx(p, 0, i - 1, j, k)]) / p->dx[0] +
                                   (F[fidx(p, 1, i, j, k)] - F[fidx(p, 1, i, j - 1, k)]) / p->dx[1] +
                                   (F[fidx(p, 2, i, j, k)] - F[fidx(p, 2, i, j, k - 1)]) / p->dx[2];
}

/* ------------------------------------------------------------------------------------------ */
/* FDTD leap-frog, PAPER.md:131-134 (Eq. 17-18), Fig. 8                                        */

/* B -= frac*dt * curl+ E   (Eq. 18; frac = 1/2 twice per step) */
void orc_push_b(const orc_params *p, const double *E, double *B, double frac) {
  const int64_t nc = ncells(p);
  double *curl = (double *)malloc(sizeof(double) * 3 * nc);
  orc_curl_plus(p, E, curl);
  for (int64_t a = 0; a < 3 * nc; a++) B[a] -= frac * p->dt * curl[a];
  free(curl);
}

/* E += frac*dt * (curl- B - J)   (Eq. 17 with c = eps0 = 1; frac = 1 in Fig. 8) */
void orc_push_e(const orc_params *p, double *E, const double *B, const double *J, double frac) {
  const int64_t nc = ncells(p);
  double *curl = (double *)malloc(sizeof(double) * 3 * nc);
  orc_curl_minus(p, B, curl);
  for (int64_t a = 0; a < 3 * nc; a++) E[a] += frac * p->dt * (curl[a] - J[a]);
  free(curl);
}

/* ------------------------------------------------------------------------------------------ */
/* B-splines, PAPER.md:183-193 (Eq. 29, 31)                                                    */

static inline double b1(double xi) {
  if (xi >= -1.0 && xi <= 0.0) return 1.0 + xi;
  if (xi >= 0.0 && xi <= 1.0) return 1.0 - xi;
  return 0.0;
}

static inline double b2(double xi) {
  if (xi >= -1.5 && xi <= -0.5) return 0.5 * (1.5 + xi) * (1.5 + xi);
  if (xi >= -0.5 && xi <= 0.5) return 0.75 - xi * xi;
  if (xi >= 0.5 && xi <= 1.5) return 0.5 * (1.5 - xi) * (1.5 - xi);
  return 0.0;
}

/* ------------------------------------------------------------------------------------------ */
/* gather, PAPER.md:88-92 (Eq. 11), 196: each component interpolated from its own staggered    */
/* points with b1 (order 1) or b2 (order 2); factor 1 along an invariant direction.  With the   */
/* alternating-order scheme the weight along a half-staggered direction of the   */
/* component is one order lower; the deposit, and with it charge conservation, is unchanged.    */

/* 1-d stencil for a sample point xi (in units of cells, measured from the first staggered
 * location of this component, i.e. stag already subtracted): fills idx0, npts, w[].           */
static inline void stencil(int order, int n, double xi, int *idx0, int *npts, double w[3]) {
  if (n == 1) {
    *idx0 = 0;
    *npts = 1;
    w[0] = 1.0;
    return;
  }
  if (order == 0) { /* b0: the nearest point (alternating-order gather of first-order particles) */
    *idx0 = (int)floor(xi + 0.5);
    *npts = 1;
    w[0] = 1.0;
  } else if (order == 1) {
    int i0 = (int)floor(xi);
    *idx0 = i0;
    *npts = 2;
    w[0] = b1(xi - i0);
    w[1] = b1(xi - (i0 + 1));
  } else {
    int i0 = (int)floor(xi + 0.5);
    *idx0 = i0 - 1;
    *npts = 3;
    w[0] = b2(xi - (i0 - 1));
    w[1] = b2(xi - i0);
    w[2] = b2(xi - (i0 + 1));
  }
}

static double gather_one(const orc_params *p, const double *F, int c, const double stag[3],
                         const double x[3]) {
  int i0[3], np[3];
  double w[3][3];
  for (int d = 0; d < 3; d++)
    stencil(p->order - ((p->scheme == 1 && stag[d] != 0.0) ? 1 : 0), p->n[d], x[d] / p->dx[d] - stag[d],
            &i0[d], &np[d], w[d]);
  double s = 0.0;
  for (int c2 = 0; c2 < np[2]; c2++)
    for (int c1 = 0; c1 < np[1]; c1++)
      for (int c0 = 0; c0 < np[0]; c0++)
        s += F[fidx(p, c, i0[0] + c0, i0[1] + c1, i0[2] + c2)] * w[0][c0] * w[1][c1] * w[2][c2];
  return s;
}

static const double STAG_E[3][3] = {{0.5, 0, 0}, {0, 0.5, 0}, {0, 0, 0.5}};
static const double STAG_B[3][3] = {{0, 0.5, 0.5}, {0.5, 0, 0.5}, {0.5, 0.5, 0}};

static void gather_eb(const orc_params *p, const double *E, const double *B, const double x[3],
                      double Ep[3], double Bp[3]) {
  for (int c = 0; c < 3; c++) {
    Ep[c] = gather_one(p, E, c, STAG_E[c], x);
    Bp[c] = gather_one(p, B, c, STAG_B[c], x);
  }
}

/* out: EB[6*n] = (Ex,Ey,Ez,Bx,By,Bz) per particle */
void orc_gather(const orc_params *p, const double *E, const double *B, int64_t n, const double *x,
                const double *y, const double *z, double *EB) {
  for (int64_t a = 0; a < n; a++) {
    double pos[3] = {x[a], y[a], z[a]};
    gather_eb(p, E, B, pos, EB + 6 * a, EB + 6 * a + 3);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* Boris push, PAPER.md:171-179 (Eq. 27-28); gamma^{n+1/2} read as Boris's gamma^- (A6)        */

static void boris(double u[3], const double Ep[3], const double Bp[3], double h /* q dt/(2m) */) {
  double um[3], t[3], s[3], up[3], upl[3];
  for (int c = 0; c < 3; c++) um[c] = u[c] + h * Ep[c]; /* half electric kick */
  double gm = sqrt(1.0 + um[0] * um[0] + um[1] * um[1] + um[2] * um[2]);
  for (int c = 0; c < 3; c++) t[c] = h * Bp[c] / gm;
  double t2 = t[0] * t[0] + t[1] * t[1] + t[2] * t[2];
  for (int c = 0; c < 3; c++) s[c] = 2.0 * t[c] / (1.0 + t2);
  /* u' = u- + u- x t */
  up[0] = um[0] + (um[1] * t[2] - um[2] * t[1]);
  up[1] = um[1] + (um[2] * t[0] - um[0] * t[2]);
  up[2] = um[2] + (um[0] * t[1] - um[1] * t[0]);
  /* u+ = u- + u' x s */
  upl[0] = um[0] + (up[1] * s[2] - up[2] * s[1]);
  upl[1] = um[1] + (up[2] * s[0] - up[0] * s[2]);
  upl[2] = um[2] + (up[0] * s[1] - up[1] * s[0]);
  for (int c = 0; c < 3; c++) u[c] = upl[c] + h * Ep[c]; /* second half kick */
}

/* Momentum update only, with given per-particle fields EB[6*n]; u updated in place. */
void orc_boris(const orc_params *p, int64_t n, double *ux, double *uy, double *uz,
               const int32_t *species, const double *EB) {
  for (int64_t a = 0; a < n; a++) {
    const int s = species[a];
    double u[3] = {ux[a], uy[a], uz[a]};
    boris(u, EB + 6 * a, EB + 6 * a + 3, p->q[s] * p->dt / (2.0 * p->m[s]));
    ux[a] = u[0];
    uy[a] = u[1];
    uz[a] = u[2];
  }
}

/* ------------------------------------------------------------------------------------------ */
/* charge density on nodes (diagnostic): rho = sum qw/dV * s(xi_x-i)s(xi_y-j)s(xi_z-k) */

void orc_rho(const orc_params *p, int64_t n, const double *x, const double *y, const double *z,
             const double *qw, double *rho) {
  const int64_t nc = ncells(p);
  const double dV = p->dx[0] * p->dx[1] * p->dx[2];
  const double zero[3] = {0, 0, 0};
  memset(rho, 0, sizeof(double) * nc);
#pragma omp parallel
  {
    double *loc = (double *)calloc(nc, sizeof(double));
#pragma omp for schedule(static)
    for (int64_t a = 0; a < n; a++) {
      const double pos[3] = {x[a], y[a], z[a]};
      int i0[3], np[3];
      double w[3][3];
      for (int d = 0; d < 3; d++)
        stencil(p->order, p->n[d], pos[d] / p->dx[d] - zero[d], &i0[d], &np[d], w[d]);
      for (int c2 = 0; c2 < np[2]; c2++)
        for (int c1 = 0; c1 < np[1]; c1++)
          for (int c0 = 0; c0 < np[0]; c0++)
            loc[fidx(p, 0, i0[0] + c0, i0[1] + c1, i0[2] + c2)] +=
                qw[a] / dV * w[0][c0] * w[1][c1] * w[2][c2];
    }
#pragma omp for ordered schedule(static, 1)
    for (int t = 0; t < team_size(); t++) {
#pragma omp ordered
      for (int64_t a = 0; a < nc; a++) rho[a] += loc[a];
    }
    free(loc);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* order 1: Villasenor-Buneman.  The current is the exact flux of the charge  */
/* cloud moving on the straight line x0 -> x1 during the step; evaluated by splitting the line  */
/* at every cell face it crosses (<= 1 per direction since c dt < dx).            */

/* one segment a -> b (in-cell offsets, units of cells) inside `cell`, lasting the fraction tau
 * of the step.  For direction c with transverse directions e,f:
 *   j_c(cell_c + 1/2, cell_e + al, cell_f + be) += (qw/dV) * (del_c dx_c / dt) * W_{al,be}
 *   W_00 = (1-m_e)(1-m_f) + del_e del_f/12   W_10 = m_e(1-m_f) - del_e del_f/12
 *   W_01 = (1-m_e)m_f - del_e del_f/12       W_11 = m_e m_f + del_e del_f/12
 * with m = (a+b)/2, del = b-a.  Along an invariant direction the weight is 1 at index 0 and
 * del = 0; the current ALONG an invariant direction uses v_c * tau in place of del_c dx_c/dt
 * (time average of v_c S_e S_f over the segment; A12). */
static void vb_segment(const orc_params *p, double *J, const int cell[3], const double a[3],
                       const double b[3], double tau, const double v[3], double qw_dV) {
  double m[3], del[3];
  for (int d = 0; d < 3; d++) {
    if (p->n[d] == 1) {
      m[d] = 0.0;
      del[d] = 0.0;
    } else {
      m[d] = 0.5 * (a[d] + b[d]);
      del[d] = b[d] - a[d];
    }
  }
  for (int c = 0; c < 3; c++) {
    const int e = (c + 1) % 3, f = (c + 2) % 3;
    const double cur = qw_dV * (p->n[c] == 1 ? v[c] * tau : del[c] * p->dx[c] / p->dt);
    const int ne = p->n[e] == 1 ? 1 : 2, nf = p->n[f] == 1 ? 1 : 2;
    for (int be = 0; be < nf; be++)
      for (int al = 0; al < ne; al++) {
        const double we = ne == 1 ? 1.0 : (al ? m[e] : 1.0 - m[e]);
        const double wf = nf == 1 ? 1.0 : (be ? m[f] : 1.0 - m[f]);
        double W = we * wf;
        if (ne == 2 && nf == 2) W += (al == be ? 1.0 : -1.0) * del[e] * del[f] / 12.0;
        int ijk[3];
        ijk[c] = cell[c];
        ijk[e] = cell[e] + al;
        ijk[f] = cell[f] + be;
        J[fidx(p, c, ijk[0], ijk[1], ijk[2])] += cur * W;
      }
  }
}

static void vb_deposit(const orc_params *p, double *J, const double x0[3], const double x1[3],
                       const double v[3], double qw) {
  const double qw_dV = qw / (p->dx[0] * p->dx[1] * p->dx[2]);
  double xi0[3], xi1[3];
  int cell[3];
  /* crossing events */
  double et[3];
  int ed[3], edir[3], ne = 0;
  for (int d = 0; d < 3; d++) {
    if (p->n[d] == 1) {
      xi0[d] = xi1[d] = 0.0;
      cell[d] = 0;
      continue;
    }
    xi0[d] = x0[d] / p->dx[d];
    xi1[d] = x1[d] / p->dx[d];
    cell[d] = (int)floor(xi0[d]);
    const int c1 = (int)floor(xi1[d]);
    if (c1 != cell[d]) {
      const int dir = c1 > cell[d] ? 1 : -1;
      const double face = dir > 0 ? cell[d] + 1 : cell[d];
      et[ne] = (face - xi0[d]) / (xi1[d] - xi0[d]);
      ed[ne] = d;
      edir[ne] = dir;
      ne++;
    }
  }
  /* sort events by parametric time (insertion sort, <= 3 entries) */
  for (int a = 1; a < ne; a++)
    for (int b = a; b > 0 && et[b] < et[b - 1]; b--) {
      double tt = et[b]; et[b] = et[b - 1]; et[b - 1] = tt;
      int ti = ed[b]; ed[b] = ed[b - 1]; ed[b - 1] = ti;
      ti = edir[b]; edir[b] = edir[b - 1]; edir[b - 1] = ti;
    }
  double pos[3] = {xi0[0], xi0[1], xi0[2]};
  double tprev = 0.0;
  for (int ev = 0; ev <= ne; ev++) {
    double end[3], t;
    if (ev < ne) {
      t = et[ev];
      for (int d = 0; d < 3; d++) end[d] = xi0[d] + t * (xi1[d] - xi0[d]);
      end[ed[ev]] = edir[ev] > 0 ? cell[ed[ev]] + 1 : cell[ed[ev]]; /* exactly on the face */
    } else {
      t = 1.0;
      for (int d = 0; d < 3; d++) end[d] = xi1[d];
    }
    double a[3], b[3];
    for (int d = 0; d < 3; d++) {
      a[d] = pos[d] - cell[d];
      b[d] = end[d] - cell[d];
    }
    if (t > tprev) vb_segment(p, J, cell, a, b, t - tprev, v, qw_dV);
    if (ev < ne) cell[ed[ev]] += edir[ev];
    for (int d = 0; d < 3; d++) pos[d] = end[d];
    tprev = t;
  }
}

/* ------------------------------------------------------------------------------------------ */
/* order 2: Esirkepov density decomposition, PAPER.md:204 (A13).                     */
/*   i0_d = floor(xi0_d + 1/2); on nodes i0_d-2 .. i0_d+2: S0 = b2(xi0 - node), S1 = b2(xi1 - node),
 *   DS = S1 - S0;
 *   W_c[i_c, i_e, i_f] = DS_c[i_c] (S0_e S0_f + DS_e S0_f/2 + S0_e DS_f/2 + DS_e DS_f/3)
 *   j_c(i_c + 1/2, i_e, i_f) = j_c(i_c - 1/2, i_e, i_f) - (qw/dV)(dx_c/dt) W_c   (running sum from 0).
 * Along an invariant direction c: j_c(i_e,i_f) = (qw/dV) v_c * bracket.                         */
static void esirkepov_deposit(const orc_params *p, double *J, const double x0[3],
                              const double x1[3], const double v[3], double qw) {
  const double qw_dV = qw / (p->dx[0] * p->dx[1] * p->dx[2]);
  int i0[3], np[3];
  double S0[3][5], DS[3][5];
  for (int d = 0; d < 3; d++) {
    if (p->n[d] == 1) {
      i0[d] = 0;
      np[d] = 1;
      S0[d][0] = 1.0;
      DS[d][0] = 0.0;
      continue;
    }
    const double xi0 = x0[d] / p->dx[d], xi1 = x1[d] / p->dx[d];
    const int c = (int)floor(xi0 + 0.5);
    i0[d] = c - 2;
    np[d] = 5;
    for (int s = 0; s < 5; s++) {
      S0[d][s] = b2(xi0 - (c - 2 + s));
      DS[d][s] = b2(xi1 - (c - 2 + s)) - S0[d][s];
    }
  }
  for (int c = 0; c < 3; c++) {
    const int e = (c + 1) % 3, f = (c + 2) % 3;
    for (int jf = 0; jf < np[f]; jf++)
      for (int je = 0; je < np[e]; je++) {
        const double br = S0[e][je] * S0[f][jf] + 0.5 * DS[e][je] * S0[f][jf] +
                          0.5 * S0[e][je] * DS[f][jf] + DS[e][je] * DS[f][jf] / 3.0;
        int ijk[3];
        ijk[e] = i0[e] + je;
        ijk[f] = i0[f] + jf;
        if (p->n[c] == 1) {
          ijk[c] = 0;
          J[fidx(p, c, ijk[0], ijk[1], ijk[2])] += qw_dV * v[c] * br;
        } else {
          double run = 0.0;
          for (int s = 0; s < 5; s++) {
            run -= qw_dV * (p->dx[c] / p->dt) * DS[c][s] * br;
            ijk[c] = i0[c] + s;
            J[fidx(p, c, ijk[0], ijk[1], ijk[2])] += run;
          }
        }
      }
  }
}

/* Deposit only: J += current of particles moving x0 -> x1 (x1 unwrapped).  v* are used only for
 * the current along invariant directions.  Serial; for the pins. */
void orc_deposit(const orc_params *p, double *J, int64_t n, const double *x0, const double *y0,
                 const double *z0, const double *x1, const double *y1, const double *z1,
                 const double *vx, const double *vy, const double *vz, const double *qw) {
  for (int64_t a = 0; a < n; a++) {
    const double p0[3] = {x0[a], y0[a], z0[a]}, p1[3] = {x1[a], y1[a], z1[a]};
    const double v[3] = {vx[a], vy[a], vz[a]};
    if (p->order == 1)
      vb_deposit(p, J, p0, p1, v, qw[a]);
    else
      esirkepov_deposit(p, J, p0, p1, v, qw[a]);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* the particle loop of Fig. 8: gather at x^{n+1/2}, p^n -> p^{n+1},         */
/* x^{n+1/2} -> x^{n+3/2}, deposit j^{n+1}, then periodic wrap (A14).  J is zeroed first.        */

static inline double wrap_pos(double x, double L) {
  if (x < 0.0) x += L;
  if (x >= L) x -= L;
  if (x >= L) x = 0.0;
  return x;
}

void orc_push_particles(const orc_params *p, const double *E, const double *B, double *J,
                        int64_t n, double *x, double *y, double *z, double *ux, double *uy,
                        double *uz, const double *qw, const int32_t *species) {
  const int64_t nc = ncells(p);
  memset(J, 0, sizeof(double) * 3 * nc);
#pragma omp parallel
  {
    double *loc = (double *)calloc(3 * nc, sizeof(double));
#pragma omp for schedule(static)
    for (int64_t a = 0; a < n; a++) {
      const int s = species[a];
      double x0[3] = {x[a], y[a], z[a]};
      double u[3] = {ux[a], uy[a], uz[a]};
      double Ep[3], Bp[3];
      gather_eb(p, E, B, x0, Ep, Bp);
      boris(u, Ep, Bp, p->q[s] * p->dt / (2.0 * p->m[s]));
      const double g = sqrt(1.0 + u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
      const double v[3] = {u[0] / g, u[1] / g, u[2] / g};
      double x1[3];
      for (int d = 0; d < 3; d++) x1[d] = p->n[d] == 1 ? x0[d] : x0[d] + p->dt * v[d]; /* Eq. 26 */
      if (p->order == 1)
        vb_deposit(p, loc, x0, x1, v, qw[a]);
      else
        esirkepov_deposit(p, loc, x0, x1, v, qw[a]);
      for (int d = 0; d < 3; d++)
        if (p->n[d] != 1) x1[d] = wrap_pos(x1[d], p->n[d] * p->dx[d]);
      x[a] = x1[0]; y[a] = x1[1]; z[a] = x1[2];
      ux[a] = u[0]; uy[a] = u[1]; uz[a] = u[2];
    }
#pragma omp for ordered schedule(static, 1)
    for (int t = 0; t < team_size(); t++) {
#pragma omp ordered
      for (int64_t a = 0; a < 3 * nc; a++) J[a] += loc[a];
    }
    free(loc);
  }
}

/* ------------------------------------------------------------------------------------------ */
/* one full step, Fig. 8; the sort is not part of the physics.              */

void orc_step(const orc_params *p, double *E, double *B, double *J, int64_t n, double *x, double *y,
              double *z, double *ux, double *uy, double *uz, const double *qw,
              const int32_t *species, int nsteps) {
  for (int s = 0; s < nsteps; s++) {
    orc_push_b(p, E, B, 0.5);                                          /* B^n -> B^{n+1/2} */
    orc_push_particles(p, E, B, J, n, x, y, z, ux, uy, uz, qw, species); /* p, x, j^{n+1} */
    orc_push_b(p, E, B, 0.5);                                          /* B^{n+1/2} -> B^{n+1} */
    orc_push_e(p, E, B, J, 1.0);                                       /* E^{n+1/2} -> E^{n+3/2} */
  }
}

/* ------------------------------------------------------------------------------------------ */
/* energies (diagnostic; quantities as stored, staggered time levels, A22)                     */

/* out[0] = 1/2 sum E^2 dV, out[1] = 1/2 sum B^2 dV, out[2] = sum_p w m_s (gamma - 1) */
void orc_energy(const orc_params *p, const double *E, const double *B, int64_t n, const double *ux,
                const double *uy, const double *uz, const double *qw, const int32_t *species,
                double out[3]) {
  const int64_t nc = ncells(p);
  const double dV = p->dx[0] * p->dx[1] * p->dx[2];
  double e = 0, b = 0, k = 0;
  for (int64_t a = 0; a < 3 * nc; a++) {
    e += E[a] * E[a];
    b += B[a] * B[a];
  }
  for (int64_t a = 0; a < n; a++) {
    const int s = species[a];
    const double u2 = ux[a] * ux[a] + uy[a] * uy[a] + uz[a] * uz[a];
    /* gamma - 1 = u^2/(gamma + 1), stable for small u */
    k += (qw[a] / p->q[s]) * p->m[s] * u2 / (sqrt(1.0 + u2) + 1.0);
  }
  out[0] = 0.5 * e * dV;
  out[1] = 0.5 * b * dV;
  out[2] = k;
}

/* ------------------------------------------------------------------------------------------ */
/* Marder's Gauss-law correction, PAPER.md:206 ("the iterative method by Marder [24] to dissipate  */
/* violations of Gauss's Law"; the paper cites only, A28 records the reading):           */
/*   f = div- E - rho   on nodes  (Eq. 16, the Gauss residual of Eq. 24)                           */
/*   E <- E + D grad+ f,  (grad+ f)_x,i+1/2,j,k = (f[i+1,j,k] - f[i,j,k]) / dx  (cyclic),          */
/* repeated `iters` times with rho fixed.  D = d * dt is the diffusion number (units length^2):    */
/* since div- grad+ is the 7-point Laplacian, every pass multiplies a Fourier mode of the residual */
/* by 1 - D sum_d K_d^2, K_d = (2/dx_d) sin(k_d dx_d / 2); E with div- E = rho is left untouched.  */
void orc_marder(const orc_params *p, double *E, const double *rho, double D, int iters) {
  const int nx = p->n[0], ny = p->n[1], nz = p->n[2];
  const int64_t nc = ncells(p);
  double *f = (double *)malloc(sizeof(double) * nc);
  for (int it = 0; it < iters; it++) {
    orc_div_minus(p, E, f);
    for (int64_t a = 0; a < nc; a++) f[a] -= rho[a];
    for (int k = 0; k < nz; k++)
      for (int j = 0; j < ny; j++)
        for (int i = 0; i < nx; i++) {
          const double f0 = f[fidx(p, 0, i, j, k)];
          E[fidx(p, 0, i, j, k)] += D * (f[fidx(p, 0, i + 1, j, k)] - f0) / p->dx[0];
          E[fidx(p, 1, i, j, k)] += D * (f[fidx(p, 0, i, j + 1, k)] - f0) / p->dx[1];
          E[fidx(p, 2, i, j, k)] += D * (f[fidx(p, 0, i, j, k + 1)] - f0) / p->dx[2];
        }
  }
  free(f);
}

/* ------------------------------------------------------------------------------------------ */
/* cell-key counting sort.  One key orders by block (supercell) and by cell    */
/* inside the block at once.  Positions are the fp32 values the GPU path sees; the cell index   */
/* is floor of the fp32 product x * (1/dx) (both operands fp32), as the parity protocol fixes.  */
/* Returns 0, or -1 if a particle lies outside [0, n_d dx_d).                                    */

int orc_sort(const orc_params *p, int64_t n, const float *x, const float *y, const float *z,
             int32_t *cell_idx, int32_t *key, int32_t *perm, int32_t *cell_offsets) {
  const int64_t nk = ncells(p);
  const float *pos[3] = {x, y, z};
  int nb[3], bs[3];
  float inv_dx[3];
  for (int d = 0; d < 3; d++) {
    bs[d] = p->block[d];
    nb[d] = p->n[d] / bs[d];
    inv_dx[d] = 1.0f / (float)p->dx[d];
  }
  int64_t *count = (int64_t *)calloc(nk + 1, sizeof(int64_t));
  for (int64_t a = 0; a < n; a++) {
    int c[3];
    for (int d = 0; d < 3; d++) {
      if (p->n[d] == 1) {
        c[d] = 0;
        continue;
      }
      volatile float xi = pos[d][a] * inv_dx[d]; /* fp32 product, rounded once */
      c[d] = (int)floorf(xi);
      if (c[d] < 0 || c[d] >= p->n[d]) {
        free(count);
        return -1;
      }
    }
    const int b[3] = {c[0] / bs[0], c[1] / bs[1], c[2] / bs[2]};
    const int l[3] = {c[0] % bs[0], c[1] % bs[1], c[2] % bs[2]};
    const int64_t kk = (((int64_t)b[2] * nb[1] + b[1]) * nb[0] + b[0]) * ((int64_t)bs[0] * bs[1] * bs[2]) +
                       ((int64_t)l[2] * bs[1] + l[1]) * bs[0] + l[0];
    key[a] = (int32_t)kk;
    cell_idx[a] = (int32_t)(((int64_t)c[2] * p->n[1] + c[1]) * p->n[0] + c[0]);
    count[kk + 1]++;
  }
  for (int64_t a = 0; a < nk; a++) count[a + 1] += count[a]; /* exclusive scan of the histogram */
  for (int64_t a = 0; a <= nk; a++) cell_offsets[a] = (int32_t)count[a];
  /* stable scatter: ascending input index inside a key (A17) */
  for (int64_t a = 0; a < n; a++) perm[count[key[a]]++] = (int32_t)a;
  free(count);
  return 0;
}

/* The same stable counting sort with the cell of every particle GIVEN as integer
 * coordinates -- used on a list that a push has advanced: which cell a particle is in is then a
 * decision the GPU path has already taken in its own precision (where
 * floating point decides an integer, both sides take that decision in the kernel's precision), and
 * what is compared is everything that follows from it: keys, offsets, the stable permutation.
 * Returns 0, or -1 if a cell lies outside the grid.                                             */
int orc_sort_cells(const orc_params *p, int64_t n, const int32_t *cx, const int32_t *cy,
                   const int32_t *cz, int32_t *cell_idx, int32_t *key, int32_t *perm,
                   int32_t *cell_offsets) {
  const int64_t nk = ncells(p);
  const int32_t *cc[3] = {cx, cy, cz};
  int nb[3], bs[3];
  for (int d = 0; d < 3; d++) {
    bs[d] = p->block[d];
    nb[d] = p->n[d] / bs[d];
  }
  int64_t *count = (int64_t *)calloc(nk + 1, sizeof(int64_t));
  for (int64_t a = 0; a < n; a++) {
    int c[3];
    for (int d = 0; d < 3; d++) {
      c[d] = cc[d][a];
      if (c[d] < 0 || c[d] >= p->n[d]) {
        free(count);
        return -1;
      }
    }
    const int b[3] = {c[0] / bs[0], c[1] / bs[1], c[2] / bs[2]};
    const int l[3] = {c[0] % bs[0], c[1] % bs[1], c[2] % bs[2]};
    const int64_t kk = (((int64_t)b[2] * nb[1] + b[1]) * nb[0] + b[0]) * ((int64_t)bs[0] * bs[1] * bs[2]) +
                       ((int64_t)l[2] * bs[1] + l[1]) * bs[0] + l[0];
    key[a] = (int32_t)kk;
    cell_idx[a] = (int32_t)(((int64_t)c[2] * p->n[1] + c[1]) * p->n[0] + c[0]);
    count[kk + 1]++;
  }
  for (int64_t a = 0; a < nk; a++) count[a + 1] += count[a];
  for (int64_t a = 0; a <= nk; a++) cell_offsets[a] = (int32_t)count[a];
  for (int64_t a = 0; a < n; a++) perm[count[key[a]]++] = (int32_t)a; /* stable (A17) */
  free(count);
  return 0;
}
