/* tslb_ref.c -- CPU ORACLE (test infrastructure, not the product).  See tslb_ref.h.
 *
 * Everything is written from PAPER.md (arXiv 2501.00846) equation by equation.  Citations are
 * "P:<line>" = PAPER.md line, "Rk" = reading k of DESIGN.md.  No blocking, fusion or
 * reordering beyond the paper's own sequence of stages.
 */
#include "tslb_ref.h"
#include <math.h>
#include <stdlib.h>
#include <string.h>

#define Q 27
/* Order of the sums over the 27 directions (stencils, Eq. 18-19; moments, Eq. 11-13).  The paper
 * does not fix it (R22).  The oracle sums in index order; -DTSLB_REF_REVERSE_SUMS builds the
 * conditioning twin that sums in reverse order (make_golden.py --twin-rev): another correct
 * rounding of the same program, never a source of expected values. */
#ifdef TSLB_REF_REVERSE_SUMS
#define FOR_SUM_Q(i) for (int i = Q - 1; i >= 0; --i)
#else
#define FOR_SUM_Q(i) for (int i = 0; i < Q; ++i)
#endif
#define OMP_MIN_NODES 8192   /* below this a pass runs on one thread (team start-up costs more) */
static const double CS2 = 1.0 / 3.0;     /* R1: cs^2 of D3Q27                       */
static const double EPS_N = 1e-12;       /* R13: n = grad(phi)/sqrt(|grad(phi)|^2 + eps^2) */

/* ---------------------------------------------------------------- L0 lattice (R1) ------ */
/* direction i <-> (cx,cy,cz) = (i%3 - 1, (i/3)%3 - 1, i/9 - 1); weights are products of the
 * one-dimensional weights 1/6, 2/3, 1/6. */
static int    Ci[Q][3];
static double Wi[Q];
static int    OPP[Q];
static double H2[Q][3][3];     /* c_a c_b - cs^2 d_ab  */
static double H3[Q][3][3][3];  /* c_a c_b c_g - cs^2 (c_g d_ab + c_a d_bg + c_b d_ag)  */
static int    tables_ready = 0;

static void build_tables(void) {
  if (tables_ready) return;
  const double w1[3] = {1.0 / 6.0, 2.0 / 3.0, 1.0 / 6.0};
  for (int i = 0; i < Q; ++i) {
    Ci[i][0] = i % 3 - 1; Ci[i][1] = (i / 3) % 3 - 1; Ci[i][2] = i / 9 - 1;
    Wi[i] = w1[Ci[i][0] + 1] * w1[Ci[i][1] + 1] * w1[Ci[i][2] + 1];
  }
  for (int i = 0; i < Q; ++i)
    for (int j = 0; j < Q; ++j)
      if (Ci[j][0] == -Ci[i][0] && Ci[j][1] == -Ci[i][1] && Ci[j][2] == -Ci[i][2]) OPP[i] = j;
  for (int i = 0; i < Q; ++i)
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) {
        H2[i][a][b] = Ci[i][a] * Ci[i][b] - CS2 * (a == b);
        for (int g = 0; g < 3; ++g)
          H3[i][a][b][g] = Ci[i][a] * Ci[i][b] * Ci[i][g]
                         - CS2 * (Ci[i][g] * (a == b) + Ci[i][a] * (b == g) + Ci[i][b] * (a == g));
      }
  tables_ready = 1;
}

void tslb_ref_lattice(int c[27][3], double w[27], int opp[27]) {
  build_tables();
  for (int i = 0; i < Q; ++i) {
    c[i][0] = Ci[i][0]; c[i][1] = Ci[i][1]; c[i][2] = Ci[i][2];
    w[i] = Wi[i]; opp[i] = OPP[i];
  }
}

/* symmetric tensor stored as 6 values xx,yy,zz,xy,xz,yz */
static const int SYM[3][3] = {{0, 3, 4}, {3, 1, 5}, {4, 5, 2}};

/* ---------------------------------------------------------------- L1 per-node physics -- */
/* Eq. 9: third-order Hermite equilibrium, zeroth moment is p*. */
void tslb_ref_feq(double pstar, const double u[3], double out[27]) {
  build_tables();
  double uu[3][3], uuu[3][3][3];            /* the tensors u_a u_b and u_a u_b u_g of Eq. 9 */
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b) {
      uu[a][b] = u[a] * u[b];
      for (int g = 0; g < 3; ++g) uuu[a][b][g] = u[a] * u[b] * u[g];
    }
  for (int i = 0; i < Q; ++i) {
    double t1 = 0.0, t2 = 0.0, t3 = 0.0;
    for (int a = 0; a < 3; ++a) t1 += Ci[i][a] * u[a];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) t2 += H2[i][a][b] * uu[a][b];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        for (int g = 0; g < 3; ++g) t3 += H3[i][a][b][g] * uuu[a][b][g];
    out[i] = Wi[i] * (pstar + t1 / CS2 + t2 / (2.0 * CS2 * CS2) + t3 / (6.0 * CS2 * CS2 * CS2));
  }
}

/* Eq. 10 with R2: weight w_i and the full second-order Hermite tensor;
 * a3_abg = u_a A_bg + u_b A_ag + u_g A_ab (recursive relation). */
void tslb_ref_fneq(const double u[3], const double A[6], double out[27]) {
  build_tables();
  double a3[3][3][3];
  for (int a = 0; a < 3; ++a)
    for (int b = 0; b < 3; ++b)
      for (int g = 0; g < 3; ++g)
        a3[a][b][g] = u[a] * A[SYM[b][g]] + u[b] * A[SYM[a][g]] + u[g] * A[SYM[a][b]];
  for (int i = 0; i < Q; ++i) {
    double t2 = 0.0, t3 = 0.0;
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b) t2 += H2[i][a][b] * A[SYM[a][b]];
    for (int a = 0; a < 3; ++a)
      for (int b = 0; b < 3; ++b)
        for (int g = 0; g < 3; ++g) t3 += H3[i][a][b][g] * a3[a][b][g];
    out[i] = Wi[i] * (t2 / (2.0 * CS2 * CS2) + t3 / (6.0 * CS2 * CS2 * CS2));
  }
}

/* Eq. 14 with R5: the "force" is the acceleration a = F/rho. */
void tslb_ref_forcing(const double u[3], const double a[3], double out[27]) {
  build_tables();
  for (int i = 0; i < Q; ++i) {
    double cu = 0.0;
    for (int b = 0; b < 3; ++b) cu += Ci[i][b] * u[b];
    double s = 0.0;
    for (int al = 0; al < 3; ++al)
      s += ((Ci[i][al] - u[al]) / CS2 + cu * Ci[i][al] / (CS2 * CS2)) * a[al];
    out[i] = Wi[i] * s;
  }
}

/* Mixture rules (R14, R15): phi is clamped to [0,1] here and only here. */
static double clamp01(double x) { return x < 0.0 ? 0.0 : (x > 1.0 ? 1.0 : x); }
static double mix_rho(const tslb_ref_params *p, double phi) {
  return p->rho_g + clamp01(phi) * (p->rho_l - p->rho_g);
}
static double mix_nu(const tslb_ref_params *p, double phi) {
  double mu = p->mu_g + clamp01(phi) * (p->mu_l - p->mu_g);
  return mu / mix_rho(p, phi);
}
double tslb_ref_omega(const tslb_ref_params *p, double phi) {
  return 1.0 / (mix_nu(p, phi) / CS2 + 0.5);
}

/* ---------------------------------------------------------------- ghost rules (R19) ---- */
/* Index of the real node that supplies position i on an axis of n nodes.  Periodic axes wrap.
 * On a wall axis the wall sits half a cell outside the first/last node and positions beyond
 * it are mirrored: -1 -> 0, -2 -> 1, n -> n-1, n+1 -> n-2.  *crossed is set when mirrored. */
static int ghost_index(int i, int n, int bc, int *crossed) {
  *crossed = 0;
  if (bc == TSLB_REF_PERIODIC) return ((i % n) + n) % n;
  if (i < 0)  { *crossed = 1; return -1 - i; }
  if (i >= n) { *crossed = 1; return 2 * n - 1 - i; }
  return i;
}

typedef struct { long idx; int cross[3]; } nbr_t;

static nbr_t neighbour(int ix, int iy, int iz, int nx, int ny, int nz, const int bc[3]) {
  nbr_t r;
  int jx = ghost_index(ix, nx, bc[0], &r.cross[0]);
  int jy = ghost_index(iy, ny, bc[1], &r.cross[1]);
  int jz = ghost_index(iz, nz, bc[2], &r.cross[2]);
  r.idx = jx + (long)nx * (jy + (long)ny * jz);
  return r;
}

/* sign of component al of a vector field at a ghost position.
 * rule 0 (velocity-like, no slip): every component flips once per wall crossed.
 * rule 1 (field built from evenly mirrored scalars): component al flips iff axis al crossed. */
static double ghost_sign(const nbr_t *nb, int al, int rule) {
  if (rule == 0) return ((nb->cross[0] + nb->cross[1] + nb->cross[2]) & 1) ? -1.0 : 1.0;
  return nb->cross[al] ? -1.0 : 1.0;
}

/* ---------------------------------------------------------------- stencils ------------- */
/* Eq. 18: d_al Psi = (1/cs^2) sum_i w_i Psi(x + c_i) c_i,al ; scalars mirror evenly. */
static void grad_at(const double *psi, int ix, int iy, int iz, int nx, int ny, int nz,
                    const int bc[3], double g[3]) {
  g[0] = g[1] = g[2] = 0.0;
  FOR_SUM_Q(i) {
    nbr_t nb = neighbour(ix + Ci[i][0], iy + Ci[i][1], iz + Ci[i][2], nx, ny, nz, bc);
    for (int al = 0; al < 3; ++al) g[al] += Wi[i] * psi[nb.idx] * Ci[i][al];
  }
  for (int al = 0; al < 3; ++al) g[al] /= CS2;
}

/* Eq. 19 as repaired by R10: (2/cs^2) sum_{i != 0} w_i (Psi(x+c_i) - Psi(x)). */
static double lap_at(const double *psi, int ix, int iy, int iz, int nx, int ny, int nz,
                     const int bc[3]) {
  long x = ix + (long)nx * (iy + (long)ny * iz);
  double s = 0.0;
  FOR_SUM_Q(i) {
    if (Ci[i][0] == 0 && Ci[i][1] == 0 && Ci[i][2] == 0) continue;
    nbr_t nb = neighbour(ix + Ci[i][0], iy + Ci[i][1], iz + Ci[i][2], nx, ny, nz, bc);
    s += Wi[i] * (psi[nb.idx] - psi[x]);
  }
  return 2.0 * s / CS2;
}

/* Eq. 18 applied component-wise to a vector field (R17): div G = (1/cs^2) sum_i w_i c_i,al
 * G_al(x + c_i).  G3 is 3 planes of N. */
static double div_at(const double *G3, long N, int ix, int iy, int iz, int nx, int ny, int nz,
                     const int bc[3], int rule) {
  double s = 0.0;
  FOR_SUM_Q(i) {
    nbr_t nb = neighbour(ix + Ci[i][0], iy + Ci[i][1], iz + Ci[i][2], nx, ny, nz, bc);
    for (int al = 0; al < 3; ++al)
      s += Wi[i] * Ci[i][al] * ghost_sign(&nb, al, rule) * G3[al * N + nb.idx];
  }
  return s / CS2;
}

void tslb_ref_gradient(const double *psi, int nx, int ny, int nz, const int bc[3], double *out3) {
  build_tables();
  long N = (long)nx * ny * nz;
#pragma omp parallel for if ((long)nx * ny * nz >= OMP_MIN_NODES)
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < nx; ++ix) {
        long x = ix + (long)nx * (iy + (long)ny * iz);
        double g[3];
        grad_at(psi, ix, iy, iz, nx, ny, nz, bc, g);
        out3[x] = g[0]; out3[N + x] = g[1]; out3[2 * N + x] = g[2];
      }
}

void tslb_ref_laplacian(const double *psi, int nx, int ny, int nz, const int bc[3], double *out) {
  build_tables();
#pragma omp parallel for if ((long)nx * ny * nz >= OMP_MIN_NODES)
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < nx; ++ix)
        out[ix + (long)nx * (iy + (long)ny * iz)] = lap_at(psi, ix, iy, iz, nx, ny, nz, bc);
}

void tslb_ref_divergence(const double *G3, int nx, int ny, int nz, const int bc[3], int ghost_rule,
                         double *out) {
  build_tables();
  long N = (long)nx * ny * nz;
#pragma omp parallel for if ((long)nx * ny * nz >= OMP_MIN_NODES)
  for (int iz = 0; iz < nz; ++iz)
    for (int iy = 0; iy < ny; ++iy)
      for (int ix = 0; ix < nx; ++ix)
        out[ix + (long)nx * (iy + (long)ny * iz)] =
            div_at(G3, N, ix, iy, iz, nx, ny, nz, bc, ghost_rule);
}

/* ---------------------------------------------------------------- L2/L3 state ---------- */
struct tslb_ref {
  int nx, ny, nz; long N;
  tslb_ref_params p;
  double beta, kappa_mu, kappa_ac;    /* P:136 ; P:71 (R12: two different kappas) */
  double *pstar, *u, *A, *a, *phi;    /* time-n state: 1 + 3 + 6 + 3 + 1 planes   */
  double *f, *fpost;                  /* explicit populations, 27 planes each     */
  double *g, *nrm, *phin;             /* grad(phi^n), normal, phi^{n+1}           */
  int inited;
};

int tslb_ref_create(int nx, int ny, int nz, const tslb_ref_params *p, tslb_ref **out) {
  if (!p || !out || nx < 1 || ny < 1 || nz < 1) return -1;
  if (!(p->rho_l > 0 && p->rho_g > 0 && p->mu_l > 0 && p->mu_g > 0 && p->delta > 0 &&
        p->mobility > 0 && p->sigma >= 0)) return -1;
  const int n[3] = {nx, ny, nz};
  for (int d = 0; d < 3; ++d) {
    if (p->bc[d] != TSLB_REF_PERIODIC && p->bc[d] != TSLB_REF_WALL) return -1;
    if (n[d] < (p->bc[d] == TSLB_REF_PERIODIC ? 4 : 2)) return -1;
  }
  build_tables();
  tslb_ref *h = (tslb_ref *)calloc(1, sizeof(*h));
  if (!h) return -3;
  h->nx = nx; h->ny = ny; h->nz = nz; h->N = (long)nx * ny * nz; h->p = *p;
  h->beta = 12.0 * p->sigma / p->delta;
  h->kappa_mu = 3.0 * p->sigma * p->delta / 2.0;
  h->kappa_ac = 4.0 * p->mobility / p->delta;
  long N = h->N;
  h->pstar = calloc(N, sizeof(double));     h->u = calloc(3 * N, sizeof(double));
  h->A = calloc(6 * N, sizeof(double));     h->a = calloc(3 * N, sizeof(double));
  h->phi = calloc(N, sizeof(double));       h->phin = calloc(N, sizeof(double));
  h->f = calloc(Q * N, sizeof(double));     h->fpost = calloc(Q * N, sizeof(double));
  h->g = calloc(3 * N, sizeof(double));     h->nrm = calloc(3 * N, sizeof(double));
  if (!h->pstar || !h->u || !h->A || !h->a || !h->phi || !h->phin || !h->f || !h->fpost ||
      !h->g || !h->nrm) { tslb_ref_destroy(h); return -3; }
  *out = h;
  return 0;
}

void tslb_ref_destroy(tslb_ref *h) {
  if (!h) return;
  free(h->pstar); free(h->u); free(h->A); free(h->a); free(h->phi); free(h->phin);
  free(h->f); free(h->fpost); free(h->g); free(h->nrm); free(h);
}

/* O5 forces (Eq. 3, 15-19; R5, R7, R8, R18, R20) at one node.
 * phi   : the phase field whose gradient/Laplacian the forces see (phi^{n+1} in a step)
 * pstar : new p* ; Pineq : Pi - p* cs^2 delta - u^n u^n (R7), 3x3 ; returns a = F / rho. */
static void forces_at(const tslb_ref *h, const double *phi, int ix, int iy, int iz,
                      double pstar, double Pineq[3][3], double a[3]) {
  const tslb_ref_params *p = &h->p;
  long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
  double gphi[3];
  grad_at(phi, ix, iy, iz, h->nx, h->ny, h->nz, p->bc, gphi);
  double lap = lap_at(phi, ix, iy, iz, h->nx, h->ny, h->nz, p->bc);
  double ph = phi[x];
  /* chemical potential, P:136 with phi_l = 1, phi_g = 0, phi_0 = 1/2 */
  double mu_phi = 4.0 * h->beta * (ph - 1.0) * (ph - 0.0) * (ph - 0.5) - h->kappa_mu * lap;
  double rho = mix_rho(p, ph);
  double nu = mix_nu(p, ph);
  double om = tslb_ref_omega(p, ph);
  for (int al = 0; al < 3; ++al) {
    double grho_al = (p->rho_l - p->rho_g) * gphi[al];                 /* R18 */
    double Fs = mu_phi * gphi[al];                                     /* Eq. 3  */
    double Fp = -pstar * CS2 * grho_al;                                /* Eq. 16 */
    double Fnu = 0.0;                                                  /* Eq. 17, R7 */
    for (int be = 0; be < 3; ++be)
      Fnu += Pineq[al][be] * (p->rho_l - p->rho_g) * gphi[be];
    Fnu *= -(nu * om / CS2);
    double Fb = (rho - (p->body_heavy ? p->rho_g : p->rho_l)) * p->body_accel[al];  /* R20, R20b */
    a[al] = (Fs + Fp + Fnu + Fb) / rho;                                /* R5  */
  }
}

int tslb_ref_init(tslb_ref *h, const double *phi, const double *u) {
  if (!h || !phi || !u) return -1;
  long N = h->N;
  memcpy(h->phi, phi, N * sizeof(double));
  memcpy(h->u, u, 3 * N * sizeof(double));
  memset(h->pstar, 0, N * sizeof(double));          /* R9 */
  memset(h->A, 0, 6 * N * sizeof(double));          /* R9 */
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (int iz = 0; iz < h->nz; ++iz)
    for (int iy = 0; iy < h->ny; ++iy)
      for (int ix = 0; ix < h->nx; ++ix) {
        long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
        double zero[3][3] = {{0}}, a[3];
        forces_at(h, h->phi, ix, iy, iz, 0.0, zero, a);   /* F^p = F^nu = 0 at start */
        for (int al = 0; al < 3; ++al) h->a[al * N + x] = a[al];
      }
  h->inited = 1;
  return 0;
}

/* ---------------------------------------------------------------- one time step -------- */
/* O1 collide (Eq. 7-10, 14; R2, R3, R5): post-collision populations of every node
 * from its own time-n macroscopic fields.  omega is local, from phi^n (R14, R15). */
static void pass_collide(tslb_ref *h) {
  long N = h->N;
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (long x = 0; x < N; ++x) {
    double u[3] = {h->u[x], h->u[N + x], h->u[2 * N + x]};
    double a[3] = {h->a[x], h->a[N + x], h->a[2 * N + x]};
    double A[6];
    for (int k = 0; k < 6; ++k) A[k] = h->A[k * N + x];
    double feq[Q], fneq[Q], S[Q];
    tslb_ref_feq(h->pstar[x], u, feq);
    tslb_ref_fneq(u, A, fneq);
    tslb_ref_forcing(u, a, S);
    double om = tslb_ref_omega(&h->p, h->phi[x]);
    for (int i = 0; i < Q; ++i)
      h->fpost[i * N + x] = feq[i] + (1.0 - om) * fneq[i] + 0.5 * S[i];   /* R3 */
  }
}

/* O2 stream (Eq. 8): f_i(x, n+1) = fpost_i(x - c_i, n).  A direction whose source lies
 * beyond a wall is bounced back: f_i(x) = fpost_ibar(x) (R19); the wall test comes first. */
static void pass_stream(tslb_ref *h) {
  long N = h->N;
  const int *bc = h->p.bc;
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (int iz = 0; iz < h->nz; ++iz)
    for (int iy = 0; iy < h->ny; ++iy)
      for (int ix = 0; ix < h->nx; ++ix) {
        long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
        for (int i = 0; i < Q; ++i) {
          nbr_t nb = neighbour(ix - Ci[i][0], iy - Ci[i][1], iz - Ci[i][2],
                               h->nx, h->ny, h->nz, bc);
          if (nb.cross[0] || nb.cross[1] || nb.cross[2])
            h->f[i * N + x] = h->fpost[OPP[i] * N + x];
          else
            h->f[i * N + x] = h->fpost[i * N + nb.idx];
        }
      }
}

/* O3 Allen-Cahn, FTCS (Eq. 4, 20; R10, R13, R16, R17, R19), all at time n.
 * Pass 1: g = grad(phi), nrm = g / sqrt(g.g + eps^2).
 * Pass 2: phi^{n+1} = phi - div(phi u) + D lap(phi) - kappa_AC div(phi (1 - phi) nrm). */
static void pass_allen_cahn(tslb_ref *h) {
  long N = h->N;
  const int *bc = h->p.bc;
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (int iz = 0; iz < h->nz; ++iz)
    for (int iy = 0; iy < h->ny; ++iy)
      for (int ix = 0; ix < h->nx; ++ix) {
        long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
        double g[3];
        grad_at(h->phi, ix, iy, iz, h->nx, h->ny, h->nz, bc, g);
        double inv = 1.0 / sqrt(g[0] * g[0] + g[1] * g[1] + g[2] * g[2] + EPS_N * EPS_N);
        for (int al = 0; al < 3; ++al) {
          h->g[al * N + x] = g[al];
          h->nrm[al * N + x] = g[al] * inv;
        }
      }
  /* the two fluxes as whole arrays: adv = phi u (velocity-like ghosts), shp = phi(1-phi) nrm
   * (normal-odd ghosts).  g is reused as scratch for adv, nrm is overwritten by shp. */
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (long x = 0; x < N; ++x) {
    double ph = h->phi[x];
    for (int al = 0; al < 3; ++al) {
      h->g[al * N + x] = ph * h->u[al * N + x];
      h->nrm[al * N + x] = ph * (1.0 - ph) * h->nrm[al * N + x];
    }
  }
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (int iz = 0; iz < h->nz; ++iz)
    for (int iy = 0; iy < h->ny; ++iy)
      for (int ix = 0; ix < h->nx; ++ix) {
        long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
        double adv = div_at(h->g, N, ix, iy, iz, h->nx, h->ny, h->nz, bc, 0);
        double shp = div_at(h->nrm, N, ix, iy, iz, h->nx, h->ny, h->nz, bc, 1);
        double lap = lap_at(h->phi, ix, iy, iz, h->nx, h->ny, h->nz, bc);
        h->phin[x] = h->phi[x] - adv + h->p.mobility * lap - h->kappa_ac * shp;
      }
}

/* O4-O7: raw moments (Eq. 11-13), forces from phi^{n+1} (R8), velocity (Eq. 12,
 * R4), pre-regularisation (Eq. 13, computed literally with fbar_eq = feq - S/2). */
static void pass_moments(tslb_ref *h) {
  long N = h->N;
#pragma omp parallel for if (h->N >= OMP_MIN_NODES)
  for (int iz = 0; iz < h->nz; ++iz)
    for (int iy = 0; iy < h->ny; ++iy)
      for (int ix = 0; ix < h->nx; ++ix) {
        long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
        double fi[Q];
        for (int i = 0; i < Q; ++i) fi[i] = h->f[i * N + x];
        double pst = 0.0, m[3] = {0, 0, 0}, Pi[3][3] = {{0}};
        FOR_SUM_Q(i) {
          pst += fi[i];                                                     /* Eq. 11 */
          for (int al = 0; al < 3; ++al) {
            m[al] += fi[i] * Ci[i][al];
            for (int be = 0; be < 3; ++be) Pi[al][be] += fi[i] * Ci[i][al] * Ci[i][be];
          }
        }
        double uold[3] = {h->u[x], h->u[N + x], h->u[2 * N + x]};          /* R7 */
        double Pineq[3][3];
        for (int al = 0; al < 3; ++al)
          for (int be = 0; be < 3; ++be)
            Pineq[al][be] = Pi[al][be] - pst * CS2 * (al == be) - uold[al] * uold[be];
        double a[3], u[3];
        forces_at(h, h->phin, ix, iy, iz, pst, Pineq, a);
        for (int al = 0; al < 3; ++al) u[al] = m[al] + 0.5 * a[al];        /* Eq. 12, R4 */
        double feq[Q], S[Q], A[3][3] = {{0}};
        tslb_ref_feq(pst, u, feq);
        tslb_ref_forcing(u, a, S);
        FOR_SUM_Q(i)                                        /* Eq. 13 */
          for (int al = 0; al < 3; ++al)
            for (int be = 0; be < 3; ++be)
              A[al][be] += H2[i][al][be] * (fi[i] - (feq[i] - 0.5 * S[i]));
        h->pstar[x] = pst;
        for (int al = 0; al < 3; ++al) { h->u[al * N + x] = u[al]; h->a[al * N + x] = a[al]; }
        h->A[0 * N + x] = A[0][0]; h->A[1 * N + x] = A[1][1]; h->A[2 * N + x] = A[2][2];
        h->A[3 * N + x] = A[0][1]; h->A[4 * N + x] = A[0][2]; h->A[5 * N + x] = A[1][2];
      }
}

int tslb_ref_step(tslb_ref *h, int n) {
  if (!h || n < 0) return -1;
  if (!h->inited) return -4;
  for (int it = 0; it < n; ++it) {
    pass_collide(h);        /* TSLB fused streaming-collision, P:174 (collision half)  */
    pass_stream(h);         /*                                        (streaming half) */
    pass_allen_cahn(h);     /* interface tracking, P:178 (needs u^n, so before moments) */
    pass_moments(h);        /* moments + pre-regularisation of the next iteration */
    double *t = h->phi; h->phi = h->phin; h->phin = t;
  }
  return 0;
}

int tslb_ref_get(tslb_ref *h, double *rho, double *p, double *u, double *phi) {
  if (!h) return -1;
  if (!h->inited) return -4;
  long N = h->N;
  for (long x = 0; x < N; ++x) {
    double r = mix_rho(&h->p, h->phi[x]);                 /* P:142, R15 */
    if (rho) rho[x] = r;
    if (p) p[x] = h->pstar[x] * r * CS2;                  /* P:144, R21 */
  }
  if (u) memcpy(u, h->u, 3 * N * sizeof(double));
  if (phi) memcpy(phi, h->phi, N * sizeof(double));
  return 0;
}

int tslb_ref_get_state(tslb_ref *h, double *pstar, double *u, double *A, double *a, double *phi) {
  if (!h) return -1;
  long N = h->N;
  if (pstar) memcpy(pstar, h->pstar, N * sizeof(double));
  if (u) memcpy(u, h->u, 3 * N * sizeof(double));
  if (A) memcpy(A, h->A, 6 * N * sizeof(double));
  if (a) memcpy(a, h->a, 3 * N * sizeof(double));
  if (phi) memcpy(phi, h->phi, N * sizeof(double));
  return 0;
}

/* Restart aid for the segment-parity tests: replace the whole state by the
 * caller's arrays.  Copies only, no arithmetic; afterwards tslb_ref_step continues from it. */
int tslb_ref_set_state(tslb_ref *h, const double *pstar, const double *u, const double *A,
                       const double *a, const double *phi) {
  if (!h || !pstar || !u || !A || !a || !phi) return -1;
  long N = h->N;
  memcpy(h->pstar, pstar, N * sizeof(double));
  memcpy(h->u, u, 3 * N * sizeof(double));
  memcpy(h->A, A, 6 * N * sizeof(double));
  memcpy(h->a, a, 3 * N * sizeof(double));
  memcpy(h->phi, phi, N * sizeof(double));
  h->inited = 1;
  return 0;
}

/* Diagnostics of the current state: the box reductions behind what the
 * paper plots (centre-of-mass velocity of a bubble, Fig. 4) and what
 * BASELINE.json checks (conservation of sum(phi), Laplace's law).  Plain loops in node order,
 * long double accumulators.  out[16]:
 *    0 sum(phi)   1 sum(p*)   2 max |u|
 *    3..5  sum(phi ix), sum(phi iy), sum(phi iz)          (node indices as coordinates)
 *    6..8  sum(phi u)        9..11 sum(u)
 *   12 sum of p over nodes with phi > 0.99, 13 their count           (p = p* rho cs^2)
 *   14 sum of p over nodes with phi < 0.01, 15 their count */
int tslb_ref_diag(tslb_ref *h, double out[16]) {
  if (!h || !out) return -1;
  if (!h->inited) return -4;
  long N = h->N;
  long double s[16];
  for (int k = 0; k < 16; ++k) s[k] = 0.0L;
  double umax = 0.0;
  for (int iz = 0; iz < h->nz; ++iz)
    for (int iy = 0; iy < h->ny; ++iy)
      for (int ix = 0; ix < h->nx; ++ix) {
        long x = ix + (long)h->nx * (iy + (long)h->ny * iz);
        double ph = h->phi[x];
        double ux = h->u[x], uy = h->u[N + x], uz = h->u[2 * N + x];
        double p = h->pstar[x] * mix_rho(&h->p, ph) * CS2;
        double um = sqrt(ux * ux + uy * uy + uz * uz);
        if (um > umax) umax = um;
        s[0] += ph; s[1] += h->pstar[x];
        s[3] += ph * ix; s[4] += ph * iy; s[5] += ph * iz;
        s[6] += ph * ux; s[7] += ph * uy; s[8] += ph * uz;
        s[9] += ux; s[10] += uy; s[11] += uz;
        if (ph > 0.99) { s[12] += p; s[13] += 1.0L; }
        if (ph < 0.01) { s[14] += p; s[15] += 1.0L; }
      }
  for (int k = 0; k < 16; ++k) out[k] = (double)s[k];
  out[2] = umax;
  return 0;
}
