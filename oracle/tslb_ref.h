/* tslb_ref.h -- CPU ORACLE for the thread-safe lattice Boltzmann (TSLB) + conservative
 * Allen-Cahn step of arXiv 2501.00846.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or helper with the CUDA path under paper_2501_00846_b200/csrc and include/.
 *
 * Plain C, fp64, host pointers only.  Explicit populations, whole-array passes in the paper's
 * order, brute-force tensor contractions over alpha,beta,gamma and i = 0..26
 * straight from the printed formulas (Eq. 7-20) as repaired by the readings R1-R24 listed in
 * DESIGN.md.  OpenMP "parallel for" over nodes is the only concession to speed.
 *
 * Readings that DEPART from the printed text (each also in DESIGN.md):
 *   R2  Eq. 10 is evaluated with the weight w_i and the full Hermite tensor c c - cs^2 delta.
 *   R3  f_post = f_eq + (1-omega) f_neq + S/2 (the redefined equilibrium of PAPER.md:122-126).
 *   R4  Eq. 12: u = sum_i f_i c_i + a/2 (the printed sum_i S_i is identically zero).
 *   R5  S_i and Eq. 12 use the acceleration a = F/rho.
 *   R10 Eq. 19 is the isotropic Laplacian (2/cs^2) sum_{i!=0} w_i (Psi(x+c_i) - Psi(x)).
 *   R16 Eq. 20 advects in divergence form div(phi u) (the printed u.grad(phi) does not conserve).
 * Parity unpinned (nothing in the paper or the physics selects among O(dt)-equivalent
 * variants; the reading is the contract): R7 (velocity level inside F^nu), R8 (forces see
 * phi^{n+1}), R9 (p* = 0, A = 0 start), R13 (epsilon in the normal), R14 (linear mu(phi)),
 * R15 (clamp of phi inside the mixture rules).
 */
#ifndef TSLB_REF_H
#define TSLB_REF_H

#ifdef __cplusplus
extern "C" {
#endif

enum { TSLB_REF_PERIODIC = 0, TSLB_REF_WALL = 1 };

typedef struct tslb_ref_params {
  double rho_l, rho_g;   /* rho = rho_g + phi (rho_l - rho_g) */
  double mu_l, mu_g;     /* dynamic viscosities, mixed linearly in phi   R14          */
  double sigma;          /* beta = 12 sigma/delta, kappa_mu = 3 sigma delta/2 */
  double delta;          /* interface width  */
  double mobility;       /* D of Eq. 4; kappa_AC = 4 D/delta */
  double body_accel[3];  /* g ; force density (rho - rho_l) g            PAPER.md:256, R20 */
  int bc[3];             /* TSLB_REF_PERIODIC / TSLB_REF_WALL per axis */
  int body_heavy;        /* 0: force density (rho - rho_l) g ; 1: (rho - rho_g) g, the
                            dispersed phase being the liquid            PAPER.md:358, R20b */
} tslb_ref_params;

typedef struct tslb_ref tslb_ref;

/* Whole-lattice driver.  All arrays are host fp64, x fastest: idx = ix + nx (iy + ny iz);
 * vectors are 3 consecutive planes (x, y, z); the tensor A is 6 planes xx,yy,zz,xy,xz,yz. */
int  tslb_ref_create (int nx, int ny, int nz, const tslb_ref_params *p, tslb_ref **out);
int  tslb_ref_init   (tslb_ref *h, const double *phi, const double *u);
int  tslb_ref_step   (tslb_ref *h, int n);
int  tslb_ref_get    (tslb_ref *h, double *rho, double *p, double *u, double *phi); /* NULL = skip */
int  tslb_ref_get_state(tslb_ref *h, double *pstar, double *u, double *A, double *a, double *phi);
void tslb_ref_destroy(tslb_ref *h);
/* Restart aid for segment parity (copies only): replace the whole state; A is a2_neq itself. */
int  tslb_ref_set_state(tslb_ref *h, const double *pstar, const double *u, const double *A,
                        const double *a, const double *phi);
/* Box reductions of the current state (Fig. 4, 292):
 * out[16] = sum(phi), sum(p*), max|u|, sum(phi ix,iy,iz), sum(phi u), sum(u),
 * sum and count of p = p* rho cs^2 over phi > 0.99, the same over phi < 0.01. */
int  tslb_ref_diag(tslb_ref *h, double out[16]);

/* Single-node pieces, the same functions the passes call, exported so the pins can reach them. */
void tslb_ref_lattice(int c[27][3], double w[27], int opp[27]);          /* R1            */
void tslb_ref_feq    (double pstar, const double u[3], double out[27]);   /* Eq. 9         */
void tslb_ref_fneq   (const double u[3], const double A[6], double out[27]); /* Eq. 10, R2 */
void tslb_ref_forcing(const double u[3], const double a[3], double out[27]); /* Eq. 14, R5 */
double tslb_ref_omega(const tslb_ref_params *p, double phi);              /* R14, R15      */

/* Stencils on whole arrays (Eq. 18, repaired Eq. 19), with the ghost rules of R19.
 * ghost_rule for vector fields: 0 = every component changes sign across a wall (velocity-like),
 * 1 = only the wall-normal component changes sign (a field built from mirrored scalars). */
void tslb_ref_gradient  (const double *psi, int nx, int ny, int nz, const int bc[3], double *out3);
void tslb_ref_laplacian (const double *psi, int nx, int ny, int nz, const int bc[3], double *out);
void tslb_ref_divergence(const double *G3, int nx, int ny, int nz, const int bc[3], int ghost_rule,
                         double *out);

#ifdef __cplusplus
}
#endif
#endif
