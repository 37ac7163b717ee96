/* tslb.h -- C ABI of the B200-native TSLB + conservative Allen-Cahn hot path.
 *
 * Method: "Thread-safe multiphase lattice Boltzmann model for droplet and bubble dynamics at
 * high density and viscosity contrasts", arXiv 2501.00846.  Citations "P:<line>" refer to the
 * paper text and "Rk" to the readings listed in DESIGN.md.
 *
 * The library stores hydrodynamic moments, not populations: per lattice node the 14
 * scalars p* (Eq. 11), u (Eq. 12), a2_neq (Eq. 13, 6 components), a = F/rho (Eq. 14-17, R5) and
 * phi (Eq. 20), as structure-of-arrays planes, double buffered, x fastest:
 *     idx = ix + nx * (iy + ny * iz).
 * One tslb_step performs, for every node, the paper's four stages: interface
 * tracking (Eq. 20), fused streaming-collision with recursive Hermite reconstruction
 * (Eq. 7-10, 14), moments and forces (Eq. 11, 12, 3, 16, 17), pre-regularisation (Eq. 13).
 *
 * Everything runs in hand-written CUDA kernels for sm_100a; there is no CPU fallback.  All
 * functions are thread-compatible (one handle per thread at a time) and enqueue work on the
 * handle's stream without synchronising; the caller synchronises the stream.
 *
 * Errors: 0 on success, negative otherwise; tslb_last_error() returns a thread-local text.
 *   TSLB_EINVAL   (-1) bad argument (non-positive size, n < 0, NULL, non-positive rho/mu/
 *                      delta/mobility, sigma < 0, unknown enum, axis shorter than the stencil)
 *   TSLB_EWORKSPACE(-2) workspace NULL, too small or not 256-byte aligned
 *   TSLB_ECUDA    (-3) a CUDA call failed (text holds cudaGetErrorString)
 *   TSLB_ESTATE   (-4) tslb_step / tslb_get before tslb_init (or tslb_set_state)
 */
#ifndef TSLB_H
#define TSLB_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct tslb_handle tslb_handle; /* opaque; host memory owned by the library */

enum { TSLB_BC_PERIODIC = 0, TSLB_BC_WALL = 1 }; /* per axis, both ends */
enum { TSLB_F32 = 0, TSLB_F64 = 1 };
enum { TSLB_OK = 0, TSLB_EINVAL = -1, TSLB_EWORKSPACE = -2, TSLB_ECUDA = -3, TSLB_ESTATE = -4 };

/* flags (bit field): validation selectors.  0 = the library chooses (production).  Every flag
 * forces another kernel of the product that computes the SAME step (same arithmetic contract,
 * same tolerances); there are no tuning or timing variants behind this field and any other bit
 * makes tslb_create fail with TSLB_EINVAL. */
enum {
  TSLB_FLAG_NAIVE = 1,      /* one-thread-per-node global-memory kernels (validation path)        */
  TSLB_FLAG_GENERIC = 2,    /* the wall-capable tiled pair (explicit populations, normals
                               recomputed) instead of the lean pair, on any box                  */
  TSLB_FLAG_K2_CPASYNC = 4, /* lean stream-collide kernel with cp.async staging, even where the
                               TMA-staged one would be chosen                                    */
  TSLB_FLAG_K2_TMA = 8,     /* ... with TMA tensor staging wherever it is usable (nx % 32 == 0,
                               nx >= 64, ny > 8, periodic x and y), even where cp.async would be
                               chosen                                                            */
  TSLB_FLAG_K1_FLUX = 16,   /* on an all-periodic box, the one-node-per-thread flux-form interface
                               kernel instead of the row kernel                                  */
  TSLB_FLAG_ALL = 31
};

/* flags, second group: NOT a kernel selector but part of the problem statement.  The paper's
 * body force acts "exclusively on the dispersed phase": the gas of a rising bubble (the
 * default, force density (rho - rho_l) g, zero in the liquid) or the liquid of droplets falling
 * through gas (force density (rho - rho_g) g, zero in the gas; reading R20b).
 * Every kernel of the library honours it. */
enum {
  TSLB_FLAG_BODY_HEAVY = 32 /* body force (rho - rho_g) g : heavy (liquid) phase only             */
};

typedef struct tslb_params {
  double rho_l, rho_g;   /* > 0 ; rho = rho_g + phi (rho_l - rho_g)      */
  double mu_l, mu_g;     /* > 0 ; dynamic viscosities, mixed linearly in phi (R14) */
  double sigma;          /* >= 0 ; beta = 12 sigma/delta, kappa_mu = 3 sigma delta/2 P:136     */
  double delta;          /* > 0 ; interface width in lattice units */
  double mobility;       /* > 0 ; D of Eq. 4 ; kappa_AC = 4 D/delta    */
  double body_accel[3];  /* g ; force density (rho - rho_l) g : light phase only    P:256, R20 ;
                            (rho - rho_g) g with TSLB_FLAG_BODY_HEAVY               P:358, R20b */
  int bc[3];             /* TSLB_BC_* for x, y, z                                              */
  int precision;         /* TSLB_F32 / TSLB_F64 : type of every field pointer and of all math  */
  int flags;             /* TSLB_FLAG_* ; 0 (or TSLB_FLAG_BODY_HEAVY alone) = production path   */
} tslb_params;

/* Bytes of device workspace tslb_create needs for this size and precision (0 on bad input). */
size_t tslb_workspace_bytes(int nx, int ny, int nz, const tslb_params *params);

/* Create a solver on the CALLER-OWNED device buffer `workspace` (>= tslb_workspace_bytes,
 * 256-byte aligned, kept alive until tslb_destroy).  The library carves out of it two state
 * buffers of 14 SoA planes, 3 more planes for the Allen-Cahn flux Q that the two kernels of a step
 * hand to each other (31 planes while the step is a split pair), and the partial-sum
 * rows of tslb_diag; it allocates nothing else on the device.  `stream` is a cudaStream_t (NULL =
 * legacy default stream).  Minimum size: 4 nodes on a periodic axis, 2 on a wall axis.  No
 * kernel is launched. */
int tslb_create(int nx, int ny, int nz, const tslb_params *params, void *workspace, void *stream,
                tslb_handle **out);

/* Set the initial state from DEVICE arrays in the handle's precision: phi[N], u[3][N] (three
 * consecutive planes ux, uy, uz).  p* = 0 and a2_neq = 0 (R9); a = (F^s + F^b)/rho from phi with
 * the same ghost rules as the step (R19).  The arrays are not retained.  May be called again. */
int tslb_init(tslb_handle *h, const void *phi, const void *u);

/* Advance n >= 0 time steps (n = 0 is a no-op).  No host synchronisation inside. */
int tslb_step(tslb_handle *h, int n);

/* Write rho = rho_g + clamp(phi)(rho_l - rho_g) (R15), p = p* rho cs^2, the
 * velocity u of Eq. 12 ([3][N]) and phi into DEVICE arrays of the handle's precision.  A NULL
 * pointer skips that field. */
int tslb_get(tslb_handle *h, void *rho, void *p, void *u, void *phi);

/* Full internal state (debug / parity of the unexposed fields): p*[N], u[3][N], a2_neq[6][N] in
 * the order xx,yy,zz,xy,xz,yz, a[3][N], phi[N]; DEVICE arrays, NULL skips. */
int tslb_get_state(tslb_handle *h, void *pstar, void *u, void *A, void *a, void *phi);

/* Restart / resume: the inverse of tslb_get_state.  DEVICE arrays in the handle's precision,
 * same shapes and order (A holds what tslb_get_state returns: (1 - omega(phi)) a2_neq); all
 * five are required.  Replaces the whole state, so it may be called instead of tslb_init; the
 * arrays are not retained.  get_state -> set_state -> step continues a run to rounding (the
 * flux of Eq. 20 handed between the two kernels of a step is rebuilt from phi and u with another
 * summation order), not bit for bit. */
int tslb_set_state(tslb_handle *h, const void *pstar, const void *u, const void *A, const void *a,
                   const void *phi);

/* z-slab decomposition support (the paper's own multi-GPU runs).
 * A slab of a lattice that is periodic along z is a handle created on nz_local + 4 planes with a
 * periodic z axis: two ghost planes at each end.  One step needs neighbour data one plane deep
 * for the interface update (Eq. 20) and one more for the stream-collide kernel (Eq. 8), so ONE
 * exchange of two planes per face and step keeps planes [2, nz-2) exact; what the step writes into
 * the ghost planes is overwritten by the next exchange.
 *   tslb_halo_pack(h, face, buf):   copy the owned planes next to the face, [2, 4) for face 0
 *                                   (low z) or [nz-4, nz-2) for face 1, of every internal array
 *                                   (13 moments, phi, the flux of Eq. 20: 17 scalars per node)
 *                                   into the DEVICE buffer buf of tslb_halo_bytes(h) bytes;
 *   tslb_halo_unpack(h, face, buf): write such a buffer into the ghost planes [0, 2) (face 0)
 *                                   or [nz-2, nz) (face 1).
 * The low neighbour's face-1 buffer goes into this slab's face 0 and vice versa.  The format of
 * the buffer is private to the library (same size, precision and flags on both sides).  One
 * launch each on the handle's stream, no synchronisation; after tslb_init and after every
 * tslb_step(1).  Needs >= 6 planes along z, flags NAIVE / GENERIC unset (the flux planes belong
 * to the lean kernel pair), ghost planes at that end (next paragraph) and, in a box with walls on
 * any axis, nx a multiple of the 128-bit vector width (2 in fp64, 4 in fp32: other rows take an
 * interface kernel of radius 2, for which two ghost planes are too few).
 *
 * Boxes with walls on z (the paper's rising bubble, and its droplet train, a
 * 500 x 500 x 3000 box) are cut the same way: every slab is created with bc z = TSLB_BC_WALL,
 * the first and the last one carry ghost planes at their inner end only, and
 *   tslb_slab_set_ends(h, ghost_low, ghost_high)
 * says which ends have them (default: both on a periodic z axis, none on a wall axis; an end
 * without ghosts must be a wall).  An end with ghosts never applies the wall rules: what the
 * kernels compute in the ghost planes is overwritten by the exchange and the owned planes do not
 * read beyond them.  Walls on x or y need nothing special (every slab has them).
 * paper_2501_00846_b200/slab.py drives it over torch.distributed. */
size_t tslb_halo_bytes(const tslb_handle *h);
int tslb_halo_pack(tslb_handle *h, int face, void *buf);
int tslb_halo_unpack(tslb_handle *h, int face, const void *buf);
int tslb_slab_set_ends(tslb_handle *h, int ghost_low, int ghost_high);

/* The same step of a slab in two stages, so that the exchange overlaps the interior sweep
 * (the paper's decompositions and their communication cost: P:194-238):
 *   tslb_slab_step_faces(h):    interface update (Eq. 20) on planes [1, nz-1), stream-collide on
 *                               the owned planes next to the faces, [2, 4) and [nz-4, nz-2); the
 *                               state buffers swap, so tslb_halo_pack now packs the NEW faces;
 *   tslb_slab_step_interior(h): stream-collide on the interior [4, nz-4): the step is complete.
 * (An end without ghosts has no face piece: its planes, from the wall on, belong to the interior.)
 * Between the two only tslb_halo_pack / tslb_halo_unpack may be called (anything else returns
 * TSLB_ESTATE): pack, start the transfer, run the interior, wait, unpack.  The ghost planes are
 * never computed (the exchange fills them), so the owned planes come out bit-identical to
 * tslb_step(1) + exchange and to the undivided lattice.  Requirements of tslb_halo_pack, and nx
 * a multiple of the 128-bit vector width (2 in fp64, 4 in fp32).  Three or four launches on the
 * handle's stream, no synchronisation. */
int tslb_slab_step_faces(tslb_handle *h);
int tslb_slab_step_interior(tslb_handle *h);

/* On-device diagnostics: box reductions of the current state, the
 * quantities behind the paper's validation plots (centre-of-mass velocity of a rising bubble,
 * Fig. 4) and BASELINE.json's checks (sum(phi) conserved; Laplace's law
 * Delta p R/(2 sigma) on configs[1]), so that no whole field has to be read back.
 * out = TSLB_NDIAG doubles (fp64 accumulation in both precisions), indexed by TSLB_D_*:
 *   SUM_PHI, SUM_PSTAR, MAX_U (max |u|; NaN if any velocity is NaN), SUM_PHI_X/Y/Z (sum phi * node index: centre of mass of
 *   the liquid = SUM_PHI_X / SUM_PHI on a non-periodic axis), SUM_PHI_UX/UY/UZ (its momentum per
 *   unit liquid density), SUM_UX/UY/UZ (so the light phase's is sum(u) - sum(phi u)),
 *   SUM_P_IN / N_IN: sum and count of p = p* rho cs^2 over nodes with phi > 0.99,
 *   SUM_P_OUT / N_OUT: the same over phi < 0.01 (Delta p = SUM_P_IN/N_IN - SUM_P_OUT/N_OUT).
 * Two launches on the handle's stream, deterministic (fixed reduction order, no atomics); the
 * partial sums live in the caller's workspace.  tslb_diag writes a DEVICE array and does not
 * synchronise; tslb_diag_host writes a HOST array and synchronises the stream. */
enum { TSLB_D_SUM_PHI = 0, TSLB_D_SUM_PSTAR = 1, TSLB_D_MAX_U = 2,
       TSLB_D_SUM_PHI_X = 3, TSLB_D_SUM_PHI_Y = 4, TSLB_D_SUM_PHI_Z = 5,
       TSLB_D_SUM_PHI_UX = 6, TSLB_D_SUM_PHI_UY = 7, TSLB_D_SUM_PHI_UZ = 8,
       TSLB_D_SUM_UX = 9, TSLB_D_SUM_UY = 10, TSLB_D_SUM_UZ = 11,
       TSLB_D_SUM_P_IN = 12, TSLB_D_N_IN = 13, TSLB_D_SUM_P_OUT = 14, TSLB_D_N_OUT = 15,
       TSLB_NDIAG = 16 };
int tslb_diag(tslb_handle *h, double *out);
int tslb_diag_host(tslb_handle *h, double *out);

/* Allocation-free variant of tslb_diag, for callers that cannot provide or allocate scratch
 * (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc): same kernels, same
 * result bit for bit, but the partial sums live in a static device array inside the library
 * (512 KB, held by every GPU that loads the library until the process exits) instead of the
 * workspace.  The call allocates nothing and synchronises nothing; `out` is a DEVICE array of
 * TSLB_NDIAG doubles; the handle's device must be the current device.
 * Limit: lattices of at most TSLB_DIAG_STATIC_MAX_NODES nodes (256^3 and 320^3 fit, 384^3 does
 * not); larger ones return TSLB_EINVAL with a text that says so (use tslb_diag).
 * The array is shared by every handle and every call in the process and keeps the last call's
 * contents (no call depends on them: every row read is overwritten first): calls whose kernels
 * may overlap on the GPU (different streams, no ordering between them) RACE on it; calls on one
 * stream, or ordered by events, are safe. */
enum { TSLB_DIAG_STATIC_MAX_NODES = 4096 * 8192 };
int tslb_diag_static(tslb_handle *h, double *out);

/* Host-buffer convenience for end-to-end use: same as tslb_init / tslb_get but the field
 * pointers are HOST arrays (pinned memory makes the copies asynchronous); the library stages
 * them through the spare state buffer, so no extra device memory is needed.  tslb_get_host
 * synchronises the stream before returning. */
int tslb_init_host(tslb_handle *h, const void *phi, const void *u);
int tslb_get_host(tslb_handle *h, void *rho, void *p, void *u, void *phi);

/* Same as tslb_step, but brackets every kernel with CUDA events on the handle's stream,
 * synchronises, and ADDS the elapsed milliseconds per kernel kind into kernel_ms[TSLB_NKERNELS]
 * (caller-zeroed HOST array).  Used by bench.py for the per-kernel roofline. */
enum { TSLB_K_NORMAL = 0,          /* naive path only: sharpening-flux kernel            */
       TSLB_K_ALLEN_CAHN = 1,      /* interface tracking, Eq. 20                          */
       TSLB_K_STREAM_COLLIDE = 2,  /* fused stream-collide-moments-forces, Eq. 7-17       */
       TSLB_NKERNELS = 4 };
int tslb_step_timed(tslb_handle *h, int n, float *kernel_ms);

/* ALU side of the roofline: measured throughput, in TFLOP/s (2 flops per FMA), of
 * dependent-chain-free fused multiply-adds in the given precision on the current device, timed
 * with CUDA events on `stream` (synchronises).  A micro-benchmark for bench.py's
 * roofline.alu_frac, not part of the path; needs no handle and allocates nothing. */
int tslb_fma_peak(int precision, void *stream, double *tflops);

/* Number of kernel launches the handle has enqueued so far (for bench.py's gpu_launches). */
long long tslb_launch_count(const tslb_handle *h);

void tslb_destroy(tslb_handle *h); /* frees host memory only; NULL is allowed */

const char *tslb_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* TSLB_H */
