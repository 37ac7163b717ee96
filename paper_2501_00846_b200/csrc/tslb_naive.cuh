// tslb_naive.cuh -- one-thread-per-node global-memory kernels (TSLB_FLAG_NAIVE).
//
// Validation path: same arithmetic contract as the tiled kernels, no shared memory, every
// neighbour value fetched through L1/L2.  Also hosts the init and get kernels, which are not on
// the per-step path.
#pragma once
#include "tslb_device.cuh"

namespace tslb {

template <typename T>
__device__ __forceinline__ void node_coords(const DevParams<T>& P, long long idx, int& ix, int& iy,
                                            int& iz) {
  ix = int(idx % P.nx);
  long long r = idx / P.nx;
  iy = int(r % P.ny);
  iz = int(r / P.ny);
}

// Neighbour at offset (dx,dy,dz), |d| <= 2: linear index and per-axis wall-crossing flags.
template <typename T>
__device__ __forceinline__ long long nbr(const DevParams<T>& P, int ix, int iy, int iz, int dx,
                                         int dy, int dz, int& kx, int& ky, int& kz) {
  int jx = ghost_index(ix + dx, P.nx, P.bcx, kx);
  int jy = ghost_index(iy + dy, P.ny, P.bcy, ky);
  int jz = ghost_index(iz + dz, P.nz, P.bcz, kz);
  return jx + (long long)P.nx * (jy + (long long)P.ny * jz);
}

// Isotropic gradient (Eq. 18) and Laplacian (Eq. 19 as repaired by R10) of a scalar plane.
template <typename T>
__device__ __forceinline__ void grad_lap(const DevParams<T>& P, const T* __restrict__ phi, int ix,
                                         int iy, int iz, T& gx, T& gy, T& gz, T& lap) {
  T sx = 0, sy = 0, sz = 0, sw = 0;
  const T p0 = phi[ix + (long long)P.nx * (iy + (long long)P.ny * iz)];
#pragma unroll
  for (int i = 0; i < 27; ++i) {
    const int cx = i % 3 - 1, cy = (i / 3) % 3 - 1, cz = i / 9 - 1;
    int kx, ky, kz;
    T v = phi[nbr(P, ix, iy, iz, cx, cy, cz, kx, ky, kz)];
    T w = w1<T>(cx) * w1<T>(cy) * w1<T>(cz);
    sw = fma(w, v - p0, sw);                      // differences first: exactly 0 on constants
    if (cx) sx = fma(w * T(cx), v, sx);
    if (cy) sy = fma(w * T(cy), v, sy);
    if (cz) sz = fma(w * T(cz), v, sz);
  }
  gx = T(3) * sx; gy = T(3) * sy; gz = T(3) * sz;
  // (2/cs^2) sum_{i!=0} w_i (phi_i - phi_0) = 6 sum_i w_i (phi_i - phi_0)
  lap = T(6) * sw;
}

// ---- stage K4a: sharpening flux  Qs = phi (1 - phi) grad(phi)/sqrt(|grad(phi)|^2 + eps^2)  (R13)
template <typename T>
__global__ void __launch_bounds__(256) k_normal_naive(DevParams<T> P, long long nodes,
                                                      const T* __restrict__ S,
                                                      T* __restrict__ Q) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  int ix, iy, iz;
  node_coords(P, idx, ix, iy, iz);
  const T* phi = S + F_PHI * P.N;
  T gx, gy, gz, lap;
  grad_lap(P, phi, ix, iy, iz, gx, gy, gz, lap);
  T ph = phi[idx];
  T s = ph * (T(1) - ph) * rsqrt_t(gx * gx + gy * gy + gz * gz + T(1e-24));
  Q[idx] = s * gx;
  Q[P.N + idx] = s * gy;
  Q[2 * P.N + idx] = s * gz;
}

// ---- stage K4b: phi^{n+1} = phi - div(phi u) + D lap(phi) - kappa_AC div(Qs)   (Eq. 20, R16)
template <typename T>
__global__ void __launch_bounds__(256) k_allen_cahn_naive(DevParams<T> P, long long nodes,
                                                          const T* __restrict__ S,
                                                          const T* __restrict__ Q,
                                                          T* __restrict__ phin) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  int ix, iy, iz;
  node_coords(P, idx, ix, iy, iz);
  const T* phi = S + F_PHI * P.N;
  T div = 0, sw = 0;
  const T p0 = phi[idx];
#pragma unroll
  for (int i = 0; i < 27; ++i) {
    const int cx = i % 3 - 1, cy = (i / 3) % 3 - 1, cz = i / 9 - 1;
    int kx, ky, kz;
    long long j = nbr(P, ix, iy, iz, cx, cy, cz, kx, ky, kz);
    T w = w1<T>(cx) * w1<T>(cy) * w1<T>(cz);
    T pj = phi[j];
    sw = fma(w, pj - p0, sw);                     // differences first: exactly 0 on constants
    if (cx || cy || cz) {
      // velocity-like ghosts: every component flips once per wall crossed (R19)
      T s0 = ((kx + ky + kz) & 1) ? T(-1) : T(1);
      T fl = 0, ux, uy, uz;
      load_u(S, P.N, j, ux, uy, uz);
      if (cx) fl += T(cx) * (s0 * pj * ux + (kx ? -P.kappa_ac : P.kappa_ac) * Q[j]);
      if (cy) fl += T(cy) * (s0 * pj * uy + (ky ? -P.kappa_ac : P.kappa_ac) * Q[P.N + j]);
      if (cz) fl += T(cz) * (s0 * pj * uz + (kz ? -P.kappa_ac : P.kappa_ac) * Q[2 * P.N + j]);
      div = fma(w, fl, div);
    }
  }
  phin[idx] = p0 - T(3) * div + P.mob * T(6) * sw;
}

// ---- stage K3+K1+K2: pull-stream with per-source reconstruction, moments, forces, closing
template <typename T>
__device__ __forceinline__ Coef<T> load_coef(const T* __restrict__ S, long long N, long long j) {
  T m[13];
  load13(S, N, j, m);
  return coef_from13(m);
}

template <typename T, int I>
__device__ __forceinline__ void pull_dir(const DevParams<T>& P, const T* __restrict__ S, int ix,
                                         int iy, int iz, long long idx, const Coef<T>& self,
                                         Mom<T>& m) {
  constexpr int CX = I % 3 - 1, CY = (I / 3) % 3 - 1, CZ = I / 9 - 1;
  int kx, ky, kz;
  long long j = nbr(P, ix, iy, iz, -CX, -CY, -CZ, kx, ky, kz);
  T f;
  if (kx | ky | kz) {
    f = fpost_dir<T, -CX, -CY, -CZ>(self);        // halfway bounce-back (R19)
  } else if (CX == 0 && CY == 0 && CZ == 0) {
    f = fpost_dir<T, 0, 0, 0>(self);
  } else {
    Coef<T> c = load_coef(S, P.N, j);
    f = fpost_dir<T, CX, CY, CZ>(c);
  }
  accumulate<T, CX, CY, CZ>(m, f);
  (void)idx;
}

template <typename T, int I>
struct PullAll {
  static __device__ __forceinline__ void run(const DevParams<T>& P, const T* __restrict__ S, int ix,
                                             int iy, int iz, long long idx, const Coef<T>& self,
                                             Mom<T>& m) {
    pull_dir<T, I>(P, S, ix, iy, iz, idx, self, m);
    PullAll<T, I + 1>::run(P, S, ix, iy, iz, idx, self, m);
  }
};
template <typename T>
struct PullAll<T, 27> {
  static __device__ __forceinline__ void run(const DevParams<T>&, const T* __restrict__, int, int,
                                             int, long long, const Coef<T>&, Mom<T>&) {}
};

template <typename T>
__device__ __forceinline__ void store_node(T* __restrict__ D, long long N, long long idx,
                                           const NodeOut<T>& o) {
  store_out(D, N, idx, o);
}

template <typename T>
__global__ void __launch_bounds__(128) k_stream_collide_naive(DevParams<T> P, long long nodes,
                                                              const T* __restrict__ S,
                                                              T* __restrict__ D) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  int ix, iy, iz;
  node_coords(P, idx, ix, iy, iz);
  Coef<T> self = load_coef(S, P.N, idx);
  Mom<T> m = {};
  PullAll<T, 0>::run(P, S, ix, iy, iz, idx, self, m);
  const T* phin = D + F_PHI * P.N;              // phi^{n+1}, written by the Allen-Cahn stage
  T gx, gy, gz, lap;
  grad_lap(P, phin, ix, iy, iz, gx, gy, gz, lap);
  T uox, uoy, uoz;
  load_u(S, P.N, idx, uox, uoy, uoz);
  NodeOut<T> o = close_node(P, m, phin[idx], gx, gy, gz, lap, uox, uoy, uoz);
  store_node(D, P.N, idx, o);
}

// ---- tslb_init: p* = 0, Ahat = 0 (R9), a = (F^s + F^b)/rho from phi (R19 ghosts)
template <typename T>
__global__ void __launch_bounds__(256) k_init(DevParams<T> P, long long nodes,
                                              const T* __restrict__ phi0,
                                              const T* __restrict__ u0, long long us,
                                              T* __restrict__ D, T* __restrict__ Q) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  int ix, iy, iz;
  node_coords(P, idx, ix, iy, iz);
  T gx, gy, gz, lap;
  grad_lap(P, phi0, ix, iy, iz, gx, gy, gz, lap);
  T ph = phi0[idx];
  Mix<T> mx = mixture(P, ph);
  T mu_phi = P.beta4 * ph * (ph - T(1)) * (ph - T(0.5)) - P.kappa_mu * lap;
  T db = mx.rho - P.rho_b;
  NodeOut<T> o = {};
  o.ux = u0[idx]; o.uy = u0[us + idx]; o.uz = u0[2 * us + idx];
  o.ax = fma(db, P.gx, mu_phi * gx) * mx.inv_rho;
  o.ay = fma(db, P.gy, mu_phi * gy) * mx.inv_rho;
  o.az = fma(db, P.gz, mu_phi * gz) * mx.inv_rho;
  store_node(D, P.N, idx, o);
  D[F_PHI * P.N + idx] = ph;
  T q[3];                                    // flux of Eq. 20 for the first interface update
  flux_q(P, ph, gx, gy, gz, o.ux, o.uy, o.uz, q);
  store_q(Q, P.N, idx, q);
}

// ---- tslb_get: rho, p = p* rho cs^2, u, phi
template <typename T>
__global__ void __launch_bounds__(256) k_get(DevParams<T> P, long long nodes,
                                             const T* __restrict__ S, T* __restrict__ rho,
                                             T* __restrict__ p, T* __restrict__ u, long long us,
                                             T* __restrict__ phi) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  T ph = S[F_PHI * P.N + idx];
  T r = fma(clamp01(ph), P.drho, P.rho_g);
  if (rho) rho[idx] = r;
  if (p) p[idx] = S[field_off<T>(P.N, idx, F_P)] * r * T(1.0 / 3.0);
  if (u) {
    T ux, uy, uz;
    load_u(S, P.N, idx, ux, uy, uz);
    u[idx] = ux; u[us + idx] = uy; u[2 * us + idx] = uz;
  }
  if (phi) phi[idx] = ph;
}

}  // namespace tslb

namespace tslb {
// ---- tslb_set_state: the inverse of tslb_get_state (restart / resume).  The flux Q of Eq. 20 that
// the periodic interface kernel expects is rebuilt from phi and u as in tslb_init.
template <typename T>
__global__ void __launch_bounds__(256) k_set_state(DevParams<T> P, long long nodes,
                                                   const T* __restrict__ pstar,
                                                   const T* __restrict__ u, const T* __restrict__ A,
                                                   const T* __restrict__ a,
                                                   const T* __restrict__ phi, T* __restrict__ D,
                                                   T* __restrict__ Q) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  int ix, iy, iz;
  node_coords(P, idx, ix, iy, iz);
  T m[13];
  m[F_P] = pstar[idx];
  for (int k = 0; k < 3; ++k) m[F_UX + k] = u[k * nodes + idx];
  for (int k = 0; k < 6; ++k) m[F_AXX + k] = A[k * nodes + idx];
  for (int k = 0; k < 3; ++k) m[F_AX + k] = a[k * nodes + idx];
  store13(D, P.N, idx, m);
  const T ph = phi[idx];
  D[F_PHI * P.N + idx] = ph;
  T gx, gy, gz, lap;
  grad_lap(P, phi, ix, iy, iz, gx, gy, gz, lap);
  T q[3];
  flux_q(P, ph, gx, gy, gz, m[F_UX], m[F_UY], m[F_UZ], q);
  store_q(Q, P.N, idx, q);
}

// ---- tslb_get_state: de-interleave the stored fields into plain planes (NULL = skip)
template <typename T>
__global__ void __launch_bounds__(256) k_get_state(DevParams<T> P, long long nodes,
                                                   const T* __restrict__ S, T* __restrict__ pstar,
                                                   T* __restrict__ u, T* __restrict__ A,
                                                   T* __restrict__ a, T* __restrict__ phi) {
  long long idx = blockIdx.x * (long long)blockDim.x + threadIdx.x;
  if (idx >= nodes) return;
  T m[13];
  load13(S, P.N, idx, m);
  if (pstar) pstar[idx] = m[F_P];
  if (u) for (int k = 0; k < 3; ++k) u[k * nodes + idx] = m[F_UX + k];
  if (A) for (int k = 0; k < 6; ++k) A[k * nodes + idx] = m[F_AXX + k];
  if (a) for (int k = 0; k < 3; ++k) a[k * nodes + idx] = m[F_AX + k];
  if (phi) phi[idx] = S[F_PHI * P.N + idx];
}
}  // namespace tslb

namespace tslb {
// ---- halo planes of the z-slab decomposition -----------
// A slab keeps HALO_DEPTH ghost planes at each end of its z range.  Every internal array (the
// 128-bit field-vector planes, az, phi of the current state buffer, the three flux planes) is
// contiguous over consecutive z planes, so the planes of one face are a handful of contiguous
// segments: one kernel copies them to / from a packed buffer, element by element.
constexpr int HALO_DEPTH = 2;      // K1 reaches one plane, K2 one more: one exchange per step
constexpr int HALO_MAXSEG = 12;
struct HaloSegs {
  int n;
  long long arr_off[HALO_MAXSEG];   // element offset of the segment inside the state buffer (or
                                    // inside the flux scratch when in_q is set)
  long long len[HALO_MAXSEG];       // elements
  int in_q[HALO_MAXSEG];
};
template <typename T, bool PACK>
__global__ void __launch_bounds__(256) k_halo_copy(HaloSegs sg, T* __restrict__ state,
                                                   T* __restrict__ q, T* __restrict__ buf) {
  long long total = 0;
  for (int i = 0; i < sg.n; ++i) total += sg.len[i];
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
       e += (long long)gridDim.x * blockDim.x) {
    long long r = e;
    int i = 0;
    while (r >= sg.len[i]) { r -= sg.len[i]; ++i; }
    T* a = (sg.in_q[i] ? q : state) + sg.arr_off[i] + r;
    if (PACK) buf[e] = *a; else *a = buf[e];
  }
}
}  // namespace tslb
