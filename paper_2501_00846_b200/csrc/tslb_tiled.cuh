// tslb_tiled.cuh -- production kernels: xy tile + z marching.
//
// A thread block owns a TX x TY tile of (x,y) columns and marches through a chunk of z planes.
// Main threads (one per column) produce outputs; extra "halo" threads own the ring of H columns
// around the tile and only feed shared memory.  Every node's 27 post-collision populations are
// reconstructed ONCE, by the thread that owns the node (Eq. 7-10, 14), and reach their 27
// destinations through shared memory (the 8 in-plane neighbours) and a register pipeline along
// z (the planes above and below).  Populations never touch global memory.
#pragma once
#include "tslb_device.cuh"

namespace tslb {

// ---- thread <-> tile-local column (lx, ly), lx in [-H, TX+H), ly in [-H, TY+H)
template <int TX, int TY, int H>
struct TileMap {
  static constexpr int W = TX + 2 * H;            // shared-memory row length
  static constexpr int HT = TY + 2 * H;
  static constexpr int NMAIN = TX * TY;
  static constexpr int NROWH = 2 * H * W;         // halo rows, full width
  static constexpr int NCOLH = 2 * H * TY;        // halo columns beside the main rows
  static constexpr int NHALO = NROWH + NCOLH;
  static constexpr int NTHREADS = NMAIN + ((NHALO + 31) / 32) * 32;
  static constexpr int CELLS = W * HT;

  __device__ static __forceinline__ bool coords(int tid, int& lx, int& ly) {
    if (tid < NMAIN) { lx = tid % TX; ly = tid / TX; return true; }
    int h = tid - NMAIN;
    if (h < NROWH) {
      int r = h / W;
      lx = h % W - H;
      ly = (r < H) ? r - H : TY + (r - H);
      return true;
    }
    h -= NROWH;
    if (h < NCOLH) {
      int c = h % (2 * H);
      ly = h / (2 * H);
      lx = (c < H) ? c - H : TX + (c - H);
      return true;
    }
    lx = 0; ly = 0;
    return false;
  }
  __device__ static __forceinline__ int cell(int lx, int ly) { return (ly + H) * W + (lx + H); }
};

// shared-memory slot of the population with in-plane direction (CX,CY) != (0,0) and CZ
__host__ __device__ constexpr int pop_slot(int cx, int cy, int cz) {
  int q = (cy + 1) * 3 + (cx + 1);
  q = q > 4 ? q - 1 : q;
  return q * 3 + (cz + 1);
}

// ------------------------------------------------------------------------------------------
// Kernel K2: fused stream-collide-moments-forces (Eq. 7-17).  H = 1.
// ------------------------------------------------------------------------------------------
template <typename T, int TX, int TY>
struct K2Smem {
  using M = TileMap<TX, TY, 1>;
  T pop[24][M::CELLS];     // in-plane-moving populations of the current source plane
  T pz[M::CELLS];          // sum_cz w(cz) phi^{n+1}(z + cz)   at the output plane
  T dz[M::CELLS];          // sum_cz w(cz) cz phi^{n+1}(z + cz)
};

template <typename T, int I, int TX, int TY>
__device__ __forceinline__ void k2_store_pop(K2Smem<T, TX, TY>& sm, int c, const Coef<T>& cf,
                                             T (&own)[27]) {
  constexpr int CX = I % 3 - 1, CY = (I / 3) % 3 - 1, CZ = I / 9 - 1;
  T f = fpost_dir<T, CX, CY, CZ>(cf);
  own[I] = f;
  if (CX != 0 || CY != 0) sm.pop[pop_slot(CX, CY, CZ)][c] = f;
}

template <typename T, int TX, int TY, int I = 0>
struct K2StoreAll {
  static __device__ __forceinline__ void run(K2Smem<T, TX, TY>& sm, int c, const Coef<T>& cf,
                                             T (&own)[27]) {
    k2_store_pop<T, I, TX, TY>(sm, c, cf, own);
    K2StoreAll<T, TX, TY, I + 1>::run(sm, c, cf, own);
  }
};
template <typename T, int TX, int TY>
struct K2StoreAll<T, TX, TY, 27> {
  static __device__ __forceinline__ void run(K2Smem<T, TX, TY>&, int, const Coef<T>&, T (&)[27]) {}
};

// wall flags of one output column at one source plane
struct WallFlags { bool xm, xp, ym, yp, zm, zp; };
template <int D> __device__ __forceinline__ bool crosses(bool m, bool p) {
  return D < 0 ? m : (D > 0 ? p : false);
}

// Gather direction I at iteration j: the population (CX,CY,CZ) emitted by (x-CX, y-CY, j) arrives
// at (x, y, j+CZ).  mom[CZ+1] accumulates destination plane j+CZ.  With walls: the arrival is
// dropped if its source lies beyond a wall (x,y) or its destination plane does not exist (z),
// and the node's own outgoing population in direction I that would cross a wall comes back to
// the node itself with the opposite direction (halfway bounce-back, R19).
template <typename T, int I, bool WALLS, int TX, int TY>
__device__ __forceinline__ void k2_gather(const K2Smem<T, TX, TY>& sm, int c, const T (&own)[27],
                                          const WallFlags& wf, Mom<T> (&mom)[3]) {
  using M = TileMap<TX, TY, 1>;
  constexpr int CX = I % 3 - 1, CY = (I / 3) % 3 - 1, CZ = I / 9 - 1;
  T f;
  if (CX == 0 && CY == 0) f = own[I];
  else f = sm.pop[pop_slot(CX, CY, CZ)][c - CY * M::W - CX];
  if (WALLS) {
    bool drop = crosses<-CX>(wf.xm, wf.xp) || crosses<-CY>(wf.ym, wf.yp) ||
                crosses<CZ>(wf.zm, wf.zp);
    if (!drop) accumulate<T, CX, CY, CZ>(mom[CZ + 1], f);
    bool bounce = crosses<CX>(wf.xm, wf.xp) || crosses<CY>(wf.ym, wf.yp) ||
                  crosses<CZ>(wf.zm, wf.zp);
    if (bounce) accumulate<T, -CX, -CY, -CZ>(mom[1], own[I]);
  } else {
    accumulate<T, CX, CY, CZ>(mom[CZ + 1], f);
  }
}

template <typename T, bool WALLS, int TX, int TY, int I = 0>
struct K2GatherAll {
  static __device__ __forceinline__ void run(const K2Smem<T, TX, TY>& sm, int c,
                                             const T (&own)[27], const WallFlags& wf,
                                             Mom<T> (&mom)[3]) {
    k2_gather<T, I, WALLS, TX, TY>(sm, c, own, wf, mom);
    K2GatherAll<T, WALLS, TX, TY, I + 1>::run(sm, c, own, wf, mom);
  }
};
template <typename T, bool WALLS, int TX, int TY>
struct K2GatherAll<T, WALLS, TX, TY, 27> {
  static __device__ __forceinline__ void run(const K2Smem<T, TX, TY>&, int, const T (&)[27],
                                             const WallFlags&, Mom<T> (&)[3]) {}
};

template <typename T>
__device__ __forceinline__ int wrap_plane(int j, int n) { return j < 0 ? j + n : (j >= n ? j - n : j); }

template <typename T, int TX, int TY, bool WALLS, int MINB>
__global__ void __launch_bounds__((TileMap<TX, TY, 1>::NTHREADS), MINB)
k_stream_collide_tiled(DevParams<T> P, const T* __restrict__ S, T* __restrict__ D, int zchunk) {
  using M = TileMap<TX, TY, 1>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  K2Smem<T, TX, TY>& sm = *reinterpret_cast<K2Smem<T, TX, TY>*>(smem_raw);

  const int tid = threadIdx.x;
  int lx, ly;
  const bool mapped = M::coords(tid, lx, ly);
  const int gx = blockIdx.x * TX + lx, gy = blockIdx.y * TY + ly;
  const int z0 = blockIdx.z * zchunk;
  const int z1 = min(P.nz, z0 + zchunk);
  const int c = M::cell(lx, ly);

  // which role does this thread play?
  const bool in_ring = mapped && gx >= -1 && gx <= P.nx && gy >= -1 && gy <= P.ny;
  int kx = 0, ky = 0;
  const int sx = ghost_index(min(max(gx, -1), P.nx), P.nx, P.bcx, kx);   // wrapped / mirrored
  const int sy = ghost_index(min(max(gy, -1), P.ny), P.ny, P.bcy, ky);
  const bool has_mom = in_ring && !kx && !ky;        // a real node whose populations exist
  const bool is_out = tid < M::NMAIN && gx < P.nx && gy < P.ny;
  const long long col = sx + (long long)P.nx * sy;   // in-plane offset of the source column
  const long long plane = (long long)P.nx * P.ny;
  const T* phin = D + F_PHI * P.N;                   // phi^{n+1} (written by the Allen-Cahn stage)

  WallFlags wf;
  wf.xm = WALLS && P.bcx && gx == 0;       wf.xp = WALLS && P.bcx && gx == P.nx - 1;
  wf.ym = WALLS && P.bcy && gy == 0;       wf.yp = WALLS && P.bcy && gy == P.ny - 1;
  wf.zm = false; wf.zp = false;

  Mom<T> mom[3] = {};                // destination planes j-1, j, j+1
  T ph_m = 0, ph_0 = 0, ph_p = 0;    // phi^{n+1} of the own column at planes j-2, j-1, j
  T uo[2][3] = {};                   // u^n of the own node at planes j-1 (slot 0) and j (slot 1)

  for (int j = z0 - 1; j <= z1; ++j) {
    // ---- source plane j: real, wrapped, or beyond a wall
    int kz = 0;
    const int jz = ghost_index(j, P.nz, P.bcz, kz);          // mirrored index if beyond a wall
    const bool plane_real = !kz;
    if (WALLS) { wf.zm = P.bcz && j == 0; wf.zp = P.bcz && j == P.nz - 1; }

    // phi^{n+1} pipeline (ghost planes mirror evenly, R19)
    ph_m = ph_0; ph_0 = ph_p;
    if (in_ring) ph_p = phin[col + plane * jz];

    T own[27];
    uo[0][0] = uo[1][0]; uo[0][1] = uo[1][1]; uo[0][2] = uo[1][2];
    if (has_mom && plane_real) {
      const long long s = col + plane * jz;
      const T ux = S[F_UX * P.N + s], uy = S[F_UY * P.N + s], uz = S[F_UZ * P.N + s];
      Coef<T> cf = coefficients<T>(S[F_P * P.N + s], ux, uy, uz, S[F_AXX * P.N + s],
                                   S[F_AYY * P.N + s], S[F_AZZ * P.N + s], S[F_AXY * P.N + s],
                                   S[F_AXZ * P.N + s], S[F_AYZ * P.N + s], S[F_AX * P.N + s],
                                   S[F_AY * P.N + s], S[F_AZ * P.N + s]);
      uo[1][0] = ux; uo[1][1] = uy; uo[1][2] = uz;
      K2StoreAll<T, TX, TY>::run(sm, c, cf, own);
    }
    // z-combinations of phi^{n+1} for the output plane k = j-1 (Eq. 18-19 are separable)
    if (in_ring) {
      sm.pz[c] = T(1.0 / 6.0) * (ph_m + ph_p) + T(2.0 / 3.0) * ph_0;
      sm.dz[c] = T(1.0 / 6.0) * (ph_p - ph_m);
    }
    __syncthreads();

    if (is_out) {
      if (plane_real) K2GatherAll<T, WALLS, TX, TY>::run(sm, c, own, wf, mom);
      const int k = j - 1;
      if (k >= z0) {
        // gradient and Laplacian of phi^{n+1} at (gx, gy, k) from the 3x3 in-plane neighbourhood
        T sx_ = 0, sy_ = 0, sz_ = 0, sw_ = 0;
#pragma unroll
        for (int q = 0; q < 9; ++q) {
          const int cx = q % 3 - 1, cy = q / 3 - 1;
          const T w = w1<T>(cx) * w1<T>(cy);
          const T a = sm.pz[c + cy * M::W + cx], b = sm.dz[c + cy * M::W + cx];
          sw_ = fma(w, a, sw_);
          sz_ = fma(w, b, sz_);
          if (cx) sx_ = fma(w * T(cx), a, sx_);
          if (cy) sy_ = fma(w * T(cy), a, sy_);
        }
        const T lap = T(6) * (sw_ - ph_0);
        NodeOut<T> o = close_node(P, mom[0], ph_0, T(3) * sx_, T(3) * sy_, T(3) * sz_, lap,
                                  uo[0][0], uo[0][1], uo[0][2]);
        const long long d = gx + (long long)P.nx * gy + plane * k;
        D[F_P * P.N + d] = o.p;
        D[F_UX * P.N + d] = o.ux; D[F_UY * P.N + d] = o.uy; D[F_UZ * P.N + d] = o.uz;
        D[F_AXX * P.N + d] = o.axx; D[F_AYY * P.N + d] = o.ayy; D[F_AZZ * P.N + d] = o.azz;
        D[F_AXY * P.N + d] = o.axy; D[F_AXZ * P.N + d] = o.axz; D[F_AYZ * P.N + d] = o.ayz;
        D[F_AX * P.N + d] = o.ax; D[F_AY * P.N + d] = o.ay; D[F_AZ * P.N + d] = o.az;
      }
      mom[0] = mom[1]; mom[1] = mom[2]; mom[2] = Mom<T>{};
    }
    __syncthreads();
  }
}

// ------------------------------------------------------------------------------------------
// Kernel K1: conservative Allen-Cahn, FTCS (Eq. 20; R10, R13, R16, R17, R19).  H = 2.
//   phi^{n+1} = phi - div(Q) + D lap(phi),  Q = phi u + kappa_AC phi (1-phi) n,
//   n = grad(phi)/sqrt(|grad(phi)|^2 + eps^2).
// Ghost columns/planes beyond a wall are evaluated from mirrored inputs (phi even, u odd), which
// yields the odd normal component of the sharpening flux that R19 prescribes.
// ------------------------------------------------------------------------------------------
template <typename T, int TX, int TY>
struct K1Smem {
  using M = TileMap<TX, TY, 2>;
  T pz[M::CELLS], dz[M::CELLS];            // z-combinations of phi^n at the flux plane j
  T X[M::CELLS], Y[M::CELLS], Z[M::CELLS]; // z-combinations of Q at the output plane k
};

template <typename T, int TX, int TY, int MINB>
__global__ void __launch_bounds__((TileMap<TX, TY, 2>::NTHREADS), MINB)
k_allen_cahn_tiled(DevParams<T> P, const T* __restrict__ S, T* __restrict__ phin, int zchunk) {
  using M = TileMap<TX, TY, 2>;
  __shared__ K1Smem<T, TX, TY> sm;

  const int tid = threadIdx.x;
  int lx, ly;
  const bool mapped = M::coords(tid, lx, ly);
  const int gx = blockIdx.x * TX + lx, gy = blockIdx.y * TY + ly;
  const int z0 = blockIdx.z * zchunk;
  const int z1 = min(P.nz, z0 + zchunk);
  const int c = M::cell(lx, ly);

  const bool ring2 = mapped && gx >= -2 && gx <= P.nx + 1 && gy >= -2 && gy <= P.ny + 1;
  const bool ring1 = ring2 && lx >= -1 && lx <= TX && ly >= -1 && ly <= TY && gx >= -1 &&
                     gx <= P.nx && gy >= -1 && gy <= P.ny;
  const bool is_out = tid < M::NMAIN && gx < P.nx && gy < P.ny;
  int kx = 0, ky = 0;
  const int sx = ghost_index(min(max(gx, -2), P.nx + 1), P.nx, P.bcx, kx);
  const int sy = ghost_index(min(max(gy, -2), P.ny + 1), P.ny, P.bcy, ky);
  const long long col = sx + (long long)P.nx * sy;
  const long long plane = (long long)P.nx * P.ny;
  const T* phi = S + F_PHI * P.N;
  const T* u = S + F_UX * P.N;

  int kz;
  T q_m = 0, q_0 = 0, q_p = 0;                 // phi^n at planes j-1, j, j+1 of the own column
  if (ring2) {
    q_0 = phi[col + plane * ghost_index(z0 - 2, P.nz, P.bcz, kz)];
    q_p = phi[col + plane * ghost_index(z0 - 1, P.nz, P.bcz, kz)];
  }
  T Qa[3] = {}, Qb[3] = {}, Qc[3] = {};        // Q at planes j-2, j-1, j
  T sw_prev = 0, phi_prev = 0;                 // in-plane smoothing of pz and phi at plane j-1

  for (int j = z0 - 1; j <= z1; ++j) {
    q_m = q_0; q_0 = q_p;
    if (ring2) {
      q_p = phi[col + plane * ghost_index(j + 1, P.nz, P.bcz, kz)];
      sm.pz[c] = T(1.0 / 6.0) * (q_m + q_p) + T(2.0 / 3.0) * q_0;
      sm.dz[c] = T(1.0 / 6.0) * (q_p - q_m);
    }
    __syncthreads();

    T sw_now = 0;
    if (ring1) {
      T sx_ = 0, sy_ = 0, sz_ = 0;
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        const T w = w1<T>(cx) * w1<T>(cy);
        const T a = sm.pz[c + cy * M::W + cx], b = sm.dz[c + cy * M::W + cx];
        sw_now = fma(w, a, sw_now);
        sz_ = fma(w, b, sz_);
        if (cx) sx_ = fma(w * T(cx), a, sx_);
        if (cy) sy_ = fma(w * T(cy), a, sy_);
      }
      const T g0 = T(3) * sx_, g1 = T(3) * sy_, g2 = T(3) * sz_;
      const T s = P.kappa_ac * q_0 * (T(1) - q_0) *
                  rsqrt_t(g0 * g0 + g1 * g1 + g2 * g2 + T(1e-24));
      const int jz = ghost_index(j, P.nz, P.bcz, kz);
      const long long n = col + plane * jz;
      const T sgn = ((kx + ky + kz) & 1) ? -q_0 : q_0;      // phi u with velocity-like ghosts
#pragma unroll
      for (int al = 0; al < 3; ++al) { Qa[al] = Qb[al]; Qb[al] = Qc[al]; }
      Qc[0] = fma(sgn, u[n], s * g0);
      Qc[1] = fma(sgn, u[P.N + n], s * g1);
      Qc[2] = fma(sgn, u[2 * P.N + n], s * g2);
      // z-combinations of Q for the output plane k = j-1 (Eq. 18, component-wise: R17)
      sm.X[c] = T(1.0 / 6.0) * (Qa[0] + Qc[0]) + T(2.0 / 3.0) * Qb[0];
      sm.Y[c] = T(1.0 / 6.0) * (Qa[1] + Qc[1]) + T(2.0 / 3.0) * Qb[1];
      sm.Z[c] = T(1.0 / 6.0) * (Qc[2] - Qa[2]);
    }
    __syncthreads();

    const int k = j - 1;
    if (is_out && k >= z0) {
      T div = 0;
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        const T w = w1<T>(cx) * w1<T>(cy);
        const int cc = c + cy * M::W + cx;
        div = fma(w, sm.Z[cc], div);
        if (cx) div = fma(w * T(cx), sm.X[cc], div);
        if (cy) div = fma(w * T(cy), sm.Y[cc], div);
      }
      const T lap = T(6) * (sw_prev - phi_prev);
      phin[gx + (long long)P.nx * gy + plane * k] = phi_prev - T(3) * div + P.mob * lap;
    }
    sw_prev = sw_now;
    phi_prev = q_0;
  }
}

// ------------------------------------------------------------------------------------------
// Launch of one time step.
// ------------------------------------------------------------------------------------------
template <typename T> struct TileCfg;
template <> struct TileCfg<double> { static constexpr int TX = 32, TY = 8, ZC = 32; };
template <> struct TileCfg<float>  { static constexpr int TX = 32, TY = 8, ZC = 32; };

template <typename T>
int launch_step_tiled(const DevParams<T>& P, const T* S, T* D, cudaStream_t stream,
                      long long* launches, const Marker& mk) {
  constexpr int TX = TileCfg<T>::TX, TY = TileCfg<T>::TY, ZC = TileCfg<T>::ZC;
  const dim3 grid((P.nx + TX - 1) / TX, (P.ny + TY - 1) / TY, (P.nz + ZC - 1) / ZC);
  using M1 = TileMap<TX, TY, 2>;
  using M2 = TileMap<TX, TY, 1>;
  const bool walls = P.bcx || P.bcy || P.bcz;

  k_allen_cahn_tiled<T, TX, TY, 1><<<grid, M1::NTHREADS, 0, stream>>>(P, S, D + F_PHI * P.N, ZC);
  mk.mark(1);

  const size_t smem2 = sizeof(K2Smem<T, TX, TY>);
  static bool attr_set = false;
  if (!attr_set) {
    cudaError_t e;
    e = cudaFuncSetAttribute(k_stream_collide_tiled<T, TX, TY, false, 1>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem2));
    if (e != cudaSuccess) return int(e);
    e = cudaFuncSetAttribute(k_stream_collide_tiled<T, TX, TY, true, 1>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, int(smem2));
    if (e != cudaSuccess) return int(e);
    attr_set = true;
  }
  if (walls)
    k_stream_collide_tiled<T, TX, TY, true, 1><<<grid, M2::NTHREADS, smem2, stream>>>(P, S, D, ZC);
  else
    k_stream_collide_tiled<T, TX, TY, false, 1><<<grid, M2::NTHREADS, smem2, stream>>>(P, S, D, ZC);
  mk.mark(2);
  *launches += 2;
  return int(cudaGetLastError());
}

}  // namespace tslb
