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

// NSTAGE = 1: the 14 scalars of the thread's own node for the next plane are fetched with
// cp.async into a private shared-memory slot while the current plane is processed.
template <typename T, int TX, int TY, bool WALLS, int MINB, int NSTAGE = 0>
__global__ void __launch_bounds__((TileMap<TX, TY, 1>::NTHREADS), MINB)
k_stream_collide_tiled(DevParams<T> P, const T* __restrict__ S, T* __restrict__ D, int zchunk) {
  using M = TileMap<TX, TY, 1>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  K2Smem<T, TX, TY>& sm = *reinterpret_cast<K2Smem<T, TX, TY>*>(smem_raw);
  StageBuf<T, M::CELLS>& stg =
      *reinterpret_cast<StageBuf<T, M::CELLS>*>(smem_raw + sizeof(K2Smem<T, TX, TY>));

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

  auto stage_issue = [&](int j) {
    if (NSTAGE > 0) {
      if (in_ring && j <= z1) {
        using V = typename VecOf<T>::type;
        int kz2 = 0;
        const long long s = col + plane * ghost_index(j, P.nz, P.bcz, kz2);
        cp_async_small(&stg.ph[c], phin + s);
        if (has_mom && !kz2) {
          const V* g = reinterpret_cast<const V*>(S);
#pragma unroll
          for (int k = 0; k < 12 / VecOf<T>::W; ++k) cp_async16(&stg.vec[k][c], g + k * P.N + s);
          cp_async_small(&stg.az[c], S + 12 * P.N + s);
        }
      }
      cp_async_commit();
    }
  };
  stage_issue(z0 - 1);

  for (int j = z0 - 1; j <= z1; ++j) {
    // ---- source plane j: real, wrapped, or beyond a wall
    int kz = 0;
    const int jz = ghost_index(j, P.nz, P.bcz, kz);          // mirrored index if beyond a wall
    const bool plane_real = !kz;
    if (WALLS) { wf.zm = P.bcz && j == 0; wf.zp = P.bcz && j == P.nz - 1; }

    // phi^{n+1} pipeline (ghost planes mirror evenly, R19)
    ph_m = ph_0; ph_0 = ph_p;
    if (NSTAGE > 0) cp_async_wait<0>();
    if (in_ring) ph_p = NSTAGE > 0 ? stg.ph[c] : phin[col + plane * jz];

    T own[27];
    uo[0][0] = uo[1][0]; uo[0][1] = uo[1][1]; uo[0][2] = uo[1][2];
    T m13[13];
    const bool src_here = has_mom && plane_real;
    if (src_here) {
      if (NSTAGE > 0) {
        constexpr int W = VecOf<T>::W;
#pragma unroll
        for (int k = 0; k < 12 / W; ++k) unpack(stg.vec[k][c], &m13[k * W]);
        m13[12] = stg.az[c];
      } else {
        load13(S, P.N, col + plane * jz, m13);
      }
    }
    stage_issue(j + 1);                        // refill the slot just consumed
    if (src_here) {
      Coef<T> cf = coef_from13(m13);
      uo[1][0] = m13[F_UX]; uo[1][1] = m13[F_UY]; uo[1][2] = m13[F_UZ];
      K2StoreAll<T, TX, TY>::run(sm, c, cf, own);
    }
    // z-combinations of phi^{n+1} for the output plane k = j-1 (Eq. 18-19 are separable)
    if (in_ring) {
      sm.pz[c] = fma(T(4), ph_0, ph_m + ph_p);     // integer weights (1,4,1); 1/216 deferred
      sm.dz[c] = ph_p - ph_m;
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
          const T w = T((cx ? 1 : 4) * (cy ? 1 : 4));
          const T a = sm.pz[c + cy * M::W + cx], b = sm.dz[c + cy * M::W + cx];
          sw_ = fma(w, a, sw_);
          sz_ = fma(w, b, sz_);
          if (cx) sx_ = fma(w * T(cx), a, sx_);
          if (cy) sy_ = fma(w * T(cy), a, sy_);
        }
        // Laplacian in difference form (exactly 0 on constants, like the oracle's Eq. 19)
        const T lap = T(6.0 / 216.0) * fma(T(-216), ph_0, sw_);
        const T g3 = T(3.0 / 216.0);
        NodeOut<T> o = close_node(P, mom[0], ph_0, g3 * sx_, g3 * sy_, g3 * sz_, lap,
                                  uo[0][0], uo[0][1], uo[0][2]);
        const long long d = gx + (long long)P.nx * gy + plane * k;
        store_out(D, P.N, d, o);
      }
      mom[0] = mom[1]; mom[1] = mom[2]; mom[2] = Mom<T>{};
    }
    __syncthreads();
  }
  if (NSTAGE > 0) cp_async_wait<0>();
}

// ------------------------------------------------------------------------------------------
// Kernel K1: conservative Allen-Cahn, FTCS (Eq. 20; R10, R13, R16, R17, R19).  H = 2.
//   phi^{n+1} = phi - div(Q) + D lap(phi),  Q = phi u + kappa_AC phi (1-phi) n,
//   n = grad(phi)/sqrt(|grad(phi)|^2 + eps^2).
// Ghost columns/planes beyond a wall are evaluated from mirrored inputs (phi even, u odd), which
// yields the odd normal component of the sharpening flux that R19 prescribes.
// ------------------------------------------------------------------------------------------
// Shared-memory cells of K1, double buffered along the marching index (one barrier per plane).
template <typename T> struct Pair2;
template <> struct Pair2<double> { using type = double2; };
template <> struct Pair2<float> { using type = float2; };
template <typename T, int CELLS> struct K1Buf {
  typename Pair2<T>::type pd[CELLS];   // z-combinations of phi^n at a flux plane:
                                       //   (phi(z-1)+phi(z+1)) + 4 phi(z),  phi(z+1) - phi(z-1)
  T dv[8][CELLS];                      // divergence contributions sent to the 8 in-plane neighbours
};

// Software pipeline of iteration j (all inside one barrier interval):
//   (a) ring-2 threads publish the z-combinations of phi^n for plane j+1,
//   (b) ring-1 threads turn the combinations of plane j (published one iteration ago) into the
//       flux Q(j), combine Q(j-2), Q(j-1), Q(j) along z (Eq. 18 is separable) and SCATTER the
//       in-plane part of div Q for plane j-1: the neighbour in direction d receives
//       w(dx) w(dy) (Z - dx X - dy Y), with integer weights (1,4,1) and the factor 1/216 deferred,
//   (c) main threads sum the 8 contributions published one iteration ago for plane j-2, add
//       their own 16 Z, and write phi^{n+1}(j-2).
// Global loads (phi two planes ahead, u one plane ahead) are issued one iteration before use.
template <typename T, int TX, int TY, int MINB, bool WALLS>
__global__ void __launch_bounds__((TileMap<TX, TY, 2>::NTHREADS), MINB)
k_allen_cahn_tiled(DevParams<T> P, const T* __restrict__ S, T* __restrict__ phin, int zchunk) {
  using M = TileMap<TX, TY, 2>;
  using P2 = typename Pair2<T>::type;
  extern __shared__ __align__(16) unsigned char k1_smem_raw[];
  K1Buf<T, M::CELLS>* sm = reinterpret_cast<K1Buf<T, M::CELLS>*>(k1_smem_raw);

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
  const int sx = ghost_index(min(max(gx, -2), P.nx + 1), P.nx, WALLS ? P.bcx : 0, kx);
  const int sy = ghost_index(min(max(gy, -2), P.ny + 1), P.ny, WALLS ? P.bcy : 0, ky);
  const int col = sx + P.nx * sy;
  const int plane = P.nx * P.ny;
  const T* phic = S + F_PHI * P.N + col;
  const int bcz = WALLS ? P.bcz : 0, nz = P.nz;

  // plane index of z in [-nz, 2nz): periodic wrap or even mirror (R19); kz = crossed a wall
  auto zsrc = [&](int z, int& kz) {
    kz = 0;
    if (z < 0) { if (bcz) { kz = 1; return -1 - z; } return z + nz; }
    if (z >= nz) { if (bcz) { kz = 1; return 2 * nz - 1 - z; } return z - nz; }
    return z;
  };
  auto load_phi = [&](int z) { int kz; return __ldg(phic + plane * zsrc(z, kz)); };
  // u at plane z; velocity-like ghosts change sign once per wall crossed (R19): the sign is
  // returned and applied where the value is consumed, so the load stays a prefetch
  auto load_uz = [&](int z, T& ux, T& uy, T& uz, bool& neg) {
    int kz;
    const int jz = zsrc(z, kz);
    load_u(S, P.N, col + plane * jz, ux, uy, uz);
    neg = WALLS && ((kx + ky + kz) & 1);
  };

  T f0 = 0, f1 = 0, f2 = 0, fn = 0;              // phi^n of the own column at planes j, j+1, j+2
  T un[3] = {};                                  // prefetched u of the next flux plane
  bool un_neg = false;
  T Qa[3] = {}, Qb[3] = {};                      // Q at planes j-2, j-1
  T sw1 = 0, sw2 = 0, ph1 = 0, ph2 = 0;          // smoothing of pz and phi at planes j-1, j-2
  T zz1 = 0;                                     // own Z of plane j-2 (computed in iteration j-1)

  if (ring2) {                                   // prologue: publish plane z0-1
    const T a = load_phi(z0 - 2);
    f1 = load_phi(z0 - 1);
    f2 = load_phi(z0);
    fn = load_phi(z0 + 1);
    P2 v; v.x = fma(T(4), f1, a + f2); v.y = f2 - a;
    sm[0].pd[c] = v;
  }
  if (ring1) load_uz(z0 - 1, un[0], un[1], un[2], un_neg);
  __syncthreads();

  for (int j = z0 - 1; j <= z1 + 1; ++j) {
    const int b = (j - z0 + 1) & 1;
    // (a) publish plane j+1
    f0 = f1; f1 = f2; f2 = fn;
    if (ring2 && j + 1 <= z1) {
      P2 v; v.x = fma(T(4), f1, f0 + f2); v.y = f2 - f0;
      sm[b ^ 1].pd[c] = v;
      if (j + 3 <= z1 + 1) fn = load_phi(j + 3);
    }
    // (b) flux of plane j, scatter of div Q for plane j-1
    T sw0 = 0, zz0 = 0;
    if (ring1 && j <= z1) {
      const T fs = un_neg ? -f0 : f0;              // phi u with the ghost sign of u
      const T u0 = un[0], u1 = un[1], u2 = un[2];
      if (j + 1 <= z1) load_uz(j + 1, un[0], un[1], un[2], un_neg);
      T rs[3], rd[3], zs[3];
#pragma unroll
      for (int r = 0; r < 3; ++r) {
        const int cc = c + (r - 1) * M::W;
        const P2 m = sm[b].pd[cc - 1], o = sm[b].pd[cc], p = sm[b].pd[cc + 1];
        rs[r] = fma(T(4), o.x, m.x + p.x);
        rd[r] = p.x - m.x;
        zs[r] = fma(T(4), o.y, m.y + p.y);
      }
      sw0 = fma(T(4), rs[1], rs[0] + rs[2]);
      const T g0 = fma(T(4), rd[1], rd[0] + rd[2]) * T(3.0 / 216.0);
      const T g1 = (rs[2] - rs[0]) * T(3.0 / 216.0);
      const T g2 = fma(T(4), zs[1], zs[0] + zs[2]) * T(3.0 / 216.0);
      const T s = P.kappa_ac * f0 * (T(1) - f0) * rsqrt_t(g0 * g0 + g1 * g1 + g2 * g2 + T(1e-24));
      const T Qc0 = fma(fs, u0, s * g0), Qc1 = fma(fs, u1, s * g1), Qc2 = fma(fs, u2, s * g2);
      const T X = fma(T(4), Qb[0], Qa[0] + Qc0), Y = fma(T(4), Qb[1], Qa[1] + Qc1);
      zz0 = Qc2 - Qa[2];
      Qa[0] = Qb[0]; Qa[1] = Qb[1]; Qa[2] = Qb[2];
      Qb[0] = Qc0; Qb[1] = Qc1; Qb[2] = Qc2;
      // direction d = (dx,dy): slot order (-1,-1) (0,-1) (1,-1) (-1,0) (1,0) (-1,1) (0,1) (1,1)
      const T zpx = zz0 + X, zmx = zz0 - X;
      sm[b].dv[0][c] = zpx + Y;                    // d = (-1,-1):  Z + X + Y
      sm[b].dv[1][c] = T(4) * (zz0 + Y);           // d = ( 0,-1):  4 (Z + Y)
      sm[b].dv[2][c] = zmx + Y;                    // d = ( 1,-1):  Z - X + Y
      sm[b].dv[3][c] = T(4) * zpx;                 // d = (-1, 0):  4 (Z + X)
      sm[b].dv[4][c] = T(4) * zmx;                 // d = ( 1, 0):  4 (Z - X)
      sm[b].dv[5][c] = zpx - Y;                    // d = (-1, 1):  Z + X - Y
      sm[b].dv[6][c] = T(4) * (zz0 - Y);           // d = ( 0, 1):  4 (Z - Y)
      sm[b].dv[7][c] = zmx - Y;                    // d = ( 1, 1):  Z - X - Y
    }
    // (c) output plane k = j-2: arrivals from the source at -d, published one iteration ago
    const int k = j - 2;
    if (is_out && k >= z0) {
      const K1Buf<T, M::CELLS>& r = sm[b ^ 1];
      T div = T(16) * zz1;
      div += (r.dv[0][c + M::W + 1] + r.dv[7][c - M::W - 1]) + (r.dv[2][c + M::W - 1] + r.dv[5][c - M::W + 1]);
      div += (r.dv[1][c + M::W] + r.dv[6][c - M::W]) + (r.dv[3][c + 1] + r.dv[4][c - 1]);
      const T lap = T(6.0 / 216.0) * fma(T(-216), ph2, sw2);   // difference form: 0 on constants
      phin[gx + P.nx * gy + plane * k] = ph2 - T(3.0 / 216.0) * div + P.mob * lap;
    }
    sw2 = sw1; sw1 = sw0; ph2 = ph1; ph1 = f0; zz1 = zz0;
    __syncthreads();
  }
}

}  // namespace tslb
