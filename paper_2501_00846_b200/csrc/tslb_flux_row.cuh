// tslb_flux_row.cuh -- interface tracking (Eq. 20) in flux form, ROW kernel (periodic axes and walls).
//
// Same arithmetic as tslb_flux.cuh (phi^{n+1} = phi - div Q + D lap(phi), Eq. 18 / repaired
// Eq. 19, R10, R16), other work distribution.  The kernel moves only 5 scalars per update, so it
// must spend very few instructions per node to stay on the HBM roofline:
//   * a thread owns V = 128 bit / sizeof(T) CONSECUTIVE x nodes of one row (4 in fp32, 2 in fp64):
//     every global access is a 128-bit vector, a warp moves 512 contiguous bytes per instruction;
//   * a warp owns one row segment of 32 V nodes and marches along z; the z-combinations
//       X = Qx(k-1) + 4 Qx(k) + Qx(k+1),  Y likewise,  Z = Qz(k+1) - Qz(k-1),
//       pz = phi(k-1) + 4 phi(k) + phi(k+1)
//     live in two running accumulators per quantity;
//   * with A = c1 Z + c2 pz, Bx = c1 X, By = c1 Y (c1 = -3/216, c2 = 6 D/216) the in-plane part is
//     separable:  R(x) = (A - Bx)(x-1) + 4 A(x) + (A + Bx)(x+1),  S(x) = By(x-1) + 4 By(x) + By(x+1)
//     are formed in registers, the two row ends come from the neighbour lanes by warp shuffle;
//     phi^{n+1}(y) = (1 - 6 D) phi + (R - S)(y-1) + 4 R(y) + (R + S)(y+1) takes two 128-bit
//     shared-memory words from the rows below / above;
//   * the columns left and right of the tile are single-node columns owned by the lanes of one
//     extra warp, which runs one plane ahead and hands (A -+ Bx, By) over in shared memory;
//   * global loads are cp.async copies into a private staging slot, NSTAGE planes ahead.
// Requires nx % V == 0 (vector alignment of every row); otherwise tslb_flux.cuh is used.
#pragma once
#include "tslb_device.cuh"

namespace tslb {

template <typename T> struct RowVec;
template <> struct RowVec<float> {
  static constexpr int V = 4;
  using vec = float4;
  static __device__ __forceinline__ void get(const float4& v, float (&a)[4]) {
    a[0] = v.x; a[1] = v.y; a[2] = v.z; a[3] = v.w;
  }
  static __device__ __forceinline__ float4 make(const float (&a)[4]) {
    return make_float4(a[0], a[1], a[2], a[3]);
  }
};
template <> struct RowVec<double> {
  static constexpr int V = 2;
  using vec = double2;
  static __device__ __forceinline__ void get(const double2& v, double (&a)[2]) { a[0] = v.x; a[1] = v.y; }
  static __device__ __forceinline__ double2 make(const double (&a)[2]) { return make_double2(a[0], a[1]); }
};

template <typename T, int TY, int NSTAGE>
struct RowSmem {
  using vec = typename RowVec<T>::vec;
  static constexpr int ROWS = TY + 2;
  vec um[2][ROWS][32];              // (Dx - S) of the V nodes of a thread, double buffered over k
  vec up[2][ROWS][32];              // (Dx + S)
  vec aa[2][ROWS][32];              // A itself (the rows above and below difference it with theirs)
  T xh[2][ROWS][2][2];              // [k & 1][row][side]{A -+ Bx, By} of the columns beside the tile
  vec stage[NSTAGE][4][ROWS][32];   // Qx, Qy, Qz, phi of the thread's nodes, one slot per plane
  T xstage[NSTAGE][4][2 * ROWS];    // the same for the single-node columns of the extra warp
};

// running z-combination  c(k) = v(k-1) + 4 v(k) + v(k+1):  returns c(k) when v(k+1) arrives
template <typename T>
__device__ __forceinline__ T zsum141(T v, T& a, T& b) {
  const T r = a + v;
  a = fma(T(4), v, b);
  b = v;
  return r;
}

// WXY: walls on x or y are possible; false compiles their ghost handling out (the periodic and
// z-wall instantiations keep their registers)
template <typename T, int TY, int MINB, int NSTAGE, bool WXY = false>
__global__ void __launch_bounds__((TY + 3) * 32, MINB)
k_allen_cahn_row(DevParams<T> P, const T* __restrict__ S, const T* __restrict__ Q,
                 T* __restrict__ phin, int zchunk) {
  using RV = RowVec<T>;
  using vec = typename RV::vec;
  constexpr int V = RV::V;
  constexpr int ROWS = TY + 2;
  using SM = RowSmem<T, TY, NSTAGE>;
  extern __shared__ __align__(16) unsigned char row_smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(row_smem_raw);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const bool xhalo = warp == ROWS;                 // the extra warp: columns beside the tile
  const int gx0 = blockIdx.x * (32 * V);
  const int nact = min(32, (P.nx - gx0) / V);      // lanes of a row warp that own nodes
  const int z0 = P.zbeg + blockIdx.z * zchunk;
  const int z1 = min(P.zend, z0 + zchunk);
  const int plane = P.nx * P.ny;
  const T* phi = S + F_PHI * P.N;
  const T c1 = T(-3.0 / 216.0), c2 = P.c2;

  // row of this thread: row warps own row `warp`; lane h of the extra warp owns row h / 2
  const int row = xhalo ? (lane >> 1) : warp;
  const int side = lane & 1;
  const int gy = blockIdx.y * TY + row - 1;
  const bool row_used = row < ROWS && gy <= P.ny;  // rows beyond the +1 halo of a ragged tile idle
  // source of a position beyond the lattice: the periodic image, or (wall, R19) the mirrored node
  auto src = [](int g, int n, int bc, int& crossed) {
    crossed = 0;
    if (g < 0) { crossed = bc; return bc ? -1 - g : g + n; }
    if (g >= n) { crossed = bc; return bc ? 2 * n - 1 - g : g - n; }
    return g;
  };
  int kx_ = 0, ky_ = 0;                            // this thread's nodes lie beyond an x / y wall
  const int sy = src(gy, P.ny, WXY ? P.bcy : 0, ky_);
  int sx;                                          // first (row warps) or only (extra warp) column
  if (xhalo) sx = src(side == 0 ? gx0 - 1 : gx0 + nact * V, P.nx, WXY ? P.bcx : 0, kx_);
  else sx = gx0 + lane * V;
  const int kx = WXY ? kx_ : 0, ky = WXY ? ky_ : 0;
  const bool active = row_used && (xhalo || lane < nact);
  const bool is_out = !xhalo && active && row >= 1 && row <= TY && gy < P.ny;
  const int col = active ? sx + P.nx * sy : 0;

  // Walls (R19).  A ghost position (beyond a wall of any axis: the plane j = -1 / nz of the
  // marching axis, a halo row beyond a y wall, a side column beyond an x wall) holds the mirrored
  // node m with phi even, the advective flux phi u odd in every component once per wall crossed
  // (no slip) and the sharpening flux odd in the components of the crossed axes only (neutral
  // wetting).  In terms of the stored total flux Q = phi u + kappa phi (1-phi) n, with
  // sa = (-1)^(walls crossed) and s_al = -1 if axis al was crossed, else +1:
  //   Q_al(ghost) = s_al Q_al(m) + (sa - s_al) phi(m) u_al(m),      phi(ghost) = phi(m),
  // so ghost positions also read u of the mirrored node (one wall on z: Qx - 2 phi ux, Qy - 2 phi
  // uy, -Qz).
  auto zsrc = [&](int j) {
    if (j < 0) return P.bcz ? -1 - j : j + P.nz;
    if (j >= P.nz) return P.bcz ? 2 * P.nz - 1 - j : j - P.nz;
    return j;
  };
  auto ghostify = [&](int j, T (&qx)[V], T (&qy)[V], T (&qz)[V], const T (&f)[V]) {
    const int kz = (P.bcz && (j < 0 || j >= P.nz)) ? 1 : 0;
    if (!(kx | ky | kz) || !active) return;
    const T sa = ((kx + ky + kz) & 1) ? T(-1) : T(1);
    const T s0 = kx ? T(-1) : T(1), s1 = ky ? T(-1) : T(1), s2 = kz ? T(-1) : T(1);
    const long long s = col + (long long)plane * zsrc(j);
#pragma unroll
    for (int i = 0; i < V; ++i) {
      if (xhalo && i > 0) break;
      T ux, uy, uz;
      load_u(S, P.N, s + i, ux, uy, uz);
      qx[i] = fma((sa - s0) * f[i], ux, s0 * qx[i]);
      qy[i] = fma((sa - s1) * f[i], uy, s1 * qy[i]);
      qz[i] = fma((sa - s2) * f[i], uz, s2 * qz[i]);
    }
  };
  auto issue = [&](int j, int slot) {              // one commit group per plane, possibly empty
    if (active && j <= z1) {
      const int jz = zsrc(j);
      const long long s = col + (long long)plane * jz;
      if (xhalo) {
        cp_async_small(&sm.xstage[slot][0][lane], Q + s);
        cp_async_small(&sm.xstage[slot][1][lane], Q + P.N + s);
        cp_async_small(&sm.xstage[slot][2][lane], Q + 2 * P.N + s);
        cp_async_small(&sm.xstage[slot][3][lane], phi + s);
      } else {
        cp_async16(&sm.stage[slot][0][row][lane], Q + s);
        cp_async16(&sm.stage[slot][1][row][lane], Q + P.N + s);
        cp_async16(&sm.stage[slot][2][row][lane], Q + 2 * P.N + s);
        cp_async16(&sm.stage[slot][3][row][lane], phi + s);
      }
    }
    cp_async_commit();
  };

  // running accumulators (see zsum141) and the two older planes of Qz
  T xa[V] = {}, xb[V] = {}, ya[V] = {}, yb[V] = {}, pm[V] = {}, pb[V] = {}, zm[V] = {}, z0v[V] = {};
  T A[V], Bx[V], By[V], fb[V], g0[V];

  // receive one plane of the own nodes: afterwards A, Bx, By, fb describe the plane before it
  auto receive = [&](const T (&qx)[V], const T (&qy)[V], const T (&qz)[V], const T (&f)[V]) {
#pragma unroll
    for (int i = 0; i < V; ++i) {
      fb[i] = pb[i];
      const T X = zsum141(qx[i], xa[i], xb[i]);
      const T Y = zsum141(qy[i], ya[i], yb[i]);
      // phi along z in DIFFERENCE form: d2z = phi(k-1) - 2 phi(k) + phi(k+1), pz = 6 phi(k) + d2z
      const T d2z = (pm[i] - pb[i]) + (f[i] - pb[i]);
      const T pz = fma(T(6), pb[i], d2z);
      pm[i] = pb[i]; pb[i] = f[i];
      const T Z = qz[i] - zm[i];
      zm[i] = z0v[i]; z0v[i] = qz[i];
      A[i] = fma(c1, Z, c2 * pz);          // carries 6 c2 phi: only ever used in differences
      g0[i] = fma(c1, Z, c2 * d2z);        // the same without it: the node's own small part
      Bx[i] = c1 * X;
      By[i] = c1 * Y;
    }
  };
  auto take = [&](int slot, int j) {
    T qx[V] = {}, qy[V] = {}, qz[V] = {}, f[V] = {};
    if (active) {
      if (xhalo) {
        qx[0] = sm.xstage[slot][0][lane]; qy[0] = sm.xstage[slot][1][lane];
        qz[0] = sm.xstage[slot][2][lane]; f[0] = sm.xstage[slot][3][lane];
      } else {
        RV::get(sm.stage[slot][0][row][lane], qx);
        RV::get(sm.stage[slot][1][row][lane], qy);
        RV::get(sm.stage[slot][2][row][lane], qz);
        RV::get(sm.stage[slot][3][row][lane], f);
      }
    }
    ghostify(j, qx, qy, qz, f);
    receive(qx, qy, qz, f);
  };

  // Plane schedule.  Row warps receive plane j in iteration j (j = z0-1 .. z1) and finish output
  // plane k = j-1.  The extra warp is one plane ahead: it receives plane j+1 in iteration j and
  // leaves the combinations of plane j in xh[j & 1], which the row warps read in iteration j+1.
  const int lead = xhalo ? 1 : 0;
  int slot = 0;
  if (xhalo) {                                      // plane z0-1 of the extra warp, before the loop
    T qx[V] = {}, qy[V] = {}, qz[V] = {}, f[V] = {};
    if (active) {
      const long long s = col + (long long)plane * zsrc(z0 - 1);
      qx[0] = __ldg(Q + s); qy[0] = __ldg(Q + P.N + s); qz[0] = __ldg(Q + 2 * P.N + s);
      f[0] = __ldg(phi + s);
    }
    ghostify(z0 - 1, qx, qy, qz, f);
    receive(qx, qy, qz, f);
  }
#pragma unroll
  for (int d = 0; d < NSTAGE; ++d) issue(z0 - 1 + lead + d, d);

  for (int j = z0 - 1; j <= z1; ++j) {
    const int k = j - 1;
    cp_async_wait<NSTAGE - 1>();                    // the group of plane j + lead has landed
    take(slot, j + lead);
    issue(j + lead + NSTAGE, slot);
    slot = (slot + 1 == NSTAGE) ? 0 : slot + 1;

    T Dx[V], Sy[V];
    if (xhalo) {
      // combinations of plane j (= k + 1) for the row warps' next iteration
      if (active) {
        sm.xh[j & 1][row][side][0] = side == 0 ? A[0] - Bx[0] : A[0] + Bx[0];
        sm.xh[j & 1][row][side][1] = By[0];
      }
    } else {
      // row ends: (A - Bx, By) of the node on the left, (A + Bx, By) of the node on the right
      T lm = __shfl_up_sync(0xffffffffu, A[V - 1] - Bx[V - 1], 1);
      T lby = __shfl_up_sync(0xffffffffu, By[V - 1], 1);
      T rp = __shfl_down_sync(0xffffffffu, A[0] + Bx[0], 1);
      T rby = __shfl_down_sync(0xffffffffu, By[0], 1);
      if (row_used) {
        if (lane == 0) { lm = sm.xh[k & 1][row][0][0]; lby = sm.xh[k & 1][row][0][1]; }
        if (lane == nact - 1) { rp = sm.xh[k & 1][row][1][0]; rby = sm.xh[k & 1][row][1][1]; }
      }
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const T left = i == 0 ? lm : A[i - 1] - Bx[i - 1];
        const T right = i == V - 1 ? rp : A[i + 1] + Bx[i + 1];
        const T bl = i == 0 ? lby : By[i - 1];
        const T br = i == V - 1 ? rby : By[i + 1];
        Dx[i] = (left - A[i]) + (right - A[i]);      // R = 6 A + Dx is never formed
        Sy[i] = fma(T(4), By[i], bl + br);
      }
      if (active) {
        T d[V], s[V];
#pragma unroll
        for (int i = 0; i < V; ++i) { d[i] = Dx[i] - Sy[i]; s[i] = Dx[i] + Sy[i]; }
        if (row <= TY - 1) sm.um[k & 1][row][lane] = RV::make(d);      // read by row + 1
        if (row >= 2) sm.up[k & 1][row][lane] = RV::make(s);           // read by row - 1
        sm.aa[k & 1][row][lane] = RV::make(A);                         // read by rows +- 1
      }
    }
    __syncthreads();
    if (is_out && k >= z0) {
      // phi' = c0 phi + sum_y w_y (R -+ S)(y) with R = 6 A + Dx, A = g0 + 6 c2 phi and
      // c0 + 216 c2 = 1 becomes, with every O(phi) term cancelled symbolically,
      //   phi' = phi + 36 g0 + 6 [(A(y-1) - A) + (A(y+1) - A)] + 4 Dx + (Dx - S)(y-1) + (Dx + S)(y+1):
      // an increment of small terms on top of phi, as in the oracle's phi - div Q + D lap(phi)
      // with the Laplacian as a sum of differences; the flux form's own c0 phi + 0.3 phi-sized
      // partial sums cost ~10x more rounding noise in phi per step.
      T lo[V], hi[V], alo[V], ahi[V], o[V];
      RV::get(sm.um[k & 1][row - 1][lane], lo);
      RV::get(sm.up[k & 1][row + 1][lane], hi);
      RV::get(sm.aa[k & 1][row - 1][lane], alo);
      RV::get(sm.aa[k & 1][row + 1][lane], ahi);
#pragma unroll
      for (int i = 0; i < V; ++i) {
        const T ty = (alo[i] - A[i]) + (ahi[i] - A[i]);
        const T inc = fma(T(36), g0[i], fma(T(6), ty, fma(T(4), Dx[i], lo[i] + hi[i])));
        o[i] = fb[i] + inc;
      }
      *reinterpret_cast<vec*>(phin + (sx + P.nx * gy + (long long)plane * k)) = RV::make(o);
    }
  }
  cp_async_wait<0>();
}

}  // namespace tslb
