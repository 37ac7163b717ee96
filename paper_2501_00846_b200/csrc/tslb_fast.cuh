// tslb_fast.cuh -- lean stream-collide kernel for all-periodic boxes.
//
// Same tiling as tslb_tiled.cuh, but the arithmetic uses the tensor-product structure of D3Q27:
//   * the post-collision population of a node is the polynomial  w(c) P(c),
//       P(cx,cy,cz) = E(cx,cy) + cz O(cx,cy) + (cz^2 - 1/3) Qq(cx,cy)          (Eq. 7-10, 14)
//     so the source evaluates the three in-plane fields E, O, Qq (9 values each) instead of 27
//     populations, and ships E, O, Qq of the 8 moving in-plane directions through shared memory;
//   * the lattice weights are products of (1,4,1)/6 per axis, so the receiver applies them while
//     it reduces (adds become FMAs with the constant 4) and the common factor 1/216 is folded
//     into the source's constants;
//   * raw moments (Eq. 11-13) are linear in the populations, so the receiver reduces the FIELDS
//     (3 x 17 operations) and only then forms the cz = +1 / 0 / -1 combinations.
#pragma once
#include "tslb_device.cuh"
#include "tslb_tiled.cuh"

namespace tslb {

__host__ __device__ constexpr int dir_slot(int cx, int cy) {
  int q = (cy + 1) * 3 + (cx + 1);
  return q > 4 ? q - 1 : q;
}

// Exchange buffers, double buffered over the marching index so that one __syncthreads per plane
// is enough.  Per direction: (E,O) as one pair word (128 bit in fp64, 64 bit in fp32) and Qq as a
// scalar, indexed by the RECEIVER (main thread index ly TX + lx): a source writes direction
// (cx,cy) at its own index + cy TX + cx, and only if that node lies inside the tile, so ring
// cells and tile-edge cells skip the directions nobody reads; a receiver finds all 8 arrivals at
// its own index.  Every access is contiguous across the warp (no bank conflicts).
template <typename T, int CELLS, int NMAIN> struct ExBuf;
template <int CELLS, int NMAIN> struct ExBuf<double, CELLS, NMAIN> {
  double2 eo[8][NMAIN];
  double q[8][NMAIN];
  double2 pd[CELLS];      // (pz, dz) of phi^{n+1}: (phi(z-1)+phi(z+1)) + 4 phi(z),  phi(z+1) - phi(z-1)
  __device__ __forceinline__ void put(int slot, int c, double E, double O, double Q) {
    eo[slot][c] = make_double2(E, O);
    q[slot][c] = Q;
  }
  __device__ __forceinline__ void get(int slot, int c, double& E, double& O, double& Q) const {
    const double2 v = eo[slot][c];
    E = v.x; O = v.y; Q = q[slot][c];
  }
  __device__ __forceinline__ void get_eo(int slot, int c, double& E, double& O) const {
    const double2 v = eo[slot][c]; E = v.x; O = v.y;
  }
  __device__ __forceinline__ void get_q(int slot, int c, double& Q) const { Q = q[slot][c]; }
  __device__ __forceinline__ void put_pd(int c, double a, double b) { pd[c] = make_double2(a, b); }
  __device__ __forceinline__ void get_pd(int c, double& a, double& b) const {
    const double2 v = pd[c]; a = v.x; b = v.y;
  }
};
template <int CELLS, int NMAIN> struct ExBuf<float, CELLS, NMAIN> {
  float2 eo[8][NMAIN];
  float q[8][NMAIN];
  float2 pd[CELLS];
  __device__ __forceinline__ void put(int slot, int c, float E, float O, float Q) {
    eo[slot][c] = make_float2(E, O);
    q[slot][c] = Q;
  }
  __device__ __forceinline__ void get(int slot, int c, float& E, float& O, float& Q) const {
    const float2 v = eo[slot][c];
    E = v.x; O = v.y; Q = q[slot][c];
  }
  __device__ __forceinline__ void get_eo(int slot, int c, float& E, float& O) const {
    const float2 v = eo[slot][c]; E = v.x; O = v.y;
  }
  __device__ __forceinline__ void get_q(int slot, int c, float& Q) const { Q = q[slot][c]; }
  __device__ __forceinline__ void put_pd(int c, float a, float b) { pd[c] = make_float2(a, b); }
  __device__ __forceinline__ void get_pd(int c, float& a, float& b) const {
    const float2 v = pd[c]; a = v.x; b = v.y;
  }
};
template <typename T, int CELLS, int NMAIN>
struct K2FastSmem { ExBuf<T, CELLS, NMAIN> buf[2]; };

// which of the 8 in-plane directions of the ring cell (lx, ly) have their receiver inside the tile
template <int TX, int TY>
__device__ __forceinline__ unsigned dir_mask(int lx, int ly) {
  unsigned m = 0;
#pragma unroll
  for (int q = 0; q < 9; ++q) {
    const int cx = q % 3 - 1, cy = q / 3 - 1;
    if (cx == 0 && cy == 0) continue;
    const int rx = lx + cx, ry = ly + cy;
    if (rx >= 0 && rx < TX && ry >= 0 && ry < TY) m |= 1u << dir_slot(cx, cy);
  }
  return m;
}

// E, O, Qq on the 3x3 in-plane directions, index [cx+1][cy+1], all scaled by 1/216.
template <typename T> struct SrcFields { T E[3][3], O[3][3], Q[3][3]; };

template <typename T>
__device__ __forceinline__ void source_fields(const Coef<T>& c, SrcFields<T>& s) {
  const T k = T(1.0 / 216.0);
  T a0[3], a1[3], a2[3];
  {   // E = a0(cx) + cy a1(cx) + (cy^2 - 1/3) a2(cx)
    const T m0 = k * c.c0;
    a0[1] = fma(T(-1.5) * k, c.xx, m0);
    const T t = fma(T(3) * k, c.xx, m0);
    a0[0] = fma(T(-3) * k, c.c1x, t);
    a0[2] = fma(T(3) * k, c.c1x, t);
    const T m1 = (T(3) * k) * c.c1y;
    a1[1] = fma(T(-4.5) * k, c.xxy, m1);
    const T t1 = fma(T(9) * k, c.xxy, m1);
    a1[0] = fma(T(-9) * k, c.xy, t1);
    a1[2] = fma(T(9) * k, c.xy, t1);
    a2[1] = (T(4.5) * k) * c.yy;
    a2[0] = fma(T(-13.5) * k, c.xyy, a2[1]);
    a2[2] = fma(T(13.5) * k, c.xyy, a2[1]);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      s.E[i][1] = fma(T(-1.0 / 3.0), a2[i], a0[i]);
      const T te = fma(T(2.0 / 3.0), a2[i], a0[i]);
      s.E[i][0] = te - a1[i];
      s.E[i][2] = te + a1[i];
    }
  }
  {   // O = b0(cx) + cy b1(cx) + (cy^2 - 1/3) b2
    const T m0 = (T(3) * k) * c.c1z;
    a0[1] = fma(T(-4.5) * k, c.xxz, m0);
    const T t = fma(T(9) * k, c.xxz, m0);
    a0[0] = fma(T(-9) * k, c.xz, t);
    a0[2] = fma(T(9) * k, c.xz, t);
    a1[1] = (T(9) * k) * c.yz;
    a1[0] = fma(T(-27) * k, c.xyz, a1[1]);
    a1[2] = fma(T(27) * k, c.xyz, a1[1]);
    const T b2 = (T(13.5) * k) * c.yyz;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      s.O[i][1] = fma(T(-1.0 / 3.0), b2, a0[i]);
      const T to = fma(T(2.0 / 3.0), b2, a0[i]);
      s.O[i][0] = to - a1[i];
      s.O[i][2] = to + a1[i];
    }
  }
  {   // Qq = d0(cx) + cy d1
    a0[1] = (T(4.5) * k) * c.zz;
    a0[0] = fma(T(-13.5) * k, c.xzz, a0[1]);
    a0[2] = fma(T(13.5) * k, c.xzz, a0[1]);
    const T d1 = (T(13.5) * k) * c.yzz;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      s.Q[i][1] = a0[i];
      s.Q[i][0] = a0[i] - d1;
      s.Q[i][2] = a0[i] + d1;
    }
  }
}

__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) {      // a - b, one rounding
  return __ffma2_rn(b, make_float2(-1.f, -1.f), a);
}
__device__ __forceinline__ float2 fma4(float2 v, float2 r) {      // 4 v + r
  return __ffma2_rn(make_float2(4.f, 4.f), v, r);
}

// fp32: the E and the O polynomial have the same shape (O's lower-order rows are E's with some
// coefficients zero), so they are evaluated as the two lanes of packed fp32x2 instructions; a lane
// that has no term there multiplies by 0 (fma(0, x, m) = m exactly), so every component is rounded
// exactly as in the scalar sequence above.
__device__ __forceinline__ void source_fields(const Coef<float>& c, SrcFields<float>& s) {
  const float k = float(1.0 / 216.0);
  auto f2 = [](float a, float b) { return make_float2(a, b); };
  float2 A0[3], A1[3], A2[3];                     // lanes: (E's a_n(cx), O's b_n(cx))
  {
    const float2 base = __fmul2_rn(f2(k, 3.f * k), f2(c.c0, c.c1z));
    const float2 q = f2(c.xx, c.xxz), l = f2(c.c1x, c.xz);
    A0[1] = __ffma2_rn(f2(-1.5f * k, -4.5f * k), q, base);
    const float2 t = __ffma2_rn(f2(3.f * k, 9.f * k), q, base);
    A0[0] = __ffma2_rn(f2(-3.f * k, -9.f * k), l, t);
    A0[2] = __ffma2_rn(f2(3.f * k, 9.f * k), l, t);
  }
  {
    const float2 m1 = __fmul2_rn(f2(3.f * k, 9.f * k), f2(c.c1y, c.yz));
    const float2 q = f2(c.xxy, 0.f), l = f2(c.xy, c.xyz);
    A1[1] = __ffma2_rn(f2(-4.5f * k, 0.f), q, m1);
    const float2 t1 = __ffma2_rn(f2(9.f * k, 0.f), q, m1);
    A1[0] = __ffma2_rn(f2(-9.f * k, -27.f * k), l, t1);
    A1[2] = __ffma2_rn(f2(9.f * k, 27.f * k), l, t1);
  }
  {
    A2[1] = __fmul2_rn(f2(4.5f * k, 13.5f * k), f2(c.yy, c.yyz));
    const float2 q = f2(c.xyy, 0.f);
    A2[0] = __ffma2_rn(f2(-13.5f * k, 0.f), q, A2[1]);
    A2[2] = __ffma2_rn(f2(13.5f * k, 0.f), q, A2[1]);
  }
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    const float2 mid = __ffma2_rn(f2(float(-1.0 / 3.0), float(-1.0 / 3.0)), A2[i], A0[i]);
    const float2 te = __ffma2_rn(f2(float(2.0 / 3.0), float(2.0 / 3.0)), A2[i], A0[i]);
    const float2 lo = sub2(te, A1[i]), hi = add2(te, A1[i]);
    s.E[i][1] = mid.x; s.O[i][1] = mid.y;
    s.E[i][0] = lo.x; s.O[i][0] = lo.y;
    s.E[i][2] = hi.x; s.O[i][2] = hi.y;
  }
  {   // Qq = d0(cx) + cy d1 (scalar)
    float a0[3];
    a0[1] = (4.5f * k) * c.zz;
    a0[0] = fmaf(-13.5f * k, c.xzz, a0[1]);
    a0[2] = fmaf(13.5f * k, c.xzz, a0[1]);
    const float d1 = (13.5f * k) * c.yzz;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
      s.Q[i][1] = a0[i];
      s.Q[i][0] = a0[i] - d1;
      s.Q[i][2] = a0[i] + d1;
    }
  }
}

// In-plane moments {1, x, y, xx, yy, xy} of a field given on the 3x3 arrival directions, with the
// lattice weights (1,4,1) (x) (1,4,1) (the factor 1/36 lives in the source constants).
template <typename T> struct Red6 { T s1, sx, sy, sxx, syy, sxy; };

template <typename T>
__device__ __forceinline__ Red6<T> reduce6(const T (&v)[3][3]) {   // v[cx+1][cy+1]
  T r0[3], r1[3], r2[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r2[i] = v[i][2] + v[i][0];
    r1[i] = v[i][2] - v[i][0];
    r0[i] = fma(T(4), v[i][1], r2[i]);
  }
  Red6<T> r;
  r.sxx = r0[2] + r0[0];
  r.sx = r0[2] - r0[0];
  r.s1 = fma(T(4), r0[1], r.sxx);
  r.sxy = r1[2] - r1[0];
  r.sy = fma(T(4), r1[1], r1[2] + r1[0]);
  r.syy = fma(T(4), r2[1], r2[2] + r2[0]);
  return r;
}

// Receiver side, fields E and O: gather the 8 arrivals, add the own resting direction, reduce both
// to their six in-plane moments.  fp32: E and O travel as one float2 and the two reductions are
// the same operation sequence on independent data, so they run as ONE sequence of packed
// fp32x2 instructions (fma.rn.f32x2 / add.f32x2, sm_100: per component the same rounding as the
// scalar ones, half the issue slots; K2 fp32 is issue-bound, profiles/r2_kernels_f32.txt).
template <typename T, typename XB>
__device__ __forceinline__ void receive_eo(const XB& xb, int tid, T ownE, T ownO, Red6<T>& rE,
                                           Red6<T>& rO) {
  T vE[3][3], vO[3][3];
  vE[1][1] = ownE; vO[1][1] = ownO;
#pragma unroll
  for (int q = 0; q < 9; ++q) {
    const int cx = q % 3 - 1, cy = q / 3 - 1;
    if (cx == 0 && cy == 0) continue;
    xb.get_eo(dir_slot(cx, cy), tid, vE[cx + 1][cy + 1], vO[cx + 1][cy + 1]);
  }
  rE = reduce6(vE);
  rO = reduce6(vO);
}
template <typename XB>
__device__ __forceinline__ void receive_eo(const XB& xb, int tid, float ownE, float ownO,
                                           Red6<float>& rE, Red6<float>& rO) {
  float2 v[3][3];
  v[1][1] = make_float2(ownE, ownO);
#pragma unroll
  for (int q = 0; q < 9; ++q) {
    const int cx = q % 3 - 1, cy = q / 3 - 1;
    if (cx == 0 && cy == 0) continue;
    v[cx + 1][cy + 1] = xb.eo[dir_slot(cx, cy)][tid];
  }
  float2 r0[3], r1[3], r2[3];                      // the operation order of reduce6, two lanes
#pragma unroll
  for (int i = 0; i < 3; ++i) {
    r2[i] = add2(v[i][2], v[i][0]);
    r1[i] = sub2(v[i][2], v[i][0]);
    r0[i] = fma4(v[i][1], r2[i]);
  }
  const float2 sxx = add2(r0[2], r0[0]);
  const float2 sx = sub2(r0[2], r0[0]);
  const float2 s1 = fma4(r0[1], sxx);
  const float2 sxy = sub2(r1[2], r1[0]);
  const float2 sy = fma4(r1[1], add2(r1[2], r1[0]));
  const float2 syy = fma4(r2[1], add2(r2[2], r2[0]));
  rE.s1 = s1.x; rE.sx = sx.x; rE.sy = sy.x; rE.sxx = sxx.x; rE.syy = syy.x; rE.sxy = sxy.x;
  rO.s1 = s1.y; rO.sx = sx.y; rO.sy = sy.y; rO.sxx = sxx.y; rO.syy = syy.y; rO.sxy = sxy.y;
}

// Source plane of marching index j in [-1, nz]: periodic wrap, or (walls at z = 0 / top, R19) the
// evenly mirrored plane: -1 -> 0, nz -> nz-1.
__device__ __forceinline__ int source_plane(int j, int nz, int bcz) {
  if (j < 0) return bcz ? -1 - j : j + nz;
  if (j >= nz) return bcz ? 2 * nz - 1 - j : j - nz;
  return j;
}

// A source node publishes E, O, Qq of its 8 moving in-plane directions at the receivers' indices
// and keeps the resting direction in registers.
// Walls on the marching axis (halfway bounce-back, R19: f_c(x) = fpost_{-c}(x) when x - c lies
// beyond the wall): a GHOST source plane (j = -1 or nz, loaded from the mirrored plane 0 / nz-1)
// sends nothing across; every node of the wall plane instead receives ITS OWN populations
// reversed: the arrival with in-plane direction a and vertical direction cz is
//   P_own(-a, -cz) = E_own(-a) - cz O_own(-a) + (cz^2 - 1/3) Qq_own(-a),
// i.e. the fields (E_own(-a), -O_own(-a), Qq_own(-a)) in the node's own receiver slots.  The
// receiver code is the same in both cases: the ghost plane's cz = +1 combination lands on plane 0,
// its cz = -1 combination on plane nz-1, and the rest falls on planes that do not exist.
template <typename T, int TX, int TY, typename XB>
__device__ __forceinline__ void publish(XB& xb, const SrcFields<T>& sf, bool ghost, bool is_main,
                                        unsigned need, int rb, T& ownE, T& ownO, T& ownQ,
                                        unsigned wmask = 0u) {
  if (!ghost) {
    ownE = sf.E[1][1]; ownO = sf.O[1][1]; ownQ = sf.Q[1][1];
#pragma unroll
    for (int q = 0; q < 9; ++q) {
      const int cx = q % 3 - 1, cy = q / 3 - 1;
      if (cx == 0 && cy == 0) continue;
      if (need >> dir_slot(cx, cy) & 1u)
        xb.put(dir_slot(cx, cy), rb + cy * TX + cx, sf.E[cx + 1][cy + 1], sf.O[cx + 1][cy + 1], sf.Q[cx + 1][cy + 1]);
    }
  } else if (is_main) {
    ownE = sf.E[1][1]; ownO = -sf.O[1][1]; ownQ = sf.Q[1][1];
#pragma unroll
    for (int q = 0; q < 9; ++q) {
      const int cx = q % 3 - 1, cy = q / 3 - 1;
      if (cx == 0 && cy == 0) continue;
      if (wmask >> dir_slot(cx, cy) & 1u) continue;      // owned by the in-plane wall accounting
      xb.put(dir_slot(cx, cy), rb, sf.E[1 - cx][1 - cy], -sf.O[1 - cx][1 - cy], sf.Q[1 - cx][1 - cy]);
    }
  }
}

// Walls on the TILE axes x, y (halfway bounce-back, R19).  A receiver r next to such a wall has
// in-plane arrival directions a whose source r - a lies beyond the wall (bit dir_slot(a) of
// wmask).  For those, all three vertical directions bounce: the arrival (a, cz) at plane k is the
// node's own fpost(-a, -cz) of plane k, i.e. the fields (E(-a), -O(-a), Qq(-a)) of the node's OWN
// plane-k source evaluation -- not distributed over planes k-1, k, k+1 like a neighbour's, but
// all three landing on plane k.  Summed over cz with the lattice weights (1, 4, 1):
//   in-plane moments {1,x,y,xx,yy,xy}: 6 red(E')        (the Qq parts cancel: 2/3 - 4/3 + 2/3 = 0)
//   mz, xz, yz: 2 red(O').{1,x,y}        zz: 2 red(E' + 2/3 Qq').1
// which is added to the accumulators of plane k when the node's own fields of plane k exist
// (iteration j = k, before the barrier).  The receiver slots of those directions are zeroed once
// and never written by anybody, so the regular reduction adds nothing for them.
template <typename T>
__device__ __forceinline__ void wall_bounce(const SrcFields<T>& sf, unsigned wmask, T (&aB)[6],
                                            T (&zB)[3], T& zcB) {
  T bE[3][3], bO[3][3], bQ[3][3];
#pragma unroll
  for (int q = 0; q < 9; ++q) {
    const int cx = q % 3 - 1, cy = q / 3 - 1;
    const bool on = (cx != 0 || cy != 0) && (wmask >> dir_slot(cx, cy) & 1u);
    bE[cx + 1][cy + 1] = on ? sf.E[1 - cx][1 - cy] : T(0);
    bO[cx + 1][cy + 1] = on ? -sf.O[1 - cx][1 - cy] : T(0);
    bQ[cx + 1][cy + 1] = on ? sf.Q[1 - cx][1 - cy] : T(0);
  }
  const Red6<T> e = reduce6(bE), o = reduce6(bO), qq = reduce6(bQ);
  aB[0] = fma(T(6), e.s1, aB[0]);   aB[1] = fma(T(6), e.sx, aB[1]);   aB[2] = fma(T(6), e.sy, aB[2]);
  aB[3] = fma(T(6), e.sxx, aB[3]);  aB[4] = fma(T(6), e.syy, aB[4]);  aB[5] = fma(T(6), e.sxy, aB[5]);
  zB[0] = fma(T(2), o.s1, zB[0]);   zB[1] = fma(T(2), o.sx, zB[1]);   zB[2] = fma(T(2), o.sy, zB[2]);
  zcB += T(2) * (fma(T(2.0 / 3.0), qq.s1, e.s1) - o.s1);
}

// mirrored (wall) or wrapped (periodic) index of a ring coordinate g in [-1, n]
__device__ __forceinline__ int ring_source(int g, int n, int bc) {
  if (g < 0) return bc ? -1 - g : g + n;
  if (g >= n) return bc ? 2 * n - 1 - g : g - n;
  return g;
}

// cp.async staging NSTAGE >= 1 planes ahead: each thread copies the 14 scalars of ITS OWN node
// for plane j + NSTAGE straight into a private shared-memory slot (StageBuf, tslb_device.cuh)
// and picks them up NSTAGE iterations later; only cp.async.wait_group is needed.
// WXY: walls on x or y are possible (wall_bounce); false compiles the accounting out so that the
// all-periodic instantiations keep their registers
template <typename T, int TX, int TY, int MINB, int NSTAGE, bool WXY = false>
__global__ void __launch_bounds__((TileMap<TX, TY, 1>::NTHREADS), MINB)
k_stream_collide_fast(DevParams<T> P, const T* __restrict__ S, T* __restrict__ D,
                      T* __restrict__ Qout, int zchunk) {
  static_assert(NSTAGE >= 1, "the kernel is latency-bound without staging");
  using M = TileMap<TX, TY, 1>;
  using SM = K2FastSmem<T, M::CELLS, M::NMAIN>;
  using XB = ExBuf<T, M::CELLS, M::NMAIN>;
  using STG = StageBuf<T, M::CELLS>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  STG* stg = reinterpret_cast<STG*>(smem_raw + sizeof(SM));      // NSTAGE slots

  const int tid = threadIdx.x;
  int lx, ly;
  const bool mapped = M::coords(tid, lx, ly);
  const int gx = blockIdx.x * TX + lx, gy = blockIdx.y * TY + ly;
  const int z0 = P.zbeg + blockIdx.z * zchunk;
  const int z1 = min(P.zend, z0 + zchunk);
  const int c = M::cell(lx, ly);
  const int rb = ly * TX + lx;                                  // index as a receiver (main: tid)
  const bool in_ring = mapped && gx >= -1 && gx <= P.nx && gy >= -1 && gy <= P.ny;
  const bool is_out = tid < M::NMAIN && gx < P.nx && gy < P.ny;
  // a ring cell beyond a wall of the tile axes is no source: it only supplies the mirrored
  // phi^{n+1} ghost (R19); every other ring cell is the periodic image
  const bool beyond = WXY && ((P.bcx && (gx < 0 || gx >= P.nx)) || (P.bcy && (gy < 0 || gy >= P.ny)));
  const unsigned need = (mapped && !beyond) ? dir_mask<TX, TY>(lx, ly) : 0u;   // directions somebody reads
  const int sx = ring_source(gx, P.nx, WXY ? P.bcx : 0);
  const int sy = ring_source(gy, P.ny, WXY ? P.bcy : 0);
  const int plane = P.nx * P.ny;
  const int col = in_ring ? sx + P.nx * sy : 0;
  const T* phin = D + F_PHI * P.N;
  // receiver's in-plane arrival directions whose source lies beyond a wall (wall_bounce)
  unsigned wmask = 0u;
  if (WXY && is_out && (P.bcx || P.bcy)) {
#pragma unroll
    for (int q = 0; q < 9; ++q) {
      const int cx = q % 3 - 1, cy = q / 3 - 1;
      if (cx == 0 && cy == 0) continue;
      const bool out = (P.bcx && ((cx == 1 && gx == 0) || (cx == -1 && gx == P.nx - 1))) ||
                       (P.bcy && ((cy == 1 && gy == 0) || (cy == -1 && gy == P.ny - 1)));
      if (out) {
        wmask |= 1u << dir_slot(cx, cy);
        sm.buf[0].put(dir_slot(cx, cy), tid, T(0), T(0), T(0));     // nobody else writes these
        sm.buf[1].put(dir_slot(cx, cy), tid, T(0), T(0), T(0));
      }
    }
  }

  // cp.async pipeline: one commit group per plane, issued by every thread (possibly empty)
  auto stage_issue = [&](int j, int slot) {
    if (in_ring && j <= z1) {
      using V = typename VecOf<T>::type;
      const int jz = source_plane(j, P.nz, P.bcz);
      const int s = col + plane * jz;
      const V* g = reinterpret_cast<const V*>(S);
#pragma unroll
      for (int k = 0; k < 12 / VecOf<T>::W; ++k) cp_async16(&stg[slot].vec[k][c], g + k * P.N + s);
      cp_async_small(&stg[slot].az[c], S + 12 * P.N + s);
      cp_async_small(&stg[slot].ph[c], phin + s);
    }
    cp_async_commit();
  };
  auto stage_take = [&](int slot, T (&m)[13], T& ph) {
    constexpr int W = VecOf<T>::W;
#pragma unroll
    for (int k = 0; k < 12 / W; ++k) unpack(stg[slot].vec[k][c], &m[k * W]);
    m[12] = stg[slot].az[c];
    ph = stg[slot].ph[c];
  };
#pragma unroll
  for (int d = 0; d < NSTAGE; ++d) stage_issue(z0 - 1 + d, d);

  // Register pipeline along z.  Two slots alternate roles every plane ("A" = destination plane
  // j-1, completed in iteration j; "B" = destination plane j), so the marching loop is unrolled
  // by two and no register is moved to shift the pipeline.
  T acc0[6] = {}, acc1[6] = {}, zo0[3] = {}, zo1[3] = {}, u0[3] = {}, u1[3] = {};
  T zc0 = 0, zc1 = 0;                          // zz of the in-plane wall bounce (wall_bounce)
  T ph_m = 0, ph_0 = 0, ph_p = 0;

  auto body = [&](const int j, const int slot, XB& xb, T (&aA)[6], T (&aB)[6],
                  T (&zA)[3], T (&zB)[3], T& zcA, T& zcB, const T (&uPrev)[3], T (&uCur)[3]) {
    T ownE = 0, ownO = 0, ownQ = 0;
    ph_m = ph_0; ph_0 = ph_p;
    if (in_ring) {
      T cur[13];
      cp_async_wait<NSTAGE - 1>();                             // the group of plane j has landed
      stage_take(slot, cur, ph_p);
      uCur[0] = cur[F_UX]; uCur[1] = cur[F_UY]; uCur[2] = cur[F_UZ];
      SrcFields<T> sf;
      const Coef<T> cf = coef_from13(cur);
      source_fields(cf, sf);
      const bool ghost = P.bcz && (j < 0 || j >= P.nz);
      publish<T, TX, TY>(xb, sf, ghost, tid < M::NMAIN, need, rb, ownE, ownO, ownQ, wmask);
      if (WXY && wmask != 0u && !ghost) wall_bounce(sf, wmask, aB, zB, zcB);
      xb.put_pd(c, fma(T(4), ph_0, ph_m + ph_p), ph_p - ph_m);
    }
    stage_issue(j + NSTAGE, slot);             // refill the slot just consumed
    __syncthreads();

    if (is_out) {
      Red6<T> rE, rO, rQ;
      receive_eo(xb, tid, ownE, ownO, rE, rO);
      if (sizeof(T) == 8) asm volatile("" ::: "memory");   // keep the Qq loads behind the E/O work
      {
        T vQ[3][3];
        vQ[1][1] = ownQ;
#pragma unroll
        for (int q = 0; q < 9; ++q) {
          const int cx = q % 3 - 1, cy = q / 3 - 1;
          if (cx == 0 && cy == 0) continue;
          xb.get_q(dir_slot(cx, cy), tid, vQ[cx + 1][cy + 1]);
        }
        rQ = reduce6(vQ);
      }
      const T e[6] = {rE.s1, rE.sx, rE.sy, rE.sxx, rE.syy, rE.sxy};
      const T o[6] = {rO.s1, rO.sx, rO.sy, rO.sxx, rO.syy, rO.sxy};
      const T qq[6] = {rQ.s1, rQ.sx, rQ.sy, rQ.sxx, rQ.syy, rQ.sxy};
      T up[6], dn[3];
#pragma unroll
      for (int i = 0; i < 6; ++i) {
        const T t = fma(T(2.0 / 3.0), qq[i], e[i]);          // cz = +-1 : E + (2/3) Qq +- O
        up[i] = t + o[i];
        const T d = t - o[i];
        if (i < 3) dn[i] = d;
        aA[i] += d;                                          // arrives at plane j-1
        aB[i] += fma(T(-4.0 / 3.0), qq[i], T(4) * e[i]);     // cz = 0 : 4 (E - Qq/3)
      }
      const int k = j - 1;
      if (k >= z0) {
        Mom<T> m;
        m.p = aA[0]; m.mx = aA[1]; m.my = aA[2];
        m.xx = aA[3]; m.yy = aA[4]; m.xy = aA[5];
        m.mz = zA[0] - dn[0]; m.xz = zA[1] - dn[1]; m.yz = zA[2] - dn[2];
        m.zz = zA[0] + dn[0];
        if (WXY) m.zz += zcA;
        if (sizeof(T) == 8) asm volatile("" ::: "memory");
        // separable gradient / Laplacian of phi^{n+1} at plane k (Eq. 18, repaired Eq. 19)
        T rs[3], rd[3], zs[3];
#pragma unroll
        for (int r = 0; r < 3; ++r) {
          const int cc = c + (r - 1) * M::W;
          T am, a0, ap, bm, b0, bp;
          xb.get_pd(cc - 1, am, bm);
          xb.get_pd(cc, a0, b0);
          xb.get_pd(cc + 1, ap, bp);
          rs[r] = fma(T(4), a0, am + ap);
          rd[r] = ap - am;
          zs[r] = fma(T(4), b0, bm + bp);
        }
        const T sw = fma(T(4), rs[1], rs[0] + rs[2]);
        const T gx_ = fma(T(4), rd[1], rd[0] + rd[2]) * T(3.0 / 216.0);
        const T gy_ = (rs[2] - rs[0]) * T(3.0 / 216.0);
        const T gz_ = fma(T(4), zs[1], zs[0] + zs[2]) * T(3.0 / 216.0);
        const T lap = T(6.0 / 216.0) * fma(T(-216), ph_0, sw);   // difference form: 0 on constants
        const NodeOut<T> out = close_node(P, m, ph_0, gx_, gy_, gz_, lap, uPrev[0], uPrev[1], uPrev[2]);
        const long long idx = gx + P.nx * gy + (long long)plane * k;
        store_out(D, P.N, idx, out);
        if (Qout != nullptr) {                      // flux of Eq. 20 for the next step (K1 flux form)
          T q[3];
          flux_q(P, ph_0, gx_, gy_, gz_, out.ux, out.uy, out.uz, q);
          store_q(Qout, P.N, idx, q);
        }
      }
      // slot A is free now: it becomes the accumulator of destination plane j+1
#pragma unroll
      for (int i = 0; i < 6; ++i) aA[i] = up[i];
#pragma unroll
      for (int i = 0; i < 3; ++i) zA[i] = up[i];
      zcA = T(0);
    }
  };

  int slot = 0;                                 // staging slot of plane j: (j - z0 + 1) % NSTAGE
  auto next_slot = [&]() { if (NSTAGE > 1) slot = (slot + 1 == NSTAGE) ? 0 : slot + 1; };
  for (int j = z0 - 1; j <= z1; j += 2) {
    body(j, slot, sm.buf[0], acc0, acc1, zo0, zo1, zc0, zc1, u0, u1);
    next_slot();
    if (j + 1 <= z1) {
      body(j + 1, slot, sm.buf[1], acc1, acc0, zo1, zo0, zc1, zc0, u1, u0);
      next_slot();
    }
  }
  cp_async_wait<0>();
}

}  // namespace tslb
