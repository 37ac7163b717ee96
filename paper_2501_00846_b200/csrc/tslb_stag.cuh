// tslb_stag.cuh -- lean periodic stream-collide kernel with STAGGERED warp groups.
//
// Same arithmetic and exchange format as tslb_fast.cuh.  The difference is the schedule inside
// a thread block.  One marching iteration j consists of two pieces of work per thread,
//     S(j)   : "source"  -- reconstruct the fields of the own node at plane j and publish them,
//     R(j-1) : "receive" -- gather the fields published for plane j-1, finish destination plane
//                           j-2 (moments, forces, closing) and store it,
// which are independent of each other.  The main warps are split in two groups that run the two
// pieces in opposite order, with a block barrier between the pieces:
//     group A :  S(j)    | barrier |  R(j-1)  | barrier
//     group B :  R(j-1)  | barrier |  S(j)    | barrier        (halo warps: S(j) with group B)
// so at any time half of the main warps stream shared-memory reads into FP work while the other
// half computes polynomials and issues shared-memory writes: the L1/shared data pipe and the FP
// pipe are both busy in both halves of the iteration instead of taking turns.
// Hazards: buffer j&1 is written during iteration j and read during iteration j+1; every read
// of S(j-1) comes after the barrier that ends iteration j-1.
#pragma once
#include "tslb_fast.cuh"

namespace tslb {

template <typename T, int TX, int TY, int MINB, int NSTAGE = 0>
__global__ void __launch_bounds__((TileMap<TX, TY, 1>::NTHREADS), MINB)
k_stream_collide_stag(DevParams<T> P, const T* __restrict__ S, T* __restrict__ D,
                      T* __restrict__ Qout, int zchunk) {
  using M = TileMap<TX, TY, 1>;
  using SM = K2FastSmem<T, M::CELLS>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  SM& sm = *reinterpret_cast<SM*>(smem_raw);
  StageBuf<T, M::CELLS>& stg = *reinterpret_cast<StageBuf<T, M::CELLS>*>(smem_raw + sizeof(SM));

  const int tid = threadIdx.x;
  int lx, ly;
  const bool mapped = M::coords(tid, lx, ly);
  const int gx = blockIdx.x * TX + lx, gy = blockIdx.y * TY + ly;
  const int z0 = blockIdx.z * zchunk;
  const int z1 = min(P.nz, z0 + zchunk);
  const int c = M::cell(lx, ly);
  const bool in_ring = mapped && gx >= -1 && gx <= P.nx && gy >= -1 && gy <= P.ny;
  const bool is_out = tid < M::NMAIN && gx < P.nx && gy < P.ny;
  const bool group_a = tid < M::NMAIN / 2;           // warp-uniform: rows 0 .. TY/2-1
  const int sx = gx < 0 ? gx + P.nx : (gx >= P.nx ? gx - P.nx : gx);      // periodic wrap
  const int sy = gy < 0 ? gy + P.ny : (gy >= P.ny ? gy - P.ny : gy);
  const int plane = P.nx * P.ny;
  const int col = in_ring ? sx + P.nx * sy : 0;
  const T* phin = D + F_PHI * P.N;

  // z pipeline of the receive side: two accumulator slots that swap roles every plane
  T acc0[6] = {}, acc1[6] = {}, zo0[3] = {}, zo1[3] = {};
  // carried from S to R: phi^{n+1}, u^n and the own (0,0)-direction fields of recent planes
  T ph_a = 0, ph_b = 0, ph_c = 0;                    // phi^{n+1} at planes s-2, s-1, s (s = last S)
  T u_b[3] = {}, u_c[3] = {}, u_a[3] = {};           // u^n at planes s-2 (a), s-1 (b), s (c)
  T own_c[3] = {}, own_b[3] = {};                    // E,O,Qq(0,0) of planes s (c) and s-1 (b)
  T nxt[13], nxt_phi = 0;                            // prefetched state of the next source plane

  auto load_plane = [&](int j, T (&m)[13], T& ph) {
    const int jz = j < 0 ? j + P.nz : (j >= P.nz ? j - P.nz : j);
    const int s = col + plane * jz;
    load13(S, P.N, s, m);
    ph = __ldg(phin + s);
  };
  auto stage_issue = [&](int j) {
    if (in_ring && j <= z1) {
      using V = typename VecOf<T>::type;
      const int jz = j < 0 ? j + P.nz : (j >= P.nz ? j - P.nz : j);
      const int s = col + plane * jz;
      const V* g = reinterpret_cast<const V*>(S);
#pragma unroll
      for (int k = 0; k < 12 / VecOf<T>::W; ++k) cp_async16(&stg.vec[k][c], g + k * P.N + s);
      cp_async_small(&stg.az[c], S + 12 * P.N + s);
      cp_async_small(&stg.ph[c], phin + s);
    }
    cp_async_commit();
  };
  if (NSTAGE > 0) stage_issue(z0 - 1);
  else if (in_ring) load_plane(z0 - 1, nxt, nxt_phi);

  // ---- S(j): publish plane j into buffer xb, prefetch plane j+1
  auto source = [&](const int j, ExBuf<T, M::CELLS>& xb) {
    ph_a = ph_b; ph_b = ph_c;
#pragma unroll
    for (int i = 0; i < 3; ++i) { u_a[i] = u_b[i]; u_b[i] = u_c[i]; own_b[i] = own_c[i]; }
    if (NSTAGE > 0) cp_async_wait<0>();
    T cur[13];
    if (in_ring) {
      if (NSTAGE > 0) {
        constexpr int W = VecOf<T>::W;
#pragma unroll
        for (int k = 0; k < 12 / W; ++k) unpack(stg.vec[k][c], &cur[k * W]);
        cur[12] = stg.az[c];
        ph_c = stg.ph[c];
      } else {
#pragma unroll
        for (int f = 0; f < 13; ++f) cur[f] = nxt[f];
        ph_c = nxt_phi;
        if (j < z1) load_plane(j + 1, nxt, nxt_phi);
      }
    }
    if (NSTAGE > 0) stage_issue(j + 1);
    if (in_ring) {
      u_c[0] = cur[F_UX]; u_c[1] = cur[F_UY]; u_c[2] = cur[F_UZ];
      const Coef<T> cf = coef_from13(cur);
      SrcFields<T> sf;
      source_fields(cf, sf);
      own_c[0] = sf.E[1][1]; own_c[1] = sf.O[1][1]; own_c[2] = sf.Q[1][1];
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        if (cx == 0 && cy == 0) continue;
        xb.put(dir_slot(cx, cy), c, sf.E[cx + 1][cy + 1], sf.O[cx + 1][cy + 1], sf.Q[cx + 1][cy + 1]);
      }
      xb.put_pd(c, fma(T(4), ph_b, ph_a + ph_c), ph_c - ph_a);    // combos for plane j-1
    }
  };

  // ---- R(jr): gather plane jr from xb, finish destination plane jr-1.
  //      own = E,O,Qq(0,0) of plane jr ; phk, uk = phi^{n+1}, u^n of the own node at plane jr-1
  auto receive = [&](const int jr, const ExBuf<T, M::CELLS>& xb, T (&aA)[6], T (&aB)[6],
                     T (&zA)[3], const T (&own)[3], const T phk, const T (&uk)[3]) {
    Red6<T> rE, rO, rQ;
    {
      T vE[3][3], vO[3][3];
      vE[1][1] = own[0]; vO[1][1] = own[1];
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        if (cx == 0 && cy == 0) continue;
        xb.get_eo(dir_slot(cx, cy), c - cy * M::W - cx, vE[cx + 1][cy + 1], vO[cx + 1][cy + 1]);
      }
      rE = reduce6(vE);
      rO = reduce6(vO);
    }
    if (sizeof(T) == 8) asm volatile("" ::: "memory");
    {
      T vQ[3][3];
      vQ[1][1] = own[2];
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        if (cx == 0 && cy == 0) continue;
        xb.get_q(dir_slot(cx, cy), c - cy * M::W - cx, vQ[cx + 1][cy + 1]);
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
      aA[i] += d;                                          // arrives at plane jr-1
      aB[i] += fma(T(-4.0 / 3.0), qq[i], T(4) * e[i]);     // cz = 0 : 4 (E - Qq/3)
    }
    const int k = jr - 1;
    if (k >= z0) {
      Mom<T> m;
      m.p = aA[0]; m.mx = aA[1]; m.my = aA[2];
      m.xx = aA[3]; m.yy = aA[4]; m.xy = aA[5];
      m.mz = zA[0] - dn[0]; m.xz = zA[1] - dn[1]; m.yz = zA[2] - dn[2];
      m.zz = zA[0] + dn[0];
      if (sizeof(T) == 8) asm volatile("" ::: "memory");
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
      const T lap = fma(T(6.0 / 216.0), sw, T(-6) * phk);
      const NodeOut<T> out = close_node(P, m, phk, gx_, gy_, gz_, lap, uk[0], uk[1], uk[2]);
      store_out(D, P.N, gx + P.nx * gy + plane * k, out);
      if (Qout != nullptr) {
        T q[3];
        flux_q(P, phk, gx_, gy_, gz_, out.ux, out.uy, out.uz, q);
        store_q(Qout, P.N, gx + P.nx * gy + plane * k, q);
      }
    }
#pragma unroll
    for (int i = 0; i < 6; ++i) aA[i] = up[i];
#pragma unroll
    for (int i = 0; i < 3; ++i) zA[i] = up[i];
  };

  // iteration j: S(j) for j <= z1, R(j-1) for j-1 >= z0-1.  Buffers by parity of the plane.
  auto iteration = [&](const int j, T (&aA)[6], T (&aB)[6], T (&zA)[3]) {
    ExBuf<T, M::CELLS>& bs = sm.buf[(j - z0 + 1) & 1];
    const ExBuf<T, M::CELLS>& br = sm.buf[(j - z0) & 1];
    const bool do_s = j <= z1, do_r = is_out && j >= z0;
    if (group_a) {
      if (do_s) source(j, bs);
      __syncthreads();
      // after S(j): planes (a,b,c) = (j-2, j-1, j); R(j-1) needs own(j-1), phi/u of plane j-2.
      // (when S(j) was skipped, j = z1+1: (a,b,c) = (j-3, j-2, j-1))
      if (do_r) {
        if (do_s) receive(j - 1, br, aA, aB, zA, own_b, ph_a, u_a);
        else receive(j - 1, br, aA, aB, zA, own_c, ph_b, u_b);
      }
      __syncthreads();
    } else {
      // before S(j): planes (a,b,c) = (j-3, j-2, j-1)
      if (do_r) receive(j - 1, br, aA, aB, zA, own_c, ph_b, u_b);
      __syncthreads();
      if (do_s) source(j, bs);
      __syncthreads();
    }
  };

  for (int j = z0 - 1; j <= z1 + 1; j += 2) {
    iteration(j, acc0, acc1, zo0);
    if (j + 1 <= z1 + 1) iteration(j + 1, acc1, acc0, zo1);
  }
  if (NSTAGE > 0) cp_async_wait<0>();
}

}  // namespace tslb
