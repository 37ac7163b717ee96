// tslb_ws.cuh -- WARP-SPECIALISED lean periodic stream-collide kernel (sm_100a).
//
// Same arithmetic as k_stream_collide_fast / _tma; different division of labour.  In those
// kernels a main thread does everything for its column (source reconstruction, exchange,
// moments, closing: ~500 instructions per plane) while the ring threads only reconstruct
// (~180) and then idle at the block barrier, and all warps run the same phase at the same time,
// so the FP pipe and the shared-memory pipe take turns instead of overlapping
// (profiles/r1b_*: issue 36 %, FP64 40 %, LSU data pipe 59 %, nothing saturated).  Here:
//   * 8 SOURCE warps reconstruct the post-collision fields E, O, Qq of all 340 ring cells
//     (Eq. 7-10, 14) from the TMA staging slot, which every thread can read, and publish them;
//   * 8 RECEIVER warps (one tile row each) gather the 8 arrivals + their own centre values,
//     reduce to raw moments (Eq. 11-13), close the node (forces, velocity, Eq. 13) and store;
//   * the two groups are decoupled by mbarriers on the double-buffered exchange (full / empty),
//     so sources work on plane j+1 while receivers finish plane j: per-plane time is the
//     maximum of the two roles, not their sum, and the pipes overlap;
//   * registers follow the roles (setmaxnreg): receivers hold the z pipeline of accumulators,
//     sources only one node at a time;
//   * lanes of the last source warp issue the TMA boxes (tslb_fast_tma.cuh), NSTAGE planes ahead.
// A source thread owns the same one or two ring cells for the whole march, so the phi history
// of a column (z-combinations of Eq. 18/19) stays in its registers.  Besides the 8 directions a
// main cell publishes a centre record for its receiver: E, O, Qq of the rest direction, u^n of
// the node (R7) and phi^{n+1} of the plane being closed.
// Requires nx % TX == 0, nx >= 2 TX, ny > TY (as the TMA staging does).
#pragma once
#include "tslb_fast_tma.cuh"

namespace tslb {

__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}

template <typename T, int CELLS, int NMAIN> struct WsBuf {
  using P2 = typename Pair2<T>::type;
  P2 eo[8][NMAIN];       // (E, O) of direction d, indexed by the receiver
  T q[8][NMAIN];         // Qq
  P2 ceo[NMAIN];         // centre record of a main cell: (E, O) of the rest direction,
  P2 cqf[NMAIN];         //   (Qq of the rest direction, phi^{n+1} of the plane being closed),
  P2 cuxy[NMAIN];        //   (ux, uy) of the source plane,
  T cuz[NMAIN];          //   uz
  P2 pd[CELLS];          // z-combinations of phi^{n+1} at the plane being closed
};

template <typename T, int TX, int TY, int NSTAGE>
struct WsSmem {
  TmaStage<T, TX, TY> stage[NSTAGE];
  WsBuf<T, TileMap<TX, TY, 1>::CELLS, TX * TY> buf[2];
  unsigned long long stage_full[NSTAGE], stage_empty[NSTAGE], ex_full[2], ex_empty[2];
};

template <typename T> struct WsRegs;     // register budgets per role (launch: 128 x 512 threads)
template <> struct WsRegs<double> { static constexpr int SRC = 104, RCV = 152; };
template <> struct WsRegs<float> { static constexpr int SRC = 104, RCV = 152; };

template <typename T, int TX, int TY, int NSTAGE>
__global__ void __launch_bounds__(512, 1)
k_stream_collide_ws(DevParams<T> P, const __grid_constant__ TmaMaps maps, T* __restrict__ D,
                    T* __restrict__ Qout, int zchunk) {
  using M = TileMap<TX, TY, 1>;
  using STG = TmaStage<T, TX, TY>;
  using XB = WsBuf<T, M::CELLS, M::NMAIN>;
  using V = typename VecOf<T>::type;
  using P2 = typename Pair2<T>::type;
  constexpr int W = VecOf<T>::W;
  constexpr int NSRC_WARPS = 8, NRCV_WARPS = 8;
  static_assert(M::NMAIN == 256, "one source thread and one receiver thread per tile node");
  extern __shared__ __align__(128) unsigned char ws_smem_raw[];
  WsSmem<T, TX, TY, NSTAGE>& sm = *reinterpret_cast<WsSmem<T, TX, TY, NSTAGE>*>(ws_smem_raw);

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int z0 = blockIdx.z * zchunk;
  const int z1 = min(P.nz, z0 + zchunk);
  const int plane = P.nx * P.ny;
  const int gx0 = blockIdx.x * TX, gy0 = blockIdx.y * TY;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) {
      mbar_init(&sm.stage_full[s], 1);
      mbar_init(&sm.stage_empty[s], NSRC_WARPS);
    }
#pragma unroll
    for (int b = 0; b < 2; ++b) {
      mbar_init(&sm.ex_full[b], NSRC_WARPS);
      mbar_init(&sm.ex_empty[b], NRCV_WARPS);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp >= NRCV_WARPS) {
    // ================================================================== source warps
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(WsRegs<T>::SRC));
    const int t = tid - 32 * NRCV_WARPS;                       // 0 .. 255
    // periodic images needed by this tile (host guarantees at most one column and one row)
    const int xw_l = gx0 == 0, xw_r = gx0 + TX == P.nx;
    const int yw_b = gy0 == 0, yw_t = gy0 + TY >= P.ny;
    const int r_w = yw_b ? 0 : P.ny - gy0 + 1;
    const bool issuer = warp == NRCV_WARPS + NSRC_WARPS - 1;
    const bool xw_any = xw_l || xw_r, yw_any = yw_b || yw_t;
    const unsigned bytes = STG::B_MAIN + (xw_any ? STG::B_WX : 0u) + (yw_any ? STG::B_WY : 0u) +
                           (xw_any && yw_any ? STG::B_WXY : 0u);

    auto produce = [&](int j, int slot) {                      // executed by the whole issuer warp
      if (j > z1) return;
      const int jz = j < 0 ? j + P.nz : (j >= P.nz ? j - P.nz : j);
      STG& st = sm.stage[slot];
      unsigned long long* bar = &sm.stage_full[slot];
      if (lane == 0) mbar_expect_tx(bar, bytes);
      __syncwarp();
      const int kind = lane / 3, what = lane % 3;              // kind: main, wx, wy, wxy
      if (lane >= 12) return;
      if (kind == 1 && !xw_any) return;
      if (kind == 2 && !yw_any) return;
      if (kind == 3 && !(xw_any && yw_any)) return;
      const bool colw = kind == 1 || kind == 3, roww = kind == 2 || kind == 3;
      const int y = roww ? (yw_b ? P.ny - 1 : 0) : gy0 - 1;
      if (what == 0) {
        const int x = (colw ? (xw_l ? P.nx - 1 : 0) : gx0 - 1) * W;
        void* dst = kind == 0 ? (void*)&st.vec[0][0] : kind == 1 ? (void*)&st.vwx[0][0]
                  : kind == 2 ? (void*)&st.vwy[0][0] : (void*)&st.vwxy[0];
        tma_load_4d(dst, &maps.vec[kind], x, y, jz, 0, bar);
      } else {
        const int x = colw ? (xw_l ? P.nx - STG::PAD : 0) : gx0 - STG::PAD;
        void* dst;
        if (what == 1)
          dst = kind == 0 ? (void*)&st.az[0][0] : kind == 1 ? (void*)&st.azx[0][0]
              : kind == 2 ? (void*)&st.azy[0] : (void*)&st.azxy[0];
        else
          dst = kind == 0 ? (void*)&st.ph[0][0] : kind == 1 ? (void*)&st.phx[0][0]
              : kind == 2 ? (void*)&st.phy[0] : (void*)&st.phxy[0];
        tma_load_3d(dst, what == 1 ? &maps.az[kind] : &maps.ph[kind], x, y, jz, bar);
      }
    };

    // the one or two ring cells of this thread: cell A = main node t, cell B = halo cell t
    struct Cell { unsigned voff, vstride, azoff, phoff, need; int c, rb; bool on; };
    auto make_cell = [&](int idx, bool exists) {
      Cell k;
      int lx = 0, ly = 0;
      const bool mapped = exists && M::coords(idx, lx, ly);
      const int gy = gy0 + ly;
      k.on = mapped && gy >= -1 && gy <= P.ny;
      k.c = M::cell(lx, ly);
      k.rb = ly * TX + lx;
      k.need = k.on ? dir_mask<TX, TY>(lx, ly) : 0u;
      const bool xw = (lx == -1 && xw_l) || (lx == TX && xw_r);
      const bool yw = yw_any && ly + 1 == r_w;
      const int r = ly + 1, xa = lx == -1 ? STG::PAD - 1 : 0;
      if (!xw && !yw) {
        k.voff = offsetof(STG, vec) + k.c * 16; k.vstride = M::CELLS * 16;
        k.azoff = offsetof(STG, az) + (r * STG::PITCH + lx + STG::PAD) * sizeof(T);
        k.phoff = offsetof(STG, ph) + (r * STG::PITCH + lx + STG::PAD) * sizeof(T);
      } else if (xw && !yw) {
        k.voff = offsetof(STG, vwx) + r * 16; k.vstride = M::HT * 16;
        k.azoff = offsetof(STG, azx) + (r * STG::PAD + xa) * sizeof(T);
        k.phoff = offsetof(STG, phx) + (r * STG::PAD + xa) * sizeof(T);
      } else if (!xw && yw) {
        k.voff = offsetof(STG, vwy) + (lx + 1) * 16; k.vstride = M::W * 16;
        k.azoff = offsetof(STG, azy) + (lx + STG::PAD) * sizeof(T);
        k.phoff = offsetof(STG, phy) + (lx + STG::PAD) * sizeof(T);
      } else {
        k.voff = offsetof(STG, vwxy); k.vstride = 16;
        k.azoff = offsetof(STG, azxy) + xa * sizeof(T);
        k.phoff = offsetof(STG, phxy) + xa * sizeof(T);
      }
      return k;
    };
    const Cell ca = make_cell(t, true);
    const bool has_b = t < M::NHALO;                           // warp-uniform up to warp 2 of 8
    const Cell cb = make_cell(M::NMAIN + t, has_b);
    T pa_m = 0, pa_0 = 0, pa_p = 0, pb_m = 0, pb_0 = 0, pb_p = 0;

    auto src_cell = [&](const Cell& k, const bool is_main, const unsigned char* sb, XB& xb,
                        T& ph_m, T& ph_0, T& ph_p) {
      ph_m = ph_0; ph_0 = ph_p;
      if (!k.on) return;
      T cur[13];
#pragma unroll
      for (int i = 0; i < STG::KV; ++i)
        unpack(*reinterpret_cast<const V*>(sb + k.voff + i * k.vstride), &cur[i * W]);
      cur[12] = *reinterpret_cast<const T*>(sb + k.azoff);
      ph_p = *reinterpret_cast<const T*>(sb + k.phoff);
      SrcFields<T> sf;
      const Coef<T> cf = coef_from13(cur);
      source_fields(cf, sf);
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        if (cx == 0 && cy == 0) continue;
        if (k.need >> dir_slot(cx, cy) & 1u) {
          P2 v; v.x = sf.E[cx + 1][cy + 1]; v.y = sf.O[cx + 1][cy + 1];
          xb.eo[dir_slot(cx, cy)][k.rb + cy * TX + cx] = v;
          xb.q[dir_slot(cx, cy)][k.rb + cy * TX + cx] = sf.Q[cx + 1][cy + 1];
        }
      }
      if (is_main) {
        P2 v;
        v.x = sf.E[1][1]; v.y = sf.O[1][1]; xb.ceo[k.rb] = v;
        v.x = sf.Q[1][1]; v.y = ph_0; xb.cqf[k.rb] = v;
        v.x = cur[F_UX]; v.y = cur[F_UY]; xb.cuxy[k.rb] = v;
        xb.cuz[k.rb] = cur[F_UZ];
      }
      P2 pdv; pdv.x = fma(T(4), ph_0, ph_m + ph_p); pdv.y = ph_p - ph_m;
      xb.pd[k.c] = pdv;
    };

    if (issuer) {
#pragma unroll
      for (int d = 0; d < NSTAGE; ++d) produce(z0 - 1 + d, d);
    }
    int slot = 0;
    unsigned spar = 0;                                         // parity of the slot's current use
    for (int j = z0 - 1; j <= z1; ++j) {
      const int n = j - (z0 - 1);
      const int b = n & 1;
      const unsigned epar = ((n >> 1) & 1) ^ 1;                // receivers done with use n/2 - 1
      mbar_wait(&sm.stage_full[slot], spar);                   // plane j has landed
      mbar_wait(&sm.ex_empty[b], epar);                        // exchange buffer b is free
      const unsigned char* sb = reinterpret_cast<const unsigned char*>(&sm.stage[slot]);
      src_cell(ca, true, sb, sm.buf[b], pa_m, pa_0, pa_p);
      if (has_b) src_cell(cb, false, sb, sm.buf[b], pb_m, pb_0, pb_p);
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(&sm.ex_full[b]);
        mbar_arrive(&sm.stage_empty[slot]);
      }
      if (issuer) {
        if (j + NSTAGE <= z1) {
          mbar_wait(&sm.stage_empty[slot], spar);              // all source warps left the slot
          produce(j + NSTAGE, slot);
        }
      }
      if (slot + 1 == NSTAGE) { slot = 0; spar ^= 1u; } else { ++slot; }
    }
    return;
  }

  // ==================================================================== receiver warps
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(WsRegs<T>::RCV));
  const int lx = tid % TX, ly = tid / TX;
  const int gx = gx0 + lx, gy = gy0 + ly;
  const int c = M::cell(lx, ly);
  const bool is_out = gy < P.ny;

  T acc0[6] = {}, acc1[6] = {}, zo0[3] = {}, zo1[3] = {}, u0[3] = {}, u1[3] = {};

  auto body = [&](const int j, XB& xb, unsigned long long* full, unsigned long long* empty,
                  const unsigned parity, T (&aA)[6], T (&aB)[6], T (&zA)[3], T (&zB)[3],
                  const T (&uPrev)[3], T (&uCur)[3]) {
    mbar_wait(full, parity);                                   // sources of plane j are published
    Red6<T> rE, rO, rQ;
    T ph_0;
    {
      T vE[3][3], vO[3][3];
      { const P2 v = xb.ceo[tid]; vE[1][1] = v.x; vO[1][1] = v.y; }
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        if (cx == 0 && cy == 0) continue;
        const P2 v = xb.eo[dir_slot(cx, cy)][tid];
        vE[cx + 1][cy + 1] = v.x; vO[cx + 1][cy + 1] = v.y;
      }
      rE = reduce6(vE);
      rO = reduce6(vO);
    }
    if (sizeof(T) == 8) asm volatile("" ::: "memory");         // keep the Qq loads behind the E/O work
    {
      T vQ[3][3];
      { const P2 v = xb.cqf[tid]; vQ[1][1] = v.x; ph_0 = v.y; }
#pragma unroll
      for (int q = 0; q < 9; ++q) {
        const int cx = q % 3 - 1, cy = q / 3 - 1;
        if (cx == 0 && cy == 0) continue;
        vQ[cx + 1][cy + 1] = xb.q[dir_slot(cx, cy)][tid];
      }
      rQ = reduce6(vQ);
    }
    { const P2 v = xb.cuxy[tid]; uCur[0] = v.x; uCur[1] = v.y; uCur[2] = xb.cuz[tid]; }
    // separable gradient / Laplacian of phi^{n+1} at plane k = j-1 (Eq. 18, repaired Eq. 19)
    T rs[3], rd[3], zs[3];
#pragma unroll
    for (int r = 0; r < 3; ++r) {
      const int cc = c + (r - 1) * M::W;
      const P2 m = xb.pd[cc - 1], o = xb.pd[cc], p = xb.pd[cc + 1];
      rs[r] = fma(T(4), o.x, m.x + p.x);
      rd[r] = p.x - m.x;
      zs[r] = fma(T(4), o.y, m.y + p.y);
    }
    // everything this warp needs from buffer b is in registers (the arrive orders behind the loads)
    __syncwarp();
    if (lane == 0) mbar_arrive(empty);

    const T e[6] = {rE.s1, rE.sx, rE.sy, rE.sxx, rE.syy, rE.sxy};
    const T o[6] = {rO.s1, rO.sx, rO.sy, rO.sxx, rO.syy, rO.sxy};
    const T qq[6] = {rQ.s1, rQ.sx, rQ.sy, rQ.sxx, rQ.syy, rQ.sxy};
    T up[6], dn[3];
#pragma unroll
    for (int i = 0; i < 6; ++i) {
      const T t = fma(T(2.0 / 3.0), qq[i], e[i]);              // cz = +-1 : E + (2/3) Qq +- O
      up[i] = t + o[i];
      const T d = t - o[i];
      if (i < 3) dn[i] = d;
      aA[i] += d;                                              // arrives at plane j-1
      aB[i] += fma(T(-4.0 / 3.0), qq[i], T(4) * e[i]);         // cz = 0 : 4 (E - Qq/3)
    }
    const int k = j - 1;
    if (k >= z0 && is_out) {
      Mom<T> m;
      m.p = aA[0]; m.mx = aA[1]; m.my = aA[2];
      m.xx = aA[3]; m.yy = aA[4]; m.xy = aA[5];
      m.mz = zA[0] - dn[0]; m.xz = zA[1] - dn[1]; m.yz = zA[2] - dn[2];
      m.zz = zA[0] + dn[0];
      const T sw = fma(T(4), rs[1], rs[0] + rs[2]);
      const T gx_ = fma(T(4), rd[1], rd[0] + rd[2]) * T(3.0 / 216.0);
      const T gy_ = (rs[2] - rs[0]) * T(3.0 / 216.0);
      const T gz_ = fma(T(4), zs[1], zs[0] + zs[2]) * T(3.0 / 216.0);
      const T lap = fma(T(6.0 / 216.0), sw, T(-6) * ph_0);
      const NodeOut<T> out = close_node(P, m, ph_0, gx_, gy_, gz_, lap, uPrev[0], uPrev[1], uPrev[2]);
      const long long idx = gx + P.nx * gy + (long long)plane * k;
      store_out(D, P.N, idx, out);
      T q[3];                                       // flux of Eq. 20 for the next step (K1 flux form)
      flux_q(P, ph_0, gx_, gy_, gz_, out.ux, out.uy, out.uz, q);
      store_q(Qout, P.N, idx, q);
    }
    // slot A is free now: it becomes the accumulator of destination plane j+1
#pragma unroll
    for (int i = 0; i < 6; ++i) aA[i] = up[i];
#pragma unroll
    for (int i = 0; i < 3; ++i) zA[i] = up[i];
  };

  unsigned par = 0;                                            // parity of use n/2 of either buffer
  for (int j = z0 - 1; j <= z1; j += 2) {
    body(j, sm.buf[0], &sm.ex_full[0], &sm.ex_empty[0], par, acc0, acc1, zo0, zo1, u0, u1);
    if (j + 1 <= z1)
      body(j + 1, sm.buf[1], &sm.ex_full[1], &sm.ex_empty[1], par, acc1, acc0, zo1, zo0, u1, u0);
    par ^= 1u;
  }
}

}  // namespace tslb
