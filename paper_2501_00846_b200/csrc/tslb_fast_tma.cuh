// tslb_fast_tma.cuh -- lean periodic stream-collide kernel with TMA tensor staging (sm_100a).
//
// Same arithmetic and exchange as k_stream_collide_fast (tslb_fast.cuh); what changes is how the
// source planes reach shared memory.  There every thread copies the 14 scalars of its own node
// with 8 cp.async instructions per plane; their shared-memory writes arrive sector by sector and
// cost about three times the ideal number of wavefronts in the LSU data pipe, which the
// population exchange already loads to ~60 % (profiles/r1_tuning_evidence.md).  Here ONE extra warp issues
// cp.async.bulk.tensor copies (TMA) for the whole ring of the tile, NSTAGE planes ahead,
// completing on an mbarrier per staging slot:
//   * one 4-d box (x, y, z, f) per 128-bit field-vector plane of the ring (6 boxes
//     in fp64; a single box for all planes is 4.5 % slower), one 3-d box each for the
//     scalar planes az and phi^{n+1} (staged with a 16-byte pad on both sides of a row so that
//     the box is 16-byte granular): 8 copies per plane for an interior tile in fp64;
//   * the parts of a box beyond the lattice are zero-filled by the TMA unit; the periodic images
//     (one column, one row, one corner cell at most) come with up to 9 small extra boxes into
//     separate arrays, and the threads of a wrapped column / row read those instead;
//   * compute threads never touch the load path: they wait on the slot's mbarrier (parity),
//     read their node, and the block barrier of the plane frees the slot for the producer warp.
// Requires nx % TX == 0, nx >= 2 TX, ny > TY; other sizes use k_stream_collide_fast.
// (A first version with non-tensor cp.async.bulk row pieces, 150-240 copies per plane, ran
// 4-5 times SLOWER than cp.async: about 37 ns per bulk copy whatever its size.)
#pragma once
#include <cstddef>

#include "tslb_fast.cuh"

namespace tslb {

__device__ __forceinline__ unsigned smem_u32(const void* p) {
  return (unsigned)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)),
               "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra WAIT_DONE;\n"
      "bra WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// ---- tensor maps (built on the host by tslb_api.cu, passed as a __grid_constant__ parameter) ----
// Per state buffer: the KV 128-bit field-vector planes as ONE 4-d tensor (x, y, z, f) and the
// scalar plane az as a 3-d tensor (x, y, z); phi^{n+1} is a 3-d tensor in the destination buffer.
// Each exists with four box shapes: the whole ring (main), one wrapped column (wx), one wrapped
// row (wy), one wrapped corner cell (wxy).  128-byte opaque blobs (CUtensorMap).
struct alignas(64) TmaMap { unsigned long long opaque[16]; };
struct TmaMaps { TmaMap vec[4], az[4], ph[4], vecf; };   // [main, wx, wy, wxy]; vecf: one field plane of main

__device__ __forceinline__ void tma_load_4d(void* dst, const TmaMap* map, int c0, int c1, int c2,
                                            int c3, unsigned long long* bar) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const TmaMap* map, int c0, int c1, int c2,
                                            unsigned long long* bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes"
      " [%0], [%1, {%2, %3, %4}], [%5];" ::"r"(smem_u32(dst)),
      "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar))
      : "memory");
}

// staging slot of one source plane: the ring of the tile, all 14 scalars.  Out-of-range parts of
// the main boxes are zero-filled by the TMA unit; the periodic images land in the w* arrays and
// the threads on a wrapped column / row read those instead.
template <typename T, int TX, int TY>
struct TmaStage {
  using M = TileMap<TX, TY, 1>;
  // cells per field plane, padded to a multiple of 128 bytes (every plane is its own box)
  static constexpr int VP = (TileMap<TX, TY, 1>::CELLS + 7) / 8 * 8;
  using V = typename VecOf<T>::type;
  static constexpr int KV = 12 / VecOf<T>::W;          // 128-bit field-vector planes
  static constexpr int PAD = 16 / int(sizeof(T));      // scalars in 16 bytes
  static constexpr int PITCH = TX + 2 * PAD;
  alignas(128) V vec[KV][VP];                          // box (W, HT, 1, KV)
  alignas(128) V vwx[KV][M::HT];                       // box (1, HT, 1, KV)
  alignas(128) V vwy[KV][M::W];                        // box (W, 1, 1, KV)
  alignas(128) V vwxy[KV];                             // box (1, 1, 1, KV)
  alignas(128) T az[M::HT][PITCH];                     // box (PITCH, HT, 1): columns -PAD .. TX+PAD-1
  alignas(128) T azx[M::HT][PAD];
  alignas(128) T azy[PITCH];
  alignas(128) T azxy[PAD];
  alignas(128) T ph[M::HT][PITCH];
  alignas(128) T phx[M::HT][PAD];
  alignas(128) T phy[PITCH];
  alignas(128) T phxy[PAD];
  static constexpr unsigned B_MAIN = KV * M::CELLS * 16 + 2 * M::HT * PITCH * int(sizeof(T));
  static constexpr unsigned B_WX = KV * M::HT * 16 + 2 * M::HT * 16;
  static constexpr unsigned B_WY = KV * M::W * 16 + 2 * PITCH * int(sizeof(T));
  static constexpr unsigned B_WXY = KV * 16 + 2 * 16;
};

template <typename T, int TX, int TY, int MINB, int NSTAGE>
__global__ void __launch_bounds__((TileMap<TX, TY, 1>::NTHREADS + 32), MINB)
k_stream_collide_tma(DevParams<T> P, const __grid_constant__ TmaMaps maps, T* __restrict__ D,
                     T* __restrict__ Qout, int zchunk) {
  using M = TileMap<TX, TY, 1>;
  using SM = K2FastSmem<T, M::CELLS, M::NMAIN>;
  using XB = ExBuf<T, M::CELLS, M::NMAIN>;
  using STG = TmaStage<T, TX, TY>;
  using V = typename VecOf<T>::type;
  constexpr int W = VecOf<T>::W;
  extern __shared__ __align__(128) unsigned char tma_smem_raw[];
  STG* stg = reinterpret_cast<STG*>(tma_smem_raw);                        // 128-byte aligned slots
  SM& sm = *reinterpret_cast<SM*>(tma_smem_raw + NSTAGE * sizeof(STG));
  unsigned long long* full =
      reinterpret_cast<unsigned long long*>(tma_smem_raw + NSTAGE * sizeof(STG) + sizeof(SM));

  const int tid = threadIdx.x;
  const int z0 = P.zbeg + blockIdx.z * zchunk;
  const int z1 = min(P.zend, z0 + zchunk);
  const int plane = P.nx * P.ny;
  const int gx0 = blockIdx.x * TX, gy0 = blockIdx.y * TY;
  // periodic images needed by this tile (host guarantees nx >= 2 TX, ny > TY: at most one each)
  const int xw_l = gx0 == 0, xw_r = gx0 + TX == P.nx;          // wrapped ring column: lx = -1 / TX
  const int yw_b = gy0 == 0, yw_t = gy0 + TY >= P.ny;          // wrapped ring row: gy = -1 / ny
  const int r_w = yw_b ? 0 : P.ny - gy0 + 1;                   // ring row that wraps (if any)

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < NSTAGE; ++s) mbar_init(&full[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  // ------------------------------------------------------------------ producer warp
  if (tid >= M::NTHREADS) {
    const int lane = tid - M::NTHREADS;
    const bool xw = xw_l || xw_r, yw = yw_b || yw_t;
    const unsigned bytes = STG::B_MAIN + (xw ? STG::B_WX : 0u) + (yw ? STG::B_WY : 0u) +
                           (xw && yw ? STG::B_WXY : 0u);
    const int xs_w = xw_l ? P.nx - 1 : 0;                      // source column of the wrapped cell
    const int xsa_w = xw_l ? P.nx - STG::PAD : 0;              // ... of the 16-byte scalar group
    const int ys_w = yw_b ? P.ny - 1 : 0;                      // source row of the wrapped row
    auto produce = [&](int j, int slot) {
      if (j > z1) return;
      const int jz = source_plane(j, P.nz, P.bcz);
      STG& st = stg[slot];
      unsigned long long* bar = &full[slot];
      if (lane == 0) mbar_expect_tx(bar, bytes);
      __syncwarp();
      // lanes 20 .. 20+KV-1: one box per 128-bit field-vector plane of the whole ring
      if (lane >= 20 && lane < 20 + STG::KV)
        tma_load_4d(&st.vec[lane - 20][0], &maps.vecf, (gx0 - 1) * W, gy0 - 1, jz, lane - 20, bar);
      // lanes 1 .. 11: kind = lane / 3 (main, wx, wy, wxy), what = lane % 3 (vectors, az, phi);
      // lane 0 (the main vector box) is covered by the per-plane boxes above
      if (lane == 0 || lane >= 12) return;
      const int kind = lane / 3, what = lane % 3;
      if (kind == 1 && !xw) return;
      if (kind == 2 && !yw) return;
      if (kind == 3 && !(xw && yw)) return;
      const bool colw = kind == 1 || kind == 3, roww = kind == 2 || kind == 3;
      const int y = roww ? ys_w : gy0 - 1;
      if (what == 0) {
        const int x = (colw ? xs_w : gx0 - 1) * W;
        void* dst = kind == 1 ? (void*)&st.vwx[0][0]
                  : kind == 2 ? (void*)&st.vwy[0][0] : (void*)&st.vwxy[0];
        tma_load_4d(dst, &maps.vec[kind], x, y, jz, 0, bar);
      } else {
        const int x = colw ? xsa_w : gx0 - STG::PAD;
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
#pragma unroll
    for (int d = 0; d < NSTAGE; ++d) produce(z0 - 1 + d, d);
    int slot = 0;
    for (int j = z0 - 1; j <= z1; ++j) {
      __syncthreads();                                 // every thread has taken plane j
      produce(j + NSTAGE, slot);
      slot = (slot + 1 == NSTAGE) ? 0 : slot + 1;
    }
    return;
  }

  // ------------------------------------------------------------------ compute threads
  int lx, ly;
  const bool mapped = M::coords(tid, lx, ly);
  const int gx = gx0 + lx, gy = gy0 + ly;
  const int c = M::cell(lx, ly);
  const int rb = ly * TX + lx;                                  // index as a receiver (main: tid)
  const unsigned need = mapped ? dir_mask<TX, TY>(lx, ly) : 0u; // directions somebody reads
  const bool in_ring = mapped && gy >= -1 && gy <= P.ny;            // nx % TX == 0: x always in
  const bool is_out = tid < M::NMAIN && gy < P.ny;
  // where this thread's node lands in a staging slot (byte offsets from the slot base)
  unsigned voff, vstride, azoff, phoff;
  {
    const bool xw = (lx == -1 && xw_l) || (lx == TX && xw_r);
    const bool yw = (yw_b || yw_t) && ly + 1 == r_w;
    const int r = ly + 1, xa = lx == -1 ? STG::PAD - 1 : 0;          // scalar inside its 16-byte group
    if (!xw && !yw) {
      voff = offsetof(STG, vec) + c * 16; vstride = STG::VP * 16;
      azoff = offsetof(STG, az) + (r * STG::PITCH + lx + STG::PAD) * sizeof(T);
      phoff = offsetof(STG, ph) + (r * STG::PITCH + lx + STG::PAD) * sizeof(T);
    } else if (xw && !yw) {
      voff = offsetof(STG, vwx) + r * 16; vstride = M::HT * 16;
      azoff = offsetof(STG, azx) + (r * STG::PAD + xa) * sizeof(T);
      phoff = offsetof(STG, phx) + (r * STG::PAD + xa) * sizeof(T);
    } else if (!xw && yw) {
      voff = offsetof(STG, vwy) + (lx + 1) * 16; vstride = M::W * 16;
      azoff = offsetof(STG, azy) + (lx + STG::PAD) * sizeof(T);
      phoff = offsetof(STG, phy) + (lx + STG::PAD) * sizeof(T);
    } else {
      voff = offsetof(STG, vwxy); vstride = 16;
      azoff = offsetof(STG, azxy) + xa * sizeof(T);
      phoff = offsetof(STG, phxy) + xa * sizeof(T);
    }
  }

  T acc0[6] = {}, acc1[6] = {}, zo0[3] = {}, zo1[3] = {}, u0[3] = {}, u1[3] = {};
  T ph_m = 0, ph_0 = 0, ph_p = 0;

  auto body = [&](const int j, const int slot, const unsigned parity, XB& xb,
                  T (&aA)[6], T (&aB)[6], T (&zA)[3], T (&zB)[3], const T (&uPrev)[3],
                  T (&uCur)[3]) {
    T ownE = 0, ownO = 0, ownQ = 0;
    ph_m = ph_0; ph_0 = ph_p;
    mbar_wait(&full[slot], parity);                    // plane j has landed
    if (in_ring) {
      T cur[13];
      const unsigned char* sb = reinterpret_cast<const unsigned char*>(&stg[slot]);
#pragma unroll
      for (int k = 0; k < STG::KV; ++k)
        unpack(*reinterpret_cast<const V*>(sb + voff + k * vstride), &cur[k * W]);
      cur[12] = *reinterpret_cast<const T*>(sb + azoff);
      ph_p = *reinterpret_cast<const T*>(sb + phoff);
      uCur[0] = cur[F_UX]; uCur[1] = cur[F_UY]; uCur[2] = cur[F_UZ];
      SrcFields<T> sf;
      const Coef<T> cf = coef_from13(cur);
      source_fields(cf, sf);
      publish<T, TX, TY>(xb, sf, P.bcz && (j < 0 || j >= P.nz), tid < M::NMAIN, need, rb, ownE, ownO, ownQ);
      xb.put_pd(c, fma(T(4), ph_0, ph_m + ph_p), ph_p - ph_m);
    }
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
        T q[3];                                     // flux of Eq. 20 for the next step (K1 flux form)
        flux_q(P, ph_0, gx_, gy_, gz_, out.ux, out.uy, out.uz, q);
        store_q(Qout, P.N, idx, q);
      }
      // slot A is free now: it becomes the accumulator of destination plane j+1
#pragma unroll
      for (int i = 0; i < 6; ++i) aA[i] = up[i];
#pragma unroll
      for (int i = 0; i < 3; ++i) zA[i] = up[i];
    }
  };

  int slot = 0;
  unsigned parity = 0;
  auto next_slot = [&]() {
    if (slot + 1 == NSTAGE) { slot = 0; parity ^= 1u; } else { ++slot; }
  };
  for (int j = z0 - 1; j <= z1; j += 2) {
    body(j, slot, parity, sm.buf[0], acc0, acc1, zo0, zo1, u0, u1);
    next_slot();
    if (j + 1 <= z1) {
      body(j + 1, slot, parity, sm.buf[1], acc1, acc0, zo1, zo0, u1, u0);
      next_slot();
    }
  }
}

}  // namespace tslb
