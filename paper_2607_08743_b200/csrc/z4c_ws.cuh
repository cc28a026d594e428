// z4c_ws.cuh -- warp-specialised variant of the fused substage kernel (sm_100a): DERIVATIVE warps and ALGEBRA warps.
//
// The point-wise algebra needs ~250 registers per point, which caps a one-thread-per-point CTA at 8 warps per SM,
// and with two warps per scheduler the ~9-cycle FP64 dependency latency is not hidden. Here a CTA has 16
// warps for the same 16 x 4 x 4 tile: for every point one D thread and one A thread.
//   D warps (8-15, `setmaxnreg.dec`): own the TMA box ring and the e exchange; for each field, in stream order, they
//     evaluate the stencils at their point and publish the derivative bundle (u0, D_a, D_ab, advection, KO: 3 to 12
//     doubles) in a bundle ring of SACRA_WS_NB slots in shared memory.
//   A warps (0-7, `setmaxnreg.inc`): run z4c_point() exactly as before, but src.derivs<F>() only reads the bundle;
//     they own the centre-value tile, the RK-input ring and the stores.
// Bundle slots are handed over with full/empty mbarriers (one arrival per warp). Each role keeps its own warps in
// lockstep with a named barrier (bar.sync 1 / 2 over 256 threads), so the schedulers always have two D and two A warps
// in different phases to pick from.
// Status (round 1): runs, bit-identical to the one-role kernel on every GPU test, 8.07 ms per 256^3
// substage against 7.19 -- an experimental build (-DSACRA_WS), not the default.
#pragma once
#include "z4c_tile.cuh"

#ifndef SACRA_WS_NB
#define SACRA_WS_NB 3   // bundle slots: how far the derivative warps may run ahead of the algebra warps
#endif

namespace sacra {

__host__ __device__ constexpr bool field_has_d1(int f) { return !(f >= F_A && f < F_A + 6) && !(f >= F_B && f < F_B + 3); }
__host__ __device__ constexpr bool field_has_d2(int f) {
  return f == F_W || (f >= F_G && f < F_G + 6) || f == F_ALP || (f >= F_BET && f < F_BET + 3);
}

template <int TX_, int TY_, int TZ_, int NS_, int REG_D_, int REG_A_>
struct WsCfg {
  static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NS = NS_;
  static constexpr int REG_D = REG_D_, REG_A = REG_A_;          // setmaxnreg targets; (REG_D + REG_A) * 256 <= 65536
  static constexpr int NT = TX * TY * TZ;                      // points per tile = threads per role
  static constexpr int NTHREADS = 2 * NT, NWR = NT / 32;       // CTA size; warps per role
  static constexpr int XC = NG + 1;
  static constexpr int PX = TX + 2 * NG + 2, PY = TY + 2 * NG, PZ = TZ + 2 * NG;
  static constexpr int BOX = PX * PY * PZ, BOX_BYTES = BOX * 8, SLOT = (BOX + 15) / 16 * 16;
  static constexpr int RKD = 5, NB = SACRA_WS_NB, BW = 12;     // RK ring depth; bundle slots; doubles per bundle
  // shared-memory map (doubles): ring | mbarriers + tile descriptors | centre tile | RK ring | bundles | e arrays
  static constexpr int BAR_OFF = NS * SLOT;
  static constexpr int CEN_OFF = BAR_OFF + 32;
  static constexpr int CEN_BYTES = NF * NT * 8;
  static constexpr int RK_OFF = CEN_OFF + NF * NT;
  static constexpr int BUN_OFF = RK_OFF + RKD * 2 * NT;        // slot b, entry k, point p: BUN_OFF + (b*BW + k)*NT + p
  static constexpr int EX = TX + 4;
  static constexpr int EY_OFF = BUN_OFF + NB * BW * NT;
  static constexpr int EZ_OFF = EY_OFF + TZ * TY * EX;
  static constexpr int SMEM_BYTES = (EZ_OFF + TZ * (TY + 4) * EX) * 8;
  // mbarrier indices; tile descriptors sit in slots 28..31
  static constexpr int B_FULL = 0, B_CFULL = NS, B_RFULL = NS + 1, B_BFULL = NS + 1 + RKD, B_BEMPTY = NS + 1 + RKD + NB,
                       B_END = NS + 1 + RKD + 2 * NB, DESC_SLOT = 28;
  static_assert(B_END <= DESC_SLOT && SMEM_BYTES <= 232448, "mbarrier area / shared memory");
  static_assert(REG_D % 8 == 0 && REG_A % 8 == 0, "register split");
  static_assert(TY == 4 && NT == 256 && NF % RKD == 0 && NS >= 2 && NS <= 5 && (PX * 8) % 16 == 0, "configuration");
};

template <class C>
struct WsBars {
  __device__ __forceinline__ static uint64_t* bar(int i) { return reinterpret_cast<uint64_t*>(tile_smem + C::BAR_OFF) + i; }
  __device__ static void init() {
    for (int i = 0; i < C::NS; ++i) tma::mbar_init(bar(C::B_FULL + i), 1);
    tma::mbar_init(bar(C::B_CFULL), 1);
    for (int i = 0; i < C::RKD; ++i) tma::mbar_init(bar(C::B_RFULL + i), 1);
    for (int i = 0; i < C::NB; ++i) { tma::mbar_init(bar(C::B_BFULL + i), C::NWR); tma::mbar_init(bar(C::B_BEMPTY + i), C::NWR); }
    tma::fence_mbar_init();
  }
  // warp-uniform wait (every lane leaves in the same iteration)
  __device__ __forceinline__ static void wait(int b, uint32_t parity) {
    while (!__all_sync(0xffffffffu, tma::mbar_try_wait(bar(b), parity))) {}
  }
};

// ---------------------------------------------------------------------------------------------------------------
// D side: boxes -> derivative bundles
// ---------------------------------------------------------------------------------------------------------------
template <class C>
struct DSide {
  int p, lane;             // point of the tile (0..NT-1), lane
  int sc, ey, ez, xh, yh;  // tile loader indices (TileLoader)
  uint32_t iter;
  bool has_next;
  TileCoord cur, nxt;
  using Bars = WsBars<C>;

  __device__ __forceinline__ static uint32_t ring_slot(uint32_t it, int s) { return (it * NF + s) % C::NS; }
  __device__ __forceinline__ static uint32_t ring_use(uint32_t it, int s) { return (it * NF + s) / C::NS; }

  template <int S>   // stream position S of this tile (S >= NF: of the next tile)
  __device__ __forceinline__ void issue() const {
    if (S >= NF && !has_next) return;
    constexpr int f = stream_field(S % NF);
    const TileCoord& t = S < NF ? cur : nxt;
    const uint32_t slot = ring_slot(iter, S);
    tma::mbar_expect_tx(Bars::bar(C::B_FULL + slot), C::BOX_BYTES);
    tma::load_box(tile_smem + slot * C::SLOT, t.m.box, Bars::bar(C::B_FULL + slot), t.x - C::XC, t.y - NG, t.z - NG, f,
                  tma::L2_EVICT_NORMAL);
  }
  __device__ __forceinline__ void prime() const {
    issue<0>();
    if constexpr (C::NS > 2) issue<1>();
    if constexpr (C::NS > 3) issue<2>();
    if constexpr (C::NS > 4) issue<3>();
  }

  // the shift at this point from the boxes of beta^x, beta^y, beta^z (stream positions 0, 1, 2; NS >= 4 keeps all
  // three resident at the start of a tile)
  __device__ __forceinline__ void shift_at_point(double (&beta)[3]) const {
    static_assert(C::NS >= 4 && stream_field(0) == F_BET && stream_field(1) == F_BET + 1 && stream_field(2) == F_BET + 2, "");
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      const uint32_t slot = ring_slot(iter, a);
      Bars::wait(C::B_FULL + slot, ring_use(iter, a) & 1u);
      beta[a] = tile_smem[sc + (int)slot * C::SLOT];
    }
  }

  template <int s>
  __device__ __forceinline__ void field(const PointCoef& pc) const {
    constexpr int F = stream_field(s);
    constexpr bool D1 = field_has_d1(F), D2 = field_has_d2(F);
    group_sync<1, C::NT>();   // every D thread is done with the box of field s-1 (and with the e arrays)
    if (p == 0) issue<s + C::NS - 1>();
    const uint32_t slot = ring_slot(iter, s);
    Bars::wait(C::B_FULL + slot, ring_use(iter, s) & 1u);
    Stencil S;
    field_derivs<D1, D2>(TileLoader<C, 1>{sc + (int)slot * C::SLOT, ey, ez, xh, yh, nullptr}, pc, S);
    // bundle slot of sequence number g = iter*NF + s (NF is odd: the slot alternates across tiles too)
    const uint32_t g = iter * NF + s, b = g % C::NB, use = g / C::NB;
    if (use > 0) Bars::wait(C::B_BEMPTY + b, (use - 1) & 1u);
    double* o = tile_smem + C::BUN_OFF + b * C::BW * C::NT + p;
    o[0] = S.u0;
    if (D1) {
#pragma unroll
      for (int k = 0; k < 3; ++k) o[(1 + k) * C::NT] = S.d1[k];
    }
    if (D2) {
#pragma unroll
      for (int k = 0; k < 6; ++k) o[(4 + k) * C::NT] = S.d2[k];
    }
    o[10 * C::NT] = S.adv;
    o[11 * C::NT] = S.ko;
    __syncwarp();
    if (lane == 0) tma::mbar_arrive(Bars::bar(C::B_BFULL + b));
  }
  template <int s>
  __device__ __forceinline__ void fields_from(const PointCoef& pc) const {
    if constexpr (s < NF) {
      field<s>(pc);
      fields_from<s + 1>(pc);
    }
  }
};

// ---------------------------------------------------------------------------------------------------------------
// A side: the Src of z4c_point()
// ---------------------------------------------------------------------------------------------------------------
// Geo::next(iter) -> TileCoord of the CTA's next tile. The D leader decodes it at the top of ITS tile; the A side may
// read it only after it has taken a bundle of the same tile (mbarrier release / acquire orders the two).
template <class C, int RK, class Geo>
struct ASide {
  Geo geo;
  int tid, lane;           // point of the tile, lane
  int cen;                 // this thread's entry of field 0 in the centre tile
  uint32_t iter;
  bool has_next;
  TileCoord cur, nxt;
  using Bars = WsBars<C>;

  __device__ __forceinline__ double centre(int f) const { return tile_smem[cen + f * C::NT]; }

  __device__ __forceinline__ void issue_centre(const TileCoord& t) const {
    tma::mbar_expect_tx(Bars::bar(C::B_CFULL), C::CEN_BYTES);
    tma::load_box(tile_smem + C::CEN_OFF, t.m.cen, Bars::bar(C::B_CFULL), t.x, t.y, t.z, 0, tma::L2_EVICT_LAST);
  }
  template <int E>   // emit index of this tile (E >= NF: of the next tile)
  __device__ __forceinline__ void issue_rk() const {
    if (E >= NF && !has_next) return;
    constexpr int r = E % C::RKD, f = emit_field(E % NF);
    const TileCoord& t = E < NF ? cur : nxt;
    tma::mbar_expect_tx(Bars::bar(C::B_RFULL + r), 2 * C::NT * 8);
    tma::load_box(tile_smem + C::RK_OFF + 2 * r * C::NT, t.m.un, Bars::bar(C::B_RFULL + r), t.x, t.y, t.z, f,
                  tma::L2_EVICT_FIRST);
    tma::load_box(tile_smem + C::RK_OFF + (2 * r + 1) * C::NT, t.m.acc, Bars::bar(C::B_RFULL + r), t.x, t.y, t.z, f,
                  tma::L2_EVICT_FIRST);
  }
  template <int LO, int HI>
  __device__ __forceinline__ void issue_rk_range() const {
    if constexpr (LO < HI) {
      issue_rk<LO + 1>();
      issue_rk_range<LO + 1, HI>();
    }
  }
  __device__ __forceinline__ void prime() const {   // first tile of the CTA
    issue_centre(cur);
    if constexpr (RK == 2) issue_rk_range<-1, C::RKD - 2>();
  }
  // start of a tile: all A threads are done with the previous tile's centre values; request this tile's
  __device__ __forceinline__ void begin_tile() const {
    group_sync<2, C::NT>();
    if (tid == 0 && iter > 0) issue_centre(cur);
    Bars::wait(C::B_CFULL, iter & 1u);
  }

  template <int F, bool D1, bool D2>
  __device__ __forceinline__ void derivs(const PointCoef&, Stencil& S) const {
    constexpr int s = stream_slot(F);
    static_assert(D1 == field_has_d1(F) && D2 == field_has_d2(F), "the D side publishes what the A side reads");
    group_sync<2, C::NT>();   // A warps in lockstep: every RK slot read so far is free
    if (tid == 0) {
      if constexpr (RK == 2) {
        constexpr int hi = emits_before(s) + C::RKD - 1;
        constexpr int lo = s == 0 ? C::RKD - 2 : emits_before(s - 1) + C::RKD - 1;
        issue_rk_range<lo, hi>();
      }
    }
    const uint32_t g = iter * NF + s, b = g % C::NB, use = g / C::NB;
    Bars::wait(C::B_BFULL + b, use & 1u);
    const double* o = tile_smem + C::BUN_OFF + b * C::BW * C::NT + tid;
    S.u0 = o[0];
    if (D1) {
#pragma unroll
      for (int k = 0; k < 3; ++k) S.d1[k] = o[(1 + k) * C::NT];
    }
    if (D2) {
#pragma unroll
      for (int k = 0; k < 6; ++k) S.d2[k] = o[(4 + k) * C::NT];
    }
    S.adv = o[10 * C::NT];
    S.ko = o[11 * C::NT];
    __syncwarp();
    if (lane == 0) tma::mbar_arrive(Bars::bar(C::B_BEMPTY + b));
    if constexpr (s == 0) {
      if (has_next) const_cast<ASide*>(this)->nxt = geo.next(iter);   // now visible: written before this bundle
    }
  }

  template <int F>
  __device__ __forceinline__ void rk_inputs(double& un, double& acc) const {
    constexpr int e = emit_slot(F), r = e % C::RKD;
    Bars::wait(C::B_RFULL + r, (iter * (NF / C::RKD) + e / C::RKD) & 1u);
    un = tile_smem[C::RK_OFF + 2 * r * C::NT + tid];
    acc = tile_smem[C::RK_OFF + (2 * r + 1) * C::NT + tid];
  }
};

}  // namespace sacra
