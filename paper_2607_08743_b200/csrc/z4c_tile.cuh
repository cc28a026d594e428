// z4c_tile.cuh -- TMA-staged field tiles for the fused Z4c substage kernel (sm_100a).
//
// One CTA owns a TX x TY x TZ tile of active points, one thread per point (the per-point running tensors of
// z4c_fused.cuh live in registers). The 25 fields are streamed through shared memory ONE FIELD AT A TIME in
// the order z4c_point() consumes them: for every field a single cp.async.bulk.tensor (TMA) instruction, issued
// by thread 0, copies the (TX+8) x (TY+6) x (TZ+6) box -- tile plus the 3-cell halo of the upwind and
// Kreiss-Oliger stencils -- from HBM/L2 into one of NS ring buffers and signals an mbarrier.
// The ring runs NS-1 fields ahead of the arithmetic and carries on across the tiles of a persistent CTA
// (the first fields of the next tile are in flight while the last fields of the current one are computed).
// NS divides 25, so the ring slot of every field is a compile-time constant and every shared-memory load of
// the stencils has an immediate offset.
#pragma once
#include <cstdint>
#include <cuda.h>   // CUtensorMap (types only; the encoder is fetched through cudaGetDriverEntryPoint)

#include "z4c_stencil.cuh"

namespace sacra {

// ---- field streaming order = the order of the field<F>() calls in z4c_point() -------------------------------
//   beta^i -> Gt^i -> gt_ij -> W -> alpha -> K-hat -> Theta -> B^i -> At_ij
__host__ __device__ constexpr int stream_field(int s) {
  constexpr int order[NF] = {19, 20, 21, 14, 15, 16, 1, 2, 3, 4, 5, 6, 0, 18, 7, 17, 22, 23, 24, 8, 9, 10, 11, 12, 13};
  return order[s];
}
__host__ __device__ constexpr int stream_slot(int f) {
  for (int s = 0; s < NF; ++s)
    if (stream_field(s) == f) return s;
  return -1;
}

namespace tma {
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t ok;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!ok);
}
// box load of a rank-4 tensor (x, y, z, field); coordinates in elements, innermost first
__device__ __forceinline__ void load_box(void* dst, const CUtensorMap* map, uint64_t* bar, int x, int y, int z, int f) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5, %6}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z), "r"(f)
      : "memory");
}
}  // namespace tma

template <int TX_, int TY_, int TZ_, int NS_>
struct TileCfg {
  static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NS = NS_;
  static constexpr int NT = TX * TY * TZ;                      // threads = points per tile
  // box extents. x: the box must start on a 16-byte boundary of global memory (TMA rule for the innermost
  // coordinate, found by probing: an odd FP64 start coordinate raises "illegal instruction"); storage cell
  // bx*TX of a row sits at an odd double (sacra.h), so the box starts one cell earlier and is one cell wider
  // on each side: centre of thread 0 at x offset XC = NG + 1.
  static constexpr int XC = NG + 1;
  static constexpr int PX = TX + 2 * NG + 2, PY = TY + 2 * NG, PZ = TZ + 2 * NG;
  static constexpr int BOX = PX * PY * PZ;                     // doubles per box
  static constexpr int BOX_BYTES = BOX * 8;
  static constexpr int SLOT = (BOX + 15) / 16 * 16;            // doubles per ring slot (128-byte multiple)
  static constexpr int SMEM_BYTES = NS * SLOT * 8 + NS * 8 + 128;
  static_assert(NF % NS == 0, "the ring depth must divide the number of fields");
  static_assert((PX * 8) % 16 == 0, "TMA: the innermost box extent must be a multiple of 16 bytes");
};

// sample loader of one field for field_derivs(): shared-memory tile, compile-time strides
template <class C>
struct TileLoader {
  const double* c;   // this thread's centre inside the ring slot of the field
  __device__ __forceinline__ double operator()(int a, int k) const {
    return c[k * (a == 0 ? 1 : (a == 1 ? C::PX : C::PX * C::PY))];
  }
  __device__ __forceinline__ double mixed(int a, int ka, int b, int kb) const {
    return c[ka * (a == 0 ? 1 : (a == 1 ? C::PX : C::PX * C::PY)) + kb * (b == 0 ? 1 : (b == 1 ? C::PX : C::PX * C::PY))];
  }
};

struct TileCoord {   // box origin of a tile in the coordinates of its patch's tensor map, and the map
  const CUtensorMap* map;
  int x, y, z;
};

// Source for z4c_point(): field<F>() advances the TMA ring to field F and returns its tile loader.
template <class C>
struct TileSource {
  const double* gcentre;   // global memory: field 0 at this thread's (clamped) point -- centre values
  long long fstride;
  const double* sc;        // shared memory: this thread's centre in ring slot 0
  double* ring;            // ring slot 0
  uint64_t* full;          // NS mbarriers
  TileCoord cur, nxt;      // this tile and the CTA's next tile
  bool has_next;
  uint32_t iter;           // tiles done by this CTA (ring phase)

  __device__ __forceinline__ double centre(int f) const { return __ldg(gcentre + (long long)f * fstride); }

  template <int S>
  __device__ __forceinline__ static void issue(double* ring, uint64_t* full, const TileCoord& t) {
    constexpr int slot = S % C::NS, f = stream_field(S);
    tma::mbar_expect_tx(full + slot, C::BOX_BYTES);
    tma::load_box(ring + slot * C::SLOT, t.map, full + slot, t.x, t.y, t.z, f);
  }

  template <int F>
  __device__ __forceinline__ TileLoader<C> field() const {
    constexpr int s = stream_slot(F);
    // every thread is done with the slot of field s-1: refill it with the field NS-1 ahead
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) {
      constexpr int sn = s + C::NS - 1;
      if constexpr (sn < NF) issue<sn>(ring, full, cur);
      else if (has_next) issue<sn - NF>(ring, full, nxt);
    }
    tma::mbar_wait(full + s % C::NS, (iter * (NF / C::NS) + s / C::NS) & 1u);
    return TileLoader<C>{sc + (s % C::NS) * C::SLOT};
  }
};

}  // namespace sacra
