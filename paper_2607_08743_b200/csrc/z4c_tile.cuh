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
  // shared-memory map (in doubles): ring | mbarriers | E_y | E_z | halo-item table
  static constexpr int BAR_OFF = NS * SLOT;                    // NS mbarriers (8 slots reserved)
  static constexpr int EX = TX + 4;                            // x extent of the e arrays (x halo of 2)
  static constexpr int EY_OFF = BAR_OFF + 8;                   // e_y on  TZ x TY x (TX+4)
  static constexpr int EZ_OFF = EY_OFF + TZ * TY * EX;         // e_z on  TZ x (TY+4) x (TX+4)
  static constexpr int TAB_OFF = (EZ_OFF + TZ * (TY + 4) * EX + 1) / 2 * 2;   // int4 table, 16-byte aligned
  static constexpr int N_EYX = 4 * TY * TZ, N_EZX = 4 * TY * TZ, N_EZY = 4 * TX * TZ;
  static constexpr int NITEMS = N_EYX + N_EZX + N_EZY;         // halo entries of e_y, e_z per field
  static constexpr int ITEMS_PER_THREAD = (NITEMS + NT - 1) / NT;
  static constexpr int SMEM_BYTES = (TAB_OFF + 2 * NITEMS) * 8;
  static_assert(NS <= 8, "mbarrier area");
  static_assert(NF % NS == 0, "the ring depth must divide the number of fields");
  static_assert((PX * 8) % 16 == 0, "TMA: the innermost box extent must be a multiple of 16 bytes");
};

// The CTA's dynamic shared memory: NS ring slots of SLOT doubles, then NS mbarriers. Always indexed as an
// array (never through a stored generic pointer), so that every access compiles to LDS with an immediate offset.
extern __shared__ __align__(1024) double tile_smem[];

// sample loader of one field for field_derivs(): shared-memory tile, compile-time strides
template <class C>
struct TileLoader {
  int c;     // index of this thread's centre inside the ring slot of the field
  int slot;  // index of the ring slot (start of the box)
  int ey, ez;  // this thread's entries of the e arrays
  __device__ __forceinline__ static constexpr int stride(int a) { return a == 0 ? 1 : (a == 1 ? C::PX : C::PX * C::PY); }
  __device__ __forceinline__ double operator()(int a, int k) const { return tile_smem[c + k * stride(a)]; }

  // Mixed second derivatives (item 4): D_ab = D_a(e_b), e_b = 8 (u(+1)-u(-1)) - (u(+2)-u(-2)) along the later
  // axis b. e_y and e_z of a point are the numerators of its own D_y, D_z; every thread publishes its pair,
  // the entries two cells outside the tile (x halo of e_y, e_z; y halo of e_z) are computed from the box by the
  // threads the table assigns them to, and after one barrier the outer difference reads four neighbours.
  __device__ __forceinline__ void publish_e(double e_y, double e_z) const {
    tile_smem[ey] = e_y;
    tile_smem[ez] = e_z;
    const int tid = threadIdx.x + C::TX * (threadIdx.y + C::TY * threadIdx.z);
    const int4* tab = reinterpret_cast<const int4*>(tile_smem + C::TAB_OFF);
#pragma unroll
    for (int r = 0; r < C::ITEMS_PER_THREAD; ++r) {
      const int j = tid + r * C::NT;
      if (j < C::NITEMS) {                       // warp-uniform when NITEMS is a multiple of 32
        const int4 t = tab[j];                   // {centre in the box, stride, destination, -}
        const double* u = tile_smem + slot + t.x;
        tile_smem[t.z] = d1_num(u[-2 * t.y], u[-t.y], u[t.y], u[2 * t.y]);
      }
    }
    __syncthreads();
  }
  __device__ __forceinline__ double e_y_x(int k) const { return tile_smem[ey + k]; }            // e_y at x + k
  __device__ __forceinline__ double e_z_x(int k) const { return tile_smem[ez + k]; }            // e_z at x + k
  __device__ __forceinline__ double e_z_y(int k) const { return tile_smem[ez + k * C::EX]; }    // e_z at y + k
};

// halo-item table of the e exchange: built once per CTA (the same for every field and tile)
template <class C>
__device__ __forceinline__ void build_e_table() {
  const int tid = threadIdx.x + C::TX * (threadIdx.y + C::TY * threadIdx.z);
  int4* tab = reinterpret_cast<int4*>(tile_smem + C::TAB_OFF);
  for (int j = tid; j < C::NITEMS; j += C::NT) {
    int x, y, z, st, dst;
    if (j < C::N_EYX + C::N_EZX) {               // x halo: columns -2, -1, TX, TX+1
      const int jj = j < C::N_EYX ? j : j - C::N_EYX;
      const int col = jj % 4;
      x = col < 2 ? col - 2 : C::TX + col - 2;
      y = (jj / 4) % C::TY;
      z = jj / (4 * C::TY);
      if (j < C::N_EYX) { st = C::PX; dst = C::EY_OFF + (z * C::TY + y) * C::EX + (x + 2); }
      else { st = C::PX * C::PY; dst = C::EZ_OFF + (z * (C::TY + 4) + (y + 2)) * C::EX + (x + 2); }
    } else {                                     // y halo of e_z: rows -2, -1, TY, TY+1
      const int jj = j - C::N_EYX - C::N_EZX;
      x = jj % C::TX;
      const int row = (jj / C::TX) % 4;
      y = row < 2 ? row - 2 : C::TY + row - 2;
      z = jj / (4 * C::TX);
      st = C::PX * C::PY;
      dst = C::EZ_OFF + (z * (C::TY + 4) + (y + 2)) * C::EX + (x + 2);
    }
    tab[j] = make_int4(((z + NG) * C::PY + (y + NG)) * C::PX + (x + C::XC), st, dst, 0);
  }
}

struct TileCoord {   // box origin of a tile in the coordinates of its patch's tensor map, and the map
  const CUtensorMap* map;
  int x, y, z;
};

// Source for z4c_point(): field<F>() advances the TMA ring to field F and returns its tile loader.
template <class C>
struct TileSource {
  const double* gcentre;   // global memory: field 0 at this thread's (clamped) point -- centre values
  long long fstride;
  int sc;                  // shared memory: index of this thread's centre in ring slot 0
  int ey, ez;              // shared memory: this thread's entries of the e arrays
  TileCoord cur, nxt;      // this tile and the CTA's next tile
  bool has_next;
  uint32_t iter;           // tiles done by this CTA (ring phase)

  __device__ __forceinline__ double centre(int f) const { return __ldg(gcentre + (long long)f * fstride); }

  __device__ __forceinline__ static uint64_t* full(int slot) {   // mbarrier "box landed" of a ring slot
    return reinterpret_cast<uint64_t*>(tile_smem + C::BAR_OFF) + slot;
  }
  template <int S>
  __device__ __forceinline__ static void issue(const TileCoord& t) {
    constexpr int slot = S % C::NS, f = stream_field(S);
    tma::mbar_expect_tx(full(slot), C::BOX_BYTES);
    tma::load_box(tile_smem + slot * C::SLOT, t.map, full(slot), t.x, t.y, t.z, f);
  }

  template <int F>
  __device__ __forceinline__ TileLoader<C> field() const {
    constexpr int s = stream_slot(F);
    // every thread is done with the slot of field s-1: refill it with the field NS-1 ahead
    __syncthreads();
    if (threadIdx.x == 0 && threadIdx.y == 0 && threadIdx.z == 0) {
      constexpr int sn = s + C::NS - 1;
      if constexpr (sn < NF) issue<sn>(cur);
      else if (has_next) issue<sn - NF>(nxt);
    }
    tma::mbar_wait(full(s % C::NS), (iter * (NF / C::NS) + s / C::NS) & 1u);
    return TileLoader<C>{sc + (s % C::NS) * C::SLOT, (s % C::NS) * C::SLOT, ey, ez};
  }
};

}  // namespace sacra
