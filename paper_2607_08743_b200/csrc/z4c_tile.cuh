// z4c_tile.cuh -- TMA-staged field tiles for the fused Z4c substage kernel (sm_100a).
//
// One CTA owns a TX x TY x TZ tile of active points, one thread per point (the per-point running tensors of
// z4c_fused.cuh live in registers). The 25 fields are streamed through shared memory ONE FIELD AT A TIME in
// the order z4c_point() consumes them: for every field a single cp.async.bulk.tensor (TMA) instruction, issued
// by thread 0, copies the (TX+8) x (TY+6) x (TZ+6) box -- tile plus the 3-cell halo of the upwind and
// Kreiss-Oliger stencils -- from HBM/L2 into one of NS ring buffers and signals an mbarrier.
// The ring runs NS-1 fields ahead of the arithmetic and carries on across the tiles of a persistent CTA
// (the first fields of the next tile are in flight while the last fields of the current one are computed).
// The ring slot of a field is (tile count * stream length + stream position) % NS: one register per field holds the
// slot base, every shared-memory load of the stencils has an immediate offset from it.
// The same machinery serves three more TMA streams: the centre-value tile of all 25 fields (no halo; the values
// the algebra needs before a field's own box arrives; every thread copies its 25 values into its Tensor Memory
// strip at the start of a tile, z4c_tmem.cuh, which frees the buffer for the next tile's values), the ring of RK
// inputs u_n / acc in emit order (stages 2-4), and -- with a 15-field stream -- the constraint monitor.
#pragma once
#include <cstdint>
#include <type_traits>
#include <cuda.h>   // CUtensorMap (types only; the encoder is fetched through cudaGetDriverEntryPoint)

#include "z4c_stencil.cuh"
#include "z4c_tmem.cuh"

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

// the fields a kernel streams, in order: the full Z4c right-hand side, and the constraint monitor (SURVEY 8(f) f-1:
// W, gt_ij, K-hat, Theta, At_ij -- the gauge fields and Gt^i do not enter Eqs. 20-21)
struct Z4cStream {
  static constexpr int N = NF;
  __host__ __device__ static constexpr int field(int s) { return stream_field(s); }
  __host__ __device__ static constexpr int slot(int f) { return stream_slot(f); }
};
struct ConStream {
  static constexpr int N = 15;
  __host__ __device__ static constexpr int field(int s) {
    constexpr int order[N] = {0, 1, 2, 3, 4, 5, 6, 7, 17, 8, 9, 10, 11, 12, 13};
    return order[s];
  }
  __host__ __device__ static constexpr int slot(int f) {
    for (int s = 0; s < N; ++s)
      if (field(s) == f) return s;
    return -1;
  }
};

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
// wait of a PRODUCER thread: it has nothing else to do, but its probes take issue slots from the compute warps of its
// scheduler (measured: 380 M try_wait instructions per 256^3 substage, 12 % of all instructions executed) -- so it
// suspends in the probe for up to ~1 us
__device__ __forceinline__ void mbar_wait_idle(uint64_t* bar, uint32_t parity) {
  for (;;) {
    uint32_t ok;
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n selp.u32 %0, 1, 0, p;\n}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity), "r"(1000u)
        : "memory");
    if (ok) return;
  }
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {   // one (possibly suspending) probe
  uint32_t ok;
  asm volatile(
      "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}"
      : "=r"(ok)
      : "r"(smem_u32(bar)), "r"(parity)
      : "memory");
  return ok != 0;
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// L2 eviction policies (the encodings createpolicy.fractional.L2::evict_*.b64 produces for fraction 1.0).
// The centre tile of a tile is requested one tile ahead of its stencil boxes and covers the same cells, so it
// should stay in L2 (evict last) for the boxes of this tile and of its neighbours to hit; u_n / acc tiles are read
// exactly once (evict first). Measured at 256^3, stage 2: 17.6 GB read from DRAM per launch (19.7 GB with the
// centre tile evict-first, 28.8 GB before the super-block tile order), 10.3 GB of it compulsory.
constexpr uint64_t L2_EVICT_FIRST = 0x12F0000000000000ull, L2_EVICT_LAST = 0x14F0000000000000ull,
                   L2_EVICT_NORMAL = 0x1000000000000000ull;
#ifndef SACRA_CEN_POLICY
#define SACRA_CEN_POLICY L2_EVICT_LAST
#endif
#ifndef SACRA_BOX_POLICY
#define SACRA_BOX_POLICY L2_EVICT_NORMAL
#endif
// box load of a rank-4 tensor (x, y, z, field); coordinates in elements, innermost first
__device__ __forceinline__ void load_box(void* dst, const CUtensorMap* map, uint64_t* bar, int x, int y, int z, int f,
                                         uint64_t policy) {
  asm volatile(
      "cp.async.bulk.tensor.4d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint"
      " [%0], [%1, {%3, %4, %5, %6}], [%2], %7;"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z), "r"(f), "l"(policy)
      : "memory");
}
}  // namespace tma

// ---- the Tensor Memory strip of a thread (z4c_tmem.cuh), in doubles ------------------------------------------------
// centre values of the 25 fields, grouped the way z4c_point() pulls them (aligned groups of 4 / 2 / 1 doubles):
//   0-5 gt_ij | 6 alpha | 7 W | 8-10 beta^i | 11 K-hat | 12-14 B^i | 15 Theta | 16-21 At_ij | 22-24 Gt^i
// then the parked tensors of the algebra.
__host__ __device__ constexpr int cen_slot(int f) {
  return (f >= F_G && f < F_G + 6) ? f - F_G
       : f == F_ALP ? 6 : f == F_W ? 7
       : (f >= F_BET && f < F_BET + 3) ? 8 + (f - F_BET)
       : f == F_KH ? 11
       : (f >= F_B && f < F_B + 3) ? 12 + (f - F_B)
       : f == F_TH ? 15
       : (f >= F_A && f < F_A + 6) ? 16 + (f - F_A)
       : 22 + (f - F_GAM);
}
__host__ __device__ constexpr int cen_field(int slot) {
  for (int f = 0; f < NF; ++f)
    if (cen_slot(f) == slot) return f;
  return -1;
}
constexpr int PK_DB = 28;    // d_k beta^i, 3 groups k of 4 doubles (i = 0..2, pad)
constexpr int PK_DG = 40;    // d_k gt_n,   6 groups n of 4 doubles (k = 0..2, pad); later Gt^k_n in the same place
constexpr int PK_GU = PK_DG;
constexpr int PK_AUU = 64;   // At^ij,      3 groups i of 4 doubles (j = 0..2, pad)
constexpr int PK_AG = 76;    // advection and KO of Gt^k, 3 groups k of 2 doubles
constexpr int PK_END = 82;

#ifndef SACRA_RKD
#define SACRA_RKD 8
#endif
template <int TX_, int TY_, int TZ_, int NS_>
struct TileCfg {
  static constexpr int TX = TX_, TY = TY_, TZ = TZ_, NS = NS_;
  static constexpr int NT = TX * TY * TZ;                      // threads = points per tile
  // Tensor Memory: 512 columns shared by the warps of a lane quarter (warps w, w + 4, ...): doubles per thread
  static constexpr int TM_WARPS = (NT / 32 + 3) / 4;
  static constexpr int TM_DOUBLES = (512 / TM_WARPS) / 2 / 2 * 2;
  static_assert(NT % 64 == 0 && PK_END <= TM_DOUBLES, "Tensor Memory strip of a thread");
  // box extents. x: the box must start on a 16-byte boundary of global memory (TMA rule for the innermost
  // coordinate, found by probing: an odd FP64 start coordinate raises "illegal instruction"); storage cell
  // bx*TX of a row sits at an odd double (sacra.h), so the box starts one cell earlier and is one cell wider
  // on each side: centre of thread 0 at x offset XC = NG + 1.
  static constexpr int XC = NG + 1;
  static constexpr int PX = TX + 2 * NG + 2, PY = TY + 2 * NG, PZ = TZ + 2 * NG;
  static constexpr int BOX = PX * PY * PZ;                     // doubles per box
  static constexpr int BOX_BYTES = BOX * 8;
  static constexpr int SLOT = (BOX + 15) / 16 * 16;            // doubles per ring slot (128-byte multiple)
  // shared-memory map (in doubles):
  //   ring | mbarriers | centre tile (NF x NT) | RK ring (RKD x {u_n, acc} x NT) | E_y | E_z
  static constexpr int RKD = SACRA_RKD;                               // depth of the RK-input ring (a power of two)
  static constexpr int NW = NT / 32;                           // compute warps of the CTA
  // threads of the CTA: the compute warps + one producer warpgroup (setmaxnreg moves registers between whole
  // warpgroups: the producer's three idle warps only donate theirs)
  static constexpr int NTH = NT + 128;
  static constexpr int REG_PRODUCER = 32;
  static constexpr int REG_COMPUTE = (65536 - 128 * REG_PRODUCER) / NT / 8 * 8;
  static_assert(NT % 128 == 0 && REG_COMPUTE >= 128 && REG_COMPUTE <= 255, "register split between the roles");
  // mbarrier area (32 doubles): "full" NS box + 1 centre + RKD rk, "empty" NS box + 1 centre + RKD rk; then the base
  // address of the CTA's Tensor Memory and two tile descriptors
  static constexpr int BAR_OFF = NS * SLOT;
  static constexpr int NBAR = 2 * NS + 2 + 2 * RKD;
  static constexpr int TMB_OFF = BAR_OFF + NBAR;               // uint32 base address of the Tensor Memory allocation
  static constexpr int DESC_OFF = BAR_OFF + 28;                // 2 x TileId (16 bytes each)
  static constexpr int CEN_OFF = BAR_OFF + 32;                 // unpadded tiles of all NF fields
  static constexpr int CEN_BYTES = NF * NT * 8;
  static constexpr int RK_OFF = CEN_OFF + NF * NT;             // slot r: u_n tile at RK_OFF + 2 r NT, acc tile + NT
  static constexpr int EX = TX + 4;                            // x extent of the e arrays (x halo of 2)
  static constexpr int EY_OFF = RK_OFF + RKD * 2 * NT;         // e_y on  TZ x TY x (TX+4)
  static constexpr int EZ_OFF = EY_OFF + TZ * TY * EX;         // e_z on  TZ x (TY+4) x (TX+4)
  static constexpr int ESZ = TZ * TY * EX + TZ * (TY + 4) * EX;   // one set of e arrays
  static constexpr int SMEM_BYTES = (EY_OFF + ESZ) * 8;
  static_assert(SMEM_BYTES + 1024 <= 233472, "shared memory of one SM");
  static_assert((RKD & (RKD - 1)) == 0 && NBAR < 28, "mbarrier area / RK ring depth");
  static_assert(TX * TY == 64, "e exchange: one z-plane of the tile = two warps = one named barrier of 64 threads");
  static_assert(TZ + 1 <= 15, "named barriers 1 .. TZ");
  static_assert(TY == 4 && TX >= 4, "e exchange: one y-halo row of e_z per thread row, x-halo columns by the edge lanes");
  static_assert((NT * 8) % 128 == 0 && SLOT % 16 == 0, "TMA destinations are 128-byte aligned");
  static_assert(NS >= 2 && NS <= 5, "ring depth");
  static_assert((PX * 8) % 16 == 0, "TMA: the innermost box extent must be a multiple of 16 bytes");
};

// The CTA's dynamic shared memory: NS ring slots of SLOT doubles, then NS mbarriers. Always indexed as an
// array (never through a stored generic pointer), so that every access compiles to LDS with an immediate offset.
extern __shared__ __align__(1024) double tile_smem[];

// Barrier among the threads that exchange e values. The mixed derivatives D_xy, D_xz, D_yz of a point need e_y / e_z
// of points of the SAME z-plane only, and a z-plane of the tile is TX x TY = 64 threads = two warps: named barrier
// 1 + z, 64 threads. No barrier of the kernel's tile loop spans the CTA: the warps of different planes drift apart by
// up to NS - 1 fields (TileSource::field()), so that the stencil loads of one warp overlap the arithmetic of another.
__device__ __forceinline__ void plane_sync() {   // 1-D block: thread t is point (t % TX, t / TX % TY, t / 64)
  asm volatile("bar.sync %0, 64;" ::"r"(1u + threadIdx.x / 64u) : "memory");
}

// sample loader of one field for field_derivs(): shared-memory tile, compile-time strides
template <class C>
struct TileLoader {
  int c;       // index of this thread's centre inside the ring slot of the field
  int ey, ez;  // this thread's entries of the e arrays
  int xh;      // x-halo duty of this thread: 0 none, else the x offset (-2 or +2) of the column it also computes
  int yh;      // y offset (-2 or +2 rows... in units of rows) of the e_z y-halo entry this thread computes
  __device__ __forceinline__ static constexpr int stride(int a) { return a == 0 ? 1 : (a == 1 ? C::PX : C::PX * C::PY); }
  __device__ __forceinline__ double operator()(int a, int k) const { return tile_smem[c + k * stride(a)]; }
  __device__ __forceinline__ double e_at(int o, int st) const {   // inner difference along stride st at centre + o
    const double* u = tile_smem + c + o;
    return d1_num(u[-2 * st], u[-st], u[st], u[2 * st]);
  }

  // Mixed second derivatives (item 4): D_ab = D_a(e_b), e_b = 8 (u(+1)-u(-1)) - (u(+2)-u(-2)) along the later
  // axis b. e_y and e_z of a point are the numerators of its own D_y, D_z; every thread publishes its pair.
  // The entries two cells outside the tile are computed from the box without any table: thread row y computes
  // the e_z entry of y-halo row {-2, -1, TY, TY+1}[y] in its own column (TY = 4: one each), and the lanes of
  // columns 0, 1 / TX-2, TX-1 compute e_y, e_z two columns to their left / right. Two barriers of the plane's two
  // warps (one set of e arrays: the previous exchange has been read; this one has been written), then the outer
  // difference reads four neighbours.
  __device__ __forceinline__ void publish_e(double e_y, double e_z) const {
    plane_sync();   // the partner warp has read the e values of the previous exchange
    tile_smem[ey] = e_y;
    tile_smem[ez] = e_z;
    tile_smem[ez + yh * C::EX] = e_at(yh * C::PX, C::PX * C::PY);
    if (xh) {
      tile_smem[ey + xh] = e_at(xh, C::PX);
      tile_smem[ez + xh] = e_at(xh, C::PX * C::PY);
    }
    plane_sync();
  }
  __device__ __forceinline__ double e_y_x(int k) const { return tile_smem[ey + k]; }            // e_y at x + k
  __device__ __forceinline__ double e_z_x(int k) const { return tile_smem[ez + k]; }            // e_z at x + k
  __device__ __forceinline__ double e_z_y(int k) const { return tile_smem[ez + k * C::EX]; }    // e_z at y + k
};

// ---- emit order = the order in which z4c_point() finishes the RHS values ------------------------------------
// Every field is emitted right after its own derivative stage, except Gt^i, whose RHS needs the gradients of
// K-hat and Theta and leaves after Theta.
__host__ __device__ constexpr int emit_field(int e) {
  constexpr int order[NF] = {19, 20, 21, 1, 2, 3, 4, 5, 6, 0, 18, 7, 17, 14, 15, 16, 22, 23, 24, 8, 9, 10, 11, 12, 13};
  return order[e];
}
__host__ __device__ constexpr int emit_slot(int f) {
  for (int e = 0; e < NF; ++e)
    if (emit_field(e) == f) return e;
  return -1;
}
// number of emits that precede the field<>() call of stream position s in program order
__host__ __device__ constexpr int emits_before(int s) {
  int n = 0;
  for (int e = 0; e < NF; ++e) {
    const int f = emit_field(e);
    const int pos = (f >= F_GAM && f < F_GAM + 3) ? stream_slot(F_TH) : stream_slot(f);
    if (pos < s) ++n;
  }
  return n;
}

constexpr int MAXP = 16;   // patch descriptors carried in kernel parameters per launch
struct alignas(64) TileMaps {   // rank-4 (x, y, z, field) tensor maps of every patch of the launch
  CUtensorMap box[MAXP];   // stage input u_in, box  PX x PY x PZ x 1   (stencil tiles)
  CUtensorMap cen[MAXP];   // stage input u_in, box  TX x TY x TZ x NF  (centre values of every field)
  CUtensorMap un[MAXP];    // u_n,              box  TX x TY x TZ x 1   (stages 2-4)
  CUtensorMap acc[MAXP];   // acc,              box  TX x TY x TZ x 1   (stages 2-4)
};
struct TileId {   // a tile of the launch: patch and tile indices
  int ip, bx, by, bz;
};

// Source for z4c_point(): field<F>() advances the TMA ring to field F and returns its tile loader;
// centre(f) reads the centre-value tile; rk_un / rk_acc read the RK-input ring (stages 2-4).
// RK = 0: no RK inputs (plain RHS); 1: u_n is the stage input itself (centre tile); 2: u_n and acc ring.
template <class C, int RK, class Stream = Z4cStream>
struct TileSource {
  int tid;                 // linear thread index = point of the tile
  int sc;                  // shared memory: index of this thread's centre in ring slot 0
  uint32_t tm;             // Tensor Memory: address of double 0 of this thread's strip (a double = 2 columns)
  int ey, ez;              // shared memory: this thread's entries of the e arrays
  int xh, yh;              // halo duties of the e exchange (TileLoader)
  uint32_t iter;           // tiles done by this CTA (ring phases)

  __device__ __forceinline__ static uint64_t* bar(int i) { return reinterpret_cast<uint64_t*>(tile_smem + C::BAR_OFF) + i; }
  __device__ __forceinline__ static uint64_t* full(int slot) { return bar(slot); }            // box landed
  __device__ __forceinline__ static uint64_t* cen_full() { return bar(C::NS); }               // centre tile landed
  __device__ __forceinline__ static uint64_t* rk_full(int r) { return bar(C::NS + 1 + r); }   // RK inputs landed
  // "empty" barriers, one arrival per warp: every warp is done with the ring slot / with the centre-value tile
  __device__ __forceinline__ static uint64_t* empty(int slot) { return bar(C::NS + 1 + C::RKD + slot); }
  __device__ __forceinline__ static uint64_t* cen_empty() { return bar(2 * C::NS + 1 + C::RKD); }
  __device__ __forceinline__ static uint64_t* rk_empty(int r) { return bar(2 * C::NS + 2 + C::RKD + r); }
  __device__ __forceinline__ static void init_barriers() {   // one thread
    for (int i = 0; i < C::NS + 1; ++i) tma::mbar_init(bar(i), 1);
    for (int i = C::NS + 1; i < C::NS + 1 + C::RKD; ++i) tma::mbar_init(bar(i), 2);   // the u_n and the acc producer
    for (int i = C::NS + 1 + C::RKD; i < C::NBAR; ++i) tma::mbar_init(bar(i), C::NW);   // "empty": one arrival per warp
    tma::fence_mbar_init();
  }

  // descriptors of this tile and of the CTA's next tile: two slots in shared memory, written by the producer
  __device__ __forceinline__ static TileId* desc() { return reinterpret_cast<TileId*>(tile_smem + C::DESC_OFF); }
  // map coordinates of the first active cell of a tile: map x coordinate c <-> storage cell c-1 (the maps start one
  // double before storage cell 0, on a 16-byte boundary), active cell i <-> storage cell i + NG
  __device__ __forceinline__ static int cx(const TileId& t) { return t.bx * C::TX + NG + 1; }
  __device__ __forceinline__ static int cy(const TileId& t) { return t.by * C::TY + NG; }
  __device__ __forceinline__ static int cz(const TileId& t) { return t.bz * C::TZ + NG; }

  __device__ __forceinline__ uint32_t strip(int d) const { return tm + 2u * (uint32_t)d; }    // double d of the strip

  // ring slot and use count of stream position s of tile `it` of this CTA: global sequence number it*NF + s
  __device__ __forceinline__ static uint32_t ring_slot(uint32_t it, int s) { return (it * Stream::N + s) % C::NS; }
  __device__ __forceinline__ static uint32_t ring_use(uint32_t it, int s) { return (it * Stream::N + s) / C::NS; }

  // ---- the producers' work: TMA requests with run-time field / slot numbers ---------------------------------------
  // stream position S of tile `it` (S >= N: position S - N of tile it + 1, whose descriptor is `t`)
  __device__ __forceinline__ static void issue_box(const TileMaps* maps, uint32_t it, int S, const TileId& t) {
    const int f = stream_field_rt(S >= Stream::N ? S - Stream::N : S);
    const uint32_t slot = ring_slot(it, S);
    tma::mbar_expect_tx(full(slot), C::BOX_BYTES);
    // the box starts XC cells before the first active cell in x (an even map coordinate) and NG in y, z
    tma::load_box(tile_smem + slot * C::SLOT, &maps->box[t.ip], full(slot), cx(t) - C::XC, cy(t) - NG, cz(t) - NG, f,
                  tma::SACRA_BOX_POLICY);
  }
  __device__ __forceinline__ static void issue_centre(const TileMaps* maps, const TileId& t) {
    tma::mbar_expect_tx(cen_full(), C::CEN_BYTES);
    tma::load_box(tile_smem + C::CEN_OFF, &maps->cen[t.ip], cen_full(), cx(t), cy(t), cz(t), 0, tma::SACRA_CEN_POLICY);
  }
  // RK input `which` (0: u_n, 1: acc) of emit e of tile t, the CTA's emit number q
  __device__ __forceinline__ static void issue_rk(const CUtensorMap* map, int which, uint32_t q, int e, const TileId& t) {
    const int f = emit_field_rt(e);
    const uint32_t r = q % C::RKD;
    tma::mbar_expect_tx(rk_full(r), C::NT * 8);
    tma::load_box(tile_smem + C::RK_OFF + (2 * r + which) * C::NT, map + t.ip, rk_full(r), cx(t), cy(t), cz(t), f,
                  tma::L2_EVICT_FIRST);
  }
  // field of stream position s / of emit e for a run-time index: the orders packed 5 bits per entry into constants
  template <class Fn>
  __host__ __device__ static constexpr uint64_t pack5(Fn fn, int first, int n) {
    uint64_t v = 0;
    for (int q = 0; q < n; ++q) v |= (uint64_t)fn(first + q) << (5 * q);
    return v;
  }
  __device__ __forceinline__ static int stream_field_rt(int sp) {
    constexpr int n0 = Stream::N < 12 ? Stream::N : 12, n1 = Stream::N - n0 < 12 ? Stream::N - n0 : 12;
    constexpr uint64_t a = pack5(Stream::field, 0, n0), b = pack5(Stream::field, 12, n1),
                       c = pack5(Stream::field, 24, Stream::N - n0 - n1);
    return (int)(((sp < 12 ? a >> (5 * sp) : sp < 24 ? b >> (5 * (sp - 12)) : c >> (5 * (sp - 24)))) & 31u);
  }
  __device__ __forceinline__ static int emit_field_rt(int e) {
    constexpr uint64_t a = pack5(emit_field, 0, 12), b = pack5(emit_field, 12, 12), c = pack5(emit_field, 24, 1);
    return (int)(((e < 12 ? a >> (5 * e) : e < 24 ? b >> (5 * (e - 12)) : c >> (5 * (e - 24)))) & 31u);
  }
  // The PRODUCERS: one lane each of up to three warps of the CTA's extra warpgroup owns the TMA requests of the CTA --
  // role 0 the stencil boxes and the centre-value tile, roles 1 and 2 (RK stages 2-4) the u_n and the acc tile of
  // every emit, so that the ~150 cycles one request costs its issuing thread are not spent in series. Each is a plain
  // ring producer: it walks the CTA's sequence of tiles and stream positions (emits), and before it refills a slot it
  // waits for the NW arrivals of the compute warps on the slot's "empty" barrier (box ring: made at the start of the
  // warps' field<>() call for the next position; RK ring: right after the emit has read its inputs). Every producer
  // waits for every phase of its barriers in order, and a phase cannot complete before the producer has filled the
  // slot for it, so the parity waits never alias.
  // Tile descriptors stay in the producers' registers; role 0 publishes them to the compute warps:
  // desc()[(it + 1) & 1] is written at the top of tile `it`, when every compute warp is inside tile it - 1 or later (it
  // read that entry at the end of tile it - 2); the compute warps read it at the end of tile `it`, after many waits
  // on "full" barriers armed later than the write.
  // `advance(t)`: the CTA's next tile after t (t + gridDim.x, or further when a partial launch skips tiles), >= ntiles
  // if there is none. Role 0 always publishes the next descriptor, with ip = -1 for "no more tiles": that is how the
  // compute warps learn that they are done.
  template <class Locate, class Advance>
  __device__ __forceinline__ static void producer(int role, const TileMaps* maps, int t, int ntiles, Locate locate,
                                                  Advance advance) {
    if (RK != 2 && role != 0) return;
    uint32_t it = 0;
    TileId cur = desc()[0], nxt = cur;
    int tn = advance(t);
    bool has_next = tn < ntiles;
    if (role == 0) {
      if (has_next) nxt = locate(tn);
      else nxt.ip = -1;
      desc()[1] = nxt;
      issue_centre(maps, cur);
#pragma unroll 1
      for (int S = 0; S < C::NS - 1; ++S) issue_box(maps, it, S, cur);
#pragma unroll 1
      for (;;) {
#pragma unroll 1
        for (int sp = 0; sp < Stream::N; ++sp) {
          const uint32_t g = it * Stream::N + sp;
          if (g > 0) tma::mbar_wait_idle(empty((g - 1u) % C::NS), ((g - 1u) / C::NS) & 1u);
          if (sp == 0 && has_next) {
            tma::mbar_wait_idle(cen_empty(), it & 1u);
            issue_centre(maps, nxt);
          }
          const int S = sp + C::NS - 1;
          if (S < Stream::N) issue_box(maps, it, S, cur);
          else if (has_next) issue_box(maps, it, S, nxt);
        }
        if (!has_next) break;
        t = tn;
        ++it;
        cur = nxt;
        tn = advance(t);
        has_next = tn < ntiles;
        if (has_next) nxt = locate(tn);
        else nxt.ip = -1;
        desc()[(it + 1u) & 1u] = nxt;
      }
    } else {
      const CUtensorMap* map = role == 1 ? maps->un : maps->acc;
      uint32_t q = 0;                                           // emit number of the CTA
#pragma unroll 1
      for (;;) {
#pragma unroll 1
        for (int e = 0; e < NF; ++e, ++q) {
          if (q >= (uint32_t)C::RKD) tma::mbar_wait_idle(rk_empty(q % C::RKD), (q / C::RKD - 1u) & 1u);
          issue_rk(map, role - 1, q, e, cur);
        }
        if (!has_next) break;
        t = tn;
        cur = locate(t);
        tn = advance(t);
        has_next = tn < ntiles;
      }
    }
  }

  // one arrival per warp on an "empty" barrier, after every lane's reads
  __device__ __forceinline__ void warp_arrive(uint64_t* b) const {
    __syncwarp();
    if ((tid & 31) == 0) tma::mbar_arrive(b);
  }
  // start of a tile: every thread copies its centre values from the shared-memory tile into its Tensor Memory strip
  // (slot order of cen_slot()). When every warp has done so the buffer is free and the producer requests the next
  // tile's values.
  __device__ __forceinline__ void begin_tile() const {
    tma::mbar_wait(cen_full(), iter & 1u);
    const double* c = tile_smem + C::CEN_OFF + tid;
#pragma unroll
    for (int q = 0; q < 24; q += 4)
      tmem::st4(strip(q), c[cen_field(q) * C::NT], c[cen_field(q + 1) * C::NT], c[cen_field(q + 2) * C::NT],
                c[cen_field(q + 3) * C::NT]);
    tmem::st1(strip(24), c[cen_field(24) * C::NT]);
    warp_arrive(cen_empty());
    tmem::wait_st();
  }

  // Advance to field F. No CTA-wide barrier: the warp releases the ring slot of the previous stream position (one
  // arrival per warp on its "empty" barrier; program order puts every read of that slot, and every read of the RK
  // ring by the emits so far, before it) and waits for the box of F. The producer refills a slot when all NW warps
  // have released it, so a warp runs at most NS - 1 fields ahead of the slowest one.
  template <int F>
  __device__ __forceinline__ auto field() const {
    constexpr int s = Stream::slot(F);
    static_assert(s >= 0, "field not in this kernel's stream");
    const uint32_t g = iter * Stream::N + s;         // sequence number of this stream position in the CTA's ring
    if (s > 0 || iter > 0) {
      const uint32_t prev = g - 1u;
      warp_arrive(empty(prev % C::NS));
    }
    tma::mbar_wait(full(g % C::NS), (g / C::NS) & 1u);
    return TileLoader<C>{sc + (int)(g % C::NS) * C::SLOT, ey, ez, xh, yh};
  }

  // derivative bundle of field F: its tile from the ring, then the stencils
  template <int F, bool D1, bool D2>
  __device__ __forceinline__ void derivs(const PointCoef& pc, Stencil& S) const {
    field_derivs<D1, D2>(field<F>(), pc, S);
  }

  // RK inputs of field F at this point (stages 2-4): waits for the ring slot of its emit
  template <int F>
  __device__ __forceinline__ void rk_inputs(double& un, double& acc) const {
    constexpr int e = emit_slot(F);
    const uint32_t q = iter * NF + e, r = q % C::RKD;          // emit sequence number of the CTA, ring position
    tma::mbar_wait(rk_full(r), (q / C::RKD) & 1u);
    un = tile_smem[C::RK_OFF + 2 * r * C::NT + tid];
    acc = tile_smem[C::RK_OFF + (2 * r + 1) * C::NT + tid];
    warp_arrive(rk_empty(r));
  }
};

}  // namespace sacra
