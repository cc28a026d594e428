// sacra.cu -- libsacra: C ABI (include/sacra.h) and the CUDA kernels behind it, sm_100a only.
//
// Kernels
//   k_fill_ghosts   halo fill, periodic or mirror per axis
//   k_z4c<EPI>      derivative stage + algebra + KO + epilogue (EPI 0: RHS store, 1..4: RK4 substage), one thread
//                   per active point, persistent CTAs on TMA-staged tiles;
//                   EPI -1: the constraint monitor on the same machinery
//   k_con_partial, k_con_final   deterministic volume-normalised L2 norms of the constraints (Eq. 22)
// There is no CPU path: every entry point enqueues kernels on the caller's stream or returns an error.
#include <cmath>
#include <cstdint>
#include <mutex>
#include <cuda_runtime.h>
#include <type_traits>

#include "../../include/sacra.h"
#include "z4c_fused.cuh"
#include "z4c_tile.cuh"
#include "z4c_constraints.cuh"

namespace sacra {

struct DevPatch {
  int nx, ny, nz;
  long long pitch, sz;     // doubles per x-row, doubles per z-plane
  long long fstride, offset;
  double dx, dt;
  GridCoef gc;             // 1/(12 h) ... of the derivative stage (launch_z4c fills in the KO factor)
  unsigned shell;          // bit 2a + side: that face is a Sommerfeld face (its 3 outermost layers are the boundary shell)
  unsigned xshell;         // bit 2a + side: ghosts behind that face come from a halo exchange (partial launches, below)
};
struct PatchBatch {
  DevPatch p[MAXP];
  int first_block[MAXP + 1];   // prefix sum of blocks per patch (block -> patch lookup)
  int np;
  // 0: every active cell. Partial launches for the overlap of the halo exchange with the computation: 1 = the cells
  // that need no exchanged ghost (more than 3 cells from every xshell face), 2 = the others, tiles without any skipped
  int part;
};

// ---------------------------------------------------------------------------------------------------
// Halo fill. Per axis: periodic (item 2; stands in for the paper's ghost exchange) or mirror (SURVEY 8(f) f-2,
// reflection symmetry about a face; the value comes with the parity of the field under x^a -> -x^a).
// Only ghost cells are written and only active cells are read (every source index is mapped into the active range),
// so reads and writes never overlap.
// ---------------------------------------------------------------------------------------------------
struct RkArgs {   // RK4 inputs / outputs of a substage (stage table of item 11)
  const double* u_n;
  double* u_out;
  double* acc;
};

struct FillModes {
  unsigned char m[MAXP][6];   // per patch and face (x- x+ y- y+ z- z+): 0 periodic, 1 mirror, 2 Sommerfeld, 3 none
};
// -1 for the a-component of a vector and for tensor components with exactly one index a
__device__ __forceinline__ double field_parity(int f, int axis) {
  if (f >= F_GAM && f < F_GAM + 3) return f - F_GAM == axis ? -1.0 : 1.0;
  if (f >= F_BET && f < F_BET + 3) return f - F_BET == axis ? -1.0 : 1.0;
  if (f >= F_B && f < F_B + 3) return f - F_B == axis ? -1.0 : 1.0;
  int n = -1;
  if (f >= F_G && f < F_G + 6) n = f - F_G;
  if (f >= F_A && f < F_A + 6) n = f - F_A;
  if (n < 0) return 1.0;
  // packed xx xy xz yy yz zz: components with exactly one index equal to `axis`
  const int one[3] = {0b000110, 0b010010, 0b010100};   // x: xy xz | y: xy yz | z: xz yz
  return (one[axis] >> n) & 1 ? -1.0 : 1.0;
}
// storage index of the source cell of storage index I along an axis with n active cells and face modes lo / hi;
// *refl: a mirror was used; *skip: the cell lies behind a face whose ghosts are not ours to fill (Sommerfeld, none)
__device__ __forceinline__ int fill_source(int I, int n, int lo, int hi, bool* refl, bool* skip) {
  const int i = I - NG;
  *refl = false;
  if (i >= 0 && i < n) return I;
  const int mode = i < 0 ? lo : hi;
  if (mode >= 2) {
    *skip = true;
    return I;
  }
  if (mode == 0) return (i < 0 ? i + n : i - n) + NG;
  *refl = true;
  return (i < 0 ? -1 - i : 2 * n - 1 - i) + NG;
}

__global__ void __launch_bounds__(256) k_fill_ghosts(const __grid_constant__ PatchBatch B, const __grid_constant__ FillModes modes,
                                                     double* __restrict__ u) {
  int ip = 0;
#pragma unroll 1
  while (ip + 1 < B.np && (int)blockIdx.x >= B.first_block[ip + 1]) ++ip;
  const DevPatch& p = B.p[ip];
  const unsigned char* m = modes.m[ip];
  const int sx = p.nx + 2 * NG, sy = p.ny + 2 * NG;
  // one block = one storage plane K of one field: a ghost plane is copied whole, an active plane only
  // has its 6 ghost rows and the 3+3 x-ghosts of its active rows
  const int f = blockIdx.y;
  const int Kk = (int)blockIdx.x - B.first_block[ip];
  bool rz, ry, rx, skz = false;
  const int Ks = fill_source(Kk, p.nz, m[4], m[5], &rz, &skz);
  if (skz) return;
  const bool plane_ghost = Ks != Kk;
  const double pz = rz ? field_parity(f, 2) : 1.0, py = field_parity(f, 1), px = field_parity(f, 0);
  double* fld = u + p.offset + (long long)f * p.fstride;
  double* dst = fld + (long long)Kk * p.sz;
  const double* src = fld + (long long)Ks * p.sz;
  auto copy_row = [&](int J) {   // one warp: the whole storage row J of this plane
    bool sky = false;
    const int Js = fill_source(J, p.ny, m[2], m[3], &ry, &sky);
    if (sky) return;
    const double s = pz * (ry ? py : 1.0);
    for (int I = threadIdx.x % 32; I < sx; I += 32) {
      bool skx = false;
      const int Is = fill_source(I, p.nx, m[0], m[1], &rx, &skx);
      if (!skx) dst[(long long)J * p.pitch + I] = (rx ? s * px : s) * src[(long long)Js * p.pitch + Is];
    }
  };
  // blockIdx.z splits the work of a plane: a whole ghost plane copied by one block is a chain of ~300 dependent
  // DRAM round trips per warp (measured 0.31 ms per call at 256^3, all of it the six ghost planes)
  const int nw = (blockDim.x / 32) * gridDim.z, w = (threadIdx.x / 32) * gridDim.z + blockIdx.z;   // warps of the plane
  if (plane_ghost) {
    for (int J = w; J < sy; J += nw) copy_row(J);
  } else {
    for (int r = w; r < 2 * NG; r += nw) copy_row(r < NG ? r : p.ny + r);   // ghost rows
    for (int q = threadIdx.x + blockDim.x * blockIdx.z; q < p.ny * 2 * NG; q += blockDim.x * gridDim.z) {   // x-ghosts
      const int J = q / (2 * NG) + NG, c = q % (2 * NG);
      const int I = c < NG ? c : p.nx + c;
      bool skx = false;
      const int Is = fill_source(I, p.nx, m[0], m[1], &rx, &skx);
      if (!skx) dst[(long long)J * p.pitch + I] = (rx ? px : 1.0) * src[(long long)J * p.pitch + Is];
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// Sommerfeld boundary shell (Eq. 13): on the active cells within NG cells of a
// Sommerfeld face the right-hand side of every field is  -( x^i d_i Q / r + Q / r ),  Q = u - flat value, with 4th-order
// differences that use existing cells only (centred / lopsided / one-sided). Same operation order as the oracle
// (oracle-independent restatement of DESIGN.md section 5.4; the library is built without FMA contraction): bit-identical.
// EPI as in the substage kernel: 0 stores the RHS, 1..5 apply the RK4 stage table to the shell cells.
// One block per active z-plane and field; threads walk the plane and skip the cells outside the shell.
// ---------------------------------------------------------------------------------------------------
struct ShellGeom {
  double origin[MAXP][3];
};
__device__ __forceinline__ bool in_shell(unsigned s, const DevPatch& p, int i, int j, int k) {
  return ((s & 1u) && i < NG) || ((s & 2u) && i >= p.nx - NG) || ((s & 4u) && j < NG) || ((s & 8u) && j >= p.ny - NG) ||
         ((s & 16u) && k < NG) || ((s & 32u) && k >= p.nz - NG);
}
// does the tile [x0, x0 + tx) x [y0, y0 + ty) x [z0, z0 + tz) hold a cell within NG cells of a flagged exchange face?
__device__ __forceinline__ bool tile_touches_xshell(const DevPatch& p, int x0, int y0, int z0, int tx, int ty, int tz) {
  const unsigned s = p.xshell;
  return ((s & 1u) && x0 < NG) || ((s & 2u) && x0 + tx > p.nx - NG) || ((s & 4u) && y0 < NG) || ((s & 8u) && y0 + ty > p.ny - NG) ||
         ((s & 16u) && z0 < NG) || ((s & 32u) && z0 + tz > p.nz - NG);
}
// first derivative along a stride at index i of an axis whose usable index range is [lo, hi]
__device__ __forceinline__ double d1_bounded(const double* u, long long st, int i, int lo, int hi, double inv12h) {
  if (i - 2 >= lo && i + 2 <= hi) return (8.0 * (u[st] - u[-st]) - (u[2 * st] - u[-2 * st])) * inv12h;
  const int s = (i - 2 < lo) ? 1 : -1;
  const long long t = s * st;
  const double u0 = u[0];
  if (i - s >= lo && i - s <= hi)
    return (double)s * ((((18.0 * (u[t] - u0) - 3.0 * (u[-t] - u0)) - 6.0 * (u[2 * t] - u0)) + (u[3 * t] - u0)) * inv12h);
  return (double)s * ((((48.0 * (u[t] - u0) - 36.0 * (u[2 * t] - u0)) + 16.0 * (u[3 * t] - u0)) - 3.0 * (u[4 * t] - u0)) * inv12h);
}
template <int EPI>
__global__ void __launch_bounds__(256) k_sommerfeld(const __grid_constant__ PatchBatch B, const __grid_constant__ ShellGeom G,
                                                    const double* __restrict__ u_in, double* __restrict__ rhs,
                                                    const __grid_constant__ RkArgs rk) {
  int ip = 0;
#pragma unroll 1
  while (ip + 1 < B.np && (int)blockIdx.x >= B.first_block[ip + 1]) ++ip;
  const DevPatch& p = B.p[ip];
  if (!p.shell) return;
  const int k = (int)blockIdx.x - B.first_block[ip], f = blockIdx.y;
  const double h = p.dx, inv12h = 1.0 / (12.0 * h);
  const int lo[3] = {(p.shell & 1u) ? 0 : -NG, (p.shell & 4u) ? 0 : -NG, (p.shell & 16u) ? 0 : -NG};
  const int hi[3] = {(p.shell & 2u) ? p.nx - 1 : p.nx - 1 + NG, (p.shell & 8u) ? p.ny - 1 : p.ny - 1 + NG,
                     (p.shell & 32u) ? p.nz - 1 : p.nz - 1 + NG};
  const bool flat1 = f == F_W || f == F_G || f == F_G + 3 || f == F_G + 5 || f == F_ALP;
  const long long fo = p.offset + (long long)f * p.fstride;
  const double z = G.origin[ip][2] + (double)k * h;
  // Only the shell cells of plane k are visited (at 256^3 the shell is 7 % of the cells): a plane inside a z-shell is
  // shell as a whole; elsewhere the rows of the y-shells come first (ys rows of nx cells), then the xs = 0, 3 or 6
  // x-shell cells of each remaining row. n >= 6 keeps the low and high shell of an axis apart.
  const bool zsh = ((p.shell & 16u) && k < NG) || ((p.shell & 32u) && k >= p.nz - NG);
  const int ylo = (p.shell & 4u) ? NG : 0, yhi = (p.shell & 8u) ? NG : 0, ys = zsh ? p.ny : ylo + yhi;
  const int xlo = (p.shell & 1u) ? NG : 0, xs = xlo + ((p.shell & 2u) ? NG : 0);
  const int nrow = ys * p.nx, ncell = nrow + (p.ny - ys) * xs;
  for (int q = threadIdx.x; q < ncell; q += blockDim.x) {
    int i, j;
    if (q < nrow) {
      const int r = q / p.nx;
      i = q - r * p.nx;
      j = (zsh || r < ylo) ? r : p.ny - NG + (r - ylo);
    } else {
      const int r = (q - nrow) / xs, c = (q - nrow) - r * xs;
      j = ylo + r;
      i = c < xlo ? c : p.nx - NG + (c - xlo);
    }
    const long long c = fo + (long long)(k + NG) * p.sz + (long long)(j + NG) * p.pitch + (i + NG);
    const double* uc = u_in + c;
    const double x = G.origin[ip][0] + (double)i * h, y = G.origin[ip][1] + (double)j * h;
    const double dx_ = d1_bounded(uc, 1, i, lo[0], hi[0], inv12h);
    const double dy_ = d1_bounded(uc, p.pitch, j, lo[1], hi[1], inv12h);
    const double dz_ = d1_bounded(uc, p.sz, k, lo[2], hi[2], inv12h);
    const double r = sqrt((x * x + y * y) + z * z);
    const double Q = uc[0] - (flat1 ? 1.0 : 0.0);
    const double kk = -((((x * dx_ + y * dy_) + z * dz_) / r) + Q / r);
    if (EPI == 0) {
      rhs[c] = kk;
      continue;
    }
    const double un = rk.u_n[c], dt = p.dt;
    double acc_new, u_new;
    if (EPI == 1) {
      acc_new = kk;
      u_new = un + (dt / 2.0) * kk;
    } else if (EPI == 2) {
      acc_new = rk.acc[c] + 2.0 * kk;
      u_new = un + (dt / 2.0) * kk;
    } else if (EPI == 3) {
      acc_new = rk.acc[c] + 2.0 * kk;
      u_new = un + dt * kk;
    } else {
      acc_new = (rk.acc[c] + kk) * (1.0 / 6.0);
      u_new = un + dt * acc_new;
    }
    if (EPI != 5) rk.acc[c] = acc_new;
    rk.u_out[c] = u_new;
  }
}

// ---------------------------------------------------------------------------------------------------
// Fused substage kernel: persistent CTAs, one thread per active point of a TX x TY x TZ tile; the 25 fields
// are streamed through a TMA ring in shared memory (z4c_tile.cuh).
// ---------------------------------------------------------------------------------------------------
#ifndef SACRA_TX   // tile shape (threads per CTA = TX*TY*TZ) and ring depth: tuning builds
#define SACRA_TX 16
#define SACRA_TY 4
#define SACRA_TZ 6
#define SACRA_NS 4
#endif
using Tile = TileCfg<SACRA_TX, SACRA_TY, SACRA_TZ, SACRA_NS>;

// EPI: 0 = store RHS; 1..4 = RK4 substage (item 11 table); 5 = substage 4 without the store of the increment S
__host__ __device__ constexpr int rk_mode(int epi) { return epi == 0 ? 0 : (epi == 1 ? 1 : 2); }

// Consumes the finished RHS values. The RK4 inputs never come from global loads: at stage 1 u_n is the stage
// input itself (the centre sample of the field's own box), from stage 2 on u_n and acc arrive through the TMA ring
// of TileSource.
// active: out-of-range threads of a ragged tile run the same instruction stream on zero-filled data (they
// must reach every barrier) and store nothing.
template <int EPI, class Src>
struct Emitter {
  const Src& src;
  double* rhs;             // EPI == 0
  double* u_out;
  double* acc;
  long long o, fstride;    // offset of field 0 at this point, field stride
  double dt;
  bool active;
  // u0: the field's value at the point, which is u_n at stage 1
  template <int F>
  __device__ __forceinline__ void put(double kk, double u0) {
    const long long a = o + (long long)F * fstride;
    if (EPI == 0) {
      if (active) __stcs(rhs + a, kk);   // streaming store: written once, not re-read by this launch
      return;
    }
    double un = u0, ac = 0.0;
    if (EPI != 1) src.template rk_inputs<F>(un, ac);
    double acc_new, u_new;
    if (EPI == 1) {
      acc_new = kk;
      u_new = __dadd_rn(un, __dmul_rn(dt / 2.0, kk));
    } else if (EPI == 2) {
      acc_new = __dadd_rn(ac, __dmul_rn(2.0, kk));
      u_new = __dadd_rn(un, __dmul_rn(dt / 2.0, kk));
    } else if (EPI == 3) {
      acc_new = __dadd_rn(ac, __dmul_rn(2.0, kk));
      u_new = __dadd_rn(un, __dmul_rn(dt, kk));
    } else {   // stage 4; EPI 5: the same without the store of S (SACRA_FLAG_SKIP_INCREMENT)
      acc_new = __dmul_rn(__dadd_rn(ac, kk), 1.0 / 6.0);
      u_new = __dadd_rn(un, __dmul_rn(dt, acc_new));
    }
    if (active) {
      if (EPI != 5) __stcs(acc + a, acc_new);   // streaming stores: they must not evict the stencil boxes from L2
      __stcs(u_out + a, u_new);
    }
  }
};

// Tile order. Tile t of a patch is NOT tile (t % nbx, ...): consecutive tiles fill SUPER-BLOCKS of SBX x SBY x SBZ
// tiles (64 x 64 x 32 points; 512 tiles = 3.5 waves of the persistent grid), x fastest inside a super-block,
// super-blocks x fastest across the patch. The tiles in flight at any time then share their halos through L2
// (a super-block's boxes of all 25 fields are 38 MB of the 126 MB), and only super-block faces are read twice
// from HBM. With the plain x-y-z order a 256^3 patch re-read every z-halo plane from DRAM (one sweep of a 4-plane
// slab of 25 fields is 131 MB): 28.8 GB read per launch against 6.7 GB algorithmic.
// Only thread 0 decodes tile indices (several integer divisions); the CTA gets them through shared memory.
#ifndef SACRA_SBX
#define SACRA_SBX 16
#define SACRA_SBY 4
#define SACRA_SBZ 4
#endif
#ifndef SACRA_L2PROMO
#define SACRA_L2PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_128B
#endif
constexpr int SBX = SACRA_SBX, SBY = SACRA_SBY, SBZ = SACRA_SBZ;
template <class C>
__device__ __forceinline__ TileId locate_inl(const PatchBatch& B, int t) {
  TileId id;
  id.ip = 0;
#pragma unroll 1
  while (id.ip + 1 < B.np && t >= B.first_block[id.ip + 1]) ++id.ip;
  const DevPatch& p = B.p[id.ip];
  const int nbx = (p.nx + C::TX - 1) / C::TX, nby = (p.ny + C::TY - 1) / C::TY, nbz = (p.nz + C::TZ - 1) / C::TZ;
  int r = t - B.first_block[id.ip];
  // layers of super-blocks in z, rows in y, super-blocks in x: every earlier one is full along that axis
  const int sz = r / (nbx * nby * SBZ);
  r -= sz * (nbx * nby * SBZ);
  const int lz = min(SBZ, nbz - sz * SBZ);
  const int sy = r / (nbx * SBY * lz);
  r -= sy * (nbx * SBY * lz);
  const int ly = min(SBY, nby - sy * SBY);
  const int sx = r / (SBX * ly * lz);
  r -= sx * (SBX * ly * lz);
  const int lx = min(SBX, nbx - sx * SBX);
  id.bx = sx * SBX + r % lx;
  r /= lx;
  id.by = sy * SBY + r % ly;
  id.bz = sz * SBZ + r / ly;
  return id;
}
// EPI 0..4: Z4c right-hand side / RK4 substage; EPI == -1: constraint monitor (rhs receives H, M^x, M^y, M^z in
// fields 0..3)
template <int EPI>
__global__ void __launch_bounds__(Tile::NTH, 1) k_z4c(const __grid_constant__ PatchBatch B,
                                                      const __grid_constant__ Params P,
                                                      const __grid_constant__ TileMaps M,
                                                      double* __restrict__ rhs, const __grid_constant__ RkArgs rk) {
  using C = Tile;
  using Src = TileSource<C, rk_mode(EPI < 0 ? 0 : EPI), std::conditional_t<EPI < 0, ConStream, Z4cStream>>;
  const int ntiles = B.first_block[B.np];
  if ((int)blockIdx.x >= ntiles) return;
  // the CTA's tiles: blockIdx.x, + gridDim.x, ...; a shell-only launch (B.part == 2) skips the tiles without a shell cell
  auto selected = [&](int tt) {
    if (B.part != 2) return true;
    const TileId q = locate_inl<C>(B, tt);
    const DevPatch& pq = B.p[q.ip];
    return tile_touches_xshell(pq, q.bx * C::TX, q.by * C::TY, q.bz * C::TZ, C::TX, C::TY, C::TZ);
  };
  auto advance = [&](int tt) {
    do tt += (int)gridDim.x;
    while (tt < ntiles && !selected(tt));
    return tt;
  };
  // 1-D block of NT compute threads (thread q = point (q % TX, q / TX % TY, q / (TX TY)) of the tile) + one producer warp
  const int tid = threadIdx.x;
  TileId* desc = Src::desc();
  uint32_t* tm_base = reinterpret_cast<uint32_t*>(tile_smem + C::TMB_OFF);
  static_assert(sizeof(TileId) == 16, "descriptor slots");
  if (tid == 0) {
    int t0 = blockIdx.x;
    if (!selected(t0)) t0 = advance(t0);
    tm_base[1] = (uint32_t)t0;
    if (t0 < ntiles) desc[0] = locate_inl<C>(B, t0);
    Src::init_barriers();
  }
  if (tid < 32) tmem::alloc_all(tm_base);   // warp 0 owns the allocation (and frees it at the end)
  tmem::fence_before_sync();
  __syncthreads();
  tmem::fence_after_sync();
  const int t = (int)tm_base[1];   // the CTA's first tile
  // The kernel starts with 65536 / NTH = 128 registers per thread; the producer warpgroup hands its registers to the
  // compute warpgroups (a kernel that uses setmaxnreg must not contain calls: locate_inl)
  if (t >= ntiles) {
    // nothing to do for this CTA (partial launch)
  } else if (tid >= C::NT) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(C::REG_PRODUCER));
    if (tid % 32 == 0 && tid < C::NT + 96)
      Src::producer((tid - C::NT) / 32, &M, t, ntiles, [&](int tt) { return locate_inl<C>(B, tt); }, advance);
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(C::REG_COMPUTE));
    const int tx = tid % C::TX, ty = tid / C::TX % C::TY, tz = tid / (C::TX * C::TY);
    Src src;
    src.tid = tid;
    {
      // the strip of this thread: Tensor Memory lane 32 (warp % 4) + lane, columns of warp / 4
      const uint32_t warp = (uint32_t)tid / 32u;
      src.tm = *tm_base + (((warp & 3u) * 32u) << 16) + (warp >> 2) * (2u * C::TM_DOUBLES);
    }
    src.ey = C::EY_OFF + (tz * C::TY + ty) * C::EX + (tx + 2);
    src.ez = C::EZ_OFF + (tz * (C::TY + 4) + (ty + 2)) * C::EX + (tx + 2);
    src.xh = tx < 2 ? -2 : (tx >= C::TX - 2 ? 2 : 0);
    src.yh = ty < 2 ? -2 : 2;   // rows y-2 (y = 0, 1 -> -2, -1) and y+2 (y = 2, 3 -> TY, TY+1)
    src.sc = ((tz + NG) * C::PY + (ty + NG)) * C::PX + (tx + C::XC);
    TileId id = desc[0];
#pragma unroll 1
    for (uint32_t iter = 0;; ++iter) {
      const DevPatch& p = B.p[id.ip];
      src.iter = iter;
      const int i = id.bx * C::TX + tx, j = id.by * C::TY + ty, k = id.bz * C::TZ + tz;
      // cells of the Sommerfeld boundary shell belong to k_sommerfeld; a partial launch takes the cells inside / outside
      // the exchange shell only
      bool active = (i < p.nx) & (j < p.ny) & (k < p.nz) && !(p.shell && in_shell(p.shell, p, i, j, k));
      if (B.part) active = active && (in_shell(p.xshell, p, i, j, k) == (B.part == 2));
      const long long c = (long long)(k + NG) * p.sz + (long long)(j + NG) * p.pitch + (i + NG);
      Emitter<(EPI < 0 ? 0 : EPI), Src> emit{src, rhs, rk.u_out, rk.acc, p.offset + c, p.fstride, p.dt, active};
      src.begin_tile();
      if constexpr (EPI < 0) constraints_point(src, p.gc, emit);
      else z4c_point(src, P, p.gc, emit);
      id = desc[(iter + 1) & 1u];   // written by the producer at the top of this tile; ip < 0: no more tiles
      if (id.ip < 0) break;
    }
  }
  tmem::fence_before_sync();
  __syncthreads();                // every thread is done with its strip
  if (tid < 32) tmem::dealloc_all(*tm_base);
}


// ---------------------------------------------------------------------------------------------------
// Norms of the constraints, Eq. 22: sqrt( sum C^2 dV / sum dV ) over the active cells of all
// patches. Deterministic: k_con_partial sums C^2 over one storage plane per block in a fixed order (thread t sums
// cells t, t + 256, ... of the plane; fixed-shape tree over the threads), k_con_final adds the per-plane sums in
// plane order with one thread per constraint. The same input gives the same bits on every run.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_con_partial(const __grid_constant__ PatchBatch B, const double* __restrict__ con,
                                                     double* __restrict__ part, int part_base) {
  __shared__ double red[4][256];
  int ip = 0;
#pragma unroll 1
  while (ip + 1 < B.np && (int)blockIdx.x >= B.first_block[ip + 1]) ++ip;
  const DevPatch& p = B.p[ip];
  const int k = (int)blockIdx.x - B.first_block[ip];                 // active plane
  const double* base = con + p.offset + (long long)(k + NG) * p.sz + (long long)NG * p.pitch + NG;
  double acc[4] = {0.0, 0.0, 0.0, 0.0};
  for (int q = threadIdx.x; q < p.nx * p.ny; q += 256) {
    const long long c = (long long)(q / p.nx) * p.pitch + (q % p.nx);
#pragma unroll
    for (int n = 0; n < 4; ++n) {
      const double v = base[(long long)n * p.fstride + c];
      acc[n] = fma(v, v, acc[n]);
    }
  }
#pragma unroll
  for (int n = 0; n < 4; ++n) red[n][threadIdx.x] = acc[n];
  __syncthreads();
  for (int s = 128; s > 0; s >>= 1) {
    if ((int)threadIdx.x < s)
#pragma unroll
      for (int n = 0; n < 4; ++n) red[n][threadIdx.x] += red[n][threadIdx.x + s];
    __syncthreads();
  }
  if (threadIdx.x < 4) part[(long long)(part_base + blockIdx.x) * 4 + threadIdx.x] = red[threadIdx.x][0] * ((p.dx * p.dx) * p.dx);
}
// part: nplanes x 4 weighted sums, vol = sum of dV over all active cells; one block of 4 threads
__global__ void k_con_final(const double* __restrict__ part, int nplanes, double vol, double* __restrict__ norms) {
  const int n = threadIdx.x;
  double s = 0.0;
  for (int q = 0; q < nplanes; ++q) s += part[(long long)q * 4 + n];
  norms[n] = sqrt(s / vol);
}

// ---------------------------------------------------------------------------------------------------
// Spatial inter-level operators of the box-in-box hierarchy, 2:1 cell-centred
// staggered grids: along each axis the parent cell org + m holds the child cells 2m and 2m+1. Tensor products of
// 1-D Lagrange interpolation; the weights are exact dyadic fractions. One thread per target cell and field, sums
// nested z(y(x)) like the oracle's. HBM/L2-bound and small next to the substage kernel.
// ---------------------------------------------------------------------------------------------------
struct LevelPair {
  DevPatch parent, child;
  int org[3];
};
// restriction: 4 points per axis at the midpoint between child cells 2m and 2m+1 (nodes 2m-1 .. 2m+2)
__global__ void __launch_bounds__(128) k_restrict(const __grid_constant__ LevelPair L, double* __restrict__ u_parent,
                                                  const double* __restrict__ u_child) {
  const DevPatch& pp = L.parent;
  const DevPatch& pc = L.child;
  const int hx = pc.nx / 2, hy = pc.ny / 2, hz = pc.nz / 2;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= hx * hy * hz) return;
  const int mx = t % hx, my = (t / hx) % hy, mz = t / (hx * hy);
  const double w[4] = {-1.0 / 16.0, 9.0 / 16.0, 9.0 / 16.0, -1.0 / 16.0};
  const double* fc = u_child + pc.offset + (long long)blockIdx.y * pc.fstride +
                     (long long)(2 * mz - 1 + NG) * pc.sz + (long long)(2 * my - 1 + NG) * pc.pitch + (2 * mx - 1 + NG);
  double az = 0.0;
#pragma unroll
  for (int kz = 0; kz < 4; ++kz) {
    double ay = 0.0;
#pragma unroll
    for (int ky = 0; ky < 4; ++ky) {
      double ax = 0.0;
#pragma unroll
      for (int kx = 0; kx < 4; ++kx) ax = ax + w[kx] * fc[(long long)kz * pc.sz + (long long)ky * pc.pitch + kx];
      ay = ay + w[ky] * ax;
    }
    az = az + w[kz] * ay;
  }
  u_parent[pp.offset + (long long)blockIdx.y * pp.fstride + (long long)(L.org[2] + mz + NG) * pp.sz +
           (long long)(L.org[1] + my + NG) * pp.pitch + (L.org[0] + mx + NG)] = az;
}
// prolongation of the child's ghost cells: 6 points per axis a quarter of a parent spacing off the parent cell that
// holds the child cell (to the left for an even child cell, to the right for an odd one: mirrored weights).
// One thread per PARENT cell m = (mx, my, mz) of the child's storage range (m = -2 .. n/2 + 1 per axis) and field: the
// up to eight child cells 2m + (0|1) it holds share the 7 x 7 x 7 parent values m - 3 .. m + 3 (an even child cell uses
// the first six per axis, an odd one the last six with the mirrored weights), so the x sums of a parent row serve two
// cells, the y sums four and a thread makes 343 loads for eight cells instead of 8 x 216. Every cell's sum is still
// nested z(y(x)), terms in ascending order from 0.0: the same bits as the one-cell-per-thread form and as the oracle.
// Only ghost cells are written; parent values that no ghost cell of the group needs are not loaded (they may lie
// outside the parent's storage at the last group of an axis).
__global__ void __launch_bounds__(128) k_prolong_ghosts(const __grid_constant__ LevelPair L, const double* __restrict__ u_parent,
                                                        double* __restrict__ u_child) {
  const DevPatch& pp = L.parent;
  const DevPatch& pc = L.child;
  const int gx = pc.nx / 2 + 4, gy = pc.ny / 2 + 4, gz = pc.nz / 2 + 4;     // parent cells that hold storage cells of the child
  // the groups that hold ghost cells form a shell two parent cells thick: 4 whole z layers, then 4 rows of every other
  // layer, then 4 cells of every other row (x fastest inside each part, so that a warp works on neighbouring groups)
  const int nzs = 4 * gx * gy, nys = 4 * gx * (gz - 4), nxs = 4 * (gy - 4) * (gz - 4);
  int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= nzs + nys + nxs) return;
  int m[3];
  auto edge = [](int q, int g) { return q < 2 ? q - 2 : g - 6 + q; };   // q = 0..3 -> -2, -1, g - 4, g - 3
  if (t < nzs) {
    m[0] = t % gx - 2; m[1] = (t / gx) % gy - 2; m[2] = edge(t / (gx * gy), gz);
  } else if (t < nzs + nys) {
    t -= nzs;
    m[0] = t % gx - 2; m[1] = edge((t / gx) % 4, gy); m[2] = t / (gx * 4);
  } else {
    t -= nzs + nys;
    m[0] = edge(t % 4, gx); m[1] = (t / 4) % (gy - 4); m[2] = t / (4 * (gy - 4));
  }
  const int nc[3] = {pc.nx, pc.ny, pc.nz};
  // per axis and parity: is child cell i = 2m + parity inside the child's storage, and is it a ghost cell along that axis?
  bool in[3][2], gh[3][2];
  bool any_ghost_axis = false;
#pragma unroll
  for (int a = 0; a < 3; ++a)
#pragma unroll
    for (int q = 0; q < 2; ++q) {
      const int i = 2 * m[a] + q;
      in[a][q] = i >= -NG && i < nc[a] + NG;
      gh[a][q] = in[a][q] && (i < 0 || i >= nc[a]);
      any_ghost_axis = any_ghost_axis || gh[a][q];
    }
  if (!any_ghost_axis) return;   // a group of active cells only
  const double we[6] = {63.0 / 8192.0, -495.0 / 8192.0, 2310.0 / 8192.0, 6930.0 / 8192.0, -693.0 / 8192.0, 77.0 / 8192.0};
  const double* fp = u_parent + pp.offset + (long long)blockIdx.y * pp.fstride + (long long)(L.org[2] + m[2] - 3 + NG) * pp.sz +
                     (long long)(L.org[1] + m[1] - 3 + NG) * pp.pitch + (L.org[0] + m[0] - 3 + NG);
  double az[2][2][2];            // [z parity][y parity][x parity]
#pragma unroll
  for (int c = 0; c < 8; ++c) az[c >> 2][(c >> 1) & 1][c & 1] = 0.0;
#pragma unroll
  for (int kz = 0; kz < 7; ++kz) {
    // plane kz serves the even cell if kz < 6 and the odd one if kz > 0
    if (!((kz < 6 && in[2][0]) || (kz > 0 && in[2][1]))) continue;
    double ay[2][2];             // [y parity][x parity]
    ay[0][0] = ay[0][1] = ay[1][0] = ay[1][1] = 0.0;
#pragma unroll
    for (int ky = 0; ky < 7; ++ky) {
      if (!((ky < 6 && in[1][0]) || (ky > 0 && in[1][1]))) continue;
      const double* row = fp + (long long)kz * pp.sz + (long long)ky * pp.pitch;
      double v[7];
#pragma unroll
      for (int kx = 0; kx < 7; ++kx) v[kx] = ((kx < 6 && in[0][0]) || (kx > 0 && in[0][1])) ? row[kx] : 0.0;
      double axe = 0.0, axo = 0.0;
#pragma unroll
      for (int kx = 0; kx < 6; ++kx) {
        axe = axe + we[kx] * v[kx];            // even cell: nodes m-3 .. m+2
        axo = axo + we[5 - kx] * v[kx + 1];    // odd cell:  nodes m-2 .. m+3, mirrored weights
      }
      if (ky < 6) { ay[0][0] = ay[0][0] + we[ky] * axe; ay[0][1] = ay[0][1] + we[ky] * axo; }
      if (ky > 0) { ay[1][0] = ay[1][0] + we[6 - ky] * axe; ay[1][1] = ay[1][1] + we[6 - ky] * axo; }
    }
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      if (kz < 6) az[0][c >> 1][c & 1] = az[0][c >> 1][c & 1] + we[kz] * ay[c >> 1][c & 1];
      if (kz > 0) az[1][c >> 1][c & 1] = az[1][c >> 1][c & 1] + we[6 - kz] * ay[c >> 1][c & 1];
    }
  }
  double* fc = u_child + pc.offset + (long long)blockIdx.y * pc.fstride;
#pragma unroll
  for (int c = 0; c < 8; ++c) {
    const int qz = c >> 2, qy = (c >> 1) & 1, qx = c & 1;
    if (!(in[0][qx] && in[1][qy] && in[2][qz])) continue;
    if (!(gh[0][qx] || gh[1][qy] || gh[2][qz])) continue;       // an active cell
    fc[(long long)(2 * m[2] + qz + NG) * pc.sz + (long long)(2 * m[1] + qy + NG) * pc.pitch + (2 * m[0] + qx + NG)] = az[qz][qy][qx];
  }
}

// Halo exchange between the patches of a block decomposition ("pack, then non-blocking
// GPU-aware exchange"): the NG outermost ACTIVE layers at a face go into a contiguous buffer [field][layer][row][col]
// (the two other axes over their whole STORAGE extent, so that exchanging x, then y, then z also fills edges and
// corners), and a received buffer goes into the NG GHOST layers of a face. PACK: true = pack, false = unpack.
template <bool PACK>
__global__ void __launch_bounds__(256) k_face(const __grid_constant__ DevPatch p, int axis, int side,
                                              double* __restrict__ u, double* __restrict__ buf) {
  const int s[3] = {p.nx + 2 * NG, p.ny + 2 * NG, p.nz + 2 * NG}, n[3] = {p.nx, p.ny, p.nz};
  const int a1 = axis == 0 ? 1 : 0, a2 = axis == 2 ? 1 : 2;       // the other two axes, the faster one first
  const long long st[3] = {1, p.pitch, p.sz};
  const int f = blockIdx.y, l = blockIdx.x;                          // field, layer
  // storage index of the layer: active layers [NG, 2NG) / [n, n + NG) when packing, ghost layers when unpacking
  const int L = PACK ? (side == 0 ? NG + l : n[axis] + l) : (side == 0 ? l : n[axis] + NG + l);
  double* base = u + p.offset + (long long)f * p.fstride + (long long)L * st[axis];
  double* b = buf + ((long long)f * NG + l) * s[a1] * s[a2];
  for (int q = threadIdx.x + blockDim.x * blockIdx.z; q < s[a1] * s[a2]; q += blockDim.x * gridDim.z) {
    const long long c = (long long)(q % s[a1]) * st[a1] + (long long)(q / s[a1]) * st[a2];
    if (PACK) b[q] = base[c];
    else base[c] = b[q];
  }
}

// linear combination of up to three states on every storage cell of a patch (time interpolation of the parent levels,
// SURVEY 8(f) f-3): out = (w0 u0 + w1 u1) [+ w2 u2], one rounding per operation like the oracle's
struct LinComb {
  const double* u[3];
  double w[3];
  int n;
  int lo[3], hi[3];   // storage-index box [lo, hi) per axis (x, y, z) the combination is formed on
};
__global__ void __launch_bounds__(256) k_lincomb(const __grid_constant__ DevPatch p, const __grid_constant__ LinComb L,
                                                 double* __restrict__ out) {
  const int sx = L.hi[0] - L.lo[0], sy = L.hi[1] - L.lo[1];
  const long long c0 = p.offset + (long long)blockIdx.y * p.fstride + (long long)(L.lo[2] + (int)blockIdx.x) * p.sz +
                       (long long)L.lo[1] * p.pitch + L.lo[0];
  for (int q = threadIdx.x; q < sx * sy; q += blockDim.x) {
    const long long c = c0 + (long long)(q / sx) * p.pitch + (q % sx);
    double s = L.w[0] * L.u[0][c] + L.w[1] * L.u[1][c];
    if (L.n == 3) s = s + L.w[2] * L.u[2][c];
    out[c] = s;
  }
}

// ---------------------------------------------------------------------------------------------------
// Host side: validation and launches
// ---------------------------------------------------------------------------------------------------
static bool aligned16(const void* q) { return (reinterpret_cast<uintptr_t>(q) & 15u) == 0; }

static int check_patches(const sacra_patch_t* p, int npatch) {
  if (!p) return SACRA_ERR_NULL;
  if (npatch < 1) return SACRA_ERR_BADARG;
  for (int q = 0; q < npatch; ++q) {
    const sacra_patch_t& a = p[q];
    if (a.ng != SACRA_NG) return SACRA_ERR_UNSUPPORTED;
    if (a.nx < 6 || a.ny < 6 || a.nz < 6) return SACRA_ERR_BADARG;
    if (!(a.dx > 0.0) || !std::isfinite(a.dx) || !std::isfinite(a.dt)) return SACRA_ERR_BADARG;
    if (a.pitch_x < a.nx + 2 * SACRA_NG) return SACRA_ERR_BADARG;
    if (a.patch_offset < 0) return SACRA_ERR_BADARG;
    const long long need = (long long)a.pitch_x * (a.ny + 2 * SACRA_NG) * (a.nz + 2 * SACRA_NG);
    if (a.field_stride < need) return SACRA_ERR_BADARG;
    if ((a.pitch_x & 1) || (a.field_stride & 1) || ((a.patch_offset + SACRA_NG) & 1)) return SACRA_ERR_ALIGN;
  }
  return SACRA_OK;
}

// doubles from a state's base pointer to the end of its last patch
static long long state_extent(const sacra_patch_t* p, int npatch) {
  long long ext = 0;
  for (int q = 0; q < npatch; ++q) {
    const long long need = (long long)p[q].pitch_x * (p[q].ny + 2 * SACRA_NG) * (p[q].nz + 2 * SACRA_NG);
    const long long e = p[q].patch_offset + (long long)(SACRA_NF - 1) * p[q].field_stride + need;
    if (e > ext) ext = e;
  }
  return ext;
}
// do [a, a + na) and [b, b + nb) (in doubles) share a byte?
static bool overlap(const double* a, long long na, const double* b, long long nb) {
  const uintptr_t a0 = reinterpret_cast<uintptr_t>(a), b0 = reinterpret_cast<uintptr_t>(b);
  return a0 < b0 + (uintptr_t)nb * 8u && b0 < a0 + (uintptr_t)na * 8u;
}

static DevPatch to_dev(const sacra_patch_t& a) {
  DevPatch d;
  d.nx = a.nx; d.ny = a.ny; d.nz = a.nz;
  d.pitch = a.pitch_x; d.sz = a.pitch_x * (long long)(a.ny + 2 * NG);
  d.fstride = a.field_stride; d.offset = a.patch_offset; d.dx = a.dx; d.dt = a.dt;
  d.shell = 0;
  d.xshell = 0;
  d.gc = grid_coef(a.dx, 0.0);
  return d;
}

static Params to_dev(const sacra_params_t& a) {
  Params P;
  P.kappa1 = a.kappa1; P.kappa2 = a.kappa2; P.eta = a.eta; P.shift_coef = a.shift_coef;
  P.ko_sigma = a.ko_sigma; P.lapse_uses_khat = a.lapse_uses_khat;
  return P;
}

// face modes of every patch: `axis_mode` (one mode per axis, both faces, every patch) or `bnd` (per patch and face)
static int launch_fill(const sacra_patch_t* p, int npatch, double* u, cudaStream_t st, const int32_t* axis_mode = nullptr,
                       const sacra_boundary_t* bnd = nullptr) {
  for (int q0 = 0; q0 < npatch; q0 += MAXP) {
    PatchBatch B;
    B.part = 0;
    FillModes M;
    B.np = (npatch - q0 < MAXP) ? npatch - q0 : MAXP;
    int nb = 0, split = 1;
    for (int q = 0; q < B.np; ++q) {
      B.p[q] = to_dev(p[q0 + q]);
      for (int a = 0; a < 6; ++a)
        M.m[q][a] = (unsigned char)(bnd ? bnd[q0 + q].face[a] : (axis_mode ? axis_mode[a / 2] : SACRA_BC_PERIODIC));
      B.first_block[q] = nb;
      nb += p[q0 + q].nz + 2 * NG;
      const long long plane = (long long)(p[q0 + q].nx + 2 * NG) * (p[q0 + q].ny + 2 * NG);
      const int want = plane / 8192 < 1 ? 1 : (plane / 8192 > 8 ? 8 : (int)(plane / 8192));
      if (want > split) split = want;   // blocks per plane: only big planes are worth splitting
    }
    B.first_block[B.np] = nb;
    k_fill_ghosts<<<dim3(nb, NF, split), 256, 0, st>>>(B, M, u);
    if (cudaGetLastError() != cudaSuccess) return SACRA_ERR_CUDA;
  }
  return SACRA_OK;
}

static int check_boundaries(const sacra_boundary_t* bnd, int npatch) {
  if (!bnd) return SACRA_ERR_NULL;
  for (int q = 0; q < npatch; ++q) {
    for (int a = 0; a < 6; ++a)
      if (bnd[q].face[a] < SACRA_BC_PERIODIC || bnd[q].face[a] > SACRA_BC_NONE) return SACRA_ERR_BADARG;
    for (int a = 0; a < 3; ++a) {
      if (!std::isfinite(bnd[q].origin[a])) return SACRA_ERR_BADARG;
      // a periodic axis is periodic on both faces
      if ((bnd[q].face[2 * a] == SACRA_BC_PERIODIC) != (bnd[q].face[2 * a + 1] == SACRA_BC_PERIODIC)) return SACRA_ERR_BADARG;
    }
  }
  return SACRA_OK;
}
static unsigned shell_bits(const sacra_boundary_t& b) {
  unsigned s = 0;
  for (int a = 0; a < 6; ++a)
    if (b.face[a] == SACRA_BC_SOMMERFELD) s |= 1u << a;
  return s;
}
// Eq. 13 divides by r: a cell of a Sommerfeld shell that sits exactly at the coordinate origin (r = 0 in the kernel's
// own arithmetic, x = origin + i h with a rounded product) would put NaN into u_out and acc without any error.
// Checked on the host before anything is launched (sacra.h: "the origin of the coordinates must not be a cell of a
// boundary shell").
static int check_shell_origin(const sacra_patch_t* p, const sacra_boundary_t* bnd, int npatch) {
  for (int q = 0; q < npatch; ++q) {
    const unsigned s = shell_bits(bnd[q]);
    if (!s) continue;
    const int n[3] = {p[q].nx, p[q].ny, p[q].nz};
    int zero[3] = {-1, -1, -1};   // index of the cell whose coordinate along the axis is exactly 0, if any
    for (int a = 0; a < 3; ++a) {
      const double g = -bnd[q].origin[a] / p[q].dx;
      if (!(g > -1.0 && g < (double)n[a])) continue;
      for (long long i = (long long)g - 1; i <= (long long)g + 2; ++i) {
        if (i < 0 || i >= n[a]) continue;
        volatile double prod = (double)i * p[q].dx;   // rounded product, as the kernel forms it (no FMA there)
        if (bnd[q].origin[a] + prod == 0.0) zero[a] = (int)i;
      }
    }
    if (zero[0] < 0 || zero[1] < 0 || zero[2] < 0) continue;
    bool hit = false;
    for (int a = 0; a < 3; ++a)
      hit = hit || ((s >> (2 * a) & 1u) && zero[a] < NG) || ((s >> (2 * a + 1) & 1u) && zero[a] >= n[a] - NG);
    if (hit) return SACRA_ERR_BADARG;
  }
  return SACRA_OK;
}

// Sommerfeld shell of every patch that has one: EPI 0 stores the RHS into `rhs`, 1..5 apply the RK4 stage table
static int launch_sommerfeld(const sacra_patch_t* p, int npatch, const sacra_boundary_t* bnd, int epi, const double* u_in,
                             double* rhs, const double* u_n, double* u_out, double* acc, cudaStream_t st) {
  RkArgs rk{u_n, u_out, acc};
  for (int q0 = 0; q0 < npatch; q0 += MAXP) {
    PatchBatch B;
    B.part = 0;
    ShellGeom G;
    B.np = (npatch - q0 < MAXP) ? npatch - q0 : MAXP;
    int nb = 0;
    bool any = false;
    for (int q = 0; q < B.np; ++q) {
      B.p[q] = to_dev(p[q0 + q]);
      B.p[q].shell = shell_bits(bnd[q0 + q]);
      any = any || B.p[q].shell;
      for (int a = 0; a < 3; ++a) G.origin[q][a] = bnd[q0 + q].origin[a];
      B.first_block[q] = nb;
      nb += p[q0 + q].nz;
    }
    B.first_block[B.np] = nb;
    if (!any) continue;
    const dim3 grid(nb, NF);
    switch (epi) {
      case 0: k_sommerfeld<0><<<grid, 256, 0, st>>>(B, G, u_in, rhs, rk); break;
      case 1: k_sommerfeld<1><<<grid, 256, 0, st>>>(B, G, u_in, rhs, rk); break;
      case 2: k_sommerfeld<2><<<grid, 256, 0, st>>>(B, G, u_in, rhs, rk); break;
      case 3: k_sommerfeld<3><<<grid, 256, 0, st>>>(B, G, u_in, rhs, rk); break;
      case 4: k_sommerfeld<4><<<grid, 256, 0, st>>>(B, G, u_in, rhs, rk); break;
      default: k_sommerfeld<5><<<grid, 256, 0, st>>>(B, G, u_in, rhs, rk); break;
    }
    if (cudaGetLastError() != cudaSuccess) return SACRA_ERR_CUDA;
  }
  return SACRA_OK;
}

// cuTensorMapEncodeTiled through the runtime (libsacra does not link libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn encode_tiled() {
  static EncodeTiledFn fn = [] {
    void* f = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &f, cudaEnableDefault, &q) != cudaSuccess ||
        q != cudaDriverEntryPointSuccess)
      f = nullptr;
    return reinterpret_cast<EncodeTiledFn>(f);
  }();
  return fn;
}

// Rank-4 (x, y, z, field) map of one patch of state `u` with box bx x by x bz x bf. Storage cell 0 of a row
// sits at an odd double (sacra.h: active cell 0 is 16-byte aligned and ng = 3), so the map starts ONE double
// earlier, which is 16-byte aligned and inside the caller's buffer (patch_offset >= 1): map x coordinate
// c <-> storage cell c - 1.
static int make_map(const sacra_patch_t& a, const double* u, int bx, int by, int bz, int bf, CUtensorMap* out) {
  EncodeTiledFn enc = encode_tiled();
  if (!enc) return SACRA_ERR_CUDA;
  const cuuint64_t dims[4] = {(cuuint64_t)a.nx + 2 * NG + 1, (cuuint64_t)a.ny + 2 * NG, (cuuint64_t)a.nz + 2 * NG, NF};
  const cuuint64_t strides[3] = {(cuuint64_t)a.pitch_x * 8, (cuuint64_t)a.pitch_x * (a.ny + 2 * NG) * 8,
                                 (cuuint64_t)a.field_stride * 8};
  const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, (cuuint32_t)bz, (cuuint32_t)bf};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  void* base = const_cast<double*>(u + a.patch_offset - 1);
  const CUresult r = enc(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, base, dims, strides, box, estr,
                         CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                         SACRA_L2PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? SACRA_OK : SACRA_ERR_CUDA;
}

// Encoding a tensor map costs a few microseconds on the host and a substage launch needs 2-4 per patch, which is most
// of the cost of a step on the small configurations. A map depends only on (address, layout, box), and callers step
// the same buffers over and over: keep the last MAPCACHE maps (a tensor map holds no device state; it stays valid as
// long as the address range it describes is what the caller passes again).
struct MapKey {
  const void* base;
  long long pitch, fstride;
  int nx, ny, nz, bx, by, bz, bf;
  bool operator==(const MapKey& o) const {
    return base == o.base && pitch == o.pitch && fstride == o.fstride && nx == o.nx && ny == o.ny && nz == o.nz &&
           bx == o.bx && by == o.by && bz == o.bz && bf == o.bf;
  }
};
constexpr int MAPCACHE = 256;
static std::mutex map_mutex;
static MapKey map_keys[MAPCACHE];
static CUtensorMap map_vals[MAPCACHE];
static int map_count = 0, map_next = 0;

static int cached_map(const sacra_patch_t& a, const double* u, int bx, int by, int bz, int bf, CUtensorMap* out) {
  const MapKey k{u + a.patch_offset, a.pitch_x, a.field_stride, a.nx, a.ny, a.nz, bx, by, bz, bf};
  std::lock_guard<std::mutex> lock(map_mutex);
  for (int i = 0; i < map_count; ++i)
    if (map_keys[i] == k) {
      *out = map_vals[i];
      return SACRA_OK;
    }
  if (int e = make_map(a, u, bx, by, bz, bf, out)) return e;
  const int slot = map_count < MAPCACHE ? map_count++ : (map_next++ % MAPCACHE);
  map_keys[slot] = k;
  map_vals[slot] = *out;
  return SACRA_OK;
}

// per-device facts are asked for at every launch (one process may drive several devices)
static int num_sms() {
  int dev = 0, v = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 0;
  if (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 0;
  return v;
}


template <int EPI>
static cudaError_t launch_one(int grid, cudaStream_t st, const PatchBatch& B, const Params& P, const TileMaps& M,
                              double* rhs, const RkArgs& rk) {
  // the opt-in to > 48 KB of dynamic shared memory is per device: set it at every launch (a host-side table lookup)
  const cudaError_t attr =
      cudaFuncSetAttribute(k_z4c<EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, Tile::SMEM_BYTES);
  if (attr != cudaSuccess) return attr;
  k_z4c<EPI><<<grid, Tile::NTH, Tile::SMEM_BYTES, st>>>(B, P, M, rhs, rk);
  return cudaGetLastError();
}

static int launch_z4c(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int epi,
                      const double* u_in, double* rhs, const double* u_n, double* u_out, double* acc,
                      cudaStream_t st, const sacra_boundary_t* bnd = nullptr, int part = 0, unsigned xfaces = 0) {
  const Params P = to_dev(*prm);
  RkArgs rk{u_n, u_out, acc};
  const int sms = num_sms();
  if (sms <= 0) return SACRA_ERR_CUDA;
  for (int q0 = 0; q0 < npatch; q0 += MAXP) {
    PatchBatch B;
    B.part = 0;
    TileMaps M;
    B.np = (npatch - q0 < MAXP) ? npatch - q0 : MAXP;
    int nb = 0;
    for (int q = 0; q < B.np; ++q) {
      const sacra_patch_t& a = p[q0 + q];
      B.p[q] = to_dev(a);
      B.p[q].gc = grid_coef(a.dx, prm->ko_sigma);
      if (bnd) B.p[q].shell = shell_bits(bnd[q0 + q]);
      B.p[q].xshell = xfaces;
      B.first_block[q] = nb;
      nb += ((a.nx + Tile::TX - 1) / Tile::TX) * ((a.ny + Tile::TY - 1) / Tile::TY) * ((a.nz + Tile::TZ - 1) / Tile::TZ);
      if (int e = cached_map(a, u_in, Tile::PX, Tile::PY, Tile::PZ, 1, &M.box[q])) return e;
      if (int e = cached_map(a, u_in, Tile::TX, Tile::TY, Tile::TZ, NF, &M.cen[q])) return e;
      if (epi >= 2) {
        if (int e = cached_map(a, u_n, Tile::TX, Tile::TY, Tile::TZ, 1, &M.un[q])) return e;
        if (int e = cached_map(a, acc, Tile::TX, Tile::TY, Tile::TZ, 1, &M.acc[q])) return e;
      }
    }
    B.first_block[B.np] = nb;
    B.part = part;
    const int grid = nb < sms ? nb : sms;   // persistent CTAs (one per SM: the kernel owns the SM's Tensor Memory)
    cudaError_t err;
    switch (epi) {
      case -1: err = launch_one<-1>(grid, st, B, P, M, rhs, rk); break;
      case 0: err = launch_one<0>(grid, st, B, P, M, rhs, rk); break;
      case 1: err = launch_one<1>(grid, st, B, P, M, rhs, rk); break;
      case 2: err = launch_one<2>(grid, st, B, P, M, rhs, rk); break;
      case 3: err = launch_one<3>(grid, st, B, P, M, rhs, rk); break;
      case 4: err = launch_one<4>(grid, st, B, P, M, rhs, rk); break;
      default: err = launch_one<5>(grid, st, B, P, M, rhs, rk); break;
    }
    if (err != cudaSuccess) return SACRA_ERR_CUDA;
  }
  return SACRA_OK;
}

}  // namespace sacra

using namespace sacra;

// ---------------------------------------------------------------------------------------------------
// Scratch of sacra_constraint_norms_static (sacra.h): the per-plane partial sums of k_con_partial for callers that
// cannot provide a device buffer. It sits in the library image, so every GPU that loads libsacra carries these
// 128 KiB until the process ends. One array per device, shared by all calls on that device.
// In HOST code the name `con_part_static` is only a handle for the runtime, not a device address: a kernel handed
// `con_part_static` itself would write to the wrong place. static_norm_scratch() asks the runtime for the real
// address, once per device and with that device current, and remembers it.
// ---------------------------------------------------------------------------------------------------
static __device__ __align__(256) double con_part_static[4 * SACRA_NORMS_STATIC_MAX_PLANES];

static const int STATIC_MAXDEV = 64;
static std::mutex static_scratch_mutex;
static double* static_scratch_addr[STATIC_MAXDEV];   // zero-initialised: not looked up yet

// device address of con_part_static on the current device; nullptr if the runtime refuses
static double* static_norm_scratch() {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= STATIC_MAXDEV) return nullptr;
  std::lock_guard<std::mutex> lock(static_scratch_mutex);
  if (!static_scratch_addr[dev]) {
    double* ptr = nullptr;
    if (cudaGetSymbolAddress((void**)&ptr, con_part_static) != cudaSuccess) {
      (void)cudaGetLastError();   // leave no sticky error behind for the caller's next launch check
      return nullptr;
    }
    static_scratch_addr[dev] = ptr;
  }
  return static_scratch_addr[dev];
}

extern "C" {

int sacra_fill_ghosts(const sacra_patch_t* p, int npatch, double* u, void* cuda_stream) {
  if (!p || !u) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(u)) return SACRA_ERR_ALIGN;
  return launch_fill(p, npatch, u, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_fill_ghosts_bc(const sacra_patch_t* p, int npatch, const int32_t* axis_mode, double* u, void* cuda_stream) {
  if (!p || !u || !axis_mode) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(u)) return SACRA_ERR_ALIGN;
  for (int a = 0; a < 3; ++a)
    if (axis_mode[a] != SACRA_BC_PERIODIC && axis_mode[a] != SACRA_BC_MIRROR) return SACRA_ERR_BADARG;
  return launch_fill(p, npatch, u, static_cast<cudaStream_t>(cuda_stream), axis_mode);
}

int sacra_z4c_rhs(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const double* u, double* rhs,
                  void* cuda_stream) {
  if (!p || !prm || !u || !rhs) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(u) || !aligned16(rhs)) return SACRA_ERR_ALIGN;
  const long long ext = state_extent(p, npatch);
  if (overlap(u, ext, rhs, ext)) return SACRA_ERR_BADARG;
  return launch_z4c(p, npatch, prm, 0, u, rhs, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_rk4_substep(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int stage, const double* u_n,
                      const double* u_in, double* u_out, double* acc, void* cuda_stream) {
  if (!p || !prm || !u_n || !u_in || !u_out || !acc) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (stage < 1 || stage > 4) return SACRA_ERR_BADARG;
  if (!aligned16(u_n) || !aligned16(u_in) || !aligned16(u_out) || !aligned16(acc)) return SACRA_ERR_ALIGN;
  // aliasing: two states are either the same buffer (where the stage table allows it) or disjoint ranges
  const long long ext = state_extent(p, npatch);
  if (stage == 1 && u_n != u_in) return SACRA_ERR_BADARG;           // stage 1 takes u_n from the stage input
  if (overlap(u_out, ext, u_in, ext)) return SACRA_ERR_BADARG;      // u_in is read through the stencil
  if (overlap(acc, ext, u_in, ext) || overlap(acc, ext, u_n, ext) || overlap(acc, ext, u_out, ext))
    return SACRA_ERR_BADARG;
  if (u_n != u_in && overlap(u_n, ext, u_in, ext)) return SACRA_ERR_BADARG;
  if (u_n != u_out && overlap(u_n, ext, u_out, ext)) return SACRA_ERR_BADARG;
  const int epi = (stage == 4 && (prm->flags & SACRA_FLAG_SKIP_INCREMENT)) ? 5 : stage;
  return launch_z4c(p, npatch, prm, epi, u_in, nullptr, u_n, u_out, acc, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_rk4_substep_part(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int stage, int part,
                           const int32_t* exchange_faces, const double* u_n, const double* u_in, double* u_out, double* acc,
                           void* cuda_stream) {
  if (!p || !prm || !exchange_faces || !u_n || !u_in || !u_out || !acc) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (stage < 1 || stage > 4 || (part != SACRA_PART_INTERIOR && part != SACRA_PART_SHELL)) return SACRA_ERR_BADARG;
  if (!aligned16(u_n) || !aligned16(u_in) || !aligned16(u_out) || !aligned16(acc)) return SACRA_ERR_ALIGN;
  const long long ext = state_extent(p, npatch);
  if (stage == 1 && u_n != u_in) return SACRA_ERR_BADARG;
  if (overlap(u_out, ext, u_in, ext)) return SACRA_ERR_BADARG;
  if (overlap(acc, ext, u_in, ext) || overlap(acc, ext, u_n, ext) || overlap(acc, ext, u_out, ext)) return SACRA_ERR_BADARG;
  if (u_n != u_in && overlap(u_n, ext, u_in, ext)) return SACRA_ERR_BADARG;
  if (u_n != u_out && overlap(u_n, ext, u_out, ext)) return SACRA_ERR_BADARG;
  unsigned faces = 0;
  for (int a = 0; a < 6; ++a)
    if (exchange_faces[a]) faces |= 1u << a;
  const int epi = (stage == 4 && (prm->flags & SACRA_FLAG_SKIP_INCREMENT)) ? 5 : stage;
  return launch_z4c(p, npatch, prm, epi, u_in, nullptr, u_n, u_out, acc, static_cast<cudaStream_t>(cuda_stream), nullptr, part,
                    faces);
}

int sacra_rk4_step(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, double* u, double* work,
                   int64_t state_doubles, void* cuda_stream) {
  if (!p || !prm || !u || !work) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (state_doubles < 1 || (state_doubles & 1)) return SACRA_ERR_BADARG;
  for (int q = 0; q < npatch; ++q) {
    const int64_t need = (int64_t)p[q].pitch_x * (p[q].ny + 2 * SACRA_NG) * (p[q].nz + 2 * SACRA_NG);
    if (p[q].patch_offset + (int64_t)(SACRA_NF - 1) * p[q].field_stride + need > state_doubles)
      return SACRA_ERR_BADARG;   // the patch would run past the end of a state
  }
  if (!aligned16(u) || !aligned16(work)) return SACRA_ERR_ALIGN;
  if (overlap(u, state_doubles, work, 3 * state_doubles)) return SACRA_ERR_BADARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int last = (prm->flags & SACRA_FLAG_SKIP_INCREMENT) ? 5 : 4;
  double* w0 = work;
  double* w1 = work + state_doubles;
  double* acc = work + 2 * state_doubles;
  int e;
  // (a periodic write-through of the ghosts from the substage kernel was measured: +2.4 ms per 256^3 stage
  //  against 0.31 ms for the fill it replaces -- DESIGN.md "What was tried")
  if ((e = launch_fill(p, npatch, u, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 1, u, nullptr, u, w0, acc, st))) return e;
  if ((e = launch_fill(p, npatch, w0, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 2, w0, nullptr, u, w1, acc, st))) return e;
  if ((e = launch_fill(p, npatch, w1, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 3, w1, nullptr, u, w0, acc, st))) return e;
  if ((e = launch_fill(p, npatch, w0, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, last, w0, nullptr, u, u, acc, st))) return e;
  return launch_fill(p, npatch, u, st);
}

int sacra_fill_ghosts_faces(const sacra_patch_t* p, int npatch, const sacra_boundary_t* bnd, double* u, void* cuda_stream) {
  if (!p || !u || !bnd) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (int e = check_boundaries(bnd, npatch)) return e;
  if (!aligned16(u)) return SACRA_ERR_ALIGN;
  return launch_fill(p, npatch, u, static_cast<cudaStream_t>(cuda_stream), nullptr, bnd);
}

int sacra_sommerfeld_rhs(const sacra_patch_t* p, int npatch, const sacra_boundary_t* bnd, const double* u, double* rhs,
                         void* cuda_stream) {
  if (!p || !u || !rhs || !bnd) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (int e = check_boundaries(bnd, npatch)) return e;
  if (int e = check_shell_origin(p, bnd, npatch)) return e;
  if (!aligned16(u) || !aligned16(rhs)) return SACRA_ERR_ALIGN;
  const long long ext = state_extent(p, npatch);
  if (overlap(u, ext, rhs, ext)) return SACRA_ERR_BADARG;
  return launch_sommerfeld(p, npatch, bnd, 0, u, rhs, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_rk4_substep_bc(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const sacra_boundary_t* bnd,
                         int stage, const double* u_n, const double* u_in, double* u_out, double* acc, void* cuda_stream) {
  if (!p || !prm || !bnd || !u_n || !u_in || !u_out || !acc) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (int e = check_boundaries(bnd, npatch)) return e;
  if (int e = check_shell_origin(p, bnd, npatch)) return e;
  if (stage < 1 || stage > 4) return SACRA_ERR_BADARG;
  if (!aligned16(u_n) || !aligned16(u_in) || !aligned16(u_out) || !aligned16(acc)) return SACRA_ERR_ALIGN;
  const long long ext = state_extent(p, npatch);
  if (stage == 1 && u_n != u_in) return SACRA_ERR_BADARG;
  if (overlap(u_out, ext, u_in, ext)) return SACRA_ERR_BADARG;
  if (overlap(acc, ext, u_in, ext) || overlap(acc, ext, u_n, ext) || overlap(acc, ext, u_out, ext)) return SACRA_ERR_BADARG;
  if (u_n != u_in && overlap(u_n, ext, u_in, ext)) return SACRA_ERR_BADARG;
  if (u_n != u_out && overlap(u_n, ext, u_out, ext)) return SACRA_ERR_BADARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int epi = (stage == 4 && (prm->flags & SACRA_FLAG_SKIP_INCREMENT)) ? 5 : stage;
  if (int e = launch_z4c(p, npatch, prm, epi, u_in, nullptr, u_n, u_out, acc, st, bnd)) return e;
  return launch_sommerfeld(p, npatch, bnd, epi, u_in, nullptr, u_n, u_out, acc, st);
}

int sacra_rk4_step_bc(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const sacra_boundary_t* bnd, double* u,
                      double* work, int64_t state_doubles, void* cuda_stream) {
  if (!p || !prm || !bnd || !u || !work) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (int e = check_boundaries(bnd, npatch)) return e;
  if (int e = check_shell_origin(p, bnd, npatch)) return e;
  if (state_doubles < 1 || (state_doubles & 1) || state_extent(p, npatch) > state_doubles) return SACRA_ERR_BADARG;
  if (!aligned16(u) || !aligned16(work)) return SACRA_ERR_ALIGN;
  if (overlap(u, state_doubles, work, 3 * state_doubles)) return SACRA_ERR_BADARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const int last = (prm->flags & SACRA_FLAG_SKIP_INCREMENT) ? 5 : 4;
  double* w0 = work;
  double* w1 = work + state_doubles;
  double* acc = work + 2 * state_doubles;
  const double* in[4] = {u, w0, w1, w0};
  double* out[4] = {w0, w1, w0, u};
  int e;
  for (int s = 0; s < 4; ++s) {
    if ((e = launch_fill(p, npatch, const_cast<double*>(in[s]), st, nullptr, bnd))) return e;
    const int epi = s == 3 ? last : s + 1;
    if ((e = launch_z4c(p, npatch, prm, epi, in[s], nullptr, u, out[s], acc, st, bnd))) return e;
    if ((e = launch_sommerfeld(p, npatch, bnd, epi, in[s], nullptr, u, out[s], acc, st))) return e;
  }
  return launch_fill(p, npatch, u, st, nullptr, bnd);
}

int sacra_constraints(const sacra_patch_t* p, int npatch, const double* u, double* con, void* cuda_stream) {
  if (!p || !u || !con) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(u) || !aligned16(con)) return SACRA_ERR_ALIGN;
  if (overlap(u, state_extent(p, npatch), con, state_extent(p, npatch))) return SACRA_ERR_BADARG;
  const sacra_params_t none = {0.0, 0.0, 0.0, 0.0, 0.0, 1, 0};   // the constraints have no parameters
  return launch_z4c(p, npatch, &none, -1, u, con, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

int64_t sacra_constraint_scratch_doubles(const sacra_patch_t* p, int npatch) {
  if (!p || npatch < 1) return 0;
  int64_t planes = 0;
  for (int q = 0; q < npatch; ++q) planes += p[q].nz > 0 ? p[q].nz : 0;
  return 4 * planes;
}

int sacra_constraint_norms(const sacra_patch_t* p, int npatch, const double* con, double* scratch, double* norms,
                           void* cuda_stream) {
  if (!p || !con || !scratch || !norms) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(con)) return SACRA_ERR_ALIGN;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double vol = 0.0;
  int planes = 0;
  for (int q0 = 0; q0 < npatch; q0 += MAXP) {
    PatchBatch B;
    B.part = 0;
    B.np = (npatch - q0 < MAXP) ? npatch - q0 : MAXP;
    int nb = 0;
    for (int q = 0; q < B.np; ++q) {
      const sacra_patch_t& a = p[q0 + q];
      B.p[q] = to_dev(a);
      B.first_block[q] = nb;
      nb += a.nz;
      vol += (double)a.nx * a.ny * a.nz * ((a.dx * a.dx) * a.dx);
    }
    B.first_block[B.np] = nb;
    k_con_partial<<<nb, 256, 0, st>>>(B, con, scratch, planes);
    if (cudaGetLastError() != cudaSuccess) return SACRA_ERR_CUDA;
    planes += nb;
  }
  k_con_final<<<1, 4, 0, st>>>(scratch, planes, vol, norms);
  return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
}

// sacra_constraint_norms for callers that cannot allocate (sacra.h has the contract): the capacity check comes
// first, so a batch that is too large launches nothing; then the partial sums go to the library's own array through
// the unchanged path above. No allocation happens here or below. The array's old contents do not matter:
// k_con_partial writes entries 0 .. 4*planes-1 and k_con_final reads exactly those.
int sacra_constraint_norms_static(const sacra_patch_t* p, int npatch, const double* con, double* norms,
                                  void* cuda_stream) {
  if (!p || !con || !norms) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  int64_t planes = 0;
  for (int q = 0; q < npatch; ++q) planes += p[q].nz;
  if (planes > SACRA_NORMS_STATIC_MAX_PLANES) return SACRA_ERR_TOOLARGE;
  double* part = static_norm_scratch();   // first call on this device: cudaGetSymbolAddress
  if (!part) return SACRA_ERR_CUDA;
  return sacra_constraint_norms(p, npatch, con, part, norms, cuda_stream);
}

// f-3: geometry checks shared by the two inter-level calls
static int check_levels(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org, bool prolong) {
  if (!parent || !child || !org) return SACRA_ERR_NULL;
  if (int e = check_patches(parent, 1)) return e;
  if (int e = check_patches(child, 1)) return e;
  if (std::fabs(2.0 * child->dx - parent->dx) > 1e-12 * parent->dx) return SACRA_ERR_BADARG;   // 2:1 refinement
  const int nc[3] = {child->nx, child->ny, child->nz}, np[3] = {parent->nx, parent->ny, parent->nz};
  for (int a = 0; a < 3; ++a) {
    if (nc[a] & 1) return SACRA_ERR_BADARG;                                  // a parent cell holds two child cells
    if (org[a] < 0 || org[a] + nc[a] / 2 > np[a]) return SACRA_ERR_BADARG;   // covered cells are parent active cells
    // prolongation reads the parent cells org + floor(i/2) - 3 .. + 3 for child cells i = -3 .. n+2: inside the
    // parent's storage (ghosts included)
    if (prolong && (org[a] - 2 - 3 < -SACRA_NG || org[a] + (nc[a] + 2) / 2 + 3 > np[a] + SACRA_NG - 1)) return SACRA_ERR_BADARG;
  }
  return SACRA_OK;
}
static LevelPair level_pair(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org) {
  LevelPair L;
  L.parent = to_dev(*parent);
  L.child = to_dev(*child);
  for (int a = 0; a < 3; ++a) L.org[a] = org[a];
  return L;
}

int sacra_restrict(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org, double* u_parent,
                   const double* u_child, void* cuda_stream) {
  if (!u_parent || !u_child) return SACRA_ERR_NULL;
  if (int e = check_levels(parent, child, org, false)) return e;
  if (!aligned16(u_parent) || !aligned16(u_child)) return SACRA_ERR_ALIGN;
  if (overlap(u_parent, state_extent(parent, 1), u_child, state_extent(child, 1))) return SACRA_ERR_BADARG;
  const LevelPair L = level_pair(parent, child, org);
  const int n = (child->nx / 2) * (child->ny / 2) * (child->nz / 2);
  k_restrict<<<dim3((n + 127) / 128, NF), 128, 0, static_cast<cudaStream_t>(cuda_stream)>>>(L, u_parent, u_child);
  return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
}

int sacra_prolong_ghosts(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org,
                         const double* u_parent, double* u_child, void* cuda_stream) {
  if (!u_parent || !u_child) return SACRA_ERR_NULL;
  if (int e = check_levels(parent, child, org, true)) return e;
  if (!aligned16(u_parent) || !aligned16(u_child)) return SACRA_ERR_ALIGN;
  if (overlap(u_parent, state_extent(parent, 1), u_child, state_extent(child, 1))) return SACRA_ERR_BADARG;
  const LevelPair L = level_pair(parent, child, org);
  const int gx = child->nx / 2 + 4, gy = child->ny / 2 + 4, gz = child->nz / 2 + 4;
  const int n = 4 * (gx * gy + gx * (gz - 4) + (gy - 4) * (gz - 4));   // parent cells that hold ghost cells of the child
  k_prolong_ghosts<<<dim3((n + 127) / 128, NF), 128, 0, static_cast<cudaStream_t>(cuda_stream)>>>(L, u_parent, u_child);
  return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
}

int64_t sacra_face_doubles(const sacra_patch_t* p, int axis) {
  if (!p || axis < 0 || axis > 2) return 0;
  const int64_t s[3] = {p->nx + 2 * SACRA_NG, p->ny + 2 * SACRA_NG, p->nz + 2 * SACRA_NG};
  return (int64_t)SACRA_NF * SACRA_NG * (s[0] * s[1] * s[2] / s[axis]);
}

static int face_call(bool pack, const sacra_patch_t* p, double* u, int axis, int side, double* buf, void* cuda_stream) {
  if (!p || !u || !buf) return SACRA_ERR_NULL;
  if (int e = check_patches(p, 1)) return e;
  if (axis < 0 || axis > 2 || side < 0 || side > 1) return SACRA_ERR_BADARG;
  if (!aligned16(u) || !aligned16(buf)) return SACRA_ERR_ALIGN;
  if (overlap(u, state_extent(p, 1), buf, sacra_face_doubles(p, axis))) return SACRA_ERR_BADARG;
  const long long plane = sacra_face_doubles(p, axis) / (SACRA_NF * SACRA_NG);
  const int split = plane / 16384 < 1 ? 1 : (plane / 16384 > 8 ? 8 : (int)(plane / 16384));
  const dim3 grid(NG, NF, split);
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (pack) k_face<true><<<grid, 256, 0, st>>>(to_dev(*p), axis, side, u, buf);
  else k_face<false><<<grid, 256, 0, st>>>(to_dev(*p), axis, side, u, buf);
  return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
}
int sacra_pack_face(const sacra_patch_t* p, const double* u, int axis, int side, double* buf, void* cuda_stream) {
  return face_call(true, p, const_cast<double*>(u), axis, side, buf, cuda_stream);
}
int sacra_unpack_face(const sacra_patch_t* p, double* u, int axis, int side, const double* buf, void* cuda_stream) {
  return face_call(false, p, u, axis, side, const_cast<double*>(buf), cuda_stream);
}

int sacra_time_weights(int nlevels, double theta, double* w) {
  if (!w) return SACRA_ERR_NULL;
  if ((nlevels != 2 && nlevels != 3) || !std::isfinite(theta)) return SACRA_ERR_BADARG;
  if (nlevels == 2) {            // straight line through theta = 0, 1
    w[0] = 1.0 - theta; w[1] = theta; w[2] = 0.0;
  } else {                       // parabola through theta = -1, 0, 1 (Lagrange basis)
    w[0] = (theta * (theta - 1.0)) / 2.0;
    w[1] = ((theta + 1.0) * (theta - 1.0)) / -1.0;
    w[2] = ((theta + 1.0) * theta) / 2.0;
  }
  return SACRA_OK;
}

// box: storage-index bounds [lo, hi) per axis, or nullptr for the whole storage of the patch
static int launch_lincomb(const sacra_patch_t* p, int n, const double* u0, const double* u1, const double* u2,
                          const double* w, double* out, cudaStream_t st, const int* lo = nullptr, const int* hi = nullptr) {
  LinComb L;
  L.u[0] = u0; L.u[1] = u1; L.u[2] = n == 3 ? u2 : u0;
  L.w[0] = w[0]; L.w[1] = w[1]; L.w[2] = n == 3 ? w[2] : 0.0;
  L.n = n;
  const int s[3] = {p->nx + 2 * NG, p->ny + 2 * NG, p->nz + 2 * NG};
  for (int a = 0; a < 3; ++a) {
    L.lo[a] = lo ? (lo[a] < 0 ? 0 : lo[a]) : 0;
    L.hi[a] = hi ? (hi[a] > s[a] ? s[a] : hi[a]) : s[a];
  }
  k_lincomb<<<dim3(L.hi[2] - L.lo[2], NF), 256, 0, st>>>(to_dev(*p), L, out);
  return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
}

int sacra_lincomb(const sacra_patch_t* p, int nlevels, const double* u0, const double* u1, const double* u2, const double* w,
                  double* out, void* cuda_stream) {
  if (!p || !u0 || !u1 || !w || !out || (nlevels == 3 && !u2)) return SACRA_ERR_NULL;
  if (int e = check_patches(p, 1)) return e;
  if (nlevels != 2 && nlevels != 3) return SACRA_ERR_BADARG;
  if (!aligned16(u0) || !aligned16(u1) || !aligned16(out) || (nlevels == 3 && !aligned16(u2))) return SACRA_ERR_ALIGN;
  const long long ext = state_extent(p, 1);
  if (overlap(out, ext, u0, ext) || overlap(out, ext, u1, ext) || (nlevels == 3 && overlap(out, ext, u2, ext)))
    return SACRA_ERR_BADARG;
  return launch_lincomb(p, nlevels, u0, u1, u2, w, out, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_subcycle_step(const sacra_patch_t* parent, const sacra_patch_t* child, const int32_t* org,
                        const sacra_params_t* prm, const sacra_boundary_t* parent_bnd, double* u_parent,
                        double* u_parent_prev, int have_prev, double* u_child, double* work_parent,
                        int64_t parent_doubles, double* work_child, int64_t child_doubles, void* cuda_stream) {
  if (!prm || !parent_bnd || !u_parent || !u_parent_prev || !u_child || !work_parent || !work_child) return SACRA_ERR_NULL;
  if (int e = check_levels(parent, child, org, true)) return e;
  if (int e = check_boundaries(parent_bnd, 1)) return e;
  if (int e = check_shell_origin(parent, parent_bnd, 1)) return e;
  if (std::fabs(2.0 * child->dt - parent->dt) > 1e-12 * std::fabs(parent->dt)) return SACRA_ERR_BADARG;   // halved time step
  if (parent_doubles < state_extent(parent, 1) || child_doubles < state_extent(child, 1) || (parent_doubles & 1) ||
      (child_doubles & 1))
    return SACRA_ERR_BADARG;
  if (!aligned16(u_parent) || !aligned16(u_parent_prev) || !aligned16(u_child) || !aligned16(work_parent) ||
      !aligned16(work_child))
    return SACRA_ERR_ALIGN;
  const double* bufs[5] = {u_parent, u_parent_prev, u_child, work_parent, work_child};
  const long long len[5] = {parent_doubles, parent_doubles, child_doubles, 5 * parent_doubles, 3 * child_doubles};
  for (int a = 0; a < 5; ++a)
    for (int b = a + 1; b < 5; ++b)
      if (overlap(bufs[a], len[a], bufs[b], len[b])) return SACRA_ERR_BADARG;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double* old = work_parent;
  double* tmp = work_parent + parent_doubles;
  double* wk = work_parent + 2 * parent_doubles;
  int e;
  // (1) the parent: t_n -> t_n + dt
  if (cudaMemcpyAsync(old, u_parent, (size_t)parent_doubles * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return SACRA_ERR_CUDA;
  if ((e = sacra_rk4_step_bc(parent, 1, prm, parent_bnd, u_parent, wk, parent_doubles, cuda_stream))) return e;
  // (2) the child: two steps of dt / 2, ghosts of every stage input from the parent levels interpolated in time
  const int nlev = have_prev ? 3 : 2;
  const double* lev[3] = {have_prev ? u_parent_prev : old, have_prev ? old : u_parent, have_prev ? u_parent : nullptr};
  double* w0 = work_child;
  double* w1 = work_child + child_doubles;
  double* acc = work_child + 2 * child_doubles;
  const double cs[4] = {0.0, 0.5, 0.5, 1.0};
  const LevelPair L = level_pair(parent, child, org);
  const int pgx = child->nx / 2 + 4, pgy = child->ny / 2 + 4, pgz = child->nz / 2 + 4;
  const int nshell = 4 * (pgx * pgy + pgx * (pgz - 4) + (pgy - 4) * (pgz - 4));   // parent cells that hold ghost cells
  auto prolong = [&](const double* up, double* uc) {
    k_prolong_ghosts<<<dim3((nshell + 127) / 128, NF), 128, 0, st>>>(L, up, uc);
    return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
  };
  // the prolongation reads the parent's active cells org - 5 .. org + n_child / 2 + 3 per axis: the time
  // interpolation is formed on that box only, not on the whole parent
  int blo[3], bhi[3];
  const int ncs[3] = {child->nx, child->ny, child->nz};
  for (int a = 0; a < 3; ++a) {
    blo[a] = org[a] - 5 + NG;
    bhi[a] = org[a] + ncs[a] / 2 + 3 + NG + 1;
  }
  for (int m = 0; m < 2; ++m) {
    const double* in[4] = {u_child, w0, w1, w0};
    double* out[4] = {w0, w1, w0, u_child};
    for (int s = 0; s < 4; ++s) {
      double w[3];
      sacra_time_weights(nlev, ((double)m + cs[s]) / 2.0, w);
      if ((e = launch_lincomb(parent, nlev, lev[0], lev[1], lev[2], w, tmp, st, blo, bhi))) return e;
      if ((e = prolong(tmp, const_cast<double*>(in[s])))) return e;
      if ((e = launch_z4c(child, 1, prm, s + 1, in[s], nullptr, u_child, out[s], acc, st))) return e;
    }
  }
  // (3) child ghosts at the new time, restriction, parent ghosts; U^n goes to the caller for the next step
  if ((e = prolong(u_parent, u_child))) return e;
  const int nr = (child->nx / 2) * (child->ny / 2) * (child->nz / 2);
  k_restrict<<<dim3((nr + 127) / 128, NF), 128, 0, st>>>(L, u_parent, u_child);
  if (cudaGetLastError() != cudaSuccess) return SACRA_ERR_CUDA;
  if ((e = launch_fill(parent, 1, u_parent, st, nullptr, parent_bnd))) return e;
  if (cudaMemcpyAsync(u_parent_prev, old, (size_t)parent_doubles * 8, cudaMemcpyDeviceToDevice, st) != cudaSuccess) return SACRA_ERR_CUDA;
  return SACRA_OK;
}

// Recursive Berger-Oliger step (sacra.h: sacra_hierarchy_step). Level l's buffers: old = work, tmp = work + n (its data
// interpolated in time for its child), then w0, w1, acc of its RK4 step.
namespace {
struct HierCtx {
  sacra_level_t* L;
  int nlevels;
  const sacra_params_t* prm;
  const sacra_boundary_t* bnd0;
  cudaStream_t st;
};
// ghosts of `target` (a state of level l) from the time levels of level l - 1 at theta
int hier_parent_ghosts(const HierCtx& c, int l, double theta, double* target) {
  sacra_level_t& pa = c.L[l - 1];
  sacra_level_t& me = c.L[l];
  const int nlev = pa.nsteps > 0 ? 3 : 2;
  double* old = pa.work;
  double* tmp = pa.work + pa.state_doubles;
  const double* lev[3] = {nlev == 3 ? pa.u_prev : old, nlev == 3 ? old : pa.u, nlev == 3 ? pa.u : nullptr};
  double w[3];
  sacra_time_weights(nlev, theta, w);
  int blo[3], bhi[3];
  const int ncs[3] = {me.patch->nx, me.patch->ny, me.patch->nz};
  for (int a = 0; a < 3; ++a) {
    blo[a] = me.org[a] - 5 + NG;
    bhi[a] = me.org[a] + ncs[a] / 2 + 3 + NG + 1;
  }
  if (int e = launch_lincomb(pa.patch, nlev, lev[0], lev[1], lev[2], w, tmp, c.st, blo, bhi)) return e;
  const LevelPair P = level_pair(pa.patch, me.patch, me.org);
  const int gx = ncs[0] / 2 + 4, gy = ncs[1] / 2 + 4, gz = ncs[2] / 2 + 4;
  const int n = 4 * (gx * gy + gx * (gz - 4) + (gy - 4) * (gz - 4));
  k_prolong_ghosts<<<dim3((n + 127) / 128, NF), 128, 0, c.st>>>(P, tmp, target);
  return cudaGetLastError() == cudaSuccess ? SACRA_OK : SACRA_ERR_CUDA;
}
int hier_advance(const HierCtx& c, int l, int m) {
  sacra_level_t& me = c.L[l];
  const int64_t n = me.state_doubles;
  double* old = me.work;
  double* w0 = me.work + 2 * n;
  double* w1 = me.work + 3 * n;
  double* acc = me.work + 4 * n;
  int e;
  if (cudaMemcpyAsync(old, me.u, (size_t)n * 8, cudaMemcpyDeviceToDevice, c.st) != cudaSuccess) return SACRA_ERR_CUDA;
  if (l == 0) {
    if ((e = sacra_rk4_step_bc(me.patch, 1, c.prm, c.bnd0, me.u, w0, n, c.st))) return e;
  } else {
    const double cs[4] = {0.0, 0.5, 0.5, 1.0};
    const double* in[4] = {me.u, w0, w1, w0};
    double* out[4] = {w0, w1, w0, me.u};
    for (int s = 0; s < 4; ++s) {
      if ((e = hier_parent_ghosts(c, l, ((double)m + cs[s]) / 2.0, const_cast<double*>(in[s])))) return e;
      if ((e = launch_z4c(me.patch, 1, c.prm, s + 1, in[s], nullptr, me.u, out[s], acc, c.st))) return e;
    }
  }
  if (l + 1 < c.nlevels) {
    // stage 4 wrote active cells only: an intermediate level brings its ghosts to the time just reached before its
    // child advances, whose prolongation box reads them when the child sits within 4 cells of this level's edge
    // (level 0: sacra_rk4_step_bc ended with its fill)
    if (l > 0 && (e = hier_parent_ghosts(c, l, ((double)m + 1.0) / 2.0, me.u))) return e;
    if ((e = hier_advance(c, l + 1, 0))) return e;
    if ((e = hier_advance(c, l + 1, 1))) return e;
    sacra_level_t& ch = c.L[l + 1];
    if ((e = sacra_prolong_ghosts(me.patch, ch.patch, ch.org, me.u, ch.u, c.st))) return e;
    if ((e = sacra_restrict(me.patch, ch.patch, ch.org, me.u, ch.u, c.st))) return e;
  }
  if (l == 0) {
    if ((e = launch_fill(me.patch, 1, me.u, c.st, nullptr, c.bnd0))) return e;
  } else if ((e = hier_parent_ghosts(c, l, ((double)m + 1.0) / 2.0, me.u))) {
    return e;
  }
  if (cudaMemcpyAsync(me.u_prev, old, (size_t)n * 8, cudaMemcpyDeviceToDevice, c.st) != cudaSuccess) return SACRA_ERR_CUDA;
  me.nsteps += 1;
  return SACRA_OK;
}
}  // namespace

int sacra_hierarchy_step(sacra_level_t* levels, int nlevels, const sacra_params_t* prm, const sacra_boundary_t* bnd0,
                         void* cuda_stream) {
  if (!levels || !prm || !bnd0) return SACRA_ERR_NULL;
  if (nlevels < 1 || nlevels > 16) return SACRA_ERR_BADARG;
  if (int e = check_boundaries(bnd0, 1)) return e;
  for (int l = 0; l < nlevels; ++l) {
    const sacra_level_t& a = levels[l];
    if (!a.patch || !a.u || !a.u_prev || !a.work) return SACRA_ERR_NULL;
    if (int e = check_patches(a.patch, 1)) return e;
    if (a.state_doubles < state_extent(a.patch, 1) || (a.state_doubles & 1) || a.nsteps < 0) return SACRA_ERR_BADARG;
    if (!aligned16(a.u) || !aligned16(a.u_prev) || !aligned16(a.work)) return SACRA_ERR_ALIGN;
    if (overlap(a.u, a.state_doubles, a.u_prev, a.state_doubles) || overlap(a.u, a.state_doubles, a.work, 5 * a.state_doubles) ||
        overlap(a.u_prev, a.state_doubles, a.work, 5 * a.state_doubles))
      return SACRA_ERR_BADARG;
    if (l > 0) {
      const sacra_level_t& pa = levels[l - 1];
      if (int e = check_levels(pa.patch, a.patch, a.org, true)) return e;
      if (std::fabs(2.0 * a.patch->dt - pa.patch->dt) > 1e-12 * std::fabs(pa.patch->dt)) return SACRA_ERR_BADARG;
      for (int k = 0; k < l; ++k) {      // buffers of different levels are disjoint
        const sacra_level_t& b = levels[k];
        const double* A[3] = {a.u, a.u_prev, a.work};
        const double* Bq[3] = {b.u, b.u_prev, b.work};
        const long long na[3] = {a.state_doubles, a.state_doubles, 5 * a.state_doubles};
        const long long nb[3] = {b.state_doubles, b.state_doubles, 5 * b.state_doubles};
        for (int i = 0; i < 3; ++i)
          for (int j = 0; j < 3; ++j)
            if (overlap(A[i], na[i], Bq[j], nb[j])) return SACRA_ERR_BADARG;
      }
    }
  }
  if (int e = check_shell_origin(levels[0].patch, bnd0, 1)) return e;
  HierCtx c{levels, nlevels, prm, bnd0, static_cast<cudaStream_t>(cuda_stream)};
  return hier_advance(c, 0, 0);
}

const char* sacra_strerror(int code) {
  switch (code) {
    case SACRA_OK: return "ok";
    case SACRA_ERR_NULL: return "null pointer argument";
    case SACRA_ERR_BADARG: return "bad argument (size, spacing, stage, layout or aliasing)";
    case SACRA_ERR_UNSUPPORTED: return "unsupported ghost width (ng must be 3)";
    case SACRA_ERR_ALIGN: return "pointer or layout breaks the 16-byte alignment rule";
    case SACRA_ERR_CUDA: return "CUDA launch failed";
    case SACRA_ERR_TOOLARGE: return "problem exceeds a fixed capacity of the library (see sacra.h)";
    default: return "unknown sacra status";
  }
}

const char* sacra_version(void) { return "0.2"; }

}  // extern "C"
