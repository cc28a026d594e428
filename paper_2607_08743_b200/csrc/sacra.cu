// sacra.cu -- libsacra: C ABI (include/sacra.h) and the CUDA kernels behind it, sm_100a only.
//
// Kernels
//   k_fill_ghosts   periodic halo fill, one thread per ghost-shell storage cell
//   k_z4c           derivative stage + algebra + KO + epilogue (RHS store or RK4 substage), one thread
//                   per active point
// There is no CPU path: every entry point enqueues kernels on the caller's stream or returns an error.
#include <cmath>
#include <cstdint>
#include <cuda_runtime.h>

#include "../../include/sacra.h"
#include "z4c_point.cuh"

namespace sacra {

constexpr int MAXP = 16;   // patch descriptors carried in kernel parameters per launch

struct DevPatch {
  int nx, ny, nz;
  long long pitch, sz;     // doubles per x-row, doubles per z-plane
  long long fstride, offset;
  double dx, dt;
};
struct PatchBatch {
  DevPatch p[MAXP];
  int first_block[MAXP + 1];   // prefix sum of blocks per patch (block -> patch lookup)
  int np;
};

// ---------------------------------------------------------------------------------------------------
// Periodic halo fill. The ghost shell of a patch is enumerated as storage cells of the full box; active
// cells return immediately (they are never written, so reads and writes never overlap: item 2).
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_fill_ghosts(const __grid_constant__ PatchBatch B, double* __restrict__ u) {
  int ip = 0;
#pragma unroll 1
  while (ip + 1 < B.np && (int)blockIdx.x >= B.first_block[ip + 1]) ++ip;
  const DevPatch& p = B.p[ip];
  const int sx = p.nx + 2 * NG, sy = p.ny + 2 * NG;
  // one block = one (row J, plane K) pair group: blockDim.x threads stride along x
  const int row = (int)blockIdx.x - B.first_block[ip];     // 0 .. sy*sz-1
  const int J = row % sy, Kk = row / sy;
  const bool row_ghost = (J < NG) | (J >= NG + p.ny) | (Kk < NG) | (Kk >= NG + p.nz);
  int j = J - NG, k = Kk - NG;
  j = j < 0 ? j + p.ny : (j >= p.ny ? j - p.ny : j);
  k = k < 0 ? k + p.nz : (k >= p.nz ? k - p.nz : k);
  const long long dst_row = (long long)Kk * p.sz + (long long)J * p.pitch;
  const long long src_row = (long long)(k + NG) * p.sz + (long long)(j + NG) * p.pitch;
  for (int f = blockIdx.y; f < NF; f += gridDim.y) {
    double* fld = u + p.offset + (long long)f * p.fstride;
    if (row_ghost) {
      for (int I = threadIdx.x; I < sx; I += blockDim.x) {
        int i = I - NG;
        i = i < 0 ? i + p.nx : (i >= p.nx ? i - p.nx : i);
        fld[dst_row + I] = fld[src_row + i + NG];
      }
    } else if (threadIdx.x < 2 * NG) {
      // active row: only the 3+3 x-ghosts
      const int I = threadIdx.x < NG ? threadIdx.x : p.nx + threadIdx.x;   // 0..2, nx+3..nx+5
      const int i = threadIdx.x < NG ? p.nx - NG + threadIdx.x : threadIdx.x - NG;
      fld[dst_row + I] = fld[src_row + i + NG];
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// Derivative stage, direct from global memory through L1/L2 (version 1: no staging).
// ---------------------------------------------------------------------------------------------------
template <int F>
__device__ __forceinline__ void derivs_of_field(const double* __restrict__ c, long long sy, long long sz,
                                                const Coef& cf, const double (&beta)[3],
                                                const double (&sg)[3], Derivs& D, double& u0_out) {
  const long long st[3] = {1, sy, sz};
  const double u0 = __ldg(c);
  u0_out = u0;
  double qsum = 0.0, adv[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    const long long s = st[a];
    const double m3 = __ldg(c - 3 * s), m2 = __ldg(c - 2 * s), m1 = __ldg(c - s);
    const double p1 = __ldg(c + s), p2 = __ldg(c + 2 * s), p3 = __ldg(c + 3 * s);
    if (d1slot(F) >= 0) D.d1[d1slot(F)][a] = __dmul_rn(d1_num(m2, m1, p1, p2), cf.inv12h);
    const double s1 = pair_sum(m1, u0, p1), s2 = pair_sum(m2, u0, p2), s3 = pair_sum(m3, u0, p3);
    if (d2slot(F) >= 0) D.d2[d2slot(F)][sym(a, a)] = __dmul_rn(d2_num(s1, s2), cf.inv12h2);
    const double q = ko_num(s1, s2, s3);
    qsum = (a == 0) ? q : __dadd_rn(qsum, q);
    // upwind: v_k = u(x + sg k h); select mirrored samples by the sign of beta^a (same instructions for
    // both signs: item 13)
    const bool pos = sg[a] > 0.0;
    const double vm1 = pos ? m1 : p1, v1 = pos ? p1 : m1, v2 = pos ? p2 : m2, v3 = pos ? p3 : m3;
    adv[a] = __dmul_rn(beta[a], __dmul_rn(up_num(vm1, u0, v1, v2, v3, sg[a]), cf.inv12h));
  }
  D.adv[F] = __dadd_rn(__dadd_rn(adv[0], adv[1]), adv[2]);
  D.ko[F] = __dmul_rn(qsum, cf.kofac);
  if (d2slot(F) >= 0) {
    // mixed second derivatives D_ab = D_a(D_b u), a < b, inner (unscaled) difference along the later axis b
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
      for (int b = a + 1; b < 3; ++b) {
        const long long sa = st[a], sb = st[b];
        auto e = [&](long long o) {
          const double* v = c + o;
          return d1_num(__ldg(v - 2 * sb), __ldg(v - sb), __ldg(v + sb), __ldg(v + 2 * sb));
        };
        const double em2 = e(-2 * sa), em1 = e(-sa), ep1 = e(sa), ep2 = e(2 * sa);
        D.d2[d2slot(F)][sym(a, b)] = __dmul_rn(d1_num(em2, em1, ep1, ep2), cf.inv144h2);
      }
  }
}

template <int F>
struct FieldLoop {
  static __device__ __forceinline__ void run(const double* __restrict__ base, long long fstride, long long c,
                                             long long sy, long long sz, const Coef& cf,
                                             const double (&beta)[3], const double (&sg)[3], Derivs& D,
                                             double (&u)[NF]) {
    derivs_of_field<F>(base + (long long)F * fstride + c, sy, sz, cf, beta, sg, D, u[F]);
    FieldLoop<F + 1>::run(base, fstride, c, sy, sz, cf, beta, sg, D, u);
  }
};
template <>
struct FieldLoop<NF> {
  static __device__ __forceinline__ void run(const double* __restrict__, long long, long long, long long,
                                             long long, const Coef&, const double (&)[3], const double (&)[3],
                                             Derivs&, double (&)[NF]) {}
};

// EPI: 0 = store RHS; 1..4 = RK4 substage (item 11 table)
struct RkArgs {
  const double* u_n;
  double* u_out;
  double* acc;
};

template <int EPI>
__global__ void __launch_bounds__(128) k_z4c(const __grid_constant__ PatchBatch B, const __grid_constant__ Params P,
                                             const double* __restrict__ u_in, double* __restrict__ rhs,
                                             const __grid_constant__ RkArgs rk) {
  int ip = 0;
#pragma unroll 1
  while (ip + 1 < B.np && (int)blockIdx.x >= B.first_block[ip + 1]) ++ip;
  const DevPatch& p = B.p[ip];
  // block -> (x-chunk, j-chunk, k) ; blockDim = (32, 4)
  const int nbx = (p.nx + 31) / 32, nby = (p.ny + 3) / 4;
  int b = (int)blockIdx.x - B.first_block[ip];
  const int bx = b % nbx; b /= nbx;
  const int by = b % nby; const int k = b / nby;
  const int i = bx * 32 + threadIdx.x, j = by * 4 + threadIdx.y;
  if (i >= p.nx || j >= p.ny) return;
  const long long c = (long long)(k + NG) * p.sz + (long long)(j + NG) * p.pitch + (i + NG);
  const double* base = u_in + p.offset;

  const Coef cf = make_coef(p.dx, P.ko_sigma);
  double beta[3], sg[3];
#pragma unroll
  for (int a = 0; a < 3; ++a) {
    beta[a] = __ldg(base + (long long)(F_BET + a) * p.fstride + c);
    sg[a] = beta[a] >= 0.0 ? 1.0 : -1.0;
  }
  Derivs D;
  double u[NF], out[NF];
  FieldLoop<0>::run(base, p.fstride, c, p.pitch, p.sz, cf, beta, sg, D, u);
  z4c_algebra(u, D, P, out);

  const long long o = p.offset + c;
  if (EPI == 0) {
#pragma unroll
    for (int f = 0; f < NF; ++f) rhs[o + (long long)f * p.fstride] = out[f];
  } else {
    const double dt = p.dt;
    const double hdt = dt / 2.0, c6 = 1.0 / 6.0;
#pragma unroll
    for (int f = 0; f < NF; ++f) {
      const long long a = o + (long long)f * p.fstride;
      const double kk = out[f];
      const double un = rk.u_n[a];
      if (EPI == 1) {
        rk.acc[a] = kk;
        rk.u_out[a] = __dadd_rn(un, __dmul_rn(hdt, kk));
      } else if (EPI == 2) {
        rk.acc[a] = __dadd_rn(rk.acc[a], __dmul_rn(2.0, kk));
        rk.u_out[a] = __dadd_rn(un, __dmul_rn(hdt, kk));
      } else if (EPI == 3) {
        rk.acc[a] = __dadd_rn(rk.acc[a], __dmul_rn(2.0, kk));
        rk.u_out[a] = __dadd_rn(un, __dmul_rn(dt, kk));
      } else {
        const double S = __dmul_rn(__dadd_rn(rk.acc[a], kk), c6);
        rk.acc[a] = S;
        rk.u_out[a] = __dadd_rn(un, __dmul_rn(dt, S));
      }
    }
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

static DevPatch to_dev(const sacra_patch_t& a) {
  DevPatch d;
  d.nx = a.nx; d.ny = a.ny; d.nz = a.nz;
  d.pitch = a.pitch_x; d.sz = a.pitch_x * (long long)(a.ny + 2 * NG);
  d.fstride = a.field_stride; d.offset = a.patch_offset; d.dx = a.dx; d.dt = a.dt;
  return d;
}

static Params to_dev(const sacra_params_t& a) {
  Params P;
  P.kappa1 = a.kappa1; P.kappa2 = a.kappa2; P.eta = a.eta; P.shift_coef = a.shift_coef;
  P.ko_sigma = a.ko_sigma; P.lapse_uses_khat = a.lapse_uses_khat;
  return P;
}

static int launch_fill(const sacra_patch_t* p, int npatch, double* u, cudaStream_t st) {
  for (int q0 = 0; q0 < npatch; q0 += MAXP) {
    PatchBatch B;
    B.np = (npatch - q0 < MAXP) ? npatch - q0 : MAXP;
    int nb = 0;
    for (int q = 0; q < B.np; ++q) {
      B.p[q] = to_dev(p[q0 + q]);
      B.first_block[q] = nb;
      nb += (p[q0 + q].ny + 2 * NG) * (p[q0 + q].nz + 2 * NG);
    }
    B.first_block[B.np] = nb;
    k_fill_ghosts<<<dim3(nb, NF), 64, 0, st>>>(B, u);
    if (cudaGetLastError() != cudaSuccess) return SACRA_ERR_CUDA;
  }
  return SACRA_OK;
}

static int launch_z4c(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int epi,
                      const double* u_in, double* rhs, const double* u_n, double* u_out, double* acc,
                      cudaStream_t st) {
  const Params P = to_dev(*prm);
  RkArgs rk{u_n, u_out, acc};
  for (int q0 = 0; q0 < npatch; q0 += MAXP) {
    PatchBatch B;
    B.np = (npatch - q0 < MAXP) ? npatch - q0 : MAXP;
    int nb = 0;
    for (int q = 0; q < B.np; ++q) {
      B.p[q] = to_dev(p[q0 + q]);
      B.first_block[q] = nb;
      nb += ((p[q0 + q].nx + 31) / 32) * ((p[q0 + q].ny + 3) / 4) * p[q0 + q].nz;
    }
    B.first_block[B.np] = nb;
    const dim3 blk(32, 4);
    switch (epi) {
      case 0: k_z4c<0><<<nb, blk, 0, st>>>(B, P, u_in, rhs, rk); break;
      case 1: k_z4c<1><<<nb, blk, 0, st>>>(B, P, u_in, rhs, rk); break;
      case 2: k_z4c<2><<<nb, blk, 0, st>>>(B, P, u_in, rhs, rk); break;
      case 3: k_z4c<3><<<nb, blk, 0, st>>>(B, P, u_in, rhs, rk); break;
      default: k_z4c<4><<<nb, blk, 0, st>>>(B, P, u_in, rhs, rk); break;
    }
    if (cudaGetLastError() != cudaSuccess) return SACRA_ERR_CUDA;
  }
  return SACRA_OK;
}

}  // namespace sacra

using namespace sacra;

extern "C" {

int sacra_fill_ghosts(const sacra_patch_t* p, int npatch, double* u, void* cuda_stream) {
  if (!p || !u) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(u)) return SACRA_ERR_ALIGN;
  return launch_fill(p, npatch, u, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_z4c_rhs(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, const double* u, double* rhs,
                  void* cuda_stream) {
  if (!p || !prm || !u || !rhs) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (!aligned16(u) || !aligned16(rhs)) return SACRA_ERR_ALIGN;
  if (u == rhs) return SACRA_ERR_BADARG;
  return launch_z4c(p, npatch, prm, 0, u, rhs, nullptr, nullptr, nullptr, static_cast<cudaStream_t>(cuda_stream));
}

int sacra_rk4_substep(const sacra_patch_t* p, int npatch, const sacra_params_t* prm, int stage, const double* u_n,
                      const double* u_in, double* u_out, double* acc, void* cuda_stream) {
  if (!p || !prm || !u_n || !u_in || !u_out || !acc) return SACRA_ERR_NULL;
  if (int e = check_patches(p, npatch)) return e;
  if (stage < 1 || stage > 4) return SACRA_ERR_BADARG;
  if (!aligned16(u_n) || !aligned16(u_in) || !aligned16(u_out) || !aligned16(acc)) return SACRA_ERR_ALIGN;
  if (u_out == u_in || acc == u_in || acc == u_n || acc == u_out) return SACRA_ERR_BADARG;
  return launch_z4c(p, npatch, prm, stage, u_in, nullptr, u_n, u_out, acc, static_cast<cudaStream_t>(cuda_stream));
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
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  double* w0 = work;
  double* w1 = work + state_doubles;
  double* acc = work + 2 * state_doubles;
  int e;
  if ((e = launch_fill(p, npatch, u, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 1, u, nullptr, u, w0, acc, st))) return e;
  if ((e = launch_fill(p, npatch, w0, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 2, w0, nullptr, u, w1, acc, st))) return e;
  if ((e = launch_fill(p, npatch, w1, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 3, w1, nullptr, u, w0, acc, st))) return e;
  if ((e = launch_fill(p, npatch, w0, st))) return e;
  if ((e = launch_z4c(p, npatch, prm, 4, w0, nullptr, u, u, acc, st))) return e;
  return launch_fill(p, npatch, u, st);
}

const char* sacra_strerror(int code) {
  switch (code) {
    case SACRA_OK: return "ok";
    case SACRA_ERR_NULL: return "null pointer argument";
    case SACRA_ERR_BADARG: return "bad argument (size, spacing, stage, layout or aliasing)";
    case SACRA_ERR_UNSUPPORTED: return "unsupported ghost width (ng must be 3)";
    case SACRA_ERR_ALIGN: return "pointer or layout breaks the 16-byte alignment rule";
    case SACRA_ERR_CUDA: return "CUDA launch failed";
    default: return "unknown sacra status";
  }
}

const char* sacra_version(void) { return "0.1"; }

}  // extern "C"
