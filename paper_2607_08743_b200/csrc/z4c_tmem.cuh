// z4c_tmem.cuh -- Tensor Memory (TMEM, 256 KB per SM on sm_100a) as per-thread scratch for the fused Z4c kernel.
//
// The point-wise algebra of the Z4c right-hand side keeps ~100 FP64 values per grid point
// alive across the 25 field passes; in registers alone that pins the kernel at 255 registers per thread and 8 warps
// per SM. The kernel uses no tensor cores, so TMEM is free: every thread parks its long-lived tensors (d_k beta^i,
// d_k gt_ij, Gt^k_ij, At^ij, the centre values of all fields) in a private strip of TMEM and pulls them back with
// tcgen05.ld when a block of the algebra needs them. TMEM is 128 lanes x 512 columns x 32 bit; warp w of a CTA may
// touch lanes 32 (w % 4) .. + 31 only, so thread (w, lane l) owns lane 32 (w % 4) + l and a column range chosen by
// w / 4. A double takes two columns. Measured on B200 (256 / 384 / 512 threads per SM): a dependent ld + wait round
// trip 54-60 cycles, 660-740 B per clock and SM for loads, about the same for stores -- five times the shared-memory
// pipe, and not competing with the stencil loads for it.
// Accesses are .32x32b (lane l of the warp <-> TMEM lane base + l), x2 / x4 / x8 / x16 = 1 / 2 / 4 / 8 doubles.
#pragma once
#include <cstdint>

namespace sacra {
namespace tmem {

__device__ __forceinline__ void alloc_all(uint32_t* smem_result) {   // one warp: all 512 columns (one CTA per SM)
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"(
                   (uint32_t)__cvta_generic_to_shared(smem_result))
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void dealloc_all(uint32_t base) {         // the same warp
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(base) : "memory");
}
__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;"); }

#define SACRA_LO(x) __double2loint(x)
#define SACRA_HI(x) __double2hiint(x)
__device__ __forceinline__ void st1(uint32_t a, double v0) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(a), "r"(SACRA_LO(v0)), "r"(SACRA_HI(v0)));
}
__device__ __forceinline__ void st2(uint32_t a, double v0, double v1) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(SACRA_LO(v0)),
               "r"(SACRA_HI(v0)), "r"(SACRA_LO(v1)), "r"(SACRA_HI(v1)));
}
__device__ __forceinline__ void st4(uint32_t a, double v0, double v1, double v2, double v3) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(a),
               "r"(SACRA_LO(v0)), "r"(SACRA_HI(v0)), "r"(SACRA_LO(v1)), "r"(SACRA_HI(v1)), "r"(SACRA_LO(v2)),
               "r"(SACRA_HI(v2)), "r"(SACRA_LO(v3)), "r"(SACRA_HI(v3)));
}
#undef SACRA_LO
#undef SACRA_HI

// The st / ld wrappers carry no "memory" clobber (they touch no ordinary memory; volatile keeps them ordered among
// themselves and with the barriers), so the compiler stays free to schedule the stencil's shared-memory loads around them.
// loads are asynchronous: the destination registers are valid after wait_ld(). The Pack types keep the raw 32-bit
// halves; get(i) assembles double i (a register pair, no instruction).
struct Pack1 { uint32_t r[2]; __device__ __forceinline__ double get(int i) const { return __hiloint2double(r[2 * i + 1], r[2 * i]); } };
struct Pack2 { uint32_t r[4]; __device__ __forceinline__ double get(int i) const { return __hiloint2double(r[2 * i + 1], r[2 * i]); } };
struct Pack4 { uint32_t r[8]; __device__ __forceinline__ double get(int i) const { return __hiloint2double(r[2 * i + 1], r[2 * i]); } };

__device__ __forceinline__ void ld1(uint32_t a, Pack1& p) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(p.r[0]), "=r"(p.r[1]) : "r"(a));
}
__device__ __forceinline__ void ld2(uint32_t a, Pack2& p) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
               : "=r"(p.r[0]), "=r"(p.r[1]), "=r"(p.r[2]), "=r"(p.r[3])
               : "r"(a));
}
__device__ __forceinline__ void ld4(uint32_t a, Pack4& p) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(p.r[0]), "=r"(p.r[1]), "=r"(p.r[2]), "=r"(p.r[3]), "=r"(p.r[4]), "=r"(p.r[5]), "=r"(p.r[6]),
                 "=r"(p.r[7])
               : "r"(a));
}

// wait for every outstanding load of this thread. The packs that were loaded are passed through the asm as in/out
// operands, so the compiler cannot move a use of their registers above the wait.
__device__ __forceinline__ void touch(Pack1& p) { asm volatile("" : "+r"(p.r[0]), "+r"(p.r[1])); }
__device__ __forceinline__ void touch(Pack2& p) { asm volatile("" : "+r"(p.r[0]), "+r"(p.r[1]), "+r"(p.r[2]), "+r"(p.r[3])); }
__device__ __forceinline__ void touch(Pack4& p) {
  asm volatile("" : "+r"(p.r[0]), "+r"(p.r[1]), "+r"(p.r[2]), "+r"(p.r[3]), "+r"(p.r[4]), "+r"(p.r[5]), "+r"(p.r[6]), "+r"(p.r[7]));
}
template <class... P>
__device__ __forceinline__ void wait_ld(P&... p) {
  asm volatile("tcgen05.wait::ld.sync.aligned;");
  (touch(p), ...);
}

}  // namespace tmem
}  // namespace sacra
