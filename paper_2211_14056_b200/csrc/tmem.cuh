// tmem.cuh — tensor memory (Blackwell TMEM, 512 columns x 128 lanes x 32 bit per SM) used as a parking lot for
// register-resident accumulators: the colour-flow vector J of me_eval is the accumulator of the dot stages and is
// dead while the next round's currents are computed, so it is moved out of the register file with tcgen05.st and
// back with tcgen05.ld (shape 32x32b: register k of lane l of warp w <-> TMEM lane 32 (w % 4) + l, column c0 + k).
// No tensor-core instruction touches it.  Measured on B200: 96 registers per thread, 8 warps at once, store + load
// round trip in 334 cycles (profiles/r2_probes.md).
#pragma once
#include <stdint.h>

namespace madme {

constexpr int tmem_cols(int need) { return need <= 32 ? 32 : need <= 64 ? 64 : need <= 128 ? 128 : need <= 256 ? 256 : 512; }

// Allocate COLS columns for the CTA (warp 0 allocates, every thread gets the base address).  Ends with a barrier.
template <int COLS> __device__ __forceinline__ uint32_t tmem_alloc() {
  static_assert(COLS >= 32 && COLS <= 512 && (COLS & (COLS - 1)) == 0, "power of two between 32 and 512");
  __shared__ uint32_t base_s;
  if ((threadIdx.x >> 5) == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;"
                 :: "r"(static_cast<uint32_t>(__cvta_generic_to_shared(&base_s))), "n"(COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
  return base_s;
}
// Every warp must be done with its columns: call after a CTA barrier-free tail is acceptable because it barriers itself.
template <int COLS> __device__ __forceinline__ void tmem_free(uint32_t base) {
  asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
  __syncthreads();
  if ((threadIdx.x >> 5) == 0)
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" :: "r"(base), "n"(COLS) : "memory");
}

__device__ __forceinline__ void tmem_st_x32(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};"
               :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]), "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]), "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]), "r"(r[31]) : "memory");
}
__device__ __forceinline__ void tmem_ld_x32(uint32_t taddr, uint32_t* r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st_x8(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};"
               :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}
__device__ __forceinline__ void tmem_ld_x8(uint32_t taddr, uint32_t* r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr) : "memory");
}
__device__ __forceinline__ void tmem_st_x4(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1,%2,%3,%4};"
               :: "r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]) : "memory");
}
__device__ __forceinline__ void tmem_ld_x4(uint32_t taddr, uint32_t* r) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(taddr) : "memory");
}

// N registers per thread (a multiple of 4) to / from columns taddr .. taddr + N - 1 of the warp's lanes; both wait for
// completion (the registers may be reused / are valid on return).
template <int N> __device__ __forceinline__ void tmem_store(uint32_t taddr, const uint32_t* r) {
  static_assert(N % 4 == 0, "multiples of four registers");
  int k = 0;
#pragma unroll
  for (; k + 32 <= N; k += 32) tmem_st_x32(taddr + k, r + k);
#pragma unroll
  for (; k + 8 <= N; k += 8) tmem_st_x8(taddr + k, r + k);
#pragma unroll
  for (; k + 4 <= N; k += 4) tmem_st_x4(taddr + k, r + k);
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}
template <int N> __device__ __forceinline__ void tmem_load(uint32_t taddr, uint32_t* r) {
  static_assert(N % 4 == 0, "multiples of four registers");
  int k = 0;
#pragma unroll
  for (; k + 32 <= N; k += 32) tmem_ld_x32(taddr + k, r + k);
#pragma unroll
  for (; k + 8 <= N; k += 8) tmem_ld_x8(taddr + k, r + k);
#pragma unroll
  for (; k + 4 <= N; k += 4) tmem_ld_x4(taddr + k, r + k);
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

}  // namespace madme
