// psr_ptx.cuh -- thin wrappers over the sm_100a PTX the kernels use: mbarriers, 1-D bulk (TMA) copies,
// cp.async, non-coherent global loads and shared-memory access by 32-bit address.  Internal to the library.
#ifndef PSR_PTX_CUH_
#define PSR_PTX_CUH_
#include <cuda_runtime.h>
#include <stdint.h>

namespace psr {

// ------------------------------------------------------------------ mbarrier / bulk copy
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.b32 %0, 1, 0, p;\n}"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
  } while (!done);
}

__device__ __forceinline__ void cp_async8(double* dst_smem, const double* src_global) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(smem_u32(dst_smem)), "l"(src_global) : "memory");
}
__device__ __forceinline__ double ldg_nc(const double* p) {
  double v;
  asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(v) : "l"(p));
  return v;
}

// ------------------------------------------------------------------ shared-memory access by 32-bit address
// (volatile so that loads are neither merged across tiles nor moved over barriers by the front end)
__device__ __forceinline__ double lds64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}
__device__ __forceinline__ void sts64(uint32_t addr, double v) {
  asm volatile("st.shared.f64 [%0], %1;" ::"r"(addr), "d"(v));
}
// non-blocking arrive (release) on an mbarrier of this CTA
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// barrier among a subset of the CTA's warps (id 1..15, count a multiple of 32)
__device__ __forceinline__ void named_bar_sync(int id, int count) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// ------------------------------------------------------------------ tensor memory as a per-lane scratchpad
// TMEM is [128 lanes][512 columns of 32 bits] per SM; warp w of a CTA reaches the 32 lanes of quadrant w % 4, thread
// l <-> lane 32 (w % 4) + l (.32x32b shape), at a column address that is the same in every thread.  A [row][32 lanes]
// tile of doubles maps to lane <-> reactor, row r <-> columns 2r, 2r + 1.  Its read path (64 B/clk/SM, 12 clk) is
// separate from the shared-memory pipe, which is what the reaction loops are short of.
// Address = (lane << 16) | column.  Whole-warp instructions (.sync.aligned): call them converged.
__device__ __forceinline__ void tm_alloc(uint32_t* slot_smem, uint32_t ncols) {   // ncols: power of two, 32..512
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot_smem)), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_dealloc(uint32_t base, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(ncols) : "memory");
}
// four rows (eight columns) of this thread's lane
__device__ __forceinline__ void tm_st64x4(uint32_t taddr, double v0, double v1, double v2, double v3) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"r"(taddr), "r"(__double2loint(v0)),
               "r"(__double2hiint(v0)), "r"(__double2loint(v1)), "r"(__double2hiint(v1)), "r"(__double2loint(v2)),
               "r"(__double2hiint(v2)), "r"(__double2loint(v3)), "r"(__double2hiint(v3))
               : "memory");
}
__device__ __forceinline__ void tm_st64(uint32_t taddr, double v) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(__double2loint(v)), "r"(__double2hiint(v)) : "memory");
}
// one row of this thread's lane; the registers are valid after tm_wait_ld* only
struct TmF64 {
  uint32_t lo, hi;
  __device__ __forceinline__ double get() const { return __hiloint2double((int)hi, (int)lo); }
};
__device__ __forceinline__ void tm_ld64(uint32_t taddr, TmF64& v) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(v.lo), "=r"(v.hi) : "r"(taddr));
}
// every tcgen05.ld of this thread so far has landed (the registers pass through the statement, so no use of them can
// be scheduled above it)
__device__ __forceinline__ void tm_wait_ld6(TmF64& a, TmF64& b, TmF64& c, TmF64& d, TmF64& e, TmF64& f) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(a.lo), "+r"(a.hi), "+r"(b.lo), "+r"(b.hi), "+r"(c.lo), "+r"(c.hi), "+r"(d.lo), "+r"(d.hi), "+r"(e.lo),
                 "+r"(e.hi), "+r"(f.lo), "+r"(f.hi)::"memory");
}
__device__ __forceinline__ void tm_wait_ld4(TmF64& a, TmF64& b, TmF64& c, TmF64& d) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(a.lo), "+r"(a.hi), "+r"(b.lo), "+r"(b.hi), "+r"(c.lo), "+r"(c.hi), "+r"(d.lo), "+r"(d.hi)::"memory");
}
__device__ __forceinline__ void tm_wait_ld1(TmF64& a) {
  asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(a.lo), "+r"(a.hi)::"memory");
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// order this thread's tcgen05 operations against a barrier / mbarrier operation that follows (before) or precedes (after)
__device__ __forceinline__ void tm_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ------------------------------------------------------------------ bounds checks of the -DPSR_CHECK build
// compute-sanitizer is refused on the GPU pool this library is developed on.  In its place the
// PSR_CHECK build asserts, on the device, every shared-memory offset the kernels take from the mechanism tables and
// every global output index against its bound: PSR_CHK(cond, code) counts a failure and keeps the first code (the
// access still happens: with all checks green nothing is out of range).  In the product build the macro is empty and
// its arguments are not evaluated.  Each translation unit has its own counter (no relocatable device code);
// psr_check_failures (psr_api.cu) sums them.
#ifdef PSR_CHECK
static __device__ unsigned int g_psr_chk[2];   // failures, first failing code
#define PSR_CHK(cond, code)                                                       \
  do {                                                                            \
    if (!(cond)) {                                                                \
      if (atomicAdd(&g_psr_chk[0], 1u) == 0u) g_psr_chk[1] = (unsigned)(code);    \
    }                                                                             \
  } while (0)
// host: read and reset this translation unit's counter (synchronises the device)
static inline cudaError_t psr_chk_read_reset(unsigned int* count, unsigned int* first_code) {
  unsigned int h[2] = {0u, 0u}, z[2] = {0u, 0u};
  cudaError_t e = cudaDeviceSynchronize();
  if (e == cudaSuccess) e = cudaMemcpyFromSymbol(h, g_psr_chk, sizeof h);
  if (e == cudaSuccess) e = cudaMemcpyToSymbol(g_psr_chk, z, sizeof z);
  *count = h[0];
  *first_code = h[1];
  return e;
}
#define PSR_CHK_TU_READER(name) \
  cudaError_t name(unsigned int* count, unsigned int* first_code) { return psr_chk_read_reset(count, first_code); }
#else
#define PSR_CHK(cond, code) ((void)0)
#define PSR_CHK_TU_READER(name) \
  cudaError_t name(unsigned int* count, unsigned int* first_code) { *count = 0u; *first_code = 0u; return cudaSuccess; }
#endif

}  // namespace psr
#endif
