// tmem.cuh — tensor memory (TMEM, 128 lanes x 512 columns x 32 bit per SM) as a per-thread parking place.
//
// Nothing in this library is a tensor-core contraction, but the 256 KB of TMEM are there and idle: the fused row kernels keep
// one packed field of a line waiting while another is transformed (the "stash", touched by its owner thread only).  In TMEM that
// costs no shared memory and none of the shared-memory data pipe's wavefronts: tcgen05.st / tcgen05.ld (SASS STTM / LDTM) have
// their own datapath.  Shape 32x32b: thread i of warp w addresses lane 32 (w mod 4) + i and N consecutive columns, i.e. a warp owns
// a private 32-lane x N-column tile; warps w and w + 4 share a lane quarter and take different columns.
//
// Protocol (blackwell_cuda_programming.md, "TMEM"): one warp allocates a power-of-two number of columns (>= 32) and publishes the
// base address through shared memory (fence, barrier, fence); the same warp frees them before the kernel ends.
#pragma once
#include "ttsh_common.cuh"

namespace ttsh {

// called by ONE full warp; ncols = 32, 64, 128, 256 or 512
__device__ __forceinline__ void tmem_alloc(unsigned* smem_holder, unsigned ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(smem_holder)),
               "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(unsigned base, unsigned ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// address of this warp's tile: lane quarter of the warp, column col0 (relative to the allocation)
__device__ __forceinline__ unsigned tmem_warp_addr(unsigned base, int warp, int col0) {
  return base + ((unsigned)(32 * (warp & 3)) << 16) + (unsigned)col0;
}

// 16 columns = 4 complex doubles (or 8 complex floats) of the calling thread.  Warp-collective (.sync.aligned).
__device__ __forceinline__ void tmem_st16(unsigned taddr, const unsigned (&r)[16]) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
               "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
               "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
               : "memory");
}
__device__ __forceinline__ void tmem_ld16(unsigned taddr, unsigned (&r)[16]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
               : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                 "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
               : "r"(taddr)
               : "memory");
}

// 16 columns hold TmemPack<T>::CH complex values of the calling thread: four complex doubles or eight complex floats
template <typename T> struct TmemPack { static constexpr int CH = 16 / (2 * (int)sizeof(T) / 4); };
__device__ __forceinline__ void tmem_stc(unsigned taddr, const cplx<double>* v) {
  unsigned r[16];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    r[4 * i + 0] = (unsigned)__double2loint(v[i].x); r[4 * i + 1] = (unsigned)__double2hiint(v[i].x);
    r[4 * i + 2] = (unsigned)__double2loint(v[i].y); r[4 * i + 3] = (unsigned)__double2hiint(v[i].y);
  }
  tmem_st16(taddr, r);
}
__device__ __forceinline__ void tmem_stc(unsigned taddr, const cplx<float>* v) {
  unsigned r[16];
#pragma unroll
  for (int i = 0; i < 8; ++i) { r[2 * i] = __float_as_uint(v[i].x); r[2 * i + 1] = __float_as_uint(v[i].y); }
  tmem_st16(taddr, r);
}
struct TmemQuad { unsigned r[16]; };
__device__ __forceinline__ void tmem_ldc_issue(unsigned taddr, TmemQuad& q) { tmem_ld16(taddr, q.r); }
// tcgen05.ld is asynchronous: its registers are valid after tcgen05.wait::ld.  The registers are in/out operands of the wait, so
// that no use of them can be scheduled above it.
__device__ __forceinline__ void tmem_wait_ld(TmemQuad& q) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+r"(q.r[0]), "+r"(q.r[1]), "+r"(q.r[2]), "+r"(q.r[3]), "+r"(q.r[4]), "+r"(q.r[5]), "+r"(q.r[6]), "+r"(q.r[7]), "+r"(q.r[8]),
                 "+r"(q.r[9]), "+r"(q.r[10]), "+r"(q.r[11]), "+r"(q.r[12]), "+r"(q.r[13]), "+r"(q.r[14]), "+r"(q.r[15])
               :
               : "memory");
}
// value i of the 16 columns, after tmem_wait_ld(q); the last argument selects the scalar type
__device__ __forceinline__ cplx<double> tmem_getc(const TmemQuad& q, int i, double) {
  return mk<double>(__hiloint2double((int)q.r[4 * i + 1], (int)q.r[4 * i + 0]), __hiloint2double((int)q.r[4 * i + 3], (int)q.r[4 * i + 2]));
}
__device__ __forceinline__ cplx<float> tmem_getc(const TmemQuad& q, int i, float) {
  return mk<float>(__uint_as_float(q.r[2 * i]), __uint_as_float(q.r[2 * i + 1]));
}

}  // namespace ttsh
