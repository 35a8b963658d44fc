// tmem.cuh -- tensor memory (TMEM, the accumulator store of the sm_100a tensor cores) used as per-lane scratch memory.
//
// TMEM is 128 lanes x 512 columns of 32 bits per SM.  With the 32x32b shape of tcgen05.ld / tcgen05.st a thread reads and
// writes consecutive columns of ITS OWN lane (lane = 32 (warp % 4) + lane of the warp: a warp reaches the 32 lanes of its
// quadrant only), the column index being a warp-uniform run-time value: per-thread storage that is indexed dynamically
// (which registers are not) and whose read path does not share the shared-memory pipe.  Measured on B200
// (16 warps per SM, four x4 loads + wait per trip): >= 330 B/cycle/SM, 40 cycles for a lone warp's four loads.
// Allocation: one warp of the block calls tm_alloc (a power of two >= 32 columns; the blocks resident on an SM must
// fit the 512 columns together, otherwise the allocation waits for another block to free its columns).
#pragma once
#include <stdint.h>

namespace crf {

__device__ __forceinline__ void tm_alloc(unsigned *smem_result, unsigned cols)
{
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(smem_result)),
                 "r"(cols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tm_dealloc(unsigned base, unsigned cols)
{
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(cols) : "memory");
}
// around a block-wide barrier that orders tensor-memory accesses of different warps
__device__ __forceinline__ void tm_fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// the address of column `col` in the quadrant of warp `warp`
__device__ __forceinline__ unsigned tm_quadrant(unsigned base, int warp) { return base + (((unsigned)(warp & 3) * 32u) << 16); }

// ---- rows of PPL doubles ---------------------------------------------------------------------------------------------
// A row of PPL doubles is 2 PPL columns.  Loads are asynchronous: the registers are valid after tm_wait, which takes
// them as operands so that no use can be scheduled before it.
template <int PPL>
struct TmRow {
    unsigned r[2 * PPL];
};
template <int PPL>
__device__ __forceinline__ void tm_ld(unsigned taddr, TmRow<PPL> &t)
{
    if (PPL == 2)
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(t.r[0]), "=r"(t.r[1]), "=r"(t.r[2 * PPL - 2]), "=r"(t.r[2 * PPL - 1])
                     : "r"(taddr));
    else
        asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(t.r[0]), "=r"(t.r[1]) : "r"(taddr));
}
template <int PPL>
__device__ __forceinline__ void tm_st(unsigned taddr, const double (&v)[PPL])
{
    if (PPL == 2)
        asm volatile("tcgen05.st.sync.aligned.32x32b.x4.b32 [%0], {%1, %2, %3, %4};" ::"r"(taddr), "r"(__double2loint(v[0])),
                     "r"(__double2hiint(v[0])), "r"(__double2loint(v[PPL - 1])), "r"(__double2hiint(v[PPL - 1]))
                     : "memory");
    else
        asm volatile("tcgen05.st.sync.aligned.32x32b.x2.b32 [%0], {%1, %2};" ::"r"(taddr), "r"(__double2loint(v[0])),
                     "r"(__double2hiint(v[0]))
                     : "memory");
}
template <int PPL>
__device__ __forceinline__ void tm_wait1(TmRow<PPL> &a)
{
    if (PPL == 2)
        asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(a.r[0]), "+r"(a.r[1]), "+r"(a.r[2 * PPL - 2]), "+r"(a.r[2 * PPL - 1]));
    else
        asm volatile("tcgen05.wait::ld.sync.aligned;" : "+r"(a.r[0]), "+r"(a.r[1]));
}
template <int PPL>
__device__ __forceinline__ void tm_get(const TmRow<PPL> &t, double (&v)[PPL])
{
#pragma unroll
    for (int u = 0; u < PPL; ++u) v[u] = __hiloint2double((int)t.r[2 * u + 1], (int)t.r[2 * u]);
}

// one wait for four rows in flight (a wait covers every earlier load of the thread; the operands order the uses)
__device__ __forceinline__ void tm_wait4(TmRow<2> &a, TmRow<2> &b, TmRow<2> &c, TmRow<2> &d)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a.r[0]), "+r"(a.r[1]), "+r"(a.r[2]), "+r"(a.r[3]), "+r"(b.r[0]), "+r"(b.r[1]), "+r"(b.r[2]), "+r"(b.r[3]),
                   "+r"(c.r[0]), "+r"(c.r[1]), "+r"(c.r[2]), "+r"(c.r[3]), "+r"(d.r[0]), "+r"(d.r[1]), "+r"(d.r[2]), "+r"(d.r[3]));
}
__device__ __forceinline__ void tm_wait4(TmRow<1> &a, TmRow<1> &b, TmRow<1> &c, TmRow<1> &d)
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a.r[0]), "+r"(a.r[1]), "+r"(b.r[0]), "+r"(b.r[1]), "+r"(c.r[0]), "+r"(c.r[1]), "+r"(d.r[0]), "+r"(d.r[1]));
}
__device__ __forceinline__ double2 tm_pair(const TmRow<2> &t)
{
    return make_double2(__hiloint2double((int)t.r[1], (int)t.r[0]), __hiloint2double((int)t.r[3], (int)t.r[2]));
}
__device__ __forceinline__ double tm_one(const TmRow<1> &t) { return __hiloint2double((int)t.r[1], (int)t.r[0]); }

}  // namespace crf
