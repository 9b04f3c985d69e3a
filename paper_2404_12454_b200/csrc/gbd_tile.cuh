// gbd_tile.cuh -- device helpers shared by the field-sum kernels (gbd_field.cu, gbd_sep.cu): mbarrier / 1-D bulk
// async copy wrappers (PTX) and the stream-K work partition.  Product code; nothing here is shared with oracle/.
#pragma once

#include "gbd_common.cuh"

namespace {

constexpr int KB = 128;                      // beamlets per shared-memory record stage

// ------------------------------------------------------------------ mbarrier / bulk copy (PTX)
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t *bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void bulk_g2s(void *dst, const void *src, uint32_t bytes, uint64_t *bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity)
        : "memory");
}

// One contiguous piece of a CTA's share: beamlets [j0, j1) of one pixel tile of one problem.  With a
// grouped launch (L.n_probs > 0) the problem is found by bisection on the concatenated work list.
struct Piece {
    const double *rec, *rec_abs;
    void *out;
    long n_b, tile, gtile, j0, j1;
};
template <bool GROUPED>
__device__ __forceinline__ Piece piece_at(const GbdFieldLaunch &L, long long pos, long long b1)
{
    Piece p;
    long long wbeg = 0;
    long ip = 0;
    if (GROUPED) {
        int lo = 0, hi = L.n_probs - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (L.probs[mid].work_begin <= pos) lo = mid; else hi = mid - 1;
        }
        ip = lo;
        p.rec = L.probs[lo].rec; p.out = L.probs[lo].out; p.n_b = L.probs[lo].n_b;
        p.rec_abs = L.probs[lo].rec_abs;
        wbeg = L.probs[lo].work_begin;
    } else {
        p.rec = L.rec; p.out = L.out; p.n_b = L.n_b; p.rec_abs = L.rec_abs;
    }
    const long long local = pos - wbeg;
    p.tile = (long)(local / p.n_b);
    p.j0 = (long)(local - (long long)p.tile * p.n_b);
    p.j1 = (long)min((long long)p.n_b, (long long)p.j0 + (b1 - pos));
    p.gtile = ip * L.tiles_per_problem + p.tile;
    return p;
}

}  // namespace
