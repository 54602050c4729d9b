// sm_100a bulk-asynchronous copy (TMA, 1-D `cp.async.bulk`, SASS UBLKCP) + mbarrier wrappers, and the
// chunk-stage helper used by the step and damage kernels: one thread streams every contiguous array of a
// chunk into shared memory in a single burst, all threads wait on one mbarrier.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace pff {

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}

// one arrival + the number of bytes the bulk copies will signal
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    const uint32_t addr = smem_u32(bar);
    uint32_t done;
    do {
        asm volatile(
            "{\n"
            ".reg .pred p;\n"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
            "selp.u32 %0, 1, 0, p;\n"
            "}\n" : "=r"(done) : "r"(addr), "r"(parity) : "memory");
    } while (!done);
}

// orders earlier generic-proxy accesses of shared memory before later asynchronous-proxy (TMA) writes to it
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// generic-proxy writes to global memory before a grid-wide barrier / asynchronous-proxy reads of them after it
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }

// Ampere-style asynchronous copy of ONE small element global -> shared (SASS LDGSTS): used for the indexed
// halo gathers, which must not hold register scoreboards across a whole chunk iteration.
template <int BYTES>
__device__ __forceinline__ void cp_async(void* dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], %2;" ::"r"(smem_u32(dst)), "l"(src), "n"(BYTES) : "memory");
}
// every cp.async this thread has issued so far arrives on `bar` when it completes (counts against the mbarrier's
// expected arrivals: .noinc), so ONE mbarrier wait covers the bulk copies and all threads' gathers of a stage
__device__ __forceinline__ void cp_async_mbar_arrive(uint64_t* bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// global -> shared bulk copy; dst, src 16-byte aligned, bytes a multiple of 16; completion on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(dst)), "l"(src), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}

// One contiguous array of a chunk stage.  kind selects the index range of the chunk that is copied:
// 0 = elements [elem_start, +n_elem) of Ne, 1 = interior nodes [node_start, +n_int) of N,
// 2 = gather-table entries [ell_off, +ell_w * nloc) of ell_total, 3 = halo entries [halo_off, +n_halo) of n_slots,
// 4 = halo entries of the NEXT chunk of a persistent CTA [next_halo_off, +next_n_halo) of n_slots.
struct StageDesc {
    const void* src;
    uint32_t dst_off;      // byte offset inside the stage (16-byte aligned)
    uint16_t esize_log2;   // log2 of the element size in bytes (0..4)
    uint16_t kind;
};
constexpr int kMaxStageArrays = 20;
struct StagePlan {
    StageDesc d[kMaxStageArrays];
    int n;
};

// One lane's share of a stage burst: lane `lane` of the issuing warp copies the array described by d (if have):
// element start + i of the global array lands at byte offset dst_off + ((start % A) + i) * esize, A = 16 / esize.
// The copy is widened to 16-byte boundaries: the source range stays inside [0, total) of its array by construction
// (a0 >= 0, a1 <= total rounded down) and the destination inside the stage region sized for it (verified on the host
// for every chunk by verify_stage_extents, mesh_setup.cpp); whatever would reach past the last full 16-byte group of
// the array is fetched with plain loads.  Lane 0 then
// arrives on the mbarrier with the total byte count of the warp.
struct ChunkRange {  // index ranges of one chunk, per descriptor kind
    int elem_start, n_elem, Ne, node_start, n_int, N, ell_off, ell_cnt, ell_total, halo_off, n_halo, n_slots, next_halo_off,
        next_n_halo;
};
__device__ __forceinline__ void stage_issue_desc(const StageDesc& d, bool have, unsigned char* stage, uint64_t* bar, int lane,
                                                 const ChunkRange& c)
{
    uint32_t bytes = 0;
    if (have) {
        int start = c.elem_start, count = c.n_elem, total = c.Ne;
        if (d.kind == 1) { start = c.node_start; count = c.n_int; total = c.N; }
        else if (d.kind == 2) { start = c.ell_off; count = c.ell_cnt; total = c.ell_total; }
        else if (d.kind == 3) { start = c.halo_off; count = c.n_halo; total = c.n_slots; }
        else if (d.kind == 4) { start = c.next_halo_off; count = c.next_n_halo; total = c.n_slots; }
        if (count > 0) {
            const int l = d.esize_log2, A1 = (16 >> l) - 1;
            const int a0 = start & ~A1, end = start + count;
            int a1 = min((end + A1) & ~A1, total & ~A1);
            const unsigned char* src = reinterpret_cast<const unsigned char*>(d.src);
            unsigned char* dst = stage + d.dst_off;
            if (a1 > a0) {
                bytes = uint32_t(a1 - a0) << l;
                bulk_g2s(dst, src + (size_t(a0) << l), bytes, bar);
            } else {
                a1 = a0;
            }
            for (size_t b = size_t(a1) << l; b < (size_t(end) << l); ++b) dst[b - (size_t(a0) << l)] = src[b];
        }
    }
    for (int o = 16; o > 0; o >>= 1) bytes += __shfl_xor_sync(0xffffffffu, bytes, o);
    if (lane == 0) mbar_arrive_expect_tx(bar, bytes);
}

// Grid-wide barrier of the cooperatively launched kernels (all CTAs are co-resident): one arrival per CTA on a counter that
// only grows (the epoch it starts from is kept on the device), thread 0 spins with acquire loads until the epoch's target.
__device__ __forceinline__ void grid_barrier(unsigned int* counter, unsigned int& target, unsigned int G)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        target += G;
        // release-arrive (orders this CTA's writes, observed through the block barrier above, before the arrival) and
        // acquire-poll; the comparison is wrap-safe
        asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(counter) : "memory");
        unsigned int seen;
        do {
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(seen) : "l"(counter) : "memory");
        } while ((int)(seen - target) < 0);
    }
    __syncthreads();
}

__host__ __device__ __forceinline__ int round_up(int v, int a) { return (v + a - 1) / a * a; }

}  // namespace pff
