// adft_rys_host.cuh -- host-side launch helpers of the Rys kernels, shared by adft_rys.cu (the f classes) and the
// generated instantiation units of the g classes (generated/rys_<tag>.cu).
#pragma once
#include <atomic>

#include "adft_internal.h"
#include "adft_rys.cuh"

namespace adft {

// resident blocks of the persistent grid, per device (occupancy x SM count), computed once per device
template <class C, bool WJ, bool WK>
inline int resident_blocks()
{
    constexpr int MAXDEV = 64;
    static std::atomic<int> cache[MAXDEV];
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev < 0 || dev >= MAXDEV) dev = 0;
    int nb = cache[dev].load(std::memory_order_relaxed);
    if (nb == 0) {
        int sms = 0, occ = 0;
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaFuncSetAttribute(jk_rys_kernel<C, WJ, WK>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, jk_rys_kernel<C, WJ, WK>, C::NT, C::SMEM_BYTES);
        nb = sms * (occ > 0 ? occ : 1);
        cache[dev].store(nb, std::memory_order_relaxed);
    }
    return nb;
}

template <class C, bool WJ, bool WK>
inline cudaError_t run_jk_variant(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, cudaStream_t st)
{
    const int nblocks = resident_blocks<C, WJ, WK>();
    const long long want = (p.total_warps - p.shard_rank + p.shard_count - 1) / p.shard_count;      // tiles of this rank
    if (want <= 0) return cudaSuccess;
    return launch_jk_rys<C, WJ, WK>(p, rt, tile_counter, (int)(want < nblocks ? want : nblocks), st);
}

template <class C>
inline cudaError_t run_jk(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, cudaStream_t st,
                          bool want_j, bool want_k)
{
    if (want_j && want_k) return run_jk_variant<C, true, true>(p, rt, tile_counter, st);
    if (want_j) return run_jk_variant<C, true, false>(p, rt, tile_counter, st);
    return run_jk_variant<C, false, true>(p, rt, tile_counter, st);
}

template <class C>
inline cudaError_t run_sw(const PairTable &t, const RysTable &rt, int pair_base, int prim_base, int n, int K, double *Qout,
                          cudaStream_t st)
{
    // persistent grid: as many blocks as fit on the device (one block works on one pair at a time)
    int dev = 0, sms = 0, occ = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    cudaFuncSetAttribute(schwarz_rys_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, schwarz_rys_kernel<C>, C::NT, C::SMEM_BYTES);
    return launch_schwarz_rys<C>(t, rt, pair_base, prim_base, n, K, Qout, sms * (occ > 0 ? occ : 1), st);
}

}  // namespace adft
