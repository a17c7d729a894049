// adft_rys.cu -- instantiations of the block-cooperative Rys kernels (adft_rys.cuh) for the quartet classes without
// straight-line code, and of the Schwarz kernels of every pair class.
#include <atomic>

#include "adft_internal.h"
#include "adft_rys.cuh"

namespace adft {

// resident blocks of the persistent grid, per device (occupancy x SM count), computed once per device
template <class C, bool WJ, bool WK>
static int resident_blocks()
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
static cudaError_t run_jk_variant(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, cudaStream_t st)
{
    const int nblocks = resident_blocks<C, WJ, WK>();
    const long long want = (p.total_warps - p.shard_rank + p.shard_count - 1) / p.shard_count;      // tiles of this rank
    if (want <= 0) return cudaSuccess;
    return launch_jk_rys<C, WJ, WK>(p, rt, tile_counter, (int)(want < nblocks ? want : nblocks), st);
}

template <class C>
static cudaError_t run_jk(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, cudaStream_t st,
                          bool want_j, bool want_k)
{
    if (want_j && want_k) return run_jk_variant<C, true, true>(p, rt, tile_counter, st);
    if (want_j) return run_jk_variant<C, true, false>(p, rt, tile_counter, st);
    return run_jk_variant<C, false, true>(p, rt, tile_counter, st);
}

template <class C>
static cudaError_t run_sw(const PairTable &t, const RysTable &rt, int pair_base, int prim_base, int n, int K, double *Qout,
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

// X(la, lb, lc, ld, NCH): NCH = number of cd chunks = thread groups per quartet.  Phase 2 is bound by shared-memory
// bandwidth (3*(lc+1)(ld+1) loads per 2*CH FP64 instructions per batch item), so NCH is as small as the register file
// allows (CH = ceil(NC*ND/NCH) contracted integrals per thread, <= 50).
#define ADFT_RYS_CLASSES(X) \
    X(3, 1, 3, 1, 2)        \
    X(3, 3, 1, 1, 1)        \
    X(3, 2, 2, 1, 1)        \
    X(3, 3, 3, 0, 1)        \
    X(3, 1, 2, 2, 2)        \
    X(3, 2, 3, 1, 1)        \
    X(3, 3, 2, 1, 1)        \
    X(3, 2, 2, 2, 1)        \
    X(3, 3, 3, 1, 1)        \
    X(3, 2, 3, 2, 2)        \
    X(3, 3, 2, 2, 1)        \
    X(3, 3, 3, 2, 2)        \
    X(3, 3, 3, 3, 2)

rys_jk_fn rys_jk_launcher(int la, int lb, int lc, int ld)
{
#define X(A, B, C_, D, NCH) \
    if (la == A && lb == B && lc == C_ && ld == D) return run_jk<RysCfg<A, B, C_, D, NCH>>;
    ADFT_RYS_CLASSES(X)
#undef X
    return nullptr;
}

rys_sw_fn rys_schwarz_launcher(int la, int lb)
{
    // every pair class: the Rys kernel chooses the recurrence centre per primitive pair (R-22), so the bounds
    // agree with the oracle's to 1e-10 relative also where a tight shell receives its angular momentum by transfer
    if (la == 0 && lb == 0) return run_sw<RysCfg<0, 0, 0, 0, 1>>;
    if (la == 1 && lb == 0) return run_sw<RysCfg<1, 0, 1, 0, 1>>;
    if (la == 1 && lb == 1) return run_sw<RysCfg<1, 1, 1, 1, 1>>;
    if (la == 2 && lb == 0) return run_sw<RysCfg<2, 0, 2, 0, 1>>;
    if (la == 2 && lb == 1) return run_sw<RysCfg<2, 1, 2, 1, 1>>;
    if (la == 2 && lb == 2) return run_sw<RysCfg<2, 2, 2, 2, 1>>;
    if (la == 3 && lb == 0) return run_sw<RysCfg<3, 0, 3, 0, 1>>;
    if (la == 3 && lb == 1) return run_sw<RysCfg<3, 1, 3, 1, 2>>;
    if (la == 3 && lb == 2) return run_sw<RysCfg<3, 2, 3, 2, 2>>;
    if (la == 3 && lb == 3) return run_sw<RysCfg<3, 3, 3, 3, 2>>;
    return nullptr;
}

}  // namespace adft
