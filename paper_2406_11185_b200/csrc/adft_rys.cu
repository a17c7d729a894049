// adft_rys.cu -- instantiations of the block-cooperative Rys kernels (adft_rys.cuh) for the quartet classes without
// straight-line code, and of the Schwarz kernels of the pair classes (fp), (fd), (ff).
#include "adft_internal.h"
#include "adft_rys.cuh"

namespace adft {

template <class C>
static cudaError_t run_jk(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, cudaStream_t st)
{
    static int nblocks = 0;
    if (nblocks == 0) {
        int dev = 0, sms = 0, occ = 0;
        cudaGetDevice(&dev);
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        cudaFuncSetAttribute(jk_rys_kernel<C>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)C::SMEM_BYTES);
        cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, jk_rys_kernel<C>, C::NT, C::SMEM_BYTES);
        nblocks = sms * (occ > 0 ? occ : 1);
    }
    const long long want = p.total_warps;
    return launch_jk_rys<C>(p, rt, tile_counter, (int)(want < nblocks ? want : nblocks), st);
}

template <class C>
static cudaError_t run_sw(const PairTable &t, const RysTable &rt, int pair_base, int prim_base, int n, int K, double *Qout,
                          cudaStream_t st)
{
    int dev = 0, sms = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    return launch_schwarz_rys<C>(t, rt, pair_base, prim_base, n, K, Qout, 2 * sms, st);
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
    if (la == 3 && lb == 1) return run_sw<RysCfg<3, 1, 3, 1, 2>>;
    if (la == 3 && lb == 2) return run_sw<RysCfg<3, 2, 3, 2, 2>>;
    if (la == 3 && lb == 3) return run_sw<RysCfg<3, 3, 3, 3, 2>>;
    return nullptr;
}

}  // namespace adft
