// adft_rys.cu -- instantiations of the block-cooperative Rys kernels (adft_rys.cuh) for the quartet classes without
// straight-line code, and of the Schwarz kernels of every pair class.
#include "adft_rys_host.cuh"

namespace adft {

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
    if (la == 4) return rys_jk_launcher_g(lb, lc, ld);      // g classes: generated/rys_g_registry.cu
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
    if (la == 4) return rys_schwarz_launcher_g(lb);
    return nullptr;
}

}  // namespace adft
