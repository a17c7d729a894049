// adft_internal.h -- host-side structures shared by the C-ABI translation unit and the class instantiation units.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string>
#include <vector>

#include "../../include/adft.h"
#include "adft_device.cuh"

namespace adft {

constexpr int NPAIRCLASS = 15;     // (la>=lb), la<=4:  pc = la(la+1)/2+lb
constexpr int NQCLASS = 120;       // X(X+1)/2+Y, X>=Y
static_assert(NQCLASS == ADFT_MAX_CLASSES, "adft_jk_stats_t is sized by ADFT_MAX_CLASSES");

inline int pair_class(int la, int lb) { return la * (la + 1) / 2 + lb; }       // requires la >= lb
inline int quartet_class(int X, int Y) { return X * (X + 1) / 2 + Y; }          // requires X >= Y

// Per-class launchers, filled by the instantiation units (one per generated class).
struct ClassEntry {
    void (*launch_jk)(const JKParams &p, cudaStream_t st, bool want_j, bool want_k, bool fp32) = nullptr;
    int la = 0, lb = 0, lc = 0, ld = 0;
    int vrr_ops = 0, hrr_ops = 0, nint = 0;   // FP64 instruction counts from the generator
    const char *impl = "none";                // "straightline" | "rys"
    bool use_rys = false;                     // this class runs through the block-cooperative Rys kernels (adft_rys.cuh)
};

// Rys kernels (adft_rys.cu): launchers per class, nullptr where none is instantiated
struct RysTable;
typedef cudaError_t (*rys_jk_fn)(const JKParams &p, const RysTable &rt, unsigned long long *tile_counter, cudaStream_t st,
                                 bool want_j, bool want_k);
typedef cudaError_t (*rys_sw_fn)(const PairTable &t, const RysTable &rt, int pair_base, int prim_base, int n, int K,
                                 double *Qout, cudaStream_t st);
rys_jk_fn rys_jk_launcher(int la, int lb, int lc, int ld);
rys_sw_fn rys_schwarz_launcher(int la, int lb);
rys_jk_fn rys_jk_launcher_g(int lb, int lc, int ld);      // classes with a g shell on the bra: generated/rys_g_registry.cu
rys_sw_fn rys_schwarz_launcher_g(int lb);
ClassEntry *class_table();                    // [NQCLASS]
void register_all_classes();                  // defined in generated registry.cu

void set_error(const std::string &msg);

}  // namespace adft
