// adft_lib.cu -- the C ABI of include/adft.h: basis ingest (a1), shell-pair table + Schwarz (a2),
// screening plan (a3), class launches (a4/a5), finalise (a6), stats, FP64 peak microbenchmark.
#include <algorithm>
#include <cfloat>
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <numeric>

#include <mutex>

#include "adft_internal.h"
#include "adft_rys.cuh"
#include "adft_sph.cuh"
#include "../../include/adft_noalloc.h"

namespace adft {

static thread_local std::string g_last_error;
void set_error(const std::string &msg) { g_last_error = msg; }

static ClassEntry g_classes[NQCLASS];
ClassEntry *class_table() { return g_classes; }
static std::once_flag g_register_once;

}  // namespace adft
// Rys root/weight tables (generated/rys_tables.bin from csrc/gen/gen_rys.py, linked in through generated/rys_blob.S)
extern "C" const double adft_rys_blob[];
extern "C" const double adft_rys_blob_end[];
namespace adft {

// Fill the class table once per process: the generated straight-line classes register themselves (generated/registry.cu);
// every other class of generated/class_meta.inc (angular momenta and the generator's FP64 instruction counts, used for
// the model flops) runs through the block-cooperative Rys kernels.
static void ensure_registered()
{
    std::call_once(g_register_once, [] {
        register_all_classes();
        static const struct { int qc, la, lb, lc, ld, vrr_ops, hrr_ops, nint; } meta[] = {
#define ADFT_CLASS_META(qc, la, lb, lc, ld, vrr_ops, hrr_ops, nint) {qc, la, lb, lc, ld, vrr_ops, hrr_ops, nint},
#include "generated/class_meta.inc"
#undef ADFT_CLASS_META
        };
        for (const auto &m : meta) {
            ClassEntry &e = g_classes[m.qc];
            if (e.launch_jk || !rys_jk_launcher(m.la, m.lb, m.lc, m.ld)) continue;
            e.use_rys = true;
            e.impl = "rys";
            e.la = m.la; e.lb = m.lb; e.lc = m.lc; e.ld = m.ld;
            e.vrr_ops = m.vrr_ops; e.hrr_ops = m.hrr_ops; e.nint = m.nint;
        }
    });
}

#define CUDA_TRY(expr)                                                                           \
    do {                                                                                         \
        cudaError_t e__ = (expr);                                                                \
        if (e__ != cudaSuccess) {                                                                \
            set_error(std::string(#expr) + ": " + cudaGetErrorString(e__));                      \
            return ADFT_ERR_CUDA;                                                                \
        }                                                                                        \
    } while (0)

static inline int ncart(int l) { return (l + 1) * (l + 2) / 2; }
static inline size_t prim_chunks(size_t nprimpairs) { return (nprimpairs + 7) / 8; }      // 8 records per chunk (PairTable::prim)
#define ADFT_MAX_PRIM_PAIRS (ADFT_MAX_NPRIM * ADFT_MAX_NPRIM)     // primitive pairs of one shell pair the sorter holds

// ------------------------------------------------------------------ small kernels
// (a2) primitive screening estimate of primitive pair (alpha on A, beta on B) of a shell pair with angular momenta
// (la, lb): the primitive Schwarz factor sqrt|(ij|ij)|.  For s functions it is exact,
//   sqrt( 2 pi^(5/2) / (zeta^2 sqrt(2 zeta)) ) |d_a d_b| exp(-alpha beta |AB|^2 / zeta);
// for l > 0 every Cartesian factor (x - A_x) is bounded on the support of the product Gaussian by
// |P - A| + 1/sqrt(zeta) (distance of the product centre plus its width).  DESIGN.md reading R-11.
__device__ __forceinline__ double prim_pair_estimate(double a, double b, double da, double db, double AB2, int la, int lb)
{
    const double z = a + b, iz = 1.0 / z;
    const double w = sqrt(iz);
    const double rAB = sqrt(AB2);
    const double pa = b * iz * rAB + w, pb = a * iz * rAB + w;       // |P-A| + width, |P-B| + width
    double f = fabs(da * db) * exp(-a * b * iz * AB2) * sqrt(34.986836655249725 * iz * iz * sqrt(0.5 * iz));  // 2 pi^2.5
    for (int i = 0; i < la; ++i) f *= pa;
    for (int i = 0; i < lb; ++i) f *= pb;
    return f;
}

// Which primitive pairs of shell pair (sa, sb) survive the primitive screen: bit ia*npb+ib of `keep` (ADFT_MAX_PRIM_PAIRS
// bits) is set iff the estimate reaches thr; if none does, the largest one is kept.  Returns the number of set bits.
// The count pass and the write pass of pair_prim_kernel both call THIS function (never inlined), so the two passes
// cannot disagree on a borderline pair.
__device__ __noinline__ int prim_keep_mask(int npa, int npb, const double *__restrict__ ea, const double *__restrict__ eb,
                                           const double *__restrict__ ca, const double *__restrict__ cb, double AB2, int la,
                                           int lb, double thr, uint32_t *keep)
{
    for (int w = 0; w < ADFT_MAX_PRIM_PAIRS / 32; ++w) keep[w] = 0u;
    int cnt = 0, best = 0;
    double best_est = -1.0;
    for (int ia = 0; ia < npa; ++ia)
        for (int ib = 0; ib < npb; ++ib) {
            const int idx = ia * npb + ib;
            const double est = prim_pair_estimate(ea[ia], eb[ib], ca[ia], cb[ib], AB2, la, lb);
            if (est >= thr) { keep[idx >> 5] |= 1u << (idx & 31); ++cnt; }
            if (est > best_est) { best_est = est; best = idx; }
        }
    if (cnt == 0) { keep[best >> 5] |= 1u << (best & 31); cnt = 1; }
    return cnt;
}

// (a2) primitive-pair records of one sublist.  Two modes:
//   kcount != NULL : write, per pair, the number of primitive pairs that survive the primitive screen to kcount[g];
//   kcount == NULL : write the records of the surviving primitive pairs to slots k = 0..K-1 of the sublist (all its pairs
//                    have K survivors; a pair whose count differs from K raises *err and writes nothing).
// The survivors are stored in DESCENDING order of zeta = alpha + beta (ties: nominal order ia major, ib minor).  All
// lanes of a warp walk primitive lists of the same length; with the lists ranked by exponent the Boys argument
// T = rho |PQ|^2 of step (kb, kk) is large in most lanes together (tight x tight first) or small together, so the
// T < / >= switch branches of boys_scaled are taken warp-uniformly more often.  The slot of a survivor is its rank
// (the number of survivors that sort before it), so no per-thread sort buffer is needed.
__global__ void pair_prim_kernel(int pair_base, int prim_base, int n, int K, int la, int lb, double thr, int32_t *kcount,
                                 int32_t *err, const int32_t *__restrict__ sha,
                                 const int32_t *__restrict__ shb, const int32_t *__restrict__ sh_atom,
                                 const int32_t *__restrict__ sh_nprim, const int32_t *__restrict__ sh_off,
                                 const double *__restrict__ xyz, const double *__restrict__ expo,
                                 const double *__restrict__ coef, double2 *prim, float *primf, size_t npp)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= n) return;
    const int g = pair_base + j;
    const int sa = sha[g], sb = shb[g];
    const double Ax = xyz[3 * sh_atom[sa]], Ay = xyz[3 * sh_atom[sa] + 1], Az = xyz[3 * sh_atom[sa] + 2];
    const double Bx = xyz[3 * sh_atom[sb]], By = xyz[3 * sh_atom[sb] + 1], Bz = xyz[3 * sh_atom[sb] + 2];
    const double AB2 = (Ax - Bx) * (Ax - Bx) + (Ay - By) * (Ay - By) + (Az - Bz) * (Az - Bz);
    const int npa = sh_nprim[sa], npb = sh_nprim[sb];
    const double *ea = expo + sh_off[sa], *eb = expo + sh_off[sb], *ca = coef + sh_off[sa], *cb = coef + sh_off[sb];
    uint32_t keep[ADFT_MAX_PRIM_PAIRS / 32];
    const int cnt = prim_keep_mask(npa, npb, ea, eb, ca, cb, AB2, la, lb, thr, keep);
    if (kcount) { kcount[g] = cnt; return; }
    if (cnt != K) { atomicExch(err, 1); return; }
    const double c0 = 5.9149671727956128778;     // sqrt(2) * pi^(5/4)
    const int np = npa * npb;
    for (int idx = 0; idx < np; ++idx) {
        if (!(keep[idx >> 5] >> (idx & 31) & 1u)) continue;
        const int ia = idx / npb, ib = idx - ia * npb;
        const double a = ea[ia], b = eb[ib];
        const double z = a + b;
        int k = 0;                               // rank among the survivors: larger zeta first, ties in nominal order
        for (int o = 0; o < np; ++o) {
            if (!(keep[o >> 5] >> (o & 31) & 1u)) continue;
            const double zo = ea[o / npb] + eb[o % npb];
            k += (zo > z || (zo == z && o < idx)) ? 1 : 0;
        }
        const double iz = 1.0 / z;
        const double px = (a * Ax + b * Bx) * iz, py = (a * Ay + b * By) * iz, pz = (a * Az + b * Bz) * iz;
        const int slot = prim_base + k * n + j;
        const double ccv = c0 * ca[ia] * cb[ib] * exp(-a * b * iz * AB2) * iz;
        // chunked record layout of PairTable::prim, one float array per field in primf (adft_device.cuh)
        double2 *r = prim + (size_t)(slot >> 3) * 40 + (slot & 7);
        r[0] = make_double2(z, ccv);
        r[8] = make_double2(px, py);
        r[16] = make_double2(pz, 0.5 * iz);
        r[24] = make_double2(px - Ax, py - Ay);
        r[32] = make_double2(pz - Az, 0.0);
        primf[slot] = (float)z;  primf[npp + slot] = (float)(0.5 * iz);
        primf[2 * npp + slot] = (float)(px - Ax);  primf[3 * npp + slot] = (float)(py - Ay);  primf[4 * npp + slot] = (float)(pz - Az);
        primf[5 * npp + slot] = (float)ccv;
    }
}

// (a3) max|D| with non-finite detection.  out[0] = bit pattern of the max (non-negative doubles order like
// their bit patterns), out[1] = 1 if any element is NaN/Inf.
__global__ void dmax_kernel(const double *__restrict__ D, size_t n, unsigned long long *out)
{
    double m = 0.0;
    int bad = 0;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const double a = fabs(D[i]);
        if (!(a <= DBL_MAX)) bad = 1;
        m = fmax(m, a);
    }
    for (int o = 16; o > 0; o >>= 1) {
        m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
        bad |= __shfl_xor_sync(0xffffffffu, bad, o);
    }
    if ((threadIdx.x & 31) == 0) {
        atomicMax(out, (unsigned long long)__double_as_longlong(m));
        if (bad) atomicOr(out + 1, 1ull);
    }
}

// (f3) |D|_XY = max over the shell block (X, Y) of max(|D_ij|, |D_ji|): the table of the block-density screen (R-23).
// One thread per shell pair X >= Y (blocks hold at most 10 x 10 elements).
__global__ void dshell_kernel(const double *__restrict__ D, int N, const int32_t *__restrict__ bfoff, int ns, double *__restrict__ Dsh)
{
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (long long)ns * ns) return;
    const int X = (int)(idx / ns), Y = (int)(idx - (long long)X * ns);
    if (Y > X) return;
    double m = 0.0;
    for (int i = bfoff[X]; i < bfoff[X + 1]; ++i)
        for (int j = bfoff[Y]; j < bfoff[Y + 1]; ++j)
            m = fmax(m, fmax(fabs(__ldg(D + (size_t)i * N + j)), fabs(__ldg(D + (size_t)j * N + i))));
    Dsh[(size_t)X * ns + Y] = Dsh[(size_t)Y * ns + X] = m;
}

// (f3) incremental build: out = a - b;  and  J += Js, K += Ks, Dprev = D
__global__ void diff_kernel(const double *__restrict__ a, const double *__restrict__ b, double *__restrict__ out, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) out[i] = a[i] - b[i];
}
__global__ void incr_finish_kernel(double *J, const double *__restrict__ Js, double *K, const double *__restrict__ Ks,
                                   double *Dprev, const double *__restrict__ D, size_t n)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        if (J) J[i] += Js[i];
        if (K) K[i] += Ks[i];
        Dprev[i] = D[i];
    }
}

// (a6) M <- M + M^T in place (M holds the one-sided accumulations of the digestion).
__global__ void symmetrize_kernel(double *M, int N)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y * blockDim.y + threadIdx.y;
    if (i >= N || j >= N || j > i) return;
    const double a = M[(size_t)i * N + j], b = M[(size_t)j * N + i];
    const double s = a + b;
    M[(size_t)i * N + j] = s;
    M[(size_t)j * N + i] = s;
}

// FP64 peak microbenchmark: 8 independent register-resident FMA chains per thread.
__global__ void fp64_peak_kernel(double *out, int iters, double seed)
{
    double a0 = seed, a1 = seed + 1, a2 = seed + 2, a3 = seed + 3, a4 = seed + 4, a5 = seed + 5, a6 = seed + 6, a7 = seed + 7;
    const double m = 0.999999, c = 1e-9;
    for (int i = 0; i < iters; ++i) {
        a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
        a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
    }
    const double s = a0 + a1 + a2 + a3 + a4 + a5 + a6 + a7;
    if (s == 1234.5678) out[0] = s;      // never true; keeps the chains alive
}

}  // namespace adft

using namespace adft;

// ------------------------------------------------------------------ handles
struct adft_basis {
    int natoms = 0, nshells = 0, nbf = 0, nprim = 0;
    std::vector<double> xyz, expo, coef;
    std::vector<int32_t> atom, l, nprimv, off, bf_off;
};

struct Sublist {
    int pc, la, lb, K, n, pair_base, prim_base;
};

struct adft_shellpairs {
    const adft_basis *basis = nullptr;
    int64_t npairs = 0, nprimpairs = 0, nprimpairs_nominal = 0;
    int sm_count = 148;                // of the device the table lives on
    double prim_threshold = 0.0;
    std::vector<Sublist> subl;
    std::vector<int> subl_of_class[NPAIRCLASS];
    std::vector<double> hQ;            // sorted order
    std::vector<double> Qmat;          // [nshells*nshells]
    // device: basis
    double *d_xyz = nullptr, *d_expo = nullptr, *d_coef = nullptr;
    int32_t *d_atom = nullptr, *d_nprim = nullptr, *d_off = nullptr;
    // device: pair table
    double *d_Q = nullptr, *d_AB = nullptr /* 3*npairs */, *d_prim = nullptr /* chunked records: 80 doubles per 8 slots */;
    float *d_primf = nullptr;                 // single-precision copies, one array per field: 6*nprimpairs floats
    float *d_boysf = nullptr;                 // the per-order Boys tables rounded to float (fp32 launches)
    int32_t *d_pint = nullptr /* 5*npairs: bfa,bfb,sha,shb,knom */;
    double *d_boysp = nullptr;                // per-order Taylor tables [BOYS_MORD][BOYS_NT][BOYS_NC] (generated kernels)
    PairTable tab{};
    // per-build workspaces
    Segment *d_segs = nullptr, *h_segs = nullptr;
    size_t segs_cap = 0;
    int32_t *d_coarse = nullptr, *h_coarse = nullptr;      // JKParams::coarse of every launch of a build, back to back
    size_t coarse_cap = 0;
    unsigned long long *d_counters = nullptr, *d_dmax = nullptr, *h_small = nullptr;
    int32_t *d_prim_err = nullptr;     // raised by pair_prim_kernel when a pair's survivor count is not its sublist's K
    cudaEvent_t ev[4 * NQCLASS + 8] = {};      // [0,2N) fp64 class launches, [2N,2N+8) phases, [2N+8,4N+8) fp32 class launches
    bool ev_ok = false;
    // last build
    adft_jk_stats_t stats{};
    bool class_ran[NQCLASS] = {}, class_ran32[NQCLASS] = {};
    bool have_build = false;
    cudaStream_t last_stream = nullptr;
    // staging for adft_jk_build_host
    double *d_stage = nullptr;
    size_t stage_n = 0;
    double *d_rys = nullptr;                  // device copy of the Rys tables
    RysTable rys{};
    int32_t *d_bfoff = nullptr;               // [nshells+1] first basis function of every shell
    double *d_dsh = nullptr;                  // [nshells*nshells] |D|_XY of the block-density screen (R-23)
    double *d_incr = nullptr;                 // 3 N^2 scratch of adft_jk_build_incremental: dD, J(dD), K(dD)
    // Cartesian -> spherical output transform (adft_sph.cuh), built on first use
    SphTables *d_sph = nullptr;
    int32_t *d_sph_map = nullptr;             // [2*nsph + nshells]: shell of spherical function i, m + l of it, l of every shell
    int nsph = 0;
};

// ------------------------------------------------------------------ misc API
extern "C" const char *adft_status_string(adft_status_t s)
{
    switch (s) {
        case ADFT_OK: return "ok";
        case ADFT_ERR_INVALID_ARG: return "invalid argument";
        case ADFT_ERR_UNSUPPORTED_L: return "unsupported angular momentum";
        case ADFT_ERR_ALLOC: return "allocation failed";
        case ADFT_ERR_CUDA: return "CUDA error";
        case ADFT_ERR_NOT_FINITE: return "density matrix is not finite";
        case ADFT_ERR_INTERNAL: return "internal error";
    }
    return "unknown status";
}
extern "C" const char *adft_last_error(void) { return g_last_error.c_str(); }

// ------------------------------------------------------------------ (a1) basis
extern "C" adft_status_t adft_basis_create(int32_t natoms, const double *xyz, int32_t nshells, const adft_shell_t *shells,
                                           const double *exponents, const double *coefficients, uint32_t flags,
                                           adft_basis_t **out)
{
    if (!xyz || !shells || !exponents || !coefficients || !out || natoms <= 0 || nshells <= 0) {
        set_error("adft_basis_create: NULL pointer or non-positive size");
        return ADFT_ERR_INVALID_ARG;
    }
    if (flags & ~1u) { set_error("adft_basis_create: unknown flags"); return ADFT_ERR_INVALID_ARG; }
    for (int i = 0; i < 3 * natoms; ++i)
        if (!std::isfinite(xyz[i])) { set_error("adft_basis_create: non-finite coordinate"); return ADFT_ERR_INVALID_ARG; }
    adft_basis *b = new (std::nothrow) adft_basis;
    if (!b) return ADFT_ERR_ALLOC;
    b->natoms = natoms; b->nshells = nshells;
    b->xyz.assign(xyz, xyz + 3 * natoms);
    b->bf_off.push_back(0);
    for (int s = 0; s < nshells; ++s) {
        const adft_shell_t &sh = shells[s];
        if (sh.l < 0 || sh.l > 4) {
            set_error("adft_basis_create: shell " + std::to_string(s) + " has l=" + std::to_string(sh.l) + " (supported 0..4)");
            delete b; return ADFT_ERR_UNSUPPORTED_L;
        }
        if (sh.atom < 0 || sh.atom >= natoms || sh.nprim < 1 || sh.nprim > ADFT_MAX_NPRIM || sh.prim_offset < 0) {
            set_error("adft_basis_create: shell " + std::to_string(s) + " has a bad atom index, nprim or offset");
            delete b; return ADFT_ERR_INVALID_ARG;
        }
        b->atom.push_back(sh.atom); b->l.push_back(sh.l); b->nprimv.push_back(sh.nprim);
        b->off.push_back((int32_t)b->expo.size());
        for (int k = 0; k < sh.nprim; ++k) {
            const double a = exponents[sh.prim_offset + k], c = coefficients[sh.prim_offset + k];
            if (!(a > 0.0) || !std::isfinite(a) || !std::isfinite(c)) {
                set_error("adft_basis_create: non-positive or non-finite exponent / coefficient in shell " + std::to_string(s));
                delete b; return ADFT_ERR_INVALID_ARG;
            }
            b->expo.push_back(a); b->coef.push_back(c);
        }
        b->bf_off.push_back(b->bf_off.back() + ncart(sh.l));
    }
    b->nbf = b->bf_off.back();
    b->nprim = (int)b->expo.size();
    if (flags & ADFT_NORMALIZE_SHELLS) {
        // DESIGN R-1: d_k = c_k N_k / sqrt(S); N_k norm of the (L,0,0) primitive, S contracted self-overlap of (L,0,0)
        const double pi = 3.14159265358979323846;
        for (int s = 0; s < nshells; ++s) {
            const int L = b->l[s], o = b->off[s], n = b->nprimv[s];
            double df = 1.0;
            for (int k = 2 * L - 1; k > 1; k -= 2) df *= k;
            for (int k = 0; k < n; ++k) {
                const double a = b->expo[o + k];
                b->coef[o + k] *= std::pow(2.0 * a / pi, 0.75) * std::pow(4.0 * a, 0.5 * L) / std::sqrt(df);
            }
            double S = 0.0;
            for (int i = 0; i < n; ++i)
                for (int j = 0; j < n; ++j) {
                    const double p = b->expo[o + i] + b->expo[o + j];
                    S += b->coef[o + i] * b->coef[o + j] * std::pow(pi / p, 1.5) * df / std::pow(2.0 * p, (double)L);
                }
            if (!(S > 0.0)) { set_error("adft_basis_create: shell with zero norm"); delete b; return ADFT_ERR_INVALID_ARG; }
            const double r = 1.0 / std::sqrt(S);
            for (int k = 0; k < n; ++k) b->coef[o + k] *= r;
        }
    }
    *out = b;
    return ADFT_OK;
}

extern "C" adft_status_t adft_basis_nbf(const adft_basis_t *b, int32_t *nbf)
{
    if (!b || !nbf) { set_error("adft_basis_nbf: NULL"); return ADFT_ERR_INVALID_ARG; }
    *nbf = b->nbf;
    return ADFT_OK;
}
extern "C" adft_status_t adft_basis_shell_offsets(const adft_basis_t *b, int32_t *bf_offset)
{
    if (!b || !bf_offset) { set_error("adft_basis_shell_offsets: NULL"); return ADFT_ERR_INVALID_ARG; }
    std::copy(b->bf_off.begin(), b->bf_off.end(), bf_offset);
    return ADFT_OK;
}
extern "C" adft_status_t adft_basis_coefficients(const adft_basis_t *b, double *c)
{
    if (!b || !c) { set_error("adft_basis_coefficients: NULL"); return ADFT_ERR_INVALID_ARG; }
    std::copy(b->coef.begin(), b->coef.end(), c);
    return ADFT_OK;
}
extern "C" void adft_basis_destroy(adft_basis_t *b) { delete b; }

// ------------------------------------------------------------------ Boys table (library's own; long double series)
static void fill_boys_table(std::vector<double> &tab)
{
    tab.assign((size_t)BOYS_NT * BOYS_NM, 0.0);
    for (int k = 0; k < BOYS_NT; ++k) {
        const long double T = (long double)k / 8.0L;
        const long double eT = expl(-T);
        for (int m = 0; m < BOYS_NM; ++m) {
            // F_m(T) = exp(-T) sum_i (2T)^i / ((2m+1)(2m+3)...(2m+2i+1))
            long double term = 1.0L / (2 * m + 1), sum = term;
            for (int i = 1; i < 4000; ++i) {
                term *= 2.0L * T / (2 * m + 2 * i + 1);
                sum += term;
                if (term < sum * 1e-21L) break;
            }
            tab[(size_t)k * BOYS_NM + m] = (double)(eT * sum);
        }
    }
}

// ------------------------------------------------------------------ (a2) shell pairs
static void free_pairs(adft_shellpairs *p)
{
    if (!p) return;
    cudaFree(p->d_xyz); cudaFree(p->d_expo); cudaFree(p->d_coef); cudaFree(p->d_atom); cudaFree(p->d_nprim);
    cudaFree(p->d_off); cudaFree(p->d_Q); cudaFree(p->d_AB); cudaFree(p->d_prim); cudaFree(p->d_pint);
    cudaFree(p->d_boysp); cudaFree(p->d_segs); cudaFree(p->d_counters); cudaFree(p->d_dmax); cudaFree(p->d_stage);
    cudaFree(p->d_rys); cudaFree(p->d_prim_err); cudaFree(p->d_bfoff); cudaFree(p->d_dsh); cudaFree(p->d_incr);
    cudaFree(p->d_primf); cudaFree(p->d_boysf); cudaFree(p->d_sph); cudaFree(p->d_sph_map);
    if (p->h_segs) cudaFreeHost(p->h_segs);
    cudaFree(p->d_coarse); if (p->h_coarse) cudaFreeHost(p->h_coarse);
    if (p->h_small) cudaFreeHost(p->h_small);
    if (p->ev_ok) for (auto &e : p->ev) cudaEventDestroy(e);
    delete p;
}
extern "C" void adft_shellpairs_destroy(adft_shellpairs_t *p) { free_pairs(p); }

struct HostPair { int sa, sb; double Q; int knom; };

static void set_table_pointers(adft_shellpairs *p)
{
    const size_t np = (size_t)p->npairs;
    PairTable &t = p->tab;
    t.Q = p->d_Q;
    t.ABx = p->d_AB; t.ABy = p->d_AB + np; t.ABz = p->d_AB + 2 * np;
    t.bfa = p->d_pint; t.bfb = p->d_pint + np; t.sha = p->d_pint + 2 * np; t.shb = p->d_pint + 3 * np;
    t.knom = p->d_pint + 4 * np;
    t.prim = reinterpret_cast<const double2 *>(p->d_prim);
    t.primf = p->d_primf;
    t.primf_stride = (size_t)p->nprimpairs;
}

static adft_status_t upload_pairs_and_prims(adft_shellpairs *p, const std::vector<HostPair> &hp, double thr, cudaStream_t st)
{
    const adft_basis *b = p->basis;
    const size_t np = hp.size();
    std::vector<double> AB(3 * np);
    std::vector<int32_t> pint(5 * np);
    for (size_t g = 0; g < np; ++g) {
        const int sa = hp[g].sa, sb = hp[g].sb;
        for (int i = 0; i < 3; ++i) AB[i * np + g] = b->xyz[3 * b->atom[sa] + i] - b->xyz[3 * b->atom[sb] + i];
        pint[g] = b->bf_off[sa]; pint[np + g] = b->bf_off[sb]; pint[2 * np + g] = sa; pint[3 * np + g] = sb;
        pint[4 * np + g] = hp[g].knom;
    }
    CUDA_TRY(cudaMemcpyAsync(p->d_AB, AB.data(), AB.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemcpyAsync(p->d_pint, pint.data(), pint.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    CUDA_TRY(cudaMemsetAsync(p->d_prim_err, 0, sizeof(int32_t), st));
    CUDA_TRY(cudaStreamSynchronize(st));     // host vectors go out of scope
    for (const Sublist &s : p->subl) {
        if (s.n == 0) continue;
        pair_prim_kernel<<<(s.n + 127) / 128, 128, 0, st>>>(s.pair_base, s.prim_base, s.n, s.K, s.la, s.lb, thr, nullptr,
                                                             p->d_prim_err, p->tab.sha, p->tab.shb, p->d_atom,
                                                             p->d_nprim, p->d_off, p->d_xyz, p->d_expo, p->d_coef,
                                                             reinterpret_cast<double2 *>(p->d_prim), p->d_primf, (size_t)p->nprimpairs);
    }
    CUDA_TRY(cudaGetLastError());
    int32_t bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, p->d_prim_err, sizeof(int32_t), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (bad) { set_error("adft_shellpairs_build: primitive-pair count of a pair differs from its sublist's depth"); return ADFT_ERR_INTERNAL; }
    return ADFT_OK;
}

// Group (key, pair) records into sublists (same pair class and contraction depth): fills p->subl, p->subl_of_class,
// hp (pairs in sublist order) and returns the number of primitive-pair records.
struct BucketKey { int pc, K; bool operator<(const BucketKey &o) const { return pc != o.pc ? pc < o.pc : K < o.K; } };
static int64_t make_sublists(adft_shellpairs *p, std::vector<std::pair<BucketKey, HostPair>> &all, std::vector<HostPair> &hp)
{
    const adft_basis *b = p->basis;
    std::stable_sort(all.begin(), all.end(), [](const auto &x, const auto &y) { return x.first < y.first; });
    hp.resize(all.size());
    p->subl.clear();
    for (auto &v : p->subl_of_class) v.clear();
    int64_t prim_total = 0;
    for (size_t g = 0; g < all.size();) {
        size_t e = g;
        while (e < all.size() && !(all[g].first < all[e].first)) ++e;
        Sublist s;
        s.pc = all[g].first.pc; s.K = all[g].first.K; s.n = (int)(e - g);
        s.la = b->l[all[g].second.sa]; s.lb = b->l[all[g].second.sb];
        s.pair_base = (int)g; s.prim_base = (int)prim_total;
        prim_total += (int64_t)s.K * s.n;
        p->subl_of_class[s.pc].push_back((int)p->subl.size());
        p->subl.push_back(s);
        for (size_t q = g; q < e; ++q) hp[q] = all[q].second;
        g = e;
    }
    return prim_total;
}

extern "C" adft_status_t adft_shellpairs_build(const adft_basis_t *b, void *cuda_stream, adft_shellpairs_t **out)
{
    return adft_shellpairs_build_ex(b, ADFT_DEFAULT_PRIM_THRESHOLD, cuda_stream, out);
}

extern "C" adft_status_t adft_shellpairs_build_ex(const adft_basis_t *b, double prim_threshold, void *cuda_stream,
                                                  adft_shellpairs_t **out)
{
    if (!b || !out) { set_error("adft_shellpairs_build: NULL"); return ADFT_ERR_INVALID_ARG; }
    if (!(prim_threshold >= 0.0) || !std::isfinite(prim_threshold)) {
        set_error("adft_shellpairs_build_ex: prim_threshold must be finite and >= 0");
        return ADFT_ERR_INVALID_ARG;
    }
    ensure_registered();
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        set_error("adft_shellpairs_build: no CUDA device (there is no CPU fallback)");
        return ADFT_ERR_CUDA;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    adft_shellpairs *p = new (std::nothrow) adft_shellpairs;
    if (!p) return ADFT_ERR_ALLOC;
    p->basis = b;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
            p->sm_count = sms;
    }
    const int ns = b->nshells;

    p->prim_threshold = prim_threshold;
    // bucket pairs (A >= B) by pair class and contraction depth; a = the higher-l shell
    std::vector<std::pair<BucketKey, HostPair>> all;
    all.reserve((size_t)ns * (ns + 1) / 2);
    for (int A = 0; A < ns; ++A)
        for (int B = 0; B <= A; ++B) {
            // orientation of the pair: a = the shell the vertical recurrences build on, b receives angular momentum
            // through the horizontal recurrence (a,b+1_i| = (a+1_i,b| + (A_i-B_i)(ab|.  The class needs la >= lb; for
            // equal l the choice is free and a = the TIGHTER shell (larger smallest exponent): the dominant Gaussian
            // product centres P then lie next to A, |P-A| stays small and the HRR does not cancel (measured on cfg 1
            // shells (23,32): Q relative error 4e-7 with a = the diffuse shell).
            int sa = A, sb = B;
            if (b->l[sa] < b->l[sb]) std::swap(sa, sb);
            else if (b->l[sa] == b->l[sb] && sa != sb) {
                auto min_exp = [&](int s) {
                    double m = b->expo[b->off[s]];
                    for (int k = 1; k < b->nprimv[s]; ++k) m = std::min(m, b->expo[b->off[s] + k]);
                    return m;
                };
                if (min_exp(sb) > min_exp(sa)) std::swap(sa, sb);
            }
            const int knom = b->nprimv[sa] * b->nprimv[sb];
            all.push_back({BucketKey{pair_class(b->l[sa], b->l[sb]), knom}, HostPair{sa, sb, 0.0, knom}});
        }
    std::vector<HostPair> hp;
    p->npairs = (int64_t)all.size();
    const int64_t prim_total = make_sublists(p, all, hp);
    if (prim_total > 0x7fffffffLL) { set_error("adft_shellpairs_build: too many primitive pairs"); free_pairs(p); return ADFT_ERR_ALLOC; }
    p->nprimpairs = p->nprimpairs_nominal = prim_total;
    // every needed Schwarz class must exist
    for (const Sublist &s : p->subl) {
        if (!rys_schwarz_launcher(s.la, s.lb)) {
            set_error("adft_shellpairs_build: no kernel for pair class (" + std::to_string(s.la) + "," + std::to_string(s.lb) + ")");
            free_pairs(p); return ADFT_ERR_UNSUPPORTED_L;
        }
    }

    const size_t np = (size_t)p->npairs, npp = (size_t)p->nprimpairs;
#define ALLOC(ptr, bytes)                                                                                   \
    if (cudaMalloc((void **)&(ptr), (bytes)) != cudaSuccess) {                                              \
        set_error("adft_shellpairs_build: cudaMalloc of " + std::to_string((size_t)(bytes)) + " bytes failed"); \
        cudaGetLastError(); free_pairs(p); return ADFT_ERR_ALLOC;                                           \
    }
    ALLOC(p->d_xyz, b->xyz.size() * sizeof(double));
    ALLOC(p->d_expo, b->expo.size() * sizeof(double));
    ALLOC(p->d_coef, b->coef.size() * sizeof(double));
    ALLOC(p->d_atom, ns * sizeof(int32_t));
    ALLOC(p->d_nprim, ns * sizeof(int32_t));
    ALLOC(p->d_off, ns * sizeof(int32_t));
    ALLOC(p->d_Q, np * sizeof(double));
    ALLOC(p->d_AB, 3 * np * sizeof(double));
    ALLOC(p->d_pint, 5 * np * sizeof(int32_t));
    ALLOC(p->d_prim, prim_chunks(npp) * 80 * sizeof(double));
    ALLOC(p->d_primf, 6 * npp * sizeof(float));
    ALLOC(p->d_boysf, (size_t)BOYS_MORD * BOYS_NT * BOYS_NC * sizeof(float));
    ALLOC(p->d_boysp, (size_t)BOYS_MORD * BOYS_NT * BOYS_NC * sizeof(double));
    ALLOC(p->d_counters, 8 * NQCLASS * sizeof(unsigned long long));     // [0,4N) all launches' fp64 part, [4N,8N) fp32 launches
    ALLOC(p->d_dmax, 2 * sizeof(unsigned long long));
    ALLOC(p->d_prim_err, sizeof(int32_t));
    ALLOC(p->d_rys, (size_t)(adft_rys_blob_end - adft_rys_blob) * sizeof(double));
    ALLOC(p->d_bfoff, (ns + 1) * sizeof(int32_t));
    ALLOC(p->d_dsh, (size_t)ns * ns * sizeof(double));
#undef ALLOC
    {
        // Rys tables (gen_rys.py layout): header[8] = magic, NMAX, TMAX, H, NCOEF
        const double *h = adft_rys_blob;
        const int nmax = (int)h[1], ncoef = (int)h[4];
        const int nint = (int)std::lround(h[2] / h[3]);
        if (h[0] != 5259531.0 || nmax != RYS_NMAX) { set_error("adft_shellpairs_build: bad Rys table blob"); free_pairs(p); return ADFT_ERR_INTERNAL; }
        p->rys.tab = p->d_rys; p->rys.nint = nint; p->rys.ncoef = ncoef; p->rys.tmax = h[2]; p->rys.inv_h = 1.0 / h[3];
        int off = 8;
        for (int n = 1; n <= RYS_NMAX; ++n) { p->rys.off_cheb[n] = off; off += nint * 2 * n * ncoef; }
        for (int n = 1; n <= RYS_NMAX; ++n) { p->rys.off_asym[n] = off; off += 2 * n; }
        if (off != (int)(adft_rys_blob_end - adft_rys_blob)) { set_error("adft_shellpairs_build: Rys table size mismatch"); free_pairs(p); return ADFT_ERR_INTERNAL; }
    }
    if (cudaMallocHost((void **)&p->h_small, 8 * NQCLASS * sizeof(unsigned long long)) != cudaSuccess) {
        set_error("adft_shellpairs_build: cudaMallocHost failed"); free_pairs(p); return ADFT_ERR_ALLOC;
    }
    for (auto &e : p->ev)
        if (cudaEventCreate(&e) != cudaSuccess) { set_error("cudaEventCreate failed"); free_pairs(p); return ADFT_ERR_CUDA; }
    p->ev_ok = true;
    set_table_pointers(p);

    adft_status_t rc = ADFT_OK;
    auto fail = [&](adft_status_t r) { free_pairs(p); return r; };
#define TRY2(expr)                                                                         \
    do {                                                                                   \
        cudaError_t e__ = (expr);                                                          \
        if (e__ != cudaSuccess) {                                                          \
            set_error(std::string(#expr) + ": " + cudaGetErrorString(e__));                \
            return fail(ADFT_ERR_CUDA);                                                    \
        }                                                                                  \
    } while (0)
    TRY2(cudaMemcpyAsync(p->d_xyz, b->xyz.data(), b->xyz.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_expo, b->expo.data(), b->expo.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_coef, b->coef.data(), b->coef.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_atom, b->atom.data(), ns * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_nprim, b->nprimv.data(), ns * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_off, b->off.data(), ns * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_bfoff, b->bf_off.data(), (ns + 1) * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    TRY2(cudaMemcpyAsync(p->d_rys, adft_rys_blob, (size_t)(adft_rys_blob_end - adft_rys_blob) * sizeof(double),
                         cudaMemcpyHostToDevice, st));
    std::vector<double> boys;
    fill_boys_table(boys);
    // per-order tables: a_j = F_{M+j}(T_k) / j!, j = 0..9  (Taylor coefficients of F_M about T_k in d = T_k - T)
    std::vector<double> boysp((size_t)BOYS_MORD * BOYS_NT * BOYS_NC);
    for (int M = 0; M < BOYS_MORD; ++M)
        for (int k = 0; k < BOYS_NT; ++k) {
            long double fact = 1.0L;
            for (int j = 0; j < BOYS_NC; ++j) {
                if (j > 0) fact *= (long double)j;
                boysp[((size_t)M * BOYS_NT + k) * BOYS_NC + j] = (double)((long double)boys[(size_t)k * BOYS_NM + M + j] / fact);
            }
        }
    TRY2(cudaMemcpyAsync(p->d_boysp, boysp.data(), boysp.size() * sizeof(double), cudaMemcpyHostToDevice, st));
    std::vector<float> boysf(boysp.begin(), boysp.end());
    TRY2(cudaMemcpyAsync(p->d_boysf, boysf.data(), boysf.size() * sizeof(float), cudaMemcpyHostToDevice, st));
    TRY2(cudaStreamSynchronize(st));

    // pass 1: records of ALL primitive pairs in bucket order, Schwarz bounds from the full contraction
    rc = upload_pairs_and_prims(p, hp, 0.0, st);
    if (rc) return fail(rc);
    for (const Sublist &s : p->subl) {
        if (s.n == 0) continue;
        TRY2(rys_schwarz_launcher(s.la, s.lb)(p->tab, p->rys, s.pair_base, s.prim_base, s.n, s.K, p->d_Q, st));
    }
    TRY2(cudaGetLastError());
    std::vector<double> Q(np);
    TRY2(cudaMemcpyAsync(Q.data(), p->d_Q, np * sizeof(double), cudaMemcpyDeviceToHost, st));
    TRY2(cudaStreamSynchronize(st));
    for (size_t g = 0; g < np; ++g) {
        if (!std::isfinite(Q[g])) { set_error("adft_shellpairs_build: non-finite Schwarz bound"); return fail(ADFT_ERR_INTERNAL); }
        hp[g].Q = Q[g];
    }
    // primitive screening (DESIGN R-11): number of primitive pairs of every pair whose estimate reaches the threshold
    {
        int32_t *d_kcount = p->d_pint + 4 * np;          // the knom slot is rewritten in pass 2
        for (const Sublist &s : p->subl) {
            if (s.n == 0) continue;
            pair_prim_kernel<<<(s.n + 127) / 128, 128, 0, st>>>(s.pair_base, s.prim_base, s.n, s.K, s.la, s.lb, prim_threshold,
                                                                 d_kcount, p->d_prim_err, p->tab.sha, p->tab.shb, p->d_atom, p->d_nprim,
                                                                 p->d_off, p->d_xyz, p->d_expo, p->d_coef, nullptr, nullptr, 0);
        }
        TRY2(cudaGetLastError());
        std::vector<int32_t> kc(np);
        TRY2(cudaMemcpyAsync(kc.data(), d_kcount, np * sizeof(int32_t), cudaMemcpyDeviceToHost, st));
        TRY2(cudaStreamSynchronize(st));
        // pass 2: re-bucket by (pair class, surviving depth), sort every sublist by Q descending (ties: by shell
        // indices, for determinism) and rebuild the records
        for (size_t g = 0; g < np; ++g) {
            if (kc[g] < 1 || kc[g] > hp[g].knom) { set_error("adft_shellpairs_build: bad primitive count"); return fail(ADFT_ERR_INTERNAL); }
            all[g] = {BucketKey{pair_class(b->l[hp[g].sa], b->l[hp[g].sb]), kc[g]}, hp[g]};
        }
        p->nprimpairs = make_sublists(p, all, hp);
        if (p->nprimpairs < p->nprimpairs_nominal) {      // compact table: release the records of the dropped primitives
            TRY2(cudaFree(p->d_prim));
            p->d_prim = nullptr;
            TRY2(cudaMalloc((void **)&p->d_prim, prim_chunks((size_t)p->nprimpairs) * 80 * sizeof(double)));
            TRY2(cudaFree(p->d_primf));
            p->d_primf = nullptr;
            TRY2(cudaMalloc((void **)&p->d_primf, 6 * (size_t)p->nprimpairs * sizeof(float)));
        }
        set_table_pointers(p);
    }
    for (const Sublist &s : p->subl)
        std::sort(hp.begin() + s.pair_base, hp.begin() + s.pair_base + s.n, [](const HostPair &x, const HostPair &y) {
            if (x.Q != y.Q) return x.Q > y.Q;
            if (x.sa != y.sa) return x.sa < y.sa;
            return x.sb < y.sb;
        });
    p->hQ.resize(np);
    p->Qmat.assign((size_t)ns * ns, 0.0);
    for (size_t g = 0; g < np; ++g) {
        p->hQ[g] = hp[g].Q;
        p->Qmat[(size_t)hp[g].sa * ns + hp[g].sb] = p->Qmat[(size_t)hp[g].sb * ns + hp[g].sa] = hp[g].Q;
    }
    TRY2(cudaMemcpyAsync(p->d_Q, p->hQ.data(), np * sizeof(double), cudaMemcpyHostToDevice, st));
    rc = upload_pairs_and_prims(p, hp, prim_threshold, st);
    if (rc) return fail(rc);
    TRY2(cudaStreamSynchronize(st));
#undef TRY2
    *out = p;
    return ADFT_OK;
}

extern "C" adft_status_t adft_shellpairs_schwarz(const adft_shellpairs_t *p, double *Q)
{
    if (!p || !Q) { set_error("adft_shellpairs_schwarz: NULL"); return ADFT_ERR_INVALID_ARG; }
    std::copy(p->Qmat.begin(), p->Qmat.end(), Q);
    return ADFT_OK;
}
extern "C" adft_status_t adft_shellpairs_counts(const adft_shellpairs_t *p, int64_t *npairs, int64_t *nprimpairs)
{
    if (!p) { set_error("adft_shellpairs_counts: NULL"); return ADFT_ERR_INVALID_ARG; }
    if (npairs) *npairs = p->npairs;
    if (nprimpairs) *nprimpairs = p->nprimpairs;
    return ADFT_OK;
}
extern "C" adft_status_t adft_shellpairs_prim_counts(const adft_shellpairs_t *p, int64_t *nominal, int64_t *kept, double *threshold)
{
    if (!p) { set_error("adft_shellpairs_prim_counts: NULL"); return ADFT_ERR_INVALID_ARG; }
    if (nominal) *nominal = p->nprimpairs_nominal;
    if (kept) *kept = p->nprimpairs;
    if (threshold) *threshold = p->prim_threshold;
    return ADFT_OK;
}

// ------------------------------------------------------------------ (a3) launch plan (host; Q lists are sorted descending)
// number of leading elements q of a descending list with (qfix*q)*dmax >= tau   (monotone predicate, DESIGN R-7)
static int prefix_len(const double *q, int n, double qfix, double dmax, double tau)
{
    int lo = 0, hi = n;
    while (lo < hi) {
        const int mid = (lo + hi) >> 1;
        if ((qfix * q[mid]) * dmax >= tau) lo = mid + 1; else hi = mid;
    }
    return lo;
}

// tau_skip > 0 (the fp32 launch of the mixed-precision dispatch, global-Dmax rule only): tile columns that lie, for EVERY
// row of the segment, inside the fp64 prefix (S >= tau_skip) are left out of the launch.  The last row has the smallest
// Q_ab and therefore the shortest fp64 prefix; columns below it are fp64 for all rows.
// tile_c = ket pairs per tile row: TILE_C, or 2*TILE_C for the packed single-precision kernel (two quartets per lane).
static long long plan_class(const adft_shellpairs *p, int X, int Y, double dmax, double tau, std::vector<Segment> &segs,
                            double tau_skip = 0.0, int tile_c = TILE_C)
{
    // A (bra sublist, ket sublist) pair keeps the quartets under the staircase Q_ab*Q_cd >= tau/dmax of its rows x columns
    // matrix (both lists descending in Q).  One rectangle around it would launch two empty tiles for every kept one (cfg 4:
    // 31% of the launched warps of (ps|ss) held a quartet, and the prologue of the empty ones was a third of that kernel's
    // instructions), so the rows are cut into bands: a band ends where the row's tile count has fallen to BAND_F of the
    // band's first row, bands are whole tile rows, and a remainder of fewer than BAND_MIN_TILES tiles stays one band.
    constexpr double BAND_F = 0.75;
    constexpr long long BAND_MIN_TILES = 1024;
    segs.clear();
    for (int i1 : p->subl_of_class[X])
        for (int i2 : p->subl_of_class[Y]) {
            if (X == Y && i2 > i1) continue;
            const Sublist &s1 = p->subl[i1], &s2 = p->subl[i2];
            if (s1.n == 0 || s2.n == 0) continue;
            const double *q1 = p->hQ.data() + s1.pair_base, *q2 = p->hQ.data() + s2.pair_base;
            const int rows = prefix_len(q1, s1.n, q2[0], dmax, tau);
            const bool same = (i1 == i2);
            int r0 = 0;
            while (r0 < rows) {
                // kept prefix of the band's first row (the longest of the band); j <= i on the diagonal block
                int cols = prefix_len(q2, s2.n, q1[r0], dmax, tau);
                if (cols == 0) break;                                  // cannot happen for r0 < rows; guards the loop
                const int tiles0 = (std::min(cols, same ? rows : cols) + tile_c - 1) / tile_c;
                int r1 = rows;
                if ((long long)((rows - r0 + TILE_R - 1) / TILE_R) * tiles0 >= BAND_MIN_TILES) {
                    // rows whose prefix still needs at least tmin tiles: q1[r] * q2[(tmin-1)*tile_c] * dmax >= tau
                    const int tmin = std::max(1, (int)std::ceil(BAND_F * tiles0));
                    const int cneed = (tmin - 1) * tile_c;             // index of the first column of tile tmin-1
                    int rb = cneed < s2.n ? prefix_len(q1, rows, q2[cneed], dmax, tau) : r0 + 1;
                    if (same) rb = std::min(rb, std::max(r0 + TILE_R, (int)((r0 + 1) / BAND_F)));   // diagonal: cols <= i + 1
                    rb = r0 + std::max(1, (rb - r0) / TILE_R) * TILE_R;                              // whole tile rows
                    r1 = std::min(rows, rb);
                }
                if (same) cols = std::min(cols, r1);
                Segment sg{};
                sg.bra_pair_base = s1.pair_base; sg.bra_prim_base = s1.prim_base; sg.bra_n = s1.n; sg.bra_K = s1.K;
                sg.ket_pair_base = s2.pair_base; sg.ket_prim_base = s2.prim_base; sg.ket_n = s2.n; sg.ket_K = s2.K;
                sg.row_begin = r0; sg.rows = r1; sg.tiles_per_row = (cols + tile_c - 1) / tile_c; sg.same = same ? 1 : 0;
                if (tau_skip > 0.0) {
                    sg.col_tile_begin = prefix_len(q2, s2.n, q1[r1 - 1], dmax, tau_skip) / tile_c;
                    sg.tiles_per_row -= sg.col_tile_begin;
                }
                if (sg.tiles_per_row > 0) segs.push_back(sg);
                r0 = r1;
            }
        }
    // heaviest tiles first (per-tile cost ~ K1*K2), so the tail of the launch is made of cheap tiles
    std::stable_sort(segs.begin(), segs.end(), [](const Segment &a, const Segment &b) {
        return (long long)a.bra_K * a.ket_K > (long long)b.bra_K * b.ket_K;
    });
    long long w = 0;
    for (Segment &s : segs) { s.warp_begin = w; w += (long long)((s.rows - s.row_begin + TILE_R - 1) / TILE_R) * s.tiles_per_row; }
    return w;
}

// ------------------------------------------------------------------ the J/K build
extern "C" adft_status_t adft_jk_build(adft_shellpairs_t *p, const double *D, double *J, double *K, double tau,
                                       void *cuda_stream)
{
    return adft_jk_build_ex(p, D, J, K, tau, nullptr, cuda_stream);
}

extern "C" adft_status_t adft_jk_build_ex(adft_shellpairs_t *p, const double *D, double *J, double *K, double tau,
                                          const adft_jk_options_t *opt, void *cuda_stream)
{
    if (!p || !D || (!J && !K)) { set_error("adft_jk_build: NULL handle or D, or both J and K NULL"); return ADFT_ERR_INVALID_ARG; }
    const uint32_t flags = opt ? opt->flags : 0u;
    const int shard_count = opt && opt->shard_count > 1 ? opt->shard_count : 1;
    const int shard_rank = opt ? opt->shard_rank : 0;
    if (flags & ~(ADFT_JK_BLOCK_DENSITY | ADFT_JK_MIXED_PRECISION)) { set_error("adft_jk_build_ex: unknown option flags"); return ADFT_ERR_INVALID_ARG; }
    const bool mixed = (flags & ADFT_JK_MIXED_PRECISION) != 0;
    const double band = opt && opt->fp32_band != 0.0 ? opt->fp32_band : ADFT_DEFAULT_FP32_BAND;
    if (mixed && (!J || !K)) { set_error("adft_jk_build_ex: ADFT_JK_MIXED_PRECISION needs both J and K"); return ADFT_ERR_INVALID_ARG; }
    if (mixed && (!(band >= 1.0) || !std::isfinite(band))) { set_error("adft_jk_build_ex: fp32_band must be finite and >= 1"); return ADFT_ERR_INVALID_ARG; }
    const double tau64 = tau * band;          // S >= tau64: double precision; tau <= S < tau64: single precision
    if (opt && (opt->shard_count < 0 || shard_rank < 0 || shard_rank >= shard_count)) {
        set_error("adft_jk_build_ex: shard_rank must lie in [0, shard_count)");
        return ADFT_ERR_INVALID_ARG;
    }
    const bool block_density = (flags & ADFT_JK_BLOCK_DENSITY) != 0;
    if (!(tau >= 0.0) || !std::isfinite(tau)) { set_error("adft_jk_build: schwarz_threshold must be finite and >= 0"); return ADFT_ERR_INVALID_ARG; }
    if (D == J || D == K || J == K) { set_error("adft_jk_build: D, J and K must not alias one another"); return ADFT_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int N = p->basis->nbf;
    const size_t n2 = (size_t)N * N;
    int launches = 0;
    // every class that can occur must have a kernel
    for (int X = 0; X < NPAIRCLASS; ++X)
        for (int Y = 0; Y <= X; ++Y)
            if (!p->subl_of_class[X].empty() && !p->subl_of_class[Y].empty() && !class_table()[quartet_class(X, Y)].launch_jk &&
                !class_table()[quartet_class(X, Y)].use_rys) {
                set_error("adft_jk_build: no kernel compiled for quartet class " + std::to_string(quartet_class(X, Y)));
                return ADFT_ERR_UNSUPPORTED_L;
            }
    cudaEvent_t *ev = p->ev;
    cudaEvent_t ev_begin = ev[2 * NQCLASS], ev_dmax = ev[2 * NQCLASS + 1], ev_plan = ev[2 * NQCLASS + 2],
                ev_eri = ev[2 * NQCLASS + 3], ev_end = ev[2 * NQCLASS + 4];
    CUDA_TRY(cudaEventRecord(ev_begin, st));
    // (a3) Dmax
    CUDA_TRY(cudaMemsetAsync(p->d_dmax, 0, 2 * sizeof(unsigned long long), st));
    dmax_kernel<<<(unsigned)std::min<size_t>((n2 + 255) / 256, (size_t)p->sm_count * 4), 256, 0, st>>>(D, n2, p->d_dmax); ++launches;
    CUDA_TRY(cudaMemcpyAsync(p->h_small, p->d_dmax, 2 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaEventRecord(ev_dmax, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    if (p->h_small[1]) { set_error("adft_jk_build: D contains NaN or Inf"); return ADFT_ERR_NOT_FINITE; }
    double dmax;
    std::memcpy(&dmax, &p->h_small[0], sizeof(double));
    if (block_density) {
        // (f3) shell-block maxima of |D|; the host plan below still bounds the rectangles with the global Dmax (a
        // superset of what the block rule keeps), the exact rule is applied per lane
        const int ns = p->basis->nshells;
        const long long nn = (long long)ns * ns;
        dshell_kernel<<<(unsigned)((nn + 255) / 256), 256, 0, st>>>(D, N, p->d_bfoff, ns, p->d_dsh); ++launches;
        CUDA_TRY(cudaGetLastError());
    }

    // plan: segments of every class
    // (f1, mixed precision) the straight-line classes get two launches: the fp64 kernel over the rectangles of the rule
    // S >= tau64 and the fp32 kernel over those of S >= tau minus the leading all-fp64 columns; each lane applies the exact
    // band test, so every kept quartet is evaluated exactly once.  The Rys classes (f shells) stay fp64 throughout.
    std::vector<std::vector<Segment>> plan(NQCLASS), plan32(NQCLASS);
    long long warps[NQCLASS] = {}, warps32[NQCLASS] = {};
    size_t nseg_total = 0;
    for (int X = 0; X < NPAIRCLASS; ++X)
        for (int Y = 0; Y <= X; ++Y) {
            const int qc = quartet_class(X, Y);
            const bool two = mixed && tau > 0.0 && !class_table()[qc].use_rys;
            warps[qc] = plan_class(p, X, Y, dmax, two ? tau64 : tau, plan[qc]);
            if (two) warps32[qc] = plan_class(p, X, Y, dmax, tau, plan32[qc], block_density ? 0.0 : tau64, 2 * TILE_C);
            nseg_total += plan[qc].size() + plan32[qc].size();
        }
    if (nseg_total > p->segs_cap) {
        cudaFree(p->d_segs); if (p->h_segs) cudaFreeHost(p->h_segs);
        p->d_segs = nullptr; p->h_segs = nullptr; p->segs_cap = 0;
        const size_t cap = nseg_total + nseg_total / 4 + 64;
        CUDA_TRY(cudaMalloc((void **)&p->d_segs, cap * sizeof(Segment)));
        CUDA_TRY(cudaMallocHost((void **)&p->h_segs, cap * sizeof(Segment)));
        p->segs_cap = cap;
    }
    size_t seg_off[NQCLASS] = {}, seg_off32[NQCLASS] = {};
    {
        size_t o = 0;
        for (int qc = 0; qc < NQCLASS; ++qc) {
            seg_off[qc] = o;
            std::copy(plan[qc].begin(), plan[qc].end(), p->h_segs + o);
            o += plan[qc].size();
            seg_off32[qc] = o;
            std::copy(plan32[qc].begin(), plan32[qc].end(), p->h_segs + o);
            o += plan32[qc].size();
        }
        if (o) CUDA_TRY(cudaMemcpyAsync(p->d_segs, p->h_segs, o * sizeof(Segment), cudaMemcpyHostToDevice, st));
    }
    // coarse index of every launch (find_segment): entry k = segment of tile k << COARSE_SHIFT, one entry past the last
    size_t co_off[NQCLASS] = {}, co_off32[NQCLASS] = {};
    {
        auto entries = [](long long w) { return w > 0 ? (size_t)(((w - 1) >> COARSE_SHIFT) + 2) : (size_t)0; };
        size_t total = 0;
        for (int qc = 0; qc < NQCLASS; ++qc) {
            co_off[qc] = total;  total += entries(warps[qc]);
            co_off32[qc] = total;  total += entries(warps32[qc]);
        }
        if (total > p->coarse_cap) {
            cudaFree(p->d_coarse); if (p->h_coarse) cudaFreeHost(p->h_coarse);
            p->d_coarse = nullptr; p->h_coarse = nullptr; p->coarse_cap = 0;
            const size_t cap = total + total / 4 + 64;
            CUDA_TRY(cudaMalloc((void **)&p->d_coarse, cap * sizeof(int32_t)));
            CUDA_TRY(cudaMallocHost((void **)&p->h_coarse, cap * sizeof(int32_t)));
            p->coarse_cap = cap;
        }
        auto fill = [&](const std::vector<Segment> &sg, long long w, int32_t *out) {
            const size_t n = entries(w);
            int sidx = 0;
            const int ns = (int)sg.size();
            for (size_t k = 0; k < n; ++k) {
                const long long t = (long long)k << COARSE_SHIFT;
                while (sidx + 1 < ns && sg[sidx + 1].warp_begin <= t) ++sidx;
                out[k] = sidx;
            }
        };
        for (int qc = 0; qc < NQCLASS; ++qc) {
            fill(plan[qc], warps[qc], p->h_coarse + co_off[qc]);
            fill(plan32[qc], warps32[qc], p->h_coarse + co_off32[qc]);
        }
        if (total) CUDA_TRY(cudaMemcpyAsync(p->d_coarse, p->h_coarse, total * sizeof(int32_t), cudaMemcpyHostToDevice, st));
    }
    CUDA_TRY(cudaMemsetAsync(p->d_counters, 0, 8 * NQCLASS * sizeof(unsigned long long), st));
    if (J) CUDA_TRY(cudaMemsetAsync(J, 0, n2 * sizeof(double), st));
    if (K) CUDA_TRY(cudaMemsetAsync(K, 0, n2 * sizeof(double), st));
    CUDA_TRY(cudaEventRecord(ev_plan, st));

    // (a4)+(a5) one launch per class, heavy classes first
    int order[NQCLASS];
    std::iota(order, order + NQCLASS, 0);
    std::stable_sort(order, order + NQCLASS, [&](int a, int b) { return a > b; });
    for (int qi = 0; qi < NQCLASS; ++qi) {
        const int qc = order[qi];
        p->class_ran[qc] = p->class_ran32[qc] = false;
        if (warps[qc] == 0 && warps32[qc] == 0) continue;
        const ClassEntry &ce = class_table()[qc];
        const bool two = mixed && tau > 0.0 && !ce.use_rys;
        JKParams prm{};
        prm.t = p->tab; prm.segs = p->d_segs + seg_off[qc]; prm.nsegs = (int)plan[qc].size(); prm.total_warps = warps[qc];
        prm.coarse = p->d_coarse + co_off[qc];
        prm.D = D; prm.J = J; prm.K = K; prm.N = N; prm.tau = two ? tau64 : tau; prm.tau_hi = HUGE_VAL; prm.dmax = dmax;
        prm.boys = p->d_boysp; prm.boys_f = p->d_boysf;
        prm.counters = p->d_counters + 4 * qc; prm.zero = 0;
        prm.Dsh = block_density ? p->d_dsh : nullptr; prm.nshells = p->basis->nshells;
        prm.shard_rank = shard_rank; prm.shard_count = shard_count;
        if (warps[qc] > 0) {
            CUDA_TRY(cudaEventRecord(ev[2 * qc], st));
            if (ce.use_rys) {
                CUDA_TRY(rys_jk_launcher(ce.la, ce.lb, ce.lc, ce.ld)(prm, p->rys, p->d_counters + 4 * qc + 3, st, J != nullptr, K != nullptr));
            } else {
                ce.launch_jk(prm, st, J != nullptr, K != nullptr, false);
            }
            ++launches;
            CUDA_TRY(cudaEventRecord(ev[2 * qc + 1], st));
            p->class_ran[qc] = true;
        }
        if (two && warps32[qc] > 0) {
            // the single-precision band tau <= S < tau64 of this class
            prm.segs = p->d_segs + seg_off32[qc]; prm.nsegs = (int)plan32[qc].size(); prm.total_warps = warps32[qc];
            prm.coarse = p->d_coarse + co_off32[qc];
            prm.tau = tau; prm.tau_hi = tau64;
            prm.counters = p->d_counters + 4 * NQCLASS + 4 * qc;
            cudaEvent_t *e32 = ev + 2 * NQCLASS + 8;
            CUDA_TRY(cudaEventRecord(e32[2 * qc], st));
            ce.launch_jk(prm, st, true, true, true);
            ++launches;
            CUDA_TRY(cudaEventRecord(e32[2 * qc + 1], st));
            p->class_ran32[qc] = true;
        }
    }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaEventRecord(ev_eri, st));
    // (a6) finalise
    dim3 blk(32, 8), grd((N + 31) / 32, (N + 7) / 8);
    if (J) { symmetrize_kernel<<<grd, blk, 0, st>>>(J, N); ++launches; }
    if (K) { symmetrize_kernel<<<grd, blk, 0, st>>>(K, N); ++launches; }
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaEventRecord(ev_end, st));
    p->stats = adft_jk_stats_t{};
    p->stats.dmax = dmax;
    p->stats.quartets_unique = p->npairs * (p->npairs + 1) / 2;
    p->stats.kernel_launches = launches;
    p->have_build = true;
    p->last_stream = st;
    return ADFT_OK;
}

extern "C" adft_status_t adft_jk_stats(adft_shellpairs_t *p, adft_jk_stats_t *out)
{
    if (!p || !out) { set_error("adft_jk_stats: NULL"); return ADFT_ERR_INVALID_ARG; }
    if (!p->have_build) { set_error("adft_jk_stats: no build yet"); return ADFT_ERR_INVALID_ARG; }
    cudaStream_t st = p->last_stream;
    CUDA_TRY(cudaMemcpyAsync(p->h_small, p->d_counters, 8 * NQCLASS * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    adft_jk_stats_t &s = p->stats;
    cudaEvent_t *ev = p->ev;
    s.quartets_kept = 0; s.prim_quartets = 0; s.prim_quartets_evaluated = 0; s.model_flops = 0.0; s.quartets_fp32 = 0;
    for (int qc = 0; qc < NQCLASS; ++qc) {
        const unsigned long long *c32 = p->h_small + 4 * NQCLASS + 4 * qc;      // the fp32 launch of this class
        s.class_quartets_fp32[qc] = (int64_t)c32[0];
        s.quartets_fp32 += (int64_t)c32[0];
        s.class_quartets[qc] = (int64_t)(p->h_small[4 * qc] + c32[0]);
        const int64_t prim = (int64_t)(p->h_small[4 * qc + 1] + c32[1]);       // evaluated (after primitive screening)
        s.quartets_kept += s.class_quartets[qc];
        s.prim_quartets_evaluated += prim;
        s.class_prim_quartets[qc] = prim;
        s.prim_quartets += (int64_t)(p->h_small[4 * qc + 2] + c32[2]);
        const ClassEntry &ce = class_table()[qc];
        const int L = ce.la + ce.lb + ce.lc + ce.ld;
        // model flops: per primitive quartet 60+4L (geometry, prefactor, Boys) + generated VRR instructions
        // counted as 2 flops each; per contracted quartet 2*HRR + 12 per integral (6 FMAs of the digestion)
        s.class_model_flops[qc] = (double)prim * (60.0 + 4.0 * L + 2.0 * ce.vrr_ops)
                                + (double)s.class_quartets[qc] * (2.0 * ce.hrr_ops + 12.0 * ce.nint);
        s.model_flops += s.class_model_flops[qc];
        float ms = 0.f;
        s.class_ms[qc] = 0.0;
        if (p->class_ran[qc] && cudaEventElapsedTime(&ms, ev[2 * qc], ev[2 * qc + 1]) == cudaSuccess) s.class_ms[qc] = ms;
        s.class_ms_fp32[qc] = 0.0;
        if (p->class_ran32[qc] && cudaEventElapsedTime(&ms, ev[2 * NQCLASS + 8 + 2 * qc], ev[2 * NQCLASS + 8 + 2 * qc + 1]) == cudaSuccess)
            s.class_ms_fp32[qc] = ms;
    }
    float ms = 0.f;
    const int B = 2 * NQCLASS;
    if (cudaEventElapsedTime(&ms, ev[B], ev[B + 1]) == cudaSuccess) s.ms_dmax = ms;
    if (cudaEventElapsedTime(&ms, ev[B + 1], ev[B + 2]) == cudaSuccess) s.ms_plan = ms;
    if (cudaEventElapsedTime(&ms, ev[B + 2], ev[B + 3]) == cudaSuccess) s.ms_eri = ms;
    if (cudaEventElapsedTime(&ms, ev[B + 3], ev[B + 4]) == cudaSuccess) s.ms_finalize = ms;
    if (cudaEventElapsedTime(&ms, ev[B], ev[B + 4]) == cudaSuccess) s.ms_total = ms;
    cudaGetLastError();
    *out = s;
    return ADFT_OK;
}

extern "C" adft_status_t adft_jk_build_incremental(adft_shellpairs_t *p, const double *D, double *Dprev, double *J, double *K,
                                                   double tau, const adft_jk_options_t *opt, void *cuda_stream)
{
    if (!p || !D || !Dprev || (!J && !K)) { set_error("adft_jk_build_incremental: NULL handle, D or D_prev, or both J and K NULL"); return ADFT_ERR_INVALID_ARG; }
    if (Dprev == D || Dprev == J || Dprev == K) { set_error("adft_jk_build_incremental: D_prev must not alias D, J or K"); return ADFT_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n2 = (size_t)p->basis->nbf * p->basis->nbf;
    if (!p->d_incr) CUDA_TRY(cudaMalloc((void **)&p->d_incr, 3 * n2 * sizeof(double)));
    double *dD = p->d_incr, *Js = J ? p->d_incr + n2 : nullptr, *Ks = K ? p->d_incr + 2 * n2 : nullptr;
    const unsigned nb = (unsigned)std::min<size_t>((n2 + 255) / 256, (size_t)p->sm_count * 8);
    diff_kernel<<<nb, 256, 0, st>>>(D, Dprev, dD, n2);
    CUDA_TRY(cudaGetLastError());
    adft_jk_options_t o{};
    if (opt) o = *opt;
    o.flags |= ADFT_JK_BLOCK_DENSITY;
    adft_status_t rc = adft_jk_build_ex(p, dD, Js, Ks, tau, &o, cuda_stream);
    if (rc) return rc;
    incr_finish_kernel<<<nb, 256, 0, st>>>(J, Js, K, Ks, Dprev, D, n2);
    CUDA_TRY(cudaGetLastError());
    p->stats.kernel_launches += 2;
    return ADFT_OK;
}

extern "C" adft_status_t adft_jk_build_host(adft_shellpairs_t *p, const double *Dh, double *Jh, double *Kh, double tau,
                                            void *cuda_stream)
{
    if (!p || !Dh || (!Jh && !Kh)) { set_error("adft_jk_build_host: NULL handle or D, or both J and K NULL"); return ADFT_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n2 = (size_t)p->basis->nbf * p->basis->nbf;
    if (p->stage_n < 3 * n2) {
        cudaFree(p->d_stage); p->d_stage = nullptr; p->stage_n = 0;
        CUDA_TRY(cudaMalloc((void **)&p->d_stage, 3 * n2 * sizeof(double)));
        p->stage_n = 3 * n2;
    }
    double *dD = p->d_stage, *dJ = Jh ? p->d_stage + n2 : nullptr, *dK = Kh ? p->d_stage + 2 * n2 : nullptr;
    CUDA_TRY(cudaMemcpyAsync(dD, Dh, n2 * sizeof(double), cudaMemcpyHostToDevice, st));
    adft_status_t rc = adft_jk_build(p, dD, dJ, dK, tau, cuda_stream);
    if (rc) return rc;
    if (Jh) CUDA_TRY(cudaMemcpyAsync(Jh, dJ, n2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    if (Kh) CUDA_TRY(cudaMemcpyAsync(Kh, dK, n2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return ADFT_OK;
}

extern "C" adft_status_t adft_basis_nsph(const adft_basis_t *b, int32_t *nsph)
{
    if (!b || !nsph) { set_error("adft_basis_nsph: NULL"); return ADFT_ERR_INVALID_ARG; }
    int n = 0;
    for (int l : b->l) n += 2 * l + 1;
    *nsph = n;
    return ADFT_OK;
}

extern "C" adft_status_t adft_cart_to_spherical(adft_shellpairs_t *p, const double *M_cart, double *M_sph, void *cuda_stream)
{
    if (!p || !M_cart || !M_sph) { set_error("adft_cart_to_spherical: NULL"); return ADFT_ERR_INVALID_ARG; }
    if (M_cart == M_sph) { set_error("adft_cart_to_spherical: input and output must not alias"); return ADFT_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const adft_basis *b = p->basis;
    const int ns = b->nshells;
    if (!p->d_sph) {
        std::vector<int32_t> map;
        for (int s = 0; s < ns; ++s) for (int m = 0; m < 2 * b->l[s] + 1; ++m) map.push_back(s);
        const int nsph = (int)map.size();
        for (int s = 0; s < ns; ++s) for (int m = 0; m < 2 * b->l[s] + 1; ++m) map.push_back(m);
        for (int s = 0; s < ns; ++s) map.push_back(b->l[s]);
        SphTables tab;
        sph_fill_tables(tab);
        CUDA_TRY(cudaMalloc((void **)&p->d_sph, sizeof(SphTables)));
        CUDA_TRY(cudaMalloc((void **)&p->d_sph_map, map.size() * sizeof(int32_t)));
        CUDA_TRY(cudaMemcpyAsync(p->d_sph, &tab, sizeof(SphTables), cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaMemcpyAsync(p->d_sph_map, map.data(), map.size() * sizeof(int32_t), cudaMemcpyHostToDevice, st));
        CUDA_TRY(cudaStreamSynchronize(st));      // the host copies go out of scope
        p->nsph = nsph;
    }
    const int Ns = p->nsph;
    dim3 blk(32, 8), grd((Ns + 31) / 32, (Ns + 7) / 8);
    cart_to_sph_kernel<<<grd, blk, 0, st>>>(M_cart, b->nbf, M_sph, Ns, p->d_sph_map, p->d_sph_map + Ns, p->d_bfoff,
                                            p->d_sph_map + 2 * Ns, p->d_sph);
    CUDA_TRY(cudaGetLastError());
    return ADFT_OK;
}

extern "C" adft_status_t adft_fp64_peak_tflops(void *cuda_stream, double *tflops)
{
    if (!tflops) { set_error("adft_fp64_peak_tflops: NULL"); return ADFT_ERR_INVALID_ARG; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    double *d = nullptr;
    CUDA_TRY(cudaMalloc((void **)&d, sizeof(double)));
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0)); CUDA_TRY(cudaEventCreate(&e1));
    const int iters = 1 << 16, blocks = sms * 8, threads = 256;
    fp64_peak_kernel<<<blocks, threads, 0, st>>>(d, 1 << 10, 1.0);       // warm-up
    double best = 0.0;
    for (int rep = 0; rep < 5; ++rep) {
        cudaEventRecord(e0, st);
        fp64_peak_kernel<<<blocks, threads, 0, st>>>(d, iters, 1.0 + rep);
        cudaEventRecord(e1, st);
        CUDA_TRY(cudaEventSynchronize(e1));
        float ms = 0.f;
        CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
        const double fl = 2.0 * 8.0 * (double)iters * blocks * threads;
        best = std::max(best, fl / (ms * 1e-3) / 1e12);
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
    *tflops = best;
    return ADFT_OK;
}

// ------------------------------------------------------------------ the entry point that allocates nothing
// include/adft_noalloc.h: adft_cart_to_spherical with its working memory (the transform tables, the index map of the
// basis) in one file-scope device array instead of per-handle cudaMalloc'ed buffers.  Every call on a device shares the
// array; the basis-dependent part is rebuilt by noalloc_sph_map_kernel on the caller's stream ahead of the transform.
namespace adft {

struct NoAllocScratch {
    SphTables tab;                                    // written once per device at set-up
    int32_t sph_shell[ADFT_NOALLOC_MAX_NSPH];         // rebuilt by every call: shell of spherical function i,
    int32_t sph_m[ADFT_NOALLOC_MAX_NSPH];             //   m + l of it,
    int32_t shell_l[ADFT_NOALLOC_MAX_SHELLS];         //   l of every shell
};
constexpr size_t NOALLOC_BYTES = (sizeof(NoAllocScratch) + 255) / 256 * 256;

// In host code this name is a host-side stand-in, not a device address: host code takes the address with
// cudaGetSymbolAddress (noalloc_scratch_ptr below); device code may name the array directly.
static __device__ __align__(256) unsigned char g_noalloc_scratch[NOALLOC_BYTES];

// One block: l of every shell from its Cartesian size, an exclusive scan of 2l+1 over the shells, then the map.
// Overwrites everything the transform of this call reads; nothing has to be zero on entry.
__global__ void noalloc_sph_map_kernel(const int32_t *__restrict__ bfoff, int ns)
{
    NoAllocScratch *s = reinterpret_cast<NoAllocScratch *>(g_noalloc_scratch);
    __shared__ int part[1024];
    const int t = threadIdx.x, per = (ns + (int)blockDim.x - 1) / (int)blockDim.x;
    const int lo = min(t * per, ns), hi = min(lo + per, ns);
    int sum = 0;
    for (int sh = lo; sh < hi; ++sh) {
        const int nc = bfoff[sh + 1] - bfoff[sh];
        int l = 0;
        while ((l + 1) * (l + 2) / 2 < nc) ++l;
        s->shell_l[sh] = l;
        sum += 2 * l + 1;
    }
    part[t] = sum;
    __syncthreads();
    for (int d = 1; d < (int)blockDim.x; d <<= 1) {          // inclusive scan over the threads
        const int v = t >= d ? part[t - d] : 0;
        __syncthreads();
        part[t] += v;
        __syncthreads();
    }
    int o = part[t] - sum;
    for (int sh = lo; sh < hi; ++sh) {
        const int n = 2 * s->shell_l[sh] + 1;
        for (int m = 0; m < n; ++m) { s->sph_shell[o + m] = sh; s->sph_m[o + m] = m; }
        o += n;
    }
}

// The array's device address, once per device, taken with that device current.
static adft_status_t noalloc_scratch_ptr(NoAllocScratch **out)
{
    constexpr int MAXDEV = 64;
    static std::mutex mtx;
    static NoAllocScratch *ptr[MAXDEV] = {};
    int dev = -1;
    CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= MAXDEV) { set_error("adft_cart_to_spherical_noalloc: device ordinal out of range"); return ADFT_ERR_INVALID_ARG; }
    std::lock_guard<std::mutex> lk(mtx);
    if (!ptr[dev]) {
        void *a = nullptr;
        CUDA_TRY(cudaGetSymbolAddress(&a, g_noalloc_scratch));
        if (!a) { set_error("adft_cart_to_spherical_noalloc: cudaGetSymbolAddress returned NULL"); return ADFT_ERR_CUDA; }
        SphTables tab;                                       // 5.4 KB on the stack
        sph_fill_tables(tab);
        CUDA_TRY(cudaMemcpy(a, &tab, sizeof(SphTables), cudaMemcpyHostToDevice));      // tab is the first member
        ptr[dev] = static_cast<NoAllocScratch *>(a);
    }
    *out = ptr[dev];
    return ADFT_OK;
}

}  // namespace adft

extern "C" adft_status_t adft_cart_to_spherical_noalloc(adft_shellpairs_t *p, const double *M_cart, double *M_sph, void *cuda_stream)
{
    if (!p || !M_cart || !M_sph) { set_error("adft_cart_to_spherical_noalloc: NULL"); return ADFT_ERR_INVALID_ARG; }
    if (M_cart == M_sph) { set_error("adft_cart_to_spherical_noalloc: input and output must not alias"); return ADFT_ERR_INVALID_ARG; }
    const adft_basis *b = p->basis;
    const int ns = b->nshells;
    long long Ns = 0;
    for (int s = 0; s < ns; ++s) Ns += 2 * b->l[s] + 1;
    if (ns > ADFT_NOALLOC_MAX_SHELLS || Ns > ADFT_NOALLOC_MAX_NSPH) {
        set_error("adft_cart_to_spherical_noalloc: basis of " + std::to_string(ns) + " shells / " + std::to_string(Ns) +
                  " spherical functions exceeds the static scratch (at most " + std::to_string(ADFT_NOALLOC_MAX_SHELLS) +
                  " shells and " + std::to_string(ADFT_NOALLOC_MAX_NSPH) + " spherical functions); use adft_cart_to_spherical");
        return ADFT_ERR_INVALID_ARG;
    }
    NoAllocScratch *s = nullptr;
    adft_status_t rc = noalloc_scratch_ptr(&s);
    if (rc) return rc;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    noalloc_sph_map_kernel<<<1, 1024, 0, st>>>(p->d_bfoff, ns);
    CUDA_TRY(cudaGetLastError());
    dim3 blk(32, 8), grd(((int)Ns + 31) / 32, ((int)Ns + 7) / 8);
    cart_to_sph_kernel<<<grd, blk, 0, st>>>(M_cart, b->nbf, M_sph, (int)Ns, s->sph_shell, s->sph_m, p->d_bfoff, s->shell_l, &s->tab);
    CUDA_TRY(cudaGetLastError());
    return ADFT_OK;
}
