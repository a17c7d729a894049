/* adft.h -- C ABI of the B200-native direct-SCF Coulomb/exchange (J/K) builder.
 *
 * The operation (Eq. 1;  PAPER.md:68-70, the ERI;  PAPER.md:78-82, class batching and
 * Cauchy-Schwarz screening): for a contracted Cartesian Gaussian basis {phi_mu} and a symmetric density D,
 *
 *     J_mu,nu     = sum_{lambda,sigma} D_lambda,sigma (mu nu|lambda sigma)
 *     K_mu,lambda = sum_{nu,sigma}     D_nu,sigma     (mu nu|lambda sigma)
 *     (mu nu|lambda sigma) = iint phi_mu(r) phi_nu(r) |r-r'|^-1 phi_lambda(r') phi_sigma(r') d3r d3r'
 *
 * evaluated on the fly over the unique shell quartets (8-fold permutational symmetry) that pass
 *     (Q_AB * Q_CD) * max|D|  >=  schwarz_threshold ,   Q_AB = sqrt(max_{mu in A, nu in B} |(mu nu|mu nu)|)
 * ("If S(AB|CD) < TOLERANCE -> there will not be dispatch").  All arithmetic is fp64 unless the caller asks
 * for the paper's mixed-precision dispatch (ADFT_JK_MIXED_PRECISION of adft_jk_build_ex).
 *
 * Call sequence:  adft_basis_create -> adft_shellpairs_build -> adft_jk_build (any number of times)
 *                 -> adft_shellpairs_destroy -> adft_basis_destroy.
 *
 * Conventions
 *  - Every function returns adft_status_t (0 = success); nothing throws, aborts or prints.
 *  - "host" pointers are ordinary CPU memory, "device" pointers are CUDA global memory of the current device.
 *  - Units: bohr, Hartree.  Shell angular momentum l = 0..4 (s, p, d, f, g), Cartesian components.
 *  - Basis-function order: shells in input order; inside a shell the components (lx,ly,lz) with lx descending,
 *    then ly descending (p: x,y,z; d: xx,xy,xz,yy,yz,zz; f: xxx,xxy,xxz,xyy,xyz,xzz,yyy,yyz,yzz,zzz; g: xxxx,xxxy,...,zzzz).
 *  - All components of a shell share the contraction coefficients d_k:
 *       phi(r) = (x-Ax)^lx (y-Ay)^ly (z-Az)^lz sum_k d_k exp(-alpha_k |r-A|^2).
 *  - There is no CPU fallback: without a CUDA device the compute entry points return ADFT_ERR_CUDA.
 */
#ifndef ADFT_H
#define ADFT_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    ADFT_OK = 0,
    ADFT_ERR_INVALID_ARG = 1,   /* NULL pointer, negative size, bad index, non-positive exponent, tau < 0 or NaN */
    ADFT_ERR_UNSUPPORTED_L = 2, /* a shell has l > 4 (or l < 0) */
    ADFT_ERR_ALLOC = 3,         /* host or device allocation failed */
    ADFT_ERR_CUDA = 4,          /* CUDA runtime error; text in adft_last_error() */
    ADFT_ERR_NOT_FINITE = 5,    /* D contains NaN or Inf */
    ADFT_ERR_INTERNAL = 6
} adft_status_t;

/* One shell = one contraction of one angular momentum. */
typedef struct {
    int32_t atom;         /* index into atom_xyz_bohr */
    int32_t l;            /* 0..4 */
    int32_t nprim;        /* >= 1 */
    int32_t prim_offset;  /* first primitive of this shell in exponents[] / coefficients[] */
} adft_shell_t;

typedef struct adft_basis adft_basis_t;           /* opaque; owned by the library */
typedef struct adft_shellpairs adft_shellpairs_t; /* opaque; owns every device workspace */

/* flags for adft_basis_create */
#define ADFT_COEFFS_FINAL 0u      /* coefficients[] are the final d_k, used as given */
#define ADFT_NORMALIZE_SHELLS 1u  /* coefficients[] are raw c_k: d_k = c_k N_k / sqrt(S), N_k the primitive norm of
                                     the (L,0,0) component, S its contracted self-overlap (reading R-1) */

#define ADFT_MAX_CLASSES 120      /* quartet classes for l <= 4: 15 pair classes, 15*16/2 (the l <= 3 classes are 0..54) */

/* Counts and device times of the last adft_jk_build on a pairs handle. */
typedef struct {
    int64_t quartets_unique;      /* unique shell quartets before screening = P(P+1)/2 */
    int64_t quartets_kept;        /* unique shell quartets that pass the screen (the metric's numerator) */
    int64_t prim_quartets;        /* primitive quartets inside the kept quartets, nominal (full contraction depth) */
    int64_t prim_quartets_evaluated; /* primitive quartets actually evaluated (after primitive-pair screening) */
    int64_t class_quartets[ADFT_MAX_CLASSES]; /* kept per class; class = X(X+1)/2+Y, X >= Y pair classes,
                                                 pair class = hi(hi+1)/2+lo of the two angular momenta */
    int64_t class_prim_quartets[ADFT_MAX_CLASSES]; /* evaluated primitive quartets per class */
    double  class_ms[ADFT_MAX_CLASSES];       /* device time of each class kernel (CUDA events) */
    double  class_model_flops[ADFT_MAX_CLASSES]; /* model FP64 flops of each class launch */
    double  model_flops;          /* FP64 flops of the generated recurrences for the kept work */
    double  dmax;                 /* max|D| used by the screen */
    double  ms_dmax, ms_plan, ms_eri, ms_finalize, ms_total; /* device ms; ms_total = whole call */
    int32_t kernel_launches;      /* kernels launched by the call */
    int32_t reserved;
    /* mixed-precision dispatch (ADFT_JK_MIXED_PRECISION): the part of the counts above evaluated in single precision */
    int64_t quartets_fp32;
    int64_t class_quartets_fp32[ADFT_MAX_CLASSES];
    double  class_ms_fp32[ADFT_MAX_CLASSES];  /* device time of each class's single-precision launch */
} adft_jk_stats_t;

#define ADFT_MAX_NPRIM 32        /* largest contraction depth of one shell */

/* Copy and validate a basis.  All input arrays are HOST memory and are copied; the caller may free them on return.
 *   atom_xyz_bohr [natoms*3], shells [nshells], exponents / coefficients [sum of nprim] (indexed via prim_offset).
 * Errors: NULL / sizes <= 0 / atom index out of range / nprim < 1 or > ADFT_MAX_NPRIM / exponent <= 0 or non-finite
 *         -> INVALID_ARG;
 *         l outside 0..4 -> UNSUPPORTED_L.  *out is written only on success.  Needs no GPU. */
adft_status_t adft_basis_create(int32_t natoms, const double *atom_xyz_bohr,
                                int32_t nshells, const adft_shell_t *shells,
                                const double *exponents, const double *coefficients,
                                uint32_t flags, adft_basis_t **out);

/* Number of Cartesian basis functions N. */
adft_status_t adft_basis_nbf(const adft_basis_t *basis, int32_t *nbf);

/* bf_offset[s] = index of the first function of shell s; bf_offset[nshells] = N.  HOST array [nshells+1]. */
adft_status_t adft_basis_shell_offsets(const adft_basis_t *basis, int32_t *bf_offset);

/* Final contraction coefficients d_k as used by the library (after optional normalisation). HOST [nprim_total]. */
adft_status_t adft_basis_coefficients(const adft_basis_t *basis, double *coefficients);

/* Build the shell-pair table on the current CUDA device ("reordering"; PAPER.md:81 the bound):
 * for every shell pair A >= B the primitive-pair records (Gaussian product centre, exponent, prefactor) and the
 * Schwarz bound Q_AB; pairs are bucketed by angular-momentum pair class and contraction depth and sorted by Q
 * descending inside a bucket.  Work is enqueued on cuda_stream (a cudaStream_t, may be NULL = default stream) and the
 * call synchronises that stream before returning.  The basis must outlive the pairs handle. */
adft_status_t adft_shellpairs_build(const adft_basis_t *basis, void *cuda_stream, adft_shellpairs_t **out);

/* The same with an explicit primitive-pair threshold (reading R-11; the paper is silent on primitive
 * screening).  After the Schwarz bounds have been computed from the FULL contraction, a primitive pair (i on A, j on B)
 * is dropped from the table when its estimated primitive Schwarz factor
 *   sqrt|(ij|ij)| ~ |d_i d_j| exp(-a b |AB|^2/(a+b)) sqrt(2 pi^(5/2)/((a+b)^2 sqrt(2(a+b)))) (|PA|+(a+b)^-1/2)^la (|PB|+(a+b)^-1/2)^lb
 * is below prim_threshold (absolute, in sqrt(Hartree)); the largest primitive pair of a shell pair is always kept.
 * prim_threshold = 0 keeps every primitive pair (the plain definition, what the oracle evaluates).
 * adft_shellpairs_build uses ADFT_DEFAULT_PRIM_THRESHOLD.  Errors: negative or non-finite threshold -> INVALID_ARG. */
#define ADFT_DEFAULT_PRIM_THRESHOLD 1e-15
adft_status_t adft_shellpairs_build_ex(const adft_basis_t *basis, double prim_threshold, void *cuda_stream,
                                       adft_shellpairs_t **out);

/* Primitive-pair records before / after primitive screening and the threshold used. */
adft_status_t adft_shellpairs_prim_counts(const adft_shellpairs_t *pairs, int64_t *nominal, int64_t *kept,
                                          double *threshold);

/* Schwarz bounds as a full symmetric HOST matrix Q[nshells*nshells] (row-major, shell order of the basis). */
adft_status_t adft_shellpairs_schwarz(const adft_shellpairs_t *pairs, double *Q);

/* The J/K build.  D, J, K are DEVICE pointers to N*N row-major fp64 matrices owned by the caller.
 *   D  symmetric (precondition, not checked), must not alias J or K.
 *   J, K  overwritten (not accumulated) with the full symmetric matrices; either may be NULL to skip it.
 *         No exchange factor, sign or 1/2 is applied:  E_J = 1/2 tr(DJ), E_K = -1/4 tr(DK).
 *   schwarz_threshold  tau >= 0; a quartet is skipped iff (Q_AB*Q_CD)*max|D| < tau.
 * All device work is enqueued on cuda_stream; the call makes small host synchronisations (max|D|, the launch plan)
 * and may return before the last kernel finishes: results are valid after the caller synchronises the stream.
 * One build in flight per pairs handle.
 * Errors: NULL handle or D, both J and K NULL, tau < 0 or NaN -> INVALID_ARG (outputs untouched);
 *         non-finite D -> NOT_FINITE (outputs untouched);  CUDA failures -> ERR_CUDA. */
adft_status_t adft_jk_build(adft_shellpairs_t *pairs, const double *D, double *J, double *K,
                            double schwarz_threshold, void *cuda_stream);

/* Options of adft_jk_build_ex.  Zero-initialise the struct: every field at 0 means "as adft_jk_build".
 *
 *  ADFT_JK_BLOCK_DENSITY (Haeser-Ahlrichs density screening; reading R-23):
 *     the single max|D| of the screen is replaced, per quartet, by
 *         Dblk(AB|CD) = max(|D|_AB, |D|_CD, |D|_AC, |D|_AD, |D|_BC, |D|_BD),  |D|_XY = max over the shell block,
 *     i.e. a quartet is skipped iff (Q_AB*Q_CD)*Dblk < tau.  Dblk <= max|D|, so the kept set is a subset of the default
 *     rule's; adft_jk_stats reports the kept counts of the rule that was used.
 *  shard_rank / shard_count (replicated D, independent quartet batches, one
 *     reduction): the call evaluates only the warp tiles t of every class launch with t % shard_count == shard_rank
 *     and writes the PARTIAL symmetric J, K of those quartets; the sum over all ranks of a group is the full result
 *     (one all-reduce, done by the caller -- the Python binding uses torch.distributed).  shard_count 0 or 1 = all
 *     tiles.  adft_jk_stats then reports the counts of this rank's share.
 *  ADFT_JK_MIXED_PRECISION (the paper's "mixed single and double precision strategy"):
 *     with S = (Q_AB*Q_CD)*density, the number the screen already forms (reading R-24),
 *         S < tau                     -> not evaluated                       ("there will not be dispatch")
 *         tau <= S < fp32_band * tau  -> evaluated in SINGLE precision       ("the single precision version is enough")
 *         S >= fp32_band * tau        -> evaluated in double precision       ("the double precision version is necessary")
 *     Single precision = Boys function, recurrences, contraction and per-quartet digestion sums in fp32; the product
 *     centre difference P - Q and every reduction into J and K stay fp64.  The kept set and its counts are those of
 *     the fp64 build.  Each single-precision integral carries a relative error of order 1e-6 on a contribution bounded
 *     by fp32_band*tau, i.e. an absolute error per quartet of the order of the screening threshold itself; J and K
 *     then differ from the fp64 build by more than the 1e-10 of the default path (DESIGN.md section 7 has the measured
 *     error study).  Needs both J and K; the quartet classes with f shells that run through the Rys kernels stay fp64.
 *  Errors: unknown flag bits, shard_rank outside [0, shard_count), mixed precision with J or K NULL, fp32_band < 1
 *  or non-finite -> INVALID_ARG. */
#define ADFT_JK_BLOCK_DENSITY 1u
#define ADFT_JK_MIXED_PRECISION 2u
#define ADFT_DEFAULT_FP32_BAND 1e5
typedef struct {
    uint32_t flags;
    int32_t shard_rank, shard_count;
    int32_t reserved0;
    double fp32_band;             /* ADFT_JK_MIXED_PRECISION: width of the single-precision band; 0 = 1e5 */
    double reserved[3];
} adft_jk_options_t;

/* adft_jk_build with options (NULL options = adft_jk_build). */
adft_status_t adft_jk_build_ex(adft_shellpairs_t *pairs, const double *D, double *J, double *K,
                               double schwarz_threshold, const adft_jk_options_t *options, void *cuda_stream);

/* Incremental build ("incremental Fock"): J and K are linear in D, so given the matrices
 * of a previous density only the difference has to be evaluated, and with the block-density screen a small, localised
 * dD keeps few quartets.  All pointers DEVICE, N*N fp64:
 *   on entry  J, K hold the matrices that belong to D_prev (either may be NULL);
 *   the call forms dD = D - D_prev, builds J(dD), K(dD) with ADFT_JK_BLOCK_DENSITY (always on here; the other
 *   options apply as given) into internal buffers, and then
 *   on exit   J += J(dD), K += K(dD), D_prev = D.
 * The screening error of a sequence of incremental builds accumulates: callers rebuild from scratch every few
 * iterations.  Stats are those of the dD build.  Errors as adft_jk_build; D_prev must not alias D, J or K. */
adft_status_t adft_jk_build_incremental(adft_shellpairs_t *pairs, const double *D, double *D_prev, double *J, double *K,
                                        double schwarz_threshold, const adft_jk_options_t *options, void *cuda_stream);

/* Spherical-harmonic output.  nsph = sum over shells of 2l+1. */
adft_status_t adft_basis_nsph(const adft_basis_t *basis, int32_t *nsph);

/* M_sph = T^T M_cart T for a DEVICE N*N matrix in the Cartesian basis (J or K of adft_jk_build): M_sph is a DEVICE
 * nsph*nsph row-major matrix in the basis of real solid harmonics, shells in input order, m = -l, ..., +l inside a shell
 * (p: y, z, x;  d: xy, yz, 2zz-xx-yy, xz, xx-yy;  f, g: the textbook forms listed in csrc/adft_sph.cuh), each function
 * normalised to unit self-overlap given the shell's radial function (the one whose (L,0,0) Cartesian component is
 * normalised, R-1).  Enqueued on cuda_stream; the first call on a handle synchronises once.
 * Errors: NULL or aliasing pointers -> INVALID_ARG. */
adft_status_t adft_cart_to_spherical(adft_shellpairs_t *pairs, const double *M_cart, double *M_sph, void *cuda_stream);

/* Convenience for host callers: D, J, K are HOST N*N arrays; the call stages them through internal device buffers
 * on cuda_stream (host->device copy of D, the build, device->host copies of J and K) and synchronises. */
adft_status_t adft_jk_build_host(adft_shellpairs_t *pairs, const double *D_host, double *J_host, double *K_host,
                                 double schwarz_threshold, void *cuda_stream);

/* Counts and timings of the last build; synchronises the build's stream to read the event timers. */
adft_status_t adft_jk_stats(adft_shellpairs_t *pairs, adft_jk_stats_t *out);

/* Number of shell pairs (A >= B) in the table and number of primitive-pair records. */
adft_status_t adft_shellpairs_counts(const adft_shellpairs_t *pairs, int64_t *npairs, int64_t *nprimpairs);

void adft_shellpairs_destroy(adft_shellpairs_t *pairs);
void adft_basis_destroy(adft_basis_t *basis);

const char *adft_status_string(adft_status_t status);
const char *adft_last_error(void);  /* thread-local detail message of the last failing call */

/* Microbenchmark used by bench.py for the roofline denominator: runs a register-resident chain of
 * dependent-free fp64 FMAs on every SM of the current device and returns achieved FP64 TFLOP/s (2 flops per FMA)
 * measured with CUDA events on cuda_stream. */
adft_status_t adft_fp64_peak_tflops(void *cuda_stream, double *tflops);

#ifdef __cplusplus
}
#endif
#endif /* ADFT_H */
