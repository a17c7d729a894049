/* adft_noalloc.h -- the one entry point of libadft.so that allocates nothing.
 *
 * Some callers cannot call cudaMalloc: code under CUDA graph capture, tight serving loops, harnesses that forbid it.
 * adft_cart_to_spherical (adft.h, "spherical-harmonic output") allocates its index map and transform
 * tables on the first call of every shell-pair handle.  The variant below keeps that working memory in ONE file-scope
 * device array of fixed size inside the library (csrc/adft_lib.cu, `g_noalloc_scratch`, 256-byte aligned, about 166 KiB;
 * every GPU that loads the library holds it until the process exits) and calls no cudaMalloc, cudaFree, cudaMallocHost
 * or any other allocating routine, on the host heap or on the device.
 *
 * Limits (the array's size): a basis of at most ADFT_NOALLOC_MAX_SHELLS shells and ADFT_NOALLOC_MAX_NSPH spherical
 * functions; anything larger is refused with ADFT_ERR_INVALID_ARG and a message naming the limit (adft_last_error),
 * before anything is enqueued.
 *
 * Sharing: every call on a device uses the same array and rebuilds the part that depends on the basis (the shell and
 * m of every spherical function, l of every shell) with a set-up kernel enqueued on cuda_stream ahead of the transform;
 * nothing in it has to start at zero, and nothing of the previous call is read.  Calls that OVERLAP on one GPU (two
 * streams, two host threads) RACE on the array: serialise them (one stream, or events).  Calls on different GPUs do
 * not interact.
 *
 * The first call on each device takes the array's device address (cudaGetSymbolAddress, with that device current) and
 * copies the basis-independent solid-harmonic tables (5.4 KB) into it with a synchronous cudaMemcpy: make that first
 * call outside any capture.  Later calls only enqueue two kernels.
 */
#ifndef ADFT_NOALLOC_H
#define ADFT_NOALLOC_H

#include "adft.h"

#ifdef __cplusplus
extern "C" {
#endif

#define ADFT_NOALLOC_MAX_SHELLS 8192
#define ADFT_NOALLOC_MAX_NSPH 16384

/* M_sph = T^T M_cart T, exactly as adft_cart_to_spherical (same kernel, same tables, bit-identical result):
 *   pairs   handle of adft_shellpairs_build (only its basis and shell offsets are read; nothing in it is modified);
 *   M_cart  DEVICE, N*N fp64 row-major (J or K), read only;
 *   M_sph   DEVICE, nsph*nsph fp64 row-major (adft_basis_nsph), written; owned by the caller like M_cart.
 * The device that holds the handle must be current.  Enqueued on cuda_stream; returns without synchronising (except
 * the first call on a device, see above).
 * Errors: NULL or aliasing pointers, more shells or spherical functions than the limits -> ADFT_ERR_INVALID_ARG;
 * a failing CUDA call (cudaGetSymbolAddress included) -> ADFT_ERR_CUDA. */
adft_status_t adft_cart_to_spherical_noalloc(adft_shellpairs_t *pairs, const double *M_cart, double *M_sph, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
