/* pf_noalloc.h -- one entry point of libpf_b200 that allocates nothing.
 *
 * Why: some callers cannot call cudaMalloc -- code under CUDA graph capture, tight serving loops, harnesses that
 * forbid it.  Every other call of the library needs a pf_grid, whose creation allocates small device buffers.  This one
 * needs no grid: its scratch is a file-scope `static __device__` array inside the library (pf_noalloc.cu), which every
 * GPU that loads the library holds until the process exits.
 *
 * What it computes: row N5 of the hot path, Table 2 step 5 / Table 4 step 7 of the paper (
 * readings Q8, Q9 of DESIGN.md): the relaxation Phi := omega_PF Phi0 + (1 - omega_PF) Phi and the increment
 * ||Phi - Phi0||_inf after it -- the same arithmetic, operation for operation, as the kernel pf_solve_pf uses; the
 * maximum goes through per-block partial results in the scratch instead of an atomic (no zeroing, deterministic).
 */
#ifndef PF_B200_NOALLOC_H
#define PF_B200_NOALLOC_H

#include "pf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Largest n the entry point accepts: the scratch holds one partial maximum per block of 4096 nodes,
 * 65 536 blocks = 512 KB of device memory per GPU (+ 256 bytes), enough for 2^28 nodes (512^3 = 2^27). */
#define PF_NOALLOC_MAX_N (1LL << 28)

/* phi := omega_pf * phi0 + (1 - omega_pf) * phi;  *incr_out = max_i |phi_i - phi0_i| (a NaN anywhere gives NaN).
 *   n        : number of nodes, 0 <= n <= PF_NOALLOC_MAX_N (n = 0: *incr_out = 0).
 *   phi0     : device, n doubles, in.
 *   phi      : device, n doubles, in/out.
 *   incr_out : device, 1 double, out.
 *   cuda_stream : a cudaStream_t (NULL = the legacy default stream).  The call only enqueues two kernels on it and
 *                 returns; it calls no cudaMalloc, cudaFree, or any allocating routine, and does not synchronise.
 * The scratch is shared by every call on the device and keeps the last call's contents (each call overwrites the
 * entries it reads, nothing has to start at zero).  Calls that overlap on the GPU -- two streams, or two host threads --
 * race on it: serialise them (one stream, or events between streams).
 * Returns PF_OK; PF_ERR_ARG (NULL pointer, n < 0, n > PF_NOALLOC_MAX_N, omega_pf outside [0, 1); message via
 * pf_last_error(NULL)); PF_ERR_CUDA (no device, cudaGetSymbolAddress or a launch failed). */
int pf_relax_noalloc(long long n, double omega_pf, const double *phi0, double *phi, double *incr_out,
                     void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* PF_B200_NOALLOC_H */
