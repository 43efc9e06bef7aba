/* pf_debug.h -- introspection entry points of libpf_b200 for the tests, bench.py and report.py.
 *
 * Not part of the solver's boundary (include/pf.h is): these calls expose assembled
 * arrays, layouts, counters and the host-side planner so that the parity tests can compare rows L1/L2 bit for
 * bit with the oracle and the bench can count launches and time single kernels.  Same conventions as pf.h
 * (host/device, ownership, return codes).
 */
#ifndef PF_B200_DEBUG_H
#define PF_B200_DEBUG_H

#include "pf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Accumulated device time (ms) and launch count of the three per-iteration kernels since
 * PF_OPT_PROFILE was set: index 0 = p-update + matvec + r~.v (row L4), 1 = s-update + matvec + t.s,
 * t.t (row L5), 2 = x, r update + r~.r, r.r (row L6).  ms_out, launches_out: host, 3 entries. */
int pf_grid_profile(pf_grid *g, double *ms_out, long long *launches_out);

/* Kernel launches issued by the library in this process so far. */
long long pf_launch_count(void);

/* Row N5 alone through the kernel and the per-grid scratch that pf_solve_pf uses (Table 2 step 5):
 * phi := omega_pf phi0 + (1 - omega_pf) phi over the grid's N nodes; *incr_out (host) = ||phi - phi0||_inf.
 * phi0, phi: device, N doubles.  The reference the no-allocation entry point (pf_noalloc.h) is tested against. */
int pf_grid_relax(pf_grid *g, double omega_pf, const double *phi0, double *phi, double *incr_out);

/* BiCGSTAB iterations of the Laplace solve for phi^L (charge model 1). */
int pf_grid_laplace_iters(const pf_grid *g);

/* Number of linear solves of this grid that were repeated by the direct kernels because the tiled kernels met
 * operands outside the range of their branch-free division (reading D4 of DESIGN.md). */
int pf_grid_fault_repeats(const pf_grid *g);

/* Decomposition the cooperative kernel (PF_OPT_KERNELS = 3; pf_krylov_coop.cu) would use for an nx x ny x nz box
 * on a device with max_blocks SMs and smem_cap bytes of dynamic shared memory per block: one brick per block,
 * brick k of nb along an axis of n nodes = nodes floor(k n/nb) .. floor((k+1) n/nb) - 1.  Host arithmetic only
 * (no device is touched).  out (host, 8 ints): bricks per direction nbx, nby, nbz; array extents of the largest
 * brick: own nodes (rounded up to even), nodes with one halo layer, halo nodes; threads per block; bytes of
 * dynamic shared memory.  Returns PF_OK, or PF_ERR_ARG when no decomposition fits (the solver then uses the
 * three-kernel families) or an argument is invalid. */
int pf_coop_plan(int nx, int ny, int nz, int max_blocks, size_t smem_cap, int *out);

/* How the persistent tiled kernels (pf_krylov_tma.cu) hand the tiles x z ranges of an nx x ny x nz box to their blocks
 * on a device with sm_count SMs, for tiles of tile_rows (13 or 16) rows and PF_OPT_SEGMENTS = mode (-1, 0, 1).  Host
 * arithmetic only.  out (host, 9 ints): mode chosen (0 equal chunks, 1 two groups); tiles along x; tiles; mode 0: chunk
 * depth, mode 1: layer depth of the main group; mode 0: items = tiles * chunks, mode 1: blocks of the main group; mode 1:
 * first plane of the rest group, its number of planes, and the flattened (tile-major) positions per rest block; blocks
 * launched.  Block b works on: mode 0 -- items b, b + blocks, ... with item i = tile i % tiles, planes
 * [(i / tiles) * depth, min(+ depth, nz)); mode 1, b < main -- tile b % tiles, planes [(b / tiles) * depth, + depth);
 * mode 1, rest block r = b - main -- positions [r q, min((r + 1) q, tiles * erest)), position p = tile p / erest, plane
 * zrest + p % erest, cut into one segment per tile.  Mode 2 (out[3] = depth of the lower layer, out[4] = tiles, zrest =
 * that depth, erest = nz - zrest, q = pieces): block b < tiles -- tile b, planes [0, depth); block b >= tiles, r = b -
 * tiles, R = blocks - tiles, L = tiles - R -- first tile r, planes [zrest, nz), then, if r < L q, tile R + r % L, planes
 * [zrest + (r / L) dp, min(+ dp, nz)) with dp = ceil(erest / q).  Returns PF_OK or PF_ERR_ARG. */
int pf_tile_plan(int nx, int ny, int nz, int tile_rows, int sm_count, int mode, int *out);

/* Introspection used by the tests: 1 = stored, 2 = on-the-fly; number of palette entries. */
int pf_grid_stencil(const pf_grid *g);
int pf_grid_palette_size(const pf_grid *g);

/* Layout of the stencil codes of the on-the-fly variant: bits per code (16: six 2-bit fields, 32: six
 * 4-bit fields, 0: none -- more than 4 distinct eps values), row pitch in codes (nx rounded up to 8;
 * code of node (ix,iy,iz) at ix + pitch*(iy + ny*iz)), bytes of one code array.  Field d-1 (d = 1..6 in
 * the order east, west, south, north, down, up of PAPER.md:219) indexes the coefficient table; index 0
 * is the coefficient 0.  Out-pointers: host, may be NULL. */
int pf_grid_code_layout(const pf_grid *g, int *bits_out, int *pitch_out, size_t *bytes_out);

/* Copy an assembled array into caller memory (device), for the assembly parity tests (rows L1/L2):
 * which = 0: Poisson diagonal A0 (N doubles); 1..6: stored off-diagonals A1..A6 (stored variant
 * only); 7: deposited fixed-charge vector (N doubles); 8: Poisson stencil codes (pf_grid_code_layout
 * bytes); 9: PF1 diagonal (N doubles, after a pf_solve_pf); 10: Poisson coefficient table (16 doubles);
 * 11: PF1 stencil codes; 12: PF1 coefficient table; 13: Psi of the last pf_solve_pf (N doubles);
 * 14: phi^L, 15: phi* on Omega_m (N doubles each, charge model 1; with it, 7 is b^IF).
 * Returns PF_ERR_ARG if unavailable. */
int pf_grid_copy_array(pf_grid *g, int which, void *dst_device);

#ifdef __cplusplus
}
#endif
#endif /* PF_B200_DEBUG_H */
