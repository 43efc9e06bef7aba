/* pf.h -- C ABI of libpf_b200: the Poisson-Fermi hot path of arXiv 1711.04060 on one B200.
 *
 * Citations are PAPER.md:<line> (the paper's text) or a reading R0..R5 / Q1..Q29 of DESIGN.md.
 *
 * What the library computes
 *   - operator assembly from a relative-permittivity map: the 7-point finite-difference rows of
 *     -div(eps grad u) + sigma u with the simplified matched-interface rows of Eqs (15)-(18)
 *     (they reduce to harmonic-mean face coefficients, reading R2), identity rows
 *     on Dirichlet nodes, omitted outward flux on zero-Neumann faces (Eq (4));
 *   - the Jacobi-preconditioned BiCGSTAB of Table 3 (reading R3);
 *   - the inexact-Newton PF loop of Table 2 steps 2-5 / Table 4 steps 4-7 (PAPER.md:217-228,
 *     281-291): pointwise Fermi-like distribution Eq (1), PF1/PF2 of Eqs (12)-(14)
 *     (PAPER.md:122-133), relaxation and the test on the potential increment.
 *
 * Conventions
 *   Grid nx*ny*nz nodes INCLUDING the boundary layer, linear index i = ix + nx*(iy + ny*iz)
 *   (x fastest); node (ix,iy,iz) sits at (ix*h, iy*h, iz*h) Angstrom.
 *   phi in k_B T/e, lengths in Angstrom, concentrations in 1/A^3, charges in e, all fp64.
 *   "device" = pointer to CUDA device memory of the current device, "host" = ordinary host memory.
 *   All device work is enqueued on the stream given to pf_grid_create; a call returns after the
 *   stream work its out-parameters depend on has completed.
 *   Ownership: the caller owns every array it passes.  eps_map and the workspace are BORROWED for
 *   the lifetime of the grid.  The library itself allocates only small (KB-sized) device buffers.
 *   Return value: 0 = PF_OK; < 0 = error (message via pf_last_error); > 0 = soft status.
 *   No exceptions or aborts cross this boundary.  There is no CPU fallback: without a CUDA device
 *   every compute call returns PF_ERR_CUDA.
 */
#ifndef PF_B200_H
#define PF_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define PF_OK                0
#define PF_NOT_CONVERGED     1   /* maxit (or max outer iterations) reached; outputs hold the last iterate */
#define PF_INNER_NOT_CONVERGED 2 /* pf_solve_pf: the increment met the tolerance, but at least one of the linear solves
                                    stopped at PF_OPT_LINEAR_MAXIT and its last iterate was used as it stood */
#define PF_ERR_ARG          -1
#define PF_ERR_CUDA         -2
#define PF_ERR_BREAKDOWN    -3   /* rho = 0, r~.v = 0 or omega = 0 before convergence (reading Q5); a reduced scalar or
                                    the potential increment is not finite (NaN/inf input, divergence; reading D7) */
#define PF_ERR_NONPHYSICAL  -4   /* bath not neutral or Gamma^B <= 0 (reading Q26) */
#define PF_ERR_WORKSPACE    -5   /* workspace missing or too small */

/* Boundary faces in the order -x,+x,-y,+y,-z,+z (Eq (4)). */
#define PF_BC_DIRICHLET 0        /* phi = value[face] (k_B T/e) */
#define PF_BC_NEUMANN   1        /* zero normal derivative: outward face flux omitted (Q21) */

typedef struct pf_grid pf_grid;                  /* opaque */
typedef struct { int type[6]; double value[6]; } pf_bc;
typedef struct { double x, y, z, q; } pf_charge; /* position in Angstrom (node 0 at the origin), charge in e */

/* Option keys for pf_grid_set_option.  Values are doubles; integer options are rounded. */
#define PF_OPT_STENCIL         1  /* 0 = auto, 1 = stored coefficients A1..A6 (the paper's diagonal
                                     format), 2 = on-the-fly coefficients: per node a packed
                                     code of six indices into the table of distinct face coefficients of
                                     the eps map.  auto = on-the-fly when the map has <= 4 distinct
                                     values, else stored.  Both give bit-identical results.  Must be
                                     set before pf_grid_set_workspace. */
#define PF_OPT_OMEGA_PF        2  /* relaxation parameter of Table 2 step 5; default 0.3 */
#define PF_OPT_LINEAR_TOL      3  /* relative tolerance of the solves inside pf_solve_pf; default 1e-10 */
#define PF_OPT_LINEAR_MAXIT    4  /* their iteration cap; default 10000 */
#define PF_OPT_CHECK_INTERVAL  5  /* BiCGSTAB iterations enqueued between two host polls of the
                                     device-side convergence flag (PF_OPT_GRAPH 0 and 1); default 16; >= 1 */
#define PF_OPT_WATER_MOLAR     6  /* bath concentration of water, mol/L; default 55.5 (Q12) */
#define PF_OPT_MAX_OUTER       7  /* cap on outer (Newton) iterations; default 1000 */
#define PF_OPT_PRECOND         8  /* 1 = Jacobi M = diag(A) (default, reading Q2); 0 = M = I, Table 3 verbatim */
#define PF_OPT_HISTORY         9  /* >0: keep the relative residual of every BiCGSTAB iteration of the
                                     last linear solve (up to that many entries); see pf_grid_history */
#define PF_OPT_KERNELS        10  /* 0 = auto, 1 = direct (one thread per node, neighbours through L1/L2),
                                     2 = tiled (planes staged in shared memory by TMA, z-marched; needs
                                     nx >= 32, ny >= 16, nz >= 8, 16-byte aligned vectors, and for an odd nx
                                     the on-the-fly stencil: the solve then runs on the box widened by one
                                     column of decoupled identity rows),
                                     3 = cooperative (a whole solve in one persistent kernel, one brick of
                                     the box per SM with its vectors in shared memory, three grid-wide
                                     barriers per iteration; needs the on-the-fly stencil and a grid of at
                                     most about 72^3 nodes).  Same arithmetic, bit-identical vectors. */

#define PF_OPT_PROFILE        11  /* n > 0: bracket the three kernels of the first n iterations of every
                                     linear solve with CUDA events and accumulate their durations
                                     (pf_grid_profile); setting it resets the sums; 0 = off */

#define PF_OPT_GRAPH          12  /* how the iterations of a linear solve reach the GPU (three-kernel families).
                                     0: plain stream launches; the host polls the device-side flag every
                                     PF_OPT_CHECK_INTERVAL iterations.  1: each polling chunk is replayed as one CUDA
                                     graph.  2: device-side loop -- one CUDA graph launch per solve whose WHILE
                                     conditional node repeats a body of 8 or 16 iterations until the solve is over
                                     (converged, breakdown) or the whole bodies below maxit are done; the host does not
                                     poll; the fewer-than-a-body iterations up to maxit follow as stream launches.
                                     3 (default): 2 for solves expected to take fewer than 192 iterations (by the
                                     previous solve with the same operator, e.g. the inner solves of pf_solve_pf),
                                     1 for longer ones.  All give the same bits.  2 falls back to 1, and 1 to 0, if a
                                     graph cannot be built. */

#define PF_OPT_NORM           13  /* stopping test of every linear solve.  0 (default, reading Q3): ||r||_2 <= tol ||b||_2;
                                     1: the paper's own test, Table 3 steps 18-19: ||r||_inf < tol,
                                     absolute.  With 1, relres_out, true_relres_out and the history are absolute
                                     maximum norms. */

#define PF_OPT_CHARGE_MODEL   14  /* how the fixed point charges enter.  0 (default, reading Q22): trilinear deposition on
                                     the 8 surrounding nodes.  1: the singular-charge decomposition of Eqs (5)-(10)
                                     (PAPER.md:85-111): phi = phi~ + phi* + phi^L in Omega_m (the low-eps nodes, Q17),
                                     phi* the Coulomb sum with eps_m = min eps, phi^L from a Laplace solve in Omega_m run
                                     inside pf_grid_set_workspace (Table 2 step 1), the charges entering the equations
                                     for phi~ only through the interface vector b^IF (flux-jump terms of Eqs (17)-(18)).
                                     pf_solve_pf then returns the total phi.  Needs 3 more workspace vectors; must be
                                     set before pf_grid_set_workspace; all charges are assumed to lie in Omega_m. */

#define PF_OPT_DIAG_FROM_CODE 15  /* 1: in Poisson solves without sigma (pf_solve_linear, the initial guess of
                                     pf_solve_pf) with 2-byte stencil codes, the tiled kernel of row L4 looks the
                                     diagonal A0 = sum of the six face coefficients up from the code instead of
                                     reading it (8 bytes per unknown less; same bits), together with the divisor's
                                     half of the Jacobi division.  2: the kernel of row L5 as well.  0: A0 is read. */

#define PF_OPT_SOLVER         16  /* 0 (default): BiCGSTAB as Table 3 writes it, three kernels and three reduction points per
                                     iteration.  1: the merged recurrence (SURVEY 8(d) "fully merged"; reading M1 of
                                     DESIGN.md): rho_i = (r~.r_{i-1} - alpha r~.v) - omega r~.t, two kernels and two
                                     reduction points per iteration (s, t = A M^-1 s | r, x, p, v = A M^-1 p fused), fewer
                                     bytes per unknown.  The same method; iterates differ from Table 3's in rounding,
                                     so its parity reference is the oracle's bicgstab_merged().  Applies to every linear
                                     solve of the grid, those inside pf_solve_pf included.  Direct and tiled kernel families
                                     (tiled: on-the-fly stencil); the cooperative kernel implements Table 3 only. */

#define PF_OPT_STERIC_MODE    17  /* how pf_solve_pf reads the three mutually dependent definitions of Eq (11).
                                     0 (default, reading Q11): solved simultaneously per node.  1 (readings G1, G2): as
                                     assignments in the order written -- C_k from phi_0 and the S^trc of the previous outer
                                     iteration (0 before the first), then Gamma_0, floored at 1e-12, gives the next S^trc.
                                     Same fixed point; converges for potentials of a few kT/e and two-cycles on crowded
                                     nodes (on configs[0] as stated), which is why it is not the default. */

#define PF_OPT_TILE_ROWS      18  /* tiled kernels: rows of a tile = main warps of a block.  0 (default): chosen per kernel
                                     and grid size (16 rows / 19 warps / 96 registers, or 13 rows / 16 warps / 128
                                     registers); 13 or 16 force one geometry.  Same bits either way; a tuning and
                                     measurement knob. */

#define PF_OPT_SEGMENTS       19  /* tiled kernels: how tiles x z ranges are handed to the persistent blocks.  -1 (default):
                                     chosen per grid; 0: z cut into equal chunks, blocks take (tile, chunk) items
                                     round-robin; 1: for grids with at most half as many tiles as SMs, whole layers in step
                                     on most SMs and the remaining planes split evenly over the other SMs; 2: for grids
                                     with between half and two thirds as many tiles as SMs, a deep lower layer on one
                                     block per tile, the upper layer of as many tiles as blocks are left, and the upper
                                     layer of the other tiles in pieces afterwards.  A forced plan that does not exist
                                     for the grid falls back to 0.  Same bits either way; a tuning and measurement knob. */

/* Create a grid: store geometry and boundary conditions, scan eps_map for its palette of distinct
 * values, keep a device copy of the charges.  Assembly itself runs in pf_grid_set_workspace.
 *   eps_map : device, nx*ny*nz doubles, relative permittivity per node; borrowed.
 *   charges : host, ncharges entries (may be NULL when ncharges = 0); copied.
 *   bc      : host; copied.
 *   cuda_stream : a cudaStream_t (NULL = the legacy default stream).
 * Errors: PF_ERR_ARG (n < 3 in a direction, h <= 0, NULL pointers, bad bc type), PF_ERR_CUDA. */
int pf_grid_create(pf_grid **out, int nx, int ny, int nz, double h,
                   const double *eps_map, const pf_charge *charges, int ncharges,
                   const pf_bc *bc, void *cuda_stream);

/* Omega_f (readings F1-F3 of DESIGN.md): `count` nodes whose potential an atomic model
 * prescribes.  idx_host[k] is the linear index of a node, val_host[k] its potential in k_B T/e; both host, copied.
 * These nodes become interior Dirichlet nodes of every system built on the grid (identity rows, neighbours keep
 * their coupling, Q20), carry Psi = 0 in PF1, and are excluded from the Fermi distribution (C_k = 0 there).
 * Must be called before pf_grid_workspace_bytes / pf_grid_set_workspace (one more workspace vector); count = 0
 * removes them.  Errors: PF_ERR_ARG (index outside the grid, NaN value, called after assembly). */
int pf_grid_set_fixed_nodes(pf_grid *g, const long long *idx_host, const double *val_host, int count);

/* Bytes of device scratch the grid needs with its current options (stencil variant). */
size_t pf_grid_workspace_bytes(const pf_grid *g);

/* Hand the grid its scratch (device, 256-byte aligned, >= pf_grid_workspace_bytes) and run the
 * operator assembly (rows L1, L2 of DESIGN.md): node classes, diagonals, optionally the stored
 * off-diagonals, the deposited fixed-charge right-hand side (reading R2).  With charge model 1 the Laplace solve for
 * phi^L runs here; PF_NOT_CONVERGED is returned (the grid stays usable) when it stopped at PF_OPT_LINEAR_MAXIT. */
int pf_grid_set_workspace(pf_grid *g, void *dev_ptr, size_t bytes);

int pf_grid_set_option(pf_grid *g, int key, double value);

/* Jacobi-BiCGSTAB solve of the grid's operator  -div(eps grad x) + sigma x = rhs  (Table 3).
 *   rhs   : device N; entries at Dirichlet nodes are ignored (the boundary value is used, Q20).
 *   x     : device N; in: initial guess (its Dirichlet nodes are overwritten, Q4), out: solution.
 *           With the Jacobi preconditioner x is written once, at the end of the solve (x = x0 + M^-1 y,
 *           reading D3 of DESIGN.md).
 *   sigma : device N or NULL (zero); added to the diagonal (PF2's -rho' term, Eq (13)).
 *   Stops when ||r||_2 <= tol*||rhs||_2 on the recurrence residual (Q3); tol = 0 runs exactly maxit
 *   iterations and returns PF_NOT_CONVERGED (the fixed-iteration timing mode).
 *   iters_out, relres_out (recurrence), true_relres_out (||b - A x||/||b||): host, may be NULL.
 * Returns PF_OK, PF_NOT_CONVERGED, PF_ERR_BREAKDOWN, PF_ERR_WORKSPACE, PF_ERR_CUDA, PF_ERR_ARG. */
int pf_solve_linear(pf_grid *g, const double *rhs, double *x, const double *sigma,
                    double tol, int maxit,
                    int *iters_out, double *relres_out, double *true_relres_out);

/* The same solve with HOST buffers (pinned or pageable): rhs and x are copied to the device into
 * grid scratch, solved, and x copied back, all on the grid's stream.  sigma stays a device pointer. */
int pf_solve_linear_host(pf_grid *g, const double *rhs_host, double *x_host, const double *sigma,
                         double tol, int maxit,
                         int *iters_out, double *relres_out, double *true_relres_out);

/* Start the upload of the host buffers of a later pf_solve_linear_host(g, rhs_host, x_host, ...) on a copy stream of
 * the grid's own and return at once: the copy then overlaps whatever the grid's stream does in between (assembly of
 * another operator, a pf_solve_pf).  rhs_host, x_host: host (pinned, or the copy is not asynchronous), N doubles; they
 * must stay unchanged until that pf_solve_linear_host, which recognises the pair by its addresses and then waits for
 * the copy instead of uploading again; any other pair of addresses is uploaded as usual.  Needs the workspace. */
int pf_grid_stage_host(pf_grid *g, const double *rhs_host, const double *x_host);

/* Nonlinear PF solve (Table 2 steps 2-5): initial guess from PF2 with rho' = Psi = 0, then
 * { Fermi update at phi0 -> PF1 for Psi -> PF2 for phi -> relax -> test ||phi - phi0||_inf <= tol }.
 *   nions K; valence, bath_conc (mol/L): host, K entries; radii: host, K+1 entries in Angstrom,
 *   water last; all radii 0 switches the steric term off (Q25).  l_c in Angstrom.
 *   phi    : device N, out.
 *   conc   : device (K+1)*N or NULL, out: C_k at the final phi (species-major), 0 outside the solvent.
 *   steric : device N or NULL, out: S^trc at the final phi.
 *   outer_iters_out, linear_iters_out (sum over all linear solves): host, may be NULL.
 * Returns PF_OK, PF_NOT_CONVERGED (outer cap reached), PF_INNER_NOT_CONVERGED, or an error. */
int pf_solve_pf(pf_grid *g, int nions, const double *valence, const double *bath_conc,
                const double *radii, double l_c, double tol,
                double *phi, double *conc, double *steric,
                int *outer_iters_out, int *linear_iters_out);

/* The pointwise part alone (row N1): Eq (1) solved per node (reading R4).
 *   phi: device N, in.  rho, sigma, steric: device N or NULL, out.  conc: device (K+1)*N or NULL. */
int pf_fermi_pointwise(pf_grid *g, int nions, const double *valence, const double *bath_conc,
                       const double *radii, const double *phi,
                       double *rho, double *sigma, double *steric, double *conc);

/* Copy out up to cap entries of the residual history of the last linear solve (PF_OPT_HISTORY):
 * hist[k] = ||r_k||/||b||, k = 0..iters.  Returns the number of entries written, < 0 on error. */
int pf_grid_history(pf_grid *g, double *hist_host, int cap);

/* Per-solve iteration counts of the last pf_solve_pf in call order (initial guess, PF1, PF2, ...). */
int pf_grid_linear_iters(pf_grid *g, int *iters_host, int cap);

/* ||Phi - Phi0||_inf (after relaxation, Table 2 step 5) of every outer iteration of the last pf_solve_pf.
 * Returns the number of entries written (<= cap). */
int pf_grid_increments(pf_grid *g, double *incr_host, int cap);

void pf_grid_destroy(pf_grid *g);
const char *pf_last_error(const pf_grid *g);   /* g may be NULL: last error of pf_grid_create */
const char *pf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* PF_B200_H */
