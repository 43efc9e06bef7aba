// pf_launch.h -- host-side launch interface between the solver driver (pf_api.cu) and the kernel
// translation units.  Internal; the public boundary is include/pf.h.
#pragma once
#include "pf_common.cuh"
#include "pf_krylov.cuh"

namespace pf {

// Kernel launches issued by this library since load (bench.py reports the difference over the timed region).
extern long long g_launch_count;
// First error a kernel launch of this thread returned since the driver last cleared it (pf_api.cu checks it after
// it has enqueued the iterations of a solve, so a failed launch is reported where it happened).
extern thread_local cudaError_t g_launch_error;
inline void note_launch(cudaError_t e) { if (e != cudaSuccess && g_launch_error == cudaSuccess) g_launch_error = e; }

// Launch with programmatic dependent launch allowed: the grid may be scheduled while the preceding kernel of
// the stream drains (its blocks run their prologue on SMs that are already free); the kernel itself calls
// pdl_wait() before it touches anything the preceding kernel wrote.
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(bool pdl, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream,
                              Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl ? 1 : 0;      // off while a CUDA graph is being captured
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

struct LaunchCtx {
    cudaStream_t stream;
    GridDims g;
    Scalars* sc[2];   // device: the two alternating copies of the scalars (pf_common.cuh)
    int* flip;        // host: index of the copy the next kernel reads
    ReduceBuf rb;     // device
    int sm_count;
    int device;       // CUDA device of the grid (per-device kernel attributes)
    int solver;       // 0: Table 3, three kernels per iteration; 1: merged recurrence, two (pf_krylov.cuh)
    int tile_rows;    // tiled family: 0 = chosen per kernel and grid, 13 or 16 = forced (PF_OPT_TILE_ROWS)
    int seg_mode;     // tiled family: -1 = decomposition chosen per grid, 0 = equal chunks, 1 = two groups (PF_OPT_SEGMENTS)
    bool pdl;         // programmatic dependent launch allowed
    // the next kernel reads sc[*flip] and its block 0 writes sc[*flip ^ 1]
    void next_scalars(const Scalars*& in, Scalars*& out) const { in = sc[*flip]; out = sc[*flip ^ 1]; *flip ^= 1; }
    Scalars* current_scalars() const { return sc[*flip]; }
};

// dst (rows of g.nx + 1 doubles) = src (rows of g.nx doubles) with `fill` in the extra column, and back.
void launch_widen(cudaStream_t s, const GridDims& g, const double* src, double* dst, double fill);
void launch_narrow(cudaStream_t s, const GridDims& g, const double* src, double* dst);

// ---- Krylov kernels -----------------------------------------------------------------------
// mode 0: r = b - A x, r~ = r, ||b||, ||r|| (Table 3 step 2); mode 1: ||b - A x||^2 only.
void launch_residual_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, int mode);
void launch_k1_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond);
void launch_k2_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond);
void launch_k3(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond);
// The two kernels of an iteration of the merged solver (pf_krylov.cuh): current (p, v) = (kv.p_in, kv.v_in), current
// r = kv.r; K31 writes kv.r_out, kv.p_out, kv.v_out.
void launch_k2m_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond);
void launch_k31_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond);
// One-block kernel that takes the pending scalar step in place, before the host reads the scalars.
void launch_finalize(const LaunchCtx& c, double* hist);
// The same, and sets the condition of the WHILE node whose body it closes (merged solver, device-side loop).
void launch_finalize_loop(const LaunchCtx& c, double* hist);
// x += M^-1 y at the end of a preconditioned solve (reading D3).
void launch_finish_x(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv);

// Tiled family (pf_krylov_tma.cu): TMA-staged planes, z-marched.  Needs an even nx (16-byte row
// strides; the driver widens an odd-nx box by one column of identity rows, pf_api.cu bicgstab_device) and
// 16-byte aligned vectors; tma_supported() says whether the grid qualifies.
struct TmaSet;                                   // tensor maps of one solve (opaque here)
bool tma_available();                            // driver entry point for tensor-map encoding found
bool tma_supported(const GridDims& g);
bool tma_pointers_ok(const KrylovVecs& kv, const Operator& op);
TmaSet* tma_set_create();
void tma_set_destroy(TmaSet* t);
// (Re)build the tensor maps for the vectors and operator of a solve; false on failure.
bool tma_set_build(TmaSet* t, const GridDims& g, const Operator& op, const KrylovVecs& kv);
void launch_residual_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, int mode,
                         bool precond = false);
void launch_k1_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond,
                   int parity /* which of the two (p, v) buffer pairs is the input */);
void launch_k2_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond,
                   int parity);
// Merged solver, iteration k of a solve (0-based): r lives in buffer k & 1, the current (p, v) pair in buffer (k & 1) ^ 1
// (buffer 0 = the pointers of the KrylovVecs the set was built from, buffer 1 = its r_out, p_out, v_out).
void launch_k2m_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond, int k);
void launch_k31_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond, int k);
// The decomposition the persistent tiled kernels use on a device with sm_count SMs (SegPlan of pf_krylov_tma.cu; host
// arithmetic only): out[9] = mode, x tiles, tiles, chunk / layer depth, items / main blocks, zrest, erest, q, blocks.
void tma_plan(const GridDims& g, int tile_rows, int sm_count, int mode, int* out);
// Whether the tiled family has the merged kernels for this operator (code form; the stored variant uses the direct ones).
bool tma_merged_supported(const Operator& op);
bool tma_merged_ok(const TmaSet* t);             // the set just built holds the maps of the merged kernels

// Cooperative family (pf_krylov_coop.cu): one persistent kernel per solve, one brick of the box per block, the
// brick's vectors in shared memory.  For grids small enough that a brick fits one SM (about <= 72^3) and
// operators in code form.
struct CoopPlan { int nbx, nby, nbz, vmax, hmax, nhmax, threads; size_t smem; };
size_t coop_smem_cap();        // usable dynamic shared memory per block, 0 if cooperative launch is unsupported
bool coop_plan(const GridDims& g, const Operator& op, int max_blocks, size_t smem_cap, CoopPlan* out);
cudaError_t launch_solve_coop(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond,
                              const CoopPlan& plan);

// ---- assembly (pf_assembly.cu) ----------------------------------------------------------------
// Boundary data handed to the assembly and pointwise kernels: the six box faces, and Omega_f (PAPER.md:213,
// 224-226; readings F1-F3): fixv[i] = prescribed potential of node i, NaN where the node is free; null = none.
struct BcDev { int type[6]; double value[6]; const double* fixv; };
__host__ __device__ inline bool is_fixed_node(const BcDev& bc, long long i) {
    return bc.fixv != nullptr && bc.fixv[i] == bc.fixv[i];
}

struct Palette {
    int count;                         // distinct eps values found (PF_MAX_PALETTE+1 = overflow)
    double value[PF_MAX_PALETTE + 1];  // ascending
};

// Scan eps for its distinct values and its range.  scratch: device, >= 256 bytes, zeroed by the call.
cudaError_t scan_eps(cudaStream_t s, long long n, const double* eps, void* scratch, Palette* out,
                     double* eps_min, double* eps_max);

// Poisson operator of Eq (3)/(13) without sigma: diagonal A0, stencil codes (code_mode 0 none, 1 uint16,
// 2 uint32; rows padded to cpitch), optionally A1..A6.
void launch_assemble_poisson(cudaStream_t s, const GridDims& g, double h, const BcDev& bc, const double* eps,
                             const Palette& pal, int code_mode, double* A0, void* code, int cpitch,
                             double* const offd[6] /* entries null unless stored */);
// PF1 operator eps(l_c^2 Lap - 1), sign flipped (Eq (12)), identity rows on the
// box boundary and outside the solvent (Q15).
void launch_assemble_pf1(cudaStream_t s, const GridDims& g, double h, double lc, const BcDev& bc, const double* eps,
                         double eps_mid, bool uniform, const Palette& pal, int code_mode, double* A0, void* code,
                         int cpitch, double* const offd[6]);
// fixv[idx[k]] = val[k] (fixv pre-filled with NaN).
void launch_scatter_fixed(cudaStream_t s, const long long* idx_dev, const double* val_dev, int count, double* fixv);
// Coefficient tables of the on-the-fly variant (host side; PF_CTAB doubles each).
void build_ctab_poisson(const Palette& pal, double h, double* ctab_host);
void build_ctab_pf1(const Palette& pal, double h, double lc, double* ctab_host);

// Trilinear deposition of the fixed charges (reading R2): fixed[i] += kappa q w / h^3, in charge order.
void launch_deposit(cudaStream_t s, const GridDims& g, double h, double kappa, const double* charges_dev, int m,
                    double* fixed);
// x[i] = g_face at Dirichlet nodes (Q4, Q20).
void launch_set_dirichlet(cudaStream_t s, const GridDims& g, const BcDev& bc, double* x);
// b_work = rhs with Dirichlet values forced.
void launch_copy_with_dirichlet(cudaStream_t s, const GridDims& g, const BcDev& bc, const double* src, double* dst);

// ---- singular-charge decomposition (pf_singular.cu), Eqs (5)-(10), readings S1-S5 ----------------------
// Laplace problem for phi^L in Omega_m: diagonal, uint16 stencil codes (table {0, -1/h^2}), right-hand side b
// and start vector x0 (prescribed values on identity rows).
void launch_laplace_m(cudaStream_t s, const GridDims& g, double h, const double* eps, double eps_mid, double eps_m,
                      double kappa, const double* charges_dev, int m, double* A0, void* code, int cpitch, double* b,
                      double* x0);
// phi* on the Omega_m nodes (0 on Omega_s).
void launch_phistar(cudaStream_t s, const GridDims& g, double h, const double* eps, double eps_mid, double eps_m,
                    double kappa, const double* charges_dev, int m, double* out);
// b^IF from the flux jumps of the interface faces (c0, d0 of Eqs (17)-(18)).
void launch_interface_rhs(cudaStream_t s, const GridDims& g, double h, const double* eps, double eps_mid, double eps_m,
                          double kappa, const double* charges_dev, int m, const double* phiL, double* b);
// phi := phi + phi* + phi^L.
void launch_recombine(cudaStream_t s, long long n, const double* phistar, const double* phiL, double* phi);

// ---- pointwise PF kernels (pf_pointwise.cu) ------------------------------------------------
struct SpeciesDev {
    int K;                              // ions; water is index K
    int steric;
    double z[PF_MAX_SPECIES];
    double cb[PF_MAX_SPECIES];          // bath concentration, 1/A^3
    double lam[PF_MAX_SPECIES];         // v_k/v_0
    double lnvc[PF_MAX_SPECIES];        // ln(v_k C_k^B) (unused when v_k = 0)
    double vol[PF_MAX_SPECIES];
    double ln_gammaB, gammaB;
    double kappa;
};

// Row N1: Fermi-like distribution at phi per solvent node; writes whichever outputs are non-null:
// rho, sigma = kappa sum z^2 C, S, conc[(K+1)][N], b1 = PF1 right-hand side (-(kappa rho), 0 on
// identity rows), a2 = a0 + sigma (PF2 diagonal).
void launch_diag_plus_sigma(cudaStream_t s, const GridDims& g, const BcDev& bc, const double* a0, const double* sigma,
                            double* a2);
void launch_fermi(cudaStream_t s, const GridDims& g, const BcDev& bc, const SpeciesDev& sp, const double* eps, double eps_mid,
                  bool uniform, const double* phi, double* rho, double* sigma, double* S, double* conc,
                  double* b1, const double* a0, double* a2,
                  double* S_state = nullptr /* lagged reading (G1): S^trc at hand, N doubles; null = solve Eq (1) per node */,
                  bool lag_update = false /* ... and replace it by ln(max(Gamma_0, 1e-12)/Gamma^B) of these C_k */);
// Row N3 right-hand side: b = [solvent](-(eps psi) + sigma phi0) + fixed, Dirichlet values forced.
void launch_rhs_pf2(cudaStream_t s, const GridDims& g, const BcDev& bc, const double* eps, double eps_mid,
                    bool uniform, const double* psi, const double* sigma, const double* phi0,
                    const double* fixed, double* b);
// Row N5: phi = w phi0 + (1-w) phi; returns max|phi - phi0| through *dmax (device, via ordered-int atomicMax).
void launch_relax(cudaStream_t s, long long n, double w, const double* phi0, double* phi, unsigned long long* dmax_bits);

}  // namespace pf
