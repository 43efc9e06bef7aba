// pf_api.cu -- the C ABI of include/pf.h (+ the introspection calls of include/pf_debug.h) and the host-side solver driver: launch sequencing of the
// three-kernel BiCGSTAB iteration, device-resident scalars, pipelined polling of the device-side
// convergence flag (row L8), and the PF outer loop (rows N1-N5).
#include "../../include/pf.h"
#include "../../include/pf_debug.h"
#include "pf_launch.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

using namespace pf;

namespace pf { void set_create_error(const char* msg); }

long long pf::g_launch_count = 0;
thread_local cudaError_t pf::g_launch_error = cudaSuccess;

namespace {

// Table 1, reading R0: kappa = e^2/(eps_0 k_B T) in Angstrom, phi in k_B T/e.
const double K_BOLTZ = 1.38e-23;       // J/K
const double T_KELVIN = 298.15;        // K
const double E_CHARGE = 1.602e-19;     // C
const double EPS0_F_PER_CM = 8.85e-14; // F/cm
const double MOLAR_TO_PER_A3 = 6.02214076e-4;

double kappa_angstrom() {
    const double eps0_per_m = EPS0_F_PER_CM * 100.0;
    return E_CHARGE * E_CHARGE / (eps0_per_m * K_BOLTZ * T_KELVIN) * 1e10;
}

thread_local std::string g_create_error;

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// The small per-grid buffers (device scalars, reduction partials, coefficient tables, charge list, pinned
// mirrors of the scalars, two events) are recycled through a process-wide free list: cudaMalloc,
// cudaMallocHost and their frees cost milliseconds and synchronise the device, which would dominate the
// creation of a grid (rows L1/L2).  A set is owned by one grid at a time.
struct SmallSet {
    int device = -1;
    char* dev = nullptr;            // one device allocation, carved up below
    size_t charge_cap = 0;          // pf_charge entries the tail of `dev` holds
    char* host = nullptr;           // pinned, 2 x 256 bytes
    cudaEvent_t ev[2] = {nullptr, nullptr};
};
// Iterations per turn of the device-side loop (even: the (p, v) double buffers are back in place).  A turn costs 6-7 us
// (the body drains, the condition is read, the body is launched again), the kernels that return at once after
// the end of the solve 1.5-8 us each: short solves (the inner solves of a PF iteration, 40-100 iterations) want the
// short body, long ones the long body.  The choice follows the previous solve with the same operator.
constexpr int LOOP_BODY_SHORT = 8, LOOP_BODY_LONG = 16, LOOP_LONG_SOLVE = 192;
constexpr long long COOP_AUTO_MAX_N = 64ll * 64 * 64;     // largest grid the cooperative solver is chosen for by itself
                                                          // (measured: 1.1x at 64^3 to 1.7x at 32^3 over the next best family)
constexpr size_t SS_SC = 0 /* two copies, 256 bytes each */, SS_FAULT = 512, SS_DMAX = 768, SS_CTAB0 = 1024,
                 SS_CTAB1 = 1280, SS_PARTIAL = 1536,
                 SS_CHARGES = SS_PARTIAL + sizeof(dd) * 3 * PF_PARTIAL_QUANTITIES * PF_MAX_PARTIAL_BLOCKS;
static_assert(sizeof(Scalars) <= 256, "Scalars slots of the small set");
std::mutex g_pool_mutex;
std::vector<SmallSet*> g_pool;

void small_set_free(SmallSet* s) {
    if (!s) return;
    cudaFree(s->dev);
    if (s->host) cudaFreeHost(s->host);
    if (s->ev[0]) cudaEventDestroy(s->ev[0]);
    if (s->ev[1]) cudaEventDestroy(s->ev[1]);
    delete s;
}

cudaError_t small_set_acquire(int device, size_t ncharges, SmallSet** out) {
    {
        std::lock_guard<std::mutex> lock(g_pool_mutex);
        for (size_t k = 0; k < g_pool.size(); ++k)
            if (g_pool[k]->device == device && g_pool[k]->charge_cap >= ncharges) {
                *out = g_pool[k];
                g_pool.erase(g_pool.begin() + k);
                return cudaSuccess;
            }
    }
    SmallSet* s = new SmallSet();
    s->device = device;
    s->charge_cap = std::max<size_t>(4096, ncharges);
    cudaError_t e = cudaMalloc(&s->dev, SS_CHARGES + sizeof(pf_charge) * s->charge_cap);
    if (e == cudaSuccess) e = cudaMallocHost(&s->host, 512);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev[0], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&s->ev[1], cudaEventDisableTiming);
    if (e != cudaSuccess) { small_set_free(s); return e; }
    *out = s;
    return cudaSuccess;
}

void small_set_release(SmallSet* s) {
    if (!s) return;
    std::lock_guard<std::mutex> lock(g_pool_mutex);
    if (g_pool.size() < 8) g_pool.push_back(s); else small_set_free(s);
}

}  // namespace

struct pf_grid {
    GridDims g;
    double h;
    BcDev bc;
    cudaStream_t stream;
    int sm_count, device;
    const double* eps;
    Palette pal;
    double eps_min, eps_max, eps_mid;
    bool uniform;
    int ncharges;
    SmallSet* small;         // recycled small buffers; the pointers below point into it
    double* charges_dev;
    // options
    // Odd nx: the tiled kernels need an even row length, so the Krylov layer can work on the box widened by one
    // column of identity rows (gk); A0p, bp, xp are the widened copies of the diagonal, right-hand side and iterate
    GridDims gk;
    bool padx;
    double *A0p, *bp, *xp;
    double* offdp[6];          // stored variant: the six off-diagonals in the widened layout
    int coop_state;            // 0 not planned yet, 1 plan valid, -1 not applicable
    CoopPlan coop;
    int opt_stencil, opt_kernels, opt_check, opt_lin_maxit, opt_max_outer, opt_precond, opt_history;
    double opt_omega_pf, opt_lin_tol, opt_water;
    // small owned device buffers
    Scalars* sc[2];          // the two alternating device copies of the scalars
    int flip;                // which one the next kernel reads
    ReduceBuf rb;
    double* ctab_poisson;    // PF_CTAB doubles each
    double* ctab_pf1;
    TmaSet* tma;
    unsigned long long* dmax_bits;
    double* hist;
    int hist_cap;
    Scalars* sc_host[2];     // pinned
    cudaEvent_t ev[2];
    // workspace carve-up
    void* ws;
    size_t ws_bytes;
    bool stored;
    bool assembled;
    double pf1_lc;           // l_c the PF1 operator was assembled for (NaN = none)
    double *r, *r1, *rt, *p0, *p1, *v0, *v1, *t, *y, *bw, *xw;      // r1: second residual buffer of the merged solver
    // host-buffer flavour (pf_solve_linear_host, pf_grid_stage_host): device staging of rhs and x, their own vectors so
    // that an upload can run on the copy stream while other work of the grid (assembly, a PF solve) uses the scratch
    double *hb, *hx;
    double* sstate;          // S^trc state of the lagged reading of Eq (11) (PF_OPT_STERIC_MODE = 1)
    int opt_steric_mode;
    cudaStream_t copy_stream;
    cudaEvent_t staged_ev, main_ev;
    const void *staged_rhs, *staged_x;
    double *A0, *A0_pf1, *A0_s, *fixed, *psi, *phi0, *phiw, *sigma, *bpf;
    void *code, *code_pf1;   // stencil codes of the on-the-fly variant (pf_common.cuh Operator)
    int code_mode;           // 0 none (palette overflow), 1 uint16, 2 uint32
    int cpitch;
    double* offd[6];
    double* offd_pf1[6];
    std::vector<int> lin_iters;
    std::vector<double> increments;      // ||Phi - Phi0||_inf of every outer iteration of the last pf_solve_pf
    // per-kernel timing (PF_OPT_PROFILE): events around k1, k2, k3 of every iteration
    std::vector<cudaEvent_t> prof_ev;
    double prof_ms[3];
    long long prof_launches[3];
    int opt_profile;
    int last_iters;
    // CUDA graphs of one polling chunk of iterations, for grids small enough to be launch-bound
    struct ChunkGraph { const void *a0, *code, *b, *x, *y, *hist; int precond, tiled, chunk; cudaGraphExec_t exec; };
    std::vector<ChunkGraph> graphs;
    std::vector<std::pair<const void*, int>> solve_len;     // iterations of the last solve per operator (by its A0)
    cudaStream_t capture_stream;
    int opt_graph;
    int opt_diag_code;       // k1 forms the Poisson diagonal from the stencil codes (PF_OPT_DIAG_FROM_CODE)
    int opt_norm;            // 0: relative 2-norm (Q3), 1: the paper's absolute maximum norm
    int opt_solver;          // 0: Table 3 (three kernels per iteration), 1: merged recurrence (two; reading M1)
    int opt_tile_rows;       // tiled kernels: 0 auto, 13 or 16 forced
    int opt_seg_mode;        // tiled kernels: -1 auto, 0 equal chunks, 1 two groups (PF_OPT_SEGMENTS)
    int opt_charge_model;    // 0: trilinear deposition (Q22), 1: singular-charge decomposition (Eqs 5-10)
    int charge_model;        // the model the workspace was laid out and assembled for
    double *phiL, *phistar, *A0_L;
    void* code_L;
    double* ctab_L;
    int laplace_iters;
    // Omega_f: nodes with prescribed potential (readings F1-F3); fixv lives in the workspace
    std::vector<long long> fix_idx;
    std::vector<double> fix_val;
    double* fixv;
    int fault_repeats;       // solves repeated by the direct kernels after a division range fault (D4)
    std::vector<const void*> fault_ops;   // operators (by their A0) whose tiled solve faulted: they go straight to the direct family
    std::string err;
};

namespace {

int fail(pf_grid* g, int code, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof(buf), fmt, ap);
    va_end(ap);
    if (g) g->err = buf; else g_create_error = buf;
    return code;
}

#define PF_CUDA(g, call)                                                                          \
    do {                                                                                          \
        cudaError_t e_ = (call);                                                                  \
        if (e_ != cudaSuccess) return fail((g), PF_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_)); \
    } while (0)

int n_vectors(bool stored, int charge_model, bool fixed_nodes, bool padx) {
    return 23 + (stored ? 12 : 0) + (charge_model == 1 ? 3 : 0) + (fixed_nodes ? 1 : 0) + (padx ? 3 + (stored ? 6 : 0) : 0);
}

int code_mode_of(const pf_grid* g) { return g->pal.count > PF_MAX_PALETTE ? 0 : (g->pal.count <= 2 ? 1 : 2); }
int cpitch_of(const pf_grid* g) { return (g->g.nx + 7) & ~7; }
size_t code_bytes_of(const pf_grid* g) {
    const int m = code_mode_of(g);
    return m == 0 ? 0 : align_up((size_t)cpitch_of(g) * g->g.ny * g->g.nz * (m == 1 ? 2 : 4), 256);
}

bool want_stored(const pf_grid* g) {
    if (g->opt_stencil == 1) return true;
    if (g->opt_stencil == 2) return false;
    return g->pal.count > PF_MAX_PALETTE;
}

bool use_tiled(const pf_grid* g, const GridDims& dims) {
    if (g->opt_kernels == 1) return false;
    // auto: below about 40^3 a launch of the one-thread-per-node kernels is shorter than one of the tiled kernels
    // (16.7 against 22.2 us per iteration at 32^3, 49 against 24 at 64^3)
    if (g->opt_kernels == 0 && dims.n < 70000) return false;
    return tma_supported(dims) && tma_available();
}

// The cooperative single-kernel solver: asked for (PF_OPT_KERNELS = 3), or chosen on small grids.
bool use_coop(pf_grid* g, const Operator& op, CoopPlan* plan) {
    if (g->opt_kernels != 3 && g->opt_kernels != 0) return false;
    if (op.stored) return false;
    if (g->coop_state == 0) {
        const size_t cap = coop_smem_cap();
        g->coop_state = (cap > 0 && coop_plan(g->g, op, g->sm_count, cap, &g->coop)) ? 1 : -1;
    }
    if (g->coop_state < 0) return false;
    // auto: small grids only; a per-kernel profile needs the three-kernel families
    if (g->opt_kernels == 0 && (g->opt_profile || g->g.n > COOP_AUTO_MAX_N)) return false;
    *plan = g->coop;
    return true;
}

Operator make_op(const pf_grid* g, int which /*0 poisson, 1 pf1, 2 poisson+sigma, 3 Laplace in Omega_m*/) {
    Operator op;
    std::memset(&op, 0, sizeof(op));
    op.stored = g->stored ? 1 : 0;
    op.code32 = g->code_mode == 2 ? 1 : 0;
    op.cpitch = g->cpitch;
    if (which == 3) {             // always in code form: two coefficient values, 0 and -1/h^2
        op.stored = 0; op.code32 = 0;
        op.A0 = g->A0_L; op.code = g->code_L; op.ctab = g->ctab_L;
    } else if (which == 1) {
        op.A0 = g->A0_pf1; op.code = g->code_pf1; op.ctab = g->ctab_pf1;
        for (int d = 0; d < 6; ++d) op.offd[d] = g->offd_pf1[d];
    } else {
        op.A0 = which == 2 ? g->A0_s : g->A0; op.code = g->code; op.ctab = g->ctab_poisson;
        op.diag_code = (which == 0 && !op.stored && !op.code32) ? g->opt_diag_code : 0;
        for (int d = 0; d < 6; ++d) op.offd[d] = g->offd[d];
    }
    return op;
}

LaunchCtx make_ctx(const pf_grid* g) {
    LaunchCtx c;
    c.stream = g->stream; c.g = g->g; c.sc[0] = g->sc[0]; c.sc[1] = g->sc[1]; c.flip = const_cast<int*>(&g->flip);
    c.rb = g->rb; c.sm_count = g->sm_count; c.device = g->device; c.pdl = true; c.solver = g->opt_solver; c.tile_rows = g->opt_tile_rows;
    c.seg_mode = g->opt_seg_mode;
    return c;
}

// One BiCGSTAB iteration = three launches (rows L4, L5, L6).  kv's (p, v) buffers are swapped on return.
// Merged solver (c.solver = 1): two launches (K2M, K31); the current (p, v) pair is (kv.p_in, kv.v_in), K31 writes the
// other pair and the other r buffer, which become current on return.  The events bracket k1 (nothing), K2M, K31.
void enqueue_iteration(const LaunchCtx& c, const Operator& op, KrylovVecs& kv, const TmaSet* tma, bool tiled,
                       bool precond, int parity, cudaEvent_t* pe) {
    if (c.solver == 1) {
        if (pe) { cudaEventRecord(pe[0], c.stream); cudaEventRecord(pe[1], c.stream); }
        if (tiled) launch_k2m_tma(c, op, kv, tma, precond, parity); else launch_k2m_direct(c, op, kv, precond);
        if (pe) cudaEventRecord(pe[2], c.stream);
        if (tiled) launch_k31_tma(c, op, kv, tma, precond, parity); else launch_k31_direct(c, op, kv, precond);
        if (pe) cudaEventRecord(pe[3], c.stream);
        std::swap(kv.p_in, kv.p_out);
        std::swap(kv.v_in, kv.v_out);
        std::swap(kv.r, kv.r_out);
        return;
    }
    if (pe) cudaEventRecord(pe[0], c.stream);
    if (tiled) launch_k1_tma(c, op, kv, tma, precond, parity); else launch_k1_direct(c, op, kv, precond);
    if (pe) cudaEventRecord(pe[1], c.stream);
    if (tiled) launch_k2_tma(c, op, kv, tma, precond, parity); else launch_k2_direct(c, op, kv, precond);
    if (pe) cudaEventRecord(pe[2], c.stream);
    launch_k3(c, op, kv, precond);
    if (pe) cudaEventRecord(pe[3], c.stream);
    std::swap(kv.p_in, kv.p_out);     // k1 read (p_in, v_in) and wrote (p_out, v_out)
    std::swap(kv.v_in, kv.v_out);
}

// One polling chunk of iterations (an even number, so the (p, v) double buffers are back in place) is captured
// once into a CUDA graph per (operator, vectors, kernel family) and replayed: kernels that follow each other
// inside a graph start 1-2 us apart, stream launches (even programmatic dependent ones) 4 us: 5 % of an
// iteration at 256^3, 7 % at 192^3, 17 % at 128^3.  Returns null when graphs do not apply.
cudaGraphExec_t chunk_graph(pf_grid* g, const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool tiled,
                            bool precond, int chunk) {
    if (!g->opt_graph || (chunk & 1)) return nullptr;
    for (const auto& cg : g->graphs)
        if (cg.a0 == op.A0 && cg.code == op.code && cg.b == kv.b && cg.x == kv.x && cg.y == kv.y && cg.hist == kv.hist &&
            cg.precond == (int)precond && cg.tiled == ((int)tiled | (op.diag_code << 1) | (c.solver ? 8 : 0)) && cg.chunk == chunk)
            return cg.exec;
    if (!g->capture_stream &&
        cudaStreamCreateWithFlags(&g->capture_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); g->opt_graph = 0; return nullptr;
    }
    LaunchCtx cc = c;
    cc.stream = g->capture_stream; cc.pdl = false;     // (programmatic edges in the captured graph: slower, measured)
    KrylovVecs kc = kv;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    const long long launches0 = pf::g_launch_count;
    bool ok = cudaStreamBeginCapture(cc.stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
    if (ok) {
        for (int k = 0; k < chunk; ++k) enqueue_iteration(cc, op, kc, g->tma, tiled, precond, k & 1, nullptr);
        ok = cudaStreamEndCapture(cc.stream, &graph) == cudaSuccess && graph;
    }
    pf::g_launch_count = launches0;            // nothing ran; replays are counted where they are launched
    if (ok) ok = cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    if (!ok) { cudaGetLastError(); g->opt_graph = 0; return nullptr; }
    if (g->graphs.size() >= 16) {              // callers that keep changing x: drop the oldest graph
        cudaGraphExecDestroy(g->graphs.front().exec);
        g->graphs.erase(g->graphs.begin());
    }
    g->graphs.push_back({op.A0, op.code, kv.b, kv.x, kv.y, kv.hist, (int)precond, (int)tiled | (op.diag_code << 1) | (c.solver ? 8 : 0), chunk, exec});
    return exec;
}

// The whole iteration loop on the device: a graph whose only node is a WHILE conditional node with a body of `body`
// iterations (an even number).  The k3 of every iteration, once it has taken the scalar step its predecessor left
// pending, sets the node's condition to "the solve is not over" (begin_kernel<true>, ReduceBuf::more), so the device
// repeats the body until the state says done (converged, maxit, breakdown) and the kernels of at most one more
// body return at once: no host poll, no chunk enqueued ahead.  A loop turn costs 1 us with empty kernels and 6-7 us
// with these (B200, driver 580; profiles/r1_v8_loop.md).  Cached like the chunk graphs (chunk = -body).  Null when it cannot be built.
cudaGraphExec_t loop_graph(pf_grid* g, const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool tiled,
                           bool precond, int body) {
    if (g->opt_graph < 2 || (body & 1) || body < 2) return nullptr;
    for (const auto& cg : g->graphs)
        if (cg.a0 == op.A0 && cg.code == op.code && cg.b == kv.b && cg.x == kv.x && cg.y == kv.y && cg.hist == kv.hist &&
            cg.precond == (int)precond && cg.tiled == ((int)tiled | (op.diag_code << 1) | (c.solver ? 8 : 0)) && cg.chunk == -body)
            return cg.exec;
    if (!g->capture_stream &&
        cudaStreamCreateWithFlags(&g->capture_stream, cudaStreamNonBlocking) != cudaSuccess) {
        cudaGetLastError(); g->opt_graph = 1; return nullptr;
    }
    LaunchCtx cc = c;
    cc.stream = g->capture_stream; cc.pdl = false;
    KrylovVecs kc = kv;
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    const long long launches0 = pf::g_launch_count;
    cudaGraphConditionalHandle more;
    bool ok = cudaGraphCreate(&graph, 0) == cudaSuccess &&
              cudaGraphConditionalHandleCreate(&more, graph, 1, cudaGraphCondAssignDefault) == cudaSuccess;
    if (ok) {
        cudaGraphNodeParams np = {};
        np.type = cudaGraphNodeTypeConditional;
        np.conditional.handle = more;
        np.conditional.type = cudaGraphCondTypeWhile;
        np.conditional.size = 1;
        cudaGraphNode_t node;
        ok = cudaGraphAddNode(&node, graph, nullptr, 0, &np) == cudaSuccess;
        if (ok) ok = cudaStreamBeginCaptureToGraph(cc.stream, np.conditional.phGraph_out[0], nullptr, nullptr, 0,
                                                   cudaStreamCaptureModeThreadLocal) == cudaSuccess;
        if (ok) {
            cc.rb.more = (unsigned long long)more;
            for (int k = 0; k < body; ++k) enqueue_iteration(cc, op, kc, g->tma, tiled, precond, k & 1, nullptr);
            if (cc.solver == 1) launch_finalize_loop(cc, kv.hist);    // takes the pending step, then sets the condition
            cudaGraph_t captured = nullptr;
            ok = cudaStreamEndCapture(cc.stream, &captured) == cudaSuccess;
        }
    }
    pf::g_launch_count = launches0;            // nothing ran; the kernels of a loop are counted after the solve
    if (ok) ok = cudaGraphInstantiate(&exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    if (!ok) { cudaGetLastError(); g->opt_graph = 1; return nullptr; }     // back to polled chunk replays
    if (g->graphs.size() >= 16) {
        cudaGraphExecDestroy(g->graphs.front().exec);
        g->graphs.erase(g->graphs.begin());
    }
    g->graphs.push_back({op.A0, op.code, kv.b, kv.x, kv.y, kv.hist, (int)precond, (int)tiled | (op.diag_code << 1) | (c.solver ? 8 : 0), -body, exec});
    return exec;
}

// Tail of a linear solve: Q3, the true residual of the returned x (row L8) and the outputs.
int finish_solve(pf_grid* g, const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, Scalars fin, bool tiled,
                 int* iters_out, double* relres_out, double* true_relres_out) {
    double* x = kv.x;
    if (!fin.done) { fin.status = PF_NOT_CONVERGED; }
    if (fin.bb == 0.0) PF_CUDA(g, cudaMemsetAsync(x, 0, sizeof(double) * c.g.n, g->stream));   // Q3
    double true_rel = 0.0;
    if (true_relres_out && fin.bb != 0.0) {
        if (tiled) launch_residual_tma(c, op, kv, g->tma, 1); else launch_residual_direct(c, op, kv, 1);
        launch_finalize(c, nullptr);
        PF_CUDA(g, cudaMemcpyAsync(g->sc_host[0], c.current_scalars(), sizeof(Scalars), cudaMemcpyDeviceToHost, g->stream));
        PF_CUDA(g, cudaStreamSynchronize(g->stream));
        true_rel = g->opt_norm == 1 ? g->sc_host[0]->true_rmax : std::sqrt(g->sc_host[0]->true_rr) / fin.bnorm;
    }
    PF_CUDA(g, cudaGetLastError());
    g->last_iters = fin.it;
    if (iters_out) *iters_out = fin.it;
    if (relres_out) *relres_out = fin.bb == 0.0 ? 0.0 : fin.rnorm / fin.bnorm;
    if (true_relres_out) *true_relres_out = true_rel;
    if (fin.status == PF_ERR_BREAKDOWN) return fail(g, PF_ERR_BREAKDOWN, "BiCGSTAB breakdown at iteration %d", fin.it);
    return fin.status;
}


// ---- Table 3 on the device ----------------------------------------------------------------
// b: device, dims.n entries with Dirichlet values already forced; x: device, in/out, Dirichlet values forced.
// dims: the grid's box, or the box widened by one column of identity rows (bicgstab_device below).
int bicgstab_core(pf_grid* g, const GridDims& dims, const Operator& op, const double* b, double* x, double tol, int maxit,
                  int* iters_out, double* relres_out, double* true_relres_out, bool allow_tiled, bool allow_coop) {
    if (maxit < 0) return fail(g, PF_ERR_ARG, "maxit < 0");
    if (!(tol >= 0.0)) return fail(g, PF_ERR_ARG, "tol must be >= 0");
    LaunchCtx c = make_ctx(g);
    c.g = dims;
    pf::g_launch_error = cudaSuccess;
    bool op_faulted = false;      // an earlier tiled solve with this operator left dvd_nb's range (D4)
    for (const void* f : g->fault_ops) op_faulted |= f == op.A0;
    const bool precond = g->opt_precond != 0;
    Scalars init;
    std::memset(&init, 0, sizeof(init));
    init.tol = tol; init.maxit = maxit; init.hist_cap = g->hist ? g->hist_cap : 0; init.norm_mode = g->opt_norm;
    init.solver = g->opt_solver;
    const bool merged = g->opt_solver == 1;
    const int kpi = merged ? 2 : 3;           // kernels per iteration
    // How the iterations reach the GPU (PF_OPT_GRAPH).  The iterations that are bracketed by profiling events are
    // launched one by one (an even number of them); of the others, a device-side loop runs the whole bodies that fit
    // below maxit and the rest follows as stream launches.  Auto: the loop for solves expected to be short (the inner
    // solves of a PF iteration: what counts is what is left behind after convergence), polled graph replays for long
    // ones (what counts is the cost per iteration); the expectation is the previous solve with the same operator.
    const int nprof_all = g->opt_profile ? std::min(maxit & ~1, ((int)(g->prof_ev.size() / 4) + 1) & ~1) : 0;
    int* prev_len = nullptr;
    for (auto& e : g->solve_len) if (e.first == op.A0) prev_len = &e.second;
    if (!prev_len) {
        if (g->solve_len.size() >= 8) g->solve_len.erase(g->solve_len.begin());
        g->solve_len.push_back({op.A0, LOOP_LONG_SOLVE});
        prev_len = &g->solve_len.back().second;
    }
    const bool expect_long = std::min(maxit, *prev_len) >= LOOP_LONG_SOLVE;
    const int LOOP_BODY = expect_long ? LOOP_BODY_LONG : LOOP_BODY_SHORT;
    const int loop_end = nprof_all + (maxit - nprof_all) / LOOP_BODY * LOOP_BODY;
    const bool want_loop = (g->opt_graph == 2 || (g->opt_graph == 3 && !expect_long)) && loop_end > nprof_all;
    init.loop_end = loop_end;
    // pageable source: the runtime stages it before returning, so a stack object is safe
    g->flip = 0;
    PF_CUDA(g, cudaMemcpyAsync(g->sc[0], &init, sizeof(init), cudaMemcpyHostToDevice, g->stream));
    PF_CUDA(g, cudaMemsetAsync(g->rb.fault, 0, sizeof(int), g->stream));
    KrylovVecs kv;
    kv.b = b; kv.x = x; kv.r = g->r; kv.rt = g->rt; kv.t = g->t; kv.hist = g->hist;
    kv.p_in = g->p0; kv.p_out = g->p1; kv.v_in = g->v0; kv.v_out = g->v1;
    kv.r_out = merged ? g->r1 : nullptr;
    // D3: with the Jacobi preconditioner step 16 accumulates y = sum(alpha p + omega s); x = x0 + M^-1 y at the end
    kv.y = precond ? g->y : x;
    if (precond) PF_CUDA(g, cudaMemsetAsync(g->y, 0, sizeof(double) * dims.n, g->stream));
    bool tiled = allow_tiled && !op_faulted && use_tiled(g, dims) && tma_pointers_ok(kv, op);
    if (tiled && !tma_set_build(g->tma, dims, op, kv)) {
        if (g->opt_kernels == 2) return fail(g, PF_ERR_CUDA, "tensor-map encoding failed");
        tiled = false;
    }
    if (tiled && merged && !tma_merged_ok(g->tma)) {
        // the merged kernels of the tiled family exist for operators in code form; stored coefficients use the direct ones
        if (g->opt_kernels == 2) return fail(g, PF_ERR_ARG, "the tiled kernels of the merged solver need the on-the-fly stencil");
        tiled = false;
    }
    if (g->opt_kernels == 2 && allow_tiled && !op_faulted && !tiled)
        return fail(g, PF_ERR_ARG, "the tiled kernels need 16-byte aligned vectors");
    // Small grids: the whole solve in one cooperative kernel (pf_krylov_coop.cu)
    CoopPlan plan;
    const bool coop = allow_tiled && allow_coop && !merged && use_coop(g, op, &plan);
    if (g->opt_kernels == 3 && merged)
        return fail(g, PF_ERR_ARG, "the cooperative kernel implements Table 3 only (PF_OPT_SOLVER = 0)");
    if (g->opt_kernels == 3 && allow_tiled && !coop)
        return fail(g, PF_ERR_ARG, "the cooperative kernel needs an operator in code form and a grid whose bricks "
                                   "fit the shared memory of the SMs (about <= 72^3)");
    bool coop_launched = false;
    if (coop) {
        const int flip0 = g->flip;
        const cudaError_t le = launch_solve_coop(c, op, kv, precond, plan);
        if (le == cudaSuccess) {
            coop_launched = true;
        } else if (g->opt_kernels == 0) {
            // chosen automatically, but the device cannot hold the grid right now (e.g. fewer SMs available to this
            // context than the plan assumed): not an error, the three-kernel families take over for this grid
            cudaGetLastError();
            g->coop_state = -1;
            g->flip = flip0;
        } else {
            return fail(g, PF_ERR_CUDA, "cooperative launch: %s", cudaGetErrorString(le));
        }
    }
    if (coop_launched) {
        Scalars fin;
        PF_CUDA(g, cudaMemcpyAsync(g->sc_host[0], c.current_scalars(), sizeof(Scalars), cudaMemcpyDeviceToHost, g->stream));
        PF_CUDA(g, cudaMemcpyAsync(g->sc_host[1], g->rb.fault, sizeof(int), cudaMemcpyDeviceToHost, g->stream));
        PF_CUDA(g, cudaStreamSynchronize(g->stream));
        if (*reinterpret_cast<const int*>(g->sc_host[1]) != 0)
            return fail(g, PF_ERR_CUDA, "cooperative solve: a grid-wide barrier timed out");
        fin = *g->sc_host[0];
        return finish_solve(g, c, op, kv, fin, false, iters_out, relres_out, true_relres_out);
    }
    if (tiled) launch_residual_tma(c, op, kv, g->tma, 0, precond); else launch_residual_direct(c, op, kv, 0);
    if (merged && maxit > 0) {
        // the merged recurrence starts from v = A M^-1 r0 (and r~.v): the ordinary k1 with p = r (first = 1)
        if (tiled) launch_k1_tma(c, op, kv, g->tma, precond, 0); else launch_k1_direct(c, op, kv, precond);
        std::swap(kv.p_in, kv.p_out);
        std::swap(kv.v_in, kv.v_out);
    }

    const int chunk = g->opt_check < 1 ? 1 : g->opt_check;
    int launched = 0, slot = 0;
    bool pending[2] = {false, false};
    bool done = false;
    Scalars fin;
    std::memset(&fin, 0, sizeof(fin));
    // Pipelined polling: enqueue chunk k+1 before waiting for the flag copy of chunk k, so the GPU
    // never idles on the host; kernels launched after convergence return at once (sc->done).
    cudaGraphExec_t loop = want_loop ? loop_graph(g, c, op, kv, tiled, precond, LOOP_BODY) : nullptr;
    if (loop) {
        for (int k = 0; k < nprof_all; ++k) {
            const bool prof = (size_t)(4 * k + 3) < g->prof_ev.size();
            enqueue_iteration(c, op, kv, g->tma, tiled, precond, k & 1, prof ? &g->prof_ev[4 * k] : nullptr);
        }
        PF_CUDA(g, cudaGraphLaunch(loop, g->stream));
        for (int k = loop_end; k < maxit; ++k)      // fewer than a body; they return at once if the solve is over
            enqueue_iteration(c, op, kv, g->tma, tiled, precond, k & 1, nullptr);
        launch_finalize(c, kv.hist);          // the scalar step the last kernel left pending
        PF_CUDA(g, cudaMemcpyAsync(g->sc_host[0], c.current_scalars(), sizeof(Scalars), cudaMemcpyDeviceToHost, g->stream));
        PF_CUDA(g, cudaStreamSynchronize(g->stream));
        fin = *g->sc_host[0];
        // kernels the loop ran: whole bodies of 3 per iteration, up to loop_end; if the solve ended before that, the
        // body in which its last iteration ran is the last one unless that iteration was the body's last (its k3's
        // step is then taken by the next body's first kernel)
        // (merged solver: a body ends with the finalize that sets the condition, so the state is exact: the body in
        // which the last iteration ran is the last one)
        const int bodies = fin.it >= loop_end ? (loop_end - nprof_all) / LOOP_BODY
                         : (merged ? std::max((std::max(fin.it - nprof_all, 0) + LOOP_BODY - 1) / LOOP_BODY, 1)
                                   : std::max(fin.it - nprof_all, 0) / LOOP_BODY + 1);
        pf::g_launch_count += ((long long)kpi * LOOP_BODY + (merged ? 1 : 0)) * bodies;
        done = true;
    }
    while (!done) {
        int todo = std::min(chunk, maxit - launched);
        // iterations that are bracketed by profiling events are launched one by one (an even number of them, so
        // that graph replays start with the buffers in place), the others as a graph
        const int nprof = g->opt_profile ? (((int)(g->prof_ev.size() / 4) + 1) & ~1) : 0;
        const bool profiled = launched < nprof;
        if (profiled) todo = std::min(todo, nprof - launched);
        cudaGraphExec_t exec = (todo == chunk && !profiled) ? chunk_graph(g, c, op, kv, tiled, precond, chunk) : nullptr;
        if (exec) {
            PF_CUDA(g, cudaGraphLaunch(exec, g->stream));
            pf::g_launch_count += (long long)kpi * chunk;
        } else {
            for (int k = 0; k < todo; ++k) {
                const bool prof = g->opt_profile && (size_t)(4 * (launched + k) + 3) < g->prof_ev.size();
                enqueue_iteration(c, op, kv, g->tma, tiled, precond, (launched + k) & 1,
                                  prof ? &g->prof_ev[4 * (launched + k)] : nullptr);
            }
        }
        launched += todo;
        launch_finalize(c, kv.hist);          // the scalar step the last kernel left pending
        PF_CUDA(g, cudaMemcpyAsync(g->sc_host[slot], c.current_scalars(), sizeof(Scalars), cudaMemcpyDeviceToHost,
                                   g->stream));
        PF_CUDA(g, cudaEventRecord(g->ev[slot], g->stream));
        pending[slot] = true;
        const int other = slot ^ 1;
        if (pending[other]) {
            PF_CUDA(g, cudaEventSynchronize(g->ev[other]));
            pending[other] = false;
            if (g->sc_host[other]->done) { fin = *g->sc_host[other]; done = true; }
        }
        if (!done && (launched >= maxit || todo == 0)) {
            PF_CUDA(g, cudaEventSynchronize(g->ev[slot]));
            pending[slot] = false;
            fin = *g->sc_host[slot];
            done = true;
        }
        slot ^= 1;
    }
    *prev_len = fin.it;
    if (pf::g_launch_error != cudaSuccess) {
        const cudaError_t le = pf::g_launch_error;
        pf::g_launch_error = cudaSuccess;
        cudaGetLastError();
        return fail(g, PF_ERR_CUDA, "kernel launch: %s", cudaGetErrorString(le));
    }
    if (tiled && fin.fault) {
        // operands outside the range of the tiled kernels' branch-free division (pf_common.cuh dvd_nb): x has
        // not been touched yet (D3), so the solve is simply repeated with the kernels that use __ddiv_rn
        PF_CUDA(g, cudaStreamSynchronize(g->stream));
        ++g->fault_repeats;
        if (g->fault_ops.size() < 16) g->fault_ops.push_back(op.A0);    // later solves with it skip the tiled family
        return bicgstab_core(g, dims, op, b, x, tol, maxit, iters_out, relres_out, true_relres_out, false, false);
    }
    if (precond) launch_finish_x(c, op, kv);
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    if (g->opt_profile) {       // only iterations that ran (kernels after convergence return at once)
        const int nprof = std::min<int>(fin.it, (int)g->prof_ev.size() / 4);
        for (int k = 0; k < nprof; ++k)
            for (int j = 0; j < 3; ++j) {
                float ms = 0.f;
                if (cudaEventElapsedTime(&ms, g->prof_ev[4 * k + j], g->prof_ev[4 * k + j + 1]) == cudaSuccess) {
                    g->prof_ms[j] += ms; g->prof_launches[j] += 1;
                }
            }
    }
    return finish_solve(g, c, op, kv, fin, tiled, iters_out, relres_out, true_relres_out);
}

// A linear solve of the grid.  Odd nx (rows of an odd number of doubles cannot be described to the TMA unit, whose
// strides are multiples of 16 bytes): where the tiled kernels would otherwise apply, the system is embedded in the
// box widened by one column x = nx of identity rows (diagonal 1, stencil code 0, b = x = 0): the extra unknowns are
// decoupled and exactly 0 in every vector, so they add exact zeros to the inner products and the iterates of the
// real unknowns keep their bits.  Costs eight vector passes per solve (about half an iteration; twelve more with
// stored coefficients).
int bicgstab_device(pf_grid* g, const Operator& op, const double* b, double* x, double tol, int maxit,
                    int* iters_out, double* relres_out, double* true_relres_out) {
    CoopPlan plan;
    const bool widen = g->padx && (!op.stored || g->offdp[0]) && g->opt_kernels != 1 && g->opt_kernels != 3 &&
                       use_tiled(g, g->gk) && (g->opt_solver == 1 || !use_coop(g, op, &plan));
    if (!widen)
        return bicgstab_core(g, g->g, op, b, x, tol, maxit, iters_out, relres_out, true_relres_out, true, true);
    launch_widen(g->stream, g->g, op.A0, g->A0p, 1.0);
    launch_widen(g->stream, g->g, b, g->bp, 0.0);
    launch_widen(g->stream, g->g, x, g->xp, 0.0);
    Operator opk = op;
    opk.A0 = g->A0p;
    if (op.stored)
        for (int d = 0; d < 6; ++d) { launch_widen(g->stream, g->g, op.offd[d], g->offdp[d], 0.0); opk.offd[d] = g->offdp[d]; }
    const int rc = bicgstab_core(g, g->gk, opk, g->bp, g->xp, tol, maxit, iters_out, relres_out, true_relres_out, true, false);
    if (rc == PF_ERR_CUDA || rc == PF_ERR_ARG) return rc;
    launch_narrow(g->stream, g->g, g->xp, x);
    PF_CUDA(g, cudaGetLastError());
    return rc;
}

int check_ready(pf_grid* g) {
    if (!g) return PF_ERR_ARG;
    if (!g->ws || !g->assembled) return fail(g, PF_ERR_WORKSPACE, "workspace not set (pf_grid_set_workspace)");
    return PF_OK;
}

// Species table of Eq (1): v_k = 4 pi a_k^3/3, v_0 = mean volume, lam_k = v_k/v_0,
// Gamma^B = 1 - sum v_k C_k^B; Q25 (all radii 0 => steric off), Q26 (neutral bath).
int make_species(pf_grid* g, int K, const double* valence, const double* bath, const double* radii, SpeciesDev* sp) {
    if (K < 0 || K + 1 > PF_MAX_SPECIES) return fail(g, PF_ERR_ARG, "nions must be in 0..%d", PF_MAX_SPECIES - 1);
    if ((K > 0 && (!valence || !bath)) || !radii) return fail(g, PF_ERR_ARG, "null species table");
    std::memset(sp, 0, sizeof(*sp));
    sp->K = K;
    sp->kappa = kappa_angstrom();
    double vsum = 0.0;
    for (int k = 0; k <= K; ++k) {
        sp->z[k] = k < K ? valence[k] : 0.0;
        sp->cb[k] = (k < K ? bath[k] : g->opt_water) * MOLAR_TO_PER_A3;
        sp->vol[k] = 4.0 * M_PI * radii[k] * radii[k] * radii[k] / 3.0;
        vsum += sp->vol[k];
    }
    const double v0 = vsum / (K + 1);
    sp->steric = vsum > 0.0 ? 1 : 0;
    double occ = 0.0;
    for (int k = 0; k <= K; ++k) {
        sp->lam[k] = sp->steric ? sp->vol[k] / v0 : 0.0;
        occ += sp->vol[k] * sp->cb[k];
        sp->lnvc[k] = sp->vol[k] > 0.0 ? std::log(sp->vol[k] * sp->cb[k]) : 0.0;
    }
    const double gammaB = 1.0 - occ;
    if (!(gammaB > 0.0)) return fail(g, PF_ERR_NONPHYSICAL, "Gamma^B = %g <= 0", gammaB);
    sp->ln_gammaB = std::log(gammaB);
    sp->gammaB = gammaB;
    double net = 0.0, tot = 0.0;
    for (int k = 0; k < K; ++k) { net += sp->z[k] * sp->cb[k]; tot += std::fabs(sp->z[k]) * sp->cb[k]; }
    if (std::fabs(net) > 1e-12 * tot) return fail(g, PF_ERR_NONPHYSICAL, "bath is not neutral");
    return PF_OK;
}

}  // namespace

// the message pf_last_error(NULL) returns, for entry points that take no grid (pf_noalloc.cu)
void pf::set_create_error(const char* msg) { g_create_error = msg ? msg : ""; }

// =========================================================================================
// C ABI
// =========================================================================================
extern "C" {

const char* pf_version(void) { return "pf_b200 0.1 (sm_100a)"; }

const char* pf_last_error(const pf_grid* g) { return g ? g->err.c_str() : g_create_error.c_str(); }

int pf_grid_create(pf_grid** out, int nx, int ny, int nz, double h, const double* eps_map,
                   const pf_charge* charges, int ncharges, const pf_bc* bc, void* cuda_stream) {
    if (!out) return fail(nullptr, PF_ERR_ARG, "out is NULL");
    *out = nullptr;
    if (nx < 3 || ny < 3 || nz < 3) return fail(nullptr, PF_ERR_ARG, "grid needs >= 3 nodes per direction");
    if (!(h > 0.0)) return fail(nullptr, PF_ERR_ARG, "h must be > 0");
    if (!eps_map || !bc) return fail(nullptr, PF_ERR_ARG, "eps_map and bc must not be NULL");
    if (ncharges < 0 || (ncharges > 0 && !charges)) return fail(nullptr, PF_ERR_ARG, "bad charge list");
    for (int f = 0; f < 6; ++f)
        if (bc->type[f] != PF_BC_DIRICHLET && bc->type[f] != PF_BC_NEUMANN)
            return fail(nullptr, PF_ERR_ARG, "bc type of face %d is %d", f, bc->type[f]);
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        return fail(nullptr, PF_ERR_CUDA, "no CUDA device: this library has no CPU fallback");
    }
    pf_grid* g = new pf_grid();
    g->g.nx = nx; g->g.ny = ny; g->g.nz = nz; g->g.n = (long long)nx * ny * nz;
    g->gk = g->g; g->padx = (nx & 1) != 0; g->A0p = g->bp = g->xp = nullptr;
    for (int d = 0; d < 6; ++d) g->offdp[d] = nullptr;
    if (g->padx) { g->gk.nx = nx + 1; g->gk.n = (long long)(nx + 1) * ny * nz; }
    g->h = h;
    for (int f = 0; f < 6; ++f) { g->bc.type[f] = bc->type[f]; g->bc.value[f] = bc->value[f]; }
    g->stream = (cudaStream_t)cuda_stream;
    g->eps = eps_map;
    g->ncharges = ncharges;
    g->coop_state = 0;
    g->opt_stencil = 0; g->opt_kernels = 0; g->opt_check = 16; g->opt_lin_maxit = 10000; g->opt_max_outer = 1000;
    g->opt_precond = 1; g->opt_history = 0;
    g->opt_omega_pf = 0.3; g->opt_lin_tol = 1e-10; g->opt_water = 55.5;
    g->ws = nullptr; g->ws_bytes = 0; g->assembled = false; g->stored = false;
    g->pf1_lc = std::nan("");
    g->opt_profile = 0; g->prof_ms[0] = g->prof_ms[1] = g->prof_ms[2] = 0.0;
    g->prof_launches[0] = g->prof_launches[1] = g->prof_launches[2] = 0;
    g->hist = nullptr; g->hist_cap = 0; g->last_iters = 0; g->fault_repeats = 0;
    g->hb = g->hx = g->sstate = nullptr; g->opt_steric_mode = 0; g->copy_stream = nullptr; g->staged_ev = g->main_ev = nullptr;
    g->staged_rhs = g->staged_x = nullptr;
    g->capture_stream = nullptr; g->opt_graph = 3; g->opt_diag_code = 1; g->opt_norm = 0; g->opt_solver = 0; g->opt_tile_rows = 0; g->opt_seg_mode = -1;
    g->opt_charge_model = 0; g->charge_model = 0; g->phiL = g->phistar = g->A0_L = nullptr; g->code_L = nullptr;
    g->ctab_L = nullptr; g->laplace_iters = 0; g->fixv = nullptr; g->bc.fixv = nullptr;
    g->small = nullptr;
    g->charges_dev = nullptr; g->sc[0] = g->sc[1] = nullptr; g->flip = 0; g->rb.partial = nullptr; g->rb.fault = nullptr; g->rb.more = 0;
    g->ctab_poisson = g->ctab_pf1 = nullptr; g->dmax_bits = nullptr; g->tma = nullptr;
    g->code = g->code_pf1 = nullptr; g->code_mode = 0; g->cpitch = 0;
    g->sc_host[0] = g->sc_host[1] = nullptr; g->ev[0] = g->ev[1] = nullptr;
#define PF_CREATE_CUDA(call)                                                                         \
    do {                                                                                             \
        cudaError_t e_ = (call);                                                                     \
        if (e_ != cudaSuccess) {                                                                     \
            int rc_ = fail(nullptr, PF_ERR_CUDA, "%s: %s", #call, cudaGetErrorString(e_));           \
            pf_grid_destroy(g);                                                                      \
            return rc_;                                                                              \
        }                                                                                            \
    } while (0)
    PF_CREATE_CUDA(cudaGetDevice(&dev));
    g->device = dev;
    PF_CREATE_CUDA(cudaDeviceGetAttribute(&g->sm_count, cudaDevAttrMultiProcessorCount, dev));
    PF_CREATE_CUDA(small_set_acquire(dev, (size_t)ncharges, &g->small));
    g->sc[0] = reinterpret_cast<Scalars*>(g->small->dev + SS_SC);
    g->sc[1] = reinterpret_cast<Scalars*>(g->small->dev + SS_SC + 256);
    g->rb.fault = reinterpret_cast<int*>(g->small->dev + SS_FAULT);
    g->dmax_bits = reinterpret_cast<unsigned long long*>(g->small->dev + SS_DMAX);
    g->ctab_poisson = reinterpret_cast<double*>(g->small->dev + SS_CTAB0);
    g->ctab_pf1 = reinterpret_cast<double*>(g->small->dev + SS_CTAB1);
    g->ctab_L = reinterpret_cast<double*>(g->small->dev + SS_CTAB1 + 128);
    g->rb.partial = reinterpret_cast<dd*>(g->small->dev + SS_PARTIAL);
    g->sc_host[0] = reinterpret_cast<Scalars*>(g->small->host);
    g->sc_host[1] = reinterpret_cast<Scalars*>(g->small->host + 256);
    g->ev[0] = g->small->ev[0]; g->ev[1] = g->small->ev[1];
    PF_CREATE_CUDA(cudaMemsetAsync(g->rb.fault, 0, 256, g->stream));
    g->tma = tma_set_create();
    if (ncharges > 0) {
        g->charges_dev = reinterpret_cast<double*>(g->small->dev + SS_CHARGES);
        PF_CREATE_CUDA(cudaMemcpyAsync(g->charges_dev, charges, sizeof(pf_charge) * ncharges, cudaMemcpyHostToDevice,
                                       g->stream));
    }
    PF_CREATE_CUDA(scan_eps(g->stream, g->g.n, eps_map, g->dmax_bits, &g->pal, &g->eps_min, &g->eps_max));
#undef PF_CREATE_CUDA
    // (the scan orders bit patterns: a negative entry shows up as a 'maximum' below the minimum)
    if (!(g->eps_min > 0.0) || !std::isfinite(g->eps_max) || !(g->eps_max >= g->eps_min)) {
        int rc = fail(nullptr, PF_ERR_ARG, "eps_map must be finite and > 0 (range %g..%g)", g->eps_min, g->eps_max);
        pf_grid_destroy(g);
        return rc;
    }
    g->uniform = g->eps_min == g->eps_max;
    g->eps_mid = 0.5 * (g->eps_min + g->eps_max);     // Q17
    *out = g;
    return PF_OK;
}

void pf_grid_destroy(pf_grid* g) {
    if (!g) return;
    cudaStreamSynchronize(g->stream);
    small_set_release(g->small);
    for (auto& cg : g->graphs) cudaGraphExecDestroy(cg.exec);
    if (g->capture_stream) cudaStreamDestroy(g->capture_stream);
    if (g->copy_stream) { cudaStreamSynchronize(g->copy_stream); cudaStreamDestroy(g->copy_stream); }
    if (g->staged_ev) cudaEventDestroy(g->staged_ev);
    if (g->main_ev) cudaEventDestroy(g->main_ev);
    cudaFree(g->hist);
    if (g->tma) tma_set_destroy(g->tma);
    for (cudaEvent_t e : g->prof_ev) cudaEventDestroy(e);
    cudaGetLastError();
    delete g;
}

size_t pf_grid_workspace_bytes(const pf_grid* g) {
    if (!g) return 0;
    const size_t vec = align_up(sizeof(double) * (size_t)g->gk.n, 256);
    const size_t code_l = g->opt_charge_model == 1 ? align_up((size_t)cpitch_of(g) * g->g.ny * g->g.nz * 2, 256) : 0;
    return (size_t)n_vectors(want_stored(g), g->opt_charge_model, !g->fix_idx.empty(), g->padx) * vec + 2 * code_bytes_of(g) + code_l;
}

int pf_grid_set_option(pf_grid* g, int key, double value) {
    if (!g) return PF_ERR_ARG;
    const int iv = (int)std::llround(value);
    switch (key) {
        case PF_OPT_STENCIL:
            if (iv < 0 || iv > 2) return fail(g, PF_ERR_ARG, "stencil must be 0, 1 or 2");
            if (iv == 2 && g->pal.count > PF_MAX_PALETTE)
                return fail(g, PF_ERR_ARG, "on-the-fly stencil needs <= %d distinct eps values", PF_MAX_PALETTE);
            if (g->assembled && (iv == 1) != g->stored && iv != 0)
                return fail(g, PF_ERR_ARG, "set the stencil variant before pf_grid_set_workspace");
            g->opt_stencil = iv;
            return PF_OK;
        case PF_OPT_OMEGA_PF:
            if (!(value >= 0.0 && value < 1.0)) return fail(g, PF_ERR_ARG, "omega_PF must be in [0,1)");
            g->opt_omega_pf = value; return PF_OK;
        case PF_OPT_LINEAR_TOL:
            if (!(value >= 0.0)) return fail(g, PF_ERR_ARG, "tolerance must be >= 0");
            g->opt_lin_tol = value; return PF_OK;
        case PF_OPT_LINEAR_MAXIT:
            if (iv < 0) return fail(g, PF_ERR_ARG, "maxit must be >= 0");
            g->opt_lin_maxit = iv; return PF_OK;
        case PF_OPT_CHECK_INTERVAL:
            if (iv < 1) return fail(g, PF_ERR_ARG, "check interval must be >= 1");
            g->opt_check = iv; return PF_OK;
        case PF_OPT_WATER_MOLAR:
            if (!(value >= 0.0)) return fail(g, PF_ERR_ARG, "water concentration must be >= 0");
            g->opt_water = value; return PF_OK;
        case PF_OPT_MAX_OUTER:
            if (iv < 1) return fail(g, PF_ERR_ARG, "max outer iterations must be >= 1");
            g->opt_max_outer = iv; return PF_OK;
        case PF_OPT_PRECOND:
            g->opt_precond = iv != 0; return PF_OK;
        case PF_OPT_HISTORY: {
            if (iv < 0) return fail(g, PF_ERR_ARG, "history length must be >= 0");
            cudaStreamSynchronize(g->stream);
            cudaFree(g->hist); g->hist = nullptr; g->hist_cap = 0;
            if (iv > 0) {
                PF_CUDA(g, cudaMalloc(&g->hist, sizeof(double) * (size_t)iv));
                g->hist_cap = iv;
            }
            g->opt_history = iv;
            return PF_OK;
        }
        case PF_OPT_PROFILE: {
            if (iv < 0 || iv > 100000) return fail(g, PF_ERR_ARG, "profile: iterations to time must be in 0..100000");
            cudaStreamSynchronize(g->stream);
            for (cudaEvent_t e : g->prof_ev) cudaEventDestroy(e);
            g->prof_ev.clear();
            for (int k = 0; k < 4 * iv; ++k) {
                cudaEvent_t e;
                PF_CUDA(g, cudaEventCreate(&e));
                g->prof_ev.push_back(e);
            }
            g->opt_profile = iv;
            for (int j = 0; j < 3; ++j) { g->prof_ms[j] = 0.0; g->prof_launches[j] = 0; }
            return PF_OK;
        }
        case PF_OPT_NORM:
            if (iv != 0 && iv != 1) return fail(g, PF_ERR_ARG, "norm must be 0 or 1");
            g->opt_norm = iv; return PF_OK;
        case PF_OPT_CHARGE_MODEL:
            if (iv != 0 && iv != 1) return fail(g, PF_ERR_ARG, "charge model must be 0 or 1");
            if (g->assembled && iv != g->charge_model)
                return fail(g, PF_ERR_ARG, "set the charge model before pf_grid_set_workspace");
            g->opt_charge_model = iv; return PF_OK;
        case PF_OPT_DIAG_FROM_CODE:
            if (iv < 0 || iv > 2) return fail(g, PF_ERR_ARG, "diag-from-code must be 0, 1 (k1) or 2 (k1 and k2)");
            g->opt_diag_code = iv; return PF_OK;
        case PF_OPT_TILE_ROWS:
            if (iv != 0 && iv != 13 && iv != 16) return fail(g, PF_ERR_ARG, "tile rows must be 0 (auto), 13 or 16");
            if (iv != g->opt_tile_rows) {          // cached graphs hold kernels of the other geometry
                cudaStreamSynchronize(g->stream);
                for (auto& cg : g->graphs) cudaGraphExecDestroy(cg.exec);
                g->graphs.clear();
            }
            g->opt_tile_rows = iv; return PF_OK;
        case PF_OPT_SEGMENTS:
            if (iv < -1 || iv > 2) return fail(g, PF_ERR_ARG, "segments must be -1 (auto), 0 (equal chunks), 1 (layers + rest) or 2 (two layers + pieces)");
            if (iv != g->opt_seg_mode) {           // cached graphs hold launches of the other decomposition
                cudaStreamSynchronize(g->stream);
                for (auto& cg : g->graphs) cudaGraphExecDestroy(cg.exec);
                g->graphs.clear();
            }
            g->opt_seg_mode = iv; return PF_OK;
        case PF_OPT_STERIC_MODE:
            if (iv != 0 && iv != 1) return fail(g, PF_ERR_ARG, "steric mode must be 0 (simultaneous) or 1 (lagged)");
            g->opt_steric_mode = iv; return PF_OK;
        case PF_OPT_SOLVER:
            if (iv != 0 && iv != 1) return fail(g, PF_ERR_ARG, "solver must be 0 (Table 3) or 1 (merged)");
            g->opt_solver = iv; return PF_OK;
        case PF_OPT_GRAPH:
            if (iv < 0 || iv > 3) return fail(g, PF_ERR_ARG, "graph must be 0, 1, 2 or 3");
            g->opt_graph = iv; return PF_OK;
        case PF_OPT_KERNELS:
            if (iv < 0 || iv > 3) return fail(g, PF_ERR_ARG, "kernels must be 0, 1, 2 or 3");
            if (iv == 2 && !(tma_supported(g->gk) && tma_available()))
                return fail(g, PF_ERR_ARG, "the tiled kernels need nx >= 32, ny >= 16, nz >= 8");
            g->opt_kernels = iv; return PF_OK;
        default:
            return fail(g, PF_ERR_ARG, "unknown option key %d", key);
    }
}

int pf_grid_set_workspace(pf_grid* g, void* dev_ptr, size_t bytes) {
    if (!g) return PF_ERR_ARG;
    if (!dev_ptr) return fail(g, PF_ERR_ARG, "workspace pointer is NULL");
    if (((uintptr_t)dev_ptr & 255u) != 0) return fail(g, PF_ERR_ARG, "workspace must be 256-byte aligned");
    const size_t need = pf_grid_workspace_bytes(g);
    if (bytes < need) return fail(g, PF_ERR_WORKSPACE, "workspace has %zu bytes, %zu needed", bytes, need);
    g->stored = want_stored(g);
    g->ws = dev_ptr; g->ws_bytes = bytes;
    bool laplace_maxit = false;
    // everything that was derived from an earlier workspace: cached graphs (they bake in the vector, scalar and
    // partial-sum pointers and the tensor maps), expected solve lengths, the cooperative plan, faulted operators
    cudaStreamSynchronize(g->stream);
    for (auto& cg : g->graphs) cudaGraphExecDestroy(cg.exec);
    g->graphs.clear();
    g->solve_len.clear();
    g->fault_ops.clear();
    g->coop_state = 0;
    const size_t vec = align_up(sizeof(double) * (size_t)g->gk.n, 256);     // every vector has room for the widened box
    char* base = (char*)dev_ptr;
    auto take = [&]() { double* p = (double*)base; base += vec; return p; };
    g->r = take(); g->r1 = take(); g->rt = take(); g->p0 = take(); g->p1 = take(); g->v0 = take(); g->v1 = take();
    g->t = take(); g->y = take(); g->bw = take(); g->xw = take(); g->hb = take(); g->hx = take(); g->sstate = take();
    g->staged_rhs = g->staged_x = nullptr;
    g->A0 = take(); g->A0_pf1 = take(); g->A0_s = take(); g->fixed = take(); g->psi = take();
    g->phi0 = take(); g->phiw = take(); g->sigma = take(); g->bpf = take();
    g->charge_model = g->opt_charge_model;
    if (g->charge_model == 1) { g->phiL = take(); g->phistar = take(); g->A0_L = take(); }
    g->fixv = g->fix_idx.empty() ? nullptr : take();
    if (g->padx) { g->A0p = take(); g->bp = take(); g->xp = take(); }
    for (int d = 0; d < 6; ++d) g->offdp[d] = (g->padx && g->stored) ? take() : nullptr;
    for (int d = 0; d < 6; ++d) { g->offd[d] = g->stored ? take() : nullptr; }
    for (int d = 0; d < 6; ++d) { g->offd_pf1[d] = g->stored ? take() : nullptr; }
    g->code_mode = code_mode_of(g);
    g->cpitch = cpitch_of(g);
    const size_t cb = code_bytes_of(g);
    g->code = cb ? (void*)base : nullptr; base += cb;
    g->code_pf1 = cb ? (void*)base : nullptr; base += cb;
    if (g->charge_model == 1) { g->code_L = (void*)base; base += align_up((size_t)g->cpitch * g->g.ny * g->g.nz * 2, 256); }
    g->bc.fixv = g->fixv;
    if (g->fixv) {            // Omega_f: NaN = free node, then the prescribed values (r, r~ serve as staging)
        const int cnt = (int)g->fix_idx.size();
        PF_CUDA(g, cudaMemsetAsync(g->fixv, 0xFF, sizeof(double) * (size_t)g->g.n, g->stream));
        PF_CUDA(g, cudaMemcpyAsync(g->rt, g->fix_idx.data(), sizeof(long long) * cnt, cudaMemcpyHostToDevice, g->stream));
        PF_CUDA(g, cudaMemcpyAsync(g->r, g->fix_val.data(), sizeof(double) * cnt, cudaMemcpyHostToDevice, g->stream));
        launch_scatter_fixed(g->stream, reinterpret_cast<const long long*>(g->rt), g->r, cnt, g->fixv);
    }
    // rows L1, L2: Poisson operator, coefficient table, fixed charges
    if (cb) PF_CUDA(g, cudaMemsetAsync(g->code, 0, 2 * cb, g->stream));    // padding columns of the code rows
    launch_assemble_poisson(g->stream, g->g, g->h, g->bc, g->eps, g->pal, g->code_mode, g->A0, g->code, g->cpitch,
                            g->offd);
    if (g->code_mode) {
        double ctab[PF_CTAB];
        build_ctab_poisson(g->pal, g->h, ctab);
        PF_CUDA(g, cudaMemcpyAsync(g->ctab_poisson, ctab, sizeof(ctab), cudaMemcpyHostToDevice, g->stream));
    }
    if (g->charge_model == 0) {
        launch_deposit(g->stream, g->g, g->h, kappa_angstrom(), g->charges_dev, g->ncharges, g->fixed);
    } else {
        // Table 2 step 1 / Table 4 steps 2-3: phi^L by the Krylov core, then the interface vector b^IF (in `fixed`)
        if (g->uniform) return fail(g, PF_ERR_ARG, "the singular-charge model needs a map with a low-eps region (Omega_m)");
        const double kap = kappa_angstrom();
        double ctab[PF_CTAB] = {0.0};
        ctab[1] = -(1.0 / (g->h * g->h));
        PF_CUDA(g, cudaMemcpyAsync(g->ctab_L, ctab, sizeof(ctab), cudaMemcpyHostToDevice, g->stream));
        PF_CUDA(g, cudaMemsetAsync(g->code_L, 0, align_up((size_t)g->cpitch * g->g.ny * g->g.nz * 2, 256), g->stream));
        PF_CUDA(g, cudaMemsetAsync(g->p0, 0, vec * 4, g->stream));
        launch_laplace_m(g->stream, g->g, g->h, g->eps, g->eps_mid, g->eps_min, kap, g->charges_dev, g->ncharges, g->A0_L,
                         g->code_L, g->cpitch, g->bpf, g->phiL);
        g->assembled = true;                  // the solver core may run now
        int rc = bicgstab_device(g, make_op(g, 3), g->bpf, g->phiL, g->opt_lin_tol, g->opt_lin_maxit, &g->laplace_iters,
                                 nullptr, nullptr);
        if (rc < 0) { g->assembled = false; return rc; }
        laplace_maxit = rc == PF_NOT_CONVERGED;
        launch_phistar(g->stream, g->g, g->h, g->eps, g->eps_mid, g->eps_min, kap, g->charges_dev, g->ncharges, g->phistar);
        launch_interface_rhs(g->stream, g->g, g->h, g->eps, g->eps_mid, g->eps_min, kap, g->charges_dev, g->ncharges,
                             g->phiL, g->fixed);
    }
    PF_CUDA(g, cudaMemsetAsync(g->p0, 0, vec * 4, g->stream));   // p0,p1,v0,v1 finite before first use
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    PF_CUDA(g, cudaGetLastError());
    g->pf1_lc = std::nan("");
    g->assembled = true;
    if (laplace_maxit) {
        g->err = "the Laplace solve for phi^L stopped at PF_OPT_LINEAR_MAXIT: b^IF was built from an unconverged phi^L";
        return PF_NOT_CONVERGED;
    }
    return PF_OK;
}

int pf_solve_linear(pf_grid* g, const double* rhs, double* x, const double* sigma, double tol, int maxit,
                    int* iters_out, double* relres_out, double* true_relres_out) {
    int rc = check_ready(g);
    if (rc) return rc;
    if (!rhs || !x) return fail(g, PF_ERR_ARG, "rhs and x must not be NULL");
    launch_copy_with_dirichlet(g->stream, g->g, g->bc, rhs, g->bw);   // Q20
    // an iterate that is not 16-byte aligned (a view into a larger array) would keep the solve off the tiled
    // kernels: it is solved in the workspace copy instead
    double* xs = x;
    const size_t nbytes = sizeof(double) * (size_t)g->g.n;
    if (((uintptr_t)x & 15u) != 0 && x != g->xw) {
        PF_CUDA(g, cudaMemcpyAsync(g->xw, x, nbytes, cudaMemcpyDeviceToDevice, g->stream));
        xs = g->xw;
    }
    launch_set_dirichlet(g->stream, g->g, g->bc, xs);                  // Q4
    int which = 0;
    if (sigma) { launch_diag_plus_sigma(g->stream, g->g, g->bc, g->A0, sigma, g->A0_s); which = 2; }
    rc = bicgstab_device(g, make_op(g, which), g->bw, xs, tol, maxit, iters_out, relres_out, true_relres_out);
    if (xs != x && rc != PF_ERR_CUDA && rc != PF_ERR_ARG)
        PF_CUDA(g, cudaMemcpyAsync(x, xs, nbytes, cudaMemcpyDeviceToDevice, g->stream));
    return rc;
}

int pf_grid_stage_host(pf_grid* g, const double* rhs_host, const double* x_host) {
    int rc = check_ready(g);
    if (rc) return rc;
    if (!rhs_host || !x_host) return fail(g, PF_ERR_ARG, "rhs and x must not be NULL");
    if (!g->copy_stream) {
        PF_CUDA(g, cudaStreamCreateWithFlags(&g->copy_stream, cudaStreamNonBlocking));
        PF_CUDA(g, cudaEventCreateWithFlags(&g->staged_ev, cudaEventDisableTiming));
        PF_CUDA(g, cudaEventCreateWithFlags(&g->main_ev, cudaEventDisableTiming));
    }
    const size_t nbytes = sizeof(double) * (size_t)g->g.n;
    // work already enqueued on the grid's stream may still read the staging vectors (an earlier host solve)
    PF_CUDA(g, cudaEventRecord(g->main_ev, g->stream));
    PF_CUDA(g, cudaStreamWaitEvent(g->copy_stream, g->main_ev, 0));
    PF_CUDA(g, cudaMemcpyAsync(g->hb, rhs_host, nbytes, cudaMemcpyHostToDevice, g->copy_stream));
    PF_CUDA(g, cudaMemcpyAsync(g->hx, x_host, nbytes, cudaMemcpyHostToDevice, g->copy_stream));
    PF_CUDA(g, cudaEventRecord(g->staged_ev, g->copy_stream));
    g->staged_rhs = rhs_host; g->staged_x = x_host;
    return PF_OK;
}

int pf_solve_linear_host(pf_grid* g, const double* rhs_host, double* x_host, const double* sigma, double tol,
                         int maxit, int* iters_out, double* relres_out, double* true_relres_out) {
    int rc = check_ready(g);
    if (rc) return rc;
    if (!rhs_host || !x_host) return fail(g, PF_ERR_ARG, "rhs and x must not be NULL");
    const size_t nbytes = sizeof(double) * (size_t)g->g.n;
    if (g->staged_rhs == rhs_host && g->staged_x == x_host) {
        // uploaded ahead by pf_grid_stage_host on the copy stream: the solve only waits for that copy
        PF_CUDA(g, cudaStreamWaitEvent(g->stream, g->staged_ev, 0));
    } else {
        PF_CUDA(g, cudaMemcpyAsync(g->hb, rhs_host, nbytes, cudaMemcpyHostToDevice, g->stream));
        PF_CUDA(g, cudaMemcpyAsync(g->hx, x_host, nbytes, cudaMemcpyHostToDevice, g->stream));
    }
    g->staged_rhs = g->staged_x = nullptr;
    rc = pf_solve_linear(g, g->hb, g->hx, sigma, tol, maxit, iters_out, relres_out, true_relres_out);
    if (rc < 0) return rc;
    PF_CUDA(g, cudaMemcpyAsync(x_host, g->hx, nbytes, cudaMemcpyDeviceToHost, g->stream));
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    return rc;
}

int pf_fermi_pointwise(pf_grid* g, int nions, const double* valence, const double* bath_conc, const double* radii,
                       const double* phi, double* rho, double* sigma, double* steric, double* conc) {
    int rc = check_ready(g);
    if (rc) return rc;
    if (!phi) return fail(g, PF_ERR_ARG, "phi must not be NULL");
    SpeciesDev sp;
    rc = make_species(g, nions, valence, bath_conc, radii, &sp);
    if (rc) return rc;
    launch_fermi(g->stream, g->g, g->bc, sp, g->eps, g->eps_mid, g->uniform, phi, rho, sigma, steric, conc, nullptr,
                 nullptr, nullptr);
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    PF_CUDA(g, cudaGetLastError());
    return PF_OK;
}

int pf_solve_pf(pf_grid* g, int nions, const double* valence, const double* bath_conc, const double* radii,
                double l_c, double tol, double* phi, double* conc, double* steric, int* outer_iters_out,
                int* linear_iters_out) {
    int rc = check_ready(g);
    if (rc) return rc;
    if (!phi) return fail(g, PF_ERR_ARG, "phi must not be NULL");
    if (!(l_c >= 0.0) || !(tol >= 0.0)) return fail(g, PF_ERR_ARG, "l_c and tol must be >= 0");
    SpeciesDev sp;
    rc = make_species(g, nions, valence, bath_conc, radii, &sp);
    if (rc) return rc;
    const size_t nbytes = sizeof(double) * (size_t)g->g.n;
    if (!(g->pf1_lc == l_c)) {      // row N2: PF1 operator, once per (grid, l_c)
        launch_assemble_pf1(g->stream, g->g, g->h, l_c, g->bc, g->eps, g->eps_mid, g->uniform, g->pal, g->code_mode, g->A0_pf1,
                            g->code_pf1, g->cpitch, g->offd_pf1);
        if (g->code_mode) {
            double ctab[PF_CTAB];
            build_ctab_pf1(g->pal, g->h, l_c, ctab);
            PF_CUDA(g, cudaMemcpyAsync(g->ctab_pf1, ctab, sizeof(ctab), cudaMemcpyHostToDevice, g->stream));
        }
        g->pf1_lc = l_c;
    }
    g->lin_iters.clear();
    g->increments.clear();
    int total = 0, its = 0;
    bool inner_maxit = false;      // a linear solve stopped at its iteration cap: its result was used as it stood
    // row N4 (Table 2 step 2): initial guess from PF2 with rho' = Psi = 0
    launch_copy_with_dirichlet(g->stream, g->g, g->bc, g->fixed, g->bpf);
    PF_CUDA(g, cudaMemsetAsync(g->phi0, 0, nbytes, g->stream));
    launch_set_dirichlet(g->stream, g->g, g->bc, g->phi0);
    rc = bicgstab_device(g, make_op(g, 0), g->bpf, g->phi0, g->opt_lin_tol, g->opt_lin_maxit, &its, nullptr, nullptr);
    g->lin_iters.push_back(its); total += its;
    if (rc < 0) return rc;
    inner_maxit |= rc == PF_NOT_CONVERGED;
    PF_CUDA(g, cudaMemsetAsync(g->psi, 0, nbytes, g->stream));
    const bool lagged = g->opt_steric_mode == 1;
    if (lagged) PF_CUDA(g, cudaMemsetAsync(g->sstate, 0, nbytes, g->stream));       // S^trc = 0: the bath (G1)
    int status = PF_NOT_CONVERGED, outer = 0;
    double* phi0 = g->phi0;
    double* phiw = g->phiw;
    while (outer < g->opt_max_outer) {
        ++outer;
        // row N1: concentrations, steric potential, PF1 right-hand side, PF2 diagonal -- one kernel
        launch_fermi(g->stream, g->g, g->bc, sp, g->eps, g->eps_mid, g->uniform, phi0, nullptr, g->sigma, nullptr,
                     nullptr, g->bpf, g->A0, g->A0_s, lagged ? g->sstate : nullptr, lagged);
        // row N2 (step 3): PF1 -> Psi, warm start from the previous Psi
        rc = bicgstab_device(g, make_op(g, 1), g->bpf, g->psi, g->opt_lin_tol, g->opt_lin_maxit, &its, nullptr, nullptr);
        g->lin_iters.push_back(its); total += its;
        if (rc < 0) return rc;
        inner_maxit |= rc == PF_NOT_CONVERGED;
        // row N3 (step 4): PF2 -> phi, warm start from phi0
        launch_rhs_pf2(g->stream, g->g, g->bc, g->eps, g->eps_mid, g->uniform, g->psi, g->sigma, phi0, g->fixed, g->bpf);
        PF_CUDA(g, cudaMemcpyAsync(phiw, phi0, nbytes, cudaMemcpyDeviceToDevice, g->stream));
        rc = bicgstab_device(g, make_op(g, 2), g->bpf, phiw, g->opt_lin_tol, g->opt_lin_maxit, &its, nullptr, nullptr);
        g->lin_iters.push_back(its); total += its;
        if (rc < 0) return rc;
        inner_maxit |= rc == PF_NOT_CONVERGED;
        // row N5 (step 5): relax, then test the increment
        launch_relax(g->stream, g->g.n, g->opt_omega_pf, phi0, phiw, g->dmax_bits);
        unsigned long long bits = 0;
        PF_CUDA(g, cudaMemcpyAsync(&bits, g->dmax_bits, sizeof(bits), cudaMemcpyDeviceToHost, g->stream));
        PF_CUDA(g, cudaStreamSynchronize(g->stream));
        double d;
        std::memcpy(&d, &bits, sizeof(d));
        g->increments.push_back(d);
        if (!std::isfinite(d))          // reading D7: a NaN fails "d > tol" and would otherwise read as converged
            return fail(g, PF_ERR_BREAKDOWN, "non-finite potential increment in outer iteration %d", outer);
        std::swap(phi0, phiw);
        if (!(d > tol)) { status = PF_OK; break; }
    }
    PF_CUDA(g, cudaMemcpyAsync(phi, phi0, nbytes, cudaMemcpyDeviceToDevice, g->stream));
    if (g->charge_model == 1) launch_recombine(g->stream, g->g.n, g->phistar, g->phiL, phi);   // Eq (5)
    if (conc || steric)       // (lagged: the fields that belong to the state -- C_k at the final phi with the S at hand)
        launch_fermi(g->stream, g->g, g->bc, sp, g->eps, g->eps_mid, g->uniform, phi0, nullptr, nullptr, steric, conc,
                     nullptr, nullptr, nullptr, lagged ? g->sstate : nullptr, false);
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    PF_CUDA(g, cudaGetLastError());
    if (outer_iters_out) *outer_iters_out = outer;
    if (linear_iters_out) *linear_iters_out = total;
    if (status == PF_OK && inner_maxit) {
        g->err = "the increment met the tolerance, but at least one linear solve stopped at PF_OPT_LINEAR_MAXIT";
        return PF_INNER_NOT_CONVERGED;
    }
    return status;
}

int pf_grid_history(pf_grid* g, double* hist_host, int cap) {
    if (!g || !hist_host || cap < 0) return PF_ERR_ARG;
    if (!g->hist) return fail(g, PF_ERR_ARG, "history not enabled (PF_OPT_HISTORY)");
    const int n = std::min(std::min(cap, g->hist_cap), g->last_iters + 1);
    PF_CUDA(g, cudaMemcpyAsync(hist_host, g->hist, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost, g->stream));
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    return n;
}

int pf_grid_linear_iters(pf_grid* g, int* iters_host, int cap) {
    if (!g || !iters_host || cap < 0) return PF_ERR_ARG;
    const int n = std::min<int>(cap, (int)g->lin_iters.size());
    for (int k = 0; k < n; ++k) iters_host[k] = g->lin_iters[k];
    return n;
}

int pf_grid_increments(pf_grid* g, double* incr_host, int cap) {
    if (!g || !incr_host || cap < 0) return PF_ERR_ARG;
    const int n = std::min<int>(cap, (int)g->increments.size());
    for (int k = 0; k < n; ++k) incr_host[k] = g->increments[k];
    return n;
}

long long pf_launch_count(void) { return pf::g_launch_count; }

int pf_grid_profile(pf_grid* g, double* ms_out, long long* launches_out) {
    if (!g || !ms_out || !launches_out) return PF_ERR_ARG;
    for (int j = 0; j < 3; ++j) { ms_out[j] = g->prof_ms[j]; launches_out[j] = g->prof_launches[j]; }
    return PF_OK;
}

int pf_grid_set_fixed_nodes(pf_grid* g, const long long* idx_host, const double* val_host, int count) {
    if (!g) return PF_ERR_ARG;
    if (g->assembled) return fail(g, PF_ERR_ARG, "set the fixed nodes before pf_grid_set_workspace");
    if (count < 0 || (count > 0 && (!idx_host || !val_host))) return fail(g, PF_ERR_ARG, "bad fixed-node list");
    if ((long long)count > g->g.n) return fail(g, PF_ERR_ARG, "more fixed nodes than grid nodes");
    for (int k = 0; k < count; ++k) {
        if (idx_host[k] < 0 || idx_host[k] >= g->g.n) return fail(g, PF_ERR_ARG, "fixed node %d is outside the grid", k);
        if (!(val_host[k] == val_host[k])) return fail(g, PF_ERR_ARG, "fixed node %d has a NaN value", k);
    }
    g->fix_idx.assign(idx_host, idx_host + count);
    g->fix_val.assign(val_host, val_host + count);
    return PF_OK;
}

int pf_grid_relax(pf_grid* g, double omega_pf, const double* phi0, double* phi, double* incr_out) {
    if (!g || !phi0 || !phi || !incr_out) return PF_ERR_ARG;
    launch_relax(g->stream, g->g.n, omega_pf, phi0, phi, g->dmax_bits);      // the kernel and scratch pf_solve_pf uses
    unsigned long long bits = 0;
    PF_CUDA(g, cudaMemcpyAsync(&bits, g->dmax_bits, sizeof(bits), cudaMemcpyDeviceToHost, g->stream));
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    std::memcpy(incr_out, &bits, sizeof(double));
    return PF_OK;
}

int pf_grid_laplace_iters(const pf_grid* g) { return g ? g->laplace_iters : PF_ERR_ARG; }

int pf_grid_fault_repeats(const pf_grid* g) { return g ? g->fault_repeats : PF_ERR_ARG; }

int pf_coop_plan(int nx, int ny, int nz, int max_blocks, size_t smem_cap, int* out) {
    if (!out || nx < 3 || ny < 3 || nz < 3 || max_blocks < 1) return PF_ERR_ARG;
    GridDims gd;
    gd.nx = nx; gd.ny = ny; gd.nz = nz; gd.n = (long long)nx * ny * nz;
    Operator op;
    std::memset(&op, 0, sizeof(op));
    CoopPlan plan;
    if (!coop_plan(gd, op, max_blocks, smem_cap, &plan)) return PF_ERR_ARG;
    out[0] = plan.nbx; out[1] = plan.nby; out[2] = plan.nbz; out[3] = plan.vmax; out[4] = plan.hmax;
    out[5] = plan.nhmax; out[6] = plan.threads; out[7] = (int)plan.smem;
    return PF_OK;
}

int pf_tile_plan(int nx, int ny, int nz, int tile_rows, int sm_count, int mode, int* out) {
    if (!out || nx < 1 || ny < 1 || nz < 1 || sm_count < 1 || (tile_rows != 13 && tile_rows != 16) || mode < -1 || mode > 2)
        return PF_ERR_ARG;
    GridDims gd;
    gd.nx = nx; gd.ny = ny; gd.nz = nz; gd.n = (long long)nx * ny * nz;
    tma_plan(gd, tile_rows, sm_count, mode, out);
    return PF_OK;
}

int pf_grid_stencil(const pf_grid* g) { return g ? (want_stored(g) ? 1 : 2) : PF_ERR_ARG; }
int pf_grid_palette_size(const pf_grid* g) { return g ? g->pal.count : PF_ERR_ARG; }

int pf_grid_code_layout(const pf_grid* g, int* bits_out, int* pitch_out, size_t* bytes_out) {
    if (!g) return PF_ERR_ARG;
    const int m = code_mode_of(g);
    if (bits_out) *bits_out = m == 0 ? 0 : (m == 1 ? 16 : 32);
    if (pitch_out) *pitch_out = cpitch_of(g);
    if (bytes_out) *bytes_out = code_bytes_of(g);
    return PF_OK;
}

int pf_grid_copy_array(pf_grid* g, int which, void* dst) {
    if (!g || !dst) return PF_ERR_ARG;
    if (!g->assembled) return fail(g, PF_ERR_WORKSPACE, "workspace not set");
    const void* src = nullptr;
    size_t nbytes = sizeof(double) * (size_t)g->g.n;
    if (which == 0) src = g->A0;
    else if (which >= 1 && which <= 6) src = g->offd[which - 1];
    else if (which == 7) src = g->fixed;
    else if (which == 8) { src = g->code; nbytes = code_bytes_of(g); }
    else if (which == 9) src = (g->pf1_lc == g->pf1_lc) ? g->A0_pf1 : nullptr;
    else if (which == 10) { src = g->code_mode ? g->ctab_poisson : nullptr; nbytes = sizeof(double) * PF_CTAB; }
    else if (which == 11) { src = (g->pf1_lc == g->pf1_lc) ? g->code_pf1 : nullptr; nbytes = code_bytes_of(g); }
    else if (which == 13) src = (g->pf1_lc == g->pf1_lc) ? g->psi : nullptr;
    else if (which == 14) src = g->charge_model == 1 ? g->phiL : nullptr;
    else if (which == 15) src = g->charge_model == 1 ? g->phistar : nullptr;
    else if (which == 12) { src = (g->pf1_lc == g->pf1_lc && g->code_mode) ? g->ctab_pf1 : nullptr; nbytes = sizeof(double) * PF_CTAB; }
    if (!src) return fail(g, PF_ERR_ARG, "array %d is not available", which);
    PF_CUDA(g, cudaMemcpyAsync(dst, src, nbytes, cudaMemcpyDeviceToDevice, g->stream));
    PF_CUDA(g, cudaStreamSynchronize(g->stream));
    return PF_OK;
}

}  // extern "C"
