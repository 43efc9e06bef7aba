// pf_krylov.cuh -- pieces shared by the direct, the tiled and the cooperative Krylov kernels: the elementwise
// statements of Table 3 (reading R3) and the scalar work at each of the three reduction
// points of an iteration (rows L4-L8), taken by thread 0 of EVERY block at the start of the next kernel
// (begin_kernel below: same data, same order, same bits in all blocks; block 0 stores the new state).
#pragma once
#include "pf_common.cuh"

namespace pf {

// Vectors of one solve.  p and v are double-buffered: the fused kernel of steps 9+11 reads the old
// p, v at neighbour nodes while other blocks already write the new ones.
struct KrylovVecs {
    const double* b;     // right-hand side with Dirichlet values in place
    double* x;
    double* y;           // preconditioned solves accumulate step 16 here (reading D3); == x when M = I
    double* r;
    double* r_out;       // merged solver: its fused kernel reads r at neighbour nodes while other blocks write the new r
    double* rt;          // r~ = r0
    double* p_in;  double* p_out;
    double* v_in;  double* v_out;
    double* t;
    double* hist;        // relative residual per iteration, or null
};

// Step 9 (+ the Jacobi step of reading Q2): value the first matvec is applied to, at node j.
//   p_j = r_j + beta (p_j - omega v_j)   (p = r in the first iteration, steps 5-6)
template <bool PRECOND>
__device__ __forceinline__ double p_new_at(bool first, double beta, double omega, double r, double p, double v) {
    (void)PRECOND;
    return first ? r : add(r, mul(beta, sub(p, mul(omega, v))));
}

// Step 13: s_j = r_j - alpha v_j.
__device__ __forceinline__ double s_at(double alpha, double r, double v) { return sub(r, mul(alpha, v)); }

template <bool PRECOND>
__device__ __forceinline__ double jacobi(double u, double a0) { return PRECOND ? dvd(u, a0) : u; }

// ---- reduction-point epilogues (the scalar steps; thread 0 of every block, see begin_kernel) -----

// After r0 = b - A x0 (step 2): ||b||, ||r0||, rho_0 = r~.r0 = r0.r0, early exits.
// norm_mode 1 (Table 3 steps 18-19 as written): the measure is ||r||_inf, absolute, the test
// strict; rnorm then holds the maximum norm and bnorm the scale 1.
__device__ __forceinline__ bool converged(const Scalars* sc) {
    return sc->norm_mode == 1 ? sc->rnorm < sc->tol : sc->rnorm <= mul(sc->tol, sc->bnorm);
}

// Reading D7: a reduced scalar that is not finite (NaN or infinite right-hand side, overflow of a
// diverging iterate) ends the solve as a breakdown -- a NaN fails every comparison, so without this test it would
// pass "rho == 0" and never pass the convergence test, and with the maximum norm it could even look converged.
__device__ __forceinline__ bool finite2(double a, double b) { return isfinite(a) && isfinite(b); }

__device__ __forceinline__ void finish_init(Scalars* sc, double* hist, double bb, double rr, double rmax) {
    sc->bb = bb; sc->rr = rr; sc->rmax = rmax;
    sc->bnorm = sc->norm_mode == 1 ? 1.0 : __dsqrt_rn(bb);
    sc->rnorm = sc->norm_mode == 1 ? rmax : __dsqrt_rn(rr);
    sc->it = 0; sc->first = 1; sc->done = 0; sc->status = 1;
    sc->rho = rr; sc->rho_old = 1.0; sc->alpha = 1.0; sc->omega = 1.0; sc->beta = 0.0;
    sc->rhat = rr; sc->rho_next = rr; sc->rtt = 0.0;
    if (!finite2(bb, sc->rnorm)) {                      // D7
        sc->done = 1; sc->status = -3;
        if (hist && sc->hist_cap > 0) hist[0] = sc->rnorm;
        return;
    }
    if (bb == 0.0) {                       // Q3: b = 0 => x = 0, no iterations (host zeroes x)
        sc->done = 1; sc->status = 0; sc->rnorm = 0.0; sc->bnorm = 0.0;
        if (hist && sc->hist_cap > 0) hist[0] = 0.0;
        return;
    }
    if (hist && sc->hist_cap > 0) hist[0] = dvd(sc->rnorm, sc->bnorm);
    if (converged(sc)) { sc->done = 1; sc->status = 0; return; }
    if (sc->maxit <= 0) { sc->done = 1; sc->status = 1; return; }
    if (rr == 0.0) { sc->done = 1; sc->status = -3; }
}

// After v = A M^-1 p (step 11): alpha = rho/(r~.v) (step 12).
__device__ __forceinline__ void finish_k1(Scalars* sc, double rtv) {
    sc->rtv = rtv;
    if (rtv == 0.0 || !isfinite(rtv)) { sc->done = 1; sc->status = -3; return; }     // Q5, D7
    sc->alpha = dvd(sc->rho, rtv);
}

// After t = A M^-1 s (step 14): omega = t.s/t.t (step 15); t.t = 0 => omega = 0 (Q5).
__device__ __forceinline__ void finish_k2(Scalars* sc, double ts, double tt) {
    sc->ts = ts; sc->tt = tt;
    sc->omega = (tt == 0.0) ? 0.0 : dvd(ts, tt);
    if (!finite2(ts, tt)) { sc->done = 1; sc->status = -3; }                          // D7
}

// After the x and r updates (steps 16-17): ||r|| test (steps 18-20), then rho and beta of the next
// iteration (steps 4, 8).
__device__ __forceinline__ void finish_k3(Scalars* sc, double* hist, double rho_new, double rr, double rmax) {
    sc->rr = rr; sc->rmax = rmax;
    sc->rnorm = sc->norm_mode == 1 ? rmax : __dsqrt_rn(rr);
    const int it = sc->it + 1;
    sc->it = it;
    if (hist && it < sc->hist_cap) hist[it] = dvd(sc->rnorm, sc->bnorm);
    const double rho_old = sc->rho;
    sc->rho_old = rho_old;
    if (!isfinite(sc->rnorm)) { sc->done = 1; sc->status = -3; return; }              // D7
    if (converged(sc)) { sc->done = 1; sc->status = 0; return; }
    if (sc->omega == 0.0) { sc->done = 1; sc->status = -3; return; }
    if (it >= sc->maxit) { sc->done = 1; sc->status = 1; return; }
    sc->rho = rho_new;
    if (rho_new == 0.0 || !isfinite(rho_new)) { sc->done = 1; sc->status = -3; return; }     // Q5, D7
    sc->beta = mul(dvd(rho_new, rho_old), dvd(sc->alpha, sc->omega));   // step 8
    sc->first = 0;
}

// ---- the merged solver (SURVEY 8(d) "fully merged", 8(f) #3; reading M1 of DESIGN.md) ----------------------------
// Two kernels and two reduction points per iteration instead of three:
//   K2M  s = r - alpha v; t = A M^-1 s;                                   reduces t.s, t.t, r~.t
//   K31  r' = s - omega t; y += alpha p + omega s; p' = r' + beta (p - omega v); v' = A M^-1 p';
//                                                                         reduces r~.v', r'.r' (max |r'|), r~.r'
// with rho_i = (r~.r_{i-1} - alpha r~.v) - omega r~.t, so that beta is known when K31 starts.  The first v = A M^-1 r0
// comes from the ordinary k1 (first = 1).  Statement for statement the oracle's bicgstab_merged().

// After K2M: omega (step 15), rho_i and beta.  Whether iteration i was the last one (convergence, omega = 0, maxit)
// is only known once K31 has reduced ||r'||; beta may therefore be meaningless in the last iteration (its p', v' are
// never used).
__device__ __forceinline__ void finish_k2m(Scalars* sc, double ts, double tt, double rtt) {
    sc->ts = ts; sc->tt = tt; sc->rtt = rtt;
    sc->omega = (tt == 0.0) ? 0.0 : dvd(ts, tt);
    if (!finite2(ts, tt)) { sc->done = 1; sc->status = -3; return; }                   // D7
    const double rho_new = sub(sub(sc->rhat, mul(sc->alpha, sc->rtv)), mul(sc->omega, rtt));   // M1
    sc->rho_next = rho_new;
    sc->beta = mul(dvd(rho_new, sc->rho), dvd(sc->alpha, sc->omega));
}

// After K31: close iteration i (||r|| test, steps 18-20), then alpha of iteration i + 1.
__device__ __forceinline__ void finish_k31(Scalars* sc, double* hist, double rtv, double rr, double rhat, double rmax) {
    sc->rr = rr; sc->rmax = rmax;
    sc->rnorm = sc->norm_mode == 1 ? rmax : __dsqrt_rn(rr);
    const int it = sc->it + 1;
    sc->it = it;
    if (hist && it < sc->hist_cap) hist[it] = dvd(sc->rnorm, sc->bnorm);
    sc->rho_old = sc->rho;
    if (!isfinite(sc->rnorm)) { sc->done = 1; sc->status = -3; return; }              // D7
    if (converged(sc)) { sc->done = 1; sc->status = 0; return; }
    if (sc->omega == 0.0) { sc->done = 1; sc->status = -3; return; }
    if (it >= sc->maxit) { sc->done = 1; sc->status = 1; return; }
    const double rho_new = sc->rho_next;
    if (rho_new == 0.0 || !isfinite(rho_new)) { sc->done = 1; sc->status = -3; return; }     // Q5, D7
    sc->rho = rho_new; sc->rhat = rhat; sc->rtv = rtv;
    sc->first = 0;
    if (rtv == 0.0 || !isfinite(rtv)) { sc->done = 1; sc->status = -3; return; }
    sc->alpha = dvd(rho_new, rtv);
}

// ---- start of every kernel of a solve (rows L7, L8) ---------------------------------------------
// Copy the device scalars into the block's shared memory, combine the partial sums the previous kernel left
// (pf_common.cuh), take the scalar step that was waiting for them, and note what THIS kernel (kind `kind`, a
// PEND_* value; PEND_NONE for the one-block finalize kernel) will leave pending.  Every block does the same
// arithmetic on the same data; block 0 stores the new state to sc_out.  Returns false when the solve is over
// (the block returns at once).  All threads of the block must call; S and scratch are shared memory
// (scratch: 3*32 dd).  hist: residual history or null.
// LOOP: the kernel is the one of a loop body that keeps the condition of the body's WHILE node up to date
// (pf_api.cu loop_graph; only k3 is compiled that way -- Nsight Compute does not profile kernel nodes that can set
// conditional handles, in graphs of any kind, so every other kernel stays free of the call).
// Which producer's partial sums a kernel of kind `kind` can find pending (besides none).  `kind` is a compile-time
// constant at every call, so the tests fold and a kernel carries the combine and the scalar step of its possible
// predecessors only: k1 follows k3 or the initial residual, k2 follows k1, k3 follows k2; K2M follows k1 (the first
// matvec of a merged solve) or K31, K31 follows K2M; the residual kernels find nothing pending; the one-block finalize
// follows anything.
__device__ __forceinline__ bool may_follow(int kind, int pend) {
    switch (kind) {
        case PEND_K1:  return pend == PEND_K3 || pend == PEND_INIT;
        case PEND_K2:  return pend == PEND_K1;
        case PEND_K3:  return pend == PEND_K2;
        case PEND_K2M: return pend == PEND_K1 || pend == PEND_K31;
        case PEND_K31: return pend == PEND_K2M;
        case PEND_INIT:                          // the residual kernels start a solve (fresh scalars) or follow the
        case PEND_TRUE: return false;            // one-block finalize: nothing is ever pending for them
        default:       return true;              // the finalize itself follows anything
    }
}

template <bool LOOP = false>
__device__ __forceinline__ bool begin_kernel(int kind, Scalars* S, const Scalars* sc_in, Scalars* sc_out,
                                             const ReduceBuf& rb, double* hist, dd* scratch) {
    constexpr int NWORDS = (int)(sizeof(Scalars) / sizeof(int));
    // what usually precedes a kernel of this kind (k3 or the initial residual before k1, k1 before k2, k2 before
    // k3): its partials are requested together with the scalars
    const PartialPrefetch pre = prefetch_partials(
        rb, kind == PEND_K1 ? PEND_K3 : (kind == PEND_K2 ? PEND_K1 : (kind == PEND_K3 ? PEND_K2
          : (kind == PEND_K2M ? PEND_K31 : (kind == PEND_K31 ? PEND_K2M : PEND_NONE)))));
    if ((int)threadIdx.x < NWORDS)
        reinterpret_cast<int*>(S)[threadIdx.x] = reinterpret_cast<const int*>(sc_in)[threadIdx.x];
    // a division range fault raised by an earlier kernel of this solve (dvd_nb, reading D4): requested with the scalars
    const int faulted = threadIdx.x == 0 ? *rb.fault : 0;
    __syncthreads();
    const int pend = S->pending, nblk = S->pending_nblk;        // the same in every thread of every block
    // Thread 0 rewrites S->pending below.  With partial sums pending, the barriers of the combine separate these
    // reads from that write; without (the first kernel after a finalize, i.e. at every polling-chunk boundary) nothing
    // did, and a warp that read late saw the NEW value, entered a combine the other warps skipped and left the block
    // with mismatched barriers: wrong sums or a hang, depending on timing (found in round 2 when two unrelated
    // one-instruction changes each made it appear).
    __syncthreads();
    dd q[2] = {dd_zero(), dd_zero()};
    dd q3[3] = {dd_zero(), dd_zero(), dd_zero()};
    double m = 0.0;
    const bool any2t = may_follow(kind, PEND_K3) || may_follow(kind, PEND_INIT) || may_follow(kind, PEND_TRUE);
    bool unexpected = false;
    if (may_follow(kind, PEND_K1) && pend == PEND_K1) { dd q1[1]; combine_partials<1, false>(q1, m, nblk, scratch, rb, pend, pre); q[0] = q1[0]; }
    else if (may_follow(kind, PEND_K2) && pend == PEND_K2) combine_partials<2, false>(q, m, nblk, scratch, rb, pend, pre);
    else if (may_follow(kind, PEND_K2M) && pend == PEND_K2M) combine_partials<3, false>(q3, m, nblk, scratch, rb, pend, pre);
    else if (may_follow(kind, PEND_K31) && pend == PEND_K31) combine_partials<3, true>(q3, m, nblk, scratch, rb, pend, pre);
    else if (any2t && may_follow(kind, pend) && (pend == PEND_K3 || pend == PEND_INIT || pend == PEND_TRUE))
        combine_partials<2, true>(q, m, nblk, scratch, rb, pend, pre);
    else if (pend != PEND_NONE) unexpected = true;       // (a launch order the driver never produces)
    if (threadIdx.x == 0) {
        const bool lead = linear_block_id() == 0;
        double* h = lead ? hist : nullptr;                       // one writer for the history
        if (unexpected) { S->done = 1; S->status = -2; }
        else if (may_follow(kind, PEND_INIT) && pend == PEND_INIT) finish_init(S, h, dd_round(q[0]), dd_round(q[1]), m);
        else if (may_follow(kind, PEND_K1) && pend == PEND_K1) finish_k1(S, dd_round(q[0]));
        else if (may_follow(kind, PEND_K2) && pend == PEND_K2) finish_k2(S, dd_round(q[0]), dd_round(q[1]));
        else if (may_follow(kind, PEND_K3) && pend == PEND_K3) finish_k3(S, h, dd_round(q[0]), dd_round(q[1]), m);
        else if (may_follow(kind, PEND_K2M) && pend == PEND_K2M) finish_k2m(S, dd_round(q3[0]), dd_round(q3[1]), dd_round(q3[2]));
        else if (may_follow(kind, PEND_K31) && pend == PEND_K31) finish_k31(S, h, dd_round(q3[0]), dd_round(q3[1]), dd_round(q3[2]), m);
        else if (may_follow(kind, PEND_TRUE) && pend == PEND_TRUE) { S->true_rr = dd_round(q[1]); S->true_rmax = m; }
        // the iterates are invalid from the faulting kernel on: stop here (status stays PF_NOT_CONVERGED) instead of
        // iterating on them up to maxit; the host repeats the solve with the __ddiv_rn kernels (x is untouched, D3).
        // Blocks of one launch may disagree for one kernel (a block of THIS launch can raise the flag while others
        // read it); what they compute is discarded anyway, and the next launch sees done in every block.
        if (faulted && kind != PEND_INIT && kind != PEND_TRUE) { S->done = 1; S->fault = 1; }
        const bool runs = kind == PEND_INIT || kind == PEND_TRUE || (kind != PEND_NONE && !S->done);
        S->pending = runs ? kind : PEND_NONE;
        S->pending_nblk = (int)linear_grid_size();
        if (kind == PEND_NONE) S->fault = faulted;               // finalize: what the host is about to read
        if (lead) *sc_out = *S;
        // body of a device-side loop: is there another turn?  Not when the solve is over (known with a lag of one
        // iteration: the k1 of iteration i + 1 takes the step that ends iteration i), nor when this k3 closes the
        // last iteration the loop is meant to run (the whole bodies that fit below maxit), whatever its sums turn
        // out to be.
        if (LOOP && lead && rb.more) {
            const bool last = S->it + 1 >= S->loop_end;
            cudaGraphSetConditional((cudaGraphConditionalHandle)rb.more, (S->done || last) ? 0u : 1u);
        }
    }
    __syncthreads();
    return S->pending != PEND_NONE;
}

}  // namespace pf
