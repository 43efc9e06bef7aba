// pf_krylov_direct.cu -- "direct" Krylov kernels: one thread per node in a grid-stride loop,
// neighbours fetched straight from global memory through L1/L2.  Same arithmetic, statement for
// statement, as the tiled kernels (pf_krylov_tma.cu) and the cooperative kernel (pf_krylov_coop.cu);
// this variant is the simple one the other two are tested against, and the one used for grids too
// small to fill the tiles when the cooperative kernel does not apply.
//
// One BiCGSTAB iteration (Table 3) is three launches, one per reduction point:
//   k1: steps 5-11   p = r + beta(p - omega v);  v = A M^-1 p;           reduces r~.v        (row L4)
//   k2: steps 12-14  alpha; s = r - alpha v;  t = A M^-1 s;              reduces t.s, t.t    (row L5)
// Each kernel starts by combining the partial sums its predecessor left and taking the scalar step that waited
// for them (alpha in k2, omega in k3, the convergence test, rho and beta in k1; begin_kernel, pf_krylov.cuh),
// and ends by writing its own partial sums.
//   k3: steps 15-18  omega; y += alpha p + omega s (x = x0 + M^-1 y at the end, reading D3);
//                    r = s - omega t; reduces r~.r (step 4 of the next iteration) and r.r     (row L6)
#include "pf_krylov.cuh"
#include "pf_launch.h"

namespace pf {

namespace {

constexpr int DIRECT_THREADS = 256;

struct Nbr {
    long long j[6];
    bool in[6];
    int ix, iy, iz;
};

__device__ __forceinline__ Nbr neighbours(const GridDims& g, long long i) {
    const int ix = (int)(i % g.nx);
    const long long q = i / g.nx;
    const int iy = (int)(q % g.ny);
    const int iz = (int)(q / g.ny);
    const long long sx = 1, sy = g.nx, sz = (long long)g.nx * g.ny;
    Nbr n;
    n.ix = ix; n.iy = iy; n.iz = iz;
    n.j[0] = i + sx; n.in[0] = ix + 1 < g.nx;
    n.j[1] = i - sx; n.in[1] = ix > 0;
    n.j[2] = i - sy; n.in[2] = iy > 0;
    n.j[3] = i + sy; n.in[3] = iy + 1 < g.ny;
    n.j[4] = i - sz; n.in[4] = iz > 0;
    n.j[5] = i + sz; n.in[5] = iz + 1 < g.nz;
    return n;
}

// Off-diagonal coefficients of row i (0 where the neighbour is outside the box or the row is an
// identity row).
__device__ __forceinline__ void row_coeffs(const Operator& op, const GridDims& g, const double* ctab_s, long long i,
                                           const Nbr& n, double (&c)[6]) {
    if (op.stored) {
#pragma unroll
        for (int d = 0; d < 6; ++d) c[d] = n.in[d] ? __ldg(op.offd[d] + i) : 0.0;
    } else {
        const unsigned int code = load_code(op, g, n.ix, n.iy, n.iz);
#pragma unroll
        for (int d = 0; d < 6; ++d) c[d] = ctab_s[code_field(code, op.code32, d)];
    }
}

__device__ __forceinline__ void load_ctab(const Operator& op, double* ctab_s) {
    if (!op.stored)
        for (int k = threadIdx.x; k < PF_CTAB; k += blockDim.x) ctab_s[k] = op.ctab[k];
    __syncthreads();
}

// MODE 0: r = b - A x, r~ = r, reduces b.b and r.r (step 2).  MODE 1: reduces ||b - A x||^2 only.
template <int MODE>
__global__ void __launch_bounds__(DIRECT_THREADS)
k_residual(GridDims g, Operator op, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb) {
    __shared__ double ctab_s[PF_CTAB];
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    begin_kernel(MODE == 0 ? PEND_INIT : PEND_TRUE, &S, sc_in, sc_out, rb, kv.hist, scratch);
    load_ctab(op, ctab_s);
    dd q[2] = {dd_zero(), dd_zero()};
    double rmax = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, g, ctab_s, i, n, c);
        double acc = mul(op.A0[i], kv.x[i]);
#pragma unroll
        for (int d = 0; d < 6; ++d)
            if (c[d] != 0.0) acc = add(acc, mul(c[d], kv.x[n.j[d]]));
        const double bi = kv.b[i];
        const double ri = sub(bi, acc);
        if (MODE == 0) {
            kv.r[i] = ri;
            kv.rt[i] = ri;
            dd_fma(q[0], bi, bi);
        }
        dd_fma(q[1], ri, ri);
        rmax = max_abs(rmax, ri);
    }
    store_partials<2, true>(q, rmax, scratch, rb, MODE == 0 ? PEND_INIT : PEND_TRUE);
}

template <bool PRECOND>
__global__ void __launch_bounds__(DIRECT_THREADS)
k1_direct(GridDims g, Operator op, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb) {
    __shared__ double ctab_s[PF_CTAB];
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    if (!begin_kernel(PEND_K1, &S, sc_in, sc_out, rb, kv.hist, scratch)) return;
    load_ctab(op, ctab_s);
    const bool first = S.first != 0;
    const double beta = S.beta, omega = S.omega;
    dd q[1] = {dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, g, ctab_s, i, n, c);
        const double a0 = op.A0[i];
        const double pi = p_new_at<PRECOND>(first, beta, omega, kv.r[i], kv.p_in[i], kv.v_in[i]);
        double acc = mul(a0, jacobi<PRECOND>(pi, a0));
#pragma unroll
        for (int d = 0; d < 6; ++d)
            if (c[d] != 0.0) {
                const long long j = n.j[d];
                const double pj = p_new_at<PRECOND>(first, beta, omega, kv.r[j], kv.p_in[j], kv.v_in[j]);
                acc = add(acc, mul(c[d], jacobi<PRECOND>(pj, op.A0[j])));
            }
        kv.p_out[i] = pi;
        kv.v_out[i] = acc;
        dd_fma(q[0], kv.rt[i], acc);
    }
    store_partials<1, false>(q, 0.0, scratch, rb, PEND_K1);
}

template <bool PRECOND>
__global__ void __launch_bounds__(DIRECT_THREADS)
k2_direct(GridDims g, Operator op, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb) {
    __shared__ double ctab_s[PF_CTAB];
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    if (!begin_kernel(PEND_K2, &S, sc_in, sc_out, rb, kv.hist, scratch)) return;
    load_ctab(op, ctab_s);
    const double alpha = S.alpha;
    dd q[2] = {dd_zero(), dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, g, ctab_s, i, n, c);
        const double a0 = op.A0[i];
        const double si = s_at(alpha, kv.r[i], kv.v_out[i]);
        double acc = mul(a0, jacobi<PRECOND>(si, a0));
#pragma unroll
        for (int d = 0; d < 6; ++d)
            if (c[d] != 0.0) {
                const long long j = n.j[d];
                const double sj = s_at(alpha, kv.r[j], kv.v_out[j]);
                acc = add(acc, mul(c[d], jacobi<PRECOND>(sj, op.A0[j])));
            }
        kv.t[i] = acc;
        dd_fma(q[0], acc, si);
        dd_fma(q[1], acc, acc);
    }
    store_partials<2, false>(q, 0.0, scratch, rb, PEND_K2);
}

// ---- the merged solver (pf_krylov.cuh; reading M1): two kernels per iteration -----------------------------------
// K2M = k2 that also reduces r~.t.  The current (p, v) pair is (kv.p_in, kv.v_in).
template <bool PRECOND>
__global__ void __launch_bounds__(DIRECT_THREADS)
k2m_direct(GridDims g, Operator op, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb) {
    __shared__ double ctab_s[PF_CTAB];
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    if (!begin_kernel(PEND_K2M, &S, sc_in, sc_out, rb, kv.hist, scratch)) return;
    load_ctab(op, ctab_s);
    const double alpha = S.alpha;
    dd q[3] = {dd_zero(), dd_zero(), dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, g, ctab_s, i, n, c);
        const double a0 = op.A0[i];
        const double si = s_at(alpha, kv.r[i], kv.v_in[i]);
        double acc = mul(a0, jacobi<PRECOND>(si, a0));
#pragma unroll
        for (int d = 0; d < 6; ++d)
            if (c[d] != 0.0) {
                const long long j = n.j[d];
                const double sj = s_at(alpha, kv.r[j], kv.v_in[j]);
                acc = add(acc, mul(c[d], jacobi<PRECOND>(sj, op.A0[j])));
            }
        kv.t[i] = acc;
        dd_fma(q[0], acc, si);
        dd_fma(q[1], acc, acc);
        dd_fma(q[2], kv.rt[i], acc);
    }
    store_partials<3, false>(q, 0.0, scratch, rb, PEND_K2M);
}

// K31 = steps 16-17 of iteration i fused with steps 5-11 of iteration i + 1: r' = s - omega t, y += alpha p + omega s,
// p' = r' + beta (p - omega v), v' = A M^-1 p'; reduces r~.v', r'.r' (and max |r'|), r~.r'.  r' and p' are formed at
// the node and at its six neighbours from the OLD r, p, v, t, which is why r', p', v' go to second buffers.
template <bool PRECOND>
__global__ void __launch_bounds__(DIRECT_THREADS)
k31_direct(GridDims g, Operator op, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb) {
    __shared__ double ctab_s[PF_CTAB];
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    if (!begin_kernel(PEND_K31, &S, sc_in, sc_out, rb, kv.hist, scratch)) return;
    load_ctab(op, ctab_s);
    const double alpha = S.alpha, omega = S.omega, beta = S.beta;
    dd q[3] = {dd_zero(), dd_zero(), dd_zero()};
    double rmax = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, g, ctab_s, i, n, c);
        const double a0 = op.A0[i];
        const double pi = kv.p_in[i], vi = kv.v_in[i];
        const double si = s_at(alpha, kv.r[i], vi);
        const double rn = sub(si, mul(omega, kv.t[i]));                          // step 17
        const double pn = p_new_at<PRECOND>(false, beta, omega, rn, pi, vi);     // step 9 of the next iteration
        double acc = mul(a0, jacobi<PRECOND>(pn, a0));
#pragma unroll
        for (int d = 0; d < 6; ++d)
            if (c[d] != 0.0) {
                const long long j = n.j[d];
                const double vj = kv.v_in[j];
                const double rj = sub(s_at(alpha, kv.r[j], vj), mul(omega, kv.t[j]));
                const double pj = p_new_at<PRECOND>(false, beta, omega, rj, kv.p_in[j], vj);
                acc = add(acc, mul(c[d], jacobi<PRECOND>(pj, op.A0[j])));
            }
        kv.y[i] = add(add(kv.y[i], mul(alpha, pi)), mul(omega, si));             // step 16 (reading D3)
        kv.r_out[i] = rn;
        kv.p_out[i] = pn;
        kv.v_out[i] = acc;
        const double rti = kv.rt[i];
        dd_fma(q[0], rti, acc);
        dd_fma(q[1], rn, rn);
        dd_fma(q[2], rti, rn);
        rmax = max_abs(rmax, rn);
    }
    store_partials<3, true>(q, rmax, scratch, rb, PEND_K31);
}

}  // namespace

// Steps 16-17 are pointwise; this kernel serves both kernel families.  Reads r, v, p, y, t, r~ and
// writes y, r: a pure streaming kernel, 128-bit accesses, two independent groups in flight per thread.
// With M = I the accumulator y IS x and the statement is Table 3 step 16 verbatim; with the Jacobi
// preconditioner y collects alpha p + omega s and x = x0 + M^-1 y is formed once (k_finish_x, D3).
struct K3Elem { double r, v, p, y, t, rt; };

__device__ __forceinline__ void k3_point(const K3Elem& e, double alpha, double omega, double& y_new, double& r_new,
                                         dd& q0, dd& q1, double& rmax) {
    const double s = s_at(alpha, e.r, e.v);
    y_new = add(add(e.y, mul(alpha, e.p)), mul(omega, s));       // step 16
    r_new = sub(s, mul(omega, e.t));                              // step 17
    dd_fma(q0, e.rt, r_new);
    dd_fma(q1, r_new, r_new);
    rmax = max_abs(rmax, r_new);             // ||r||_inf of Table 3 step 18 (a NaN is kept)
}

template <bool VEC, bool LOOP>
__global__ void __launch_bounds__(256, 3)
k3_update(long long n, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb) {
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    pdl_launch_dependents();
    pdl_wait();
    if (!begin_kernel<LOOP>(PEND_K3, &S, sc_in, sc_out, rb, kv.hist, scratch)) return;
    const double alpha = S.alpha, omega = S.omega;
    dd qa[2] = {dd_zero(), dd_zero()}, qb[2] = {dd_zero(), dd_zero()};
    double rmax = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long tid = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (VEC) {
        const long long n2 = n >> 1;
        const double2* r2 = reinterpret_cast<const double2*>(kv.r);
        const double2* v2 = reinterpret_cast<const double2*>(kv.v_out);
        const double2* p2 = reinterpret_cast<const double2*>(kv.p_out);
        const double2* y2 = reinterpret_cast<const double2*>(kv.y);
        const double2* t2 = reinterpret_cast<const double2*>(kv.t);
        const double2* rt2 = reinterpret_cast<const double2*>(kv.rt);
        double2* yo = reinterpret_cast<double2*>(kv.y);
        double2* ro = reinterpret_cast<double2*>(kv.r);
        long long i = tid;
        for (; i + stride < n2; i += 2 * stride) {
            const long long j = i + stride;
            const double2 ra = r2[i], va = v2[i], pa = p2[i], ya = y2[i], ta = t2[i], wa = rt2[i];
            const double2 rb2 = r2[j], vb = v2[j], pb = p2[j], yb = y2[j], tb = t2[j], wb = rt2[j];
            double2 yn, rn;
            k3_point({ra.x, va.x, pa.x, ya.x, ta.x, wa.x}, alpha, omega, yn.x, rn.x, qa[0], qa[1], rmax);
            k3_point({ra.y, va.y, pa.y, ya.y, ta.y, wa.y}, alpha, omega, yn.y, rn.y, qb[0], qb[1], rmax);
            yo[i] = yn; ro[i] = rn;
            k3_point({rb2.x, vb.x, pb.x, yb.x, tb.x, wb.x}, alpha, omega, yn.x, rn.x, qa[0], qa[1], rmax);
            k3_point({rb2.y, vb.y, pb.y, yb.y, tb.y, wb.y}, alpha, omega, yn.y, rn.y, qb[0], qb[1], rmax);
            yo[j] = yn; ro[j] = rn;
        }
        for (; i < n2; i += stride) {
            const double2 ra = r2[i], va = v2[i], pa = p2[i], ya = y2[i], ta = t2[i], wa = rt2[i];
            double2 yn, rn;
            k3_point({ra.x, va.x, pa.x, ya.x, ta.x, wa.x}, alpha, omega, yn.x, rn.x, qa[0], qa[1], rmax);
            k3_point({ra.y, va.y, pa.y, ya.y, ta.y, wa.y}, alpha, omega, yn.y, rn.y, qb[0], qb[1], rmax);
            yo[i] = yn; ro[i] = rn;
        }
        if ((n & 1) && tid == 0) {                    // odd tail
            const long long k = n - 1;
            double yn, rn;
            k3_point({kv.r[k], kv.v_out[k], kv.p_out[k], kv.y[k], kv.t[k], kv.rt[k]}, alpha, omega, yn, rn, qa[0], qa[1], rmax);
            kv.y[k] = yn; kv.r[k] = rn;
        }
    } else {
        for (long long i = tid; i < n; i += stride) {
            double yn, rn;
            k3_point({kv.r[i], kv.v_out[i], kv.p_out[i], kv.y[i], kv.t[i], kv.rt[i]}, alpha, omega, yn, rn, qa[0], qa[1], rmax);
            kv.y[i] = yn; kv.r[i] = rn;
        }
    }
    dd_add(qa[0], qb[0]);
    dd_add(qa[1], qb[1]);
    store_partials<2, true>(qa, rmax, scratch, rb, PEND_K3);
}

// One block: take the scalar step that is still pending (so that the host reads a finished state), in place.
__global__ void __launch_bounds__(256)
k_finalize(Scalars* sc, ReduceBuf rb, double* hist) {
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    begin_kernel(PEND_NONE, &S, sc, sc, rb, hist, scratch);
}

// The same at the end of a body of the device-side loop of the merged solver (pf_api.cu loop_graph): the state is then
// exact, and the body's WHILE node repeats while the solve is not over and iterations of the loop are left.  (The
// three-kernel solver keeps this call in its k3 instead; kernels that can set a conditional handle are invisible to
// Nsight Compute, so the hot kernels of the merged solver stay free of it.)
__global__ void __launch_bounds__(256)
k_finalize_loop(Scalars* sc, ReduceBuf rb, double* hist) {
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    begin_kernel(PEND_NONE, &S, sc, sc, rb, hist, scratch);
    if (threadIdx.x == 0 && rb.more)
        cudaGraphSetConditional((cudaGraphConditionalHandle)rb.more, (S.done || S.it >= S.loop_end) ? 0u : 1u);
}

// x = x + M^-1 y (reading D3).  y is exactly 0 on identity rows, so Dirichlet values of x are kept.
__global__ void __launch_bounds__(256)
k_finish_x(long long n, const double* __restrict__ A0, const double* __restrict__ y, double* __restrict__ x) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        x[i] = add(x[i], dvd(y[i], A0[i]));
}

// Rows of nx doubles <-> rows of nx + 1 doubles (odd nx, pf_api.cu bicgstab_device).
__global__ void __launch_bounds__(256)
k_widen(int nx, long long rows, const double* __restrict__ src, double* __restrict__ dst, double fill) {
    const long long total = rows * (nx + 1);
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
        const long long row = k / (nx + 1);
        const int ix = (int)(k - row * (nx + 1));
        dst[k] = ix < nx ? src[row * nx + ix] : fill;
    }
}
__global__ void __launch_bounds__(256)
k_narrow(int nx, long long rows, const double* __restrict__ src, double* __restrict__ dst) {
    const long long total = rows * nx;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < total; k += stride) {
        const long long row = k / nx;
        dst[k] = src[k + row];
    }
}

void launch_widen(cudaStream_t s, const GridDims& g, const double* src, double* dst, double fill) {
    const long long rows = (long long)g.ny * g.nz;
    const long long want = (rows * (g.nx + 1) + 255) / 256;
    ++g_launch_count;
    k_widen<<<(int)(want < 4736 ? want : 4736), 256, 0, s>>>(g.nx, rows, src, dst, fill);
}
void launch_narrow(cudaStream_t s, const GridDims& g, const double* src, double* dst) {
    const long long rows = (long long)g.ny * g.nz;
    const long long want = (rows * g.nx + 255) / 256;
    ++g_launch_count;
    k_narrow<<<(int)(want < 4736 ? want : 4736), 256, 0, s>>>(g.nx, rows, src, dst);
}

static int direct_blocks(long long n, int sm_count) {
    long long want = (n + DIRECT_THREADS - 1) / DIRECT_THREADS;
    long long cap = (long long)sm_count * 8;
    if (cap > PF_MAX_PARTIAL_BLOCKS) cap = PF_MAX_PARTIAL_BLOCKS;
    return (int)(want < cap ? (want < 1 ? 1 : want) : cap);
}

void launch_residual_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, int mode) {
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (mode == 0) { ++g_launch_count; k_residual<0><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb); }
    else           { ++g_launch_count; k_residual<1><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb); }
}

void launch_k1_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (precond) { ++g_launch_count; k1_direct<true><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb); }
    else         { ++g_launch_count; k1_direct<false><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb); }
}

void launch_k2_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (precond) { ++g_launch_count; k2_direct<true><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb); }
    else         { ++g_launch_count; k2_direct<false><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb); }
}

void launch_k2m_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    const int nb = direct_blocks(c.g.n, c.sm_count);
    ++g_launch_count;
    if (precond) k2m_direct<true><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb);
    else         k2m_direct<false><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb);
}

void launch_k31_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    const int nb = direct_blocks(c.g.n, c.sm_count);
    ++g_launch_count;
    if (precond) k31_direct<true><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb);
    else         k31_direct<false><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, sc_in, sc_out, c.rb);
}

void launch_k3(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    (void)op; (void)precond;
    // 3 blocks of 256 threads per SM, each thread two 16-byte groups in flight per vector
    long long want = (c.g.n / 2 + 255) / 256;
    long long cap = (long long)c.sm_count * 3;
    if (cap > PF_MAX_PARTIAL_BLOCKS) cap = PF_MAX_PARTIAL_BLOCKS;
    const int nb = (int)(want < cap ? (want < 1 ? 1 : want) : cap);
    const bool vec = (((uintptr_t)kv.y | (uintptr_t)kv.r | (uintptr_t)kv.v_out | (uintptr_t)kv.p_out | (uintptr_t)kv.t |
                       (uintptr_t)kv.rt) & 15u) == 0;
    ++g_launch_count;
    // inside the body of a device-side loop (c.rb.more) the instance that sets the loop condition
    auto kern = c.rb.more ? (vec ? k3_update<true, true> : k3_update<false, true>)
                          : (vec ? k3_update<true, false> : k3_update<false, false>);
    note_launch(launch_pdl(c.pdl, kern, dim3(nb), dim3(256), 0, c.stream, c.g.n, kv, sc_in, sc_out, c.rb));
}

void launch_finalize(const LaunchCtx& c, double* hist) {
    ++g_launch_count;
    k_finalize<<<1, 256, 0, c.stream>>>(c.current_scalars(), c.rb, hist);
}

void launch_finalize_loop(const LaunchCtx& c, double* hist) {
    ++g_launch_count;
    k_finalize_loop<<<1, 256, 0, c.stream>>>(c.current_scalars(), c.rb, hist);
}

void launch_finish_x(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv) {
    const int nb = direct_blocks(c.g.n, c.sm_count);
    ++g_launch_count;
    k_finish_x<<<nb, 256, 0, c.stream>>>(c.g.n, op.A0, kv.y, kv.x);
}

}  // namespace pf
