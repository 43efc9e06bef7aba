// pf_krylov_direct.cu -- "direct" Krylov kernels: one thread per node in a grid-stride loop,
// neighbours fetched straight from global memory through L1/L2.  Same arithmetic, statement for
// statement, as the tiled kernels (pf_krylov_tiled.cu); this variant is the simple one the tiled
// kernels are tested against, and the one used for grids too small to fill the tiles.
//
// One BiCGSTAB iteration (Table 3) is three launches, one per reduction point:
//   k1: steps 5-11   p = r + beta(p - omega v);  v = A M^-1 p;           reduces r~.v        (row L4)
//   k2: steps 12-14  alpha; s = r - alpha v;  t = A M^-1 s;              reduces t.s, t.t    (row L5)
//   k3: steps 15-18  omega; x += alpha M^-1 p + omega M^-1 s; r = s - omega t;
//                    reduces r~.r (step 4 of the next iteration) and r.r (step 18)            (row L6)
#include "pf_krylov.cuh"
#include "pf_launch.h"

namespace pf {

namespace {

constexpr int DIRECT_THREADS = 256;

struct Nbr {
    long long j[6];
    bool in[6];
};

__device__ __forceinline__ Nbr neighbours(const GridDims& g, long long i) {
    const int ix = (int)(i % g.nx);
    const long long q = i / g.nx;
    const int iy = (int)(q % g.ny);
    const int iz = (int)(q / g.ny);
    const long long sx = 1, sy = g.nx, sz = (long long)g.nx * g.ny;
    Nbr n;
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
__device__ __forceinline__ void row_coeffs(const Operator& op, const double* lut_s, long long i, const Nbr& n,
                                           double (&c)[6]) {
    if (op.stored) {
#pragma unroll
        for (int d = 0; d < 6; ++d) c[d] = n.in[d] ? __ldg(op.offd[d] + i) : 0.0;
    } else {
        const int ci = op.cls[i] * op.ncls;
#pragma unroll
        for (int d = 0; d < 6; ++d) c[d] = n.in[d] ? lut_s[ci + op.cls[n.j[d]]] : 0.0;
    }
}

__device__ __forceinline__ void load_lut(const Operator& op, double* lut_s) {
    if (!op.stored)
        for (int k = threadIdx.x; k < op.ncls * op.ncls; k += blockDim.x) lut_s[k] = op.lut[k];
    __syncthreads();
}

// MODE 0: r = b - A x, r~ = r, reduces b.b and r.r (step 2).  MODE 1: reduces ||b - A x||^2 only.
template <int MODE>
__global__ void __launch_bounds__(DIRECT_THREADS)
k_residual(GridDims g, Operator op, KrylovVecs kv, Scalars* sc, ReduceBuf rb) {
    __shared__ double lut_s[PF_MAX_CLASSES * PF_MAX_CLASSES];
    __shared__ dd scratch[2 * 32];
    load_lut(op, lut_s);
    dd q[2] = {dd_zero(), dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, lut_s, i, n, c);
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
    }
    if (grid_reduce_dd<2>(q, scratch, rb)) {
        if (MODE == 0) finish_init(sc, kv.hist, dd_round(q[0]), dd_round(q[1]));
        else sc->true_rr = dd_round(q[1]);
    }
}

template <bool PRECOND>
__global__ void __launch_bounds__(DIRECT_THREADS)
k1_direct(GridDims g, Operator op, KrylovVecs kv, Scalars* sc, ReduceBuf rb) {
    if (sc->done) return;
    __shared__ double lut_s[PF_MAX_CLASSES * PF_MAX_CLASSES];
    __shared__ dd scratch[32];
    load_lut(op, lut_s);
    const bool first = sc->first != 0;
    const double beta = sc->beta, omega = sc->omega;
    dd q[1] = {dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, lut_s, i, n, c);
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
    if (grid_reduce_dd<1>(q, scratch, rb)) finish_k1(sc, dd_round(q[0]));
}

template <bool PRECOND>
__global__ void __launch_bounds__(DIRECT_THREADS)
k2_direct(GridDims g, Operator op, KrylovVecs kv, Scalars* sc, ReduceBuf rb) {
    if (sc->done) return;
    __shared__ double lut_s[PF_MAX_CLASSES * PF_MAX_CLASSES];
    __shared__ dd scratch[2 * 32];
    load_lut(op, lut_s);
    const double alpha = sc->alpha;
    dd q[2] = {dd_zero(), dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        Nbr n = neighbours(g, i);
        double c[6];
        row_coeffs(op, lut_s, i, n, c);
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
    if (grid_reduce_dd<2>(q, scratch, rb)) finish_k2(sc, dd_round(q[0]), dd_round(q[1]));
}

}  // namespace

// Steps 16-17 are pointwise; this kernel serves both kernel families.
template <bool PRECOND>
__global__ void __launch_bounds__(256)
k3_update(long long n, const double* __restrict__ A0, KrylovVecs kv, Scalars* sc, ReduceBuf rb) {
    if (sc->done) return;
    __shared__ dd scratch[2 * 32];
    const double alpha = sc->alpha, omega = sc->omega;
    dd q[2] = {dd_zero(), dd_zero()};
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double a0 = PRECOND ? A0[i] : 1.0;
        const double s = s_at(alpha, kv.r[i], kv.v_out[i]);
        const double ph = jacobi<PRECOND>(kv.p_out[i], a0);
        const double sh = jacobi<PRECOND>(s, a0);
        kv.x[i] = add(add(kv.x[i], mul(alpha, ph)), mul(omega, sh));   // step 16
        const double rn = sub(s, mul(omega, kv.t[i]));                  // step 17
        kv.r[i] = rn;
        dd_fma(q[0], kv.rt[i], rn);
        dd_fma(q[1], rn, rn);
    }
    if (grid_reduce_dd<2>(q, scratch, rb)) finish_k3(sc, kv.hist, dd_round(q[0]), dd_round(q[1]));
}

static int direct_blocks(long long n, int sm_count) {
    long long want = (n + DIRECT_THREADS - 1) / DIRECT_THREADS;
    long long cap = (long long)sm_count * 8;
    if (cap > PF_MAX_PARTIAL_BLOCKS) cap = PF_MAX_PARTIAL_BLOCKS;
    return (int)(want < cap ? (want < 1 ? 1 : want) : cap);
}

void launch_residual_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, int mode) {
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (mode == 0) { ++g_launch_count; k_residual<0><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb); }
    else           { ++g_launch_count; k_residual<1><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb); }
}

void launch_k1_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (precond) { ++g_launch_count; k1_direct<true><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb); }
    else         { ++g_launch_count; k1_direct<false><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb); }
}

void launch_k2_direct(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (precond) { ++g_launch_count; k2_direct<true><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb); }
    else         { ++g_launch_count; k2_direct<false><<<nb, DIRECT_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb); }
}

void launch_k3(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const int nb = direct_blocks(c.g.n, c.sm_count);
    if (precond) { ++g_launch_count; k3_update<true><<<nb, 256, 0, c.stream>>>(c.g.n, op.A0, kv, c.sc, c.rb); }
    else         { ++g_launch_count; k3_update<false><<<nb, 256, 0, c.stream>>>(c.g.n, op.A0, kv, c.sc, c.rb); }
}

}  // namespace pf
