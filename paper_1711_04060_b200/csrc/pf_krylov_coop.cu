// pf_krylov_coop.cu -- one persistent kernel for a whole Jacobi-BiCGSTAB solve on small grids
// (on the GPU the solver's time goes to matvecs, inner products and
// synchronisation -- on a grid of <= 64^3 nodes the three launches per iteration of the other kernel families
// ARE the time).
//
// The box is cut into one brick per block, at most one block per SM, launched cooperatively so that all blocks
// are resident.  A block keeps the vectors of its brick (r, p, v, y, r~, t, the diagonal and the stencil codes)
// in shared memory for the whole solve; the arithmetic is Table 3 statement for statement,
// the same device functions as the direct kernels (pf_krylov.cuh), so the iterates are bit-identical to theirs.
// What crosses blocks:
//   * halo values of the vector a matvec is applied to.  They are not exchanged but recomputed (as the direct
//     and tiled kernels do at their tile edges): every block also writes its r, p, v to the global vectors,
//     and a neighbour forms p^_j = (r_j + beta(p_j - omega v_j))/a0_j or s^_j = (r_j - alpha v_j)/a0_j of its
//     halo nodes from them.  p and v alternate between two global buffers, r is only written in a phase in
//     which no block reads halos, so no exchange barrier is needed: three grid-wide barriers per iteration,
//     one per reduction point.
//   * the inner products.  Barrier and reduction are one step (sync_reduce): a block writes its double-double
//     partial sums to its record, thread 0 adds 1 to an arrival counter (after a fence) and waits until the
//     counter shows that all blocks of this generation have arrived; then thread b of every block takes block
//     b's record, and every block sums the records in the same order and takes the same scalar step (alpha,
//     omega, beta, the convergence test), so all blocks leave the loop in the same iteration.
// A wait is bounded: a block that does not see the arrivals within about a second sets the abort flag and leaves
// (the host reports PF_ERR_CUDA); the cooperative launch makes that unreachable in normal operation.
//
// Measured (B200, profiles/r1_coop.md): a barrier-reduction costs 2.5-3.5 us (two block-wide double-double
// trees, a fence, the atomic round trip, the record reads), so an iteration costs 12 us at 32^3 and 19 us at
// 64^3 against 16-22 / 24 us for three launches; a flag per block polled by all blocks was 2x slower (hot lines),
// cooperative_groups' grid.sync() alone costs 1.2 us.
#include <algorithm>
#include <cstring>
#include "pf_krylov.cuh"
#include "pf_launch.h"

namespace pf {

namespace {

constexpr unsigned COOP_SPIN_LIMIT = 1u << 22;
constexpr int COOP_MAX_THREADS = 1024;
constexpr int COOP_MAX_BLOCKS = 256;            // flags / records reserved per generation

struct CoopArgs {
    GridDims g;
    Operator op;
    KrylovVecs kv;
    const Scalars* sc_in;
    Scalars* sc_out;
    dd* rec;                 // [4 generations][nblk][3] partial records
    unsigned long long* count;   // arrivals since the launch
    int* abort;
    int nbx, nby, nbz;       // bricks per direction
    int vmax, hmax, nhmax;   // array extents in shared memory (largest brick)
};

__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_relaxed_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}

// Grid-wide barrier + reduction.  In: this thread's sums q (and maximum m).  Out (thread 0): totals over all
// blocks, the same bits in every block.  Returns false if the wait timed out.  Every global write the block
// made before the call is visible to every block after it.  One arrival counter (thread 0 of a block adds 1 and
// waits for gen * nblk), then thread b of every block takes block b's record.
template <int NQ, bool MAX>
__device__ __forceinline__ bool sync_reduce(dd (&q)[NQ], double& m, unsigned gen, const CoopArgs& a, dd* scratch) {
    const int nblk = (int)gridDim.x;
    __shared__ int ok_s;
    double* mxs = reinterpret_cast<double*>(scratch + 2 * 32);
    block_reduce_dd<NQ>(q, scratch);
    if (MAX) m = block_reduce_max(m, mxs);
    if (threadIdx.x == 0) {
        dd* rec = a.rec + ((size_t)(gen & 3u) * COOP_MAX_BLOCKS + blockIdx.x) * 3;
#pragma unroll
        for (int k = 0; k < NQ; ++k) rec[k] = q[k];
        if (MAX) { dd pm; pm.hi = m; pm.lo = 0.0; rec[NQ] = pm; }
        __threadfence();
        atomicAdd(a.count, 1ull);
        const unsigned long long target = (unsigned long long)gen * (unsigned)nblk;
        unsigned spins = 0;
        int ok = 1;
        while (ld_relaxed_u64(a.count) < target)
            if (++spins > COOP_SPIN_LIMIT) { ok = 0; *a.abort = 1; break; }
        (void)ld_acquire_u64(a.count);          // orders everything after the barrier behind the arrivals
        ok_s = ok;
    }
    __syncthreads();
    if (!ok_s) return false;
#pragma unroll
    for (int k = 0; k < NQ; ++k) q[k] = dd_zero();
    m = 0.0;
    for (int b = threadIdx.x; b < nblk; b += blockDim.x) {
        const double2* rec = reinterpret_cast<const double2*>(a.rec + ((size_t)(gen & 3u) * COOP_MAX_BLOCKS + b) * 3);
        double2 w[NQ + (MAX ? 1 : 0)];
#pragma unroll
        for (int k = 0; k < NQ + (MAX ? 1 : 0); ++k) w[k] = __ldcg(rec + k);
#pragma unroll
        for (int k = 0; k < NQ; ++k) { dd part; part.hi = w[k].x; part.lo = w[k].y; dd_add(q[k], part); }
        if (MAX) m = max_abs(m, w[NQ].x);
    }
    block_reduce_dd<NQ>(q, scratch, (nblk + 31) >> 5);     // thread b holds block b's record
    if (MAX) m = block_reduce_max(m, mxs, (nblk + 31) >> 5);
    return true;
}

// Bounds of brick k of nb along an axis of n nodes (balanced split, never empty for nb <= n).
__host__ __device__ __forceinline__ int brick_lo(int k, int nb, int n) { return (int)((long long)k * n / nb); }

// Shared-memory image of a brick.  u and aH are indexed over the brick plus one halo layer (strides 1, hx,
// hx*hy); the other arrays over the brick's own nodes in x-fastest order.
struct Brick {
    double *r, *p, *v, *y, *rt, *t;      // own nodes
    double *aH, *u;                      // halo'd: diagonal (1.0 outside the box), operand of the matvec
    unsigned* code;                      // own nodes: six coefficient indices (pf_common.cuh Operator)
    int* gidx;                           // own nodes: global index
    int2* hlist;                         // halo nodes inside the box: (index into u, global index)
    unsigned short* uidx;                // own nodes: index into u
    int V, nh, hx, hxy;
};

__host__ __device__ inline size_t coop_smem_bytes(int vmax, int hmax, int nhmax) {
    // vmax is even, so every array below starts on an 8-byte boundary
    return (size_t)vmax * (6 * 8 + 4 + 4 + 2) + (size_t)hmax * 16 + (size_t)nhmax * 8 + 16;
}

// Row i of A applied to the halo'd operand u (Table 3 steps 11 and 14; same order of terms as the direct kernels:
// diagonal, then faces 1..6, zero coefficients skipped).
__device__ __forceinline__ double brick_row(const Brick& B, const double* ctab_s, int code32, int e, int ui) {
    const unsigned code = B.code[e];
    double acc = mul(B.aH[ui], B.u[ui]);
    const int off[6] = {1, -1, -B.hx, B.hx, -B.hxy, B.hxy};
#pragma unroll
    for (int d = 0; d < 6; ++d) {
        const double c = ctab_s[code_field(code, code32, d)];
        if (c != 0.0) acc = add(acc, mul(c, B.u[ui + off[d]]));
    }
    return acc;
}

template <bool PRECOND>
__global__ void __launch_bounds__(COOP_MAX_THREADS, 1) k_solve_coop(const CoopArgs a) {
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ dd scratch[3 * 32];
    __shared__ Scalars S;
    __shared__ double ctab_s[PF_CTAB];
    __shared__ int nh_s;
    const int tid = threadIdx.x, NT = blockDim.x;
    const GridDims g = a.g;
    const KrylovVecs kv = a.kv;

    // ---- this block's brick ------------------------------------------------------------------------
    const int bid = blockIdx.x;
    const int kx = bid % a.nbx, ky = (bid / a.nbx) % a.nby, kz = bid / (a.nbx * a.nby);
    const int x0 = brick_lo(kx, a.nbx, g.nx), bx = brick_lo(kx + 1, a.nbx, g.nx) - x0;
    const int y0 = brick_lo(ky, a.nby, g.ny), by = brick_lo(ky + 1, a.nby, g.ny) - y0;
    const int z0 = brick_lo(kz, a.nbz, g.nz), bz = brick_lo(kz + 1, a.nbz, g.nz) - z0;
    Brick B;
    B.V = bx * by * bz; B.hx = bx + 2; B.hxy = (bx + 2) * (by + 2);
    const int H = B.hxy * (bz + 2);
    {
        double* d = reinterpret_cast<double*>(smem_raw);
        B.r = d; d += a.vmax; B.p = d; d += a.vmax; B.v = d; d += a.vmax; B.y = d; d += a.vmax;
        B.rt = d; d += a.vmax; B.t = d; d += a.vmax; B.aH = d; d += a.hmax; B.u = d; d += a.hmax;
        B.hlist = reinterpret_cast<int2*>(d);
        B.code = reinterpret_cast<unsigned*>(B.hlist + a.nhmax);
        B.gidx = reinterpret_cast<int*>(B.code + a.vmax);
        B.uidx = reinterpret_cast<unsigned short*>(B.gidx + a.vmax);
    }
    constexpr int NWORDS = (int)(sizeof(Scalars) / sizeof(int));
    if (tid < NWORDS) reinterpret_cast<int*>(&S)[tid] = reinterpret_cast<const int*>(a.sc_in)[tid];
    if (tid < PF_CTAB) ctab_s[tid] = a.op.ctab[tid];
    if (tid == 0) nh_s = 0;
    __syncthreads();
    for (int e = tid; e < B.V; e += NT) {
        const int ex = e % bx, q = e / bx, ey = q % by, ez = q / by;
        const int gx = x0 + ex, gy = y0 + ey, gz = z0 + ez;
        B.gidx[e] = gx + g.nx * (gy + g.ny * gz);
        B.uidx[e] = (unsigned short)((ex + 1) + B.hx * (ey + 1) + B.hxy * (ez + 1));
        B.code[e] = load_code(a.op, g, gx, gy, gz);
    }
    for (int c = tid; c < H; c += NT) {
        const int cx = c % B.hx, q = c / B.hx, cy = q % (by + 2), cz = q / (by + 2);
        const int gx = x0 + cx - 1, gy = y0 + cy - 1, gz = z0 + cz - 1;
        const bool inbox = gx >= 0 && gx < g.nx && gy >= 0 && gy < g.ny && gz >= 0 && gz < g.nz;
        const int outside = (cx == 0 || cx == bx + 1) + (cy == 0 || cy == by + 1) + (cz == 0 || cz == bz + 1);
        const int gi = gx + g.nx * (gy + g.ny * gz);
        B.aH[c] = (inbox && outside <= 1) ? a.op.A0[gi] : 1.0;
        B.u[c] = 0.0;
        if (inbox && outside == 1) B.hlist[atomicAdd(&nh_s, 1)] = make_int2(c, gi);
    }
    __syncthreads();
    B.nh = nh_s;
    const bool lead = bid == 0;
    double* hist = lead ? kv.hist : nullptr;
    unsigned gen = 0;

    // ---- step 2: r0 = b - A x0, r~ = r0; ||b||, ||r0|| ---------------------------------------------
    {
        for (int h = tid; h < B.nh; h += NT) { const int2 hh = B.hlist[h]; B.u[hh.x] = kv.x[hh.y]; }
        for (int e = tid; e < B.V; e += NT) B.u[B.uidx[e]] = kv.x[B.gidx[e]];
        __syncthreads();
        dd q[2] = {dd_zero(), dd_zero()};
        double rmax = 0.0;
        for (int e = tid; e < B.V; e += NT) {
            const int ui = B.uidx[e], gi = B.gidx[e];
            const double bi = kv.b[gi];
            const double ri = sub(bi, brick_row(B, ctab_s, a.op.code32, e, ui));
            B.r[e] = ri; B.rt[e] = ri;
            B.p[e] = 0.0; B.v[e] = 0.0; B.t[e] = 0.0;
            B.y[e] = PRECOND ? 0.0 : B.u[ui];
            kv.r[gi] = ri;
            dd_fma(q[0], bi, bi);
            dd_fma(q[1], ri, ri);
            rmax = max_abs(rmax, ri);
        }
        if (!sync_reduce<2, true>(q, rmax, ++gen, a, scratch)) return;
        if (tid == 0) finish_init(&S, hist, dd_round(q[0]), dd_round(q[1]), rmax);
        __syncthreads();
    }

    // ---- iterations ----------------------------------------------------------------------------------
    int parity = 0;
    while (!S.done) {
        const double* p_in = parity ? kv.p_out : kv.p_in;
        double* p_out = parity ? kv.p_in : kv.p_out;
        const double* v_in = parity ? kv.v_out : kv.v_in;
        double* v_out = parity ? kv.v_in : kv.v_out;
        {   // steps 5-11: p = r + beta(p - omega v); v = A M^-1 p; r~.v
            const bool first = S.first != 0;
            const double beta = S.beta, omega = S.omega;
            for (int h = tid; h < B.nh; h += NT) {
                const int2 hh = B.hlist[h];
                const double rj = __ldcg(kv.r + hh.y);
                const double pj = first ? 0.0 : __ldcg(p_in + hh.y);
                const double vj = first ? 0.0 : __ldcg(v_in + hh.y);
                B.u[hh.x] = jacobi<PRECOND>(p_new_at<PRECOND>(first, beta, omega, rj, pj, vj), B.aH[hh.x]);
            }
            for (int e = tid; e < B.V; e += NT) {
                const int ui = B.uidx[e];
                const double pn = p_new_at<PRECOND>(first, beta, omega, B.r[e], B.p[e], B.v[e]);
                B.p[e] = pn;
                B.u[ui] = jacobi<PRECOND>(pn, B.aH[ui]);
                p_out[B.gidx[e]] = pn;
            }
            __syncthreads();
            dd q[1] = {dd_zero()};
            double m = 0.0;
            for (int e = tid; e < B.V; e += NT) {
                const double vn = brick_row(B, ctab_s, a.op.code32, e, B.uidx[e]);
                B.v[e] = vn;
                v_out[B.gidx[e]] = vn;
                dd_fma(q[0], B.rt[e], vn);
            }
            if (!sync_reduce<1, false>(q, m, ++gen, a, scratch)) return;
            if (tid == 0) finish_k1(&S, dd_round(q[0]));
            __syncthreads();
            if (S.done) break;
        }
        {   // steps 12-14: s = r - alpha v; t = A M^-1 s; t.s, t.t
            const double alpha = S.alpha;
            for (int h = tid; h < B.nh; h += NT) {
                const int2 hh = B.hlist[h];
                const double sj = s_at(alpha, __ldcg(kv.r + hh.y), __ldcg(v_out + hh.y));
                B.u[hh.x] = jacobi<PRECOND>(sj, B.aH[hh.x]);
            }
            for (int e = tid; e < B.V; e += NT) {
                const int ui = B.uidx[e];
                B.u[ui] = jacobi<PRECOND>(s_at(alpha, B.r[e], B.v[e]), B.aH[ui]);
            }
            __syncthreads();
            dd q[2] = {dd_zero(), dd_zero()};
            double m = 0.0;
            for (int e = tid; e < B.V; e += NT) {
                const double tn = brick_row(B, ctab_s, a.op.code32, e, B.uidx[e]);
                const double si = s_at(alpha, B.r[e], B.v[e]);
                B.t[e] = tn;
                dd_fma(q[0], tn, si);
                dd_fma(q[1], tn, tn);
            }
            if (!sync_reduce<2, false>(q, m, ++gen, a, scratch)) return;
            if (tid == 0) finish_k2(&S, dd_round(q[0]), dd_round(q[1]));
            __syncthreads();
            if (S.done) break;            // non-finite t.s or t.t (reading D7)
        }
        {   // steps 15-18: y += alpha p + omega s (reading D3); r = s - omega t; r~.r, r.r, ||r||_inf
            const double alpha = S.alpha, omega = S.omega;
            dd q[2] = {dd_zero(), dd_zero()};
            double rmax = 0.0;
            for (int e = tid; e < B.V; e += NT) {
                const double s = s_at(alpha, B.r[e], B.v[e]);
                B.y[e] = add(add(B.y[e], mul(alpha, B.p[e])), mul(omega, s));
                const double rn = sub(s, mul(omega, B.t[e]));
                B.r[e] = rn;
                kv.r[B.gidx[e]] = rn;
                dd_fma(q[0], B.rt[e], rn);
                dd_fma(q[1], rn, rn);
                rmax = max_abs(rmax, rn);
            }
            if (!sync_reduce<2, true>(q, rmax, ++gen, a, scratch)) return;
            if (tid == 0) finish_k3(&S, hist, dd_round(q[0]), dd_round(q[1]), rmax);
            __syncthreads();
        }
        parity ^= 1;
    }

    // ---- x = x0 + M^-1 y (D3); with M = I y is x itself ------------------------------------------------
    for (int e = tid; e < B.V; e += NT) {
        const int gi = B.gidx[e];
        kv.x[gi] = PRECOND ? add(kv.x[gi], dvd(B.y[e], B.aH[B.uidx[e]])) : B.y[e];
    }
    if (lead && tid == 0) {
        S.pending = PEND_NONE; S.pending_nblk = 0; S.fault = 0;
        *a.sc_out = S;
    }
}

int ceil_div(int a, int b) { return (a + b - 1) / b; }

}  // namespace

// Decomposition: bricks per direction with at most max_blocks bricks, the largest brick within the shared
// memory of one SM, the work of the largest brick (own nodes + recomputed halo nodes) minimal.
bool coop_plan(const GridDims& g, const Operator& op, int max_blocks, size_t smem_cap, CoopPlan* out) {
    if (op.stored || g.n > (long long)max_blocks * 4096 || g.n >= (1ll << 31)) return false;
    if (max_blocks > COOP_MAX_BLOCKS) max_blocks = COOP_MAX_BLOCKS;
    double best = 1e300;
    for (int nbz = 1; nbz <= std::min(g.nz, max_blocks); ++nbz)
        for (int nby = 1; nby <= std::min(g.ny, max_blocks / nbz); ++nby)
            for (int nbx = 1; nbx <= std::min(g.nx, max_blocks / (nbz * nby)); ++nbx) {
                const int bx = ceil_div(g.nx, nbx), by = ceil_div(g.ny, nby), bz = ceil_div(g.nz, nbz);
                const int V = (bx * by * bz + 1) & ~1, H = (bx + 2) * (by + 2) * (bz + 2);
                const int nh = 2 * (bx * by + by * bz + bx * bz);
                const size_t smem = coop_smem_bytes(V, H, nh);
                if (smem > smem_cap || H > 65535) continue;
                // a halo node costs about as much as an own node in each of the two matvec phases
                // (ties: the longest bricks along x, the contiguous direction)
                const double cost = V + 0.7 * nh + 1e-3 * nbx;
                if (cost < best) {
                    best = cost;
                    out->nbx = nbx; out->nby = nby; out->nbz = nbz;
                    out->vmax = V; out->hmax = H; out->nhmax = nh; out->smem = smem;
                }
            }
    if (best == 1e300) return false;
    const int v = out->vmax;
    out->threads = v <= 256 ? 256 : (v <= 1024 ? 512 : COOP_MAX_THREADS);
    return true;
}

size_t coop_smem_cap() {
    int dev = 0, cap = 0, coop = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return 0;
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) return 0;
    if (cudaDeviceGetAttribute(&cap, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) != cudaSuccess) return 0;
    return cap > 4096 ? (size_t)cap - 4096 : 0;        // static shared memory of the kernel comes on top
}

// Whole solve: Table 3 from step 2 to the last x update.  Reads the initial scalars from the current copy and
// leaves the final ones in the other (which becomes the current one).
cudaError_t launch_solve_coop(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond,
                              const CoopPlan& plan) {
    CoopArgs a;
    std::memset(&a, 0, sizeof(a));
    a.g = c.g; a.op = op; a.kv = kv;
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    a.sc_in = sc_in; a.sc_out = sc_out;
    a.rec = c.rb.partial;
    a.count = reinterpret_cast<unsigned long long*>(c.rb.partial + (size_t)4 * COOP_MAX_BLOCKS * 3);
    a.abort = c.rb.fault;
    a.nbx = plan.nbx; a.nby = plan.nby; a.nbz = plan.nbz;
    a.vmax = plan.vmax; a.hmax = plan.hmax; a.nhmax = plan.nhmax;
    const int nblk = plan.nbx * plan.nby * plan.nbz;
    cudaError_t e = cudaMemsetAsync(a.count, 0, sizeof(unsigned long long), c.stream);
    if (e != cudaSuccess) return e;
    const void* fn = precond ? reinterpret_cast<const void*>(&k_solve_coop<true>)
                             : reinterpret_cast<const void*>(&k_solve_coop<false>);
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)plan.smem);
    if (e != cudaSuccess) return e;
    void* args[] = {&a};
    e = cudaLaunchCooperativeKernel(fn, dim3(nblk), dim3(plan.threads), args, plan.smem, c.stream);
    if (e == cudaSuccess) ++g_launch_count;
    return e;
}

}  // namespace pf
