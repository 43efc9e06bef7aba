// pf_krylov_tiled.cu -- the fused stencil kernels of the BiCGSTAB iteration, tiled for B200.
//
// Work decomposition: the xy plane is cut into tiles of TX x TY nodes (TX = 64: one warp owns one
// 512-byte row segment, each lane two x-adjacent nodes, so every global access is a 128-bit
// coalesced load/store); a block marches its tile along z over a chunk of planes.
//
// What is fused (rows L3-L5 of DESIGN.md): the vector update that precedes a matvec in Table 3
// is recomputed on the fly at the tile AND at its one-node halo ring, so the
// updated vector is never written and re-read for the matvec:
//   MODE_K1  u = M^-1 (r + beta (p - omega v))  (steps 5-9, Jacobi Q2), v' = A u (step 11), r~.v'
//   MODE_K2  u = M^-1 (r - alpha v)             (step 13),            t  = A u (step 14), t.s, t.t
//   MODE_R0  u = x,  r = b - A u, r~ = r, b.b, r.r (step 2);  MODE_R1: ||b - A x||^2 only
// The plane of u being differenced sits in shared memory (xy neighbours); the z neighbours stay in
// registers of the marching thread.  Next-plane operands are requested before the current plane is
// differenced, so about one plane per SM of loads is always in flight.
//
// Arithmetic is the same statement-for-statement as the direct kernels (pf_krylov_direct.cu): both
// families give bit-identical vectors.
#include "pf_krylov.cuh"
#include "pf_launch.h"
#include <algorithm>

namespace pf {

namespace {

constexpr int TX = 64;               // tile width in nodes (32 lanes x 2)
constexpr int TY = 16;               // tile height = warps per block
constexpr int TILE_THREADS = 32 * TY;
constexpr int SW = TX + 2;           // shared row: halo column, TX nodes, halo column
constexpr int SH = TY + 2;
constexpr int CLS_OUT = 2 * PF_MAX_PALETTE;
static_assert(TY == 16 && TX == 64, "halo duty of warps 0-2 is written for 64 x 16 tiles");

enum { MODE_R0 = 0, MODE_R1 = 1, MODE_K1 = 2, MODE_K2 = 3 };

struct Raw2 { double2 r, p, v, a; };   // operands of u at two x-adjacent nodes
struct Raw1 { double r, p, v, a; };

template <int MODE, bool PRECOND>
__device__ __forceinline__ double u_of(double r, double p, double v, double a, bool first, double c1, double c2,
                                       double& numer) {
    if (MODE == MODE_K1) { numer = p_new_at<PRECOND>(first, c1, c2, r, p, v); return jacobi<PRECOND>(numer, a); }
    if (MODE == MODE_K2) { numer = s_at(c1, r, v); return jacobi<PRECOND>(numer, a); }
    numer = r;           // residual modes: the field is x itself (passed in r)
    return r;
}

template <int MODE, bool PRECOND, bool STORED>
__global__ void __launch_bounds__(TILE_THREADS, 1)
k_tiled(GridDims g, Operator op, KrylovVecs kv, Scalars* sc, ReduceBuf rb, int zchunk) {
    if (MODE >= MODE_K1 && sc->done) return;
    __shared__ double u_s[2][SH][SW];
    __shared__ uint8_t c_s[2][SH][SW + 6];
    __shared__ double lut_s[PF_MAX_CLASSES * PF_MAX_CLASSES];
    __shared__ dd scratch[2 * 32];

    const int lane = threadIdx.x & 31, ty = threadIdx.x >> 5;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, g.nz);
    if (!STORED) for (int k = threadIdx.x; k < op.ncls * op.ncls; k += TILE_THREADS) lut_s[k] = op.lut[k];

    // which stencil operand goes where
    const double* fr; const double* fp = nullptr; const double* fv = nullptr; const double* fa = op.A0;
    bool first = false; double c1 = 0.0, c2 = 0.0;
    if (MODE == MODE_K1) { fr = kv.r; fp = kv.p_in; fv = kv.v_in; first = sc->first != 0; c1 = sc->beta; c2 = sc->omega; }
    else if (MODE == MODE_K2) { fr = kv.r; fv = kv.v_out; c1 = sc->alpha; }
    else { fr = kv.x; }
    constexpr bool NEED_P = MODE == MODE_K1, NEED_V = MODE == MODE_K1 || MODE == MODE_K2;
    constexpr bool NEED_A = (MODE == MODE_K1 || MODE == MODE_K2) && PRECOND;

    // own slot: nodes (x, y) and (x+1, y); nx is even so both are inside or both outside
    const int x = x0 + 2 * lane, y = y0 + ty;
    const bool own_ok = x < g.nx && y < g.ny;
    const long long plane = (long long)g.nx * g.ny;
    const long long own_off = x + (long long)g.nx * y;
    // halo slot: warp 0 -> row y0-1, warp 1 -> row y0+TY (two nodes per lane); warp 2 -> the columns
    // x0-1 (lanes 0..15) and x0+TX (lanes 16..31), one node per lane
    int hx = 0, hy = 0, hsx = 0, hsy = 0;
    bool h_two = false, h_ok = false;
    if (ty == 0) { hx = x; hy = y0 - 1; hsx = 1 + 2 * lane; hsy = 0; h_two = true; h_ok = hx < g.nx && hy >= 0; }
    else if (ty == 1) { hx = x; hy = y0 + TY; hsx = 1 + 2 * lane; hsy = SH - 1; h_two = true; h_ok = hx < g.nx && hy < g.ny; }
    else if (ty == 2) {
        const int row = lane & 15;
        hy = y0 + row; hsy = 1 + row;
        if (lane < 16) { hx = x0 - 1; hsx = 0; } else { hx = x0 + TX; hsx = SW - 1; }
        h_ok = hx >= 0 && hx < g.nx && hy < g.ny;
    }
    const bool h_any = ty <= 2;
    const long long h_off = hx + (long long)g.nx * hy;

    Raw2 own; Raw2 hal;                   // operands of the next plane, in flight
    uchar2 own_c = make_uchar2(CLS_OUT, CLS_OUT), hal_c = make_uchar2(CLS_OUT, CLS_OUT);
    const double2 zero2 = make_double2(0.0, 0.0);

    auto request = [&](int z) {            // issue the loads of plane z
        const bool zin = z >= 0 && z < g.nz;
        own.r = own.p = own.v = zero2; own.a = make_double2(1.0, 1.0);
        hal.r = hal.p = hal.v = zero2; hal.a = make_double2(1.0, 1.0);
        own_c = make_uchar2(CLS_OUT, CLS_OUT); hal_c = make_uchar2(CLS_OUT, CLS_OUT);
        if (zin && own_ok) {
            const long long i = own_off + plane * z;
            own.r = *reinterpret_cast<const double2*>(fr + i);
            if (NEED_P) own.p = *reinterpret_cast<const double2*>(fp + i);
            if (NEED_V) own.v = *reinterpret_cast<const double2*>(fv + i);
            own.a = *reinterpret_cast<const double2*>(fa + i);     // also the diagonal of the row
            if (!STORED) own_c = *reinterpret_cast<const uchar2*>(op.cls + i);
        }
        if (h_any && zin && h_ok) {
            const long long i = h_off + plane * z;
            if (h_two) {
                hal.r = *reinterpret_cast<const double2*>(fr + i);
                if (NEED_P) hal.p = *reinterpret_cast<const double2*>(fp + i);
                if (NEED_V) hal.v = *reinterpret_cast<const double2*>(fv + i);
                if (NEED_A) hal.a = *reinterpret_cast<const double2*>(fa + i);
                if (!STORED) hal_c = *reinterpret_cast<const uchar2*>(op.cls + i);
            } else {
                hal.r.x = fr[i];
                if (NEED_P) hal.p.x = fp[i];
                if (NEED_V) hal.v.x = fv[i];
                if (NEED_A) hal.a.x = fa[i];
                if (!STORED) hal_c.x = op.cls[i];
            }
        }
    };

    // u of the plane whose operands are in (own, hal); own nodes -> registers (+ shared), halo -> shared
    double u_dn[2] = {0, 0}, u_c[2] = {0, 0}, u_up[2] = {0, 0};
    double n_c[2] = {0, 0}, n_up[2] = {0, 0};              // numerators: p' (K1) or s (K2)
    double a_c[2] = {1, 1}, a_up[2] = {1, 1};
    uint8_t k_dn[2] = {CLS_OUT, CLS_OUT}, k_c[2] = {CLS_OUT, CLS_OUT}, k_up[2] = {CLS_OUT, CLS_OUT};

    auto consume = [&](int z, bool to_shared) {
        const int buf = z & 1;
        u_up[0] = u_of<MODE, PRECOND>(own.r.x, own.p.x, own.v.x, own.a.x, first, c1, c2, n_up[0]);
        u_up[1] = u_of<MODE, PRECOND>(own.r.y, own.p.y, own.v.y, own.a.y, first, c1, c2, n_up[1]);
        a_up[0] = own.a.x; a_up[1] = own.a.y;
        k_up[0] = own_c.x; k_up[1] = own_c.y;
        if (MODE == MODE_K1 && own_ok && z >= z0 && z < z1)       // p' is an output of steps 5-9
            *reinterpret_cast<double2*>(kv.p_out + own_off + plane * z) = make_double2(n_up[0], n_up[1]);
        if (to_shared) {
            u_s[buf][1 + ty][1 + 2 * lane] = u_up[0];
            u_s[buf][1 + ty][2 + 2 * lane] = u_up[1];
            if (!STORED) { c_s[buf][1 + ty][1 + 2 * lane] = own_c.x; c_s[buf][1 + ty][2 + 2 * lane] = own_c.y; }
            if (h_any) {
                double dummy;
                u_s[buf][hsy][hsx] = u_of<MODE, PRECOND>(hal.r.x, hal.p.x, hal.v.x, hal.a.x, first, c1, c2, dummy);
                if (!STORED) c_s[buf][hsy][hsx] = hal_c.x;
                if (h_two) {
                    u_s[buf][hsy][hsx + 1] = u_of<MODE, PRECOND>(hal.r.y, hal.p.y, hal.v.y, hal.a.y, first, c1, c2, dummy);
                    if (!STORED) c_s[buf][hsy][hsx + 1] = hal_c.y;
                }
            }
        }
    };
    auto rotate = [&]() {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            u_dn[e] = u_c[e]; u_c[e] = u_up[e]; n_c[e] = n_up[e]; a_c[e] = a_up[e];
            k_dn[e] = k_c[e]; k_c[e] = k_up[e];
        }
    };

    dd q[2] = {dd_zero(), dd_zero()};

    request(z0 - 1);
    __syncthreads();                       // lut_s
    consume(z0 - 1, false); rotate();
    request(z0);
    consume(z0, true); rotate();
    request(z0 + 1);
    __syncthreads();

    for (int z = z0; z < z1; ++z) {
        const int buf = z & 1;
        const long long i = own_off + plane * z;
        // operands that are needed only at the row's own node
        double2 w0 = zero2, w1 = zero2;    // K1: r~ ; K2: - ; R0/R1: b
        double2 cf[6];
        if (own_ok) {
            if (MODE == MODE_K1) w0 = *reinterpret_cast<const double2*>(kv.rt + i);
            if (MODE == MODE_R0 || MODE == MODE_R1) w0 = *reinterpret_cast<const double2*>(kv.b + i);
            if (STORED) {
#pragma unroll
                for (int d = 0; d < 6; ++d) cf[d] = *reinterpret_cast<const double2*>(op.offd[d] + i);
            }
        }
        (void)w1;
        consume(z + 1, true);              // u(z+1): registers + the other shared buffer
        request(z + 2);                    // in flight while plane z is differenced
        if (own_ok) {
            double out[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                const int sx = 1 + 2 * lane + e, sy = 1 + ty;
                double c[6];
                if (STORED) {
#pragma unroll
                    for (int d = 0; d < 6; ++d) c[d] = e == 0 ? cf[d].x : cf[d].y;
                } else {
                    const double* row = lut_s + k_c[e] * PF_MAX_CLASSES;
                    c[0] = row[e == 0 ? k_c[1] : c_s[buf][sy][sx + 1]];
                    c[1] = row[e == 1 ? k_c[0] : c_s[buf][sy][sx - 1]];
                    c[2] = row[c_s[buf][sy - 1][sx]];
                    c[3] = row[c_s[buf][sy + 1][sx]];
                    c[4] = row[k_dn[e]];
                    c[5] = row[k_up[e]];
                }
                double acc = mul(a_c[e], u_c[e]);
                const double ue = e == 0 ? u_c[1] : u_s[buf][sy][sx + 1];
                const double uw = e == 1 ? u_c[0] : u_s[buf][sy][sx - 1];
                if (c[0] != 0.0) acc = add(acc, mul(c[0], ue));
                if (c[1] != 0.0) acc = add(acc, mul(c[1], uw));
                if (c[2] != 0.0) acc = add(acc, mul(c[2], u_s[buf][sy - 1][sx]));
                if (c[3] != 0.0) acc = add(acc, mul(c[3], u_s[buf][sy + 1][sx]));
                if (c[4] != 0.0) acc = add(acc, mul(c[4], u_dn[e]));
                if (c[5] != 0.0) acc = add(acc, mul(c[5], u_up[e]));
                out[e] = acc;
            }
            if (MODE == MODE_K1) {
                *reinterpret_cast<double2*>(kv.v_out + i) = make_double2(out[0], out[1]);
                dd_fma(q[0], w0.x, out[0]); dd_fma(q[0], w0.y, out[1]);
            } else if (MODE == MODE_K2) {
                *reinterpret_cast<double2*>(kv.t + i) = make_double2(out[0], out[1]);
                dd_fma(q[0], out[0], n_c[0]); dd_fma(q[0], out[1], n_c[1]);
                dd_fma(q[1], out[0], out[0]); dd_fma(q[1], out[1], out[1]);
            } else {
                const double r0 = sub(w0.x, out[0]), r1 = sub(w0.y, out[1]);
                if (MODE == MODE_R0) {
                    *reinterpret_cast<double2*>(kv.r + i) = make_double2(r0, r1);
                    *reinterpret_cast<double2*>(kv.rt + i) = make_double2(r0, r1);
                    dd_fma(q[0], w0.x, w0.x); dd_fma(q[0], w0.y, w0.y);
                }
                dd_fma(q[1], r0, r0); dd_fma(q[1], r1, r1);
            }
        }
        rotate();
        __syncthreads();
    }

    if (MODE == MODE_K1) {
        dd q1[1] = {q[0]};
        if (grid_reduce_dd<1>(q1, scratch, rb)) finish_k1(sc, dd_round(q1[0]));
    } else if (grid_reduce_dd<2>(q, scratch, rb)) {
        if (MODE == MODE_K2) finish_k2(sc, dd_round(q[0]), dd_round(q[1]));
        else if (MODE == MODE_R0) finish_init(sc, kv.hist, dd_round(q[0]), dd_round(q[1]));
        else sc->true_rr = dd_round(q[1]);
    }
}

// z-chunking: enough blocks to fill the SMs in whole waves, chunks deep enough that the two extra
// planes per chunk stay a small fraction.
int choose_zchunks(const GridDims& g, int tiles, int sm_count) {
    int best = 1;
    double best_score = -1.0;
    const int max_chunks = std::max(1, std::min(g.nz / 4, PF_MAX_PARTIAL_BLOCKS / tiles));
    for (int zc = 1; zc <= max_chunks; ++zc) {
        const int depth = (g.nz + zc - 1) / zc;
        const int chunks = (g.nz + depth - 1) / depth;
        const long long blocks = (long long)tiles * chunks;
        const long long waves = (blocks + sm_count - 1) / sm_count;
        const double fill = (double)blocks / (double)(waves * sm_count);
        const double halo = (double)depth / (double)(depth + 2);
        const double score = fill * halo;
        if (score > best_score + 1e-9) { best_score = score; best = chunks; }
    }
    return best;
}

bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

template <int MODE>
void launch_mode(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    const int tx = (c.g.nx + TX - 1) / TX, tyb = (c.g.ny + TY - 1) / TY;
    const int chunks = choose_zchunks(c.g, tx * tyb, c.sm_count);
    const int depth = (c.g.nz + chunks - 1) / chunks;
    dim3 grid(tx, tyb, (c.g.nz + depth - 1) / depth);
    ++g_launch_count;
    if (op.stored) {
        if (precond) k_tiled<MODE, true, true><<<grid, TILE_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb, depth);
        else         k_tiled<MODE, false, true><<<grid, TILE_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb, depth);
    } else {
        if (precond) k_tiled<MODE, true, false><<<grid, TILE_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb, depth);
        else         k_tiled<MODE, false, false><<<grid, TILE_THREADS, 0, c.stream>>>(c.g, op, kv, c.sc, c.rb, depth);
    }
}

}  // namespace

// The tiled family needs an even nx (128-bit accesses) and a grid that fills at least a few tiles.
bool tiled_supported(const GridDims& g) {
    return (g.nx % 2 == 0) && g.nx >= 32 && g.ny >= 16 && g.nz >= 8;
}

bool tiled_pointers_ok(const KrylovVecs& kv) { return aligned16(kv.x) && aligned16(kv.b); }

void launch_residual_tiled(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, int mode) {
    if (mode == 0) launch_mode<MODE_R0>(c, op, kv, false); else launch_mode<MODE_R1>(c, op, kv, false);
}
void launch_k1_tiled(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    launch_mode<MODE_K1>(c, op, kv, precond);
}
void launch_k2_tiled(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, bool precond) {
    launch_mode<MODE_K2>(c, op, kv, precond);
}

}  // namespace pf
