// pf_krylov_tma.cu -- the fused stencil kernels of the BiCGSTAB iteration for B200: planes staged in
// shared memory by TMA, z marched in registers.
//
// Work decomposition.  The xy plane is cut into tiles of TX x TY = 64 x 16 nodes; a block of 512 threads
// (warp = one 512-byte row, lane = two x-adjacent nodes) marches its tile along z over a chunk of planes.
// One elected thread keeps a ring of S stages filled: per plane one 3-D tensor-map copy
// (cp.async.bulk.tensor, completion on an mbarrier) per operand, of the tile PLUS its halo ring -- box
// (TX+4) x (TY+2) so that every thread's pair of nodes is 16-byte aligned in shared memory.  Nodes outside
// the grid are zero-filled by the TMA unit, so no thread computes an address or a bounds test for a load.
//
// What is fused (rows L3-L5 of DESIGN.md).  The vector update that precedes a matvec in Table 3
// is recomputed on the fly at the tile AND at its halo ring, so the updated vector is
// never written and re-read for the matvec:
//   MODE_K1  u = M^-1 (r + beta (p - omega v))  (steps 5-9, Jacobi Q2), v' = A u (step 11), r~.v'
//   MODE_K2  u = M^-1 (r - alpha v)             (step 13),            t  = A u (step 14), t.s, t.t
//   MODE_R0  u = x,  r = b - A u, r~ = r, b.b, r.r (step 2);  MODE_R1: ||b - A x||^2 only
// u of the plane being differenced sits in shared memory (xy neighbours, double-buffered); the z
// neighbours stay in registers of the marching thread.  Per plane: wait for the stage, form u(z+1),
// difference plane z, one __syncthreads, refill the stage just consumed (S-1 planes of loads in flight).
//
// Arithmetic is the same statement for statement as the direct kernels (pf_krylov_direct.cu): both
// families give bit-identical vectors.
#include "pf_krylov.cuh"
#include "pf_launch.h"

#include <cuda.h>      // CUtensorMap and its enums (types only; the encoder is fetched at run time)
#include <algorithm>
#include <cstring>

namespace pf {

namespace {

constexpr int TX = 64;                   // tile width in nodes (32 lanes x 2)
constexpr int TY = 16;                   // tile height = warps per block
constexpr int NT = 32 * TY;
constexpr int BX = TX + 4;               // box: two halo columns each side (one used; two keep 16-byte alignment)
constexpr int BY = TY + 2;
constexpr int FIELD_BYTES = ((BX * BY * 8 + 127) / 128) * 128;   // 9856
constexpr int OWN_BYTES = TX * TY * 8;                            // 8192
constexpr int NHALO = 2 * TX + 2 * TY;                            // 160 halo nodes per plane
static_assert(NHALO <= NT, "one halo node per thread");

enum { MODE_R0 = 0, MODE_R1 = 1, MODE_K1 = 2, MODE_K2 = 3 };

template <int MODE> struct ModeTraits;
template <> struct ModeTraits<MODE_R0> { static constexpr int NF = 2; static constexpr bool OWN = true;  static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_R1> { static constexpr int NF = 2; static constexpr bool OWN = true;  static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_K1> { static constexpr int NF = 4; static constexpr bool OWN = true;  static constexpr int STAGES = 3; };
template <> struct ModeTraits<MODE_K2> { static constexpr int NF = 3; static constexpr bool OWN = false; static constexpr int STAGES = 4; };

// Halo fields in stage order.  K1: r, p, v, A0.  K2: r, v, A0.  R0/R1: x, A0.
// Own-only field (tile without halo): K1: r~;  R0/R1: b.
struct TmaArgs {
    CUtensorMap f[4];
    CUtensorMap own;
    CUtensorMap code;
};

template <int MODE, bool STORED, bool CODE32>
struct Layout {
    using T = ModeTraits<MODE>;
    static constexpr int CODE_BYTES = STORED ? 0 : TX * TY * (CODE32 ? 4 : 2);
    static constexpr int STAGE_BYTES = T::NF * FIELD_BYTES + (T::OWN ? OWN_BYTES : 0) + CODE_BYTES;
    static constexpr int OWN_OFF = T::NF * FIELD_BYTES;
    static constexpr int CODE_OFF = OWN_OFF + (T::OWN ? OWN_BYTES : 0);
    static constexpr int U_BYTES = BX * BY * 8;                     // one buffer of u
    static constexpr int U_OFF = T::STAGES * STAGE_BYTES;
    static constexpr int CTAB_OFF = U_OFF + 2 * FIELD_BYTES;
    static constexpr int SCRATCH_OFF = CTAB_OFF + PF_CTAB * 8;
    static constexpr int BAR_OFF = SCRATCH_OFF + 2 * 32 * (int)sizeof(dd);
    static constexpr int TOTAL = BAR_OFF + 8 * T::STAGES;
    static constexpr unsigned TX_BYTES = (unsigned)(T::NF * BX * BY * 8 + (T::OWN ? OWN_BYTES : 0) + CODE_BYTES);
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned long long* bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, unsigned long long* bar, int x, int y,
                                            int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(x), "r"(y), "r"(z)
        : "memory");
}

template <int MODE, bool PRECOND>
__device__ __forceinline__ double u_of(double r, double p, double v, double a, bool first, double c1, double c2,
                                       double& numer) {
    if (MODE == MODE_K1) { numer = p_new_at<PRECOND>(first, c1, c2, r, p, v); return jacobi<PRECOND>(numer, a); }
    if (MODE == MODE_K2) { numer = s_at(c1, r, v); return jacobi<PRECOND>(numer, a); }
    numer = r;           // residual modes: the field is x itself (passed in r)
    return r;
}

// Byte offset into the coefficient table of field d of node e (0 or 1) of the thread's code word(s).
template <bool CODE32>
__device__ __forceinline__ unsigned ctab_off(unsigned w0, unsigned w1, int e, int d) {
    if (CODE32) {
        const unsigned w = e ? w1 : w0;
        const int sh = 4 * d - 3;
        return (sh >= 0 ? (w >> sh) : (w << -sh)) & 0x78u;
    } else {
        const int sh = 16 * e + 2 * d - 3;
        return (sh >= 0 ? (w0 >> sh) : (w0 << -sh)) & 0x18u;
    }
}

template <int MODE, bool PRECOND, bool STORED, bool CODE32>
__global__ void __launch_bounds__(NT, 1)
k_tma(const __grid_constant__ TmaArgs tm, GridDims g, Operator op, KrylovVecs kv, Scalars* sc, ReduceBuf rb, int zchunk) {
    using L = Layout<MODE, STORED, CODE32>;
    using T = ModeTraits<MODE>;
    constexpr int S = T::STAGES;
    constexpr int NF = T::NF;
    if (MODE >= MODE_K1 && sc->done) return;
    extern __shared__ __align__(128) unsigned char smem[];
    double* ctab_s = reinterpret_cast<double*>(smem + L::CTAB_OFF);
    dd* scratch = reinterpret_cast<dd*>(smem + L::SCRATCH_OFF);
    unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem + L::BAR_OFF);

    const int tid = threadIdx.x, lane = tid & 31, ty = tid >> 5;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY;
    const int z0 = blockIdx.z * zchunk, z1 = min(z0 + zchunk, g.nz);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < S; ++s) mbar_init(&bars[s], 1);
        fence_proxy_async();
    }
    if (!STORED && tid < PF_CTAB) ctab_s[tid] = op.ctab[tid];
    __syncthreads();

    // plane q of this block's load sequence is z0 - 1 + q; q = 0 .. nq-1
    const int nq = z1 - z0 + 2;
    auto issue = [&](int q) {                       // tid 0 only
        const int s = q % S;
        unsigned char* st = smem + s * L::STAGE_BYTES;
        const int z = z0 - 1 + q;
        mbar_expect_tx(&bars[s], L::TX_BYTES);
#pragma unroll
        for (int f = 0; f < NF; ++f) tma_load_3d(st + f * FIELD_BYTES, &tm.f[f], &bars[s], x0 - 2, y0 - 1, z);
        if (T::OWN) tma_load_3d(st + L::OWN_OFF, &tm.own, &bars[s], x0, y0, z);
        if (!STORED) tma_load_3d(st + L::CODE_OFF, &tm.code, &bars[s], x0, y0, z);
    };
    if (tid == 0)
        for (int q = 0; q < S && q < nq; ++q) issue(q);

    bool first = false; double c1 = 0.0, c2 = 0.0;
    if (MODE == MODE_K1) { first = sc->first != 0; c1 = sc->beta; c2 = sc->omega; }
    else if (MODE == MODE_K2) { c1 = sc->alpha; }

    // own slot: nodes (x, y) and (x+1, y); nx is even so both are inside or both outside
    const int x = x0 + 2 * lane, y = y0 + ty;
    const bool own_ok = x < g.nx && y < g.ny;
    const long long plane = (long long)g.nx * g.ny;
    const long long own_off = x + (long long)g.nx * y;
    const int own_box = (ty + 1) * BX + 2 + 2 * lane;              // element offset in a halo box
    const int own_tile = ty * TX + 2 * lane;                        // element offset in an own-only box
    // halo slot: one node per thread, threads 0..NHALO-1
    int hbox = 0; bool h_ok = false;
    const bool h_any = tid < NHALO;
    if (h_any) {
        int hx, hy;
        if (tid < TX)            { hx = 2 + tid;        hy = 0; }
        else if (tid < 2 * TX)   { hx = 2 + tid - TX;   hy = BY - 1; }
        else if (tid < 2 * TX + TY) { hx = 1;           hy = 1 + tid - 2 * TX; }
        else                     { hx = BX - 2;         hy = 1 + tid - 2 * TX - TY; }
        hbox = hy * BX + hx;
        const int gx = x0 - 2 + hx, gy = y0 - 1 + hy;
        h_ok = gx >= 0 && gx < g.nx && gy >= 0 && gy < g.ny;
    }

    double u_dn[2] = {0, 0}, u_c[2] = {0, 0}, u_up[2] = {0, 0};
    double n_c[2] = {0, 0}, n_up[2] = {0, 0};              // numerators: p' (K1) or s (K2)
    double a_c[2] = {1, 1}, a_up[2] = {1, 1};
    double2 w_c = make_double2(0, 0), w_up = make_double2(0, 0);    // own-only operand: r~ (K1) or b (R0/R1)
    unsigned k0_c = 0, k1_c = 0, k0_up = 0, k1_up = 0;              // code word(s) of the thread's two nodes

    // form u of plane z0-1+q from its stage: own nodes -> registers (+ shared), halo nodes -> shared
    auto prepare = [&](int q, bool to_shared) {
        const int s = q % S;
        const unsigned par = (unsigned)(q / S) & 1u;
        while (!mbar_try_wait(&bars[s], par)) {}
        const unsigned char* st = smem + s * L::STAGE_BYTES;
        const int z = z0 - 1 + q;
        const bool zin = z >= 0 && z < g.nz;
        double* u_s = reinterpret_cast<double*>(smem + L::U_OFF + (q & 1) * FIELD_BYTES);
        const double* F0 = reinterpret_cast<const double*>(st);
        const double* F1 = reinterpret_cast<const double*>(st + FIELD_BYTES);
        const double* F2 = reinterpret_cast<const double*>(st + 2 * FIELD_BYTES);
        const double* F3 = reinterpret_cast<const double*>(st + 3 * FIELD_BYTES);
        double2 fr = *reinterpret_cast<const double2*>(F0 + own_box), fp = make_double2(0, 0), fv = make_double2(0, 0), fa;
        if (MODE == MODE_K1) {
            fp = *reinterpret_cast<const double2*>(F1 + own_box);
            fv = *reinterpret_cast<const double2*>(F2 + own_box);
            fa = *reinterpret_cast<const double2*>(F3 + own_box);
        } else if (MODE == MODE_K2) {
            fv = *reinterpret_cast<const double2*>(F1 + own_box);
            fa = *reinterpret_cast<const double2*>(F2 + own_box);
        } else {
            fa = *reinterpret_cast<const double2*>(F1 + own_box);
        }
        const bool ok = own_ok && zin;
        if (!ok) fa = make_double2(1.0, 1.0);                       // zero-filled nodes: keep u finite (0/1)
        u_up[0] = u_of<MODE, PRECOND>(fr.x, fp.x, fv.x, fa.x, first, c1, c2, n_up[0]);
        u_up[1] = u_of<MODE, PRECOND>(fr.y, fp.y, fv.y, fa.y, first, c1, c2, n_up[1]);
        a_up[0] = fa.x; a_up[1] = fa.y;
        if (T::OWN) w_up = *reinterpret_cast<const double2*>(reinterpret_cast<const double*>(st + L::OWN_OFF) + own_tile);
        if (!STORED) {
            if (CODE32) {
                const uint2 cw = *reinterpret_cast<const uint2*>(st + L::CODE_OFF + 4 * own_tile);
                k0_up = cw.x; k1_up = cw.y;
            } else {
                k0_up = *reinterpret_cast<const unsigned*>(st + L::CODE_OFF + 2 * own_tile);
            }
        }
        if (MODE == MODE_K1 && ok && z >= z0 && z < z1)             // p' is an output of steps 5-9
            *reinterpret_cast<double2*>(kv.p_out + own_off + plane * z) = make_double2(n_up[0], n_up[1]);
        if (to_shared) {
            *reinterpret_cast<double2*>(u_s + own_box) = make_double2(u_up[0], u_up[1]);
            if (h_any) {
                double hr = F0[hbox], hp = 0.0, hv = 0.0, ha;
                if (MODE == MODE_K1) { hp = F1[hbox]; hv = F2[hbox]; ha = F3[hbox]; }
                else if (MODE == MODE_K2) { hv = F1[hbox]; ha = F2[hbox]; }
                else ha = 1.0;
                if (!(h_ok && zin)) ha = 1.0;
                double dummy;
                u_s[hbox] = u_of<MODE, PRECOND>(hr, hp, hv, ha, first, c1, c2, dummy);
            }
        }
    };
    auto rotate = [&]() {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
            u_dn[e] = u_c[e]; u_c[e] = u_up[e]; n_c[e] = n_up[e]; a_c[e] = a_up[e];
        }
        w_c = w_up; k0_c = k0_up; k1_c = k1_up;
    };

    dd q[2] = {dd_zero(), dd_zero()};

    prepare(0, false); rotate();           // plane z0-1: registers only
    prepare(1, true);  rotate();           // plane z0
    __syncthreads();
    if (tid == 0) {                        // stages of q = 0, 1 are consumed
        if (S + 0 < nq) issue(S + 0);
        if (S + 1 < nq) issue(S + 1);
    }

    for (int z = z0; z < z1; ++z) {
        const int qn = z - z0 + 2;         // load-sequence index of plane z+1
        const long long i = own_off + plane * z;
        double2 cf[6];
        if (STORED && own_ok) {
#pragma unroll
            for (int d = 0; d < 6; ++d) cf[d] = *reinterpret_cast<const double2*>(op.offd[d] + i);
        }
        prepare(qn, true);                 // u(z+1): registers + the other shared buffer
        if (own_ok) {
            const double* u_s = reinterpret_cast<const double*>(smem + L::U_OFF + ((qn - 1) & 1) * FIELD_BYTES);
            const double2 us = *reinterpret_cast<const double2*>(u_s + own_box - BX);
            const double2 un = *reinterpret_cast<const double2*>(u_s + own_box + BX);
            const double uw = u_s[own_box - 1], ue = u_s[own_box + 2];
            double out[2];
#pragma unroll
            for (int e = 0; e < 2; ++e) {
                double c[6];
                if (STORED) {
#pragma unroll
                    for (int d = 0; d < 6; ++d) c[d] = e == 0 ? cf[d].x : cf[d].y;
                } else {
#pragma unroll
                    for (int d = 0; d < 6; ++d)
                        c[d] = *reinterpret_cast<const double*>(reinterpret_cast<const unsigned char*>(ctab_s) +
                                                                ctab_off<CODE32>(k0_c, k1_c, e, d));
                }
                double acc = mul(a_c[e], u_c[e]);
                acc = add(acc, mul(c[0], e == 0 ? u_c[1] : ue));
                acc = add(acc, mul(c[1], e == 1 ? u_c[0] : uw));
                acc = add(acc, mul(c[2], e == 0 ? us.x : us.y));
                acc = add(acc, mul(c[3], e == 0 ? un.x : un.y));
                acc = add(acc, mul(c[4], u_dn[e]));
                acc = add(acc, mul(c[5], u_up[e]));
                out[e] = acc;
            }
            if (MODE == MODE_K1) {
                *reinterpret_cast<double2*>(kv.v_out + i) = make_double2(out[0], out[1]);
                dd_fma(q[0], w_c.x, out[0]); dd_fma(q[1], w_c.y, out[1]);
            } else if (MODE == MODE_K2) {
                *reinterpret_cast<double2*>(kv.t + i) = make_double2(out[0], out[1]);
                dd_fma(q[0], out[0], n_c[0]); dd_fma(q[0], out[1], n_c[1]);
                dd_fma(q[1], out[0], out[0]); dd_fma(q[1], out[1], out[1]);
            } else {
                const double r0 = sub(w_c.x, out[0]), r1 = sub(w_c.y, out[1]);
                if (MODE == MODE_R0) {
                    *reinterpret_cast<double2*>(kv.r + i) = make_double2(r0, r1);
                    *reinterpret_cast<double2*>(kv.rt + i) = make_double2(r0, r1);
                    dd_fma(q[0], w_c.x, w_c.x); dd_fma(q[0], w_c.y, w_c.y);
                }
                dd_fma(q[1], r0, r0); dd_fma(q[1], r1, r1);
            }
        }
        rotate();
        __syncthreads();
        if (tid == 0 && qn + S < nq) issue(qn + S);     // the stage of plane z+1 is consumed: refill it
    }

    if (MODE == MODE_K1) {
        dd_add(q[0], q[1]);                // two chains for instruction-level parallelism, one quantity
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

// ---- tensor maps ------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encoder() {
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) != cudaSuccess ||
            qres != cudaDriverEntryPointSuccess) {
            cudaGetLastError();
            return nullptr;
        }
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// 3-D map over an nx x ny x nz array of `elem`-byte entries with row pitch `pitch` entries.
bool make_map(CUtensorMap* m, const void* base, CUtensorMapDataType dt, int elem, const GridDims& g, long long pitch,
              int bx, int by) {
    EncodeTiledFn fn = encoder();
    if (!fn) return false;
    cuuint64_t dims[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz};
    cuuint64_t strides[2] = {(cuuint64_t)pitch * elem, (cuuint64_t)pitch * g.ny * elem};
    cuuint32_t box[3] = {(cuuint32_t)bx, (cuuint32_t)by, 1u};
    cuuint32_t es[3] = {1u, 1u, 1u};
    return fn(m, dt, 3, const_cast<void*>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

bool halo_map(CUtensorMap* m, const double* base, const GridDims& g) {
    return make_map(m, base, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, g, g.nx, BX, BY);
}
bool own_map(CUtensorMap* m, const double* base, const GridDims& g) {
    return make_map(m, base, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, g, g.nx, TX, TY);
}

template <int MODE, bool PRECOND, bool STORED, bool CODE32>
void launch_inst(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaArgs& tm, dim3 grid, int depth) {
    using L = Layout<MODE, STORED, CODE32>;
    static bool configured = false;
    auto kern = k_tma<MODE, PRECOND, STORED, CODE32>;
    if (!configured) {
        cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL);
        configured = true;
    }
    ++g_launch_count;
    kern<<<grid, NT, L::TOTAL, c.stream>>>(tm, c.g, op, kv, c.sc, c.rb, depth);
}

template <int MODE>
void launch_mode(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaArgs& tm, bool precond) {
    const int tx = (c.g.nx + TX - 1) / TX, tyb = (c.g.ny + TY - 1) / TY;
    const int chunks = choose_zchunks(c.g, tx * tyb, c.sm_count);
    const int depth = (c.g.nz + chunks - 1) / chunks;
    dim3 grid(tx, tyb, (c.g.nz + depth - 1) / depth);
    const bool c32 = op.code32 != 0;
    if (op.stored) {
        if (precond) launch_inst<MODE, true, true, false>(c, op, kv, tm, grid, depth);
        else         launch_inst<MODE, false, true, false>(c, op, kv, tm, grid, depth);
    } else if (c32) {
        if (precond) launch_inst<MODE, true, false, true>(c, op, kv, tm, grid, depth);
        else         launch_inst<MODE, false, false, true>(c, op, kv, tm, grid, depth);
    } else {
        if (precond) launch_inst<MODE, true, false, false>(c, op, kv, tm, grid, depth);
        else         launch_inst<MODE, false, false, false>(c, op, kv, tm, grid, depth);
    }
}

}  // namespace

// Tensor maps of one solve: every vector a kernel reads through TMA.
struct TmaSet {
    CUtensorMap r, p[2], v[2], a0, rt, x, b, code;
    bool have_code;
};

bool tma_available() { return encoder() != nullptr; }

// Even nx (16-byte row strides) and a grid that fills at least a few tiles.
bool tma_supported(const GridDims& g) {
    return (g.nx % 2 == 0) && g.nx >= 32 && g.ny >= 16 && g.nz >= 8;
}

bool tma_pointers_ok(const KrylovVecs& kv, const Operator& op) {
    return aligned16(kv.x) && aligned16(kv.b) && aligned16(op.A0) && aligned16(kv.r) && aligned16(kv.rt) &&
           aligned16(kv.p_in) && aligned16(kv.p_out) && aligned16(kv.v_in) && aligned16(kv.v_out) && aligned16(kv.t);
}

TmaSet* tma_set_create() { return new TmaSet(); }
void tma_set_destroy(TmaSet* t) { delete t; }

bool tma_set_build(TmaSet* t, const GridDims& g, const Operator& op, const KrylovVecs& kv) {
    bool ok = halo_map(&t->r, kv.r, g) && halo_map(&t->p[0], kv.p_in, g) && halo_map(&t->p[1], kv.p_out, g) &&
              halo_map(&t->v[0], kv.v_in, g) && halo_map(&t->v[1], kv.v_out, g) && halo_map(&t->a0, op.A0, g) &&
              own_map(&t->rt, kv.rt, g) && halo_map(&t->x, kv.x, g) && own_map(&t->b, kv.b, g);
    t->have_code = false;
    if (ok && !op.stored) {
        ok = op.code32 ? make_map(&t->code, op.code, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, g, op.cpitch, TX, TY)
                       : make_map(&t->code, op.code, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, g, op.cpitch, TX, TY);
        t->have_code = ok;
    }
    return ok;
}

void launch_residual_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, int mode) {
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    a.f[0] = t->x; a.f[1] = t->a0; a.own = t->b; a.code = t->code;
    if (mode == 0) launch_mode<MODE_R0>(c, op, kv, a, false); else launch_mode<MODE_R1>(c, op, kv, a, false);
}

void launch_k1_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond,
                   int parity) {
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    a.f[0] = t->r; a.f[1] = t->p[parity]; a.f[2] = t->v[parity]; a.f[3] = t->a0; a.own = t->rt; a.code = t->code;
    launch_mode<MODE_K1>(c, op, kv, a, precond);
}

void launch_k2_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond,
                   int parity) {
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    a.f[0] = t->r; a.f[1] = t->v[parity ^ 1]; a.f[2] = t->a0; a.code = t->code;   // v' = the buffer k1 just wrote
    launch_mode<MODE_K2>(c, op, kv, a, precond);
}

}  // namespace pf
