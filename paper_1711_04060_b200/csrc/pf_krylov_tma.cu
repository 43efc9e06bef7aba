// pf_krylov_tma.cu -- the fused stencil kernels of the BiCGSTAB iteration for B200: planes staged in
// shared memory by TMA, z marched in registers, warp-specialised.
//
// Work decomposition.  The xy plane is cut into tiles of TX x TY = 64 x 16 nodes and z into chunks; a work item
// is one tile marched along z over one chunk.  min(#SMs, #items) persistent blocks take the items round-robin in
// the order x tile, y tile, chunk (neighbouring tiles run at the same time and share halo rows in L2), with the
// stage ring running on from one item to the next.  Roles of a block's 19 warps:
//   producer (1 warp, one lane)  keeps a ring of S stages filled: per plane one 3-D tensor-map copy
//       (cp.async.bulk.tensor, completion on a "full" mbarrier) per operand, of the tile PLUS its halo ring --
//       box (TX+4) x (TY+2) so that every thread's pair of nodes is 16-byte aligned in shared memory.  Nodes
//       outside the grid are zero-filled by the TMA unit: no thread computes an address or a bounds test for
//       a load.  A stage is refilled as soon as the 18 consumer warps have released it ("empty" mbarrier).
//   main (16 warps)  warp = one 512-byte tile row, lane = two x-adjacent nodes: form u at the own nodes,
//       difference the plane, store, accumulate the inner products.
//   halo (2 warps)   form u on the halo ring (rows y0-1 and y0+TY, columns x0-1 and x0+TX), off the main
//       warps' critical path.
//
// What is fused (rows L3-L5 of DESIGN.md).  The vector update that precedes a matvec in Table 3
// is recomputed on the fly at the tile AND at its halo ring, so the updated vector is
// never written and re-read for the matvec:
//   MODE_K1  u = M^-1 (r + beta (p - omega v))  (steps 5-9, Jacobi Q2), v' = A u (step 11), r~.v'
//   MODE_K2  u = M^-1 (r - alpha v)             (step 13),            t  = A u (step 14), t.s, t.t
//   MODE_R0  u = x,  r = b - A u, r~ = r, b.b, r.r (step 2);  MODE_R1: ||b - A x||^2 only
// u of the plane being differenced sits in shared memory (xy neighbours, three buffers); the z
// neighbours stay in registers of the marching thread (three register slots renamed, not moved, by a
// three-way unrolled loop).  Per plane: wait for the stage, form u(z+1), publish it and release the stage,
// difference plane z.  There is no block-wide barrier in the loop: a "ready" mbarrier per u buffer (one
// arrival per consumer warp) orders the writers and readers of the buffers, so warps drift by up to a plane.
//
// Reductions: a block ends by writing its double-double partial sums; the next kernel of the stream combines
// them in every block and takes the scalar step (begin_kernel, pf_krylov.cuh), while its producer warp has
// already requested the first stages.
//
// Arithmetic is the same statement for statement as the direct kernels (pf_krylov_direct.cu): both
// families give bit-identical vectors.
#include "pf_krylov.cuh"
#include "pf_launch.h"

#include <cuda.h>      // CUtensorMap and its enums (types only; the encoder is fetched at run time)
#include <algorithm>
#include <atomic>
#include <type_traits>
#include <cstring>

namespace pf {

namespace {

constexpr int TX = 64;                   // tile width in nodes (32 lanes x 2)
constexpr int BX = TX + 4;               // box: two halo columns each side (one used; two keep 16-byte alignment)
constexpr int NU = 3;                    // shared buffers of u (planes k, k+1 live, k+2 being written)

// Tile height = main warps per block.  Two geometries are compiled:
//   16 rows: 16 main + 2 halo + 1 producer = 19 warps; five warps share an SM quarter, which caps a thread at 96 registers;
//   13 rows: 13 + 2 + 1 = 16 warps, four per quarter, 128 registers: no spills and room to overlap the long dependent
//            chains of a plane (K31 of the merged solver, and every kernel on grids where fixed costs dominate).
// tile_rows() below picks per kernel and grid; the arithmetic does not depend on the tiling.
template <int TYV>
struct Geo {
    static constexpr int TY = TYV;
    static constexpr int NW_CONSUMER = TY + 2;
    static constexpr int NT_CONSUMER = 32 * NW_CONSUMER;
    static constexpr int NT = NT_CONSUMER + 32;     // + the producer warp
    static constexpr int BY = TY + 2;
    static constexpr int FIELD_BYTES = ((BX * BY * 8 + 127) / 128) * 128;   // 9856 (16 rows), 8192 (13 rows)
    static constexpr int OWN_BYTES = TX * TY * 8;                            // 8192, 6656
    static_assert(TY <= 16, "one halo column node per lane of a halo warp (lanes 0..15 left, 16..31 unused)");
};
constexpr int TY_WIDE = 16, TY_DEEP = 13;

enum { MODE_R0 = 0, MODE_R1 = 1, MODE_K1 = 2, MODE_K2 = 3, MODE_K1D = 4, MODE_K2M = 5, MODE_K31 = 6, MODE_K31D = 7,
       MODE_K2D = 8, MODE_K2MD = 9 };
// MODE_K1D: k1 for operators whose diagonal is the sum of their face coefficients (Poisson without sigma): A0 is
// not read but looked up, together with the reciprocal the Jacobi division needs, in a table indexed by the node's
// stencil code, whose box then covers the halo ring too.  MODE_K2D: the same for k2.
// MODE_K2M, MODE_K31 (MODE_K2MD, MODE_K31D: diagonal from the codes): the two kernels of the merged solver (pf_krylov.cuh).
constexpr int CXO = 8;                   // code box with halo: starts CXO nodes left of the tile (the TMA unit wants the
constexpr int BXC = TX + 2 * CXO;        // box to start on a 16-byte boundary of the row: 8 two-byte entries), rows of 160 bytes

// ---- work decomposition ------------------------------------------------------------------------
// A segment is one tile marched along z over [z0, z1): z1 - z0 + 2 plane steps (the two extra planes only form u).
// Two ways to hand segments to the persistent blocks (plan_segments below picks the one with the shorter longest block):
//   mode 0  z is cut into equal chunks; item i = (tile i % ntiles, chunk i / ntiles); block b takes items b, b + G, ...
//           Blocks that run at the same time work on neighbouring tiles of the same chunk, plane for plane, so halo
//           rows are shared in L2.
//   mode 1  for grids with fewer tiles than SMs, where mode 0 cannot fill the SMs evenly (256^3: 64 tiles x 9 chunks on
//           148 SMs = 4 rounds of 31 steps with the last round short: 124 steps against 111 of the volume itself):
//           `full` = #SMs / ntiles layers of `zchunk` planes are taken by ntiles * full blocks, one segment each, all
//           in step; the remaining planes z >= zrest of all tiles, flattened tile-major, are split evenly over the
//           remaining blocks (a few short segments each).  256^3: 114 steps.
//   mode 2  for grids with more tiles than half the SMs but fewer than two thirds (256^3 with 13-row tiles: 80 tiles, 6
//           rounds of 26 steps = 156 against 138 of the volume): every tile's planes [0, zchunk) on one block each
//           (group A, in step); the planes above on the other R = #SMs - tiles blocks for the first R tiles (group B, in
//           step, shallower); the same planes of the remaining tiles, cut into q pieces along z, are taken by group B's
//           blocks when they are done (piece j of all these tiles by consecutive blocks, in step).  256^3: 143 steps.
struct SegPlan {
    int mode, ntx, ntiles;
    int zchunk, nitems;       // mode 0: chunk depth and tiles * chunks; mode 1: layer depth of the main group, nmain;
                              // mode 2: depth of group A's layer, tiles
    int zrest, erest, q;      // mode 1: the rest group's planes [zrest, zrest + erest), q flattened positions per block
                              // mode 2: the upper layer [zrest, zrest + erest), q pieces per leftover tile
    int blocks;               // host: blocks to launch
    int m2_rest, m2_left, m2_depth;   // mode 2, precomputed so that the kernels divide by nothing: blocks of group B, tiles
                                      // whose upper layer comes second, depth of a piece
};
// The segments of block b, one after the other (every thread of the block walks the same sequence).  PERSIST = false:
// the block's one item of the equal-chunk plan (the stored variant has no registers to spare for a loop).
// M2: the instance walks a plan of mode 2 (its own template parameter: kept apart, the walks of modes 0 / 1 are the code
// they were before mode 2 existed -- with all three in one function the kernels, which sit at their register cap, lost
// 3-5 % at 128^3 to a different register allocation and to divisions the compiler hoisted out of untaken branches).
template <bool PERSIST, bool M2>
struct SegIter {
    int pos, end;
    __device__ __forceinline__ void init(const SegPlan& P, int b, int nblocks) {
        if (PERSIST && M2) {
            // group A: one segment; group B block r: its own upper layer, then piece r / L of leftover tile R + r % L
            // (plan_segments names non-empty pieces only)
            (void)nblocks;
            pos = 0; end = (b >= P.ntiles && b - P.ntiles < P.m2_left * P.q) ? 2 : 1;
        }
        else if (PERSIST && P.mode == 1 && b >= P.nitems) { pos = (b - P.nitems) * P.q; end = min(pos + P.q, P.ntiles * P.erest); }
        else if (PERSIST && P.mode == 1) { pos = b; end = b + 1; }
        else { pos = b; end = PERSIST ? P.nitems : min(b + 1, P.nitems); }
    }
    __device__ __forceinline__ bool next(const SegPlan& P, int nz, int b, int nblocks, int& tile, int& z0, int& z1) {
        if (pos >= end) return false;
        if (PERSIST && M2) {
            if (b < P.ntiles) { tile = b; z0 = 0; z1 = P.zchunk; }
            else if (pos == 0) { tile = b - P.ntiles; z0 = P.zrest; z1 = nz; }
            else {
                // r = piece * L + t with piece < q <= 8: found by subtraction (an integer division here would be
                // evaluated, predicated off, by every thread of every kernel: the compiler hoists it)
                int t = b - P.ntiles, piece = 0;
                while (t >= P.m2_left) { t -= P.m2_left; ++piece; }
                tile = P.m2_rest + t;
                z0 = P.zrest + piece * P.m2_depth; z1 = min(z0 + P.m2_depth, nz);
            }
            ++pos;
        } else if (PERSIST && P.mode == 1 && b >= P.nitems) {   // rest group: flattened positions, one segment per tile
            tile = pos / P.erest;
            const int zz = pos - tile * P.erest, len = min(P.erest - zz, end - pos);
            z0 = P.zrest + zz; z1 = z0 + len; pos += len;
        } else {
            tile = pos % P.ntiles;
            z0 = (pos / P.ntiles) * P.zchunk; z1 = min(z0 + P.zchunk, (PERSIST && P.mode == 1) ? P.zrest : nz);
            pos += PERSIST ? nblocks : 1;
        }
        return true;
    }
};

template <int MODE> struct ModeTraits;
template <> struct ModeTraits<MODE_R0> { static constexpr int NF = 2; static constexpr bool OWN = true;  static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_R1> { static constexpr int NF = 2; static constexpr bool OWN = true;  static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_K1> { static constexpr int NF = 4; static constexpr bool OWN = true;  static constexpr int STAGES = 3; };
template <> struct ModeTraits<MODE_K1D> { static constexpr int NF = 3; static constexpr bool OWN = true; static constexpr int STAGES = 3; };   // (4 fit, within 1.2 KB of the limit: 1 % faster)
template <> struct ModeTraits<MODE_K2> { static constexpr int NF = 3; static constexpr bool OWN = false; static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_K2M> { static constexpr int NF = 3; static constexpr bool OWN = true; static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_K31> { static constexpr int NF = 5; static constexpr bool OWN = true; static constexpr int STAGES = 3; };
template <> struct ModeTraits<MODE_K31D> { static constexpr int NF = 4; static constexpr bool OWN = true; static constexpr int STAGES = 3; };
template <> struct ModeTraits<MODE_K2D> { static constexpr int NF = 2; static constexpr bool OWN = false; static constexpr int STAGES = 4; };
template <> struct ModeTraits<MODE_K2MD> { static constexpr int NF = 2; static constexpr bool OWN = true; static constexpr int STAGES = 4; };

// Halo fields in stage order.  K1: r, p, v, A0.  K1D: r, p, v.  K2, K2M: r, v, A0.  K2D, K2MD: r, v.  K31: r, p, v, t, A0.
// K31D: r, p, v, t.
// R0/R1: x, A0.  Own-only field (tile without halo): K1, K2M, K31: r~;  R0/R1: b.
struct TmaArgs {
    CUtensorMap f[5];
    CUtensorMap own;
    CUtensorMap code;
};

template <int MODE, bool STORED, bool CODE32, int TYV>
struct Layout {
    using T = ModeTraits<MODE>;
    static constexpr int TY = Geo<TYV>::TY, BY = Geo<TYV>::BY, FIELD_BYTES = Geo<TYV>::FIELD_BYTES,
                         OWN_BYTES = Geo<TYV>::OWN_BYTES;
    static constexpr bool DIAG = MODE == MODE_K1D || MODE == MODE_K31D || MODE == MODE_K2D || MODE == MODE_K2MD;
    // (the wide K31D, which no policy picks, makes room for the table with a stage less)
    // k1 on the deep tiles has room for a fourth stage (measured at 256^3, same box: k1 0.152 -> 0.142 ms with it, against
    // 0.150 on the wide tiles; a fifth stage for k2 / K2M changes nothing)
    static constexpr int STAGES = (MODE == MODE_K31D && TYV == 16) ? 2
        : ((MODE == MODE_K1 || MODE == MODE_K1D) && TYV == 13 && !STORED) ? 4
        : T::STAGES;
    static constexpr int CODE_TX = DIAG ? BXC * BY * 2 : TX * TY * (CODE32 ? 4 : 2);   // bytes the TMA unit delivers
    static constexpr int CODE_BYTES = STORED ? 0 : ((CODE_TX + 127) / 128) * 128;
    static constexpr int STAGE_BYTES = T::NF * FIELD_BYTES + (T::OWN ? OWN_BYTES : 0) + CODE_BYTES;
    static constexpr int OWN_OFF = T::NF * FIELD_BYTES;
    static constexpr int CODE_OFF = OWN_OFF + (T::OWN ? OWN_BYTES : 0);
    static constexpr int U_OFF = STAGES * STAGE_BYTES;
    static constexpr int CTAB_OFF = U_OFF + NU * FIELD_BYTES;
    // 2-bit codes: the coefficients of three faces at once from a 64-entry table of 32-byte entries, placed at
    // the first 2048-byte boundary inside a 4 KB region (its address is ORed with the entry offset)
    static constexpr int T3_OFF = CTAB_OFF + PF_CTAB * 8;
    static constexpr int T3_BYTES = (STORED || CODE32) ? 0 : 4096;
    // DIAG modes: the diagonal and the reciprocal half of the Jacobi division (recip_nb) as functions of the 12-bit
    // code of a node, 4096 pairs of doubles, built by the block at its start
    static constexpr int DTAB_OFF = T3_OFF + T3_BYTES;
    static constexpr int DTAB_BYTES = DIAG ? 4096 * 16 : 0;
    static constexpr int SCRATCH_OFF = DTAB_OFF + DTAB_BYTES;
    static constexpr int BAR_OFF = SCRATCH_OFF + 3 * 32 * (int)sizeof(dd);
    static constexpr int SC_OFF = ((BAR_OFF + 16 * STAGES + 8 * NU + 15) / 16) * 16;   // after full[S], empty[S], ready[NU]
    static constexpr int TOTAL = SC_OFF + 256;                       // the block's copy of the scalars
    static_assert(TOTAL <= 232448, "dynamic shared memory of a block (227 KB)");
    static_assert(CTAB_OFF % 128 == 0, "ctab_at ORs table offsets into the table address");
    static constexpr unsigned TX_BYTES = (unsigned)(T::NF * BX * BY * 8 + (T::OWN ? OWN_BYTES : 0) + (STORED ? 0 : CODE_TX));
};

__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }

// The mbarriers are addressed by 32-bit shared-memory addresses that every thread derives once from the block's
// base (kept opaque to the compiler, which otherwise re-derives the base from special registers at every use).
__device__ __forceinline__ unsigned opaque_u32(unsigned v) {
    unsigned r;
    asm volatile("mov.u32 %0, %1;" : "=r"(r) : "r"(v));
    return r;
}
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) { while (!mbar_try_wait(bar, parity)) {} }
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* map, unsigned bar, int x, int y, int z) {
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
        ::"r"(dst), "l"(map), "r"(bar), "r"(x), "r"(y), "r"(z)
        : "memory");
}

// Position in a ring of N slots that is walked one slot at a time: slot index and the parity of the current lap
// (the phase bit an mbarrier of the slot is waited on with).  Advancing costs an add, a compare and two selects,
// whatever N is -- the rings run on across the work items of a persistent block, so the position is run-time state.
template <int N>
struct Ring {
    unsigned idx, par;
    __device__ __forceinline__ void reset() { idx = 0u; par = 0u; }
    __device__ __forceinline__ void next() {
        const bool wrap = idx == (unsigned)(N - 1);
        idx = wrap ? 0u : idx + 1u;
        par ^= wrap ? 1u : 0u;
    }
};

// rc: recip_nb(a) from the table of the DIAG modes (unused otherwise)
template <int MODE, bool PRECOND>
__device__ __forceinline__ double u_of(double r, double p, double v, double a, double rc, bool first, double c1, double c2,
                                       double& numer, DivRange& range) {
    constexpr bool TAB = MODE == MODE_K1D || MODE == MODE_K2D || MODE == MODE_K2MD;
    if (MODE == MODE_K1 || MODE == MODE_K1D) numer = p_new_at<PRECOND>(first, c1, c2, r, p, v);
    else if (MODE == MODE_K2 || MODE == MODE_K2M || MODE == MODE_K2D || MODE == MODE_K2MD) numer = s_at(c1, r, v);
    else { numer = r; return r; }    // residual modes: the field is x itself (passed in r)
    // == jacobi<PRECOND>(numer, a) of the direct kernels
    return PRECOND ? (TAB ? dvd_rcp(numer, a, rc, range) : dvd_nb(numer, a, range)) : numer;
}

// Merged solver, K31: from the old r, p, v, t of a node: s (step 13), the new r (step 17), the new p (step 9 of the next
// iteration) and u = M^-1 p'.
template <bool PRECOND, bool TAB>
__device__ __forceinline__ double u31_of(double r, double p, double v, double t, double a, double rc, double alpha,
                                         double omega, double beta, double& s, double& rn, double& pn, DivRange& range) {
    s = s_at(alpha, r, v);
    rn = sub(s, mul(omega, t));
    pn = p_new_at<PRECOND>(false, beta, omega, rn, p, v);
    return PRECOND ? (TAB ? dvd_rcp(pn, a, rc, range) : dvd_nb(pn, a, range)) : pn;
}

// Coefficient of field d of node e (0 or 1) of the thread's code word(s): one shift, one three-input logic
// operation that masks the field and ORs in the (128-byte aligned) shared address of the table, one load.
template <bool CODE32>
__device__ __forceinline__ double ctab_at(unsigned ctab_addr, unsigned w0, unsigned w1, int e, int d) {
    unsigned off;
    if (CODE32) {
        const unsigned w = e ? w1 : w0;
        const int sh = 4 * d - 3;
        off = ((sh >= 0 ? (w >> sh) : (w << -sh)) & 0x78u) | ctab_addr;
    } else {
        const int sh = 16 * e + 2 * d - 3;
        off = ((sh >= 0 ? (w0 >> sh) : (w0 << -sh)) & 0x18u) | ctab_addr;
    }
    double c;
    asm("ld.shared.f64 %0, [%1];" : "=d"(c) : "r"(off));
    return c;
}

// 2-bit codes: the coefficients of faces 3g+1 .. 3g+3 (g = 0, 1) of node e of the thread's code word, from the
// table whose entry i holds ctab[i & 3], ctab[(i >> 2) & 3], ctab[(i >> 4) & 3]: one shift, one logic operation
// (mask the six code bits, scaled by 32, and OR in the 2048-byte aligned table address), two loads.
__device__ __forceinline__ void ctab3_at(unsigned t3_addr, unsigned w0, int e, int g, double (&c)[3]) {
    const int sh = 16 * e + 6 * g - 5;
    const unsigned off = ((sh >= 0 ? (w0 >> sh) : (w0 << -sh)) & 0x7e0u) | t3_addr;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(c[0]), "=d"(c[1]) : "r"(off));
    asm("ld.shared.f64 %0, [%1+16];" : "=d"(c[2]) : "r"(off));
}

// DIAG modes: the diagonal of a node as a function of its 12-bit code (six 2-bit fields).  The Poisson assembly adds
// the six face coefficients in the order of the fields, starting from 0.0, and the table holds their negatives, so
// the negated sum of the table entries has the same bits; rows without a face (code 0) are the identity rows,
// diagonal 1.  Every block tabulates the 4096 values once at its start (ctab: the 16-entry coefficient table), each
// with recip_nb of it: the divisor's half of the branch-free division, so that a Jacobi division costs a multiplication
// and two fused operations per node instead of nine (same bits: the same instruction sequence, split in two).
__device__ __forceinline__ double diag_of_code12(const double* ctab, unsigned code) {
    double sacc = 0.0;
#pragma unroll
    for (int d = 0; d < 6; ++d) sacc = add(sacc, ctab[(code >> (2 * d)) & 3u]);
    return code == 0u ? 1.0 : -sacc;
}
__device__ __forceinline__ double dtab_at(unsigned dtab_addr, unsigned w0, int e) {             // the diagonal alone
    const unsigned off = (e ? (w0 >> 12) & 0xfff0u : (w0 << 4) & 0xfff0u) + dtab_addr;
    double a;
    asm("ld.shared.f64 %0, [%1];" : "=d"(a) : "r"(off));
    return a;
}
__device__ __forceinline__ void dtab2_at(unsigned dtab_addr, unsigned w0, int e, double& a, double& rc) {   // with its reciprocal
    const unsigned off = (e ? (w0 >> 12) & 0xfff0u : (w0 << 4) & 0xfff0u) + dtab_addr;
    asm("ld.shared.v2.f64 {%0, %1}, [%2];" : "=d"(a), "=d"(rc) : "r"(off));
}

// Registers of one plane of a main thread: u at its two nodes, the numerators (p' or s), the diagonal,
// the own-only operand (r~ or b) and the stencil code word(s).
struct Slot {
    double u[2], n[2], a[2];
    double2 w;
    unsigned k0, k1;
};

template <int MODE, bool PRECOND, bool STORED, bool CODE32, int TYV, bool M2>
__global__ void __launch_bounds__(Geo<TYV>::NT, 1)
k_tma(const __grid_constant__ TmaArgs tm, GridDims g, Operator op, KrylovVecs kv, const Scalars* sc_in, Scalars* sc_out, ReduceBuf rb,
      SegPlan plan) {
    using L = Layout<MODE, STORED, CODE32, TYV>;
    constexpr int TY = Geo<TYV>::TY, NW_CONSUMER = Geo<TYV>::NW_CONSUMER, NT_CONSUMER = Geo<TYV>::NT_CONSUMER,
                  BY = Geo<TYV>::BY, FIELD_BYTES = Geo<TYV>::FIELD_BYTES;
    using T = ModeTraits<MODE>;
    constexpr int NS = L::STAGES;
    constexpr int NF = T::NF;
    constexpr bool DIAG = L::DIAG;                   // the diagonal is formed from the codes
    constexpr bool K1 = MODE == MODE_K1 || MODE == MODE_K1D;
    constexpr bool K2M = MODE == MODE_K2M || MODE == MODE_K2MD;     // the k2 of the merged solver: + r~.t
    constexpr bool K2 = MODE == MODE_K2 || MODE == MODE_K2D || K2M;
    constexpr bool K31 = MODE == MODE_K31 || MODE == MODE_K31D;     // the fused k3 + k1 of the merged solver
    constexpr bool RES = MODE == MODE_R0 || MODE == MODE_R1;
    static_assert(!DIAG || (!STORED && !CODE32), "the diagonal is formed from 2-bit codes");
    static_assert(!(K2M || K31) || !STORED, "the merged kernels exist for operators in code form");
    pdl_launch_dependents();
    extern __shared__ __align__(128) unsigned char smem[];
    double* ctab_s = reinterpret_cast<double*>(smem + L::CTAB_OFF);
    dd* scratch = reinterpret_cast<dd*>(smem + L::SCRATCH_OFF);
    // full[s]: the TMA copies of stage s have landed; empty[s]: all 18 consumer warps are done with stage s;
    // ready[b]: all 18 consumer warps have written their part of u buffer b
    const unsigned sbase = opaque_u32(smem_u32(smem));
    const unsigned full_a = sbase + (unsigned)L::BAR_OFF, empty_a = full_a + 8u * NS, ready_a = empty_a + 8u * NS;

    const int tid = threadIdx.x, lane = tid & 31, wid = tid >> 5;
    // Persistent blocks: work item i = (tile i % ntiles, z chunk i / ntiles), x tiles fastest, so that the
    // blocks running at any moment work on neighbouring tiles of the same chunk and share their halo rows in
    // L2.  Block b takes items b, b + gridDim.x, ...; the stage and u-buffer rings run on across items, so
    // the producer already loads the next item while the consumers finish the current one, and a launch leaves
    // at most one set of partial sums per SM for the next kernel to combine.
    // (The stored variant, short of registers, runs one item per block.)
    constexpr bool PERSIST = !STORED;
    Scalars* S = reinterpret_cast<Scalars*>(smem + L::SC_OFF);

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < NS; ++s) { mbar_init(full_a + 8u * s, 1); mbar_init(empty_a + 8u * s, NW_CONSUMER); }
#pragma unroll
        for (int b = 0; b < NU; ++b) mbar_init(ready_a + 8u * b, NW_CONSUMER);
        fence_proxy_async();
    }
    if (!STORED && tid < PF_CTAB) ctab_s[tid] = op.ctab[tid];
    unsigned t3_addr = 0u;
    if (!STORED && !CODE32) {
        unsigned char* region = smem + L::T3_OFF;
        const unsigned a = smem_u32(region);
        t3_addr = (a + 2047u) & ~2047u;
        double* T3 = reinterpret_cast<double*>(region + (t3_addr - a));
        if (tid < 256) T3[tid] = (tid & 3) < 3 ? op.ctab[((tid >> 2) >> (2 * (tid & 3))) & 3] : 0.0;
    }
    const unsigned ctab_addr = smem_u32(ctab_s);           // 128-byte aligned: CTAB_OFF and the smem base are
    __syncthreads();
    unsigned dtab_addr = 0u;
    if (DIAG) {
        double* dtab = reinterpret_cast<double*>(smem + L::DTAB_OFF);
        dtab_addr = smem_u32(dtab);
        for (int k = tid; k < 4096; k += blockDim.x) {
            const double a = diag_of_code12(ctab_s, (unsigned)k);
            reinterpret_cast<double2*>(dtab)[k] = make_double2(a, recip_nb(a));
        }
        __syncthreads();
    }
    pdl_wait();                                            // everything above is independent of the previous kernel
    constexpr int KIND = K1 ? PEND_K1 : (K2M ? PEND_K2M : (K2 ? PEND_K2 : (K31 ? PEND_K31 : (MODE == MODE_R0 ? PEND_INIT : PEND_TRUE))));
    const int ntx = plan.ntx;
    // plane k of the load sequence of the segment (tile, z0) into stage sidx; the producer lane only
    auto issue_plane = [&](int tile, int z0, int k, unsigned sidx) {
        const int px = (tile % ntx) * TX, py = (tile / ntx) * TY, pz = z0 - 1 + k;
        const unsigned st = sbase + sidx * (unsigned)L::STAGE_BYTES, bar = full_a + 8u * sidx;
        mbar_expect_tx(bar, L::TX_BYTES);
#pragma unroll
        for (int f = 0; f < NF; ++f) tma_load_3d(st + f * FIELD_BYTES, &tm.f[f], bar, px - 2, py - 1, pz);
        if (T::OWN) tma_load_3d(st + L::OWN_OFF, &tm.own, bar, px, py, pz);
        if (!STORED) tma_load_3d(st + L::CODE_OFF, &tm.code, bar, DIAG ? px - CXO : px, DIAG ? py - 1 : py, pz);
    };
    // The first stages do not depend on the scalars: they are requested before the block combines the previous
    // kernel's partial sums, so the loads fly while the scalar step is taken.
    int pre_issued = 0;
    if (tid == NT_CONSUMER) {
        SegIter<PERSIST, M2> it0;
        it0.init(plan, (int)blockIdx.x, (int)gridDim.x);
        int tile_f, z0f, z1f;
        if (it0.next(plan, g.nz, (int)blockIdx.x, (int)gridDim.x, tile_f, z0f, z1f)) {
            const int nqf = z1f - z0f + 2;
            for (; pre_issued < NS && pre_issued < nqf; ++pre_issued) issue_plane(tile_f, z0f, pre_issued, (unsigned)pre_issued);
        }
    }
    if (!begin_kernel(KIND, S, sc_in, sc_out, rb, kv.hist, scratch)) {
        // the solve is over: let the requested stages land before the block's shared memory is released
        for (int k = 0; k < pre_issued; ++k) mbar_wait(full_a + 8u * k, 0u);
        return;
    }

    dd q[3] = {dd_zero(), dd_zero(), dd_zero()};
    double rmax = 0.0;                     // residual modes: ||b - A x||_inf; K31: ||r'||_inf
    DivRange range;                        // quotients of the branch-free division (reading D4)
    range.reset();
    bool diag_bad = false;                 // MODE_R0 of a preconditioned solve: the diagonal itself, once per solve

    // Ring positions (run-time state: the rings run on across the items of a persistent block).
    //   cr: stage of the next plane this thread consumes / (producer lane) fills
    //   ur: u buffer of the next plane to be published; its predecessor in the ring is the plane published before
    Ring<NS> cr;
    Ring<NU> ur;
    cr.reset(); ur.reset();
    bool have_prev = false;                // a plane has been published before (by an earlier item)
    if (wid == NW_CONSUMER) { for (int k = 0; k < pre_issued; ++k) cr.next(); }
    int issued = pre_issued;               // producer: planes requested so far

    bool first = false; double c1 = 0.0, c2 = 0.0, c3 = 0.0;     // (K31 reads its scalars from S where it uses them)
    if (K1) { first = S->first != 0; c1 = S->beta; c2 = S->omega; }
    else if (K2) { c1 = S->alpha; }
    (void)c3;
    const bool is_main = wid < TY;
    // main thread: nodes (x, y) and (x+1, y) of box row wid+1; nx is even so both are inside or both outside.
    // halo warp TY: box row 0 (pairs) and box column 1 (lanes 0..15); halo warp TY+1: row BY-1 and column BX-2.
    const int brow = is_main ? wid + 1 : (wid == TY ? 0 : BY - 1);
    const long long plane = (long long)g.nx * g.ny;
    const int pair_box = brow * BX + 2 + 2 * lane;                 // element offset in a halo box
    const int own_tile = (brow - 1) * TX + 2 * lane;               // element offset in an own-only box (main)
    const int pair_code = brow * BXC + CXO + 2 * lane;             // MODE_K1D: element offset in the code box with halo

    SegIter<PERSIST, M2> seg;
    seg.init(plan, (int)blockIdx.x, (int)gridDim.x);
    int skip = pre_issued;                 // producer: planes of the first segment that are already requested
    int tile, z0, z1;
    while (seg.next(plan, g.nz, (int)blockIdx.x, (int)gridDim.x, tile, z0, z1)) {
    const int x0 = (tile % ntx) * TX, y0 = (tile / ntx) * TY;
    const int nq = z1 - z0 + 2;            // plane k of this segment's load sequence is z0 - 1 + k

    if (wid == NW_CONSUMER) {
        // ---- producer warp: one lane keeps the ring of stages filled ----------------------------
        if (lane == 0) {
            for (int k = skip; k < nq; ++k) {
                if (issued >= NS) mbar_wait(empty_a + 8u * cr.idx, cr.par ^ 1u);   // the consumers' release of the lap before
                issue_plane(tile, z0, k, cr.idx);
                cr.next();
                ++issued;
            }
            skip = 0;
        }
        __syncwarp();
    } else {
        const int x = x0 + 2 * lane, y = y0 - 1 + brow;
        const bool pair_ok = x < g.nx && y >= 0 && y < g.ny;
        const long long own_off = x + (long long)g.nx * y;

        // operands of the thread's pair of nodes in a plane -> u, numerator, diagonal (K31: also s, the new r and the old p)
        auto form_pair = [&](const unsigned char* st, bool ok, double (&u)[2], double (&n)[2], double (&a)[2],
                             double (&sx)[2], double (&rx)[2], double (&px)[2]) {
            const double* F0 = reinterpret_cast<const double*>(st);
            const double* F1 = reinterpret_cast<const double*>(st + FIELD_BYTES);
            const double* F2 = reinterpret_cast<const double*>(st + 2 * FIELD_BYTES);
            const double* F3 = reinterpret_cast<const double*>(st + 3 * FIELD_BYTES);
            const double* F4 = reinterpret_cast<const double*>(st + 4 * FIELD_BYTES);
            double2 fr = *reinterpret_cast<const double2*>(F0 + pair_box), fp = make_double2(0, 0),
                    fv = make_double2(0, 0), ft = make_double2(0, 0), fa, frc = make_double2(1.0, 1.0);
            if (K1 || K31) {
                fp = *reinterpret_cast<const double2*>(F1 + pair_box);
                fv = *reinterpret_cast<const double2*>(F2 + pair_box);
                if (K31) ft = *reinterpret_cast<const double2*>(F3 + pair_box);
                if (!DIAG) fa = *reinterpret_cast<const double2*>((K31 ? F4 : F3) + pair_box);
            } else if (K2) {
                fv = *reinterpret_cast<const double2*>(F1 + pair_box);
                if (!DIAG) fa = *reinterpret_cast<const double2*>(F2 + pair_box);
            } else {
                fa = *reinterpret_cast<const double2*>(F1 + pair_box);
            }
            if (DIAG) {
                const unsigned cw = *reinterpret_cast<const unsigned*>(st + L::CODE_OFF + 2 * pair_code);
                dtab2_at(dtab_addr, cw, 0, fa.x, frc.x);
                dtab2_at(dtab_addr, cw, 1, fa.y, frc.y);
            }
            // the divisor of the branch-free division is tested once per solve, here (D4)
            if (MODE == MODE_R0 && PRECOND && ok) diag_bad |= DivRange::diag_bad(fa.x) | DivRange::diag_bad(fa.y);
            if (!ok) { fa = make_double2(1.0, 1.0); frc = make_double2(1.0, 1.0); }   // zero-filled nodes: keep u finite (0/1)
            if (K31) {
                // alpha, omega, beta from the block's copy of the scalars at every use: three shared loads per plane
                // instead of six registers held through the loop (this kernel is the one short of registers)
                const double al = S->alpha, om = S->omega, be = S->beta;
                u[0] = u31_of<PRECOND, DIAG>(fr.x, fp.x, fv.x, ft.x, fa.x, frc.x, al, om, be, sx[0], rx[0], n[0], range);
                u[1] = u31_of<PRECOND, DIAG>(fr.y, fp.y, fv.y, ft.y, fa.y, frc.y, al, om, be, sx[1], rx[1], n[1], range);
                px[0] = fp.x; px[1] = fp.y;
            } else {
                u[0] = u_of<MODE, PRECOND && !RES>(fr.x, fp.x, fv.x, fa.x, frc.x, first, c1, c2, n[0], range);
                u[1] = u_of<MODE, PRECOND && !RES>(fr.y, fp.y, fv.y, fa.y, frc.y, first, c1, c2, n[1], range);
            }
            a[0] = fa.x; a[1] = fa.y;
        };
        // the stage of the next plane: wait until its copies have landed; data pointer
        auto wait_full = [&]() -> const unsigned char* {
            mbar_wait(full_a + 8u * cr.idx, cr.par);
            return smem + cr.idx * (unsigned)L::STAGE_BYTES;
        };
        // u of plane k (k >= 1) lives in the u buffer at ring position ur when it is published.  No block-wide
        // barrier: a warp that waits for plane k before it overwrites plane k-2's buffer with plane k+1 cannot race
        // a reader (every warp that published plane k has finished differencing plane k-2).
        auto u_ptr = [&](unsigned idx) -> double* { return reinterpret_cast<double*>(smem + L::U_OFF + idx * (unsigned)FIELD_BYTES); };

        if (!is_main) {
            // ---- halo warps: u on the halo ring of every plane that gets differenced ---------------
            int col_box = 0; bool col_ok = false;
            const bool col_any = lane < TY;
            if (col_any) {
                const int hx = wid == TY ? 1 : BX - 2, hy = 1 + lane;
                col_box = hy * BX + hx;
                const int gx = x0 - 2 + hx, gy = y0 - 1 + hy;
                col_ok = gx >= 0 && gx < g.nx && gy < g.ny;
            }
            wait_full();                                                // plane z0-1 has no xy neighbours to serve
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_a + 8u * cr.idx);
            cr.next();
            for (int k = 1; k < nq; ++k) {
                if (have_prev) {                                         // the plane published before this one: the buffer
                    const unsigned pi = ur.idx == 0u ? (unsigned)(NU - 1) : ur.idx - 1u;     // written 3 publishes ago is free
                    mbar_wait(ready_a + 8u * pi, ur.par ^ (ur.idx == 0u ? 1u : 0u));
                }
                const unsigned char* st = wait_full();
                const int z = z0 - 1 + k;
                const bool zin = z >= 0 && z < g.nz;
                double* u_s = u_ptr(ur.idx);
                double u[2], n[2], a[2], sx[2], rx[2], px[2];
                form_pair(st, pair_ok && zin, u, n, a, sx, rx, px);
                *reinterpret_cast<double2*>(u_s + pair_box) = make_double2(u[0], u[1]);
                if (col_any) {
                    const double* F0 = reinterpret_cast<const double*>(st);
                    const double* F1 = reinterpret_cast<const double*>(st + FIELD_BYTES);
                    const double* F2 = reinterpret_cast<const double*>(st + 2 * FIELD_BYTES);
                    const double* F3 = reinterpret_cast<const double*>(st + 3 * FIELD_BYTES);
                    const double* F4 = reinterpret_cast<const double*>(st + 4 * FIELD_BYTES);
                    double hr = F0[col_box], hp = 0.0, hv = 0.0, ht = 0.0, ha = 1.0, hrc = 1.0;
                    if (K1 || K31) {
                        hp = F1[col_box]; hv = F2[col_box];
                        if (K31) ht = F3[col_box];
                        if (!DIAG) ha = (K31 ? F4 : F3)[col_box];
                    }
                    else if (K2) { hv = F1[col_box]; if (!DIAG) ha = F2[col_box]; }
                    if (DIAG) {
                        const int hxc = (wid == TY ? 1 : BX - 2) + CXO - 2;     // the code box starts CXO - 2 columns further left
                        const unsigned cw = *reinterpret_cast<const unsigned short*>(st + L::CODE_OFF + 2 * ((1 + lane) * BXC + hxc));
                        dtab2_at(dtab_addr, cw, 0, ha, hrc);
                    }
                    if (!(col_ok && zin)) { ha = 1.0; hrc = 1.0; }
                    double d0, d1, d2;
                    if (K31) u_s[col_box] = u31_of<PRECOND, DIAG>(hr, hp, hv, ht, ha, hrc, S->alpha, S->omega, S->beta, d0, d1, d2, range);
                    else u_s[col_box] = u_of<MODE, PRECOND && !RES>(hr, hp, hv, ha, hrc, first, c1, c2, d0, range);
                }
                __syncwarp();                                           // publish: this warp's part of plane k is written
                if (lane == 0) { mbar_arrive(ready_a + 8u * ur.idx); mbar_arrive(empty_a + 8u * cr.idx); }
                ur.next(); cr.next();
                have_prev = true;
            }
        } else {
            // ---- main warps -------------------------------------------------------------------------
            // form u(z+1) into slot `up` (+ the other shared buffer) and difference plane z (slot c, z neighbours
            // in dn and up, xy neighbours from shared).  Everything between the wait and the stage release is
            // one basic block: the divisions of plane z+1 and the stencil chain of plane z are independent and
            // get interleaved by the scheduler.  Nodes outside the grid see zero operands and zero codes, give
            // exact zeros and add nothing to the inner products; only their stores are predicated.
            // Running global positions: op_row = index of the thread's pair in the plane that load_slot forms next
            // (z0 - 1 + k), out_row = in the plane that step differences next.
            long long form_i = own_off + plane * (z0 - 1);
            long long out_i = own_off + plane * z0;
            int zf = z0 - 1;                                            // plane load_slot forms next
            // K31: y of the plane that load_slot forms next, requested one plane ahead (a global load in front of the
            // dependent additions of step 16 would stall the whole basic block).  The request is issued right AFTER the
            // warp's mbarrier arrivals, never before them: an arrive is a release, and the hardware holds it back until
            // the thread's outstanding loads have returned -- with the load in front of it every `ready` barrier, and
            // with it the whole block, waited a DRAM round trip per plane (0.287 ms per launch instead of ...).
            double2 ypre = make_double2(0, 0);
            auto y_prefetch = [&]() {
                if (K31 && pair_ok && zf >= z0 && zf < z1) {
                    ypre = *reinterpret_cast<const double2*>(kv.y + form_i);
                    // (an additional prefetch.global.L2 two planes ahead was measured and removed: 0.260 -> 0.258 ms
                    // without it at 256^3, 2.18 -> 2.13 ms at 512^3, same DRAM bytes)
                }
            };
            auto load_slot = [&](Slot& up, bool to_shared, double* u_dst) {
                const unsigned char* st = wait_full();
                const bool zown = zf >= z0 && zf < z1;
                const bool ok = pair_ok && zf >= 0 && zf < g.nz;
                double sx[2], rx[2], px[2];
                form_pair(st, ok, up.u, up.n, up.a, sx, rx, px);
                if (T::OWN)
                    up.w = *reinterpret_cast<const double2*>(reinterpret_cast<const double*>(st + L::OWN_OFF) + own_tile);
                if (!STORED) {
                    if (CODE32) {
                        const uint2 cw = *reinterpret_cast<const uint2*>(st + L::CODE_OFF + 4 * own_tile);
                        up.k0 = cw.x; up.k1 = cw.y;
                    } else if (DIAG) {
                        up.k0 = *reinterpret_cast<const unsigned*>(st + L::CODE_OFF + 2 * pair_code);
                    } else {
                        up.k0 = *reinterpret_cast<const unsigned*>(st + L::CODE_OFF + 2 * own_tile);
                    }
                }
                if (K1 && ok && zown)                                   // p' is an output of steps 5-9
                    *reinterpret_cast<double2*>(kv.p_out + form_i) = make_double2(up.n[0], up.n[1]);
                if (K31 && zown) {                                      // (uniform over the block)
                    // steps 16-17 of the closing iteration and step 9 of the next: y, r', p' at the thread's own nodes;
                    // r'.r', r~.r', max |r'| (nodes outside the grid hold zeros and add nothing)
                    if (ok) {
                        const double al = S->alpha, om = S->omega;
                        const double y0n = add(add(ypre.x, mul(al, px[0])), mul(om, sx[0]));
                        const double y1n = add(add(ypre.y, mul(al, px[1])), mul(om, sx[1]));
                        *reinterpret_cast<double2*>(kv.y + form_i) = make_double2(y0n, y1n);
                        *reinterpret_cast<double2*>(kv.r_out + form_i) = make_double2(rx[0], rx[1]);
                        *reinterpret_cast<double2*>(kv.p_out + form_i) = make_double2(up.n[0], up.n[1]);
                    }
                    dd_fma(q[1], rx[0], rx[0]); dd_fma(q[1], rx[1], rx[1]);
                    dd_fma(q[2], up.w.x, rx[0]); dd_fma(q[2], up.w.y, rx[1]);
                    rmax = max_abs(max_abs(rmax, rx[0]), rx[1]);
                }
                if (to_shared) *reinterpret_cast<double2*>(u_dst + pair_box) = make_double2(up.u[0], up.u[1]);
                form_i += plane; ++zf;
            };
            constexpr bool DEFER = !STORED && !K31 && !K2M;  // the stored variant, K31 and K2M have no registers to spare for it
            double pa[2] = {0.0, 0.0}, pb[2] = {0.0, 0.0};   // operands of the deferred inner products (zeros add nothing)
            double pc[2] = {0.0, 0.0};                       // K2M: r~ of the plane whose t is in pa
            // The loop below is unrolled three ways and NU = 3, so the u buffer of plane z0 + 3m + J is a fixed
            // rotation J of the item's first one and the parity of its `ready` barrier a fixed bit xor (m & 1):
            // three addresses and three bits per item instead of ring arithmetic per plane and use.
            static_assert(NU == 3, "the rotation below is written for three u buffers");
            unsigned bj[3];                                             // buffer of rotation j
            unsigned pbits = 0u;                                        // bit j: parity of rotation j at m = 0
            {
                Ring<NU> t = ur;
#pragma unroll
                for (int j = 0; j < 3; ++j) { bj[j] = t.idx; pbits |= t.par << j; t.next(); }
            }
            unsigned mp = 0u;                                           // (z - z0) / 3 & 1
            auto U = [&](int j) { return u_ptr(bj[j]); };
            auto R = [&](int j) { return ready_a + 8u * bj[j]; };
            auto step = [&](auto Jc, const Slot& dn, const Slot& c, Slot& up) {
                constexpr int J = decltype(Jc)::value, J1 = (J + 1) % 3;
                const long long i = out_i;
                const double* u_s = U(J);
                mbar_wait(R(J), ((pbits >> J) & 1u) ^ mp);               // every warp has published the plane to difference
                load_slot(up, true, U(J1));
                // Publish at once: u(z+1) is in shared memory and the stage is consumed.  Arriving here, before this
                // plane's stencil, rather than after it lets the other warps (and the producer) run on up to a plane
                // ahead.  Still race-free: whoever overwrites the buffer of plane z (with plane z+3) first waits for
                // `ready` of plane z+2, on which this warp arrives in its next step, i.e. after the reads below.
                __syncwarp();
                if (lane == 0) { mbar_arrive(R(J1)); mbar_arrive(empty_a + 8u * cr.idx); }
                cr.next();
                y_prefetch();
                // inner products of the PREVIOUS plane: a third independent chain beside the divisions of plane
                // z+1 and the 7-point sums of plane z
                if (DEFER && K1) {
                    dd_fma(q[0], pa[0], pb[0]); dd_fma(q[1], pa[1], pb[1]);
                } else if (DEFER && K31) {
                    dd_fma(q[0], pa[0], pb[0]); dd_fma(q[0], pa[1], pb[1]);
                } else if (DEFER && K2) {
                    dd_fma(q[0], pa[0], pb[0]); dd_fma(q[0], pa[1], pb[1]);
                    dd_fma(q[1], pa[0], pa[0]); dd_fma(q[1], pa[1], pa[1]);
                    if (K2M) { dd_fma(q[2], pc[0], pa[0]); dd_fma(q[2], pc[1], pa[1]); }
                }
                const double2 us = *reinterpret_cast<const double2*>(u_s + pair_box - BX);
                const double2 un = *reinterpret_cast<const double2*>(u_s + pair_box + BX);
                const double uw = u_s[pair_box - 1], ue = u_s[pair_box + 2];
                double2 cf[6];
                if (STORED) {
#pragma unroll
                    for (int d = 0; d < 6; ++d)
                        cf[d] = pair_ok ? *reinterpret_cast<const double2*>(op.offd[d] + i) : make_double2(0, 0);
                }
                double out[2], c5[2];
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    double cc[6];
                    if (STORED) {
#pragma unroll
                        for (int d = 0; d < 6; ++d) cc[d] = e == 0 ? cf[d].x : cf[d].y;
                    } else if (CODE32) {
#pragma unroll
                        for (int d = 0; d < 6; ++d)
                            cc[d] = ctab_at<CODE32>(ctab_addr, c.k0, c.k1, e, d);
                    } else {
                        double c3[3];
                        ctab3_at(t3_addr, c.k0, e, 0, c3); cc[0] = c3[0]; cc[1] = c3[1]; cc[2] = c3[2];
                        ctab3_at(t3_addr, c.k0, e, 1, c3); cc[3] = c3[0]; cc[4] = c3[1]; cc[5] = c3[2];
                    }
                    // (DIAG: looked up again from the code rather than kept in three register slots)
                    const double a_own = (DIAG && K31) ? dtab_at(dtab_addr, c.k0, e) : c.a[e];
                    double acc = mul(a_own, c.u[e]);
                    acc = add(acc, mul(cc[0], e == 0 ? c.u[1] : ue));
                    acc = add(acc, mul(cc[1], e == 1 ? c.u[0] : uw));
                    acc = add(acc, mul(cc[2], e == 0 ? us.x : us.y));
                    acc = add(acc, mul(cc[3], e == 0 ? un.x : un.y));
                    acc = add(acc, mul(cc[4], dn.u[e]));
                    out[e] = acc;
                    c5[e] = cc[5];
                }
                out[0] = add(out[0], mul(c5[0], up.u[0]));
                out[1] = add(out[1], mul(c5[1], up.u[1]));
                if (K1 || K31) {
                    if (pair_ok) *reinterpret_cast<double2*>(kv.v_out + i) = make_double2(out[0], out[1]);
                    if (DEFER) { pa[0] = c.w.x; pa[1] = c.w.y; pb[0] = out[0]; pb[1] = out[1]; }   // r~ . v', next step
                    else if (K31) { dd_fma(q[0], c.w.x, out[0]); dd_fma(q[0], c.w.y, out[1]); }
                    else { dd_fma(q[0], c.w.x, out[0]); dd_fma(q[1], c.w.y, out[1]); }
                } else if (K2) {
                    if (pair_ok) *reinterpret_cast<double2*>(kv.t + i) = make_double2(out[0], out[1]);
                    if (DEFER) {                                        // t . s, t . t (K2M: r~ . t), next step
                        pa[0] = out[0]; pa[1] = out[1]; pb[0] = c.n[0]; pb[1] = c.n[1];
                        if (K2M) { pc[0] = c.w.x; pc[1] = c.w.y; }
                    }
                    else {
                        dd_fma(q[0], out[0], c.n[0]); dd_fma(q[0], out[1], c.n[1]);
                        dd_fma(q[1], out[0], out[0]); dd_fma(q[1], out[1], out[1]);
                        if (K2M) { dd_fma(q[2], c.w.x, out[0]); dd_fma(q[2], c.w.y, out[1]); }
                    }
                } else {
                    const double r0 = sub(c.w.x, out[0]), r1 = sub(c.w.y, out[1]);
                    if (MODE == MODE_R0) {
                        if (pair_ok) {
                            *reinterpret_cast<double2*>(kv.r + i) = make_double2(r0, r1);
                            *reinterpret_cast<double2*>(kv.rt + i) = make_double2(r0, r1);
                        }
                        dd_fma(q[0], c.w.x, c.w.x); dd_fma(q[0], c.w.y, c.w.y);
                    }
                    dd_fma(q[1], r0, r0); dd_fma(q[1], r1, r1);
                    rmax = max_abs(max_abs(rmax, r0), r1);
                }
                out_i += plane;
            };

            Slot s0, s1, s2;
            s0.w = s1.w = s2.w = make_double2(0, 0);
            s0.k0 = s0.k1 = s1.k0 = s1.k1 = s2.k0 = s2.k1 = 0u;
            load_slot(s0, false, nullptr);         // plane z0-1: registers only
            __syncwarp();
            if (lane == 0) mbar_arrive(empty_a + 8u * cr.idx);
            cr.next();
            y_prefetch();
            if (have_prev) {                       // last plane of the previous item: its buffer-mates are free
                const unsigned pi = ur.idx == 0u ? (unsigned)(NU - 1) : ur.idx - 1u;
                mbar_wait(ready_a + 8u * pi, ur.par ^ (ur.idx == 0u ? 1u : 0u));
            }
            load_slot(s1, true, U(0));             // plane z0
            __syncwarp();
            if (lane == 0) { mbar_arrive(R(0)); mbar_arrive(empty_a + 8u * cr.idx); }
            cr.next();
            y_prefetch();
            for (int z = z0; z < z1; z += 3) {     // slots rotate by renaming, not by moving registers
                step(std::integral_constant<int, 0>{}, s0, s1, s2);
                if (z + 1 >= z1) break;
                step(std::integral_constant<int, 1>{}, s1, s2, s0);
                if (z + 2 >= z1) break;
                step(std::integral_constant<int, 2>{}, s2, s0, s1);
                mp ^= 1u;
            }
            if (DEFER && K1) {                               // the last plane's inner products
                dd_fma(q[0], pa[0], pb[0]); dd_fma(q[1], pa[1], pb[1]);
            } else if (DEFER && K31) {
                dd_fma(q[0], pa[0], pb[0]); dd_fma(q[0], pa[1], pb[1]);
            } else if (DEFER && K2) {
                dd_fma(q[0], pa[0], pb[0]); dd_fma(q[0], pa[1], pb[1]);
                dd_fma(q[1], pa[0], pa[0]); dd_fma(q[1], pa[1], pa[1]);
                if (K2M) { dd_fma(q[2], pc[0], pa[0]); dd_fma(q[2], pc[1], pa[1]); }
            }
            pa[0] = pa[1] = pb[0] = pb[1] = pc[0] = pc[1] = 0.0;     // (the next item starts with nothing deferred)
            // the item published nq - 1 planes
            {
                const int adv = nq - 1;
                ur.par ^= (unsigned)(adv / NU) & 1u;
                for (int r = adv % NU; r > 0; --r) ur.next();
            }
            have_prev = true;
        }
    }
    }

    if (range.bad() || diag_bad) *rb.fault = 1;     // the host repeats the solve with the __ddiv_rn kernels
    // this block's partial sums; the next kernel of the stream combines them (pf_common.cuh)
    if (K1) {
        dd_add(q[0], q[1]);                // two chains for instruction-level parallelism, one quantity
        dd q1[1] = {q[0]};
        store_partials<1, false>(q1, 0.0, scratch, rb, PEND_K1);
    } else if (K2M) {
        store_partials<3, false>(q, 0.0, scratch, rb, PEND_K2M);
    } else if (K2) {
        dd q2[2] = {q[0], q[1]};
        store_partials<2, false>(q2, 0.0, scratch, rb, PEND_K2);
    } else if (K31) {
        store_partials<3, true>(q, rmax, scratch, rb, PEND_K31);
    } else {
        dd q2[2] = {q[0], q[1]};
        store_partials<2, true>(q2, rmax, scratch, rb, KIND);
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

bool halo_map(CUtensorMap* m, const double* base, const GridDims& g, int ty) {
    return make_map(m, base, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, g, g.nx, BX, ty + 2);
}
bool own_map(CUtensorMap* m, const double* base, const GridDims& g, int ty) {
    return make_map(m, base, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 8, g, g.nx, TX, ty);
}

// The decomposition of a launch for tiles of `ty` rows (SegPlan above): the equal-chunk plan, or the two-group plan
// where its longest block is shorter by 3 % or more.  `persist`: blocks loop over segments (else one item per block).
// Lengths are counted in plane steps, z1 - z0 + 2 per segment, which is what a block's time is proportional to.
SegPlan plan_segments(const GridDims& g, int ty, int sm_count, bool persist, int mode_forced /* -1: choose */) {
    SegPlan P;
    std::memset(&P, 0, sizeof(P));
    const int tx = (g.nx + TX - 1) / TX, tyb = (g.ny + ty - 1) / ty, T = tx * tyb;
    P.ntx = tx; P.ntiles = T;
    const int chunks0 = choose_zchunks(g, T, sm_count);
    P.zchunk = (g.nz + chunks0 - 1) / chunks0;
    const int chunks = (g.nz + P.zchunk - 1) / P.zchunk;
    P.nitems = T * chunks;
    P.blocks = persist ? std::min(sm_count, P.nitems) : P.nitems;
    if (!persist || mode_forced == 0 || T >= sm_count) return P;
    // longest block of the equal-chunk plan
    long long span0 = 0;
    for (int b = 0; b < P.blocks; ++b) {
        long long w = 0;
        for (int i = b; i < P.nitems; i += P.blocks) {
            const int z0 = (i / T) * P.zchunk;
            w += std::min(P.zchunk, g.nz - z0) + 2;
        }
        span0 = std::max(span0, w);
    }
    const int full = sm_count / T, R = sm_count - full * T;
    if (full == 1) {
        if (ty != TY_DEEP) return P;               // (the kernels of mode 2 are compiled for the 13-row tiles)
        // Mode 2.  (A plan like mode 1 with ONE layer in step, whose rest group takes almost half of the volume tile by
        // tile, gives up the sharing of halo rows in L2 between neighbouring tiles -- measured: K31 at 256^3 with 80
        // tiles, 0.233 -> 0.266 ms -- so here every group marches neighbouring tiles in step.)
        const int L = T - R;                       // tiles whose upper layer waits for group B
        if (mode_forced == 1 || L <= 0 || R / L < 1) return P;
        const int pieces = std::min(R / L, 8);
        long long best = -1; int bestD = 0, bestq = 0;
        for (int D = (g.nz + 1) / 2; D < g.nz - 4; ++D) {
            const int E = g.nz - D;
            int q = pieces, dp = (E + q - 1) / q;
            if (dp < 4) break;
            // as many pieces as there are non-empty ones of that depth (the kernel derives the depth from the count)
            for (int q2 = (E + dp - 1) / dp; q2 != q; q2 = (E + dp - 1) / dp) { q = q2; dp = (E + q - 1) / q; }
            const long long span = std::max<long long>(D + 2, (E + 2) + (dp + 2));
            if (best < 0 || span < best) { best = span; bestD = D; bestq = q; }
        }
        if (best < 0 || (mode_forced != 2 && best * 100 > span0 * 97)) return P;
        P.mode = 2; P.zchunk = bestD; P.nitems = T; P.zrest = bestD; P.erest = g.nz - bestD; P.q = bestq; P.blocks = sm_count;
        P.m2_rest = R; P.m2_left = L; P.m2_depth = (P.erest + bestq - 1) / bestq;
        return P;
    }
    if (mode_forced == 2) return P;
    // two-group plans: `full` layers of depth D in step, the rest flattened over the R remaining blocks
    long long best = -1; int bestD = 0, bestq = 0;
    for (int D = 4; D * full <= g.nz; ++D) {
        const int E = g.nz - D * full;
        long long span = D + 2;
        int q = 0;
        if (E > 0) {
            if (R == 0) continue;
            q = (int)(((long long)T * E + R - 1) / R);
            for (int r = 0; r < R; ++r) {
                long long pos = (long long)r * q, end = std::min(pos + q, (long long)T * E), w = 0;
                while (pos < end) {
                    const long long zz = pos % E, len = std::min((long long)E - zz, end - pos);
                    w += len + 2; pos += len;
                }
                span = std::max(span, w);
            }
        }
        if (best < 0 || span < best) { best = span; bestD = D; bestq = q; }
    }
    if (best < 0 || (mode_forced != 1 && best * 100 > span0 * 97)) return P;
    P.mode = 1; P.zchunk = bestD; P.nitems = T * full; P.zrest = bestD * full; P.erest = g.nz - P.zrest; P.q = bestq;
    P.blocks = P.erest > 0 ? sm_count : P.nitems;
    if (P.erest == 0) P.erest = 1;       // (never dereferenced: no rest block exists; keeps the divisions defined)
    return P;
}

template <int MODE, bool PRECOND, bool STORED, bool CODE32, int TYV>
void launch_geo(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaArgs& tm) {
    // The stored variant (six more arrays per node straight from global memory, no registers to spare for the
    // segment loop) keeps one item per block.  The plan of a grid is computed once per geometry and process.
    // Plans of mode 2 exist for the 13-row tiles (their kernels are instances of their own).
    constexpr bool M2_OK = !STORED && TYV == TY_DEEP;
    static thread_local struct { GridDims g; int sm, forced; SegPlan P; bool valid; } cache = {};
    if (!cache.valid || cache.g.nx != c.g.nx || cache.g.ny != c.g.ny || cache.g.nz != c.g.nz || cache.sm != c.sm_count ||
        cache.forced != c.seg_mode) {
        cache.P = plan_segments(c.g, TYV, c.sm_count, !STORED, c.seg_mode);
        cache.g = c.g; cache.sm = c.sm_count; cache.forced = c.seg_mode; cache.valid = true;
    }
    const SegPlan& plan = cache.P;
    const int blocks = plan.blocks;
    const Scalars* sc_in; Scalars* sc_out;
    c.next_scalars(sc_in, sc_out);
    using L = Layout<MODE, STORED, CODE32, TYV>;
    static std::atomic<unsigned long long> configured{0ull};      // bit d: the attribute is set on device d
    auto kern = k_tma<MODE, PRECOND, STORED, CODE32, TYV, false>;
    if constexpr (M2_OK) { if (plan.mode == 2) kern = k_tma<MODE, PRECOND, STORED, CODE32, TYV, true>; }
    const unsigned long long bit = 1ull << (c.device & 63);
    if (c.device >= 64 || !(configured.load(std::memory_order_relaxed) & bit)) {
        note_launch(cudaFuncSetAttribute(k_tma<MODE, PRECOND, STORED, CODE32, TYV, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL));
        if constexpr (M2_OK)
            note_launch(cudaFuncSetAttribute(k_tma<MODE, PRECOND, STORED, CODE32, TYV, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, L::TOTAL));
        configured.fetch_or(bit, std::memory_order_relaxed);
    }
    ++g_launch_count;
    note_launch(launch_pdl(c.pdl, kern, dim3(blocks), dim3(Geo<TYV>::NT), (size_t)L::TOTAL, c.stream, tm, c.g, op, kv, sc_in, sc_out,
                           c.rb, plan));
}

// ty: tile rows (TY_WIDE or TY_DEEP); the stored variant is compiled for the wide tiles only
template <int MODE, bool PRECOND, bool STORED, bool CODE32>
void launch_inst(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaArgs& tm, int ty) {
    if (!STORED && ty == TY_DEEP) launch_geo<MODE, PRECOND, STORED, CODE32, STORED ? TY_WIDE : TY_DEEP>(c, op, kv, tm);
    else launch_geo<MODE, PRECOND, STORED, CODE32, TY_WIDE>(c, op, kv, tm);
}

template <int MODE>
void launch_mode(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaArgs& tm, bool precond, int ty) {
    const bool c32 = op.code32 != 0;
    constexpr bool MERGED = MODE == MODE_K2M || MODE == MODE_K31 || MODE == MODE_K31D || MODE == MODE_K2MD;    // code form only
    if constexpr (!MERGED) {
        if (op.stored) {
            if (precond) launch_inst<MODE, true, true, false>(c, op, kv, tm, ty);
            else         launch_inst<MODE, false, true, false>(c, op, kv, tm, ty);
            return;
        }
    }
    if (c32) {
        if (precond) launch_inst<MODE, true, false, true>(c, op, kv, tm, ty);
        else         launch_inst<MODE, false, false, true>(c, op, kv, tm, ty);
    } else {
        if (precond) launch_inst<MODE, true, false, false>(c, op, kv, tm, ty);
        else         launch_inst<MODE, false, false, false>(c, op, kv, tm, ty);
    }
}

// Tile rows of a launch.  Measured on one B200 (profiles/r2_tiles.md, r2_plans.md): the deep tiles (16 warps, 128
// registers, no spills) win for both kernels of the merged solver at every size (K31 -8 to -16 %, K2M -2 to -11 %); for k1
// since it has a fourth stage there (k1 with the diagonal from the codes 0.149 -> 0.142 ms at 256^3, 1.22 -> 1.07 at
// 512^3; with the diagonal read, where the wide kernel spills, 0.182 -> 0.157 at 256^3, 1.62 -> 1.27 at 512^3); and for
// k2 at every size once the decomposition of mode 2 exists (256^3: 0.112 wide with the plan of mode 1, 0.109 deep;
// 192^3: 0.053 / 0.051; 512^3: equal).  So operators in code form run on the deep tiles; the wide ones serve the
// stored variant (only geometry compiled for it).  c.tile_rows != 0 forces one geometry (PF_OPT_TILE_ROWS).
int tile_rows(const LaunchCtx& c, const Operator& op, int mode) {
    (void)mode;
    if (op.stored) return TY_WIDE;
    if (c.tile_rows == TY_WIDE || c.tile_rows == TY_DEEP) return c.tile_rows;
    return TY_DEEP;
}

}  // namespace

// Tensor maps of one solve: every vector a kernel reads through TMA, once per tile geometry (the boxes differ).
struct TmaMaps {
    CUtensorMap r, p[2], v[2], a0, rt, x, b, code;
    CUtensorMap codeh;       // 2-byte codes with the halo ring (MODE_K1D, MODE_K31D)
    CUtensorMap r1, th;      // merged solver: the second r buffer, and t with its halo ring
};
struct TmaSet {
    TmaMaps m[2];            // [0]: TY_WIDE, [1]: TY_DEEP
    bool have_code, have_codeh, have_merged;
    bool k2_diag;            // k2 / K2M take the diagonal from the codes too (op.diag_code >= 2)
    const TmaMaps& of(int ty) const { return m[ty == TY_DEEP ? 1 : 0]; }
};

bool tma_available() { return encoder() != nullptr; }

// Even nx (16-byte row strides) and a grid that fills at least a few tiles.
bool tma_supported(const GridDims& g) {
    return (g.nx % 2 == 0) && g.nx >= 32 && g.ny >= 16 && g.nz >= 8;
}

bool tma_merged_ok(const TmaSet* t) { return t->have_merged; }

bool tma_pointers_ok(const KrylovVecs& kv, const Operator& op) {
    return aligned16(kv.x) && aligned16(kv.b) && aligned16(op.A0) && aligned16(kv.r) && aligned16(kv.rt) &&
           aligned16(kv.p_in) && aligned16(kv.p_out) && aligned16(kv.v_in) && aligned16(kv.v_out) && aligned16(kv.t);
}

TmaSet* tma_set_create() { return new TmaSet(); }
void tma_set_destroy(TmaSet* t) { delete t; }

bool tma_set_build(TmaSet* t, const GridDims& g, const Operator& op, const KrylovVecs& kv) {
    bool ok = true;
    t->have_code = !op.stored;
    t->have_codeh = !op.stored && !op.code32 && op.diag_code;
    t->k2_diag = op.diag_code >= 2;
    t->have_merged = kv.r_out && !op.stored && aligned16(kv.r_out);
    for (int k = 0; k < (op.stored ? 1 : 2) && ok; ++k) {
        TmaMaps& M = t->m[k];
        const int ty = k ? TY_DEEP : TY_WIDE;
        ok = halo_map(&M.r, kv.r, g, ty) && halo_map(&M.p[0], kv.p_in, g, ty) && halo_map(&M.p[1], kv.p_out, g, ty) &&
             halo_map(&M.v[0], kv.v_in, g, ty) && halo_map(&M.v[1], kv.v_out, g, ty) && halo_map(&M.a0, op.A0, g, ty) &&
             own_map(&M.rt, kv.rt, g, ty) && halo_map(&M.x, kv.x, g, ty) && own_map(&M.b, kv.b, g, ty);
        if (ok && t->have_code)
            ok = op.code32 ? make_map(&M.code, op.code, CU_TENSOR_MAP_DATA_TYPE_UINT32, 4, g, op.cpitch, TX, ty)
                           : make_map(&M.code, op.code, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, g, op.cpitch, TX, ty);
        if (ok && t->have_codeh)
            t->have_codeh = make_map(&M.codeh, op.code, CU_TENSOR_MAP_DATA_TYPE_UINT16, 2, g, op.cpitch, BXC, ty + 2);
        if (ok && t->have_merged) t->have_merged = halo_map(&M.r1, kv.r_out, g, ty) && halo_map(&M.th, kv.t, g, ty);
    }
    if (!ok) t->have_code = t->have_codeh = t->have_merged = false;
    return ok;
}

bool tma_merged_supported(const Operator& op) { return !op.stored; }

void tma_plan(const GridDims& g, int tile_rows, int sm_count, int mode, int* out) {
    const SegPlan P = plan_segments(g, tile_rows == TY_DEEP ? TY_DEEP : TY_WIDE, sm_count, true, mode);
    out[0] = P.mode; out[1] = P.ntx; out[2] = P.ntiles; out[3] = P.zchunk; out[4] = P.nitems; out[5] = P.zrest;
    out[6] = P.erest; out[7] = P.q; out[8] = P.blocks;
}

// precond: mode 0 of a preconditioned solve also tests the diagonal against the range of the branch-free division
// that k1 and k2 will divide by it with (reading D4; the residual itself involves no division).
void launch_residual_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, int mode,
                         bool precond) {
    const int ty = tile_rows(c, op, mode == 0 ? MODE_R0 : MODE_R1);
    const TmaMaps& M = t->of(ty);
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    a.f[0] = M.x; a.f[1] = M.a0; a.own = M.b; a.code = M.code;
    if (mode == 0) launch_mode<MODE_R0>(c, op, kv, a, precond, ty); else launch_mode<MODE_R1>(c, op, kv, a, false, ty);
}

void launch_k1_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond,
                   int parity) {
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    if (t->have_codeh) {     // the diagonal is the sum of the face coefficients: formed from the codes, A0 not read
        const int ty = tile_rows(c, op, MODE_K1D);
        const TmaMaps& M = t->of(ty);
        a.f[0] = M.r; a.f[1] = M.p[parity]; a.f[2] = M.v[parity]; a.own = M.rt; a.code = M.codeh;
        if (precond) launch_inst<MODE_K1D, true, false, false>(c, op, kv, a, ty);
        else         launch_inst<MODE_K1D, false, false, false>(c, op, kv, a, ty);
        return;
    }
    const int ty = tile_rows(c, op, MODE_K1);
    const TmaMaps& M = t->of(ty);
    a.f[0] = M.r; a.f[1] = M.p[parity]; a.f[2] = M.v[parity]; a.f[3] = M.a0; a.own = M.rt; a.code = M.code;
    launch_mode<MODE_K1>(c, op, kv, a, precond, ty);
}

void launch_k2m_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond, int k) {
    const bool diag = t->have_codeh && t->k2_diag;
    const int ty = tile_rows(c, op, diag ? MODE_K2MD : MODE_K2M);
    const TmaMaps& M = t->of(ty);
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    const int rb = k & 1, pb = rb ^ 1;
    a.f[0] = rb ? M.r1 : M.r; a.f[1] = M.v[pb]; a.own = M.rt;
    if (diag) {
        a.code = M.codeh;
        if (precond) launch_inst<MODE_K2MD, true, false, false>(c, op, kv, a, ty);
        else         launch_inst<MODE_K2MD, false, false, false>(c, op, kv, a, ty);
        return;
    }
    a.f[2] = M.a0; a.code = M.code;
    launch_mode<MODE_K2M>(c, op, kv, a, precond, ty);
}

void launch_k31_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond, int k) {
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    const int rb = k & 1, pb = rb ^ 1;
    const int ty = tile_rows(c, op, t->have_codeh ? MODE_K31D : MODE_K31);
    const TmaMaps& M = t->of(ty);
    a.f[0] = rb ? M.r1 : M.r; a.f[1] = M.p[pb]; a.f[2] = M.v[pb]; a.f[3] = M.th; a.own = M.rt;
    if (t->have_codeh) {     // the diagonal is the sum of the face coefficients: formed from the codes, A0 not read
        a.code = M.codeh;
        if (precond) launch_inst<MODE_K31D, true, false, false>(c, op, kv, a, ty);
        else         launch_inst<MODE_K31D, false, false, false>(c, op, kv, a, ty);
        return;
    }
    a.f[4] = M.a0; a.code = M.code;
    launch_mode<MODE_K31>(c, op, kv, a, precond, ty);
}

void launch_k2_tma(const LaunchCtx& c, const Operator& op, const KrylovVecs& kv, const TmaSet* t, bool precond,
                   int parity) {
    const bool diag = t->have_codeh && t->k2_diag;
    const int ty = tile_rows(c, op, diag ? MODE_K2D : MODE_K2);
    const TmaMaps& M = t->of(ty);
    TmaArgs a;
    std::memset(&a, 0, sizeof(a));
    a.f[0] = M.r; a.f[1] = M.v[parity ^ 1];                                   // v' = the buffer k1 just wrote
    if (diag) {              // diagonal and reciprocal from the code table: A0 is not read
        a.code = M.codeh;
        if (precond) launch_inst<MODE_K2D, true, false, false>(c, op, kv, a, ty);
        else         launch_inst<MODE_K2D, false, false, false>(c, op, kv, a, ty);
        return;
    }
    a.f[2] = M.a0; a.code = M.code;
    launch_mode<MODE_K2>(c, op, kv, a, precond, ty);
}

}  // namespace pf
