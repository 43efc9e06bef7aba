// pf_assembly.cu -- operator assembly on the device (rows L1, L2 of DESIGN.md).
//
// The paper builds A0..A6 and b on the GPU each outer iteration and finds that the weak part of its
// design (7.7x against 22.8x for the solver).  Here the flux part of every
// operator is assembled ONCE per grid: per node the diagonal and either the six stored off-diagonals
// (the paper's format) or a packed code of six table indices, one per face, into the
// short table of distinct face coefficients of the map (on-the-fly variant; pf_common.cuh Operator).
// PF2's sigma only shifts the diagonal.
#include "pf_launch.h"
#include <algorithm>
#include <cstring>

namespace pf {

namespace {

constexpr int ASM_THREADS = 256;
// Table index of the face between palette entries a and b (unordered pair), 1-based; 0 = no coupling.
__host__ __device__ inline int pair_index(int a, int b, int count) {
    const int lo = a < b ? a : b, hi = a < b ? b : a;
    return 1 + lo * count - lo * (lo - 1) / 2 + (hi - lo);
}

__device__ __forceinline__ void store_code(void* code, int code_mode, long long k, unsigned int c) {
    if (code_mode == 1) static_cast<unsigned short*>(code)[k] = (unsigned short)c;
    else if (code_mode == 2) static_cast<unsigned int*>(code)[k] = c;
}

struct ScanBuf {
    unsigned long long tab[PF_MAX_PALETTE + 1];  // bit patterns of the distinct values, 0 = empty
    unsigned long long min_bits, max_bits;
    int overflow;
};

// Distinct values (up to PF_MAX_PALETTE + 1, then overflow), minimum and maximum of eps.  A thread keeps the
// values it has met in registers and goes to the shared table only for a value that is new to it, so the scan
// runs at memory speed (one 8-byte load and a few compares per node).
__global__ void __launch_bounds__(ASM_THREADS) k_scan_eps(long long n, const double* __restrict__ eps, ScanBuf* sb) {
    unsigned long long lo = ~0ull, hi = 0ull;
    unsigned long long known[PF_MAX_PALETTE + 1];
    int nknown = 0;
    bool lost = false;                  // more distinct values than the table holds
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const unsigned long long bits = (unsigned long long)__double_as_longlong(eps[i]);
        lo = bits < lo ? bits : lo;
        hi = bits > hi ? bits : hi;
        bool seen = lost;
#pragma unroll
        for (int k = 0; k <= PF_MAX_PALETTE; ++k) seen = seen || (k < nknown && known[k] == bits);
        if (seen) continue;
        bool found = false;                 // new to this thread: look in the shared table, claim a free slot if absent
        int k = 0;
        for (; k <= PF_MAX_PALETTE; ++k) {
            const unsigned long long v = ((volatile unsigned long long*)sb->tab)[k];
            if (v == bits) { found = true; break; }
            if (v == 0ull) break;
        }
        for (; !found && k <= PF_MAX_PALETTE; ++k) {
            const unsigned long long old = atomicCAS(&sb->tab[k], 0ull, bits);
            if (old == 0ull || old == bits) found = true;
        }
        if (!found) { sb->overflow = 1; lost = true; continue; }
#pragma unroll
        for (int k = 0; k <= PF_MAX_PALETTE; ++k)
            if (k == nknown) known[k] = bits;
        ++nknown;
    }
    for (int d = 16; d > 0; d >>= 1) {
        unsigned long long a = __shfl_xor_sync(0xffffffffu, lo, d), b = __shfl_xor_sync(0xffffffffu, hi, d);
        lo = a < lo ? a : lo;
        hi = b > hi ? b : hi;
    }
    if ((threadIdx.x & 31) == 0) { atomicMin(&sb->min_bits, lo); atomicMax(&sb->max_bits, hi); }
}

// First Dirichlet face the node lies on (order -x,+x,-y,+y,-z,+z), else -1 (reading Q20).
__device__ __forceinline__ int dirichlet_face(const GridDims& g, const BcDev& bc, int ix, int iy, int iz) {
    if (ix == 0 && bc.type[0] == 0) return 0;
    if (ix == g.nx - 1 && bc.type[1] == 0) return 1;
    if (iy == 0 && bc.type[2] == 0) return 2;
    if (iy == g.ny - 1 && bc.type[3] == 0) return 3;
    if (iz == 0 && bc.type[4] == 0) return 4;
    if (iz == g.nz - 1 && bc.type[5] == 0) return 5;
    return -1;
}

__device__ __forceinline__ void decode(const GridDims& g, long long i, int& ix, int& iy, int& iz) {
    ix = (int)(i % g.nx);
    const long long q = i / g.nx;
    iy = (int)(q % g.ny);
    iz = (int)(q / g.ny);
}

__device__ __forceinline__ int palette_index(const Palette& pal, double e) {
    int k = 0;
#pragma unroll
    for (int m = 1; m < PF_MAX_PALETTE; ++m)
        if (m < pal.count && e == pal.value[m]) k = m;
    return k;
}

// Face coefficient: harmonic mean of eps over h^2 -- Eqs (17)-(18) with the interface at the face
// midpoint (reading R2/Q16).
__device__ __forceinline__ double face_coeff(double ea, double eb, double hh) {
    return dvd(dvd(mul(mul(2.0, ea), eb), add(ea, eb)), hh);
}

// code_mode: 0 = no codes (palette overflow), 1 = uint16 / 2-bit fields, 2 = uint32 / 4-bit fields.
__global__ void __launch_bounds__(ASM_THREADS)
k_assemble_poisson(GridDims g, double h, BcDev bc, const double* __restrict__ eps, Palette pal, int code_mode,
                   double* __restrict__ A0, void* __restrict__ code, int cpitch, double* o0, double* o1, double* o2,
                   double* o3, double* o4, double* o5) {
    double* offd[6] = {o0, o1, o2, o3, o4, o5};
    const double hh = mul(h, h);
    const long long off[6] = {1, -1, -(long long)g.nx, (long long)g.nx, -(long long)g.nx * g.ny,
                              (long long)g.nx * g.ny};
    const int fbits = code_mode == 2 ? 4 : 2;
    // With a palette the map has at most ten distinct face coefficients: each block forms them once (the same
    // expression, so the same bits, as a node would) instead of two divisions per face and node.
    __shared__ double pair_coeff[PF_CTAB];
    if (code_mode && (int)threadIdx.x < pal.count * pal.count) {
        const int a = threadIdx.x / pal.count, b = threadIdx.x % pal.count;
        if (a <= b) pair_coeff[pair_index(a, b, pal.count)] = face_coeff(pal.value[a], pal.value[b], hh);
    }
    __syncthreads();
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        int ix, iy, iz;
        decode(g, i, ix, iy, iz);
        const long long k = ix + (long long)cpitch * (iy + (long long)g.ny * iz);
        const double ei = eps[i];
        const bool ident = dirichlet_face(g, bc, ix, iy, iz) >= 0 || is_fixed_node(bc, i);   // Q20, F2
        if (ident) {
            A0[i] = 1.0;
            store_code(code, code_mode, k, 0u);
#pragma unroll
            for (int d = 0; d < 6; ++d) if (offd[d]) offd[d][i] = 0.0;
            continue;
        }
        const bool in[6] = {ix + 1 < g.nx, ix > 0, iy > 0, iy + 1 < g.ny, iz > 0, iz + 1 < g.nz};
        const int pi = code_mode ? palette_index(pal, ei) : 0;
        double diag = 0.0;
        unsigned int cw = 0u;
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            double c = 0.0;
            if (in[d]) {
                const double en = eps[i + off[d]];
                if (code_mode) {
                    const int pj = pair_index(pi, palette_index(pal, en), pal.count);
                    c = pair_coeff[pj];
                    cw |= (unsigned int)pj << (fbits * d);
                } else {
                    c = face_coeff(ei, en, hh);
                }
                diag = add(diag, c);
            }
            if (offd[d]) offd[d][i] = in[d] ? -c : 0.0;
        }
        A0[i] = diag;
        store_code(code, code_mode, k, cw);
    }
}

__global__ void __launch_bounds__(ASM_THREADS)
k_assemble_pf1(GridDims g, double h, double lc, BcDev bc, const double* __restrict__ eps, double eps_mid, bool uniform,
               Palette pal, int code_mode, double* __restrict__ A0, void* __restrict__ code, int cpitch, double* o0,
               double* o1, double* o2, double* o3, double* o4, double* o5) {
    double* offd[6] = {o0, o1, o2, o3, o4, o5};
    const double hh = mul(h, h), ll = mul(lc, lc);
    const int fbits = code_mode == 2 ? 4 : 2;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        int ix, iy, iz;
        decode(g, i, ix, iy, iz);
        const long long k = ix + (long long)cpitch * (iy + (long long)g.ny * iz);
        const double ei = eps[i];
        const bool boundary = ix == 0 || ix == g.nx - 1 || iy == 0 || iy == g.ny - 1 || iz == 0 || iz == g.nz - 1;
        const bool solvent = uniform || ei > eps_mid;           // Q17
        const bool ident = boundary || !solvent || is_fixed_node(bc, i);   // Q15, F2
        if (ident) {
            A0[i] = 1.0;
            store_code(code, code_mode, k, 0u);
#pragma unroll
            for (int d = 0; d < 6; ++d) if (offd[d]) offd[d][i] = 0.0;
            continue;
        }
        const double c = dvd(mul(ei, ll), hh);
        A0[i] = add(mul(6.0, c), ei);
        if (code_mode) {           // all six faces carry the node's own coefficient: table index 1 + palette index
            const unsigned int f = 1u + (unsigned int)palette_index(pal, ei);
            unsigned int cw = 0u;
#pragma unroll
            for (int d = 0; d < 6; ++d) cw |= f << (fbits * d);
            store_code(code, code_mode, k, cw);
        }
#pragma unroll
        for (int d = 0; d < 6; ++d) if (offd[d]) offd[d][i] = -c;
    }
}

// Deposits of different charges can hit the same node and floating-point addition is not associative,
// so they must be applied in charge order (reading R2).  One block walks the list in chunks of DEP_CHUNK
// charges, one charge per thread, in rounds: a charge is applied once every earlier charge of the chunk
// whose cell is adjacent to its own (the only ones that can share a node with it) has been applied.
// Charges applied in the same round touch disjoint nodes.  The result is identical to the serial loop.
constexpr int DEP_CHUNK = 256;

__device__ __forceinline__ void deposit_one(const GridDims& g, double h, double h3, double kappa,
                                            const double* __restrict__ ch, int c, double* fixed) {
    const double px = dvd(ch[4 * c], h), py = dvd(ch[4 * c + 1], h), pz = dvd(ch[4 * c + 2], h);
    const double q = ch[4 * c + 3];
    const int ix = min(max((int)floor(px), 0), g.nx - 2);
    const int iy = min(max((int)floor(py), 0), g.ny - 2);
    const int iz = min(max((int)floor(pz), 0), g.nz - 2);
    const double fx = sub(px, (double)ix), fy = sub(py, (double)iy), fz = sub(pz, (double)iz);
    const double amp = dvd(mul(kappa, q), h3);
    for (int dz = 0; dz < 2; ++dz)
        for (int dy = 0; dy < 2; ++dy)
            for (int dx = 0; dx < 2; ++dx) {
                const double wx = dx ? fx : sub(1.0, fx), wy = dy ? fy : sub(1.0, fy), wz = dz ? fz : sub(1.0, fz);
                const double w = mul(mul(wx, wy), wz);
                const long long i = (ix + dx) + (long long)g.nx * ((iy + dy) + (long long)g.ny * (iz + dz));
                fixed[i] = add(fixed[i], mul(amp, w));
            }
}

__global__ void __launch_bounds__(DEP_CHUNK)
k_deposit(GridDims g, double h, double kappa, const double* __restrict__ ch, int m, double* fixed) {
    __shared__ int cell[DEP_CHUNK][3];
    __shared__ unsigned char done[DEP_CHUNK];
    const double h3 = mul(mul(h, h), h);
    const int t = threadIdx.x;
    for (int base = 0; base < m; base += DEP_CHUNK) {
        const int c = base + t;
        bool pending = c < m;
        done[t] = 0;
        if (pending) {
            cell[t][0] = min(max((int)floor(dvd(ch[4 * c], h)), 0), g.nx - 2);
            cell[t][1] = min(max((int)floor(dvd(ch[4 * c + 1], h)), 0), g.ny - 2);
            cell[t][2] = min(max((int)floor(dvd(ch[4 * c + 2], h)), 0), g.nz - 2);
        }
        while (__syncthreads_or(pending)) {
            bool ready = pending;
            if (pending)
                for (int k = 0; k < t && ready; ++k)
                    if (!done[k] && abs(cell[k][0] - cell[t][0]) <= 1 && abs(cell[k][1] - cell[t][1]) <= 1 &&
                        abs(cell[k][2] - cell[t][2]) <= 1)
                        ready = false;
            __syncthreads();                  // every thread has read done[] of this round
            if (ready) {
                deposit_one(g, h, h3, kappa, ch, c, fixed);
                __threadfence_block();
                done[t] = 1;
                pending = false;
            }
        }
        __syncthreads();
    }
}

__global__ void __launch_bounds__(ASM_THREADS)
k_set_dirichlet(GridDims g, BcDev bc, const double* __restrict__ src, double* __restrict__ dst) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        int ix, iy, iz;
        decode(g, i, ix, iy, iz);
        const int f = dirichlet_face(g, bc, ix, iy, iz);
        if (f >= 0) dst[i] = bc.value[f];
        else if (is_fixed_node(bc, i)) dst[i] = bc.fixv[i];
        else if (src != dst) dst[i] = src[i];
    }
}

int asm_blocks(long long n) {
    long long b = (n + ASM_THREADS - 1) / ASM_THREADS;
    return (int)std::min<long long>(std::max<long long>(b, 1), 148 * 16);
}

double host_face_coeff(double ea, double eb, double h) { return (2.0 * ea * eb / (ea + eb)) / (h * h); }

}  // namespace

cudaError_t scan_eps(cudaStream_t s, long long n, const double* eps, void* scratch, Palette* out, double* eps_min,
                     double* eps_max) {
    ScanBuf init;
    std::memset(&init, 0, sizeof(init));
    init.min_bits = ~0ull;
    cudaError_t e = cudaMemcpyAsync(scratch, &init, sizeof(init), cudaMemcpyHostToDevice, s);
    if (e != cudaSuccess) return e;
    ++g_launch_count;
    k_scan_eps<<<asm_blocks(n), ASM_THREADS, 0, s>>>(n, eps, (ScanBuf*)scratch);
    ScanBuf res;
    e = cudaMemcpyAsync(&res, scratch, sizeof(res), cudaMemcpyDeviceToHost, s);
    if (e != cudaSuccess) return e;
    e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) return e;
    int cnt = 0;
    double vals[PF_MAX_PALETTE + 1];
    for (int k = 0; k <= PF_MAX_PALETTE; ++k)
        if (res.tab[k] != 0ull) { std::memcpy(&vals[cnt], &res.tab[k], 8); ++cnt; }
    std::sort(vals, vals + cnt);
    out->count = res.overflow ? PF_MAX_PALETTE + 1 : cnt;
    for (int k = 0; k <= PF_MAX_PALETTE; ++k) out->value[k] = k < cnt ? vals[k] : 0.0;
    std::memcpy(eps_min, &res.min_bits, 8);
    std::memcpy(eps_max, &res.max_bits, 8);
    return cudaSuccess;
}

void launch_assemble_poisson(cudaStream_t s, const GridDims& g, double h, const BcDev& bc, const double* eps,
                             const Palette& pal, int code_mode, double* A0, void* code, int cpitch,
                             double* const offd[6]) {
    ++g_launch_count;
    k_assemble_poisson<<<asm_blocks(g.n), ASM_THREADS, 0, s>>>(g, h, bc, eps, pal, code_mode, A0, code, cpitch, offd[0],
                                                                offd[1], offd[2], offd[3], offd[4], offd[5]);
}

__global__ void k_scatter_fixed(const long long* __restrict__ idx, const double* __restrict__ val, int count,
                                double* __restrict__ fixv) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k < count) fixv[idx[k]] = val[k];
}

void launch_scatter_fixed(cudaStream_t s, const long long* idx_dev, const double* val_dev, int count, double* fixv) {
    if (count <= 0) return;
    ++g_launch_count;
    k_scatter_fixed<<<(count + 255) / 256, 256, 0, s>>>(idx_dev, val_dev, count, fixv);
}

void launch_assemble_pf1(cudaStream_t s, const GridDims& g, double h, double lc, const BcDev& bc, const double* eps,
                         double eps_mid, bool uniform, const Palette& pal, int code_mode, double* A0, void* code,
                         int cpitch, double* const offd[6]) {
    ++g_launch_count;
    k_assemble_pf1<<<asm_blocks(g.n), ASM_THREADS, 0, s>>>(g, h, lc, bc, eps, eps_mid, uniform, pal, code_mode, A0, code,
                                                            cpitch, offd[0], offd[1], offd[2], offd[3], offd[4], offd[5]);
}

// Coefficient tables of the on-the-fly variant (host side, PF_CTAB doubles): entry 0 is 0.0, entry
// pair_index(a, b) the off-diagonal -H(eps_a, eps_b)/h^2 (Poisson) resp. entry 1 + a the off-diagonal
// -eps_a l_c^2/h^2 (PF1), computed with the same operations in the same order as the kernels above.
void build_ctab_poisson(const Palette& pal, double h, double* ctab) {
    for (int k = 0; k < PF_CTAB; ++k) ctab[k] = 0.0;
    for (int a = 0; a < pal.count && a < PF_MAX_PALETTE; ++a)
        for (int b = a; b < pal.count && b < PF_MAX_PALETTE; ++b)
            ctab[pair_index(a, b, pal.count)] = -host_face_coeff(pal.value[a], pal.value[b], h);
}

void build_ctab_pf1(const Palette& pal, double h, double lc, double* ctab) {
    for (int k = 0; k < PF_CTAB; ++k) ctab[k] = 0.0;
    for (int a = 0; a < pal.count && a < PF_MAX_PALETTE; ++a) ctab[1 + a] = -(pal.value[a] * (lc * lc) / (h * h));
}

void launch_deposit(cudaStream_t s, const GridDims& g, double h, double kappa, const double* charges_dev, int m,
                    double* fixed) {
    cudaMemsetAsync(fixed, 0, sizeof(double) * g.n, s);
    if (m > 0) { ++g_launch_count; k_deposit<<<1, DEP_CHUNK, 0, s>>>(g, h, kappa, charges_dev, m, fixed); }
}

void launch_set_dirichlet(cudaStream_t s, const GridDims& g, const BcDev& bc, double* x) {
    ++g_launch_count;
    k_set_dirichlet<<<asm_blocks(g.n), ASM_THREADS, 0, s>>>(g, bc, x, x);
}

void launch_copy_with_dirichlet(cudaStream_t s, const GridDims& g, const BcDev& bc, const double* src, double* dst) {
    ++g_launch_count;
    k_set_dirichlet<<<asm_blocks(g.n), ASM_THREADS, 0, s>>>(g, bc, src, dst);
}

}  // namespace pf
