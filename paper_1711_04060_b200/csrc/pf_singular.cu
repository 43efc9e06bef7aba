// pf_singular.cu -- singular-charge decomposition, Eqs (5)-(10) and the flux-jump terms c0, d0 of
// Eqs (17)-(18) (readings S1-S5 of DESIGN.md), the step in front of the PF loop
// (Table 2 step 1, Table 4 steps 2-3).  The paper computes the interface vector
// b^IF on the CPU; here everything stays on the device:
//   k_laplace_m   : rows, right-hand side and prescribed values of the Laplace problem for phi^L in Omega_m
//                   (interface at the face midpoints, ghost-value Dirichlet data -phi*), Coulomb sums on the fly;
//   (the Laplace solve itself is the Jacobi-BiCGSTAB core with this operator)
//   k_phistar     : phi* on the Omega_m nodes;
//   k_interface   : b^IF gathered per node from the flux jumps of its interface faces.
// One thread per node; only the nodes next to the interface (and the Omega_m nodes on the box boundary) do
// Coulomb sums, M terms each, in charge order, every operation rounded once as written (the oracle does the
// same in the same order, so the vectors agree bit for bit).
#include "pf_launch.h"
#include <algorithm>

namespace pf {

namespace {

constexpr int SG_THREADS = 128;

__device__ __forceinline__ void decode3(const GridDims& g, long long i, int& ix, int& iy, int& iz) {
    ix = (int)(i % g.nx);
    const long long q = i / g.nx;
    iy = (int)(q % g.ny);
    iz = (int)(q / g.ny);
}

// faces d = 1..6 in the order of PAPER.md:219: east, west, south, north, down, up
__device__ __constant__ int c_fdx[7] = {0, 1, -1, 0, 0, 0, 0};
__device__ __constant__ int c_fdy[7] = {0, 0, 0, -1, 1, 0, 0};
__device__ __constant__ int c_fdz[7] = {0, 0, 0, 0, 0, -1, 1};
__device__ __constant__ int c_faxis[7] = {0, 0, 0, 1, 1, 2, 2};
__device__ __constant__ int c_fsign[7] = {0, 1, -1, -1, 1, -1, 1};
__device__ __constant__ int c_fopp[7] = {0, 2, 1, 4, 3, 6, 5};

struct Coulomb {
    const double* ch;      // M x 4: x, y, z, q
    int m;
    double pref;           // kappa / (4 pi eps_m)
};

// phi*(x, y, z) = pref * sum_j q_j / |r - r_j|   (Eq 5)
__device__ __forceinline__ double coulomb_potential(const Coulomb& c, double x, double y, double z) {
    double s = 0.0;
    for (int j = 0; j < c.m; ++j) {
        const double dx = sub(x, c.ch[4 * j]), dy = sub(y, c.ch[4 * j + 1]), dz = sub(z, c.ch[4 * j + 2]);
        const double r = __dsqrt_rn(add(add(mul(dx, dx), mul(dy, dy)), mul(dz, dz)));
        s = add(s, dvd(c.ch[4 * j + 3], r));
    }
    return mul(c.pref, s);
}

// d phi*/d x_axis = -pref * sum_j q_j (x_axis - r_j,axis) / |r - r_j|^3
__device__ __forceinline__ double coulomb_gradient(const Coulomb& c, double x, double y, double z, int axis) {
    double s = 0.0;
    for (int j = 0; j < c.m; ++j) {
        const double dx = sub(x, c.ch[4 * j]), dy = sub(y, c.ch[4 * j + 1]), dz = sub(z, c.ch[4 * j + 2]);
        const double r2 = add(add(mul(dx, dx), mul(dy, dy)), mul(dz, dz));
        const double r = __dsqrt_rn(r2);
        const double comp = axis == 0 ? dx : (axis == 1 ? dy : dz);
        s = add(s, dvd(mul(c.ch[4 * j + 3], comp), mul(r2, r)));
    }
    return -mul(c.pref, s);
}

__device__ __forceinline__ bool is_solvent(const double* eps, double eps_mid, long long i) { return eps[i] > eps_mid; }

// midpoint of face d of node (ix, iy, iz)
__device__ __forceinline__ void face_point(int ix, int iy, int iz, int d, double h, double& x, double& y, double& z) {
    x = mul(add((double)ix, mul(0.5, (double)c_fdx[d])), h);
    y = mul(add((double)iy, mul(0.5, (double)c_fdy[d])), h);
    z = mul(add((double)iz, mul(0.5, (double)c_fdz[d])), h);
}

// Laplace system for phi^L (readings S2, S3): diagonal, 2-bit stencil codes (table {0, -1/h^2}), right-hand
// side, and the start vector = prescribed values on identity rows, 0 elsewhere.
__global__ void __launch_bounds__(SG_THREADS)
k_laplace_m(GridDims g, double h, const double* __restrict__ eps, double eps_mid, Coulomb cl,
            double* __restrict__ A0, unsigned short* __restrict__ code, int cpitch, double* __restrict__ b,
            double* __restrict__ x0) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    int ix, iy, iz;
    decode3(g, i, ix, iy, iz);
    const long long k = ix + (long long)cpitch * (iy + (long long)g.ny * iz);
    if (is_solvent(eps, eps_mid, i)) { A0[i] = 1.0; code[k] = 0; b[i] = 0.0; x0[i] = 0.0; return; }
    if (ix == 0 || ix == g.nx - 1 || iy == 0 || iy == g.ny - 1 || iz == 0 || iz == g.nz - 1) {
        const double v = -coulomb_potential(cl, mul((double)ix, h), mul((double)iy, h), mul((double)iz, h));
        A0[i] = 1.0; code[k] = 0; b[i] = v; x0[i] = v;
        return;
    }
    const long long off[7] = {0, 1, -1, -(long long)g.nx, (long long)g.nx, -(long long)g.nx * g.ny,
                              (long long)g.nx * g.ny};
    const double c = dvd(1.0, mul(h, h));
    const double c2 = mul(2.0, c);
    double diag = 0.0, rhs = 0.0;
    unsigned cw = 0u;
    for (int d = 1; d < 7; ++d) {
        if (!is_solvent(eps, eps_mid, i + off[d])) { cw |= 1u << (2 * (d - 1)); diag = add(diag, c); continue; }
        double xf, yf, zf;
        face_point(ix, iy, iz, d, h, xf, yf, zf);
        const double gf = -coulomb_potential(cl, xf, yf, zf);
        diag = add(diag, c2);
        rhs = add(rhs, mul(c2, gf));
    }
    A0[i] = diag; code[k] = (unsigned short)cw; b[i] = rhs; x0[i] = 0.0;
}

__global__ void __launch_bounds__(SG_THREADS)
k_phistar(GridDims g, double h, const double* __restrict__ eps, double eps_mid, Coulomb cl, double* __restrict__ out) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    int ix, iy, iz;
    decode3(g, i, ix, iy, iz);
    out[i] = is_solvent(eps, eps_mid, i) ? 0.0
                                         : coulomb_potential(cl, mul((double)ix, h), mul((double)iy, h), mul((double)iz, h));
}

// Flux jump of the interface face d of the Omega_m node (ix, iy, iz) = im, n pointing into the solvent:
//   J = eps_m-node [ dphi*/dn (x_f) + 2 (g_f - phi^L_m)/h ],  g_f = -phi*(x_f)      (Eq 8, reading S2)
__device__ __forceinline__ double face_jump(const Coulomb& cl, double h, double eps_node, double phiL_node, int ix, int iy,
                                            int iz, int d) {
    double xf, yf, zf;
    face_point(ix, iy, iz, d, h, xf, yf, zf);
    const double gf = -coulomb_potential(cl, xf, yf, zf);
    const double dn_star = mul((double)c_fsign[d], coulomb_gradient(cl, xf, yf, zf, c_faxis[d]));
    const double dn_L = dvd(mul(2.0, sub(gf, phiL_node)), h);
    return mul(eps_node, add(dn_star, dn_L));
}

// b^IF: every node gathers the faces it shares with a node of the other kind, d = 1..6 (c0, d0 of Eqs 17-18):
//   b_i += -eps_i J_f / ((eps_i + eps_j) h)
__global__ void __launch_bounds__(SG_THREADS)
k_interface(GridDims g, double h, const double* __restrict__ eps, double eps_mid, Coulomb cl,
            const double* __restrict__ phiL, double* __restrict__ b) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= g.n) return;
    int ix, iy, iz;
    decode3(g, i, ix, iy, iz);
    const long long off[7] = {0, 1, -1, -(long long)g.nx, (long long)g.nx, -(long long)g.nx * g.ny,
                              (long long)g.nx * g.ny};
    const bool in[7] = {true, ix + 1 < g.nx, ix > 0, iy > 0, iy + 1 < g.ny, iz > 0, iz + 1 < g.nz};
    const bool si = is_solvent(eps, eps_mid, i);
    const double ei = eps[i];
    double acc = 0.0;
    for (int d = 1; d < 7; ++d) {
        if (!in[d]) continue;
        const long long j = i + off[d];
        if (is_solvent(eps, eps_mid, j) == si) continue;
        const double ej = eps[j];
        // the jump belongs to the Omega_m node of the pair and is evaluated from its indices
        const double Jf = si ? face_jump(cl, h, ej, phiL[j], ix + c_fdx[d], iy + c_fdy[d], iz + c_fdz[d], c_fopp[d])
                             : face_jump(cl, h, ei, phiL[i], ix, iy, iz, d);
        acc = add(acc, dvd(-mul(ei, Jf), mul(add(ei, ej), h)));
    }
    b[i] = acc;
}

// phi := phi + phi* + phi^L  (Eq 5; both are 0 on Omega_s)
__global__ void __launch_bounds__(256)
k_recombine(long long n, const double* __restrict__ phistar, const double* __restrict__ phiL, double* __restrict__ phi) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
        phi[i] = add(add(phi[i], phistar[i]), phiL[i]);
}

int sg_blocks(long long n) { return (int)((n + SG_THREADS - 1) / SG_THREADS); }

Coulomb make_coulomb(const double* charges_dev, int m, double kappa, double eps_m) {
    Coulomb c;
    c.ch = charges_dev; c.m = m;
    c.pref = kappa / ((4.0 * M_PI) * eps_m);
    return c;
}

}  // namespace

void launch_laplace_m(cudaStream_t s, const GridDims& g, double h, const double* eps, double eps_mid, double eps_m,
                      double kappa, const double* charges_dev, int m, double* A0, void* code, int cpitch, double* b,
                      double* x0) {
    ++g_launch_count;
    k_laplace_m<<<sg_blocks(g.n), SG_THREADS, 0, s>>>(g, h, eps, eps_mid, make_coulomb(charges_dev, m, kappa, eps_m), A0,
                                                       static_cast<unsigned short*>(code), cpitch, b, x0);
}

void launch_phistar(cudaStream_t s, const GridDims& g, double h, const double* eps, double eps_mid, double eps_m,
                    double kappa, const double* charges_dev, int m, double* out) {
    ++g_launch_count;
    k_phistar<<<sg_blocks(g.n), SG_THREADS, 0, s>>>(g, h, eps, eps_mid, make_coulomb(charges_dev, m, kappa, eps_m), out);
}

void launch_interface_rhs(cudaStream_t s, const GridDims& g, double h, const double* eps, double eps_mid, double eps_m,
                          double kappa, const double* charges_dev, int m, const double* phiL, double* b) {
    ++g_launch_count;
    k_interface<<<sg_blocks(g.n), SG_THREADS, 0, s>>>(g, h, eps, eps_mid, make_coulomb(charges_dev, m, kappa, eps_m), phiL, b);
}

void launch_recombine(cudaStream_t s, long long n, const double* phistar, const double* phiL, double* phi) {
    ++g_launch_count;
    const int nb = (int)std::min<long long>((n + 255) / 256, 148 * 16);
    k_recombine<<<nb, 256, 0, s>>>(n, phistar, phiL, phi);
}

}  // namespace pf
