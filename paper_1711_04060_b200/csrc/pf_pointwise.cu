// pf_pointwise.cu -- the pointwise nonlinear part of the PF outer loop (rows N1, N3, N5).
//
// N1: Fermi-like distribution, Eq (1): C_k = C_k^B exp(-z_k phi + lam_k S),
//     S = ln(Gamma/Gamma^B), Gamma = 1 - sum v_k C_k, solved simultaneously per node (reading R4):
//     S is the root of g(S) = log sum_{k=0..K+1} exp(a_k + lam_k S), a_0 = ln Gamma^B, lam_0 = 1,
//     a_k = ln(v_k C_k^B) - z_k phi; Newton from S = 0 with the maximum subtracted.
//     One fused kernel also emits what the two linear systems need: PF1's right-hand side
//     -kappa rho (Eq (12)) and PF2's diagonal A0 + sigma, sigma = -kappa rho'
//     with S held fixed (Eq (11)) -- so A^PF2 is never rebuilt.
#include "pf_launch.h"
#include <algorithm>

namespace pf {

namespace {

constexpr int PW_THREADS = 256;

int pw_blocks(long long n) {
    long long b = (n + PW_THREADS - 1) / PW_THREADS;
    return (int)std::min<long long>(std::max<long long>(b, 1), 148 * 16);
}

__device__ __forceinline__ bool on_boundary(const GridDims& g, long long i) {
    const int ix = (int)(i % g.nx);
    const long long q = i / g.nx;
    const int iy = (int)(q % g.ny);
    const int iz = (int)(q / g.ny);
    return ix == 0 || ix == g.nx - 1 || iy == 0 || iy == g.ny - 1 || iz == 0 || iz == g.nz - 1;
}

__device__ __forceinline__ int dirichlet_face_pw(const GridDims& g, const BcDev& bc, long long i) {
    const int ix = (int)(i % g.nx);
    const long long q = i / g.nx;
    const int iy = (int)(q % g.ny);
    const int iz = (int)(q / g.ny);
    if (ix == 0 && bc.type[0] == 0) return 0;
    if (ix == g.nx - 1 && bc.type[1] == 0) return 1;
    if (iy == 0 && bc.type[2] == 0) return 2;
    if (iy == g.ny - 1 && bc.type[3] == 0) return 3;
    if (iz == 0 && bc.type[4] == 0) return 4;
    if (iz == g.nz - 1 && bc.type[5] == 0) return 5;
    return -1;
}

__global__ void __launch_bounds__(PW_THREADS)
k_fermi(GridDims g, BcDev bc, SpeciesDev sp, const double* __restrict__ eps, double eps_mid, bool uniform,
        const double* __restrict__ phi, double* __restrict__ rho_o, double* __restrict__ sigma_o,
        double* __restrict__ S_o, double* __restrict__ conc, double* __restrict__ b1,
        const double* __restrict__ a0, double* __restrict__ a2, double* S_state, int lag_update) {
    const int K = sp.K;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        // Q17; Eq (1) lives in Omega_s only, and not in Omega_f (F3)
        const bool solvent = (uniform || eps[i] > eps_mid) && !is_fixed_node(bc, i);
        double S = 0.0, rho = 0.0, sig = 0.0;
        double c[PF_MAX_SPECIES];
#pragma unroll
        for (int k = 0; k < PF_MAX_SPECIES; ++k) c[k] = 0.0;
        if (solvent) {
            const double ph = phi[i];
            // Lagged reading of Eq (11) (PF_OPT_STERIC_MODE = 1; readings G1, G2): S^trc is the state left by the previous
            // outer iteration (0 before the first); no simultaneous solve
            if (S_state) S = S_state[i];
            if (sp.steric && !S_state) {
                for (int itn = 0; itn < 50; ++itn) {
                    const double t0 = sp.ln_gammaB + S;
                    double tmax = t0;
                    double tk[PF_MAX_SPECIES];
#pragma unroll
                    for (int k = 0; k < PF_MAX_SPECIES; ++k)
                        if (k <= K && sp.vol[k] > 0.0) {
                            tk[k] = sp.lnvc[k] - sp.z[k] * ph + sp.lam[k] * S;
                            tmax = fmax(tmax, tk[k]);
                        }
                    const double e0 = exp(t0 - tmax);
                    double sum = e0, dsum = e0;
#pragma unroll
                    for (int k = 0; k < PF_MAX_SPECIES; ++k)
                        if (k <= K && sp.vol[k] > 0.0) {
                            const double e = exp(tk[k] - tmax);
                            sum += e;
                            dsum += sp.lam[k] * e;
                        }
                    const double gval = tmax + log(sum);
                    const double dS = -gval / (dsum / sum);
                    S += dS;
                    if (fabs(dS) <= 1e-14 * fmax(1.0, fabs(S))) break;
                }
            }
#pragma unroll
            for (int k = 0; k < PF_MAX_SPECIES; ++k)
                if (k <= K) {
                    const double ck = sp.cb[k] * exp(-sp.z[k] * ph + sp.lam[k] * S);   // Eq (1)
                    c[k] = ck;
                    if (k < K) { rho += sp.z[k] * ck; sig += sp.z[k] * sp.z[k] * ck; }
                }
            sig = sp.kappa * sig;
            if (S_state && lag_update && sp.steric) {
                // Gamma_0 from the C_k^0 just formed, floored (G2), gives S^trc of the NEXT outer iteration
                double occ = 0.0;
#pragma unroll
                for (int k = 0; k < PF_MAX_SPECIES; ++k)
                    if (k <= K) occ += sp.vol[k] * c[k];
                S_state[i] = log(fmax(1.0 - occ, 1e-12) / sp.gammaB);
            }
        }
        if (rho_o) rho_o[i] = rho;
        if (sigma_o) sigma_o[i] = sig;
        if (S_o) S_o[i] = S;
        if (conc) {
#pragma unroll
            for (int k = 0; k < PF_MAX_SPECIES; ++k)
                if (k <= K) conc[(long long)k * g.n + i] = c[k];
        }
        if (b1) b1[i] = (!solvent || on_boundary(g, i)) ? 0.0 : -(sp.kappa * rho);
        if (a2) a2[i] = (dirichlet_face_pw(g, bc, i) >= 0 || is_fixed_node(bc, i)) ? a0[i] : add(a0[i], sig);   // identity rows stay identity
    }
}

// PF2 right-hand side, Eq (13): -eps Psi - rho' phi0 in the solvent, plus the
// fixed charges; Dirichlet rows carry the boundary value.
__global__ void __launch_bounds__(PW_THREADS)
k_rhs_pf2(GridDims g, BcDev bc, const double* __restrict__ eps, double eps_mid, bool uniform,
          const double* __restrict__ psi, const double* __restrict__ sigma, const double* __restrict__ phi0,
          const double* __restrict__ fixed, double* __restrict__ b) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride) {
        const int f = dirichlet_face_pw(g, bc, i);
        if (f >= 0) { b[i] = bc.value[f]; continue; }
        if (is_fixed_node(bc, i)) { b[i] = bc.fixv[i]; continue; }
        const double e = eps[i];
        const bool solvent = uniform || e > eps_mid;
        const double addv = solvent ? add(-mul(e, psi[i]), mul(sigma[i], phi0[i])) : 0.0;
        b[i] = add(addv, fixed[i]);
    }
}

// Table 2 step 5 (Q8, Q9): Phi := w Phi0 + (1-w) Phi, then ||Phi - Phi0||_inf.
__global__ void __launch_bounds__(PW_THREADS)
k_relax(long long n, double w, double w1, const double* __restrict__ phi0, double* __restrict__ phi,
        unsigned long long* dmax_bits) {
    double d = 0.0;
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride) {
        const double p0 = phi0[i];
        const double pn = add(mul(w, p0), mul(w1, phi[i]));
        phi[i] = pn;
        d = max_abs(d, sub(pn, p0));
    }
    // d >= 0 or NaN: the bit pattern orders like the value and a NaN (a diverged solve) has the largest pattern, so
    // every level of the reduction keeps it (max_abs, pf_common.cuh); the host turns it into PF_ERR_BREAKDOWN
    for (int s = 16; s > 0; s >>= 1) d = max_abs(d, __shfl_xor_sync(0xffffffffu, d, s));
    if ((threadIdx.x & 31) == 0) atomicMax(dmax_bits, (unsigned long long)__double_as_longlong(d));
}

}  // namespace

// a2 = a0 + sigma off the Dirichlet rows (pf_solve_linear with a caller-supplied sigma).
__global__ void __launch_bounds__(PW_THREADS)
k_diag_plus_sigma(GridDims g, BcDev bc, const double* __restrict__ a0, const double* __restrict__ sigma,
                  double* __restrict__ a2) {
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < g.n; i += stride)
        a2[i] = (dirichlet_face_pw(g, bc, i) >= 0 || is_fixed_node(bc, i)) ? a0[i] : add(a0[i], sigma[i]);
}

void launch_diag_plus_sigma(cudaStream_t s, const GridDims& g, const BcDev& bc, const double* a0, const double* sigma,
                            double* a2) {
    ++g_launch_count;
    k_diag_plus_sigma<<<pw_blocks(g.n), PW_THREADS, 0, s>>>(g, bc, a0, sigma, a2);
}

void launch_fermi(cudaStream_t s, const GridDims& g, const BcDev& bc, const SpeciesDev& sp, const double* eps, double eps_mid,
                  bool uniform, const double* phi, double* rho, double* sigma, double* S, double* conc, double* b1,
                  const double* a0, double* a2, double* S_state, bool lag_update) {
    ++g_launch_count;
    k_fermi<<<pw_blocks(g.n), PW_THREADS, 0, s>>>(g, bc, sp, eps, eps_mid, uniform, phi, rho, sigma, S, conc, b1, a0, a2,
                                                  S_state, lag_update ? 1 : 0);
}

void launch_rhs_pf2(cudaStream_t s, const GridDims& g, const BcDev& bc, const double* eps, double eps_mid,
                    bool uniform, const double* psi, const double* sigma, const double* phi0, const double* fixed,
                    double* b) {
    ++g_launch_count;
    k_rhs_pf2<<<pw_blocks(g.n), PW_THREADS, 0, s>>>(g, bc, eps, eps_mid, uniform, psi, sigma, phi0, fixed, b);
}

void launch_relax(cudaStream_t s, long long n, double w, const double* phi0, double* phi,
                  unsigned long long* dmax_bits) {
    cudaMemsetAsync(dmax_bits, 0, sizeof(unsigned long long), s);
    ++g_launch_count;
    k_relax<<<pw_blocks(n), PW_THREADS, 0, s>>>(n, w, 1.0 - w, phi0, phi, dmax_bits);
}

}  // namespace pf
