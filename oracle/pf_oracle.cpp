// pf_oracle.cpp -- CPU ORACLE for the Poisson-Fermi hot path of arXiv 1711.04060.
//
// THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke()
// and bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code
// with the CUDA path (paper_1711_04060_b200/csrc) and neither includes the other.
//
// Plain, slow, single-threaded C++17, fp64.  Inner products are evaluated as if in twice the
// working precision (Dot2, see dot()) so that the reduced scalars do not depend on summation
// order.  Build with -O2 -ffp-contract=off: every arithmetic operation below is rounded once,
// as written (std::fma appears only inside dot()).
// No blocking, fusion or reordering beyond what the paper's tables state.
//
// Citations are PAPER.md:<line> (+ equation/table) or the SURVEY.md section 8(c)
// reading (R0..R5, Q1..Q29) that DESIGN.md lists.
//
// Conventions: grid nx*ny*nz nodes INCLUDING boundary nodes, i = ix + nx*(iy + ny*iz)
// (PAPER.md:219).  phi in k_BT/e, lengths in Angstrom, concentrations in 1/A^3, charges
// in e.  Matrix in the paper's 7-vector diagonal format A0..A6, stored
// here as one array A[7*N] with A[d*N+i]:
//   d=0 diagonal, 1: j=i+1 (east), 2: i-1 (west), 3: i-nx (south), 4: i+nx (north),
//   5: i-nx*ny (down), 6: i+nx*ny (up).
// bc: faces in the order -x,+x,-y,+y,-z,+z; type 0 = Dirichlet(value), 1 = zero-Neumann.
//
// Pins (tests/test_oracle_*.py, all -m "not gpu"):
//   assembly      : SMIB identities of Eqs (17)-(18); row sums; symmetry; 1-D two-dielectric slab
//   linear solver : discrete sine-mode closed form; O(h^2) manufactured solution; dense LU on 8^3;
//                   scipy sparse LU; M=I reproduces Table 3 transcribed independently in numpy;
//                   1-D Debye-Hueckel sinh profile (pins the sigma diagonal)
//   pointwise     : phi=0 => S=0, C=C^B; equal-radii closed form; sum v_k C_k + Gamma = 1;
//                   saturation C_k < 1/v_k; radii->0 => Boltzmann
//   outer loop    : l_c=0 + steric off => nonlinear PB (Gouy-Chapman closed form in 1-D);
//                   independence of omega_PF; fixed-point residuals of PF1/PF2 at convergence
//                   l_c > 0 coupling: closed form of the discrete split system for a sine-mode source
//   full PF with l_c>0, steric term (unequal radii) and strong nonlinearity together, 3-D: a manufactured discrete
//                   solution (independent Fermi root finder + sine-transform PF1 solve in numpy) that the outer loop
//                   must converge to, and second-order grid refinement (tests/test_oracle_pf.py)
//   merged BiCGSTAB (reading M1): dense LU, numpy transcription, the identity rho_i = r~.r_i, agreement with Table 3
//                   (tests/test_oracle_merged.py);  lagged reading of Eq (11) (G1, G2): same fixed point, first step
//                   by hand, the two-cycle on configs[0];  non-finite data (D7): breakdown, not success
//   singular charges (Eqs 5-10): Coulomb sums vs numpy; 1-D closed form with a prescribed flux jump (c0, d0 of
//                   Eqs 17-18); discrete Gauss law sum b^IF h^3 = kappa sum q; harmonic phi^L; Born ion;
//                   agreement with the independent deposition model in the solvent (tests/test_oracle_singular.py)

#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>
#include <algorithm>

namespace {

// ---- R0: constants from Table 1, computed, not retyped -------------
const double K_B = 1.38e-23;      // J/K
const double T_ABS = 298.15;      // K
const double E_CH = 1.602e-19;    // C
const double EPS0 = 8.85e-14;     // F/cm
const double AVOGADRO_PER_A3 = 6.02214076e-4;  // 1 mol/L in 1/A^3

double kappa_angstrom() {
    // kappa = e^2/(eps0 kB T); eps0 in F/cm -> F/m is *100; metres -> Angstrom is *1e10.
    double eps0_m = EPS0 * 100.0;
    return E_CH * E_CH / (eps0_m * K_B * T_ABS) * 1e10;
}

struct Grid {
    int nx, ny, nz;
    double h;
    int bc_type[6];
    double bc_value[6];
    // Omega_f (readings F1-F3): nodes whose potential is prescribed by an atomic model the
    // caller brings.  fix_mask[i] != 0 => phi_i = fix_val[i] (an interior Dirichlet node).  Null = no such nodes.
    const uint8_t* fix_mask = nullptr;
    const double* fix_val = nullptr;
    int64_t n() const { return (int64_t)nx * ny * nz; }
};

// First Dirichlet face (in the order -x,+x,-y,+y,-z,+z) the node lies on, else -1.  (Q20)
int dirichlet_face(const Grid& g, int ix, int iy, int iz) {
    if (ix == 0 && g.bc_type[0] == 0) return 0;
    if (ix == g.nx - 1 && g.bc_type[1] == 0) return 1;
    if (iy == 0 && g.bc_type[2] == 0) return 2;
    if (iy == g.ny - 1 && g.bc_type[3] == 0) return 3;
    if (iz == 0 && g.bc_type[4] == 0) return 4;
    if (iz == g.nz - 1 && g.bc_type[5] == 0) return 5;
    return -1;
}

bool on_box_boundary(const Grid& g, int ix, int iy, int iz) {
    return ix == 0 || ix == g.nx - 1 || iy == 0 || iy == g.ny - 1 || iz == 0 || iz == g.nz - 1;
}

// Face coefficient between two nodes: harmonic mean of eps over h^2.  This IS the paper's
// SMIB row pair, Eqs (17)-(18): eps_m*c2 = eps_s*d1 = 2 eps_m eps_s/(eps_m+eps_s)
// and 2-c1 = 1+c2, 2-d2 = 1+d1 (reading R2/Q16: interface at the face midpoint).
double face_coeff(double ea, double eb, double h) {
    return (2.0 * ea * eb / (ea + eb)) / (h * h);
}

// ---- L1/L2: assembly of  -div(eps grad u) + sigma u  with boundary rows ----------------
// Interior row: (sum_f c_f + sigma_i) u_i - sum_f c_f u_nb.  Dirichlet node: identity row.
// Zero-Neumann face: the outward face flux is omitted (Q21).  Neighbours keep their coupling
// to Dirichlet nodes (Q20, uniform stencil).
void assemble_poisson(const Grid& g, const double* eps, const double* sigma, double* A) {
    const int64_t N = g.n();
    const int64_t off[7] = {0, 1, -1, -(int64_t)g.nx, (int64_t)g.nx,
                            -(int64_t)g.nx * g.ny, (int64_t)g.nx * g.ny};
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                if (dirichlet_face(g, ix, iy, iz) >= 0 || (g.fix_mask && g.fix_mask[i])) {   // Q20, F2
                    A[i] = 1.0;
                    for (int d = 1; d < 7; ++d) A[d * N + i] = 0.0;
                    continue;
                }
                bool inside[7] = {true, ix + 1 < g.nx, ix - 1 >= 0, iy - 1 >= 0, iy + 1 < g.ny,
                                  iz - 1 >= 0, iz + 1 < g.nz};
                double diag = 0.0;
                for (int d = 1; d < 7; ++d) {
                    if (!inside[d]) { A[d * N + i] = 0.0; continue; }
                    double c = face_coeff(eps[i], eps[i + off[d]], g.h);
                    A[d * N + i] = -c;
                    diag = diag + c;
                }
                A[i] = diag + (sigma ? sigma[i] : 0.0);
            }
}

// ---- N2: PF1 operator  eps (l_c^2 Lap - 1) Psi = kappa rho, times -1 ----
// (eps_i l_c^2/h^2)(6 Psi_i - sum Psi_nb) + eps_i Psi_i on solvent nodes strictly inside the box;
// identity rows (Psi = 0) at every non-solvent node and every box-boundary node (Q15).
void assemble_pf1(const Grid& g, const double* eps, const uint8_t* solvent, double lc, double* A) {
    const int64_t N = g.n();
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                if (on_box_boundary(g, ix, iy, iz) || !solvent[i]) {
                    A[i] = 1.0;
                    for (int d = 1; d < 7; ++d) A[d * N + i] = 0.0;
                    continue;
                }
                double c = eps[i] * (lc * lc) / (g.h * g.h);
                A[i] = 6.0 * c + eps[i];
                for (int d = 1; d < 7; ++d) A[d * N + i] = -c;
            }
}

// ---- K2: y = A x in diagonal format --------------------------------------
// Coefficients that point outside the index range are exactly 0 by construction and are
// never read together with an out-of-range x.
void dia_spmv(const Grid& g, const double* A, const double* x, double* y) {
    const int64_t N = g.n();
    const int64_t off[7] = {0, 1, -1, -(int64_t)g.nx, (int64_t)g.nx,
                            -(int64_t)g.nx * g.ny, (int64_t)g.nx * g.ny};
    for (int64_t i = 0; i < N; ++i) {
        double acc = A[i] * x[i];
        for (int d = 1; d < 7; ++d) {
            int64_t j = i + off[d];
            double a = A[d * N + i];
            if (a != 0.0 && j >= 0 && j < N) acc = acc + a * x[j];
        }
        y[i] = acc;
    }
}

// K3: inner product.  The value of sum a_i b_i does not depend on the order of
// summation, but a floating-point sum does, and BiCGSTAB amplifies such last-bit differences into
// iteration counts that differ by several per cent (D2).  The oracle therefore computes
// the inner product as if in twice the working precision and rounds once at the end: algorithm
// Dot2 of Ogita, Rump & Oishi, "Accurate sum and dot product", SIAM J. Sci. Comput. 26 (2005):
// TwoProduct (exact product via fma) and Knuth's TwoSum (exact sum), error terms accumulated
// separately.  The result is the correctly rounded inner product except with negligible
// probability, i.e. it is (for all practical purposes) independent of summation order.
// Pinned against exact rational arithmetic in tests/test_oracle_linear.py.
double dot(int64_t N, const double* a, const double* b) {
    double hi = 0.0, lo = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        double p = a[i] * b[i];
        double ep = std::fma(a[i], b[i], -p);       // TwoProduct: a*b = p + ep exactly
        double s = hi + p;                           // TwoSum: hi + p = s + es exactly
        double z = s - hi;
        double es = (hi - (s - z)) + (p - z);
        hi = s;
        lo = lo + (es + ep);
    }
    return hi + lo;
}

double norm2(int64_t N, const double* a) { return std::sqrt(dot(N, a, a)); }

// K4: maximum norm (Table 3 step 18).
// A NaN entry makes the norm NaN (std::max would drop it: every comparison with a NaN is false).
double norm_inf(int64_t N, const double* a) {
    double m = 0.0;
    for (int64_t i = 0; i < N; ++i) {
        double v = std::fabs(a[i]);
        if (std::isnan(v) || v > m) m = v;
        if (std::isnan(m)) break;
    }
    return m;
}

// Q4/Q20: force Dirichlet values into a vector.
void set_dirichlet(const Grid& g, double* x) {
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int f = dirichlet_face(g, ix, iy, iz);
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                if (f >= 0) x[i] = g.bc_value[f];
                else if (g.fix_mask && g.fix_mask[i]) x[i] = g.fix_val[i];
            }
}

// ---- Table 3 with the Templates Jacobi step (R3, Q2) -----------------
// Return: 0 converged, 1 maxit reached, -3 breakdown.
// precond = 1: M = diag(A) (right preconditioning: p^ = M^-1 p, v = A p^, ...); 0: M = I, which
// is Table 3 verbatim.  Stopping on the recurrence residual: norm_mode 0 (Q3, BASELINE): ||r||_2 <= tol*||b||_2;
// norm_mode 1 (the paper's own test, Table 3 steps 18-19): ||r||_inf < tol, absolute.
// In mode 1 relres_out, true_relres_out and hist carry the absolute maximum norms.
// Reading D7: a scalar that is not finite (||b||, ||r||, rho, r~.v, t.s, t.t) is a breakdown (-3);
// Table 3 is silent, and a NaN would otherwise fail "== 0" and never pass the convergence test.
int bicgstab(const Grid& g, const double* A, const double* b, double* x, double tol, int maxit,
             int precond, int* iters_out, double* relres_out, double* true_relres_out,
             double* hist /* maxit+1 or null */, int norm_mode = 0) {
    const int64_t N = g.n();
    std::vector<double> r(N), rt(N), p(N, 0.0), v(N, 0.0), s(N), t(N), ph(N), sh(N);
    *iters_out = 0;
    double bnorm = norm2(N, b);
    if (bnorm == 0.0) {  // Q3: b = 0 => x = 0, zero iterations
        std::fill(x, x + N, 0.0);
        if (relres_out) *relres_out = 0.0;
        if (true_relres_out) *true_relres_out = 0.0;
        return 0;
    }
    // step 2: r0 = b - A x0, r~ = r0
    dia_spmv(g, A, x, r.data());
    for (int64_t i = 0; i < N; ++i) r[i] = b[i] - r[i];
    rt = r;
    auto measure = [&](const double* u) { return norm_mode == 1 ? norm_inf(N, u) : norm2(N, u); };
    auto converged = [&](double rn) { return norm_mode == 1 ? rn < tol : rn <= tol * bnorm; };
    const double scale = norm_mode == 1 ? 1.0 : bnorm;
    double rnorm = measure(r.data());
    if (hist) hist[0] = rnorm / scale;
    int status = 1;
    double rho_old = 1.0, alpha = 1.0, omega = 1.0;
    if (!std::isfinite(bnorm) || !std::isfinite(rnorm)) status = -3;                  // D7
    else if (converged(rnorm)) status = 0;  // warm start already converged (DESIGN reading D1)
    int it = 0;
    while (status == 1 && it < maxit) {
        ++it;
        // step 4
        double rho = dot(N, rt.data(), r.data());
        if (rho == 0.0 || !std::isfinite(rho)) { status = -3; --it; break; }
        // steps 5-10
        if (it == 1) {
            p = r;
        } else {
            double beta = (rho / rho_old) * (alpha / omega);
            for (int64_t i = 0; i < N; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
        }
        // step 11 (+ Jacobi)
        for (int64_t i = 0; i < N; ++i) ph[i] = precond ? p[i] / A[i] : p[i];
        dia_spmv(g, A, ph.data(), v.data());
        // step 12
        double rtv = dot(N, rt.data(), v.data());
        if (rtv == 0.0 || !std::isfinite(rtv)) { status = -3; --it; break; }
        alpha = rho / rtv;
        // step 13
        for (int64_t i = 0; i < N; ++i) s[i] = r[i] - alpha * v[i];
        // step 14 (+ Jacobi)
        for (int64_t i = 0; i < N; ++i) sh[i] = precond ? s[i] / A[i] : s[i];
        dia_spmv(g, A, sh.data(), t.data());
        // step 15
        double ts = dot(N, t.data(), s.data());
        double tt = dot(N, t.data(), t.data());
        omega = (tt == 0.0) ? 0.0 : ts / tt;   // Q5
        if (!std::isfinite(ts) || !std::isfinite(tt)) { status = -3; --it; break; }   // D7
        // step 16
        for (int64_t i = 0; i < N; ++i) x[i] = x[i] + alpha * ph[i] + omega * sh[i];
        // step 17
        for (int64_t i = 0; i < N; ++i) r[i] = s[i] - omega * t[i];
        // steps 18-20
        rnorm = measure(r.data());
        if (hist) hist[it] = rnorm / scale;
        rho_old = rho;
        if (!std::isfinite(rnorm)) { status = -3; break; }                            // D7
        if (converged(rnorm)) { status = 0; break; }
        if (omega == 0.0) { status = -3; break; }
    }
    *iters_out = it;
    if (relres_out) *relres_out = rnorm / scale;
    if (true_relres_out) {
        dia_spmv(g, A, x, t.data());
        for (int64_t i = 0; i < N; ++i) t[i] = b[i] - t[i];
        *true_relres_out = measure(t.data()) / scale;
    }
    return status;
}

// ---- Merged BiCGSTAB: two reduction points per iteration (SURVEY.md section 8(d) "fully merged", 8(f) #3) --------
// The same Krylov method as Table 3 with the Jacobi step of R3, rearranged so that an iteration has two
// synchronisation points instead of three (PAPER.md:279 names inner products and synchronisation as where the
// solver's time goes).  Reading M1: from r_i = s - omega t and s = r_{i-1} - alpha v,
//     rho_i = r~.r_i = (r~.r_{i-1} - alpha r~.v) - omega r~.t ,
// a combination of inner products that are all known as soon as omega is: r~.t is reduced together with t.s and
// t.t, and r~.r_{i-1} together with r~.v and ||r_{i-1}|| one synchronisation earlier.  beta and the next p then need
// no reduction of their own:
//     start   r0 = b - A x0; r~ = r0; rho_0 = rhat_0 = r~.r0; p = r0; v = A M^-1 p;                 [r~.v]
//     i >= 1  alpha = rho_{i-1}/(r~.v); s = r - alpha v; t = A M^-1 s;                              [t.s, t.t, r~.t]
//             omega = t.s/t.t; x += alpha M^-1 p + omega M^-1 s; r = s - omega t;
//             rho_i = (rhat_{i-1} - alpha (r~.v)) - omega (r~.t); beta = (rho_i/rho_{i-1})(alpha/omega);
//             p = r + beta (p - omega v); v = A M^-1 p;                                             [r~.v, rhat_i = r~.r, ||r||]
//             stop if ||r|| meets the test.
// SURVEY 8(d) drops the bracket (it vanishes in exact arithmetic by the choice of alpha, leaving rho_i = -omega r~.t).
// In floating point it must stay: without it the rounding error of rho is never corrected, stays at eps |r~| |r_0|
// while |r_i| shrinks, and the recurrence stalls near a relative residual of 1e-6..1e-8 (measured with this oracle
// before the term was restored; tests/test_oracle_merged.py::test_merged_rho_identity_in_the_recurrence).  With it,
// rho_i differs from the directly reduced r~.r_i only by the rounding of s, r and three scalar operations.
// The iterates equal Table 3's in exact arithmetic; iteration paths separate from bicgstab() after O(100) iterations
// like those of any two roundings of the method.  Every elementwise statement is rounded as
// written; inner products through dot().  The test on ||r|| is made before the next p and v are formed (they are
// not needed when it passes); statuses, breakdown tests (Q5, D7) and outputs as bicgstab().
// rho_rec (maxit+1 or null) receives the rho_i the recurrence used, rho_direct (maxit+1 or null) the directly
// reduced r~.r_i: the pin of the identity compares them.
int bicgstab_merged(const Grid& g, const double* A, const double* b, double* x, double tol, int maxit,
                    int precond, int* iters_out, double* relres_out, double* true_relres_out,
                    double* hist /* maxit+1 or null */, int norm_mode, double* rho_rec, double* rho_direct) {
    const int64_t N = g.n();
    std::vector<double> r(N), rt(N), p(N), v(N), s(N), t(N), ph(N), sh(N);
    *iters_out = 0;
    double bnorm = norm2(N, b);
    if (bnorm == 0.0) {  // Q3
        std::fill(x, x + N, 0.0);
        if (relres_out) *relres_out = 0.0;
        if (true_relres_out) *true_relres_out = 0.0;
        return 0;
    }
    dia_spmv(g, A, x, r.data());
    for (int64_t i = 0; i < N; ++i) r[i] = b[i] - r[i];
    rt = r;
    auto measure = [&](const double* u) { return norm_mode == 1 ? norm_inf(N, u) : norm2(N, u); };
    auto converged = [&](double rn) { return norm_mode == 1 ? rn < tol : rn <= tol * bnorm; };
    const double scale = norm_mode == 1 ? 1.0 : bnorm;
    double rnorm = measure(r.data());
    if (hist) hist[0] = rnorm / scale;
    int status = 1;
    if (!std::isfinite(bnorm) || !std::isfinite(rnorm)) status = -3;                  // D7
    else if (converged(rnorm)) status = 0;                                            // D1
    double rho = dot(N, rt.data(), r.data());                                         // rho_0
    double rhat = rho;                                                                // r~.r of the current iterate
    if (rho_direct) rho_direct[0] = rho;
    if (rho_rec) rho_rec[0] = rho;
    int it = 0;
    double rtv = 0.0;
    if (status == 1 && maxit > 0) {
        if (rho == 0.0 || !std::isfinite(rho)) status = -3;
        else {
            p = r;
            for (int64_t i = 0; i < N; ++i) ph[i] = precond ? p[i] / A[i] : p[i];
            dia_spmv(g, A, ph.data(), v.data());
            rtv = dot(N, rt.data(), v.data());
        }
    }
    while (status == 1 && it < maxit) {
        ++it;
        if (rtv == 0.0 || !std::isfinite(rtv)) { status = -3; --it; break; }
        double alpha = rho / rtv;
        for (int64_t i = 0; i < N; ++i) s[i] = r[i] - alpha * v[i];
        for (int64_t i = 0; i < N; ++i) sh[i] = precond ? s[i] / A[i] : s[i];
        dia_spmv(g, A, sh.data(), t.data());
        double ts = dot(N, t.data(), s.data());
        double tt = dot(N, t.data(), t.data());
        double rtt = dot(N, rt.data(), t.data());
        double omega = (tt == 0.0) ? 0.0 : ts / tt;                                   // Q5
        if (!std::isfinite(ts) || !std::isfinite(tt)) { status = -3; --it; break; }   // D7
        for (int64_t i = 0; i < N; ++i) x[i] = x[i] + alpha * ph[i] + omega * sh[i];
        for (int64_t i = 0; i < N; ++i) r[i] = s[i] - omega * t[i];
        rnorm = measure(r.data());
        if (hist) hist[it] = rnorm / scale;
        double rho_new = (rhat - alpha * rtv) - omega * rtt;                          // M1
        rhat = dot(N, rt.data(), r.data());                                           // reduced with r~.v and ||r||
        if (rho_direct) rho_direct[it] = rhat;
        if (rho_rec) rho_rec[it] = rho_new;
        if (!std::isfinite(rnorm)) { status = -3; break; }                            // D7
        if (converged(rnorm)) { status = 0; break; }
        if (omega == 0.0) { status = -3; break; }
        if (it >= maxit) break;
        if (rho_new == 0.0 || !std::isfinite(rho_new)) { status = -3; break; }
        double beta = (rho_new / rho) * (alpha / omega);
        rho = rho_new;
        for (int64_t i = 0; i < N; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
        for (int64_t i = 0; i < N; ++i) ph[i] = precond ? p[i] / A[i] : p[i];
        dia_spmv(g, A, ph.data(), v.data());
        rtv = dot(N, rt.data(), v.data());
    }
    *iters_out = it;
    if (relres_out) *relres_out = rnorm / scale;
    if (true_relres_out) {
        dia_spmv(g, A, x, t.data());
        for (int64_t i = 0; i < N; ++i) t[i] = b[i] - t[i];
        *true_relres_out = measure(t.data()) / scale;
    }
    return status;
}

// solver 0: Table 3 (bicgstab); 1: the merged two-reduction form (bicgstab_merged).
int krylov(int solver, const Grid& g, const double* A, const double* b, double* x, double tol, int maxit,
           int precond, int* iters_out, double* relres_out, double* true_relres_out, double* hist, int norm_mode) {
    return solver == 1 ? bicgstab_merged(g, A, b, x, tol, maxit, precond, iters_out, relres_out, true_relres_out, hist,
                                         norm_mode, nullptr, nullptr)
                       : bicgstab(g, A, b, x, tol, maxit, precond, iters_out, relres_out, true_relres_out, hist, norm_mode);
}

// ---- R2: fixed point charges, trilinear deposition (Eq (3)) ----------------
// b_i += kappa q w_i / h^3 over the 8 corners of the cell containing the charge.
void deposit_charges(const Grid& g, const double* ch /* M x 4 */, int M, double* b) {
    const double kap = kappa_angstrom();
    for (int m = 0; m < M; ++m) {
        double px = ch[4 * m] / g.h, py = ch[4 * m + 1] / g.h, pz = ch[4 * m + 2] / g.h;
        double q = ch[4 * m + 3];
        int ix = std::min(std::max((int)std::floor(px), 0), g.nx - 2);
        int iy = std::min(std::max((int)std::floor(py), 0), g.ny - 2);
        int iz = std::min(std::max((int)std::floor(pz), 0), g.nz - 2);
        double fx = px - ix, fy = py - iy, fz = pz - iz;
        double amp = kap * q / (g.h * g.h * g.h);
        for (int dz = 0; dz < 2; ++dz)
            for (int dy = 0; dy < 2; ++dy)
                for (int dx = 0; dx < 2; ++dx) {
                    double w = (dx ? fx : 1.0 - fx) * (dy ? fy : 1.0 - fy) * (dz ? fz : 1.0 - fz);
                    int64_t i = (ix + dx) + (int64_t)g.nx * ((iy + dy) + (int64_t)g.ny * (iz + dz));
                    b[i] = b[i] + amp * w;
                }
    }
}

// ---- R4: Fermi-like distribution, Eq (1), solved pointwise --------------
struct SpeciesTab {
    int K;                       // ions; water is index K
    std::vector<double> z;       // K+1 (water 0)
    std::vector<double> cb;      // K+1, 1/A^3
    std::vector<double> vol;     // K+1, A^3
    std::vector<double> lam;     // K+1, v_k/v_0
    double gammaB;
    bool steric;
};

// returns 0 ok, -4 nonphysical
int make_species(int K, const double* valence, const double* bath_molar, const double* radii,
                 double water_molar, SpeciesTab& sp) {
    sp.K = K;
    sp.z.assign(K + 1, 0.0); sp.cb.assign(K + 1, 0.0); sp.vol.assign(K + 1, 0.0); sp.lam.assign(K + 1, 0.0);
    double vsum = 0.0;
    for (int k = 0; k <= K; ++k) {
        sp.z[k] = k < K ? valence[k] : 0.0;
        sp.cb[k] = (k < K ? bath_molar[k] : water_molar) * AVOGADRO_PER_A3;
        sp.vol[k] = 4.0 * M_PI * radii[k] * radii[k] * radii[k] / 3.0;   // v_i = 4 pi a_i^3/3
        vsum += sp.vol[k];
    }
    double v0 = vsum / (K + 1);
    sp.steric = vsum > 0.0;
    double occ = 0.0;
    for (int k = 0; k <= K; ++k) {
        sp.lam[k] = sp.steric ? sp.vol[k] / v0 : 0.0;                    // Q25
        occ += sp.vol[k] * sp.cb[k];
    }
    sp.gammaB = 1.0 - occ;
    if (!(sp.gammaB > 0.0)) return -4;
    double net = 0.0, tot = 0.0;                                         // Q26 bath neutrality
    for (int k = 0; k < K; ++k) { net += sp.z[k] * sp.cb[k]; tot += std::fabs(sp.z[k]) * sp.cb[k]; }
    if (std::fabs(net) > 1e-12 * tot) return -4;
    return 0;
}

// One node.  Solves the three simultaneous definitions of Eq (1) exactly (R4, Q11):
// g(S) = log sum_{k=0..K+1} exp(a_k + lam_k S) = 0 with a_0 = ln Gamma^B, lam_0 = 1,
// a_k = ln(v_k C_k^B) - z_k phi.  Newton from S = 0.  Outputs C_k, S, rho, sigma = -kappa rho'.
void fermi_node(const SpeciesTab& sp, double kap, double phi, double* conc /*K+1*/, double* S_out,
                double* rho_out, double* sigma_out) {
    const int K = sp.K;
    double S = 0.0;
    if (sp.steric) {
        for (int itn = 0; itn < 50; ++itn) {
            // terms t_k = a_k + lam_k S, k = 0 is the void term
            double tmax = std::log(sp.gammaB) + S;
            for (int k = 0; k <= K; ++k)
                if (sp.vol[k] > 0.0)
                    tmax = std::max(tmax, std::log(sp.vol[k] * sp.cb[k]) - sp.z[k] * phi + sp.lam[k] * S);
            double e0 = std::exp(std::log(sp.gammaB) + S - tmax);
            double sum = e0, dsum = e0;   // lam_0 = 1
            for (int k = 0; k <= K; ++k)
                if (sp.vol[k] > 0.0) {
                    double e = std::exp(std::log(sp.vol[k] * sp.cb[k]) - sp.z[k] * phi + sp.lam[k] * S - tmax);
                    sum += e;
                    dsum += sp.lam[k] * e;
                }
            double gval = tmax + std::log(sum);
            double dS = -gval / (dsum / sum);
            S += dS;
            if (std::fabs(dS) <= 1e-14 * std::max(1.0, std::fabs(S))) break;
        }
    }
    double rho = 0.0, sig = 0.0;
    for (int k = 0; k <= K; ++k) {
        double c = sp.cb[k] * std::exp(-sp.z[k] * phi + sp.lam[k] * S);  // Eq (1)
        conc[k] = c;
        if (k < K) { rho += sp.z[k] * c; sig += sp.z[k] * sp.z[k] * c; }
    }
    *S_out = S;
    *rho_out = rho;
    *sigma_out = kap * sig;   // sigma = -kappa rho', rho' = -sum z_k^2 C_k with S held fixed
}

// Q17: solvent nodes are those with eps above the midpoint of the map's range; uniform => all.
void solvent_mask(int64_t N, const double* eps, uint8_t* mask) {
    double lo = eps[0], hi = eps[0];
    for (int64_t i = 1; i < N; ++i) { lo = std::min(lo, eps[i]); hi = std::max(hi, eps[i]); }
    double mid = 0.5 * (lo + hi);
    for (int64_t i = 0; i < N; ++i) mask[i] = (lo == hi) ? 1 : (eps[i] > mid ? 1 : 0);
}

void fermi_field(const SpeciesTab& sp, int64_t N, const double* phi, const uint8_t* solvent,
                 double* rho, double* sigma, double* S, double* conc /* (K+1)*N or null */) {
    const double kap = kappa_angstrom();
    std::vector<double> c(sp.K + 1);
    for (int64_t i = 0; i < N; ++i) {
        double s = 0.0, r = 0.0, sg = 0.0;
        if (solvent[i]) fermi_node(sp, kap, phi[i], c.data(), &s, &r, &sg);
        else std::fill(c.begin(), c.end(), 0.0);          // defined only in Omega_s
        if (rho) rho[i] = r;
        if (sigma) sigma[i] = sg;
        if (S) S[i] = s;
        if (conc) for (int k = 0; k <= sp.K; ++k) conc[(int64_t)k * N + i] = c[k];
    }
}

// ---- Lagged reading of Eq (11) (readings G1-G2 of DESIGN.md) --------------------
// Eq (11) writes C_k^0, S_0^trc and Gamma_0 with the same subscript 0 although each is defined through the others.
// Besides solving the three definitions simultaneously per node (fermi_node, the default), one can take them as
// assignments in the order written: C_k^0 from phi_0 and the S^trc that is at hand (that of the previous outer
// iteration, 0 = the bath value before the first), then Gamma_0 from these C_k^0, then S_0^trc from Gamma_0 for the
// NEXT outer iteration.  Both readings have the same fixed point.  G2: nothing keeps sum v_k C_k^0 below 1 here
// (the saturation property C_k < 1/v_k of PAPER.md:45 belongs to the simultaneous solution), so Gamma_0 is floored
// at GAMMA_FLOOR before the logarithm.  S (N, in/out): the state; null entries of the outputs are skipped.
const double GAMMA_FLOOR = 1e-12;

void fermi_field_lagged(const SpeciesTab& sp, int64_t N, const double* phi, const uint8_t* solvent, double* S,
                        bool update, double* rho, double* sigma, double* conc /* (K+1)*N or null */) {
    const double kap = kappa_angstrom();
    std::vector<double> c(sp.K + 1);
    for (int64_t i = 0; i < N; ++i) {
        double r = 0.0, sg = 0.0;
        if (solvent[i]) {
            double occ = 0.0;
            for (int k = 0; k <= sp.K; ++k) {
                c[k] = sp.cb[k] * std::exp(-sp.z[k] * phi[i] + sp.lam[k] * S[i]);        // Eq (1) with the S at hand
                if (k < sp.K) { r += sp.z[k] * c[k]; sg += sp.z[k] * sp.z[k] * c[k]; }
                occ += sp.vol[k] * c[k];
            }
            sg = kap * sg;
            if (update && sp.steric) S[i] = std::log(std::max(1.0 - occ, GAMMA_FLOOR) / sp.gammaB);   // G2
        } else {
            std::fill(c.begin(), c.end(), 0.0);
        }
        if (rho) rho[i] = r;
        if (sigma) sigma[i] = sg;
        if (conc) for (int k = 0; k <= sp.K; ++k) conc[(int64_t)k * N + i] = c[k];
    }
}

// N2/N3 right-hand sides.
void rhs_pf1(const Grid& g, const uint8_t* solvent, const double* rho, double* b) {
    const double kap = kappa_angstrom();
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                b[i] = (on_box_boundary(g, ix, iy, iz) || !solvent[i]) ? 0.0 : -(kap * rho[i]);
            }
}

void rhs_pf2(const Grid& g, const double* eps, const uint8_t* solvent, const double* psi,
             const double* sigma, const double* phi0, const double* fixed, double* b) {
    const int64_t N = g.n();
    for (int64_t i = 0; i < N; ++i) {
        double add = solvent[i] ? (-(eps[i] * psi[i]) + sigma[i] * phi0[i]) : 0.0;
        b[i] = add + fixed[i];
    }
    set_dirichlet(g, b);
}

}  // namespace

// =========================================================================================
// Singular-charge decomposition, Eqs (5)-(10) and the flux-jump terms of Eqs (17)-(18)
// (readings S1-S5 of DESIGN.md).
//   phi = phi~ + phi* + phi^L in Omega_m (the non-solvent nodes),  phi = phi~ in Omega_s.
//   phi*(r) = kappa/(4 pi eps_m) sum_j q_j/|r - r_j|                              (Eq 5, units R0)
//   Laplace phi^L = 0 in Omega_m,  phi^L = -phi* on the boundary of Omega_m        (Eqs 9-10, S1)
//   [eps grad phi~ . n] = eps_m grad(phi* + phi^L) . n on the interface            (Eq 8)
// Discretisation (S2): the interface cuts every face between an Omega_m node i and an Omega_s
// node j at its midpoint x_f (Q16).  Laplace rows at interior Omega_m nodes: (u_i - u_nb)/h^2 per
// face towards an Omega_m neighbour, 2 (u_i - g_f)/h^2 per interface face (ghost value 2 g_f - u_i,
// g_f = -phi*(x_f)); Omega_m nodes on the box boundary carry u = -phi* (S3: Eq (10) on ALL of the
// boundary of Omega_m); Omega_s nodes are identity rows with u = 0.
// Flux jump on an interface face, n from i (Omega_m) to j (Omega_s):
//   J_f = eps_i [ dphi*/dn (x_f) + 2 (g_f - u_i)/h ]                                (Eq 8)
// enters the two rows next to the face exactly as c0, d0 of Eqs (17)-(18):
//   b_i += -eps_i J_f/((eps_i + eps_j) h),   b_j += -eps_j J_f/((eps_i + eps_j) h).
// =========================================================================================
namespace {

const double FOUR_PI = 4.0 * M_PI;

// phi* at the point (x, y, z) [Angstrom]; charges summed in list order.
double coulomb_potential(const double* ch, int M, double eps_m, double x, double y, double z) {
    double s = 0.0;
    for (int j = 0; j < M; ++j) {
        double dx = x - ch[4 * j], dy = y - ch[4 * j + 1], dz = z - ch[4 * j + 2];
        double r = std::sqrt(dx * dx + dy * dy + dz * dz);
        s = s + ch[4 * j + 3] / r;
    }
    return (kappa_angstrom() / (FOUR_PI * eps_m)) * s;
}

// d phi*/d x_axis at the point: -kappa/(4 pi eps_m) sum q (x_axis - r_j,axis)/r^3.
double coulomb_gradient(const double* ch, int M, double eps_m, double x, double y, double z, int axis) {
    double s = 0.0;
    for (int j = 0; j < M; ++j) {
        double dx = x - ch[4 * j], dy = y - ch[4 * j + 1], dz = z - ch[4 * j + 2];
        double r2 = dx * dx + dy * dy + dz * dz;
        double r = std::sqrt(r2);
        double comp = axis == 0 ? dx : (axis == 1 ? dy : dz);
        s = s + ch[4 * j + 3] * comp / (r2 * r);
    }
    return -((kappa_angstrom() / (FOUR_PI * eps_m)) * s);
}

// Face d (1..6, PAPER.md:219 order) of node (ix,iy,iz): neighbour offset, axis and outward sign.
const int FACE_DX[7] = {0, 1, -1, 0, 0, 0, 0};
const int FACE_DY[7] = {0, 0, 0, -1, 1, 0, 0};
const int FACE_DZ[7] = {0, 0, 0, 0, 0, -1, 1};
const int FACE_AXIS[7] = {0, 0, 0, 1, 1, 2, 2};
const int FACE_SIGN[7] = {0, 1, -1, -1, 1, -1, 1};

// Laplace system for phi^L in Omega_m (S2, S3): matrix in the diagonal format, right-hand side, and the
// vector of prescribed values (identity rows: Omega_s nodes 0, boundary Omega_m nodes -phi*).
void assemble_laplace_m(const Grid& g, const uint8_t* solvent, const double* ch, int M, double eps_m,
                        double* A, double* b) {
    const int64_t N = g.n();
    const int64_t off[7] = {0, 1, -1, -(int64_t)g.nx, (int64_t)g.nx, -(int64_t)g.nx * g.ny, (int64_t)g.nx * g.ny};
    const double c = 1.0 / (g.h * g.h);
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                for (int d = 1; d < 7; ++d) A[d * N + i] = 0.0;
                if (solvent[i]) { A[i] = 1.0; b[i] = 0.0; continue; }
                if (on_box_boundary(g, ix, iy, iz)) {
                    A[i] = 1.0;
                    b[i] = -coulomb_potential(ch, M, eps_m, ix * g.h, iy * g.h, iz * g.h);
                    continue;
                }
                double diag = 0.0, rhs = 0.0;
                for (int d = 1; d < 7; ++d) {
                    int64_t j = i + off[d];
                    if (!solvent[j]) { A[d * N + i] = -c; diag = diag + c; continue; }
                    double xf = (ix + 0.5 * FACE_DX[d]) * g.h, yf = (iy + 0.5 * FACE_DY[d]) * g.h,
                           zf = (iz + 0.5 * FACE_DZ[d]) * g.h;
                    double gf = -coulomb_potential(ch, M, eps_m, xf, yf, zf);
                    diag = diag + 2.0 * c;
                    rhs = rhs + (2.0 * c) * gf;
                }
                A[i] = diag;
                b[i] = rhs;
            }
}

// Flux jumps J_f on the interface faces, stored at the Omega_m node: J[(d-1)*N + i] for face d of node i
// (0 where face d of i is not an interface face).  Box-boundary Omega_m nodes have no rows of their own in
// the Poisson system beyond what the boundary condition gives, but their interface faces still separate two
// materials and carry a jump like any other.
void face_jumps(const Grid& g, const double* eps, const uint8_t* solvent, const double* ch, int M, double eps_m,
                const double* phiL, double* J) {
    const int64_t N = g.n();
    const int64_t off[7] = {0, 1, -1, -(int64_t)g.nx, (int64_t)g.nx, -(int64_t)g.nx * g.ny, (int64_t)g.nx * g.ny};
    std::fill(J, J + 6 * N, 0.0);
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                if (solvent[i]) continue;
                bool inside[7] = {true, ix + 1 < g.nx, ix - 1 >= 0, iy - 1 >= 0, iy + 1 < g.ny, iz - 1 >= 0, iz + 1 < g.nz};
                for (int d = 1; d < 7; ++d) {
                    if (!inside[d] || !solvent[i + off[d]]) continue;
                    double xf = (ix + 0.5 * FACE_DX[d]) * g.h, yf = (iy + 0.5 * FACE_DY[d]) * g.h,
                           zf = (iz + 0.5 * FACE_DZ[d]) * g.h;
                    double gf = -coulomb_potential(ch, M, eps_m, xf, yf, zf);
                    double dn_star = FACE_SIGN[d] * coulomb_gradient(ch, M, eps_m, xf, yf, zf, FACE_AXIS[d]);
                    double dn_L = 2.0 * (gf - phiL[i]) / g.h;
                    J[(d - 1) * N + i] = eps[i] * (dn_star + dn_L);
                }
            }
}

// b^IF from the jumps: every node gathers the faces it shares with a node of the other kind, d = 1..6.
void interface_rhs(const Grid& g, const double* eps, const uint8_t* solvent, const double* J, double* b) {
    const int64_t N = g.n();
    const int64_t off[7] = {0, 1, -1, -(int64_t)g.nx, (int64_t)g.nx, -(int64_t)g.nx * g.ny, (int64_t)g.nx * g.ny};
    const int opposite[7] = {0, 2, 1, 4, 3, 6, 5};
    for (int iz = 0; iz < g.nz; ++iz)
        for (int iy = 0; iy < g.ny; ++iy)
            for (int ix = 0; ix < g.nx; ++ix) {
                int64_t i = ix + (int64_t)g.nx * (iy + (int64_t)g.ny * iz);
                bool inside[7] = {true, ix + 1 < g.nx, ix - 1 >= 0, iy - 1 >= 0, iy + 1 < g.ny, iz - 1 >= 0, iz + 1 < g.nz};
                double acc = 0.0;
                for (int d = 1; d < 7; ++d) {
                    if (!inside[d]) continue;
                    int64_t j = i + off[d];
                    if (solvent[i] == solvent[j]) continue;
                    // the jump is stored at the Omega_m node of the pair
                    double Jf = solvent[i] ? J[(opposite[d] - 1) * N + j] : J[(d - 1) * N + i];
                    acc = acc + (-(eps[i] * Jf) / ((eps[i] + eps[j]) * g.h));
                }
                b[i] = acc;
            }
}

}  // namespace

// =========================================================================================
// C interface (ctypes).  All pointers are host pointers.
// =========================================================================================
extern "C" {

double pfo_kappa(void) { return kappa_angstrom(); }
double pfo_kT_over_e_volt(void) { return K_B * T_ABS / E_CH; }
double pfo_molar_to_per_A3(void) { return AVOGADRO_PER_A3; }

static Grid mk(int nx, int ny, int nz, double h, const int* bct, const double* bcv,
               const uint8_t* fix_mask = nullptr, const double* fix_val = nullptr) {
    Grid g; g.nx = nx; g.ny = ny; g.nz = nz; g.h = h;
    for (int f = 0; f < 6; ++f) { g.bc_type[f] = bct[f]; g.bc_value[f] = bcv[f]; }
    g.fix_mask = fix_mask; g.fix_val = fix_val;
    return g;
}

void pfo_assemble_poisson(int nx, int ny, int nz, double h, const int* bct, const double* bcv,
                          const double* eps, const double* sigma, double* A,
                          const uint8_t* fix_mask, const double* fix_val) {
    assemble_poisson(mk(nx, ny, nz, h, bct, bcv, fix_mask, fix_val), eps, sigma, A);
}

void pfo_assemble_pf1(int nx, int ny, int nz, double h, const int* bct, const double* bcv,
                      const double* eps, const uint8_t* solvent, double lc, double* A) {
    assemble_pf1(mk(nx, ny, nz, h, bct, bcv), eps, solvent, lc, A);
}

void pfo_solvent_mask(int64_t N, const double* eps, uint8_t* mask) { solvent_mask(N, eps, mask); }

void pfo_dia_spmv(int nx, int ny, int nz, const double* A, const double* x, double* y) {
    int t[6] = {0, 0, 0, 0, 0, 0}; double v[6] = {0, 0, 0, 0, 0, 0};
    dia_spmv(mk(nx, ny, nz, 1.0, t, v), A, x, y);
}

double pfo_dot(int64_t N, const double* a, const double* b) { return dot(N, a, b); }

void pfo_set_dirichlet(int nx, int ny, int nz, const int* bct, const double* bcv, double* x,
                       const uint8_t* fix_mask, const double* fix_val) {
    set_dirichlet(mk(nx, ny, nz, 1.0, bct, bcv, fix_mask, fix_val), x);
}

void pfo_deposit_charges(int nx, int ny, int nz, double h, const double* charges, int M, double* b) {
    int t[6] = {0, 0, 0, 0, 0, 0}; double v[6] = {0, 0, 0, 0, 0, 0};
    deposit_charges(mk(nx, ny, nz, h, t, v), charges, M, b);
}

int pfo_bicgstab(int nx, int ny, int nz, const double* A, const double* b, double* x, double tol,
                 int maxit, int precond, int* iters, double* relres, double* true_relres, double* hist,
                 int norm_mode) {
    int t[6] = {0, 0, 0, 0, 0, 0}; double v[6] = {0, 0, 0, 0, 0, 0};
    return bicgstab(mk(nx, ny, nz, 1.0, t, v), A, b, x, tol, maxit, precond, iters, relres, true_relres, hist,
                    norm_mode);
}

int pfo_bicgstab_merged(int nx, int ny, int nz, const double* A, const double* b, double* x, double tol,
                        int maxit, int precond, int* iters, double* relres, double* true_relres, double* hist,
                        int norm_mode, double* rho_rec, double* rho_direct) {
    int t[6] = {0, 0, 0, 0, 0, 0}; double v[6] = {0, 0, 0, 0, 0, 0};
    return bicgstab_merged(mk(nx, ny, nz, 1.0, t, v), A, b, x, tol, maxit, precond, iters, relres, true_relres, hist,
                           norm_mode, rho_rec, rho_direct);
}

// The library-level call the GPU path mirrors (pf_solve_linear): Poisson operator of the grid,
// Dirichlet values forced into rhs and x0 (Q4, Q20).
int pfo_solve_linear(int nx, int ny, int nz, double h, const int* bct, const double* bcv,
                     const double* eps, const double* sigma, const double* rhs, double* x,
                     double tol, int maxit, int precond, int* iters, double* relres,
                     double* true_relres, double* hist, int norm_mode,
                     const uint8_t* fix_mask, const double* fix_val, int solver /* 0 Table 3, 1 merged */) {
    Grid g = mk(nx, ny, nz, h, bct, bcv, fix_mask, fix_val);
    const int64_t N = g.n();
    std::vector<double> A(7 * N), b(rhs, rhs + N);
    assemble_poisson(g, eps, sigma, A.data());
    set_dirichlet(g, b.data());
    set_dirichlet(g, x);
    return krylov(solver, g, A.data(), b.data(), x, tol, maxit, precond, iters, relres, true_relres, hist, norm_mode);
}

int pfo_fermi_pointwise(int K, const double* valence, const double* bath_molar, const double* radii,
                        double water_molar, int64_t N, const double* phi, const uint8_t* solvent,
                        double* rho, double* sigma, double* S, double* conc, double* gammaB_out) {
    SpeciesTab sp;
    int rc = make_species(K, valence, bath_molar, radii, water_molar, sp);
    if (gammaB_out) *gammaB_out = sp.gammaB;
    if (rc) return rc;
    fermi_field(sp, N, phi, solvent, rho, sigma, S, conc);
    return 0;
}

// ---- R5: the outer loop, Table 2 steps 2-5 / Table 4 steps 4-7 ----
// Returns 0 converged, 1 max_outer reached, 2 converged on the increment although at least one linear solve stopped
// at lin_maxit, <0 error (-3: breakdown of a linear solve or a non-finite increment, D7).  lin_iters_hist (may be null) receives the
// BiCGSTAB iteration count of every linear solve in call order (initial guess, then PF1, PF2, ...),
// up to hist_cap entries; incr_hist the increment ||phi - phi0||_inf of every outer iteration.
int pfo_solve_pf(int nx, int ny, int nz, double h, const int* bct, const double* bcv,
                 const double* eps, const double* charges, int M,
                 int K, const double* valence, const double* bath_molar, const double* radii,
                 double water_molar, double lc, double tol, double omega_pf,
                 double lin_tol, int lin_maxit, int max_outer, int norm_mode,
                 double* phi /* out */, double* psi /* out or null */, double* conc /* out or null */,
                 double* steric /* out or null */,
                 int* outer_iters, int* linear_iters, int* lin_iters_hist, int hist_cap,
                 double* incr_hist, const double* fixed_override /* b^IF of the singular-charge model, or null */,
                 const uint8_t* fix_mask, const double* fix_val /* Omega_f, or null */,
                 int solver /* linear solver of every step: 0 Table 3, 1 merged */,
                 int steric_mode /* 0: Eq (1) solved simultaneously per node (Q11); 1: lagged (G1) */) {
    Grid g = mk(nx, ny, nz, h, bct, bcv, fix_mask, fix_val);
    const int64_t N = g.n();
    SpeciesTab sp;
    int rc = make_species(K, valence, bath_molar, radii, water_molar, sp);
    if (rc) return rc;
    std::vector<uint8_t> solv(N);
    solvent_mask(N, eps, solv.data());
    // F2, F3: in Omega_f neither Eq (1) nor PF1 applies: treat its nodes like non-solvent ones (C = rho = sigma = 0,
    // Psi = 0); their PF2 rows are the identity rows that assemble_poisson and set_dirichlet produce
    if (fix_mask) for (int64_t i = 0; i < N; ++i) if (fix_mask[i]) solv[i] = 0;
    std::vector<double> fixed(N, 0.0), A0(7 * N), A1(7 * N), A2(7 * N), b(N);
    std::vector<double> phi0(N, 0.0), Psi(N, 0.0), ph(N), rho(N), sigma(N), S(N), Slag(steric_mode == 1 ? N : 0, 0.0);
    if (fixed_override) std::memcpy(fixed.data(), fixed_override, N * sizeof(double));
    else deposit_charges(g, charges, M, fixed.data());
    int nsolve = 0, total = 0, its = 0;
    double rr, tr;
    bool inner_maxit = false;     // a linear solve stopped at lin_maxit (status 1): its last iterate is used as it stands
    auto record = [&](int n) { if (lin_iters_hist && nsolve < hist_cap) lin_iters_hist[nsolve] = n; ++nsolve; total += n; };
    // step 2 / 4: initial guess, PF2 with rho' = Psi = 0
    assemble_poisson(g, eps, nullptr, A0.data());
    b = fixed; set_dirichlet(g, b.data());
    set_dirichlet(g, phi0.data());
    rc = krylov(solver, g, A0.data(), b.data(), phi0.data(), lin_tol, lin_maxit, 1, &its, &rr, &tr, nullptr, norm_mode);
    record(its);
    if (rc < 0) return rc;
    inner_maxit |= rc == 1;
    assemble_pf1(g, eps, solv.data(), lc, A1.data());
    int status = 1, outer = 0;
    while (outer < max_outer) {
        ++outer;
        if (steric_mode == 1) fermi_field_lagged(sp, N, phi0.data(), solv.data(), Slag.data(), true, rho.data(), sigma.data(), nullptr);
        else fermi_field(sp, N, phi0.data(), solv.data(), rho.data(), sigma.data(), S.data(), nullptr);
        // step 3 / 5: PF1 -> Psi (warm start: previous Psi)
        rhs_pf1(g, solv.data(), rho.data(), b.data());
        rc = krylov(solver, g, A1.data(), b.data(), Psi.data(), lin_tol, lin_maxit, 1, &its, &rr, &tr, nullptr, norm_mode);
        record(its);
        if (rc < 0) return rc;
        inner_maxit |= rc == 1;
        // step 4 / 6: PF2 -> phi (warm start: phi0)
        assemble_poisson(g, eps, sigma.data(), A2.data());
        rhs_pf2(g, eps, solv.data(), Psi.data(), sigma.data(), phi0.data(), fixed.data(), b.data());
        ph = phi0;
        rc = krylov(solver, g, A2.data(), b.data(), ph.data(), lin_tol, lin_maxit, 1, &its, &rr, &tr, nullptr, norm_mode);
        record(its);
        if (rc < 0) return rc;
        inner_maxit |= rc == 1;
        // step 5 / 7: relax, then test the increment (Q8, Q9)
        for (int64_t i = 0; i < N; ++i) ph[i] = omega_pf * phi0[i] + (1.0 - omega_pf) * ph[i];
        for (int64_t i = 0; i < N; ++i) b[i] = ph[i] - phi0[i];
        double d = norm_inf(N, b.data());
        if (incr_hist) incr_hist[outer - 1] = d;
        if (!std::isfinite(d)) return -3;                  // D7: a NaN fails "d > tol" and would read as converged
        phi0 = ph;
        if (!(d > tol)) { status = 0; break; }
    }
    std::memcpy(phi, phi0.data(), N * sizeof(double));
    if (psi) std::memcpy(psi, Psi.data(), N * sizeof(double));
    if (steric_mode == 1) {          // the fields that belong to the state: C_k from the final phi and the S at hand
        if (conc) fermi_field_lagged(sp, N, phi0.data(), solv.data(), Slag.data(), false, nullptr, nullptr, conc);
        if (steric) std::memcpy(steric, Slag.data(), N * sizeof(double));
    } else if (conc || steric) fermi_field(sp, N, phi0.data(), solv.data(), nullptr, nullptr, steric, conc);
    *outer_iters = outer;
    *linear_iters = total;
    if (status == 0 && inner_maxit) return 2;    // converged on the increment, but an inner solve was cut off
    return status;
}

// Fixed-point residuals of the split system at given (phi, Psi): PF1 with rho(phi) and PF2 with
// phi0 = phi, both relative to their right-hand sides.  Used for the any-size property check.
int pfo_pf_residuals(int nx, int ny, int nz, double h, const int* bct, const double* bcv,
                     const double* eps, const double* charges, int M,
                     int K, const double* valence, const double* bath_molar, const double* radii,
                     double water_molar, double lc, const double* phi, const double* psi,
                     double* res_pf1, double* res_pf2) {
    Grid g = mk(nx, ny, nz, h, bct, bcv);
    const int64_t N = g.n();
    SpeciesTab sp;
    int rc = make_species(K, valence, bath_molar, radii, water_molar, sp);
    if (rc) return rc;
    std::vector<uint8_t> solv(N);
    solvent_mask(N, eps, solv.data());
    std::vector<double> fixed(N, 0.0), A(7 * N), b(N), y(N), rho(N), sigma(N), S(N);
    deposit_charges(g, charges, M, fixed.data());
    fermi_field(sp, N, phi, solv.data(), rho.data(), sigma.data(), S.data(), nullptr);
    assemble_pf1(g, eps, solv.data(), lc, A.data());
    rhs_pf1(g, solv.data(), rho.data(), b.data());
    dia_spmv(g, A.data(), psi, y.data());
    for (int64_t i = 0; i < N; ++i) y[i] = b[i] - y[i];
    double bn = norm2(N, b.data());
    *res_pf1 = bn > 0 ? norm2(N, y.data()) / bn : norm2(N, y.data());
    assemble_poisson(g, eps, sigma.data(), A.data());
    rhs_pf2(g, eps, solv.data(), psi, sigma.data(), phi, fixed.data(), b.data());
    dia_spmv(g, A.data(), phi, y.data());
    for (int64_t i = 0; i < N; ++i) y[i] = b[i] - y[i];
    bn = norm2(N, b.data());
    *res_pf2 = bn > 0 ? norm2(N, y.data()) / bn : norm2(N, y.data());
    return 0;
}

// ---- singular-charge decomposition (see the block comment above assemble_laplace_m) -----------------
double pfo_coulomb_potential(const double* charges, int M, double eps_m, double x, double y, double z) {
    return coulomb_potential(charges, M, eps_m, x, y, z);
}

double pfo_coulomb_gradient(const double* charges, int M, double eps_m, double x, double y, double z, int axis) {
    return coulomb_gradient(charges, M, eps_m, x, y, z, axis);
}

void pfo_interface_rhs(int nx, int ny, int nz, double h, const double* eps, const uint8_t* solvent,
                       const double* J, double* b) {
    int t[6] = {0, 0, 0, 0, 0, 0}; double v[6] = {0, 0, 0, 0, 0, 0};
    interface_rhs(mk(nx, ny, nz, h, t, v), eps, solvent, J, b);
}

// Everything that precedes the PF loop in Table 2 step 1 / Table 4 steps 2-3:
// phi* on the Omega_m nodes, the Laplace solve for phi^L, the flux jumps and b^IF.
// eps_m = the smallest eps of the map (S4).  Returns the status of the Laplace solve.
int pfo_singular_setup(int nx, int ny, int nz, double h, const double* eps, const double* charges, int M,
                       double lin_tol, int lin_maxit,
                       double* phiL /* N */, double* phistar /* N, 0 on Omega_s */, double* bIF /* N */,
                       double* Jout /* 6N or null */, int* laplace_iters) {
    int t[6] = {0, 0, 0, 0, 0, 0}; double v[6] = {0, 0, 0, 0, 0, 0};
    Grid g = mk(nx, ny, nz, h, t, v);
    const int64_t N = g.n();
    std::vector<uint8_t> solv(N);
    solvent_mask(N, eps, solv.data());
    double eps_m = eps[0];
    for (int64_t i = 1; i < N; ++i) eps_m = std::min(eps_m, eps[i]);
    std::vector<double> A(7 * N), b(N), J(6 * N);
    assemble_laplace_m(g, solv.data(), charges, M, eps_m, A.data(), b.data());
    // initial guess: the prescribed values on identity rows, 0 elsewhere (the Krylov vectors then vanish there)
    for (int64_t i = 0; i < N; ++i) phiL[i] = (A[i] == 1.0 && A[1 * N + i] == 0.0 && A[2 * N + i] == 0.0 &&
                                               A[3 * N + i] == 0.0 && A[4 * N + i] == 0.0 && A[5 * N + i] == 0.0 &&
                                               A[6 * N + i] == 0.0) ? b[i] : 0.0;
    double rr, tr;
    int rc = bicgstab(g, A.data(), b.data(), phiL, lin_tol, lin_maxit, 1, laplace_iters, &rr, &tr, nullptr);
    if (rc < 0) return rc;
    for (int iz = 0; iz < nz; ++iz)
        for (int iy = 0; iy < ny; ++iy)
            for (int ix = 0; ix < nx; ++ix) {
                int64_t i = ix + (int64_t)nx * (iy + (int64_t)ny * iz);
                phistar[i] = solv[i] ? 0.0 : coulomb_potential(charges, M, eps_m, ix * h, iy * h, iz * h);
            }
    face_jumps(g, eps, solv.data(), charges, M, eps_m, phiL, J.data());
    interface_rhs(g, eps, solv.data(), J.data(), bIF);
    if (Jout) std::memcpy(Jout, J.data(), 6 * N * sizeof(double));
    return rc;
}

// ---- dense LU with partial pivoting (pin for the 8^3 case; no LAPACK) --------------------
void pfo_dia_to_dense(int nx, int ny, int nz, const double* A, double* dense /* N*N row-major */) {
    const int64_t N = (int64_t)nx * ny * nz;
    const int64_t off[7] = {0, 1, -1, -(int64_t)nx, (int64_t)nx, -(int64_t)nx * ny, (int64_t)nx * ny};
    std::fill(dense, dense + N * N, 0.0);
    for (int64_t i = 0; i < N; ++i)
        for (int d = 0; d < 7; ++d) {
            int64_t j = i + off[d];
            double a = A[d * N + i];
            if (a != 0.0 && j >= 0 && j < N) dense[i * N + j] = a;
        }
}

int pfo_dense_lu_solve(int64_t n, double* a /* n*n row-major, destroyed */, const double* b, double* x) {
    std::vector<int64_t> piv(n);
    std::vector<double> y(b, b + n);
    for (int64_t k = 0; k < n; ++k) {
        int64_t p = k; double best = std::fabs(a[k * n + k]);
        for (int64_t i = k + 1; i < n; ++i)
            if (std::fabs(a[i * n + k]) > best) { best = std::fabs(a[i * n + k]); p = i; }
        if (best == 0.0) return -1;
        if (p != k) {
            for (int64_t j = 0; j < n; ++j) std::swap(a[k * n + j], a[p * n + j]);
            std::swap(y[k], y[p]);
        }
        for (int64_t i = k + 1; i < n; ++i) {
            double m = a[i * n + k] / a[k * n + k];
            if (m == 0.0) continue;
            a[i * n + k] = m;
            for (int64_t j = k + 1; j < n; ++j) a[i * n + j] -= m * a[k * n + j];
            y[i] -= m * y[k];
        }
    }
    for (int64_t i = n - 1; i >= 0; --i) {
        double s = y[i];
        for (int64_t j = i + 1; j < n; ++j) s -= a[i * n + j] * x[j];
        x[i] = s / a[i * n + i];
    }
    return 0;
}

}  // extern "C"
