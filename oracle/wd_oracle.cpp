// wd_oracle.cpp -- TEST INFRASTRUCTURE ONLY.  Plain, slow, fp64 CPU oracle for the hot path of
// arxiv/paper_1009_5169 (blocked quark solve D X = Phi, D^dag Y = X, force F_mu += f[x_i, y_i];
// PAPER.md:51-58 Algorithm 2, eq. 2.3).
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
// load this.  It shares no code with the CUDA path under paper_1009_5169_b200/ and is never used by
// it.  Every function works on the CANONICAL layouts documented in wd_inputs/__init__.py:
//   gauge   double [mu=4][T][Lz][Ly][Lx][3][3][2]     spinor  double [n_rhs][T][Lz][Ly][Lx][4][3][2]
//   force   double [mu=4][T][Lz][Ly][Lx][3][3][2]
//
// The paper does not write down the operator, the gamma basis, the SF boundary treatment or the
// force functional; the readings used are those of SURVEY.md §8(c.1)/(c.5), restated in DESIGN.md:
//   D = 1 - kappa H,
//   (H psi)(x) = sum_mu [ (1 - gamma_mu) U_mu(x) psi(x+mu) + (1 + gamma_mu) U_mu(x-mu)^dag psi(x-mu) ]
//   D^dag: gamma_mu -> -gamma_mu  (== gamma5 D gamma5)
//   SF: T slices stored, psi(t=0) = psi(t=T) = 0, D_SF = P (1 - kappa H) P, P = projector on t >= 1
//   F_mu(x) = sum_i 2 kappa TA[ U_mu(x) W^(i)_mu(x) ],
//   W = sum_spin [ x(x+mu) (x) ((1-gamma_mu) y(x))^dag + ((1+gamma_mu) y(x+mu)) (x) x(x)^dag ]
//   TA(M) = (M - M^dag)/2 - tr(M - M^dag)/6
// No even/odd split, no mixed precision, no half-spinor tricks: the definition written out.
//
// Pins (tests/test_oracle_pins.py, all -m "not gpu"): free-field and twisted-abelian closed forms,
// gamma5-hermiticity, gauge covariance, Gamma D Gamma = 2 - D, SF boundary-link independence,
// dense LU inverse on 2^3x4, finite-difference derivative of S = sum |D^-1 phi|^2 for the force.
// Parity with values printed in the paper: unpinned -- the paper prints no worked example.
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef std::complex<double> cplx;

namespace {

const cplx I_(0.0, 1.0);

// Chiral gamma basis, SURVEY.md Appendix A.  GAMMA[mu][row][col], mu = x,y,z,t.
const cplx GAMMA[4][4][4] = {
    {{0, 0, 0, -I_}, {0, 0, -I_, 0}, {0, I_, 0, 0}, {I_, 0, 0, 0}},
    {{0, 0, 0, -1}, {0, 0, 1, 0}, {0, 1, 0, 0}, {-1, 0, 0, 0}},
    {{0, 0, -I_, 0}, {0, 0, 0, I_}, {I_, 0, 0, 0}, {0, -I_, 0, 0}},
    {{0, 0, 1, 0}, {0, 0, 0, 1}, {1, 0, 0, 0}, {0, 1, 0, 0}},
};

struct Lattice {
    int L[4];   // Lx, Ly, Lz, T
    long V;
    int bc;     // 0 periodic, 1 SF
    long idx(const int c[4]) const { return c[0] + (long)L[0] * (c[1] + (long)L[1] * (c[2] + (long)L[2] * c[3])); }
    void coords(long s, int c[4]) const {
        c[0] = (int)(s % L[0]); s /= L[0];
        c[1] = (int)(s % L[1]); s /= L[1];
        c[2] = (int)(s % L[2]); s /= L[2];
        c[3] = (int)s;
    }
    // neighbour in direction mu, step +1/-1.  Returns -1 if the neighbour is a zero SF slice
    // (t = 0 stored slice or the virtual t = T slice).
    long nbr(long s, int mu, int step) const {
        int c[4]; coords(s, c);
        c[mu] += step;
        if (c[mu] >= L[mu]) { if (mu == 3 && bc == 1) return -1; c[mu] -= L[mu]; }
        if (c[mu] < 0)      { if (mu == 3 && bc == 1) return -1; c[mu] += L[mu]; }
        if (bc == 1 && c[3] == 0) return -1;
        return idx(c);
    }
    bool dynamical(long s) const { return !(bc == 1 && s < V / L[3]); }   // t >= 1 in SF mode
};

bool make_lattice(const int dims[4], int bc, Lattice& lat) {
    lat.V = 1;
    for (int i = 0; i < 4; ++i) { if (dims[i] < 1) return false; lat.L[i] = dims[i]; lat.V *= dims[i]; }
    if (bc != 0 && bc != 1) return false;
    lat.bc = bc;
    return true;
}

inline const cplx* link(const double* U, const Lattice& lat, int mu, long s) {
    return reinterpret_cast<const cplx*>(U) + ((long)mu * lat.V + s) * 9;
}

// out = D psi (dag = 0) or D^dag psi (dag = 1) for ONE right-hand side; SURVEY.md §8(c.3).
void apply_one(const Lattice& lat, double kappa, int dag, const double* U, const cplx* psi, cplx* out) {
    const double sg = dag ? -1.0 : 1.0;
#pragma omp parallel for schedule(static)
    for (long s = 0; s < lat.V; ++s) {
        cplx* o = out + s * 12;
        if (!lat.dynamical(s)) { for (int k = 0; k < 12; ++k) o[k] = 0.0; continue; }
        cplx sum[4][3];
        for (int a = 0; a < 4; ++a) for (int c = 0; c < 3; ++c) sum[a][c] = 0.0;
        for (int mu = 0; mu < 4; ++mu) {
            cplx f[4][3], b[4][3];
            const long nf = lat.nbr(s, mu, +1), nb = lat.nbr(s, mu, -1);
            // f = U_mu(x) psi(x+mu)
            if (nf >= 0) {
                const cplx* u = link(U, lat, mu, s);
                const cplx* p = psi + nf * 12;
                for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
                    cplx acc = 0.0;
                    for (int c = 0; c < 3; ++c) acc += u[a * 3 + c] * p[sp * 3 + c];
                    f[sp][a] = acc;
                }
            } else for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) f[sp][a] = 0.0;
            // b = U_mu(x-mu)^dag psi(x-mu)
            if (nb >= 0) {
                const cplx* u = link(U, lat, mu, nb);
                const cplx* p = psi + nb * 12;
                for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) {
                    cplx acc = 0.0;
                    for (int c = 0; c < 3; ++c) acc += std::conj(u[c * 3 + a]) * p[sp * 3 + c];
                    b[sp][a] = acc;
                }
            } else for (int sp = 0; sp < 4; ++sp) for (int a = 0; a < 3; ++a) b[sp][a] = 0.0;
            // sum += (1 - sg gamma_mu) f + (1 + sg gamma_mu) b
            for (int r = 0; r < 4; ++r) for (int a = 0; a < 3; ++a) {
                cplx acc = f[r][a] + b[r][a];
                for (int q = 0; q < 4; ++q) acc += sg * GAMMA[mu][r][q] * (b[q][a] - f[q][a]);
                sum[r][a] += acc;
            }
        }
        const cplx* p0 = psi + s * 12;
        for (int r = 0; r < 4; ++r) for (int a = 0; a < 3; ++a) o[r * 3 + a] = p0[r * 3 + a] - kappa * sum[r][a];
    }
}

cplx dot(long n, const cplx* a, const cplx* b) {   // <a,b> = sum conj(a) b
    double re = 0.0, im = 0.0;
#pragma omp parallel for reduction(+ : re, im) schedule(static)
    for (long i = 0; i < n; ++i) { cplx t = std::conj(a[i]) * b[i]; re += t.real(); im += t.imag(); }
    return cplx(re, im);
}
double norm2(long n, const cplx* a) { return dot(n, a, a).real(); }

// Textbook BiCGStab (SURVEY.md Appendix B.1 for one column), unpreconditioned, full lattice, zero
// start, shadow residual = r0.  Returns iterations, or -1 on breakdown.
int bicgstab_one(const Lattice& lat, double kappa, int dag, const double* U, const cplx* b, cplx* x,
                 double tol, int max_iter) {
    const long n = lat.V * 12;
    std::vector<cplx> r(b, b + n), rt(b, b + n), p(n, 0.0), v(n, 0.0), s(n), t(n);
    for (long i = 0; i < n; ++i) x[i] = 0.0;
    const double bn = std::sqrt(norm2(n, b));
    if (bn == 0.0) return 0;
    cplx rho = 1.0, alpha = 1.0, omega = 1.0;
    for (int it = 1; it <= max_iter; ++it) {
        cplx rho1 = dot(n, rt.data(), r.data());
        if (std::abs(rho1) == 0.0 || std::abs(omega) == 0.0) return -1;
        cplx beta = (rho1 / rho) * (alpha / omega);
        rho = rho1;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) p[i] = r[i] + beta * (p[i] - omega * v[i]);
        apply_one(lat, kappa, dag, U, p.data(), v.data());
        cplx sigma = dot(n, rt.data(), v.data());
        if (std::abs(sigma) == 0.0) return -1;
        alpha = rho / sigma;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) s[i] = r[i] - alpha * v[i];
        apply_one(lat, kappa, dag, U, s.data(), t.data());
        double tt = norm2(n, t.data());
        if (tt == 0.0) {   // s == 0: exact solution
#pragma omp parallel for schedule(static)
            for (long i = 0; i < n; ++i) x[i] += alpha * p[i];
            return it;
        }
        omega = dot(n, t.data(), s.data()) / tt;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) { x[i] += alpha * p[i] + omega * s[i]; r[i] = s[i] - omega * t[i]; }
        if (std::sqrt(norm2(n, r.data())) <= tol * bn) return it;
        if (!std::isfinite(norm2(n, r.data()))) return -1;
    }
    return max_iter + 1;
}

// CG on the normal equations A^dag A x = A^dag b; the fallback of SURVEY.md §8(c.4).
int cgne_one(const Lattice& lat, double kappa, int dag, const double* U, const cplx* b, cplx* x,
             double tol, int max_iter) {
    const long n = lat.V * 12;
    std::vector<cplx> r(n), p(n), q(n), w(n), res(b, b + n);
    for (long i = 0; i < n; ++i) x[i] = 0.0;
    const double bn = std::sqrt(norm2(n, b));
    if (bn == 0.0) return 0;
    apply_one(lat, kappa, !dag, U, b, r.data());   // r = A^dag b
    p = r;
    double rr = norm2(n, r.data());
    for (int it = 1; it <= max_iter; ++it) {
        apply_one(lat, kappa, dag, U, p.data(), q.data());      // q = A p
        double a = rr / norm2(n, q.data());
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) { x[i] += a * p[i]; res[i] -= a * q[i]; }
        if (std::sqrt(norm2(n, res.data())) <= tol * bn) return it;
        apply_one(lat, kappa, !dag, U, q.data(), w.data());     // w = A^dag A p
        double rr1 = 0.0;
#pragma omp parallel for reduction(+ : rr1) schedule(static)
        for (long i = 0; i < n; ++i) { r[i] -= a * w[i]; rr1 += std::norm(r[i]); }
        double be = rr1 / rr; rr = rr1;
#pragma omp parallel for schedule(static)
        for (long i = 0; i < n; ++i) p[i] = r[i] + be * p[i];
    }
    return max_iter + 1;
}

}  // namespace

extern "C" {

int orc_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

// gamma_mu (mu = 0..3) or gamma5 = gamma_x gamma_y gamma_z gamma_t (mu = 4) as [4][4][2] doubles.
int orc_gamma(int mu, double* out) {
    cplx g[4][4];
    if (mu >= 0 && mu < 4) {
        for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) g[r][c] = GAMMA[mu][r][c];
    } else if (mu == 4) {
        cplx a[4][4], b[4][4];
        for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) a[r][c] = GAMMA[0][r][c];
        for (int m = 1; m < 4; ++m) {
            for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) {
                b[r][c] = 0.0;
                for (int k = 0; k < 4; ++k) b[r][c] += a[r][k] * GAMMA[m][k][c];
            }
            std::memcpy(a, b, sizeof(a));
        }
        std::memcpy(g, a, sizeof(g));
    } else return -1;
    for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) { out[(r * 4 + c) * 2] = g[r][c].real(); out[(r * 4 + c) * 2 + 1] = g[r][c].imag(); }
    return 0;
}

// out = D in (dag=0) / D^dag in (dag=1), n_rhs columns.
int orc_apply(const int dims[4], double kappa, int bc, int dag, int n_rhs, const double* U,
              const double* in, double* out) {
    Lattice lat;
    if (!make_lattice(dims, bc, lat) || n_rhs < 0) return -1;
    for (int r = 0; r < n_rhs; ++r)
        apply_one(lat, kappa, dag, U, reinterpret_cast<const cplx*>(in) + (long)r * lat.V * 12,
                  reinterpret_cast<cplx*>(out) + (long)r * lat.V * 12);
    return 0;
}

// Solve D X = B (dag=0) or D^dag X = B (dag=1) column by column.  SURVEY.md §8(c.4): fp64
// BiCGStab to a recursive residual `tol`, then the TRUE residual |b - A x| / |b| is recomputed
// and written to relres[r]; CG on the normal equations if BiCGStab breaks down or stalls.
// iters[r] = iterations used (BiCGStab count, or 100000 + CGNE count).  Returns 0 when every
// true residual is <= 10*tol, else 1.
int orc_solve(const int dims[4], double kappa, int bc, int dag, int n_rhs, const double* U,
              const double* B, double* X, double tol, int max_iter, double* relres, int* iters) {
    Lattice lat;
    if (!make_lattice(dims, bc, lat) || n_rhs < 0) return -1;
    const long n = lat.V * 12;
    int rc = 0;
    std::vector<cplx> ax(n);
    for (int r = 0; r < n_rhs; ++r) {
        const cplx* b = reinterpret_cast<const cplx*>(B) + (long)r * n;
        cplx* x = reinterpret_cast<cplx*>(X) + (long)r * n;
        int it = bicgstab_one(lat, kappa, dag, U, b, x, tol, max_iter);
        auto true_res = [&]() {
            apply_one(lat, kappa, dag, U, x, ax.data());
            double num = 0.0;
            for (long i = 0; i < n; ++i) num += std::norm(b[i] - ax[i]);
            double bn = norm2(n, b);
            return bn > 0.0 ? std::sqrt(num / bn) : 0.0;
        };
        double rr = true_res();
        if (it < 0 || it > max_iter || !(rr <= 10 * tol)) {
            it = 100000 + cgne_one(lat, kappa, dag, U, b, x, tol, 20 * max_iter);
            rr = true_res();
        }
        if (relres) relres[r] = rr;
        if (iters) iters[r] = it;
        if (!(rr <= 10 * tol)) rc = 1;
    }
    return rc;
}

// The fallback route of orc_solve on its own (SURVEY.md §8(c.4) "fall back to CG on D^dag D x = D^dag phi"), exported so
// that tests can pin it: same arguments and outputs as orc_solve, iters[r] = CG iterations.  (Export only: cgne_one is
// unchanged.)
int orc_solve_cgne(const int dims[4], double kappa, int bc, int dag, int n_rhs, const double* U,
                   const double* B, double* X, double tol, int max_iter, double* relres, int* iters) {
    Lattice lat;
    if (!make_lattice(dims, bc, lat) || n_rhs < 0) return -1;
    const long n = lat.V * 12;
    int rc = 0;
    std::vector<cplx> ax(n);
    for (int r = 0; r < n_rhs; ++r) {
        const cplx* b = reinterpret_cast<const cplx*>(B) + (long)r * n;
        cplx* x = reinterpret_cast<cplx*>(X) + (long)r * n;
        const int it = cgne_one(lat, kappa, dag, U, b, x, tol, max_iter);
        apply_one(lat, kappa, dag, U, x, ax.data());
        double num = 0.0;
        for (long i = 0; i < n; ++i) num += std::norm(b[i] - ax[i]);
        const double bn = norm2(n, b);
        const double rr = bn > 0.0 ? std::sqrt(num / bn) : 0.0;
        if (relres) relres[r] = rr;
        if (iters) iters[r] = it;
        if (!(rr <= 10 * tol)) rc = 1;
    }
    return rc;
}

// out = P_parity in: keeps the sites with (x+y+z+t) mod 2 == parity, zero elsewhere (the even/odd-
// preconditioned-action variant has phi on even sites only).  in == out is allowed.
int orc_project_parity(const int dims[4], int parity, int n_rhs, const double* in, double* out) {
    if (parity != 0 && parity != 1) return -1;
    const long Lx = dims[0], Ly = dims[1], Lz = dims[2], Lt = dims[3], V = Lx * Ly * Lz * Lt;
    for (int r = 0; r < n_rhs; ++r)
        for (long t = 0; t < Lt; ++t) for (long z = 0; z < Lz; ++z) for (long y = 0; y < Ly; ++y) for (long x = 0; x < Lx; ++x) {
            const long s = x + Lx * (y + Ly * (z + Lz * t));
            const bool keep = ((x + y + z + t) & 1) == parity;
            for (int k = 0; k < 24; ++k) out[((long)r * V + s) * 24 + k] = keep ? in[((long)r * V + s) * 24 + k] : 0.0;
        }
    return 0;
}

// F += sum_i 2 kappa TA[ U_mu(x) W^(i)_mu(x) ]   ("F = F + f[x_i,y_i]").
int orc_force(const int dims[4], double kappa, int bc, int n_rhs, const double* U, const double* X,
              const double* Y, double* F) {
    Lattice lat;
    if (!make_lattice(dims, bc, lat) || n_rhs < 0) return -1;
    const long n = lat.V * 12;
    cplx* Fc = reinterpret_cast<cplx*>(F);
    for (int mu = 0; mu < 4; ++mu) {
#pragma omp parallel for schedule(static)
        for (long s = 0; s < lat.V; ++s) {
            if (!lat.dynamical(s)) continue;              // x(s) = y(s) = 0 and so is W
            const long nf = lat.nbr(s, mu, +1);
            if (nf < 0) continue;                         // x(s+mu) = y(s+mu) = 0
            cplx W[3][3];
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) W[a][b] = 0.0;
            for (int i = 0; i < n_rhs; ++i) {
                const cplx* x0 = reinterpret_cast<const cplx*>(X) + (long)i * n + s * 12;
                const cplx* y0 = reinterpret_cast<const cplx*>(Y) + (long)i * n + s * 12;
                const cplx* x1 = reinterpret_cast<const cplx*>(X) + (long)i * n + nf * 12;
                const cplx* y1 = reinterpret_cast<const cplx*>(Y) + (long)i * n + nf * 12;
                cplx pm[4][3], pp[4][3];   // (1 - gamma_mu) y(x),  (1 + gamma_mu) y(x+mu)
                for (int r = 0; r < 4; ++r) for (int a = 0; a < 3; ++a) {
                    cplx m = y0[r * 3 + a], p = y1[r * 3 + a];
                    for (int q = 0; q < 4; ++q) { m -= GAMMA[mu][r][q] * y0[q * 3 + a]; p += GAMMA[mu][r][q] * y1[q * 3 + a]; }
                    pm[r][a] = m; pp[r][a] = p;
                }
                for (int r = 0; r < 4; ++r) for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
                    W[a][b] += x1[r * 3 + a] * std::conj(pm[r][b]) + pp[r][a] * std::conj(x0[r * 3 + b]);
            }
            const cplx* u = link(U, lat, mu, s);
            cplx M[3][3];
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
                cplx acc = 0.0;
                for (int c = 0; c < 3; ++c) acc += u[a * 3 + c] * W[c][b];
                M[a][b] = acc;
            }
            cplx tr = 0.0;
            for (int a = 0; a < 3; ++a) tr += M[a][a] - std::conj(M[a][a]);
            cplx* f = Fc + ((long)mu * lat.V + s) * 9;
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) {
                cplx ta = 0.5 * (M[a][b] - std::conj(M[b][a]));
                if (a == b) ta -= tr / 6.0;
                f[a * 3 + b] += 2.0 * kappa * ta;
            }
        }
    }
    return 0;
}

// Number of dynamical unknowns: 12 * (sites with t >= 1 in SF mode, all sites otherwise).
long orc_dense_dim(const int dims[4], int bc) {
    Lattice lat;
    if (!make_lattice(dims, bc, lat)) return -1;
    long ns = 0;
    for (long s = 0; s < lat.V; ++s) ns += lat.dynamical(s) ? 1 : 0;
    return ns * 12;
}

// Assemble the dynamical block of D (or D^dag) column by column by applying it to unit vectors.
// A is [N][N][2] row-major; unknown index = 12 * (rank of the site among dynamical sites) + spin*3+colour.
int orc_dense_matrix(const int dims[4], double kappa, int bc, int dag, const double* U, double* A) {
    Lattice lat;
    if (!make_lattice(dims, bc, lat)) return -1;
    std::vector<long> sites;
    for (long s = 0; s < lat.V; ++s) if (lat.dynamical(s)) sites.push_back(s);
    const long N = (long)sites.size() * 12;
    std::vector<cplx> e(lat.V * 12, 0.0), col(lat.V * 12);
    cplx* Ac = reinterpret_cast<cplx*>(A);
    for (long j = 0; j < N; ++j) {
        const long src = sites[j / 12] * 12 + j % 12;
        e[src] = 1.0;
        apply_one(lat, kappa, dag, U, e.data(), col.data());
        e[src] = 0.0;
        for (long i = 0; i < N; ++i) Ac[i * N + j] = col[sites[i / 12] * 12 + i % 12];
    }
    return 0;
}

// Hand-written LU with partial pivoting; solves A x = b for nrhs columns in place.
// A [N][N][2] row-major (destroyed), b [nrhs][N][2].  Returns 0, or 1 if singular.
int orc_lu_solve(long N, double* A, double* b, int nrhs) {
    cplx* a = reinterpret_cast<cplx*>(A);
    cplx* rhs = reinterpret_cast<cplx*>(b);
    std::vector<long> piv(N);
    for (long k = 0; k < N; ++k) {
        long p = k; double best = std::abs(a[k * N + k]);
        for (long i = k + 1; i < N; ++i) { double v = std::abs(a[i * N + k]); if (v > best) { best = v; p = i; } }
        if (best == 0.0) return 1;
        piv[k] = p;
        if (p != k) {
            for (long j = 0; j < N; ++j) std::swap(a[k * N + j], a[p * N + j]);
            for (int r = 0; r < nrhs; ++r) std::swap(rhs[(long)r * N + k], rhs[(long)r * N + p]);
        }
        const cplx inv = 1.0 / a[k * N + k];
#pragma omp parallel for schedule(static)
        for (long i = k + 1; i < N; ++i) {
            const cplx l = a[i * N + k] * inv;
            if (l == 0.0) continue;
            a[i * N + k] = l;
            for (long j = k + 1; j < N; ++j) a[i * N + j] -= l * a[k * N + j];
            for (int r = 0; r < nrhs; ++r) rhs[(long)r * N + i] -= l * rhs[(long)r * N + k];
        }
    }
    for (int r = 0; r < nrhs; ++r) {
        cplx* x = rhs + (long)r * N;
        for (long i = N - 1; i >= 0; --i) {
            cplx acc = x[i];
            for (long j = i + 1; j < N; ++j) acc -= a[i * N + j] * x[j];
            x[i] = acc / a[i * N + i];
        }
    }
    return 0;
}

}  // extern "C"
