/*
 * vog_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, double-precision CPU oracle for the hot path of the 1Dx1D
 * semi-Lagrangian Vlasov-Poisson solver of "Vlasov on GPU (VOG project)"
 * (arXiv 1301.5892; PAPER.md, cited below as P:<line>).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant with the CUDA path in paper_1301_5892_b200/csrc/.
 *
 * What it computes, and how:
 *   - every constant advection is the product u' = A u of the circulant
 *     interpolation matrix A = C(a_0..a_{N-1}) of P:98-100 eq (4) with the
 *     periodic line u, applied DIRECTLY (stencil form, or a dense N x N
 *     matrix for small N) -- there is NO FFT in any advection here;
 *   - Lagrange 2d+1 weights are the product formula of P:115;
 *   - the cubic spline follows P:117-129 literally: B_0^3 by the recurrence
 *     of P:121, A = M x C(0,..,0,B(x_1),B(x_2),B(x_3))^{-1}, with M from P:129;
 *   - rho is the plain sum over v, made zero-mean as in P:205-211;
 *   - E is the Fourier solve of P:221 written as two naive O(Nx^2) DFT sums
 *     (mode 0 set to 0; Nyquist mode set to 0, reading Q12);
 *   - delta-f source of P:197 as a plain difference of two evaluations;
 *   - Strang step in the order stated in DESIGN.md reading Q1.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): integer shifts are
 * exact permutations; a Fourier mode is multiplied by the closed-form symbol;
 * dense A equals U diag(FFT(a)) U^* / N for N <= 16; LAG1 is linear
 * interpolation; Lagrange reproduces polynomials; the spline equals scipy's
 * periodic CubicSpline; mass conservation; v-advection keeps rho; E of
 * cos(kx) is sin(kx)/k; Landau damping rate 0.1533.
 * Unpinned: long-time bump-on-tail / KEEN trajectories ("parity unpinned"
 * beyond per-step parity).
 *
 * Layout: f is row-major [Nv][Nx], f[j*Nx+i] = value at (x_i, v_j).
 * Build: gcc -O2 -fopenmp -shared -fPIC -o libvog_oracle.so vog_oracle.c -lm
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_LAGRANGE 0
#define ORACLE_BSPLINE 1

typedef struct {
    int n;            /* number of Gaussians; 0 => full-f            */
    double amp[4];    /* f_eq(v) = sum_g amp_g exp(-c_g (v - mu_g)^2) */
    double mu[4];
    double c[4];
} oracle_feq_t;

/* mathematical modulo, result in [0, n) */
static long pmod(long a, long n)
{
    long r = a % n;
    return r < 0 ? r + n : r;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* beta = b + b*, (b, b*) in Z x [0,1[ -- floor also for beta < 0. */
void oracle_split_shift(double beta, long *b, double *bstar)
{
    double fl = floor(beta);
    *b = (long)fl;
    *bstar = beta - fl;
}

/* for j in {-d..d+1}, a_{b+j} = prod_{k=-d,k!=j}^{d+1} (b*-k)/(j-k).
 * w[j+d] receives the weight of index j; 2d+2 values. */
void oracle_lagrange_weights(int d, double bstar, double *w)
{
    for (int j = -d; j <= d + 1; ++j) {
        double p = 1.0;
        for (int k = -d; k <= d + 1; ++k) {
            if (k == j) continue;
            p *= (bstar - (double)k) / (double)(j - k);
        }
        w[j + d] = p;
    }
}

/* P:121 recurrence on the unit mesh (x_i = i, Delta x = 1):
 *   B_i^0(x) = 1 on [x_i, x_{i+1}[  (half-open: DESIGN.md reading Q8)
 *   B_i^k(x) = (x-x_i)/k * B_i^{k-1}(x) + (1 - (x-x_{i+1})/k) * B_{i+1}^{k-1}(x) */
double oracle_bspline(int i, int k, double x)
{
    if (k == 0) return (x >= (double)i && x < (double)(i + 1)) ? 1.0 : 0.0;
    return (x - (double)i) / (double)k * oracle_bspline(i, k - 1, x)
         + (1.0 - (x - (double)(i + 1)) / (double)k) * oracle_bspline(i + 1, k - 1, x);
}

/* First row a_0..a_{N-1} of the circulant A (eq (4)) for Lagrange
 * degree 2d+1 and normalised displacement beta.  a must hold N zeros-able
 * doubles.  Entries that fall on the same index (2d+2 > N is rejected by
 * the caller) are accumulated. */
void oracle_lagrange_first_row(int N, int d, double beta, double *a)
{
    long b; double bs;
    double w[64];
    oracle_split_shift(beta, &b, &bs);
    oracle_lagrange_weights(d, bs, w);
    for (int i = 0; i < N; ++i) a[i] = 0.0;
    for (int j = -d; j <= d + 1; ++j) a[pmod(b + j, N)] += w[j + d];
}

/* Dense circulant from its first row: A[i][i'] = a_{(i'-i) mod N} (P:100:
 * first row a_0 a_1 ..., second row a_{N-1} a_0 a_1 ...). Row-major N x N. */
void oracle_circulant(int N, const double *a, double *A)
{
    for (int i = 0; i < N; ++i)
        for (int ip = 0; ip < N; ++ip)
            A[(size_t)i * N + ip] = a[pmod((long)ip - i, N)];
}

/* u' = A u by the stencil form of the Lagrange circulant:
 * u'_i = sum_{j=-d}^{d+1} a_{b+j} u_{(i+b+j) mod N}  (row i of eq (4)). */
void oracle_lagrange_line(int N, const double *u, long stride, double beta, int d,
                          double *out, long ostride)
{
    long b; double bs;
    double w[64];
    oracle_split_shift(beta, &b, &bs);
    oracle_lagrange_weights(d, bs, w);
    for (int i = 0; i < N; ++i) {
        double s = 0.0;
        for (int j = -d; j <= d + 1; ++j)
            s += w[j + d] * u[pmod((long)i + b + j, N) * stride];
        out[(long)i * ostride] = s;
    }
}

/* Solve the dense system A x = r (A row-major n x n, destroyed) by Gaussian
 * elimination with partial pivoting.  Returns 0, or -1 if singular. */
static int dense_solve(int n, double *A, double *r)
{
    for (int c = 0; c < n; ++c) {
        int p = c;
        double best = fabs(A[(size_t)c * n + c]);
        for (int q = c + 1; q < n; ++q) {
            double v = fabs(A[(size_t)q * n + c]);
            if (v > best) { best = v; p = q; }
        }
        if (best == 0.0) return -1;
        if (p != c) {
            for (int k = 0; k < n; ++k) {
                double t = A[(size_t)c * n + k];
                A[(size_t)c * n + k] = A[(size_t)p * n + k];
                A[(size_t)p * n + k] = t;
            }
            double t = r[c]; r[c] = r[p]; r[p] = t;
        }
        for (int q = c + 1; q < n; ++q) {
            double m = A[(size_t)q * n + c] / A[(size_t)c * n + c];
            if (m == 0.0) continue;
            for (int k = c; k < n; ++k) A[(size_t)q * n + k] -= m * A[(size_t)c * n + k];
            r[q] -= m * r[c];
        }
    }
    for (int c = n - 1; c >= 0; --c) {
        double s = r[c];
        for (int k = c + 1; k < n; ++k) s -= A[(size_t)c * n + k] * r[k];
        r[c] = s / A[(size_t)c * n + c];
    }
    return 0;
}

/* First rows of the two circulants of P:125-129 for the B-spline of degree k:
 *   cc = (0,..,0 [N-k zeros], B_0^k(x_1), .., B_0^k(x_k))
 *   mm: m_{b-j} = B_0^k(x_{j+b*}), j = 0..k. */
void oracle_spline_first_rows(int N, int k, double beta, double *cc, double *mm)
{
    long b; double bs;
    oracle_split_shift(beta, &b, &bs);
    for (int i = 0; i < N; ++i) { cc[i] = 0.0; mm[i] = 0.0; }
    for (int p = 1; p <= k; ++p) cc[N - k + p - 1] += oracle_bspline(0, k, (double)p);
    for (int j = 0; j <= k; ++j) mm[pmod(b - j, N)] += oracle_bspline(0, k, (double)j + bs);
}

/* Dense A = M x C^{-1} for the B-spline of degree k, N small.
 * A row-major N x N.  Returns 0 or -1 (singular collocation matrix). */
int oracle_spline_dense_matrix(int N, int k, double beta, double *A)
{
    double *cc = malloc(sizeof(double) * N), *mm = malloc(sizeof(double) * N);
    double *C = malloc(sizeof(double) * N * N), *M = malloc(sizeof(double) * N * N);
    double *Cw = malloc(sizeof(double) * N * N), *col = malloc(sizeof(double) * N);
    int rc = 0;
    oracle_spline_first_rows(N, k, beta, cc, mm);
    oracle_circulant(N, cc, C);
    oracle_circulant(N, mm, M);
    /* column q of C^{-1}: solve C y = e_q; then A[:,q] = M y */
    for (int q = 0; q < N && rc == 0; ++q) {
        memcpy(Cw, C, sizeof(double) * N * N);
        for (int i = 0; i < N; ++i) col[i] = (i == q) ? 1.0 : 0.0;
        rc = dense_solve(N, Cw, col);
        if (rc) break;
        for (int i = 0; i < N; ++i) {
            double s = 0.0;
            for (int ip = 0; ip < N; ++ip) s += M[(size_t)i * N + ip] * col[ip];
            A[(size_t)i * N + q] = s;
        }
    }
    free(cc); free(mm); free(C); free(M); free(Cw); free(col);
    return rc;
}

/* Cubic spline (degree 3) line, production path of the oracle:
 * solve C eta = u with C = C(0,..,0,1/6,4/6,1/6), i.e.
 *   (1/6) eta_{i-3} + (4/6) eta_{i-2} + (1/6) eta_{i-1} = u_i   (indices mod N),
 * by the cyclic Thomas algorithm (Sherman-Morrison) on the re-indexed unknown
 * y_i = eta_{i-2}, then u'_i = sum_{j=0}^{3} m_{b-j} eta_{(i+b-j) mod N}. */
int oracle_spline3_line(int N, const double *u, long stride, double beta,
                        double *out, long ostride)
{
    long b; double bs;
    oracle_split_shift(beta, &b, &bs);
    double B1 = oracle_bspline(0, 3, 1.0), B2 = oracle_bspline(0, 3, 2.0), B3 = oracle_bspline(0, 3, 3.0);
    /* unknown y_i = eta_{(i-2) mod N}:  B1*y_{i-1} + B2*y_i + B3*y_{i+1} = u_i
     * (C row i has B(x_1) at column i-3, B(x_2) at i-2, B(x_3) at i-1). */
    double *y = malloc(sizeof(double) * N), *z = malloc(sizeof(double) * N);
    double *cp = malloc(sizeof(double) * N), *dd = malloc(sizeof(double) * N);
    /* cyclic tridiagonal: lower = B1, diag = B2, upper = B3, corners upper-right B1, lower-left B3 */
    double gamma = -B2;
    /* modified diagonal */
    for (int i = 0; i < N; ++i) dd[i] = B2;
    dd[0] = B2 - gamma;
    dd[N - 1] = B2 - B3 * B1 / gamma;
    /* solve T y = u and T z = w, w = (gamma,0,..,0,B3) */
    for (int pass = 0; pass < 2; ++pass) {
        double *x = pass == 0 ? y : z;
        for (int i = 0; i < N; ++i) x[i] = pass == 0 ? u[(long)i * stride] : 0.0;
        if (pass == 1) { x[0] = gamma; x[N - 1] = B3; }
        /* Thomas forward sweep */
        double denom = dd[0];
        cp[0] = B3 / denom;
        x[0] = x[0] / denom;
        for (int i = 1; i < N; ++i) {
            denom = dd[i] - B1 * cp[i - 1];
            cp[i] = B3 / denom;
            x[i] = (x[i] - B1 * x[i - 1]) / denom;
        }
        for (int i = N - 2; i >= 0; --i) x[i] -= cp[i] * x[i + 1];
    }
    /* Sherman-Morrison: v = (1,0,..,0,B1/gamma) */
    {
        double vy = y[0] + B1 / gamma * y[N - 1];
        double vz = z[0] + B1 / gamma * z[N - 1];
        double fac = vy / (1.0 + vz);
        for (int i = 0; i < N; ++i) y[i] -= fac * z[i];
    }
    /* eta_k = y_{(k+2) mod N};  u'_i = sum_j B_0^3(x_{j+b*}) eta_{(i+b-j) mod N} */
    double m[4];
    for (int j = 0; j <= 3; ++j) m[j] = oracle_bspline(0, 3, (double)j + bs);
    for (int i = 0; i < N; ++i) {
        double s = 0.0;
        for (int j = 0; j <= 3; ++j) s += m[j] * y[pmod((long)i + b - j + 2, N)];
        out[(long)i * ostride] = s;
    }
    free(y); free(z); free(cp); free(dd);
    return 0;
}

/* One line, either kind.  order = polynomial degree: Lagrange odd 1..17
 * (d = (order-1)/2), B-spline 3.  Returns 0 or -1 on bad arguments. */
int oracle_advect_line(int N, const double *u, long stride, double beta, int kind, int order,
                       double *out, long ostride)
{
    if (kind == ORACLE_LAGRANGE) {
        if (order < 1 || (order & 1) == 0 || order > 17 || order > N - 1) return -1;
        oracle_lagrange_line(N, u, stride, beta, (order - 1) / 2, out, ostride);
        return 0;
    }
    if (kind == ORACLE_BSPLINE && order == 3) return oracle_spline3_line(N, u, stride, beta, out, ostride);
    return -1;
}

/* Shift every velocity row j by beta[j] cells along x (out of place). */
int oracle_shift_x(int Nx, int Nv, const double *f, const double *beta, int kind, int order, double *out)
{
    int rc = 0;
#pragma omp parallel for schedule(static) reduction(|:rc)
    for (int j = 0; j < Nv; ++j)
        rc |= oracle_advect_line(Nx, f + (size_t)j * Nx, 1, beta[j], kind, order, out + (size_t)j * Nx, 1);
    return rc ? -1 : 0;
}

/* Shift every space column i by beta[i] cells along v (out of place). */
int oracle_shift_v(int Nx, int Nv, const double *f, const double *beta, int kind, int order, double *out)
{
    int rc = 0;
#pragma omp parallel for schedule(static) reduction(|:rc)
    for (int i = 0; i < Nx; ++i)
        rc |= oracle_advect_line(Nv, f + i, Nx, beta[i], kind, order, out + i, Nx);
    return rc ? -1 : 0;
}

/* Mesh: x_i = i dx, dx = L/Nx; v_j = vmin + j dv, dv = (vmax-vmin)/Nv (reading Q2). */
static double mesh_v(int j, int Nv, double vmin, double vmax)
{
    return vmin + (double)j * ((vmax - vmin) / (double)Nv);
}

/* transport in x over dt: for each v_j a constant advection with c = v_j,
 * beta = -c dt / dx. */
int oracle_advect_x(int Nx, int Nv, const double *f, double L, double vmin, double vmax, double dt,
                    int kind, int order, double *out)
{
    double dx = L / (double)Nx;
    double *beta = malloc(sizeof(double) * Nv);
    for (int j = 0; j < Nv; ++j) beta[j] = -mesh_v(j, Nv, vmin, vmax) * dt / dx;
    int rc = oracle_shift_x(Nx, Nv, f, beta, kind, order, out);
    free(beta);
    return rc;
}

double oracle_feq(const oracle_feq_t *q, double v)
{
    double s = 0.0;
    for (int g = 0; g < q->n; ++g) s += q->amp[g] * exp(-q->c[g] * (v - q->mu[g]) * (v - q->mu[g]));
    return s;
}

/* transport in v over dt with c = E_i, beta = -E_i dt / dv;
 * delta-f mode (feq->n > 0): add f_eq(v_j - dt E_i) - f_eq(v_j), an evaluation. */
int oracle_advect_v(int Nx, int Nv, const double *f, const double *E, double vmin, double vmax, double dt,
                    int kind, int order, const oracle_feq_t *feq, double *out)
{
    double dv = (vmax - vmin) / (double)Nv;
    double *beta = malloc(sizeof(double) * Nx);
    for (int i = 0; i < Nx; ++i) beta[i] = -E[i] * dt / dv;
    int rc = oracle_shift_v(Nx, Nv, f, beta, kind, order, out);
    free(beta);
    if (rc == 0 && feq && feq->n > 0) {
#pragma omp parallel for schedule(static)
        for (int j = 0; j < Nv; ++j) {
            double v = mesh_v(j, Nv, vmin, vmax);
            double f0 = oracle_feq(feq, v);
            for (int i = 0; i < Nx; ++i)
                out[(size_t)j * Nx + i] += oracle_feq(feq, v - dt * E[i]) - f0;
        }
    }
    return rc;
}

/* rho_i = dv * sum_j f_ji  (uniform weights on the Nv periodic nodes, reading Q10). */
void oracle_density(int Nx, int Nv, const double *f, double vmin, double vmax, double *rho)
{
    double dv = (vmax - vmin) / (double)Nv;
    for (int i = 0; i < Nx; ++i) {
        double s = 0.0;
        for (int j = 0; j < Nv; ++j) s += f[(size_t)j * Nx + i];
        rho[i] = dv * s;
    }
}

/* Field from a given density: zero-mean rho, then "Fourier":
 *   rho^_m = sum_i rho~_i e^{-2 i pi m i / Nx},
 *   E^_m = rho^_m / (i k_m), k_m = 2 pi m / L for 0 < m < Nx/2 and the mirrored
 *   negative frequencies; E^_0 = 0; E^_{Nx/2} = 0 (reading Q12),
 *   E_i = (1/Nx) sum_m E^_m e^{+2 i pi m i / Nx}.
 * Both sums are written out naively, O(Nx^2). */
void oracle_poisson(int Nx, const double *rho, double L, double *E)
{
    double mean = 0.0;
    for (int i = 0; i < Nx; ++i) mean += rho[i];
    mean /= (double)Nx;
    double *cr = malloc(sizeof(double) * Nx), *ci = malloc(sizeof(double) * Nx);
    double *er = malloc(sizeof(double) * Nx), *ei = malloc(sizeof(double) * Nx);
    /* roots of unity e^{-2 i pi q / Nx}, q = 0..Nx-1 */
    for (int q = 0; q < Nx; ++q) {
        double a = -2.0 * M_PI * (double)q / (double)Nx;
        cr[q] = cos(a); ci[q] = sin(a);
    }
#pragma omp parallel for schedule(static)
    for (int m = 0; m < Nx; ++m) {
        double sr = 0.0, si = 0.0;
        for (int i = 0; i < Nx; ++i) {
            long q = ((long)m * i) % Nx;
            double r = rho[i] - mean;
            sr += r * cr[q]; si += r * ci[q];
        }
        /* signed frequency */
        int ms = (m <= Nx / 2) ? m : m - Nx;
        if (m == 0 || 2 * m == Nx) { er[m] = 0.0; ei[m] = 0.0; }
        else {
            double k = 2.0 * M_PI * (double)ms / L;
            /* (sr + i si) / (i k) = (si - i sr) / k */
            er[m] = si / k; ei[m] = -sr / k;
        }
    }
#pragma omp parallel for schedule(static)
    for (int i = 0; i < Nx; ++i) {
        double s = 0.0;
        for (int m = 0; m < Nx; ++m) {
            long q = ((long)m * i) % Nx;
            /* e^{+i a} = conj(root): real part of (er + i ei)(cr - i ci) */
            s += er[m] * cr[q] + ei[m] * ci[q];
        }
        E[i] = s / (double)Nx;
    }
    free(cr); free(ci); free(er); free(ei);
}

void oracle_field(int Nx, int Nv, const double *f, double L, double vmin, double vmax, double *E)
{
    double *rho = malloc(sizeof(double) * Nx);
    oracle_density(Nx, Nv, f, vmin, vmax, rho);
    oracle_poisson(Nx, rho, L, E);
    free(rho);
}

/* The paper's other field solve, written out step by step:
 *   M = (1/N) sum_k rho_k;  rho~_k = rho_k - M           (zero_mean != 0)
 *                           rho~_k = rho_k - background   (zero_mean == 0: "rho~ = rho - 1"; the caller passes
 *                                                          the background, 1 minus the equilibrium's mass in delta-f mode)
 *   E~_0 = 0;  E~_{k+1} = E~_k + dx (rho~_k + rho~_{k+1}) / 2,  k = 0 .. N-2      (trapezoidal rule)
 *   M~ = (1/N) sum_k E~_k;  E_k = E~_k - M~               (zero_mean != 0); E_k = E~_k otherwise. */
void oracle_field_trapezoid(int Nx, const double *rho, double L, int zero_mean, double background, double *E)
{
    double dx = L / (double)Nx;
    double M = background;
    if (zero_mean) {
        M = 0.0;
        for (int k = 0; k < Nx; ++k) M += rho[k];
        M /= (double)Nx;
    }
    E[0] = 0.0;
    for (int k = 0; k + 1 < Nx; ++k) E[k + 1] = E[k] + dx * ((rho[k] - M) + (rho[k + 1] - M)) / 2.0;
    if (zero_mean) {
        double Mt = 0.0;
        for (int k = 0; k < Nx; ++k) Mt += E[k];
        Mt /= (double)Nx;
        for (int k = 0; k < Nx; ++k) E[k] -= Mt;
    }
}

/* Diagnostics of P:245, 253-261 from a density:  out[0] = rho^_0 = (1/N) sum_k rho_k  (the mass error is |rho^_0 - 1|,
 * P:245; in delta-f mode the caller adds the equilibrium's mass);  out[1] = |rho^_1| = |(1/N) sum_k rho_k e^{-2 i pi k/N}|
 * ("the first mode of rho in absolute value"). */
void oracle_rho_modes(int Nx, const double *rho, double *out)
{
    double s0 = 0.0, sr = 0.0, si = 0.0;
    for (int k = 0; k < Nx; ++k) {
        double a = -2.0 * M_PI * (double)k / (double)Nx;
        s0 += rho[k];
        sr += rho[k] * cos(a);
        si += rho[k] * sin(a);
    }
    out[0] = s0 / (double)Nx;
    out[1] = sqrt(sr * sr + si * si) / (double)Nx;
}

/* Kinetic energy: E_k = int int f v^2/2 dv dx ~ (1/2) dx dv sum_j v_j^2 sum_i f_ji (rectangle rule on the
 * periodic mesh, the same weights as rho).  Of the stored array: in delta-f mode the caller adds the equilibrium's part. */
double oracle_kinetic_energy(int Nx, int Nv, const double *f, double L, double vmin, double vmax)
{
    double dx = L / (double)Nx, dv = (vmax - vmin) / (double)Nv, s = 0.0;
    for (int j = 0; j < Nv; ++j) {
        double v = mesh_v(j, Nv, vmin, vmax), r = 0.0;
        for (int i = 0; i < Nx; ++i) r += f[(size_t)j * Nx + i];
        s += v * v * r;
    }
    return 0.5 * dx * dv * s;
}

/* Electric energy (1/2) ||E||^2_{L2} = (1/2) dx sum_i E_i^2. */
double oracle_electric_energy(int Nx, const double *E, double L)
{
    double s = 0.0;
    for (int i = 0; i < Nx; ++i) s += E[i] * E[i];
    return 0.5 * (L / (double)Nx) * s;
}

/* One Strang step, in place on f (reading Q1).
 * split 0 (XVX, the order BASELINE.json's configs bind): x(dt/2); E = field(f);
 *   v(dt, E + E_ext); x(dt/2).  E_out receives the self-consistent E used.
 * split 1 (VXV, the paper's order P:63-83): v(dt/2, E_in + E_ext); x(dt);
 *   E = field(f); v(dt/2, E + E_ext).  E_in is the self-consistent field at t^n
 *   (caller supplies it, e.g. from oracle_field); E_out receives E^{n+1}.
 * E_ext may be NULL.  work must hold Nx*Nv doubles. */
int oracle_step(int Nx, int Nv, double *f, double L, double vmin, double vmax, double dt,
                int kind, int order, const oracle_feq_t *feq, int split,
                const double *E_ext, const double *E_in, double *E_out, double *work)
{
    double *Et = malloc(sizeof(double) * Nx);
    int rc = 0;
    size_t bytes = sizeof(double) * (size_t)Nx * Nv;
    if (split == 0) {
        rc |= oracle_advect_x(Nx, Nv, f, L, vmin, vmax, 0.5 * dt, kind, order, work);
        oracle_field(Nx, Nv, work, L, vmin, vmax, E_out);
        for (int i = 0; i < Nx; ++i) Et[i] = E_out[i] + (E_ext ? E_ext[i] : 0.0);
        rc |= oracle_advect_v(Nx, Nv, work, Et, vmin, vmax, dt, kind, order, feq, f);
        rc |= oracle_advect_x(Nx, Nv, f, L, vmin, vmax, 0.5 * dt, kind, order, work);
        memcpy(f, work, bytes);
    } else {
        for (int i = 0; i < Nx; ++i) Et[i] = E_in[i] + (E_ext ? E_ext[i] : 0.0);
        rc |= oracle_advect_v(Nx, Nv, f, Et, vmin, vmax, 0.5 * dt, kind, order, feq, work);
        rc |= oracle_advect_x(Nx, Nv, work, L, vmin, vmax, dt, kind, order, f);
        oracle_field(Nx, Nv, f, L, vmin, vmax, E_out);
        for (int i = 0; i < Nx; ++i) Et[i] = E_out[i] + (E_ext ? E_ext[i] : 0.0);
        rc |= oracle_advect_v(Nx, Nv, f, Et, vmin, vmax, 0.5 * dt, kind, order, feq, work);
        memcpy(f, work, bytes);
    }
    free(Et);
    return rc ? -1 : 0;
}
