/*
 * clt_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU evaluation (FP64) of the hot path of CLTx
 * (arxiv 1812.00525): the resistive-MHD right-hand side in the equilibrium-subtracted
 * form, eqs (11)-(14) [PAPER.md L105-115] with Ohm/Ampere, eqs (5)-(6) [L77-79] (Hall term of eq (5)
 * optional: d_i = 0 unless oracle_set_hall() is called),
 * on a uniform cylindrical (R, phi, Z) grid with 4th-order central differences [L125],
 * advanced by the classical 4th-order Runge-Kutta scheme [L125, L139], plus the
 * kinetic/magnetic-energy and div B diagnostics [L139, L149, L430] and the SETDT CFL
 * formula [Fig. 4, L180-215].
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * may call this.  It shares no code with the CUDA path (paper_1812_00525_b200/csrc).
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (no fast-math).  OpenMP is used only
 * on the outermost loop over nodes (every node is independent); there is no blocking, fusion
 * or reordering beyond what the formulas state.
 *
 * Every discrete choice the paper leaves open is a reading listed in DESIGN.md ("Readings",
 * R1-R9, G1-G15); the ones used here are cited next to the code.
 *
 * PINS (tests/test_oracle_pins.py, all CPU):  P1 stencils exact on polynomials; P2 vacuum-field
 * static state gives K = 0; P3 4th-order convergence of every operator and of the whole RHS to
 * a sympy-derived analytic RHS of eqs (1)-(6); P4 div_c B stays at round-off over steps;
 * P5 rigid rotation annihilated by the viscous operator; P6 U0 = 0 reduces to a separately
 * written numpy evaluation of eqs (1)-(4); P7 Alfven modified-wavenumber identity; P8 RK4 order
 * on du/dt = lambda u through oracle_rk4 and on the MHD system by dt-halving.  P12 Hall term of eq (5):
 * exact discrete whistler-type response with the squared modified wavenumber, d_i = 0 reduction, and the
 * sympy convergence pin P3b run with d_i != 0.  P13 pseudo-spectral phi scheme: against numpy.fft, exact on
 * resolved Fourier modes, the Alfven identity with the exact wavenumber, P3b with the spectral scheme.
 * P10 oracle_setdt against the closed form of Fig. 4 on a uniform state; P11 oracle_diagnostics (all five
 * outputs) against closed forms; P14 oracle_step_cfl = SETDT + one RK4 step with that dt, step by step.
 * Parity unpinned: none of the exported functions (each is covered by at least one pin); the
 * absolute value of a generic RHS has no paper-printed number to compare with (PAPER.md prints
 * no worked example), so the pins above are mathematical ones.
 *
 * Layout: a scalar field is f[(j*nZ + k)*nR + i], i = R index (fastest), k = Z, j = phi -- the C
 * image of CLTx's X(JX,JZ,JY,M) [L191-196].  A state is 8 such fields in the order
 * rho, p, v_R, v_phi, v_Z, B_R, B_phi, B_Z [L191-196].  A vector field is 3 consecutive fields
 * (R, phi, Z components).
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct oracle {
    int nR, nphi, nZ;
    double Rmin, Rmax, Zmin, Zmax, Lphi;
    double dR, dZ, dphi;
    double gamma, eta, nu, D, kappa, dt;
    int phi_scheme;     /* 0 = 4th-order central differences in phi, 1 = pseudo-spectral (L125) */
    double *c1, *c2;    /* pseudo-spectral derivative weights, see oracle_set_phi_scheme         */
    double last_dt;     /* dt of the last adaptive step (oracle_step_cfl); the fixed dt is untouched */
    double d_i;         /* ion inertial length of the Hall term in eq (5); 0 = resistive MHD */
    double *R;          /* R_i = Rmin + i*dR  (reading R1; hazard H1)           */
    double *Z;          /* Z_k = Zmin + k*dZ                                     */
    size_t N;           /* nodes per field                                       */
    /* equilibrium, replicated along phi so that the same operators apply       */
    double *U0;         /* 8N                                                    */
    double *J0;         /* 3N  curl_c(B0) on interior nodes, 0 on boundary layers */
    double *divv0;      /* N   div v0                                            */
    double *v0gv0;      /* 3N  (v0.grad) v0                                      */
    /* state and work arrays                                                     */
    double *U;          /* 8N                                                    */
    double *U1;         /* 8N  perturbation U - U0                               */
    double *J1;         /* 3N                                                    */
    double *E1;         /* 3N                                                    */
    double *G;          /* 3N  Hall field (J1 x B + J0 x B1 - grad p1)/rho - rho1 (v0.grad)v0/rho on interior nodes */
    double *K1, *K2, *K3, *K4, *Us;   /* 8N each, RK4 work                      */
    int64_t step;
    double time;
} oracle;

/* ---------------------------------------------------------------------------------------- */
/* O0 grid / indexing                                                                       */

static inline size_t idx(const oracle *o, int i, int k, int j)
{
    return ((size_t)j * (size_t)o->nZ + (size_t)k) * (size_t)o->nR + (size_t)i;
}
static inline int wrapphi(const oracle *o, int j)       /* phi is periodic [L125; a1]   */
{
    int n = o->nphi;
    j %= n;
    if (j < 0) j += n;
    return j;
}
/* boundary layers: two node layers per R/Z side hold fixed values (Fig. 4 loop bounds
 * FIRST+2 .. LAST-2, L187-189; fixed boundary L123)                                       */
static inline int is_interior(const oracle *o, int i, int k)
{
    return i >= 2 && i <= o->nR - 3 && k >= 2 && k <= o->nZ - 3;
}

/* ---------------------------------------------------------------------------------------- */
/* O1 stencils: standard 4th-order central differences, radius 2 (reading R2; L125, L127)   */

static inline double d1R(const oracle *o, const double *f, int i, int k, int j)
{
    return (8.0 * (f[idx(o, i + 1, k, j)] - f[idx(o, i - 1, k, j)])
            - (f[idx(o, i + 2, k, j)] - f[idx(o, i - 2, k, j)])) / (12.0 * o->dR);
}
static inline double d1Z(const oracle *o, const double *f, int i, int k, int j)
{
    return (8.0 * (f[idx(o, i, k + 1, j)] - f[idx(o, i, k - 1, j)])
            - (f[idx(o, i, k + 2, j)] - f[idx(o, i, k - 2, j)])) / (12.0 * o->dZ);
}
static inline double d1P(const oracle *o, const double *f, int i, int k, int j)
{
    if (o->phi_scheme == 1) {       /* pseudo-spectral: sum_m c1[m] f_{j+m}, see oracle_set_phi_scheme */
        double s = 0.0;
        for (int m = 0; m < o->nphi; ++m) s += o->c1[m] * f[idx(o, i, k, wrapphi(o, j + m))];
        return s;
    }
    return (8.0 * (f[idx(o, i, k, wrapphi(o, j + 1))] - f[idx(o, i, k, wrapphi(o, j - 1))])
            - (f[idx(o, i, k, wrapphi(o, j + 2))] - f[idx(o, i, k, wrapphi(o, j - 2))]))
           / (12.0 * o->dphi);
}
/* d/dR of the product R*f, differencing the products R_{i+s} f_{i+s} (reading R4)          */
static inline double d1R_Rf(const oracle *o, const double *f, int i, int k, int j)
{
    const double *R = o->R;
    return (8.0 * (R[i + 1] * f[idx(o, i + 1, k, j)] - R[i - 1] * f[idx(o, i - 1, k, j)])
            - (R[i + 2] * f[idx(o, i + 2, k, j)] - R[i - 2] * f[idx(o, i - 2, k, j)]))
           / (12.0 * o->dR);
}
static inline double d2R(const oracle *o, const double *f, int i, int k, int j)
{
    return (-f[idx(o, i + 2, k, j)] + 16.0 * f[idx(o, i + 1, k, j)] - 30.0 * f[idx(o, i, k, j)]
            + 16.0 * f[idx(o, i - 1, k, j)] - f[idx(o, i - 2, k, j)]) / (12.0 * o->dR * o->dR);
}
static inline double d2Z(const oracle *o, const double *f, int i, int k, int j)
{
    return (-f[idx(o, i, k + 2, j)] + 16.0 * f[idx(o, i, k + 1, j)] - 30.0 * f[idx(o, i, k, j)]
            + 16.0 * f[idx(o, i, k - 1, j)] - f[idx(o, i, k - 2, j)]) / (12.0 * o->dZ * o->dZ);
}
static inline double d2P(const oracle *o, const double *f, int i, int k, int j)
{
    if (o->phi_scheme == 1) {
        double s = 0.0;
        for (int m = 0; m < o->nphi; ++m) s += o->c2[m] * f[idx(o, i, k, wrapphi(o, j + m))];
        return s;
    }
    return (-f[idx(o, i, k, wrapphi(o, j + 2))] + 16.0 * f[idx(o, i, k, wrapphi(o, j + 1))]
            - 30.0 * f[idx(o, i, k, j)]
            + 16.0 * f[idx(o, i, k, wrapphi(o, j - 1))] - f[idx(o, i, k, wrapphi(o, j - 2))])
           / (12.0 * o->dphi * o->dphi);
}

/* ---------------------------------------------------------------------------------------- */
/* O2 operators in (R, phi, Z), right-handed, R^ x phi^ = Z^ (L121)                          */

/* grad f = (d_R f, d_phi f / R, d_Z f) */
static inline void grad(const oracle *o, const double *f, int i, int k, int j, double g[3])
{
    g[0] = d1R(o, f, i, k, j);
    g[1] = d1P(o, f, i, k, j) / o->R[i];
    g[2] = d1Z(o, f, i, k, j);
}
static inline double dot3(const double a[3], const double b[3])
{
    return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}
/* div a = d_R a_R + a_R/R + d_phi a_phi / R + d_Z a_Z   (expanded form, reading R3) */
static inline double divergence(const oracle *o, const double *a, int i, int k, int j)
{
    size_t N = o->N;
    double R = o->R[i];
    return d1R(o, a, i, k, j) + a[idx(o, i, k, j)] / R + d1P(o, a + N, i, k, j) / R
           + d1Z(o, a + 2 * N, i, k, j);
}
/* conservative curl (reading R4): the radial derivative in the Z component differences R*A_phi */
static inline void curl_c(const oracle *o, const double *A, int i, int k, int j, double c[3])
{
    size_t N = o->N;
    double R = o->R[i];
    const double *AR = A, *AP = A + N, *AZ = A + 2 * N;
    c[0] = d1P(o, AZ, i, k, j) / R - d1Z(o, AP, i, k, j);
    c[1] = d1Z(o, AR, i, k, j) - d1R(o, AZ, i, k, j);
    c[2] = d1R_Rf(o, AP, i, k, j) / R - d1P(o, AR, i, k, j) / R;
}
/* matching divergence: div_c a = d_R(R a_R)/R + d_phi a_phi / R + d_Z a_Z  (reading R4) */
static inline double div_c(const oracle *o, const double *a, int i, int k, int j)
{
    size_t N = o->N;
    double R = o->R[i];
    return d1R_Rf(o, a, i, k, j) / R + d1P(o, a + N, i, k, j) / R + d1Z(o, a + 2 * N, i, k, j);
}
/* scalar Laplacian = d2_R f + d_R f / R + d2_phi f / R^2 + d2_Z f ; second derivatives use the
 * 5-point delta^2 directly, not delta applied twice (reading R2) */
static inline double laplacian(const oracle *o, const double *f, int i, int k, int j)
{
    double R = o->R[i];
    return d2R(o, f, i, k, j) + d1R(o, f, i, k, j) / R + d2P(o, f, i, k, j) / (R * R)
           + d2Z(o, f, i, k, j);
}
/* vector Laplacian (reading G4) */
static inline void vector_laplacian(const oracle *o, const double *a, int i, int k, int j,
                                    double L[3])
{
    size_t N = o->N;
    double R = o->R[i];
    const double *aR = a, *aP = a + N, *aZ = a + 2 * N;
    L[0] = laplacian(o, aR, i, k, j) - aR[idx(o, i, k, j)] / (R * R)
           - 2.0 * d1P(o, aP, i, k, j) / (R * R);
    L[1] = laplacian(o, aP, i, k, j) - aP[idx(o, i, k, j)] / (R * R)
           + 2.0 * d1P(o, aR, i, k, j) / (R * R);
    L[2] = laplacian(o, aZ, i, k, j);
}
/* (a.grad) b for vectors: components of a given as numbers at the node, b a field */
static inline void advect_vector(const oracle *o, const double a[3], const double *b, int i,
                                 int k, int j, double out[3])
{
    size_t N = o->N, n = idx(o, i, k, j);
    double R = o->R[i];
    double g[3];
    grad(o, b, i, k, j, g);
    out[0] = dot3(a, g) - a[1] * b[N + n] / R;
    grad(o, b + N, i, k, j, g);
    out[1] = dot3(a, g) + a[1] * b[n] / R;
    grad(o, b + 2 * N, i, k, j, g);
    out[2] = dot3(a, g);
}
static inline void cross(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1];
    c[1] = a[2] * b[0] - a[0] * b[2];
    c[2] = a[0] * b[1] - a[1] * b[0];
}

/* ---------------------------------------------------------------------------------------- */
/* life cycle                                                                               */

static double *zalloc(size_t n)
{
    return (double *)calloc(n ? n : 1, sizeof(double));
}

oracle *oracle_create(int nR, int nphi, int nZ, double Rmin, double Rmax, double Zmin,
                      double Zmax, double phi_extent, double gamma, double eta, double nu,
                      double D, double kappa, double dt)
{
    if (nR < 9 || nZ < 9 || nphi < 5 || !(Rmin > 0.0) || !(Rmax > Rmin) || !(Zmax > Zmin))
        return NULL;
    oracle *o = (oracle *)calloc(1, sizeof(oracle));
    if (!o) return NULL;
    o->nR = nR; o->nphi = nphi; o->nZ = nZ;
    o->Rmin = Rmin; o->Rmax = Rmax; o->Zmin = Zmin; o->Zmax = Zmax;
    o->Lphi = (phi_extent == 0.0) ? 2.0 * M_PI : phi_extent;
    o->dR = (Rmax - Rmin) / (double)(nR - 1);      /* box edge is a node (reading R1)  */
    o->dZ = (Zmax - Zmin) / (double)(nZ - 1);
    o->dphi = o->Lphi / (double)nphi;
    o->gamma = gamma; o->eta = eta; o->nu = nu; o->D = D; o->kappa = kappa; o->dt = dt;
    o->N = (size_t)nR * (size_t)nZ * (size_t)nphi;
    o->R = zalloc((size_t)nR);
    for (int i = 0; i < nR; ++i) o->R[i] = Rmin + (double)i * o->dR;
    o->Z = zalloc((size_t)nZ);
    for (int k = 0; k < nZ; ++k) o->Z[k] = Zmin + (double)k * o->dZ;
    size_t N = o->N;
    o->U0 = zalloc(8 * N); o->J0 = zalloc(3 * N); o->divv0 = zalloc(N); o->v0gv0 = zalloc(3 * N);
    o->U = zalloc(8 * N); o->U1 = zalloc(8 * N); o->J1 = zalloc(3 * N); o->E1 = zalloc(3 * N);
    o->G = zalloc(3 * N);
    o->K1 = zalloc(8 * N); o->K2 = zalloc(8 * N); o->K3 = zalloc(8 * N); o->K4 = zalloc(8 * N);
    o->Us = zalloc(8 * N);
    return o;
}

void oracle_destroy(oracle *o)
{
    if (!o) return;
    free(o->R); free(o->Z); free(o->U0); free(o->J0); free(o->divv0); free(o->v0gv0);
    free(o->U); free(o->U1); free(o->J1); free(o->E1); free(o->G); free(o->c1); free(o->c2);
    free(o->K1); free(o->K2); free(o->K3); free(o->K4); free(o->Us);
    free(o);
}

void oracle_set_dt(oracle *o, double dt) { o->dt = dt; }

/* phi scheme [L125: "in the phi direction, either 4th order finite difference or pseudo-spectrum method can be
 * used"].  scheme 1 = pseudo-spectral (reading R12): the periodic samples f_j, j = 0..N-1 on length L are
 * expanded in the discrete Fourier modes e^{i kappa q phi}, kappa = 2 pi / L, q = -Q..Q, Q = floor((N-1)/2)
 * [plus the Nyquist mode q = N/2 when N is even], each mode is differentiated exactly and the series is
 * evaluated back on the nodes.  The Nyquist mode (-1)^j has no defined phase: its first derivative is
 * taken as 0, its second derivative as -(kappa N/2)^2 times itself (the usual convention).  Written in
 * physical space that is the circulant sum  d f_j = sum_m c[m] f_{j+m}  with
 *   c1[m] = (1/N) sum_q (i kappa q) e^{-2 pi i q m/N}       = (2 kappa/N) sum_{q=1..Q} q sin(2 pi q m/N)
 *   c2[m] = (1/N) sum_q -(kappa q)^2 e^{-2 pi i q m/N}      = -(kappa^2/N)[2 sum_{q=1..Q} q^2 cos(2 pi q m/N)
 *                                                              + (N even) (N/2)^2 cos(pi m)]
 * summed here exactly as written (long double).                                                   */
void oracle_set_phi_scheme(oracle *o, int scheme)
{
    int N = o->nphi;
    o->phi_scheme = scheme ? 1 : 0;
    if (!o->phi_scheme) return;
    if (!o->c1) { o->c1 = zalloc((size_t)N); o->c2 = zalloc((size_t)N); }
    long double kappa = 2.0L * 3.141592653589793238462643383279502884L / (long double)o->Lphi;
    int Q = (N - 1) / 2;
    for (int m = 0; m < N; ++m) {
        long double s1 = 0.0L, s2 = 0.0L;
        for (int q = 1; q <= Q; ++q) {
            long double th = 2.0L * 3.141592653589793238462643383279502884L * (long double)q * (long double)m / (long double)N;
            s1 += (long double)q * sinl(th);
            s2 += 2.0L * (long double)q * (long double)q * cosl(th);
        }
        if (N % 2 == 0) s2 += (long double)(N / 2) * (long double)(N / 2) * ((m % 2) ? -1.0L : 1.0L);
        o->c1[m] = (double)(2.0L * kappa / (long double)N * s1);
        o->c2[m] = (double)(-kappa * kappa / (long double)N * s2);
    }
}
/* switches the Hall term of eq (5) [L77] on (d_i != 0) or off (d_i = 0, the default) */
void oracle_set_hall(oracle *o, double d_i) { o->d_i = d_i; }

/* O3: equilibrium U0(R,Z), axisymmetric, [8][nZ][nR]; NULL = all zero.  J0 = curl_c(B0) on
 * interior nodes, once (reading R5: 0 on the boundary layers).                              */
void oracle_set_equilibrium(oracle *o, const double *U0_2d)
{
    size_t N = o->N, plane = (size_t)o->nR * (size_t)o->nZ;
    memset(o->U0, 0, 8 * N * sizeof(double));
    if (U0_2d)
        for (int m = 0; m < 8; ++m)
            for (int j = 0; j < o->nphi; ++j)
                memcpy(o->U0 + (size_t)m * N + (size_t)j * plane, U0_2d + (size_t)m * plane,
                       plane * sizeof(double));
    memset(o->J0, 0, 3 * N * sizeof(double));
    memset(o->divv0, 0, N * sizeof(double));
    memset(o->v0gv0, 0, 3 * N * sizeof(double));
    const double *v0 = o->U0 + 2 * N, *B0 = o->U0 + 5 * N;
#pragma omp parallel for collapse(2) schedule(static)
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i) {
                size_t n = idx(o, i, k, j);
                double c[3], a[3], adv[3];
                curl_c(o, B0, i, k, j, c);
                o->J0[n] = c[0]; o->J0[N + n] = c[1]; o->J0[2 * N + n] = c[2];
                o->divv0[n] = divergence(o, v0, i, k, j);
                a[0] = v0[n]; a[1] = v0[N + n]; a[2] = v0[2 * N + n];
                advect_vector(o, a, v0, i, k, j, adv);
                o->v0gv0[n] = adv[0]; o->v0gv0[N + n] = adv[1]; o->v0gv0[2 * N + n] = adv[2];
            }
}

void oracle_set_state(oracle *o, const double *U)
{
    memcpy(o->U, U, 8 * o->N * sizeof(double));
    o->step = 0;
    o->time = 0.0;
}
void oracle_get_state(const oracle *o, double *U)
{
    memcpy(U, o->U, 8 * o->N * sizeof(double));
}
int64_t oracle_get_step(const oracle *o) { return o->step; }
double oracle_get_time(const oracle *o) { return o->time; }

/* ---------------------------------------------------------------------------------------- */
/* a2: J1 = curl_c(B - B0) on interior nodes, 0 on the boundary layers (eq 6; R4, R5).
 * The equilibrium is subtracted BEFORE differencing (hazard H2; the paper's remark at L117). */
static void compute_U1_J1_E1(oracle *o, const double *U)
{
    size_t N = o->N;
    for (size_t n = 0; n < 8 * N; ++n) o->U1[n] = U[n] - o->U0[n];
    const double *B1 = o->U1 + 5 * N;
    memset(o->J1, 0, 3 * N * sizeof(double));
#pragma omp parallel for collapse(2) schedule(static)
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i) {
                size_t n = idx(o, i, k, j);
                double c[3];
                curl_c(o, B1, i, k, j, c);
                o->J1[n] = c[0]; o->J1[N + n] = c[1]; o->J1[2 * N + n] = c[2];
            }
    /* Hall field of eq (5) [L77] in the equilibrium-subtracted form (reading R11):
     *   E - E0 with E0 = -v0 x B0 + (d_i/rho0)(J0 x B0 - grad p0) [curl-free by eq (10)] and eq (9) used exactly
     *   as eq (13) uses it gives  d_i * G,
     *   G = (J1 x B + J0 x B1 - grad p1)/rho - (rho1/rho) (v0.grad)v0      -- the force bracket of eq (13).
     * On interior nodes; G = 0 on the boundary layers (like J1, reading R5).                    */
    memset(o->G, 0, 3 * N * sizeof(double));
    if (o->d_i != 0.0) {
#pragma omp parallel for collapse(2) schedule(static)
        for (int j = 0; j < o->nphi; ++j)
            for (int k = 2; k <= o->nZ - 3; ++k)
                for (int i = 2; i <= o->nR - 3; ++i) {
                    size_t n = idx(o, i, k, j);
                    double BB[3]  = { U[5 * N + n], U[6 * N + n], U[7 * N + n] };
                    double BB1[3] = { B1[n], B1[N + n], B1[2 * N + n] };
                    double JJ1[3] = { o->J1[n], o->J1[N + n], o->J1[2 * N + n] };
                    double JJ0[3] = { o->J0[n], o->J0[N + n], o->J0[2 * N + n] };
                    double J1xB[3], J0xB1[3], gp1[3];
                    cross(JJ1, BB, J1xB);
                    cross(JJ0, BB1, J0xB1);
                    grad(o, o->U1 + N, i, k, j, gp1);
                    for (int c = 0; c < 3; ++c)
                        o->G[(size_t)c * N + n] = (J1xB[c] + J0xB1[c] - gp1[c]) / U[n]
                                                  - o->U1[n] * o->v0gv0[(size_t)c * N + n] / U[n];
                }
    }
    /* a4: E1 = -v x B + v0 x B0 + eta J1 + d_i G at every node (eq 5 minus E0, eq 10; readings G5, R11).
     * On the boundary layers J1 = 0 and G = 0.                                                  */
#pragma omp parallel for schedule(static)
    for (size_t n = 0; n < N; ++n) {
        double v[3] = { U[2 * N + n], U[3 * N + n], U[4 * N + n] };
        double B[3] = { U[5 * N + n], U[6 * N + n], U[7 * N + n] };
        double v0[3] = { o->U0[2 * N + n], o->U0[3 * N + n], o->U0[4 * N + n] };
        double B0[3] = { o->U0[5 * N + n], o->U0[6 * N + n], o->U0[7 * N + n] };
        double vxB[3], v0xB0[3];
        cross(v, B, vxB);
        cross(v0, B0, v0xB0);
        for (int c = 0; c < 3; ++c) {
            double e = -vxB[c] + v0xB0[c] + o->eta * o->J1[(size_t)c * N + n];
            if (o->d_i != 0.0) e += o->d_i * o->G[(size_t)c * N + n];
            o->E1[(size_t)c * N + n] = e;
        }
    }
}

void oracle_curl_J1(oracle *o, const double *U, double *J1_out)
{
    compute_U1_J1_E1(o, U);
    memcpy(J1_out, o->J1, 3 * o->N * sizeof(double));
}
void oracle_E1(oracle *o, const double *U, double *E1_out)
{
    compute_U1_J1_E1(o, U);
    memcpy(E1_out, o->E1, 3 * o->N * sizeof(double));
}
void oracle_hall_G(oracle *o, const double *U, double *G_out)
{
    compute_U1_J1_E1(o, U);
    memcpy(G_out, o->G, 3 * o->N * sizeof(double));
}

/* a3-a5: K = dU/dt from eqs (11)-(14) on interior nodes, K = 0 on the boundary layers.
 * Uniform D, kappa, nu, eta (reading R6); diffusion acts on the perturbation (G1, G2).       */
void oracle_rhs_of(oracle *o, const double *U, double *K)
{
    size_t N = o->N;
    compute_U1_J1_E1(o, U);
    memset(K, 0, 8 * N * sizeof(double));
    const double *rho = U, *p = U + N, *v = U + 2 * N, *B = U + 5 * N;
    const double *rho1 = o->U1, *p1 = o->U1 + N, *v1 = o->U1 + 2 * N, *B1 = o->U1 + 5 * N;
    const double *v0 = o->U0 + 2 * N;
    (void)B;
#pragma omp parallel for collapse(2) schedule(static)
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i) {
                size_t n = idx(o, i, k, j);
                double vv[3]  = { v[n],  v[N + n],  v[2 * N + n] };
                double vv1[3] = { v1[n], v1[N + n], v1[2 * N + n] };
                double vv0[3] = { v0[n], v0[N + n], v0[2 * N + n] };
                double BB[3]  = { U[5 * N + n], U[6 * N + n], U[7 * N + n] };
                double BB1[3] = { B1[n], B1[N + n], B1[2 * N + n] };
                double JJ1[3] = { o->J1[n], o->J1[N + n], o->J1[2 * N + n] };
                double JJ0[3] = { o->J0[n], o->J0[N + n], o->J0[2 * N + n] };
                double g[3], g1[3];
                double divv1 = divergence(o, v1, i, k, j);

                /* eq (11): d_t rho = -div(rho v1 + rho1 v0) + div[D grad(rho - rho0)] */
                grad(o, rho, i, k, j, g);
                grad(o, rho1, i, k, j, g1);
                K[n] = -(dot3(vv1, g) + rho[n] * divv1 + dot3(vv0, g1) + rho1[n] * o->divv0[n])
                       + o->D * laplacian(o, rho1, i, k, j);

                /* eq (12): d_t p = -v1.grad p - v0.grad p1 - Gamma(p div v1 + p1 div v0)
                 *                        + div[kappa grad(p - p0)]                           */
                grad(o, p, i, k, j, g);
                grad(o, p1, i, k, j, g1);       /* g1 = grad p1, reused in eq (13) */
                K[N + n] = -dot3(vv1, g) - dot3(vv0, g1)
                           - o->gamma * (p[n] * divv1 + p1[n] * o->divv0[n])
                           + o->kappa * laplacian(o, p1, i, k, j);

                /* eq (13): d_t v = -(v.grad v1 + v1.grad v0 + rho1 v0.grad v0 / rho)
                 *            + (J1 x B + J0 x B1 - grad p1)/rho + div[nu grad(v - v0)]       */
                double a1[3], a2[3], J1xB[3], J0xB1[3], L[3];
                advect_vector(o, vv, v1, i, k, j, a1);
                advect_vector(o, vv1, v0, i, k, j, a2);
                cross(JJ1, BB, J1xB);
                cross(JJ0, BB1, J0xB1);
                vector_laplacian(o, v1, i, k, j, L);
                for (int c = 0; c < 3; ++c)
                    K[(size_t)(2 + c) * N + n] =
                        -(a1[c] + a2[c] + rho1[n] * o->v0gv0[(size_t)c * N + n] / rho[n])
                        + (J1xB[c] + J0xB1[c] - g1[c]) / rho[n] + o->nu * L[c];

                /* eq (14): d_t B = -curl E1 (conservative curl, R4) */
                double cE[3];
                curl_c(o, o->E1, i, k, j, cE);
                for (int c = 0; c < 3; ++c) K[(size_t)(5 + c) * N + n] = -cE[c];
            }
}

void oracle_rhs(oracle *o, double *K) { oracle_rhs_of(o, o->U, K); }

/* ---------------------------------------------------------------------------------------- */
/* O5: classical RK4 (reading R7), written for any autonomous RHS so that pin P8 can run
 * du/dt = lambda u through this very routine.                                               */
typedef void (*oracle_rhs_fn)(void *user, const double *U, double *K);

void oracle_rk4(size_t len, double *U, double dt, int nsteps, oracle_rhs_fn f, void *user,
                double *K1, double *K2, double *K3, double *K4, double *Us)
{
    for (int s = 0; s < nsteps; ++s) {
        f(user, U, K1);
        for (size_t n = 0; n < len; ++n) Us[n] = U[n] + 0.5 * dt * K1[n];
        f(user, Us, K2);
        for (size_t n = 0; n < len; ++n) Us[n] = U[n] + 0.5 * dt * K2[n];
        f(user, Us, K3);
        for (size_t n = 0; n < len; ++n) Us[n] = U[n] + dt * K3[n];
        f(user, Us, K4);
        for (size_t n = 0; n < len; ++n)
            U[n] = U[n] + dt / 6.0 * (K1[n] + 2.0 * K2[n] + 2.0 * K3[n] + K4[n]);
    }
}

static void mhd_rhs_thunk(void *user, const double *U, double *K)
{
    oracle_rhs_of((oracle *)user, U, K);
}

/* n classical RK4 steps with the fixed dt (reading R8); the boundary layers never change
 * because K = 0 there.                                                                      */
void oracle_step(oracle *o, int n)
{
    oracle_rk4(8 * o->N, o->U, o->dt, n, mhd_rhs_thunk, o, o->K1, o->K2, o->K3, o->K4, o->Us);
    o->step += n;
    o->time += (double)n * o->dt;
}

/* ---------------------------------------------------------------------------------------- */
/* O6 diagnostics (reading R9).  out = { KE, ME, ME_pert, ME_n1, max|div_c B| }.
 * Sums over interior nodes, in long double; max over the deep interior i in [4,nR-5],
 * k in [4,nZ-5].                                                                            */
void oracle_diagnostics(oracle *o, double out[5])
{
    size_t N = o->N;
    const double *U = o->U;
    long double ke = 0.0L, me = 0.0L, mep = 0.0L, men1 = 0.0L;
    double maxdiv = 0.0;
    double dV = o->dR * o->dphi * o->dZ;
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i) {
                size_t n = idx(o, i, k, j);
                double w = o->R[i] * dV;
                double v2 = U[2 * N + n] * U[2 * N + n] + U[3 * N + n] * U[3 * N + n]
                            + U[4 * N + n] * U[4 * N + n];
                double b2 = U[5 * N + n] * U[5 * N + n] + U[6 * N + n] * U[6 * N + n]
                            + U[7 * N + n] * U[7 * N + n];
                double b1[3] = { U[5 * N + n] - o->U0[5 * N + n], U[6 * N + n] - o->U0[6 * N + n],
                                 U[7 * N + n] - o->U0[7 * N + n] };
                ke += (long double)(0.5 * U[n] * v2 * w);
                me += (long double)(0.5 * b2 * w);
                mep += (long double)(0.5 * (b1[0] * b1[0] + b1[1] * b1[1] + b1[2] * b1[2]) * w);
            }
    /* energy of the n = 1 toroidal harmonic of B1:  B1c ~ a cos(2 pi j/nphi) + b sin(..),
     * a, b = (2/nphi) sum_j B1c {cos, sin};  integral over phi of 1/2 (a cos + b sin)^2 R dphi
     * = 1/4 (a^2 + b^2) R Lphi                                                             */
    for (int k = 2; k <= o->nZ - 3; ++k)
        for (int i = 2; i <= o->nR - 3; ++i)
            for (int c = 0; c < 3; ++c) {
                long double a = 0.0L, b = 0.0L;
                for (int j = 0; j < o->nphi; ++j) {
                    size_t n = idx(o, i, k, j);
                    double b1 = U[(size_t)(5 + c) * N + n] - o->U0[(size_t)(5 + c) * N + n];
                    double ang = 2.0 * M_PI * (double)j / (double)o->nphi;
                    a += (long double)(b1 * cos(ang));
                    b += (long double)(b1 * sin(ang));
                }
                a *= 2.0L / (long double)o->nphi;
                b *= 2.0L / (long double)o->nphi;
                men1 += 0.25L * (a * a + b * b) * (long double)(o->R[i] * o->dR * o->dZ * o->Lphi);
            }
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 4; k <= o->nZ - 5; ++k)
            for (int i = 4; i <= o->nR - 5; ++i) {
                double d = fabs(div_c(o, U + 5 * N, i, k, j));
                if (d > maxdiv) maxdiv = d;
            }
    out[0] = (double)ke; out[1] = (double)me; out[2] = (double)mep; out[3] = (double)men1;
    out[4] = maxdiv;
}

/* div_c B at every interior node (0 elsewhere): lets tests look at div_c B(t) - div_c B(0). */
void oracle_divB(oracle *o, const double *U, double *out)
{
    size_t N = o->N;
    memset(out, 0, N * sizeof(double));
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i)
                out[idx(o, i, k, j)] = div_c(o, U + 5 * N, i, k, j);
}

/* SETDT, Fig. 4 (L180-215), transcribed: DT1 starts at 100; interior nodes FIRST+2..LAST-2;
 * the grid-type mask GDTP_EP (cut-cell boundary, L190) does not exist on a rectangular box.  */
double oracle_setdt(const oracle *o, double cfl)
{
    size_t N = o->N;
    const double *X = o->U;
    double dt1 = 100.0;
    for (int jy = 0; jy < o->nphi; ++jy)
        for (int jz = 2; jz <= o->nZ - 3; ++jz)
            for (int jx = 2; jx <= o->nR - 3; ++jx) {
                size_t n = idx(o, jx, jz, jy);
                double vx = X[2 * N + n], vy = X[3 * N + n], vz = X[4 * N + n];
                double va2 = (X[5 * N + n] * X[5 * N + n] + X[6 * N + n] * X[6 * N + n]
                              + X[7 * N + n] * X[7 * N + n]) / X[n];
                double cs2 = o->gamma * X[N + n] / X[n];
                double vpx = fabs(vx) + sqrt(fabs(cs2 + va2));
                double vpy = fabs(vy) + sqrt(fabs(cs2 + va2));
                double vpz = fabs(vz) + sqrt(fabs(cs2 + va2));
                double dtx = fabs(o->R[jx] - o->R[jx - 1]) / (vpx / cfl);
                double dtz = fabs(o->Z[jz] - o->Z[jz - 1]) / (vpz / cfl);
                double dty = fabs(o->R[jx] * o->dphi) / (vpy / cfl);
                double dt2 = fmin(dtx, dtz);
                double dt3 = fmin(dty, dt2);
                dt1 = fmin(dt1, dt3);
            }
    return dt1;
}

/* NEXT-1, adaptive time step [L139: "the time step ... is calculated based on the latest rho, p, v, B"; Fig. 3:
 * STEPON then SETDT inside the loop]: every RK4 step runs with dt = SETDT (Fig. 4) of the state at its start.  */
void oracle_step_cfl(oracle *o, int n, double cfl)
{
    for (int s = 0; s < n; ++s) {
        o->last_dt = oracle_setdt(o, cfl);
        oracle_rk4(8 * o->N, o->U, o->last_dt, 1, mhd_rhs_thunk, o, o->K1, o->K2, o->K3, o->K4, o->Us);
        o->step += 1;
        o->time += o->last_dt;
    }
}
double oracle_get_dt(const oracle *o) { return o->last_dt; }

/* ---------------------------------------------------------------------------------------- */
/* array-level wrappers around the point operators, so that the pins can exercise exactly the
 * functions the RHS uses.  which: 0 d1R, 1 d1P, 2 d1Z, 3 d2R, 4 d2P, 5 d2Z, 6 d1R_Rf,
 * 7 laplacian, 8 divergence(vector in), 9 div_c(vector in).  Output on interior nodes.       */
void oracle_apply_scalar_op(oracle *o, int which, const double *in, double *out)
{
    memset(out, 0, o->N * sizeof(double));
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i) {
                double r = 0.0;
                switch (which) {
                case 0: r = d1R(o, in, i, k, j); break;
                case 1: r = d1P(o, in, i, k, j); break;
                case 2: r = d1Z(o, in, i, k, j); break;
                case 3: r = d2R(o, in, i, k, j); break;
                case 4: r = d2P(o, in, i, k, j); break;
                case 5: r = d2Z(o, in, i, k, j); break;
                case 6: r = d1R_Rf(o, in, i, k, j); break;
                case 7: r = laplacian(o, in, i, k, j); break;
                case 8: r = divergence(o, in, i, k, j); break;
                case 9: r = div_c(o, in, i, k, j); break;
                default: break;
                }
                out[idx(o, i, k, j)] = r;
            }
}
/* which: 0 grad(scalar in, vector out), 1 curl_c, 2 vector_laplacian,
 * 3 (a.grad)b with in = [a(3 fields), b(3 fields)]                                          */
void oracle_apply_vector_op(oracle *o, int which, const double *in, double *out)
{
    size_t N = o->N;
    memset(out, 0, 3 * N * sizeof(double));
    for (int j = 0; j < o->nphi; ++j)
        for (int k = 2; k <= o->nZ - 3; ++k)
            for (int i = 2; i <= o->nR - 3; ++i) {
                size_t n = idx(o, i, k, j);
                double r[3] = { 0.0, 0.0, 0.0 };
                switch (which) {
                case 0: grad(o, in, i, k, j, r); break;
                case 1: curl_c(o, in, i, k, j, r); break;
                case 2: vector_laplacian(o, in, i, k, j, r); break;
                case 3: {
                    double a[3] = { in[n], in[N + n], in[2 * N + n] };
                    advect_vector(o, a, in + 3 * N, i, k, j, r);
                    break;
                }
                default: break;
                }
                out[n] = r[0]; out[N + n] = r[1]; out[2 * N + n] = r[2];
            }
}
