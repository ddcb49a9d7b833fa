/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain serial CPU Crank-Nicolson stepper for the 1-D TDSE in complex128, solved
 * with the Thomas algorithm.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call this file.  It
 * shares no code, header, table or helper with the CUDA path under
 * paper_2205_00856_b200/csrc/ and is never tuned for speed.
 *
 * What it computes is the paper's *definition* of one time step, which the
 * N-shaped partition method reaches exactly up to rounding (it is a direct
 * solver made of row operations only, App. I):
 *
 *   T psi(t+dt) = T^dagger psi(t),   T = 1 + (i dt/2) H          PAPER.md:48-52  Eq. 2
 *   explicit half-step  d = T^dagger psi                          PAPER.md:58     Eq. 3
 *   implicit half-step  T psi' = d                                PAPER.md:62     Eq. 4
 *   b_i psi_{i-1} + a_i psi_i + c_i psi_{i+1} = d_i,
 *   b_i = T_{i,i-1}, a_i = T_{i,i}, c_i = T_{i,i+1},
 *   psi_0 = psi_{n_tot+1} = 0 (reflecting)                        PAPER.md:80-84  Eq. 5
 *   solved serially by the Thomas algorithm
 *
 * Readings where the paper is silent:
 *   R3  (H psi)_j = -(psi_{j-1} - 2 psi_j + psi_{j+1}) / (2 dx^2) + V_j psi_j  (atomic units)
 *       => s = dt/(4 dx^2), b = c = -i s, a_j = 1 + i (2 s + dt V_j / 2).
 *   R4  T (with +i) multiplies the NEW psi.
 *   V real => T is complex symmetric => T^dagger = conj(T) element by element.
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): dense complex LU for N <= 64,
 * the closed-form Cayley phase of the discrete Dirichlet-Laplacian sine modes at V = 0,
 * norm conservation, per-step residual, time reversal.  No function here is "parity unpinned".
 *
 * Build: gcc -O2 -std=c11 -fPIC -shared -ffp-contract=off -fcx-limited-range  (no -ffast-math, no FTZ/DAZ).
 * -fcx-limited-range only selects the textbook 4-multiply complex product / quotient
 * instead of libgcc's NaN-recovering __muldc3/__divdc3; it allows no reordering.
 */
#define _POSIX_C_SOURCE 200809L
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <time.h>

typedef double complex zc;

/* ---- general complex tridiagonal system, Thomas algorithm (Eq. 5) ------------------
 * b[0] and c[n-1] are ignored (psi_{-1} = psi_n = 0).  d is overwritten by the solution.
 * scratch: n complex.  Returns 0, or 1 + row of a zero / non-finite pivot. */
int64_t cn_oracle_thomas(int64_t n, const zc *b, const zc *a, const zc *c, zc *d, zc *scratch)
{
    zc *cp = scratch;
    zc piv = a[0];
    if (!(cabs(piv) > 0.0) || !isfinite(cabs(piv))) return 1;
    cp[0] = c[0] / piv;
    d[0] = d[0] / piv;
    for (int64_t j = 1; j < n; ++j) {
        piv = a[j] - b[j] * cp[j - 1];
        if (!(cabs(piv) > 0.0) || !isfinite(cabs(piv))) return 1 + j;
        cp[j] = c[j] / piv;
        d[j] = (d[j] - b[j] * d[j - 1]) / piv;
    }
    for (int64_t j = n - 2; j >= 0; --j) d[j] = d[j] - cp[j] * d[j + 1];
    return 0;
}

/* ---- the three diagonals of T for the 3-point Hamiltonian (reading R3) --------------------------- */
void cn_oracle_diagonals(int64_t n, double dx, double dt, const double *V, zc *b, zc *a, zc *c)
{
    const double s = dt / (4.0 * dx * dx);
    for (int64_t j = 0; j < n; ++j) {
        b[j] = -I * s;
        c[j] = -I * s;
        a[j] = 1.0 + I * (2.0 * s + 0.5 * dt * V[j]);
    }
}

/* ---- explicit half-step d = T^dagger psi = conj(T) psi (Eq. 3) ---------------------------------- */
void cn_oracle_rhs(int64_t n, const zc *b, const zc *a, const zc *c, const zc *psi, zc *d)
{
    for (int64_t j = 0; j < n; ++j) {
        zc lo = (j > 0) ? psi[j - 1] : 0.0;
        zc hi = (j < n - 1) ? psi[j + 1] : 0.0;
        d[j] = conj(b[j]) * lo + conj(a[j]) * psi[j] + conj(c[j]) * hi;
    }
}

/* ---- precomputed Thomas coefficients of T (still plain Thomas: SURVEY 8c-3) ------------------------ */
typedef struct { int64_t n; zc *b, *a, *c, *cp, *ip, *d; } cn_oracle_sys;

static void sys_free(cn_oracle_sys *S)
{
    free(S->b); free(S->a); free(S->c); free(S->cp); free(S->ip); free(S->d);
    memset(S, 0, sizeof *S);
}

static int64_t sys_init(cn_oracle_sys *S, int64_t n, double dx, double dt, const double *V)
{
    memset(S, 0, sizeof *S);
    S->n = n;
    S->b = malloc(sizeof(zc) * n); S->a = malloc(sizeof(zc) * n); S->c = malloc(sizeof(zc) * n);
    S->cp = malloc(sizeof(zc) * n); S->ip = malloc(sizeof(zc) * n); S->d = malloc(sizeof(zc) * n);
    if (!S->b || !S->a || !S->c || !S->cp || !S->ip || !S->d) { sys_free(S); return -1; }
    cn_oracle_diagonals(n, dx, dt, V, S->b, S->a, S->c);
    zc piv = S->a[0];
    if (!(cabs(piv) > 0.0)) { sys_free(S); return 1; }
    S->ip[0] = 1.0 / piv;
    S->cp[0] = S->c[0] * S->ip[0];
    for (int64_t j = 1; j < n; ++j) {
        piv = S->a[j] - S->b[j] * S->cp[j - 1];
        if (!(cabs(piv) > 0.0) || !isfinite(cabs(piv))) { sys_free(S); return 1 + j; }
        S->ip[j] = 1.0 / piv;
        S->cp[j] = S->c[j] * S->ip[j];
    }
    return 0;
}

/* one CN step of one system; psi has `stride` complex elements between consecutive rows */
static void sys_step(const cn_oracle_sys *S, zc *psi, int64_t stride)
{
    const int64_t n = S->n;
    const zc *b = S->b, *a = S->a, *c = S->c, *cp = S->cp, *ip = S->ip;
    zc *d = S->d;
    /* Eq. 3 */
    for (int64_t j = 0; j < n; ++j) {
        zc lo = (j > 0) ? psi[(j - 1) * stride] : 0.0;
        zc hi = (j < n - 1) ? psi[(j + 1) * stride] : 0.0;
        d[j] = conj(b[j]) * lo + conj(a[j]) * psi[j * stride] + conj(c[j]) * hi;
    }
    /* Eq. 4 by Thomas: forward elimination, back substitution */
    d[0] = d[0] * ip[0];
    for (int64_t j = 1; j < n; ++j) d[j] = (d[j] - b[j] * d[j - 1]) * ip[j];
    psi[(n - 1) * stride] = d[n - 1];
    for (int64_t j = n - 2; j >= 0; --j) psi[j * stride] = d[j] - cp[j] * psi[(j + 1) * stride];
}

static double now_s(void)
{
    struct timespec t;
    clock_gettime(CLOCK_MONOTONIC, &t);
    return (double)t.tv_sec + 1e-9 * (double)t.tv_nsec;
}

/* ---- nsteps CN steps of one system, full variant (6 n-vectors) -----------------------------------
 * `seconds_out` times the step loop only (precompute excluded). */
int64_t cn_oracle_step(int64_t n, double dx, double dt, const double *V, zc *psi, int64_t stride,
                       int64_t nsteps, double *seconds_out)
{
    cn_oracle_sys S;
    int64_t rc = sys_init(&S, n, dx, dt, V);
    if (rc) return rc;
    double t0 = now_s();
    for (int64_t k = 0; k < nsteps; ++k) sys_step(&S, psi, stride);
    if (seconds_out) *seconds_out = now_s() - t0;
    sys_free(&S);
    return 0;
}

/* ---- lean variant for n >= 2^29: keeps only psi and the inverse pivots -------------
 * c'_j = c * ip_j with the constant c = -i s; Eq. 3 is folded into the forward sweep with a
 * one-element carry of the old psi.  Same arithmetic, same order, 2 n-vectors instead of 6. */
int64_t cn_oracle_step_lean(int64_t n, double dx, double dt, const double *V, zc *psi, int64_t nsteps,
                            double *seconds_out)
{
    const double s = dt / (4.0 * dx * dx);
    const zc b = -I * s, c = -I * s;
    zc *ip = malloc(sizeof(zc) * n);
    if (!ip) return -1;
    {
        zc piv = 1.0 + I * (2.0 * s + 0.5 * dt * V[0]);
        ip[0] = 1.0 / piv;
        for (int64_t j = 1; j < n; ++j) {
            piv = (1.0 + I * (2.0 * s + 0.5 * dt * V[j])) - b * (c * ip[j - 1]);
            if (!(cabs(piv) > 0.0) || !isfinite(cabs(piv))) { free(ip); return 1 + j; }
            ip[j] = 1.0 / piv;
        }
    }
    double t0 = now_s();
    for (int64_t k = 0; k < nsteps; ++k) {
        zc old_prev = 0.0;   /* psi_{j-1} of the OLD state */
        zc dprev = 0.0;      /* d'_{j-1} */
        for (int64_t j = 0; j < n; ++j) {
            zc cur = psi[j];
            zc hi = (j < n - 1) ? psi[j + 1] : 0.0;
            zc aj = 1.0 + I * (2.0 * s + 0.5 * dt * V[j]);
            zc dj = conj(b) * old_prev + conj(aj) * cur + conj(c) * hi;
            dprev = (dj - b * dprev) * ip[j];
            psi[j] = dprev;          /* psi now holds d' */
            old_prev = cur;
        }
        for (int64_t j = n - 2; j >= 0; --j) psi[j] = psi[j] - (c * ip[j]) * psi[j + 1];
    }
    if (seconds_out) *seconds_out = now_s() - t0;
    free(ip);
    return 0;
}

/* ---- C4: Lie-split 2-D step  psi <- CN_y(dt) CN_x(dt) psi  (reading R18) -------------
 * psi is row-major psi[y][x], ny rows of nx.  Vx: nx values, Vy: ny values (separable potential).
 * Plain loops over the independent systems; no OpenMP in the correctness oracle. */
int64_t cn_oracle_step_2d(int64_t nx, int64_t ny, double dx, double dt, const double *Vx, const double *Vy,
                          zc *psi, int64_t nsteps, double *seconds_out)
{
    cn_oracle_sys Sx, Sy;
    int64_t rc = sys_init(&Sx, nx, dx, dt, Vx);
    if (rc) return rc;
    rc = sys_init(&Sy, ny, dx, dt, Vy);
    if (rc) { sys_free(&Sx); return rc; }
    double t0 = now_s();
    for (int64_t k = 0; k < nsteps; ++k) {
        for (int64_t y = 0; y < ny; ++y) sys_step(&Sx, psi + y * nx, 1);
        for (int64_t x = 0; x < nx; ++x) sys_step(&Sy, psi + x, nx);
    }
    double acc = now_s() - t0;
    sys_free(&Sx); sys_free(&Sy);
    if (seconds_out) *seconds_out = acc;
    return 0;
}

/* ---- C4 timed on all host cores (SURVEY 8d "Oracle timing") ------------------------
 * The SAME 2-D step with the independent systems of a sweep shared out over OpenMP threads (static schedule);
 * compiled only with -fopenmp into libcn_oracle_omp.so.  Every thread runs the unchanged serial sys_step on its
 * systems with a scratch vector of its own, so the result is bit-identical to cn_oracle_step_2d
 * (tests/test_oracle_pins.py::test_step_2d_omp_is_bitwise_serial).  A CPU-baseline timing aid: parity tests use the
 * serial function above. */
#ifdef _OPENMP
#include <omp.h>
int64_t cn_oracle_step_2d_omp(int64_t nx, int64_t ny, double dx, double dt, const double *Vx, const double *Vy,
                              zc *psi, int64_t nsteps, double *seconds_out, int64_t *threads_out)
{
    cn_oracle_sys Sx, Sy;
    int64_t rc = sys_init(&Sx, nx, dx, dt, Vx);
    if (rc) return rc;
    rc = sys_init(&Sy, ny, dx, dt, Vy);
    if (rc) { sys_free(&Sx); return rc; }
    int64_t bad = 0, nthreads = 1;
    double t0 = now_s();
#pragma omp parallel
    {
        cn_oracle_sys Lx = Sx, Ly = Sy; /* shared read-only coefficients, private right-hand-side scratch */
        Lx.d = malloc(sizeof(zc) * nx);
        Ly.d = malloc(sizeof(zc) * ny);
        if (!Lx.d || !Ly.d) {
#pragma omp atomic write
            bad = 1;
        }
#pragma omp single
        nthreads = omp_get_num_threads();
#pragma omp barrier
        if (!bad) {
            for (int64_t k = 0; k < nsteps; ++k) {
#pragma omp for schedule(static)
                for (int64_t y = 0; y < ny; ++y) sys_step(&Lx, psi + y * nx, 1);
#pragma omp for schedule(static)
                for (int64_t x = 0; x < nx; ++x) sys_step(&Ly, psi + x, nx);
            }
        }
        free(Lx.d);
        free(Ly.d);
    }
    double acc = now_s() - t0;
    sys_free(&Sx); sys_free(&Sy);
    if (seconds_out) *seconds_out = acc;
    if (threads_out) *threads_out = nthreads;
    return bad ? -1 : 0;
}
#endif
