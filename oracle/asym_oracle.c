/*
 * asym_oracle.c -- CPU oracle for the explicit asymptotic kinetic-network step.
 *
 * TEST INFRASTRUCTURE ONLY.  Plain, slow, scalar C; it exists to say what the
 * CUDA path must compute.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build or call it.  It
 * shares no code, header, table or constant with paper_1409_5826_b200/.
 *
 * What it follows (P:Lnn = /root/reference/PAPER.md line nn; S:Qn / S:On =
 * SURVEY.md section 8(c) reading / oracle step, restated in DESIGN.md):
 *   O1 setup        statistical prefactor 1/prod(m!) and one edge per distinct
 *                   (reaction, species, side)                         S:Q2
 *   O2 rates        7-parameter exponential in T9, rho^(n-1), once per zone
 *                   per call                      P:L104, L197, L202; S:Q1
 *   O4 fluxes       f_r = R_r * prod Y_reactants (start-of-step Y)
 *   O5 sums         F+_i, F-_i over the edge list            P:L49-53 Eq. (1)
 *   O6 dt control   a-priori accuracy controller                 S:Q7, Q9-Q11
 *   O7 update       k dt >= kappa -> Eq. (3), else forward Euler; Jacobi
 *                                                   P:L61-69 Eq. (3); S:Q4-Q6,Q8
 *   O8/O9 advance, outputs
 *   method = 1      the QSS variant of O7 named as future work in P:L217-219.  The paper
 *                   gives no formula (its ref. [5] is not in the container): DESIGN.md
 *                   reading Q20 takes the predictor of the published alpha-QSS scheme,
 *                   y' = y + dt (F+ - k y)/(1 + alpha k dt) with the Pade alpha, for every
 *                   species, behind the same fluxes, sums and dt controller.  Pinned by
 *                   hand-worked per-step factors, the exact e^{-k dt} it approximates, the
 *                   two-species fixed point, the Euler limit and RK4 on a tiny network.
 *
 * Precision: double throughout.  precision == 32 is the paper's single-
 * precision study (S:Q13): Y, f, F+, F-, k and the update in float;
 * rates evaluated in double then rounded; t, dt and the dt minimum in double.
 *
 * Pins (tests/test_oracle_pins.py): P1 rate special cases and long-double
 * cross-check; P2 discrete closed forms of a single decay in both branches;
 * P3 continuum exp(-kt); P4 two-species fixed point; P5 sum(A Y) in the Euler
 * regime; P6 positivity; P7 brute-force small-dt Euler; P8 dense-matrix linear
 * networks; P9 permutation invariance; P10 three-body multiplicity.
 * precision == 32 has no bound in the paper: PARITY UNPINNED for it.
 *
 * precision == 80 is the ARBITER: the same O1-O9, textually the same sub-step, with
 * Y, f, F+, F-, k, the update, the rates (cbrtl/logl/expl), t, dt and the dt minimum
 * in x87 long double (64-bit significand).  It is not a different method and not a
 * reference for the CUDA path's arithmetic; it answers one question in the parity
 * tests: in a zone where the adaptive trajectory amplifies rounding,
 * is the CUDA result as close to the extended-precision trajectory as the fp64
 * oracle's own results are?  Abundances go in and come out as double.  Pinned by
 * the same closed forms as precision 64 (tests/test_oracle_pins.py).
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC (oracle/build.py).
 * OpenMP only runs independent zones on different cores; it never touches the
 * arithmetic of one zone.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define MAX_REACT 3
#define MAX_PROD 4
#define N_COEF 7

typedef struct {
    double kappa;        /* branch threshold on k*dt, P:L65 (kappa = 1)          */
    double eps_y;        /* max relative explicit change per step, S:Q7          */
    double y_floor;      /* abundance floor inside the dt controller, S:Q7       */
    double growth;       /* dt growth cap per step, S:Q7                         */
    long long max_steps; /* per call; status bit 1 when hit                      */
    int method;          /* 0 = asymptotic / forward Euler (the paper's method);
                            1 = explicit quasi-steady-state variant, P:L217-219     */
} oracle_params;

typedef struct {
    int r;    /* reaction             */
    int i;    /* species              */
    int sign; /* +1 product, -1 reactant */
    int nu;   /* multiplicity of i on that side */
} edge_t;

typedef struct {
    int N, M, n_edges;
    int *A;
    int *n_react, *react; /* [M], [M*3] */
    double *coef;         /* [M*7]      */
    double *ln_pref;      /* [M] ln(1/prod m!) */
    long double *ln_pref_ld; /* the same in long double (arbiter) */
    edge_t *edges;
    oracle_params p;
} oracle_net;

void oracle_default_params(oracle_params *p) {
    p->kappa = 1.0;
    p->eps_y = 0.05;
    p->y_floor = 1e-10;
    p->growth = 2.0;
    p->max_steps = 10000000LL;
    p->method = 0;
}

static double ln_factorial(int m) {
    double s = 0.0;
    for (int q = 2; q <= m; ++q) s += log((double)q);
    return s;
}

static long double ln_factorial_ld(int m) {
    long double s = 0.0L;
    for (int q = 2; q <= m; ++q) s += logl((long double)q);
    return s;
}

/* O1.  Returns NULL on invalid tables. */
void *oracle_create(int N, const int *A, int M, const int *n_react, const int *react,
                    const int *n_prod, const int *prod, const double *coef,
                    const oracle_params *params) {
    if (N <= 0 || M < 0) return NULL;
    for (int r = 0; r < M; ++r) {
        if (n_react[r] < 1 || n_react[r] > MAX_REACT) return NULL;
        if (n_prod[r] < 1 || n_prod[r] > MAX_PROD) return NULL;
        long sa = 0;
        for (int q = 0; q < n_react[r]; ++q) {
            int s = react[r * MAX_REACT + q];
            if (s < 0 || s >= N) return NULL;
            sa += A[s];
        }
        for (int q = 0; q < n_prod[r]; ++q) {
            int s = prod[r * MAX_PROD + q];
            if (s < 0 || s >= N) return NULL;
            sa -= A[s];
        }
        if (sa != 0) return NULL;
    }
    oracle_net *net = (oracle_net *)calloc(1, sizeof(oracle_net));
    net->N = N;
    net->M = M;
    net->A = (int *)malloc(sizeof(int) * N);
    memcpy(net->A, A, sizeof(int) * N);
    net->n_react = (int *)malloc(sizeof(int) * (M + 1));
    net->react = (int *)malloc(sizeof(int) * (M * MAX_REACT + 1));
    net->coef = (double *)malloc(sizeof(double) * (M * N_COEF + 1));
    net->ln_pref = (double *)malloc(sizeof(double) * (M + 1));
    net->ln_pref_ld = (long double *)malloc(sizeof(long double) * (M + 1));
    net->edges = (edge_t *)malloc(sizeof(edge_t) * (M * (MAX_REACT + MAX_PROD) + 1));
    memcpy(net->n_react, n_react, sizeof(int) * M);
    memcpy(net->react, react, sizeof(int) * M * MAX_REACT);
    memcpy(net->coef, coef, sizeof(double) * M * N_COEF);
    if (params) net->p = *params; else oracle_default_params(&net->p);

    int ne = 0;
    for (int r = 0; r < M; ++r) {
        double lp = 0.0;
        long double lp_ld = 0.0L;
        /* reactant side: one edge per distinct species, nu = multiplicity */
        for (int q = 0; q < n_react[r]; ++q) {
            int s = react[r * MAX_REACT + q], first = 1, m = 0;
            for (int u = 0; u < q; ++u) if (react[r * MAX_REACT + u] == s) first = 0;
            if (!first) continue;
            for (int u = 0; u < n_react[r]; ++u) if (react[r * MAX_REACT + u] == s) ++m;
            lp -= ln_factorial(m);
            lp_ld -= ln_factorial_ld(m);
            net->edges[ne++] = (edge_t){r, s, -1, m};
        }
        for (int q = 0; q < n_prod[r]; ++q) {
            int s = prod[r * MAX_PROD + q], first = 1, m = 0;
            for (int u = 0; u < q; ++u) if (prod[r * MAX_PROD + u] == s) first = 0;
            if (!first) continue;
            for (int u = 0; u < n_prod[r]; ++u) if (prod[r * MAX_PROD + u] == s) ++m;
            net->edges[ne++] = (edge_t){r, s, +1, m};
        }
        net->ln_pref[r] = lp;
        net->ln_pref_ld[r] = lp_ld;
    }
    net->n_edges = ne;
    return net;
}

void oracle_destroy(void *h) {
    oracle_net *net = (oracle_net *)h;
    if (!net) return;
    free(net->A); free(net->n_react); free(net->react); free(net->coef);
    free(net->ln_pref); free(net->ln_pref_ld); free(net->edges); free(net);
}

int oracle_num_edges(void *h) { return ((oracle_net *)h)->n_edges; }

/* O2: R_r = exp(ln p_r + (n_r - 1) ln rho + a0 + a1/T9 + a2/T9^(1/3)
 *               + a3 T9^(1/3) + a4 T9 + a5 T9^(5/3) + a6 ln T9). */
int oracle_rates(void *h, double T9, double rho, double *R) {
    oracle_net *net = (oracle_net *)h;
    double t13 = cbrt(T9);
    double t53 = T9 * t13 * t13;
    double lnT = log(T9), lnrho = log(rho);
    for (int r = 0; r < net->M; ++r) {
        const double *a = net->coef + r * N_COEF;
        double lnR = a[0] + a[1] / T9 + a[2] / t13 + a[3] * t13 + a[4] * T9 + a[5] * t53 +
                     a[6] * lnT;
        R[r] = exp(net->ln_pref[r] + (double)(net->n_react[r] - 1) * lnrho + lnR);
    }
    return 0;
}

/* O2 in long double (arbiter). */
static void rates_ld(const oracle_net *net, double T9d, double rhod, long double *R) {
    long double T9 = (long double)T9d, rho = (long double)rhod;
    long double t13 = cbrtl(T9);
    long double t53 = T9 * t13 * t13;
    long double lnT = logl(T9), lnrho = logl(rho);
    for (int r = 0; r < net->M; ++r) {
        const double *a = net->coef + r * N_COEF;
        long double lnR = (long double)a[0] + (long double)a[1] / T9 + (long double)a[2] / t13 +
                          (long double)a[3] * t13 + (long double)a[4] * T9 +
                          (long double)a[5] * t53 + (long double)a[6] * lnT;
        R[r] = expl(net->ln_pref_ld[r] + (long double)(net->n_react[r] - 1) * lnrho + lnR);
    }
}

/* Exposed for the pins of the arbiter (R: [M] long double). */
int oracle_rates_ld(void *h, double T9, double rho, long double *R) {
    rates_ld((oracle_net *)h, T9, rho, R);
    return 0;
}

/* ---- the sub-step, written once per state type ------------------------- */
#define REAL double
#define RATE double
#define TIME double
#define SUFFIX(name) name##_f64
#include "asym_substep.inc"
#undef REAL
#undef SUFFIX
#define REAL float
#define SUFFIX(name) name##_f32
#include "asym_substep.inc"
#undef REAL
#undef RATE
#undef TIME
#undef SUFFIX
#define REAL long double
#define RATE long double
#define TIME long double
#define SUFFIX(name) name##_f80
#include "asym_substep.inc"
#undef REAL
#undef RATE
#undef TIME
#undef SUFFIX

/* O4+O5 exposed for the pins: fluxes and sums for one state (double). */
int oracle_rhs(void *h, const double *R, const double *Y, double *f, double *Fp, double *Fm) {
    rhs_f64((oracle_net *)h, R, Y, f, Fp, Fm);
    return 0;
}

static int run_zones(oracle_net *net, int zones, const double *T9, const double *rho, void *Y,
                     int adaptive, double t_hydro, double *dt, double dt_fixed,
                     long long n_fixed, long long *n_steps, int *status, long long *n_asym,
                     int precision, int n_threads) {
    if (precision != 64 && precision != 32 && precision != 80) return -1;
    if (n_threads < 1) n_threads = 1;
    int N = net->N, M = net->M;
#ifdef _OPENMP
#pragma omp parallel num_threads(n_threads)
#endif
    {
        double *R = (double *)malloc(sizeof(double) * (M + 1));
        void *work = malloc(sizeof(long double) * (size_t)(M + 4 * N + 4));
        long double *R_ld = (long double *)malloc(sizeof(long double) * (M + 1));
        long double *Y_ld = (long double *)malloc(sizeof(long double) * (N + 1));
#ifdef _OPENMP
#pragma omp for schedule(dynamic, 1)
#endif
        for (int z = 0; z < zones; ++z) {
            if (precision == 80) rates_ld(net, T9[z], rho[z], R_ld);
            else oracle_rates(net, T9[z], rho[z], R);
            double dt_io = (dt != NULL) ? dt[z] : 0.0;
            long long steps = 0, asym = 0;
            int st;
            if (precision == 64)
                st = zone_f64(net, R, (double *)Y + (size_t)z * N, adaptive, t_hydro, &dt_io,
                              dt_fixed, n_fixed, &steps, &asym, work);
            else if (precision == 32)
                st = zone_f32(net, R, (float *)Y + (size_t)z * N, adaptive, t_hydro, &dt_io,
                              dt_fixed, n_fixed, &steps, &asym, work);
            else { /* arbiter: abundances in and out as double */
                double *Yz = (double *)Y + (size_t)z * N;
                for (int i = 0; i < N; ++i) Y_ld[i] = (long double)Yz[i];
                st = zone_f80(net, R_ld, Y_ld, adaptive, t_hydro, &dt_io, dt_fixed, n_fixed,
                              &steps, &asym, work);
                for (int i = 0; i < N; ++i) Yz[i] = (double)Y_ld[i];
            }
            if (dt) dt[z] = dt_io;
            if (n_steps) n_steps[z] = steps;
            if (status) status[z] = st;
            if (n_asym) n_asym[z] = asym;
        }
        free(R);
        free(work);
        free(R_ld);
        free(Y_ld);
    }
    return 0;
}

/* One hydro step for every zone, adaptive dt (O3-O9).  Y is [zones*N],
 * double or float according to precision; dt in/out may be NULL. */
int oracle_integrate(void *h, int zones, const double *T9, const double *rho, void *Y,
                     double t_hydro, double *dt, long long *n_steps, int *status,
                     long long *n_asym, int precision, int n_threads) {
    return run_zones((oracle_net *)h, zones, T9, rho, Y, 1, t_hydro, dt, 0.0, 0, n_steps,
                     status, n_asym, precision, n_threads);
}

/* Exactly n_steps sub-steps of size dt_fixed (O9, fixed-dt mode). */
int oracle_integrate_fixed(void *h, int zones, const double *T9, const double *rho, void *Y,
                           double dt_fixed, long long n_steps, long long *n_asym,
                           int precision, int n_threads) {
    return run_zones((oracle_net *)h, zones, T9, rho, Y, 0, 0.0, NULL, dt_fixed, n_steps,
                     NULL, NULL, n_asym, precision, n_threads);
}

int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
