/*
 * sso_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * A plain, slow, double-precision CPU implementation of one Fourier
 * split-operator time step, written directly from the paper
 * (Bauke & Keitel, arXiv:1012.3911; line numbers refer to PAPER.md) and the
 * readings listed in DESIGN.md ("Readings of the paper", G1..G28).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or constant with paper_1012_3911_b200/csrc (the CUDA product)
 * and neither includes the other.
 *
 * What it computes (one step, step index n, tau = dt):
 *   1. psi_c(r) <- exp(-i Vbar_n(r) tau/2) psi_c(r)      PAPER.md:98 (eq. 11, delta=1/2), 165 (eq. 22)
 *   2. psi~_c(k) = sum_j psi_c(r_j) exp(-2 pi i j.l/n)    PAPER.md:103 (eq. 12: forward = minus sign), 80
 *   3. Schroedinger: psi~ <- exp(-i tau sum_a (k_a - q Abar_a)^2 / 2m) psi~     PAPER.md:107 (eq. 13, delta=1)
 *      Dirac:        psi~ <- u(p)^+ diag(e^{-iE tau}.., e^{+iE tau}..) u(p) psi~ PAPER.md:211-232 (eq. 29-33), 240-242 (eq. 35)
 *   4. psi_c(r) = (1/N) sum_k psi~_c(k) exp(+2 pi i ...)   PAPER.md:76-78 (eq. 8)
 *   5. step 1 again with the same Vbar_n                   PAPER.md:71 (eq. 7: U_A1(t+tau,t,1/2) appears twice)
 *
 * There is no blocking, fusion or re-ordering beyond that: no merged half
 * steps, no phase tables, no closed-form Dirac exponential (the CUDA path uses
 * cos/sin; this file uses the paper's Foldy-Wouthuysen form, eq. 29-33).
 *
 * The FFT is a textbook recursive radix-2 decimation-in-time transform whose
 * twiddles are evaluated directly (cos/sin of each angle, no recurrence); it is
 * pinned to the O(N^2) DFT definition in tests/test_oracle_pins.py.
 *
 * Parity pins (tests/test_oracle_pins.py): naive DFT, F^-1 F = id, Parseval,
 * free Gaussian closed form, harmonic-well Stoermer-Verlet centroid, norm
 * conservation, reversibility, eq. 15 algebra for eq. 16/17 (matrices typed
 * from the paper in tests/golden/), expm(-iH tau) by brute force, free Dirac
 * dispersion E = +-sqrt(c^2 k^2 + c^4), field plumbing.  Full-size configs
 * 2..5 have no paper value to compare to: "parity unpinned beyond oracle +
 * invariants" for those.
 *
 * Observables (end of file): overlap / autocorrelation
 * chi(t) (eq. 40), <r>, <p>, windowed spectrum (eq. 41), eigenfunction filter
 * (eq. 42), each the plain sum.  Pins (tests/test_oracle_observables.py):
 * Gaussian-overlap closed form, plane-wave autocorrelation, packet centroid
 * and momentum, Stoermer-Verlet kick, exact Hann-window identities, and the
 * paper's soft-core ground-state energy -Z^2/2 for zeta = 1.4133 (1D) and
 * 0.791 (2D) through the whole chi -> spectrum -> filter
 * chain.
 *
 * Units: atomic units, hbar = 1.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define ORC_FIELD_NONE 0
#define ORC_FIELD_E 1 /* adds r . Ebar_n to the potential energy (length gauge) */
#define ORC_FIELD_A 2 /* pi = k - q Abar_n in the kinetic factor            */

/* ------------------------------------------------------------------ */
/* threads                                                             */
/* ------------------------------------------------------------------ */
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

/* ------------------------------------------------------------------ */
/* FFT: recursive radix-2, directly evaluated twiddles                 */
/* X_l = sum_j x_j exp(sign * 2 pi i j l / n),  sign = -1 forward       */
/* (eq. 12), +1 inverse (unscaled here).                 */
/* ------------------------------------------------------------------ */

/* w[m] = exp(sign 2 pi i m / n), m < n/2, each angle evaluated on its own */
static cplx *make_twiddles(int64_t n, int sign) {
    int64_t h = n / 2 > 0 ? n / 2 : 1;
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)h);
    for (int64_t m = 0; m < h; ++m) {
        double ang = (double)sign * 2.0 * M_PI * (double)m / (double)n;
        w[m] = cos(ang) + I * sin(ang);
    }
    return w;
}

/* out[0..n) = DFT of in[0], in[s], in[2s], ...; w holds the size-(n*ws) table */
static void fft_rec(const cplx *in, int64_t s, cplx *out, int64_t n, const cplx *w, int64_t ws) {
    if (n == 1) {
        out[0] = in[0];
        return;
    }
    int64_t h = n / 2;
    fft_rec(in, 2 * s, out, h, w, 2 * ws);         /* even samples -> out[0..h)  */
    fft_rec(in + s, 2 * s, out + h, h, w, 2 * ws); /* odd samples  -> out[h..n)  */
    for (int64_t l = 0; l < h; ++l) {
        cplx e = out[l];
        cplx o = w[l * ws] * out[l + h];
        out[l] = e + o;
        out[l + h] = e - o;
    }
}

/* transform every line along `axis` of a C-ordered array of shape n[0..ndim) */
static void fft_axis(cplx *x, int ndim, const int64_t *n, int axis, int sign) {
    int64_t len = n[axis];
    int64_t inner = 1, outer = 1;
    for (int a = axis + 1; a < ndim; ++a) inner *= n[a];
    for (int a = 0; a < axis; ++a) outer *= n[a];
    cplx *w = make_twiddles(len, sign);
    int64_t nlines = outer * inner;
#pragma omp parallel
    {
        cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)len * 2);
        cplx *res = buf + len;
#pragma omp for schedule(static)
        for (int64_t L = 0; L < nlines; ++L) {
            int64_t o = L / inner, i = L % inner;
            cplx *base = x + o * len * inner + i;
            for (int64_t j = 0; j < len; ++j) buf[j] = base[j * inner];
            fft_rec(buf, 1, res, len, w, 1);
            for (int64_t j = 0; j < len; ++j) base[j * inner] = res[j];
        }
        free(buf);
    }
    free(w);
}

/* N-d transform, sign=-1: unnormalised forward; sign=+1: inverse including 1/N */
void orc_fft(double *xri, int ndim, const int64_t *n, int sign) {
    cplx *x = (cplx *)xri;
    int64_t N = 1;
    for (int a = 0; a < ndim; ++a) N *= n[a];
    for (int a = 0; a < ndim; ++a) fft_axis(x, ndim, n, a, sign);
    if (sign > 0) {
        double inv = 1.0 / (double)N;
#pragma omp parallel for schedule(static)
        for (int64_t j = 0; j < N; ++j) x[j] *= inv;
    }
}

/* ------------------------------------------------------------------ */
/* grids (G14): r_j = (j - n/2) dx, half open;               */
/* k_j = 2 pi j/(n dx) for j < n/2, 2 pi (j-n)/(n dx) for j >= n/2     */
/* ------------------------------------------------------------------ */
static double r_of(int64_t j, int64_t n, double dx) { return ((double)j - (double)(n / 2)) * dx; }
static double k_of(int64_t j, int64_t n, double dx) {
    int64_t jj = (j < n / 2) ? j : j - n;
    return 2.0 * M_PI * (double)jj / ((double)n * dx);
}
void orc_grids(int64_t n, double dx, double *r, double *k) {
    for (int64_t j = 0; j < n; ++j) {
        r[j] = r_of(j, n, dx);
        k[j] = k_of(j, n, dx);
    }
}

/* ------------------------------------------------------------------ */
/* Dirac matrices                                                      */
/* ncomp = 4: eq. 16; ncomp = 2: eq. 17             */
/* alpha1 = sigma_x, beta = sigma_z, and for two    */
/* dimensions alpha2 = sigma_y (G7: the {1,4} block of       */
/* eq. 16 at p3 = 0).                                                  */
/* out: [4][ncomp][ncomp] = alpha1, alpha2, alpha3, beta (row major);  */
/* alpha3 is zero for ncomp = 2.                                       */
/* ------------------------------------------------------------------ */
static void dirac_matrices(int ncomp, cplx *al /*[3][C][C]*/, cplx *be /*[C][C]*/) {
    int C = ncomp;
    memset(al, 0, sizeof(cplx) * 3 * C * C);
    memset(be, 0, sizeof(cplx) * C * C);
#define AL(i, r, c) al[((i)*C + (r)) * C + (c)]
#define BE(r, c) be[(r)*C + (c)]
    if (C == 4) {
        /* alpha_1 */
        AL(0, 0, 3) = 1; AL(0, 1, 2) = 1; AL(0, 2, 1) = 1; AL(0, 3, 0) = 1;
        /* alpha_2 */
        AL(1, 0, 3) = -I; AL(1, 1, 2) = I; AL(1, 2, 1) = -I; AL(1, 3, 0) = I;
        /* alpha_3 */
        AL(2, 0, 2) = 1; AL(2, 1, 3) = -1; AL(2, 2, 0) = 1; AL(2, 3, 1) = -1;
        /* beta */
        BE(0, 0) = 1; BE(1, 1) = 1; BE(2, 2) = -1; BE(3, 3) = -1;
    } else {
        AL(0, 0, 1) = 1; AL(0, 1, 0) = 1;  /* sigma_x */
        AL(1, 0, 1) = -I; AL(1, 1, 0) = I; /* sigma_y */
        BE(0, 0) = 1; BE(1, 1) = -1;       /* sigma_z */
    }
#undef AL
#undef BE
}

void orc_dirac_matrices(int ncomp, double *out_ri /* [4][C][C] complex */) {
    cplx *out = (cplx *)out_ri;
    dirac_matrices(ncomp, out, out + 3 * ncomp * ncomp);
}

/*
 * U(p) = u(p)^+ diag(e^{-iE tau} x C/2, e^{+iE tau} x C/2) u(p)     eq. 33 / 35
 * u(p) = d+ + d- sum_i (p_i/|p|) beta alpha_i                        eq. 30
 * d+-  = sqrt(1/2 +- 1/(2 sqrt(1 + p^2/(mc)^2)))                     eq. 29
 * E    = sqrt(m^2 c^4 + p^2 c^2)                                     eq. 32
 * At p = 0, d- = 0 and u = 1 (G6).
 */
/*
 * eq. 29.  d+ is evaluated as printed.  d- as printed, sqrt(1/2 - 1/(2 s)) with
 * s = sqrt(1 + p^2/(mc)^2), cancels catastrophically for |p| << mc (absolute
 * error up to 1e-8 near |p| ~ 3e-6 a.u.; found by the expm pin).  The same
 * quantity is therefore evaluated in the algebraically identical form
 *   1/2 - 1/(2s) = (s - 1)/(2s) = (p/(mc))^2 / (2 s (s + 1)),
 * which has no subtraction (reading G29).
 */
static void fw_scalars(double p2, double mass, double c, double *dplus, double *dminus) {
    double x2 = p2 / (mass * mass * c * c);
    double s = sqrt(1.0 + x2);
    *dplus = sqrt(0.5 + 0.5 / s);
    *dminus = sqrt(x2 / (2.0 * s * (s + 1.0)));
}

static void dirac_kinetic_matrix(int C, int ndim, const double *p, double mass, double c, double tau, cplx *U /*[C][C]*/) {
    cplx al[3 * 4 * 4], be[4 * 4];
    dirac_matrices(C, al, be);
    double p2 = 0.0;
    for (int a = 0; a < ndim; ++a) p2 += p[a] * p[a];
    double pabs = sqrt(p2);
    double dplus, dminus;
    fw_scalars(p2, mass, c, &dplus, &dminus);
    double E = sqrt(mass * mass * c * c * c * c + p2 * c * c);
    cplx u[16], ud[16], D[16], t[16];
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) {
            cplx acc = (r == s) ? dplus : 0.0;
            if (pabs > 0.0) {
                for (int a = 0; a < ndim; ++a) {
                    /* (beta alpha_a)[r][s] */
                    cplx ba = 0.0;
                    for (int m = 0; m < C; ++m) ba += be[r * C + m] * al[(a * C + m) * C + s];
                    acc += dminus * (p[a] / pabs) * ba;
                }
            }
            u[r * C + s] = acc;
        }
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) ud[r * C + s] = conj(u[s * C + r]);
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) {
            cplx d = 0.0;
            if (r == s) {
                double ang = (r < C / 2) ? -E * tau : E * tau;
                d = cos(ang) + I * sin(ang);
            }
            D[r * C + s] = d;
        }
    /* t = D u ; U = u^+ t */
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) {
            cplx acc = 0.0;
            for (int m = 0; m < C; ++m) acc += D[r * C + m] * u[m * C + s];
            t[r * C + s] = acc;
        }
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) {
            cplx acc = 0.0;
            for (int m = 0; m < C; ++m) acc += ud[r * C + m] * t[m * C + s];
            U[r * C + s] = acc;
        }
}

void orc_dirac_kinetic_matrix(int ncomp, int ndim, const double *p, double mass, double c, double tau, double *U_ri) {
    dirac_kinetic_matrix(ncomp, ndim, p, mass, c, tau, (cplx *)U_ri);
}

/* u(p) of eq. 30 itself, for the pins (unitarity, u H u^+ = diag(E,E,-E,-E)) */
void orc_dirac_u(int ncomp, int ndim, const double *p, double mass, double c, double *u_ri) {
    int C = ncomp;
    cplx *u = (cplx *)u_ri;
    cplx al[3 * 4 * 4], be[4 * 4];
    dirac_matrices(C, al, be);
    double p2 = 0.0;
    for (int a = 0; a < ndim; ++a) p2 += p[a] * p[a];
    double pabs = sqrt(p2);
    double dplus, dminus;
    fw_scalars(p2, mass, c, &dplus, &dminus);
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) {
            cplx acc = (r == s) ? dplus : 0.0;
            if (pabs > 0.0)
                for (int a = 0; a < ndim; ++a) {
                    cplx ba = 0.0;
                    for (int m = 0; m < C; ++m) ba += be[r * C + m] * al[(a * C + m) * C + s];
                    acc += dminus * (p[a] / pabs) * ba;
                }
            u[r * C + s] = acc;
        }
}

/* ------------------------------------------------------------------ */
/* the step                                                            */
/* ------------------------------------------------------------------ */
typedef struct {
    int32_t ndim;       /* 1..3 */
    int32_t ncomp;      /* 1 Schroedinger, 2 or 4 Dirac */
    int64_t n[3];
    double dx[3];
    double dt;
    double mass, c, charge;
    int32_t field_kind; /* ORC_FIELD_* */
    int32_t pad_;
    int64_t nvals;      /* rows of step_avg */
} orc_params;

/* psi_c(r) <- exp(-i (V(r) + r.Ebar) tau/2) psi_c(r)   eq. 11 / 22, delta = 1/2 */
static void potential_half_step(const orc_params *P, cplx *psi, const double *V, const double *Ebar) {
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    double half = 0.5 * P->dt;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j) {
        double v = V ? V[j] : 0.0;
        if (Ebar) {
            int64_t rem = j;
            for (int a = P->ndim - 1; a >= 0; --a) {
                int64_t ja = rem % P->n[a];
                rem /= P->n[a];
                v += r_of(ja, P->n[a], P->dx[a]) * Ebar[a];
            }
        }
        double ang = -v * half;
        cplx ph = cos(ang) + I * sin(ang);
        for (int cpt = 0; cpt < P->ncomp; ++cpt) psi[(int64_t)cpt * N + j] *= ph;
    }
}

static void kinetic_step(const orc_params *P, cplx *psi, const double *Abar) {
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    int C = P->ncomp;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j) {
        double p[3] = {0, 0, 0};
        int64_t rem = j;
        for (int a = P->ndim - 1; a >= 0; --a) {
            int64_t ja = rem % P->n[a];
            rem /= P->n[a];
            p[a] = k_of(ja, P->n[a], P->dx[a]) - (Abar ? P->charge * Abar[a] : 0.0);
        }
        if (C == 1) {
            /* eq. 13 with the step average of A (G12, G17) */
            double p2 = 0.0;
            for (int a = 0; a < P->ndim; ++a) p2 += p[a] * p[a];
            double ang = -P->dt * p2 / (2.0 * P->mass);
            psi[j] *= cos(ang) + I * sin(ang);
        } else {
            cplx U[16], in[4], out[4];
            dirac_kinetic_matrix(C, P->ndim, p, P->mass, P->c, P->dt, U);
            for (int s = 0; s < C; ++s) in[s] = psi[(int64_t)s * N + j];
            for (int r = 0; r < C; ++r) {
                cplx acc = 0.0;
                for (int s = 0; s < C; ++s) acc += U[r * C + s] * in[s];
                out[r] = acc;
            }
            for (int r = 0; r < C; ++r) psi[(int64_t)r * N + j] = out[r];
        }
    }
}

/*
 * Position-space vector-potential factor of the Dirac equation (the paper's own treatment of A(x,t)):
 * the split of PAPER.md:138-144 (eq. 18a) puts c sum_i alpha_i (-q A_i(x,t)) into A_1, next to q phi; the two
 * parts commute (eq. 19-22), and the exponential of the matrix part is, by the algebra of the
 * alpha_i (eq. 23/24),
 *     exp(i sum_i a_i alpha_i) = cos(a) + i (sum_i a_i alpha_i / a) sin(a),   a = sqrt(sum_i a_i^2),
 * here with a_i = delta * q * c * Abar_i(r), Abar_i = tau * (step average of A_i at r) the time integral of
 * eq. 25a.  For q = -1 this is eq. 26 as printed (reading G4); in one dimension it is
 * eq. 34.  Aavg: [ndim][N] step averages of A on the lattice.  a = 0 leaves psi unchanged.
 */
static void position_rotation(const orc_params *P, cplx *psi, const double *Aavg, double delta) {
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    int C = P->ncomp;
    cplx al[3 * 4 * 4], be[4 * 4];
    dirac_matrices(C, al, be);
    double coef = delta * P->charge * P->c * P->dt;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < N; ++j) {
        double ai[3] = {0, 0, 0}, a2 = 0.0;
        for (int a = 0; a < P->ndim; ++a) {
            ai[a] = coef * Aavg[(int64_t)a * N + j];
            a2 += ai[a] * ai[a];
        }
        double an = sqrt(a2);
        if (an == 0.0) continue;
        cplx M[16], in[4], out[4];
        for (int r = 0; r < C; ++r)
            for (int s = 0; s < C; ++s) {
                cplx acc = (r == s) ? cos(an) : 0.0;
                for (int a = 0; a < P->ndim; ++a) acc += I * (ai[a] / an) * sin(an) * al[(a * C + r) * C + s];
                M[r * C + s] = acc;
            }
        for (int s = 0; s < C; ++s) in[s] = psi[(int64_t)s * N + j];
        for (int r = 0; r < C; ++r) {
            cplx acc = 0.0;
            for (int s = 0; s < C; ++s) acc += M[r * C + s] * in[s];
            out[r] = acc;
        }
        for (int r = 0; r < C; ++r) psi[(int64_t)r * N + j] = out[r];
    }
}

/* the matrix of the factor above for one point, for the pins: a_i given directly */
void orc_alpha_rotation(int ncomp, int ndim, const double *ai, double *M_ri) {
    int C = ncomp;
    cplx *M = (cplx *)M_ri;
    cplx al[3 * 4 * 4], be[4 * 4];
    dirac_matrices(C, al, be);
    double a2 = 0.0;
    for (int a = 0; a < ndim; ++a) a2 += ai[a] * ai[a];
    double an = sqrt(a2);
    for (int r = 0; r < C; ++r)
        for (int s = 0; s < C; ++s) {
            cplx acc = (r == s) ? (an == 0.0 ? 1.0 : cos(an)) : 0.0;
            if (an != 0.0)
                for (int a = 0; a < ndim; ++a) acc += I * (ai[a] / an) * sin(an) * al[(a * C + r) * C + s];
            M[r * C + s] = acc;
        }
}

/*
 * The step with the position-space factor: as orc_step, with U_A1(1/2) = [scalar phase] x [rotation above] on both
 * sides of the Fourier sandwich (eq. 7 with the A_1 of eq. 18a; the two parts of A_1 commute, eq. 19-22).
 * Aavg: [ndim][N] step average of the position-dependent A(r), the same for every step of the call.  Dirac only.
 */
int orc_step_apos(const orc_params *P, double *psi_ri, const double *V, const double *step_avg, const double *Aavg, int64_t n0step, int64_t nsteps) {
    cplx *psi = (cplx *)psi_ri;
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    if (P->ncomp < 2 || Aavg == NULL) return -2;
    if (P->field_kind != ORC_FIELD_NONE && (step_avg == NULL || n0step + nsteps > P->nvals)) return -1;
    for (int64_t s = 0; s < nsteps; ++s) {
        int64_t n = n0step + s;
        const double *avg = (P->field_kind != ORC_FIELD_NONE) ? step_avg + n * P->ndim : NULL;
        const double *Ebar = (P->field_kind == ORC_FIELD_E) ? avg : NULL;
        const double *Abar = (P->field_kind == ORC_FIELD_A) ? avg : NULL;
        potential_half_step(P, psi, V, Ebar);
        position_rotation(P, psi, Aavg, 0.5);
        for (int cpt = 0; cpt < P->ncomp; ++cpt) orc_fft((double *)(psi + (int64_t)cpt * N), P->ndim, P->n, -1);
        kinetic_step(P, psi, Abar);
        for (int cpt = 0; cpt < P->ncomp; ++cpt) orc_fft((double *)(psi + (int64_t)cpt * N), P->ndim, P->n, +1);
        position_rotation(P, psi, Aavg, 0.5);
        potential_half_step(P, psi, V, Ebar);
    }
    return 0;
}

/*
 * Advance psi ([ncomp][n0][n1][n2] C order, interleaved re/im doubles) by
 * nsteps steps starting at step index n0step.  V: real potential energy
 * q phi(r) on the grid or NULL.  step_avg: [nvals][ndim] averages of E or A
 * over each step (G12), or NULL when field_kind = NONE.
 * Returns 0, or -1 if the field table is too short.
 */
int orc_step(const orc_params *P, double *psi_ri, const double *V, const double *step_avg, int64_t n0step, int64_t nsteps) {
    cplx *psi = (cplx *)psi_ri;
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    if (P->field_kind != ORC_FIELD_NONE && (step_avg == NULL || n0step + nsteps > P->nvals)) return -1;
    for (int64_t s = 0; s < nsteps; ++s) {
        int64_t n = n0step + s; /* t_n = n tau from the integer counter (G21) */
        const double *avg = (P->field_kind != ORC_FIELD_NONE) ? step_avg + n * P->ndim : NULL;
        const double *Ebar = (P->field_kind == ORC_FIELD_E) ? avg : NULL;
        const double *Abar = (P->field_kind == ORC_FIELD_A) ? avg : NULL;
        potential_half_step(P, psi, V, Ebar);                                     /* 1 */
        for (int cpt = 0; cpt < P->ncomp; ++cpt)                                  /* 2 */
            orc_fft((double *)(psi + (int64_t)cpt * N), P->ndim, P->n, -1);
        kinetic_step(P, psi, Abar);                                               /* 3 */
        for (int cpt = 0; cpt < P->ncomp; ++cpt)                                  /* 4 */
            orc_fft((double *)(psi + (int64_t)cpt * N), P->ndim, P->n, +1);
        potential_half_step(P, psi, V, Ebar);                                     /* 5 */
    }
    return 0;
}

/* sum_c sum_r |psi_c(r)|^2 prod dx */
double orc_norm(const orc_params *P, const double *psi_ri) {
    const cplx *psi = (const cplx *)psi_ri;
    int64_t N = 1;
    double vol = 1.0;
    for (int a = 0; a < P->ndim; ++a) {
        N *= P->n[a];
        vol *= P->dx[a];
    }
    int64_t M = N * P->ncomp;
    double acc = 0.0;
#pragma omp parallel for reduction(+ : acc) schedule(static)
    for (int64_t j = 0; j < M; ++j) acc += creal(psi[j]) * creal(psi[j]) + cimag(psi[j]) * cimag(psi[j]);
    return acc * vol;
}

/*
 * One output sample of step 4+5 computed from the definition, for full-size
 * spot checks: given psi~ after the kinetic factor (k space, all components),
 * returns psi_c(r_j) = exp(-i Vbar tau/2) (1/N) sum_k psi~_c(k) e^{+2 pi i j.l/n}
 * by the O(N) sum for one flat grid index j.
 */
void orc_inverse_sample(const orc_params *P, const double *psik_ri, const double *V, const double *Ebar, int64_t j, double *out_ri /*[ncomp] complex*/) {
    const cplx *psik = (const cplx *)psik_ri;
    cplx *out = (cplx *)out_ri;
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    int64_t jj[3] = {0, 0, 0};
    int64_t rem = j;
    double v = V ? V[j] : 0.0;
    for (int a = P->ndim - 1; a >= 0; --a) {
        jj[a] = rem % P->n[a];
        rem /= P->n[a];
        if (Ebar) v += r_of(jj[a], P->n[a], P->dx[a]) * Ebar[a];
    }
    for (int cpt = 0; cpt < P->ncomp; ++cpt) {
        double accr = 0.0, acci = 0.0;
#pragma omp parallel for reduction(+ : accr, acci) schedule(static)
        for (int64_t l = 0; l < N; ++l) {
            int64_t r2 = l;
            double frac = 0.0;
            for (int a = P->ndim - 1; a >= 0; --a) {
                int64_t la = r2 % P->n[a];
                r2 /= P->n[a];
                /* reduce j*l mod n exactly in integers before dividing */
                frac += (double)((jj[a] * la) % P->n[a]) / (double)P->n[a];
            }
            double ang = 2.0 * M_PI * frac;
            cplx t = psik[(int64_t)cpt * N + l] * (cos(ang) + I * sin(ang));
            accr += creal(t);
            acci += cimag(t);
        }
        double ang = -v * 0.5 * P->dt;
        out[cpt] = (accr + I * acci) / (double)N * (cos(ang) + I * sin(ang));
    }
}

/* steps 1-3 only (psi -> psi~ after the kinetic factor), the first half used with orc_inverse_sample */
int orc_half_step_to_k(const orc_params *P, double *psi_ri, const double *V, const double *step_avg, int64_t n) {
    cplx *psi = (cplx *)psi_ri;
    int64_t N = 1;
    for (int a = 0; a < P->ndim; ++a) N *= P->n[a];
    if (P->field_kind != ORC_FIELD_NONE && (step_avg == NULL || n + 1 > P->nvals)) return -1;
    const double *avg = (P->field_kind != ORC_FIELD_NONE) ? step_avg + n * P->ndim : NULL;
    const double *Ebar = (P->field_kind == ORC_FIELD_E) ? avg : NULL;
    const double *Abar = (P->field_kind == ORC_FIELD_A) ? avg : NULL;
    potential_half_step(P, psi, V, Ebar);
    for (int cpt = 0; cpt < P->ncomp; ++cpt) orc_fft((double *)(psi + (int64_t)cpt * N), P->ndim, P->n, -1);
    kinetic_step(P, psi, Abar);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Observables (section V.2).  New functions only:   */
/* nothing above is changed.  All are the plain definitions, written   */
/* as sums over the lattice (integrals -> sum * prod dx, reading G30). */
/* Pins: tests/test_oracle_observables.py.                             */
/* ------------------------------------------------------------------ */

/* <a|b> = sum_c sum_r conj(a_c(r)) b_c(r) prod dx: the autocorrelation chi(t) of eq. 40
 * with a = Psi(.,0), b = Psi(.,t).  out = (re, im). */
void orc_overlap(const orc_params *P, const double *a_ri, const double *b_ri, double *out) {
    const cplx *a = (const cplx *)a_ri, *b = (const cplx *)b_ri;
    int64_t N = 1;
    double vol = 1.0;
    for (int ax = 0; ax < P->ndim; ++ax) {
        N *= P->n[ax];
        vol *= P->dx[ax];
    }
    int64_t M = N * P->ncomp;
    double re = 0.0, im = 0.0;
#pragma omp parallel for reduction(+ : re, im) schedule(static)
    for (int64_t j = 0; j < M; ++j) {
        cplx t = conj(a[j]) * b[j];
        re += creal(t);
        im += cimag(t);
    }
    out[0] = re * vol;
    out[1] = im * vol;
}

/* <r_a> = sum_c sum_r r_a |psi_c(r)|^2 prod dx, a < ndim, on the grid r_j = (j - n/2) dx (G14) */
void orc_expect_r(const orc_params *P, const double *psi_ri, double *out /*[ndim]*/) {
    const cplx *psi = (const cplx *)psi_ri;
    int64_t N = 1;
    double vol = 1.0;
    for (int ax = 0; ax < P->ndim; ++ax) {
        N *= P->n[ax];
        vol *= P->dx[ax];
    }
    for (int ax = 0; ax < P->ndim; ++ax) {
        int64_t inner = 1;
        for (int b = ax + 1; b < P->ndim; ++b) inner *= P->n[b];
        double acc = 0.0;
#pragma omp parallel for reduction(+ : acc) schedule(static)
        for (int64_t j = 0; j < N; ++j) {
            double r = r_of((j / inner) % P->n[ax], P->n[ax], P->dx[ax]);
            double d = 0.0;
            for (int cpt = 0; cpt < P->ncomp; ++cpt) {
                cplx v = psi[(int64_t)cpt * N + j];
                d += creal(v) * creal(v) + cimag(v) * cimag(v);
            }
            acc += r * d;
        }
        out[ax] = acc * vol;
    }
}

/* <p_a> = sum_c sum_k k_a |psi~_c(k)|^2 prod dx / N  (canonical momentum, hbar = 1; psi~ = unnormalised forward DFT of
 * eq. 12, so sum_k |psi~|^2 = N sum_r |psi|^2), k on the grid of G14 */
void orc_expect_p(const orc_params *P, const double *psi_ri, double *out /*[ndim]*/) {
    int64_t N = 1;
    double vol = 1.0;
    for (int ax = 0; ax < P->ndim; ++ax) {
        N *= P->n[ax];
        vol *= P->dx[ax];
    }
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)(N * P->ncomp));
    memcpy(w, psi_ri, sizeof(cplx) * (size_t)(N * P->ncomp));
    for (int cpt = 0; cpt < P->ncomp; ++cpt) orc_fft((double *)(w + (int64_t)cpt * N), P->ndim, P->n, -1);
    for (int ax = 0; ax < P->ndim; ++ax) {
        int64_t inner = 1;
        for (int b = ax + 1; b < P->ndim; ++b) inner *= P->n[b];
        double acc = 0.0;
#pragma omp parallel for reduction(+ : acc) schedule(static)
        for (int64_t j = 0; j < N; ++j) {
            double k = k_of((j / inner) % P->n[ax], P->n[ax], P->dx[ax]);
            double d = 0.0;
            for (int cpt = 0; cpt < P->ncomp; ++cpt) {
                cplx v = w[(int64_t)cpt * N + j];
                d += creal(v) * creal(v) + cimag(v) * cimag(v);
            }
            acc += k * d;
        }
        out[ax] = acc * vol / (double)N;
    }
    free(w);
}

/* chi~(E) = int_0^T chi(t) (1 - cos(2 pi t/T)) exp(i t E) dt  (eq. 41) from samples chi(t_n),
 * t_n = n dts, n < nt, T = nt dts, as the plain sum over samples times dts (reading G30; the window vanishes at both
 * ends, so rectangle and trapezoid rule coincide).  chi_ri: [nt] complex; E: [nE]; out_ri: [nE] complex. */
void orc_spectrum(const double *chi_ri, int64_t nt, double dts, const double *E, int64_t nE, double *out_ri) {
    const cplx *chi = (const cplx *)chi_ri;
    cplx *out = (cplx *)out_ri;
    double T = (double)nt * dts;
#pragma omp parallel for schedule(static)
    for (int64_t e = 0; e < nE; ++e) {
        cplx acc = 0.0;
        for (int64_t n = 0; n < nt; ++n) {
            double t = (double)n * dts;
            double wdw = 1.0 - cos(2.0 * M_PI * t / T);
            acc += chi[n] * wdw * (cos(t * E[e]) + I * sin(t * E[e]));
        }
        out[e] = acc * dts;
    }
}

/* one term of eq. 42: acc(x) += Psi(x, t) (1 - cos(2 pi t/T)) exp(i E t) dts, every component */
void orc_filter_accumulate(const orc_params *P, double *acc_ri, const double *psi_ri, double t, double T, double E, double dts) {
    cplx *acc = (cplx *)acc_ri;
    const cplx *psi = (const cplx *)psi_ri;
    int64_t N = 1;
    for (int ax = 0; ax < P->ndim; ++ax) N *= P->n[ax];
    int64_t M = N * P->ncomp;
    cplx wgt = (1.0 - cos(2.0 * M_PI * t / T)) * (cos(E * t) + I * sin(E * t)) * dts;
#pragma omp parallel for schedule(static)
    for (int64_t j = 0; j < M; ++j) acc[j] += wgt * psi[j];
}
