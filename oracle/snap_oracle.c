/*
 * snap_oracle.c -- TEST INFRASTRUCTURE ONLY.
 *
 * Plain, slow, fp64 CPU definition of the SNAP bispectrum grid descriptor of
 * MALA (arXiv 2411.19617).  It exists so that tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs have something
 * independent to compare the CUDA path with.  Nothing in the product path
 * (paper_2411_19617_b200/) may import, link or execute it, and it shares no
 * code, header, table or constant generator with the CUDA path.
 *
 * What it follows (PAPER.md = /root/reference/PAPER.md):
 *   - neighbor density with cutoff, element weight and self term:
 *       Eq. (24)
 *   - hyperspherical-harmonic expansion coefficients u_j "computed using
 *     orthogonality" (= sum over neighbors of c * D^J(g)):  Eq. (25),
 *       PAPER.md:256-259
 *   - bispectrum = "scalar triple products of the expansion coefficients",
 *       PAPER.md:261; component count Eq. (26)
 *   - f_c, theta0 map, rfac0, rmin0, wself:  BASELINE.json north_star
 *   - the U / CG / B formulas themselves are not printed in the paper; they are
 *     the standard definitions of its Ref. [41], written out
 *     as mathematics in SURVEY.md 8(c) steps 5-8 (readings #1-#6 in DESIGN.md).
 *
 * Method, on purpose the plain definition (no recursion, no symmetry tricks,
 * no cells, no neighbor lists):
 *   U^J(g) is the explicit Wigner-D matrix = the matrix of g in SU(2) acting
 *   on homogeneous polynomials of degree J (double binomial sum);
 *   Clebsch-Gordan coefficients by Racah's closed form;
 *   B = Re sum_{m,m'} conj(U^j[m,m']) sum CG CG U^{j1} U^{j2}, full sums;
 *   neighbors = all atoms x all lattice images.
 *
 * All angular momenta are DOUBLED integers (J = 2 j_true); matrix indices
 * run 0..J and stand for m_true = idx - J/2.
 *
 * Pins (tests/test_oracle_pins.py, run with -m "not gpu"): Eq. (26) counts,
 * D unitarity / homomorphism / Chebyshev trace, CG orthogonality and sympy
 * cross-check, B_000 closed form, zero- and one-neighbor closed forms,
 * Chebyshev closed form of B_{j,0,j}, index symmetries of B, rotation /
 * reflection / permutation / translation invariances.
 * oracle_bj0j_grid (Chebyshev closed form of B_{j,0,j}, whole grids) and
 * oracle_gaussian_points (Gaussian descriptors, row f2) have their own
 * pins in tests/test_oracle_pins.py and tests/test_gaussian_descriptors.py.
 * Parity unpinned: component ORDER versus LAMMPS/MALA files (no such file in
 * the container); the order is the loop order of oracle_triples().
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double complex cplx;

#define ORACLE_MAX_TWOJ 16

/* ------------------------------------------------------------------ */
/* Triple enumeration; count pinned by Eq. (26) */
/* ------------------------------------------------------------------ */
int oracle_ntriples(int twojmax)
{
    int n = 0;
    for (int j1 = 0; j1 <= twojmax; j1++)
        for (int j2 = 0; j2 <= j1; j2++)
            for (int j = j1 - j2; j <= (twojmax < j1 + j2 ? twojmax : j1 + j2); j += 2)
                if (j >= j1) n++;
    return n;
}

void oracle_triples(int twojmax, int *out /* [n*3] */)
{
    int n = 0;
    for (int j1 = 0; j1 <= twojmax; j1++)
        for (int j2 = 0; j2 <= j1; j2++)
            for (int j = j1 - j2; j <= (twojmax < j1 + j2 ? twojmax : j1 + j2); j += 2)
                if (j >= j1) {
                    out[3 * n + 0] = j1;
                    out[3 * n + 1] = j2;
                    out[3 * n + 2] = j;
                    n++;
                }
}

/* ------------------------------------------------------------------ */
/* factorials (exact in fp64 up to 22!) and binomials                   */
/* ------------------------------------------------------------------ */
static double FACT[2 * ORACLE_MAX_TWOJ + 8];
static double BINOM[ORACLE_MAX_TWOJ + 1][ORACLE_MAX_TWOJ + 1];
static int tables_ready = 0;

static void tables_init(void)
{
    if (tables_ready) return;
    FACT[0] = 1.0;
    for (int i = 1; i < 2 * ORACLE_MAX_TWOJ + 8; i++) FACT[i] = FACT[i - 1] * (double)i;
    for (int n = 0; n <= ORACLE_MAX_TWOJ; n++)
        for (int k = 0; k <= ORACLE_MAX_TWOJ; k++)
            BINOM[n][k] = (k <= n) ? FACT[n] / (FACT[k] * FACT[n - k]) : 0.0;
    tables_ready = 1;
}

static double fact(int n) { return FACT[n]; }

static double binom(int n, int k)
{
    if (k < 0 || k > n) return 0.0;
    return BINOM[n][k];
}

/* ------------------------------------------------------------------ */
/* Clebsch-Gordan, Racah's closed form, Condon-Shortley phases.         */
/* SURVEY.md 8(c) step 7.  Arguments are doubled: J = 2j, M = 2m.       */
/* ------------------------------------------------------------------ */
double oracle_cg(int J1, int M1, int J2, int M2, int J, int M)
{
    tables_init();
    if (M1 + M2 != M) return 0.0;
    if ((J1 + J2 + J) % 2 != 0) return 0.0;
    if (J < abs(J1 - J2) || J > J1 + J2) return 0.0;
    if (abs(M1) > J1 || abs(M2) > J2 || abs(M) > J) return 0.0;
    if ((J1 + M1) % 2 != 0 || (J2 + M2) % 2 != 0 || (J + M) % 2 != 0) return 0.0;

    /* integer factorial arguments */
    int a = (J1 + J2 - J) / 2;  /* j1+j2-j  */
    int b = (J1 - J2 + J) / 2;  /* j1-j2+j  */
    int c = (-J1 + J2 + J) / 2; /* -j1+j2+j */
    int d = (J1 + J2 + J) / 2 + 1;
    int j1pm1 = (J1 + M1) / 2, j1mm1 = (J1 - M1) / 2;
    int j2pm2 = (J2 + M2) / 2, j2mm2 = (J2 - M2) / 2;
    int jpm = (J + M) / 2, jmm = (J - M) / 2;
    int e = (J - J2 + M1) / 2; /* j-j2+m1 */
    int f = (J - J1 - M2) / 2; /* j-j1-m2 */

    double pref = sqrt((double)(J + 1)) *
                  sqrt(fact(a) * fact(b) * fact(c) / fact(d)) *
                  sqrt(fact(j1pm1) * fact(j1mm1) * fact(j2pm2) * fact(j2mm2) * fact(jpm) * fact(jmm));
    double sum = 0.0;
    for (int z = 0; z <= d; z++) {
        int t1 = a - z, t2 = j1mm1 - z, t3 = j2pm2 - z, t4 = e + z, t5 = f + z;
        if (t1 < 0 || t2 < 0 || t3 < 0 || t4 < 0 || t5 < 0) continue;
        double term = 1.0 / (fact(z) * fact(t1) * fact(t2) * fact(t3) * fact(t4) * fact(t5));
        sum += (z % 2) ? -term : term;
    }
    return pref * sum;
}

/* ------------------------------------------------------------------ */
/* Pair geometry, SURVEY.md 8(c) step 5 / north_star.                   */
/* d = R_neighbor - r_point.  Returns 0 if not a neighbor (r >= rcut).  */
/* a = q0 - i q3, b = q2 - i q1, q = (cos th0, sin th0 * d/r).          */
/* r -> 0 limit (reading #11): a = 1, b = 0, fc = 1 (for rmin0 > 0 the  */
/* direction is undefined at r = 0 and the same U = I is used).         */
/* ------------------------------------------------------------------ */
int oracle_pair(const double d[3], double rcut, double rfac0, double rmin0,
                double ab[4] /* a.re a.im b.re b.im */, double *fc)
{
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(r < rcut)) return 0;
    if (r < 1e-10 * rcut) {
        ab[0] = 1.0; ab[1] = 0.0; ab[2] = 0.0; ab[3] = 0.0;
        *fc = 1.0;
        return 1;
    }
    /* reading #22: for r <= rmin0 the switching function
     * saturates at 1, while the theta0 map stays the same linear function of r
     * (theta0 < 0 there); only rmin0 = 0 occurs in the five configs. */
    double x = (r - rmin0) / (rcut - rmin0);
    *fc = (x <= 0.0) ? 1.0 : 0.5 * (cos(M_PI * x) + 1.0);
    double th0 = rfac0 * M_PI * x;
    double q0 = cos(th0), s = sin(th0);
    double q1 = s * d[0] / r, q2 = s * d[1] / r, q3 = s * d[2] / r;
    ab[0] = q0;  ab[1] = -q3;
    ab[2] = q2;  ab[3] = -q1;
    return 1;
}

/* ------------------------------------------------------------------ */
/* Explicit Wigner-D, SURVEY.md 8(c) step 6.                            */
/* g = [[a, -conj(b)],[b, conj(a)]] acts on degree-J polynomials in     */
/* (xi, eta), orthonormal basis e_m = xi^m eta^(J-m)/sqrt(m!(J-m)!).    */
/* D[m'][m] = sqrt(m'!(J-m')!/(m!(J-m)!)) *                             */
/*   sum_{k=0..m} sum_{l=0..J-m, k+l=m'} C(m,k) C(J-m,l)                */
/*        g00^k g01^(m-k) g10^l g11^(J-m-l)                             */
/* D is written row-major, (J+1)x(J+1), interleaved re/im.              */
/* ------------------------------------------------------------------ */
static void wigner_D(int J, cplx a, cplx b, cplx *D)
{
    cplx g00 = a, g01 = -conj(b), g10 = b, g11 = conj(a);
    cplx p00[ORACLE_MAX_TWOJ + 1], p01[ORACLE_MAX_TWOJ + 1], p10[ORACLE_MAX_TWOJ + 1], p11[ORACLE_MAX_TWOJ + 1];
    p00[0] = p01[0] = p10[0] = p11[0] = 1.0;
    for (int i = 1; i <= J; i++) {
        p00[i] = p00[i - 1] * g00;
        p01[i] = p01[i - 1] * g01;
        p10[i] = p10[i - 1] * g10;
        p11[i] = p11[i - 1] * g11;
    }
    for (int mp = 0; mp <= J; mp++)
        for (int m = 0; m <= J; m++) {
            cplx s = 0.0;
            for (int k = 0; k <= m; k++) {
                int l = mp - k;
                if (l < 0 || l > J - m) continue;
                s += binom(m, k) * binom(J - m, l) * p00[k] * p01[m - k] * p10[l] * p11[J - m - l];
            }
            double nrm = sqrt(fact(mp) * fact(J - mp) / (fact(m) * fact(J - m)));
            D[mp * (J + 1) + m] = nrm * s;
        }
}

void oracle_wigner_D(int J, const double ab[4], double *D_out /* (J+1)^2*2 */)
{
    tables_init();
    cplx *D = (cplx *)malloc(sizeof(cplx) * (J + 1) * (J + 1));
    wigner_D(J, ab[0] + I * ab[1], ab[2] + I * ab[3], D);
    for (int i = 0; i < (J + 1) * (J + 1); i++) {
        D_out[2 * i] = creal(D[i]);
        D_out[2 * i + 1] = cimag(D[i]);
    }
    free(D);
}

/* offset of level J in the packed U array: sum_{K<J} (K+1)^2 */
static int uoff(int J)
{
    int o = 0;
    for (int K = 0; K < J; K++) o += (K + 1) * (K + 1);
    return o;
}

int oracle_usize(int twojmax) { return uoff(twojmax + 1); }

/* ------------------------------------------------------------------ */
/* System description                                                   */
/* ------------------------------------------------------------------ */
typedef struct {
    int twojmax;
    double rcutfac, rfac0, rmin0, wself;
    int ntypes;
    const double *radelem, *wj;
    int natoms;
    const double *pos; /* [natoms*3] as given */
    const int *types;
    const double *box; /* rows a1,a2,a3 */
    const double *origin;
    const int *pbc;
    /* derived */
    double *wpos; /* wrapped positions */
    int nimg[3];
    double rcutmax;
} sys_t;

static void cross3(const double *u, const double *v, double *w)
{
    w[0] = u[1] * v[2] - u[2] * v[1];
    w[1] = u[2] * v[0] - u[0] * v[2];
    w[2] = u[0] * v[1] - u[1] * v[0];
}

static double dot3(const double *u, const double *v) { return u[0] * v[0] + u[1] * v[1] + u[2] * v[2]; }

/* wrap atoms along periodic axes (reading #14) and fix the image range
 * N_i = ceil(rcutmax / h_i) + 1 on periodic axes, 0 otherwise (step 4). */
static int sys_prepare(sys_t *s)
{
    const double *a1 = s->box, *a2 = s->box + 3, *a3 = s->box + 6;
    double c23[3], c31[3], c12[3];
    cross3(a2, a3, c23);
    cross3(a3, a1, c31);
    cross3(a1, a2, c12);
    double det = dot3(a1, c23);
    if (!(fabs(det) > 0.0)) return -1;
    s->rcutmax = 0.0;
    for (int t = 0; t < s->ntypes; t++) {
        double rc = 2.0 * s->rcutfac * s->radelem[t];
        if (rc > s->rcutmax) s->rcutmax = rc;
    }
    double h[3] = {fabs(det) / sqrt(dot3(c23, c23)), fabs(det) / sqrt(dot3(c31, c31)), fabs(det) / sqrt(dot3(c12, c12))};
    for (int i = 0; i < 3; i++) s->nimg[i] = s->pbc[i] ? (int)ceil(s->rcutmax / h[i]) + 1 : 0;
    s->wpos = (double *)malloc(sizeof(double) * 3 * (s->natoms > 0 ? s->natoms : 1));
    /* reciprocal rows: f_i = (x - origin) . c_jk / det */
    for (int n = 0; n < s->natoms; n++) {
        double x[3] = {s->pos[3 * n] - s->origin[0], s->pos[3 * n + 1] - s->origin[1], s->pos[3 * n + 2] - s->origin[2]};
        double f[3] = {dot3(x, c23) / det, dot3(x, c31) / det, dot3(x, c12) / det};
        for (int i = 0; i < 3; i++)
            if (s->pbc[i]) f[i] -= floor(f[i]);
        for (int k = 0; k < 3; k++)
            s->wpos[3 * n + k] = s->origin[k] + f[0] * a1[k] + f[1] * a2[k] + f[2] * a3[k];
    }
    return 0;
}

/* ------------------------------------------------------------------ */
/* U_tot at one point: wself*I + sum over all atoms x all images of     */
/* c * D^J(g)  (Eq. 24-25).  U packed by level, row-major [m'][m].      */
/* Also returns the neighbor count.                                     */
/* ------------------------------------------------------------------ */
static int utot_point(const sys_t *s, const double rp[3], cplx *U, cplx *Dtmp,
                      double *nbr_q /* optional [cap*5]: c,q0,q1,q2,q3 */, int nbr_cap)
{
    int tj = s->twojmax;
    int usz = uoff(tj + 1);
    for (int i = 0; i < usz; i++) U[i] = 0.0;
    for (int J = 0; J <= tj; J++)
        for (int m = 0; m <= J; m++) U[uoff(J) + m * (J + 1) + m] = s->wself;
    int nn = 0;
    const double *a1 = s->box, *a2 = s->box + 3, *a3 = s->box + 6;
    for (int n = 0; n < s->natoms; n++) {
        int t = s->types[n];
        double rcut = 2.0 * s->rcutfac * s->radelem[t];
        double w = s->wj[t];
        for (int n1 = -s->nimg[0]; n1 <= s->nimg[0]; n1++)
            for (int n2 = -s->nimg[1]; n2 <= s->nimg[1]; n2++)
                for (int n3 = -s->nimg[2]; n3 <= s->nimg[2]; n3++) {
                    double d[3];
                    for (int k = 0; k < 3; k++)
                        d[k] = s->wpos[3 * n + k] + n1 * a1[k] + n2 * a2[k] + n3 * a3[k] - rp[k];
                    /* correctness-neutral early rejection on one coordinate */
                    if (fabs(d[0]) >= rcut || fabs(d[1]) >= rcut || fabs(d[2]) >= rcut) continue;
                    double ab[4], fc;
                    if (!oracle_pair(d, rcut, s->rfac0, s->rmin0, ab, &fc)) continue;
                    double c = w * fc;
                    cplx a = ab[0] + I * ab[1], b = ab[2] + I * ab[3];
                    for (int J = 0; J <= tj; J++) {
                        wigner_D(J, a, b, Dtmp);
                        cplx *UJ = U + uoff(J);
                        for (int i = 0; i < (J + 1) * (J + 1); i++) UJ[i] += c * Dtmp[i];
                    }
                    if (nbr_q && nn < nbr_cap) {
                        /* q0 = Re a, q3 = -Im a, q2 = Re b, q1 = -Im b */
                        nbr_q[5 * nn + 0] = c;
                        nbr_q[5 * nn + 1] = ab[0];
                        nbr_q[5 * nn + 2] = -ab[3];
                        nbr_q[5 * nn + 3] = ab[2];
                        nbr_q[5 * nn + 4] = -ab[1];
                    }
                    nn++;
                }
    }
    return nn;
}

/* ------------------------------------------------------------------ */
/* CG cache for a list of triples: table[t][i1*(J2+1)+i2] =             */
/*   C^{j m}_{j1 m1 j2 m2} with m = m1+m2 (0 where |m| > j)             */
/* ------------------------------------------------------------------ */
typedef struct {
    int n;
    int *tr;
    double **tab;
} cgcache_t;

static void cg_build(cgcache_t *c, int n, const int *tr)
{
    c->n = n;
    c->tr = (int *)malloc(sizeof(int) * 3 * n);
    memcpy(c->tr, tr, sizeof(int) * 3 * n);
    c->tab = (double **)malloc(sizeof(double *) * n);
    for (int t = 0; t < n; t++) {
        int J1 = tr[3 * t], J2 = tr[3 * t + 1], J = tr[3 * t + 2];
        c->tab[t] = (double *)malloc(sizeof(double) * (J1 + 1) * (J2 + 1));
        for (int i1 = 0; i1 <= J1; i1++)
            for (int i2 = 0; i2 <= J2; i2++) {
                int M1 = 2 * i1 - J1, M2 = 2 * i2 - J2;
                c->tab[t][i1 * (J2 + 1) + i2] = oracle_cg(J1, M1, J2, M2, J, M1 + M2);
            }
    }
}

static void cg_free(cgcache_t *c)
{
    for (int t = 0; t < c->n; t++) free(c->tab[t]);
    free(c->tab);
    free(c->tr);
}

/* ------------------------------------------------------------------ */
/* B from U_tot, full sums:                      */
/* B = Re sum_{m,m'} conj(U^j[m,m']) sum_{m1+m2=m} sum_{m1'+m2'=m'}     */
/*        C(m1,m2) C(m1',m2') U^{j1}[m1,m1'] U^{j2}[m2,m2']             */
/* index relation: idx = idx1 + idx2 - (J1+J2-J)/2.                     */
/* Returns also the imaginary part (rounding noise) if imag != NULL.    */
/* ------------------------------------------------------------------ */
static void b_from_u(const cgcache_t *cg, const cplx *U, double *B, double *imag)
{
    for (int t = 0; t < cg->n; t++) {
        int J1 = cg->tr[3 * t], J2 = cg->tr[3 * t + 1], J = cg->tr[3 * t + 2];
        const cplx *U1 = U + uoff(J1), *U2 = U + uoff(J2), *UJ = U + uoff(J);
        const double *C = cg->tab[t];
        int sh = (J1 + J2 - J) / 2;
        cplx acc = 0.0;
        for (int m = 0; m <= J; m++)
            for (int mp = 0; mp <= J; mp++) {
                cplx z = 0.0;
                for (int m1 = 0; m1 <= J1; m1++) {
                    int m2 = m + sh - m1;
                    if (m2 < 0 || m2 > J2) continue;
                    double c1 = C[m1 * (J2 + 1) + m2];
                    for (int m1p = 0; m1p <= J1; m1p++) {
                        int m2p = mp + sh - m1p;
                        if (m2p < 0 || m2p > J2) continue;
                        double c2 = C[m1p * (J2 + 1) + m2p];
                        z += c1 * c2 * U1[m1 * (J1 + 1) + m1p] * U2[m2 * (J2 + 1) + m2p];
                    }
                }
                acc += conj(UJ[m * (J + 1) + mp]) * z;
            }
        B[t] = creal(acc);
        if (imag) imag[t] = cimag(acc);
    }
}

/* ------------------------------------------------------------------ */
/* Public entry points                                                  */
/* ------------------------------------------------------------------ */

/* B (and optionally U_tot, Im B, neighbor quaternions) at explicit points,
 * for an arbitrary list of triples (test mode: unordered triples allowed as
 * long as they satisfy the triangle and parity conditions). */
int oracle_bispectrum_points(int twojmax, double rcutfac, double rfac0, double rmin0, double wself,
                             int ntypes, const double *radelem, const double *wj,
                             int natoms, const double *pos, const int *types,
                             const double *box, const double *origin, const int *pbc,
                             int npoints, const double *points /* [npoints*3] */,
                             int ntriples, const int *triples /* [ntriples*3] */,
                             double *B /* [npoints*ntriples] */,
                             double *Bimag /* optional */,
                             double *U_out /* optional [npoints*usize*2] */,
                             int *nnbr_out /* optional [npoints] */,
                             double *nbr_q /* optional [npoints*nbr_cap*5] */, int nbr_cap)
{
    if (twojmax < 0 || twojmax > ORACLE_MAX_TWOJ) return -1;
    tables_init();
    sys_t s = {twojmax, rcutfac, rfac0, rmin0, wself, ntypes, radelem, wj, natoms, pos, types, box, origin, pbc, NULL, {0, 0, 0}, 0.0};
    if (sys_prepare(&s)) return -1;
    cgcache_t cg;
    cg_build(&cg, ntriples, triples);
    int usz = uoff(twojmax + 1);
#pragma omp parallel
    {
        cplx *U = (cplx *)malloc(sizeof(cplx) * usz);
        cplx *D = (cplx *)malloc(sizeof(cplx) * (twojmax + 1) * (twojmax + 1));
#pragma omp for schedule(dynamic, 8)
        for (int p = 0; p < npoints; p++) {
            int nn = utot_point(&s, points + 3 * p, U, D, nbr_q ? nbr_q + (size_t)p * nbr_cap * 5 : NULL, nbr_cap);
            if (nnbr_out) nnbr_out[p] = nn;
            if (U_out)
                for (int i = 0; i < usz; i++) {
                    U_out[((size_t)p * usz + i) * 2] = creal(U[i]);
                    U_out[((size_t)p * usz + i) * 2 + 1] = cimag(U[i]);
                }
            b_from_u(&cg, U, B + (size_t)p * ntriples, Bimag ? Bimag + (size_t)p * ntriples : NULL);
        }
        free(U);
        free(D);
    }
    cg_free(&cg);
    free(s.wpos);
    return 0;
}

/* Grid form (step 3 + step 9): point (ix,iy,iz) at
 * origin + ix/nx a1 + iy/ny a2 + iz/nz a3, ix fastest, z-slab [z_begin,z_end);
 * out[((iz-z_begin)*ny+iy)*nx+ix][k], k in oracle_triples() order.
 * Optional subsampling: if nsample > 0, only the listed flat point indices
 * (relative to the slab) are evaluated and written densely to out[nsample][ncomp]. */
int oracle_bispectrum_grid(int twojmax, double rcutfac, double rfac0, double rmin0, double wself,
                           int ntypes, const double *radelem, const double *wj,
                           int natoms, const double *pos, const int *types,
                           const double *box, const double *origin, const int *pbc,
                           const int *ngrid, int z_begin, int z_end,
                           long nsample, const long *sample,
                           double *out)
{
    int nx = ngrid[0], ny = ngrid[1], nz = ngrid[2];
    if (nx <= 0 || ny <= 0 || nz <= 0 || z_begin < 0 || z_end > nz || z_begin > z_end) return -1;
    long npts = nsample > 0 ? nsample : (long)(z_end - z_begin) * ny * nx;
    if (npts > 2000000000L) return -1;
    double *pts = (double *)malloc(sizeof(double) * 3 * (npts > 0 ? npts : 1));
    for (long q = 0; q < npts; q++) {
        long f = nsample > 0 ? sample[q] : q;
        int ix = (int)(f % nx);
        int iy = (int)((f / nx) % ny);
        int iz = (int)(f / ((long)nx * ny)) + z_begin;
        double fx = (double)ix / nx, fy = (double)iy / ny, fz = (double)iz / nz;
        for (int k = 0; k < 3; k++)
            pts[3 * q + k] = origin[k] + fx * box[k] + fy * box[3 + k] + fz * box[6 + k];
    }
    int nt = oracle_ntriples(twojmax);
    int *tr = (int *)malloc(sizeof(int) * 3 * nt);
    oracle_triples(twojmax, tr);
    int rc = oracle_bispectrum_points(twojmax, rcutfac, rfac0, rmin0, wself, ntypes, radelem, wj,
                                      natoms, pos, types, box, origin, pbc,
                                      (int)npts, pts, nt, tr, out, NULL, NULL, NULL, NULL, 0);
    free(tr);
    free(pts);
    return rc;
}

/* ------------------------------------------------------------------ */
/* Gaussian descriptors ("a sum of  */
/* Gaussians centered at R", Eqs. (40)-(43) PAPER.md:396-412).          */
/* Reading: per atom type t one channel,         */
/*   G_t(r) = w_t (2 pi sigma^2)^(-3/2) sum exp(-|R - r|^2 / (2 sigma^2)) */
/* over the atoms of type t and their periodic images with              */
/* |R - r| < rcut_t (strict), i.e. unit-integral Gaussians of width     */
/* sigma = w_G truncated at the descriptor cutoff.  Plain definition:   */
/* all atoms x all images.                                              */
/* ------------------------------------------------------------------ */
int oracle_gaussian_points(double rcutfac, double sigma, int ntypes, const double *radelem, const double *wj, int natoms,
                           const double *pos, const int *types, const double *box, const double *origin, const int *pbc,
                           int npoints, const double *points, double *out /* [npoints*ntypes] */)
{
    if (!(sigma > 0.0) || ntypes < 1 || natoms < 0 || npoints < 0) return -1;
    sys_t s;
    memset(&s, 0, sizeof(s));
    s.rcutfac = rcutfac; s.ntypes = ntypes; s.radelem = radelem; s.wj = wj;
    s.natoms = natoms; s.pos = pos; s.types = types; s.box = box; s.origin = origin; s.pbc = pbc;
    if (sys_prepare(&s)) return -1;
    const double pi = 3.14159265358979323846;
    const double pref = 1.0 / (pow(2.0 * pi, 1.5) * sigma * sigma * sigma);
    const double *a1 = box, *a2 = box + 3, *a3 = box + 6;
#pragma omp parallel for schedule(dynamic, 16)
    for (int p = 0; p < npoints; p++) {
        const double *rp = points + 3 * p;
        double *g = out + (size_t)p * ntypes;
        for (int t = 0; t < ntypes; t++) g[t] = 0.0;
        for (int n = 0; n < natoms; n++) {
            int t = types[n];
            double rcut = 2.0 * rcutfac * radelem[t];
            for (int n1 = -s.nimg[0]; n1 <= s.nimg[0]; n1++)
                for (int n2 = -s.nimg[1]; n2 <= s.nimg[1]; n2++)
                    for (int n3 = -s.nimg[2]; n3 <= s.nimg[2]; n3++) {
                        double d[3];
                        for (int k = 0; k < 3; k++)
                            d[k] = s.wpos[3 * n + k] + n1 * a1[k] + n2 * a2[k] + n3 * a3[k] - rp[k];
                        double r2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                        if (!(sqrt(r2) < rcut)) continue;
                        g[t] += wj[t] * pref * exp(-r2 / (2.0 * sigma * sigma));
                    }
        }
    }
    free(s.wpos);
    return 0;
}

/* ------------------------------------------------------------------ */
/* Second, independent oracle for the 11 components B_{j,0,j}           */
/* (SURVEY.md 8(c) pins): with the self term (c = wself, q = (1,0,0,0)) */
/* and the neighbors (c = w f_c, unit quaternion q = (cos t0, sin t0    */
/* d/r)) indexed together,                                              */
/*   B_{j,0,j} = (sum_k c_k) * sum_{k,l} c_k c_l U_j(<q_k, q_l>),        */
/* U_j the Chebyshev polynomial of the second kind of degree j          */
/* (doubled j).  Needs neither Wigner-D nor Clebsch-Gordan, only the     */
/* neighbor gather, f_c and the theta0 map -- cheap enough for whole     */
/* grids.  Pinned against oracle_bispectrum_points (the Wigner-D / CG    */
/* path) in tests/test_oracle_pins.py.  out[(z1-z0)*ny*nx][twojmax+1],   */
/* or out[nsample][twojmax+1] when a list of point indices is given.     */
/* ------------------------------------------------------------------ */
int oracle_bj0j_grid(int twojmax, double rcutfac, double rfac0, double rmin0, double wself, int ntypes, const double *radelem,
                     const double *wj, int natoms, const double *pos, const int *types, const double *box,
                     const double *origin, const int *pbc, const int *ngrid, int z0, int z1,
                     long nsample, const long *sample /* optional flat point indices relative to the slab */, double *out)
{
    if (twojmax < 0 || twojmax > ORACLE_MAX_TWOJ || ntypes < 1 || z0 < 0 || z1 > ngrid[2] || z0 > z1) return -1;
    sys_t s;
    memset(&s, 0, sizeof(s));
    s.twojmax = twojmax; s.rcutfac = rcutfac; s.rfac0 = rfac0; s.rmin0 = rmin0; s.wself = wself;
    s.ntypes = ntypes; s.radelem = radelem; s.wj = wj;
    s.natoms = natoms; s.pos = pos; s.types = types; s.box = box; s.origin = origin; s.pbc = pbc;
    if (sys_prepare(&s)) return -1;
    const double *a1 = box, *a2 = box + 3, *a3 = box + 6;
    const int nx = ngrid[0], ny = ngrid[1], nz = ngrid[2];
    const long npts = nsample > 0 ? nsample : (long)(z1 - z0) * ny * nx;
    int bad = 0;
#pragma omp parallel for schedule(dynamic, 64)
    for (long ip = 0; ip < npts; ip++) {
        const long fp = nsample > 0 ? sample[ip] : ip;
        const int ix = (int)(fp % nx), iy = (int)((fp / nx) % ny), iz = z0 + (int)(fp / ((long)nx * ny));
        double rp[3];
        for (int k = 0; k < 3; k++)
            rp[k] = origin[k] + ((double)ix / nx) * a1[k] + ((double)iy / ny) * a2[k] + ((double)iz / nz) * a3[k];
        int cap = 128, n = 1;
        double *c = (double *)malloc(sizeof(double) * cap), *q = (double *)malloc(sizeof(double) * 4 * cap);
        c[0] = wself; q[0] = 1.0; q[1] = q[2] = q[3] = 0.0;
        for (int a = 0; a < natoms; a++) {
            const int t = types[a];
            const double rcut = 2.0 * rcutfac * radelem[t];
            for (int n1 = -s.nimg[0]; n1 <= s.nimg[0]; n1++)
                for (int n2 = -s.nimg[1]; n2 <= s.nimg[1]; n2++)
                    for (int n3 = -s.nimg[2]; n3 <= s.nimg[2]; n3++) {
                        double d[3];
                        for (int k = 0; k < 3; k++)
                            d[k] = s.wpos[3 * a + k] + n1 * a1[k] + n2 * a2[k] + n3 * a3[k] - rp[k];
                        if (fabs(d[0]) >= rcut || fabs(d[1]) >= rcut || fabs(d[2]) >= rcut) continue;
                        double ab[4], fc;
                        if (!oracle_pair(d, rcut, rfac0, rmin0, ab, &fc)) continue;
                        if (n == cap) {
                            cap *= 2;
                            c = (double *)realloc(c, sizeof(double) * cap);
                            q = (double *)realloc(q, sizeof(double) * 4 * cap);
                        }
                        /* a = q0 - i q3, b = q2 - i q1 (oracle_pair) */
                        c[n] = wj[t] * fc;
                        q[4 * n + 0] = ab[0]; q[4 * n + 1] = -ab[3]; q[4 * n + 2] = ab[2]; q[4 * n + 3] = -ab[1];
                        n++;
                    }
        }
        double csum = 0.0, acc[ORACLE_MAX_TWOJ + 1];
        for (int j = 0; j <= twojmax; j++) acc[j] = 0.0;
        for (int k = 0; k < n; k++) csum += c[k];
        for (int k = 0; k < n; k++)
            for (int l = 0; l < n; l++) {
                const double x = q[4 * k] * q[4 * l] + q[4 * k + 1] * q[4 * l + 1] + q[4 * k + 2] * q[4 * l + 2] + q[4 * k + 3] * q[4 * l + 3];
                double um = 0.0, u = 1.0; /* U_{-1}, U_0 */
                const double w = c[k] * c[l];
                for (int j = 0; j <= twojmax; j++) {
                    acc[j] += w * u;
                    const double un = 2.0 * x * u - um;
                    um = u;
                    u = un;
                }
            }
        for (int j = 0; j <= twojmax; j++) out[(size_t)ip * (twojmax + 1) + j] = csum * acc[j];
        free(c);
        free(q);
        if (n < 1) bad = 1;
    }
    free(s.wpos);
    return bad ? -1 : 0;
}

/* ------------------------------------------------------------------ */
/* Row f3: derivative of the descriptors with respect to the atom       */
/* positions, dB(r, j)/dR_alpha (Eq. (45): the third  */
/* factor of the chain rule, applied to a per-grid-point vector).       */
/* Plain forward differentiation of the definition above, term by term: */
/*   d/dR of f_c, theta0, the quaternion, (a, b);                       */
/*   dD^J by the product rule on the double binomial sum;               */
/*   dB = T(dU,U,U) + T(U,dU,U) + T(U,U,dU) for the trilinear form      */
/*   T(X,Y,W) = Re sum conj(W^j) sum CG CG X^{j1} Y^{j2}, full sums.    */
/* All images of atom alpha move with it.  No adjoint trick, no         */
/* symmetry: the CUDA path (Y contraction + dU recursion) shares        */
/* nothing with this.  Pinned in tests/test_force_oracle.py by central  */
/* finite differences of oracle_bispectrum_points, by the closed forms  */
/* of the one-neighbor case and of B_000, by sum_alpha dB/dR_alpha =    */
/* -dB/dr (point moved instead of atoms) and by rotation covariance.    */
/* ------------------------------------------------------------------ */

/* d(a, b, fc)/dR_k for k = x, y, z (d = R - r_point).  Returns 0 if not a neighbor. */
static int pair_grad(const double d[3], double rcut, double rfac0, double rmin0, cplx *a, cplx *b, double *fc,
                     cplx da[3], cplx db[3], double dfc[3])
{
    double r = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    if (!(r < rcut)) return 0;
    if (r < 1e-10 * rcut) { /* reading #11: U = I, weight w; the direction is undefined, the derivative is taken as 0 */
        *a = 1.0; *b = 0.0; *fc = 1.0;
        for (int k = 0; k < 3; k++) { da[k] = 0.0; db[k] = 0.0; dfc[k] = 0.0; }
        return 1;
    }
    double x = (r - rmin0) / (rcut - rmin0);
    double dxdr = 1.0 / (rcut - rmin0);
    double fcp; /* dfc/dr */
    if (x <= 0.0) { *fc = 1.0; fcp = 0.0; }
    else { *fc = 0.5 * (cos(M_PI * x) + 1.0); fcp = -0.5 * M_PI * sin(M_PI * x) * dxdr; }
    double th0 = rfac0 * M_PI * x, th0p = rfac0 * M_PI * dxdr;
    double c0 = cos(th0), s0 = sin(th0);
    double u[3] = {d[0] / r, d[1] / r, d[2] / r};
    double q[4] = {c0, s0 * u[0], s0 * u[1], s0 * u[2]};
    *a = q[0] - I * q[3];
    *b = q[2] - I * q[1];
    for (int k = 0; k < 3; k++) {
        double dr = u[k]; /* dr/dR_k */
        double dq0 = -s0 * th0p * dr;
        double dq[3];
        for (int i = 0; i < 3; i++) dq[i] = c0 * th0p * dr * u[i] + s0 * (((i == k) ? 1.0 : 0.0) - u[i] * u[k]) / r;
        da[k] = dq0 - I * dq[2];
        db[k] = dq[1] - I * dq[0];
        dfc[k] = fcp * dr;
    }
    return 1;
}

/* D^J(g) and its directional derivative for (da, db): product rule on every factor of the double binomial sum */
static void wigner_dD(int J, cplx a, cplx b, cplx da, cplx db, cplx *dD)
{
    cplx g[4] = {a, -conj(b), b, conj(a)};          /* g00 g01 g10 g11 */
    cplx dg[4] = {da, -conj(db), db, conj(da)};
    cplx pw[4][ORACLE_MAX_TWOJ + 1];
    for (int f = 0; f < 4; f++) {
        pw[f][0] = 1.0;
        for (int i = 1; i <= J; i++) pw[f][i] = pw[f][i - 1] * g[f];
    }
    for (int mp = 0; mp <= J; mp++)
        for (int m = 0; m <= J; m++) {
            cplx s = 0.0;
            for (int k = 0; k <= m; k++) {
                int l = mp - k;
                if (l < 0 || l > J - m) continue;
                int e[4] = {k, m - k, l, J - m - l};    /* exponents of g00 g01 g10 g11 */
                cplx term = 0.0;
                for (int f = 0; f < 4; f++) {
                    if (e[f] == 0) continue;
                    cplx t = (double)e[f] * pw[f][e[f] - 1] * dg[f];
                    for (int h = 0; h < 4; h++)
                        if (h != f) t *= pw[h][e[h]];
                    term += t;
                }
                s += binom(m, k) * binom(J - m, l) * term;
            }
            double nrm = sqrt(fact(mp) * fact(J - mp) / (fact(m) * fact(J - m)));
            dD[mp * (J + 1) + m] = nrm * s;
        }
}

/* T(X, Y, W)[t] = Re sum_{m,m'} conj(W^j[m,m']) sum CG CG X^{j1}[m1,m1'] Y^{j2}[m2,m2'], full sums (b_from_u with three arrays) */
static void b_trilinear(const cgcache_t *cg, const cplx *X, const cplx *Y, const cplx *W, double *out)
{
    for (int t = 0; t < cg->n; t++) {
        int J1 = cg->tr[3 * t], J2 = cg->tr[3 * t + 1], J = cg->tr[3 * t + 2];
        const cplx *U1 = X + uoff(J1), *U2 = Y + uoff(J2), *UJ = W + uoff(J);
        const double *C = cg->tab[t];
        int sh = (J1 + J2 - J) / 2;
        cplx acc = 0.0;
        for (int m = 0; m <= J; m++)
            for (int mp = 0; mp <= J; mp++) {
                cplx z = 0.0;
                for (int m1 = 0; m1 <= J1; m1++) {
                    int m2 = m + sh - m1;
                    if (m2 < 0 || m2 > J2) continue;
                    double c1 = C[m1 * (J2 + 1) + m2];
                    for (int m1p = 0; m1p <= J1; m1p++) {
                        int m2p = mp + sh - m1p;
                        if (m2p < 0 || m2p > J2) continue;
                        double c2 = C[m1p * (J2 + 1) + m2p];
                        z += c1 * c2 * U1[m1 * (J1 + 1) + m1p] * U2[m2 * (J2 + 1) + m2p];
                    }
                }
                acc += conj(UJ[m * (J + 1) + mp]) * z;
            }
        out[t] = creal(acc);
    }
}

/* dB at explicit points.  dB_out (optional) [npoints][natoms][3][ncomp]; beta (optional) [npoints][ncomp] and
 * g_out [natoms][3] = sum_p sum_t beta[p][t] dB[p][alpha][k][t]  (Eq. (45): "apply dB/dR_alpha to an array"). */
int oracle_bispectrum_grad_points(int twojmax, double rcutfac, double rfac0, double rmin0, double wself, int ntypes, const double *radelem,
                                  const double *wj, int natoms, const double *pos, const int *types, const double *box,
                                  const double *origin, const int *pbc, int npoints, const double *points, double *dB_out,
                                  const double *beta, double *g_out)
{
    if (twojmax < 0 || twojmax > ORACLE_MAX_TWOJ) return -1;
    tables_init();
    sys_t s = {twojmax, rcutfac, rfac0, rmin0, wself, ntypes, radelem, wj, natoms, pos, types, box, origin, pbc, NULL, {0, 0, 0}, 0.0};
    if (sys_prepare(&s)) return -1;
    int nt = oracle_ntriples(twojmax);
    int *tr = (int *)malloc(sizeof(int) * 3 * nt);
    oracle_triples(twojmax, tr);
    cgcache_t cg;
    cg_build(&cg, nt, tr);
    int usz = uoff(twojmax + 1);
    const double *a1 = box, *a2 = box + 3, *a3 = box + 6;
    if (g_out)
        for (int i = 0; i < 3 * natoms; i++) g_out[i] = 0.0;
#pragma omp parallel
    {
        cplx *U = (cplx *)malloc(sizeof(cplx) * usz);
        cplx *dU = (cplx *)malloc(sizeof(cplx) * usz * 3);
        cplx *D = (cplx *)malloc(sizeof(cplx) * (twojmax + 1) * (twojmax + 1));
        cplx *dD = (cplx *)malloc(sizeof(cplx) * (twojmax + 1) * (twojmax + 1));
        double *t1 = (double *)malloc(sizeof(double) * nt * 3), *gl = (double *)calloc(3 * (natoms > 0 ? natoms : 1), sizeof(double));
#pragma omp for schedule(dynamic, 1)
        for (int p = 0; p < npoints; p++) {
            const double *rp = points + 3 * p;
            utot_point(&s, rp, U, D, NULL, 0);
            for (int n = 0; n < natoms; n++) {
                int t = types[n];
                double rcut = 2.0 * rcutfac * radelem[t], w = wj[t];
                for (int i = 0; i < 3 * usz; i++) dU[i] = 0.0;
                int hits = 0;
                for (int n1 = -s.nimg[0]; n1 <= s.nimg[0]; n1++)
                    for (int n2 = -s.nimg[1]; n2 <= s.nimg[1]; n2++)
                        for (int n3 = -s.nimg[2]; n3 <= s.nimg[2]; n3++) {
                            double d[3];
                            for (int k = 0; k < 3; k++) d[k] = s.wpos[3 * n + k] + n1 * a1[k] + n2 * a2[k] + n3 * a3[k] - rp[k];
                            cplx a, b, da[3], db[3];
                            double fc, dfc[3];
                            if (!pair_grad(d, rcut, rfac0, rmin0, &a, &b, &fc, da, db, dfc)) continue;
                            hits++;
                            for (int J = 0; J <= twojmax; J++) {
                                wigner_D(J, a, b, D);
                                for (int k = 0; k < 3; k++) {
                                    wigner_dD(J, a, b, da[k], db[k], dD);
                                    cplx *dUJ = dU + (size_t)k * usz + uoff(J);
                                    for (int i = 0; i < (J + 1) * (J + 1); i++) dUJ[i] += w * (dfc[k] * D[i] + fc * dD[i]);
                                }
                            }
                        }
                double *dst = dB_out ? dB_out + (((size_t)p * natoms + n) * 3) * nt : NULL;
                if (!hits) {
                    if (dst) for (int i = 0; i < 3 * nt; i++) dst[i] = 0.0;
                    continue;
                }
                for (int k = 0; k < 3; k++) {
                    const cplx *dUk = dU + (size_t)k * usz;
                    b_trilinear(&cg, dUk, U, U, t1);
                    b_trilinear(&cg, U, dUk, U, t1 + nt);
                    b_trilinear(&cg, U, U, dUk, t1 + 2 * nt);
                    double acc = 0.0;
                    for (int i = 0; i < nt; i++) {
                        double v = t1[i] + t1[nt + i] + t1[2 * nt + i];
                        if (dst) dst[k * nt + i] = v;
                        if (beta) acc += beta[(size_t)p * nt + i] * v;
                    }
                    gl[3 * n + k] += acc;
                }
            }
        }
        if (g_out) {
#pragma omp critical
            for (int i = 0; i < 3 * natoms; i++) g_out[i] += gl[i];
        }
        free(U); free(dU); free(D); free(dD); free(t1); free(gl);
    }
    cg_free(&cg);
    free(tr);
    free(s.wpos);
    return 0;
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    omp_set_num_threads(n);
#else
    (void)n;
#endif
}
